// gmapp_voxel.cuh -- sphere-world builder: point cloud -> workspace crop -> voxelise at pitch
// 2 r_O -> occupied-voxel centres = spheres of the sphere world S_W (Sec. IV-B; "voxelise
// at 2 r_O", Eq. 5), written straight into the context's packed sphere array: no host round trip.
//
// Deterministic and exact (integer work): a bitmap over the voxel grid is marked with atomicOr, then compacted in
// voxel-index order by a popcount scan, so the sphere list is the sorted list of occupied voxels and is bit-identical
// run to run and to the numpy oracle in tests/.  Two launches per build (mark, compact); HBM-bound: 12 bytes read per point.
//
//   voxel index  i_c = floor((p_c - lo_c) / pitch)  (FP32, IEEE division), kept if lo_c <= p_c < hi_c and i_c < dim_c
//   linear index v = (i_z * dim_y + i_y) * dim_x + i_x
//   sphere       centre_c = fma(i_c + 0.5, pitch, lo_c), radius pitch / 2
//
// Shares nothing with oracle/.  Compiled in gmapp.cu only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gmapp {

struct VoxelGrid {
    float lo[3], hi[3];
    float pitch;
    int dim[3];
    int n_words;          // bitmap words = ceil(dim_x dim_y dim_z / 32)
};

// voxel of a point, or -1 (outside the box, NaN, or beyond the last voxel of an axis)
__device__ __forceinline__ int vox_of_point(const float* __restrict__ pts, int i, const VoxelGrid& G) {
    const float x = pts[3 * size_t(i)], y = pts[3 * size_t(i) + 1], z = pts[3 * size_t(i) + 2];
    if (!(x >= G.lo[0] && x < G.hi[0] && y >= G.lo[1] && y < G.hi[1] && z >= G.lo[2] && z < G.hi[2])) return -1;   // NaN fails too
    const int ix = int(floorf(__fdiv_rn(x - G.lo[0], G.pitch)));
    const int iy = int(floorf(__fdiv_rn(y - G.lo[1], G.pitch)));
    const int iz = int(floorf(__fdiv_rn(z - G.lo[2], G.pitch)));
    if (ix >= G.dim[0] || iy >= G.dim[1] || iz >= G.dim[2]) return -1;
    return int((unsigned(iz) * G.dim[1] + iy) * G.dim[0] + ix);
}
__device__ __forceinline__ float4 vox_sphere(unsigned vox, const VoxelGrid& G) {
    const int ix = vox % G.dim[0], iy = (vox / G.dim[0]) % G.dim[1], iz = vox / (G.dim[0] * G.dim[1]);
    return make_float4(__fmaf_rn(float(ix) + 0.5f, G.pitch, G.lo[0]), __fmaf_rn(float(iy) + 0.5f, G.pitch, G.lo[1]),
                       __fmaf_rn(float(iz) + 0.5f, G.pitch, G.lo[2]), 0.5f * G.pitch);
}

// large grids (more than kVoxSmallWords bitmap words): mark the global bitmap directly
__global__ void k_vox_mark(const float* __restrict__ pts, int n, const __grid_constant__ VoxelGrid G, unsigned* bitmap) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int v = vox_of_point(pts, i, G);
    if (v < 0) return;
    // most points fall into a voxel that is already marked: test first (a stale 0 only costs a redundant atomic)
    const unsigned bit = 1u << (v & 31);
    if (!(__ldcg(&bitmap[v >> 5]) & bit)) atomicOr(&bitmap[v >> 5], bit);
}

// ---------------------------------------------------------------------------------------------
// Everything after the marking in ONE kernel: popcount scan of the bitmap (chained over blocks with decoupled
// look-back), emission of the spheres in voxel-index order into the float4 array AND the sphere-pair arrays of the
// packed kernels, the sentinel tail, the count -- and the bitmap and the scan state are left zeroed for the next build,
// so a build is two launches (mark, compact) with no memset.  Scan block b (ticket b < n_scan) owns bitmap words
// [1024 b, 1024 b + 1024); the blocks with later tickets are FILL helpers: they wait for the total and write the
// sentinel tail in parallel (one block filling 32768 slots alone took longer than everything else together).
//   state[b] = (status << 32) | value; status 0 = nothing yet, 1 = the block's own total, 2 = inclusive prefix
//   sync[0] = dynamic block id ticket (tickets are handed out in start order, so a block only ever waits for blocks
//   that are already running), sync[1] = finished blocks
// ---------------------------------------------------------------------------------------------
// ---------------------------------------------------------------------------------------------
// Small grids (<= kVoxSmallWords bitmap words = 262144 voxels; the paper's workspace at pitch 2 r_O = 4 cm is 15625): the
// whole build in ONE launch.  ncu showed where the time of the first version went: not into its seven launches but into
// k_vox_mark's global atomics -- a depth cloud marks a few hundred bitmap words from 8e5 points, ~3000 same-address
// atomics per word at L2 (78 us, 98 % stalled on long_scoreboard / drain).  Here every block marks a PRIVATE bitmap in
// shared memory (grid-stride over the points), writes its slice of the sentinel tail, ORs its non-zero words into the
// global bitmap (<= one atomic per word and block), and the block that finishes last scans the bitmap, emits the spheres
// in voxel-index order over the sentinels, writes the count and leaves the bitmap zeroed.
// ---------------------------------------------------------------------------------------------
constexpr int kVoxSmallWords = 8192;
__device__ __forceinline__ void vox_store_sphere(float4* sph, float4* pairs, int stride, int rank, float x, float y, float z, float r);

__global__ void __launch_bounds__(1024) k_vox_build_small(const float* __restrict__ pts, int n_points, const __grid_constant__ VoxelGrid G,
                                                          unsigned* bitmap, int* sync, int capacity, int n_fill,
                                                          float4* sph, float4* svel, float4* pairs, int stride,
                                                          int* count, int* count_out) {
    extern __shared__ unsigned sbits[];                      // [n_words] this block's bitmap; the last block: the merged one
    __shared__ int s[32];
    __shared__ int s_last;
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5, nw = G.n_words;
    for (int w = t; w < nw; w += 1024) sbits[w] = 0u;
    __syncthreads();
    for (int i = blockIdx.x * 1024 + t; i < n_points; i += gridDim.x * 1024) {
        const int v = vox_of_point(pts, i, G);
        if (v >= 0) {
            const unsigned bit = 1u << (v & 31);
            if (!(sbits[v >> 5] & bit)) atomicOr(&sbits[v >> 5], bit);
        }
    }
    // sentinel tail: every slot now, the last block writes the real spheres over the front of it afterwards
    for (int i = blockIdx.x * 1024 + t; i < n_fill; i += gridDim.x * 1024) {
        vox_store_sphere(sph, pairs, stride, i, kFar, kFar, kFar, 0.0f);
        svel[i] = make_float4(0, 0, 0, 0);
    }
    __syncthreads();
    for (int w = t; w < nw; w += 1024) {
        const unsigned m = sbits[w];
        if (m && (m & ~__ldcg(&bitmap[w]))) atomicOr(&bitmap[w], m);
    }
    __threadfence();
    __syncthreads();
    if (t == 0) s_last = (atomicAdd(&sync[1], 1) == int(gridDim.x) - 1) ? 1 : 0;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // the last block: thread t owns the contiguous words [t * per, t * per + per)
    const int per = (nw + 1023) / 1024;
    int mine = 0;
    for (int k = 0; k < per; ++k) {
        const int w = t * per + k;
        unsigned m = 0u;
        if (w < nw) { m = __ldcg(&bitmap[w]); if (m) bitmap[w] = 0u; }      // leave the bitmap clean for the next build
        if (w < nw) sbits[w] = m;
        mine += __popc(m);
    }
    int inc = mine;
    for (int off = 1; off < 32; off <<= 1) { int o = __shfl_up_sync(0xffffffffu, inc, off); if (lane >= off) inc += o; }
    if (lane == 31) s[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int ws = s[lane], wi = ws;
        for (int off = 1; off < 32; off <<= 1) { int o = __shfl_up_sync(0xffffffffu, wi, off); if (lane >= off) wi += o; }
        s[lane] = wi - ws;
        if (lane == 31) { *count = wi; if (count_out) *count_out = wi; sync[1] = 0; }
    }
    __syncthreads();
    int rank = s[wid] + inc - mine;
    for (int k = 0; k < per; ++k) {
        const int w = t * per + k;
        if (w >= nw) break;
        unsigned bits = sbits[w];
        while (bits) {
            const int bpos = __ffs(bits) - 1;
            bits &= bits - 1;
            if (rank < capacity) {
                const float4 c = vox_sphere((unsigned(w) << 5) + bpos, G);
                vox_store_sphere(sph, pairs, stride, rank, c.x, c.y, c.z, c.w);
            }
            ++rank;
        }
    }
}

__device__ __forceinline__ void vox_store_sphere(float4* sph, float4* pairs, int stride, int rank, float x, float y, float z, float r) {
    sph[rank] = make_float4(x, y, z, r);
    float* a = reinterpret_cast<float*>(pairs + (rank >> 1)) + (rank & 1);             // A = (cx0,cx1,cy0,cy1)
    float* b = reinterpret_cast<float*>(pairs + stride + (rank >> 1)) + (rank & 1);    // B = (cz0,cz1,-R0,-R1)
    a[0] = x; a[2] = y; b[0] = z; b[2] = -r;
}

__global__ void __launch_bounds__(1024) k_vox_compact(unsigned* __restrict__ bitmap, unsigned long long* state, int* sync,
                                                      const __grid_constant__ VoxelGrid G, int capacity, int n_fill, int n_scan,
                                                      float4* sph, float4* svel, float4* pairs, int stride,
                                                      int* count, int* count_out) {
    __shared__ int s[32];
    __shared__ int s_bid, s_base, s_last;
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
    if (t == 0) s_bid = atomicAdd(&sync[0], 1);
    __syncthreads();
    const int b = s_bid, nb = n_scan, n_all = gridDim.x;
    if (b >= nb) {                                           // fill helper: sentinel tail and zero velocities of its slice
        if (t == 0) {
            volatile unsigned long long* st = state;
            unsigned long long e;
            do { e = st[nb - 1]; } while ((e >> 32) != 2ull);
            s_base = int(unsigned(e));
        }
        __syncthreads();
        const int n = min(s_base, capacity), nh = n_all - nb, h = b - nb;
        for (int i = h * 1024 + t; i < n_fill; i += nh * 1024) {
            if (i >= n) vox_store_sphere(sph, pairs, stride, i, kFar, kFar, kFar, 0.0f);
            svel[i] = make_float4(0, 0, 0, 0);
        }
        __threadfence();
        __syncthreads();
        if (t == 0) s_last = (atomicAdd(&sync[1], 1) == n_all - 1) ? 1 : 0;
        __syncthreads();
        if (s_last) {
            for (int j = t; j < nb; j += 1024) state[j] = 0ull;
            if (t == 0) { *count = s_base; if (count_out) *count_out = s_base; sync[0] = 0; sync[1] = 0; }
        }
        return;
    }
    const int w = b * 1024 + t;
    unsigned bits = 0u;
    if (w < G.n_words) { bits = bitmap[w]; if (bits) bitmap[w] = 0u; }                  // leave the bitmap clean for the next build
    const int v = __popc(bits);
    int inc = v;
    for (int off = 1; off < 32; off <<= 1) { int o = __shfl_up_sync(0xffffffffu, inc, off); if (lane >= off) inc += o; }
    if (lane == 31) s[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int ws = s[lane], wi = ws;
        for (int off = 1; off < 32; off <<= 1) { int o = __shfl_up_sync(0xffffffffu, wi, off); if (lane >= off) wi += o; }
        s[lane] = wi - ws;                                   // exclusive warp offsets
        const int total = __shfl_sync(0xffffffffu, wi, 31);
        if (lane == 0) {
            // decoupled look-back: publish the block total, add up the predecessors' totals back to the first prefix
            volatile unsigned long long* st = state;
            if (b > 0) { st[b] = (1ull << 32) | unsigned(total); __threadfence(); }
            int base = 0;
            for (int j = b - 1; j >= 0; --j) {
                unsigned long long e;
                do { e = st[j]; } while ((e >> 32) == 0ull);
                base += int(unsigned(e));
                if ((e >> 32) == 2ull) break;
            }
            __threadfence();
            st[b] = (2ull << 32) | unsigned(base + total);
            s_base = base;
        }
    }
    __syncthreads();
    int rank = s_base + s[wid] + inc - v;
    while (bits) {
        const int bpos = __ffs(bits) - 1;
        bits &= bits - 1;
        if (rank < capacity) {
            const float4 c = vox_sphere((unsigned(w) << 5) + bpos, G);
            vox_store_sphere(sph, pairs, stride, rank, c.x, c.y, c.z, c.w);
        }
        ++rank;
    }
    // the block that finishes last (of all: scan blocks and fill helpers) writes the count and resets the scan state
    __threadfence();
    __syncthreads();
    if (t == 0) s_last = (atomicAdd(&sync[1], 1) == n_all - 1) ? 1 : 0;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    const int total = int(unsigned(reinterpret_cast<volatile unsigned long long*>(state)[nb - 1]));
    for (int j = t; j < nb; j += 1024) state[j] = 0ull;
    if (t == 0) { *count = total; if (count_out) *count_out = total; sync[0] = 0; sync[1] = 0; }
}

}  // namespace gmapp
