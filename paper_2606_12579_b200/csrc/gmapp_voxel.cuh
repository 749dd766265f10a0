// gmapp_voxel.cuh -- sphere-world builder: point cloud -> workspace crop -> voxelise at pitch
// 2 r_O -> occupied-voxel centres = spheres of the sphere world S_W (Sec. IV-B; "voxelise
// at 2 r_O", Eq. 5), written straight into the context's packed sphere array: no host round trip.
//
// Deterministic and exact (integer work): a bitmap over the voxel grid is marked with atomicOr, then compacted in
// voxel-index order by a three-kernel popcount scan, so the sphere list is the sorted list of occupied voxels and
// is bit-identical run to run and to the numpy oracle in tests/.  HBM-bound: 12 bytes read per point.
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

__global__ void k_vox_mark(const float* __restrict__ pts, int n, const __grid_constant__ VoxelGrid G, unsigned* bitmap) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float x = pts[3 * size_t(i)], y = pts[3 * size_t(i) + 1], z = pts[3 * size_t(i) + 2];
    if (!(x >= G.lo[0] && x < G.hi[0] && y >= G.lo[1] && y < G.hi[1] && z >= G.lo[2] && z < G.hi[2])) return;   // NaN fails too
    const int ix = int(floorf(__fdiv_rn(x - G.lo[0], G.pitch)));
    const int iy = int(floorf(__fdiv_rn(y - G.lo[1], G.pitch)));
    const int iz = int(floorf(__fdiv_rn(z - G.lo[2], G.pitch)));
    if (ix >= G.dim[0] || iy >= G.dim[1] || iz >= G.dim[2]) return;
    const unsigned v = (unsigned(iz) * G.dim[1] + iy) * G.dim[0] + ix;
    // most points fall into a voxel that is already marked: test first (a stale 0 only costs a redundant atomic), so
    // the atomics per word drop from thousands to a handful and the kernel stays bound by reading the points
    const unsigned bit = 1u << (v & 31);
    if (!(__ldcg(&bitmap[v >> 5]) & bit)) atomicOr(&bitmap[v >> 5], bit);
}

// block sums of popcounts: 1024 words per block
__global__ void __launch_bounds__(1024) k_vox_count(const unsigned* __restrict__ bitmap, int n_words, int* block_sums) {
    __shared__ int s[32];
    const int w = blockIdx.x * 1024 + threadIdx.x;
    int c = w < n_words ? __popc(bitmap[w]) : 0;
    for (int off = 16; off > 0; off >>= 1) c += __shfl_xor_sync(0xffffffffu, c, off);
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x < 32) {
        c = s[threadIdx.x];
        for (int off = 16; off > 0; off >>= 1) c += __shfl_xor_sync(0xffffffffu, c, off);
        if (threadIdx.x == 0) block_sums[blockIdx.x] = c;
    }
}

// exclusive scan of the block sums in place (n_blocks <= 1024, one block); total -> *count
__global__ void __launch_bounds__(1024) k_vox_scan(int* block_sums, int n_blocks, int* count) {
    __shared__ int s[32];
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
    const int v = t < n_blocks ? block_sums[t] : 0;
    int inc = v;
    for (int off = 1; off < 32; off <<= 1) { int o = __shfl_up_sync(0xffffffffu, inc, off); if (lane >= off) inc += o; }
    if (lane == 31) s[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int ws = s[lane], wi = ws;
        for (int off = 1; off < 32; off <<= 1) { int o = __shfl_up_sync(0xffffffffu, wi, off); if (lane >= off) wi += o; }
        s[lane] = wi - ws;                                  // exclusive warp offsets
        if (lane == 31) *count = wi;
    }
    __syncthreads();
    if (t < n_blocks) block_sums[t] = s[wid] + inc - v;
}

// emit the spheres of the occupied voxels in voxel-index order; ranks >= capacity are dropped
__global__ void __launch_bounds__(1024) k_vox_emit(const unsigned* __restrict__ bitmap, const int* __restrict__ block_off,
                                                   const __grid_constant__ VoxelGrid G, int capacity, float4* sph) {
    __shared__ int s[32];
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
    const int w = blockIdx.x * 1024 + t;
    unsigned bits = w < G.n_words ? bitmap[w] : 0u;
    const int v = __popc(bits);
    int inc = v;
    for (int off = 1; off < 32; off <<= 1) { int o = __shfl_up_sync(0xffffffffu, inc, off); if (lane >= off) inc += o; }
    if (lane == 31) s[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int ws = s[lane], wi = ws;
        for (int off = 1; off < 32; off <<= 1) { int o = __shfl_up_sync(0xffffffffu, wi, off); if (lane >= off) wi += o; }
        s[lane] = wi - ws;
    }
    __syncthreads();
    int rank = block_off[blockIdx.x] + s[wid] + inc - v;
    const float r = 0.5f * G.pitch;
    while (bits) {
        const int b = __ffs(bits) - 1;
        bits &= bits - 1;
        if (rank < capacity) {
            const unsigned vox = (unsigned(w) << 5) + b;
            const int ix = vox % G.dim[0], iy = (vox / G.dim[0]) % G.dim[1], iz = vox / (G.dim[0] * G.dim[1]);
            sph[rank] = make_float4(__fmaf_rn(float(ix) + 0.5f, G.pitch, G.lo[0]), __fmaf_rn(float(iy) + 0.5f, G.pitch, G.lo[1]),
                                    __fmaf_rn(float(iz) + 0.5f, G.pitch, G.lo[2]), r);
        }
        ++rank;
    }
}

// slots [min(count, capacity), n_fill) become sentinels (far away, never gated, never the minimum); velocities zero
__global__ void k_vox_fill(const int* __restrict__ count, int capacity, int n_fill, float4* sph, float4* svel) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_fill) return;
    const int n = min(*count, capacity);
    if (i >= n) sph[i] = make_float4(kFar, kFar, kFar, 0.0f);
    svel[i] = make_float4(0, 0, 0, 0);
}

}  // namespace gmapp
