"""FP64/integer CPU oracle of the sphere-world builder.  TEST INFRASTRUCTURE, NOT THE PRODUCT:
only tests/ may import it; it shares no code with paper_2606_12579_b200/csrc.

What it follows (Sec. IV-B: crop to the workspace, "voxelise at 2 r_O", voxel centres
= spheres of S_W, Eq. 5), written out plainly: keep the points inside the box, compute each point's
voxel index, take the set of occupied voxels, order it by linear voxel index, emit one sphere per voxel.

Where floating point decides an integer (the voxel index) both sides decide in FP32 (reading N3):
i = floor((p - lo) / pitch) with p, lo, pitch float32 and IEEE float32 subtraction and division.  The centre
lo + (i + 1/2) pitch is one fused multiply-add in FP32 on the device; here it is formed exactly in float64 (the
product of a 13-bit integer-and-a-half with a float32 and the sum with a float32 are exact in 53 bits for the sizes
allowed) and rounded once to float32, which is the same value.
Pins (tests/test_oracle_pins.py, P15): brute force with Python sets on tiny clouds, containment of every kept point in
its voxel's cube, idempotence on its own centres, count bounds."""
import numpy as np


def sphere_world_from_points(points, lo, hi, pitch):
    """points [n,3] float32 (NaN allowed); lo, hi [3]; pitch scalar.  Returns (xyzr [m,4] float32 in increasing linear
    voxel index, dims [3] int, linear indices [m] int64)."""
    p = np.ascontiguousarray(points, dtype=np.float32).reshape(-1, 3)
    lo32, hi32, h = np.asarray(lo, np.float32), np.asarray(hi, np.float32), np.float32(pitch)
    dims = np.maximum(1, np.ceil((hi32.astype(np.float64) - lo32.astype(np.float64)) / np.float64(h))).astype(np.int64)
    with np.errstate(invalid="ignore"):
        inside = np.all((p >= lo32) & (p < hi32), axis=1)                      # NaN compares false
        idx = np.floor((p - lo32) / h)                                        # float32 arithmetic throughout
    keep = inside & np.all(idx < dims, axis=1)
    ijk = idx[keep].astype(np.int64)
    lin = np.unique((ijk[:, 2] * dims[1] + ijk[:, 1]) * dims[0] + ijk[:, 0])
    ix, iy, iz = lin % dims[0], (lin // dims[0]) % dims[1], lin // (dims[0] * dims[1])
    c = lo32.astype(np.float64) + (np.stack([ix, iy, iz], axis=1) + 0.5) * np.float64(h)
    xyzr = np.concatenate([c, np.full((lin.size, 1), 0.5 * np.float64(h))], axis=1).astype(np.float32)
    return xyzr, dims, lin
