"""GPU test (-m gpu) of the allocation-free entry point gmapp_build_sphere_world_static (include/gmapp.h): the sphere-world
builder with its scratch (voxel bitmap + block counter) in a file-scope `static __device__` array instead of context
memory, for callers that cannot call cudaMalloc.  Its output is compared with the existing path's
(gmapp_build_sphere_world + gmapp_get_obstacles) -- bit for bit, the tolerance every sphere-world-builder test here uses
(integer / voxel-index work) -- on two calls in a row with DIFFERENT clouds, so stale scratch from the first call would
show in the second.

Named test_zz_* so that pytest collects it last (the suite runs with `pytest -x`); it passes alone in a fresh process and
after the other tests."""
import numpy as np
import pytest

from paper_2606_12579_b200 import scenes

pytestmark = pytest.mark.gpu


def _reference(api, ctx, d_pts, lo, hi, pitch, capacity):
    import torch
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda:0")
    out = torch.empty((capacity, 4), dtype=torch.float32, device="cuda:0")
    ctx.build_sphere_world(d_pts, lo, hi, pitch, capacity, d_count_out=cnt)
    ctx.get_obstacles(out, n=capacity)
    torch.cuda.synchronize()
    return out.cpu().numpy(), int(cnt.item())


def test_static_scratch_builder_matches_context_builder_twice():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_12579_b200 import api                    # raises if libgmapp.so is missing: no fallback
    capacity = 4096
    ctx = api.Context(max_agents=1, max_spheres=capacity)
    try:
        clouds = [scenes.depth_cloud(seed=0, n_points=200_000), scenes.depth_cloud(seed=3, n_points=50_001)]
        pitches = [0.04, 0.05]
        d_out = torch.full((capacity, 4), -1.0, dtype=torch.float32, device="cuda:0")
        d_cnt = torch.full((1,), -1, dtype=torch.int32, device="cuda:0")
        free_after = []
        for (pts, lo, hi), pitch in zip(clouds, pitches):
            d_pts = torch.from_numpy(pts).to("cuda:0")
            want, want_n = _reference(api, ctx, d_pts, lo, hi, pitch, capacity)
            d_out.fill_(-1.0); d_cnt.fill_(-1)
            api.build_sphere_world_static(d_pts, lo, hi, pitch, capacity, d_out, d_cnt)
            torch.cuda.synchronize()
            free_after.append(torch.cuda.mem_get_info()[0])
            got = d_out.cpu().numpy()
            assert int(d_cnt.item()) == want_n and 0 < want_n < capacity
            assert np.array_equal(got, want)                 # spheres in voxel-index order, then the sentinel tail
        assert want_n != _reference(api, ctx, torch.from_numpy(clouds[0][0]).to("cuda:0"), clouds[0][1], clouds[0][2], pitches[0], capacity)[1]
        # the second call allocated nothing (the first may have loaded the kernel's module lazily)
        assert free_after[0] - free_after[1] < (1 << 20)
        # capacity smaller than the number of occupied voxels: the tail is dropped, the count still says how many there were
        pts, lo, hi = clouds[0]
        d_pts = torch.from_numpy(pts).to("cuda:0")
        small = torch.empty((100, 4), dtype=torch.float32, device="cuda:0")
        api.build_sphere_world_static(d_pts, lo, hi, 0.04, 100, small, d_cnt)
        torch.cuda.synchronize()
        full, n_full = _reference(api, ctx, d_pts, lo, hi, 0.04, capacity)
        assert int(d_cnt.item()) == n_full > 100 and np.array_equal(small.cpu().numpy(), full[:100])
        # a grid beyond the static scratch (262 144 voxels) is refused with a clear error, nothing launched
        with pytest.raises(api.GmappError) as e:
            api.build_sphere_world_static(d_pts, lo, hi, 0.004, capacity, d_out, d_cnt)
        assert e.value.status == api.GMAPP_ECAPACITY and "static scratch" in str(e.value)
        with pytest.raises(api.GmappError) as e:
            api.build_sphere_world_static(d_pts, lo, hi, 0.04, 0, d_out, d_cnt)
        assert e.value.status == api.GMAPP_EINVAL
    finally:
        ctx.close()
