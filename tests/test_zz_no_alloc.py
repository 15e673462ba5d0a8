"""-m gpu: gadep_trace_rays_static -- the ray cast for callers that must not allocate (scratch in a file-scope static
device array of libgadep.so, at most GADEP_STATIC_MAX_RAYS rays per call) -- against the existing gadep_trace_rays.

Collected last on purpose (the suite runs with pytest -x).  The two paths launch the same kernel on the same hierarchy,
so the bar is the one the other ray tests use for two traversals of one mesh: facet index and distance bit for bit
(tests/test_gpu_acceptance.py::test_compressed_wide_nodes_give_the_same_hits).  Two calls in a row with different rays
show that nothing of the first call's scratch contents (ray-fetch counter, work counters, staged rays and results)
leaks into the second.  Runs alone in a fresh process or after the other tests.
"""
import numpy as np
import pytest

import detmesh as dm
from detmesh.configs import make_rays

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2605_25963_b200 as pkg
    w = dm.make_config(1)
    g = pkg.Gadep(0)
    g.load_workload(w)
    return pkg, w, g


def _rays(n, seed):
    # the recipe of the other ray tests: isotropic rays from uniform points in the bounding cylinder of the endcap
    return make_rays(n, seed, 41.9, -101.9, 6.0)


def test_static_scratch_ray_cast_equals_the_allocating_path_twice_in_a_row(ctx):
    import torch
    from paper_2605_25963_b200.binding import STATIC_MAX_RAYS
    pkg, w, g = ctx
    # two calls in a row: different rays, different counts (the second smaller, so stale staging lies behind it),
    # one with a from-side material filter and a negative window
    calls = [(200_000, 11, pkg.FILTER_NONE, 0.0), (77_777, 12, 1, -1e-4)]
    for n, seed, filt, t_min in calls:
        assert n <= STATIC_MAX_RAYS
        org, d = _rays(n, seed)
        # HOST arrays: staged in the static array
        tri_s, t_s = g.trace_rays_static(org, d, filter_material=filt, t_min=t_min)
        cs = g.get_counters()
        tri_a, t_a = g.trace_rays(org, d, filter_material=filt, t_min=t_min)
        ca = g.get_counters()
        assert np.array_equal(tri_s, tri_a)
        assert np.array_equal(t_s.view(np.uint32), t_a.view(np.uint32))
        assert (tri_a >= 0).sum() > 0.5 * n                     # the comparison is not about empty results
        assert cs["n_queries"] == ca["n_queries"] == n          # the counters started at zero, not at the last call's
        # the order in which warps fetch rays is free, the work per ray is not
        assert cs["n_box_tests"] == ca["n_box_tests"] and cs["n_tri_tests"] == ca["n_tri_tests"]
        # DEVICE arrays: only the two counters live in the static array
        to, td = torch.from_numpy(org).cuda(), torch.from_numpy(d).cuda()
        tri_d = torch.full((n,), -7, dtype=torch.int32, device="cuda")
        t_d = torch.full((n,), -7.0, dtype=torch.float32, device="cuda")
        g.trace_rays_static(to, td, filter_material=filt, t_min=t_min, tri_out=tri_d, t_out=t_d)
        assert g.get_counters()["n_queries"] == n
        assert np.array_equal(tri_d.cpu().numpy(), tri_a)
        assert np.array_equal(t_d.cpu().numpy().view(np.uint32), t_a.view(np.uint32))


def test_static_scratch_ray_cast_does_not_allocate_and_rejects_oversize(ctx):
    import torch
    from paper_2605_25963_b200.binding import STATIC_MAX_RAYS
    pkg, w, g = ctx
    org, d = _rays(50_000, 13)
    g.trace_rays_static(org, d)                                  # the address of the array is resolved by now
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        g.trace_rays_static(org, d)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                        # device memory in use did not move
    # the maximum itself is accepted, one more is refused with a text that names the limit; nothing is launched
    n = STATIC_MAX_RAYS
    org, d = _rays(n + 1, 14)
    tri, t = g.trace_rays_static(org[:n], d[:n])
    ref, _ = g.trace_rays(org[:n], d[:n])
    assert np.array_equal(tri, ref)
    with pytest.raises(pkg.GadepError) as ei:
        g.trace_rays_static(org, d)
    assert ei.value.code == -3 and "GADEP_STATIC_MAX_RAYS" in str(ei.value)
    # empty input is a no-op, mixed memory spaces and a missing hierarchy are argument / order errors
    e3, e1 = np.empty((0, 3), np.float32), np.empty(0, np.float32)
    g.trace_rays_static(e3, e3, tri_out=np.empty(0, np.int32), t_out=e1)
    dev = torch.zeros((4, 3), dtype=torch.float32, device="cuda")
    with pytest.raises(pkg.GadepError) as ei:
        g.trace_rays_static(dev, dev, tri_out=np.empty(4, np.int32), t_out=np.empty(4, np.float32))
    assert ei.value.code == -3
    g2 = pkg.Gadep(0)
    with pytest.raises(pkg.GadepError) as ei:
        g2.trace_rays_static(org[:4], d[:4])
    assert ei.value.code == -2
