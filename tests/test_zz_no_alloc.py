"""dos_uncollided_static (include/dos.h): the ray trace for callers that cannot allocate device memory -- no context, no
workspace, the kernel's scratch in a static device array shared by all calls. Checked against the existing path
(dos_create + dos_uncollided) on two calls in a row with DIFFERENT problems, so that stale scratch contents of the first
call (a larger table, a set bad-material flag) would show in the second. Named test_zz_* so that pytest collects it last:
the suite runs with pytest -x. Self-contained: passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from parity import TOL_UNCOLLIDED

pytestmark = pytest.mark.gpu


def _existing_path(dos, p, source_index):
    import torch
    ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
    out = ctx.new_field()
    ctx.dos_uncollided(p["sources"][source_index], p["spectrum"], out)
    torch.cuda.synchronize()
    res = out.cpu().numpy().copy()
    ctx.close()
    return res


def _assert_same(got, ref, label):
    assert got.shape == ref.shape, label
    assert np.array_equal(got == 0.0, ref == 0.0), f"{label}: beam membership differs"
    for g in range(ref.shape[0]):
        peak = np.abs(ref[g]).max()
        m = np.abs(ref[g]) > 1e-6 * peak
        if m.any():
            err = (np.abs(got[g].astype(np.float64) - ref[g])[m] / np.abs(ref[g])[m]).max()
            assert err <= TOL_UNCOLLIDED, f"{label}: group {g} max rel {err:.3e}"


def test_static_scratch_ray_trace_equals_the_workspace_path_twice_in_a_row():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1811_12391_b200 import dos
    from paper_1811_12391_b200.inputs import make_problem
    dev = torch.device("cuda:0")
    # call 1: 19 groups (a large table), cone beam, heterogeneous phantom, ragged mesh; one voxel inside the beam gets an
    # id >= n_mat so that the bad-material flag is SET when call 2 starts
    pa = make_problem("config4", nx=37, ny=29, nz=11, voxel=1.2, n_iter=1, n_pos=3)
    # call 2: 4 groups, isotropic point source, another mesh: a smaller table over the same scratch
    pb = make_problem("config1")
    mat_a = torch.from_numpy(np.ascontiguousarray(pa["material"], dtype=np.uint8)).to(dev)
    mat_b = torch.from_numpy(np.ascontiguousarray(pb["material"], dtype=np.uint8)).to(dev)
    n_mat_a = pa["sigma_t"].shape[0]
    ref_a = _existing_path(dos, pa, 1)
    ref_b = _existing_path(dos, pb, 0)
    lit = np.argwhere(ref_a[0] > 0)
    assert len(lit) > 100, "the test problem must have voxels inside the beam"
    k, j, i = lit[len(lit) // 2]
    mat_a_bad = mat_a.clone()
    mat_a_bad[k, j, i] = n_mat_a                      # out of range
    out_a = torch.full((pa["n_group"],) + tuple(mat_a.shape), -1.0, dtype=torch.float32, device=dev)
    out_a2 = torch.full_like(out_a, -1.0)
    out_b = torch.full((pb["n_group"],) + tuple(mat_b.shape), -1.0, dtype=torch.float32, device=dev)
    flag_a = torch.full((1,), 7, dtype=torch.int32, device=dev)
    flag_a2 = torch.full((1,), 7, dtype=torch.int32, device=dev)
    flag_b = torch.full((1,), 7, dtype=torch.int32, device=dev)
    before = torch.cuda.memory_allocated(dev)
    # three calls back to back on one stream, nothing synchronised in between
    dos.dos_uncollided_static(pa["mesh"], mat_a, pa["sigma_t"], pa["sources"][1], pa["spectrum"], out_a, flag_a)
    dos.dos_uncollided_static(pa["mesh"], mat_a_bad, pa["sigma_t"], pa["sources"][1], pa["spectrum"], out_a2, flag_a2)
    dos.dos_uncollided_static(pb["mesh"], mat_b, pb["sigma_t"], pb["sources"][0], pb["spectrum"], out_b, flag_b)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated(dev) == before
    _assert_same(out_a.cpu().numpy(), ref_a, "call 1")
    _assert_same(out_b.cpu().numpy(), ref_b, "call 3 (after a call that set the flag and held a larger table)")
    assert int(flag_a.item()) == 0 and int(flag_a2.item()) == 1 and int(flag_b.item()) == 0, "bad-material flag must be per call"
    # the same kernel on the same table: not merely within tolerance
    assert np.array_equal(out_a.cpu().numpy(), ref_a) and np.array_equal(out_b.cpu().numpy(), ref_b)
    # away from the bad voxel's rays the second call equals the first
    a2 = out_a2.cpu().numpy()
    assert (a2 == ref_a).mean() > 0.9

    # beyond the stated maximum: a clear error, nothing launched
    G_big = 65
    with pytest.raises(dos.DosError) as ei:
        dos.dos_uncollided_static(pb["mesh"], mat_b, np.ones((2, G_big), np.float32), pb["sources"][0], np.ones(G_big, np.float32) / G_big,
                                  out_b, None)
    assert ei.value.status == -6 and "exceeds the static scratch" in str(ei.value)
    with pytest.raises(dos.DosError) as ei:
        dos.dos_uncollided_static(pb["mesh"], mat_b, np.ones((17, 4), np.float32), pb["sources"][0], pb["spectrum"], out_b, None)
    assert ei.value.status == -6
    # and the scratch still serves the next call
    out_b.fill_(-1.0)
    dos.dos_uncollided_static(pb["mesh"], mat_b, pb["sigma_t"], pb["sources"][0], pb["spectrum"], out_b, None)
    torch.cuda.synchronize()
    assert np.array_equal(out_b.cpu().numpy(), ref_b)
