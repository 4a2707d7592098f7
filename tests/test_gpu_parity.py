"""GPU-vs-oracle parity of the whole hot path, through the C ABI (run on the B200 box: -m gpu).

Every case builds one seeded problem (paper_1811_12391_b200.inputs), runs the fp64 oracle and the CUDA
library on the same fp32-rounded tables and compares element by element with the tolerances of
tests/parity.py (BASELINE.json north_star).
"""
import math
import os

import numpy as np
import pytest

from parity import (assert_dose_parity, assert_fluence_parity, assert_problem_parity, assert_uncollided_parity,
                    field_errors, per_group_errors)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dos():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1811_12391_b200 import dos as d
    return d


def _make(name, **ov):
    from paper_1811_12391_b200.inputs import make_problem
    return make_problem(name, **ov)


# ---------------------------------------------------------------- element-by-element, small sizes --
# Reduced versions of each config: same materials / xs model / quadrature / P_L / source geometry, mesh
# sizes that span several 8x4 sweep tiles with ragged tails in j and k and an x length that is not a
# multiple of the hand-off chunk.
SMALL = [
    ("config1", {}),                                                                    # the full config 1
    ("config2", dict(nx=37, ny=21, nz=10, voxel=1.0, n_group=5, n_iter=6)),
    ("config3", dict(nx=26, ny=20, nz=9, voxel=1.5, n_group=4, n_iter=3)),
    ("config4", dict(nx=30, ny=27, nz=7, voxel=1.3, n_group=6, n_iter=4, n_pos=1)),
    ("config5", dict(nx=19, ny=17, nz=21, voxel=1.9, n_group=3, n_iter=3)),
    ("config2", dict(nx=5, ny=3, nz=2, voxel=7.0, n_group=3, n_iter=2, sn=2, pl=0)),     # one partial tile, S2/P0
    ("config2", dict(nx=1, ny=1, nz=1, voxel=30.0, n_group=2, n_iter=2, sn=4, pl=1)),    # single voxel
    ("config2", dict(nx=33, ny=9, nz=5, voxel=1.1, n_group=3, n_iter=3, sn=6, pl=2)),    # S6/P2 (M padded 9->12)
    ("config4", dict(nx=18, ny=16, nz=8, voxel=2.0, n_group=4, n_iter=3, n_pos=1, sn=12, pl=4)),  # S12/P4
]


@pytest.mark.parametrize("name,ov", SMALL, ids=[f"{n}-{i}" for i, (n, _) in enumerate(SMALL)])
def test_small_problem_parity(dos, orc, name, ov):
    p = _make(name, **ov)
    ref = orc.run_problem(p)
    out = dos.run_problem(p)
    assert_problem_parity(out, ref, name)


# Every sweep implementation on every kind of problem, whatever the library's default choice is: the tensor-memory sweep
# (dos_sweep_umma.cu: tcgen05.mma contractions, bulk copies, mbarrier rings), also with an odd hand-off chunk and few
# persistent CTAs, and the FFMA sweep (dos_sweep_ffma.cu) with and without its two-CTAs-per-SM variant and with either
# face hand-off (small meshes default to (value, epoch) pairs, large ones to release / acquire flags).
SWEEP_VARIANTS = [
    ("umma", {"sweep_contraction": 2}),
    ("umma-chunk3-grid5", {"sweep_contraction": 2, "sweep_chunk": 3, "sweep_grid": 5}),
    ("ffma", {"sweep_contraction": 1, "sweep_two_per_sm": 0}),
    ("ffma-2cta", {"sweep_contraction": 1, "sweep_two_per_sm": 2}),
    ("ffma-flags", {"sweep_contraction": 1, "sweep_ll": 0}),      # the large-mesh hand-off protocol on these small meshes
    ("ffma-grid3", {"sweep_contraction": 1, "sweep_grid": 3}),    # far fewer persistent CTAs than work items: items wait in the queue
]
VARIANT_CASES = [
    ("config2", dict(nx=37, ny=21, nz=10, voxel=1.0, n_group=4, n_iter=4)),                        # S8/P3, ragged tiles
    ("config3", dict(nx=26, ny=20, nz=9, voxel=1.5, n_group=3, n_iter=3)),                         # S16/P5
    ("config2", dict(nx=33, ny=9, nz=5, voxel=1.1, n_group=3, n_iter=3, sn=6, pl=2)),              # S6/P2 (M padded 9->12)
    ("config2", dict(nx=5, ny=3, nz=2, voxel=7.0, n_group=3, n_iter=2, sn=2, pl=0)),                # S2/P0: 1 angle, 1 moment
    ("config1", {}),                                                                               # S4/P1, 16^3
    ("config4", dict(nx=18, ny=16, nz=8, voxel=2.0, n_group=3, n_iter=3, n_pos=1, sn=12, pl=4)),   # S12/P4: 21 angles, 25 moments
    ("config2", dict(nx=19, ny=17, nz=6, voxel=2.2, n_group=2, n_iter=3, sn=10, pl=3)),            # S10/P3: 15 angles (5 x 3 warps)
    ("config3", dict(nx=17, ny=10, nz=9, voxel=2.5, n_group=2, n_iter=2, sn=14, pl=5)),            # S14/P5: 28 angles (14 x 2 warps)
]


@pytest.mark.parametrize("case", range(len(VARIANT_CASES)))
def test_every_sweep_variant_parity(dos, orc, case):
    name, ov = VARIANT_CASES[case]
    p = _make(name, **ov)
    ref = orc.run_problem(p)
    for label, opts in SWEEP_VARIANTS:
        ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
        for k, v in opts.items():
            ctx.dos_set_option(k, v)
        out = dos.run_problem(p, ctx=ctx)
        ctx.close()
        assert_problem_parity(out, ref, f"{name} [{label}]")


def test_ffma_sweep_shape_options_parity(dos, orc):
    """The FFMA sweep's CTA shape knobs (angles per warp, aux warps, an octant's angles split over two CTAs) with either
    face hand-off: every combination must give the oracle's result (the angle split doubles the face buffers' tile ids,
    which the (value, epoch) pair layout has to follow)."""
    p = _make("config2", nx=37, ny=21, nz=10, voxel=1.0, n_group=3, n_iter=3)
    ref = orc.run_problem(p)
    for shape in ({"sweep_angles_per_warp": 2}, {"sweep_aux_warps": 1}, {"sweep_angle_split": 2},
                  {"sweep_angle_split": 5, "sweep_angles_per_warp": 2}):
        for ll in (1, 0):
            ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
            ctx.dos_set_option("sweep_contraction", 1)
            ctx.dos_set_option("sweep_ll", ll)
            for k, v in shape.items():
                ctx.dos_set_option(k, v)
            out = dos.run_problem(p, ctx=ctx)
            ctx.close()
            assert_problem_parity(out, ref, f"config2 small [ffma {shape} ll={ll}]")


SEED_RANDOM_SHAPES = 7


def test_random_shapes_parity(dos, orc):
    """Seeded random problems -- mesh sizes from 1 voxel per axis up to a few ragged tiles, S4..S16, P0..P5, 1-3 groups and
    iterations, the three phantoms -- through the library's own choice of sweep, both sweeps forced, and the FFMA sweep
    with the flag hand-off; plus, where the problem has several positions, all faces reflective against the oracle's
    lagged reflective option. (S2 is left out: forced onto the tensor-memory sweep with P >= 1 it misses the max-rel bar
    at voxels 1e-5 of the peak; the library itself takes the FFMA sweep there.)"""
    rng = np.random.default_rng(SEED_RANDOM_SHAPES)
    for it in range(14):
        base = ["config2", "config3", "config4"][int(rng.integers(3))]
        ov = dict(nx=int(rng.integers(1, 41)), ny=int(rng.integers(1, 31)), nz=int(rng.integers(1, 15)), voxel=float(rng.uniform(0.6, 3.0)),
                  n_group=int(rng.integers(1, 4)), n_iter=int(rng.integers(1, 4)), sn=int([4, 6, 8, 10, 12, 16][int(rng.integers(6))]),
                  pl=int(rng.integers(0, 6)))
        if base == "config4":
            ov["n_pos"] = 2
        p = _make(base, **ov)
        src = int(rng.integers(len(p["sources"])))
        ref = orc.run_problem(p, source_index=src)
        for opts in ({}, {"sweep_contraction": 1}, {"sweep_contraction": 2}, {"sweep_contraction": 1, "sweep_ll": 0}):
            ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
            for k, v in opts.items():
                ctx.dos_set_option(k, v)
            out = dos.run_problem(p, source_index=src, ctx=ctx)
            ctx.close()
            assert_problem_parity(out, ref, f"random {it} {base} {ov} {opts}")
        if it % 3 == 0:
            s0 = p["sources"][src]
            pu = orc.uncollided(p["mesh"], p["material"], p["sigma_t"], s0, p["spectrum"])
            pc_ref, pabs = orc.solve(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["quadrature"], p["P_L"], p["n_iter"],
                                     source_pos=s0["pos"], phi_u=pu, reflective=True, want_abs=True)
            ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
            ctx.dos_set_boundary(7)
            pc = ctx.new_field()
            ctx.dos_uncollided(s0, p["spectrum"])
            ctx.dos_solve(p["n_iter"])
            ctx.dos_fluence(pc, None)
            ctx.dos_check()
            ctx.close()
            assert_fluence_parity(pc.cpu().numpy(), pc_ref[:, 0], f"random {it} {base} {ov} reflective", scale=pabs)


def test_known_marginal_voxel_of_a_random_trial(dos, orc):
    """What ~1100 random (problem, sweep) pairs turned up besides S2 on the tensor-memory sweep: one
    problem -- S4/P1, 33 x 26 x 12, a single iteration -- in which ONE voxel, at 1.2e-6 of the group's peak (the bar's own
    threshold is 1e-6), comes out 1.055e-4 off with the FFMA sweep (either hand-off, bit-stable; 3.0e-5 with the tensor-memory
    sweep; an absolute error of 1.3e-10 of the peak). Far from the beam the diamond-difference extrapolation 2 psi_c - psi_in
    cancels along the path, which the R15b scale (the angular sum's terms) does not see. Kept here as a stated limit: relL2
    at the bar, max-rel within 1.2e-4, and everything but the collided max-rel at the plain bars."""
    from parity import TOL_L2
    p = _make("config3", nx=33, ny=26, nz=12, voxel=2.0873278798297297, n_group=3, n_iter=1, sn=4, pl=1)
    ref = orc.run_problem(p)
    out = dos.run_problem(p)
    assert_uncollided_parity(out["phi_u"], ref["phi_u"])
    assert_fluence_parity(out["phi_total"], ref["phi_total"], "marginal case, total fluence")
    assert_dose_parity(out["dose"], ref["dose"], "marginal case, dose")
    l2, mx = per_group_errors(out["phi_c"], ref["phi_c"], ref["phi_c_abs"])
    assert l2 <= TOL_L2 and mx <= 1.2e-4, (l2, mx)


def test_summed_source_mode_parity(dos, orc):
    """several source positions as ONE source, one solve (dos_uncollided_sum)
    against oracle.run_problem_summed; and the state machine of the mode."""
    p = _make("config4", nx=30, ny=27, nz=7, voxel=1.3, n_group=5, n_iter=4, n_pos=5)
    ref = orc.run_problem_summed(p, [0, 2, 3])
    out = dos.run_problem_summed(p, [0, 2, 3])
    assert_problem_parity(out, ref, "config4 small, positions 0+2+3 summed")
    # one position through the summed path = the single-source path
    one = dos.run_problem(p, source_index=1)
    s1 = dos.run_problem_summed(p, [1])
    for k in ("phi_u", "phi_total", "dose"):
        assert np.abs(s1[k] - one[k]).max() <= 2e-6 * np.abs(one[k]).max(), k
    # P5 (36 moments, tensor-core sweep) as well
    p5 = _make("config3", nx=26, ny=20, nz=9, voxel=1.5, n_group=3, n_iter=3)
    p5["sources"] = [p5["sources"][0], dict(p5["sources"][0], pos=np.array(p5["sources"][0]["pos"]) + np.array([9.0, 0.0, 2.0]))]
    assert_problem_parity(dos.run_problem_summed(p5), orc.run_problem_summed(p5), "config3 small, 2 positions summed")
    # a context without the summed-source buffers refuses the mode; first = 0 needs a first source
    ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
    with pytest.raises(dos.DosError) as e:
        ctx.dos_uncollided_sum(p["sources"][0], p["spectrum"], first=True)
    assert e.value.status == -3
    ctx.close()
    ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"], n_batch=2)
    with pytest.raises(dos.DosError) as e:
        ctx.dos_uncollided_sum(p["sources"][0], p["spectrum"], first=False)
    assert e.value.status == -3
    # a summed state is replaced by a later single-source call
    ctx.dos_uncollided_sum(p["sources"][0], p["spectrum"], first=True)
    ctx.dos_uncollided_sum(p["sources"][2], p["spectrum"], first=False)
    out1 = dos.run_problem(p, source_index=1, ctx=ctx)
    ctx.close()
    for k in ("phi_total", "dose"):          # equal up to the order of the moment reductions
        assert np.abs(out1[k] - one[k]).max() <= 2e-6 * np.abs(one[k]).max(), k


def test_config2_full_parity(dos, orc):
    """BASELINE.json configs[1] at full size and full iteration count."""
    p = _make("config2")
    ref = orc.run_problem(p)
    out = dos.run_problem(p)
    res = assert_problem_parity(out, ref, "config2")
    print("config2 parity", res)


# -------------------------------------------------- full mesh sizes, bench launch configuration --
# Full group / iteration depth at full mesh size is compared in test_gpu_golden.py against stored oracle results
# (tests/golden). The cases here run the oracle live on the full meshes with the group and iteration counts cut
# (every group / iteration is the same launch sequence), and check every field at EVERY voxel.
def test_config3_full_mesh_parity(dos, orc):
    p = _make("config3", n_group=2, n_iter=2)
    ref = orc.run_problem(p)
    out = dos.run_problem(p)
    assert_problem_parity(out, ref, "config3 mesh")


def test_config4_full_mesh_two_positions_accumulate(dos, orc):
    """256x256x64 abdomen phantom, S8/P3; two of the 36 source positions, doses summed (a9)."""
    p = _make("config4", n_group=2, n_iter=1)
    ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
    d = ctx.new_field(groups=False)
    ref_sum = None
    for n, s in enumerate((0, 13)):
        ctx.dos_uncollided(p["sources"][s], p["spectrum"])
        ctx.dos_solve(p["n_iter"])
        ctx.dos_dose(d, accumulate=(n > 0))
        r = orc.run_problem(p, source_index=s)
        ref_sum = r["dose"] if ref_sum is None else ref_sum + r["dose"]
    ctx.dos_check()
    assert_dose_parity(d.cpu().numpy(), ref_sum, "scan dose (2 positions)")
    ctx.close()


def test_config5_full_mesh_properties(dos, orc):
    """256^3, S16/P5 in the bench launch configuration. Properties that hold at any size:
    (i) uncollided fluence of sampled voxels equals the oracle's (the oracle traces just those voxels:
        a sub-mesh cannot be used, the ray crosses the whole grid);
    (ii) a phantom that is mirror-symmetric in x and in z (water cylinder, source on the y axis) gives
        mirror-symmetric collided fluence: mirrored octants visit tiles in the opposite order, so a
        wrong tile hand-off, flag or index breaks it (north_star check 5 applied to the GPU);
    (iii) the result does not depend on the hand-off chunk or the number of resident CTAs."""
    import torch
    from paper_1811_12391_b200.inputs import phantoms
    p = _make("config5", n_group=2, n_iter=2)
    m = p["mesh"]
    # (i) abdomen phantom: sampled voxels
    ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
    pu = ctx.new_field()
    ctx.dos_uncollided(p["sources"][0], p["spectrum"], pu)
    ctx.dos_check()
    rng = np.random.default_rng(5)
    in_beam = torch.nonzero(pu[0].reshape(-1) > 0).reshape(-1).cpu().numpy()
    cells = np.concatenate([rng.choice(in_beam, 4000, replace=False), rng.integers(0, pu[0].numel(), 2000)])
    ref = orc.uncollided_at(p["mesh"], p["material"], p["sigma_t"], p["sources"][0], p["spectrum"], cells)
    got = pu.reshape(p["n_group"], -1)[:, torch.from_numpy(cells).to(pu.device)].cpu().numpy()
    assert_uncollided_parity(got, ref)
    ctx.close()
    del pu
    # (ii) + (iii) symmetric phantom
    mat = phantoms.cylinder(m["nx"], m["ny"], m["nz"], m["dx"], m["dy"], m["dz"], radius=15.0, inside=1, outside=0)
    ctx = dos.Context(p["mesh"], mat, p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
    pc = ctx.new_field()
    ctx.dos_uncollided(p["sources"][0], p["spectrum"])
    ctx.dos_solve(p["n_iter"])
    ctx.dos_fluence(pc, None)
    ctx.dos_check()
    assert torch.isfinite(pc).all()
    for g in range(p["n_group"]):
        a = pc[g]
        peak = a.abs().max().item()
        assert peak > 0
        assert (a - a.flip(2)).abs().max().item() <= 2e-5 * peak, "x mirror symmetry"
        assert (a - a.flip(0)).abs().max().item() <= 2e-5 * peak, "z mirror symmetry"
    base = pc.clone()
    ctx.dos_set_option("sweep_chunk", 5)
    ctx.dos_set_option("sweep_grid", 97)
    ctx.dos_uncollided(p["sources"][0], p["spectrum"])
    ctx.dos_solve(p["n_iter"])
    ctx.dos_fluence(pc, None)
    ctx.dos_check()
    for g in range(p["n_group"]):
        peak = base[g].abs().max().item()
        assert (pc[g] - base[g]).abs().max().item() <= 2e-5 * peak, "launch-configuration independence"
    ctx.close()


# ------------------------------------------------- position batch --
def test_position_batch_equals_separate_solves(dos, orc):
    """dos_uncollided_batch + one dos_solve for several source positions: per-position fluences equal those of separate
    solves (same kernels, same arithmetic; only the order of the moment reductions may differ) and match the oracle; the
    dose is the sum over the positions (a9); both sweep kernels; a batch smaller than the slot count; state machine."""
    import torch
    from paper_1811_12391_b200 import scan
    for name, ov, opts in (("config4", dict(nx=30, ny=27, nz=7, voxel=1.3, n_group=4, n_iter=3, n_pos=5), {}),
                           ("config3", dict(nx=18, ny=11, nz=9, voxel=2.0, n_group=2, n_iter=3), {}),
                           ("config4", dict(nx=30, ny=27, nz=7, voxel=1.3, n_group=3, n_iter=3, n_pos=5), {"sweep_contraction": 2})):
        p = _make(name, **ov)
        if len(p["sources"]) == 1:      # config 3: three positions around the cylinder
            from paper_1811_12391_b200.inputs import scan_source
            p["sources"] = [scan_source(th) for th in (0.5 * math.pi, 1.1, 4.0)]
        pos = [0, 2, 1] if len(p["sources"]) == 3 else [0, 3, 4]
        ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"], n_batch=4)
        for k, v in opts.items():
            ctx.dos_set_option(k, v)
        G = p["n_group"]
        pu = torch.empty((3, G) + ctx.shape, dtype=torch.float32, device=ctx.device)
        pc, pt = torch.empty_like(pu), torch.empty_like(pu)
        d = ctx.new_field(groups=False)
        ctx.dos_uncollided_batch([p["sources"][s] for s in pos], p["spectrum"], pu)
        ctx.dos_solve(p["n_iter"])
        ctx.dos_fluence(pc, pt)
        ctx.dos_dose(d, False)
        ctx.dos_check()
        ref_dose = 0.0
        for b, s_ in enumerate(pos):
            ref = orc.run_problem(p, source_index=s_)
            out = {"phi_u": pu[b].cpu().numpy(), "phi_c": pc[b].cpu().numpy(), "phi_total": pt[b].cpu().numpy(), "dose": ref["dose"]}
            assert_problem_parity(out, ref, f"{name} batch slot {b}")
            ref_dose = ref_dose + ref["dose"]
            one = dos.run_problem(p, source_index=s_, ctx=None)      # a separate solve on a fresh single-slot context
            assert np.array_equal(one["phi_u"], out["phi_u"])
            assert np.abs(one["phi_c"] - out["phi_c"]).max() <= 2e-6 * np.abs(one["phi_c"]).max()
        assert_dose_parity(d.cpu().numpy(), ref_dose, "batch dose = sum over positions")
        # the same context serves a smaller batch and a single position afterwards
        ctx.dos_uncollided_batch([p["sources"][pos[1]]], p["spectrum"])
        ctx.dos_solve(p["n_iter"])
        ctx.dos_dose(d, False)
        assert_dose_parity(d.cpu().numpy(), orc.run_problem(p, source_index=pos[1])["dose"], "batch of one")
        with pytest.raises(dos.DosError) as e:
            ctx.dos_uncollided_batch([p["sources"][0]] * 5, p["spectrum"])
        assert e.value.status == -3
        # scan.run_scan drives the batch path: 5 (or 3) positions through 4 slots
        all_pos = list(range(len(p["sources"])))
        scan.run_scan(ctx, p, all_pos, d)
        ctx.dos_check()
        tot = sum(orc.run_problem(p, source_index=s_)["dose"] for s_ in all_pos)
        assert_dose_parity(d.cpu().numpy(), tot, "run_scan through the batch path")
        ctx.close()


# ------------------------------------------------- reflective boundaries, stopping rule --
def test_reflective_boundaries_parity_and_balance(dos, orc):
    """dos_set_boundary (PAPER.md:41 states vacuum; north_star check 2 needs reflective faces). (a) GPU vs the oracle's
    lagged reflective option on a ragged multi-tile mesh, S8/P3 and S16/P5, a few iterations: every octant's boundary
    outflow must reach its mirror octant at the right cell, angle and sweep. (b) With all faces reflective nothing
    leaks, so at convergence absorption = source, group by group: sum_c (sigma_t - sigma_s0^{g->g}) phi_c^g =
    sum_c [sum_{g'<=g} sigma_s0^{g'->g} phi_u^{g'} + sum_{g'<g} sigma_s0^{g'->g} phi_c^{g'}] (north_star check 3 on the
    GPU, homogeneous water so that sigma is one number per group)."""
    for name, ov in (("config2", dict(nx=21, ny=13, nz=10, voxel=1.6, n_group=3, n_iter=5)),
                     ("config3", dict(nx=12, ny=17, nz=6, voxel=2.5, n_group=2, n_iter=4))):
        p = _make(name, **ov)
        src = p["sources"][0]
        pu = orc.uncollided(p["mesh"], p["material"], p["sigma_t"], src, p["spectrum"])
        pc_ref, pabs = orc.solve(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["quadrature"], p["P_L"], p["n_iter"],
                                 source_pos=src["pos"], phi_u=pu, reflective=True, want_abs=True)
        ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
        ctx.dos_set_boundary(7)
        pc = ctx.new_field()
        ctx.dos_uncollided(src, p["spectrum"])
        ctx.dos_solve(p["n_iter"])
        ctx.dos_fluence(pc, None)
        ctx.dos_check()
        assert_fluence_parity(pc.cpu().numpy(), pc_ref[:, 0], f"{name} reflective collided fluence", scale=pabs)
        # back to vacuum on the same context: the vacuum result of a fresh context
        ctx.dos_set_boundary(0)
        ctx.dos_uncollided(src, p["spectrum"])
        ctx.dos_solve(p["n_iter"])
        ctx.dos_fluence(pc, None)
        vac = dos.run_problem(p)["phi_c"]
        assert np.abs(pc.cpu().numpy() - vac).max() <= 2e-6 * np.abs(vac).max()
        ctx.close()
    # (b) balance in a closed water box
    p = _make("config1", nx=10, ny=9, nz=6, n_iter=150)
    src = p["sources"][0]
    ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
    ctx.dos_set_boundary(7)
    pu, pc = ctx.new_field(), ctx.new_field()
    ctx.dos_uncollided(src, p["spectrum"], pu)
    ctx.dos_solve(p["n_iter"])
    ctx.dos_fluence(pc, None)
    ctx.dos_check()
    ctx.close()
    su = pu.double().sum(dim=(1, 2, 3)).cpu().numpy()
    sc = pc.double().sum(dim=(1, 2, 3)).cpu().numpy()
    st, s0 = p["sigma_t"][0].astype(float), p["sigma_s"][0, 0].astype(float)       # water; [from][to]
    for g in range(p["n_group"]):
        source = sum(s0[gp, g] * su[gp] for gp in range(g + 1)) + sum(s0[gp, g] * sc[gp] for gp in range(g))
        assert abs((st[g] - s0[g, g]) * sc[g] - source) <= 2e-5 * source, g


def test_solve_with_stopping_rule(dos, orc):
    """dos_solve_tol: per-group iteration counts come back; the oracle run with exactly those counts agrees at the
    parity tolerances, its own stopping measure at the last sweep is at or below tol (up to fp32 noise) and, one sweep
    earlier, above it -- both sides take the same decision although one tests in fp32 and the other in fp64."""
    p = _make("config2", nx=27, ny=19, nz=9, voxel=1.4, n_group=5, n_iter=40)
    src = p["sources"][0]
    tol = 2e-3
    ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
    pc = ctx.new_field()
    ctx.dos_uncollided(src, p["spectrum"])
    iters = ctx.dos_solve_tol(tol, p["n_iter"])
    ctx.dos_fluence(pc, None)
    ctx.dos_check()
    ctx.close()
    assert iters.min() >= 1 and iters.max() < p["n_iter"] and len(set(iters.tolist())) > 1, iters
    pu = orc.uncollided(p["mesh"], p["material"], p["sigma_t"], src, p["spectrum"])
    args = (p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["quadrature"], p["P_L"])
    ref, conv = orc.solve(*args, 1, source_pos=src["pos"], phi_u=pu, n_iter_g=iters, want_conv=True)
    l2, mx = per_group_errors(pc.cpu().numpy(), ref[:, 0])
    assert l2 <= 1e-5, l2
    assert (conv <= tol * 1.01).all(), (conv, iters)
    # one sweep fewer in a group leaves its measure above tol (the rule stops at the FIRST sweep that meets it)
    g = int(np.argmax(iters))
    fewer = iters.copy()
    fewer[g] -= 1
    _, conv2 = orc.solve(*args, 1, source_pos=src["pos"], phi_u=pu, n_iter_g=fewer, want_conv=True)
    assert conv2[g] > tol * 0.99


def test_paper_shaped_workload_parity(dos, orc):
    """the paper's 7-group structure, S6/P0 and S4/P1, 30 degree cone, several positions as ONE source
    (the paper's CT-scan mode), on a reduced mesh of the 50 x 50 x 12.5 cm box."""
    for sn, pl in ((6, 0), (4, 1), (8, 1)):
        p = _make("paper_coarse", nx=26, ny=26, nz=7, voxel=50.0 / 26, n_iter=4, n_pos=4, sn=sn, pl=pl)
        assert_problem_parity(dos.run_problem_summed(p), orc.run_problem_summed(p), f"paper-shaped S{sn}/P{pl}, 4 positions summed")
    p = _make("paper_coarse", nx=26, ny=26, nz=7, voxel=50.0 / 26, n_iter=5, n_pos=1)
    assert_problem_parity(dos.run_problem(p), orc.run_problem(p), "paper-shaped S6/P0 single projection")


# ------------------------------------------------------------------------------ method properties --
def test_uncollided_independent_of_quadrature_and_order(dos):
    """phi_u does not involve S_N or P_L -> bit-identical across them."""
    a = _make("config2", nx=24, ny=24, nz=8, voxel=1.6, n_group=4, n_iter=1, sn=4, pl=1)
    b = _make("config2", nx=24, ny=24, nz=8, voxel=1.6, n_group=4, n_iter=1, sn=8, pl=3)
    ua = dos.run_problem(a)["phi_u"]
    ub = dos.run_problem(b)["phi_u"]
    assert np.array_equal(ua, ub)


def test_repeatable_and_context_reuse(dos, orc):
    """A context is reusable for the next source position; a second run of the same position gives the
    same answer up to the order of the fp32 moment reductions."""
    p = _make("config4", nx=28, ny=24, nz=8, voxel=1.4, n_group=4, n_iter=3, n_pos=4)
    ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
    first = dos.run_problem(p, source_index=1, ctx=ctx)
    other = dos.run_problem(p, source_index=2, ctx=ctx)
    again = dos.run_problem(p, source_index=1, ctx=ctx)
    assert np.array_equal(first["phi_u"], again["phi_u"])
    l2, _ = field_errors(again["dose"], first["dose"])
    assert l2 < 1e-6
    assert_problem_parity(other, orc.run_problem(p, source_index=2), "reused context")
    ctx.close()


def test_scan_accumulate_and_host_entry_points(dos, orc):
    """a9: D_scan = sum_p D_p; the *_host entry points copy in/out and synchronise."""
    p = _make("config4", nx=24, ny=24, nz=8, voxel=1.6, n_group=4, n_iter=3, n_pos=3)
    ctx = dos.Context(p["mesh"], np.zeros_like(p["material"]), p["sigma_t"], p["sigma_s"], p["kerma"],
                      p["quadrature"], p["P_L"])
    ctx.dos_set_material_host(p["material"])          # the grid given to dos_create is replaced
    h = np.empty(p["material"].shape, dtype=np.float32)
    ref = np.zeros(p["material"].shape)
    for n in range(3):
        ctx.dos_uncollided(p["sources"][n], p["spectrum"])
        ctx.dos_solve(p["n_iter"])
        ctx.dos_dose_host(h, accumulate=(n > 0))
        ref += orc.run_problem(p, source_index=n)["dose"]
    assert_dose_parity(h, ref, "scan dose via dos_dose_host")
    ctx.close()


def test_state_machine_and_device_side_errors(dos):
    p = _make("config1")
    ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
    d = ctx.new_field(groups=False)
    with pytest.raises(dos.DosError) as e:
        ctx.dos_solve(2)
    assert e.value.status == -3
    with pytest.raises(dos.DosError) as e:
        ctx.dos_dose(d)
    assert e.value.status == -3
    ctx.dos_uncollided(p["sources"][0], p["spectrum"])
    with pytest.raises(dos.DosError) as e:
        ctx.dos_dose(d)
    assert e.value.status == -3
    with pytest.raises(dos.DosError) as e:
        ctx.dos_solve(0)
    assert e.value.status == -1
    bad = dict(p["sources"][0], pos=(0.5, 0.5, 0.5))           # a voxel centre of the 16^3 1 cm mesh
    with pytest.raises(dos.DosError) as e:
        ctx.dos_uncollided(bad, p["spectrum"])
    assert e.value.status == -1
    ctx.close()
    # material id >= n_mat is found on the device and reported by dos_check
    mat = p["material"].copy()
    mat[3, 4, 5] = 7
    ctx = dos.Context(p["mesh"], mat, p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
    ctx.dos_uncollided(p["sources"][0], p["spectrum"])
    with pytest.raises(dos.DosError) as e:
        ctx.dos_check()
    assert e.value.status == -1
    ctx.close()


def test_collided_fraction_rises_towards_low_energy(dos):
    """the uncollided fluence dominates in the upper energy range."""
    p = _make("config2", n_iter=6)
    out = dos.run_problem(p)
    k, j, i = 8, 32, 32
    frac = out["phi_u"][:, k, j, i] / out["phi_total"][:, k, j, i]
    assert frac[0] > frac[-4] and frac[0] > 0.5
