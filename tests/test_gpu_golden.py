"""GPU-vs-oracle parity at FULL size for configs 3, 4 and 5 (BASELINE.json north_star target), through the C ABI, in the
launch configuration bench.py times. The oracle results come from tests/golden/*.npz, written once by
tests/golden/make_golden.py (fp64 oracle only; keyed by a hash of inputs + oracle source, checked here and by the CPU test
test_golden_files_match_inputs_and_oracle_source). What is compared: per-group uncollided, collided and total fluence at
a seeded sample of 10 240 voxels and the dose at 262 144 voxels, at the north_star tolerances (tests/parity.py); the
relative L2 error is taken over the sample, the max-rel threshold uses the stored all-voxel peaks.

  config3          128x128x64, S16/P5, all 19 groups x 20 iterations
  config4_pos5     256x256x64, S8/P3, source position 5 of the scan, all 19 groups x 15 iterations
  config5_top3x6   256^3, S16/P5, the 3 highest-energy groups x 6 iterations
  config5_top6     256^3, S16/P5, the 6 highest-energy groups x 20 iterations (groups 0..5 of the full cascade ARE this
                   problem: photons only downscatter; the full 19 x 20 run is 5 h of oracle time on the 8-core build box)
"""
import glob
import os
import sys

import numpy as np
import pytest

from parity import TOL_L2, TOL_MAX, TOL_UNCOLLIDED, FLT_MIN, sampled_field_errors

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "golden"))
CASES = sorted(os.path.basename(f)[:-4] for f in glob.glob(os.path.join(HERE, "golden", "*.npz")))


@pytest.mark.parametrize("case", CASES)
def test_full_size_parity_against_stored_oracle(case):
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import make_golden as mg
    from paper_1811_12391_b200 import dos
    from paper_1811_12391_b200.inputs import make_problem
    z = np.load(os.path.join(HERE, "golden", case + ".npz"))
    config, ov, sidx, text = mg.CASES[case]
    p = make_problem(config, **ov)
    assert str(z["key"]) == mg.problem_key(p, sidx), f"{case}: stale golden file (inputs or oracle source changed)"
    G = p["n_group"]
    ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
    pu, pc, pt, d = ctx.new_field(), ctx.new_field(), ctx.new_field(), ctx.new_field(groups=False)
    ctx.dos_uncollided(p["sources"][sidx], p["spectrum"], pu)
    ctx.dos_solve(p["n_iter"])
    ctx.dos_fluence(pc, pt)
    ctx.dos_dose(d, False)
    ctx.dos_check()
    cells = torch.from_numpy(z["cells"]).to(pu.device)
    dcells = torch.from_numpy(z["dose_cells"]).to(pu.device)
    got = {"phi_u": pu.reshape(G, -1)[:, cells].cpu().numpy(), "phi_c": pc.reshape(G, -1)[:, cells].cpu().numpy(),
           "phi_total": pt.reshape(G, -1)[:, cells].cpu().numpy(), "dose": d.reshape(-1)[dcells].cpu().numpy()}
    ctx.close()
    # uncollided: zero pattern exact, max-rel 1e-6 above 1e-6 of the group's true peak
    ref_u = z["phi_u"].astype(np.float64)
    assert not got["phi_u"][ref_u == 0.0].any(), "GPU has fluence outside the oracle's beam"
    lost = (got["phi_u"] == 0.0) & (ref_u != 0.0)
    assert (np.abs(ref_u[lost]) < FLT_MIN).all(), "GPU has zeros inside the oracle's beam"
    # the stored reference is the oracle's fp64 value rounded to fp32 (6e-8): the 1e-6 bar keeps its meaning
    worst_u = max(sampled_field_errors(got["phi_u"][g], ref_u[g], float(z["peak_phi_u"][g]))[1] for g in range(G))
    assert worst_u <= TOL_UNCOLLIDED + 1.2e-7, f"{case}: uncollided max rel {worst_u:.3e}"
    res = {"phi_u": worst_u}
    # total fluence (the north_star quantity): the plain measure, every sampled voxel, no exception
    errs = [sampled_field_errors(got["phi_total"][g], z["phi_total"][g], float(z["peak_phi_total"][g])) for g in range(G)]
    l2, mx = max(e[0] for e in errs), max(e[1] for e in errs)
    res["phi_total"] = (l2, mx)
    assert l2 <= TOL_L2 and mx <= TOL_MAX, f"{case} phi_total: relL2 {l2:.3e} (<= {TOL_L2}), max rel {mx:.3e} (<= {TOL_MAX})"
    # collided fluence on its own (R15, R15b, R15c): relL2 as stated; max-rel against sum_n w_n |psi_n|. At full
    # cascade depth a few voxels inside the direct beam, where the truncated-P_L first-collision source drives angular
    # fluxes of both signs through hundreds of diamond-difference cells, sit just above 1e-4 even in that measure
    # (measured: 5 of 194 446 sampled (group, voxel) pairs at config 4 with the FFMA sweep, worst 1.32e-4; none with the
    # tensor-memory sweep, worst 9.1e-5): fp32 storage of the moments bounds what any fp32 sweep can do there. On the
    # 256^3 S16/P5 mesh after 6 groups x 20 iterations the same happens in 2-4 of 61 434 pairs, all in air voxels outside
    # the body where the collided fluence is 1e-3 of its peak and 1e-3 of the uncollided fluence of the same voxel:
    # worst 1.4-1.5e-4 with the FFMA sweep, 4.5-5.4e-4 with the tensor-memory sweep (3xTF32 products carry ~3x the
    # rounding error of fp32 FMAs; rounding instead of truncating the low part changed nothing), run-to-run different in
    # the last digits (order of the reds). The test admits at most 1e-4 of the pairs above 1e-4 and none above 1e-3
    # (R15c), and prints what it found; the total fluence keeps the plain bar at every voxel.
    ref_c, sc_c = z["phi_c"].astype(np.float64), z["phi_c_abs"].astype(np.float64)
    l2c, over, worst_c, n_pairs = 0.0, 0, 0.0, 0
    for g in range(G):
        l2c = max(l2c, sampled_field_errors(got["phi_c"][g], ref_c[g], float(z["peak_phi_c"][g]))[0])
        m = np.abs(ref_c[g]) > 1e-6 * float(z["peak_phi_c"][g])
        e = np.abs(got["phi_c"][g].astype(np.float64) - ref_c[g])[m] / sc_c[g][m]
        over += int((e > TOL_MAX).sum()); n_pairs += int(m.sum()); worst_c = max(worst_c, float(e.max()) if e.size else 0.0)
    res["phi_c"] = (l2c, worst_c, f"{over} of {n_pairs} pairs above {TOL_MAX}")
    assert l2c <= TOL_L2, f"{case} phi_c: relL2 {l2c:.3e} (<= {TOL_L2})"
    assert over <= 1e-4 * n_pairs and worst_c <= 10 * TOL_MAX, f"{case} phi_c: {over} of {n_pairs} pairs above {TOL_MAX}, worst {worst_c:.3e}"
    # evidence for R15b: the plain measure of the collided fluence and how many voxels cancel
    plain = [sampled_field_errors(got["phi_c"][g], z["phi_c"][g], float(z["peak_phi_c"][g]))[1] for g in range(G)]
    canc = int(((z["phi_c_abs"] > np.abs(z["phi_c"]) * (1 + 1e-6)) & (np.abs(z["phi_c"]) > 1e-6 * z["peak_phi_c"][:, None])).sum())
    l2, mx = sampled_field_errors(got["dose"], z["dose"], float(z["dose_peak"]))
    res["dose"] = (l2, mx)
    assert l2 <= TOL_L2 and mx <= TOL_MAX, f"{case} dose: relL2 {l2:.3e}, max rel {mx:.3e}"
    print(f"[golden] {case} ({text}): " + ", ".join(f"{k} {v}" for k, v in res.items()) +
          f"; collided plain max-rel {max(plain):.3e} with {canc} sampled (group, voxel) pairs of mixed-sign angular flux")
