"""Error measures and tolerances of the GPU-vs-oracle parity tests (BASELINE.json north_star).

  scalar fluence (total and collided, per group) and dose:
      relative L2 error over all voxels  <= 1e-5
      max relative error over voxels above 1e-6 of the field's peak  <= 1e-4
  uncollided fluence: max relative error over voxels above 1e-6 of the group's peak <= 1e-6, and the
      zero pattern (beam membership) must match exactly. The GPU stores fp32, so an oracle value below
      the smallest normal fp32 (1.18e-38) may legitimately read back as 0 or as a denormal.
"""
import numpy as np

TOL_L2 = 1e-5
TOL_MAX = 1e-4
TOL_UNCOLLIDED = 1e-6
FLT_MIN = 1.1754943508222875e-38


def field_errors(gpu, ref):
    """(relL2, max rel error above 1e-6 of peak) of one field (any shape)."""
    g = np.asarray(gpu, dtype=np.float64).ravel()
    r = np.asarray(ref, dtype=np.float64).ravel()
    peak = np.abs(r).max()
    if peak == 0.0:
        return (0.0 if not g.any() else np.inf), (0.0 if not g.any() else np.inf)
    l2 = np.linalg.norm(g - r) / np.linalg.norm(r)
    m = np.abs(r) > 1e-6 * peak
    return l2, (np.abs(g - r)[m] / np.abs(r)[m]).max()


def conditioned_field_errors(gpu, ref, scale):
    """field_errors for the collided fluence, which is a quadrature sum (eq. 3) of angular
    fluxes that go negative where the truncated P_L source is negative (reading R11): the sum
    can cancel to a value far below its terms, and no fp32 evaluation can then be relatively accurate
    in the RESULT (reading R15b). The denominator is therefore the oracle's sum of the terms'
    magnitudes, scale = sum_n w_n |psi_n| >= |phi_c|; where all psi_n >= 0 (no cancellation) it equals
    |phi_c| and the measure is exactly the north_star one."""
    g = np.asarray(gpu, dtype=np.float64).ravel()
    r = np.asarray(ref, dtype=np.float64).ravel()
    s = np.asarray(scale, dtype=np.float64).ravel()
    peak = np.abs(r).max()
    if peak == 0.0:
        return field_errors(g, r)
    assert (s >= np.abs(r) * (1.0 - 1e-12)).all()
    l2 = np.linalg.norm(g - r) / np.linalg.norm(r)
    m = np.abs(r) > 1e-6 * peak
    return l2, (np.abs(g - r)[m] / s[m]).max()


def per_group_errors(gpu, ref, scale=None):
    errs = np.array([field_errors(gpu[g], ref[g]) if scale is None else
                     conditioned_field_errors(gpu[g], ref[g], scale[g]) for g in range(ref.shape[0])])
    return errs[:, 0].max(), errs[:, 1].max()


def assert_fluence_parity(gpu, ref, what, scale=None):
    l2, mx = per_group_errors(gpu, ref, scale)
    assert l2 <= TOL_L2 and mx <= TOL_MAX, f"{what}: relL2 {l2:.3e} (<= {TOL_L2}), max rel {mx:.3e} (<= {TOL_MAX})"
    return l2, mx


def assert_dose_parity(gpu, ref, what="dose"):
    l2, mx = field_errors(gpu, ref)
    assert l2 <= TOL_L2 and mx <= TOL_MAX, f"{what}: relL2 {l2:.3e}, max rel {mx:.3e}"
    return l2, mx


def assert_uncollided_parity(gpu, ref):
    gpu = np.asarray(gpu)
    ref = np.asarray(ref, dtype=np.float64)
    # beam membership: exact zeros of the oracle are exact zeros on the GPU, and nothing else is zero
    # unless the oracle's value is below fp32 range
    assert not gpu[ref == 0.0].any(), "GPU has fluence outside the oracle's beam"
    lost = (gpu == 0.0) & (ref != 0.0)
    assert (np.abs(ref[lost]) < FLT_MIN).all(), "GPU has zeros inside the oracle's beam"
    worst = 0.0
    for g in range(ref.shape[0]):
        _, mx = field_errors(gpu[g], ref[g])
        worst = max(worst, mx)
    assert worst <= TOL_UNCOLLIDED, f"uncollided max rel error {worst:.3e} (<= {TOL_UNCOLLIDED})"
    return worst


def cancellation_report(gpu, ref, scale, what=""):
    """Evidence for reading R15b, printed by every parity case: the plain north_star max-rel of the collided fluence
    (denominator |phi_c|), the conditioned one (denominator sum_n w_n |psi_n|), and on how many of the voxels above the
    1e-6-of-peak threshold the two denominators differ at all (i.e. some angular flux is negative there)."""
    out = []
    for g in range(ref.shape[0]):
        r = np.asarray(ref[g], dtype=np.float64).ravel()
        s = np.asarray(scale[g], dtype=np.float64).ravel()
        d = np.abs(np.asarray(gpu[g], dtype=np.float64).ravel() - r)
        peak = np.abs(r).max()
        if peak == 0.0:
            continue
        m = np.abs(r) > 1e-6 * peak
        canc = m & (s > np.abs(r) * (1.0 + 1e-9))
        plain = (d[m] / np.abs(r[m])).max()
        cond = (d[m] / s[m]).max()
        plain_nc = (d[m & ~canc] / np.abs(r[m & ~canc])).max() if (m & ~canc).any() else 0.0
        out.append((g, plain, cond, int(canc.sum()), int(m.sum()), plain_nc))
    worst = max(out, key=lambda t: t[1]) if out else None
    if worst:
        print(f"[R15b] {what}: worst group {worst[0]}: plain max-rel {worst[1]:.3e}, conditioned {worst[2]:.3e}; "
              f"{worst[3]} of {worst[4]} voxels above threshold have angular fluxes of both signs; plain max-rel on the "
              f"others {worst[5]:.3e}")
    return out


def sampled_field_errors(gpu_s, ref_s, peak, scale_s=None):
    """(relL2 over the sample, max rel error over sampled voxels above 1e-6 of the field's TRUE peak) for a seeded
    sample of voxels of a stored full-size oracle result (tests/golden): a uniform subset estimates the all-voxel ratio
    of mean squares without bias; the threshold uses the peak over all voxels, stored with the sample."""
    g = np.asarray(gpu_s, dtype=np.float64).ravel()
    r = np.asarray(ref_s, dtype=np.float64).ravel()
    den = np.abs(r) if scale_s is None else np.asarray(scale_s, dtype=np.float64).ravel()
    if peak == 0.0:
        return (0.0 if not g.any() else np.inf), (0.0 if not g.any() else np.inf)
    l2 = np.linalg.norm(g - r) / max(np.linalg.norm(r), 1e-300)
    m = np.abs(r) > 1e-6 * peak
    return l2, ((np.abs(g - r)[m] / den[m]).max() if m.any() else 0.0)


def assert_problem_parity(out, ref, name=""):
    cancellation_report(out["phi_c"], ref["phi_c"], ref["phi_c_abs"], name)
    res = {"phi_u": assert_uncollided_parity(out["phi_u"], ref["phi_u"]),
           "phi_c": assert_fluence_parity(out["phi_c"], ref["phi_c"], name + " collided fluence", scale=ref["phi_c_abs"]),
           "phi_total": assert_fluence_parity(out["phi_total"], ref["phi_total"], name + " total fluence"),
           "dose": assert_dose_parity(out["dose"], ref["dose"], name + " dose")}
    return res
