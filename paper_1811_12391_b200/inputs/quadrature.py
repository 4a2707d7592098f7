"""Level-symmetric S_N quadrature sets, built by construction (no recalled tables).

Input generator only: it produces the (mu, eta, xi, w) table that is an INPUT to both the
oracle and the CUDA library (dos_quadrature). It holds none of the transport arithmetic.

Cites: PAPER.md:43-45 (eq. 3: N(N+2) directions, weights w_n), PAPER.md:79 (S2..S8 =
8/24/48/80 directions); construction recipe SURVEY.md section 8(c) "Quadrature" pin.

Construction (level-symmetric LQ_N):
  levels    mu_i^2 = mu_1^2 + (i-1) * 2 (1 - 3 mu_1^2) / (N - 2),  i = 1..N/2
  points    (mu_i, mu_j, mu_k) with i + j + k = N/2 + 2 in the first octant, reflected to 8 octants
  weights   one per permutation class of (i, j, k); solved from the even-moment conditions
            sum_n w_n mu_n^(2k) = 1/(2k+1), k = 0, 2, 3, .., N/2 (k = 1 holds by symmetry),
            with sum_n w_n = 1 over the whole sphere
  mu_1      the value that makes that linear system consistent (1-D search around a start value)

Octant numbering (matches SURVEY.md 8(c) O4): bit0 set <=> mu < 0, bit1 <=> eta < 0, bit2 <=> xi < 0.
Angles are ordered octant-major: n = octant * (N_a/8) + index within the first-octant list.
"""
from __future__ import annotations

import itertools
import numpy as np

# start values for the 1-D search on mu_1; the search polishes them
_MU1_START = {2: 0.5773502691896258, 4: 0.3500212, 6: 0.2666355, 8: 0.2182179,
              10: 0.1893213, 12: 0.1672126, 14: 0.1519859, 16: 0.1389568}


def _levels(n_order: int, mu1: float) -> np.ndarray:
    h = n_order // 2
    if n_order == 2:
        return np.array([mu1])
    delta = 2.0 * (1.0 - 3.0 * mu1 * mu1) / (n_order - 2)
    return np.sqrt(mu1 * mu1 + np.arange(h) * delta)


def _octant_points(n_order: int):
    """First-octant level-index triples (i, j, k), 1-based, i + j + k = N/2 + 2, and their class id."""
    h = n_order // 2
    triples = [(i, j, k) for i in range(1, h + 1) for j in range(1, h + 1)
               for k in range(1, h + 1) if i + j + k == h + 2]
    classes = sorted({tuple(sorted(t)) for t in triples})
    cid = [classes.index(tuple(sorted(t))) for t in triples]
    return triples, cid, len(classes)


def _moment_system(n_order: int, mu1: float):
    lv = _levels(n_order, mu1)
    triples, cid, ncls = _octant_points(n_order)
    ks = [0] + list(range(2, n_order // 2 + 1))
    a = np.zeros((len(ks), ncls))
    for (i, _, _), c in zip(triples, cid):
        for r, k in enumerate(ks):
            a[r, c] += 8.0 * lv[i - 1] ** (2 * k)      # 8 octants, all carry the same |mu|
    b = np.array([1.0 / (2 * k + 1) for k in ks])
    return a, b


def _residual(n_order: int, mu1: float) -> float:
    a, b = _moment_system(n_order, mu1)
    w, *_ = np.linalg.lstsq(a, b, rcond=None)
    return float(np.linalg.norm(a @ w - b))


def _solve_mu1(n_order: int) -> float:
    if n_order == 2:
        return _MU1_START[2]
    x0 = _MU1_START[n_order]
    # golden-section search on the least-squares residual in a small bracket, then refine
    lo, hi = x0 - 2e-5, x0 + 2e-5
    g = (np.sqrt(5.0) - 1.0) / 2.0
    c, d = hi - g * (hi - lo), lo + g * (hi - lo)
    fc, fd = _residual(n_order, c), _residual(n_order, d)
    for _ in range(200):
        if fc < fd:
            hi, d, fd = d, c, fc
            c = hi - g * (hi - lo)
            fc = _residual(n_order, c)
        else:
            lo, c, fc = c, d, fd
            d = lo + g * (hi - lo)
            fd = _residual(n_order, d)
        if hi - lo < 1e-16:
            break
    return 0.5 * (lo + hi)


def level_symmetric(n_order: int):
    """Return dict(mu, eta, xi, w) as float64 arrays of length N(N+2), sum(w) = 1, octant-major."""
    if n_order % 2 or n_order < 2 or n_order not in _MU1_START:
        raise ValueError(f"unsupported S_N order {n_order}")
    mu1 = _solve_mu1(n_order)
    lv = _levels(n_order, mu1)
    triples, cid, _ = _octant_points(n_order)
    a, b = _moment_system(n_order, mu1)
    wcls, *_ = np.linalg.lstsq(a, b, rcond=None)          # min-norm when rank-deficient (S16)
    per = len(triples)
    n_ang = 8 * per
    mu = np.empty(n_ang); eta = np.empty(n_ang); xi = np.empty(n_ang); w = np.empty(n_ang)
    for o in range(8):
        sx = -1.0 if (o & 1) else 1.0
        sy = -1.0 if (o & 2) else 1.0
        sz = -1.0 if (o & 4) else 1.0
        for t, ((i, j, k), c) in enumerate(zip(triples, cid)):
            n = o * per + t
            mu[n], eta[n], xi[n] = sx * lv[i - 1], sy * lv[j - 1], sz * lv[k - 1]
            w[n] = wcls[c]
    w /= w.sum()
    return {"mu": mu, "eta": eta, "xi": xi, "w": w, "n_order": n_order, "mu1": mu1}


def as_float32(q):
    """Round the table to fp32 (the values both sides consume); weights renormalised in fp64 first."""
    return {k: (np.asarray(v, dtype=np.float32) if k in ("mu", "eta", "xi", "w") else v) for k, v in q.items()}
