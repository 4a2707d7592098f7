"""Synthetic multigroup photon cross sections, dose factors and source spectrum (input generator).

Stands in for the ORNL 47-group / ENDF/B-VII.0 library, the ICRP 116 factors and the 100 kVp
spectrum of PAPER.md:79-81, :93, none of which is in the container. The model is
analytic: photoelectric ~ rho*C*Z^4/E^3 plus Klein-Nishina Compton from electron density, collapsed
to groups by Gauss-Legendre quadrature with a flat weight. Everything is computed in fp64 and
rounded to fp32; those fp32 values are the inputs to BOTH the oracle and the CUDA library.

This module holds no transport arithmetic (no ray trace, no sweep, no harmonics of directions).
"""
from __future__ import annotations

import numpy as np

MEC2_KEV = 510.99895
RE2_CM2 = 7.940787e-26            # classical electron radius squared
C_PE = 1.3535                      # cm^2 keV^3 / g ; tuned so water has a 13.9 mm mfp at 20 keV

# name: (rho g/cm3, n_e 1e23 e/cm3, Z_eff)  -- nominal, synthetic
MATERIALS = {
    "air": (0.001205, 0.003622, 7.64),
    "water": (1.00, 3.343, 7.42),
    "soft": (1.05, 3.48, 7.46),
    "fat": (0.95, 3.18, 6.3),
    "bone": (1.92, 5.95, 13.8),
    "liver": (1.06, 3.51, 7.5),
    "aluminium": (2.699, 7.83, 13.0),
}


def group_edges(n_group: int, e_hi: float, e_lo: float) -> np.ndarray:
    """Uniform-width groups, index 0 = highest energy. Returns G+1 descending edges."""
    return e_hi - np.arange(n_group + 1) * (e_hi - e_lo) / n_group


def mu_pe(name: str, e_kev):
    rho, _, z = MATERIALS[name]
    return rho * C_PE * z ** 4 / np.asarray(e_kev, dtype=np.float64) ** 3


def kn_dsigma_domega(e_kev, cos_t):
    """Klein-Nishina differential cross section per electron [cm^2/sr] and the ratio k = E_out/E."""
    k = 1.0 / (1.0 + (e_kev / MEC2_KEV) * (1.0 - cos_t))
    return 0.5 * RE2_CM2 * k * k * (k + 1.0 / k - (1.0 - cos_t * cos_t)), k


def _legendre_table(n_leg: int, x: np.ndarray) -> np.ndarray:
    p = np.zeros((n_leg + 1,) + x.shape)
    p[0] = 1.0
    if n_leg >= 1:
        p[1] = x
    for l in range(2, n_leg + 1):
        p[l] = ((2 * l - 1) * x * p[l - 1] - (l - 1) * p[l - 2]) / l
    return p


def make_xs(material_names, n_group: int, e_hi: float, e_lo: float, n_leg: int,
            n_e_nodes: int = 16, n_mu_nodes: int = 128, edges=None):
    """Multigroup table for the listed materials.

    Returns dict with float32 arrays
      sigma_t [n_mat][G]                 1/cm
      sigma_s [n_mat][n_leg+1][G][G]     [from][to], zero for to < from (downscatter only; eq. 2)
      kerma   [n_mat][G]                 keV cm^2 / g  (collision kerma per unit fluence), air row = 0
    and 'edges' (float64, descending). `edges` (G+1 descending values, keV) replaces the uniform-width structure,
    e.g. the paper's 7 groups 100/75/70/60/45/30/20/10 keV.
    """
    edges = group_edges(n_group, e_hi, e_lo) if edges is None else np.asarray(edges, dtype=np.float64)
    assert edges.shape == (n_group + 1,) and np.all(np.diff(edges) < 0)
    xe, we = np.polynomial.legendre.leggauss(n_e_nodes)
    xm, wm = np.polynomial.legendre.leggauss(n_mu_nodes)
    pl = _legendre_table(n_leg, xm)                           # [l][mu-node]
    n_mat = len(material_names)
    sigma_t = np.zeros((n_mat, n_group))
    sigma_s = np.zeros((n_mat, n_leg + 1, n_group, n_group))
    kerma = np.zeros((n_mat, n_group))
    for im, name in enumerate(material_names):
        rho, ne23, _ = MATERIALS[name]
        n_e = ne23 * 1e23
        for gp in range(n_group):
            hi, lo = edges[gp], edges[gp + 1]
            e_nodes = 0.5 * (hi + lo) + 0.5 * (hi - lo) * xe
            e_wts = 0.5 * we                                   # flat weight, normalised to 1
            for e, wq in zip(e_nodes, e_wts):
                ds, k = kn_dsigma_domega(e, xm)
                dmu = 2.0 * np.pi * n_e * ds * wm             # macroscopic, per cos-theta node
                e_out = e * k
                sigma_t[im, gp] += wq * (mu_pe(name, e) + dmu.sum())
                kerma[im, gp] += wq * (e * mu_pe(name, e) + (dmu * (e - e_out)).sum()) / rho
                # destination group of each node: edges descending, group g holds (edges[g+1], edges[g]]
                g_to = np.searchsorted(-edges, -e_out, side="left") - 1
                for g in range(gp, n_group):
                    sel = g_to == g
                    if sel.any():
                        sigma_s[im, :, gp, g] += wq * (pl[:, sel] * dmu[sel]).sum(axis=1)
        if name == "air":
            kerma[im, :] = 0.0                                 # dose in air neglected
    return {"sigma_t": sigma_t.astype(np.float32), "sigma_s": sigma_s.astype(np.float32),
            "kerma": kerma.astype(np.float32), "edges": edges, "materials": list(material_names),
            "n_leg": n_leg}


def uniform_spectrum(n_group: int) -> np.ndarray:
    return np.full(n_group, 1.0 / n_group, dtype=np.float32)


def kramers_spectrum(n_group: int, e_hi: float, e_lo: float, kvp: float = 120.0, al_cm: float = 0.2,
                     seed: int = 1, n_e_nodes: int = 16, edges=None) -> np.ndarray:
    """Seeded synthetic Kramers spectrum with Al filtration, group-integrated, sum = 1."""
    edges = group_edges(n_group, e_hi, e_lo) if edges is None else np.asarray(edges, dtype=np.float64)
    xe, we = np.polynomial.legendre.leggauss(n_e_nodes)
    _, ne23, _ = MATERIALS["aluminium"]
    s = np.zeros(n_group)
    for g in range(n_group):
        hi, lo = edges[g], edges[g + 1]
        e = 0.5 * (hi + lo) + 0.5 * (hi - lo) * xe
        mu_al = mu_pe("aluminium", e) + np.array(
            [(2.0 * np.pi * ne23 * 1e23 * kn_dsigma_domega(ei, _XM)[0] * _WM).sum() for ei in e])
        s[g] = (0.5 * (hi - lo) * we * np.maximum(kvp / e - 1.0, 0.0) * np.exp(-mu_al * al_cm)).sum()
    u = np.random.default_rng(seed).uniform(-1.0, 1.0, n_group)
    s *= 1.0 + 0.02 * u
    s /= s.sum()
    s32 = s.astype(np.float32)
    return s32


_XM, _WM = np.polynomial.legendre.leggauss(128)
