"""The five BASELINE.json workloads, and the paper-shaped workload of SURVEY.md 8(f) N4, as seeded synthetic problems
(SURVEY.md 8(d) recipe).

`make_problem(name)` returns a plain dict of numpy arrays / scalars; the same dict feeds the oracle
(tests, bench cpu_baseline) and the CUDA library. No transport arithmetic lives here.
"""
from __future__ import annotations

import math
import numpy as np

from . import phantoms, quadrature, xs


def _source(pos, axis, up, tan_half_fan, tan_half_cone, isotropic):
    return {"pos": tuple(float(v) for v in pos), "axis": tuple(float(v) for v in axis),
            "up": tuple(float(v) for v in up), "tan_half_fan": float(tan_half_fan),
            "tan_half_cone": float(tan_half_cone), "isotropic": int(isotropic)}


def scan_source(theta: float, radius: float = 54.0, tan_half_fan=None, tan_half_cone=None):
    """Cone-beam source on a circle of `radius` cm in the z = 0 plane, axis pointing at the origin; by default
    4 cm axial collimation at the isocentre (tan_half_cone = 2/54) and a 21 degree half fan."""
    c, s = math.cos(theta), math.sin(theta)
    return _source((radius * c, radius * s, 0.0), (-c, -s, 0.0), (0.0, 0.0, 1.0),
                   math.tan(math.radians(21.0)) if tan_half_fan is None else tan_half_fan,
                   2.0 / 54.0 if tan_half_cone is None else tan_half_cone, 0)


# the SHAPE of the paper's own workload (BASELINE.md "What the paper reports"):
# 7 energy groups with edges 100/75/70/60/45/30/20/10 keV, a 100 kVp spectrum, a 35 cm water cylinder in a
# 50 x 50 x 12.5 cm box on a 64x64x16 ("coarse", 7.81 mm) or 256x256x64 ("fine", 1.95 mm) mesh, S2-S8 x P0-P1
# (default S6/P0, the setting of the paper's CT-scan runs and of its Table 6), 16 source positions, 30 degree cone.
# The cross sections, spectrum and phantom are the synthetic stand-ins of this package, not the paper's data.
PAPER_EDGES = (100.0, 75.0, 70.0, 60.0, 45.0, 30.0, 20.0, 10.0)


_SPECS = {
    # name: nx ny nz voxel  G  SN PL n_iter  phantom   positions
    "config1": (16, 16, 16, 1.0, 4, 4, 1, 10, "water_cube", 1),
    "config2": (64, 64, 16, 0.6, 19, 8, 3, 20, "cylinder", 1),
    "config3": (128, 128, 64, 0.3, 19, 16, 5, 20, "cylinder", 1),
    "config4": (256, 256, 64, 0.15, 19, 8, 3, 15, "abdomen", 36),
    "config5": (256, 256, 256, 0.14, 19, 16, 5, 20, "abdomen", 1),
    "paper_coarse": (64, 64, 16, 50.0 / 64, 7, 6, 0, 20, "paper_cylinder", 16),
    "paper_fine": (256, 256, 64, 50.0 / 256, 7, 6, 0, 20, "paper_cylinder", 16),
}


def make_problem(name: str, **override):
    """Build a workload. `override` may replace nx, ny, nz, voxel, n_group, sn, pl, n_iter (for reduced
    parity cases that keep the structure of a config at a size the oracle finishes in seconds).
    `top_groups=k` keeps only the k highest-energy groups of the config's own group structure (tables and spectrum
    cut, not re-generated or re-normalised): photons only downscatter, so groups 0..k-1 of the full problem ARE
    this problem, and a parity run of it is a parity run of the head of the full cascade."""
    nx, ny, nz, vox, n_group, sn, pl, n_iter, kind, n_pos = _SPECS[name]
    nx = override.get("nx", nx); ny = override.get("ny", ny); nz = override.get("nz", nz)
    vox = override.get("voxel", vox); n_group = override.get("n_group", n_group)
    sn = override.get("sn", sn); pl = override.get("pl", pl); n_iter = override.get("n_iter", n_iter)
    n_pos = override.get("n_pos", n_pos)
    mesh = {"nx": nx, "ny": ny, "nz": nz, "dx": vox, "dy": vox, "dz": vox,
            "x0": -0.5 * nx * vox, "y0": -0.5 * ny * vox, "z0": -0.5 * nz * vox}
    quad = quadrature.as_float32(quadrature.level_symmetric(sn))
    if kind == "water_cube":
        mats = ["water"]
        mat = phantoms.homogeneous(nx, ny, nz, 0)
        table = xs.make_xs(mats, n_group, 120.0, 20.0, pl)
        spectrum = xs.uniform_spectrum(n_group)                   # seed 0 recorded, unused
        s = 30.0 / 7.0
        sources = [_source((2 * s, -3 * s, 6 * s), (0, 0, -1), (0, 1, 0), 0.0, 0.0, 1)]
    elif kind == "cylinder":
        mats = ["air", "water"]
        mat = phantoms.cylinder(nx, ny, nz, vox, vox, vox, radius=17.5 * (nx * vox) / 38.4)
        table = xs.make_xs(mats, n_group, 120.0, 10.0, pl)
        spectrum = xs.kramers_spectrum(n_group, 120.0, 10.0, seed=1)
        sources = [scan_source(0.5 * math.pi)]                    # (0, 54, 0), axis (0, -1, 0)
    elif kind == "paper_cylinder":
        if n_group != 7:
            raise ValueError("the paper-shaped workload has the paper's 7 groups")
        mats = ["air", "water"]
        mat = phantoms.cylinder(nx, ny, nz, vox, vox, vox, radius=17.5)
        table = xs.make_xs(mats, 7, 100.0, 10.0, pl, edges=PAPER_EDGES)
        spectrum = xs.kramers_spectrum(7, 100.0, 10.0, kvp=100.0, seed=1, edges=PAPER_EDGES)
        t15 = math.tan(math.radians(15.0))                       # "30 degree cone": 15 degree half angles both ways
        sources = [scan_source(2.0 * math.pi * q / n_pos, tan_half_fan=t15, tan_half_cone=t15) for q in range(n_pos)]
    else:
        mats = phantoms.ABDOMEN_MATERIALS
        mat = phantoms.abdomen(nx, ny, nz, seed=3)
        table = xs.make_xs(mats, n_group, 120.0, 10.0, pl)
        spectrum = xs.kramers_spectrum(n_group, 120.0, 10.0, seed=1)
        if n_pos == 1:
            sources = [scan_source(2.0 * math.pi * 9 / 36)]
        else:
            sources = [scan_source(2.0 * math.pi * p / n_pos) for p in range(n_pos)]
    top = override.get("top_groups")
    if top is not None and top < n_group:
        table = {"sigma_t": np.ascontiguousarray(table["sigma_t"][:, :top]),
                 "sigma_s": np.ascontiguousarray(table["sigma_s"][:, :, :top, :top]),
                 "kerma": np.ascontiguousarray(table["kerma"][:, :top]), "edges": table["edges"][:top + 1]}
        spectrum = np.ascontiguousarray(spectrum[:top])
        n_group = top
    return {"name": name, "mesh": mesh, "material": mat, "materials": mats,
            "sigma_t": table["sigma_t"], "sigma_s": table["sigma_s"], "kerma": table["kerma"],
            "edges": table["edges"], "n_group": n_group, "n_leg": pl, "P_L": pl, "quadrature": quad,
            "sn": sn, "spectrum": spectrum, "sources": sources, "n_iter": n_iter}


def n_updates(p) -> int:
    """Cell-angle-group updates of the whole problem (the BASELINE.json metric's numerator)."""
    m = p["mesh"]
    return m["nx"] * m["ny"] * m["nz"] * len(p["quadrature"]["w"]) * p["n_group"] * p["n_iter"] * len(p["sources"])
