"""Seeded synthetic voxel phantoms shaped like the paper's: a 35 cm water cylinder in
air and an abdomen-like body. Input generator only (material-id grids); recipe: SURVEY.md 8(d).

Material-id arrays are uint8 [nz][ny][nx] (x fastest). The mesh is centred at the origin:
x0 = -nx*dx/2, voxel (i, j, k) centre at x0 + (i + 1/2) dx, etc.
"""
from __future__ import annotations

import numpy as np


def centres(n: int, d: float) -> np.ndarray:
    return -0.5 * n * d + (np.arange(n) + 0.5) * d


def homogeneous(nx, ny, nz, mat_id=0) -> np.ndarray:
    return np.full((nz, ny, nx), mat_id, dtype=np.uint8)


def cylinder(nx, ny, nz, dx, dy, dz, radius=17.5, inside=1, outside=0) -> np.ndarray:
    """Water (id `inside`) where the voxel centre has x^2 + y^2 <= radius^2, else air (id `outside`)."""
    x = centres(nx, dx)[None, None, :]
    y = centres(ny, dy)[None, :, None]
    m = np.where(x * x + y * y <= radius * radius, inside, outside).astype(np.uint8)
    return np.broadcast_to(m, (nz, ny, nx)).copy()


# ids used by the abdomen-like phantom
AIR, SOFT, FAT, BONE, LIVER = 0, 1, 2, 3, 4
ABDOMEN_MATERIALS = ["air", "soft", "fat", "bone", "liver"]


def abdomen(nx, ny, nz, seed=3) -> np.ndarray:
    """Abdomen-like phantom in normalised coordinates u, v, t in [-1, 1] (so an axially longer mesh holds
    'the same phantom extended axially'). Painted in order, later wins: body soft tissue, fat shell,
    liver, spine, ribs, air-filled bowel pockets. All semi-axes jittered +-5 %, centres +-0.02."""
    rng = np.random.default_rng(seed)

    def jit_ax(a):
        return a * (1.0 + 0.05 * rng.uniform(-1.0, 1.0))

    def jit_c(c):
        return c + 0.02 * rng.uniform(-1.0, 1.0)

    u = (2.0 * (np.arange(nx) + 0.5) / nx - 1.0)[None, None, :]
    v = (2.0 * (np.arange(ny) + 0.5) / ny - 1.0)[None, :, None]
    t = (2.0 * (np.arange(nz) + 0.5) / nz - 1.0)[:, None, None]
    m = np.zeros((nz, ny, nx), dtype=np.uint8)

    au, av = jit_ax(0.88), jit_ax(0.62)
    body = (u / au) ** 2 + (v / av) ** 2 <= 1.0
    inner = (u / (0.90 * au)) ** 2 + (v / (0.90 * av)) ** 2 <= 1.0
    m[np.broadcast_to(body, m.shape)] = SOFT
    m[np.broadcast_to(body & ~inner, m.shape)] = FAT
    cu, cv, ct = jit_c(-0.35), jit_c(0.10), jit_c(0.0)
    a1, a2, a3 = jit_ax(0.33), jit_ax(0.26), jit_ax(0.8)
    m[((u - cu) / a1) ** 2 + ((v - cv) / a2) ** 2 + ((t - ct) / a3) ** 2 <= 1.0] = LIVER
    cu, cv = jit_c(0.0), jit_c(-0.30)
    a1, a2 = jit_ax(0.11), jit_ax(0.11)
    m[np.broadcast_to(((u - cu) / a1) ** 2 + ((v - cv) / a2) ** 2 <= 1.0, m.shape)] = BONE
    for r in range(5):                                           # 5 ribs, each mirrored -> 10
        th = rng.uniform(0.15 * np.pi, 0.85 * np.pi)
        tc = rng.uniform(-0.8, 0.8)
        for sgn in (1.0, -1.0):
            cu, cv, ct = jit_c(sgn * 0.72 * np.cos(th)), jit_c(0.50 * np.sin(th)), jit_c(tc)
            a1, a2, a3 = jit_ax(0.05), jit_ax(0.03), jit_ax(0.25)
            m[((u - cu) / a1) ** 2 + ((v - cv) / a2) ** 2 + ((t - ct) / a3) ** 2 <= 1.0] = BONE
    for b in range(8):
        cu, cv, ct = jit_c(rng.uniform(-0.1, 0.5)), jit_c(rng.uniform(-0.1, 0.35)), jit_c(rng.uniform(-0.8, 0.8))
        a1, a2, a3 = jit_ax(rng.uniform(0.03, 0.07)), jit_ax(rng.uniform(0.03, 0.07)), jit_ax(rng.uniform(0.1, 0.3))
        m[((u - cu) / a1) ** 2 + ((v - cv) / a2) ** 2 + ((t - ct) / a3) ** 2 <= 1.0] = AIR
    return m
