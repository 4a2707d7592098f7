"""fp64 CPU oracle of the discrete-ordinates CT dose hot path -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this
package. It shares nothing with paper_1811_12391_b200/csrc (the CUDA path) and does not import it.

The arithmetic lives in dos_oracle.c (plain C, fp64); this module is the ctypes loader plus thin
argument marshalling. `build()` compiles the C file with gcc.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dos_oracle.c")
_SRC_BLOCKED = os.path.join(_HERE, "dos_oracle_blocked.c")     # second loop arrangement, bit-identical (golden runs)
_LIB = os.path.join(_HERE, "libdos_oracle.so")
_lib = None


class _Mesh(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("x0", C.c_double), ("y0", C.c_double), ("z0", C.c_double)]


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -shared; rebuilt when a source is newer than the library. -ffp-contract=off: no fused
    multiply-add, so the two loop arrangements round identically; the vectoriser flags change no result."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_BLOCKED)):
        subprocess.check_call(["gcc", "-O2", "-ftree-vectorize", "-fvect-cost-model=dynamic", "-std=c11", "-fopenmp", "-fPIC",
                               "-shared", "-ffp-contract=off", "-o", _LIB, _SRC, _SRC_BLOCKED, "-lm"])
    return _LIB


def source_files():
    """The C sources whose text keys the stored golden results (tests/golden)."""
    return [_SRC, _SRC_BLOCKED]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_harmonics.restype = None
        _lib.orc_uncollided.restype = C.c_int
        _lib.orc_uncollided_cells.restype = C.c_int
        _lib.orc_first_collision.restype = None
        _lib.orc_sweep.restype = C.c_int
        _lib.orc_solve.restype = C.c_int
        _lib.orc_solve_iters.restype = C.c_int
        _lib.orc_solve_blocked.restype = C.c_int
        _lib.orc_dose.restype = None
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _mesh(m):
    return _Mesh(m["nx"], m["ny"], m["nz"], m["dx"], m["dy"], m["dz"], m["x0"], m["y0"], m["z0"])


def n_moments(L: int) -> int:
    return (L + 1) * (L + 1)


def harmonics(mu, eta, xi, L):
    """Y_lm(Omega) for one direction -> float64 [(L+1)^2], index lm = l(l+1)+m."""
    y = np.zeros(n_moments(L))
    lib().orc_harmonics(C.c_double(mu), C.c_double(eta), C.c_double(xi), C.c_int(L), _p(y))
    return y


def uncollided(mesh, material, sigma_t, source, spectrum, want_path=False):
    """phi_u [G][nz][ny][nx] (float64). sigma_t [n_mat][G]."""
    sig = _d(sigma_t)
    n_mat, G = sig.shape
    mat = np.ascontiguousarray(material, dtype=np.uint8)
    nv = mat.size
    phi = np.zeros((G, nv))
    path = np.zeros(nv) if want_path else None
    pos, axis, up = _d(source["pos"]), _d(source["axis"]), _d(source["up"])
    ms = _mesh(mesh)
    err = lib().orc_uncollided(C.byref(ms), _p(mat), C.c_int(n_mat), C.c_int(G), _p(sig), _p(pos), _p(axis), _p(up),
                               C.c_double(source["tan_half_fan"]), C.c_double(source["tan_half_cone"]),
                               C.c_int(source["isotropic"]), _p(_d(spectrum)), _p(phi), _p(path))
    if err:
        raise ValueError("source coincides with a voxel centre")
    phi = phi.reshape((G,) + mat.shape)
    return (phi, path.reshape(mat.shape)) if want_path else phi


def uncollided_at(mesh, material, sigma_t, source, spectrum, cells):
    """phi_u [G][len(cells)] for the listed flat voxel indices (k*ny*nx + j*nx + i) only."""
    sig = _d(sigma_t)
    n_mat, G = sig.shape
    mat = np.ascontiguousarray(material, dtype=np.uint8)
    idx = np.ascontiguousarray(cells, dtype=np.int64)
    assert idx.min() >= 0 and idx.max() < mat.size
    phi = np.zeros((G, idx.size))
    pos, axis, up = _d(source["pos"]), _d(source["axis"]), _d(source["up"])
    ms = _mesh(mesh)
    err = lib().orc_uncollided_cells(C.byref(ms), _p(mat), C.c_int(n_mat), C.c_int(G), _p(sig), _p(pos), _p(axis),
                                     _p(up), C.c_double(source["tan_half_fan"]), C.c_double(source["tan_half_cone"]),
                                     C.c_int(source["isotropic"]), _p(_d(spectrum)), _p(idx), C.c_longlong(idx.size),
                                     _p(phi))
    if err:
        raise ValueError("source coincides with a voxel centre")
    return phi


def sweep(mesh, material, sig_t_g, quad, L, Q, reflective=False, bnd_state=None, want_leakage=False,
          want_psi=False):
    """One transport sweep. Q [M][nz][ny][nx] -> phi_new [M][nz][ny][nx]; optional leakage, psi [n_ang][Nv]."""
    mat = np.ascontiguousarray(material, dtype=np.uint8)
    nv = mat.size
    M = n_moments(L)
    Qd = _d(Q).reshape(M, nv)
    phi = np.zeros((M, nv))
    n_ang = len(quad["w"])
    mu, eta, xi, w = _d(quad["mu"]), _d(quad["eta"]), _d(quad["xi"]), _d(quad["w"])
    leak = C.c_double(0.0)
    psi = np.zeros((n_ang, nv)) if want_psi else None
    ms = _mesh(mesh)
    if reflective and bnd_state is None:
        raise ValueError("reflective sweep needs bnd_state")
    rc = lib().orc_sweep(C.byref(ms), _p(mat), _p(_d(sig_t_g)), C.c_int(n_ang), _p(mu), _p(eta), _p(xi), _p(w),
                         C.c_int(L), _p(Qd), _p(phi), C.c_int(int(reflective)), _p(bnd_state),
                         C.byref(leak) if want_leakage else None, _p(psi), None)
    if rc:
        raise MemoryError("orc_sweep")
    out = [phi.reshape((M,) + mat.shape)]
    if want_leakage:
        out.append(leak.value)
    if want_psi:
        out.append(psi)
    return out[0] if len(out) == 1 else tuple(out)


def bnd_state_size(mesh, n_ang):
    return n_ang * (mesh["ny"] * mesh["nz"] + mesh["nx"] * mesh["nz"] + mesh["nx"] * mesh["ny"])


def solve(mesh, material, sigma_t, sigma_s, quad, L, n_iter, source_pos=None, phi_u=None, q_ext=None,
          reflective=False, want_balance=False, want_abs=False, blocked=False, n_iter_g=None, want_conv=False):
    """Group cascade + source iteration. Returns phi_c moments [G][M][nz][ny][nx] (float64)
    (and, if want_balance, (leak[G], src_last[G]) of each group's last sweep; if want_abs, the
    diagnostic sum_n w_n |psi_n| [G][nz][ny][nx] of each group's last sweep).
    blocked=True runs dos_oracle_blocked.c, the bit-identical second loop arrangement (vacuum boundaries only).
    n_iter_g [G] replaces n_iter group by group; want_conv appends each group's last-iteration stopping measure
    max|phi00^(it) - phi00^(it-1)| / max|phi00^(it)| (the quantity dos_solve_tol tests) to the result."""
    sig_t, sig_s = _d(sigma_t), _d(sigma_s)
    n_mat, G = sig_t.shape
    n_leg = sig_s.shape[1] - 1
    assert sig_s.shape == (n_mat, n_leg + 1, G, G) and L <= n_leg
    mat = np.ascontiguousarray(material, dtype=np.uint8)
    nv = mat.size
    M = n_moments(L)
    phi_c = np.zeros((G, M, nv))
    n_ang = len(quad["w"])
    mu, eta, xi, w = _d(quad["mu"]), _d(quad["eta"]), _d(quad["xi"]), _d(quad["w"])
    leak = np.zeros(G) if want_balance else None
    src = np.zeros(G) if want_balance else None
    pu = _d(phi_u).reshape(G, nv) if phi_u is not None else None
    qe = _d(q_ext).reshape(G, M, nv) if q_ext is not None else None
    pos = _d(source_pos) if source_pos is not None else np.zeros(3)
    pabs = np.zeros((G, nv)) if want_abs else None
    ms = _mesh(mesh)
    conv = None
    if blocked:
        if reflective or want_balance or want_conv or n_iter_g is not None:
            raise ValueError("the blocked arrangement has vacuum boundaries and no balance outputs")
        rc = lib().orc_solve_blocked(C.byref(ms), _p(mat), C.c_int(n_mat), C.c_int(G), C.c_int(n_leg), C.c_int(L),
                                     _p(sig_t), _p(sig_s), C.c_int(n_ang), _p(mu), _p(eta), _p(xi), _p(w), _p(pos),
                                     _p(pu), _p(qe), C.c_int(n_iter), _p(phi_c), _p(pabs))
    else:
        nig = np.ascontiguousarray(n_iter_g, dtype=np.int32) if n_iter_g is not None else None
        assert nig is None or nig.shape == (G,)
        conv = np.zeros(G) if want_conv else None
        rc = lib().orc_solve_iters(C.byref(ms), _p(mat), C.c_int(n_mat), C.c_int(G), C.c_int(n_leg), C.c_int(L), _p(sig_t),
                                   _p(sig_s), C.c_int(n_ang), _p(mu), _p(eta), _p(xi), _p(w), _p(pos), _p(pu), _p(qe),
                                   C.c_int(n_iter), _p(nig), C.c_int(int(reflective)), _p(phi_c), _p(leak), _p(src),
                                   _p(pabs), _p(conv))
    if rc:
        raise MemoryError("orc_solve")
    phi_c = phi_c.reshape((G, M) + mat.shape)
    if want_conv:
        return phi_c, conv
    if want_abs:
        return phi_c, pabs.reshape((G,) + mat.shape)
    return (phi_c, leak, src) if want_balance else phi_c


def dose(mesh, material, kerma, phi_u, phi_c_moments, dose_in=None):
    """Returns (phi_total [G][nz][ny][nx], dose [nz][ny][nx]); dose_in (if given) is accumulated into."""
    mat = np.ascontiguousarray(material, dtype=np.uint8)
    nv = mat.size
    pc = _d(phi_c_moments)
    G, M = pc.shape[0], pc.shape[1]
    tot = np.zeros((G, nv))
    d = np.zeros(nv) if dose_in is None else _d(dose_in).reshape(nv).copy()
    pu = _d(phi_u).reshape(G, nv) if phi_u is not None else None
    ms = _mesh(mesh)
    lib().orc_dose(C.byref(ms), _p(mat), C.c_int(G), C.c_int(M), _p(_d(kerma)), _p(pu), _p(pc.reshape(G, M, nv)),
                   _p(tot), _p(d), C.c_int(0 if dose_in is None else 1))
    return tot.reshape((G,) + mat.shape), d.reshape(mat.shape)


def run_problem(p, source_index=0, n_iter=None, blocked=False):
    """Whole path O1-O5 for one source position of a problem dict from inputs.make_problem.
    Returns dict(phi_u, phi_c (scalar, [G][nz][ny][nx]), phi_total, dose, phi_c_moments, phi_c_abs
    (sum_n w_n |psi_n| of each group's last sweep: the parity tests' conditioning scale))."""
    src = p["sources"][source_index]
    pu = uncollided(p["mesh"], p["material"], p["sigma_t"], src, p["spectrum"])
    pc, pabs = solve(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["quadrature"], p["P_L"],
                     p["n_iter"] if n_iter is None else n_iter, source_pos=src["pos"], phi_u=pu, want_abs=True,
                     blocked=blocked)
    tot, d = dose(p["mesh"], p["material"], p["kerma"], pu, pc)
    return {"phi_u": pu, "phi_c": pc[:, 0], "phi_total": tot, "dose": d, "phi_c_moments": pc, "phi_c_abs": pabs}


def first_collision(mesh, material, sigma_s, L, source_pos, phi_u, q_out):
    """ADDS the first-collision source moments of one source position (O2) into q_out
    [G][M][nz*ny*nx] (float64): q_out[g][lm] += Y_lm(Omega_r) sum_{g'<=g} sigma_sl^{g'->g} phi_u^{g'}."""
    sig_s = _d(sigma_s)
    n_leg, G = sig_s.shape[1] - 1, sig_s.shape[2]
    mat = np.ascontiguousarray(material, dtype=np.uint8)
    pu = _d(phi_u).reshape(G, mat.size)
    pos = _d(source_pos)
    ms = _mesh(mesh)
    assert q_out.dtype == np.float64 and q_out.flags.c_contiguous and q_out.shape == (G, n_moments(L), mat.size)
    for g in range(G):
        lib().orc_first_collision(C.byref(ms), _p(mat), C.c_int(G), C.c_int(n_leg), C.c_int(L), _p(sig_s), _p(pos), _p(pu),
                                  C.c_int(g), C.c_void_p(q_out[g].ctypes.data))


def run_problem_summed(p, source_indices=None, n_iter=None):
    """the given source positions form ONE source. The uncollided fluence
    and the first-collision source moments of the positions are summed (each position with its own direction to
    the cell), then O3-O5 run once. Same keys as run_problem; phi_u is the summed uncollided fluence."""
    idx = list(range(len(p["sources"]))) if source_indices is None else list(source_indices)
    mat = np.ascontiguousarray(p["material"], dtype=np.uint8)
    G, M = np.asarray(p["sigma_t"]).shape[1], n_moments(p["P_L"])
    q_ext = np.zeros((G, M, mat.size))
    pu_sum = np.zeros((G,) + mat.shape)
    for s in idx:
        src = p["sources"][s]
        pu = uncollided(p["mesh"], p["material"], p["sigma_t"], src, p["spectrum"])
        pu_sum += pu
        first_collision(p["mesh"], p["material"], p["sigma_s"], p["P_L"], src["pos"], pu, q_ext)
    pc, pabs = solve(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["quadrature"], p["P_L"],
                     p["n_iter"] if n_iter is None else n_iter, phi_u=None, q_ext=q_ext, want_abs=True)
    tot, d = dose(p["mesh"], p["material"], p["kerma"], pu_sum, pc)
    return {"phi_u": pu_sum, "phi_c": pc[:, 0], "phi_total": tot, "dose": d, "phi_c_moments": pc, "phi_c_abs": pabs}
