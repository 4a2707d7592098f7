"""Thin Python binding of the C ABI in include/dos.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of csrc/libdos.so; PyTorch is used only for device
memory and the stream. There is no CPU fallback: if the library is missing it is built with nvcc, and
if that fails, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .csrc import build as _build

_LIBPATH = _build.build()
_lib = C.CDLL(_LIBPATH)

DOS_OK = 0
STATUS = {0: "DOS_OK", -1: "DOS_ERR_INVALID_ARG", -2: "DOS_ERR_SHAPE", -3: "DOS_ERR_STATE", -4: "DOS_ERR_NOMEM",
          -5: "DOS_ERR_CUDA", -6: "DOS_ERR_UNSUPPORTED"}

EXPORTS = ["dos_workspace_bytes", "dos_create", "dos_set_material_host", "dos_uncollided", "dos_uncollided_batch", "dos_uncollided_sum",
           "dos_uncollided_total", "dos_solve", "dos_solve_tol", "dos_set_boundary", "dos_fluence", "dos_dose", "dos_dose_host", "dos_check", "dos_set_option",
           "dos_profile", "dos_profile_reset", "dos_destroy", "dos_last_error", "dos_uncollided_static", "dos_static_last_error"]


class dos_mesh(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("x0", C.c_double), ("y0", C.c_double), ("z0", C.c_double)]


class dos_xs(C.Structure):
    _fields_ = [("n_mat", C.c_int32), ("n_group", C.c_int32), ("n_leg", C.c_int32),
                ("sigma_t", C.c_void_p), ("sigma_s", C.c_void_p), ("kerma", C.c_void_p)]


class dos_quadrature(C.Structure):
    _fields_ = [("n_ang", C.c_int32), ("mu", C.c_void_p), ("eta", C.c_void_p), ("xi", C.c_void_p), ("w", C.c_void_p)]


class dos_source(C.Structure):
    _fields_ = [("pos", C.c_double * 3), ("axis", C.c_double * 3), ("up", C.c_double * 3),
                ("tan_half_fan", C.c_double), ("tan_half_cone", C.c_double), ("isotropic", C.c_int32)]


class dos_profile_t(C.Structure):
    _fields_ = [("sweep_ms", C.c_double), ("sweep_launches", C.c_int64), ("raytrace_ms", C.c_double),
                ("raytrace_launches", C.c_int64), ("kernel_launches", C.c_int64)]


_lib.dos_workspace_bytes.restype = C.c_int
_lib.dos_workspace_bytes.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.POINTER(C.c_size_t)]
_lib.dos_create.restype = C.c_int
_lib.dos_create.argtypes = [C.POINTER(C.c_void_p), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32,
                            C.c_void_p, C.c_size_t, C.c_void_p]
_lib.dos_set_material_host.restype = C.c_int
_lib.dos_set_material_host.argtypes = [C.c_void_p, C.c_void_p]
_lib.dos_uncollided.restype = C.c_int
_lib.dos_uncollided.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.dos_uncollided_batch.restype = C.c_int
_lib.dos_uncollided_batch.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.dos_uncollided_sum.restype = C.c_int
_lib.dos_uncollided_sum.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]
_lib.dos_solve.restype = C.c_int
_lib.dos_solve.argtypes = [C.c_void_p, C.c_int32]
_lib.dos_solve_tol.restype = C.c_int
_lib.dos_solve_tol.argtypes = [C.c_void_p, C.c_float, C.c_int32, C.c_void_p]
_lib.dos_set_boundary.restype = C.c_int
_lib.dos_set_boundary.argtypes = [C.c_void_p, C.c_int32]
_lib.dos_fluence.restype = C.c_int
_lib.dos_fluence.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
_lib.dos_dose.restype = C.c_int
_lib.dos_dose.argtypes = [C.c_void_p, C.c_void_p, C.c_int32]
_lib.dos_dose_host.restype = C.c_int
_lib.dos_dose_host.argtypes = [C.c_void_p, C.c_void_p, C.c_int32]
_lib.dos_check.restype = C.c_int
_lib.dos_check.argtypes = [C.c_void_p]
_lib.dos_set_option.restype = C.c_int
_lib.dos_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_int64]
_lib.dos_profile.restype = C.c_int
_lib.dos_profile.argtypes = [C.c_void_p, C.c_void_p]
_lib.dos_profile_reset.restype = C.c_int
_lib.dos_profile_reset.argtypes = [C.c_void_p]
_lib.dos_uncollided_total.restype = C.c_int
_lib.dos_uncollided_total.argtypes = [C.c_void_p, C.c_void_p]
_lib.dos_destroy.restype = None
_lib.dos_destroy.argtypes = [C.c_void_p]
_lib.dos_last_error.restype = C.c_char_p
_lib.dos_last_error.argtypes = [C.c_void_p]
_lib.dos_uncollided_static.restype = C.c_int
_lib.dos_uncollided_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p,
                                       C.c_void_p, C.c_void_p, C.c_void_p]
_lib.dos_static_last_error.restype = C.c_char_p
_lib.dos_static_last_error.argtypes = []


class DosError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"{STATUS.get(status, status)}: {message}")
        self.status = status


def library_path() -> str:
    return _LIBPATH


def raw():
    """The ctypes handle (tests use it to probe error paths of the C ABI directly)."""
    return _lib


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _mesh_struct(m):
    return dos_mesh(m["nx"], m["ny"], m["nz"], m["dx"], m["dy"], m["dz"], m["x0"], m["y0"], m["z0"])


def _source_struct(s):
    out = dos_source()
    out.pos[:] = s["pos"]
    out.axis[:] = s["axis"]
    out.up[:] = s["up"]
    out.tan_half_fan = s["tan_half_fan"]
    out.tan_half_cone = s["tan_half_cone"]
    out.isotropic = s["isotropic"]
    return out


def dos_uncollided_static(mesh, material, sigma_t, source, spectrum, phi_u_out, bad_material_out=None, stream=None):
    """Ray trace without a context or workspace (include/dos.h: dos_uncollided_static): nothing is allocated; the
    kernel's scratch is a static device array shared by all calls. material: uint8 device tensor [nz][ny][nx];
    phi_u_out: float32 device tensor [G][nz][ny][nx]; bad_material_out: int32 device tensor of 1 element or None;
    stream: a torch.cuda.Stream (default: the current one). Marshalling only."""
    import torch
    sig = _f32(sigma_t)
    n_mat, G = sig.shape
    m, src, sp = _mesh_struct(mesh), _source_struct(source), _f32(spectrum)
    st = (stream if stream is not None else torch.cuda.current_stream(material.device)).cuda_stream
    rc = _lib.dos_uncollided_static(C.byref(m), material.data_ptr(), n_mat, G, sig.ctypes.data, C.byref(src), sp.ctypes.data,
                                    phi_u_out.data_ptr(), bad_material_out.data_ptr() if bad_material_out is not None else None, st)
    if rc != DOS_OK:
        raise DosError(rc, _lib.dos_static_last_error().decode())


class _Tables:
    """Keeps the host arrays alive while the C structs point at them."""

    def __init__(self, sigma_t, sigma_s, kerma, quad):
        self.sigma_t, self.sigma_s, self.kerma = _f32(sigma_t), _f32(sigma_s), _f32(kerma)
        n_mat, G = self.sigma_t.shape
        n_leg = self.sigma_s.shape[1] - 1
        if self.sigma_s.shape != (n_mat, n_leg + 1, G, G) or self.kerma.shape != (n_mat, G):
            raise ValueError("cross-section table shapes are inconsistent")
        self.xs = dos_xs(n_mat, G, n_leg, self.sigma_t.ctypes.data, self.sigma_s.ctypes.data, self.kerma.ctypes.data)
        self.mu, self.eta, self.xi, self.w = (_f32(quad[k]) for k in ("mu", "eta", "xi", "w"))
        self.quad = dos_quadrature(len(self.w), self.mu.ctypes.data, self.eta.ctypes.data, self.xi.ctypes.data,
                                   self.w.ctypes.data)


def dos_workspace_bytes(mesh, sigma_t, sigma_s, kerma, quad, P_L, n_batch=1) -> int:
    t = _Tables(sigma_t, sigma_s, kerma, quad)
    ms = _mesh_struct(mesh)
    n = C.c_size_t(0)
    st = _lib.dos_workspace_bytes(C.byref(ms), C.byref(t.xs), C.byref(t.quad), P_L, n_batch, C.byref(n))
    if st != DOS_OK:
        raise DosError(st, _lib.dos_last_error(None).decode())
    return n.value


class Context:
    """Owner of one dos_ctx plus the torch tensors (workspace, material ids) it lives in."""

    def __init__(self, mesh, material, sigma_t, sigma_s, kerma, quad, P_L, device="cuda:0", stream=None, n_batch=1):
        import torch
        self.torch = torch
        self.mesh = dict(mesh)
        self.device = torch.device(device)
        self.G = int(np.asarray(sigma_t).shape[1])
        self.n_batch = int(n_batch)
        self.shape = (mesh["nz"], mesh["ny"], mesh["nx"])
        self._tables = _Tables(sigma_t, sigma_s, kerma, quad)
        nbytes = dos_workspace_bytes(mesh, sigma_t, sigma_s, kerma, quad, P_L, n_batch)
        self.workspace_bytes = nbytes
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            mat = np.ascontiguousarray(material, dtype=np.uint8)
            if mat.shape != self.shape:
                raise ValueError("material grid shape must be [nz][ny][nx]")
            self.material = torch.from_numpy(mat).to(self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            ms = _mesh_struct(mesh)
            h = C.c_void_p(None)
            st = _lib.dos_create(C.byref(h), C.byref(ms), self.material.data_ptr(), C.byref(self._tables.xs),
                                 C.byref(self._tables.quad), P_L, self.workspace.data_ptr(), nbytes,
                                 self.stream.cuda_stream)
        if st != DOS_OK:
            raise DosError(st, _lib.dos_last_error(None).decode())
        self.handle = h

    def _check(self, st):
        if st != DOS_OK:
            raise DosError(st, _lib.dos_last_error(self.handle).decode())

    def dos_set_material_host(self, material_host):
        mat = np.ascontiguousarray(material_host, dtype=np.uint8)
        self._check(_lib.dos_set_material_host(self.handle, mat.ctypes.data))

    def dos_uncollided(self, source, spectrum, phi_u_out=None):
        src = _source_struct(source)
        sp = _f32(spectrum)
        ptr = phi_u_out.data_ptr() if phi_u_out is not None else None
        self._check(_lib.dos_uncollided(self.handle, C.byref(src), sp.ctypes.data, ptr))

    def dos_uncollided_batch(self, sources, spectrum, phi_u_out=None):
        """Up to n_batch source positions at once; the following dos_solve sweeps them in the same launches."""
        arr = (dos_source * len(sources))(*[_source_struct(s) for s in sources])
        sp = _f32(spectrum)
        ptr = phi_u_out.data_ptr() if phi_u_out is not None else None
        self._check(_lib.dos_uncollided_batch(self.handle, len(sources), arr, sp.ctypes.data, ptr))

    def dos_uncollided_sum(self, source, spectrum, first, phi_u_out=None):
        src = _source_struct(source)
        sp = _f32(spectrum)
        ptr = phi_u_out.data_ptr() if phi_u_out is not None else None
        self._check(_lib.dos_uncollided_sum(self.handle, C.byref(src), sp.ctypes.data, int(bool(first)), ptr))

    def dos_uncollided_total(self, phi_u_out):
        self._check(_lib.dos_uncollided_total(self.handle, phi_u_out.data_ptr()))

    def dos_solve(self, n_iter):
        self._check(_lib.dos_solve(self.handle, int(n_iter)))

    def dos_solve_tol(self, tol, max_iter):
        """Returns the sweeps done per group (numpy int32 [G])."""
        iters = np.zeros(self.G, dtype=np.int32)
        self._check(_lib.dos_solve_tol(self.handle, float(tol), int(max_iter), iters.ctypes.data))
        return iters

    def dos_set_boundary(self, reflective_faces):
        self._check(_lib.dos_set_boundary(self.handle, int(reflective_faces)))

    def dos_fluence(self, phi_collided=None, phi_total=None):
        self._check(_lib.dos_fluence(self.handle, phi_collided.data_ptr() if phi_collided is not None else None,
                                     phi_total.data_ptr() if phi_total is not None else None))

    def dos_dose(self, dose, accumulate=False):
        self._check(_lib.dos_dose(self.handle, dose.data_ptr(), int(bool(accumulate))))

    def dos_dose_host(self, dose_host, accumulate=False):
        assert dose_host.dtype == np.float32 and dose_host.flags["C_CONTIGUOUS"]
        self._check(_lib.dos_dose_host(self.handle, dose_host.ctypes.data, int(bool(accumulate))))

    def dos_check(self):
        self._check(_lib.dos_check(self.handle))

    def dos_set_option(self, name, value):
        self._check(_lib.dos_set_option(self.handle, name.encode(), int(value)))

    def dos_profile(self):
        p = dos_profile_t()
        self._check(_lib.dos_profile(self.handle, C.byref(p)))
        return {"sweep_ms": p.sweep_ms, "sweep_launches": p.sweep_launches, "raytrace_ms": p.raytrace_ms,
                "raytrace_launches": p.raytrace_launches, "kernel_launches": p.kernel_launches}

    def dos_profile_reset(self):
        self._check(_lib.dos_profile_reset(self.handle))

    def new_field(self, groups=True):
        shape = ((self.G,) if groups else ()) + self.shape
        return self.torch.empty(shape, dtype=self.torch.float32, device=self.device)

    def close(self):
        if getattr(self, "handle", None):
            _lib.dos_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def run_problem(p, source_index=0, n_iter=None, device="cuda:0", ctx=None):
    """Whole hot path for one source position of a problem dict (inputs.make_problem) -> numpy arrays
    phi_u, phi_c, phi_total [G][nz][ny][nx] and dose [nz][ny][nx]."""
    own = ctx is None
    if own:
        ctx = Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"],
                      device=device)
    pu, pc, pt, d = ctx.new_field(), ctx.new_field(), ctx.new_field(), ctx.new_field(groups=False)
    ctx.dos_uncollided(p["sources"][source_index], p["spectrum"], pu)
    ctx.dos_solve(p["n_iter"] if n_iter is None else n_iter)
    ctx.dos_fluence(pc, pt)
    ctx.dos_dose(d, False)
    ctx.dos_check()
    out = {"phi_u": pu.cpu().numpy(), "phi_c": pc.cpu().numpy(), "phi_total": pt.cpu().numpy(), "dose": d.cpu().numpy()}
    if own:
        ctx.close()
    return out


def run_problem_summed(p, source_indices=None, n_iter=None, device="cuda:0"):
    """Summed-source mode (dos_uncollided_sum): all the given source positions form ONE source, one solve.
    Returns the same dict as run_problem (phi_u = the summed uncollided fluence)."""
    idx = list(range(len(p["sources"]))) if source_indices is None else list(source_indices)
    ctx = Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"],
                  device=device, n_batch=max(2, len(idx)))
    pu, pc, pt, d = ctx.new_field(), ctx.new_field(), ctx.new_field(), ctx.new_field(groups=False)
    for n, s in enumerate(idx):
        ctx.dos_uncollided_sum(p["sources"][s], p["spectrum"], first=(n == 0))
    ctx.dos_uncollided_total(pu)                    # the library's own sum over the positions
    ctx.dos_solve(p["n_iter"] if n_iter is None else n_iter)
    ctx.dos_fluence(pc, pt)
    ctx.dos_dose(d, False)
    ctx.dos_check()
    out = {"phi_u": pu.cpu().numpy(), "phi_c": pc.cpu().numpy(), "phi_total": pt.cpu().numpy(), "dose": d.cpu().numpy()}
    ctx.close()
    return out
