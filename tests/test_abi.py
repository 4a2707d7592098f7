"""CPU-only checks of the C-ABI boundary (include/dos.h <-> csrc/libdos.so <-> the Python binding).

No compute call is made here: only symbol presence, struct layout, and the argument validation that
runs on the host before any CUDA call.
"""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "dos.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dos_[a-z_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_1811_12391_b200 import dos
    lib = C.CDLL(dos.library_path())
    names = _declared()
    assert {"dos_create", "dos_uncollided", "dos_solve", "dos_dose", "dos_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/dos.h but not exported"
    assert sorted(dos.EXPORTS) == names, "binding's EXPORTS list and include/dos.h disagree"


def test_library_is_sm100a_and_not_linked_to_the_oracle():
    from paper_1811_12391_b200 import dos
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", dos.library_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    ldd = subprocess.run(["ldd", dos.library_path()], capture_output=True, text=True).stdout
    assert "oracle" not in ldd


def test_product_sources_do_not_reference_the_oracle():
    pkg = os.path.join(ROOT, "paper_1811_12391_b200")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                src = open(os.path.join(d, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", src, flags=re.M), f
                assert "dos_oracle" not in src and "libdos_oracle" not in src, f


def _problem():
    from paper_1811_12391_b200.inputs import make_problem
    return make_problem("config1")


def test_struct_layouts_match_the_header():
    from paper_1811_12391_b200 import dos
    assert C.sizeof(dos.dos_mesh) == 3 * 4 + 4 + 6 * 8          # 3 int32, pad, 6 double
    assert C.sizeof(dos.dos_source) == 9 * 8 + 2 * 8 + 8        # 3x3 double, 2 double, int32 + pad
    assert C.sizeof(dos.dos_xs) == 16 + 3 * 8
    assert C.sizeof(dos.dos_quadrature) == 8 + 4 * 8


def test_workspace_bytes_and_host_side_validation():
    from paper_1811_12391_b200 import dos
    p = _problem()
    n = dos.dos_workspace_bytes(p["mesh"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"])
    nv = 16 ** 3
    assert n >= 4 * nv * 4 * (p["n_group"] + 2)                  # moments of all groups + Q_fix + Q
    with pytest.raises(dos.DosError) as e:
        dos.dos_workspace_bytes(p["mesh"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], 3)
    assert e.value.status == -2                                  # P_L > n_leg -> DOS_ERR_SHAPE
    bad = dict(p["mesh"], nx=0)
    with pytest.raises(dos.DosError) as e:
        dos.dos_workspace_bytes(bad, p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], 1)
    assert e.value.status == -1
    # n_batch > 1 adds the summed-source buffers: [G][Nv][MP] + [G][Nv] floats (MP = 4 at P1)
    n2 = dos.dos_workspace_bytes(p["mesh"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], 1, n_batch=2)
    assert n2 >= n + 4 * nv * p["n_group"] * (4 + 1)
    with pytest.raises(dos.DosError) as e:
        dos.dos_workspace_bytes(p["mesh"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], 1, n_batch=0)
    assert e.value.status == -1
    q = {k: (v[:20] if k in ("mu", "eta", "xi", "w") else v) for k, v in p["quadrature"].items()}
    with pytest.raises(dos.DosError) as e:
        dos.dos_workspace_bytes(p["mesh"], p["sigma_t"], p["sigma_s"], p["kerma"], q, 1)
    assert e.value.status == -1                                  # n_ang not a multiple of 8


def test_create_rejects_bad_tables_before_touching_cuda():
    """dos_create validates host tables first; with fake (never dereferenced) device pointers the
    failures below must come back as statuses, not crashes, on a box without a GPU."""
    from paper_1811_12391_b200 import dos
    lib = dos.raw()
    p = _problem()
    ms = dos._mesh_struct(p["mesh"])
    h = C.c_void_p(None)
    fake_dev = C.c_void_p(0x10000)          # 256-aligned, never dereferenced on these paths

    def create(sigma_t=None, sigma_s=None, quad=None, ws=fake_dev, mat=fake_dev, nbytes=1 << 40):
        t = dos._Tables(p["sigma_t"] if sigma_t is None else sigma_t, p["sigma_s"] if sigma_s is None else sigma_s,
                        p["kerma"], p["quadrature"] if quad is None else quad)
        st = lib.dos_create(C.byref(h), C.byref(ms), mat, C.byref(t.xs), C.byref(t.quad), 1, ws, nbytes, None)
        return st, lib.dos_last_error(None).decode()

    st, msg = create(sigma_t=np.zeros_like(p["sigma_t"]))
    assert st == -1 and "sigma_t" in msg
    up = p["sigma_s"].copy()
    up[0, 0, 2, 1] = 0.1                                         # upscatter entry
    st, msg = create(sigma_s=up)
    assert st == -1 and "upscatter" in msg
    q = dict(p["quadrature"])
    q["w"] = q["w"] * np.float32(1.01)
    st, msg = create(quad=q)
    assert st == -1 and "sum to 1" in msg
    q = dict(p["quadrature"])
    q["mu"] = q["mu"][::-1].copy()
    st, msg = create(quad=q)
    assert st == -1 and "octant" in msg
    st, msg = create(ws=C.c_void_p(0x10010))
    assert st == -1 and "aligned" in msg
    st, msg = create(mat=None)
    assert st == -1
    st, msg = create(nbytes=1024)
    assert st == -2 and "workspace" in msg
    assert h.value is None


def test_null_context_calls_return_status():
    from paper_1811_12391_b200 import dos
    lib = dos.raw()
    assert lib.dos_solve(None, 3) == -1
    assert lib.dos_dose(None, None, 0) == -1
    assert lib.dos_uncollided(None, None, None, None) == -1
    assert lib.dos_check(None) == -1
    lib.dos_destroy(None)                                        # no-op


def test_static_entry_point_validates_before_touching_cuda():
    """dos_uncollided_static (no context, no workspace, scratch in a static device array): null arguments and sizes
    beyond the scratch are refused on the host, with a message, before any CUDA call (so this runs without a GPU)."""
    import ctypes as C
    import numpy as np
    from paper_1811_12391_b200 import dos
    from paper_1811_12391_b200.inputs import make_problem
    lib = dos.raw()
    assert lib.dos_uncollided_static(None, None, 2, 4, None, None, None, None, None, None) == -1
    p = make_problem("config1")
    mesh, src = dos._mesh_struct(p["mesh"]), dos._source_struct(p["sources"][0])
    fake = C.c_void_p(256)                                     # never dereferenced: the size check comes first
    sig = np.ones((2, 65), np.float32)
    sp = np.ones(65, np.float32)
    rc = lib.dos_uncollided_static(C.byref(mesh), fake, 2, 65, sig.ctypes.data, C.byref(src), sp.ctypes.data, fake, None, None)
    assert rc == -6 and b"exceeds the static scratch" in lib.dos_static_last_error()
    sig = np.ones((17, 4), np.float32)
    rc = lib.dos_uncollided_static(C.byref(mesh), fake, 17, 4, sig.ctypes.data, C.byref(src), sp.ctypes.data, fake, None, None)
    assert rc == -6
    sig = np.zeros((2, 4), np.float32)                         # sigma_t must be > 0
    rc = lib.dos_uncollided_static(C.byref(mesh), fake, 2, 4, sig.ctypes.data, C.byref(src), sp.ctypes.data, fake, None, None)
    assert rc == -1 and b"sigma_t" in lib.dos_static_last_error()
    # the header states the scratch size the library holds per GPU
    text = open(os.path.join(ROOT, "include", "dos.h")).read()
    assert "#define DOS_STATIC_SCRATCH_BYTES 4352" in text


def test_paper_shaped_workload_has_the_papers_shape():
    """7 groups with edges 100/75/70/60/45/30/20/10 keV, a 50 x 50 x 12.5 cm box on
    64x64x16 or 256x256x64 voxels, 16 source positions, S6/P0 by default; spectrum normalised per source particle."""
    import numpy as np
    from paper_1811_12391_b200.inputs import make_problem
    p = make_problem("paper_coarse")
    m = p["mesh"]
    assert (m["nx"], m["ny"], m["nz"]) == (64, 64, 16) and abs(m["nx"] * m["dx"] - 50.0) < 1e-12 and abs(m["nz"] * m["dz"] - 12.5) < 1e-12
    assert list(p["edges"]) == [100.0, 75.0, 70.0, 60.0, 45.0, 30.0, 20.0, 10.0] and p["n_group"] == 7
    assert len(p["sources"]) == 16 and len(p["quadrature"]["w"]) == 48 and p["P_L"] == 0
    assert abs(float(np.sum(p["spectrum"], dtype=np.float64)) - 1.0) < 1e-6
    assert p["sigma_s"].shape == (2, 1, 7, 7) and np.all(np.triu(p["sigma_s"][1, 0]) == p["sigma_s"][1, 0])    # downscatter only
    f = make_problem("paper_fine", n_pos=1)
    assert (f["mesh"]["nx"], f["mesh"]["nz"]) == (256, 64) and abs(f["mesh"]["dx"] - 50.0 / 256) < 1e-12
