"""CPU-side checks of the product's boundary: the C-ABI library builds for sm_100a, loads without
a GPU, exports every function include/mm.h declares, validates arguments before touching CUDA,
and refuses to compute without a device (no CPU fallback).  No compute calls here."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def mm():
    from paper_2401_15233_b200 import mm as _mm
    _mm.lib()
    return _mm


def declared_functions(header="mm.h"):
    text = (ROOT / "include" / header).read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mm_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(mm):
    names = declared_functions()
    assert len(names) >= 14 and set(names) == set(mm.EXPORTS)
    lib = mm.lib()
    for n in names:
        assert getattr(lib, n) is not None
    # the measurement hooks live in their own header and library (they allocate device scratch)
    bnames = declared_functions("mm_bench.h")
    assert set(bnames) == set(mm.BENCH_EXPORTS) and not set(bnames) & set(names)
    blib = mm.bench_lib()
    for n in bnames:
        assert getattr(blib, n) is not None
        assert not hasattr(lib, n)


def test_product_library_never_allocates_device_memory():
    """include/mm.h: "the library never allocates device memory" -- no cudaMalloc* in what builds libmm.so."""
    from paper_2401_15233_b200 import build_ext
    for f in build_ext.DEPS:
        text = (build_ext.CSRC / f).resolve().read_text()
        assert not re.search(r"\bcudaMalloc|\bcudaFree\b|cudaHostAlloc", text), f


def test_binding_structs_match_header(mm):
    # field order / count of the header structs (layout is plain C, natural alignment)
    text = (ROOT / "include" / "mm.h").read_text()
    assert "typedef struct { int system; int nx, ny; double x0, x1, y0, y1; } mm_grid;" in text
    assert [f[0] for f in mm.mm_grid._fields_] == ["system", "nx", "ny", "x0", "x1", "y0", "y1"]
    assert [f[0] for f in mm.mm_collision._fields_] == ["model", "tau", "Kn", "L_ref", "rho_ref"]
    assert [f[0] for f in mm.mm_bc._fields_] == ["type", "nbands", "band_lo", "band_hi", "band_W", "default_W", "band_state"]
    assert "typedef struct { double R_gas; } mm_gas;" in text and [f[0] for f in mm.mm_gas._fields_] == ["R_gas"]
    assert re.search(r"int mm_create\(mm_solver \*\*out, const mm_grid \*grid, const mm_gas \*gas, const mm_collision \*collision,", text)
    assert [f[0] for f in mm.mm_options._fields_] == ["sigma_lim", "ws_scale", "limiter", "shared_limiter", "flux", "source_scheme", "time_scheme", "stream"]
    for name, val in [("MM_SYS5_1D", 5), ("MM_SYS14_2D", 14), ("MM_MAX_BANDS", 8)]:
        assert re.search(rf"{name}\s*=?\s*{val}\b", text)


def test_workspace_bytes_and_argument_checks(mm):
    lib = mm.lib()
    n = mm.mm_workspace_bytes(14, 2048, 2048)
    # two padded state copies of 14 planes, each as conserved moments and as primitives, dominate
    planes = 4 * 14 * (2048 + 4) * 2064 * 8
    assert planes <= n <= planes + 600000         # + control block, boundary tables, a/b table, dt history
    assert mm.mm_workspace_bytes(5, 1000, 1) > 2 * 5 * 1004 * 5 * 8
    assert mm.mm_workspace_bytes(5, 10, 2) == 0          # 1-D system needs ny = 1
    assert mm.mm_workspace_bytes(7, 10, 10) == 0
    assert mm.mm_workspace_bytes(14, 0, 4) == 0
    assert lib.mm_strerror(0) == b"ok" and b"invalid" in lib.mm_strerror(-1)
    # NULL / bad arguments are rejected before any CUDA call
    g = mm.mm_grid(14, 8, 8, 0, 1, 0, 1)
    c = mm.mm_collision(0, 0, 0, 1, 1)
    o = mm.mm_options(1e-4, 1.0, 1, 0, 0, 0, 0, None)
    b = (mm.mm_bc * 4)()
    h = C.c_void_p()
    gas = mm.mm_gas(287.0)
    assert lib.mm_create(C.byref(h), C.byref(g), C.byref(gas), C.byref(c), b, C.byref(o), None, 0) == mm.EWORKSPACE
    assert lib.mm_create(C.byref(h), C.byref(g), None, C.byref(c), b, C.byref(o), None, 0) == mm.EWORKSPACE    # gas NULL: R = 1
    gas.R_gas = 0.0
    assert lib.mm_create(C.byref(h), C.byref(g), C.byref(gas), C.byref(c), b, C.byref(o), None, 0) == mm.EINVAL
    o.sigma_lim = -1.0
    assert lib.mm_create(C.byref(h), C.byref(g), None, C.byref(c), b, C.byref(o), None, 0) == mm.EINVAL
    assert lib.mm_step(None, 1, 0.4) == mm.EINVAL
    assert lib.mm_launch_count(None) == 0


def test_no_cpu_fallback(mm):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(mm.MMError) as e:
        mm.Solver(14, 8, 8)
    assert e.value.status == mm.ECUDA
    # the C entry point itself also refuses: aligned fake workspace, still no device
    lib = mm.lib()
    g = mm.mm_grid(5, 8, 1, 0, 1, 0, 1)
    c = mm.mm_collision(0, 0, 0, 1, 1)
    o = mm.mm_options(1e-4, 1.0, 1, 0, 0, 0, 0, None)
    b = (mm.mm_bc * 4)()
    h = C.c_void_p()
    n = lib.mm_workspace_bytes(C.byref(g))
    assert lib.mm_create(C.byref(h), C.byref(g), None, C.byref(c), b, C.byref(o), C.c_void_p(4096), n) == mm.ECUDA
    assert b"CUDA" in lib.mm_strerror(mm.ECUDA)


def test_product_does_not_touch_the_oracle():
    for f in (ROOT / "paper_2401_15233_b200").rglob("*"):
        if f.suffix in (".py", ".cu", ".cuh", ".h"):
            assert "oracle" not in f.read_text().lower().replace("no cpu", ""), f
    assert "mmo" not in (ROOT / "include" / "mm.h").read_text()


def test_launch_decomposition_host_logic(mm):
    """Strips x row chunks of the 14-moment step kernel (no device needed): every cell is covered,
    the items fill whole waves of the resident warps as well as the grid allows, and no chunk is empty."""
    for nx, ny in [(2048, 2048), (4096, 4096), (512, 512), (1200, 1200), (4096, 4), (33, 9), (1, 1), (70, 37)]:
        for zsym in (True, False):
            ns, nc, w = mm.mm_decomposition(nx, ny, zsym, 148)
            assert ns == -(-nx // 30) and 1 <= nc <= ny and w >= 8
            slots = 148 * w                           # one work item per warp (mm_tm14.cuh)
            waves = -(-ns * nc // slots)
            rows = -(-ny // nc)
            # never worse than one chunk per strip, and within 15 % of the ideal split on large grids
            # (20 % at 512^2, where a chunk is only ~6 rows and whole rows are the granularity)
            assert waves * (rows + 0.8) <= -(-ns // slots) * (ny + 0.8) + 1e-9
            if nx * ny >= 512 * 512:
                ideal = ns * (ny + 0.8 * nc) / slots
                assert waves * (rows + 0.8) <= (1.15 if nx * ny >= 1024 * 1024 else 1.2) * ideal
    assert mm.mm_decomposition(2048, 2048, True, 148)[::2] == (69, 16)
    with pytest.raises(mm.MMError):
        mm.mm_decomposition(0, 5)

