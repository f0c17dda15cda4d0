"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/hz.h declares, and its
host logic (argument validation, memory plan, error strings) behaves as the header says.  No compute
call is made: there is no GPU here and no CPU fallback exists."""
import ctypes as C
import os
import re

import pytest

import paper_1102_5202_b200 as pkg
from paper_1102_5202_b200 import binding as B
from paper_1102_5202_b200 import build as hz_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    hz_build.build()
    return pkg.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "hz.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hz_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(L):
    names = declared_symbols()
    assert len(names) >= 15
    for n in names:
        assert hasattr(L, n), n
    assert sorted(B.SYMBOLS) == names  # the binding covers exactly the header


def test_default_params(L):
    p = B.HzParams()
    assert L.hz_default_params(C.byref(p)) == 0
    assert abs(p.gamma_ad - 4.0 / 3.0) < 1e-15 and p.cleaning == 1 and p.c2p_maxit == 30
    assert p.rho_atm == 1e-12 and p.p_atm == 1e-14 and p.atm_tol == 1e-3 and p.kappa == 1.0
    assert L.hz_default_params(None) == B.HZ_EINVAL


def grid(nx, ny, nz, dx=1.0, bc=(0, 0, 0)):
    return B.HzGrid(nx, ny, nz, dx, dx, dx, (C.c_int * 3)(*bc))


def test_state_bytes_plan(L):
    n = C.c_size_t()
    # 46 resident padded fields + staging: between 46 and 80 interior-field sizes at 256^3 fp64
    assert L.hz_state_bytes(C.byref(grid(256, 256, 256)), B.HZ_F64, C.byref(n)) == 0
    one = 256 ** 3 * 8
    assert 46 * one < n.value < 80 * one
    n32 = C.c_size_t()
    assert L.hz_state_bytes(C.byref(grid(256, 256, 256)), B.HZ_F32, C.byref(n32)) == 0
    assert 0.45 * n.value < n32.value < 0.6 * n.value
    # the mixed mode (fp32 storage, fp64 phase 2) stores exactly what fp32 stores
    nmix = C.c_size_t()
    assert L.hz_state_bytes(C.byref(grid(256, 256, 256)), B.HZ_F32_F64, C.byref(nmix)) == 0
    assert nmix.value == n32.value
    # an inactive axis carries no ghosts: the tube is tiny
    assert L.hz_state_bytes(C.byref(grid(400, 1, 1)), B.HZ_F64, C.byref(n)) == 0
    assert n.value < 1 << 20
    # 384^3 fp64 (largest BASELINE grid) fits a 180 GB B200 many times over
    assert L.hz_state_bytes(C.byref(grid(384, 384, 384)), B.HZ_F64, C.byref(n)) == 0
    assert n.value < 40e9


def test_state_bytes_for_matches_the_layout_built(L):
    """hz_state_bytes_for sizes the context for the reconstruction it is created with (the
    3-ghost PPM size was allocated for every context): MC needs less than the upper bound hz_state_bytes, PPM
    exactly it; at 256^3 in fp64 the MC context is the 46 + 4 + 10 resident fields DESIGN.md section 4 lists."""
    nmc, nppm, nup = C.c_size_t(), C.c_size_t(), C.c_size_t()
    g = grid(256, 256, 256)
    mc, ppm = B.HzParams.default(), B.HzParams.default(recon=1)
    assert L.hz_state_bytes_for(C.byref(g), B.HZ_F64, C.byref(mc), C.byref(nmc)) == 0
    assert L.hz_state_bytes_for(C.byref(g), B.HZ_F64, C.byref(ppm), C.byref(nppm)) == 0
    assert L.hz_state_bytes(C.byref(g), B.HZ_F64, C.byref(nup)) == 0
    assert nmc.value < nppm.value == nup.value
    assert L.hz_state_bytes_for(C.byref(g), B.HZ_F64, None, C.byref(nup)) == 0 and nup.value == nmc.value
    field = (256 + 4) * (16 + 256 + 16) * (256 + 4) * 8          # padded rows, 2 ghost layers
    assert 50 * field < nmc.value < 50 * field + 10.5 * 256 ** 3 * 8 + (1 << 22)   # + host staging, scratch
    # a 2-cell axis is fine with MC, too short for PPM's 3 ghost layers
    g2 = grid(8, 2, 8)
    assert L.hz_state_bytes_for(C.byref(g2), B.HZ_F64, C.byref(mc), C.byref(nmc)) == 0
    assert L.hz_state_bytes_for(C.byref(g2), B.HZ_F64, C.byref(ppm), C.byref(nppm)) == B.HZ_EINVAL


@pytest.mark.parametrize("g,dtype", [
    (grid(0, 4, 4), 1), (grid(4, -1, 4), 1), (grid(4, 4, 4, dx=0.0), 1), (grid(4, 4, 4, dx=float("nan")), 1),
    (grid(4, 4, 4, bc=(0, 7, 0)), 1), (grid(4, 4, 4), 5),
])
def test_bad_grid_is_einval(L, g, dtype):
    n = C.c_size_t()
    assert L.hz_state_bytes(C.byref(g), dtype, C.byref(n)) == B.HZ_EINVAL
    h = C.c_void_p()
    assert L.hz_create(C.byref(g), dtype, None, None, C.byref(h)) == B.HZ_EINVAL
    assert not h.value


def test_bad_params_is_einval(L):
    h = C.c_void_p()
    p = B.HzParams.default(gamma_ad=1.0)
    assert L.hz_create(C.byref(grid(8, 8, 8)), 1, C.byref(p), None, C.byref(h)) == B.HZ_EINVAL
    p = B.HzParams.default(c2p_maxit=0)
    assert L.hz_create(C.byref(grid(8, 8, 8)), 1, C.byref(p), None, C.byref(h)) == B.HZ_EINVAL


def test_no_gpu_means_ecuda_not_a_fallback(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    assert L.hz_create(C.byref(grid(8, 8, 8)), 1, None, None, C.byref(h)) == B.HZ_ECUDA
    assert not h.value
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        pkg.Horizon((8, 8, 8), (1, 1, 1), (0, 0, 0))


def test_null_handles(L):
    assert L.hz_step(None, 0.1, 1) == B.HZ_EINVAL
    assert L.hz_substeps(None, 0.1, 1) == B.HZ_EINVAL
    assert L.hz_set_metric(None, None, None, None) == B.HZ_EINVAL
    assert L.hz_set_primitives(None, None) == B.HZ_EINVAL
    assert L.hz_get_primitives(None, None) == B.HZ_EINVAL
    assert L.hz_diagnostics(None, None) == B.HZ_EINVAL
    assert L.hz_destroy(None) == 0
    assert L.hz_launch_count(None) == 0


def test_strerror(L):
    seen = set()
    for code in (0, -1, -2, -3, -4):
        s = L.hz_strerror(code).decode()
        assert s and s not in seen
        seen.add(s)
    assert L.hz_strerror(-99).decode() == "unknown error"
    assert [L.hz_kernel_name(k).decode() for k in range(B.HZ_NKERNELS)][0]


def test_product_path_does_not_touch_the_oracle():
    """The package and bench.py's product arm must not import oracle/ (DESIGN.md section 6)."""
    pkgdir = os.path.join(ROOT, "paper_1102_5202_b200")
    for dirpath, _, files in os.walk(pkgdir):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "hzo" not in txt and "import oracle" not in txt and "from oracle" not in txt, f
    wtxt = open(os.path.join(ROOT, "workloads", "__init__.py")).read()
    assert "import oracle" not in wtxt and "from oracle" not in wtxt and "import paper_1102" not in wtxt
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1102_5202_b200" not in txt and "from paper_1102_5202_b200" not in txt, f
            assert '#include "../' not in txt and "csrc" not in txt.replace("paper_1102_5202_b200/csrc", ""), f
