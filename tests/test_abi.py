"""Host-side checks of the C ABI (no GPU needed): the library builds for sm_100a, loads,
exports every symbol include/pyr.h declares, validates arguments before touching CUDA, and
fails loudly (PYR_ECUDA, never a CPU fallback) when no device is present."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2602_06688_b200 import build
    return build.build()


def declared_symbols():
    """Function names declared in include/pyr.h (comments stripped)."""
    src = open(os.path.join(ROOT, "include", "pyr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(pyr_[a-z_0-9]+)\s*\(", src)
    return sorted(set(names))


def test_sh_header_symbols_are_exported(libpath):
    src = open(os.path.join(ROOT, "include", "sh.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = sorted(set(re.findall(r"\b(sh_[a-z_0-9]+)\s*\(", src)))
    assert {"sh_plan_create", "sh_compute", "sh_plan_destroy"} <= set(names)
    L = ctypes.CDLL(libpath)
    for n in names:
        assert hasattr(L, n), "libpyr.so does not export %s" % n
    from paper_2602_06688_b200 import sh
    assert sorted(sh.EXPORTS) == names
    # argument validation happens before CUDA is touched
    assert not sh.lib.sh_plan_create(10, 3, 16, 1, 1) and sh.lib.sh_last_error() == 1      # n_sub does not divide P
    assert not sh.lib.sh_plan_create(16, 2, 13, 1, 1) and sh.lib.sh_last_error() == 1      # F odd
    assert not sh.lib.sh_plan_create(80, 2, 64, 1, 1) and sh.lib.sh_last_error() == 2      # p = 40 > 32
    assert sh.lib.sh_compute(None, None, None, None, None, None, None) == 1


def test_chain_header_symbols_are_exported(libpath):
    src = open(os.path.join(ROOT, "include", "chain.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = sorted(set(re.findall(r"\b((?:atmo|ccd|pupdata|modalrec|chain)_[a-z_0-9]+)\s*\(", src)))
    assert {"atmo_propagate", "ccd_integrate", "pupdata_from_frame", "modalrec_compute"} <= set(names)
    L = ctypes.CDLL(libpath)
    for n in names:
        assert hasattr(L, n), "libpyr.so does not export %s" % n
    from paper_2602_06688_b200 import chain
    assert sorted(chain.EXPORTS) == names
    # argument validation happens before CUDA is touched
    assert not chain.lib.atmo_plan_create(0, 8, 8, 1) and chain.lib.chain_last_error() == 1
    assert not chain.lib.atmo_plan_create(40, 8, 8, 4) and chain.lib.chain_last_error() == 2     # 160 > 128 shifts
    assert not chain.lib.ccd_plan_create(0, 1, 1, 1, 0.4, 0.0, 16, 1) and chain.lib.chain_last_error() == 1
    assert not chain.lib.ccd_plan_create(16, 1, 1, 1, -1.0, 0.0, 16, 1) and chain.lib.chain_last_error() == 1
    assert not chain.lib.modalrec_plan_create(0, 4, None, None, 1) and chain.lib.chain_last_error() == 1
    assert chain.lib.modalrec_compute(None, None, None, None) == 1
    assert chain.lib.atmo_propagate(None, None, None, None, None) == 1


def test_header_declares_the_three_north_star_calls():
    names = declared_symbols()
    for n in ("pyr_plan_create", "pyr_compute", "pyr_plan_destroy"):
        assert n in names


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    names = declared_symbols()
    assert len(names) >= 8
    for n in names:
        assert hasattr(L, n), "libpyr.so does not export %s" % n


def test_binding_lists_the_same_symbols(libpath):
    from paper_2602_06688_b200 import pyr
    assert sorted(pyr.EXPORTS) == declared_symbols()


def test_no_torch_or_cufft_linkage(libpath):
    """The boundary is a plain C library: no torch, no cuFFT among its dynamic dependencies."""
    import subprocess
    out = subprocess.run(["ldd", libpath], capture_output=True, text=True).stdout.lower()
    for bad in ("torch", "cufft", "c10", "python"):
        assert bad not in out


INVALID = [
    # (P, N, M, r, b, B)
    (32, 102, 8, 3.0, 2, 1),     # N not a multiple of 4
    (32, 8, 8, 3.0, 2, 1),       # N too small
    (32, 4096, 8, 3.0, 2, 1),    # N too large
    (33, 128, 8, 3.0, 1, 1),     # P odd
    (0, 128, 8, 3.0, 2, 1),      # P < 2
    (66, 128, 8, 3.0, 1, 1),     # P > N/2
    (32, 128, 0, 3.0, 2, 1),     # M < 1
    (32, 128, 8, -1.0, 2, 1),    # r < 0
    (32, 128, 8, float("nan"), 2, 1),
    (32, 128, 8, float("inf"), 2, 1),
    (32, 128, 8, 3.0, 0, 1),     # b < 1
    (32, 128, 8, 3.0, 3, 1),     # b does not divide N/4
    (30, 128, 8, 3.0, 2, 1),     # b does not divide N/4 - P/2 = 17
    (32, 128, 8, 3.0, 2, 0),     # B < 1
]


@pytest.mark.parametrize("args", INVALID)
def test_plan_create_rejects_bad_arguments(libpath, args):
    from paper_2602_06688_b200 import pyr
    P, N, M, r, b, B = args
    h = pyr.lib.pyr_plan_create(P, N, M, r, b, B)
    assert not h
    code, msg = pyr.last_error()
    assert code == pyr.PYR_EINVAL and msg


def test_null_arguments(libpath):
    from paper_2602_06688_b200 import pyr
    assert pyr.lib.pyr_compute(None, None, None, None, None, None) == pyr.PYR_EINVAL
    assert pyr.lib.pyr_compute_host(None, None, None, None, None, None) == pyr.PYR_EINVAL
    assert pyr.lib.pyr_plan_set_valid(None, None) == pyr.PYR_EINVAL
    assert pyr.lib.pyr_plan_set_mask_separable(None, None, None) == pyr.PYR_EINVAL
    assert pyr.lib.pyr_plan_get_dims(None, None, None, None) == pyr.PYR_EINVAL
    assert pyr.lib.pyr_test_line_conv(None, None, None, 1, None) == pyr.PYR_EINVAL
    assert pyr.lib.pyr_plan_launches_per_compute(None) == 0
    pyr.lib.pyr_plan_destroy(None)   # no-op


def test_no_cpu_fallback_without_a_device(libpath):
    """On a box without a GPU a valid request must fail with PYR_ECUDA, not compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2602_06688_b200 import pyr
    with pytest.raises(pyr.PyrError) as ei:
        pyr.Plan(32, 128, 8, 3.0, 2, 1)
    assert ei.value.code == pyr.PYR_ECUDA


def test_product_does_not_import_the_oracle():
    """Neither side imports, links or includes the other (the seeded generator `synth`,
    which holds none of the method's arithmetic, serves both)."""
    pkg = os.path.join(ROOT, "paper_2602_06688_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                for bad in ("import oracle", "from oracle", "liboracle", "pyr_oracle"):
                    assert bad not in txt, "%s refers to the oracle (%s)" % (f, bad)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            for bad in ("import paper_2602_06688_b200", "from paper_2602_06688_b200", "pyr.h",
                        "libpyr.so", "pyr_fft"):
                assert bad not in txt, "oracle/%s refers to the CUDA path (%s)" % (f, bad)
