"""Host-side checks of the C ABI that need no GPU: the library loads, exports every symbol
include/vipir.h declares, and rejects bad arguments before touching CUDA."""
import ctypes
import re
from pathlib import Path

import pytest

from paper_2606_11536_b200 import build, vipir

ROOT = Path(__file__).resolve().parents[1]


@pytest.fixture(scope="module")
def lib():
    build.build()
    return vipir.load()


def _declared(header_name):
    header = (ROOT / "include" / header_name).read_text()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)  # declarations only, not comments
    return set(re.findall(r"\b(vipir_[a-z0-9_]+)\s*\(", header))


def test_header_symbols_are_exported(lib):
    assert sorted(f.name for f in (ROOT / "include").glob("*.h")) == ["vipir.h", "vipir_testing.h"]
    declared = _declared("vipir.h")
    assert declared == set(vipir.SYMBOLS), declared ^ set(vipir.SYMBOLS)
    testing = _declared("vipir_testing.h")
    assert testing == set(vipir.TESTING_SYMBOLS), testing ^ set(vipir.TESTING_SYMBOLS)
    for name in declared | testing:
        assert hasattr(lib, name), name


def test_library_never_reads_the_environment():
    """No getenv in the product: every planner override is an explicit vipir_tuning argument."""
    for f in (ROOT / "paper_2606_11536_b200" / "csrc").glob("*.cu*"):
        assert "getenv" not in f.read_text(), f


def test_tuning_domain_is_checked_before_any_device_call(lib):
    def st(**fields):
        h = ctypes.c_void_p()
        tune = vipir.Tuning(**fields)
        return lib.vipir_dbmul_plan_tuned(ctypes.byref(h), 256, 1024, 8, 8, None, 0, 0, ctypes.byref(tune))
    for bad in (dict(m_sub=3), dict(m_sub=8), dict(tile_queries=129), dict(k_atoms=9), dict(stages=1), dict(stages=13),
                dict(separate_split=2), dict(whole_units=2), dict(no_collector=2), dict(host_staged=2), dict(host_slices=5)):
        assert st(**bad) == vipir.ERR_INVALID_ARG, bad
    tune = vipir.Tuning()
    tune.reserved[3] = 1
    h = ctypes.c_void_p()
    assert lib.vipir_dbmul_plan_tuned(ctypes.byref(h), 256, 1024, 8, 8, None, 0, 0, ctypes.byref(tune)) == vipir.ERR_INVALID_ARG

    def mg(**fields):
        h = ctypes.c_void_p()
        tune = vipir.ModGemmTuning(**fields)
        q = (ctypes.c_uint32 * 1)(97)
        return lib.vipir_modgemm_plan_create_tuned(ctypes.byref(h), 1, 2, 128, 128, 8, 0, q, ctypes.byref(tune))
    for bad in (dict(cta_group=3), dict(tile_cols=12), dict(tile_cols=72), dict(a_stages=3), dict(a_stages=25), dict(c_split=3), dict(r_stages=1), dict(r_stages=5),
                dict(b_stages=1), dict(b_stages=5)):
        assert mg(**bad) == vipir.ERR_INVALID_ARG, bad


def test_status_strings(lib):
    names = [lib.vipir_status_str(i).decode() for i in range(6)]
    assert names == ["VIPIR_OK", "VIPIR_ERR_INVALID_ARG", "VIPIR_ERR_UNSUPPORTED", "VIPIR_ERR_ALLOC",
                     "VIPIR_ERR_CUDA", "VIPIR_ERR_ARCH"]
    assert lib.vipir_status_str(99).decode() == "VIPIR_ERR_UNKNOWN"


def test_destroy_null_is_noop(lib):
    lib.vipir_destroy(None)


def _plan_status(lib, rows, cols, batch, db_bits, moduli=None, regime=0, count=None):
    h = ctypes.c_void_p()
    spec_p = None
    if moduli is not None or count is not None:
        arr = (ctypes.c_uint32 * max(1, len(moduli or [])))(*(moduli or [0]))
        spec = vipir.ModulusSpec(len(moduli) if count is None else count, arr if moduli is not None else None)
        spec_p = ctypes.byref(spec)
    st = lib.vipir_dbmul_plan_ex(ctypes.byref(h), rows, cols, batch, db_bits, spec_p, regime)
    assert st != vipir.OK or h.value
    if st == vipir.OK:
        lib.vipir_destroy(h)
    return st


@pytest.mark.parametrize("args", [
    dict(rows=0, cols=16, batch=1, db_bits=8),
    dict(rows=16, cols=0, batch=1, db_bits=8),
    dict(rows=16, cols=16, batch=0, db_bits=8),
    dict(rows=16, cols=16, batch=1, db_bits=12),
    dict(rows=16, cols=16, batch=1, db_bits=8, moduli=[1]),
    dict(rows=16, cols=16, batch=1, db_bits=8, moduli=[1 << 30]),
    dict(rows=16, cols=16, batch=1, db_bits=8, moduli=[97, 101, 103, 107, 109]),
    dict(rows=16, cols=16, batch=1, db_bits=8, count=2),  # count > 0 with a null moduli pointer
    dict(rows=16, cols=16, batch=1, db_bits=8, regime=9),
])
def test_invalid_arguments(lib, args):
    assert _plan_status(lib, **args) == vipir.ERR_INVALID_ARG


@pytest.mark.parametrize("args", [
    dict(rows=16, cols=24, batch=1, db_bits=8),        # row bytes not a multiple of 16
    dict(rows=16, cols=4, batch=1, db_bits=16),
    dict(rows=1 << 31, cols=16, batch=1, db_bits=8),   # beyond the stated size limit
    dict(rows=16, cols=1 << 31, batch=1, db_bits=8),
])
def test_unsupported_shapes(lib, args):
    assert _plan_status(lib, **args) == vipir.ERR_UNSUPPORTED


def test_null_out_pointer(lib):
    assert lib.vipir_dbmul_plan_ex(None, 16, 16, 1, 8, None, 0) == vipir.ERR_INVALID_ARG
    assert lib.vipir_dbmul(None, None, None, None, None) == vipir.ERR_INVALID_ARG
    assert lib.vipir_dbmul_host(None, None, None, None, None) == vipir.ERR_INVALID_ARG
    assert lib.vipir_plan_info(None, None) == vipir.ERR_INVALID_ARG
    assert lib.vipir_split_limbs(None, None, None, None) == vipir.ERR_INVALID_ARG
    assert lib.vipir_dbmul_scan(None, None, None, None) == vipir.ERR_INVALID_ARG
    assert lib.vipir_plan_set_modswitch(None, 18) == vipir.ERR_INVALID_ARG
    assert lib.vipir_plan_set_db_signed(None, 1) == vipir.ERR_INVALID_ARG
    assert lib.vipir_dbmul_plan_layout(None, 16, 16, 1, 16, None, 0, 1) == vipir.ERR_INVALID_ARG
    assert lib.vipir_dbmul_plan_tuned(None, 16, 16, 1, 8, None, 0, 0, None) == vipir.ERR_INVALID_ARG
    assert lib.vipir_testing_modgemm_limbs(None, None, None) == vipir.ERR_INVALID_ARG
    assert lib.vipir_db_split_u16(None, None, 16, 16, None) == vipir.ERR_INVALID_ARG


def test_limb_plane_layout_argument_checks(lib):
    """VIPIR_DB_LIMB_PLANES: u16 only, tensor-core regimes only, cols % 16 == 0, 2*rows < 2^31 --
    all rejected before any device call."""
    def st(rows, cols, batch, db_bits, regime, layout):
        h = ctypes.c_void_p()
        return lib.vipir_dbmul_plan_layout(ctypes.byref(h), rows, cols, batch, db_bits, None, regime, layout)
    assert st(64, 32, 1, 16, 0, 2) == vipir.ERR_INVALID_ARG
    assert st(64, 32, 1, 8, 0, 1) == vipir.ERR_UNSUPPORTED
    assert st(64, 32, 1, 16, vipir.REGIME_GEMV, 1) == vipir.ERR_UNSUPPORTED
    assert st(64, 32, 1, 16, vipir.REGIME_NAIVE, 1) == vipir.ERR_UNSUPPORTED
    assert st(64, 24, 1, 16, 0, 1) == vipir.ERR_UNSUPPORTED
    assert st(1 << 30, 32, 1, 16, 0, 1) == vipir.ERR_UNSUPPORTED
    one = ctypes.c_void_p(0x1000)
    assert lib.vipir_db_split_u16(one, ctypes.c_void_p(0x100000), 0, 16, None) == vipir.ERR_INVALID_ARG
    assert lib.vipir_db_split_u16(one, ctypes.c_void_p(0x100000), 16, 24, None) == vipir.ERR_UNSUPPORTED
    assert lib.vipir_db_split_u16(ctypes.c_void_p(0x1001), ctypes.c_void_p(0x100000), 16, 16, None) == vipir.ERR_INVALID_ARG
    assert lib.vipir_db_split_u16(one, ctypes.c_void_p(0x1100), 16, 16, None) == vipir.ERR_INVALID_ARG  # overlap


def test_no_silent_fallback_without_a_gpu(lib):
    """On a box without a B200 a valid plan request must fail loudly (CUDA/ARCH), never succeed."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    st = _plan_status(lib, 1024, 1024, 1, 8)
    assert st in (vipir.ERR_CUDA, vipir.ERR_ARCH)
    with pytest.raises(vipir.VipirError):
        vipir.dbmul_plan(1024, 1024, 1)


def test_product_never_imports_the_oracle():
    pkg = ROOT / "paper_2606_11536_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")) + [ROOT / "include" / "vipir.h"]:
        text = f.read_text()
        assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), f
        assert "vipir_oracle" not in text, f
    for f in (ROOT / "oracle").rglob("*.py"):
        assert not re.search(r"^\s*(from|import)\s+paper_2606_11536_b200\b", f.read_text(), re.M), f
    assert "#include \"" not in (ROOT / "oracle" / "vipir_oracle.c").read_text()  # system headers only


# ---- vipir_ntt_*: argument checks that need no device ------------------------------------------

def _ntt_status(lib, T, log2n, moduli, psi, scale, p_bits, centered=0):
    h = ctypes.c_void_p()
    arr = lambda xs: (ctypes.c_uint32 * max(1, len(xs)))(*xs)  # noqa: E731
    st = lib.vipir_ntt_plan_create(ctypes.byref(h), T, log2n, arr(moduli), arr(psi), arr(scale), p_bits, centered)
    if st == vipir.OK:
        lib.vipir_ntt_destroy(h)
    return st


def test_ntt_plan_argument_checks(lib):
    q, psi16 = 97, 19                     # 19^16 = -1 mod 97: a primitive 32nd root of unity
    assert pow(psi16, 16, q) == q - 1
    assert _ntt_status(lib, 0, 4, [q], [psi16], [1], 6) == vipir.ERR_INVALID_ARG            # T == 0
    assert _ntt_status(lib, 5, 4, [q] * 5, [psi16] * 5, [1] * 5, 6) == vipir.ERR_INVALID_ARG  # T > 4
    assert _ntt_status(lib, 1, 4, [q], [psi16], [1], 0) == vipir.ERR_INVALID_ARG            # p_bits
    assert _ntt_status(lib, 1, 4, [q], [psi16], [1], 30) == vipir.ERR_INVALID_ARG
    assert _ntt_status(lib, 1, 4, [q], [psi16], [1], 7) == vipir.ERR_INVALID_ARG            # p = 128 > q
    assert _ntt_status(lib, 1, 4, [q], [psi16 * psi16 % q], [1], 6) == vipir.ERR_INVALID_ARG  # order 16, not 32
    assert _ntt_status(lib, 1, 4, [q], [psi16], [1], 6, centered=2) == vipir.ERR_INVALID_ARG
    assert _ntt_status(lib, 1, 5, [q], [psi16], [1], 6) == vipir.ERR_UNSUPPORTED            # log2 N not 4/8/12
    assert lib.vipir_ntt_plan_create(None, 1, 4, None, None, None, 6, 0) == vipir.ERR_INVALID_ARG
    assert lib.vipir_ntt_lift(None, None, 1, 1, 0, None, None) == vipir.ERR_INVALID_ARG
    assert lib.vipir_ntt_bad_input(None, None) == vipir.ERR_INVALID_ARG
    lib.vipir_ntt_destroy(None)
    import torch
    if not torch.cuda.is_available():     # a valid request must fail loudly without a B200, never succeed
        assert _ntt_status(lib, 1, 4, [q], [psi16], [1], 6) in (vipir.ERR_CUDA, vipir.ERR_ARCH)


def test_header_is_plain_c_and_links_from_c(lib, tmp_path):
    """include/vipir.h compiles as strict C99 and a C program linked against libvipir.so (no Python, no
    torch) reaches the entry points: status strings, argument errors before any device call."""
    import shutil
    import subprocess
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("no gcc")
    src = tmp_path / "abi.c"
    src.write_text(r'''
#include <stdio.h>
#include <string.h>
#include "vipir.h"
int main(void) {
    vipir_plan *plan = (vipir_plan *)1;
    vipir_modulus_spec spec;
    uint32_t bad = 1u << 30;
    vipir_info info;
    spec.count = 1; spec.moduli = &bad;
    if (strcmp(vipir_status_str(VIPIR_OK), "VIPIR_OK")) return 1;
    if (vipir_dbmul_plan(&plan, 0, 16, 1, 8, NULL) != VIPIR_ERR_INVALID_ARG || plan != NULL) return 2;
    if (vipir_dbmul_plan(&plan, 16, 16, 1, 8, &spec) != VIPIR_ERR_INVALID_ARG) return 3;
    if (vipir_dbmul_plan_layout(&plan, 16, 16, 1, 8, NULL, VIPIR_REGIME_AUTO, VIPIR_DB_LIMB_PLANES) != VIPIR_ERR_UNSUPPORTED) return 4;
    if (vipir_dbmul(NULL, NULL, NULL, NULL, NULL) != VIPIR_ERR_INVALID_ARG) return 5;
    if (vipir_plan_info(NULL, &info) != VIPIR_ERR_INVALID_ARG) return 6;
    if (vipir_db_split_u16(NULL, NULL, 1, 16, NULL) != VIPIR_ERR_INVALID_ARG) return 7;
    vipir_destroy(NULL);
    vipir_modgemm_destroy(NULL);
    vipir_ntt_destroy(NULL);
    puts("c abi ok");
    return 0;
}
''')
    so = vipir.lib_path()
    exe = tmp_path / "abi"
    subprocess.run([gcc, "-std=c99", "-pedantic", "-Wall", "-Wextra", "-Werror", "-I", str(ROOT / "include"), str(src),
                    "-o", str(exe), str(so), f"-Wl,-rpath,{so.parent}"], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout
    assert "c abi ok" in out


def test_ceilings_library_loads_and_exports_its_entry_points():
    """bench.py's measured ceilings (ceilings/libvipir_ceilings.so: bench-only, not product code)."""
    from paper_2606_11536_b200 import ceilings
    lib = ceilings._load()
    for name in ("vipir_ceiling_mma_i8", "vipir_ceiling_butterflies"):
        assert hasattr(lib, name), name
    # nothing of the product links or loads it
    for f in (ROOT / "paper_2606_11536_b200" / "csrc").glob("*.cu*"):
        assert "ceilings" not in f.read_text(), f
    assert "ceilings" not in (ROOT / "paper_2606_11536_b200" / "vipir.py").read_text()
