"""Thin ctypes binding of libvipir (include/vipir.h): argument marshalling only.

Every step of the hot path runs inside csrc/libvipir.so; torch is used for device memory and
streams, nothing else.  There is no CPU fallback: if the shared library is missing or fails
to load, the first call raises.

    plan = vipir.dbmul_plan(rows, cols, batch, db_bits=8, moduli=None)
    vipir.dbmul(plan, d_db, d_query, d_answer)          # torch CUDA tensors, current stream
    vipir.destroy(plan)                                  # or use `with vipir.Plan(...) as p:`
"""
from __future__ import annotations

import ctypes
from pathlib import Path

_LIB_PATH = Path(__file__).resolve().parent / "csrc" / "libvipir.so"
_lib = None

OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_ALLOC, ERR_CUDA, ERR_ARCH = range(6)
REGIME_AUTO, REGIME_GEMV, REGIME_MMA_1SM, REGIME_MMA_2SM, REGIME_NAIVE = range(5)
REGIME_NAMES = {0: "auto", 1: "gemv", 2: "mma_1sm", 3: "mma_2sm", 4: "naive"}
DB_ROW_MAJOR, DB_LIMB_PLANES = 0, 1
MAX_MODULI = 4

# every symbol include/vipir.h declares
SYMBOLS = (
    "vipir_dbmul_plan", "vipir_dbmul_plan_ex", "vipir_dbmul_plan_layout", "vipir_dbmul_plan_tuned", "vipir_db_split_u16",
    "vipir_dbmul", "vipir_dbmul_host", "vipir_split_limbs", "vipir_dbmul_scan", "vipir_dbmul_static",
    "vipir_plan_set_modswitch", "vipir_plan_set_db_signed",
    "vipir_plan_info", "vipir_destroy", "vipir_status_str", "vipir_last_cuda_error",
    "vipir_modgemm_plan_create", "vipir_modgemm_plan_create_tuned", "vipir_modgemm_set_h", "vipir_modgemm",
    "vipir_modgemm_split_c", "vipir_modgemm_products", "vipir_modgemm_info", "vipir_modgemm_destroy",
    "vipir_ntt_plan_create", "vipir_ntt_lift", "vipir_ntt_bad_input", "vipir_ntt_destroy",
)
# include/vipir_testing.h: introspection for the test suite, not part of the product ABI
TESTING_SYMBOLS = ("vipir_testing_work_items", "vipir_testing_modgemm_limbs")


class ModulusSpec(ctypes.Structure):
    _fields_ = [("count", ctypes.c_uint32), ("moduli", ctypes.POINTER(ctypes.c_uint32))]


class Tuning(ctypes.Structure):
    """vipir_tuning: explicit planner overrides, every field 0 = the planner's own choice."""
    _fields_ = [("m_sub", ctypes.c_uint32), ("tile_queries", ctypes.c_uint32), ("k_atoms", ctypes.c_uint32),
                ("stages", ctypes.c_uint32), ("min_chunks", ctypes.c_uint32), ("separate_split", ctypes.c_uint32),
                ("whole_units", ctypes.c_uint32), ("no_collector", ctypes.c_uint32), ("host_staged", ctypes.c_uint32),
                ("host_slices", ctypes.c_uint32), ("leftover_chunks", ctypes.c_uint32), ("reserved", ctypes.c_uint32 * 5)]


class ModGemmTuning(ctypes.Structure):
    """vipir_modgemm_tuning."""
    _fields_ = [("cta_group", ctypes.c_uint32), ("tile_cols", ctypes.c_uint32), ("a_stages", ctypes.c_uint32),
                ("b_stages", ctypes.c_uint32), ("c_split", ctypes.c_uint32), ("r_stages", ctypes.c_uint32),
                ("reserved", ctypes.c_uint32 * 2)]


class Info(ctypes.Structure):
    _fields_ = [
        ("regime", ctypes.c_uint32), ("db_limbs", ctypes.c_uint32), ("limb_cols", ctypes.c_uint32),
        ("query_vectors", ctypes.c_uint32), ("k_bytes", ctypes.c_uint64), ("k_chunk_bytes", ctypes.c_uint32),
        ("n_chunks", ctypes.c_uint32), ("tile_queries", ctypes.c_uint32), ("tile_cols", ctypes.c_uint32),
        ("mma_n", ctypes.c_uint32), ("m_tiles", ctypes.c_uint32), ("n_tiles", ctypes.c_uint32),
        ("stages", ctypes.c_uint32), ("smem_bytes", ctypes.c_uint32), ("grid", ctypes.c_uint32),
        ("launches", ctypes.c_uint32), ("workspace_bytes", ctypes.c_uint64),
        ("modswitch_bits", ctypes.c_uint32), ("db_signed", ctypes.c_uint32), ("m_sub", ctypes.c_uint32),
        ("db_layout", ctypes.c_uint32), ("leftover_chunks", ctypes.c_uint32),
    ]

    def as_dict(self):
        d = {k: getattr(self, k) for k, _ in self._fields_}
        d["regime_name"] = REGIME_NAMES.get(d["regime"], "?")
        return d


class ModGemmInfo(ctypes.Structure):
    _fields_ = [
        ("problems", ctypes.c_uint64), ("k_padded", ctypes.c_uint32), ("cta_group", ctypes.c_uint32),
        ("tile_cols", ctypes.c_uint32), ("mma_n", ctypes.c_uint32), ("m_tiles", ctypes.c_uint32),
        ("n_tiles", ctypes.c_uint32), ("n_chunks", ctypes.c_uint32), ("a_stages", ctypes.c_uint32),
        ("b_stages", ctypes.c_uint32), ("acc_stages", ctypes.c_uint32), ("r_stages", ctypes.c_uint32),
        ("smem_bytes", ctypes.c_uint32),
        ("grid", ctypes.c_uint32), ("launches", ctypes.c_uint32), ("fused_split", ctypes.c_uint32),
        ("h_limb_bytes", ctypes.c_uint64), ("c_limb_bytes", ctypes.c_uint64),
    ]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class VipirError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        lib = load()
        name = lib.vipir_status_str(status).decode()
        detail = lib.vipir_last_cuda_error().decode() if status == ERR_CUDA else ""
        super().__init__(f"{what}: {name}" + (f" ({detail})" if detail else ""))


def lib_path() -> Path:
    return _LIB_PATH


def load() -> ctypes.CDLL:
    """Load csrc/libvipir.so; raises if it has not been built (no fallback exists)."""
    global _lib
    if _lib is None:
        if not _LIB_PATH.exists():
            raise RuntimeError(f"{_LIB_PATH} is missing: run `python -m paper_2606_11536_b200.build` "
                               "(the CUDA library is the only implementation; there is no CPU fallback)")
        lib = ctypes.CDLL(str(_LIB_PATH))
        u64, u32, vp, i = ctypes.c_uint64, ctypes.c_uint32, ctypes.c_void_p, ctypes.c_int
        pp = ctypes.POINTER(ctypes.c_void_p)
        ms = ctypes.POINTER(ModulusSpec)
        lib.vipir_dbmul_plan.restype = i
        lib.vipir_dbmul_plan.argtypes = [pp, u64, u64, u32, u32, ms]
        lib.vipir_dbmul_plan_ex.restype = i
        lib.vipir_dbmul_plan_ex.argtypes = [pp, u64, u64, u32, u32, ms, u32]
        lib.vipir_dbmul_plan_layout.restype = i
        lib.vipir_dbmul_plan_layout.argtypes = [pp, u64, u64, u32, u32, ms, u32, u32]
        lib.vipir_dbmul_plan_tuned.restype = i
        lib.vipir_dbmul_plan_tuned.argtypes = [pp, u64, u64, u32, u32, ms, u32, u32, ctypes.POINTER(Tuning)]
        lib.vipir_db_split_u16.restype = i
        lib.vipir_db_split_u16.argtypes = [vp, vp, u64, u64, vp]
        lib.vipir_dbmul.restype = i
        lib.vipir_dbmul.argtypes = [vp, vp, vp, vp, vp]
        lib.vipir_dbmul_static.restype = i
        lib.vipir_dbmul_static.argtypes = [u64, u64, u32, u32, ms, vp, vp, vp, vp]
        lib.vipir_dbmul_host.restype = i
        lib.vipir_dbmul_host.argtypes = [vp, vp, vp, vp, vp]
        lib.vipir_split_limbs.restype = i
        lib.vipir_split_limbs.argtypes = [vp, vp, vp, vp]
        lib.vipir_dbmul_scan.restype = i
        lib.vipir_dbmul_scan.argtypes = [vp, vp, vp, vp]
        lib.vipir_plan_set_modswitch.restype = i
        lib.vipir_plan_set_modswitch.argtypes = [vp, u32]
        lib.vipir_plan_set_db_signed.restype = i
        lib.vipir_plan_set_db_signed.argtypes = [vp, u32]
        lib.vipir_plan_info.restype = i
        lib.vipir_plan_info.argtypes = [vp, ctypes.POINTER(Info)]
        lib.vipir_destroy.restype = None
        lib.vipir_destroy.argtypes = [vp]
        lib.vipir_testing_work_items.restype = i
        lib.vipir_testing_work_items.argtypes = [u32, u32, u32, u32, u32, ctypes.POINTER(ctypes.c_uint32), u32,
                                                 ctypes.POINTER(ctypes.c_uint32)]
        lib.vipir_testing_modgemm_limbs.restype = i
        lib.vipir_testing_modgemm_limbs.argtypes = [vp, pp, pp]
        lib.vipir_modgemm_plan_create.restype = i
        lib.vipir_modgemm_plan_create.argtypes = [pp, u32, u64, u32, u32, u32, u32, ctypes.POINTER(ctypes.c_uint32)]
        lib.vipir_modgemm_plan_create_tuned.restype = i
        lib.vipir_modgemm_plan_create_tuned.argtypes = [pp, u32, u64, u32, u32, u32, u32, ctypes.POINTER(ctypes.c_uint32),
                                                        ctypes.POINTER(ModGemmTuning)]
        lib.vipir_modgemm_set_h.restype = i
        lib.vipir_modgemm_set_h.argtypes = [vp, vp, vp]
        lib.vipir_modgemm.restype = i
        lib.vipir_modgemm.argtypes = [vp, vp, vp, vp, vp]
        lib.vipir_modgemm_split_c.restype = i
        lib.vipir_modgemm_split_c.argtypes = [vp, vp, vp]
        lib.vipir_modgemm_products.restype = i
        lib.vipir_modgemm_products.argtypes = [vp, vp, vp, vp]
        lib.vipir_modgemm_info.restype = i
        lib.vipir_modgemm_info.argtypes = [vp, ctypes.POINTER(ModGemmInfo)]
        lib.vipir_modgemm_destroy.restype = None
        lib.vipir_modgemm_destroy.argtypes = [vp]
        u32p = ctypes.POINTER(ctypes.c_uint32)
        lib.vipir_ntt_plan_create.restype = i
        lib.vipir_ntt_plan_create.argtypes = [pp, u32, u32, u32p, u32p, u32p, u32, u32]
        lib.vipir_ntt_lift.restype = i
        lib.vipir_ntt_lift.argtypes = [vp, vp, u32, u32, u32, vp, vp]
        lib.vipir_ntt_bad_input.restype = i
        lib.vipir_ntt_bad_input.argtypes = [vp, u32p]
        lib.vipir_ntt_destroy.restype = None
        lib.vipir_ntt_destroy.argtypes = [vp]
        lib.vipir_status_str.restype = ctypes.c_char_p
        lib.vipir_status_str.argtypes = [i]
        lib.vipir_last_cuda_error.restype = ctypes.c_char_p
        lib.vipir_last_cuda_error.argtypes = []
        _lib = lib
    return _lib


def _check(status: int, what: str):
    if status != OK:
        raise VipirError(status, what)


def _stream_ptr(stream):
    if stream is None:
        import torch
        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return ctypes.c_void_p(stream)
    return ctypes.c_void_p(stream.cuda_stream)


def _ptr(t):
    """Device/host address of a torch tensor, numpy array or raw int."""
    if isinstance(t, int):
        return ctypes.c_void_p(t)
    if hasattr(t, "data_ptr"):
        return ctypes.c_void_p(t.data_ptr())
    return ctypes.c_void_p(t.ctypes.data)


def dbmul_plan(rows: int, cols: int, batch: int, db_bits: int = 8, moduli=None, regime: int = REGIME_AUTO,
               db_layout: int = DB_ROW_MAJOR, tuning: dict | None = None):
    """vipir_dbmul_plan[_ex|_layout|_tuned]; returns the opaque plan handle (a c_void_p).
    tuning: {field of vipir_tuning: value} -- explicit planner overrides."""
    lib = load()
    handle = ctypes.c_void_p()
    spec_p = None
    if moduli is not None and len(moduli) > 0:
        arr = (ctypes.c_uint32 * len(moduli))(*[int(m) for m in moduli])
        spec = ModulusSpec(len(moduli), arr)
        spec_p = ctypes.byref(spec)
    if tuning:
        tune = Tuning(**{k: int(v) for k, v in tuning.items()})
        _check(lib.vipir_dbmul_plan_tuned(ctypes.byref(handle), rows, cols, batch, db_bits, spec_p, regime, db_layout,
                                          ctypes.byref(tune)), "vipir_dbmul_plan_tuned")
    else:
        _check(lib.vipir_dbmul_plan_layout(ctypes.byref(handle), rows, cols, batch, db_bits, spec_p, regime, db_layout),
               "vipir_dbmul_plan")
    return handle


def db_split_u16(d_db_u16, d_db_planes, rows: int, cols: int, stream=None):
    """vipir_db_split_u16: offline de-interleave of a u16 DB into its two byte-limb planes."""
    _check(load().vipir_db_split_u16(_ptr(d_db_u16), _ptr(d_db_planes), rows, cols, _stream_ptr(stream)),
           "vipir_db_split_u16")


def dbmul(plan, d_db, d_query, d_answer, stream=None):
    """vipir_dbmul: enqueue answer = D*Q mod q on `stream` (default: torch's current stream)."""
    _check(load().vipir_dbmul(plan, _ptr(d_db), _ptr(d_query), _ptr(d_answer), _stream_ptr(stream)), "vipir_dbmul")


def dbmul_host(plan, d_db, h_query, h_answer, stream=None):
    """vipir_dbmul_host: host query in, host answer out; synchronises the stream."""
    _check(load().vipir_dbmul_host(plan, _ptr(d_db), _ptr(h_query), _ptr(h_answer), _stream_ptr(stream)),
           "vipir_dbmul_host")


STATIC_SCRATCH_BYTES = 8 << 20  # VIPIR_STATIC_SCRATCH_BYTES


def dbmul_static(rows: int, cols: int, batch: int, d_db, d_query, d_answer, db_bits: int = 8, moduli=None, stream=None):
    """vipir_dbmul_static: the batched product without a plan, for callers that may not allocate device memory
    (a server whose GPU memory is fully handed out at start-up, a request path that cannot afford the device-wide
    stall of cudaMalloc / cudaFree).  The kernel's scratch is a fixed 8 MiB array inside the library, shared by every
    call on the GPU: the query limb planes (T * batch * LC * cols * db_bits/8 bytes) must fit in
    STATIC_SCRATCH_BYTES, else VipirError(ERR_UNSUPPORTED) with the two sizes in the message; calls whose GPU work
    overlaps race.  The first call on a device does a one-time address look-up: make it before any stream capture.
    Only enqueues on `stream` (default: torch's current stream); same answer as dbmul, bit for bit."""
    lib = load()
    spec_p = None
    if moduli is not None and len(moduli) > 0:
        arr = (ctypes.c_uint32 * len(moduli))(*[int(m) for m in moduli])
        spec = ModulusSpec(len(moduli), arr)
        spec_p = ctypes.byref(spec)
    status = lib.vipir_dbmul_static(rows, cols, batch, db_bits, spec_p, _ptr(d_db), _ptr(d_query), _ptr(d_answer),
                                    _stream_ptr(stream))
    if status == ERR_UNSUPPORTED:
        why = lib.vipir_last_cuda_error().decode()
        if why:
            raise VipirError(status, why)
    _check(status, "vipir_dbmul_static")


def split_limbs(plan, d_query, d_planes_out=None, stream=None):
    """vipir_split_limbs: step a1 alone, into d_planes_out (or the plan's workspace if None)."""
    out = ctypes.c_void_p(None) if d_planes_out is None else _ptr(d_planes_out)
    _check(load().vipir_split_limbs(plan, _ptr(d_query), out, _stream_ptr(stream)), "vipir_split_limbs")


def dbmul_scan(plan, d_db, d_answer, stream=None):
    """vipir_dbmul_scan: the scan kernel alone, against the planes already in the workspace."""
    _check(load().vipir_dbmul_scan(plan, _ptr(d_db), _ptr(d_answer), _stream_ptr(stream)), "vipir_dbmul_scan")


def plan_set_modswitch(plan, out_bits: int):
    """vipir_plan_set_modswitch: fuse round(x * 2^out_bits / 2^32) into the epilogue (0 = off)."""
    _check(load().vipir_plan_set_modswitch(plan, out_bits), "vipir_plan_set_modswitch")


def plan_set_db_signed(plan, is_signed: bool = True):
    """vipir_plan_set_db_signed: read the u8 DB bytes as two's-complement int8."""
    _check(load().vipir_plan_set_db_signed(plan, 1 if is_signed else 0), "vipir_plan_set_db_signed")


def plan_info(plan) -> dict:
    info = Info()
    _check(load().vipir_plan_info(plan, ctypes.byref(info)), "vipir_plan_info")
    return info.as_dict()


def destroy(plan):
    load().vipir_destroy(plan)


class Plan:
    """Context-manager convenience around dbmul_plan / destroy."""

    def __init__(self, rows, cols, batch, db_bits=8, moduli=None, regime=REGIME_AUTO, modswitch_bits=0,
                 db_signed=False, db_layout=DB_ROW_MAJOR, tuning=None):
        self.handle = dbmul_plan(rows, cols, batch, db_bits, moduli, regime, db_layout, tuning)
        if modswitch_bits:
            plan_set_modswitch(self.handle, modswitch_bits)
        if db_signed:
            plan_set_db_signed(self.handle, True)
        self.info = plan_info(self.handle)

    def __call__(self, d_db, d_query, d_answer, stream=None):
        dbmul(self.handle, d_db, d_query, d_answer, stream)

    def host(self, d_db, h_query, h_answer, stream=None):
        dbmul_host(self.handle, d_db, h_query, h_answer, stream)

    def close(self):
        if self.handle is not None:
            destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def testing_work_items(g: int, n_groups: int, n_units: int, n_chunks: int, split: int = 1):
    """vipir_testing_work_items (include/vipir_testing.h): [(unit, chunk, must_wait), ...] for group g (host only)."""
    cap = n_units * n_chunks + 1
    buf = (ctypes.c_uint32 * (3 * cap))()
    n = ctypes.c_uint32(0)
    _check(load().vipir_testing_work_items(g, n_groups, n_units, n_chunks, split, buf, cap, ctypes.byref(n)),
           "vipir_testing_work_items")
    return [(buf[3 * i], buf[3 * i + 1], bool(buf[3 * i + 2])) for i in range(n.value)]


# ---- parallel INT32 modular GEMMs  Out = H*C + (0|G) mod q_t  (include/vipir.h, NEXT-4) ----------

def modgemm_plan_create(T: int, NC: int, M: int, K: int, ncols: int, gcols: int, moduli, tuning: dict | None = None):
    """vipir_modgemm_plan_create[_tuned]; returns the opaque plan handle."""
    handle = ctypes.c_void_p()
    arr = (ctypes.c_uint32 * max(len(moduli), 1))(*[int(m) for m in moduli])
    if len(moduli) != T:
        raise ValueError(f"{len(moduli)} moduli for T = {T}")
    if tuning:
        tune = ModGemmTuning(**{k: int(v) for k, v in tuning.items()})
        _check(load().vipir_modgemm_plan_create_tuned(ctypes.byref(handle), T, NC, M, K, ncols, gcols, arr,
                                                      ctypes.byref(tune)), "vipir_modgemm_plan_create_tuned")
    else:
        _check(load().vipir_modgemm_plan_create(ctypes.byref(handle), T, NC, M, K, ncols, gcols, arr),
               "vipir_modgemm_plan_create")
    return handle


def testing_modgemm_limbs(plan):
    """vipir_testing_modgemm_limbs (include/vipir_testing.h): device addresses (d_h_limbs, d_c_limbs)."""
    h, c = ctypes.c_void_p(), ctypes.c_void_p()
    _check(load().vipir_testing_modgemm_limbs(plan, ctypes.byref(h), ctypes.byref(c)), "vipir_testing_modgemm_limbs")
    return h.value, c.value


def modgemm_set_h(plan, d_H, stream=None):
    """vipir_modgemm_set_h: the offline re-layout of the static hint H [T][NC][M][K] u32."""
    _check(load().vipir_modgemm_set_h(plan, _ptr(d_H), _stream_ptr(stream)), "vipir_modgemm_set_h")


def modgemm(plan, d_C, d_G, d_Out, stream=None):
    """vipir_modgemm: enqueue Out = H*C + (0|G) mod q_t (C splitter + tensor-core kernel)."""
    g = ctypes.c_void_p(None) if d_G is None else _ptr(d_G)
    _check(load().vipir_modgemm(plan, _ptr(d_C), g, _ptr(d_Out), _stream_ptr(stream)), "vipir_modgemm")


def modgemm_split_c(plan, d_C, stream=None):
    _check(load().vipir_modgemm_split_c(plan, _ptr(d_C), _stream_ptr(stream)), "vipir_modgemm_split_c")


def modgemm_products(plan, d_G, d_Out, stream=None):
    g = ctypes.c_void_p(None) if d_G is None else _ptr(d_G)
    _check(load().vipir_modgemm_products(plan, g, _ptr(d_Out), _stream_ptr(stream)), "vipir_modgemm_products")


def modgemm_info(plan) -> dict:
    info = ModGemmInfo()
    _check(load().vipir_modgemm_info(plan, ctypes.byref(info)), "vipir_modgemm_info")
    return info.as_dict()


def modgemm_destroy(plan):
    load().vipir_modgemm_destroy(plan)


class ModGemmPlan:
    """Context-manager convenience around modgemm_plan_create / modgemm_destroy."""

    def __init__(self, T, NC, M, K, ncols, gcols, moduli, tuning=None):
        self.handle = modgemm_plan_create(T, NC, M, K, ncols, gcols, moduli, tuning)
        self.info = modgemm_info(self.handle)

    def set_h(self, d_H, stream=None):
        modgemm_set_h(self.handle, d_H, stream)

    def __call__(self, d_C, d_G, d_Out, stream=None):
        modgemm(self.handle, d_C, d_G, d_Out, stream)

    def close(self):
        if self.handle is not None:
            modgemm_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- lift + forward NTT producing the ring-packing operands G and H (include/vipir.h) ------------

NTT_LAYOUT_G, NTT_LAYOUT_H = 0, 1


def ntt_plan_create(log2n: int, moduli, psi, scale, p_bits: int, centered: bool = False):
    """vipir_ntt_plan_create; returns the opaque plan handle."""
    T = len(moduli)
    if len(psi) != T or len(scale) != T:
        raise ValueError("one psi and one scale per modulus")
    arr = lambda xs: (ctypes.c_uint32 * max(T, 1))(*[int(x) for x in xs])  # noqa: E731
    handle = ctypes.c_void_p()
    _check(load().vipir_ntt_plan_create(ctypes.byref(handle), T, log2n, arr(moduli), arr(psi), arr(scale), p_bits,
                                        1 if centered else 0), "vipir_ntt_plan_create")
    return handle


def ntt_lift(plan, d_X, n_a: int, M: int, out_layout: int, d_O, stream=None):
    """vipir_ntt_lift: d_X [n_a][M][N] u32 -> d_O [T][N][n_a][M] (LAYOUT_G) or [T][N][M][n_a] (LAYOUT_H)."""
    _check(load().vipir_ntt_lift(plan, _ptr(d_X), n_a, M, out_layout, _ptr(d_O), _stream_ptr(stream)), "vipir_ntt_lift")


def ntt_bad_input(plan) -> bool:
    seen = ctypes.c_uint32(0)
    _check(load().vipir_ntt_bad_input(plan, ctypes.byref(seen)), "vipir_ntt_bad_input")
    return bool(seen.value)


def ntt_destroy(plan):
    load().vipir_ntt_destroy(plan)


class NttPlan:
    """Context-manager convenience around ntt_plan_create / ntt_destroy."""

    def __init__(self, log2n, moduli, psi, scale, p_bits, centered=False):
        self.handle = ntt_plan_create(log2n, moduli, psi, scale, p_bits, centered)

    def __call__(self, d_X, n_a, M, out_layout, d_O, stream=None):
        ntt_lift(self.handle, d_X, n_a, M, out_layout, d_O, stream)

    def bad_input(self) -> bool:
        return ntt_bad_input(self.handle)

    def close(self):
        if self.handle is not None:
            ntt_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
