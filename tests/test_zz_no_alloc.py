"""vipir_dbmul_static: the batched product for callers that may not allocate device memory.

Some users of this library cannot call cudaMalloc at request time: a PIR server that gave all GPU memory to the
resident database and to one arena at start-up, or a request path that cannot afford the
device-wide stall an allocation or a free can cause.  For them the library has one entry point that needs no plan
and allocates nothing; the tensor-core kernel's scratch (query limb planes, work counters) sits in a fixed 8 MiB
array inside the library, shared by every call on the GPU.

What is checked here: the answers of that entry point equal those of the ordinary plan path (vipir_dbmul) word
for word -- the same bit-exact bar as every other parity test in this suite -- on calls made back to back on one
stream with no synchronisation between them, so the second and third call find the array as the one before left
it (other shape, other regime, other limb-column count).  And that a size the array cannot hold is refused with
a message that says so, before any device work.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide
the rest of the suite.  It does not depend on what ran before it (fresh process or after all other tests).
"""
import ctypes

import numpy as np
import pytest

from paper_2606_11536_b200 import inputs, vipir

from gpu_util import ensure_built, run_dbmul

PRIMES = inputs.rns_primes(0)


def _static(D, Q, moduli, d_db=None):
    """Enqueue one vipir_dbmul_static call on the current stream; returns the (poisoned) device answer, unsynchronised."""
    import torch
    rows, cols = D.shape
    T, batch, _ = Q.shape
    if d_db is None:
        d_db = torch.from_numpy(np.ascontiguousarray(D).view(np.uint8).reshape(rows, -1)).cuda()
    d_q = torch.from_numpy(np.ascontiguousarray(Q).view(np.int32)).cuda()
    d_a = torch.full((T, batch, rows), -1, dtype=torch.int32, device="cuda")
    vipir.dbmul_static(rows, cols, batch, d_db, d_q, d_a, db_bits=8 * D.dtype.itemsize, moduli=moduli)
    return d_a, (d_db, d_q)


# (rows, cols, batch, db_bits, moduli): shapes that land in different regimes and leave different things behind
CASE_PAIRS = {
    # CTA pairs, ragged rows and K tail, wrapping  ->  1-SM tiles, u16 x three primes (five limb columns)
    "m2_u8_then_m1_u16_primes": [(700, 2064, 24, 8, None), (300, 1040, 3, 16, PRIMES)],
    # two K chunks and more work units than CTA groups (the shared counters get used)  ->  one vector, tiny
    "chunked_then_batch1": [(5000, 40000, 8, 8, None), (130, 48, 1, 8, None)],
    # prime moduli on a u8 DB  ->  the widest tile the limit allows at cols = 8192 (256 vectors: exactly 8 MiB)
    "primes_then_full_scratch": [(260, 528, 5, 8, PRIMES), (512, 8192, 256, 8, None)],
}


@pytest.mark.gpu
@pytest.mark.parametrize("name", list(CASE_PAIRS))
def test_static_entry_point_matches_the_plan_path_on_back_to_back_calls(name):
    import torch
    ensure_built()
    first, second = CASE_PAIRS[name]
    data = []
    for i, (rows, cols, batch, db_bits, moduli) in enumerate((first, second, first)):
        seed = 900 + 7 * i
        data.append((inputs.db_rows(seed, rows, cols, db_bits), inputs.query(seed, cols, batch, moduli), moduli))
    # three calls in a row, nothing between them: the 2nd finds the 1st's scratch, the 3rd the 2nd's
    pending = [_static(D, Q, moduli) for D, Q, moduli in data]
    torch.cuda.synchronize()
    for i, ((d_a, _keep), (D, Q, moduli)) in enumerate(zip(pending, data)):
        got = d_a.cpu().numpy().view(np.uint32)
        want = run_dbmul(D, Q, moduli)  # the existing path: vipir_dbmul_plan + vipir_dbmul, regime AUTO
        bad = np.argwhere(got != want)
        assert bad.size == 0, (f"call {i}: {len(bad)} of {got.size} words differ from vipir_dbmul; first at "
                               f"[t,b,r]={bad[0].tolist()}: got {got[tuple(bad[0])]} want {want[tuple(bad[0])]}")


def test_static_entry_point_refuses_what_the_array_cannot_hold():
    """The size check comes before any device call, so it can be tested without a GPU: 16-byte-aligned dummy
    addresses are never dereferenced."""
    ensure_built()
    lib = vipir.load()
    fake = ctypes.c_void_p(4096)
    stream = ctypes.c_void_p(0)
    # u8, cols = 8192: 256 vectors are exactly 8 MiB of planes (accepted above); 257 are not
    assert lib.vipir_dbmul_static(512, 8192, 257, 8, None, fake, fake, fake, stream) == vipir.ERR_UNSUPPORTED
    msg = lib.vipir_last_cuda_error().decode()
    assert "8421376" in msg and str(vipir.STATIC_SCRATCH_BYTES) in msg and "plan" in msg, msg
    with pytest.raises(vipir.VipirError, match="built-in scratch"):
        vipir.dbmul_static(512, 131072, 17, 4096, 4096, 4096, stream=0)
    # the plain argument rules still come first
    assert lib.vipir_dbmul_static(0, 8192, 1, 8, None, fake, fake, fake, stream) == vipir.ERR_INVALID_ARG
    assert lib.vipir_dbmul_static(16, 8192, 1, 8, None, None, fake, fake, stream) == vipir.ERR_INVALID_ARG
    assert lib.vipir_dbmul_static(16, 24, 1, 8, None, fake, fake, fake, stream) == vipir.ERR_UNSUPPORTED
