"""Out-of-bounds write check without compute-sanitizer (closed on this pool): every output buffer is a
window inside a larger allocation whose guard bands hold a sentinel; after each call the bands must be
untouched and the window bit-exact.  Shapes are ragged in every dimension on purpose."""
import numpy as np
import pytest

import oracle
from paper_2606_11536_b200 import inputs, vipir

from gpu_util import ensure_built

pytestmark = pytest.mark.gpu
PRIMES = inputs.rns_primes(0)
GUARD = 4096          # words on each side
SENT = 0x5A5A5A5A


def guarded(shape):
    import torch
    n = int(np.prod(shape))
    buf = torch.full((n + 2 * GUARD,), SENT, dtype=torch.int32, device="cuda")
    return buf, buf[GUARD:GUARD + n].view(shape)


def check_bands(buf):
    host = buf.cpu().numpy().view(np.uint32)
    assert (host[:GUARD] == SENT).all() and (host[-GUARD:] == SENT).all(), "guard band overwritten"


@pytest.mark.parametrize("regime", [vipir.REGIME_GEMV, vipir.REGIME_MMA_1SM, vipir.REGIME_MMA_2SM])
@pytest.mark.parametrize("moduli", [None, PRIMES])
def test_dbmul_writes_only_its_answer(regime, moduli):
    import torch
    ensure_built()
    if regime == vipir.REGIME_GEMV and moduli:
        pytest.skip("GEMV is q = 2^32 only")
    rows, cols = 128 * 4 * 2 + 77, 32768 + 2064
    batch = 1 if regime == vipir.REGIME_GEMV else 5
    D, Q = inputs.db_rows(91, rows, cols, 8), inputs.query(91, cols, batch, moduli)
    buf, d_a = guarded((Q.shape[0], batch, rows))
    tuning = None if regime == vipir.REGIME_GEMV else {"m_sub": 4}
    with vipir.Plan(rows, cols, batch, 8, moduli, regime, tuning=tuning) as plan:
        plan(torch.from_numpy(D).cuda(), torch.from_numpy(Q.view(np.int32)).cuda(), d_a)
        torch.cuda.synchronize()
    check_bands(buf)
    assert np.array_equal(d_a.cpu().numpy().view(np.uint32), oracle.dbmul(D, Q, moduli, nthreads=8))


def test_modgemm_and_ntt_write_only_their_outputs():
    import torch
    ensure_built()
    from paper_2606_11536_b200.inputs import generator as gen
    moduli = inputs.rns_primes(0, 2, 1 << 29, 1 << 18)
    T, NC, M, K, ncols, gcols = 2, 3, 300, 200, 21, 9
    H = gen.modgemm_operand(1, gen.STREAM_MG_H, moduli, NC, M * K).reshape(T, NC, M, K)
    C = gen.modgemm_operand(1, gen.STREAM_MG_C, moduli, NC, ncols * K).reshape(T, NC, ncols, K)
    G = gen.modgemm_operand(1, gen.STREAM_MG_G, moduli, NC, gcols * M).reshape(T, NC, gcols, M)
    buf, d_O = guarded((T, NC, ncols, M))
    with vipir.ModGemmPlan(T, NC, M, K, ncols, gcols, moduli) as plan:
        plan.set_h(torch.from_numpy(H.view(np.int32)).cuda())
        plan(torch.from_numpy(C.view(np.int32)).cuda(), torch.from_numpy(G.view(np.int32)).cuda(), d_O)
        torch.cuda.synchronize()
    check_bands(buf)
    assert np.array_equal(d_O.cpu().numpy().view(np.uint32), oracle.modgemm(H, C, G, moduli, nthreads=8))

    N, n_a, Mp, p_bits = 256, 3, 37, 12
    mods = [7681, 12289]
    psi = [oracle.smallest_psi(N, q) for q in mods]
    X = np.random.default_rng(3).integers(0, 1 << p_bits, size=(n_a, Mp * N), dtype=np.uint32)
    for layout, shape in ((vipir.NTT_LAYOUT_G, (2, N, n_a, Mp)), (vipir.NTT_LAYOUT_H, (2, N, Mp, n_a))):
        buf, d_Y = guarded(shape)
        with vipir.NttPlan(8, mods, psi, [5, 7], p_bits) as plan:
            plan(torch.from_numpy(X.view(np.int32)).cuda(), n_a, Mp, layout, d_Y)
            torch.cuda.synchronize()
        check_bands(buf)
        assert np.array_equal(d_Y.cpu().numpy().view(np.uint32), oracle.ntt_lift(X, N, mods, psi, [5, 7], p_bits, False, layout))
