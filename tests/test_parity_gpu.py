"""GPU parity: libvipir (through the C ABI) against the CPU oracle, bit for bit.

All work is integer, so the bar is exact equality of every compared word (no tolerance).
Small and medium shapes are compared in full and are sized to span several tiles plus a
ragged tail in every dimension (rows, K bytes, query vectors, K chunks).  BASELINE.json's
full-size configs are in tests/test_parity_fullsize_gpu.py: configs[1] and configs[2] at B = 1 in full,
the batched ones on whole 128-row tiles plus a column-sum identity over every row, through both the
device and the host entry point.
"""
import os

import numpy as np
import pytest

import oracle
from paper_2606_11536_b200 import inputs, vipir

from gpu_util import ensure_built, run_dbmul

pytestmark = pytest.mark.gpu

PRIMES = inputs.rns_primes(0)
NT = max(1, os.cpu_count() or 1)
G, M1, M2, NAIVE, AUTO = (vipir.REGIME_GEMV, vipir.REGIME_MMA_1SM, vipir.REGIME_MMA_2SM, vipir.REGIME_NAIVE,
                          vipir.REGIME_AUTO)


def make(seed, rows, cols, batch, db_bits=8, moduli=None):
    return inputs.db_rows(seed, rows, cols, db_bits), inputs.query(seed, cols, batch, moduli)


def assert_same(got, want):
    bad = np.argwhere(got != want)
    assert bad.size == 0, (f"{len(bad)} of {got.size} words differ; first at [t,b,r]={bad[0].tolist()}: "
                           f"got {got[tuple(bad[0])]} want {want[tuple(bad[0])]}")


def check(D, Q, moduli, regime):
    got = run_dbmul(D, Q, moduli, regime)
    want = oracle.dbmul(D, Q, moduli, nthreads=NT)
    assert_same(got, want)


# ---- a1: the limb splitter on its own --------------------------------------

@pytest.mark.parametrize("db_bits,moduli,cols,batch", [
    (8, None, 1040, 3), (16, None, 520, 2), (16, PRIMES, 264, 2), (8, None, 16, 1), (8, PRIMES, 48, 1)])
def test_split_limbs_planes(db_bits, moduli, cols, batch):
    import torch
    ensure_built()
    Q = inputs.query(31, cols, batch, moduli)
    Q[0, 0, :3] = [0xFFFFFFFF, 0x01020304, 0x80000000]
    d_q = torch.from_numpy(Q.view(np.int32)).cuda()
    dl = db_bits // 8
    with vipir.Plan(256, cols, batch, db_bits, moduli, M1) as plan:
        lc, nq, kb = plan.info["limb_cols"], plan.info["query_vectors"], plan.info["k_bytes"]
        assert lc == (5 if (dl == 2 and moduli) else 4) and nq == Q.shape[0] * batch and kb == cols * dl
        assert plan.info["workspace_bytes"] == nq * lc * kb
        planes = torch.full((nq * lc * kb,), 0xAA, dtype=torch.uint8, device="cuda")
        vipir.split_limbs(plan.handle, d_q, planes)
        torch.cuda.synchronize()
    got = planes.cpu().numpy().reshape(nq, lc, kb)
    Qf = Q.reshape(nq, cols)
    limb = [((Qf >> (8 * j)) & 0xFF).astype(np.uint8) for j in range(4)]  # B_j of PAPER.md:245
    for s in range(lc):
        if dl == 1:
            want = limb[s]
        else:
            want = np.zeros((nq, kb), dtype=np.uint8)
            if s < 4:
                want[:, 0::2] = limb[s]
            if s >= 1:
                want[:, 1::2] = limb[s - 1]
        assert np.array_equal(got[:, s, :], want), f"plane s={s}"


# ---- test-only check kernel ---------------------------------------------------------------------

@pytest.mark.parametrize("db_bits,moduli", [(8, None), (16, None), (8, PRIMES), (16, PRIMES)])
def test_naive_kernel(db_bits, moduli):
    D, Q = make(41, 70, 48 // (db_bits // 8) * 4, 3, db_bits, moduli)
    check(D, Q, moduli, NAIVE)


# ---- a2: batch-1 scan (GEMV regime) ------------------------------------------------------------

@pytest.mark.parametrize("rows,cols", [(1024, 1024), (100, 4112), (33, 16), (1, 16), (257, 2064), (32, 1024), (64, 3072)])
def test_gemv_u8(rows, cols):
    D, Q = make(rows + cols, rows, cols, 1)
    check(D, Q, None, G)


@pytest.mark.parametrize("fused", ["1", "0"])
@pytest.mark.parametrize("signed,bits", [(False, 0), (True, 0), (False, 18)])
def test_gemv_fused_and_separate_split_agree_with_the_oracle(fused, signed, bits):
    """cols % 32 == 0: the query split runs inside the scan kernel (one launch); vipir_tuning.separate_split
    forces the two-launch path.  Ragged rows, a K tail shorter than a stage, several stages."""
    rows, cols = 1000, 1024 * 5 + 32 * 7
    D, Q = make(77, rows, cols, 1)
    got, info = run_dbmul(D, Q, None, G, return_info=True, modswitch_bits=bits, db_signed=signed,
                          tuning=None if fused == "1" else {"separate_split": 1})
    assert info["launches"] == (1 if fused == "1" else 2)
    want = oracle.dbmul_signed(D, Q, None) if signed else oracle.dbmul(D, Q, None, nthreads=NT)
    if bits:
        want = oracle.modswitch(want, bits)
    assert_same(got, want)


def test_gemv_u16_wrapping():
    D, Q = make(43, 70, 520, 1, 16)
    check(D, Q, None, G)


def test_gemv_extremes_and_permutation():
    rows, cols = 96, 2048
    D = np.full((rows, cols), 255, dtype=np.uint8)
    Q = np.full((1, 1, cols), 0xFFFFFFFF, dtype=np.uint32)
    got = run_dbmul(D, Q, None, G)
    assert (got == (-255 * cols) % (1 << 32)).all()  # closed form 2 of SURVEY.md 8(c)
    perm = np.random.default_rng(1).integers(0, cols, size=rows)
    D = np.zeros((rows, cols), dtype=np.uint8)
    D[np.arange(rows), perm] = 1
    Q = (np.arange(cols, dtype=np.uint32) + 1).reshape(1, 1, cols)
    assert np.array_equal(run_dbmul(D, Q, None, G)[0, 0], (perm + 1).astype(np.uint32))


# ---- a3/a4: tensor-core regimes, q = 2^32 --------------------------------------------------------

@pytest.mark.parametrize("regime", [M1, M2])
@pytest.mark.parametrize("batch", [1, 2, 3, 8, 16, 64, 100])
def test_mma_u8_wrapping(regime, batch):
    # rows: 2 full M tiles + ragged tail (44 rows); K: 12 k-steps + 16-byte tail
    D, Q = make(100 + batch, 300, 1552, batch)
    check(D, Q, None, regime)


@pytest.mark.parametrize("regime", [M1, M2])
def test_mma_permutation_probe(regime):
    # catches swizzle / descriptor / layout errors as permuted results
    rows, cols, batch = 256, 512, 8
    rng = np.random.default_rng(2)
    perm = rng.integers(0, cols, size=rows)
    D = np.zeros((rows, cols), dtype=np.uint8)
    D[np.arange(rows), perm] = 1
    Q = np.stack([(np.arange(cols, dtype=np.uint64) + 1) * (b + 1) * 0x01010101 % (1 << 32) for b in range(batch)])
    Q = Q.astype(np.uint32).reshape(1, batch, cols)
    got = run_dbmul(D, Q, None, regime)
    for b in range(batch):
        assert np.array_equal(got[0, b], Q[0, b, perm]), f"query {b}"


@pytest.mark.parametrize("regime", [M1, M2])
def test_mma_large_batch_two_n_tiles(regime):
    D, Q = make(51, 260, 1040, 256)
    got, info = run_dbmul(D, Q, None, regime, return_info=True)
    assert info["n_tiles"] >= 2
    assert_same(got, oracle.dbmul(D, Q, None, nthreads=NT))


@pytest.mark.parametrize("regime,cols", [(AUTO, 65536), (M2, 65536 - 112)])
def test_mma_config4_launch_path_compared_in_full(regime, cols):
    """The exact launch path of BASELINE.json configs[3] (four limbs, int32 accumulation per K
    chunk, shift-recombine, free wrap), every answer word compared: q = 2^32 with no fused modulus switch, CTA
    pairs, B = 256 = two N tiles of 512 accumulator columns, TWO tcgen05.mma per K slice (the second taking the
    DB operand from the collector), two K chunks -- chunk 0 stores, chunk 1 accumulates with red.global.add.
    Rows: 2 full 256-row pair tiles + 88 ragged rows; K: configs[3]'s own 65536 columns = two full 32768-byte
    chunks, and 65424 columns = the same two chunks with a 16-byte tail in the last k-step."""
    rows, batch = 600, 256
    D, Q = make(53, rows, cols, batch)
    D[:3] = 255                            # int32 accumulators at 255 * 255 * 32768 on a few rows
    Q[0, :2, :] = 0xFFFFFFFF
    got, info = run_dbmul(D, Q, None, regime, return_info=True)
    assert info["regime_name"] == "mma_2sm" and info["modswitch_bits"] == 0
    assert info["tile_cols"] == 512 and info["mma_n"] * 2 == info["tile_cols"]  # n_instr == 2
    assert info["n_tiles"] == 2 and info["n_chunks"] == 2 and info["k_chunk_bytes"] <= 32768
    assert_same(got, oracle.dbmul(D, Q, None, nthreads=NT))


# ---- M sub-tiles and chunk-granular work distribution (gemm_i8_tcgen05.cuh header) ---------------

@pytest.mark.parametrize("regime", [M1, M2])
@pytest.mark.parametrize("msub", [2, 4])
@pytest.mark.parametrize("moduli,bits", [(None, 0), (None, 18), (PRIMES, 0)])
def test_mma_m_subtiles(regime, msub, moduli, bits):
    # rows: several (128 * CG * msub)-row units + a ragged tail that leaves whole sub-tiles empty;
    # K: 3 chunks, so units are split between groups and accumulated through the answer buffer
    rows, cols, batch = 128 * 2 * msub * 2 + 128 + 37, 32768 * 2 + 2064, 6
    D, Q = make(300 + msub, rows, cols, batch, 8, moduli)
    got, info = run_dbmul(D, Q, moduli, regime, return_info=True, modswitch_bits=bits, tuning={"m_sub": msub})
    assert info["m_sub"] == msub and info["n_chunks"] == 3
    want = oracle.dbmul(D, Q, moduli, nthreads=NT)
    if bits:
        want = oracle.modswitch(want, bits)
    assert_same(got, want)


@pytest.mark.parametrize("regime", [M1, M2])
def test_mma_m_subtiles_permutation_probe(regime):
    rows, cols, batch = 128 * 2 * 4 * 2, 512, 8
    rng = np.random.default_rng(5)
    perm = rng.integers(0, cols, size=rows)
    D = np.zeros((rows, cols), dtype=np.uint8)
    D[np.arange(rows), perm] = 1
    Q = np.stack([(np.arange(cols, dtype=np.uint64) + 1) * (b + 1) * 0x01010101 % (1 << 32) for b in range(batch)])
    Q = Q.astype(np.uint32).reshape(1, batch, cols)
    got = run_dbmul(D, Q, None, regime, tuning={"m_sub": 4})
    for b in range(batch):
        assert np.array_equal(got[0, b], Q[0, b, perm]), f"query {b}"


@pytest.mark.parametrize("regime", [M1, M2])
@pytest.mark.parametrize("rows,chunks", [(128, 5), (300, 4), (9700, 3), (19000, 2), (24000, 2)])
def test_mma_split_units_and_plan_reuse(regime, rows, chunks):
    """Fewer units than CTAs (every unit dealt out chunk by chunk) up to several rounds plus a
    leftover round; the same plan is launched repeatedly, so the in-kernel reset of the ticket and
    arrival counters is exercised too."""
    import torch
    ensure_built()
    cols, batch = 32768 * (chunks - 1) + 4096, 3
    D = inputs.db_rows(400 + rows, rows, cols, 8)
    d_db = torch.from_numpy(D).cuda()
    for moduli in (None, PRIMES):
        Q = inputs.query(400 + rows, cols, batch, moduli)
        want = oracle.dbmul(D, Q, moduli, nthreads=NT)
        d_q = torch.from_numpy(Q.view(np.int32)).cuda()
        with vipir.Plan(rows, cols, batch, 8, moduli, regime) as plan:
            assert plan.info["n_chunks"] == chunks
            for it in range(3):
                d_a = torch.full((Q.shape[0], batch, rows), -1 - it, dtype=torch.int32, device="cuda")
                plan(d_db, d_q, d_a)
                torch.cuda.synchronize()
                assert_same(d_a.cpu().numpy().view(np.uint32), want)


def test_cuda_graph_replay_of_split_units():
    """vipir_dbmul only enqueues (include/vipir.h): it can be captured into a CUDA graph, and the
    in-kernel reset of the ticket / arrival counters makes every replay start from a clean state."""
    import torch
    ensure_built()
    rows, cols, batch = 9700, 32768 * 2 + 4096, 3           # units dealt out chunk by chunk (see above)
    D = inputs.db_rows(431, rows, cols, 8)
    d_db = torch.from_numpy(D).cuda()
    for moduli in (None, PRIMES):
        Q = inputs.query(431, cols, batch, moduli)
        want = oracle.dbmul(D, Q, moduli, nthreads=NT)
        d_q = torch.from_numpy(Q.view(np.int32)).cuda()
        d_a = torch.zeros((Q.shape[0], batch, rows), dtype=torch.int32, device="cuda")
        with vipir.Plan(rows, cols, batch, 8, moduli, M2) as plan:
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                plan(d_db, d_q, d_a, stream=side)             # warm-up outside capture
            torch.cuda.current_stream().wait_stream(side)
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=side):
                plan(d_db, d_q, d_a, stream=side)
            for it in range(3):
                d_a.fill_(-1 - it)
                graph.replay()
                torch.cuda.synchronize()
                assert_same(d_a.cpu().numpy().view(np.uint32), want)


# ---- K chunking: int32 accumulators at their limit (R7) ------------------------------

@pytest.mark.parametrize("regime", [M1, M2])
def test_mma_chunk_seams_adversarial(regime, golden):
    cols = 32768 * 2 + 4112  # three chunks, ragged
    rows, batch = 130, 2
    D = np.full((rows, cols), 255, dtype=np.uint8)
    Q = np.full((1, batch, cols), 0xFFFFFFFF, dtype=np.uint32)
    got, info = run_dbmul(D, Q, None, regime, return_info=True)
    assert info["n_chunks"] == 3 and info["k_chunk_bytes"] <= golden["int32_chunk_bound"]["k_chunk_contract"]
    assert (got == (-255 * cols) % (1 << 32)).all()
    D, Q = make(52, rows, cols, batch)
    D[:64] = 255
    check(D, Q, None, regime)


@pytest.mark.parametrize("regime", [M1, M2])
def test_mma_exact_chunk_of_32768_all_max(regime):
    cols = 32768
    D = np.full((128, cols), 255, dtype=np.uint8)
    Q = np.full((1, 4, cols), 0xFFFFFFFF, dtype=np.uint32)
    got = run_dbmul(D, Q, None, regime)
    assert (got == (-255 * cols) % (1 << 32)).all()
    p = PRIMES[0]
    got = run_dbmul(D, Q, [p], regime)  # true integer sums needed: no wrap may hide an overflow
    assert (got == (255 * 0xFFFFFFFF * cols) % p).all()


# ---- a4/a5: prime moduli, u16 DB -------------------------------------------------------------------

@pytest.mark.parametrize("regime", [M1, M2])
@pytest.mark.parametrize("db_bits,moduli,batch", [
    (8, PRIMES, 5), (8, [PRIMES[0]], 1), (16, None, 4), (16, PRIMES, 3), (16, PRIMES, 40), (16, [97, 1 << 29, 2, PRIMES[1]], 2)])
def test_mma_moduli_and_u16(regime, db_bits, moduli, batch):
    D, Q = make(60 + batch, 300, 776 if db_bits == 16 else 1552, batch, db_bits, moduli)
    check(D, Q, moduli, regime)


@pytest.mark.parametrize("regime", [M1, M2])
def test_mma_prime_edges(regime):
    p = PRIMES[0]
    cols = 40000
    D = np.ones((130, cols), dtype=np.uint16)
    Q = np.full((1, 2, cols), p - 1, dtype=np.uint32)
    got = run_dbmul(D, Q, [p], regime)
    assert (got == (-cols) % p).all()  # closed form 3
    D = np.full((130, cols), 0xFFFF, dtype=np.uint16)
    Q = np.full((2, 1, cols), 0xFFFFFFFF, dtype=np.uint32)  # words above the modulus are legal (R5)
    got = run_dbmul(D, Q, PRIMES, regime)
    for t, pt in enumerate(PRIMES):
        assert (got[t] == (0xFFFF * 0xFFFFFFFF * cols) % pt).all()
        assert (got[t] < pt).all()


# ---- planner / ABI behaviour on the device ------------------------------------------------------

def test_auto_regime_choice():
    ensure_built()
    with vipir.Plan(1024, 1024, 1) as p:
        assert p.info["regime_name"] == "gemv" and p.info["launches"] == 1     # query split fused into the scan
    with vipir.Plan(1024, 1040, 1) as p:                                     # cols % 32 != 0: separate splitter
        assert p.info["regime_name"] == "gemv" and p.info["launches"] == 2
    with vipir.Plan(1024, 1024, 8) as p:
        assert p.info["regime_name"] == "mma_1sm" and p.info["mma_n"] == 32
    with vipir.Plan(1024, 1024, 256) as p:
        assert p.info["regime_name"] == "mma_2sm" and p.info["tile_cols"] == 512 and p.info["n_tiles"] == 2
    with vipir.Plan(1024, 1024, 1, 8, [PRIMES[0]]) as p:
        assert p.info["regime_name"] == "mma_1sm"
    with vipir.Plan(32768, 32768, 64, 16, PRIMES) as p:
        assert p.info["limb_cols"] == 5 and p.info["k_bytes"] == 65536 and p.info["n_chunks"] == 2
    with pytest.raises(vipir.VipirError) as e:
        vipir.Plan(1024, 1024, 2, regime=G)
    assert e.value.status == vipir.ERR_UNSUPPORTED


def test_tuning_overrides_are_honoured_or_refused():
    """vipir_dbmul_plan_tuned: an override the shape or regime cannot honour is UNSUPPORTED, never ignored."""
    ensure_built()

    def status(regime, batch=8, **tuning):
        try:
            vipir.Plan(1024, 2048, batch, 8, None, regime, tuning=tuning).close()
            return vipir.OK
        except vipir.VipirError as e:
            return e.status
    assert status(M2, batch=256, m_sub=2) == vipir.ERR_UNSUPPORTED    # 2 x 512 accumulator columns > TMEM
    assert status(M1, tile_queries=6) == vipir.ERR_UNSUPPORTED         # not a multiple of 4
    assert status(M1, tile_queries=128) == vipir.ERR_UNSUPPORTED       # 512 columns need CTA pairs
    assert status(M1, min_chunks=17) == vipir.ERR_UNSUPPORTED          # only 16 k-atoms
    assert status(M1, stages=12, k_atoms=4) == vipir.ERR_UNSUPPORTED   # does not fit in shared memory
    assert status(M1, separate_split=1) == vipir.ERR_UNSUPPORTED       # a GEMV override
    assert status(G, batch=1, m_sub=2) == vipir.ERR_UNSUPPORTED        # an MMA override
    assert status(G, batch=1, stages=7) == vipir.ERR_UNSUPPORTED
    assert status(G, batch=1, host_slices=2) == vipir.ERR_UNSUPPORTED  # K slices are the tensor regimes' host pipeline
    assert status(M1, host_slices=2) == vipir.OK
    # the modular GEMMs keep the same promise: the raw-tile ring exists in the one-kernel form only
    for tuning, want in ((dict(c_split=1, r_stages=2), vipir.ERR_UNSUPPORTED), (dict(c_split=2, r_stages=2), vipir.OK),
                         (dict(r_stages=2), vipir.ERR_UNSUPPORTED)):  # 8 columns: the planner's form is two kernels
        try:
            vipir.ModGemmPlan(1, 2, 128, 128, 8, 0, [PRIMES[0]], tuning=tuning).close()
            got = vipir.OK
        except vipir.VipirError as e:
            got = e.status
        assert got == want, (tuning, got)
    with vipir.Plan(1024, 2048, 8, 8, None, M1, tuning=dict(m_sub=2, tile_queries=4, k_atoms=2, stages=3, min_chunks=4,
                                                            whole_units=1, no_collector=1)) as p:
        i = p.info
        assert (i["m_sub"], i["tile_queries"], i["stages"], i["n_chunks"], i["n_tiles"]) == (2, 4, 3, 4, 2)
    with vipir.Plan(1024, 2048, 1, 8, None, G, tuning=dict(stages=6, separate_split=1)) as p:
        assert p.info["stages"] == 6 and p.info["launches"] == 2


def test_plan_used_under_another_current_device_is_refused():
    """A plan belongs to the device current at plan time (include/vipir.h); a call under another current device
    returns INVALID_ARG and enqueues nothing.  Needs two GPUs: skipped on a one-GPU box."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    ensure_built()
    D, Q = make(5, 256, 1024, 8)
    with torch.cuda.device(0):
        d_db = torch.from_numpy(D).cuda()
        d_q = torch.from_numpy(Q.view(np.int32)).cuda()
        d_a = torch.full((1, 8, 256), -1, dtype=torch.int32, device="cuda")
        plan = vipir.Plan(256, 1024, 8)
    with torch.cuda.device(1):
        with pytest.raises(vipir.VipirError) as e:
            plan(d_db, d_q, d_a, stream=0)
        assert e.value.status == vipir.ERR_INVALID_ARG
    with torch.cuda.device(0):
        plan(d_db, d_q, d_a)
        torch.cuda.synchronize()
        assert_same(d_a.cpu().numpy().view(np.uint32), oracle.dbmul(D, Q))
        plan.close()


def test_auto_matches_oracle_on_config_1():
    # BASELINE.json configs[0]: D 1024x1024 u8, Q 1024x1 u32, q = 2^32, seed 0
    D, Q = make(0, 1024, 1024, 1)
    check(D, Q, None, AUTO)


def test_plan_reuse_with_new_buffers_and_host_entry_point():
    import torch
    ensure_built()
    rows, cols, batch = 200, 1040, 8
    with vipir.Plan(rows, cols, batch) as plan:
        for seed in (70, 71):
            D, Q = make(seed, rows, cols, batch)
            d_db = torch.from_numpy(D).cuda()
            d_q = torch.from_numpy(Q.view(np.int32)).cuda()
            d_a = torch.empty((1, batch, rows), dtype=torch.int32, device="cuda")
            plan(d_db, d_q, d_a)
            torch.cuda.synchronize()
            assert_same(d_a.cpu().numpy().view(np.uint32), oracle.dbmul(D, Q))
        h_q = torch.from_numpy(Q.view(np.int32)).pin_memory()
        h_a = torch.empty((1, batch, rows), dtype=torch.int32).pin_memory()
        plan.host(d_db, h_q, h_a)
        assert_same(h_a.numpy().view(np.uint32), oracle.dbmul(D, Q))


@pytest.mark.parametrize("bits", [0, 18])
def test_host_entry_point_batch1_pinned_and_pageable(bits):
    """vipir_dbmul_host at batch 1: into pinned (device-mapped) host memory the scan kernel stores the answer
    directly, into pageable memory it goes through the staged copy -- same words either way, also at an
    unaligned offset inside a pinned buffer and with the fused modulus switch."""
    import torch
    ensure_built()
    rows, cols = 1000, 2080
    D, Q = make(88, rows, cols, 1)
    want = oracle.dbmul(D, Q, nthreads=NT)
    if bits:
        want = oracle.modswitch(want, bits)
    d_db = torch.from_numpy(D).cuda()
    h_q = torch.from_numpy(Q.view(np.int32)).pin_memory()
    with vipir.Plan(rows, cols, 1, modswitch_bits=bits) as plan:
        assert plan.info["regime_name"] == "gemv"
        pinned = torch.full((rows + 7,), -1, dtype=torch.int32).pin_memory()
        for off in (0, 3):
            pinned.fill_(-1)
            h_a = pinned[off:off + rows]
            plan.host(d_db, h_q, h_a)
            assert_same(h_a.numpy().view(np.uint32).reshape(1, 1, rows), want)
            assert (pinned[:off] == -1).all() and (pinned[off + rows:] == -1).all()
        pageable = torch.full((1, 1, rows), -1, dtype=torch.int32)
        plan.host(d_db, h_q, pageable)
        assert_same(pageable.numpy().view(np.uint32), want)
        pageable_q = torch.from_numpy(Q.view(np.int32).copy())
        pinned.fill_(-1)
        plan.host(d_db, pageable_q, pinned[:rows])
        assert_same(pinned[:rows].numpy().view(np.uint32).reshape(1, 1, rows), want)


# the host call of the tensor-core regimes: copy / split / scan pipelined over K slices, every slice adding to the
# running sums of the ones before it, the finished words stored straight into mapped host memory (PAPER.md:245-249's
# K chunks; :176 for the server's per-request path)
@pytest.mark.parametrize("name,rows,cols,batch,bits,moduli,regime,tune,ms,signed", [
    ("M1 3 slices", 300, 2064, 8, 8, None, M1, dict(host_slices=3), 0, False),
    ("M2 4 slices ragged K", 520, 4112, 40, 8, None, M2, dict(host_slices=4), 0, False),
    ("M2 two N halves, 2 slices", 300, 1040, 130, 8, None, M2, dict(host_slices=2), 0, False),
    ("M2 slices of two chunks each", 260, 4 * 32768 + 128, 12, 8, None, M2, dict(host_slices=2), 0, False),
    ("M1 one slice two chunks", 260, 32768 + 256, 8, 8, None, M1, dict(host_slices=1), 0, False),
    ("M1 planner default (one slice)", 200, 1040, 8, 8, None, M1, None, 0, False),
    ("M2 primes 3 slices", 300, 2064, 20, 8, PRIMES, M2, dict(host_slices=3), 0, False),
    ("M1 u16 primes LC=5 3 slices", 260, 1032, 16, 16, PRIMES, M1, dict(host_slices=3), 0, False),
    ("M2 u16 2^32 byte view", 260, 1032, 24, 16, None, M2, dict(host_slices=3), 0, False),
    ("M2 modswitch 3 slices", 300, 2064, 40, 8, None, M2, dict(host_slices=3), 18, False),
    ("M1 signed primes", 300, 2064, 8, 8, PRIMES, M1, dict(host_slices=4), 0, True),
    ("M2 more groups than units", 130, 8192, 8, 8, None, M2, dict(host_slices=4, m_sub=1), 0, False),
    ("M2 staged form", 300, 2064, 40, 8, None, M2, dict(host_staged=1), 0, False),
])
def test_host_entry_point_tensor_regimes(name, rows, cols, batch, bits, moduli, regime, tune, ms, signed):
    import torch
    ensure_built()
    D, Q = make(91, rows, cols, batch, bits, moduli)
    D[0, :] = np.iinfo(D.dtype).max  # an all-max row: every slice's partial sum is large
    want = oracle.dbmul_signed(D, Q, moduli) if signed else oracle.dbmul(D, Q, moduli, nthreads=NT)
    if ms:
        want = oracle.modswitch(want, ms)
    T = Q.shape[0]
    d_db = torch.from_numpy(D.view(np.uint8).reshape(rows, -1)).cuda()
    h_q = torch.from_numpy(Q.view(np.int32)).pin_memory()
    with vipir.Plan(rows, cols, batch, bits, moduli, regime, ms, signed, tuning=tune) as plan:
        pinned = torch.full((T * batch * rows + 5,), -1, dtype=torch.int32).pin_memory()
        for off in (0, 3):  # into mapped host memory, also at an odd word offset
            pinned.fill_(-1)
            h_a = pinned[off:off + T * batch * rows]
            plan.host(d_db, h_q, h_a)
            assert_same(h_a.numpy().view(np.uint32).reshape(T, batch, rows), want)
            assert (pinned[:off] == -1).all() and (pinned[off + T * batch * rows:] == -1).all()
        pageable = torch.full((T, batch, rows), -1, dtype=torch.int32)
        plan.host(d_db, h_q, pageable)  # staged copy back
        assert_same(pageable.numpy().view(np.uint32), want)
        pinned.fill_(-1)
        plan.host(d_db, torch.from_numpy(Q.view(np.int32).copy()), pinned[:T * batch * rows])  # pageable query
        assert_same(pinned[:T * batch * rows].numpy().view(np.uint32).reshape(T, batch, rows), want)
        # the device entry point of the same plan still gives the same words (no plan state was left behind)
        d_a = torch.full((T, batch, rows), -1, dtype=torch.int32, device="cuda")
        plan(d_db, torch.from_numpy(Q.view(np.int32)).cuda(), d_a)
        torch.cuda.synchronize()
        assert_same(d_a.cpu().numpy().view(np.uint32), want)
    # a fresh plan used at once on a non-blocking side stream (plan-time zeroing of the work counters is complete
    # when the plan call returns; the copy stream is ordered after the caller's stream)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side), vipir.Plan(rows, cols, batch, bits, moduli, regime, ms, signed, tuning=tune) as plan:
        pinned.fill_(-1)
        plan.host(d_db, h_q, pinned[:T * batch * rows])
        assert_same(pinned[:T * batch * rows].numpy().view(np.uint32).reshape(T, batch, rows), want)


def test_host_entry_point_at_scale_planner_slices_several_units_per_cta():
    """The server's per-request path (PAPER.md:117 "a D1 x B x D0 ... GEMM for a batch of B queries", :176 the DB
    resident in GPU DRAM) at a size where nothing is forced: 60000 x 8192 u8, B = 256, regime AUTO.  The query is
    8 MiB, so the planner's own rule cuts the call into three K slices; there are several times more work units
    than CTA pairs, so every pair finishes several units per slice -- its two-entry copier ring wraps and its copier
    warps run behind its epilogue warps -- and the rows end in a ragged tile.  The answer, delivered into mapped
    host memory, is compared with the oracle on the first, the last (ragged) and 16 seeded random 128-row tiles,
    all 256 query vectors; the same call into pageable memory and the device call must give the same words
    everywhere."""
    import torch
    from paper_2606_11536_b200.inputs import device
    ensure_built()
    rows, cols, batch, seed = 60000, 8192, 256, 123
    d_db = device.db(seed, rows, cols, 8)
    Q = inputs.query(seed, cols, batch, None)
    assert Q.nbytes == 8 << 20  # the planner's three-slice threshold (no host_slices forced)
    h_q = torch.from_numpy(Q.view(np.int32)).pin_memory()
    h_a = torch.full((1, batch, rows), -1, dtype=torch.int32).pin_memory()
    pageable = torch.full((1, batch, rows), -1, dtype=torch.int32)
    d_a = torch.full((1, batch, rows), -1, dtype=torch.int32, device="cuda")
    with vipir.Plan(rows, cols, batch) as plan:
        i = plan.info
        assert i["regime_name"] == "mma_2sm"
        assert i["n_tiles"] * i["m_tiles"] >= 6 * i["grid"] // 2, i  # >= 6 finished units per CTA pair
        plan.host(d_db, h_q, h_a)
        plan.host(d_db, h_q, pageable)
        plan(d_db, torch.from_numpy(Q.view(np.int32)).cuda(), d_a)
        torch.cuda.synchronize()
    got = h_a.numpy().view(np.uint32)
    n_tiles = (rows + 127) // 128
    tiles = sorted({0, n_tiles - 1, *np.random.default_rng(seed).choice(n_tiles, size=16, replace=False).tolist()})
    assert np.array_equal(d_db[777].cpu().numpy(), inputs.db_rows(seed, rows, cols, 8, row0=777, nrows=1)[0])
    for t0 in tiles:
        r0, r1 = t0 * 128, min(rows, t0 * 128 + 128)
        want = oracle.dbmul(d_db[r0:r1].cpu().numpy(), Q, None, nthreads=NT)
        assert_same(got[:, :, r0:r1], want)
    assert (got[:, :, rows - 96:] != 0xFFFFFFFF).any()  # the ragged tile was written
    assert np.array_equal(pageable.numpy().view(np.uint32), got), "pageable and mapped host answers differ"
    assert np.array_equal(d_a.cpu().numpy().view(np.uint32), got), "host and device entry points differ"


@pytest.mark.parametrize("name,regime,rows,cols,batch,bits,moduli,layout,tune,ms", [
    ("M2 one chunk -> 3", M2, 24000, 2064, 24, 8, None, vipir.DB_ROW_MAJOR, dict(m_sub=1, leftover_chunks=3), 0),
    ("M1 primes one chunk -> 4", M1, 24000, 4112, 8, 8, PRIMES, vipir.DB_ROW_MAJOR, dict(m_sub=1, leftover_chunks=4), 0),
    ("M2 limb planes primes -> 2", M2, 20000, 1040, 12, 16, PRIMES, vipir.DB_LIMB_PLANES, dict(leftover_chunks=2), 0),
    ("M2 two chunks -> 5, switch", M2, 24000, 40000, 8, 8, None, vipir.DB_ROW_MAJOR, dict(m_sub=1, leftover_chunks=5), 18),
    ("M2 u16 byte view primes -> 3", M2, 20000, 1032, 8, 16, PRIMES, vipir.DB_ROW_MAJOR, dict(m_sub=1, leftover_chunks=3), 0),
])
def test_leftover_round_cut_into_finer_chunks(name, regime, rows, cols, batch, bits, moduli, layout, tune, ms):
    """More units than CTA groups, and the units of the last, partial round cut into more K chunks than those of the
    full rounds (vipir_tuning.leftover_chunks; the planner does this by itself for configs[4] held as limb planes):
    device call in full against the oracle, and the K-sliced host call of the same plan (its slices use uniform
    chunks) equal to it."""
    import torch
    D, Q = make(61, rows, cols, batch, bits, moduli)
    want = oracle.dbmul(D, Q, moduli, nthreads=NT)
    if ms:
        want = oracle.modswitch(want, ms)
    got, info = run_dbmul(D, Q, moduli, regime, return_info=True, modswitch_bits=ms, db_layout=layout, tuning=tune)
    groups = info["grid"] // (2 if regime == M2 else 1)
    assert info["m_tiles"] * info["n_tiles"] > groups and (info["m_tiles"] * info["n_tiles"]) % groups != 0, info
    assert info["leftover_chunks"] == tune["leftover_chunks"] > info["n_chunks"], info
    assert_same(got, want)
    if layout == vipir.DB_ROW_MAJOR:
        T = Q.shape[0]
        d_db = torch.from_numpy(D.view(np.uint8).reshape(rows, -1)).cuda()
        h_a = torch.full((T, batch, rows), -1, dtype=torch.int32).pin_memory()
        with vipir.Plan(rows, cols, batch, bits, moduli, regime, ms, tuning=dict(tune, host_slices=2)) as plan:
            plan.host(d_db, torch.from_numpy(Q.view(np.int32)).pin_memory(), h_a)
        assert_same(h_a.numpy().view(np.uint32), want)


def test_leftover_chunks_planner_rule_and_refusals():
    ensure_built()
    # configs[4] as limb planes: 256 one-chunk units on 74 pairs -> the 34 leftover units are cut in two (3.5 rounds, not 4)
    with vipir.Plan(32768, 32768, 64, 16, PRIMES[:2], db_layout=vipir.DB_LIMB_PLANES) as p:
        assert (p.info["n_chunks"], p.info["leftover_chunks"], p.info["m_tiles"] * p.info["n_tiles"], p.info["grid"]) == (1, 2, 256, 148)
    # configs[3]: 68 leftover units of two chunks on 74 pairs -- no finer cut shortens that round
    with vipir.Plan(65536, 65536, 256) as p:
        assert p.info["leftover_chunks"] == p.info["n_chunks"] == 2
    for tune in (dict(leftover_chunks=1, min_chunks=2), dict(leftover_chunks=2, whole_units=1), dict(leftover_chunks=17)):
        with pytest.raises(vipir.VipirError) as e:  # fewer than n_chunks; nothing is split; more than the 16 k-atoms
            vipir.Plan(1024, 2048, 8, 8, None, M1, tuning=tune)
        assert e.value.status == vipir.ERR_UNSUPPORTED, tune


def test_forced_chunk_count_that_does_not_divide_the_k_atoms():
    """6 k-atoms cut into "4" chunks are three chunks of two (a fourth, empty chunk would never complete: this shape
    hung the kernel until the planner counted the chunks that exist).  Found by a random soak of the host call."""
    D, Q = make(81, 742, 736, 28, 8, PRIMES)
    got, info = run_dbmul(D, Q, PRIMES, M1, return_info=True, tuning=dict(min_chunks=4))
    assert info["n_chunks"] == 3 and info["k_chunk_bytes"] == 256
    assert_same(got, oracle.dbmul(D, Q, PRIMES, nthreads=NT))
    for mc, cols in ((5, 896), (7, 1280), (3, 512)):  # 7 k-atoms / 5, 10 / 7, 4 / 3
        D, Q = make(82, 300, cols, 9)
        assert_same(run_dbmul(D, Q, None, M2, tuning=dict(min_chunks=mc)), oracle.dbmul(D, Q, nthreads=NT))


def _random_host_case(rng):
    regime = [M1, M2][int(rng.integers(2))]
    bits = [8, 8, 16][int(rng.integers(3))]
    moduli = [None, PRIMES][int(rng.integers(2))]
    rows = int(rng.integers(1, 700))
    cols = int(rng.integers(1, 300)) * (16 if bits == 8 else 8)
    batch = int(rng.integers(1, 70))
    tune = dict(host_slices=int(rng.integers(1, 5)))
    if rng.integers(3) == 0:
        tune["min_chunks"] = int(rng.integers(1, 4))
    ms = 18 if (moduli is None and rng.integers(3) == 0) else 0
    return regime, bits, moduli, rows, cols, batch, tune, ms


@pytest.mark.parametrize("seed", range(16))
def test_host_entry_point_random_shapes(seed):
    """Seeded random shapes through the K-sliced host call (ragged rows / K / query vectors, 1-4 slices, forced
    extra chunks so that slices hold several chunks and leftover units are shared between groups)."""
    import torch
    ensure_built()
    rng = np.random.default_rng(1000 + seed)
    regime, bits, moduli, rows, cols, batch, tune, ms = _random_host_case(rng)
    D, Q = make(200 + seed, rows, cols, batch, bits, moduli)
    want = oracle.dbmul(D, Q, moduli, nthreads=NT)
    if ms:
        want = oracle.modswitch(want, ms)
    T = Q.shape[0]
    d_db = torch.from_numpy(D.view(np.uint8).reshape(rows, -1)).cuda()
    h_q = torch.from_numpy(Q.view(np.int32)).pin_memory()
    h_a = torch.full((T, batch, rows), -1, dtype=torch.int32).pin_memory()
    try:
        plan = vipir.Plan(rows, cols, batch, bits, moduli, regime, ms, tuning=tune)
    except vipir.VipirError as e:  # an override the shape cannot honour (min_chunks > k-atoms) is refused, not ignored
        assert e.status == vipir.ERR_UNSUPPORTED and "min_chunks" in tune
        tune.pop("min_chunks")
        plan = vipir.Plan(rows, cols, batch, bits, moduli, regime, ms, tuning=tune)
    with plan:
        plan.host(d_db, h_q, h_a)
        assert_same(h_a.numpy().view(np.uint32), want)


def test_host_and_device_entry_points_seeded_soak():
    """A bounded soak in the suite (round 2's unbounded ones ran from working scripts and found the empty-chunk hang
    pinned above): 160 seeded random shapes -- both tensor regimes, u8 / u16, 2^32 / primes, 1-4 K slices, forced extra
    chunks, the fused switch -- each through vipir_dbmul_host into mapped memory AND vipir_dbmul, both against the
    oracle.  A hang shows as the kernel's own trap or the test's timeout, a race as a wrong word."""
    import torch
    ensure_built()
    rng = np.random.default_rng(20261106)
    refused = 0
    for case in range(160):
        regime, bits, moduli, rows, cols, batch, tune, ms = _random_host_case(rng)
        rows, batch = min(rows, 400), min(batch, 40)  # keeps the whole soak at a few seconds of oracle time
        D, Q = make(5000 + case, rows, cols, batch, bits, moduli)
        want = oracle.dbmul(D, Q, moduli, nthreads=NT)
        if ms:
            want = oracle.modswitch(want, ms)
        T = Q.shape[0]
        d_db = torch.from_numpy(D.view(np.uint8).reshape(rows, -1)).cuda()
        h_q = torch.from_numpy(Q.view(np.int32)).pin_memory()
        h_a = torch.full((T, batch, rows), -1, dtype=torch.int32).pin_memory()
        d_a = torch.full((T, batch, rows), -1, dtype=torch.int32, device="cuda")
        try:
            plan = vipir.Plan(rows, cols, batch, bits, moduli, regime, ms, tuning=tune)
        except vipir.VipirError as e:
            assert e.status == vipir.ERR_UNSUPPORTED and "min_chunks" in tune, (case, tune, e)
            refused += 1
            continue
        with plan:
            plan.host(d_db, h_q, h_a)
            plan(d_db, h_q.cuda(), d_a)
            torch.cuda.synchronize()
        what = f"case {case}: {rows}x{cols} B={batch} u{bits} {'primes' if moduli else '2^32'} regime {regime} {tune} ms={ms}"
        assert np.array_equal(h_a.numpy().view(np.uint32), want), "host call, " + what
        assert np.array_equal(d_a.cpu().numpy().view(np.uint32), want), "device call, " + what
    assert refused < 40


def test_two_plans_two_threads_two_streams():
    """One plan per stream (include/vipir.h): two host threads, each with its own plan, side stream and pinned buffers,
    call vipir_dbmul_host repeatedly against the same resident DB; every answer is the oracle's."""
    import threading
    import torch
    ensure_built()
    rows, cols, batch = 520, 4112, 40
    D = inputs.db_rows(95, rows, cols, 8)
    d_db = torch.from_numpy(D).cuda()
    Qs = [inputs.query(96 + i, cols, batch) for i in range(2)]
    wants = [oracle.dbmul(D, Q, nthreads=NT) for Q in Qs]
    errors = []

    def worker(i):
        try:
            torch.cuda.set_device(0)
            side = torch.cuda.Stream()
            h_q = torch.from_numpy(Qs[i].view(np.int32)).pin_memory()
            h_a = torch.full((1, batch, rows), -1, dtype=torch.int32).pin_memory()
            with torch.cuda.stream(side), vipir.Plan(rows, cols, batch, 8, None, M2, tuning=dict(host_slices=3)) as plan:
                for _ in range(25):
                    h_a.fill_(-1)
                    plan.host(d_db, h_q, h_a)
                    if not np.array_equal(h_a.numpy().view(np.uint32), wants[i]):
                        errors.append(f"thread {i}: answer differs")
                        return
        except Exception as e:  # noqa: BLE001
            errors.append(f"thread {i}: {e!r}")
    th = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not errors, errors


@pytest.mark.parametrize("regime,batch,moduli", [(G, 1, None), (M1, 8, None), (M2, 40, PRIMES)])
def test_device_call_is_cuda_graph_capturable(regime, batch, moduli):
    """vipir_dbmul only enqueues kernels (no allocation, no synchronisation, work counters reset by the kernel itself), so a
    call can be captured into a CUDA graph and replayed with new query contents in the same buffers."""
    import torch
    ensure_built()
    rows, cols = 700, 33024 if regime != G else 2080   # two K chunks in the tensor regimes: units shared between groups
    D = inputs.db_rows(77, rows, cols, 8)
    d_db = torch.from_numpy(D).cuda()
    T = 1 if moduli is None else len(moduli)
    d_q = torch.zeros((T, batch, cols), dtype=torch.int32, device="cuda")
    d_a = torch.full((T, batch, rows), -1, dtype=torch.int32, device="cuda")
    with vipir.Plan(rows, cols, batch, 8, moduli, regime) as plan:
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            plan(d_db, d_q, d_a)            # first call outside the capture: sets the kernels' attributes, encodes the maps
            side.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=side):
                plan(d_db, d_q, d_a)
        for seed in (1, 2, 3):
            Q = inputs.query(300 + seed, cols, batch, moduli)
            d_q.copy_(torch.from_numpy(Q.view(np.int32)))
            d_a.fill_(-1)
            graph.replay()
            torch.cuda.synchronize()
            assert_same(d_a.cpu().numpy().view(np.uint32), oracle.dbmul(D, Q, moduli, nthreads=NT))


def test_misaligned_pointers_are_rejected():
    import torch
    ensure_built()
    with vipir.Plan(64, 64, 1) as plan:
        buf = torch.zeros(64 * 64 + 64, dtype=torch.uint8, device="cuda")
        q = torch.zeros(64, dtype=torch.int32, device="cuda")
        a = torch.zeros(64, dtype=torch.int32, device="cuda")
        with pytest.raises(vipir.VipirError) as e:
            vipir.dbmul(plan.handle, buf.data_ptr() + 1, q, a)
        assert e.value.status == vipir.ERR_INVALID_ARG


def test_toy_lwe_roundtrip_through_the_gpu():
    """SimplePIR end to end: the GPU's answer decrypts to the
    selected DB column.  Uses the oracle package's toy client only for keys/queries/decrypt."""
    from oracle import lwe
    cols, rows, n = 1024, 200, 15  # n+1 = 16 query vectors
    g = np.random.default_rng(5)
    D = inputs.db_rows(77, rows, cols, 8)
    s = lwe.keygen(n, g)
    Q, _ = lwe.simplepir_query(cols, 321, s, g)
    A = run_dbmul(D, Q.reshape(1, n + 1, cols), None, AUTO)[0]
    assert np.array_equal(lwe.decrypt_answer(A, s), D[:, 321])


# ---- NEXT-1: fused modulus switch 2^32 -> 2^18 -----------------------

@pytest.mark.parametrize("regime,rows,cols,batch", [
    (G, 100, 4112, 1), (M1, 300, 1552, 8), (M2, 300, 1552, 40),
    (M1, 130, 32768 * 2 + 4112, 2), (M2, 260, 32768 + 528, 130),  # several K chunks: the last one rounds
])
@pytest.mark.parametrize("bits", [18, 31, 1])
def test_fused_modswitch(regime, rows, cols, batch, bits):
    D, Q = make(200 + batch, rows, cols, batch)
    D[: rows // 2] = 255  # large sums: exercise the wrap before the rounding
    got, info = run_dbmul(D, Q, None, regime, return_info=True, modswitch_bits=bits)
    assert info["modswitch_bits"] == bits
    want = oracle.modswitch(oracle.dbmul(D, Q, None, nthreads=NT), bits)
    assert_same(got, want)
    assert got.max() < (1 << bits)


def test_modswitch_rejected_for_prime_moduli():
    ensure_built()
    with vipir.Plan(256, 256, 2, 8, PRIMES) as plan:
        with pytest.raises(vipir.VipirError) as e:
            vipir.plan_set_modswitch(plan.handle, 18)
        assert e.value.status == vipir.ERR_UNSUPPORTED
    with vipir.Plan(256, 256, 2) as plan:
        with pytest.raises(vipir.VipirError) as e:
            vipir.plan_set_modswitch(plan.handle, 32)
        assert e.value.status == vipir.ERR_INVALID_ARG
        vipir.plan_set_modswitch(plan.handle, 18)
        vipir.plan_set_modswitch(plan.handle, 0)
        assert vipir.plan_info(plan.handle)["modswitch_bits"] == 0


def test_modswitched_gpu_answer_decrypts():
    from oracle import lwe
    cols, rows, n = 1024, 200, 15
    g = np.random.default_rng(6)
    D = inputs.db_rows(78, rows, cols, 8)
    s = lwe.keygen(n, g)
    Q, _ = lwe.simplepir_query(cols, 77, s, g)
    A18 = run_dbmul(D, Q.reshape(1, n + 1, cols), None, AUTO, modswitch_bits=18)[0]
    assert np.array_equal(lwe.decrypt_answer_switched(A18, s, 18), D[:, 77])


# ---- NEXT-3: signed int8 DB (centred plaintexts) ---------------------------------

@pytest.mark.parametrize("regime,rows,cols,batch,moduli", [
    (G, 100, 4112, 1, None), (NAIVE, 70, 192, 3, None), (NAIVE, 70, 192, 3, PRIMES),
    (M1, 300, 1552, 8, None), (M2, 300, 1552, 40, None), (M1, 300, 1552, 5, PRIMES), (M2, 300, 1552, 40, PRIMES),
    (M1, 130, 32768 * 2 + 4112, 2, None), (M2, 260, 32768 + 528, 70, PRIMES),  # K-chunk seams
    (AUTO, 1024, 1024, 1, None), (AUTO, 260, 1040, 256, None),
])
def test_signed_db(regime, rows, cols, batch, moduli):
    D, Q = make(400 + batch, rows, cols, batch, 8, moduli)
    D[: rows // 4] = 0x80      # all -128: most negative limb sums, every accumulator at -128*255*K_chunk
    D[rows // 4: rows // 2] = 0x7F
    if moduli is None:
        Q[0, 0, : min(cols, 64)] = 0xFFFFFFFF
    got, info = run_dbmul(D, Q, moduli, regime, return_info=True, db_signed=True)
    assert info["db_signed"] == 1
    assert_same(got, oracle.dbmul_signed(D, Q, moduli))
    if moduli:
        for t, pt in enumerate(moduli):
            assert (got[t] < pt).all()


def test_signed_db_all_min_exact_chunk():
    # every s32 accumulator at its most negative: -128 * 255 * 32768 > -2^31 (R7 holds a fortiori)
    cols = 32768
    D = np.full((128, cols), 0x80, dtype=np.uint8)
    Q = np.full((1, 4, cols), 0xFFFFFFFF, dtype=np.uint32)
    for regime in (M1, M2):
        got = run_dbmul(D, Q, None, regime, db_signed=True)
        assert (got == (-128 * 0xFFFFFFFF * cols) % (1 << 32)).all()
        p = PRIMES[1]
        got = run_dbmul(D, Q, [p], regime, db_signed=True)
        assert (got == (-128 * 0xFFFFFFFF * cols) % p).all()


def test_signed_db_with_modswitch_and_lwe():
    """A centred DB decrypts to the signed byte (m in [-p/2, p/2)); also through the
    fused modulus switch."""
    from oracle import lwe
    cols, rows, n = 1024, 200, 15
    g = np.random.default_rng(8)
    D = inputs.db_rows(79, rows, cols, 8)
    s = lwe.keygen(n, g)
    Q, _ = lwe.simplepir_query(cols, 500, s, g)
    A = run_dbmul(D, Q.reshape(1, n + 1, cols), None, AUTO, db_signed=True)[0]
    assert np.array_equal(lwe.decrypt_answer(A, s), D[:, 500])  # the byte pattern of the signed value mod 2^8
    A18 = run_dbmul(D, Q.reshape(1, n + 1, cols), None, AUTO, modswitch_bits=18, db_signed=True)[0]
    assert np.array_equal(lwe.decrypt_answer_switched(A18, s, 18), D[:, 500])


def test_signed_db_rejected_for_u16():
    ensure_built()
    with vipir.Plan(256, 256, 2, 16) as plan:
        with pytest.raises(vipir.VipirError) as e:
            vipir.plan_set_db_signed(plan.handle, True)
        assert e.value.status == vipir.ERR_UNSUPPORTED
    with vipir.Plan(256, 256, 2, 8) as plan:
        vipir.plan_set_db_signed(plan.handle, True)
        assert vipir.plan_info(plan.handle)["db_signed"] == 1
        vipir.plan_set_db_signed(plan.handle, False)
        assert vipir.plan_info(plan.handle)["db_signed"] == 0


# ---- NEXT-2: other shapes of the same product ---------------------------------

@pytest.mark.parametrize("rows,cols,batch", [
    (260, 528, 1281),   # DoublePIR-style B = n+1 = 1281 query vectors: 11 N tiles
    (4100, 144, 40),    # tall layout, rows >> cols, 17 M-pair tiles, ragged
    (130, 272, 1280),   # hint precomputation B = n = 1280
])
def test_other_shapes_of_the_product(rows, cols, batch):
    D, Q = make(300 + batch, rows, cols, batch)
    got, info = run_dbmul(D, Q, None, AUTO, return_info=True)
    assert info["regime_name"] == "mma_2sm" and info["n_tiles"] == -(-batch // info["tile_queries"])
    assert_same(got, oracle.dbmul(D, Q, None, nthreads=NT))


# ---- seeded random shapes: every regime the planner can pick, ragged everywhere ----------------

def _random_cases(n, seed):
    g = np.random.default_rng(seed)
    cases = []
    for _ in range(n):
        db_bits = int(g.choice([8, 8, 16]))
        dl = db_bits // 8
        rows = int(g.integers(1, 700))
        cols = int(g.integers(1, 260)) * (16 // dl)          # row bytes a multiple of 16
        if g.random() < 0.15:
            cols += (32768 // dl) * int(g.integers(1, 3))      # cross one or two K-chunk seams
            rows = int(g.integers(1, 200))
        kind = g.random()
        if kind < 0.35:
            moduli = None
        elif kind < 0.6:
            moduli = [int(g.integers(2, 1 << 30))]
        else:
            moduli = [int(g.integers(2, 1 << 30)) for _ in range(int(g.integers(2, 5)))]
        batch = int(g.choice([1, 1, 2, 3, 5, 8, 17, 33, 70, 150]))
        if cols * dl > 40000:
            batch = min(batch, 8)
        cases.append((rows, cols, batch, db_bits, moduli))
    return cases


@pytest.mark.parametrize("case", _random_cases(40, 2024), ids=lambda c: f"{c[0]}x{c[1]}xB{c[2]}u{c[3]}m{0 if c[4] is None else len(c[4])}")
def test_random_shapes_auto(case):
    rows, cols, batch, db_bits, moduli = case
    D, Q = make(rows * 31 + cols, rows, cols, batch, db_bits, moduli)
    if moduli is None:
        Q[0, 0, : min(cols, 5)] = 0xFFFFFFFF
    check(D, Q, moduli, AUTO)
