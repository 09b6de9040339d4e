"""GPU parity for the limb-plane u16 database layout (include/vipir.h: VIPIR_DB_LIMB_PLANES;
BASELINE.json configs[4]: "uint16 ... (split into 2 u8 limbs)").

The answer is defined on the u16 database (oracle.dbmul gets the u16 matrix); the library scans the
two byte matrices vipir_db_split_u16 made of it.  Bit-exact, no tolerance.
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
M1, M2, AUTO = vipir.REGIME_MMA_1SM, vipir.REGIME_MMA_2SM, vipir.REGIME_AUTO
LP = vipir.DB_LIMB_PLANES


def assert_same(got, want):
    bad = np.argwhere(got != want)
    assert bad.size == 0, (f"{len(bad)} of {got.size} words differ; first at [t,b,r]={bad[0].tolist()}: "
                           f"got {got[tuple(bad[0])]} want {want[tuple(bad[0])]}")


@pytest.mark.parametrize("rows,cols", [(1, 16), (3, 48), (257, 2064), (1024, 4096)])
def test_db_split_u16_is_the_byte_deinterleave(rows, cols):
    """D_lo = D & 0xFF, D_hi = D >> 8, D_hi directly behind D_lo; nothing written outside."""
    import torch
    ensure_built()
    D = inputs.db_rows(11, rows, cols, 16)
    d_db = torch.from_numpy(D.view(np.uint8).reshape(rows, -1)).cuda()
    guard = 4096
    buf = torch.full((2 * rows * cols + 2 * guard,), 0xA5, dtype=torch.uint8, device="cuda")
    out = buf[guard:guard + 2 * rows * cols]
    vipir.db_split_u16(d_db, out, rows, cols)
    torch.cuda.synchronize()
    h = buf.cpu().numpy()
    assert (h[:guard] == 0xA5).all() and (h[-guard:] == 0xA5).all()
    planes = h[guard:-guard].reshape(2, rows, cols)
    assert np.array_equal(planes[0], (D & 0xFF).astype(np.uint8))
    assert np.array_equal(planes[1], (D >> 8).astype(np.uint8))


def test_db_split_u16_argument_errors():
    import torch
    ensure_built()
    a = torch.zeros(2 * 16 * 32 + 64, dtype=torch.uint8, device="cuda")
    b = torch.zeros(2 * 16 * 32 + 64, dtype=torch.uint8, device="cuda")
    for args, status in [((a, b, 0, 32), vipir.ERR_INVALID_ARG), ((a, b, 16, 0), vipir.ERR_INVALID_ARG),
                         ((a, b, 16, 24), vipir.ERR_UNSUPPORTED), ((a[1:], b, 16, 32), vipir.ERR_INVALID_ARG),
                         ((a, a[16:], 16, 32), vipir.ERR_INVALID_ARG), ((0, b, 16, 32), vipir.ERR_INVALID_ARG)]:
        with pytest.raises(vipir.VipirError) as e:
            vipir.db_split_u16(*args)
        assert e.value.status == status, args[2:]


@pytest.mark.parametrize("regime", [M1, M2])
@pytest.mark.parametrize("moduli,batch", [(None, 1), (None, 4), (PRIMES, 1), (PRIMES, 3), (PRIMES, 40),
                                          ([97, 1 << 29, 2, PRIMES[1]], 2), ([PRIMES[0]], 100)])
def test_limb_planes_match_the_u16_definition(regime, moduli, batch):
    # rows: several tiles + ragged tail (the D_lo tail tile reads into D_hi: those rows are masked);
    # K: ragged against the 128-byte k-atom
    rows, cols = 300, 784
    D = inputs.db_rows(70 + batch, rows, cols, 16)
    Q = inputs.query(70 + batch, cols, batch, moduli)
    got, info = run_dbmul(D, Q, moduli, regime, return_info=True, db_layout=LP)
    assert info["db_layout"] == LP and info["limb_cols"] == 4 and info["db_limbs"] == 2 and info["m_sub"] % 2 == 0
    assert info["k_bytes"] == cols
    assert_same(got, oracle.dbmul(D, Q, moduli, nthreads=NT))


@pytest.mark.parametrize("regime", [M1, M2])
@pytest.mark.parametrize("msub", [2, 4])
@pytest.mark.parametrize("moduli,bits", [(None, 0), (None, 18), (PRIMES, 0)])
def test_limb_planes_subtiles_chunks_and_split_units(regime, msub, moduli, bits):
    # msub = 4: two row blocks x two limb planes per CTA; K: 3 chunks so that leftover units are dealt
    # out chunk by chunk and accumulated through the answer buffer
    rows, cols, batch = 128 * 2 * (msub // 2) * 2 + 128 + 37, 32768 * 2 + 2064, 6
    D = inputs.db_rows(400 + msub, rows, cols, 16)
    Q = inputs.query(400 + msub, cols, batch, moduli)
    got, info = run_dbmul(D, Q, moduli, regime, return_info=True, modswitch_bits=bits, db_layout=LP, tuning={"m_sub": msub})
    assert info["m_sub"] == msub and info["n_chunks"] == 3
    want = oracle.dbmul(D, Q, moduli, nthreads=NT)
    if bits:
        want = oracle.modswitch(want, bits)
    assert_same(got, want)


@pytest.mark.parametrize("regime", [M1, M2])
def test_limb_planes_permutation_probe_tells_the_planes_apart(regime):
    """One-hot rows whose single element is 1 (D_lo only), 256 (D_hi only) or 257: a swapped or
    misplaced limb tile changes the answer by a factor of 256."""
    rows, cols, batch = 128 * 2 * 2 + 50, 512, 8
    rng = np.random.default_rng(9)
    perm = rng.integers(0, cols, size=rows)
    val = np.array([1, 256, 257], dtype=np.uint64)[rng.integers(0, 3, size=rows)]
    D = np.zeros((rows, cols), dtype=np.uint16)
    D[np.arange(rows), perm] = val
    Q = np.stack([(np.arange(cols, dtype=np.uint64) + 1) * (b + 1) * 0x010101 % (1 << 32) for b in range(batch)])
    Q = Q.astype(np.uint32).reshape(1, batch, cols)
    got = run_dbmul(D, Q, None, regime, db_layout=LP)
    for b in range(batch):
        want = (Q[0, b, perm].astype(np.uint64) * val) % (1 << 32)
        assert np.array_equal(got[0, b], want.astype(np.uint32)), f"query {b}"


@pytest.mark.parametrize("regime", [M1, M2])
def test_limb_planes_all_max_at_the_chunk_bound(regime):
    """Every int32 limb sum at 255^2 * 32768 (R7) in both planes; closed forms over the integers."""
    cols = 32768 + 128
    D = np.full((130, cols), 0xFFFF, dtype=np.uint16)
    Q = np.full((2, 1, cols), 0xFFFFFFFF, dtype=np.uint32)
    got = run_dbmul(D, Q, PRIMES, regime, db_layout=LP)
    for t, pt in enumerate(PRIMES):
        assert (got[t] == (0xFFFF * 0xFFFFFFFF * cols) % pt).all()
    Q1 = np.full((1, 3, cols), 0xFFFFFFFF, dtype=np.uint32)
    got = run_dbmul(D, Q1, None, regime, db_layout=LP)
    assert (got == (0xFFFF * 0xFFFFFFFF * cols) % (1 << 32)).all()


def test_limb_planes_auto_regime_and_rejections():
    ensure_built()
    with vipir.Plan(512, 256, 1, 16, None, AUTO, db_layout=LP) as p:
        assert p.info["regime_name"] == "mma_1sm"  # no GEMV for limb planes
    with vipir.Plan(512, 256, 64, 16, PRIMES, AUTO, db_layout=LP) as p:
        assert p.info["regime_name"] == "mma_2sm" and p.info["tile_cols"] <= 256
    for kw, status in [(dict(db_bits=8), vipir.ERR_UNSUPPORTED), (dict(db_bits=16, regime=vipir.REGIME_GEMV), vipir.ERR_UNSUPPORTED),
                       (dict(db_bits=16, regime=vipir.REGIME_NAIVE), vipir.ERR_UNSUPPORTED),
                       (dict(db_bits=16, cols=24), vipir.ERR_UNSUPPORTED), (dict(db_bits=16, db_layout=2), vipir.ERR_INVALID_ARG)]:
        args = dict(rows=64, cols=32, batch=1, db_bits=16, moduli=None, regime=AUTO, db_layout=LP)
        args.update(kw)
        with pytest.raises(vipir.VipirError) as e:
            vipir.dbmul_plan(**args)
        assert e.value.status == status, kw


def test_limb_planes_host_entry_point_and_plan_reuse():
    import torch
    ensure_built()
    rows, cols, batch = 700, 1040, 5
    D = inputs.db_rows(5, rows, cols, 16)
    d_raw = torch.from_numpy(D.view(np.uint8).reshape(rows, -1)).cuda()
    d_db = torch.empty_like(d_raw)
    vipir.db_split_u16(d_raw, d_db, rows, cols)
    with vipir.Plan(rows, cols, batch, 16, PRIMES, AUTO, db_layout=LP) as plan:
        for seed in (1, 2):
            Q = inputs.query(seed, cols, batch, PRIMES)
            h_q = torch.from_numpy(Q.view(np.int32)).pin_memory()
            h_a = torch.full((2, batch, rows), -1, dtype=torch.int32).pin_memory()
            plan.host(d_db, h_q, h_a)
            assert_same(h_a.numpy().view(np.uint32), oracle.dbmul(D, Q, PRIMES, nthreads=NT))


def _random_cases(n, seed):
    g = np.random.default_rng(seed)
    cases = []
    for _ in range(n):
        rows = int(g.integers(1, 900))
        cols = int(g.integers(1, 300)) * 16
        if g.random() < 0.2:
            cols += 32768 * int(g.integers(1, 3))              # cross one or two K-chunk seams
            rows = int(g.integers(1, 300))
        kind = g.random()
        moduli = None if kind < 0.35 else [int(g.integers(2, 1 << 30)) for _ in range(int(g.integers(1, 5)))]
        batch = int(g.choice([1, 2, 3, 5, 8, 17, 33, 64, 70, 130]))
        if cols > 40000:
            batch = min(batch, 8)
        regime = int(g.choice([AUTO, M1, M2]))
        cases.append((rows, cols, batch, moduli, regime))
    return cases


@pytest.mark.parametrize("case", _random_cases(30, 2025),
                         ids=lambda c: f"{c[0]}x{c[1]}xB{c[2]}m{0 if c[3] is None else len(c[3])}r{c[4]}")
def test_random_shapes_limb_planes(case):
    rows, cols, batch, moduli, regime = case
    D = inputs.db_rows(rows * 31 + cols, rows, cols, 16)
    Q = inputs.query(rows * 31 + cols, cols, batch, moduli)
    if moduli is None:
        Q[0, 0, : min(cols, 5)] = 0xFFFFFFFF
    got = run_dbmul(D, Q, moduli, regime, db_layout=LP)
    assert_same(got, oracle.dbmul(D, Q, moduli, nthreads=NT))
