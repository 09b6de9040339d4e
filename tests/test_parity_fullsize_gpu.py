"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(VIPIR_REGIME_AUTO).  The DB is generated on the device by the input generator's device twin
(tests/test_inputs.py proves it equals the host twin); the oracle recomputes

  * sampled rows one by one (first/last rows, tile boundaries, seeded random rows) from the
    host twin's bytes -- every query vector of those rows, bit for bit; and
  * a column-sum identity over ALL rows, which holds at any size:
        sum_r answer[t][b][r]  =  sum_k (sum_r D[r][k]) * Q[t][b][k]      (mod q_t)
    (linearity, eq. (1)), with the DB column sums taken by a plain torch
    reduction that shares nothing with libvipir.

configs[1] (1 GiB, B = 1) is compared in full.
"""
import os

import numpy as np
import pytest

import oracle
from paper_2606_11536_b200 import inputs, vipir

from gpu_util import ensure_built

pytestmark = pytest.mark.gpu

PRIMES = inputs.rns_primes(0)
NT = max(1, os.cpu_count() or 1)
SEED = 0

CONFIGS = {
    # name: rows, cols, batch, db_bits, moduli, expected regime
    "C2_1GiB_B1": (32768, 32768, 1, 8, None, "gemv"),
    "C3_16GiB_B1": (131072, 131072, 1, 8, None, "gemv"),
    "C3_16GiB_B8": (131072, 131072, 8, 8, None, "mma_1sm"),
    "C4_4GiB_B256": (65536, 65536, 256, 8, None, "mma_2sm"),
    "C5_rns_u16_B64": (32768, 32768, 64, 16, PRIMES, "mma_2sm"),
}


@pytest.fixture(scope="module")
def device_db():
    """16 GiB of the seed-0 DB byte stream; every config's DB is a prefix of it."""
    import torch
    from paper_2606_11536_b200.inputs import device
    ensure_built()
    buf = device.db(SEED, 131072, 131072, 8).view(-1)
    torch.cuda.synchronize()
    yield buf
    del buf
    torch.cuda.empty_cache()


def sample_rows(rows, n_random=24):
    fixed = [0, 1, 31, 32, 127, 128, 255, 256, rows // 2 - 1, rows // 2, rows - 129, rows - 128, rows - 2, rows - 1]
    rnd = np.random.default_rng(rows).integers(0, rows, size=n_random).tolist()
    return sorted(set(r for r in fixed + rnd if 0 <= r < rows))


def run(name, device_db, limb_planes=False):
    import torch
    from paper_2606_11536_b200.inputs import device
    rows, cols, batch, db_bits, moduli, regime = CONFIGS[name]
    kb = cols * db_bits // 8
    d_db = device_db[: rows * kb].view(rows, kb)
    d_q = device.query(SEED, cols, batch, moduli)
    T = d_q.shape[0]
    d_a = torch.full((T, batch, rows), -1, dtype=torch.int32, device="cuda")
    d_scan, layout = d_db, vipir.DB_ROW_MAJOR
    if limb_planes:  # the u16 DB re-laid out once into its two byte-limb planes (vipir_db_split_u16)
        d_scan, layout = torch.empty_like(d_db), vipir.DB_LIMB_PLANES
        vipir.db_split_u16(d_db, d_scan, rows, cols)
    with vipir.Plan(rows, cols, batch, db_bits, moduli, db_layout=layout) as plan:
        assert plan.info["regime_name"] == regime
        plan(d_scan, d_q, d_a)
        torch.cuda.synchronize()
    return d_db, d_q, d_a


def check_sampled_rows(name, d_a):
    rows, cols, batch, db_bits, moduli, _ = CONFIGS[name]
    Q = inputs.query(SEED, cols, batch, moduli)
    rs = sample_rows(rows)
    D = np.concatenate([inputs.db_rows(SEED, rows, cols, db_bits, row0=r, nrows=1) for r in rs])
    want = oracle.dbmul(D, Q, moduli, nthreads=NT)  # [T][B][len(rs)]
    got = d_a[:, :, rs].cpu().numpy().view(np.uint32)
    bad = np.argwhere(got != want)
    assert bad.size == 0, f"{name}: {len(bad)} sampled words differ, first at t,b,i={bad[0].tolist()} (row {rs[bad[0][2]]})"
    if moduli:
        for t, p in enumerate(moduli):
            assert int(d_a[t].max()) < p and int(d_a[t].min()) >= 0  # canonical range, every word


def check_column_sum_identity(name, d_db, d_a):
    import torch
    rows, cols, batch, db_bits, moduli, _ = CONFIGS[name]
    Q = inputs.query(SEED, cols, batch, moduli).astype(np.uint64)
    colsum_bytes = torch.sum(d_db, dim=0, dtype=torch.int64).cpu().numpy().astype(np.uint64)
    if db_bits == 16:
        colsum = colsum_bytes[0::2] + np.uint64(256) * colsum_bytes[1::2]
    else:
        colsum = colsum_bytes
    ans_sum = (d_a.to(torch.int64) & 0xFFFFFFFF).sum(dim=-1).cpu().numpy()  # exact: < 2^32 * 2^17
    T = Q.shape[0]
    for t in range(T):
        if not moduli:
            with np.errstate(over="ignore"):
                want = (colsum[None, :] * Q[t]).sum(axis=1) & np.uint64(0xFFFFFFFF)  # u64 wrap is exact mod 2^32
            got = ans_sum[t].astype(np.uint64) & np.uint64(0xFFFFFFFF)
        else:
            p = np.uint64(moduli[t])
            want = (((colsum % p)[None, :] * Q[t]) % p).sum(axis=1) % p  # products < 2^60, sum < 2^45
            got = ans_sum[t].astype(np.uint64) % p
        assert np.array_equal(got, want), f"{name}: column-sum identity fails for modulus index {t}"


def test_config2_full_compare(device_db):
    name = "C2_1GiB_B1"
    rows, cols, batch, db_bits, moduli, _ = CONFIGS[name]
    d_db, d_q, d_a = run(name, device_db)
    D = d_db.cpu().numpy()
    assert np.array_equal(D[:2], inputs.db_rows(SEED, rows, cols, 8, 0, 2))
    want = oracle.dbmul(D, inputs.query(SEED, cols, batch), nthreads=NT)
    assert np.array_equal(d_a.cpu().numpy().view(np.uint32), want)


@pytest.mark.parametrize("name", ["C3_16GiB_B1", "C3_16GiB_B8", "C4_4GiB_B256", "C5_rns_u16_B64"])
def test_fullsize_sampled_rows_and_column_sums(name, device_db):
    d_db, d_q, d_a = run(name, device_db)
    check_sampled_rows(name, d_a)
    check_column_sum_identity(name, d_db, d_a)


def test_config5_limb_plane_layout(device_db):
    """configs[4] with the u16 DB held as its two byte-limb planes (bench.py: C5_rns_u16_B64x2_planes):
    same answer as the u16 definition -- sampled rows, every word canonical, column sums over all rows."""
    name = "C5_rns_u16_B64"
    d_db, d_q, d_a = run(name, device_db, limb_planes=True)
    check_sampled_rows(name, d_a)
    check_column_sum_identity(name, d_db, d_a)


# ---- NEXT-2 at full size: hint precomputation and a tall 4 GiB layout ---------------------------

CONFIGS["N2_hint_4GiB_B1280"] = (65536, 65536, 1280, 8, None, "mma_2sm")
CONFIGS["N2_tall_4GiB_B32"] = (1 << 20, 4096, 32, 8, None, "mma_2sm")        # D/D0 = 2^8 tall layout, :331


@pytest.mark.parametrize("name", ["N2_hint_4GiB_B1280", "N2_tall_4GiB_B32"])
def test_next2_fullsize_sampled_rows(name, device_db):
    d_db, d_q, d_a = run(name, device_db)
    check_sampled_rows(name, d_a)
    check_column_sum_identity(name, d_db, d_a)
