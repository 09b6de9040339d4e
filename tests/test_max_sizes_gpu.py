"""GPU parity at the ABI's size limits (include/vipir.h: rows and K' = cols*db_bits/8 must be < 2^31).

Two degenerate-but-legal shapes that push every row / K coordinate to its largest value:
  * rows = 2^31 - 1 (odd: ragged against every tile), cols = 16   -- 32 GiB DB, one 16-byte K step;
  * cols = 2^31 - 16, rows = 2                                     -- 4 GiB DB, 65536 K chunks of one unit
                                                                      dealt out chunk by chunk.
Inputs come from the device twin of the seeded generator (tests/test_inputs.py proves it equals the host
twin); the oracle recomputes sampled rows from the same bytes, and a column-sum identity (eq. (1),
PAPER.md:76) covers every row.  Bit-exact.  Skipped when the device has less than 100 GB free.
"""
import os

import numpy as np
import pytest

import oracle
from paper_2606_11536_b200 import inputs, vipir

from gpu_util import ensure_built

pytestmark = pytest.mark.gpu

NT = max(1, os.cpu_count() or 1)
SEED = 3
PRIMES = inputs.rns_primes(0)


def _need_memory(gb):
    import torch
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < gb * (1 << 30):
        pytest.skip(f"needs {gb} GiB of free device memory, {free >> 30} GiB available")


@pytest.mark.parametrize("batch,moduli,regime", [(1, None, "gemv"), (2, [PRIMES[0]], "mma_1sm")])
def test_maximum_rows(batch, moduli, regime):
    import torch
    from paper_2606_11536_b200.inputs import device
    ensure_built()
    _need_memory(100)
    rows, cols = (1 << 31) - 1, 16
    d_db = device.db(SEED, rows + 1, cols, 8)[:rows]          # generator fills whole 8-byte words
    d_q = device.query(SEED, cols, batch, moduli)
    T = d_q.shape[0]
    d_a = torch.full((T, batch, rows), -1, dtype=torch.int32, device="cuda")
    with vipir.Plan(rows, cols, batch, 8, moduli) as plan:
        assert plan.info["regime_name"] == regime
        plan(d_db, d_q, d_a)
        torch.cuda.synchronize()
    # sampled rows, recomputed by the oracle from the host twin's bytes
    rs = sorted(set([0, 1, 31, 32, 127, 128, rows // 2, rows - 129, rows - 128, rows - 33, rows - 32, rows - 2, rows - 1]
                    + np.random.default_rng(rows).integers(0, rows, size=40).tolist()))
    D = np.concatenate([inputs.db_rows(SEED, rows + 1, cols, 8, row0=r, nrows=1) for r in rs])
    assert np.array_equal(D, d_db[rs].cpu().numpy())
    Q = inputs.query(SEED, cols, batch, moduli)
    want = oracle.dbmul(D, Q, moduli, nthreads=NT)
    got = d_a[:, :, rs].cpu().numpy().view(np.uint32)
    assert np.array_equal(got, want), np.argwhere(got != want)[:4]
    # column sums over all rows: sum_r answer[r] = sum_k (sum_r D[r][k]) Q[k]  (mod q)
    colsum = np.zeros(cols, dtype=object)
    step = 1 << 28
    for r0 in range(0, rows, step):
        part = torch.sum(d_db[r0:r0 + step], dim=0, dtype=torch.int64).cpu().numpy()
        colsum += np.array([int(x) for x in part], dtype=object)
    q = moduli[0] if moduli else 1 << 32
    for b in range(batch):
        total = 0
        for r0 in range(0, rows, step):
            total += int((d_a[0, b, r0:r0 + step].to(torch.int64) & 0xFFFFFFFF).sum())
        want_sum = sum(int(c) * int(w) for c, w in zip(colsum, Q[0, b])) % q
        assert total % q == want_sum, f"query {b}"
    if moduli:
        assert int(d_a.max()) < q and int(d_a.min()) >= 0


@pytest.mark.parametrize("batch,moduli,regime", [(1, None, "gemv"), (2, None, "mma_1sm"), (1, [PRIMES[1]], "mma_1sm")])
def test_maximum_k(batch, moduli, regime):
    import torch
    from paper_2606_11536_b200.inputs import device
    ensure_built()
    _need_memory(40)
    rows, cols = 2, (1 << 31) - 16
    d_db = device.db(SEED, rows, cols, 8)
    d_q = device.query(SEED, cols, batch, moduli)
    T = d_q.shape[0]
    d_a = torch.full((T, batch, rows), -1, dtype=torch.int32, device="cuda")
    with vipir.Plan(rows, cols, batch, 8, moduli) as plan:
        info = plan.info
        assert info["regime_name"] == regime
        if regime != "gemv":
            assert info["n_chunks"] == 65536
        plan(d_db, d_q, d_a)
        plan(d_db, d_q, d_a)   # again: the in-kernel reset of the arrival counters
        torch.cuda.synchronize()
    D = d_db.cpu().numpy()
    # the device generator's bytes are the host twin's: slices at the start, a row seam and the very end
    from paper_2606_11536_b200.inputs import generator as gen
    key = gen.stream_key(SEED, gen.STREAM_DB)
    flat = D.reshape(-1)
    for start in (0, cols - 2048, rows * cols - 4096):
        assert np.array_equal(flat[start:start + 4096], gen.uniform_bytes(key, start, 4096)), start
    Q = d_q.cpu().numpy().view(np.uint32)
    want = oracle.dbmul(D, Q, moduli, nthreads=NT)
    assert np.array_equal(d_a.cpu().numpy().view(np.uint32), want)
