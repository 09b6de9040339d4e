"""The seeded input generator: host twin properties (no GPU) and host == device twin (GPU)."""
import numpy as np
import pytest

from paper_2606_11536_b200 import inputs


def test_random_access_matches_sequential():
    key = inputs.stream_key(0, inputs.STREAM_DB)
    full = inputs.uniform_bytes(key, 0, 4096)
    for start, n in [(0, 1), (5, 7), (8, 16), (1023, 1025), (4000, 96)]:
        assert np.array_equal(inputs.uniform_bytes(key, start, n), full[start:start + n])


def test_db_rows_slices_and_u16_view():
    full = inputs.db_rows(3, 20, 48, 8)
    assert full.dtype == np.uint8 and full.shape == (20, 48)
    assert np.array_equal(inputs.db_rows(3, 20, 48, 8, row0=7, nrows=5), full[7:12])
    d16 = inputs.db_rows(3, 20, 24, 16)
    assert d16.dtype == np.uint16 and d16.shape == (20, 24)
    raw = full.reshape(20, 24, 2).astype(np.uint16)
    assert np.array_equal(d16, raw[:, :, 0] + 256 * raw[:, :, 1])  # little-endian


def test_streams_and_seeds_differ_and_are_deterministic():
    a = inputs.db_rows(0, 4, 64, 8)
    assert np.array_equal(a, inputs.db_rows(0, 4, 64, 8))
    assert not np.array_equal(a, inputs.db_rows(1, 4, 64, 8))
    q = inputs.query(0, 64, 1)
    assert q.dtype == np.uint32 and q.shape == (1, 1, 64)
    assert not np.array_equal(q.view(np.uint8).ravel(), a.ravel())


def test_bytes_look_uniform():
    b = inputs.db_rows(0, 64, 4096, 8).ravel()
    hist = np.bincount(b, minlength=256)
    assert hist.min() > 800 and hist.max() < 1250  # expectation 1024 per value
    q = inputs.query(0, 1 << 16, 1).ravel()
    assert abs(q.mean() / 2**31 - 1) < 0.02


def test_residues_are_canonical_and_per_prime():
    p0, p1 = inputs.rns_primes(0)
    q = inputs.query(5, 512, 3, [p0, p1])
    assert q.shape == (2, 3, 512)
    assert (q[0] < p0).all() and (q[1] < p1).all()
    assert not np.array_equal(q[0], q[1])


@pytest.mark.gpu
def test_device_twin_equals_host_twin():
    import torch
    from paper_2606_11536_b200 import build
    from paper_2606_11536_b200.inputs import device
    build.build()
    for db_bits, rows, cols in [(8, 37, 1040), (16, 21, 520)]:
        d = device.db(9, rows, cols, db_bits).cpu().numpy()
        want = inputs.db_rows(9, rows, cols, db_bits)
        assert np.array_equal(d, want.view(np.uint8).reshape(rows, -1))
    q = device.query(9, 1000, 3).cpu().numpy().view(np.uint32)
    assert np.array_equal(q, inputs.query(9, 1000, 3))
    primes = inputs.rns_primes(0)
    qp = device.query(9, 1000, 3, primes).cpu().numpy().view(np.uint32)
    assert np.array_equal(qp, inputs.query(9, 1000, 3, primes))
    torch.cuda.synchronize()
