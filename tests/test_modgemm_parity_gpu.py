"""GPU parity of the parallel INT32 modular GEMMs  Out = H*C + (0|G) mod q_t  (SURVEY.md 8(f)
NEXT-4): libvipir's tensor-core path, through the C ABI, against the CPU
oracle, bit for bit (integer work: no tolerance).

Shapes span several M tiles, N tiles, k-atoms and K chunks with ragged tails in every
dimension, both CTA groupings (vipir_modgemm_tuning.cta_group), all-maximum words at the int32 accumulation
bound, operand words above the modulus, and the paper's own per-problem shape
(M = 256, K = n = 1280, ncols = 2B).
"""
import os

import numpy as np
import pytest

import oracle
from paper_2606_11536_b200 import inputs, vipir
from paper_2606_11536_b200.inputs import generator as gen

from gpu_util import ensure_built

pytestmark = pytest.mark.gpu

P29 = [536608769, 533463041, 531628033]   # < 2^29, = 1 mod 2^18; three: #RNS = 3
P30 = inputs.rns_primes(0)
NT = max(1, os.cpu_count() or 1)


def run_modgemm(H, C, G, moduli, cg=0, ct=0, return_info=False, via_parts=False):
    import torch
    ensure_built()
    T, NC, M, K = H.shape
    ncols = C.shape[2]
    gcols = 0 if G is None else G.shape[2]
    tuning = {k: v for k, v in (("cta_group", cg), ("tile_cols", ct)) if v}
    d_H = torch.from_numpy(np.ascontiguousarray(H).view(np.int32)).cuda()
    d_C = torch.from_numpy(np.ascontiguousarray(C).view(np.int32)).cuda()
    d_G = None if G is None else torch.from_numpy(np.ascontiguousarray(G).view(np.int32)).cuda()
    d_O = torch.full((T, NC, ncols, M), -1, dtype=torch.int32, device="cuda")  # poison
    fusable = K % 4 == 0
    with vipir.ModGemmPlan(T, NC, M, K, ncols, gcols, moduli, tuning=tuning) as plan:
        plan.set_h(d_H)
        assert plan.info["fused_split"] == (1 if fusable and ncols >= 16 else 0)  # the planner's rule (include/vipir.h)
        assert plan.info["launches"] == 2 - plan.info["fused_split"]
        if via_parts:
            vipir.modgemm_split_c(plan.handle, d_C)
            vipir.modgemm_products(plan.handle, d_G, d_O)
        else:
            plan(d_C, d_G, d_O)
        torch.cuda.synchronize()
        info = plan.info
    if not via_parts:
        # the other form of the same plan shape -- one kernel with C split into limbs in shared memory, or the splitter
        # pre-pass + products -- must give the same words; so every parity case covers both
        other = dict(tuning, c_split=1 if info["fused_split"] else 2)
        if info["fused_split"] or fusable:
            for extra in ({}, {"r_stages": 2}, {"r_stages": 3, "b_stages": 3}) if not info["fused_split"] else ({},):
                with vipir.ModGemmPlan(T, NC, M, K, ncols, gcols, moduli, tuning=dict(other, **extra)) as plan:
                    assert plan.info["fused_split"] == (0 if info["fused_split"] else 1)
                    plan.set_h(d_H)
                    d_O2 = torch.full_like(d_O, -1)
                    plan(d_C, d_G, d_O2)
                    torch.cuda.synchronize()
                    assert torch.equal(d_O, d_O2), f"fused and two-kernel forms differ ({extra})"
        else:
            with pytest.raises(vipir.VipirError):  # no fused form for K % 4 != 0
                vipir.ModGemmPlan(T, NC, M, K, ncols, gcols, moduli, tuning=dict(tuning, c_split=2))
    out = d_O.cpu().numpy().view(np.uint32)
    return (out, info) if return_info else out


def assert_same(got, want):
    bad = np.argwhere(got != want)
    assert bad.size == 0, (f"{len(bad)} of {got.size} words differ; first at [t,c,j,m]={bad[0].tolist()}: "
                           f"got {got[tuple(bad[0])]} want {want[tuple(bad[0])]}")


def operands(seed, moduli, NC, M, K, ncols, gcols):
    H = gen.modgemm_operand(seed, gen.STREAM_MG_H, moduli, NC, M * K).reshape(len(moduli), NC, M, K)
    C = gen.modgemm_operand(seed, gen.STREAM_MG_C, moduli, NC, ncols * K).reshape(len(moduli), NC, ncols, K)
    G = gen.modgemm_operand(seed, gen.STREAM_MG_G, moduli, NC, gcols * M).reshape(len(moduli), NC, gcols, M) \
        if gcols else None
    return H, C, G


@pytest.mark.parametrize("cg", [1, 2])
@pytest.mark.parametrize("NC,M,K,ncols,gcols,moduli", [
    (3, 128, 128, 8, 4, P29[:1]),         # one tile, one atom
    (2, 256, 1280, 2, 1, P29),            # the paper's per-problem shape at B = 1
    (2, 256, 1280, 64, 32, P29[:2]),      # ... at B = 32: ct = 64, one accumulator stage
    (5, 200, 200, 10, 5, P30),            # ragged M, K (not a multiple of 16), ncols
    (3, 300, 392, 40, 40, P30),           # 3 M tiles (cg = 1), ragged everything, gcols = ncols
    (2, 64, 1000, 100, 0, P29[:1]),       # two N tiles, no G
    (7, 17, 33, 3, 2, [97, 65537]),       # tiny moduli, tiny shapes
])
def test_modgemm_matches_oracle(cg, NC, M, K, ncols, gcols, moduli):
    H, C, G = operands(NC * 7 + M, moduli, NC, M, K, ncols, gcols)
    got, info = run_modgemm(H, C, G, moduli, cg=cg, return_info=True)
    assert info["cta_group"] == cg
    assert_same(got, oracle.modgemm(H, C, G, moduli, nthreads=NT))


@pytest.mark.parametrize("cg,ct", [(1, 8), (1, 16), (2, 24), (2, 32), (1, 64), (2, 64)])
def test_modgemm_tile_widths(cg, ct):
    moduli = P29[:2]
    H, C, G = operands(ct, moduli, 3, 260, 520, 72, 36)
    got, info = run_modgemm(H, C, G, moduli, cg=cg, ct=ct, return_info=True)
    assert info["tile_cols"] == ct and info["n_tiles"] == -(-72 // ct)
    assert_same(got, oracle.modgemm(H, C, G, moduli, nthreads=NT))


@pytest.mark.parametrize("cg", [1, 2])
def test_modgemm_any_u32_words_and_chunks(cg):
    # words above the modulus are legal; K = 8192 + 300 crosses the int32 accumulation chunk (two chunks)
    g = np.random.default_rng(5)
    moduli = [P30[0], 3]
    T, NC, M, K, ncols, gcols = 2, 2, 130, 8192 + 300, 9, 3
    H = g.integers(0, 1 << 32, size=(T, NC, M, K), dtype=np.uint64).astype(np.uint32)
    C = g.integers(0, 1 << 32, size=(T, NC, ncols, K), dtype=np.uint64).astype(np.uint32)
    G = g.integers(0, 1 << 32, size=(T, NC, gcols, M), dtype=np.uint64).astype(np.uint32)
    got, info = run_modgemm(H, C, G, moduli, cg=cg, return_info=True)
    assert info["n_chunks"] == 2
    assert_same(got, oracle.modgemm(H, C, G, moduli, nthreads=NT))


@pytest.mark.parametrize("cg", [1, 2])
def test_modgemm_all_max_words_at_chunk_bound(cg):
    # every limb 255 and K = 8192: each accumulator block s holds (number of (i,j) pairs) * 255^2 * 8192,
    # the middle one 4 * 255^2 * 8192 = 2130739200 < 2^31 -- the exact bound of the chunking rule.
    # Closed form: (2^32-1)^2 * K + (2^32-1) mod q.
    moduli = [P29[0], P30[1]]
    T, NC, M, K, ncols = 2, 1, 128, 8192, 8
    H = np.full((T, NC, M, K), 0xFFFFFFFF, dtype=np.uint32)
    C = np.full((T, NC, ncols, K), 0xFFFFFFFF, dtype=np.uint32)
    G = np.full((T, NC, ncols, M), 0xFFFFFFFF, dtype=np.uint32)
    got = run_modgemm(H, C, G, moduli, cg=cg)
    for t, q in enumerate(moduli):
        want = (((1 << 32) - 1) ** 2 * K + (1 << 32) - 1) % q
        assert (got[t] == want).all(), (t, got[t].ravel()[:4], want)


def test_modgemm_identity_and_probe():
    # H = identity per problem: Out[j][m] = C[j][m] + G ; one-hot H at (m, pi(m)), C[j][k] = k+1+j*K
    q = P29[0]
    M = K = 136
    NC, ncols = 2, 5
    H = np.zeros((1, NC, M, K), dtype=np.uint32)
    pi = np.random.default_rng(1).permutation(K)
    for c in range(NC):
        H[0, c, np.arange(M), np.roll(pi, c)] = 1
    C = (np.arange(ncols * K, dtype=np.uint32).reshape(ncols, K) + 1)[None, None].repeat(NC, axis=1)
    got = run_modgemm(H, C, None, [q], cg=1)
    for c in range(NC):
        for j in range(ncols):
            assert np.array_equal(got[0, c, j], (np.roll(pi, c) + 1 + j * K).astype(np.uint32))


def test_modgemm_planner_choices_at_the_paper_shape():
    """Form and ring depths the planner takes at the paper's per-problem shape 256 x 2B x 1280 (include/vipir.h,
    DESIGN.md section 12): two kernels below 16 columns; one kernel from there on, with the deepest raw / operand rings
    that leave the H ring its minimum."""
    ensure_built()
    for B, want in ((1, dict(fused_split=0, launches=2, cta_group=1)),
                    (8, dict(fused_split=1, launches=1, cta_group=2, tile_cols=16, r_stages=4, b_stages=4)),
                    (16, dict(fused_split=1, tile_cols=32, r_stages=4, b_stages=4, acc_stages=2)),
                    (32, dict(fused_split=1, tile_cols=64, r_stages=3, b_stages=3, a_stages=5, acc_stages=1))):
        with vipir.ModGemmPlan(3, 8, 256, 1280, 2 * B, B, P29) as plan:
            got = {k: plan.info[k] for k in want}
            assert got == want, (B, plan.info)
            assert plan.info["a_stages"] >= 5 and plan.info["smem_bytes"] <= 232448


def test_modgemm_split_kernels_layout():
    # the limb re-layouts on their own, against their stated layouts (include/vipir.h)
    import torch
    ensure_built()
    moduli = P29[:1]
    T, NC, M, K, ncols = 1, 2, 5, 150, 3
    H, C, _ = operands(3, moduli, NC, M, K, ncols, 0)
    d_H = torch.from_numpy(H.view(np.int32)).cuda()
    d_C = torch.from_numpy(C.view(np.int32)).cuda()
    with vipir.ModGemmPlan(T, NC, M, K, ncols, 0, moduli) as plan:
        plan.set_h(d_H)
        vipir.modgemm_split_c(plan.handle, d_C)
        torch.cuda.synchronize()
        Kp = plan.info["k_padded"]
        assert Kp == 256
        d_hp, d_cp = vipir.testing_modgemm_limbs(plan.handle)
        hp = _device_bytes(d_hp, plan.info["h_limb_bytes"])
        cp = _device_bytes(d_cp, plan.info["c_limb_bytes"])
    hp = hp.reshape(NC * M, Kp // 128, 4, 128)
    cp = cp.reshape(NC, 4, ncols, Kp)
    Hb = np.zeros((NC * M, Kp), dtype=np.uint32)
    Hb[:, :K] = H.reshape(NC * M, K)
    Cb = np.zeros((NC, ncols, Kp), dtype=np.uint32)
    Cb[:, :, :K] = C.reshape(NC, ncols, K)
    for i in range(4):
        assert np.array_equal(hp[:, :, i, :].reshape(NC * M, Kp), ((Hb >> (8 * i)) & 0xFF).astype(np.uint8))
        assert np.array_equal(cp[:, i], ((Cb >> (8 * i)) & 0xFF).astype(np.uint8))


def _device_bytes(ptr, nbytes):
    """Copy `nbytes` from a raw device pointer to a numpy uint8 array (cudaMemcpy through torch's runtime)."""
    import ctypes

    import torch
    out = np.empty(nbytes, dtype=np.uint8)
    rt = ctypes.CDLL(os.path.join(os.path.dirname(torch.__file__), "lib", "libcudart.so.12")) \
        if os.path.exists(os.path.join(os.path.dirname(torch.__file__), "lib", "libcudart.so.12")) \
        else ctypes.CDLL("libcudart.so.12")
    rt.cudaMemcpy.restype = ctypes.c_int
    rt.cudaMemcpy.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int]
    rc = rt.cudaMemcpy(out.ctypes.data, ctypes.c_void_p(ptr), nbytes, 2)  # cudaMemcpyDeviceToHost
    assert rc == 0, rc
    return out


def test_modgemm_parts_equal_whole_and_errors():
    moduli = P29[:1]
    H, C, G = operands(11, moduli, 2, 64, 256, 4, 2)
    a = run_modgemm(H, C, G, moduli)
    b = run_modgemm(H, C, G, moduli, via_parts=True)
    assert_same(a, b)
    lib = vipir.load()
    import ctypes
    h = ctypes.c_void_p()
    arr = (ctypes.c_uint32 * 1)(moduli[0])
    big = (ctypes.c_uint32 * 1)(1 << 30)
    assert lib.vipir_modgemm_plan_create(ctypes.byref(h), 1, 0, 4, 4, 4, 0, arr) == vipir.ERR_INVALID_ARG
    assert lib.vipir_modgemm_plan_create(ctypes.byref(h), 1, 1, 4, 4, 4, 5, arr) == vipir.ERR_INVALID_ARG
    assert lib.vipir_modgemm_plan_create(ctypes.byref(h), 1, 1, 4, 4, 4, 0, big) == vipir.ERR_INVALID_ARG
    assert lib.vipir_modgemm_plan_create(ctypes.byref(h), 5, 1, 4, 4, 4, 0, arr) == vipir.ERR_INVALID_ARG
    # products before set_h is an error, not a silent run on garbage
    import torch
    with vipir.ModGemmPlan(1, 1, 8, 16, 2, 0, moduli) as plan:
        d_O = torch.zeros((1, 1, 2, 8), dtype=torch.int32, device="cuda")
        with pytest.raises(vipir.VipirError):
            vipir.modgemm_products(plan.handle, None, d_O)


# ---- the paper's full shape (64 GiB DB, N = 2^12, D_r = 2^8, n = 1280, #RNS = 3) --------
# T*NC = 12288 problems of 256 x 2B x 1280; H is 15 GiB ("H occupies 15GiB of memory space", :222).
# Compared on sampled problems the oracle recomputes in full from the host generator's words, plus a
# row-sum identity over ALL problems that holds at any size (linearity):
#     sum_m Out[p][j][m] = sum_k (sum_m H[p][m][k]) * C[p][j][k] + sum_m G[p][j-g0][m]      (mod q_t)
# with the sums taken by plain torch reductions that share nothing with libvipir.

FULL_T, FULL_NC, FULL_M, FULL_K = 3, 4096, 256, 1280


@pytest.mark.parametrize("B", [1, 32])
def test_modgemm_paper_shape_sampled_problems_and_row_sums(B):
    import torch
    from paper_2606_11536_b200.inputs import device
    ensure_built()
    torch.cuda.empty_cache()
    moduli = P29
    T, NC, M, K = FULL_T, FULL_NC, FULL_M, FULL_K
    ncols, gcols = 2 * B, B
    g0 = ncols - gcols
    d_H = device.modgemm_operand(0, gen.STREAM_MG_H, moduli, NC, M * K).view(T, NC, M, K)
    d_C = device.modgemm_operand(0, gen.STREAM_MG_C, moduli, NC, ncols * K).view(T, NC, ncols, K)
    d_G = device.modgemm_operand(0, gen.STREAM_MG_G, moduli, NC, gcols * M).view(T, NC, gcols, M)
    d_O = torch.full((T, NC, ncols, M), -1, dtype=torch.int32, device="cuda")
    with vipir.ModGemmPlan(T, NC, M, K, ncols, gcols, moduli) as plan:
        plan.set_h(d_H)
        plan(d_C, d_G, d_O)  # the launch configuration bench.py times (the planner's own choice)
        torch.cuda.synchronize()

    # (1) sampled problems, every output word
    cs = sorted(set([0, 1, NC // 2, NC - 1] + np.random.default_rng(B).integers(0, NC, size=6).tolist()))
    for c in cs:
        H = gen.modgemm_operand(0, gen.STREAM_MG_H, moduli, NC, M * K, c0=c, nc=1).reshape(T, 1, M, K)
        C = gen.modgemm_operand(0, gen.STREAM_MG_C, moduli, NC, ncols * K, c0=c, nc=1).reshape(T, 1, ncols, K)
        G = gen.modgemm_operand(0, gen.STREAM_MG_G, moduli, NC, gcols * M, c0=c, nc=1).reshape(T, 1, gcols, M)
        want = oracle.modgemm(H, C, G, moduli, nthreads=NT)
        got = d_O[:, c:c + 1].cpu().numpy().view(np.uint32)
        assert_same(got, want)

    # (2) row-sum identity over all problems; canonical range of every word
    for t, q in enumerate(moduli):
        assert int(d_O[t].max()) < q and int(d_O[t].min()) >= 0
        for c0 in range(0, NC, 512):
            sl = slice(c0, c0 + 512)
            hs = d_H[t, sl].to(torch.int64).sum(dim=1) % q                       # [nc][K], each < q < 2^29
            terms = (hs[:, None, :] * d_C[t, sl].to(torch.int64)) % q            # products < 2^58
            want = terms.sum(dim=2)                                              # < 1280 * 2^29
            want[:, g0:] += d_G[t, sl].to(torch.int64).sum(dim=2)
            got = d_O[t, sl].to(torch.int64).sum(dim=2)
            assert torch.equal(got % q, want % q), f"row-sum identity fails: modulus {t}, problems {c0}.."
    del d_H, d_C, d_G, d_O
    torch.cuda.empty_cache()
