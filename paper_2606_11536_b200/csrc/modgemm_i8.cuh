// modgemm_i8.cuh -- SURVEY.md 8(f) NEXT-4: VIPIR's parallel INT32 modular GEMMs
//     Out = H * C + (0 | G)   mod q_t
// on the int8 tensor cores.
//
// PAPER.md:216 (section 3.5.2): "this reduces to (#RNS * N)-parallel ceil(D1/N) x 2B x n INT32
// GEMMs with additional modular reduction computations"; PAPER.md:261-265 (section 4.2): the
// paper runs them on CUDA cores in a "tile-major (GEMM-friendly)" layout with lazy reduction
// (64-bit accumulators, one reduction per 32 multiply-accumulates, primes < 2^29), because on
// H100 "modulo-q_i arithmetic ... introduces significant overheads ... under tensor-core
// execution" (:255-257).
//
// B200 design.  What is kept from the paper: a GEMM-friendly re-layout
// of the operands before the GEMMs (:263) and deferred reduction (:265) -- here deferred over
// the WHOLE K dimension.  What changes: the products run on tcgen05.mma.kind::i8.  Both
// operands are split into four 8-bit limbs, H = sum_i 2^(8i) H_i, C = sum_j 2^(8j) C_j, so
//     H*C = sum_{s=0..6} 2^(8s) S_s,     S_s = sum_{i+j=s} H_i * C_j        (over the integers)
// and every S_s <= 4 * 255^2 * K stays below 2^31 for K <= 8192 per chunk: the int32 TMEM
// accumulators hold the exact limb sums, one modular reduction per OUTPUT word (the extreme
// of the paper's lazy reduction).  16 int8 MACs replace one 32x32->64-bit MAC; the B200's int8
// tensor rate is ~130x its INT32 ALU rate, so the GEMMs become HBM-bound on streaming H.
//
// The seven sums are formed without seven separate products: the B operand holds the four
// limb planes of the C tile stacked along N in the order (j, column), N = 4*ct, and the MMA for
// H limb i writes its N accumulator columns at TMEM column offset i*ct -- so column block
// s = i + j of the accumulator receives H_i*C_j, and the four instructions (i = 0..3)
// overlap-add into 7*ct columns.
//
//   warp 0   TMA producer: per k-atom (128 k) one B box (4 limb planes x ct columns x 128 B) and
//            four A boxes (128 rows x 128 B, one per H limb) into two mbarrier rings;
//   warp 1   MMA issuer (one thread): per A box four tcgen05.mma (K = 32 each);
//   warp 2   TMEM allocator;   warps 2-3 (FUSED) converters, see below;
//   warps 4-11 epilogue: tcgen05.ld, recombine in u64 (shifts for the
//            low four sums, 2^(8s) mod q weights for the high three), + G, one Barrett reduction,
//            store (coalesced over rows).
//
// FUSED (the default from 16 columns up and K % 4 == 0): the limb split of C -- the paper fuses its prmt decomposition into
// the GEMM kernel too -- happens inside this kernel instead of a pre-pass that writes and re-reads
// 4 bytes per word of C.  The producer brings the RAW u32 words of the C tile by TMA (four 32-word x ct-column
// boxes per k-atom, 128B-swizzled so that a thread's 64-byte run reads conflict-free), two converter warps
// byte-transpose them with prmt (split_limbs.cuh) and write the limb planes straight into the swizzled K-major
// B operand slot the tensor core reads; fence.proxy.async + an mbarrier arrival hand the slot to the MMA issuer.
// With CTA pairs (CTA c stages limb planes 2c, 2c + 1 of the whole tile) each CTA reads the whole raw tile (the
// second read hits L2) and converts its two planes, so every write stays in the CTA's own shared memory.  The
// converters hand a slot over with fence.proxy.async.shared::cta and an arrival on their OWN CTA's barrier; for
// the peer CTA the otherwise idle warp 1 forwards that arrival to the leader's barrier with one cluster-scope
// release per k-atom.  (Measured alternatives: a release.cluster arrival in the converters
// themselves, or halving the raw tile per CTA and writing the peer's planes through distributed shared memory,
// cost a GPU-scope membar per converter warp and k-atom -- 1.3-1.5x slower than the two-kernel form; TMA cannot
// gather the 16-bit half of every word, element strides do not apply to dimension 0.)
#pragma once
#include <cstdint>
#include <cuda.h>
#include "gemm_i8_tcgen05.cuh"  // make_smem_desc, barrett_u64
#include "ptx.cuh"
#include "split_limbs.cuh"  // byte_transpose4

namespace vipir {

constexpr int MG_BM = 128;      // rows per CTA
constexpr int MG_BK = 128;      // k per atom = bytes per limb-plane row segment (one 128B swizzle row)
constexpr int MG_UMMA_K = 32;
constexpr int MG_EPI_WARPS = 8;  // two per TMEM lane quarter, splitting the column groups
constexpr int MG_CONV_WARPS = 2; // warps 2 and 3: raw C words -> limb planes in shared memory (FUSED)
constexpr int MG_THREADS = 32 * (4 + MG_EPI_WARPS);
constexpr int MG_A_BYTES = MG_BM * MG_BK;  // 16 KiB: one H limb of one k-atom
constexpr int MG_ZERO_BYTES = 1024;        // all-zero A operand (one 8-row swizzle atom, aliased by SBO = 0)
constexpr int MG_MAX_MODULI = 4;
constexpr uint32_t MG_MAX_CHUNK_ATOMS = 64;  // 4 * 255^2 * 8192 < 2^31

struct ModGemmParams {
    uint32_t P;        // problems = T * NC
    uint32_t NC;       // problems per modulus (modulus index = problem / NC)
    uint32_t M, ncols, gcols;
    uint32_t ct;       // C columns per N tile (multiple of 8); MMA N = 4*ct; accumulator columns = 7*ct
    uint32_t m_tiles, n_tiles;  // per problem
    uint32_t atoms;    // k-atoms = Kp / 128
    uint32_t atoms_per_chunk, n_chunks;
    uint32_t a_stages, b_stages, b_stage_bytes;  // per CTA
    uint32_t r_stages, r_stage_bytes;            // FUSED: ring of raw C tiles (ct columns x 128 words as four 32-word
                                                 // boxes), per CTA
    uint32_t tmem_cols, acc_stages;
    uint32_t idesc;
    uint32_t moduli[MG_MAX_MODULI];
    uint32_t w[MG_MAX_MODULI][3];     // 2^32, 2^40, 2^48 mod q_t: weights of the three high limb sums
    uint64_t barrett[MG_MAX_MODULI];  // floor(2^64 / q_t)
    const uint32_t* G;                // [P][gcols][M] or nullptr
    uint32_t* out;                    // [P][ncols][M]
};

// ---- operand re-layout (the paper's "layout transposition before the GEMMs", :263) -------------
// X [P][R][K] u32  ->  byte limbs.  One thread = 16 consecutive k of one row.
//   INTERLEAVED (H, the static hint; written once, offline):
//       Hp[(p*R + r)][ (k/128)*512 + i*128 + k%128 ] = byte i of X[p][r][k]      row pitch 4*Kp
//     i.e. per row the four limb segments of one k-atom are adjacent: the (atom, limb) boxes the
//     kernel loads in sequence are consecutive 128-byte column blocks of one byte matrix.
//   planes (C, every call):
//       Cp[((p*4 + i)*R + r)][k] = byte i of X[p][r][k]                           row pitch Kp
// Kp = K rounded up to 128; the padding is written as zeros.
template <bool INTERLEAVED>
__global__ void __launch_bounds__(256) mg_split_kernel(const uint32_t* __restrict__ X, uint8_t* __restrict__ out,
                                                       uint64_t n_rows /* P*R */, uint32_t R, uint32_t K,
                                                       uint32_t Kp) {
    const uint32_t groups = Kp / 16;
    const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= n_rows * groups) return;
    const uint64_t row = gid / groups;
    const uint32_t k0 = (uint32_t)(gid % groups) * 16;
    const uint32_t* src = X + row * K + k0;
    uint32_t L[4][4];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        uint32_t t[4] = {0, 0, 0, 0};
        if (k0 + 4 * w + 3 < K && (K & 3) == 0) {
            const uint4 v = *reinterpret_cast<const uint4*>(src + 4 * w);
            t[0] = v.x; t[1] = v.y; t[2] = v.z; t[3] = v.w;
        } else {
            for (int e = 0; e < 4; ++e)
                if (k0 + 4 * w + e < K) t[e] = src[4 * w + e];
        }
        byte_transpose4(t[0], t[1], t[2], t[3], L[w]);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        uint8_t* dst;
        if constexpr (INTERLEAVED) {
            dst = out + row * (4ull * Kp) + (k0 / MG_BK) * (4 * MG_BK) + i * MG_BK + (k0 % MG_BK);
        } else {
            const uint64_t p = row / R, r = row % R;
            dst = out + ((p * 4 + i) * R + r) * (uint64_t)Kp + k0;
        }
        *reinterpret_cast<uint4*>(dst) = make_uint4(L[0][i], L[1][i], L[2][i], L[3][i]);
    }
}

// zero operand: every 8-row group aliases the same 1 KiB of zeros (stride byte offset 0)
__device__ __forceinline__ uint64_t make_smem_desc_zero(uint32_t saddr) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);
    d |= (uint64_t)1 << 16;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}

// tmB: the C limb planes (FUSED = false) or the raw u32 words of C (FUSED = true)
template <int CG, bool FUSED>
__global__ void __launch_bounds__(MG_THREADS, 1)
modgemm_i8_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, ModGemmParams p) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* sA_ring = smem;
    uint8_t* sB_ring = sA_ring + (size_t)p.a_stages * MG_A_BYTES;
    uint8_t* sR_ring = sB_ring + (size_t)p.b_stages * p.b_stage_bytes;
    uint8_t* sZero = sR_ring + (FUSED ? (size_t)p.r_stages * p.r_stage_bytes : 0);
    uint64_t* fullA = reinterpret_cast<uint64_t*>(sZero + MG_ZERO_BYTES);
    uint64_t* emptyA = fullA + p.a_stages;
    uint64_t* fullB = emptyA + p.a_stages;
    uint64_t* emptyB = fullB + p.b_stages;
    uint64_t* fullR = emptyB + p.b_stages;
    uint64_t* emptyR = fullR + (FUSED ? p.r_stages : 0);
    uint64_t* tmem_full = emptyR + (FUSED ? p.r_stages : 0);  // [2]
    uint64_t* tmem_empty = tmem_full + 2;       // [2]
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(tmem_empty + 2);

    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t rank = (CG == 2) ? ptx::cluster_ctarank() : 0u;
    const uint32_t unit0 = (CG == 2) ? ptx::cluster_id_x() : blockIdx.x;
    const uint32_t unit_stride = (CG == 2) ? ptx::num_clusters_x() : gridDim.x;
    const uint32_t tiles_per_problem = p.m_tiles * p.n_tiles;
    const uint32_t n_units = p.P * tiles_per_problem;
    const uint32_t acc_cols = 7 * p.ct;

    // the zero operand (generic-proxy writes, made visible to the tensor core's async proxy)
    for (uint32_t i = threadIdx.x; i < MG_ZERO_BYTES / 4; i += MG_THREADS) reinterpret_cast<uint32_t*>(sZero)[i] = 0u;
    ptx::fence_proxy_async();
    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tmA);
        ptx::prefetch_tmap(&tmB);
    }
    if (warp == 1 && lane == 0) {
        for (uint32_t s = 0; s < p.a_stages; ++s) {
            ptx::mbar_init(&fullA[s], 1);
            ptx::mbar_init(&emptyA[s], 1);
        }
        for (uint32_t s = 0; s < p.b_stages; ++s) {
            // FUSED: the slot is filled by this CTA's converter warps; the leader also counts the peer's forwarder
            ptx::mbar_init(&fullB[s], FUSED ? MG_CONV_WARPS + ((CG == 2 && rank == 0) ? 1 : 0) : 1);
            ptx::mbar_init(&emptyB[s], 1);
        }
        if constexpr (FUSED)
            for (uint32_t s = 0; s < p.r_stages; ++s) {
                ptx::mbar_init(&fullR[s], 1);
                ptx::mbar_init(&emptyR[s], MG_CONV_WARPS);
            }
        for (uint32_t a = 0; a < 2; ++a) {
            ptx::mbar_init(&tmem_full[a], 1);
            ptx::mbar_init(&tmem_empty[a], MG_EPI_WARPS * CG);
        }
        ptx::fence_barrier_init();
    }
    if (warp == 2) {
        ptx::tmem_alloc<CG>(tmem_ptr, p.tmem_cols);
        ptx::tmem_relinquish<CG>();
    }
    ptx::tc_fence_before();
    if constexpr (CG == 2) ptx::cluster_sync(); else __syncthreads();
    ptx::tc_fence_after();
    // same in every lane: say so (shfl from lane 0), so the single-issuer loops run on the uniform datapath
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_ptr, 0);

    if (warp == 0) {
        // ===== TMA producer: the whole warp runs the (warp-uniform) loop, one elected lane issues =====
        {
            uint32_t sa = 0, pa = 0, sb = 0, pb = 0;
            // H is streamed once when there is a single N tile; sibling N tiles re-read it from L2
            const uint64_t hintA = (p.n_tiles == 1) ? ptx::kEvictFirst : ptx::kEvictNormal;
            // FUSED: the raw words of the C tiles run AHEAD of the H boxes by r_stages - 1 k-atoms (a cursor of their
            // own, across unit boundaries): they have the longer way to the tensor core (load, conversion, hand-over),
            // and requested in step with the H boxes of their k-atom they arrive late whenever the H ring is short
            // (measured at 64 columns: 5.36 / 5.07 / 4.86 ms with 4 / 6 / 8 H boxes before this)
            uint32_t ur = unit0, ar = 0;
            auto raw_next = [&]() {
                if (ur >= n_units) return;
                const uint32_t prob = ur / tiles_per_problem, nt = (ur % tiles_per_problem) % p.n_tiles;
                ptx::mbar_wait(&emptyR[sb], pb ^ 1);
                __syncwarp();
                uint8_t* dR = sR_ring + (size_t)sb * p.r_stage_bytes;
                if (ptx::elect_one()) {
                    ptx::mbar_arrive_expect_tx(&fullR[sb], p.r_stage_bytes);
#pragma unroll
                    for (uint32_t kb = 0; kb < 4; ++kb)  // every CTA its own copy: four 32-word k-blocks
                        ptx::tma_load_3d(dR + kb * (p.r_stage_bytes / 4), &tmB, &fullR[sb], (int32_t)(ar * MG_BK + kb * 32),
                                         (int32_t)(nt * p.ct), (int32_t)prob, ptx::kEvictNormal);
                }
                __syncwarp();
                if (++sb == p.r_stages) { sb = 0; pb ^= 1; }
                if (++ar == p.atoms) { ar = 0; ur += unit_stride; }
            };
            if constexpr (FUSED)
                for (uint32_t i = 0; i + 1 < p.r_stages; ++i) raw_next();
            for (uint32_t u = unit0; u < n_units; u += unit_stride) {
                const uint32_t prob = u / tiles_per_problem, rem = u % tiles_per_problem;
                const uint32_t mt = rem / p.n_tiles, nt = rem % p.n_tiles;
                const int32_t row0 = (int32_t)((mt * CG + rank) * MG_BM);
                for (uint32_t a = 0; a < p.atoms; ++a) {
                    if constexpr (FUSED) {
                        raw_next();
                    } else {
                    ptx::mbar_wait(&emptyB[sb], pb ^ 1);
                    __syncwarp();
                    uint8_t* dB = sB_ring + (size_t)sb * p.b_stage_bytes;
                    if (ptx::elect_one()) {
                    if constexpr (CG == 1) {
                        ptx::mbar_arrive_expect_tx(&fullB[sb], p.b_stage_bytes);
                        ptx::tma_load_4d(dB, &tmB, &fullB[sb], (int32_t)(a * MG_BK), (int32_t)(nt * p.ct), 0,
                                         (int32_t)prob, ptx::kEvictNormal);
                    } else {
                        if (rank == 0) ptx::mbar_arrive_expect_tx(&fullB[sb], 2 * p.b_stage_bytes);
                        // this CTA stages limb planes j = 2*rank, 2*rank+1: its half of the N = 4*ct rows
                        ptx::tma_load_4d_pair(dB, &tmB, ptx::mapa(ptx::smem_u32(&fullB[sb]), 0), (int32_t)(a * MG_BK),
                                              (int32_t)(nt * p.ct), (int32_t)(2 * rank), (int32_t)prob,
                                              ptx::kEvictNormal);
                    }
                    }
                    __syncwarp();
                    if (++sb == p.b_stages) { sb = 0; pb ^= 1; }
                    }
#pragma unroll 1
                    for (uint32_t i = 0; i < 4; ++i) {
                        ptx::mbar_wait(&emptyA[sa], pa ^ 1);
                        __syncwarp();
                        uint8_t* dA = sA_ring + (size_t)sa * MG_A_BYTES;
                        const int32_t kb = (int32_t)((a * 4 + i) * MG_BK);
                        if (ptx::elect_one()) {
                        if constexpr (CG == 1) {
                            ptx::mbar_arrive_expect_tx(&fullA[sa], MG_A_BYTES);
                            ptx::tma_load_3d(dA, &tmA, &fullA[sa], kb, row0, (int32_t)prob, hintA);
                        } else {
                            if (rank == 0) ptx::mbar_arrive_expect_tx(&fullA[sa], 2 * MG_A_BYTES);
                            ptx::tma_load_3d_pair(dA, &tmA, ptx::mapa(ptx::smem_u32(&fullA[sa]), 0), kb, row0,
                                                  (int32_t)prob, hintA);
                        }
                        }
                        __syncwarp();
                        if (++sa == p.a_stages) { sa = 0; pa ^= 1; }
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (leader CTA of the pair only) =====
        // whole warp in the (warp-uniform) loop; one elected lane -- always the same -- issues and commits
        if (rank == 0) {
            uint32_t sa = 0, pa = 0, sb = 0, pb = 0, acc_it = 0;
            const uint64_t dZ = make_smem_desc_zero(ptx::smem_u32(sZero));
            for (uint32_t u = unit0; u < n_units; u += unit_stride) {
                for (uint32_t c = 0; c < p.n_chunks; ++c, ++acc_it) {
                    const uint32_t as = acc_it % p.acc_stages;
                    const uint32_t aphase = (acc_it / p.acc_stages) & 1;
                    if constexpr (CG == 2) ptx::mbar_wait_cluster(&tmem_empty[as], aphase ^ 1);
                    else ptx::mbar_wait(&tmem_empty[as], aphase ^ 1);
                    ptx::tc_fence_after();
                    const uint32_t a_begin = c * p.atoms_per_chunk;
                    const uint32_t a_end = min(p.atoms, a_begin + p.atoms_per_chunk);
                    const uint32_t tacc = tmem_base + as * acc_cols;
                    for (uint32_t a = a_begin; a < a_end; ++a) {
                        // FUSED pairs: the peer's converter warps arrive on this barrier too (cluster-scope acquire)
                        if constexpr (FUSED && CG == 2) ptx::mbar_wait_cluster(&fullB[sb], pb);
                        else ptx::mbar_wait(&fullB[sb], pb);
                        ptx::tc_fence_after();
                        const uint64_t dB = make_smem_desc(ptx::smem_u32(sB_ring + (size_t)sb * p.b_stage_bytes));
#pragma unroll 1
                        for (uint32_t i = 0; i < 4; ++i) {
                            ptx::mbar_wait(&fullA[sa], pa);
                            ptx::tc_fence_after();
                            __syncwarp();
                            if (ptx::elect_one()) {
                            const uint64_t dA = make_smem_desc(ptx::smem_u32(sA_ring + (size_t)sa * MG_A_BYTES));
                            const bool first = (a == a_begin && i == 0);
                            // blocks 3..6 start at zero (0 * anything), then H_0*C overwrites blocks 0..3
                            if (first) ptx::mma_i8<CG>(tacc + 3 * p.ct, dZ, dB, p.idesc, 0u);
#pragma unroll
                            for (uint32_t kk = 0; kk < MG_BK / MG_UMMA_K; ++kk) {
                                const uint64_t koff = (uint64_t)((kk * MG_UMMA_K) >> 4);
                                ptx::mma_i8<CG>(tacc + i * p.ct, dA + koff, dB + koff, p.idesc,
                                                (first && kk == 0) ? 0u : 1u);
                            }
                            if constexpr (CG == 2) ptx::tc_commit_pair(&emptyA[sa], 3);
                            else ptx::tc_commit(&emptyA[sa]);
                            if (i == 3) {
                                if constexpr (CG == 2) ptx::tc_commit_pair(&emptyB[sb], 3);
                                else ptx::tc_commit(&emptyB[sb]);
                                if (a + 1 == a_end) {
                                    if constexpr (CG == 2) ptx::tc_commit_pair(&tmem_full[as], 3);
                                    else ptx::tc_commit(&tmem_full[as]);
                                }
                            }
                            }
                            __syncwarp();
                            if (++sa == p.a_stages) { sa = 0; pa ^= 1; }
                        }
                        if (++sb == p.b_stages) { sb = 0; pb ^= 1; }
                    }
                }
            }
        } else if constexpr (FUSED && CG == 2) {
            // ===== rank 1's warp 1 (the MMA issuer sits in rank 0): forwards "this CTA's operand half is written" =====
            uint32_t sb = 0, pb = 0;
            for (uint32_t u = unit0; u < n_units; u += unit_stride) {
                for (uint32_t a = 0; a < p.atoms; ++a) {
                    ptx::mbar_wait(&fullB[sb], pb);
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive_cluster(&fullB[sb], 0);  // release at cluster scope
                    if (++sb == p.b_stages) { sb = 0; pb ^= 1; }
                }
            }
        }
    } else if (FUSED && (warp == 2 || warp == 3)) {
        // ===== converter warps: raw C words -> this CTA's limb planes in the B operand slot =====
        const uint32_t tid = (warp - 2) * 32 + lane;
        uint32_t sr = 0, pr = 0, sb = 0, pb = 0;
        for (uint32_t u = unit0; u < n_units; u += unit_stride) {
            for (uint32_t a = 0; a < p.atoms; ++a) {
                ptx::mbar_wait(&fullR[sr], pr);
                ptx::mbar_wait(&emptyB[sb], pb ^ 1);  // the MMAs that read this operand slot are done
                ptx::tc_fence_after();
                const uint8_t* raw = sR_ring + (size_t)sr * p.r_stage_bytes;
                uint8_t* dst = sB_ring + (size_t)sb * p.b_stage_bytes;
                // one item = 16 consecutive k of one column, one 16-byte chunk per limb plane out.  Eight neighbouring
                // lanes take eight neighbouring columns (ct % 8 == 0): their 16-byte accesses land on eight different
                // chunk positions of the 128B swizzle, in the raw tile and in the operand
                for (uint32_t idx = tid; idx < 8 * p.ct; idx += 32 * MG_CONV_WARPS) {
                    const uint32_t r = idx % p.ct, kh = idx / p.ct, sw = r & 7;  // kh: which 16 k of the atom's 128
                    const uint8_t* src = raw + (kh >> 1) * (p.r_stage_bytes / 4) + r * 128;  // 32 words a box
                    uint8_t* d0 = dst + r * 128 + ((kh ^ sw) << 4);
                    uint32_t L[4][4];
#pragma unroll
                    for (uint32_t w = 0; w < 4; ++w) {
                        const uint4 v = *reinterpret_cast<const uint4*>(src + (((4 * (kh & 1) + w) ^ sw) << 4));
                        byte_transpose4(v.x, v.y, v.z, v.w, L[w]);
                    }
                    if constexpr (CG == 1) {
#pragma unroll
                        for (uint32_t j = 0; j < 4; ++j)
                            *reinterpret_cast<uint4*>(d0 + j * p.ct * 128) = make_uint4(L[0][j], L[1][j], L[2][j], L[3][j]);
                    } else {  // this CTA stages planes 2*rank and 2*rank + 1
                        *reinterpret_cast<uint4*>(d0) = rank ? make_uint4(L[0][2], L[1][2], L[2][2], L[3][2])
                                                             : make_uint4(L[0][0], L[1][0], L[2][0], L[3][0]);
                        *reinterpret_cast<uint4*>(d0 + p.ct * 128) = rank ? make_uint4(L[0][3], L[1][3], L[2][3], L[3][3])
                                                                          : make_uint4(L[0][1], L[1][1], L[2][1], L[3][1]);
                    }
                }
                ptx::fence_proxy_async();  // generic-proxy writes -> visible to the tensor core's async proxy
                __syncwarp();
                if (lane == 0) {
                    ptx::mbar_arrive(&emptyR[sr]);
                    ptx::mbar_arrive(&fullB[sb]);
                }
                if (++sr == p.r_stages) { sr = 0; pr ^= 1; }
                if (++sb == p.b_stages) { sb = 0; pb ^= 1; }
            }
        }
    } else if (warp >= 4) {
        // ===== epilogue warps: lane quarter = warp % 4; the two warps of a quarter take alternate
        // groups of 8 columns =====
        const uint32_t quarter = warp & 3;
        const uint32_t half = (warp - 4) >> 2;
        const uint32_t g0 = p.ncols - p.gcols;
        const uint32_t n_groups = p.ct / 8;  // <= 8
        uint32_t acc_it = 0;
        for (uint32_t u = unit0; u < n_units; u += unit_stride) {
            const uint32_t prob = u / tiles_per_problem, rem = u % tiles_per_problem;
            const uint32_t mt = rem / p.n_tiles, nt = rem % p.n_tiles;
            const uint32_t row = (mt * CG + rank) * MG_BM + quarter * 32 + lane;
            const bool row_ok = row < p.M;
            const uint32_t t = prob / p.NC;
            const uint32_t q = p.moduli[t];
            const uint32_t w4 = p.w[t][0], w5 = p.w[t][1], w6 = p.w[t][2];
            const uint64_t bm = p.barrett[t];
            const uint32_t* __restrict__ Gp = p.G + ((uint64_t)prob * p.gcols) * p.M + row;
            uint32_t* __restrict__ Op = p.out + ((uint64_t)prob * p.ncols) * p.M + row;
            for (uint32_t c = 0; c < p.n_chunks; ++c, ++acc_it) {
                const uint32_t as = acc_it % p.acc_stages;
                const uint32_t aphase = (acc_it / p.acc_stages) & 1;
                // The words added to this chunk's sums -- G on the last gcols columns ("(0 | G)") for
                // chunk 0, the running (reduced) result for later chunks -- do not depend on the
                // accumulators: all of this warp's are fetched before waiting for the MMAs, so their
                // global-load latency is paid once per tile and overlaps the products.
                uint32_t add[4][8];
#pragma unroll
                for (int gi = 0; gi < 4; ++gi) {
                    const uint32_t g = half + 2 * gi;
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const uint32_t col = nt * p.ct + g * 8 + e;
                        add[gi][e] = 0u;
                        if (g < n_groups && col < p.ncols && row_ok) {
                            if (c > 0) add[gi][e] = __ldcg(Op + (uint64_t)col * p.M);
                            else if (col >= g0) add[gi][e] = __ldg(Gp + (uint64_t)(col - g0) * p.M);
                        }
                    }
                }
                ptx::mbar_wait(&tmem_full[as], aphase);
                ptx::tc_fence_after();
                const uint32_t tacc = tmem_base + ((quarter * 32) << 16) + as * acc_cols;
                // rolled loop: the body always consumes add[0], the prefetched words shift down after
                // every group (register moves), which keeps the indices compile-time constants
#pragma unroll 1
                for (uint32_t g = half; g < n_groups; g += 2) {
                    // the group's 8 columns of all seven sums at once, then eight independent reductions (computed
                    // unconditionally so that the compiler interleaves their multiply chains; only the stores are
                    // guarded), then the stores
                    uint32_t v[7][8];
#pragma unroll
                    for (int s = 0; s < 7; ++s) ptx::tmem_ld8(tacc + s * p.ct + g * 8, v[s]);
                    ptx::tmem_ld_wait();
                    uint32_t res[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        // sum_s 2^(8s) S_s with S_s < 2^31 (one K chunk).  The low four limb sums are combined with
                        // shifts (< 2^57); the high three are weighted by 2^(8s) mod q < 2^30 (each product < 2^61),
                        // so the total stays below 2^63 and ONE Barrett reduction per output word remains.
                        uint64_t x = (uint64_t)v[0][e] + ((uint64_t)v[1][e] << 8) + ((uint64_t)v[2][e] << 16) +
                                     ((uint64_t)v[3][e] << 24);
                        x += (uint64_t)v[4][e] * w4 + (uint64_t)v[5][e] * w5 + (uint64_t)v[6][e] * w6;
                        x += add[0][e];
                        res[e] = barrett_u64(x, q, bm);
                    }
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const uint32_t col = nt * p.ct + g * 8 + e;
                        if (col < p.ncols && row_ok) Op[(uint64_t)col * p.M] = res[e];
                    }
#pragma unroll
                    for (int gi = 0; gi < 3; ++gi)
#pragma unroll
                        for (int e = 0; e < 8; ++e) add[gi][e] = add[gi + 1][e];
                }
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if constexpr (CG == 2) ptx::mbar_arrive_cluster_relaxed(&tmem_empty[as], 0);
                    else ptx::mbar_arrive(&tmem_empty[as]);
                }
            }
        }
    }

    // ===== teardown =====
    ptx::tc_fence_before();
    if constexpr (CG == 2) ptx::cluster_sync(); else __syncthreads();
    if (warp == 2) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc<CG>(tmem_base, p.tmem_cols);
    }
}

}  // namespace vipir
