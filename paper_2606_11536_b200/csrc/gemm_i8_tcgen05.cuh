// gemm_i8_tcgen05.cuh -- steps a3 + a4 (+ a5): the batched scan on the 5th-generation
// tensor cores (regime b).
//
// PAPER.md:245-249 (section 4.1): "As tensor cores support INT8 GEMMs with INT32
// accumulation, we decompose the INT32 matrix into four INT8 matrices ... to compute A*B as
//   A*B0 + 2^8 (A*B1) + 2^16 (A*B2) + 2^24 (A*B3)  mod 2^32
// where each A*Bj is computed using tensor cores, multiplications by {2^8,2^16,2^24} are
// implemented via bit shifts, and modulo-2^32 reduction is free."  Prime moduli
// replace the free wrap by an explicit reduction.
//
// B200 design: persistent, warp-specialised.
//   warp 0   TMA producer: per k-step (128 bytes of K) one 128-row x 128-byte box of the DB
//            byte view D' and the matching box(es) of the limb planes, 128B-swizzled, into an
//            mbarrier ring;
//   warp 1   MMA issuer: one thread issues tcgen05.mma.kind::i8 (u8 x u8 -> s32, M = 128 per
//            CTA, N <= 256 per instruction, K = 32 bytes), accumulators in TMEM; the limb
//            planes are laid out so that the LC limb sums of one query are LC adjacent
//            accumulator columns;
//   warp 2   TMEM allocator;
//   warps 4-7 epilogue: tcgen05.ld the accumulators of their lane quarter, recombine limbs
//            with shifts (wrap mod 2^32) or in u64 + Barrett (prime moduli), and store /
//            read-modify-write answer[q][row] (coalesced over rows).
// The K dimension is processed in chunks of <= 32768 bytes (256 k-steps): 255*255*32768 <
// 2^31, so the s32 accumulators hold the exact limb sums (reading R7); the
// accumulators are drained after every chunk.  With CG = 2 a pair of CTAs (one cluster of 2
// SMs) runs cta_group::2 MMAs: M = 256 rows per pair, each CTA stages its own 128 DB rows and
// HALF of the limb-plane tile, halving shared-memory fill and read traffic per SM.
#pragma once
#include <cstdint>
#include <cuda.h>
#include "ptx.cuh"

namespace vipir {

constexpr int GM_BM = 128;           // rows per CTA
constexpr int GM_BK = 128;           // bytes of K per stage (one 128B swizzle row)
constexpr int GM_UMMA_K = 32;        // bytes of K per tcgen05.mma.kind::i8
constexpr int GM_THREADS = 256;
constexpr int GM_A_BYTES = GM_BM * GM_BK;  // 16384
constexpr int GM_MAX_MODULI = 4;

struct GemmParams {
    uint64_t rows;
    uint32_t nq;             // query vectors = T * batch
    uint32_t batch;          // queries per modulus
    uint32_t qt;             // query vectors per N tile
    uint32_t bn;             // accumulator columns per tile = qt * LC
    uint32_t n_tiles, m_tiles;
    uint32_t ni_cols;        // N of one MMA instruction
    uint32_t n_instr;        // instructions per k-step (bn = n_instr * ni_cols)
    uint32_t total_ksteps;   // ceil(K' / 128): number of 128-byte k-atoms
    uint32_t ksteps_per_chunk;
    uint32_t n_chunks;
    uint32_t katoms;         // k-atoms per pipeline stage (>= 1): one stage = katoms x (A box + B boxes)
    uint32_t atom_bytes;     // per CTA: 16 KiB of DB + this CTA's share of the limb tile, for one k-atom
    uint32_t stages;
    uint32_t stage_bytes;    // per CTA = katoms * atom_bytes
    uint32_t tmem_cols, acc_stages;
    uint32_t idesc;
    uint32_t ms_bits;        // fused modulus switch 2^32 -> 2^ms_bits of the answer (0 = off; q = 2^32 only)
    uint32_t db_signed;      // DB bytes are s8 (A format s8 in idesc): the s32 accumulators may be negative
    uint32_t n_moduli;
    uint32_t moduli[GM_MAX_MODULI];
    uint64_t barrett[GM_MAX_MODULI];  // floor(2^64 / p)
    uint32_t* answer;
};

// K-major, 128B-swizzled shared-memory operand descriptor (8-row x 128-byte atoms, 1024 B apart)
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFF) >> 4);        // start address, bits [0,14)
    d |= (uint64_t)1 << 16;                         // leading byte offset (unused for swizzled K-major)
    d |= (uint64_t)(1024 >> 4) << 32;               // stride byte offset: 8 rows * 128 B
    d |= (uint64_t)1 << 46;                         // descriptor version (sm_100)
    d |= (uint64_t)2 << 61;                         // SWIZZLE_128B
    return d;
}

// x mod p for any u64 x, p in [2, 2^30): m = floor(2^64 / p); q' = mulhi(x, m) in {q-1, q}
__device__ __forceinline__ uint32_t barrett_u64(uint64_t x, uint32_t p, uint64_t m) {
    const uint64_t qhat = __umul64hi(x, m);
    uint64_t r = x - qhat * p;
    if (r >= p) r -= p;
    return (uint32_t)r;
}

template <int CG, int LC, bool PRIME>
__global__ void __launch_bounds__(GM_THREADS, 1)
gemm_i8_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, GemmParams p) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)p.stages * p.stage_bytes);
    uint64_t* empty = full + p.stages;
    uint64_t* tmem_full = empty + p.stages;   // [2]
    uint64_t* tmem_empty = tmem_full + 2;     // [2]
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(tmem_empty + 2);

    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t rank = (CG == 2) ? ptx::cluster_ctarank() : 0u;
    const uint32_t unit0 = (CG == 2) ? ptx::cluster_id_x() : blockIdx.x;
    const uint32_t unit_stride = (CG == 2) ? ptx::num_clusters_x() : gridDim.x;
    const uint32_t n_units = p.m_tiles * p.n_tiles;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tmA);
        ptx::prefetch_tmap(&tmB);
    }
    if (warp == 1 && lane == 0) {
        for (uint32_t s = 0; s < p.stages; ++s) {
            ptx::mbar_init(&full[s], 1);
            ptx::mbar_init(&empty[s], 1);
        }
        for (uint32_t a = 0; a < 2; ++a) {
            ptx::mbar_init(&tmem_full[a], 1);
            ptx::mbar_init(&tmem_empty[a], 4 * CG);  // one arrival per epilogue warp of every CTA
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
    const uint32_t tmem_base = *tmem_ptr;

    if (warp == 0) {
        // ===== TMA producer =====
        if (lane == 0) {
            uint32_t stage = 0, phase = 0;
            const uint32_t b_rows = p.ni_cols / CG;  // limb-plane rows this CTA stages per instruction
            const uint32_t b_bytes = b_rows * GM_BK;
            for (uint32_t u = unit0; u < n_units; u += unit_stride) {
                const uint32_t mt = u / p.n_tiles, nt = u % p.n_tiles;
                // the DB is streamed once (evict_first); with several N tiles the sibling tiles, which
                // run alongside on neighbouring clusters, re-read it from L2, so it stays evict_normal
                // (ncu: marking the last sibling evict_first raised DRAM reads from 5.6 to 8.0 GB on C4)
                const uint64_t hintA = (p.n_tiles == 1) ? ptx::kEvictFirst : ptx::kEvictNormal;
                const int32_t row0 = (int32_t)((mt * CG + rank) * GM_BM);
                for (uint32_t c = 0; c < p.n_chunks; ++c) {
                    const uint32_t ks_begin = c * p.ksteps_per_chunk;
                    const uint32_t ks_end = min(p.total_ksteps, ks_begin + p.ksteps_per_chunk);
                    // a stage never straddles a chunk: the last stage of a chunk may hold fewer atoms
                    for (uint32_t ks0 = ks_begin; ks0 < ks_end; ks0 += p.katoms) {
                        const uint32_t na = min(p.katoms, ks_end - ks0);
                        ptx::mbar_wait(&empty[stage], phase ^ 1);
                        uint8_t* sbase = smem + (size_t)stage * p.stage_bytes;
                        uint32_t bar = 0;
                        if constexpr (CG == 1) {
                            ptx::mbar_arrive_expect_tx(&full[stage], na * p.atom_bytes);
                        } else {
                            // both CTAs' bytes are counted on the leader's barrier
                            if (rank == 0) ptx::mbar_arrive_expect_tx(&full[stage], 2 * na * p.atom_bytes);
                            bar = ptx::mapa(ptx::smem_u32(&full[stage]), 0);
                        }
                        for (uint32_t a = 0; a < na; ++a) {
                            uint8_t* sA = sbase + a * p.atom_bytes;
                            uint8_t* sB = sA + GM_A_BYTES;
                            const int32_t k0 = (int32_t)((ks0 + a) * GM_BK);
                            if constexpr (CG == 1) {
                                ptx::tma_load_2d(sA, &tmA, &full[stage], k0, row0, hintA);
                                for (uint32_t j = 0; j < p.n_instr; ++j)
                                    ptx::tma_load_2d(sB + j * b_bytes, &tmB, &full[stage], k0,
                                                     (int32_t)(nt * p.bn + j * p.ni_cols), ptx::kEvictLast);
                            } else {
                                ptx::tma_load_2d_pair(sA, &tmA, bar, k0, row0, hintA);
                                for (uint32_t j = 0; j < p.n_instr; ++j)
                                    ptx::tma_load_2d_pair(sB + j * b_bytes, &tmB, bar, k0,
                                                          (int32_t)(nt * p.bn + j * p.ni_cols + rank * b_rows),
                                                          ptx::kEvictLast);
                            }
                        }
                        if (++stage == p.stages) { stage = 0; phase ^= 1; }
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (leader CTA of the pair only) =====
        if (rank == 0 && lane == 0) {
            uint32_t stage = 0, phase = 0, acc_it = 0;
            const uint32_t b_bytes = (p.ni_cols / CG) * GM_BK;
            for (uint32_t u = unit0; u < n_units; u += unit_stride) {
                for (uint32_t c = 0; c < p.n_chunks; ++c, ++acc_it) {
                    const uint32_t as = acc_it % p.acc_stages;
                    const uint32_t aphase = (acc_it / p.acc_stages) & 1;
                    if constexpr (CG == 2) ptx::mbar_wait_cluster(&tmem_empty[as], aphase ^ 1);
                    else ptx::mbar_wait(&tmem_empty[as], aphase ^ 1);
                    ptx::tc_fence_after();
                    const uint32_t ks_begin = c * p.ksteps_per_chunk;
                    const uint32_t ks_end = min(p.total_ksteps, ks_begin + p.ksteps_per_chunk);
                    const uint32_t tacc = tmem_base + as * p.bn;
                    for (uint32_t ks0 = ks_begin; ks0 < ks_end; ks0 += p.katoms) {
                        const uint32_t na = min(p.katoms, ks_end - ks0);
                        ptx::mbar_wait(&full[stage], phase);
                        ptx::tc_fence_after();
                        const uint32_t sbase = ptx::smem_u32(smem + (size_t)stage * p.stage_bytes);
                        for (uint32_t a = 0; a < na; ++a) {
                            const uint32_t sA = sbase + a * p.atom_bytes;
                            const uint32_t sB = sA + GM_A_BYTES;
                            const uint64_t dA = make_smem_desc(sA);
                            for (uint32_t j = 0; j < p.n_instr; ++j) {
                                const uint64_t dB = make_smem_desc(sB + j * b_bytes);
#pragma unroll
                                for (uint32_t kk = 0; kk < GM_BK / GM_UMMA_K; ++kk) {
                                    // advancing K inside the swizzle atom = adding the byte offset >> 4
                                    const uint64_t koff = (uint64_t)((kk * GM_UMMA_K) >> 4);
                                    ptx::mma_i8<CG>(tacc + j * p.ni_cols, dA + koff, dB + koff, p.idesc,
                                                    (ks0 + a > ks_begin || kk > 0) ? 1u : 0u);
                                }
                            }
                        }
                        // release the smem slot once these MMAs have read it
                        if constexpr (CG == 2) ptx::tc_commit_pair(&empty[stage], 3);
                        else ptx::tc_commit(&empty[stage]);
                        if (++stage == p.stages) { stage = 0; phase ^= 1; }
                    }
                    // accumulators of this chunk complete -> epilogue
                    if constexpr (CG == 2) ptx::tc_commit_pair(&tmem_full[as], 3);
                    else ptx::tc_commit(&tmem_full[as]);
                }
            }
        }
    } else if (warp >= 4) {
        // ===== epilogue warps: lane quarter = warp % 4 =====
        const uint32_t quarter = warp & 3;
        uint32_t acc_it = 0;
        for (uint32_t u = unit0; u < n_units; u += unit_stride) {
            const uint32_t mt = u / p.n_tiles, nt = u % p.n_tiles;
            const uint64_t row = (uint64_t)(mt * CG + rank) * GM_BM + quarter * 32 + lane;
            const bool row_ok = row < p.rows;
            for (uint32_t c = 0; c < p.n_chunks; ++c, ++acc_it) {
                const uint32_t as = acc_it % p.acc_stages;
                const uint32_t aphase = (acc_it / p.acc_stages) & 1;
                ptx::mbar_wait(&tmem_full[as], aphase);
                ptx::tc_fence_after();
                const uint32_t tacc = tmem_base + ((quarter * 32) << 16) + as * p.bn;
                // later chunks add to what chunk 0 stored: a fire-and-forget red.add for q = 2^32; for
                // primes the old words are fetched eight steps (32 query vectors) at a time so that
                // one global-load latency is paid per batch, not per step
                // with the fused modulus switch (q = 2^32 only) the LAST chunk needs the running sum back
                // to round it: same batched prefetch, once per tile
                constexpr uint32_t kPf = 8;
                const bool ms_final = !PRIME && p.ms_bits != 0 && c + 1 == p.n_chunks;
                const bool need_old = c > 0 && (PRIME || ms_final);
                for (uint32_t g0 = 0; g0 < p.qt / 4; g0 += kPf) {
                    uint32_t old[4 * kPf];
                    if (need_old) {
#pragma unroll
                        for (uint32_t i = 0; i < 4 * kPf; ++i) {
                            const uint32_t q = nt * p.qt + g0 * 4 + i;
                            old[i] = (q < p.nq && row_ok && g0 * 4 + i < p.qt)
                                         ? __ldcg(p.answer + (uint64_t)q * p.rows + row) : 0u;
                        }
                    }
#pragma unroll
                    for (uint32_t gg = 0; gg < kPf; ++gg) {
                        const uint32_t g = g0 + gg;
                        if (g >= p.qt / 4) break;
                        uint32_t v[4 * LC];
                        ptx::tmem_ld16(tacc + g * (4 * LC), v);
                        if constexpr (LC == 5) ptx::tmem_ld4(tacc + g * (4 * LC) + 16, v + 16);
                        ptx::tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const uint32_t q = nt * p.qt + g * 4 + i;
                            if (q < p.nq && row_ok) {
                                uint32_t* dst = p.answer + (uint64_t)q * p.rows + row;
                                if constexpr (!PRIME) {
                                    // shifts, wrap mod 2^32 (an s = 4 column would vanish)
                                    uint32_t val =
                                        v[i * LC] + (v[i * LC + 1] << 8) + (v[i * LC + 2] << 16) + (v[i * LC + 3] << 24);
                                    if (ms_final) {
                                        if (c > 0) val += old[gg * 4 + i];
                                        *dst = modswitch_word(val, p.ms_bits);
                                    } else if (c == 0) {
                                        *dst = val;
                                    } else {
                                        asm volatile("red.global.add.u32 [%0], %1;" ::"l"(dst), "r"(val) : "memory");
                                    }
                                } else {
                                    const uint32_t t = q / p.batch;
                                    const uint32_t pm = p.moduli[t];
                                    uint32_t val;
                                    if constexpr (LC == 4) {
                                        // every |P_s| < 2^31 (R7), so the s32 reading is exact for u8 and s8
                                        // DBs alike and |x| < 2^56; a negative x reduces as p - (|x| mod p)
                                        int64_t x = 0;
#pragma unroll
                                        for (int s = 0; s < LC; ++s) x += (int64_t)(int32_t)v[i * LC + s] << (8 * s);
                                        const bool neg = x < 0;
                                        val = barrett_u64((uint64_t)(neg ? -x : x), pm, p.barrett[t]);
                                        if (neg && val != 0) val = pm - val;
                                    } else {
                                        uint64_t x = 0;  // u16 DB (never signed): up to 2^63 * 1.004
#pragma unroll
                                        for (int s = 0; s < LC; ++s) x += (uint64_t)v[i * LC + s] << (8 * s);
                                        val = barrett_u64(x, pm, p.barrett[t]);
                                    }
                                    if (c > 0) {
                                        val += old[gg * 4 + i];
                                        if (val >= pm) val -= pm;
                                    }
                                    *dst = val;
                                }
                            }
                        }
                    }
                }
                // accumulator stage drained
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if constexpr (CG == 2) ptx::mbar_arrive_cluster(&tmem_empty[as], 0);
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
