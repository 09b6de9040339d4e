// gemv_b1.cuh -- step a2: the batch-1 HBM-streaming scan (regime a).
//
// PAPER.md:293 (section 5): "separate CUDA-core-based kernels for the INT8-INT32
// matrix-vector multiplications in single-batch execution as they are memory-bound and
// cannot exploit tensor-core throughput".  answer[r] = sum_k D[r][k] * Q[k] mod 2^32.
//
// B200 design: the DB is read exactly once, by TMA, into a
// multi-stage shared-memory ring (one 32-row x 1024-byte box per stage, 32 KiB, plus the
// matching 4 x 1024-byte slice of the query's limb planes); a producer warp keeps the ring
// full so ~200 KiB per SM are in flight regardless of register pressure; eight consumer
// warps read the ring with 128-bit shared loads and multiply with dp4a against the
// pre-split 8-bit query limbs (PAPER.md:245-249 limb identity): 1 integer op per DB byte
// instead of 2 for unpack+IMAD.  Each consumer thread keeps its 16 query-limb registers
// for eight DB rows, so shared-memory traffic is 1.5x the DB stream (of 128 B/clk/SM).
// Row sums are reduced with a transposing warp-shuffle reduction (31 shuffles for 32
// values) and the four limb sums recombined with shifts, wrapping mod 2^32 (:249).
//
// With FUSED (below) the kernel takes the raw query words and splits them itself; otherwise it
// Works on the byte view D' (rows x K' bytes, K' = cols*dl) against LC = 4 limb planes, so
// a u16 DB with q = 2^32 runs through the same kernel (split_limbs.cuh).
#pragma once
#include <cstdint>
#include <cuda.h>
#include "ptx.cuh"
#include "split_limbs.cuh"  // byte_transpose4 (fused query split)

namespace vipir {

constexpr int GV_R = 32;              // DB rows per stage / per CTA row block
constexpr int GV_KT = 1024;           // bytes of K per stage
constexpr int GV_CWARPS = 8;          // consumer warps: 2 along K x 4 along rows
constexpr int GV_THREADS = 32 * (GV_CWARPS + 1);
constexpr int GV_STAGE_BYTES = GV_R * GV_KT + 4 * GV_KT;  // 36864

struct GemvParams {
    uint64_t rows;
    uint32_t kbytes;     // K'
    uint32_t n_ksteps;   // ceil(K' / GV_KT)
    uint32_t n_blocks;   // ceil(rows / GV_R)
    uint32_t stages;
    uint32_t ms_bits;    // fused modulus switch 2^32 -> 2^ms_bits of the answer (0 = off)
    uint32_t* answer;
};

__device__ __forceinline__ uint4 lds128(const uint8_t* p) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "r"(ptx::smem_u32(p)));
    return v;
}

// one dp4a: four u8 (or, SIGNED, two's-complement s8) DB bytes x four u8 query-limb bytes; the
// 32-bit accumulator wraps, which is exact mod 2^32 either way
template <bool SIGNED>
__device__ __forceinline__ uint32_t dp4a_db(uint32_t d, uint32_t q, uint32_t acc) {
    if constexpr (SIGNED) {
        uint32_t r;
        asm("dp4a.s32.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(d), "r"(q), "r"(acc));
        return r;
    } else {
        return __dp4a(d, q, acc);
    }
}

// FUSED: step a1 runs inside the scan.  tmL then maps the RAW query words (u8 DB only: 1024 DB bytes of a row
// meet 1024 query words = the same 4 KiB per stage as four limb slices) as rows of 32 words, boxed 32 x 32 with
// the 128-byte swizzle so that every thread's 64-byte run of 16 words is read with four conflict-free
// ld.shared.v4; the thread transposes them into its four limb registers with prmt (two prmt per
// element) -- 32 prmt next to 128 dp4a per k-step -- and the separate splitter launch disappears.
template <bool SIGNED, bool FUSED>
__global__ void __launch_bounds__(GV_THREADS, 1)
gemv_b1_kernel(const __grid_constant__ CUtensorMap tmD, const __grid_constant__ CUtensorMap tmL, GemvParams p) {
    extern __shared__ uint8_t smem_raw[];
    // 1024-byte alignment: the swizzled query box needs it (a stage is 36 KiB = 36 * 1024)
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)p.stages * GV_STAGE_BYTES);
    uint64_t* empty = full + p.stages;
    uint32_t* red = reinterpret_cast<uint32_t*>(empty + p.stages);  // [2][GV_R]

    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (uint32_t s = 0; s < p.stages; ++s) {
            ptx::mbar_init(&full[s], 1);
            ptx::mbar_init(&empty[s], GV_CWARPS);
        }
        ptx::fence_barrier_init();
        ptx::prefetch_tmap(&tmD);
        ptx::prefetch_tmap(&tmL);
    }
    __syncthreads();

    if (warp == GV_CWARPS) {
        // ===== producer warp: one lane issues the TMA loads =====
        if (lane == 0) {
            uint32_t stage = 0, phase = 0;
            for (uint32_t blk = blockIdx.x; blk < p.n_blocks; blk += gridDim.x) {
                for (uint32_t ks = 0; ks < p.n_ksteps; ++ks) {
                    ptx::mbar_wait(&empty[stage], phase ^ 1);
                    uint8_t* dst = smem + (size_t)stage * GV_STAGE_BYTES;
                    ptx::mbar_arrive_expect_tx(&full[stage], GV_STAGE_BYTES);
                    // tensor maps are typed u32: coordinates are in 4-byte elements
                    ptx::tma_load_2d(dst, &tmD, &full[stage], (int32_t)(ks * (GV_KT / 4)), (int32_t)(blk * GV_R),
                                     ptx::kEvictFirst);
                    if constexpr (FUSED)  // query words [ks*1024, +1024): rows ks*32 .. +32 of the 32-word view
                        ptx::tma_load_2d(dst + GV_R * GV_KT, &tmL, &full[stage], 0, (int32_t)(ks * 32), ptx::kEvictLast);
                    else
                        ptx::tma_load_2d(dst + GV_R * GV_KT, &tmL, &full[stage], (int32_t)(ks * (GV_KT / 4)), 0,
                                         ptx::kEvictLast);
                    if (++stage == p.stages) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else {
        // ===== consumer warps =====
        const uint32_t kw = warp & 1;   // which 512-byte half of the K slice
        const uint32_t rw = warp >> 1;  // which 8-row group
        const uint32_t koff = kw * 512 + lane * 16;
        uint32_t stage = 0, phase = 0;
        for (uint32_t blk = blockIdx.x; blk < p.n_blocks; blk += gridDim.x) {
            uint32_t acc[32];  // acc[rr*4 + j]: row rr of this warp's 8, query limb j
#pragma unroll
            for (int i = 0; i < 32; ++i) acc[i] = 0;

            for (uint32_t ks = 0; ks < p.n_ksteps; ++ks) {
                ptx::mbar_wait(&full[stage], phase);
                const uint8_t* sD = smem + (size_t)stage * GV_STAGE_BYTES;
                const uint8_t* sL = sD + GV_R * GV_KT;
                uint4 q[4];
                if constexpr (FUSED) {
                    // words [koff, koff + 16) of this K slice: 128-byte row koff/32, 16-byte chunks
                    // (koff/4 % 8) + {0..3}, stored at chunk ^ (row % 8) (128B swizzle)
                    const uint32_t row = koff >> 5, c0 = (koff >> 2) & 7;
                    uint32_t L[4][4];
#pragma unroll
                    for (int w = 0; w < 4; ++w) {
                        const uint4 v = lds128(sL + row * 128 + (((c0 + w) ^ (row & 7)) << 4));
                        byte_transpose4(v.x, v.y, v.z, v.w, L[w]);
                    }
#pragma unroll
                    for (int j = 0; j < 4; ++j) q[j] = make_uint4(L[0][j], L[1][j], L[2][j], L[3][j]);
                } else {
#pragma unroll
                    for (int j = 0; j < 4; ++j) q[j] = lds128(sL + j * GV_KT + koff);
                }
                uint4 d[8];
#pragma unroll
                for (int rr = 0; rr < 8; ++rr) d[rr] = lds128(sD + (rw * 8 + rr) * GV_KT + koff);
#pragma unroll
                for (int rr = 0; rr < 8; ++rr) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        uint32_t a = acc[rr * 4 + j];
                        a = dp4a_db<SIGNED>(d[rr].x, q[j].x, a);
                        a = dp4a_db<SIGNED>(d[rr].y, q[j].y, a);
                        a = dp4a_db<SIGNED>(d[rr].z, q[j].z, a);
                        a = dp4a_db<SIGNED>(d[rr].w, q[j].w, a);
                        acc[rr * 4 + j] = a;
                    }
                }
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(&empty[stage]);
                if (++stage == p.stages) { stage = 0; phase ^= 1; }
            }

            // transposing warp reduction: after 5 halving steps lane l holds the warp-wide
            // sum of acc[l] (31 shuffles instead of 160)
#pragma unroll
            for (int off = 16, n = 32; off >= 1; off >>= 1, n >>= 1) {
                const bool upper = (lane & off) != 0;
#pragma unroll
                for (int i = 0; i < n / 2; ++i) {
                    const uint32_t send = upper ? acc[i] : acc[i + n / 2];
                    const uint32_t keep = upper ? acc[i + n / 2] : acc[i];
                    acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
                }
            }
            // lane = rr*4 + j: shift limb j into place and add the four limbs (mod 2^32)
            uint32_t v = acc[0] << (8 * (lane & 3));
            v += __shfl_xor_sync(0xffffffffu, v, 1);
            v += __shfl_xor_sync(0xffffffffu, v, 2);
            if ((lane & 3) == 0) red[kw * GV_R + rw * 8 + (lane >> 2)] = v;
            asm volatile("bar.sync 1, %0;" ::"n"(GV_CWARPS * 32) : "memory");
            if (threadIdx.x < GV_R) {
                const uint64_t row = (uint64_t)blk * GV_R + threadIdx.x;
                if (row < p.rows) {
                    const uint32_t v = red[threadIdx.x] + red[GV_R + threadIdx.x];
                    p.answer[row] = p.ms_bits ? modswitch_word(v, p.ms_bits) : v;
                }
            }
            asm volatile("bar.sync 1, %0;" ::"n"(GV_CWARPS * 32) : "memory");
        }
    }
}

}  // namespace vipir
