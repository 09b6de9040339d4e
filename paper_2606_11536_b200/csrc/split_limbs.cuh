// split_limbs.cuh -- step a1: the query-limb splitter.
//
// PAPER.md:245-251 (section 4.1): "we decompose the INT32 matrix into four INT8 matrices
// B0..B3 ... Given four contiguous INT32 elements from B, we use two prmt instructions
// [per element] to extract one byte from each element and pack them into a single 32-bit
// register".  The paper fuses this into its GEMM kernel; here it is a pre-pass that writes
// the byte planes in exactly the K-major layout TMA hands to the consumers.
//
// Output ("limb planes"): P[n][kb], n = q*LC + s, kb in [0, K'), K' = cols*dl, u8, row pitch
// K' bytes, for query vector q in [0, nq) and shift s in [0, LC):
//   dl = 1 (u8 DB):   P[q*LC+s][k]      = byte s of Q[q][k]                      (LC = 4)
//   dl = 2 (u16 DB):  P[q*LC+s][2k + i] = byte (s-i) of Q[q][k], 0 if s-i not in 0..3
// so that  D'(rows x K' bytes, the DB viewed as bytes) * P[q*LC+s]^T = S_s =
// sum_{i+j=s} (D_i * Q_j), and the answer is sum_s 2^(8s) S_s.  For q = 2^32 the s = 4 term
// vanishes, so LC = 4 there; prime moduli with a u16 DB need LC = 5.
#pragma once
#include <cstdint>

namespace vipir {

// 128-bit store that leaves the line in L2 with evict_last priority: the planes are re-read by
// every M tile of the scan kernel while the DB streams through the same L2.
__device__ __forceinline__ void st_evict_last(uint8_t* dst, uint4 v) {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("st.global.L2::cache_hint.v4.b32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(dst), "r"(v.x), "r"(v.y), "r"(v.z),
                 "r"(v.w), "l"(pol)
                 : "memory");
}

// 4x4 byte transpose of four consecutive query words with 8 prmt (2 per element).
__device__ __forceinline__ void byte_transpose4(uint32_t a, uint32_t b, uint32_t c, uint32_t d, uint32_t L[4]) {
    const uint32_t ab_lo = __byte_perm(a, b, 0x5140);  // a0 b0 a1 b1
    const uint32_t ab_hi = __byte_perm(a, b, 0x7362);  // a2 b2 a3 b3
    const uint32_t cd_lo = __byte_perm(c, d, 0x5140);
    const uint32_t cd_hi = __byte_perm(c, d, 0x7362);
    L[0] = __byte_perm(ab_lo, cd_lo, 0x5410);  // a0 b0 c0 d0
    L[1] = __byte_perm(ab_lo, cd_lo, 0x7632);  // a1 b1 c1 d1
    L[2] = __byte_perm(ab_hi, cd_hi, 0x5410);
    L[3] = __byte_perm(ab_hi, cd_hi, 0x7632);
}

// One thread handles 16 consecutive k of one query vector (4 x 128-bit loads).
// cols must be a multiple of 16/dl (the ABI's 16-byte row rule); tail threads are guarded.
// Only the columns [k_lo, k_hi) are split (k_lo a multiple of 16; the whole vector: 0, cols) -- the host
// entry point splits a query slice by slice along K as its copies arrive.
template <int DL, int LC>
__global__ void __launch_bounds__(256) split_limbs_kernel(const uint32_t* __restrict__ Q, uint8_t* __restrict__ P,
                                                          uint64_t cols, uint32_t nq, uint64_t k_lo, uint64_t k_hi) {
    const uint64_t groups_per_q = (k_hi - k_lo + 15) / 16;
    const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= groups_per_q * nq) return;
    const uint32_t q = (uint32_t)(gid / groups_per_q);
    const uint64_t k0 = k_lo + (gid % groups_per_q) * 16;
    const uint32_t* src = Q + (uint64_t)q * cols + k0;
    const uint64_t kp = cols * DL;  // plane pitch in bytes

    uint32_t L[4][4];  // L[word][limb]: limb bytes of k0+4w .. k0+4w+3
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        uint4 v = make_uint4(0, 0, 0, 0);
        if (k0 + 4 * w + 3 < cols) {
            v = *reinterpret_cast<const uint4*>(src + 4 * w);
        } else {
            uint32_t t[4] = {0, 0, 0, 0};
            for (int e = 0; e < 4; ++e)
                if (k0 + 4 * w + e < cols) t[e] = src[4 * w + e];
            v = make_uint4(t[0], t[1], t[2], t[3]);
        }
        byte_transpose4(v.x, v.y, v.z, v.w, L[w]);
    }

    if constexpr (DL == 1) {
#pragma unroll
        for (int s = 0; s < LC; ++s) {
            uint8_t* dst = P + ((uint64_t)q * LC + s) * kp + k0;
            if (k0 + 15 < cols) {
                st_evict_last(dst, make_uint4(L[0][s], L[1][s], L[2][s], L[3][s]));
            } else {
                for (int w = 0; w < 4; ++w)
                    for (int e = 0; e < 4; ++e)
                        if (k0 + 4 * w + e < cols) dst[4 * w + e] = (uint8_t)(L[w][s] >> (8 * e));
            }
        }
    } else {
#pragma unroll
        for (int s = 0; s < LC; ++s) {
            // bytes at 2k+0 come from limb s, bytes at 2k+1 from limb s-1
            uint32_t o[8];
#pragma unroll
            for (int w = 0; w < 4; ++w) {
                const uint32_t even = (s < 4) ? L[w][s < 4 ? s : 0] : 0u;
                const uint32_t odd = (s >= 1) ? L[w][s >= 1 ? s - 1 : 0] : 0u;
                o[2 * w] = __byte_perm(even, odd, 0x5140);      // e0 o0 e1 o1
                o[2 * w + 1] = __byte_perm(even, odd, 0x7362);  // e2 o2 e3 o3
            }
            uint8_t* dst = P + ((uint64_t)q * LC + s) * kp + 2 * k0;
            if (k0 + 15 < cols) {
                st_evict_last(dst, make_uint4(o[0], o[1], o[2], o[3]));
                st_evict_last(dst + 16, make_uint4(o[4], o[5], o[6], o[7]));
            } else {
                for (int w = 0; w < 8; ++w)
                    for (int e = 0; e < 4; ++e)
                        if (k0 + (4 * w + e) / 2 < cols) dst[4 * w + e] = (uint8_t)(o[w] >> (8 * e));
            }
        }
    }
}

}  // namespace vipir
