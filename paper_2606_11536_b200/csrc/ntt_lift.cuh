// ntt_lift.cuh -- the lift + forward negacyclic NTT that turns the scan's scalar-HE output (and,
// offline, the hint) into the ring-packing operands G and H, written straight into the modular
// GEMMs' tile-major layout (the step between vipir_dbmul and vipir_modgemm).
//
// PAPER.md:214 (section 3.5.2): "the D1 x n and D1 x B SimplePIR outputs are first transformed into
// polynomials by treating each length-N vector along the D1 dimension as a polynomial in R_q ...
// to which NTTs are applied independently.  Let H and G denote these two polynomial matrices
// after the NTTs."  PAPER.md:667 (Appendix C.1): "the server lifts the coefficients of iota(A_i)
// and iota(b) from Z_p to Z_q and transforms them into the NTT domain"; eq. (3)
// scales the b part by Delta.  PAPER.md:269-271 (section 4.3): "a single-kernel design ... For
// the NTT with N = 2^12, whose working set fits within on-chip resources"; fused with its
// neighbours ("we fuse the initial RNS decomposition with the NTT"); PAPER.md:263 (section 4.2):
// "layout transpositions before and after the GEMMs to convert between polynomial-major
// (NTT-friendly) and tile-major (GEMM-friendly) layouts".
//
// B200 design.  Kept from the paper: one kernel per transform with the
// polynomial resident on chip, RNS decomposition (the lift) fused in front, and the layout
// transposition -- here fused behind it, into the kernel's store.  Changed: Shoup/Harvey lazy
// butterflies (one mul.hi + two mul.lo per twiddle product, values kept in [0, 4q), a single
// normalisation at the end) instead of Montgomery products (four multiplies): every twiddle is a
// plan-time constant, so its Shoup companion floor(w * 2^32 / q) is precomputed with it.
//
// Algorithm: the merged (negacyclic) Cooley-Tukey transform, natural-order input, twiddles
// psi^bitrev(i); log2 N = 4 * passes, each pass = four radix-2 stages on 16 elements held in
// registers (a radix-16 step), the passes exchanging data through padded shared memory.  The
// transform leaves Y[bitrev(pos)] at position pos; the last pass writes to shared memory in natural
// order, and the CTA then stores, for every NTT coefficient c, the P results of its P polynomials
// as one contiguous run (they are neighbours along the GEMM operand's inner dimension).
#pragma once
#include <cstdint>

namespace vipir {

constexpr int NTT_THREADS = 512;
constexpr int NTT_MAX_MODULI = 4;

struct NttParams {
    uint32_t T;
    uint32_t n_outer, n_inner;   // polynomial grid in OUTPUT order: O[t][c][outer][inner]
    uint32_t in_stride_outer;    // input polynomial index = outer * in_stride_outer + inner * in_stride_inner
    uint32_t in_stride_inner;
    uint32_t p_bits, centered;
    uint32_t moduli[NTT_MAX_MODULI];
    uint32_t scale[NTT_MAX_MODULI], scale_shoup[NTT_MAX_MODULI];
    const uint32_t* twiddles;    // [T][2][N]: w[i] = psi^bitrev(i) mod q, then floor(w[i] * 2^32 / q)
    const uint32_t* X;           // polynomial-major input words, each < 2^p_bits
    uint32_t* O;
    uint32_t* bad_input;         // set to 1 if a word >= 2^p_bits was seen (its excess bits are ignored)
};

// y * w mod q, lazily: result in [0, 2q) for any 32-bit y (Harvey); ws = floor(w * 2^32 / q)
__device__ __forceinline__ uint32_t shoup_mul(uint32_t y, uint32_t w, uint32_t ws, uint32_t q) {
    const uint32_t qhat = __umulhi(y, ws);
    return y * w - qhat * q;
}

// x, y in [0, 4q) -> x + w*y, x - w*y, both in [0, 4q)
__device__ __forceinline__ void harvey_butterfly(uint32_t& x, uint32_t& y, uint32_t w, uint32_t ws, uint32_t q) {
    const uint32_t two_q = 2 * q;
    const uint32_t xr = min(x, x - two_q);  // x - 2q wraps to a huge value when x < 2q
    const uint32_t t = shoup_mul(y, w, ws, q);
    x = xr + t;
    y = xr - t + two_q;
}

// four radix-2 stages (one radix-16 step) on r[0..15]; pass rho covers stages 4*rho .. 4*rho+3,
// `hi` = the element index bits above this group's 4 bits.  tw/tws: the prime's tables (shared memory).
template <bool TW_SMEM>
__device__ __forceinline__ void radix16_pass(uint32_t (&r)[16], uint32_t rho, uint32_t hi, const uint32_t* tw,
                                             const uint32_t* tws, uint32_t q) {
#pragma unroll
    for (int sigma = 0; sigma < 4; ++sigma) {
        const int half = 8 >> sigma;
        const uint32_t base = (1u << (4 * rho + sigma)) + (hi << sigma);
#pragma unroll
        for (int b = 0; b < (1 << sigma); ++b) {
            const uint32_t w = TW_SMEM ? tw[base + b] : __ldg(tw + base + b);
            const uint32_t ws = TW_SMEM ? tws[base + b] : __ldg(tws + base + b);
#pragma unroll
            for (int k = 0; k < half; ++k) harvey_butterfly(r[b * 2 * half + k], r[b * 2 * half + k + half], w, ws, q);
        }
    }
}

// barrier among the TP threads of one polynomial.  For N = 4096 (TP = 256: whole warps) it is a named
// barrier of its own, so the Q polynomials in flight drift out of phase and one's global loads and
// barrier waits overlap the other's butterflies; smaller N (sub-warp groups) use the CTA barrier.
template <uint32_t TP, uint32_t NT>
__device__ __forceinline__ void ntt_group_sync(uint32_t group) {
    if constexpr (TP % 32 == 0 && TP < NT) {
        asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "n"(TP) : "memory");
    } else {
        __syncthreads();
    }
}

__device__ __forceinline__ uint32_t ntt_pad(uint32_t i) { return i + (i >> 4); }   // work buffer
__device__ __forceinline__ uint32_t ntt_pad_out(uint32_t c) { return c + (c >> 5); }  // natural-order staging

// L = log2 N in {4, 8, 12}.  NT threads per CTA, TP = N/16 threads per polynomial, Q = NT / TP
// polynomials in flight, R rounds: P = Q*R polynomials (neighbours along `inner`) per CTA iteration.
// TW_SMEM: twiddle tables copied to shared memory (small N), or read through L1 (N = 4096, where the
// shared memory goes to the work slots so that MINB CTAs fit on an SM and their multiply-dense and
// shared-memory-dense phases overlap).
template <int L, int NT, int R_, bool TW_SMEM, int MINB>
__global__ void __launch_bounds__(NT, MINB) ntt_lift_kernel(NttParams p) {
    constexpr uint32_t N = 1u << L;
    constexpr uint32_t TP = N / 16;
    constexpr uint32_t Q = NT / TP;
    constexpr uint32_t R = R_;
    constexpr uint32_t P = Q * R;
    constexpr uint32_t NTT_THREADS = NT;
    constexpr uint32_t PASSES = L / 4;
    constexpr uint32_t STR = N + N / 16 + 4;  // words per polynomial slot: padded, and = 4 mod 32 for N >= 512
    extern __shared__ uint32_t ntt_smem[];
    const uint32_t t = blockIdx.y;
    const uint32_t q = p.moduli[t];
    const uint32_t* tw = p.twiddles + (size_t)t * 2 * N;   // [N] w, then [N] floor(w * 2^32 / q)
    uint32_t* buf = ntt_smem;                               // [P][STR]
    if constexpr (TW_SMEM) {
        uint32_t* tw_s = ntt_smem;
        buf = ntt_smem + 2 * N;
        for (uint32_t i = threadIdx.x; i < 2 * N; i += NTT_THREADS) tw_s[i] = tw[i];
        tw = tw_s;
        __syncthreads();
    }
    const uint32_t* tws = tw + N;

    const uint32_t tid = threadIdx.x % TP;   // thread within its polynomial
    const uint32_t slot0 = threadIdx.x / TP; // polynomial slot within a round
    const uint32_t pmask = (1u << p.p_bits) - 1u;
    const uint32_t half_p = 1u << (p.p_bits - 1);
    const uint32_t groups_per_outer = (p.n_inner + P - 1) / P;
    const uint32_t n_groups = p.n_outer * groups_per_outer;
    uint32_t bad = 0;

    for (uint32_t grp = blockIdx.x; grp < n_groups; grp += gridDim.x) {
        const uint32_t outer = grp / groups_per_outer;
        const uint32_t inner0 = (grp % groups_per_outer) * P;
        // this thread's 16 input words of round rd, prefetched into the round's (still unused) work slot
        // with cp.async one round ahead: the global-load latency overlaps the previous round's butterflies
        auto prefetch = [&](uint32_t rd) {
            const uint32_t slot = rd * Q + slot0;
            const uint32_t inner = inner0 + slot;
            if (rd < R && inner < p.n_inner) {
                const uint32_t* src = p.X + ((size_t)outer * p.in_stride_outer + (size_t)inner * p.in_stride_inner) * N;
                const uint32_t dst = (uint32_t)__cvta_generic_to_shared(buf + slot * STR);
                if (STR % 4 == 0 && (reinterpret_cast<uintptr_t>(p.X) & 15) == 0) {  // slots 16-byte aligned
                    // the polynomial copied as it lies (16 bytes per thread and step, coalesced)
#pragma unroll
                    for (int i = 0; i < 4; ++i)
                        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + (i * TP + tid) * 16),
                                     "l"(src + (i * TP + tid) * 4)
                                     : "memory");
                } else {
#pragma unroll
                    for (int k = 0; k < 16; ++k)
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst + (k * TP + tid) * 4),
                                     "l"(src + k * TP + tid)
                                     : "memory");
                }
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        prefetch(0);
#pragma unroll 1
        for (uint32_t rd = 0; rd < R; ++rd) {
            const uint32_t slot = rd * Q + slot0;
            const uint32_t inner = inner0 + slot;
            const bool live = inner < p.n_inner;
            uint32_t* work = buf + slot * STR;
            uint32_t r[16];
            prefetch(rd + 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
            ntt_group_sync<TP, NT>(slot0);  // the words were copied by other threads of the polynomial
            // ---- pass 0: lift -> scale -> stages 0..3 ----
            {
#pragma unroll
                for (int k = 0; k < 16; ++k) {
                    uint32_t v = live ? work[k * TP + tid] : 0u;
                    bad |= v & ~pmask;
                    v &= pmask;
                    if (p.centered && v >= half_p) v = v - (pmask + 1u) + q;  // x - p, taken mod q
                    r[k] = shoup_mul(v, p.scale[t], p.scale_shoup[t], q);      // [0, 2q)
                }
                ntt_group_sync<TP, NT>(slot0);  // the slot is reused for the exchange below
                radix16_pass<TW_SMEM>(r, 0, 0, tw, tws, q);
            }
#pragma unroll
            for (uint32_t rho = 1; rho < PASSES; ++rho) {
                // elements of pass rho-1: idx = hi' * 2^(L-4(rho-1)) + k * 2^(L-4rho) + lo'; the padded index
                // i + i/16 is linear in k whenever k's stride is a multiple of 16
                {
                    const uint32_t lo_bits = L - 4 * rho;  // >= 4: bits of lo' = bits below k in the previous pass
                    const uint32_t lo = tid & ((1u << lo_bits) - 1u), hi = tid >> lo_bits;
                    uint32_t* w0 = work + ntt_pad((hi << (lo_bits + 4)) + lo);
#pragma unroll
                    for (int k = 0; k < 16; ++k) w0[k * ((1u << lo_bits) + (1u << (lo_bits - 4)))] = r[k];
                }
                ntt_group_sync<TP, NT>(slot0);
                const uint32_t lo_bits = L - 4 * rho - 4;
                const uint32_t lo = tid & ((1u << lo_bits) - 1u), hi = tid >> lo_bits;
                if (lo_bits >= 4) {
                    const uint32_t* r0 = work + ntt_pad((hi << (lo_bits + 4)) + lo);
#pragma unroll
                    for (int k = 0; k < 16; ++k) r[k] = r0[k * ((1u << lo_bits) + ((1u << lo_bits) >> 4))];
                } else {  // lo_bits == 0: idx = 16 hi + k, padded 17 hi + k
                    const uint32_t* r0 = work + hi * 17;
#pragma unroll
                    for (int k = 0; k < 16; ++k) r[k] = r0[k];
                }
                ntt_group_sync<TP, NT>(slot0);
                radix16_pass<TW_SMEM>(r, rho, hi, tw, tws, q);
            }
            // ---- normalise to [0, q) and stage in natural order: position pos = 16 hi + k holds
            // Y[bitrev(pos)], bitrev(pos) = bitrev4(k) * N/16 + bitrev(hi) ----
            {
                const uint32_t c0 = (L > 4) ? (__brev(tid) >> (32 - (L > 4 ? L - 4 : 1))) : 0u;
                uint32_t* s0 = work + ntt_pad_out(c0);
#pragma unroll
                for (int k = 0; k < 16; ++k) {
                    uint32_t v = r[k];
                    v = min(v, v - 2 * q);
                    v = min(v, v - q);
                    constexpr uint32_t kStep = N / 16 + N / 512;  // N/16 padded (a multiple of 32 for N = 4096)
                    const uint32_t kr = ((k & 1) << 3) | ((k & 2) << 1) | ((k & 4) >> 1) | ((k & 8) >> 3);
                    if constexpr (L == 12) s0[kr * kStep] = v;
                    else work[ntt_pad_out(c0 + kr * (N / 16))] = v;
                }
            }
        }
        __syncthreads();
        // ---- store: for each c, the P (live) polynomials' words are contiguous in the output ----
        {
            const uint32_t n_live = min(P, p.n_inner - inner0);
            uint32_t* dst = p.O + ((size_t)t * N * p.n_outer + outer) * p.n_inner + inner0;
            const size_t c_stride = (size_t)p.n_outer * p.n_inner;
            const bool vec = (P % 4 == 0) && n_live == P && (p.n_inner % 4 == 0) &&
                             ((reinterpret_cast<uintptr_t>(p.O) & 15) == 0);
            if (vec) {
                // one thread = one c and four neighbouring polynomials: a 16-byte store
                constexpr uint32_t QUADS = P / 4;
#pragma unroll 4
                for (uint32_t i = threadIdx.x; i < N * QUADS; i += NTT_THREADS) {
                    const uint32_t c = i / QUADS, s4 = (i % QUADS) * 4;
                    const uint32_t* src = buf + s4 * STR + ntt_pad_out(c);
                    const uint4 v = make_uint4(src[0], src[STR], src[2 * STR], src[3 * STR]);
                    *reinterpret_cast<uint4*>(dst + (size_t)c * c_stride + s4) = v;
                }
            } else {
                for (uint32_t i = threadIdx.x; i < N * P; i += NTT_THREADS) {
                    const uint32_t s = i % P, c = i / P;
                    if (s < n_live) dst[(size_t)c * c_stride + s] = buf[s * STR + ntt_pad_out(c)];
                }
            }
        }
        __syncthreads();
    }
    if (bad) *p.bad_input = 1u;
}

}  // namespace vipir
