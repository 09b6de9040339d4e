// ntt_host.cuh -- host side (plan, twiddle tables, dispatch, C ABI) of the lift + forward NTT
// (include/vipir.h "vipir_ntt_*"; kernel in ntt_lift.cuh).  Textually included at the end of
// vipir_api.cu: it uses that file's helpers (CK, g_cuda_err, kMaxSmem).
#pragma once
#include <vector>
#include "ntt_lift.cuh"

struct vipir_ntt_plan {
    uint32_t T, log2n, N, p_bits, centered;
    uint32_t moduli[VIPIR_MAX_MODULI], scale[VIPIR_MAX_MODULI], scale_shoup[VIPIR_MAX_MODULI];
    int num_sms;
    int device;            // the device current at plan time: every call must come with it current
    uint32_t* d_twiddles;  // [T][2][N]
    uint32_t* d_bad;       // device flag: an input word >= 2^p_bits was seen
};

namespace {

uint32_t ntt_mulmod(uint32_t a, uint32_t b, uint32_t q) { return (uint32_t)(((uint64_t)a * b) % q); }
uint32_t ntt_powmod(uint32_t b, uint64_t e, uint32_t q) {
    uint32_t r = 1 % q;
    for (; e; e >>= 1, b = ntt_mulmod(b, b, q))
        if (e & 1) r = ntt_mulmod(r, b, q);
    return r;
}
uint32_t ntt_shoup(uint32_t w, uint32_t q) { return (uint32_t)(((uint64_t)w << 32) / q); }
uint32_t ntt_bitrev(uint32_t x, uint32_t bits) {
    uint32_t r = 0;
    for (uint32_t i = 0; i < bits; ++i) r |= ((x >> i) & 1u) << (bits - 1 - i);
    return r;
}

// 512 threads, twiddle tables in shared memory.  N = 4096: two polynomials in flight, P = 8 per iteration
// (172 KB: one CTA per SM).  Measured alternative: 256-thread CTAs with P = 4 and
// the twiddles read through L1, three CTAs per SM -- 1.5x slower for G, 2.3x slower for H (twiddle loads
// from L1 instead of shared memory; 16-byte instead of 32-byte output runs).
template <int L>
int launch_ntt(vipir_ntt_plan* p, const vipir::NttParams& np, cudaStream_t st) {
    constexpr bool BIG = (L == 12);
    constexpr int NT = 512, R = BIG ? 4 : 1, MINB = 1;
    constexpr bool TW_SMEM = true;
    constexpr uint32_t N = 1u << L, TP = N / 16, Q = NT / TP, P = Q * R;
    constexpr uint32_t STR = N + N / 16 + 4;
    const uint32_t smem = ((TW_SMEM ? 2 * N : 0) + P * STR) * sizeof(uint32_t);
    auto kern = vipir::ntt_lift_kernel<L, NT, R, TW_SMEM, MINB>;
    static thread_local uint64_t attr_set = 0;  // bit d: done on device d
    if (attr_needed(attr_set)) {
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem));
    }
    const uint64_t groups = (uint64_t)np.n_outer * ((np.n_inner + P - 1) / P);
    const uint64_t cap = (uint64_t)p->num_sms * (BIG ? 1 : 4);
    const uint32_t gx = (uint32_t)(groups < cap ? groups : cap);
    kern<<<dim3(gx, p->T), NT, smem, st>>>(np);
    CK(cudaGetLastError());
    return VIPIR_OK;
}

}  // namespace

extern "C" {

int vipir_ntt_plan_create(vipir_ntt_plan** out, uint32_t T, uint32_t log2n, const uint32_t* moduli, const uint32_t* psi,
                          const uint32_t* scale, uint32_t p_bits, uint32_t centered) {
    if (!out) return VIPIR_ERR_INVALID_ARG;
    *out = nullptr;
    if (!moduli || !psi || !scale || T == 0 || T > VIPIR_MAX_MODULI || centered > 1) return VIPIR_ERR_INVALID_ARG;
    if (p_bits < 1 || p_bits > 29) return VIPIR_ERR_INVALID_ARG;
    if (log2n != 4 && log2n != 8 && log2n != 12) return VIPIR_ERR_UNSUPPORTED;
    const uint32_t N = 1u << log2n;
    for (uint32_t t = 0; t < T; ++t) {
        const uint32_t q = moduli[t];
        if (q <= (1u << p_bits) || q >= (1u << 30)) return VIPIR_ERR_INVALID_ARG;
        // psi must be a primitive 2N-th root of unity: psi^N = -1 (PAPER.md:578-582 makes one exist)
        if (ntt_powmod(psi[t] % q, N, q) != q - 1) return VIPIR_ERR_INVALID_ARG;
    }
    int dev = 0;
    CK(cudaGetDevice(&dev));
    int major = 0, minor = 0, sms = 0;
    CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    CK(cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10 || minor != 0) return VIPIR_ERR_ARCH;

    vipir_ntt_plan* p = new (std::nothrow) vipir_ntt_plan;
    if (!p) return VIPIR_ERR_ALLOC;
    memset(p, 0, sizeof *p);
    p->T = T;
    p->log2n = log2n;
    p->N = N;
    p->p_bits = p_bits;
    p->centered = centered;
    p->num_sms = sms;
    p->device = dev;
    std::vector<uint32_t> tab((size_t)T * 2 * N);
    for (uint32_t t = 0; t < T; ++t) {
        const uint32_t q = moduli[t];
        p->moduli[t] = q;
        p->scale[t] = scale[t] % q;
        p->scale_shoup[t] = ntt_shoup(p->scale[t], q);
        // w[i] = psi^bitrev(i): powers in natural order first, then scattered
        std::vector<uint32_t> pw(N);
        pw[0] = 1;
        for (uint32_t i = 1; i < N; ++i) pw[i] = ntt_mulmod(pw[i - 1], psi[t] % q, q);
        uint32_t* w = tab.data() + (size_t)t * 2 * N;
        for (uint32_t i = 0; i < N; ++i) {
            w[i] = pw[ntt_bitrev(i, log2n)];
            w[N + i] = ntt_shoup(w[i], q);
        }
    }
    if (cudaMalloc(&p->d_twiddles, tab.size() * 4) != cudaSuccess || cudaMalloc(&p->d_bad, 4) != cudaSuccess) {
        cudaGetLastError();
        vipir_ntt_destroy(p);
        return VIPIR_ERR_ALLOC;
    }
    if (cudaMemcpy(p->d_twiddles, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemset(p->d_bad, 0, 4) != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) {
        snprintf(g_cuda_err, sizeof g_cuda_err, "%s", cudaGetErrorString(cudaGetLastError()));
        vipir_ntt_destroy(p);
        return VIPIR_ERR_CUDA;
    }
    *out = p;
    return VIPIR_OK;
}

int vipir_ntt_lift(vipir_ntt_plan* p, const uint32_t* d_X, uint32_t n_a, uint32_t M, uint32_t out_layout, uint32_t* d_O,
                   void* cuda_stream) {
    if (!p || !d_X || !d_O || n_a == 0 || M == 0 || out_layout > 1) return VIPIR_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_X) & 3) || (reinterpret_cast<uintptr_t>(d_O) & 3)) return VIPIR_ERR_INVALID_ARG;
    if ((uint64_t)n_a * M >= (1ull << 31)) return VIPIR_ERR_UNSUPPORTED;
    if (!on_device(p->device)) return VIPIR_ERR_INVALID_ARG;
    vipir::NttParams np{};
    np.T = p->T;
    if (out_layout == VIPIR_NTT_LAYOUT_G) {  // O[t][c][a][m]
        np.n_outer = n_a; np.n_inner = M; np.in_stride_outer = M; np.in_stride_inner = 1;
    } else {                                 // O[t][c][m][a]
        np.n_outer = M; np.n_inner = n_a; np.in_stride_outer = 1; np.in_stride_inner = M;
    }
    np.p_bits = p->p_bits;
    np.centered = p->centered;
    for (uint32_t t = 0; t < p->T; ++t) {
        np.moduli[t] = p->moduli[t];
        np.scale[t] = p->scale[t];
        np.scale_shoup[t] = p->scale_shoup[t];
    }
    np.twiddles = p->d_twiddles;
    np.X = d_X;
    np.O = d_O;
    np.bad_input = p->d_bad;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    switch (p->log2n) {
        case 4: return launch_ntt<4>(p, np, st);
        case 8: return launch_ntt<8>(p, np, st);
        default: return launch_ntt<12>(p, np, st);
    }
}

int vipir_ntt_bad_input(vipir_ntt_plan* p, uint32_t* seen) {
    if (!p || !seen) return VIPIR_ERR_INVALID_ARG;
    if (!on_device(p->device)) return VIPIR_ERR_INVALID_ARG;
    // the flag is written by kernels on the caller's streams (possibly non-blocking ones, which the legacy
    // stream does not order against): wait for all of them before reading and clearing it
    CK(cudaDeviceSynchronize());
    CK(cudaMemcpy(seen, p->d_bad, 4, cudaMemcpyDeviceToHost));
    CK(cudaMemset(p->d_bad, 0, 4));
    CK(cudaDeviceSynchronize());
    return VIPIR_OK;
}

void vipir_ntt_destroy(vipir_ntt_plan* p) {
    if (!p) return;
    if (p->d_twiddles) cudaFree(p->d_twiddles);
    if (p->d_bad) cudaFree(p->d_bad);
    delete p;
}

}  // extern "C"
