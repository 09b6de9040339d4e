// naive.cuh -- test-only check kernel (regime VIPIR_REGIME_NAIVE): one thread per output
// word, straight u8/u16 x u32 multiply-accumulate on the INT32/INT64 ALUs.  It plays the
// role of the paper's "Base" INT32 DB GEMM without tensor cores (Fig. 7
// ablation); it is never selected by VIPIR_REGIME_AUTO.
#pragma once
#include <cstdint>

namespace vipir {

struct NaiveParams {
    uint64_t rows, cols;
    uint32_t batch, db_bits, n_moduli;
    uint32_t db_signed;  // db_bits == 8 only: elements are two's-complement int8
    uint32_t moduli[4];
};

__global__ void __launch_bounds__(128) naive_dbmul_kernel(const void* __restrict__ D, const uint32_t* __restrict__ Q,
                                                          uint32_t* __restrict__ A, NaiveParams p) {
    const uint64_t r = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t q = blockIdx.y;  // query vector index in [0, T*batch)
    if (r >= p.rows) return;
    const uint32_t t = q / p.batch;
    const uint32_t* qv = Q + (uint64_t)q * p.cols;
    uint64_t acc = 0;
    if (p.db_signed) {
        const int8_t* d = reinterpret_cast<const int8_t*>(D) + r * p.cols;
        if (p.n_moduli == 0) {
            // two's complement: wrapping accumulation is exact mod 2^32
            for (uint64_t k = 0; k < p.cols; ++k) acc += (uint64_t)((int64_t)d[k] * (int64_t)qv[k]);
            A[(uint64_t)q * p.rows + r] = (uint32_t)acc;
        } else {
            const int64_t m = p.moduli[t];
            int64_t sacc = 0;  // |term| < 2^39: reduce every 2^15 terms
            for (uint64_t k = 0; k < p.cols; ++k) {
                sacc += (int64_t)d[k] * (int64_t)qv[k];
                if ((k & 0x7FFF) == 0x7FFF) sacc %= m;
            }
            sacc %= m;
            if (sacc < 0) sacc += m;
            A[(uint64_t)q * p.rows + r] = (uint32_t)sacc;
        }
    } else if (p.n_moduli == 0) {
        // mod 2^32 divides 2^64: wrapping u64 accumulation is exact
        if (p.db_bits == 8) {
            const uint8_t* d = reinterpret_cast<const uint8_t*>(D) + r * p.cols;
            for (uint64_t k = 0; k < p.cols; ++k) acc += (uint64_t)d[k] * qv[k];
        } else {
            const uint16_t* d = reinterpret_cast<const uint16_t*>(D) + r * p.cols;
            for (uint64_t k = 0; k < p.cols; ++k) acc += (uint64_t)d[k] * qv[k];
        }
        A[(uint64_t)q * p.rows + r] = (uint32_t)acc;
    } else {
        const uint64_t m = p.moduli[t];
        // reduce every 2^15 terms: each term < 2^48, so acc < 2^63 + m
        for (uint64_t k = 0; k < p.cols; ++k) {
            const uint64_t d = (p.db_bits == 8) ? reinterpret_cast<const uint8_t*>(D)[r * p.cols + k]
                                                : reinterpret_cast<const uint16_t*>(D)[r * p.cols + k];
            acc += d * qv[k];
            if ((k & 0x7FFF) == 0x7FFF) acc %= m;
        }
        A[(uint64_t)q * p.rows + r] = (uint32_t)(acc % m);
    }
}

}  // namespace vipir
