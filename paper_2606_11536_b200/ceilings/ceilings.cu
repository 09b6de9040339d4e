// ceilings.cu -- measurement aids for bench.py: what this part can do at best on the unit a kernel of
// libvipir is bound by, measured live in the same run as the kernel ("the bench must add
// a pure tcgen05.mma.kind::i8 loop ... ceiling").  Not product code: nothing in csrc/ or vipir.py uses
// this library, and it computes nothing of the method -- operands are pseudo-random bytes that never
// leave the SM.  C ABI, loaded by ceilings/__init__.py.
//
//   vipir_ceiling_mma_i8       every SM pair issues back-to-back tcgen05.mma.cta_group::2.kind::i8
//                              (M = 256, N = 256, K = 32; u8 x u8 -> s32 in TMEM) on operands resident in
//                              shared memory: no TMA, no epilogue, no HBM traffic -- the int8 tensor pipe
//                              alone (burst: one launch after idle; sustained: launches back to back
//                              under the power cap, which bench.py does)
//   vipir_ceiling_butterflies  Harvey/Shoup radix-2 butterflies on registers only (no shared memory, no
//                              global traffic): the INT32 ALU + multiply pipes alone, the ceiling of
//                              ntt_lift_kernel's butterfly passes
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "../csrc/gemm_i8_tcgen05.cuh"  // make_smem_desc
#include "../csrc/ntt_lift.cuh"         // the butterfly itself (so that the ceiling times the same instruction mix)
#include "../csrc/ptx.cuh"

namespace {

using namespace vipir;

constexpr int CL_THREADS = 128;
constexpr uint32_t CL_OP_BYTES = 128 * 128;  // one 128-row x 128-byte K-major swizzled operand tile

__device__ __forceinline__ uint32_t mix32(uint32_t x) {
    x ^= x >> 16; x *= 0x7FEB352Du; x ^= x >> 15; x *= 0x846CA68Bu; x ^= x >> 16;
    return x;
}

// cluster of 2: rank 0 issues, both CTAs hold their half of the operands (A: own 128 rows; B: half of N)
__global__ void __launch_bounds__(CL_THREADS, 1) mma_i8_ceiling_kernel(uint32_t iters, uint32_t seed) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* sA = smem;
    uint8_t* sB = smem + CL_OP_BYTES;
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + 2 * CL_OP_BYTES);
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(bar + 1);
    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t rank = ptx::cluster_ctarank();

    // pseudo-random operand bytes: data toggling is part of what the power cap sees
    for (uint32_t i = threadIdx.x; i < 2 * CL_OP_BYTES / 4; i += CL_THREADS)
        reinterpret_cast<uint32_t*>(smem)[i] = mix32(seed + blockIdx.x * 0x9E3779B9u + i);
    ptx::fence_proxy_async();
    if (threadIdx.x == 0) {
        ptx::mbar_init(bar, 1);
        ptx::fence_barrier_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc<2>(tmem_ptr, 512);
        ptx::tmem_relinquish<2>();
    }
    ptx::tc_fence_before();
    ptx::cluster_sync();
    ptx::tc_fence_after();
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_ptr, 0);

    if (rank == 0 && warp == 0) {
        const uint32_t idesc = (2u << 4) | ((256u >> 3) << 17) | ((256u >> 4) << 24);  // D = s32, A = B = u8, N 256, M 256
        const uint64_t dA = make_smem_desc(ptx::smem_u32(sA)), dB = make_smem_desc(ptx::smem_u32(sB));
        for (uint32_t it = 0; it < iters; ++it) {
            if (ptx::elect_one()) {
#pragma unroll
                for (uint32_t kk = 0; kk < 4; ++kk) {
                    const uint64_t koff = (uint64_t)((kk * 32) >> 4);
                    // two accumulators in turn (512 TMEM columns), as a double-buffered kernel has
                    ptx::mma_i8<2>(tmem_base + (it & 1) * 256, dA + koff, dB + koff, idesc, (it > 1 || kk > 0) ? 1u : 0u);
                }
            }
            __syncwarp();
        }
        if (ptx::elect_one()) ptx::tc_commit_pair(bar, 3);
        __syncwarp();
    }
    ptx::mbar_wait(bar, 0);
    ptx::tc_fence_after();
    ptx::tc_fence_before();
    ptx::cluster_sync();
    if (warp == 1) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc<2>(tmem_base, 512);
    }
}

// 16 values per thread, `iters` rounds of the four radix-2 stages of one radix-16 pass (32 butterflies a
// round), twiddles in registers.
__global__ void __launch_bounds__(512, 1) butterfly_ceiling_kernel(uint32_t iters, uint32_t q, uint32_t w, uint32_t ws,
                                                                    uint32_t* sink) {
    uint32_t v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = mix32(threadIdx.x * 16 + i + blockIdx.x * 8192) % q;
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            const int h = 8 >> s;
#pragma unroll
            for (int i = 0; i < 16; ++i)
                if ((i & h) == 0) harvey_butterfly(v[i], v[i + h], w, ws, q);
        }
    }
    uint32_t acc = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) acc ^= v[i];
    if (acc == 0xFFFFFFFFu && sink) *sink = acc;  // never (values stay below 4q < 2^32 - 1): keeps the work alive
}

}  // namespace

extern "C" {

// Enqueue `iters` x 4 MMAs (M 256 x N 256 x K 32) on every SM pair.  int8 ops = pairs * iters * 4 * 2*256*256*32.
int vipir_ceiling_mma_i8(uint32_t iters, uint32_t* pairs_out, void* stream) {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 2;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 2;
    const uint32_t pairs = (uint32_t)sms / 2;
    if (pairs_out) *pairs_out = pairs;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(pairs * 2);
    cfg.blockDim = dim3(CL_THREADS);
    cfg.dynamicSmemBytes = 2 * CL_OP_BYTES + 1024 + 64;
    cfg.stream = static_cast<cudaStream_t>(stream);
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, mma_i8_ceiling_kernel, iters, 12345u) == cudaSuccess ? 0 : 2;
}

// Enqueue `iters` x 32 butterflies per thread on blocks x 512 threads (one CTA per SM).
int vipir_ceiling_butterflies(uint32_t iters, uint32_t q, uint32_t* blocks_out, void* stream) {
    int dev = 0, sms = 0;
    if (q < 3 || q >= (1u << 30)) return 1;
    if (cudaGetDevice(&dev) != cudaSuccess) return 2;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 2;
    if (blocks_out) *blocks_out = (uint32_t)sms;
    const uint32_t w = 3 % q, ws = (uint32_t)(((uint64_t)w << 32) / q);
    butterfly_ceiling_kernel<<<sms, 512, 0, static_cast<cudaStream_t>(stream)>>>(iters, q, w, ws, nullptr);
    return cudaGetLastError() == cudaSuccess ? 0 : 2;
}

}  // extern "C"
