// db_split.cuh -- offline re-layout of a u16 database into its two byte-limb planes.
//
// BASELINE.json configs[4]: "D 32768x32768 uint16 ... (split into 2 u8 limbs)".  The database of a PIR
// server is static and resident in GPU DRAM; like the hint it may be
// prepared once, offline.  This kernel writes  D_lo[r][k] = D[r][k] & 0xFF  and  D_hi[r][k] = D[r][k] >> 8
// as two rows x cols byte matrices, D_hi directly behind D_lo: the form gemm_i8_kernel<.., NL = 2>
// scans.  Pure data movement (one prmt pair per four elements); reads and writes 2*rows*cols bytes.
#pragma once
#include <cstdint>

namespace vipir {

// One thread handles 16 consecutive elements (two 128-bit loads, one 128-bit store per plane).
// n16 = rows*cols / 16 (cols is a multiple of 16, so a group never straddles a row... nor needs to:
// both layouts are dense, element e of the DB is byte e of each plane).
__global__ void __launch_bounds__(256) db_split_u16_kernel(const uint4* __restrict__ src, uint4* __restrict__ lo,
                                                           uint4* __restrict__ hi, uint64_t n16) {
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t g = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; g < n16; g += stride) {
        const uint4 a = __ldcs(src + 2 * g), b = __ldcs(src + 2 * g + 1);
        uint4 l, h;
        l.x = __byte_perm(a.x, a.y, 0x6420); h.x = __byte_perm(a.x, a.y, 0x7531);
        l.y = __byte_perm(a.z, a.w, 0x6420); h.y = __byte_perm(a.z, a.w, 0x7531);
        l.z = __byte_perm(b.x, b.y, 0x6420); h.z = __byte_perm(b.x, b.y, 0x7531);
        l.w = __byte_perm(b.z, b.w, 0x6420); h.w = __byte_perm(b.z, b.w, 0x7531);
        lo[g] = l;
        hi[g] = h;
    }
}

}  // namespace vipir
