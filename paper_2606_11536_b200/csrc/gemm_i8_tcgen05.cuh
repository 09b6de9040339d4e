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
//   warp 2   TMEM allocator; warps 2-3 copy finished units to final_out when the host call wants the result there;
//   warps 4-11 epilogue (two per TMEM lane quarter, taking alternate batches of 32 query vectors):
//            tcgen05.ld the accumulators of their lane quarter, recombine limbs
//            with shifts (wrap mod 2^32) or in u64 + Barrett (prime moduli), and store /
//            read-modify-write answer[q][row] (coalesced over rows).
// The K dimension is processed in chunks of <= 32768 bytes (256 k-steps): 255*255*32768 <
// 2^31, so the s32 accumulators hold the exact limb sums (reading R7); the
// accumulators are drained after every chunk.  With CG = 2 a pair of CTAs (one cluster of 2
// SMs) runs cta_group::2 MMAs: M = 256 rows per pair, each CTA stages its own 128 DB rows and
// HALF of the limb-plane tile, halving shared-memory fill and read traffic per SM.
//
// M sub-tiles (msub = 1, 2, 4): while the product is HBM-bound what limits it is the L2 -> SM
// fill (DB bytes + the limb tile re-read by every M tile), so a CTA keeps msub 128-row DB
// sub-tiles per k-atom against ONE limb-tile box: msub accumulators side by side in TMEM, the
// limb-plane traffic per DB byte divided by msub.
//
// Limb-plane u16 DB (NL = 2): a u16 DB that was de-interleaved once, offline,
// into its two byte matrices [D_lo ; D_hi] (vipir_db_split_u16) is scanned as the u8 matrix of 2*rows
// rows it then is: the two limb tiles of the same 128 rows are two of the CTA's M sub-tiles (msub is a
// multiple of 2), their accumulators sit side by side in TMEM, and the epilogue thread that owns the
// row adds them as  P_lo + 2^8 P_hi  before the one reduction.  8 int8 MACs per u16 x u32 product and
// 4 limb-plane columns per query vector instead of the byte view's 10 and 5.
//
// Work distribution.  A work item is (unit = (M tile, N tile), K chunk).  Groups (a CTA, or a
// CTA pair) take whole units round-robin for the full rounds -- so that the sibling N tiles of
// one M tile run at the same time on neighbouring groups and share the DB tile through L2 --
// and the units of the last, partial round are dealt out chunk by chunk in contiguous item
// ranges, which removes the wave-quantisation loss (e.g. 256 units on 74 pairs: 3.5 rounds
// instead of 4).  The leftover units may be cut into MORE chunks than the units of the full rounds
// (GemmParams.nc_left: the planner's choice where few chunks would deal out badly, e.g. one chunk per unit),
// which costs the extra accumulator drains only where they buy an even last round.
// A unit split between two groups is accumulated through the answer buffer
// (chunk 0 stores, later chunks add): the later group waits on a per-unit arrival counter in
// global memory before its first read-modify-write.  Group ids are tickets drawn from an atomic
// counter, a group only ever waits for lower tickets, and every group works through its
// producing items (the tail of its range) first, so the waits cannot deadlock whatever order the
// hardware starts the CTAs in -- nor when another kernel holds some SMs and part of the grid starts
// late: a ticket is drawn by a CTA that is already running, and a running CTA is never descheduled
// before it exits, so every lower ticket a group can wait for belongs to a group that is resident and
// making progress; the last group to finish resets the counters for the next launch.
#pragma once
#include <cstdint>
#include <cuda.h>
#include "ptx.cuh"

namespace vipir {

constexpr int GM_BM = 128;           // rows per CTA
constexpr int GM_BK = 128;           // bytes of K per stage (one 128B swizzle row)
constexpr int GM_UMMA_K = 32;        // bytes of K per tcgen05.mma.kind::i8
constexpr int GM_EPI_WARPS = 8;      // two per TMEM lane quarter (a warp reads the 32 lanes of quarter warp % 4)
constexpr int GM_THREADS = 32 * (4 + GM_EPI_WARPS);
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
    uint32_t k_begin;        // first k-atom of this launch's K range (0 unless the call is cut into K slices)
    uint32_t total_ksteps;   // k-atoms of this launch's K range (ceil(K' / 128) for the whole product)
    uint32_t ksteps_per_chunk;
    uint32_t n_chunks;
    uint32_t nc_left, kpc_left;  // units of the leftover round only: cut into nc_left chunks of kpc_left k-atoms instead
                             // (finer items to deal out; 0 = like every other unit)
    uint32_t katoms;         // k-atoms per pipeline stage (>= 1): one stage = katoms x (A box + B boxes)
    uint32_t atom_bytes;     // per CTA: 16 KiB of DB + this CTA's share of the limb tile, for one k-atom
    uint32_t stages;
    uint32_t stage_bytes;    // per CTA = katoms * atom_bytes
    uint32_t tmem_cols, acc_stages;
    uint32_t msub;           // 128-row DB sub-tiles per CTA and unit (1, 2 or 4): rows per unit = 128 * CG * msub / NL
    uint32_t collector;      // n_instr == 2: second N half reuses the A operand from the collector buffer
    uint32_t split;          // deal the last, partial round out chunk by chunk (1) or unit by unit (0)
    uint32_t n_groups;       // CTAs (CG = 1) or CTA pairs (CG = 2) launched
    uint32_t* sync;          // [0] ticket, [1] groups finished, [2 + i] epilogue-warp arrivals of leftover unit i
    uint32_t idesc;
    uint32_t ms_bits;        // fused modulus switch 2^32 -> 2^ms_bits of the answer (0 = off; q = 2^32 only)
    uint32_t db_signed;      // DB bytes are s8 (A format s8 in idesc): the s32 accumulators may be negative
    uint32_t n_moduli;
    uint32_t moduli[GM_MAX_MODULI];
    uint64_t barrett[GM_MAX_MODULI];  // floor(2^64 / p)
    uint32_t acc_in;         // 1: `answer` already holds the sum over the K range before k_begin (an earlier launch's)
    uint32_t* answer;        // [nq][rows]: running sums between K chunks, and the result unless final_out differs
    uint32_t* final_out;     // == answer, or where the result is wanted besides (mapped host memory): warps 2-3 of every
                             // CTA copy a unit's words there once its LAST chunk of this launch is in `answer`
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

// ---- work distribution (see the header comment) ------------------------------------------------
// Group g of G: units  r*G + g  for the full rounds r < n_units / G  (all chunks), then the item range
// [g*I/G, (g+1)*I/G) of the I = L*nc leftover items (L = n_units mod G units, unit-major), visited in
// the order  tail (chunks [0, c) of the range's last unit)  ->  whole units  ->  head (chunks
// [c0, c1) of the range's first unit, whose earlier chunks belong to group g-1 or before).
struct WorkPlan {
    uint32_t g, G, nc, nc_full, full_rounds, u_base;  // nc: chunks of a leftover unit; nc_full: of a unit of the full rounds
    uint32_t has_tail, tail_u, tail_c1;
    uint32_t mid0, mid1;
    uint32_t has_head, head_u, head_c0, head_c1;
};

__host__ __device__ __forceinline__ WorkPlan make_work_plan(uint32_t g, uint32_t G, uint32_t n_units, uint32_t nc,
                                                   uint32_t split, uint32_t nc_full = 0) {
    WorkPlan w;
    w.g = g; w.G = G; w.nc = nc; w.nc_full = nc_full ? nc_full : nc;
    w.full_rounds = n_units / G;
    w.u_base = w.full_rounds * G;
    const uint32_t L = n_units - w.u_base;
    if (!split) {  // leftover units whole, one per group
        w.has_head = w.has_tail = 0;
        w.head_u = w.head_c0 = w.head_c1 = w.tail_u = w.tail_c1 = 0;
        w.mid0 = w.u_base + (g < L ? g : L);
        w.mid1 = w.u_base + (g < L ? g + 1 : L);
        return w;
    }
    const uint64_t I = (uint64_t)L * nc;
    const uint32_t b = (uint32_t)((uint64_t)g * I / G), e = (uint32_t)((uint64_t)(g + 1) * I / G);
    const uint32_t ub = b / nc, cb = b % nc, ue = e / nc, ce = e % nc;
    w.has_head = (e > b && cb != 0) ? 1u : 0u;
    w.head_u = w.u_base + ub;
    w.head_c0 = cb;
    w.head_c1 = (ue == ub) ? ce : nc;
    const uint32_t m0 = cb ? ub + 1 : ub;
    w.mid0 = w.u_base + m0;
    w.mid1 = w.u_base + (ue > m0 ? ue : m0);
    w.has_tail = (e > b && ce != 0 && !(cb != 0 && ue == ub)) ? 1u : 0u;
    w.tail_u = w.u_base + ue;
    w.tail_c1 = ce;
    return w;
}

// f(unit, chunk, must_wait): must_wait marks the first item of a head segment -- the chunks before
// it were (or are being) accumulated into the answer by another group.
// (also instantiated with a host lambda by vipir_testing_work_items: silence the host-call-from-HD diagnostic)
#pragma nv_diag_suppress 20013
template <class F>
__host__ __device__ __forceinline__ void for_each_item(const WorkPlan& w, F&& f) {
    // four segments, one loop nest (a single copy of the caller's body)
#pragma unroll 1
    for (uint32_t seg = 0; seg < 4; ++seg) {
        uint32_t u_lo, u_hi, u_step = 1, c_lo = 0, c_hi = w.nc;
        if (seg == 0) {  // full rounds
            u_lo = w.g; u_hi = w.u_base; u_step = w.G; c_hi = w.nc_full;
        } else if (seg == 1) {  // tail of the leftover range: produces chunks another group continues
            u_lo = w.tail_u; u_hi = w.tail_u + w.has_tail; c_hi = w.tail_c1;
        } else if (seg == 2) {  // whole leftover units
            u_lo = w.mid0; u_hi = w.mid1;
        } else {  // head: continues a unit another group started
            u_lo = w.head_u; u_hi = w.head_u + w.has_head; c_lo = w.head_c0; c_hi = w.head_c1;
        }
#pragma unroll 1
        for (uint32_t u = u_lo; u < u_hi; u += u_step)
#pragma unroll 1
            for (uint32_t c = c_lo; c < c_hi; ++c) f(u, c, seg == 3 && c == c_lo);
    }
}

#pragma nv_diag_default 20013

// NL = byte-limb planes of the DB held as separate matrices (1: u8 DB or the byte view of a u16 DB;
// 2: limb-plane u16 DB, D_hi starting p.rows rows below D_lo in the tensor map).
template <int CG, int LC, bool PRIME, int NL = 1>
__global__ void __launch_bounds__(GM_THREADS, 1)
gemm_i8_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, GemmParams p) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)p.stages * p.stage_bytes);
    uint64_t* empty = full + p.stages;
    uint64_t* tmem_full = empty + p.stages;   // [2]
    uint64_t* tmem_empty = tmem_full + 2;     // [2]
    uint64_t* copy_full = tmem_empty + 2;     // [2]  finished units handed to the copier warps (final_out != answer)
    uint64_t* copy_empty = copy_full + 2;     // [2]
    uint32_t* tmem_ptr = reinterpret_cast<uint32_t*>(copy_empty + 2);
    uint32_t* ticket_ptr = tmem_ptr + 1;
    uint32_t* last_ptr = tmem_ptr + 2;
    uint32_t* copy_unit = tmem_ptr + 3;       // [2]
    const bool copier = p.final_out != p.answer;

    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t rank = (CG == 2) ? ptx::cluster_ctarank() : 0u;
    const uint32_t n_units = p.m_tiles * p.n_tiles;
    const uint32_t acc_cols = p.msub * p.bn;  // TMEM columns of one accumulator stage
    const uint32_t rsub = p.msub / NL;         // 128*CG-row blocks per unit
    static_assert(NL == 1 || (NL == 2 && LC == 4), "limb-plane DBs use the four plain query limb planes");

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tmA);
        ptx::prefetch_tmap(&tmB);
        // group id = ticket: a group only ever waits for groups that drew a lower ticket, i.e. that
        // are already running
        if (rank == 0) {
            const uint32_t t = atomicAdd(p.sync, 1u);
            *ticket_ptr = p.split ? t : ((CG == 2) ? ptx::cluster_id_x() : blockIdx.x);
        }
    }
    if (warp == 1 && lane == 0) {
        for (uint32_t s = 0; s < p.stages; ++s) {
            ptx::mbar_init(&full[s], 1);
            ptx::mbar_init(&empty[s], 1);
        }
        for (uint32_t a = 0; a < 2; ++a) {
            ptx::mbar_init(&tmem_full[a], 1);
            ptx::mbar_init(&tmem_empty[a], GM_EPI_WARPS * CG);  // one arrival per epilogue warp of every CTA
            ptx::mbar_init(&copy_full[a], GM_EPI_WARPS);        // this CTA's epilogue warps
            ptx::mbar_init(&copy_empty[a], 2);                  // this CTA's two copier warps
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
    // values read back from shared memory are the same in every lane: say so (shfl from lane 0), so
    // that the single-issuer loops below run on the uniform datapath instead of per-lane registers
    const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_ptr, 0);
    // the pair's ticket lives in the leader's shared memory (the leader outlives this read: the
    // teardown ends with a cluster barrier)
    const uint32_t ticket = __shfl_sync(
        0xffffffffu, (CG == 2 && rank == 1) ? ptx::ld_shared_cluster_u32(ticket_ptr, 0) : *ticket_ptr, 0);
    // chunks of a unit: n_chunks x ksteps_per_chunk k-atoms in the full rounds; the leftover round's units may be cut finer
    const uint32_t nc_left = p.nc_left ? p.nc_left : p.n_chunks;
    const uint32_t kpc_left = p.nc_left ? p.kpc_left : p.ksteps_per_chunk;
    const WorkPlan work = make_work_plan(ticket, p.n_groups, n_units, nc_left, p.split, p.n_chunks);

    if (warp == 0) {
        // ===== TMA producer: the whole warp runs the (warp-uniform) loop, one elected lane issues =====
        {
            uint32_t stage = 0, phase = 0;
            const uint32_t b_rows = p.ni_cols / CG;  // limb-plane rows this CTA stages per instruction
            const uint32_t b_bytes = b_rows * GM_BK;
            // the DB is streamed once (evict_first); with several N tiles the sibling tiles, which
            // run alongside on neighbouring clusters, re-read it from L2, so it stays evict_normal
            // (ncu: marking the last sibling evict_first raised DRAM reads from 5.6 to 8.0 GB on C4)
            const uint64_t hintA = (p.n_tiles == 1) ? ptx::kEvictFirst : ptx::kEvictNormal;
            for_each_item(work, [&](uint32_t u, uint32_t c, bool) {
                const uint32_t mt = u / p.n_tiles, nt = u % p.n_tiles;
                // sub-tile j of the unit = limb plane j % NL of rows [(mt*rsub + j/NL) * 128*CG, +128*CG);
                // this CTA's 128 of them
                auto sub_row = [&](uint32_t j) {
                    return (int32_t)((j % NL) * p.rows + ((uint64_t)(mt * rsub + j / NL) * CG + rank) * GM_BM);
                };
                const uint32_t kpc = (u < work.u_base) ? p.ksteps_per_chunk : kpc_left;
                const uint32_t ks_begin = c * kpc;
                const uint32_t ks_end = min(p.total_ksteps, ks_begin + kpc);
                // a stage never straddles a chunk: the last stage of a chunk may hold fewer atoms
                for (uint32_t ks0 = ks_begin; ks0 < ks_end; ks0 += p.katoms) {
                    const uint32_t na = min(p.katoms, ks_end - ks0);
                    ptx::mbar_wait(&empty[stage], phase ^ 1);
                    __syncwarp();
                    if (ptx::elect_one()) {
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
                        uint8_t* sB = sA + p.msub * GM_A_BYTES;
                        const int32_t k0 = (int32_t)((p.k_begin + ks0 + a) * GM_BK);
                        if constexpr (CG == 1) {
                            for (uint32_t j = 0; j < p.msub; ++j)
                                ptx::tma_load_2d(sA + j * GM_A_BYTES, &tmA, &full[stage], k0, sub_row(j), hintA);
                            for (uint32_t j = 0; j < p.n_instr; ++j)
                                ptx::tma_load_2d(sB + j * b_bytes, &tmB, &full[stage], k0,
                                                 (int32_t)(nt * p.bn + j * p.ni_cols), ptx::kEvictLast);
                        } else {
                            for (uint32_t j = 0; j < p.msub; ++j)
                                ptx::tma_load_2d_pair(sA + j * GM_A_BYTES, &tmA, bar, k0, sub_row(j), hintA);
                            for (uint32_t j = 0; j < p.n_instr; ++j)
                                ptx::tma_load_2d_pair(sB + j * b_bytes, &tmB, bar, k0,
                                                      (int32_t)(nt * p.bn + j * p.ni_cols + rank * b_rows),
                                                      ptx::kEvictLast);
                        }
                    }
                    }
                    __syncwarp();
                    if (++stage == p.stages) { stage = 0; phase ^= 1; }
                }
            });
        }
    } else if (warp == 1) {
        // ===== MMA issuer (leader CTA of the pair only) =====
        // the whole warp runs the (warp-uniform) loop; one elected lane -- the same one every time, so
        // that tcgen05.commit tracks the MMAs it issued -- issues
        if (rank == 0) {
            uint32_t stage = 0, phase = 0, acc_it = 0;
            const uint32_t b_bytes = (p.ni_cols / CG) * GM_BK;
            for_each_item(work, [&](uint32_t u, uint32_t c, bool) {
                const uint32_t as = acc_it % p.acc_stages;
                const uint32_t aphase = (acc_it / p.acc_stages) & 1;
                ++acc_it;
                if constexpr (CG == 2) ptx::mbar_wait_cluster(&tmem_empty[as], aphase ^ 1);
                else ptx::mbar_wait(&tmem_empty[as], aphase ^ 1);
                ptx::tc_fence_after();
                const uint32_t kpc = (u < work.u_base) ? p.ksteps_per_chunk : kpc_left;
                const uint32_t ks_begin = c * kpc;
                const uint32_t ks_end = min(p.total_ksteps, ks_begin + kpc);
                const uint32_t tacc = tmem_base + as * acc_cols;
                for (uint32_t ks0 = ks_begin; ks0 < ks_end; ks0 += p.katoms) {
                    const uint32_t na = min(p.katoms, ks_end - ks0);
                    ptx::mbar_wait(&full[stage], phase);
                    ptx::tc_fence_after();
                    __syncwarp();
                    if (ptx::elect_one()) {
                    const uint32_t sbase = ptx::smem_u32(smem + (size_t)stage * p.stage_bytes);
                    for (uint32_t a = 0; a < na; ++a) {
                        const uint32_t sA = sbase + a * p.atom_bytes;
                        const uint32_t sB = sA + p.msub * GM_A_BYTES;
                        const uint32_t accumulate = (ks0 + a > ks_begin) ? 1u : 0u;
                        for (uint32_t m = 0; m < p.msub; ++m) {
                            const uint64_t dA = make_smem_desc(sA + m * GM_A_BYTES);
                            if (p.n_instr == 2 && p.collector) {
                                // two N halves against the same DB slice: issue them back to back and let
                                // the second take A from the collector instead of shared memory
                                const uint64_t dB0 = make_smem_desc(sB), dB1 = make_smem_desc(sB + b_bytes);
#pragma unroll
                                for (uint32_t kk = 0; kk < GM_BK / GM_UMMA_K; ++kk) {
                                    const uint64_t koff = (uint64_t)((kk * GM_UMMA_K) >> 4);
                                    const uint32_t acc = (accumulate || kk > 0) ? 1u : 0u;
                                    ptx::mma_i8_collect<CG, 1>(tacc + m * p.bn, dA + koff, dB0 + koff, p.idesc, acc);
                                    ptx::mma_i8_collect<CG, 2>(tacc + m * p.bn + p.ni_cols, dA + koff, dB1 + koff, p.idesc,
                                                               acc);
                                }
                                continue;
                            }
                            for (uint32_t j = 0; j < p.n_instr; ++j) {
                                const uint64_t dB = make_smem_desc(sB + j * b_bytes);
#pragma unroll
                                for (uint32_t kk = 0; kk < GM_BK / GM_UMMA_K; ++kk) {
                                    // advancing K inside the swizzle atom = adding the byte offset >> 4
                                    const uint64_t koff = (uint64_t)((kk * GM_UMMA_K) >> 4);
                                    ptx::mma_i8<CG>(tacc + m * p.bn + j * p.ni_cols, dA + koff, dB + koff, p.idesc,
                                                    (accumulate || kk > 0) ? 1u : 0u);
                                }
                            }
                        }
                    }
                    // release the smem slot once these MMAs have read it
                    if constexpr (CG == 2) ptx::tc_commit_pair(&empty[stage], 3);
                    else ptx::tc_commit(&empty[stage]);
                    // accumulators of this chunk complete -> epilogue
                    if (ks0 + na >= ks_end) {
                        if constexpr (CG == 2) ptx::tc_commit_pair(&tmem_full[as], 3);
                        else ptx::tc_commit(&tmem_full[as]);
                    }
                    }
                    __syncwarp();
                    if (++stage == p.stages) { stage = 0; phase ^= 1; }
                }
            });
        }
    } else if (copier && warp < 4) {
        // ===== warps 2-3, only when the result is wanted in final_out (the host call's mapped answer buffer): move every
        // finished unit's words of this CTA from `answer` (device memory, just written: L2) to final_out.  The epilogue
        // warps cannot store there themselves without holding the accumulators for as long as the host link takes
        // (one unit's 64 KB per CTA is ~185 us of a saturated link, the unit's products ~210 us): measured 0.4-0.5 ms per
        // configs[3] call.  Here the stores of unit u run beside the products of unit u + 1. =====
        const uint32_t cw = warp - 2;
        const bool vec = (p.rows % 4 == 0) && ((reinterpret_cast<uintptr_t>(p.answer) | reinterpret_cast<uintptr_t>(p.final_out)) & 15) == 0;
        uint32_t n_final = 0;
        for_each_item(work, [&](uint32_t u_item, uint32_t c, bool) {
            if (c + 1 != ((u_item < work.u_base) ? p.n_chunks : nc_left)) return;
            const uint32_t slot = n_final & 1, ph = (n_final >> 1) & 1;
            ++n_final;
            ptx::mbar_wait(&copy_full[slot], ph);
            const uint32_t u = *reinterpret_cast<volatile uint32_t*>(&copy_unit[slot]);
            const uint32_t mt = u / p.n_tiles, nt = u % p.n_tiles;
            const uint32_t q_lo = nt * p.qt, q_hi = min(p.nq, q_lo + p.qt);
            for (uint32_t m = 0; m < rsub; ++m) {
                const uint64_t row0 = (uint64_t)((mt * rsub + m) * CG + rank) * GM_BM;
                if (row0 >= p.rows) break;
                const uint32_t n_rows = (uint32_t)min((uint64_t)GM_BM, p.rows - row0);
                if (vec) {  // a warp moves one query vector's 128 rows (512 bytes) per step, eight steps in flight
                    constexpr uint32_t kU = 8;
                    for (uint32_t q0 = q_lo + cw * kU; q0 < q_hi; q0 += 2 * kU) {
                        uint4 v[kU];
#pragma unroll
                        for (uint32_t j = 0; j < kU; ++j)
                            if (q0 + j < q_hi && lane * 4 < n_rows)
                                v[j] = __ldcg(reinterpret_cast<const uint4*>(p.answer + (uint64_t)(q0 + j) * p.rows + row0) + lane);
#pragma unroll
                        for (uint32_t j = 0; j < kU; ++j)
                            if (q0 + j < q_hi && lane * 4 < n_rows)
                                reinterpret_cast<uint4*>(p.final_out + (uint64_t)(q0 + j) * p.rows + row0)[lane] = v[j];
                    }
                } else {
                    for (uint32_t q = q_lo + cw; q < q_hi; q += 2)
                        for (uint32_t r = lane; r < n_rows; r += 32)
                            p.final_out[(uint64_t)q * p.rows + row0 + r] = __ldcg(p.answer + (uint64_t)q * p.rows + row0 + r);
                }
            }
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(&copy_empty[slot]);
        });
    }
    if (warp >= 4) {
        // ===== epilogue warps: lane quarter = warp % 4; the two warps of a quarter take alternate batches of kPf steps =====
        const uint32_t quarter = warp & 3;
        const uint32_t half = (warp - 4) >> 2;
        uint32_t acc_it = 0, n_final = 0;
        for_each_item(work, [&](uint32_t u, uint32_t c, bool must_wait) {
            const uint32_t mt = u / p.n_tiles, nt = u % p.n_tiles;
            const uint32_t as = acc_it % p.acc_stages;
            const uint32_t aphase = (acc_it / p.acc_stages) & 1;
            ++acc_it;
            ptx::mbar_wait(&tmem_full[as], aphase);
            ptx::tc_fence_after();
            if (must_wait) {
                // chunks [0, c) of this unit belong to another group: all of its (GM_EPI_WARPS * CG) epilogue
                // warps must have stored them before this read-modify-write (see "Work distribution")
                const uint32_t* cnt = p.sync + 2 + (u - work.u_base);
                const uint32_t want = c * GM_EPI_WARPS * CG;
                const long long t0 = clock64();
                while (ptx::ld_acquire_gpu(cnt) < want) {
                    // a bound far above any legitimate wait: the longest one is a single unit cut into 65536 chunks
                    // (rows <= 128, K = 2^31 - 16: tests/test_max_sizes_gpu.py), whose chunks are accumulated strictly
                    // in order, group after group -- 7-11 s on a B200, which the former ~11 s bound cut short on some runs
                    if (clock64() - t0 > (1ll << 38)) __trap();  // ~2.4 min at 1.9 GHz: never in a correct run
                }
            }
            // later chunks add to what chunk 0 stored: a fire-and-forget red.add for q = 2^32; for
            // primes the old words are fetched eight steps (32 query vectors) at a time so that
            // one global-load latency is paid per batch, not per step
            // with the fused modulus switch (q = 2^32 only) the LAST chunk needs the running sum back
            // to round it: same batched prefetch, once per tile
            constexpr uint32_t kPf = 8;
            const bool first = c == 0 && !p.acc_in;   // nothing accumulated yet: plain store
            const bool last = c + 1 == ((u < work.u_base) ? p.n_chunks : nc_left);
            const bool ms_final = !PRIME && p.ms_bits != 0 && last;
            const bool need_old = !first && (PRIME || ms_final);
            // every chunk lands in `answer`; when the result is wanted elsewhere (final_out: the host call's mapped
            // answer) the CTA's copier warps move a unit there once its last chunk is in (below)
            uint32_t* const obase = p.answer;
            for (uint32_t m = 0; m < rsub; ++m) {
                const uint64_t row = (uint64_t)((mt * rsub + m) * CG + rank) * GM_BM + quarter * 32 + lane;
                const bool row_ok = row < p.rows;
                const uint32_t tacc = tmem_base + ((quarter * 32) << 16) + as * acc_cols + m * NL * p.bn;
                for (uint32_t g0 = half * kPf; g0 < p.qt / 4; g0 += 2 * kPf) {
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
                        uint32_t w[NL == 2 ? 4 * LC : 1];  // the D_hi sub-tile's sums for the same row
                        if constexpr (NL == 2) ptx::tmem_ld16(tacc + p.bn + g * (4 * LC), w);
                        ptx::tmem_ld_wait();
                        if constexpr (PRIME) {
                            // the four reductions computed unconditionally, so that the compiler interleaves their
                            // multiply chains; only the stores are guarded (a tile's tail columns reduce garbage that
                            // is never stored: the modulus index is clamped)
                            uint32_t val[4];
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                const uint32_t q = nt * p.qt + g * 4 + i;
                                const uint32_t t = min(q / p.batch, p.n_moduli - 1u);
                                const uint32_t pm = p.moduli[t];
                                if constexpr (NL == 2) {
                                    // unsigned; each sum < 2^31, so x < 2^63.1
                                    uint64_t x = 0;
#pragma unroll
                                    for (int s = 0; s < LC; ++s)
                                        x += ((uint64_t)v[i * LC + s] + ((uint64_t)w[i * LC + s] << 8)) << (8 * s);
                                    val[i] = barrett_u64(x, pm, p.barrett[t]);
                                } else if constexpr (LC == 4) {
                                    // every |P_s| < 2^31 (R7), so the s32 reading is exact for u8 and s8
                                    // DBs alike and |x| < 2^56; a negative x reduces as p - (|x| mod p)
                                    int64_t x = 0;
#pragma unroll
                                    for (int s = 0; s < LC; ++s) x += (int64_t)(int32_t)v[i * LC + s] << (8 * s);
                                    const bool neg = x < 0;
                                    uint32_t r = barrett_u64((uint64_t)(neg ? -x : x), pm, p.barrett[t]);
                                    if (neg && r != 0) r = pm - r;
                                    val[i] = r;
                                } else {
                                    uint64_t x = 0;  // u16 DB (never signed): up to 2^63 * 1.004
#pragma unroll
                                    for (int s = 0; s < LC; ++s) x += (uint64_t)v[i * LC + s] << (8 * s);
                                    val[i] = barrett_u64(x, pm, p.barrett[t]);
                                }
                                if (!first) {
                                    val[i] += old[gg * 4 + i];
                                    if (val[i] >= pm) val[i] -= pm;
                                }
                            }
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                const uint32_t q = nt * p.qt + g * 4 + i;
                                if (q < p.nq && row_ok) obase[(uint64_t)q * p.rows + row] = val[i];
                            }
                        } else {
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const uint32_t q = nt * p.qt + g * 4 + i;
                            if (q < p.nq && row_ok) {
                                uint32_t* dst = obase + (uint64_t)q * p.rows + row;
                                // shifts, wrap mod 2^32 (an s = 4 column would vanish)
                                uint32_t val =
                                    v[i * LC] + (v[i * LC + 1] << 8) + (v[i * LC + 2] << 16) + (v[i * LC + 3] << 24);
                                if constexpr (NL == 2)  // D = D_lo + 2^8 D_hi; the 2^32 term of w[3] vanishes
                                    val += (w[i * LC] << 8) + (w[i * LC + 1] << 16) + (w[i * LC + 2] << 24);
                                if (ms_final) {
                                    if (!first) val += old[gg * 4 + i];
                                    *dst = modswitch_word(val, p.ms_bits);
                                } else if (first) {
                                    *dst = val;
                                } else {
                                    asm volatile("red.global.add.u32 [%0], %1;" ::"l"(dst), "r"(val) : "memory");
                                }
                            }
                        }
                        }
                    }
                }
            }
            // accumulator stage drained
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                if constexpr (CG == 2) ptx::mbar_arrive_cluster_relaxed(&tmem_empty[as], 0);
                else ptx::mbar_arrive(&tmem_empty[as]);
            }
            // this lane's answer words, before the arrivals below: for the group that continues a leftover unit,
            // and for the copier warps that move a finished unit to final_out
            if (u >= work.u_base || (copier && last)) __threadfence();
            __syncwarp();
            if (copier && last) {
                // hand the finished unit to this CTA's copier warps: a ring of two entries, the n-th finished unit of
                // this CTA in entry n % 2 (the copiers walk the same work items and count the same way)
                const uint32_t slot = n_final & 1, ph = (n_final >> 1) & 1;
                ++n_final;
                ptx::mbar_wait(&copy_empty[slot], ph ^ 1);
                if (lane == 0) {
                    if (warp == 4) *reinterpret_cast<volatile uint32_t*>(&copy_unit[slot]) = u;
                    ptx::mbar_arrive(&copy_full[slot]);  // release: the unit id (warp 4) and the fence above
                }
            }
            // units of the leftover round may be shared with another group: count this warp in
            if (lane == 0 && u >= work.u_base) ptx::red_release_gpu_add(p.sync + 2 + (u - work.u_base), 1u);
        });
    }

    // ===== teardown =====
    ptx::tc_fence_before();
    if constexpr (CG == 2) ptx::cluster_sync(); else __syncthreads();
    if (warp == 2) {
        ptx::tc_fence_after();
        ptx::tmem_dealloc<CG>(tmem_base, p.tmem_cols);
    }
    // the last group to finish leaves the ticket and the arrival counters at zero for the next launch
    if (rank == 0) {
        if (threadIdx.x == 0) {
            __threadfence();
            *last_ptr = (atomicAdd(p.sync + 1, 1u) == p.n_groups - 1) ? 1u : 0u;
        }
        __syncthreads();
        if (*last_ptr) {
            __threadfence();
            for (uint32_t i = threadIdx.x; i < 2 + p.n_groups; i += GM_THREADS) p.sync[i] = 0u;
        }
    }
}

}  // namespace vipir
