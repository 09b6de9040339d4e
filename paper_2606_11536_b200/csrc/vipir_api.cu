// vipir_api.cu -- host side of libvipir: plan (step a0), dispatch, C ABI (include/vipir.h).
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include <cuda.h>
#include <cuda_runtime.h>

#include "../../include/vipir.h"
#include "../../include/vipir_testing.h"
#include "db_split.cuh"
#include "gemm_i8_tcgen05.cuh"
#include "gemv_b1.cuh"
#include "naive.cuh"
#include "split_limbs.cuh"

namespace {

thread_local char g_cuda_err[256] = "";

int cuda_fail(cudaError_t e, const char* where) {
    snprintf(g_cuda_err, sizeof g_cuda_err, "%s: %s", where, cudaGetErrorString(e));
    return VIPIR_ERR_CUDA;
}
#define CK(call)                                                   \
    do {                                                           \
        cudaError_t e__ = (call);                                  \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call);      \
    } while (0)

// the opt-in shared-memory attribute of a kernel is per device: true the first time the calling thread
// asks on the current device
bool attr_needed(uint64_t& done_mask) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return true;
    const uint64_t bit = 1ull << (dev & 63);
    if (done_mask & bit) return false;
    done_mask |= bit;
    return true;
}
constexpr uint32_t kMaxSmem = 232448;  // 227 KiB opt-in dynamic shared memory per CTA
constexpr uint32_t kChunkBytes = 32768; // 255*255*32768 < 2^31 (R7)
constexpr uint32_t kMaxHostSlices = 4;  // K slices of one vipir_dbmul_host call (copy / split / scan pipeline)

using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// 2-D row-major tensor [dim1][dim0] of `esize`-byte elements, row pitch `pitch` bytes.
int make_tmap_2d(CUtensorMap* m, const void* base, CUtensorMapDataType dt, uint32_t esize, uint64_t dim0,
                 uint64_t dim1, uint64_t pitch, uint32_t box0, uint32_t box1, CUtensorMapSwizzle sw,
                 CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_L2_256B) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) {
        snprintf(g_cuda_err, sizeof g_cuda_err, "cuTensorMapEncodeTiled entry point not found");
        return VIPIR_ERR_CUDA;
    }
    cuuint64_t dims[2] = {dim0, dim1};
    cuuint64_t strides[1] = {pitch};
    cuuint32_t box[2] = {box0, box1};
    cuuint32_t estr[2] = {1, 1};
    (void)esize;
    CUresult r = fn(m, dt, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, sw,
                    promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof g_cuda_err, "cuTensorMapEncodeTiled failed: CUresult %d", (int)r);
        return VIPIR_ERR_CUDA;
    }
    return VIPIR_OK;
}

// A plan's workspace, tensor maps and streams belong to the device that was current when it was made: a call under
// another current device would launch there against this device's addresses.  Checked on every call.
bool on_device(int plan_device) {
    int cur = -1;
    return cudaGetDevice(&cur) == cudaSuccess && cur == plan_device;
}

uint32_t round_up(uint32_t x, uint32_t m) { return (x + m - 1) / m * m; }
uint32_t ceil_div(uint32_t x, uint32_t m) { return (x + m - 1) / m; }

}  // namespace

struct vipir_plan {
    uint64_t rows, cols, kbytes;
    uint32_t batch, db_bits, dl, lc, nq, n_moduli;
    uint32_t db_layout;  // VIPIR_DB_ROW_MAJOR or VIPIR_DB_LIMB_PLANES (u16 only)
    uint32_t kdl;        // DB bytes per k in one row of the matrix the kernels scan: dl, or 1 for limb planes
    uint32_t moduli[VIPIR_MAX_MODULI];
    uint32_t regime;
    uint32_t ms_bits;  // fused modulus switch (0 = off)
    uint32_t db_signed;  // DB elements are two's-complement int8
    vipir_tuning tune;   // explicit planner overrides (vipir_dbmul_plan_tuned); all zero = the planner's own choices
    int num_sms;
    int device;  // the device current at plan time: every call must come with it current
    // workspace
    uint8_t* d_planes;
    uint64_t planes_bytes;
    uint32_t* d_sync;  // MMA regimes: ticket, finished-groups count, per-leftover-unit arrival counters
    // host-call staging; the copy stream and events of its overlapped form (vipir_dbmul_host)
    uint32_t* d_q_stage;
    uint32_t* d_a_stage;
    cudaStream_t copy_stream;
    cudaEvent_t ev_begin, ev_slice[kMaxHostSlices];
    // kernel parameters
    vipir::GemmParams gm;
    vipir::GemvParams gv;
    uint32_t smem_bytes, grid;
    // tensor maps
    CUtensorMap tm_planes;
    CUtensorMap tm_db;
    const void* tm_db_for;  // d_db the cached tm_db was encoded for
    // GEMV with the query split fused in (u8 DB, cols % 32 == 0): tensor map over the raw query words
    bool gv_fused;
    CUtensorMap tm_query;
    const void* tm_query_for;
};

namespace {

template <int CG, int LC, bool PRIME, int NL = 1>
int launch_gemm(vipir_plan* p, const vipir::GemmParams& g, cudaStream_t st) {
    auto kern = vipir::gemm_i8_kernel<CG, LC, PRIME, NL>;
    static thread_local uint64_t attr_set = 0;  // bit d: done on device d
    if (attr_needed(attr_set)) {
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem));
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(g.n_groups * CG);
    cfg.blockDim = dim3(vipir::GM_THREADS);
    cfg.dynamicSmemBytes = p->smem_bytes;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CG;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    CK(cudaLaunchKernelEx(&cfg, kern, p->tm_db, p->tm_planes, g));
    return VIPIR_OK;
}

template <int CG>
int launch_gemm_cg(vipir_plan* p, const vipir::GemmParams& g, cudaStream_t st) {
    const bool prime = p->n_moduli > 0;
    if (p->db_layout == VIPIR_DB_LIMB_PLANES)
        return prime ? launch_gemm<CG, 4, true, 2>(p, g, st) : launch_gemm<CG, 4, false, 2>(p, g, st);
    if (p->lc == 5) return launch_gemm<CG, 5, true>(p, g, st);
    return prime ? launch_gemm<CG, 4, true>(p, g, st) : launch_gemm<CG, 4, false>(p, g, st);
}

// splits the columns [k_lo, k_hi) of every query vector (k_lo a multiple of 16)
int launch_split(vipir_plan* p, const uint32_t* d_query, uint8_t* planes, cudaStream_t st, uint64_t k_lo, uint64_t k_hi) {
    const uint64_t groups = ((k_hi - k_lo + 15) / 16) * p->nq;
    const uint32_t blocks = (uint32_t)((groups + 255) / 256);
    if (p->kdl == 1)
        vipir::split_limbs_kernel<1, 4><<<blocks, 256, 0, st>>>(d_query, planes, p->cols, p->nq, k_lo, k_hi);
    else if (p->lc == 4)
        vipir::split_limbs_kernel<2, 4><<<blocks, 256, 0, st>>>(d_query, planes, p->cols, p->nq, k_lo, k_hi);
    else
        vipir::split_limbs_kernel<2, 5><<<blocks, 256, 0, st>>>(d_query, planes, p->cols, p->nq, k_lo, k_hi);
    CK(cudaGetLastError());
    return VIPIR_OK;
}
int launch_split(vipir_plan* p, const uint32_t* d_query, uint8_t* planes, cudaStream_t st) {
    return launch_split(p, d_query, planes, st, 0, p->cols);
}

// ---- planning ------------------------------------------------------------------------------

int plan_gemm(vipir_plan* p, int cg) {
    vipir::GemmParams& g = p->gm;
    memset(&g, 0, sizeof g);
    if (p->tune.separate_split) return VIPIR_ERR_UNSUPPORTED;  // the tensor-core regimes always run the splitter
    const uint32_t lc = p->lc;
    // limb-plane u16 DB: the two limb tiles of a row block are two M sub-tiles, so msub >= 2
    const uint32_t nl = (p->db_layout == VIPIR_DB_LIMB_PLANES) ? 2u : 1u;
    const uint32_t bn_max = (cg == 1 || nl == 2) ? 256u : 512u;
    const uint32_t q_align = (lc == 5) ? 16u : 4u;       // keeps bn a multiple of 16 and of 4*LC
    const uint32_t q_align2 = (lc == 5) ? 32u : 8u;      // two instructions: bn/2 a multiple of 16
    const uint32_t qt_max = (bn_max / lc) / q_align2 * q_align2;
    uint32_t qt = round_up(p->nq, q_align);
    uint32_t n_tiles = 1;
    if (qt > qt_max) {
        n_tiles = ceil_div(p->nq, qt_max);
        qt = round_up(ceil_div(p->nq, n_tiles), q_align);
    }
    if (const uint32_t qt_force = p->tune.tile_queries) {
        if (qt_force % q_align != 0 || qt_force > qt_max) return VIPIR_ERR_UNSUPPORTED;
        qt = qt_force;
    }
    uint32_t bn = qt * lc;
    if (bn > 256) {
        qt = round_up(qt, q_align2);
        bn = qt * lc;
    }
    if (bn > bn_max) return VIPIR_ERR_UNSUPPORTED;
    g.rows = p->rows;
    g.nq = p->nq;
    g.batch = p->batch;
    g.qt = qt;
    g.bn = bn;
    g.n_tiles = ceil_div(p->nq, qt);
    g.n_instr = (bn > 256) ? 2u : 1u;
    g.ni_cols = bn / g.n_instr;
    g.total_ksteps = (uint32_t)((p->kbytes + vipir::GM_BK - 1) / vipir::GM_BK);
    const uint32_t max_ksteps = kChunkBytes / vipir::GM_BK;  // 256
    g.n_chunks = ceil_div(g.total_ksteps, max_ksteps);
    if (const uint32_t min_chunks = p->tune.min_chunks) {
        // finer work items for short K (measured: no robust gain, so not a planner rule)
        if (min_chunks > g.total_ksteps) return VIPIR_ERR_UNSUPPORTED;
        if (min_chunks > g.n_chunks) g.n_chunks = min_chunks;
    }
    g.ksteps_per_chunk = ceil_div(g.total_ksteps, g.n_chunks);
    // equal chunks of ceil(k-atoms / n) can leave the last ones empty when n was forced (6 k-atoms in 4 chunks:
    // 2 + 2 + 2 + 0), and a chunk without k-atoms would never complete its accumulator: count the chunks that exist
    g.n_chunks = ceil_div(g.total_ksteps, g.ksteps_per_chunk);
    const uint32_t max_groups = (uint32_t)p->num_sms / cg;
    // M sub-tiles per CTA (gemm_i8_tcgen05.cuh): while the product is HBM-bound every DB byte drags
    // bn / (128 * cg * msub) limb-plane bytes through L2 -> SM with it, and that fill (~8 TB/s on the
    // whole chip) is what caps the scan; so take the most sub-tiles that keep two accumulator stages
    // in TMEM, three pipeline stages in shared memory and >= 2 work items per group.
    uint32_t msub = nl;
    for (uint32_t cand = 4; cand > nl; cand >>= 1) {
        const uint64_t rows_unit = 128ull * cg * (cand / nl);
        const uint64_t units = (p->rows + rows_unit - 1) / rows_unit * g.n_tiles;
        const uint32_t atom = cand * vipir::GM_A_BYTES + g.n_instr * (g.ni_cols / cg) * vipir::GM_BK;
        if (2 * cand * bn <= 512 && 3 * atom <= kMaxSmem - 1408 && units * g.n_chunks >= 2ull * max_groups) {
            msub = cand;
            break;
        }
    }
    if (const uint32_t msub_force = p->tune.m_sub) {
        if (msub_force * bn > 512 || msub_force % nl != 0) return VIPIR_ERR_UNSUPPORTED;
        msub = msub_force;
    }
    g.msub = msub;
    const uint64_t rows_unit = 128ull * cg * (msub / nl);
    g.m_tiles = (uint32_t)((p->rows + rows_unit - 1) / rows_unit);
    g.atom_bytes = msub * vipir::GM_A_BYTES + g.n_instr * (g.ni_cols / cg) * vipir::GM_BK;
    const uint32_t overhead = 1024 + 384;  // alignment slack + barriers (ring, accumulator, copier) and the words behind them
    // k-atoms per stage and ring depth (DESIGN.md section 6 "in-flight bytes")
    // round-1 measurement on B200, not reproduced since (vipir_tuning.k_atoms / .stages reach the alternatives; round 3's
    // configs[4] sweep, profiles/r03_ncu_gemm_i8_c5_planes.txt, again has k_atoms 2 behind the default): several k-atoms per stage (longer contiguous DB
    // runs per row, fewer barrier round trips) beat deeper rings of single atoms; keep >= 3 stages
    uint32_t katoms = (kMaxSmem - overhead) / 3 / g.atom_bytes;
    if (katoms > 4) katoms = 4;
    if (p->tune.k_atoms) katoms = p->tune.k_atoms;
    if (katoms < 1) katoms = 1;
    while (katoms > 1 && 2 * katoms * g.atom_bytes > kMaxSmem - overhead) --katoms;
    if (katoms > g.ksteps_per_chunk) katoms = g.ksteps_per_chunk;
    g.katoms = katoms;
    g.stage_bytes = katoms * g.atom_bytes;
    uint32_t stages = (kMaxSmem - overhead) / g.stage_bytes;
    if (stages > 12) stages = 12;
    if (const uint32_t want = p->tune.stages) {
        if (want > stages) return VIPIR_ERR_UNSUPPORTED;
        stages = want;
    }
    if (stages < 2) return VIPIR_ERR_UNSUPPORTED;
    g.stages = stages;
    g.acc_stages = (2 * msub * bn <= 512) ? 2u : 1u;
    uint32_t cols_needed = g.acc_stages * msub * bn, tc = 32;
    while (tc < cols_needed) tc <<= 1;
    g.tmem_cols = tc;
    g.idesc = (2u << 4) /* D = s32 */ | (0u << 7) /* A = u8 */ | (0u << 10) /* B = u8 */ |
              ((g.ni_cols >> 3) << 17) | (((128u * cg) >> 4) << 24);
    g.n_moduli = p->n_moduli;
    for (uint32_t t = 0; t < p->n_moduli; ++t) {
        g.moduli[t] = p->moduli[t];
        g.barrett[t] = (uint64_t)((((unsigned __int128)1) << 64) / p->moduli[t]);
    }
    p->smem_bytes = stages * g.stage_bytes + overhead;
    // groups: one per SM (pair); fewer only when there are fewer work items (unit, K chunk) than that
    const uint64_t items = (uint64_t)g.m_tiles * g.n_tiles * g.n_chunks;
    g.split = p->tune.whole_units ? 0u : 1u;
    g.collector = p->tune.no_collector ? 0u : 1u;
    const uint64_t n_units64 = (uint64_t)g.m_tiles * g.n_tiles;
    g.n_groups = (uint32_t)(items < max_groups ? items : max_groups);
    if (!g.split && n_units64 < g.n_groups) g.n_groups = (uint32_t)n_units64;
    // The last, partial round: L = units mod groups leftover units are dealt out chunk by chunk, so it takes
    // ceil(L * nc / groups) / nc of a unit's time.  With few K chunks that rounds up badly (configs[4] as limb planes:
    // 256 units of ONE chunk on 74 pairs = 34 pairs run a fourth unit while 40 idle, ncu: SMs active 84 % of the launch),
    // so the leftover units alone may be cut finer; the units of the full rounds keep the fewest chunks (every extra chunk
    // is one more accumulator drain).  Finer only where it shortens the round by a fifth or more, chunks of >= 8 KiB of K.
    g.nc_left = g.kpc_left = 0;
    {
        uint32_t nc_left = 0;
        if (const uint32_t force = p->tune.leftover_chunks) {
            if (!g.split || force < g.n_chunks || force > g.total_ksteps) return VIPIR_ERR_UNSUPPORTED;
            nc_left = force;
        } else if (g.split && n_units64 > g.n_groups && n_units64 % g.n_groups != 0) {
            const uint64_t L = n_units64 % g.n_groups;
            auto cost = [&](uint32_t nc) { return (uint32_t)(((L * nc + g.n_groups - 1) / g.n_groups) * 1000 / nc); };
            uint32_t best = g.n_chunks, best_cost = cost(g.n_chunks);
            for (uint32_t mult = 2; mult <= 4; mult *= 2) {
                const uint32_t kpc = ceil_div(g.total_ksteps, g.n_chunks * mult);
                if (kpc < 64) break;
                const uint32_t nc = ceil_div(g.total_ksteps, kpc);
                if (cost(nc) * 10 <= best_cost * 8) best = nc, best_cost = cost(nc);
            }
            if (best != g.n_chunks) nc_left = best;
        }
        if (nc_left) {
            const uint32_t kpc = ceil_div(g.total_ksteps, nc_left);
            if (kpc != g.ksteps_per_chunk) {
                g.kpc_left = kpc;
                g.nc_left = ceil_div(g.total_ksteps, kpc);  // the chunks that exist (see n_chunks above)
            }
        }
    }
    p->grid = g.n_groups * cg;
    if (!p->d_sync) {
        const size_t sync_bytes = (2 + (size_t)max_groups) * sizeof(uint32_t);
        if (cudaMalloc(&p->d_sync, sync_bytes) != cudaSuccess) {
            cudaGetLastError();
            return VIPIR_ERR_ALLOC;
        }
        CK(cudaMemset(p->d_sync, 0, sync_bytes));
        // the first launch may come on a non-blocking stream, which the legacy stream's memset is not ordered
        // against: the plan call may block, so wait for the zeros here
        CK(cudaDeviceSynchronize());
    }
    g.sync = p->d_sync;
    // limb-plane tensor map: [nq*LC][K'] bytes, box 128 B x (ni_cols / cg) rows, 128B swizzle
    return make_tmap_2d(&p->tm_planes, p->d_planes, CU_TENSOR_MAP_DATA_TYPE_UINT8, 1, p->kbytes,
                        (uint64_t)p->nq * lc, p->kbytes, vipir::GM_BK, g.ni_cols / cg, CU_TENSOR_MAP_SWIZZLE_128B);
}

int plan_gemv(vipir_plan* p) {
    if (p->nq != 1 || p->n_moduli != 0 || p->lc != 4) return VIPIR_ERR_UNSUPPORTED;
    const vipir_tuning& tu = p->tune;  // overrides of the tensor-core regimes do not apply here
    if (tu.m_sub || tu.tile_queries || tu.k_atoms || tu.min_chunks || tu.whole_units || tu.no_collector || tu.host_slices ||
        tu.leftover_chunks)
        return VIPIR_ERR_UNSUPPORTED;
    vipir::GemvParams& g = p->gv;
    memset(&g, 0, sizeof g);
    g.rows = p->rows;
    g.kbytes = (uint32_t)p->kbytes;
    g.n_ksteps = (uint32_t)((p->kbytes + vipir::GV_KT - 1) / vipir::GV_KT);
    g.n_blocks = (uint32_t)((p->rows + vipir::GV_R - 1) / vipir::GV_R);
    g.stages = p->tune.stages ? p->tune.stages : 4;  // 4 x 36 KiB in flight per SM measured best
    if (g.stages > 6) return VIPIR_ERR_UNSUPPORTED;
    p->smem_bytes = g.stages * vipir::GV_STAGE_BYTES + 1024 + 2 * 8 * g.stages + 2 * vipir::GV_R * 4;
    // step a1 fused into the scan when the raw query can be boxed as 32-word rows (gemv_b1.cuh "FUSED")
    p->gv_fused = p->dl == 1 && p->cols % 32 == 0 && !p->tune.separate_split;
    p->grid = g.n_blocks < (uint32_t)p->num_sms ? g.n_blocks : (uint32_t)p->num_sms;
    // limb planes [4][K'] viewed as u32 elements: box 256 elements (1024 B) x 4 rows
    return make_tmap_2d(&p->tm_planes, p->d_planes, CU_TENSOR_MAP_DATA_TYPE_UINT32, 4, p->kbytes / 4, 4, p->kbytes,
                        vipir::GV_KT / 4, 4, CU_TENSOR_MAP_SWIZZLE_NONE);
}

int encode_db_map(vipir_plan* p, const void* d_db) {
    if (p->tm_db_for == d_db) return VIPIR_OK;
    int rc;
    if (p->regime == VIPIR_REGIME_GEMV)
        rc = make_tmap_2d(&p->tm_db, d_db, CU_TENSOR_MAP_DATA_TYPE_UINT32, 4, p->kbytes / 4, p->rows, p->kbytes,
                          vipir::GV_KT / 4, vipir::GV_R, CU_TENSOR_MAP_SWIZZLE_NONE);
    else
        // limb planes: D_hi lies directly behind D_lo, one u8 matrix of 2*rows rows
        rc = make_tmap_2d(&p->tm_db, d_db, CU_TENSOR_MAP_DATA_TYPE_UINT8, 1, p->kbytes,
                          p->rows * (p->db_layout == VIPIR_DB_LIMB_PLANES ? 2 : 1), p->kbytes,
                          vipir::GM_BK, vipir::GM_BM, CU_TENSOR_MAP_SWIZZLE_128B);
    if (rc == VIPIR_OK) p->tm_db_for = d_db;
    return rc;
}

}  // namespace

extern "C" {

const char* vipir_status_str(int s) {
    switch (s) {
        case VIPIR_OK: return "VIPIR_OK";
        case VIPIR_ERR_INVALID_ARG: return "VIPIR_ERR_INVALID_ARG";
        case VIPIR_ERR_UNSUPPORTED: return "VIPIR_ERR_UNSUPPORTED";
        case VIPIR_ERR_ALLOC: return "VIPIR_ERR_ALLOC";
        case VIPIR_ERR_CUDA: return "VIPIR_ERR_CUDA";
        case VIPIR_ERR_ARCH: return "VIPIR_ERR_ARCH";
        default: return "VIPIR_ERR_UNKNOWN";
    }
}

const char* vipir_last_cuda_error(void) { return g_cuda_err; }

int vipir_dbmul_plan_ex(vipir_plan** out, uint64_t rows, uint64_t cols, uint32_t batch, uint32_t db_bits,
                        const vipir_modulus_spec* mod, uint32_t regime) {
    return vipir_dbmul_plan_layout(out, rows, cols, batch, db_bits, mod, regime, VIPIR_DB_ROW_MAJOR);
}

int vipir_dbmul_plan_layout(vipir_plan** out, uint64_t rows, uint64_t cols, uint32_t batch, uint32_t db_bits,
                            const vipir_modulus_spec* mod, uint32_t regime, uint32_t db_layout) {
    return vipir_dbmul_plan_tuned(out, rows, cols, batch, db_bits, mod, regime, db_layout, nullptr);
}

int vipir_dbmul_plan_tuned(vipir_plan** out, uint64_t rows, uint64_t cols, uint32_t batch, uint32_t db_bits,
                           const vipir_modulus_spec* mod, uint32_t regime, uint32_t db_layout,
                           const vipir_tuning* tune) {
    if (!out) return VIPIR_ERR_INVALID_ARG;
    *out = nullptr;
    if (tune) {  // domain of every field; whether the shape can honour it is the planner's UNSUPPORTED
        if ((tune->m_sub != 0 && tune->m_sub != 1 && tune->m_sub != 2 && tune->m_sub != 4) || tune->tile_queries > 128 ||
            tune->k_atoms > 8 || tune->stages == 1 || tune->stages > 12 || tune->separate_split > 1 ||
            tune->whole_units > 1 || tune->no_collector > 1 || tune->host_staged > 1 || tune->host_slices > kMaxHostSlices ||
            tune->leftover_chunks > 4096)
            return VIPIR_ERR_INVALID_ARG;
        for (uint32_t r : tune->reserved)
            if (r != 0) return VIPIR_ERR_INVALID_ARG;
    }
    // ---- argument checks first: these need no device ----
    if (rows == 0 || cols == 0 || batch == 0) return VIPIR_ERR_INVALID_ARG;
    if (db_bits != 8 && db_bits != 16) return VIPIR_ERR_INVALID_ARG;
    if (regime > VIPIR_REGIME_NAIVE) return VIPIR_ERR_INVALID_ARG;
    if (db_layout > VIPIR_DB_LIMB_PLANES) return VIPIR_ERR_INVALID_ARG;
    const bool planes = db_layout == VIPIR_DB_LIMB_PLANES;
    // limb planes exist for u16 DBs and are scanned by the tensor-core regimes only
    if (planes && (db_bits != 16 || regime == VIPIR_REGIME_GEMV || regime == VIPIR_REGIME_NAIVE))
        return VIPIR_ERR_UNSUPPORTED;
    const uint32_t n_moduli = mod ? mod->count : 0;
    if (n_moduli > VIPIR_MAX_MODULI) return VIPIR_ERR_INVALID_ARG;
    if (n_moduli > 0 && !mod->moduli) return VIPIR_ERR_INVALID_ARG;
    for (uint32_t t = 0; t < n_moduli; ++t)
        if (mod->moduli[t] < 2 || mod->moduli[t] >= (1u << 30)) return VIPIR_ERR_INVALID_ARG;
    const uint32_t dl = db_bits / 8;
    const uint32_t kdl = planes ? 1u : dl;
    if (cols > (1ull << 31) || (cols * kdl) % 16 != 0) return VIPIR_ERR_UNSUPPORTED;
    const uint64_t kbytes = cols * kdl;
    if (rows >= (1ull << 31) || kbytes >= (1ull << 31)) return VIPIR_ERR_UNSUPPORTED;
    if (planes && rows >= (1ull << 30)) return VIPIR_ERR_UNSUPPORTED;  // 2*rows rows in one tensor map
    const uint32_t T = n_moduli ? n_moduli : 1;
    if ((uint64_t)T * batch * 5 >= (1ull << 31)) return VIPIR_ERR_UNSUPPORTED;

    // ---- device ----
    int dev = 0;
    CK(cudaGetDevice(&dev));
    int major = 0, minor = 0, sms = 0;
    CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    CK(cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10 || minor != 0) return VIPIR_ERR_ARCH;

    vipir_plan* p = new (std::nothrow) vipir_plan;
    if (!p) return VIPIR_ERR_ALLOC;
    memset(p, 0, sizeof *p);
    p->rows = rows;
    p->cols = cols;
    p->kbytes = kbytes;
    p->batch = batch;
    p->db_bits = db_bits;
    p->dl = dl;
    p->kdl = kdl;
    p->db_layout = db_layout;
    p->n_moduli = n_moduli;
    for (uint32_t t = 0; t < n_moduli; ++t) p->moduli[t] = mod->moduli[t];
    p->nq = T * batch;
    p->lc = (kdl == 2 && n_moduli > 0) ? 5u : 4u;  // split_limbs.cuh: the s = 4 column vanishes mod 2^32
    p->num_sms = sms;
    p->device = dev;
    if (tune) p->tune = *tune;

    if (regime == VIPIR_REGIME_AUTO) {
        if (p->nq == 1 && n_moduli == 0 && !planes) regime = VIPIR_REGIME_GEMV;
        // round-1 measurement, not reproduced since (VIPIR_REGIME_MMA_1SM / _2SM force either): CTA pairs win from 32 query vectors up, where the limb
        // tile's shared-memory traffic starts to matter; below that one CTA per tile is as fast
        else regime = ((uint64_t)p->nq * p->lc > 64 && rows > 128) ? VIPIR_REGIME_MMA_2SM : VIPIR_REGIME_MMA_1SM;
    }
    p->regime = regime;

    p->planes_bytes = (uint64_t)p->nq * p->lc * kbytes;
    if (cudaMalloc(&p->d_planes, p->planes_bytes) != cudaSuccess) {
        cudaGetLastError();
        delete p;
        return VIPIR_ERR_ALLOC;
    }
    int rc = VIPIR_OK;
    switch (regime) {
        case VIPIR_REGIME_GEMV: rc = plan_gemv(p); break;
        case VIPIR_REGIME_MMA_1SM: rc = plan_gemm(p, 1); break;
        case VIPIR_REGIME_MMA_2SM: rc = plan_gemm(p, 2); break;
        case VIPIR_REGIME_NAIVE: p->grid = (uint32_t)((rows + 127) / 128); break;
        default: rc = VIPIR_ERR_INVALID_ARG;
    }
    if (rc != VIPIR_OK) {
        vipir_destroy(p);
        return rc;
    }
    *out = p;
    return VIPIR_OK;
}

int vipir_dbmul_plan(vipir_plan** out, uint64_t rows, uint64_t cols, uint32_t batch, uint32_t db_bits,
                     const vipir_modulus_spec* mod) {
    return vipir_dbmul_plan_ex(out, rows, cols, batch, db_bits, mod, VIPIR_REGIME_AUTO);
}

int vipir_split_limbs(vipir_plan* p, const uint32_t* d_query, uint8_t* d_planes_out, void* cuda_stream) {
    if (!p || !d_query || (reinterpret_cast<uintptr_t>(d_query) & 15) ||
        (reinterpret_cast<uintptr_t>(d_planes_out) & 15))
        return VIPIR_ERR_INVALID_ARG;
    if (!on_device(p->device)) return VIPIR_ERR_INVALID_ARG;
    return launch_split(p, d_query, d_planes_out ? d_planes_out : p->d_planes, static_cast<cudaStream_t>(cuda_stream));
}

// The launch's view of the K dimension when a call is cut into K slices (vipir_dbmul_host): k-atoms
// [k_begin, k_begin + k_atoms) of the product, added to what `answer` holds when acc_in is set, the last
// chunk written to final_out.  The whole product: {0, all, 0, answer}.
struct KSlice {
    uint32_t k_begin, k_atoms, acc_in;
    uint32_t* final_out;
    bool is_last;
};

// d_query_fused != NULL: GEMV with the query split fused in (reads the raw query instead of the limb planes)
static int scan_only(vipir_plan* p, const void* d_db, uint32_t* d_answer, cudaStream_t st,
                     const uint32_t* d_query_fused = nullptr, const KSlice* slice = nullptr) {
    int rc = encode_db_map(p, d_db);
    if (rc != VIPIR_OK) return rc;
    if (p->regime == VIPIR_REGIME_GEMV) {
        static thread_local uint64_t attr_set = 0;  // bit d: done on device d
        if (attr_needed(attr_set)) {
            CK(cudaFuncSetAttribute(vipir::gemv_b1_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)kMaxSmem));
            CK(cudaFuncSetAttribute(vipir::gemv_b1_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)kMaxSmem));
            CK(cudaFuncSetAttribute(vipir::gemv_b1_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)kMaxSmem));
            CK(cudaFuncSetAttribute(vipir::gemv_b1_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    (int)kMaxSmem));
        }
        vipir::GemvParams gv = p->gv;  // per-call values go into a copy: the plan's parameters stay as planned
        gv.answer = d_answer;
        gv.ms_bits = p->ms_bits;
        if (d_query_fused) {  // raw query words, split inside the kernel
            if (p->tm_query_for != d_query_fused) {
                rc = make_tmap_2d(&p->tm_query, d_query_fused, CU_TENSOR_MAP_DATA_TYPE_UINT32, 4, 32, p->cols / 32, 128, 32,
                                  32, CU_TENSOR_MAP_SWIZZLE_128B);
                if (rc != VIPIR_OK) return rc;
                p->tm_query_for = d_query_fused;
            }
            if (p->db_signed)
                vipir::gemv_b1_kernel<true, true><<<p->grid, vipir::GV_THREADS, p->smem_bytes, st>>>(p->tm_db, p->tm_query, gv);
            else
                vipir::gemv_b1_kernel<false, true><<<p->grid, vipir::GV_THREADS, p->smem_bytes, st>>>(p->tm_db, p->tm_query, gv);
        } else if (p->db_signed) {
            vipir::gemv_b1_kernel<true, false><<<p->grid, vipir::GV_THREADS, p->smem_bytes, st>>>(p->tm_db, p->tm_planes, gv);
        } else {
            vipir::gemv_b1_kernel<false, false><<<p->grid, vipir::GV_THREADS, p->smem_bytes, st>>>(p->tm_db, p->tm_planes, gv);
        }
        CK(cudaGetLastError());
        return VIPIR_OK;
    }
    vipir::GemmParams g = p->gm;  // per-call values go into a copy: the plan's parameters stay as planned
    g.answer = d_answer;
    g.final_out = d_answer;
    g.ms_bits = p->ms_bits;
    g.db_signed = p->db_signed;
    // instruction descriptor bits [7,10): A operand format, 0 = u8, 1 = s8 (B stays u8: the limbs)
    g.idesc = (g.idesc & ~(7u << 7)) | ((p->db_signed ? 1u : 0u) << 7);
    if (slice) {
        const uint32_t max_ksteps = kChunkBytes / vipir::GM_BK;
        g.k_begin = slice->k_begin;
        g.total_ksteps = slice->k_atoms;
        g.n_chunks = ceil_div(slice->k_atoms, max_ksteps);
        g.ksteps_per_chunk = ceil_div(slice->k_atoms, g.n_chunks);
        g.nc_left = g.kpc_left = 0;  // a K slice is short already: every unit in the same chunks
        g.acc_in = slice->acc_in;
        g.final_out = slice->final_out;
        if (!slice->is_last) g.ms_bits = 0;  // the switch rounds the complete sum only
        const uint64_t items = (uint64_t)g.m_tiles * g.n_tiles * g.n_chunks;
        if (items < g.n_groups) g.n_groups = (uint32_t)items;
    }
    return (p->regime == VIPIR_REGIME_MMA_2SM) ? launch_gemm_cg<2>(p, g, st) : launch_gemm_cg<1>(p, g, st);
}

int vipir_dbmul_scan(vipir_plan* p, const void* d_db, uint32_t* d_answer, void* cuda_stream) {
    if (!p || !d_db || !d_answer) return VIPIR_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_db) & 15) || (reinterpret_cast<uintptr_t>(d_answer) & 3))
        return VIPIR_ERR_INVALID_ARG;
    if (!on_device(p->device)) return VIPIR_ERR_INVALID_ARG;
    if (p->regime == VIPIR_REGIME_NAIVE) return VIPIR_ERR_UNSUPPORTED;  // the check kernel has no limb planes
    return scan_only(p, d_db, d_answer, static_cast<cudaStream_t>(cuda_stream));
}

int vipir_dbmul(vipir_plan* p, const void* d_db, const uint32_t* d_query, uint32_t* d_answer, void* cuda_stream) {
    if (!p || !d_db || !d_query || !d_answer) return VIPIR_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_db) & 15) || (reinterpret_cast<uintptr_t>(d_query) & 15) ||
        (reinterpret_cast<uintptr_t>(d_answer) & 3))
        return VIPIR_ERR_INVALID_ARG;
    if (!on_device(p->device)) return VIPIR_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

    if (p->regime == VIPIR_REGIME_NAIVE) {
        vipir::NaiveParams np{};
        np.rows = p->rows;
        np.cols = p->cols;
        np.batch = p->batch;
        np.db_bits = p->db_bits;
        np.n_moduli = p->n_moduli;
        np.db_signed = p->db_signed;
        for (uint32_t t = 0; t < p->n_moduli; ++t) np.moduli[t] = p->moduli[t];
        vipir::naive_dbmul_kernel<<<dim3(p->grid, p->nq), 128, 0, st>>>(d_db, d_query, d_answer, np);
        CK(cudaGetLastError());
        return VIPIR_OK;
    }
    if (p->regime == VIPIR_REGIME_GEMV && p->gv_fused) return scan_only(p, d_db, d_answer, st, d_query);
    int rc = launch_split(p, d_query, p->d_planes, st);
    if (rc != VIPIR_OK) return rc;
    return scan_only(p, d_db, d_answer, st);
}

// device pointer of h if it is pinned, device-mapped host memory; else NULL
static uint32_t* mapped_device_pointer(uint32_t* h) {
    cudaPointerAttributes attr{};
    if (cudaPointerGetAttributes(&attr, h) == cudaSuccess && attr.type == cudaMemoryTypeHost && attr.devicePointer)
        return static_cast<uint32_t*>(attr.devicePointer);
    cudaGetLastError();  // not a CUDA-known pointer: pageable memory
    return nullptr;
}

// K slices of one host call (tensor-core regimes): boundaries in k-atoms.  The first slice is small so that the
// scan starts early; the copies of the later, larger slices run behind the scan of the earlier ones.
static uint32_t host_slices(const vipir_plan* p, size_t qbytes, uint32_t bounds[kMaxHostSlices + 1]) {
    const uint32_t A = p->gm.total_ksteps;
    uint32_t S = p->tune.host_slices;
    if (S == 0) S = (qbytes >= (8u << 20) && A >= 16) ? 3u : 1u;  // small queries: one copy, one launch
    if (S > A) S = A;
    bounds[0] = 0;
    // 1/8, 1/2, 1 (three slices); 1/8, 3/8, 5/8, 1 (four); 1/4, 1 (two)
    static const uint32_t frac8[kMaxHostSlices + 1][kMaxHostSlices] = {{0}, {8}, {2, 8}, {1, 4, 8}, {1, 3, 5, 8}};
    for (uint32_t i = 0; i < S; ++i) {
        uint32_t b = (uint32_t)((uint64_t)A * frac8[S][i] / 8);
        if (b <= bounds[i]) b = bounds[i] + 1;
        bounds[i + 1] = b;
    }
    bounds[S] = A;
    return S;
}

int vipir_dbmul_host(vipir_plan* p, const void* d_db, const uint32_t* h_query, uint32_t* h_answer, void* cuda_stream) {
    if (!p || !d_db || !h_query || !h_answer) return VIPIR_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(d_db) & 15) return VIPIR_ERR_INVALID_ARG;
    if (!on_device(p->device)) return VIPIR_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t qbytes = (size_t)p->nq * p->cols * 4, abytes = (size_t)p->nq * p->rows * 4;
    if (!p->d_q_stage && cudaMalloc(&p->d_q_stage, qbytes) != cudaSuccess) {
        cudaGetLastError();
        return VIPIR_ERR_ALLOC;
    }
    // with pinned, device-mapped host memory the kernels write the answer into it themselves while the scan runs
    // (batch 1: the scan's own 128-byte stores; tensor regimes: copier warps, gemm_i8_tcgen05.cuh), and the
    // device-to-host copy after it disappears
    uint32_t* d_direct = p->tune.host_staged ? nullptr : mapped_device_pointer(h_answer);
    const bool mma = p->regime == VIPIR_REGIME_MMA_1SM || p->regime == VIPIR_REGIME_MMA_2SM;

    if (p->regime == VIPIR_REGIME_GEMV && d_direct) {
        CK(cudaMemcpyAsync(p->d_q_stage, h_query, qbytes, cudaMemcpyHostToDevice, st));
        int rc = vipir_dbmul(p, d_db, p->d_q_stage, d_direct, cuda_stream);
        if (rc != VIPIR_OK) return rc;
        CK(cudaStreamSynchronize(st));
        return VIPIR_OK;
    }
    uint32_t bounds[kMaxHostSlices + 1];
    const uint32_t S = (mma && !p->tune.host_staged) ? host_slices(p, qbytes, bounds) : 1u;
    // the running sums between K chunks / slices are read back by the kernels: they stay in device memory (the
    // mapped host buffer only receives finished units)
    if (!p->d_a_stage && cudaMalloc(&p->d_a_stage, abytes) != cudaSuccess) {
        cudaGetLastError();
        return VIPIR_ERR_ALLOC;
    }
    if (!mma || p->tune.host_staged) {  // one copy in, the device call, one copy out
        CK(cudaMemcpyAsync(p->d_q_stage, h_query, qbytes, cudaMemcpyHostToDevice, st));
        int rc = vipir_dbmul(p, d_db, p->d_q_stage, p->d_a_stage, cuda_stream);
        if (rc != VIPIR_OK) return rc;
        CK(cudaMemcpyAsync(h_answer, p->d_a_stage, abytes, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        return VIPIR_OK;
    }
    // ---- tensor-core regimes: copy / split / scan pipelined over K slices ----
    // copy stream: H2D of slice i's columns of every query vector (a strided copy), its split;  caller's stream:
    // the scan of slice i, which adds to the running sums of the slices before it (device staging).  In the last
    // slice every CTA copies its finished units to the host buffer when that is mapped (final_out).
    if (!p->copy_stream) {  // all of them or none: a later call must not find a stream without its events
        cudaStream_t cs = nullptr;
        cudaEvent_t ev[kMaxHostSlices + 1] = {};
        cudaError_t e = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking);
        for (uint32_t i = 0; e == cudaSuccess && i <= kMaxHostSlices; ++i)
            e = cudaEventCreateWithFlags(&ev[i], cudaEventDisableTiming);
        if (e != cudaSuccess) {
            for (cudaEvent_t x : ev)
                if (x) cudaEventDestroy(x);
            if (cs) cudaStreamDestroy(cs);
            return cuda_fail(e, "vipir_dbmul_host: copy stream / events");
        }
        p->copy_stream = cs;
        p->ev_begin = ev[kMaxHostSlices];
        for (uint32_t i = 0; i < kMaxHostSlices; ++i) p->ev_slice[i] = ev[i];
    }
    CK(cudaEventRecord(p->ev_begin, st));  // the staging buffers may still be read by work queued on `st`
    CK(cudaStreamWaitEvent(p->copy_stream, p->ev_begin, 0));
    uint32_t* const d_final = d_direct ? d_direct : p->d_a_stage;
    const size_t pitch = (size_t)p->cols * 4;
    // From here on work is in flight on both streams.  The call promises to be complete when it returns, also
    // when it fails: an error exit first waits for whatever was enqueued (copies still reading h_query, kernels
    // still writing the staging buffers or h_answer), so the caller may free or reuse its buffers and the plan.
    auto fail = [&](int rc) {
        cudaStreamSynchronize(p->copy_stream);
        cudaStreamSynchronize(st);
        cudaGetLastError();  // the error of record is the one already in g_cuda_err
        return rc;
    };
#define CKD(call)                                                   \
    do {                                                            \
        cudaError_t e__ = (call);                                   \
        if (e__ != cudaSuccess) return fail(cuda_fail(e__, #call)); \
    } while (0)
    for (uint32_t i = 0; i < S; ++i) {
        const uint64_t c_lo = (uint64_t)bounds[i] * vipir::GM_BK / p->kdl;
        uint64_t c_hi = (uint64_t)bounds[i + 1] * vipir::GM_BK / p->kdl;
        if (c_hi > p->cols) c_hi = p->cols;
        CKD(cudaMemcpy2DAsync(p->d_q_stage + c_lo, pitch, h_query + c_lo, pitch, (size_t)(c_hi - c_lo) * 4, p->nq,
                              cudaMemcpyHostToDevice, p->copy_stream));
        int rc = launch_split(p, p->d_q_stage, p->d_planes, p->copy_stream, c_lo, c_hi);
        if (rc != VIPIR_OK) return fail(rc);
        CKD(cudaEventRecord(p->ev_slice[i], p->copy_stream));
        CKD(cudaStreamWaitEvent(st, p->ev_slice[i], 0));
        KSlice sl{bounds[i], bounds[i + 1] - bounds[i], i > 0 ? 1u : 0u, i + 1 == S ? d_final : p->d_a_stage, i + 1 == S};
        rc = scan_only(p, d_db, p->d_a_stage, st, nullptr, &sl);
        if (rc != VIPIR_OK) return fail(rc);
    }
    if (!d_direct) CKD(cudaMemcpyAsync(h_answer, p->d_a_stage, abytes, cudaMemcpyDeviceToHost, st));
    CKD(cudaStreamSynchronize(st));
#undef CKD
    return VIPIR_OK;
}

int vipir_db_split_u16(const void* d_db_u16, void* d_db_planes, uint64_t rows, uint64_t cols, void* cuda_stream) {
    if (!d_db_u16 || !d_db_planes || rows == 0 || cols == 0) return VIPIR_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_db_u16) & 15) || (reinterpret_cast<uintptr_t>(d_db_planes) & 15))
        return VIPIR_ERR_INVALID_ARG;
    if (cols % 16 != 0 || rows >= (1ull << 31) || cols >= (1ull << 31)) return VIPIR_ERR_UNSUPPORTED;
    const uint64_t bytes = rows * cols * 2;
    const uintptr_t a = reinterpret_cast<uintptr_t>(d_db_u16), b = reinterpret_cast<uintptr_t>(d_db_planes);
    if (a < b + bytes && b < a + bytes) return VIPIR_ERR_INVALID_ARG;  // not in place
    const uint64_t n16 = rows * cols / 16;
    const uint64_t want = (n16 + 255) / 256;
    const uint32_t blocks = (uint32_t)(want < 148ull * 32 ? want : 148ull * 32);
    uint8_t* lo = static_cast<uint8_t*>(d_db_planes);
    vipir::db_split_u16_kernel<<<blocks, 256, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        static_cast<const uint4*>(d_db_u16), reinterpret_cast<uint4*>(lo), reinterpret_cast<uint4*>(lo + rows * cols), n16);
    CK(cudaGetLastError());
    return VIPIR_OK;
}

int vipir_plan_set_modswitch(vipir_plan* p, uint32_t out_bits) {
    if (!p || out_bits > 31) return VIPIR_ERR_INVALID_ARG;
    if (out_bits != 0 && (p->n_moduli != 0 || p->regime == VIPIR_REGIME_NAIVE)) return VIPIR_ERR_UNSUPPORTED;
    p->ms_bits = out_bits;
    return VIPIR_OK;
}

int vipir_plan_set_db_signed(vipir_plan* p, uint32_t is_signed) {
    if (!p || is_signed > 1) return VIPIR_ERR_INVALID_ARG;
    if (is_signed && p->db_bits != 8) return VIPIR_ERR_UNSUPPORTED;
    p->db_signed = is_signed;
    return VIPIR_OK;
}

int vipir_plan_info(const vipir_plan* p, vipir_info* o) {
    if (!p || !o) return VIPIR_ERR_INVALID_ARG;
    memset(o, 0, sizeof *o);
    o->regime = p->regime;
    o->db_limbs = p->dl;
    o->limb_cols = p->lc;
    o->query_vectors = p->nq;
    o->k_bytes = p->kbytes;
    o->smem_bytes = p->smem_bytes;
    o->grid = p->grid;
    o->workspace_bytes = p->planes_bytes;
    o->modswitch_bits = p->ms_bits;
    o->db_signed = p->db_signed;
    o->db_layout = p->db_layout;
    o->launches = (p->regime == VIPIR_REGIME_NAIVE || (p->regime == VIPIR_REGIME_GEMV && p->gv_fused)) ? 1 : 2;
    if (p->regime == VIPIR_REGIME_MMA_1SM || p->regime == VIPIR_REGIME_MMA_2SM) {
        o->k_chunk_bytes = p->gm.ksteps_per_chunk * vipir::GM_BK;
        o->n_chunks = p->gm.n_chunks;
        o->leftover_chunks = p->gm.nc_left ? p->gm.nc_left : p->gm.n_chunks;
        o->tile_queries = p->gm.qt;
        o->tile_cols = p->gm.bn;
        o->mma_n = p->gm.ni_cols;
        o->m_tiles = p->gm.m_tiles;
        o->n_tiles = p->gm.n_tiles;
        o->stages = p->gm.stages;
        o->m_sub = p->gm.msub;
    } else if (p->regime == VIPIR_REGIME_GEMV) {
        o->n_chunks = 1;
        o->m_tiles = p->gv.n_blocks;
        o->n_tiles = 1;
        o->stages = p->gv.stages;
    }
    return VIPIR_OK;
}

int vipir_testing_work_items(uint32_t g, uint32_t n_groups, uint32_t n_units, uint32_t n_chunks, uint32_t split,
                             uint32_t* out_triples, uint32_t cap, uint32_t* n) {
    if (!n || n_groups == 0 || g >= n_groups || n_chunks == 0 || (cap && !out_triples)) return VIPIR_ERR_INVALID_ARG;
    const vipir::WorkPlan w = vipir::make_work_plan(g, n_groups, n_units, n_chunks, split);
    uint32_t count = 0;
    vipir::for_each_item(w, [&](uint32_t u, uint32_t c, bool must_wait) {
        if (count < cap) {
            out_triples[3 * count] = u;
            out_triples[3 * count + 1] = c;
            out_triples[3 * count + 2] = must_wait ? 1u : 0u;
        }
        ++count;
    });
    *n = count;
    return VIPIR_OK;
}

void vipir_destroy(vipir_plan* p) {
    if (!p) return;
    if (p->d_planes) cudaFree(p->d_planes);
    if (p->d_sync) cudaFree(p->d_sync);
    if (p->d_q_stage) cudaFree(p->d_q_stage);
    if (p->d_a_stage) cudaFree(p->d_a_stage);
    if (p->copy_stream) {
        cudaStreamDestroy(p->copy_stream);
        cudaEventDestroy(p->ev_begin);
        for (uint32_t i = 0; i < kMaxHostSlices; ++i) cudaEventDestroy(p->ev_slice[i]);
    }
    delete p;
}

}  // extern "C"

// ---- vipir_dbmul_static: the tensor-core product for callers that must not allocate (include/vipir.h) ----------
//
// The tensor-core kernel needs two pieces of global memory besides its inputs and outputs: the query limb planes
// the splitter writes for it, and a few work-distribution counters.  A plan gets them from cudaMalloc.  This
// entry point keeps them in an array that is part of the library image instead, so the call itself never asks
// the driver for memory.  Layout: [0, 4096) the counters, [4096, 4096 + VIPIR_STATIC_SCRATCH_BYTES) the planes.
namespace {

constexpr uint32_t kStaticSyncBytes = 4096;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticSyncBytes + VIPIR_STATIC_SCRATCH_BYTES];

// In host code `g_static_scratch` is only a handle for the runtime, not an address a kernel can use.  The real
// device address differs per GPU, so it is looked up once per device (with that device current) and remembered.
constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
unsigned char* g_static_ptr[kStaticMaxDevices] = {};
int g_static_sms[kStaticMaxDevices] = {};

int static_scratch_setup(int dev, unsigned char** ptr, int* sms) {
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        int major = 0, minor = 0, n = 0;
        CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        CK(cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev));
        CK(cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev));
        if (major != 10 || minor != 0) return VIPIR_ERR_ARCH;
        void* a = nullptr;
        CK(cudaGetSymbolAddress(&a, g_static_scratch));
        if (!a) {
            snprintf(g_cuda_err, sizeof g_cuda_err, "cudaGetSymbolAddress returned a null address");
            return VIPIR_ERR_CUDA;
        }
        g_static_sms[dev] = n;
        g_static_ptr[dev] = static_cast<unsigned char*>(a);
    }
    *ptr = g_static_ptr[dev];
    *sms = g_static_sms[dev];
    return VIPIR_OK;
}

}  // namespace

extern "C" int vipir_dbmul_static(uint64_t rows, uint64_t cols, uint32_t batch, uint32_t db_bits,
                                  const vipir_modulus_spec* mod, const void* d_db, const uint32_t* d_query,
                                  uint32_t* d_answer, void* cuda_stream) {
    g_cuda_err[0] = 0;
    // ---- the argument rules of vipir_dbmul_plan and vipir_dbmul; none of them needs a device ----
    if (!d_db || !d_query || !d_answer) return VIPIR_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_db) & 15) || (reinterpret_cast<uintptr_t>(d_query) & 15) ||
        (reinterpret_cast<uintptr_t>(d_answer) & 3))
        return VIPIR_ERR_INVALID_ARG;
    if (rows == 0 || cols == 0 || batch == 0) return VIPIR_ERR_INVALID_ARG;
    if (db_bits != 8 && db_bits != 16) return VIPIR_ERR_INVALID_ARG;
    const uint32_t n_moduli = mod ? mod->count : 0;
    if (n_moduli > VIPIR_MAX_MODULI) return VIPIR_ERR_INVALID_ARG;
    if (n_moduli > 0 && !mod->moduli) return VIPIR_ERR_INVALID_ARG;
    for (uint32_t t = 0; t < n_moduli; ++t)
        if (mod->moduli[t] < 2 || mod->moduli[t] >= (1u << 30)) return VIPIR_ERR_INVALID_ARG;
    const uint32_t dl = db_bits / 8;
    if (cols > (1ull << 31) || (cols * dl) % 16 != 0) return VIPIR_ERR_UNSUPPORTED;
    const uint64_t kbytes = cols * dl;
    if (rows >= (1ull << 31) || kbytes >= (1ull << 31)) return VIPIR_ERR_UNSUPPORTED;
    const uint32_t T = n_moduli ? n_moduli : 1;
    if ((uint64_t)T * batch * 5 >= (1ull << 31)) return VIPIR_ERR_UNSUPPORTED;
    const uint32_t nq = T * batch;
    const uint32_t lc = (dl == 2 && n_moduli > 0) ? 5u : 4u;
    // ---- the one limit of this entry point: the limb planes have to fit the built-in array ----
    const uint64_t planes_bytes = (uint64_t)nq * lc * kbytes;
    if (planes_bytes > VIPIR_STATIC_SCRATCH_BYTES) {
        snprintf(g_cuda_err, sizeof g_cuda_err,
                 "vipir_dbmul_static: the query limb planes need %llu bytes (%u query vectors x %u limb columns x %llu "
                 "row bytes), the built-in scratch holds VIPIR_STATIC_SCRATCH_BYTES = %u; use a plan for this size",
                 (unsigned long long)planes_bytes, nq, lc, (unsigned long long)kbytes, (unsigned)VIPIR_STATIC_SCRATCH_BYTES);
        return VIPIR_ERR_UNSUPPORTED;
    }
    // ---- per-device set-up (first call on this device only) ----
    int dev = 0;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return VIPIR_ERR_UNSUPPORTED;
    unsigned char* scratch = nullptr;
    int sms = 0;
    int rc = static_scratch_setup(dev, &scratch, &sms);
    if (rc != VIPIR_OK) return rc;
    if ((2 + (size_t)sms) * sizeof(uint32_t) > kStaticSyncBytes) return VIPIR_ERR_UNSUPPORTED;

    // A plan that lives on this stack frame and points into the static array: nothing to allocate, nothing to free
    // (vipir_destroy must never see it).  The planner below is the one vipir_dbmul_plan uses; with d_sync already
    // set it skips its own cudaMalloc.
    vipir_plan pl;
    memset(&pl, 0, sizeof pl);
    pl.rows = rows;
    pl.cols = cols;
    pl.kbytes = kbytes;
    pl.batch = batch;
    pl.db_bits = db_bits;
    pl.dl = dl;
    pl.kdl = dl;
    pl.db_layout = VIPIR_DB_ROW_MAJOR;
    pl.n_moduli = n_moduli;
    for (uint32_t t = 0; t < n_moduli; ++t) pl.moduli[t] = mod->moduli[t];
    pl.nq = nq;
    pl.lc = lc;
    pl.num_sms = sms;
    pl.device = dev;
    pl.regime = ((uint64_t)nq * lc > 64 && rows > 128) ? VIPIR_REGIME_MMA_2SM : VIPIR_REGIME_MMA_1SM;
    pl.planes_bytes = planes_bytes;
    pl.d_sync = reinterpret_cast<uint32_t*>(scratch);
    pl.d_planes = scratch + kStaticSyncBytes;
    rc = plan_gemm(&pl, pl.regime == VIPIR_REGIME_MMA_2SM ? 2 : 1);
    if (rc != VIPIR_OK) return rc;

    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    // The array keeps whatever the previous call (or a call that was cut short) left in it.  The kernel expects its
    // counters to start at zero, so they are cleared on the caller's stream ahead of the kernel.  The planes need no
    // clearing: the splitter rewrites every byte the kernel will read.
    CK(cudaMemsetAsync(scratch, 0, kStaticSyncBytes, st));
    rc = launch_split(&pl, d_query, pl.d_planes, st);
    if (rc != VIPIR_OK) return rc;
    return scan_only(&pl, d_db, d_answer, st);
}

#include "modgemm_host.cuh"  // vipir_modgemm_* (parallel INT32 modular GEMMs, NEXT-4)
#include "ntt_host.cuh"      // vipir_ntt_* (lift + forward NTT producing G and H)
