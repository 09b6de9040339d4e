// modgemm_host.cuh -- host side (plan, dispatch, C ABI) of the parallel INT32 modular GEMMs
// Out = H*C + (0|G) mod q_t (include/vipir.h "vipir_modgemm_*"; kernels in modgemm_i8.cuh).
// Textually included at the end of vipir_api.cu: it uses that file's helpers (CK,
// get_encode_fn, g_cuda_err).
#pragma once
#include "modgemm_i8.cuh"

struct vipir_modgemm_plan {
    uint32_t T, M, K, Kp, ncols, gcols, cg;
    uint64_t NC, P;
    uint32_t moduli[VIPIR_MAX_MODULI];
    vipir_modgemm_tuning tune;  // explicit planner overrides; all zero = the planner's own choices
    int num_sms;
    int device;          // the device current at plan time: every call must come with it current
    uint8_t* d_hp;       // H byte limbs, interleaved per k-atom: [P*M][4*Kp]   (written by vipir_modgemm_set_h)
    uint8_t* d_cp;       // C limb planes: [P][4][ncols][Kp]                    (written every call)
    uint64_t hp_bytes, cp_bytes;
    bool h_set;
    bool fused;          // vipir_modgemm splits C inside the products kernel (from 16 columns up and K % 4 == 0): one launch
    vipir::ModGemmParams mg, mg_fused;
    uint32_t smem_bytes, smem_bytes_fused, grid;
    CUtensorMap tm_h, tm_c;
    CUtensorMap tm_c_raw;      // FUSED: the caller's raw C words [P][ncols][K] u32
    const void* tm_c_raw_for;  // d_C the cached tm_c_raw was encoded for
};

namespace {

int make_tmap_nd(CUtensorMap* m, const void* base, uint32_t rank, const uint64_t* dims, const uint64_t* strides_bytes,
                 const uint32_t* box, CUtensorMapDataType dt = CU_TENSOR_MAP_DATA_TYPE_UINT8) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) {
        snprintf(g_cuda_err, sizeof g_cuda_err, "cuTensorMapEncodeTiled entry point not found");
        return VIPIR_ERR_CUDA;
    }
    cuuint64_t d[5], s[4];
    cuuint32_t b[5], e[5];
    for (uint32_t i = 0; i < rank; ++i) {
        d[i] = dims[i];
        b[i] = box[i];
        e[i] = 1;
        if (i + 1 < rank) s[i] = strides_bytes[i];
    }
    CUresult r = fn(m, dt, rank, const_cast<void*>(base), d, s, b, e,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof g_cuda_err, "cuTensorMapEncodeTiled (rank %u) failed: CUresult %d", rank, (int)r);
        return VIPIR_ERR_CUDA;
    }
    return VIPIR_OK;
}

int plan_modgemm(vipir_modgemm_plan* p) {
    vipir::ModGemmParams& g = p->mg;
    memset(&g, 0, sizeof g);
    const uint32_t cg = p->cg;
    // N tile: ct C-columns (multiple of 8) -> MMA N = 4*ct <= 256, 7*ct accumulator columns <= 512.
    // Up to 32 columns a tile keeps two accumulator stages (2*7*32 = 448), so the drain of one
    // problem overlaps the products of the next.
    const uint32_t np8 = round_up(p->ncols, 8);
    uint32_t ct, n_tiles;
    if (np8 <= 32) {
        ct = np8;
        n_tiles = 1;
    } else {
        n_tiles = ceil_div(p->ncols, 64);
        ct = round_up(ceil_div(p->ncols, n_tiles), 8);
    }
    if (const uint32_t ct_force = p->tune.tile_cols) {
        ct = ct_force;
        n_tiles = ceil_div(p->ncols, ct);
    }
    g.P = (uint32_t)p->P;
    g.NC = (uint32_t)p->NC;
    g.M = p->M;
    g.ncols = p->ncols;
    g.gcols = p->gcols;
    g.ct = ct;
    g.n_tiles = n_tiles;
    g.m_tiles = ceil_div(p->M, 128u * cg);
    g.atoms = p->Kp / vipir::MG_BK;
    g.n_chunks = ceil_div(g.atoms, vipir::MG_MAX_CHUNK_ATOMS);
    g.atoms_per_chunk = ceil_div(g.atoms, g.n_chunks);
    g.b_stage_bytes = vipir::MG_BK * ct * (4 / cg);
    g.b_stages = p->tune.b_stages ? p->tune.b_stages : 3;
    // barrier area: 2 x 8 bytes per ring slot, 4 accumulator barriers, the TMEM base word (<= 640 bytes: the
    // tuning domain caps b_stages at 4 and a_stages at 24; the raw ring has at most 4 slots)
    const uint32_t overhead = 1024 /* alignment */ + vipir::MG_ZERO_BYTES + 640 /* barriers */;
    if (overhead + g.b_stages * g.b_stage_bytes + 4 * vipir::MG_A_BYTES > kMaxSmem) return VIPIR_ERR_UNSUPPORTED;
    const uint32_t left = kMaxSmem - overhead - g.b_stages * g.b_stage_bytes;
    g.a_stages = left / vipir::MG_A_BYTES;
    if (g.a_stages > 24) g.a_stages = 24;
    if (const uint32_t a_force = p->tune.a_stages) {
        if (a_force > g.a_stages) return VIPIR_ERR_UNSUPPORTED;
        g.a_stages = a_force;
    }
    if (g.a_stages < 4) return VIPIR_ERR_UNSUPPORTED;
    static_assert(16 * 24 + 16 * 4 + 16 * 4 + 36 <= 640, "barrier area");
    g.acc_stages = (2 * 7 * ct <= 512) ? 2u : 1u;
    uint32_t tc = 32;
    while (tc < g.acc_stages * 7 * ct) tc <<= 1;
    g.tmem_cols = tc;
    g.idesc = (2u << 4) /* D = s32 */ | (0u << 7) /* A = u8 */ | (0u << 10) /* B = u8 */ | (((4 * ct) >> 3) << 17) |
              (((128u * cg) >> 4) << 24);
    for (uint32_t t = 0; t < p->T; ++t) {
        const uint32_t q = p->moduli[t];
        g.moduli[t] = q;
        for (int s = 0; s < 3; ++s) g.w[t][s] = (uint32_t)((1ull << (32 + 8 * s)) % q);
        g.barrett[t] = (uint64_t)((((unsigned __int128)1) << 64) / q);
    }
    p->smem_bytes = g.a_stages * vipir::MG_A_BYTES + g.b_stages * g.b_stage_bytes + overhead;
    // (The two-kernel parameters above are planned and checked for every plan -- vipir_modgemm_split_c + _products may be
    // called on a one-kernel plan too.  That never refuses a shape or an override the one-kernel form could run: the
    // two-kernel form has no raw ring and at most as many operand slots, so whenever the checks below pass, those did.)
    // the fused kernel: two operand slots, two to four raw-tile slots (ct columns x 128 words each), the rest to the H ring
    p->mg_fused = g;
    if (p->fused) {
        vipir::ModGemmParams& f = p->mg_fused;
        // every CTA brings the raw words of the whole tile, per k-atom four 32-word boxes of ct rows (a multiple of
        // 1 KiB, so every box starts on a swizzle atom).  The raw tiles are requested r_stages - 1 k-atoms ahead of
        // the H boxes (modgemm_i8.cuh), which makes the H ring's depth uncritical (64 columns: 4.94 / 4.95 / 4.92 ms
        // with 4 / 6 / 8 H boxes); what pays is the depth of the converted-operand ring, which decouples the
        // converters from the MMA issuer: at 64 columns b = 2 / 3 with r = 2: 4.95 / 4.59 ms, r = b = 3 (5 H boxes)
        // 4.50 ms, b = 4 no better; at 32 columns r = b = 4: 3.40 against 3.48 ms.  So: four and four slots when
        // eight H boxes remain, else three and three with at least five, else three and two, else two and two.
        f.r_stage_bytes = 4 * ct * 128;
        auto fits = [&](uint32_t r, uint32_t b, uint32_t a) {
            return overhead + b * f.b_stage_bytes + r * f.r_stage_bytes + a * vipir::MG_A_BYTES <= kMaxSmem;
        };
        if (fits(4, 4, 8)) f.r_stages = 4, f.b_stages = 4;
        else if (fits(3, 3, 5)) f.r_stages = 3, f.b_stages = 3;
        else if (fits(2, 3, 6)) f.r_stages = 2, f.b_stages = 3;
        else f.r_stages = 2, f.b_stages = 2;
        if (p->tune.b_stages) f.b_stages = p->tune.b_stages;
        if (p->tune.r_stages) f.r_stages = p->tune.r_stages;
        const uint32_t fixed = overhead + f.b_stages * f.b_stage_bytes + f.r_stages * f.r_stage_bytes;
        if (fixed + 4 * vipir::MG_A_BYTES > kMaxSmem) return VIPIR_ERR_UNSUPPORTED;
        f.a_stages = (kMaxSmem - fixed) / vipir::MG_A_BYTES;
        if (f.a_stages > 24) f.a_stages = 24;
        if (const uint32_t a_force = p->tune.a_stages) {
            if (a_force > f.a_stages) return VIPIR_ERR_UNSUPPORTED;
            f.a_stages = a_force;
        }
        p->smem_bytes_fused = f.a_stages * vipir::MG_A_BYTES + fixed;
    }
    const uint64_t units = (uint64_t)p->P * g.m_tiles * g.n_tiles;
    if (units >= (1ull << 31)) return VIPIR_ERR_UNSUPPORTED;
    const uint32_t max_units = (uint32_t)p->num_sms / cg;
    p->grid = (uint32_t)(units < max_units ? units : max_units) * cg;

    // H limbs: byte matrix [P][M][4*Kp]; box = 128 B x 128 rows of one problem
    {
        const uint64_t dims[3] = {4ull * p->Kp, p->M, p->P};
        const uint64_t str[2] = {4ull * p->Kp, 4ull * p->Kp * p->M};
        const uint32_t box[3] = {vipir::MG_BK, vipir::MG_BM, 1};
        int rc = make_tmap_nd(&p->tm_h, p->d_hp, 3, dims, str, box);
        if (rc != VIPIR_OK) return rc;
    }
    return VIPIR_OK;
}

// C limb planes [P][4][ncols][Kp]; box = 128 B x ct columns x (4/cg) planes of one problem
int ensure_c_planes(vipir_modgemm_plan* p) {
    if (p->d_cp) return VIPIR_OK;
    if (cudaMalloc(&p->d_cp, p->cp_bytes) != cudaSuccess) {
        cudaGetLastError();
        return VIPIR_ERR_ALLOC;
    }
    const uint64_t dims[4] = {p->Kp, p->ncols, 4, p->P};
    const uint64_t str[3] = {p->Kp, (uint64_t)p->Kp * p->ncols, 4ull * p->Kp * p->ncols};
    const uint32_t box[4] = {vipir::MG_BK, p->mg.ct, 4 / p->cg, 1};
    return make_tmap_nd(&p->tm_c, p->d_cp, 4, dims, str, box);
}

template <int CG, bool FUSED>
int launch_modgemm(vipir_modgemm_plan* p, const vipir::ModGemmParams& g, cudaStream_t st) {
    auto kern = vipir::modgemm_i8_kernel<CG, FUSED>;
    static thread_local uint64_t attr_set = 0;  // bit d: done on device d
    if (attr_needed(attr_set)) {
        CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem));
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p->grid);
    cfg.blockDim = dim3(vipir::MG_THREADS);
    cfg.dynamicSmemBytes = FUSED ? p->smem_bytes_fused : p->smem_bytes;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CG;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    CK(cudaLaunchKernelEx(&cfg, kern, p->tm_h, FUSED ? p->tm_c_raw : p->tm_c, g));
    return VIPIR_OK;
}

template <bool INTERLEAVED>
int launch_mg_split(const uint32_t* src, uint8_t* dst, uint64_t n_rows, uint32_t R, uint32_t K, uint32_t Kp,
                    cudaStream_t st) {
    const uint64_t threads = n_rows * (Kp / 16);
    const uint64_t blocks = (threads + 255) / 256;
    if (blocks >= (1ull << 31)) return VIPIR_ERR_UNSUPPORTED;
    vipir::mg_split_kernel<INTERLEAVED><<<(uint32_t)blocks, 256, 0, st>>>(src, dst, n_rows, R, K, Kp);
    CK(cudaGetLastError());
    return VIPIR_OK;
}

}  // namespace

extern "C" {

int vipir_modgemm_plan_create(vipir_modgemm_plan** out, uint32_t T, uint64_t NC, uint32_t M, uint32_t K, uint32_t ncols,
                              uint32_t gcols, const uint32_t* moduli) {
    return vipir_modgemm_plan_create_tuned(out, T, NC, M, K, ncols, gcols, moduli, nullptr);
}

int vipir_modgemm_plan_create_tuned(vipir_modgemm_plan** out, uint32_t T, uint64_t NC, uint32_t M, uint32_t K,
                                    uint32_t ncols, uint32_t gcols, const uint32_t* moduli,
                                    const vipir_modgemm_tuning* tune) {
    if (!out) return VIPIR_ERR_INVALID_ARG;
    *out = nullptr;
    if (tune) {
        if (tune->cta_group > 2 || tune->tile_cols > 64 || tune->tile_cols % 8 != 0 || tune->b_stages == 1 ||
            tune->b_stages > 4 || (tune->a_stages != 0 && tune->a_stages < 4) || tune->a_stages > 24 ||
            tune->c_split > 2 || tune->r_stages == 1 || tune->r_stages > 4)
            return VIPIR_ERR_INVALID_ARG;
        for (uint32_t r : tune->reserved)
            if (r != 0) return VIPIR_ERR_INVALID_ARG;
    }
    if (!moduli || T == 0 || T > VIPIR_MAX_MODULI || NC == 0 || M == 0 || K == 0 || ncols == 0 || gcols > ncols)
        return VIPIR_ERR_INVALID_ARG;
    for (uint32_t t = 0; t < T; ++t)
        if (moduli[t] < 2 || moduli[t] >= (1u << 30)) return VIPIR_ERR_INVALID_ARG;
    if (M >= (1u << 24) || K >= (1u << 24) || ncols >= (1u << 24) || NC >= (1ull << 28)) return VIPIR_ERR_UNSUPPORTED;

    int dev = 0;
    CK(cudaGetDevice(&dev));
    int major = 0, minor = 0, sms = 0;
    CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    CK(cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10 || minor != 0) return VIPIR_ERR_ARCH;

    vipir_modgemm_plan* p = new (std::nothrow) vipir_modgemm_plan;
    if (!p) return VIPIR_ERR_ALLOC;
    memset(p, 0, sizeof *p);
    p->T = T;
    p->NC = NC;
    p->P = (uint64_t)T * NC;
    p->M = M;
    p->K = K;
    p->Kp = round_up(K, vipir::MG_BK);
    p->ncols = ncols;
    p->gcols = gcols;
    p->num_sms = sms;
    p->device = dev;
    for (uint32_t t = 0; t < T; ++t) p->moduli[t] = moduli[t];
    if (tune) p->tune = *tune;
    // CTA pairs (one 256-row tile, each CTA staging half of the C limb tile) once the C tile is wide
    // enough for its shared-memory traffic to matter
    p->cg = (M > 128 && ncols >= 16) ? 2u : 1u;  // measured: pairs win from 16 columns up (8 clients: 2.64 -> 2.55 ms)
    if (p->tune.cta_group) p->cg = p->tune.cta_group;
    // One kernel (C split into limbs inside the products kernel) or two (a splitter pre-pass writes C's limb planes).
    // The raw-C tensor map needs 16-byte row strides: K % 4 == 0 (the paper's n = 1280).  Measured at the paper's shape
    // (sustained, same run): 64 columns 4.95 against 5.6 ms, 16 columns 3.01 against 2.93 ms, 2 columns 2.51 against
    // 2.42 ms -- the pre-pass costs 2 * 4 bytes per word of C, the fused form a longer dependency chain per k-atom.
    // With the raw tiles requested ahead and deeper operand rings (plan_modgemm): 64 columns 4.50 against 5.4 ms,
    // 32 columns 3.40 against 3.64, 16 columns 2.91 against 2.94, 2 columns 2.48 against 2.42: fused from 16 columns up.
    if (p->tune.c_split == 2 && K % 4 != 0) {
        delete p;
        return VIPIR_ERR_UNSUPPORTED;
    }
    p->fused = p->tune.c_split ? p->tune.c_split == 2 : (K % 4 == 0 && ncols >= 16);
    if (p->tune.r_stages && !p->fused) {  // the raw-tile ring exists in the one-kernel form only: refused, not ignored
        delete p;
        return VIPIR_ERR_UNSUPPORTED;
    }
    p->hp_bytes = p->P * M * 4ull * p->Kp;
    p->cp_bytes = p->P * 4ull * ncols * p->Kp;
    // the C limb planes are only needed by the two-kernel form: allocated here when that is the plan's form,
    // else on the first vipir_modgemm_split_c
    if (cudaMalloc(&p->d_hp, p->hp_bytes) != cudaSuccess) {
        cudaGetLastError();
        vipir_modgemm_destroy(p);
        return VIPIR_ERR_ALLOC;
    }
    int rc = plan_modgemm(p);
    if (rc == VIPIR_OK && !p->fused) rc = ensure_c_planes(p);
    if (rc != VIPIR_OK) {
        vipir_modgemm_destroy(p);
        return rc;
    }
    *out = p;
    return VIPIR_OK;
}

int vipir_modgemm_set_h(vipir_modgemm_plan* p, const uint32_t* d_H, void* cuda_stream) {
    if (!p || !d_H || (reinterpret_cast<uintptr_t>(d_H) & 15)) return VIPIR_ERR_INVALID_ARG;
    if (!on_device(p->device)) return VIPIR_ERR_INVALID_ARG;
    int rc = launch_mg_split<true>(d_H, p->d_hp, p->P * p->M, p->M, p->K, p->Kp, static_cast<cudaStream_t>(cuda_stream));
    if (rc == VIPIR_OK) p->h_set = true;
    return rc;
}

int vipir_modgemm_split_c(vipir_modgemm_plan* p, const uint32_t* d_C, void* cuda_stream) {
    if (!p || !d_C || (reinterpret_cast<uintptr_t>(d_C) & 15)) return VIPIR_ERR_INVALID_ARG;
    if (!on_device(p->device)) return VIPIR_ERR_INVALID_ARG;
    int rc = ensure_c_planes(p);
    if (rc != VIPIR_OK) return rc;
    return launch_mg_split<false>(d_C, p->d_cp, p->P * p->ncols, p->ncols, p->K, p->Kp,
                                  static_cast<cudaStream_t>(cuda_stream));
}

namespace {
int check_products_args(const vipir_modgemm_plan* p, const uint32_t* d_G, const uint32_t* d_Out) {
    if (!p || !d_Out || (p->gcols > 0 && !d_G)) return VIPIR_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_Out) & 3) || (reinterpret_cast<uintptr_t>(d_G) & 3)) return VIPIR_ERR_INVALID_ARG;
    if (!p->h_set) return VIPIR_ERR_INVALID_ARG;
    if (!on_device(p->device)) return VIPIR_ERR_INVALID_ARG;
    return VIPIR_OK;
}
}  // namespace

int vipir_modgemm_products(vipir_modgemm_plan* p, const uint32_t* d_G, uint32_t* d_Out, void* cuda_stream) {
    int rc = check_products_args(p, d_G, d_Out);
    if (rc != VIPIR_OK) return rc;
    if (!p->d_cp) return VIPIR_ERR_INVALID_ARG;  // no limb planes yet: vipir_modgemm_split_c first
    vipir::ModGemmParams g = p->mg;  // per-call values go into a copy
    g.G = d_G;
    g.out = d_Out;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    return p->cg == 2 ? launch_modgemm<2, false>(p, g, st) : launch_modgemm<1, false>(p, g, st);
}

int vipir_modgemm(vipir_modgemm_plan* p, const uint32_t* d_C, const uint32_t* d_G, uint32_t* d_Out, void* cuda_stream) {
    if (!p || !d_C || (reinterpret_cast<uintptr_t>(d_C) & 15)) return VIPIR_ERR_INVALID_ARG;
    if (!p->fused) {
        int rc = vipir_modgemm_split_c(p, d_C, cuda_stream);
        if (rc != VIPIR_OK) return rc;
        return vipir_modgemm_products(p, d_G, d_Out, cuda_stream);
    }
    int rc = check_products_args(p, d_G, d_Out);
    if (rc != VIPIR_OK) return rc;
    if (p->tm_c_raw_for != d_C) {
        // the caller's C as it lies: [P][ncols][K] u32; box = 32 words x ct columns of one problem, 128B swizzle
        const uint64_t dims[3] = {p->K, p->ncols, p->P};
        const uint64_t str[2] = {4ull * p->K, 4ull * p->K * p->ncols};
        const uint32_t box[3] = {32, p->mg.ct, 1};
        rc = make_tmap_nd(&p->tm_c_raw, d_C, 3, dims, str, box, CU_TENSOR_MAP_DATA_TYPE_UINT32);
        if (rc != VIPIR_OK) return rc;
        p->tm_c_raw_for = d_C;
    }
    vipir::ModGemmParams g = p->mg_fused;
    g.G = d_G;
    g.out = d_Out;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    return p->cg == 2 ? launch_modgemm<2, true>(p, g, st) : launch_modgemm<1, true>(p, g, st);
}

int vipir_modgemm_info(const vipir_modgemm_plan* p, vipir_modgemm_info_t* o) {
    if (!p || !o) return VIPIR_ERR_INVALID_ARG;
    memset(o, 0, sizeof *o);
    o->problems = p->P;
    o->k_padded = p->Kp;
    o->cta_group = p->cg;
    o->tile_cols = p->mg.ct;
    o->mma_n = 4 * p->mg.ct;
    o->m_tiles = p->mg.m_tiles;
    o->n_tiles = p->mg.n_tiles;
    o->n_chunks = p->mg.n_chunks;
    const vipir::ModGemmParams& g = p->fused ? p->mg_fused : p->mg;
    o->a_stages = g.a_stages;
    o->b_stages = g.b_stages;
    o->acc_stages = g.acc_stages;
    o->r_stages = p->fused ? g.r_stages : 0;
    o->smem_bytes = p->fused ? p->smem_bytes_fused : p->smem_bytes;
    o->grid = p->grid;
    o->launches = p->fused ? 1 : 2;
    o->fused_split = p->fused ? 1 : 0;
    o->h_limb_bytes = p->hp_bytes;
    o->c_limb_bytes = p->d_cp ? p->cp_bytes : 0;
    return VIPIR_OK;
}

int vipir_testing_modgemm_limbs(const vipir_modgemm_plan* p, void** d_h_limbs, void** d_c_limbs) {
    if (!p || !d_h_limbs || !d_c_limbs) return VIPIR_ERR_INVALID_ARG;
    *d_h_limbs = p->d_hp;
    *d_c_limbs = p->d_cp;
    return VIPIR_OK;
}

void vipir_modgemm_destroy(vipir_modgemm_plan* p) {
    if (!p) return;
    if (p->d_hp) cudaFree(p->d_hp);
    if (p->d_cp) cudaFree(p->d_cp);
    delete p;
}

}  // extern "C"
