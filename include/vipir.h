/*
 * vipir.h -- C ABI of libvipir: the VIPIR PIR server's database scan on one B200.
 *
 *     answer = D * Q  mod q
 *
 * the "D1 x B x D0 INT8-INT32 GEMM for a batch of B queries" that is the server's online
 * step (arxiv/paper_2606_11536, section 2.5), with the plaintext database
 * D (rows x cols small unsigned integers) and the encrypted query matrix Q (u32 words).
 * Modulus: q = 2^32, "modulo-2^32 operations as in SimplePIR ... modular reduction
 * effectively becomes free" (section 4), or per-prime RNS residues, "each row
 * corresponds to a different q_i" (section 2.3).  The method is the paper's
 * limb decomposition A*B = sum_j 2^(8j) (A*B_j) over 8-bit query limbs (PAPER.md:245-249
 * section 4.1) on int8 tensor cores (batched) or CUDA cores (batch 1).
 *
 * Definition of the result (bit-exact; no tolerance).  For modulus index t < T, query b < batch,
 * row r < rows:
 *     answer[t][b][r] = ( sum_{k < cols} D[r][k] * Q[t][b][k] )  mod q_t
 * D[r][k] the UNSIGNED value of the element (signed int8 after vipir_plan_set_db_signed), Q the unsigned 32-bit word (any u32 is legal,
 * also >= q_t), the sum over the integers, the result canonical in [0, q_t).
 * T = max(mod.count, 1); mod.count == 0 selects q = 2^32.
 *
 * Layouts (all dense, no pitch):
 *   d_db      rows x cols, row-major (cols contiguous), uint8, or little-endian uint16 when
 *             db_bits == 16.  DEVICE pointer, 16-byte aligned.  cols * db_bits/8 must be a
 *             multiple of 16 bytes.  (A uint16 database may instead be handed over as its two
 *             byte-limb planes, prepared once by vipir_db_split_u16: vipir_db_layout below.)
 *   d_query   [T][batch][cols] uint32 -- each query vector contiguous.  DEVICE pointer, 16-byte aligned.
 *   d_answer  [T][batch][rows] uint32.  DEVICE pointer.
 * Ownership: the caller owns d_db, d_query, d_answer (they must not overlap and must stay
 * valid until the stream has run the call); the plan owns its workspace (query limb planes,
 * host-call staging) and frees it in vipir_destroy.
 *
 * Execution: vipir_dbmul only ENQUEUES work on `cuda_stream` (a cudaStream_t / CUstream passed
 * as void*, NULL = legacy default stream): no host synchronisation, no allocation.  One plan
 * must not be in flight on two streams at once, nor be used from two host threads at once: it
 * owns one limb-plane workspace, one set of staging buffers and cached tensor maps.  (Per-call
 * values -- the answer pointer, the modulus-switch and signedness flags in effect -- are passed
 * to the kernels by value; the planned parameters are never rewritten by a call.)  A server
 * that overlaps requests makes one plan per stream.  After one call outside the capture (which
 * sets kernel attributes and encodes the tensor maps for these buffers) a vipir_dbmul call can be
 * captured into a CUDA graph and replayed: the kernels reset their own work counters.  All
 * kernels are sm_100a; there is no fallback of any kind.  A plan (of any of the three kinds in this header) belongs to
 * the device that was current when it was made -- its workspace, tensor maps and streams live there -- and every call
 * that takes it must come with that device current: under another one it returns VIPIR_ERR_INVALID_ARG and
 * enqueues nothing (a process that drives several GPUs, makes one plan per GPU).
 *
 * Errors: every entry point returns a vipir_status (0 = OK) and never throws or aborts.
 */
#ifndef VIPIR_H
#define VIPIR_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vipir_plan vipir_plan; /* opaque, owned by the library */

typedef enum {
    VIPIR_OK = 0,
    VIPIR_ERR_INVALID_ARG = 1, /* null pointer, zero size, db_bits not 8/16, modulus < 2 or >= 2^30, count > 4 */
    VIPIR_ERR_UNSUPPORTED = 2, /* row bytes not a multiple of 16, size beyond a stated limit, regime cannot run this shape */
    VIPIR_ERR_ALLOC = 3,       /* host or device allocation failed */
    VIPIR_ERR_CUDA = 4,        /* a CUDA call failed (no device, launch error, ...) */
    VIPIR_ERR_ARCH = 5         /* the current device is not compute capability 10.0 (B200) */
} vipir_status;

#define VIPIR_MAX_MODULI 4u

typedef struct {
    uint32_t count;         /* 0 => q = 2^32 (wrapping); else number of moduli (<= VIPIR_MAX_MODULI) */
    const uint32_t *moduli; /* HOST pointer to `count` values, each 2 <= m < 2^30; copied by the plan */
} vipir_modulus_spec;

/* Kernel regimes.  AUTO picks GEMV for one wrapping query vector,
 * otherwise the tensor-core path (1-SM tiles up to 16 query vectors, 2-SM pairs
 * above).  NAIVE is a test-only check kernel and is never picked by AUTO. */
typedef enum {
    VIPIR_REGIME_AUTO = 0,
    VIPIR_REGIME_GEMV = 1,    /* step a2: CUDA-core dp4a scan, batch 1, q = 2^32 only */
    VIPIR_REGIME_MMA_1SM = 2, /* steps a3-a5: tcgen05.mma.cta_group::1.kind::i8 */
    VIPIR_REGIME_MMA_2SM = 3, /* steps a3-a5: tcgen05.mma.cta_group::2.kind::i8, CTA pairs */
    VIPIR_REGIME_NAIVE = 4
} vipir_regime;

/* Layout of the database in device memory.  ROW_MAJOR: rows x cols
 * elements, u8 or little-endian u16, as the caller holds it.  LIMB_PLANES (u16 only; BASELINE.json
 * configs[4]: "uint16 ... (split into 2 u8 limbs)"): the two byte matrices D_lo[r][k] = D[r][k] & 0xFF
 * and D_hi[r][k] = D[r][k] >> 8, each rows x cols u8 row-major, D_hi directly behind D_lo
 * (2*rows*cols bytes) -- written once, offline, by vipir_db_split_u16; the DB of a PIR server is
 * static and resident in GPU DRAM, prepared like the hint. */
typedef enum { VIPIR_DB_ROW_MAJOR = 0, VIPIR_DB_LIMB_PLANES = 1 } vipir_db_layout;

typedef struct {
    uint32_t regime;          /* the regime in effect (never AUTO) */
    uint32_t db_limbs;        /* dl: 1 (u8) or 2 (u16) */
    uint32_t limb_cols;       /* LC: accumulator columns per query vector (4; 5 for a row-major u16 DB with prime moduli) */
    uint32_t query_vectors;   /* T * batch */
    uint64_t k_bytes;         /* K' = cols * dl: bytes per DB row (LIMB_PLANES: cols, the bytes per row of one limb plane) */
    uint32_t k_chunk_bytes;   /* K' bytes per int32 accumulation chunk (<= 32768); 0 for GEMV/NAIVE */
    uint32_t n_chunks;
    uint32_t tile_queries;    /* query vectors per N tile (MMA regimes) */
    uint32_t tile_cols;       /* accumulator columns per tile = tile_queries * LC */
    uint32_t mma_n;           /* N of one tcgen05.mma */
    uint32_t m_tiles, n_tiles; /* a work unit = one (M tile, N tile); units x n_chunks work items are dealt to the CTAs */
    uint32_t stages;          /* shared-memory ring depth */
    uint32_t smem_bytes;      /* dynamic shared memory per CTA */
    uint32_t grid;            /* CTAs launched by the main kernel */
    uint32_t launches;        /* kernels enqueued per vipir_dbmul call */
    uint64_t workspace_bytes; /* limb planes [query_vectors*LC][K'] u8, owned by the plan */
    uint32_t modswitch_bits;  /* fused output modulus switch in effect (0 = off) */
    uint32_t db_signed;       /* 1 if the DB elements are read as two's-complement int8 (vipir_plan_set_db_signed) */
    uint32_t m_sub;           /* MMA regimes: 128-row DB sub-tiles per CTA and tile (rows per tile = 128 * CTAs * m_sub;
                                 LIMB_PLANES: the two limb tiles of a row block count as two sub-tiles) */
    uint32_t db_layout;       /* vipir_db_layout the plan expects d_db in */
    uint32_t leftover_chunks; /* MMA: K chunks of a unit of the last, partial round (== n_chunks unless cut finer) */
} vipir_info;

/*
 * Build a plan for one problem shape (host only; allocates the limb-plane workspace on the
 * current device and picks regime, tiles and K chunks).  SimplePIR shapes: rows = D1,
 * cols = D0, batch = B.
 *   out      receives the plan (NULL on failure)
 *   db_bits  8 or 16
 *   mod      NULL or count == 0 for q = 2^32
 * Errors: INVALID_ARG, UNSUPPORTED (cols*db_bits/8 % 16 != 0; rows or cols*db_bits/8 >= 2^31;
 * T*batch*5 >= 2^31), ARCH, ALLOC, CUDA.
 */
int vipir_dbmul_plan(vipir_plan **out, uint64_t rows, uint64_t cols, uint32_t batch, uint32_t db_bits,
                     const vipir_modulus_spec *mod);

/* Same, forcing a regime (tests, benchmarks).  UNSUPPORTED if the regime cannot run the shape
 * (GEMV needs T*batch == 1 and q = 2^32). */
int vipir_dbmul_plan_ex(vipir_plan **out, uint64_t rows, uint64_t cols, uint32_t batch, uint32_t db_bits,
                        const vipir_modulus_spec *mod, uint32_t regime);

/*
 * Same, for a database held in `db_layout` (vipir_db_layout).  With VIPIR_DB_LIMB_PLANES the d_db
 * passed to vipir_dbmul / vipir_dbmul_scan / vipir_dbmul_host is the buffer vipir_db_split_u16
 * wrote; the answer is that of the u16 database it was made from, bit for bit.  The tensor-core
 * kernel then runs 8 int8 MACs per u16 x u32 product (two DB limbs x four query limbs)
 * against four limb-plane columns per query vector, instead of the 10 and 5 of the byte view of an
 * interleaved u16 row (DESIGN.md sections 5, 14).
 * Errors: as vipir_dbmul_plan_ex; INVALID_ARG (unknown layout); UNSUPPORTED (LIMB_PLANES with
 * db_bits != 16, with the GEMV or NAIVE regime, with cols % 16 != 0, or with rows >= 2^30).
 */
int vipir_dbmul_plan_layout(vipir_plan **out, uint64_t rows, uint64_t cols, uint32_t batch, uint32_t db_bits,
                            const vipir_modulus_spec *mod, uint32_t regime, uint32_t db_layout);

/*
 * Explicit planner overrides (DESIGN.md section 6 "Regimes" and "M sub-tiles"): every field 0 = the planner's own
 * choice, so a zeroed struct (or tune == NULL) is vipir_dbmul_plan_layout.  They select between code paths that
 * all compute the same, bit-exact answer -- for tests that must reach each path and for measurements; nothing
 * in the library reads the environment.  A value outside a field's domain is INVALID_ARG; a value the shape or
 * regime cannot honour (for example m_sub * tile_cols > 512 TMEM columns) is UNSUPPORTED -- never silently ignored.
 */
typedef struct {
    uint32_t m_sub;          /* MMA: 128-row DB sub-tiles per CTA and tile: 1, 2 or 4 */
    uint32_t tile_queries;   /* MMA: query vectors per N tile (a multiple of 4; of 16 when limb_cols == 5), <= 128 */
    uint32_t k_atoms;        /* MMA: 128-byte k-atoms per pipeline stage, 1..8 (lowered until two stages fit) */
    uint32_t stages;         /* shared-memory ring depth: MMA 2..12 (at most what fits), GEMV 2..6 */
    uint32_t min_chunks;     /* MMA: cut K into this many equal chunks of whole k-atoms instead of the fewest that respect the
                                int32 bound (finer work items; <= number of k-atoms; fewer when the k-atoms do not divide
                                that way: 6 k-atoms in "4" chunks are 3 chunks of 2) */
    uint32_t separate_split; /* GEMV: 1 = always run the query-limb splitter as its own kernel (two launches) */
    uint32_t whole_units;    /* MMA: 1 = deal the last, partial round of work units out whole, not chunk by chunk */
    uint32_t no_collector;   /* MMA: 1 = the second N half re-reads the DB operand from shared memory */
    uint32_t host_staged;    /* vipir_dbmul_host: 1 = always stage the answer in device memory and copy it back
                                (no direct stores into mapped host memory, no overlapped copies) */
    uint32_t host_slices;    /* vipir_dbmul_host, MMA: K slices of the copy / split / scan pipeline, 1..4 (0: three for
                                queries of 8 MiB and more, else one); UNSUPPORTED for a GEMV plan */
    uint32_t leftover_chunks; /* MMA: cut the units of the last, partial round (units mod CTA groups of them) into this many
                                K chunks, so that the round can be dealt out evenly; >= the plan's n_chunks, <= k-atoms;
                                UNSUPPORTED with whole_units.  0: the planner's rule (finer only where it shortens that
                                round by a fifth or more) */
    uint32_t reserved[5];    /* must be 0 */
} vipir_tuning;

/* vipir_dbmul_plan_layout with explicit planner overrides.  Errors: as vipir_dbmul_plan_layout; INVALID_ARG
 * (a field outside its domain, reserved != 0); UNSUPPORTED (an override this shape / regime cannot honour). */
int vipir_dbmul_plan_tuned(vipir_plan **out, uint64_t rows, uint64_t cols, uint32_t batch, uint32_t db_bits,
                           const vipir_modulus_spec *mod, uint32_t regime, uint32_t db_layout,
                           const vipir_tuning *tune);

/*
 * Offline, once per database: de-interleave a u16 DB (rows x cols, row-major, little-endian) into
 * the VIPIR_DB_LIMB_PLANES form.  d_db_u16, d_db_planes: DEVICE pointers, 16-byte aligned,
 * 2*rows*cols bytes each, caller-owned, not overlapping.  Enqueues one kernel on `cuda_stream`.
 * Errors: INVALID_ARG (null / misaligned / overlapping pointers, zero sizes), UNSUPPORTED
 * (cols % 16 != 0, rows or cols >= 2^31), CUDA.
 */
int vipir_db_split_u16(const void *d_db_u16, void *d_db_planes, uint64_t rows, uint64_t cols, void *cuda_stream);

/*
 * Enqueue answer = D * Q mod q on `cuda_stream`: the query-limb splitter
 * followed by the scan kernel of the plan's regime -- or, for the batch-1 scan of a u8 DB whose cols
 * are a multiple of 32, ONE kernel that splits the query words as it reads them (vipir_info.launches
 * says which).  All three pointers are DEVICE pointers.
 * Errors: INVALID_ARG (null / misaligned pointer), CUDA.
 */
int vipir_dbmul(vipir_plan *plan, const void *d_db, const uint32_t *d_query, uint32_t *d_answer,
                void *cuda_stream);

/*
 * End-to-end variant with HOST query and answer buffers (the PIR server's per-request path:
 * queries arrive from clients, answers go back; the static DB stays resident on the GPU,
 * PAPER.md:176).  Copies h_query to the device, runs the product, delivers the answer to h_answer and
 * waits for the stream: the result is complete when the call returns.  h_query / h_answer: HOST
 * pointers with the d_query / d_answer layouts; d_db: DEVICE pointer.  The first call allocates device
 * staging, a copy stream and events, all owned by the plan.
 *   Pinned memory (cudaHostAlloc / cudaHostRegister) makes the copies asynchronous.  When h_answer is
 * pinned and device-mapped, the kernels write the finished answer words into it themselves while the scan
 * runs (batch 1: the scan's own stores; tensor-core regimes: two warps of every CTA copy each finished tile
 * from device staging) and no device-to-host copy is made.
 *   Tensor-core regimes: the call is pipelined over K slices (PAPER.md:245-249's K chunks, grouped): the
 * copy stream brings slice i's columns of every query vector and splits them into limbs while the caller's
 * stream scans slice i-1; every slice adds to the running sums (device staging).  Same answer, bit for bit,
 * as vipir_dbmul.  vipir_tuning.host_staged = 1 selects the plain form
 * (one copy in, vipir_dbmul, one copy out).
 */
int vipir_dbmul_host(vipir_plan *plan, const void *d_db, const uint32_t *h_query, uint32_t *h_answer,
                     void *cuda_stream);

/* Run only the query-limb splitter (step a1): d_query [T*batch][cols] u32 ->
 * byte planes [T*batch*LC][K'] u8 (layout: csrc/split_limbs.cuh) written to d_planes_out
 * (DEVICE, 16-byte aligned, workspace_bytes long), or into the plan's workspace if NULL. */
int vipir_split_limbs(vipir_plan *plan, const uint32_t *d_query, uint8_t *d_planes_out, void *cuda_stream);

/* Run only the scan kernel (steps a2 or a3+a4) against the limb planes already in the plan's
 * workspace (written by the last vipir_dbmul or vipir_split_limbs(plan, q, NULL, ...) call).
 * vipir_dbmul == vipir_split_limbs + vipir_dbmul_scan.  For per-kernel timing and tests. */
int vipir_dbmul_scan(vipir_plan *plan, const void *d_db, uint32_t *d_answer, void *cuda_stream);

/*
 * Fuse the scalar-HE modulus switch into the scan kernel's epilogue (section 5: the
 * ciphertext modulus 2^32 "is reduced to 2^18 after each scalar-HE folding step"
 * Appendix D.2): every answer word x becomes  round(x * 2^out_bits / 2^32) mod 2^out_bits  (ties
 * up), saving a pass over the answer.  out_bits in [1, 31]; 0 switches it off (the default).
 * Only for q = 2^32 plans.  Errors: INVALID_ARG (out_bits > 31), UNSUPPORTED (prime moduli, NAIVE).
 */
int vipir_plan_set_modswitch(vipir_plan *plan, uint32_t out_bits);

/*
 * Read the database elements as SIGNED two's-complement int8 instead of unsigned (centred
 * plaintexts: the paper's decryption range is m in [-p/2, p/2), Appendix A.1; a
 * centred DB halves the |m| <= p/2 factor of the LWE noise term sum_k m_k e_k):
 *     answer[t][b][r] = ( sum_k (int8)D[r][k] * Q[t][b][k] )  mod q_t,  canonical in [0, q_t).
 * The same bytes in HBM; the tensor-core path switches the A operand format of
 * tcgen05.mma.kind::i8 to s8, the batch-1 scan uses dp4a.s32.u32.  is_signed: 0 (default) or 1.
 * Errors: INVALID_ARG (null plan, is_signed > 1), UNSUPPORTED (db_bits == 16: the byte view of a
 * signed int16 mixes an unsigned low byte with a signed high byte in one operand).
 */
int vipir_plan_set_db_signed(vipir_plan *plan, uint32_t is_signed);

/* Describe the plan.  Errors: INVALID_ARG. */
int vipir_plan_info(const vipir_plan *plan, vipir_info *out);

/* Free the plan and its workspace.  vipir_destroy(NULL) is a no-op. */
void vipir_destroy(vipir_plan *plan);

/*
 * The batched product for callers that cannot allocate device memory: no plan, no cudaMalloc, no cudaFree, no
 * library routine that allocates -- the call only encodes tensor maps on the host and enqueues a memset and two
 * kernels on `cuda_stream`.  Same definition and the same answer, bit for bit, as vipir_dbmul
 * (answer = D * Q mod q, by the limb decomposition of PAPER.md:245-249).
 *
 * Who needs this.  A PIR server keeps the whole database resident in GPU DRAM, so a deployment
 * typically hands all device memory out once at start-up -- to the database and to one arena that some other
 * runtime owns -- and a later cudaMalloc from inside a library either fails or eats into that arena behind its
 * owner's back.  Request handlers on a latency budget are in the same position for another reason: cudaMalloc
 * and cudaFree may synchronise the whole device, which stalls every other request's stream while they run.
 * Such callers cannot build a vipir_plan (it allocates the query limb planes and a few counters); they call this.
 *
 * How it works.  The tensor-core kernel's scratch (the limb planes written by the query splitter, and its
 * work-distribution counters) lives in a fixed array inside the library image, 4 KiB + VIPIR_STATIC_SCRATCH_BYTES
 * (8 MiB) long.  Every GPU on which the library's kernels are loaded holds that array until the process exits,
 * whether or not this entry point is ever used.  The caller passes inputs and outputs only:
 *   rows, cols, batch, db_bits, mod   the shape, as for vipir_dbmul_plan (database row-major; q = 2^32 or primes)
 *   d_db, d_query, d_answer           DEVICE pointers with vipir_dbmul's layouts, alignment and ownership rules
 * Always the tensor-core kernel (1-SM tiles or CTA pairs by AUTO's rule), also for batch 1, where a plan would
 * pick the faster GEMV regime.
 *
 * Limit.  The limb planes must fit: T * batch * LC * cols * db_bits/8 <= VIPIR_STATIC_SCRATCH_BYTES
 * (LC = 4; 5 for a u16 database with prime moduli).  For a u8 database that is 256 query vectors at cols = 8192,
 * 16 at cols = 131072.  Anything larger returns VIPIR_ERR_UNSUPPORTED before any device work, and
 * vipir_last_cuda_error() then holds a sentence with the bytes needed and the bytes available.
 *
 * First call on each device: looks up the array's address on that device (the current device must be the one the
 * pointers belong to) and sets the kernels' shared-memory attribute.  Make that first call during start-up, before
 * any stream capture begins.  Later calls skip the set-up.
 *
 * Shared state.  All calls on one GPU -- from any thread, on any stream -- use the same array, and it keeps the
 * previous call's contents.  The call clears the counters itself (on `cuda_stream`, ahead of the kernels) and the
 * splitter overwrites every plane byte the scan reads, so a stale array is harmless; but two calls whose GPU work
 * overlaps in time race on it and both answers are undefined.  Issue them on one stream, or order the streams with
 * events.  The call does not wait for the GPU: d_answer is valid once `cuda_stream` has run it.
 *
 * Errors: INVALID_ARG and UNSUPPORTED as for vipir_dbmul_plan / vipir_dbmul, UNSUPPORTED for the size limit above or
 * a device ordinal >= 64, ARCH, CUDA.  Never ALLOC.
 */
#define VIPIR_STATIC_SCRATCH_BYTES (8u << 20)
int vipir_dbmul_static(uint64_t rows, uint64_t cols, uint32_t batch, uint32_t db_bits, const vipir_modulus_spec *mod,
                       const void *d_db, const uint32_t *d_query, uint32_t *d_answer, void *cuda_stream);

/* Static string for a status code. */
const char *vipir_status_str(int status);

/* Last CUDA error string recorded by this library on the calling thread ("" if none). */
const char *vipir_last_cuda_error(void);

/* ===========================================================================================
 * Parallel INT32 modular GEMMs of the ring-packing stage
 *
 *     Out = H * C + (0 | G)   mod q_t
 *
 * PAPER.md:216 (section 3.5.2): after the NTTs, Tiptoe-style packing (eq. (3))
 * "reduces to (#RNS * N)-parallel ceil(D1/N) x 2B x n INT32 GEMMs with additional modular
 * reduction computations"; PAPER.md:261-265 (section 4.2) gives the paper's CUDA-core method
 * (tile-major layout, lazy reduction).  Here the products run on the int8 tensor cores with
 * both operands split into 8-bit limbs and ONE modular reduction per output word
 * (csrc/modgemm_i8.cuh).
 *
 * One problem per (modulus t < T, NTT coefficient c < NC): an M x ncols x K product of 32-bit
 * words mod q_t (M = ceil(D1/N), K = n, ncols = 2B), plus G added to the LAST gcols columns.
 * Definition (bit-exact): for t, c, column j < ncols, row m < M
 *   Out[t][c][j][m] = ( sum_{k<K} H[t][c][m][k] * C[t][c][j][k]
 *                       + (j >= ncols-gcols ? G[t][c][j-(ncols-gcols)][m] : 0) )  mod q_t
 * over the integers, canonical in [0, q_t).  Any u32 input word is legal (also >= q_t).
 *
 * Layouts (dense uint32, DEVICE pointers, 16-byte aligned; "tile-major": every problem's
 * operands contiguous):
 *   d_H   [T][NC][M][K]       K contiguous      -- the static hint after its NTTs
 *   d_C   [T][NC][ncols][K]   each column of C contiguous along K
 *   d_G   [T][NC][gcols][M]   (may be NULL when gcols == 0)
 *   d_Out [T][NC][ncols][M]
 * Ownership: the caller owns all four; the plan owns a re-laid-out byte-limb copy of H
 * (4*T*NC*M*Kp bytes, Kp = K rounded up to 128; written by vipir_modgemm_set_h, after which the
 * caller may free d_H) and the limb planes of C (4*T*NC*ncols*Kp bytes, rewritten every call).
 * Execution and errors as for vipir_dbmul: calls only enqueue on `cuda_stream`.  One plan must not be in flight
 * on two streams, nor be used from two host threads at once: vipir_modgemm keeps per-plan state between calls --
 * the tensor map of the caller's C is cached for the last d_C seen and re-encoded (a host-side call of a few
 * microseconds) whenever d_C changes, so a caller that alternates C buffers may prefer one plan per buffer; and the
 * C limb planes of the two-kernel form are allocated by the plan call when that is the plan's form, else by the
 * first vipir_modgemm_split_c (ALLOC can come from there).  A server that overlaps requests makes one plan per stream.
 * =========================================================================================== */
typedef struct vipir_modgemm_plan vipir_modgemm_plan;

typedef struct {
    uint64_t problems;      /* T * NC */
    uint32_t k_padded;      /* Kp */
    uint32_t cta_group;     /* 1, or 2 = CTA pairs (tcgen05 cta_group::2, 256-row tiles) */
    uint32_t tile_cols;     /* ct: columns of C per N tile */
    uint32_t mma_n;         /* N of one tcgen05.mma = 4 * ct */
    uint32_t m_tiles, n_tiles; /* per problem */
    uint32_t n_chunks;      /* K chunks of <= 8192 (int32 accumulation bound 4*255^2*K < 2^31) */
    uint32_t a_stages, b_stages, acc_stages; /* ring depths: H boxes, converted C operand slots; accumulator stages */
    uint32_t r_stages;      /* one-kernel form: ring depth of the raw C tiles (0 otherwise) */
    uint32_t smem_bytes, grid;
    uint32_t launches;      /* kernels enqueued per vipir_modgemm call: 1 when the C limb split is fused in */
    uint32_t fused_split;   /* 1: vipir_modgemm splits C inside the products kernel, no C limb planes */
    uint64_t h_limb_bytes, c_limb_bytes; /* plan-owned workspaces: H limbs [T*NC*M][4*Kp] u8, C limbs [T*NC][4][ncols][Kp] u8
                                            (0 for a fused plan until vipir_modgemm_split_c is called) */
} vipir_modgemm_info_t;

/* Explicit planner overrides for the modular GEMMs; every field 0 = the planner's own choice (see vipir_tuning). */
typedef struct {
    uint32_t cta_group;   /* 1, or 2 = CTA pairs */
    uint32_t tile_cols;   /* ct: columns of C per N tile, a multiple of 8, <= 64 */
    uint32_t a_stages;    /* ring depth of the H operand: 4..24 (at most what fits) */
    uint32_t b_stages;    /* ring depth of the C operand: 2..4 */
    uint32_t c_split;     /* where vipir_modgemm splits C into limbs: 1 = a splitter kernel of its own (two launches),
                             2 = inside the products kernel (one launch; UNSUPPORTED unless K % 4 == 0) */
    uint32_t r_stages;    /* one-kernel form: ring depth of the raw C tiles, 2..4; UNSUPPORTED when the plan's form is two
                             kernels.  (a_stages and b_stages apply to whichever form runs, and to both when the parts
                             are called on a one-kernel plan.) */
    uint32_t reserved[2]; /* must be 0 */
} vipir_modgemm_tuning;

/*
 * Build a plan (host; allocates the limb workspaces on the current device).
 *   moduli  HOST pointer to T values, 2 <= q_t < 2^30 (the paper's RNS primes are < 2^29)
 * Errors: INVALID_ARG (null, zero size, T > VIPIR_MAX_MODULI, gcols > ncols, modulus out of
 * range), UNSUPPORTED (M, K or ncols >= 2^24, NC >= 2^28), ARCH, ALLOC, CUDA.
 */
int vipir_modgemm_plan_create(vipir_modgemm_plan **out, uint32_t T, uint64_t NC, uint32_t M, uint32_t K,
                              uint32_t ncols, uint32_t gcols, const uint32_t *moduli);

/* Same with explicit planner overrides.  Errors: as above; INVALID_ARG (a field outside its domain),
 * UNSUPPORTED (an override the shape cannot honour). */
int vipir_modgemm_plan_create_tuned(vipir_modgemm_plan **out, uint32_t T, uint64_t NC, uint32_t M, uint32_t K,
                                    uint32_t ncols, uint32_t gcols, const uint32_t *moduli,
                                    const vipir_modgemm_tuning *tune);

/* OFFLINE step: split the static hint H into byte limbs in the plan's GEMM-friendly layout (the
 * paper's "layout transposition before the GEMMs"; H is precomputed offline,
 * PAPER.md:222).  Must run before the first vipir_modgemm / vipir_modgemm_products. */
int vipir_modgemm_set_h(vipir_modgemm_plan *plan, const uint32_t *d_H, void *cuda_stream);

/* ONLINE step: enqueue Out = H*C + (0|G) mod q_t.  From 16 columns up (and K % 4 == 0: the paper's n = 1280) ONE
 * kernel: the tensor-core kernel reads the raw words of C by TMA and splits them into limbs in shared memory (the
 * paper fuses its prmt decomposition into the GEMM kernel as well); below that, where it measures
 * faster, the C limb splitter followed by the tensor-core kernel (vipir_modgemm_info_t.launches says which;
 * vipir_modgemm_tuning.c_split overrides).
 * Errors: INVALID_ARG (null / misaligned pointer, set_h not called), ALLOC, CUDA. */
int vipir_modgemm(vipir_modgemm_plan *plan, const uint32_t *d_C, const uint32_t *d_G, uint32_t *d_Out,
                  void *cuda_stream);

/* The two-kernel form separately (per-kernel timing, tests; the form a producer that writes C's limb planes
 * itself would use): vipir_modgemm_split_c writes the plan's C limb planes (allocated on first use),
 * vipir_modgemm_products multiplies against them.  Same result as vipir_modgemm, bit for bit. */
int vipir_modgemm_split_c(vipir_modgemm_plan *plan, const uint32_t *d_C, void *cuda_stream);
int vipir_modgemm_products(vipir_modgemm_plan *plan, const uint32_t *d_G, uint32_t *d_Out, void *cuda_stream);

int vipir_modgemm_info(const vipir_modgemm_plan *plan, vipir_modgemm_info_t *out);

/* Free the plan and its workspaces.  NULL is a no-op. */
void vipir_modgemm_destroy(vipir_modgemm_plan *plan);

/* ===========================================================================================
 * Lift + forward NTT: the scan's scalar-HE words (and, offline, the hint) -> the ring-packing
 * operands G and H of vipir_modgemm
 *
 * PAPER.md:214 (section 3.5.2): "the D1 x n and D1 x B SimplePIR outputs are first transformed into
 * polynomials by treating each length-N vector along the D1 dimension as a polynomial in R_q ...
 * to which NTTs are applied independently.  Let H and G denote these two polynomial matrices after
 * the NTTs."  PAPER.md:667 (Appendix C.1): the server "lifts the coefficients of iota(A_i) and
 * iota(b) from Z_p to Z_q and transforms them into the NTT domain"; eq. (3) scales
 * the b part by Delta.  PAPER.md:269-271 (section 4.3): single-kernel NTT for N = 2^12, fused with
 * the RNS decomposition; layout transposition to the GEMM-friendly layout (fused
 * into this kernel's store).
 *
 * Definition (bit-exact).  d_X [n_a][M][N] uint32: word j of polynomial (a, m); i.e. the layout of
 * vipir_dbmul's answer [batch = n_a][rows = M*N] after vipir_plan_set_modswitch(plan, p_bits): every
 * word < p = 2^p_bits.  For RNS prime t (modulus q_t > p, primitive 2N-th root of unity psi_t, scale_t):
 *     x_j  = scale_t * lift_t(X[a][m][j])  mod q_t
 *     Y[c] = sum_{j<N} x_j * psi_t^((2c+1) j)  mod q_t,   c < N       (natural order: the polynomial
 *            evaluated at the c-th odd power of psi_t, the roots of X^N + 1)
 * lift(x) = x (centered == 0), or x - p taken mod q_t for x >= p/2 (centered == 1).
 * Output, canonical in [0, q_t):
 *     VIPIR_NTT_LAYOUT_G:  d_O[t][c][a][m]   = vipir_modgemm's d_G [T][NC = N][gcols = n_a][M]
 *     VIPIR_NTT_LAYOUT_H:  d_O[t][c][m][a]   = vipir_modgemm's d_H [T][NC = N][M][K = n_a]
 * Words >= p are a caller error: their excess bits are ignored and a flag is raised that
 * vipir_ntt_bad_input reads (and clears).
 * Ownership: the caller owns d_X and d_O (DEVICE pointers, 4-byte aligned, not overlapping); the plan
 * owns its twiddle tables.  vipir_ntt_lift only enqueues on `cuda_stream`.
 * =========================================================================================== */
typedef struct vipir_ntt_plan vipir_ntt_plan;
#define VIPIR_NTT_LAYOUT_G 0u
#define VIPIR_NTT_LAYOUT_H 1u

/*
 * Build a plan (host; computes the twiddle tables psi_t^bitrev(i) and their Shoup companions and
 * copies them to the current device).
 *   log2n   log2 N: 4, 8 or 12 (the paper's N = 2^12)
 *   moduli, psi, scale   HOST pointers to T values: 2^p_bits < q_t < 2^30, psi_t^N = -1 mod q_t,
 *           scale_t any u32 (reduced mod q_t; 1 for H, Delta mod q_t for G)
 *   p_bits  1..29 (the paper's p = 2^18)
 * Errors: INVALID_ARG (null, T == 0 or > VIPIR_MAX_MODULI, modulus out of range, psi not a primitive
 * 2N-th root of unity, p_bits out of range, centered > 1), UNSUPPORTED (log2n), ARCH, ALLOC, CUDA.
 */
int vipir_ntt_plan_create(vipir_ntt_plan **out, uint32_t T, uint32_t log2n, const uint32_t *moduli,
                          const uint32_t *psi, const uint32_t *scale, uint32_t p_bits, uint32_t centered);

/* Enqueue the transform of n_a * M polynomials.  Errors: INVALID_ARG (null / misaligned pointer, zero
 * size, out_layout > 1), UNSUPPORTED (n_a * M >= 2^31), CUDA. */
int vipir_ntt_lift(vipir_ntt_plan *plan, const uint32_t *d_X, uint32_t n_a, uint32_t M, uint32_t out_layout,
                   uint32_t *d_O, void *cuda_stream);

/* *seen = 1 if any launch since the last call read a word >= 2^p_bits.  Blocks: cudaDeviceSynchronize() before
 * the flag is read and after it is cleared, so launches on any stream (blocking or not) are covered. */
int vipir_ntt_bad_input(vipir_ntt_plan *plan, uint32_t *seen);

/* Free the plan and its tables.  NULL is a no-op. */
void vipir_ntt_destroy(vipir_ntt_plan *plan);

#ifdef __cplusplus
}
#endif
#endif /* VIPIR_H */
