/*
 * vipir_oracle.c -- CPU ORACLE for the VIPIR database scan  answer = D * Q mod q.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or helper with paper_2606_11536_b200/csrc (the CUDA path).
 *
 * What it computes (section 2.5, SimplePIR): the server multiplies the
 * D1 x D0 database of small plaintext integers by the D0 x B matrix of query words; the
 * online step is "a D1 x B x D0 INT8-INT32 GEMM for a batch of B queries".  Number types
 * (section 2.3): "regular INT8-INT32 scalar-vector multiplications and
 * INT32 vector additions"; modulus (section 4): "we perform modulo-2^32
 * operations as in SimplePIR".  Per-prime residues (section 2.3): the
 * same integer reduced "% q_i" for each RNS prime q_i.
 *
 * Two routines:
 *   vipir_oracle_dbmul        the plain definition, written out (triple loop, wide
 *                             accumulator, one explicit "% q" per output word);
 *   vipir_oracle_dbmul_limbs  the paper's METHOD followed step by step (PAPER.md:245-249
 *                             section 4.1): split each query word into four 8-bit
 *                             matrices B0..B3, form every A*Bj with 32-bit signed
 *                             accumulation, recombine with shifts, reduce.  It exists to
 *                             cross-check the definition and to state executably what a
 *                             tensor-core implementation does; it must equal the
 *                             definition on every input.
 *
 * Layout (the same one include/vipir.h documents; readings R2, R3):
 *   D  rows x cols, row-major (cols contiguous), unsigned 8-bit, or unsigned little-endian
 *      16-bit when db_bits == 16 (readings R1, R10: elements are UNSIGNED).
 *   Q  [T][batch][cols] uint32, T = max(n_moduli, 1); each query vector contiguous.
 *   A  [T][batch][rows] uint32, canonical representative in [0, q_t).
 *   n_moduli == 0 means q = 2^32 (wrapping).
 *
 *   vipir_oracle_modswitch    NEXT-1 of SURVEY.md section 8(f): the scalar-HE modulus switch
 *                             2^32 -> 2^bits applied to every answer word.
 *
 * Parity pins: tests/test_oracle_pins.py (brute force on tiny shapes, closed forms,
 * identity, permutation probe, unit vectors, linearity, toy LWE round trip, CRT).  Nothing
 * in this file is "parity unpinned".
 */
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef unsigned __int128 u128;

static inline uint64_t db_at(const void *D, int db_bits, uint64_t idx) {
    if (db_bits == 8) return ((const uint8_t *)D)[idx];
    /* little-endian u16, value = lo + 256*hi (reading R10) */
    const uint8_t *p = (const uint8_t *)D + 2 * idx;
    return (uint64_t)p[0] | ((uint64_t)p[1] << 8);
}

/*
 * The definition:
 *   A[t][b][r] = ( sum_{k<cols} D[r][k] * Q[t][b][k] ) mod q_t   over the integers.
 * The accumulator is 128 bits wide, so the sum never overflows for any cols < 2^64/2^48.
 * Returns 0, or -1 on a bad argument.  nthreads <= 1 runs serially; otherwise the row
 * loop is split with OpenMP (each thread still runs the same triple loop on its rows).
 */
int vipir_oracle_dbmul(uint64_t rows, uint64_t cols, uint32_t batch, int db_bits,
                       uint32_t n_moduli, const uint32_t *moduli,
                       const void *D, const uint32_t *Q, uint32_t *A, int nthreads) {
    if (!D || !Q || !A || rows == 0 || cols == 0 || batch == 0) return -1;
    if (db_bits != 8 && db_bits != 16) return -1;
    if (n_moduli > 0 && !moduli) return -1;
    for (uint32_t t = 0; t < n_moduli; ++t)
        if (moduli[t] < 2) return -1;
    const uint32_t T = n_moduli ? n_moduli : 1;
    if (nthreads < 1) nthreads = 1;

#pragma omp parallel for num_threads(nthreads) schedule(static)
    for (uint64_t r = 0; r < rows; ++r) {
        for (uint32_t t = 0; t < T; ++t) {
            for (uint32_t b = 0; b < batch; ++b) {
                const uint32_t *q = Q + ((uint64_t)t * batch + b) * cols;
                u128 acc = 0;
                for (uint64_t k = 0; k < cols; ++k)
                    acc += (u128)(db_at(D, db_bits, r * cols + k) * (uint64_t)q[k]);
                uint64_t red;
                if (n_moduli == 0)
                    red = (uint64_t)(acc % (((u128)1) << 32)); /* q = 2^32 */
                else
                    red = (uint64_t)(acc % (u128)moduli[t]);
                A[((uint64_t)t * batch + b) * rows + r] = (uint32_t)red;
            }
        }
    }
    return 0;
}

/*
 * The paper's method, step by step (section 4.1):
 *   "we decompose the INT32 matrix into four INT8 matrices ... B0, B1, B2, B3 to compute
 *    A*B as  A*B0 + 2^8 (A*B1) + 2^16 (A*B2) + 2^24 (A*B3)  mod 2^32  where each A*Bj is
 *    computed using tensor cores [INT8 GEMMs with INT32 accumulation], multiplications by
 *    {2^8, 2^16, 2^24} are implemented via bit shifts".
 * A 16-bit database element is likewise split into two 8-bit limbs A = A0 + 2^8 A1
 * (BASELINE.json config 5; not in the paper).  The 32-bit signed accumulation is only
 * exact while 255*255*K < 2^31, so the K dimension is cut into chunks of at most k_chunk
 * products per accumulator (reading R7: k_chunk <= 32768); each chunk's partial product
 * P_ij is held in int32 exactly as the hardware would hold it, and this routine returns
 * -2 if any P_ij would not have fitted.  Recombination: sum_ij 2^(8(i+j)) P_ij, reduced
 * mod q_t per chunk and added mod q_t across chunks.
 */
int vipir_oracle_dbmul_limbs(uint64_t rows, uint64_t cols, uint32_t batch, int db_bits,
                             uint32_t n_moduli, const uint32_t *moduli,
                             const void *D, const uint32_t *Q, uint32_t *A,
                             uint64_t k_chunk) {
    if (!D || !Q || !A || rows == 0 || cols == 0 || batch == 0 || k_chunk == 0) return -1;
    if (db_bits != 8 && db_bits != 16) return -1;
    if (n_moduli > 0 && !moduli) return -1;
    const uint32_t T = n_moduli ? n_moduli : 1;
    const int dl = db_bits / 8; /* database limbs */
    int overflow = 0;

    /* step 1: B -> B0..B3 (one byte matrix per limb) */
    uint8_t *Bj[4];
    const uint64_t nq = (uint64_t)T * batch * cols;
    for (int j = 0; j < 4; ++j) {
        Bj[j] = (uint8_t *)malloc(nq);
        if (!Bj[j]) return -3;
        for (uint64_t n = 0; n < nq; ++n) Bj[j][n] = (uint8_t)(Q[n] >> (8 * j));
    }

    for (uint64_t r = 0; r < rows; ++r) {
        for (uint32_t t = 0; t < T; ++t) {
            const u128 q = n_moduli ? (u128)moduli[t] : (((u128)1) << 32);
            for (uint32_t b = 0; b < batch; ++b) {
                const uint64_t qoff = ((uint64_t)t * batch + b) * cols;
                u128 total = 0; /* running answer, kept reduced mod q */
                for (uint64_t k0 = 0; k0 < cols; k0 += k_chunk) {
                    const uint64_t k1 = (k0 + k_chunk < cols) ? k0 + k_chunk : cols;
                    /* step 2: P_ij = A_i * B_j over this chunk, INT32 accumulation */
                    int64_t P[2][4];
                    memset(P, 0, sizeof P);
                    for (uint64_t k = k0; k < k1; ++k) {
                        const uint64_t d = db_at(D, db_bits, r * cols + k);
                        for (int i = 0; i < dl; ++i) {
                            const int64_t di = (int64_t)((d >> (8 * i)) & 0xFF);
                            for (int j = 0; j < 4; ++j) P[i][j] += di * (int64_t)Bj[j][qoff + k];
                        }
                    }
                    /* step 3: shift-recombine */
                    u128 part = 0;
                    for (int i = 0; i < dl; ++i)
                        for (int j = 0; j < 4; ++j) {
                            if (P[i][j] > (int64_t)INT32_MAX) overflow = 1;
                            part += ((u128)(uint64_t)P[i][j]) << (8 * (i + j));
                        }
                    total = (total + part % q) % q;
                }
                A[((uint64_t)t * batch + b) * rows + r] = (uint32_t)(uint64_t)total;
            }
        }
    }
    for (int j = 0; j < 4; ++j) free(Bj[j]);
    return overflow ? -2 : 0;
}

/*
 * Scalar-HE modulus switch (section 5: the ciphertext modulus 2^32 "is reduced to
 * 2^18 after each scalar-HE folding step"; Appendix D.2: "we reduce the
 * ciphertext modulus of scalar-HE ciphertexts from 2^32 to p = 2^18 ... equivalent to
 * introducing an additional rounding error term into each element", |r| < 2^13 in the 2^32
 * scale, i.e. rounding to nearest).  Plain definition, per word x in [0, 2^32):
 *     y = round( x * 2^bits / 2^32 )  mod 2^bits,   ties rounded up (reading R19)
 * written with a multiply and a divide so it can be checked by eye; in place.
 * 1 <= bits <= 31.  Returns 0, or -1 on a bad argument.
 */
int vipir_oracle_modswitch(uint32_t *A, uint64_t n, int bits) {
    if (!A || bits < 1 || bits > 31) return -1;
    const uint64_t q_in = 1ull << 32, q_out = 1ull << bits;
    for (uint64_t i = 0; i < n; ++i) {
        const uint64_t num = (uint64_t)A[i] * q_out;         /* x * 2^bits < 2^63 */
        const uint64_t y = (2 * num + q_in) / (2 * q_in);    /* floor(x*2^bits/2^32 + 1/2) */
        A[i] = (uint32_t)(y % q_out);
    }
    return 0;
}

/*
 * NEXT-3 of SURVEY.md section 8(f): SIGNED database elements (centred plaintexts: the paper's
 * decryption range is m in [-p/2, p/2)).  Same definition as vipir_oracle_dbmul
 * with D[r][k] read as a two's-complement int8 (db_bits == 8) or little-endian int16:
 *   A[t][b][r] = ( sum_k D[r][k] * Q[t][b][k] ) mod q_t,  sum over the (signed) integers,
 * result canonical in [0, q_t).  Serial; tests only.
 */
int vipir_oracle_dbmul_signed(uint64_t rows, uint64_t cols, uint32_t batch, int db_bits,
                              uint32_t n_moduli, const uint32_t *moduli,
                              const void *D, const uint32_t *Q, uint32_t *A) {
    if (!D || !Q || !A || rows == 0 || cols == 0 || batch == 0) return -1;
    if (db_bits != 8 && db_bits != 16) return -1;
    if (n_moduli > 0 && !moduli) return -1;
    const uint32_t T = n_moduli ? n_moduli : 1;
    for (uint64_t r = 0; r < rows; ++r)
        for (uint32_t t = 0; t < T; ++t) {
            const __int128 q = n_moduli ? (__int128)moduli[t] : (((__int128)1) << 32);
            for (uint32_t b = 0; b < batch; ++b) {
                const uint32_t *qv = Q + ((uint64_t)t * batch + b) * cols;
                __int128 acc = 0;
                for (uint64_t k = 0; k < cols; ++k) {
                    const uint64_t u = db_at(D, db_bits, r * cols + k);
                    const int64_t d = (db_bits == 8) ? (int64_t)(int8_t)(uint8_t)u : (int64_t)(int16_t)(uint16_t)u;
                    acc += (__int128)d * (__int128)qv[k];
                }
                __int128 red = acc % q; /* C remainder has the sign of acc */
                if (red < 0) red += q;
                A[((uint64_t)t * batch + b) * rows + r] = (uint32_t)(uint64_t)red;
            }
        }
    return 0;
}
