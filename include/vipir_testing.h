/*
 * vipir_testing.h -- introspection entry points of libvipir for its own test suite.  NOT part of the product
 * ABI (include/vipir.h): nothing here is needed to run the database scan, and a server never calls it.
 */
#ifndef VIPIR_TESTING_H
#define VIPIR_TESTING_H

#include <stdint.h>

#include "vipir.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * The tensor-core regimes' work distribution (host only, no device needed): the (unit, K chunk) items that
 * group `g` of `n_groups` visits, in order, for a problem of n_units = m_tiles * n_tiles units and n_chunks
 * chunks (csrc/gemm_i8_tcgen05.cuh "Work distribution"; split = 1: the last partial round is dealt out chunk
 * by chunk).  Writes min(*n, cap) triples (unit, chunk, must_wait) to out_triples; must_wait = 1 marks an item
 * whose earlier chunks belong to another group.  Errors: INVALID_ARG.
 */
int vipir_testing_work_items(uint32_t g, uint32_t n_groups, uint32_t n_units, uint32_t n_chunks, uint32_t split,
                             uint32_t *out_triples, uint32_t cap, uint32_t *n);

/*
 * DEVICE pointers to the plan-owned byte-limb workspaces of the modular GEMMs (read-only for the caller):
 *   *d_h_limbs  [T*NC*M][4*Kp] u8, byte (k/128)*512 + i*128 + k%128 of a row = limb i of H[..][k]
 *   *d_c_limbs  [T*NC][4][ncols][Kp] u8
 * Errors: INVALID_ARG.
 */
int vipir_testing_modgemm_limbs(const vipir_modgemm_plan *plan, void **d_h_limbs, void **d_c_limbs);

#ifdef __cplusplus
}
#endif
#endif /* VIPIR_TESTING_H */
