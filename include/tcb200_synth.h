/*
 * tcb200_synth.h -- seeded synthetic input tensors generated ON THE DEVICE (bench / test helper, not part of
 * the hot path).  The device twin of paper_2409_06759_b200/synth.py: same counter-based generator, bit-identical
 * values, used where a tensor is too large to build on the host (config 3: V is 25.6 GB).  Holds none of the
 * method's arithmetic.  Recipe: DESIGN.md "input recipe" (readings #4, #5).
 */
#ifndef TCB200_SYNTH_H
#define TCB200_SYNTH_H

#include "tcb200.h"

#ifdef __cplusplus
extern "C" {
#endif

/* t[idx] = sigma * sym( g(seed, tensor_id, canonical linear index of (idx + label_offset) in label_extents) )
 *   g: one complex draw, Re and Im i.i.d. N(0,1) (Box-Muller on two splitmix64 words);
 *   n_pairs in {0,1,2} antisymmetrised index pairs (pairs[2*n]): 1/2[(g - g(p<->q)) - (g(r<->s) - g(pq,rs))];
 *   hermitian != 0 (rank 4): W(pqrs) = 1/2 [A(pqrs) + conj A(rspq)].
 * label_offset / label_extents may be NULL (= zeros / the tensor's own extents). */
int tcbx_synth_normal(tcb_ctx *ctx, tcb_tensor *t, uint64_t seed, uint64_t tensor_id, int n_pairs,
                      const int32_t *pairs, double sigma, int hermitian, const int64_t *label_offset,
                      const int64_t *label_extents);
/* re = canonical linear index, im = -(index) - 0.5 : closed-form checkable transposition input */
int tcbx_synth_index_linear(tcb_ctx *ctx, tcb_tensor *t);
/* T(a,b,i,j) = vvoo(a,b,i,j) / ((e_i + e_j) - (e_a + e_b)), component-wise; eo[o], ev[v] are HOST arrays */
int tcbx_synth_mp2_amplitudes(tcb_ctx *ctx, tcb_tensor *T, const tcb_tensor *vvoo, const double *eo, int64_t o,
                              const double *ev, int64_t v);

#ifdef __cplusplus
}
#endif
#endif
