/*
 * mas_pcg_debug.h -- measurement probes for bench.py.  NOT part of the product ABI (include/mas_pcg.h): these two
 * entry points exist only in lib/libmas_pcg_dbg.so, which is the product source compiled with
 * -DMAS_PCG_DEBUG_PROBES.  The product library lib/libmas_pcg.so does not export them.
 */
#ifndef MAS_PCG_DEBUG_H
#define MAS_PCG_DEBUG_H
#include "mas_pcg.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Runs `nit` PCG iterations (rtol = 0) from x0 = x_dev with the loop's two kernels launched one by one and CUDA
 * events recorded around each on `stream`; synchronises.  ms_out (HOST, 4 doubles) = { mean K1, mean K2, min K1,
 * min K2 } kernel durations in milliseconds (K1 = fused matvec, K2 = fused vector kernel, K2R when q is recomputed).
 * 1 <= nit <= 256.  x_dev is overwritten. */
int mas_pcg_dbg_profile(mas_pcg_t *h, const double *b_dev, double *x_dev, int nit, void *stream, double *ms_out);

/* *ms_out (HOST) = best sustained time per launch, over `reps` back-to-back launches, of a trivial LINEAR kernel with
 * the DRAM read/write mix of K1 (which = 6: three N-vectors read, three written, one of them in place; which = 5: the
 * same without the q store) or of K2 (which = 3: two read, one written in place) and none of their structure: what
 * the memory system sustains for that mix.  Clobbers the handle's workspaces. */
int mas_pcg_dbg_mix_probe(mas_pcg_t *h, int which, int reps, void *stream, double *ms_out);

#ifdef __cplusplus
}
#endif
#endif /* MAS_PCG_DEBUG_H */
