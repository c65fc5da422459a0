/* orbit_debug.h -- A/B switch of the debug build (liborbit_dbg.so, built with -DORBIT_DEBUG_SWITCH).  NOT part of the
 * product ABI (include/orbit.h): the shipped liborbit.so has one dispatch and does not export this symbol.
 *   0 = automatic (tcgen05 tensor-core kernels for bf16 where shapes allow),
 *   1 = force the SIMT fp32-FMA kernels everywhere (cross-check),
 *   2 = single-CTA tcgen05 GEMM instead of the CTA-pair kernel,
 *   3 = mma.sync attention instead of the tcgen05 attention (forward and backward), 4 = backward only,
 *   5 = direct row-per-thread stores in the CTA-pair GEMM epilogue instead of the TMA store / reduce-add path.
 * Process-wide and unsynchronised: set it before any other call, from one thread. */
#ifndef ORBIT_DEBUG_H_
#define ORBIT_DEBUG_H_
#ifdef ORBIT_DEBUG_SWITCH
#ifdef __cplusplus
extern "C" {
#endif
void orbit_set_debug_force_simt(int mode);
/* only with -DORBIT_PROBE_TIMELINE: the forward-attention wait-cycle counters of CTA (0, 0) (attention_tc5.cu), summed over the
 * launches since the last reset */
int orbit_debug_read_probe(unsigned long long* out, int n, int reset);
#ifdef __cplusplus
}
#endif
#endif
#endif /* ORBIT_DEBUG_H_ */
