/*
 * qcldpc_profile.h -- measurement hooks of libqcldpc (used by bench.py for the roofline line).  NOT part of the decode
 * ABI of include/qcldpc.h: nothing here changes what a decode computes.  The hooks keep per-thread state (a pool of
 * CUDA events) while they are switched on; qcldpc_profile_enable(0) releases it.
 */
#ifndef QCLDPC_PROFILE_H_
#define QCLDPC_PROFILE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Launch timing for roofline reports.  qcldpc_profile_enable(stride) with stride > 0 makes the
 * following qcldpc_decode calls of this thread record a CUDA event pair, on the decode stream, around every
 * stride-th launch of the two per-iteration kernels (kind 0 = fused check/variable update k_pass, kind 1 =
 * early-exit check k_cand); stride = 0 switches it off.  qcldpc_profile_collect waits for the recorded events (host
 * blocks until they have completed), returns for each kind the summed duration in ms of the timed launches, how many
 * were timed and how many were launched since enable/collect, and clears the record.  ms_sum, timed, launched:
 * HOST arrays of 2 entries.  The events live in a per-thread pool that grows on demand while profiling is on (the one
 * place where a decode call creates CUDA objects) and is destroyed by qcldpc_profile_enable(0).
 */
int qcldpc_profile_enable(int stride);
int qcldpc_profile_collect(double* ms_sum, int64_t* timed, int64_t* launched);

#ifdef __cplusplus
}
#endif
#endif /* QCLDPC_PROFILE_H_ */
