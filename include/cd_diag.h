/*
 * cd_diag.h -- measurement and diagnostic entry points of libcd.so.
 *
 * These are exported by the same library as cd.h but are NOT part of the decoding contract
 * (SURVEY.md 8(b)): bench.py and the tests use them to time the kernels and to count launches.
 * A caller that only decodes never needs this header.  Conventions as in cd.h.
 */
#ifndef CD_DIAG_H_
#define CD_DIAG_H_

#include "cd.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * cd_loop_trace returns, for the last loop that ran in a persistent kernel on (dfa, cuda_stream),
 * the number of decoding steps it ran (*steps_out), and for the first min(cap, 256) of them the
 * rows that took the step and its duration in nanoseconds measured on the device (HOST arrays;
 * without lock-step, step k lasts from the latest publication of a row's step k to the latest
 * publication of a row's step k + 1; *steps_out = 0 if that loop took the per-step path).  It
 * synchronises the stream.
 */
CD_API cd_status cd_loop_trace(const cd_dfa_t* dfa, void* cuda_stream, int32_t cap, int64_t* t_ns_out,
                        int32_t* n_active_out, int32_t* steps_out);

/*
 * Measurement aid for the roofline: streams `bytes` (>= 8192, rounded down to
 * 8 KiB tiles) of the DEVICE buffer `buf` (16-byte aligned) through the copy machinery of the
 * step kernel -- per-warp rings of 1-D bulk async copies, 12 warps x 2 stages x 8 KiB per SM --
 * with no arithmetic, `iters` times after 2 warm-up launches, and writes the average duration
 * of one pass in milliseconds to *ms_out (HOST float).  bytes / time is what a pure-read
 * kernel of this shape reaches on this GPU; bench.py reports it beside the measured copy
 * peak.  Synchronises the stream.
 */
CD_API cd_status cd_probe_read(const void* buf, int64_t bytes, int32_t iters, float* ms_out, void* cuda_stream);

/* Number of kernel launches this library has enqueued from the calling thread's
   process so far (monotone; used by bench.py to report gpu_launches). */
CD_API int64_t cd_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* CD_DIAG_H_ */
