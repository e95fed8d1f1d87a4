/*
 * routebalance_testing.h -- entry points of librouteb.so that only the tests and bench.py use: per-stage device
 * timing of a decision (the roofline figures of bench.py) and a self-test of the dispatch
 * kernel's division.  Not part of the decision API of routebalance.h; same conventions (C ABI, plain pointers,
 * rb_status).
 */
#ifndef ROUTEBALANCE_TESTING_H_
#define ROUTEBALANCE_TESTING_H_

#include "routebalance.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Device time of the stages of the most recent rb_decide / rb_estimate on this context, measured with
 * CUDA events on the context's stream (only when the call ran with stage timing enabled through
 * rb_set_stage_timing(ctx, 1); the decision is then replayed from a graph with event-record nodes between its kernels,
 * which serialises them: each stage's interval is meaningful, their sum is longer than an untimed decision).
 *   us [host] 6 floats: stage (query staging), scan, merge, aggregate, score, dispatch. */
rb_status rb_set_stage_timing(rb_ctx* ctx, int32_t enabled);
rb_status rb_last_stage_us(rb_ctx* ctx, float us[6]);

/* Duration of the bank-scan kernel of the most recent rb_decide / rb_estimate that ran with stage timing enabled, on
 * the device's own clock: latest CTA end - earliest CTA start (globaltimer), in microseconds; 0 if not measured (fp32
 * storage, B > 128, or stage timing off).  Unlike the event interval in rb_last_stage_us it holds no launch latency. */
rb_status rb_last_scan_device_us(rb_ctx* ctx, float* us);

/* Self-test of the dispatch kernel's branch-free fp32 division (reciprocal refinement without the compiler's range check;
 * used only for operands inside the exponent window where it is exact, IEEE __fdiv_rn otherwise): compares it with the
 * IEEE division bit for bit on n_pairs pseudo-random in-window operand pairs.  *mismatches [host] must come back 0. */
rb_status rb_selftest_division(rb_ctx* ctx, uint64_t n_pairs, uint64_t seed, uint64_t* mismatches);

/* Read-only streaming bandwidth of the device (bench.py's ceiling for read-dominated kernels): a kernel of coalesced
 * 16-byte loads over a scratch buffer of `bytes` bytes (allocated and freed by the call), timed with CUDA events, best of
 * `repeats` launches.  *gb_per_s [host].  RB_ENOMEM if the buffer cannot be allocated. */
rb_status rb_testing_read_bandwidth(rb_ctx* ctx, uint64_t bytes, int32_t repeats, double* gb_per_s);

#ifdef __cplusplus
}
#endif
#endif /* ROUTEBALANCE_TESTING_H_ */
