/* abi_check.c -- plain C99 program against include/routebalance.h: the header is valid C, the library links from C,
 * defaults and argument validation behave as documented.  No GPU needed (every call below returns before any device
 * work).  Built and run by tests/test_abi.py::test_c_program_links_and_runs. */
#include <stdio.h>
#include <string.h>

#include "routebalance.h"

int main(void) {
  rb_options opt;
  memset(&opt, 0xff, sizeof opt);
  rb_options_default(&opt);
  if (opt.bank_dtype != RB_F32 || opt.store_dtype != RB_BF16 || opt.weight_mode != 0 || opt.rerank_slack != 6 ||
      opt.lpt_enabled != 1 || opt.update_enabled != 1 || opt.max_batch != 4096 || opt.use_graph != 1 ||
      opt.scan_list != 0 || opt.tiebreak_mode != 0 || opt.latency_mode != 0 || opt.pipeline != 0 || opt.stream != NULL) {
    printf("defaults differ from the header\n");
    return 1;
  }
  rb_ctx* ctx = (rb_ctx*)0x1;
  float dummy[8] = {0};
  /* bad sizes are refused before anything touches the device, and *out is cleared */
  if (rb_create(&ctx, dummy, dummy, dummy, /*N=*/0, /*d=*/8, /*M=*/1, /*k=*/1, &opt) != RB_EINVAL || ctx != NULL) return 2;
  if (rb_create(&ctx, dummy, dummy, dummy, 1, /*d=*/7, 1, 1, &opt) != RB_EINVAL) return 3;     /* d % 8 != 0 */
  if (rb_create(&ctx, dummy, dummy, dummy, 1, 8, /*M=*/17, 1, &opt) != RB_EINVAL) return 4;    /* M > 16 */
  if (rb_create(&ctx, dummy, dummy, dummy, 1, 8, 1, /*k=*/2, &opt) != RB_EINVAL) return 5;     /* k > N */
  if (rb_create(&ctx, NULL, dummy, dummy, 1, 8, 1, 1, &opt) != RB_EINVAL) return 6;
  if (rb_create(NULL, dummy, dummy, dummy, 1, 8, 1, 1, &opt) != RB_EINVAL) return 7;
  opt.latency_mode = 3;
  if (rb_create(&ctx, dummy, dummy, dummy, 1, 8, 1, 1, &opt) != RB_EINVAL) return 8;
  /* NULL contexts are refused, never dereferenced */
  {
    float w[3] = {1.0f, 0.0f, 0.0f};
    int32_t a[1];
    if (rb_decide(NULL, dummy, a, 1, w, a, NULL, NULL, NULL, NULL, NULL) != RB_EINVAL) return 9;
    if (rb_advance_state(NULL, 1.0f) != RB_EINVAL) return 10;
    if (rb_batch_target(NULL, 4, 64, a, NULL) != RB_EINVAL) return 14;
    if (rb_decide_submit(NULL, dummy, a, 1, w) != RB_EINVAL || rb_decide_collect(NULL, a, 1) != RB_EINVAL) return 15;
    if (rb_sweep_weights(NULL, dummy, dummy, a, NULL, 1, w, 1, a) != RB_EINVAL) return 13;
    if (rb_decide_from_predictions_static(NULL, dummy, dummy, a, 1, w, 0, a) != RB_EINVAL) return 16;
    if (rb_launch_count(NULL) != 0) return 11;
    if (strcmp(rb_last_error(NULL), "null context") != 0) return 12;
    rb_destroy(NULL);
  }
  printf("abi ok\n");
  return 0;
}
