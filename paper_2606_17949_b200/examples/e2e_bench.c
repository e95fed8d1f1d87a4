/* e2e_bench.c -- end-to-end latency of one decision through the C ABI alone (no Python, no torch): host buffers in,
 * assignment out, rb_advance_state + rb_decide per step.  Prints one JSON line.  Built and run by bench.py
 * (gcc ... -lrouteb); usage: e2e_bench N d B I steps [pipeline]   (pipeline = 1: rb_decide_submit / rb_decide_collect, three
 * decisions in flight)
 * The bank is synthetic (unit-norm rows around a few centres, a multiplicative congruential generator): this program
 * measures the library's host path, not parity. */
#define _POSIX_C_SOURCE 199309L
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>

#include "routebalance.h"

static unsigned long long rng_state = 88172645463325252ULL;
static double rnd(void) { /* xorshift64*, uniform in [0,1) */
  rng_state ^= rng_state >> 12;
  rng_state ^= rng_state << 25;
  rng_state ^= rng_state >> 27;
  return (double)((rng_state * 2685821657736338717ULL) >> 11) / 9007199254740992.0;
}
static double now_us(void) {
  struct timespec ts;
  clock_gettime(CLOCK_MONOTONIC, &ts);
  return ts.tv_sec * 1e6 + ts.tv_nsec * 1e-3;
}
static void unit_row(float* row, const float* centre, int d, double noise) {
  double n2 = 0.0;
  for (int c = 0; c < d; ++c) {
    row[c] = centre[c] + (float)(noise * (rnd() - 0.5) * 3.4641 / sqrt((double)d));
    n2 += (double)row[c] * row[c];
  }
  for (int c = 0; c < d; ++c) row[c] = (float)(row[c] / sqrt(n2));
}
static int cmp_double(const void* a, const void* b) { return (*(const double*)a > *(const double*)b) - (*(const double*)a < *(const double*)b); }

int main(int argc, char** argv) {
  const long N = argc > 1 ? atol(argv[1]) : 100000;
  const int d = argc > 2 ? atoi(argv[2]) : 768, B = argc > 3 ? atoi(argv[3]) : 12, I = argc > 4 ? atoi(argv[4]) : 13;
  const int steps = argc > 5 ? atoi(argv[5]) : 300, M = 4, k = 10, Kc = 64;
  const int pipeline = argc > 6 ? atoi(argv[6]) : 0;
  float* centres = malloc((size_t)Kc * d * 4);
  float* bank = malloc((size_t)N * d * 4);
  float* quality = malloc((size_t)N * M * 4);
  float* outlen = malloc((size_t)N * M * 4);
  float* query = malloc((size_t)B * d * 4);
  int32_t* plen = malloc((size_t)B * 4);
  int32_t* assignment = malloc((size_t)B * 4);
  double* t = malloc((size_t)steps * 8);
  if (!centres || !bank || !quality || !outlen || !query || !plen || !assignment || !t) return 2;
  float zero[4096];
  memset(zero, 0, sizeof zero);
  for (int c = 0; c < Kc; ++c) unit_row(centres + (size_t)c * d, zero, d, 3.4641 * sqrt((double)d) / 3.4641);
  for (long n = 0; n < N; ++n) {
    unit_row(bank + (size_t)n * d, centres + (size_t)(n % Kc) * d, d, 0.3);
    for (int m = 0; m < M; ++m) {
      quality[n * M + m] = (float)(0.2 + 0.6 * rnd());
      outlen[n * M + m] = (float)(50.0 + 500.0 * rnd());
    }
  }
  rb_options opt;
  rb_options_default(&opt);
  opt.max_batch = B > 64 ? B : 64;
  opt.pipeline = pipeline;
  rb_ctx* ctx = NULL;
  if (rb_create(&ctx, bank, quality, outlen, N, d, M, k, &opt) != RB_OK) {
    printf("{\"error\": \"rb_create: %s\"}\n", ctx ? rb_last_error(ctx) : "no context");
    return 1;
  }
  int32_t tier[1024], cap[1024], running[1024];
  float queued[1024];
  for (int i = 0; i < I; ++i) { tier[i] = i * M / I; cap[i] = 16; running[i] = (int)(rnd() * 17); queued[i] = (float)(int)(rnd() * 20000); }
  const float price[4] = {0.1f, 0.3f, 0.8f, 2.0f};
  const rb_lat_head heads[4] = {{0.05f, 10.2f, 0.02f}, {0.10f, 19.6f, 0.02f}, {0.08f, 13.9f, 0.02f}, {0.25f, 41.6f, 0.02f}};
  if (rb_set_instances(ctx, I, tier, cap, price, price, heads) != RB_OK || rb_set_state(ctx, queued, running) != RB_OK) {
    printf("{\"error\": \"%s\"}\n", rb_last_error(ctx));
    return 1;
  }
  const float w[3] = {1.0f / 3, 1.0f / 3, 1.0f / 3};
  double total_us = 0.0;
  if (!pipeline) {
    for (int s = -20; s < steps; ++s) {   /* 20 warm-up steps (graph capture, first touches) */
      for (int r = 0; r < B; ++r) {
        unit_row(query + (size_t)r * d, centres + (size_t)((int)(rnd() * Kc) % Kc) * d, d, 0.1);
        plen[r] = 1 + (int)(rnd() * 2000);
      }
      const double t0 = now_us();
      if (rb_advance_state(ctx, 40.0f) != RB_OK || rb_decide(ctx, query, plen, B, w, assignment, NULL, NULL, NULL, NULL, NULL) != RB_OK) {
        printf("{\"error\": \"%s\"}\n", rb_last_error(ctx));
        return 1;
      }
      if (s >= 0) { t[s] = now_us() - t0; total_us += t[s]; }
    }
  } else {
    /* submit(j + 2), collect(j): the inputs of every step are generated before the timed loop */
    const int n = steps + 20;
    float* allq = malloc((size_t)n * B * d * 4);
    int32_t* allp = malloc((size_t)n * B * 4);
    if (!allq || !allp) return 2;
    for (long r = 0; r < (long)n * B; ++r) {
      unit_row(allq + (size_t)r * d, centres + (size_t)((int)(rnd() * Kc) % Kc) * d, d, 0.1);
      allp[r] = 1 + (int)(rnd() * 2000);
    }
    double t_start = 0.0;
    for (int s = 0; s < n; ++s) {
      if (s == 20) t_start = now_us();
      const double t0 = now_us();
      if (rb_advance_state(ctx, 40.0f) != RB_OK ||
          rb_decide_submit(ctx, allq + (size_t)s * B * d, allp + (size_t)s * B, B, w) != RB_OK ||
          (s >= 2 && rb_decide_collect(ctx, assignment, B) != RB_OK)) {
        printf("{\"error\": \"%s\"}\n", rb_last_error(ctx));
        return 1;
      }
      if (s >= 20) t[s - 20] = now_us() - t0;
    }
    if (rb_decide_collect(ctx, assignment, B) != RB_OK || rb_decide_collect(ctx, assignment, B) != RB_OK) return 1;
    total_us = now_us() - t_start;
  }
  const double sum = total_us;
  qsort(t, (size_t)steps, 8, cmp_double);
  printf("{\"N\": %ld, \"d\": %d, \"B\": %d, \"I\": %d, \"steps\": %d, \"us_mean\": %.2f, \"us_p50\": %.2f, \"us_p99\": %.2f, "
         "\"mode\": \"%s\", \"buffers\": \"pageable host memory in, host memory out\", \"l2\": \"not flushed (bank %.1f MB)\"}\n",
         N, d, B, I, steps, sum / steps, t[steps / 2], t[(int)(steps * 0.99)],
         pipeline ? "rb_decide_submit / rb_decide_collect, three in flight (us_mean = wall clock over all steps / steps)" : "rb_decide, one at a time",
         (double)N * d * 2 / 1e6);
  rb_destroy(ctx);
  return 0;
}
