/*
 * turbochunk_sched.h — C ABI of the closed-loop scheduler of TurboServe (arxiv/paper_2606_19271 §5.2), the host-side
 * controller that consumes what the per-GPU runtime of turbochunk.h produces: the per-chunk latency model l_hat(n)
 * (measured by paper_2606_19271_b200.latency_model) and the migration primitive (ts_session_migrate).
 * Pure host code: no CUDA call, usable without a GPU.
 *
 *   PAPER.md:203-207  Algorithm 1: per event  PLACE -> SCALE -> (scale-in: PLACE under M_tar, then shrink) /
 *                     (scale-out: grow, then PLACE under the new budget) / (keep the budget).
 *   PAPER.md:193-199  PLACE: start from phi(t-) without terminated sessions; every session of
 *                     U(t) = { s_i : alpha_i = 1 and phi_i(t-) = empty }  (Eq. 3) goes to the feasible GPU that minimises
 *                     the resulting bottleneck latency L(t) = max_j l_hat(n_j), ties "preferring less-loaded GPUs".
 *   PAPER.md:201-213  migration-aware min-max rebalancing: g_max = argmax_j l_hat(n_j); over sessions i on g_max and targets
 *                     j' != g_max:  Gamma_{i,j'} = L - L' - eta * kappa_i  (Eq. 4), kappa_i by the alpha-beta model; the best
 *                     move is applied while its Gamma > 0.
 *   PAPER.md:234-236  SCALE: rho_max = max_j n_j / K; scale-out if rho_max > rho_hat + delta, scale-in if
 *                     rho_max < rho_hat - delta; M_tar = ceil(N_req / (K * rho_hat)).
 *   PAPER.md:447-464  volatility mapping: sigma(t) = std of the newly activated sessions per event over a window of W
 *                     events (Eq. 6); measure -> quantise -> look up -> replace rho_hat.
 * Readings where the paper is silent (R23-R29): stable GPU ids with an alive flag, scale-out activates the lowest
 * dead ids, scale-in removes the least-loaded alive GPUs (ties: highest id) and re-assigns their sessions by the Eq. 3
 * rule; alpha_i = 0 => phi_i = empty; one l_hat table for all GPUs; exact ties broken by (less loaded, lowest id) for
 * targets and (lowest session id) for sessions; kappa_i = kappa_alpha + kappa_beta * state_mb_i; a scale-out trigger never
 * lowers M, a scale-in trigger never raises it, M_tar is clamped to [max(1, ceil(N_req / K)), M_max].
 * All decisions are integer or exact-double arithmetic in a fixed operation order: results are bit-identical to the
 * oracle (oracle/scheduler.py), which tests/test_scheduler_parity.py checks event by event.
 *
 * Errors: TS_OK or a negative ts_status of turbochunk.h (TS_ERR_INVALID: null pointer, bad config, duplicate session id in
 * an event, negative id).  One caller thread per scheduler.
 */
#ifndef TURBOCHUNK_SCHED_H_
#define TURBOCHUNK_SCHED_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ts_sched ts_sched; /* opaque */

typedef struct ts_sched_config {
  int32_t K;           /* per-GPU session cap */
  int32_t M_max;       /* largest GPU budget */
  int32_t M0;          /* GPUs alive at start, 1 <= M0 <= M_max (ids 0..M0-1) */
  int32_t vol_window;  /* W of Eq. 6 in events; 0 = rho_hat stays fixed */
  double rho_hat;      /* target utilisation (initial value when vol_window > 0) */
  double delta;        /* hysteresis tolerance */
  double eta;          /* weight of the migration cost in Eq. 4 */
  double kappa_alpha;  /* alpha-beta model: kappa_i = kappa_alpha + kappa_beta * state_mb_i (same unit as l_hat) */
  double kappa_beta;
  const double* l_hat; /* host [K+1]: l_hat[n] = per-chunk latency of a GPU with n sessions; l_hat[0] = 0, non-decreasing. Copied. */
  int32_t n_levels;    /* volatility levels L (vol_window > 0): vol_rho[n_levels], vol_bounds[n_levels - 1] */
  int32_t reserved;
  const double* vol_bounds; /* host: ascending interval edges; level = number of edges <= sigma. Copied. */
  const double* vol_rho;    /* host: rho_hat of each level. Copied. */
} ts_sched_config;

typedef struct ts_sched_result {
  int32_t M;            /* GPUs alive after the event */
  int32_t n_migrations; /* sessions placed before and after the event, on different GPUs (what the runtime must move) */
  int32_t n_moves;      /* entries of the move log (every re-assignment PLACE made, in order) */
  int32_t n_unplaced;   /* active sessions without a GPU (every alive GPU holds K) */
  int32_t n_req;        /* N_req: sessions with alpha_i = 1 */
  int32_t reserved;
  double rho_max;       /* max_j n_j / K after the event */
  double L;             /* bottleneck latency max_j l_hat(n_j) */
  double rho_hat;       /* target utilisation in force */
  double sigma;         /* volatility of Eq. 6 (0 when vol_window == 0) */
} ts_sched_result;

int ts_sched_create(const ts_sched_config* cfg, ts_sched** out);
int ts_sched_destroy(ts_sched* s);

/* One decision epoch of Algorithm 1.  The event lists every session that exists (absent = terminated), in the order in
 * which U(t) is served: session_ids[n] (>= 0, no duplicates), active[n] = alpha_i, state_mb[n] = size of the session's
 * state for kappa_i.  phi_out[n] receives the GPU id of each session or -1 (suspended / unplaced).  All host pointers. */
int ts_sched_event(ts_sched* s, int32_t n, const int32_t* session_ids, const int32_t* active, const double* state_mb,
                   int32_t* phi_out, ts_sched_result* res);

/* Lists of the last event, up to `cap` entries; *n_out = their number.  which = 0: net migrations sorted by session id;
 * which = 1: the move log in the order PLACE made the moves. */
int ts_sched_moves(ts_sched* s, int32_t which, int32_t* sid, int32_t* from_gpu, int32_t* to_gpu, int32_t cap, int32_t* n_out);
/* alive_out[M_max] = 1 for every GPU id that is provisioned after the last event. */
int ts_sched_alive(ts_sched* s, int32_t* alive_out);

#ifdef __cplusplus
}
#endif
#endif /* TURBOCHUNK_SCHED_H_ */
