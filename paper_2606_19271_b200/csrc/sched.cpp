// Closed-loop scheduler of TurboServe (§5.2, Algorithm 1): PLACE (Eq. 3 assignment, Eq. 4 migration-aware min-max
// rebalancing), SCALE (hysteresis trigger + proportional target) and the volatility-to-parameter mapping of App. A, behind
// the C ABI of include/turbochunk_sched.h.  Host code only.  Every comparison is on integers or on doubles produced by the
// same operations in the same order as the statement of the algorithm, so decisions are reproducible bit for bit
// (built with -ffp-contract=off: no fused multiply-add may change a gain).
#include <algorithm>
#include <cmath>
#include <deque>
#include <map>
#include <set>
#include <vector>

#include "../../include/turbochunk.h"
#include "../../include/turbochunk_sched.h"

namespace {

struct Move {
  int32_t sid, from, to;
};

struct SessionIn {
  int32_t sid, active;
  double mb;
};

}  // namespace

struct ts_sched {
  int K = 0, M_max = 0, vol_window = 0;
  double rho_hat = 0, delta = 0, eta = 0, kappa_alpha = 0, kappa_beta = 0;
  std::vector<double> l_hat, vol_bounds, vol_rho;
  std::vector<char> alive;
  std::map<int32_t, int32_t> phi;    // placed sessions only, ordered by id
  std::set<int32_t> known;           // sessions with alpha = 1 at the previous event
  std::deque<int> activations;       // a_tau of Eq. 6, last W events
  std::vector<Move> moves, net;      // of the last event

  int n_alive() const { return (int)std::count(alive.begin(), alive.end(), (char)1); }

  std::vector<int> loads() const {
    std::vector<int> n(M_max, 0);
    for (const auto& kv : phi) ++n[kv.second];
    return n;
  }
  double bottleneck(const std::vector<int>& n) const {   // L = max_j l_hat(n_j) over the alive GPUs
    double L = 0.0;
    bool any = false;
    for (int j = 0; j < M_max; ++j)
      if (alive[j] && (!any || l_hat[n[j]] > L)) {
        L = l_hat[n[j]];
        any = true;
      }
    return L;
  }
  // Eq. 3: the feasible GPU that minimises the resulting bottleneck latency; ties -> less loaded -> lowest id
  bool assign(int32_t sid, std::vector<int>& n) {
    int best = -1, best_n = 0;
    double best_L = 0.0;
    for (int j = 0; j < M_max; ++j) {
      if (!alive[j] || n[j] >= K) continue;
      ++n[j];
      const double L = bottleneck(n);
      --n[j];
      if (best < 0 || L < best_L || (L == best_L && n[j] < best_n)) {
        best = j;
        best_L = L;
        best_n = n[j];
      }
    }
    if (best < 0) return false;
    phi[sid] = best;
    ++n[best];
    return true;
  }

  // PLACE(S(t), phi(t-), M) -> (phi(t), rho_max(t))
  double place(const std::vector<SessionIn>& ev, const std::map<int32_t, int32_t>* displaced) {
    std::set<int32_t> live;
    for (const SessionIn& s : ev) live.insert(s.sid);
    for (auto it = phi.begin(); it != phi.end();) {   // initialisation: drop terminated sessions (and removed GPUs)
      if (!live.count(it->first) || !alive[it->second]) it = phi.erase(it);
      else ++it;
    }
    for (const SessionIn& s : ev)
      if (!s.active) phi.erase(s.sid);                // an idle session holds no GPU slot
    std::vector<int> n = loads();
    for (const SessionIn& s : ev) {                   // session assignment, U(t), in event order
      if (!s.active || phi.count(s.sid)) continue;
      if (assign(s.sid, n) && displaced != nullptr) {
        auto d = displaced->find(s.sid);
        if (d != displaced->end()) moves.push_back({s.sid, d->second, phi[s.sid]});
      }
    }
    std::map<int32_t, double> size;
    for (const SessionIn& s : ev) size[s.sid] = s.mb;
    for (;;) {                                        // migration-aware min-max rebalancing, Eq. 4
      const double L = bottleneck(n);
      int gmax = -1;
      for (int j = 0; j < M_max && gmax < 0; ++j)
        if (alive[j] && l_hat[n[j]] == L) gmax = j;
      if (gmax < 0 || n[gmax] == 0) break;
      bool have = false;
      double best_gain = 0.0;
      int32_t best_sid = 0;
      int best_n = 0, best_j = 0;
      for (const auto& kv : phi) {                    // ascending session id
        if (kv.second != gmax) continue;
        const double kappa = kappa_alpha + kappa_beta * size[kv.first];
        for (int j = 0; j < M_max; ++j) {
          if (j == gmax || !alive[j] || n[j] >= K) continue;
          --n[gmax];
          ++n[j];
          const double Lp = bottleneck(n);
          ++n[gmax];
          --n[j];
          const double cost = eta * kappa;
          const double gain = (L - Lp) - cost;        // Gamma_{i,j'} = L - L' - eta * kappa_i
          // order: larger gain, then lower session id (the outer loop), then less-loaded target, then lower target id
          if (!have || gain > best_gain || (gain == best_gain && kv.first == best_sid && n[j] < best_n)) {
            have = true;
            best_gain = gain;
            best_sid = kv.first;
            best_n = n[j];
            best_j = j;
          }
        }
      }
      if (!have || !(best_gain > 0.0)) break;
      moves.push_back({best_sid, gmax, best_j});
      phi[best_sid] = best_j;
      --n[gmax];
      ++n[best_j];
    }
    int mx = 0;
    for (int j = 0; j < M_max; ++j)
      if (alive[j]) mx = std::max(mx, n[j]);
    return (double)mx / (double)K;
  }

  // SCALE(rho_max, M(t-)) -> M_tar
  int scale(double rho_max, int M, int n_req) const {
    int tar = (int)std::ceil((double)n_req / ((double)K * rho_hat));   // proportional target
    tar = std::min(M_max, std::max(std::max(1, (n_req + K - 1) / K), tar));
    if (rho_max > rho_hat + delta) return std::max(M, tar);            // hysteresis trigger
    if (rho_max < rho_hat - delta) return std::min(M, tar);
    return M;
  }

  double adapt(int n_new) {   // App. A: measure -> quantise -> look up -> replace
    if (vol_window <= 0) return 0.0;
    activations.push_back(n_new);
    while ((int)activations.size() > vol_window) activations.pop_front();
    long long sum = 0;
    for (int a : activations) sum += a;
    const double len = (double)activations.size();
    const double mean = (double)sum / len;
    double acc = 0.0;
    for (int a : activations) {
      const double d = (double)a - mean;
      acc += d * d;
    }
    const double sigma = std::sqrt(acc / len);
    int level = 0;
    for (double b : vol_bounds) level += sigma >= b;
    rho_hat = vol_rho[level];
    return sigma;
  }
};

extern "C" {

int ts_sched_create(const ts_sched_config* c, ts_sched** out) {
  if (out == nullptr) return TS_ERR_INVALID;
  *out = nullptr;
  if (c == nullptr || c->K < 1 || c->M_max < 1 || c->M0 < 1 || c->M0 > c->M_max || c->l_hat == nullptr) return TS_ERR_INVALID;
  if (!(c->rho_hat > 0.0) || c->rho_hat > 1.0 || c->delta < 0.0 || c->eta < 0.0 || c->vol_window < 0) return TS_ERR_INVALID;
  if (c->l_hat[0] != 0.0) return TS_ERR_INVALID;
  for (int i = 0; i < c->K; ++i)
    if (!(c->l_hat[i] <= c->l_hat[i + 1])) return TS_ERR_INVALID;
  if (c->vol_window > 0) {
    if (c->n_levels < 1 || c->vol_rho == nullptr || (c->n_levels > 1 && c->vol_bounds == nullptr)) return TS_ERR_INVALID;
    for (int i = 0; i < c->n_levels; ++i)
      if (!(c->vol_rho[i] > 0.0) || c->vol_rho[i] > 1.0) return TS_ERR_INVALID;
    for (int i = 0; i + 2 < c->n_levels; ++i)
      if (!(c->vol_bounds[i] <= c->vol_bounds[i + 1])) return TS_ERR_INVALID;
  }
  ts_sched* s = new ts_sched();
  s->K = c->K;
  s->M_max = c->M_max;
  s->vol_window = c->vol_window;
  s->rho_hat = c->rho_hat;
  s->delta = c->delta;
  s->eta = c->eta;
  s->kappa_alpha = c->kappa_alpha;
  s->kappa_beta = c->kappa_beta;
  s->l_hat.assign(c->l_hat, c->l_hat + c->K + 1);
  if (c->vol_window > 0) {
    s->vol_rho.assign(c->vol_rho, c->vol_rho + c->n_levels);
    if (c->n_levels > 1) s->vol_bounds.assign(c->vol_bounds, c->vol_bounds + c->n_levels - 1);
  }
  s->alive.assign(c->M_max, 0);
  for (int j = 0; j < c->M0; ++j) s->alive[j] = 1;
  *out = s;
  return TS_OK;
}

int ts_sched_destroy(ts_sched* s) {
  if (s == nullptr) return TS_ERR_INVALID;
  delete s;
  return TS_OK;
}

int ts_sched_event(ts_sched* s, int32_t n, const int32_t* session_ids, const int32_t* active, const double* state_mb,
                   int32_t* phi_out, ts_sched_result* res) {
  if (s == nullptr || res == nullptr || n < 0) return TS_ERR_INVALID;
  if (n > 0 && (session_ids == nullptr || active == nullptr || state_mb == nullptr || phi_out == nullptr)) return TS_ERR_INVALID;
  std::vector<SessionIn> ev(n);
  std::set<int32_t> active_now, seen;
  for (int i = 0; i < n; ++i) {
    if (session_ids[i] < 0 || !seen.insert(session_ids[i]).second) return TS_ERR_INVALID;
    ev[i] = {session_ids[i], active[i] != 0 ? 1 : 0, state_mb[i]};
    if (ev[i].active) active_now.insert(ev[i].sid);
  }
  int n_new = 0;
  for (int32_t sid : active_now) n_new += !s->known.count(sid);
  const double sigma = s->adapt(n_new);
  s->known = active_now;
  s->moves.clear();
  s->net.clear();
  const std::map<int32_t, int32_t> phi_prev = s->phi;
  const int M_prev = s->n_alive();
  double rho_max = s->place(ev, nullptr);                                   // Algorithm 1, line 1
  const int n_req = (int)active_now.size();
  const int M_tar = s->scale(rho_max, M_prev, n_req);                       // line 2
  if (M_tar < M_prev) {                                                     // lines 3-5: rebalancing precedes removal
    const std::vector<int> ld = s->loads();
    std::vector<int> order;
    for (int j = 0; j < s->M_max; ++j)
      if (s->alive[j]) order.push_back(j);
    std::sort(order.begin(), order.end(), [&](int a, int b) { return ld[a] != ld[b] ? ld[a] < ld[b] : a > b; });
    order.resize(M_prev - M_tar);                                           // least loaded first, ties: highest id
    std::map<int32_t, int32_t> displaced;
    for (const auto& kv : s->phi)
      if (std::find(order.begin(), order.end(), kv.second) != order.end()) displaced[kv.first] = kv.second;
    for (int j : order) s->alive[j] = 0;
    rho_max = s->place(ev, &displaced);
  } else if (M_tar > M_prev) {                                              // lines 6-9: expansion precedes rebalancing
    int need = M_tar - M_prev;
    for (int j = 0; j < s->M_max && need > 0; ++j)
      if (!s->alive[j]) {
        s->alive[j] = 1;
        --need;
      }
    rho_max = s->place(ev, nullptr);
  }
  for (const auto& kv : phi_prev) {
    auto it = s->phi.find(kv.first);
    if (it != s->phi.end() && it->second != kv.second) s->net.push_back({kv.first, kv.second, it->second});
  }
  int unplaced = 0;
  for (int i = 0; i < n; ++i) {
    auto it = s->phi.find(ev[i].sid);
    phi_out[i] = it == s->phi.end() ? -1 : it->second;
    unplaced += ev[i].active && it == s->phi.end();
  }
  res->M = s->n_alive();
  res->n_migrations = (int32_t)s->net.size();
  res->n_moves = (int32_t)s->moves.size();
  res->n_unplaced = unplaced;
  res->n_req = n_req;
  res->reserved = 0;
  res->rho_max = rho_max;
  res->L = s->bottleneck(s->loads());
  res->rho_hat = s->rho_hat;
  res->sigma = sigma;
  return TS_OK;
}

int ts_sched_moves(ts_sched* s, int32_t which, int32_t* sid, int32_t* from_gpu, int32_t* to_gpu, int32_t cap, int32_t* n_out) {
  if (s == nullptr || n_out == nullptr || cap < 0 || (which != 0 && which != 1)) return TS_ERR_INVALID;
  if (cap > 0 && (sid == nullptr || from_gpu == nullptr || to_gpu == nullptr)) return TS_ERR_INVALID;
  const std::vector<Move>& v = which == 0 ? s->net : s->moves;
  *n_out = (int32_t)v.size();
  for (int i = 0; i < std::min<int>(cap, (int)v.size()); ++i) {
    sid[i] = v[i].sid;
    from_gpu[i] = v[i].from;
    to_gpu[i] = v[i].to;
  }
  return TS_OK;
}

int ts_sched_alive(ts_sched* s, int32_t* alive_out) {
  if (s == nullptr || alive_out == nullptr) return TS_ERR_INVALID;
  for (int j = 0; j < s->M_max; ++j) alive_out[j] = s->alive[j];
  return TS_OK;
}

}  // extern "C"
