"""Oracle of TurboServe's closed-loop scheduler (TEST INFRASTRUCTURE).

Follows PAPER.md §5.2 step by step, in the paper's notation:
  Algorithm 1 (:203-207)   per event: PLACE -> SCALE -> (scale-in: PLACE under M_tar, then shrink) /
                           (scale-out: grow, then PLACE under the new budget) / (keep the budget).
  PLACE, §5.2.1 (:181-213) initialisation from phi(t-) (:193); session assignment of U(t), Eq. (3) (:195-199):
                           each s_i in U(t) goes to the feasible GPU that minimises the resulting bottleneck latency
                           L(t), fixed tie-break "preferring less-loaded GPUs"; migration-aware min-max rebalancing,
                           Eq. (4) (:201-213): repeat { g_max = argmax_j l_hat_j(n_j); over sessions i on g_max and
                           targets j' != g_max:  Gamma = L - L' - eta * kappa_i ; apply the best move if Gamma > 0 }.
  SCALE, §5.2.2 (:217-245) rho_max = max_j n_j / K; scale-out if rho_max > rho_hat + delta, scale-in if
                           rho_max < rho_hat - delta (:234); M_tar = ceil(N_req / (K * rho_hat)) (:236).
  Volatility mapping, App. A (:447-464): sigma(t) = std(a_{t-W+1..t}) of newly activated sessions per event (Eq. 6),
                           measure -> quantise -> look up -> replace rho_hat.
kappa_i follows the alpha-beta model (:209): kappa_i = alpha + beta * (state size of s_i).

Readings where the paper is silent (R23-R29):
  R23 GPUs have stable ids 0..M_max-1 and an `alive` flag.  Scale-out activates the lowest dead ids.  Scale-in removes the
      least-loaded alive GPUs (ties: highest id): their sessions lose their placement and are re-assigned by the Eq. (3)
      rule ("rebalancing consolidates sessions onto a reduced GPU set", :221), each counted as a migration.
  R24 An active session that fits nowhere (every alive GPU holds K) stays unplaced and is reported; N_req counts the
      sessions with alpha_i = 1 (equal to the paper's |{i : phi_i != empty}| whenever all of them are placed).
  R25 alpha_i = 0  =>  phi_i = empty (suspend releases the GPU slot, :76); a session absent from the event is terminated.
  R26 l_hat_j(n) is one non-decreasing table l_hat[0..K] for every GPU (homogeneous workers), l_hat[0] = 0.
  R27 "similar L(t)" = equal; ties: less-loaded GPU, then lowest id.  Rebalancing ties: smallest kappa_i (it is the
      larger Gamma), then lowest session id, then least-loaded target, then lowest target id; g_max ties: lowest id.
  R28 kappa_i = alpha + beta * state_mb_i.
  R29 a scale-out trigger never lowers M and a scale-in trigger never raises it; M_tar is clamped to [1, M_max]
      (to [ceil(N_req / K), M_max] so that the capacity constraint of Eq. (1) stays satisfiable).
Everything here is integer / exact-double work: the CUDA-side library (csrc/sched.cpp) must reproduce it exactly.
"""
import math
from collections import deque


class SchedulerOracle:
    def __init__(self, K, M_max, M0, l_hat, rho_hat=0.7, delta=0.1, eta=0.0, kappa_alpha=0.0, kappa_beta=0.0,
                 vol_window=0, vol_bounds=(), vol_rho=()):
        assert len(l_hat) == K + 1 and l_hat[0] == 0 and all(l_hat[i] <= l_hat[i + 1] for i in range(K))
        assert 1 <= M0 <= M_max and len(vol_rho) == (len(vol_bounds) + 1 if vol_window else 0)
        self.K, self.M_max, self.l_hat = K, M_max, [float(x) for x in l_hat]
        self.rho_hat, self.delta, self.eta = float(rho_hat), float(delta), float(eta)
        self.kappa_alpha, self.kappa_beta = float(kappa_alpha), float(kappa_beta)
        self.alive = [j < M0 for j in range(M_max)]
        self.phi = {}                    # session id -> GPU id (placed sessions only)
        self.known = set()               # sessions seen at the previous event with alpha = 1
        self.vol_window, self.vol_bounds, self.vol_rho = vol_window, list(vol_bounds), list(vol_rho)
        self.activations = deque(maxlen=vol_window if vol_window else 1)

    # ---- helpers -------------------------------------------------------------------------------------------------
    def _loads(self):
        n = [0] * self.M_max
        for g in self.phi.values():
            n[g] += 1
        return n

    def _L(self, n):
        return max((self.l_hat[n[j]] for j in range(self.M_max) if self.alive[j]), default=0.0)

    def _assign(self, sid, n):
        """Eq. (3): the feasible GPU that minimises the resulting bottleneck latency; ties -> less loaded -> lowest id."""
        best = None
        for j in range(self.M_max):
            if not self.alive[j] or n[j] >= self.K:
                continue
            n[j] += 1
            key = (self._L(n), n[j] - 1, j)
            n[j] -= 1
            if best is None or key < best:
                best = key
        if best is None:
            return False                                             # R24: every alive GPU holds K sessions
        self.phi[sid] = best[2]
        n[best[2]] += 1
        return True

    # ---- PLACE (S(t), phi(t-), M) -> (phi(t), rho_max(t)) ------------------------------------------------------------
    def place(self, sessions, migrations, displaced=None):
        """sessions: list of (sid, alpha, state_mb) in event order.  Mutates self.phi; appends (sid, from, to) moves.
        displaced: sid -> GPU it sat on before that GPU was removed (scale-in); its re-assignment is a migration."""
        displaced = displaced or {}
        live = {sid for sid, _, _ in sessions}
        for sid in list(self.phi):                                   # initialisation (:193): drop terminated sessions
            if sid not in live or not self.alive[self.phi[sid]]:
                del self.phi[sid]
        for sid, alpha, _ in sessions:                               # R25: an idle session holds no GPU slot
            if not alpha:
                self.phi.pop(sid, None)
        n = self._loads()
        for sid, alpha, _ in sessions:                               # session assignment, U(t) of Eq. (3), event order
            if alpha and sid not in self.phi:
                if self._assign(sid, n) and sid in displaced:
                    migrations.append((sid, displaced[sid], self.phi[sid]))
        size = {sid: mb for sid, _, mb in sessions}
        while True:                                                  # migration-aware min-max rebalancing, Eq. (4)
            L = self._L(n)
            gmax = next((j for j in range(self.M_max) if self.alive[j] and self.l_hat[n[j]] == L), None)
            if gmax is None or n[gmax] == 0:
                break
            best = None
            for sid in sorted(s for s, g in self.phi.items() if g == gmax):
                kappa = self.kappa_alpha + self.kappa_beta * size[sid]
                for j in range(self.M_max):
                    if j == gmax or not self.alive[j] or n[j] >= self.K:
                        continue
                    n[gmax] -= 1
                    n[j] += 1
                    gain = L - self._L(n) - self.eta * kappa         # Gamma_{i,j'} = L - L' - eta * kappa_i
                    n[gmax] += 1
                    n[j] -= 1
                    key = (-gain, sid, n[j], j)
                    if best is None or key < best:
                        best = key
            if best is None or not (-best[0] > 0):
                break
            _, sid, _, j = best
            migrations.append((sid, gmax, j))
            self.phi[sid] = j
            n[gmax] -= 1
            n[j] += 1
        return max((n[j] for j in range(self.M_max) if self.alive[j]), default=0) / self.K

    # ---- SCALE (rho_max, M(t-)) -> M_tar ------------------------------------------------------------------------------
    def scale(self, rho_max, M, n_req):
        tar = math.ceil(n_req / (self.K * self.rho_hat))             # proportional target (:236)
        tar = min(self.M_max, max(1, -(-n_req // self.K), tar))      # R29
        if rho_max > self.rho_hat + self.delta:                      # hysteresis trigger (:234)
            return max(M, tar)
        if rho_max < self.rho_hat - self.delta:
            return min(M, tar)
        return M

    # ---- volatility mapping (App. A) ------------------------------------------------------------------------------------
    def _adapt(self, n_new):
        if not self.vol_window:
            return None
        self.activations.append(n_new)                               # measure
        a = list(self.activations)
        mean = sum(a) / len(a)
        acc = 0.0
        for x in a:
            d = x - mean
            acc += d * d
        sigma = math.sqrt(acc / len(a))                              # population std over the window (Eq. 6)
        level = sum(1 for b in self.vol_bounds if sigma >= b)        # quantise: bounds are the interval edges
        self.rho_hat = float(self.vol_rho[level])                    # look up + replace
        return sigma

    # ---- Algorithm 1, one event -------------------------------------------------------------------------------------------
    def event(self, sessions):
        active_now = {sid for sid, alpha, _ in sessions if alpha}
        sigma = self._adapt(len(active_now - self.known))
        self.known = active_now
        migrations = []                                              # log of moves in the order PLACE made them
        phi_prev = dict(self.phi)
        M_prev = sum(self.alive)
        rho_max = self.place(sessions, migrations)                                    # line 1
        n_req = len(active_now)
        M_tar = self.scale(rho_max, M_prev, n_req)                                    # line 2
        if M_tar < M_prev:                                                            # lines 3-5: rebalance, then remove
            n = self._loads()
            victims = sorted((j for j in range(self.M_max) if self.alive[j]), key=lambda j: (n[j], -j))[:M_prev - M_tar]
            displaced = {sid: g for sid, g in self.phi.items() if g in victims}
            for j in victims:
                self.alive[j] = False
            rho_max = self.place(sessions, migrations, displaced)
        elif M_tar > M_prev:                                                          # lines 6-9: grow, then rebalance
            need = M_tar - M_prev
            for j in range(self.M_max):
                if need and not self.alive[j]:
                    self.alive[j] = True
                    need -= 1
            rho_max = self.place(sessions, migrations)
        n = self._loads()
        # what the runtime has to carry out: sessions placed before and after the event, on different GPUs
        net = [(sid, g, self.phi[sid]) for sid, g in sorted(phi_prev.items()) if sid in self.phi and self.phi[sid] != g]
        return {"M": sum(self.alive), "alive": [j for j in range(self.M_max) if self.alive[j]], "rho_max": rho_max,
                "L": self._L(n), "phi": {sid: self.phi.get(sid, -1) for sid, _, _ in sessions},
                "moves": migrations, "migrations": net, "unplaced": sorted(s for s in active_now if s not in self.phi),
                "rho_hat": self.rho_hat, "sigma": sigma, "n_req": n_req}
