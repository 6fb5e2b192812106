"""Expert-cache policy simulator -- ORACLE, TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Integers only.  It steps the Expert Cache Engine's policy (§3.2; §4.1,
P:L183-187) exactly as DESIGN.md §4 ("cache policy, readings R6-R13, R25") words it, one decision
at a time.  The CUDA library's cache manager (csrc/ef_api.cu) must reproduce its slot table and
counters bit for bit; the two share no code.

What the paper fixes (and what pins this file, tests/test_oracle_cache.py):
  * PLEC prefetches predicted experts in layer order into one global pool and refills it as
    layers complete -- worked example P:L124 (4 layers x 4 experts, pool of 8).
  * Real-time correction: missed experts are loaded on demand; victims are mis-prefetched experts
    first, then experts that have completed their computation -- P:L130.
  * Prefetch for the next step happens during the current step; experts needed again stay --
    worked example P:L187 ([5,6,7,8] -> [2,3,4,5]: 3 loads, expert 5 retained).
  * Every expert is backed up on the host, so eviction needs no write-back -- P:L338.
What the paper leaves open (tie-breaks, horizon, "completed" under asynchrony) is a DESIGN.md
reading (R8-R13, R25).  Each reading is pinned to a hand-worked scenario whose expected slot table and
counters are literals derived from DESIGN.md section 4's wording (tests/test_oracle_cache.py, "Hand-worked
scenarios"), and a mutation test there demands that every one-line change of the decision logic below
turns one of the pins red.  What stays unpinned is only whether the authors' unpublished code breaks
these ties the same way (there is nothing to compare with).

Baseline policies (the paper's comparison points as policy sketches, "Cache-MoE ... a fixed-size
cache per layer, using a Least-Recently-Used strategy"): `policy="lru"` -- on-demand loading, the victim is an
empty slot, else the least recently used slot of the whole pool; `policy="layer_lru"` -- the same inside the requesting
layer's own S // L slots.  Neither consults predictions; `prefetch` does nothing.  (SE-MoE-like "prefetch all experts of
the next layer", is `policy="plec"` fed an all-ones predicted path with horizon 1.)  Pins: textbook LRU on a
hand-worked reference string and an independent OrderedDict LRU (tests/test_oracle_cache.py).

Vocabulary: visit v = step * L + layer (logical clock).  g = layer * E + e (global expert id).
A slot is *pending* while it holds a prefetched expert that has not been used since its load.
"""
from __future__ import annotations

from dataclasses import dataclass, field

STAT_KEYS = ("lookups", "hits", "misses", "prefetch_issued", "prefetch_used", "prefetch_wasted",
             "ondemand_loads", "evictions", "bytes_h2d")


@dataclass
class VisitPlan:
    """What happened at one visit, in order.  waves[i] = (expert e, slot, loaded_now)."""
    hits: list = field(default_factory=list)
    misses: list = field(default_factory=list)
    waves: list = field(default_factory=list)


class CacheSim:
    def __init__(self, n_layers: int, n_experts: int, n_slots: int, expert_bytes: int, horizon: int = 0,
                 policy: str = "plec"):
        assert n_slots >= 1 and policy in ("plec", "lru", "layer_lru")
        assert policy != "layer_lru" or n_slots >= n_layers
        self.policy = policy
        self.L, self.E, self.S, self.W, self.H = n_layers, n_experts, n_slots, expert_bytes, horizon
        self.slot_expert = [-1] * n_slots     # g or -1
        self.slot_pred_for = [-1] * n_slots   # visit the expert was prefetched for; -1 = loaded on demand
        self.slot_used = [False] * n_slots    # used since load
        self.slot_stamp = [0] * n_slots       # tick of last use (or of the load, if never used): LRU order
        self.tick = 0                         # advances at every load and every use, in call order
        self.slot_of: dict[int, int] = {}     # g -> slot
        self.pred: dict[int, frozenset] = {}  # visit -> predicted batch-level active set (local ids)
        self.stats = {k: 0 for k in STAT_KEYS}
        self.log: list[tuple] = []            # (visit_now, kind, g, slot, evicted_g)

    # ------------------------------------------------------------------ helpers
    def _first_visit_of_layer_after(self, layer: int, v: int) -> int:
        return v + 1 + ((layer - (v + 1)) % self.L)

    def est_next_use(self, g: int, v: int) -> int:
        """First visit > v of g's layer at which g is predicted active; a visit with no supplied
        prediction counts as 'assume used'."""
        layer, e = divmod(g, self.E)
        v2 = self._first_visit_of_layer_after(layer, v)
        while v2 in self.pred and e not in self.pred[v2]:
            v2 += self.L
        return v2

    def _pending(self, s: int) -> bool:
        return self.slot_pred_for[s] != -1 and not self.slot_used[s]

    def _victim(self, v_now: int, target: int, allow3: bool, locked: set):
        """Smallest key wins.  class 0 empty; 1 mis-prefetched (P:L130 'first'); 2 completed with next
        use later than the target (P:L130 'then'); 3 (on-demand last resort) anything else."""
        if self.policy != "plec":
            return self._victim_lru(target % self.L, locked)
        best_key, best_slot = None, None
        for s in range(self.S):
            g = self.slot_expert[s]
            if g < 0:
                key = (0, 0, 0, s)
            elif g in locked:
                continue
            elif self._pending(s) and self.slot_pred_for[s] <= v_now:
                key = (1, 0, self.slot_stamp[s], s)
            else:
                nu = self.est_next_use(g, v_now)
                if not self._pending(s) and nu > target:
                    key = (2, -nu, self.slot_stamp[s], s)
                elif allow3:
                    key = (3, -nu, self.slot_stamp[s], s)
                else:
                    continue
            if best_key is None or key < best_key:
                best_key, best_slot = key, s
        return best_slot

    def _victim_lru(self, layer: int, locked: set):
        """Baselines: the first empty slot, else the least recently used unlocked slot -- of the whole pool ("lru") or
        of the layer's own share of S // L slots ("layer_lru")."""
        lo, hi = 0, self.S
        if self.policy == "layer_lru":
            share = self.S // self.L
            lo, hi = layer * share, (layer + 1) * share
        best = None
        for s in range(lo, hi):
            g = self.slot_expert[s]
            if g < 0:
                return s
            if g in locked:
                continue
            if best is None or self.slot_stamp[s] < self.slot_stamp[best]:
                best = s
        return best

    def _load(self, s: int, g: int, pred_for: int, v_now: int, kind: str):
        old = self.slot_expert[s]
        if old >= 0:
            self.stats["evictions"] += 1
            if self._pending(s):
                self.stats["prefetch_wasted"] += 1
            del self.slot_of[old]
        self.slot_expert[s] = g
        self.slot_pred_for[s] = pred_for
        self.slot_used[s] = False
        self.tick += 1
        self.slot_stamp[s] = self.tick
        self.slot_of[g] = s
        self.stats["bytes_h2d"] += self.W
        self.log.append((v_now, kind, g, s, old))

    # ------------------------------------------------------------------ the three calls
    def visit(self, v: int, counts) -> VisitPlan:
        """Lookup + real-time correction for visit v given the gate's actual per-expert row counts."""
        layer = v % self.L
        plan = VisitPlan()
        act = [e for e in range(self.E) if counts[e] > 0]
        gid = lambda e: layer * self.E + e
        plan.hits = [e for e in act if gid(e) in self.slot_of]
        plan.misses = [e for e in act if gid(e) not in self.slot_of]
        self.stats["lookups"] += len(act)
        self.stats["hits"] += len(plan.hits)
        self.stats["misses"] += len(plan.misses)
        locked = set()
        for e in plan.hits:
            s = self.slot_of[gid(e)]
            if self._pending(s):
                self.stats["prefetch_used"] += 1
            # wave 0 is enqueued first: 'completed' = enqueued (R9).  The lock only keeps phase A off it.
            self.slot_used[s] = True
            self.tick += 1
            self.slot_stamp[s] = self.tick
            locked.add(gid(e))
            plan.waves.append((e, s, False))
        # Phase A: on-demand loads that do not disturb this visit's hits nor still-useful prefetches
        rest = []
        for e in plan.misses:
            s = self._victim(v, v, allow3=False, locked=locked)
            if s is None:
                rest.append(e)
                continue
            self._load(s, gid(e), -1, v, "ondemand")
            self.stats["ondemand_loads"] += 1
            self.slot_used[s] = True
            locked.add(gid(e))
            plan.waves.append((e, s, True))
        # locks drop
        # Phase B: remaining misses, one wave each, may now reuse this visit's completed slots
        for e in rest:
            s = self._victim(v, v, allow3=True, locked=set())
            self._load(s, gid(e), -1, v, "ondemand")
            self.stats["ondemand_loads"] += 1
            self.slot_used[s] = True
            plan.waves.append((e, s, True))
        return plan

    def prefetch(self, v_now: int, predicted) -> int:
        """PLEC refill after visit v_now.  predicted[i] (iterable of 0/1 of length E) is the batch-level
        predicted path of visit v_now+1+i.  Returns the number of loads issued."""
        if self.policy != "plec":
            return 0                            # the LRU baselines neither predict nor prefetch
        n_ahead = len(predicted)
        for i in range(n_ahead):
            self.pred[v_now + 1 + i] = frozenset(e for e in range(self.E) if predicted[i][e])
        for key in [k for k in self.pred if k <= v_now]:
            del self.pred[key]
        hi = v_now + (min(self.H, n_ahead) if self.H > 0 else n_ahead)
        issued = 0
        for t in range(v_now + 1, hi + 1):
            layer = t % self.L
            for e in sorted(self.pred[t]):
                g = layer * self.E + e
                if g in self.slot_of:
                    s = self.slot_of[g]
                    if self._pending(s) and self.slot_pred_for[s] <= v_now:
                        self.slot_pred_for[s] = t   # R25: a stale prefetch predicted again is re-targeted
                    continue
                s = self._victim(v_now, t, allow3=False, locked=set())
                if s is None:
                    return issued               # pool is full of useful experts: stop
                self._load(s, g, t, v_now, "prefetch")
                self.stats["prefetch_issued"] += 1
                issued += 1
        return issued

    def evict(self, layer: int, experts) -> None:
        for e in experts:
            g = layer * self.E + e
            if g not in self.slot_of:
                continue
            s = self.slot_of.pop(g)
            self.stats["evictions"] += 1
            if self._pending(s):
                self.stats["prefetch_wasted"] += 1
            self.slot_expert[s] = -1
            self.slot_pred_for[s] = -1
            self.slot_used[s] = False
            self.slot_stamp[s] = 0

    # ------------------------------------------------------------------ views
    def snapshot(self):
        return list(self.slot_expert)

    def hit_ratio(self) -> float:
        return self.stats["hits"] / max(1, self.stats["lookups"])


def belady_min_loads(n_layers: int, n_experts: int, n_slots: int, actual) -> list:
    """Clairvoyant reference for the policy gap (NOT part of the library's policy): Belady's MIN [farthest next use
    is evicted] on the ACTUAL trace, with demand loading.  actual[v] = iterable of the experts active at visit v (local
    ids; layer = v mod n_layers).  A visit's active experts are served hits first, then misses in ascending id (R12); a
    miss evicts, among the residents that are not still waiting to be served at this visit, the one whose next use lies
    farthest in the future (never used again = infinitely far).  Returns the number of loads at every visit.
    Prefetching cannot lower the NUMBER of loads, only hide their latency, so on a link-bound step this is the floor that
    PLEC's and LRU's bytes_h2d are held against.  With one access per visit this is the textbook OPT (pinned to the
    classic reference string: 9 faults with 3 frames) and it is checked against exhaustive search on small traces."""
    nv = len(actual)
    acts = [sorted(set(int(e) for e in a)) for a in actual]
    gid = lambda v, e: (v % n_layers) * n_experts + e
    # next_use[v][g] = first visit > v at which g is active
    INF = 1 << 60
    nxt_at = [dict() for _ in range(nv)]
    upcoming: dict = {}
    for v in range(nv - 1, -1, -1):
        for e in acts[v]:
            g = gid(v, e)
            nxt_at[v][g] = upcoming.get(g, INF)
        for e in acts[v]:
            upcoming[gid(v, e)] = v
    next_use: dict = {}          # for residents: their next use strictly after the current visit (kept up to date on use)
    cache: set = set()
    loads = []
    for v in range(nv):
        want = [gid(v, e) for e in acts[v]]
        misses = [g for g in want if g not in cache]
        for g in want:                                      # hits are served first: from now on their next use is after v
            if g in cache:
                next_use[g] = nxt_at[v][g]
        n = 0
        for g in misses:
            if len(cache) >= n_slots:
                victim = max(cache, key=lambda r: (next_use[r], r))
                cache.discard(victim)
                del next_use[victim]
            cache.add(g)
            next_use[g] = nxt_at[v][g]
            n += 1
        loads.append(n)
    return loads
