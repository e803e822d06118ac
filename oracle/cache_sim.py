"""O3 — logical-time ProMoE expert cache + prefetcher state machine (ORACLE; test infrastructure).

Follows PAPER.md Algorithm 1 "Prefetch Worker Thread", Algorithm 2 "Prefetcher Interface"
(P:233-273), §5.2 early preemption, §5.3 reordered inference and §6.1 "standard
per-layer LRU cache ... accessing experts that are already cached [when adding prefetch tasks], thereby delaying
their eviction", under the LOGICAL-TIME reading of SURVEY.md §8(c) O3:

  In the paper the slot replacement happens when the worker thread pops chunk 0 (Alg. 1 l.3-5) — a wall-clock
  event.  Here every slot-table transition happens at PUSH time, in program order; only the byte copies are
  asynchronous and they never influence the table.  With FetchRate = 1 the two coincide.

Per MoE layer: C slots, each {expert | EMPTY, stamp, origin ∈ {RESIDENT, PRED, PRECISE}}; one global `clock`;
every touch / alloc sets stamp ← ++clock (LRU = smallest stamp).

  push_precise(m, needed)          (Alg. 2 l.11-23; called after the gate of MoE layer m)
     class A: holds a slot with origin ≠ PRED   ("already in the cache")
     class B: holds a slot with origin = PRED   ("currently being prefetched")
     class C: holds no slot                      ("prefetch has not yet begun" → HIGH task, Alg. 2 l.18-20)
     launch order = A (ascending id), B (ascending id), C (ascending id)        (Alg. 2 l.13, l.22; G13)
     touch A then B in that order                                               (Alg. 2 l.15-17 cache.hit)
     for each C in order: alloc(PRECISE); a slot holding a needed expert that has not yet been computed in the
       launch order is pinned (G2); when every slot is pinned (prefill, |needed| > C) the allocation is deferred
       until the next expert in launch order finishes and unpins its slot ("pipeline").
     finally all slots of layer m revert to RESIDENT.
  push_predicted(m, preds)         (Alg. 2 l.1-10; predictor of MoE layer m - stride)
     for e in listed order: holds a slot → touch (Alg. 2 l.3-5); else alloc(PRED); the experts of this
       same list are protected (one push never evicts its own predictions); no victim → SKIP.
     max_spec (SURVEY G3 knob): at most max_spec experts of one push may ALLOCATE (the list is ordered by
       descending predictor score, so the most confident ones go first); further non-cached ones → SKIP.
       Defaults (G3/G7): decode = top_k (every prediction may allocate, as in Alg. 2); prefill = 0 —
       with T > 1 tokens 50-100 % of the experts are needed and a per-layer LRU has no free slot, so
       an allocation only swaps one needed expert for another; predictions then only refresh LRU stamps.

alloc victim (Alg. 1 l.4 `cache.replace_with`): lowest-index EMPTY slot, else smallest stamp among unprotected
(equal stamps — only demoted slots, below — → lowest slot index).

Two switches (readings G16, G17), both off the paper's text:
  reorder=False — the ablation baseline of §7.3 / Fig. 12 WITHOUT reordered inference: the needed experts
     are processed in ascending id (the order a framework loops over them), each classified AT ITS TURN:
     holds a slot → class A / B + touch; holds none → class C, alloc with the plain LRU victim over ALL slots
     ("standard per-layer LRU") — which may be a needed expert whose turn has not come yet: it is then
     fetched again at its own turn (the cache-unfriendly order §5.3 removes).  If the victim's slot holds an expert
     that was launched EARLIER in this layer, `dep` = that launch index (its compute must finish before the copy).
  demote=True — a slot of origin PRED whose expert the gate of its layer did NOT select (a misprediction) gets
     stamp 0 at that gate, before the class-C allocations: it is the next victim, so a wrong prediction costs the
     cache one LRU victim (which the next miss would have taken anyway) instead of a most-recently-used slot.
     The paper keeps mispredicted prefetches as ordinary MRU entries.
  static_slots=S > 0 — the "static" baseline of §7.1: it "caches a fixed set of experts and utilizes two additional
     expert buffers to load any missing experts".  Slots 0..S-1 of every layer are never victims (with a warm start they hold
     experts 0..S-1 for good); only the remaining C - S slots — the staging buffers, S = C - 2 for the paper's two — take
     allocations, by LRU among themselves.  DESIGN.md reading G21.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

EMPTY = -1
RESIDENT, PRED, PRECISE = 0, 1, 2
CLASS_A, CLASS_B, CLASS_C = 0, 1, 2
ACT_TOUCH, ACT_ALLOC, ACT_SKIP = 0, 1, 2


@dataclass
class PreciseRecord:
    """One entry per needed expert, in launch order."""
    expert: List[int] = field(default_factory=list)
    cls: List[int] = field(default_factory=list)
    slot: List[int] = field(default_factory=list)
    victim: List[int] = field(default_factory=list)   # expert evicted by a class-C alloc, -1 = none / EMPTY slot
    dep: List[int] = field(default_factory=list)      # launch-order index whose finish freed the slot, -1 = none

    def as_tuples(self):
        return list(zip(self.expert, self.cls, self.slot, self.victim, self.dep))


@dataclass
class PredRecord:
    """One entry per predicted expert, in listed order."""
    expert: List[int] = field(default_factory=list)
    action: List[int] = field(default_factory=list)
    slot: List[int] = field(default_factory=list)
    victim: List[int] = field(default_factory=list)

    def as_tuples(self):
        return list(zip(self.expert, self.action, self.slot, self.victim))


@dataclass
class CacheStats:
    accesses: int = 0
    hits_resident: int = 0      # class A
    hits_prefetch: int = 0      # class B
    misses: int = 0             # class C
    evictions: int = 0
    predicted: int = 0
    predicted_correct: int = 0
    pred_allocs: int = 0
    need_experts: int = 0       # |needed \ resident at step start| summed (B_need / expert_bytes)

    @property
    def hits(self) -> int:
        return self.hits_resident + self.hits_prefetch


class ProMoECacheSim:
    def __init__(self, n_moe_layers: int, n_experts: int, slots_per_layer: int, warm: bool = True,
                 reorder: bool = True, demote: bool = False, static_slots: int = 0):
        self.L, self.E, self.C = n_moe_layers, n_experts, slots_per_layer
        self.reorder, self.demote = reorder, demote
        assert 0 <= static_slots < slots_per_layer
        self.static_slots = static_slots
        self.slot_expert = [[EMPTY] * self.C for _ in range(self.L)]
        self.stamp = [[0] * self.C for _ in range(self.L)]
        self.origin = [[RESIDENT] * self.C for _ in range(self.L)]
        self.clock = 0
        if warm:   # experts 0..C-1 resident, expert 0 oldest
            for m in range(self.L):
                for i in range(min(self.C, self.E)):
                    self.slot_expert[m][i] = i
                    self.stamp[m][i] = m * self.C + i + 1
            self.clock = self.L * self.C
        self.stats = CacheStats()
        self._pending_pred: Dict[int, List[int]] = {}   # target layer → predicted list of the current step
        self._step_start: List[set] = [set(x for x in row if x != EMPTY) for row in self.slot_expert]

    # -- helpers ---------------------------------------------------------------------------------------------
    def slot_of(self, m: int, e: int) -> int:
        row = self.slot_expert[m]
        return row.index(e) if e in row else -1

    def _touch(self, m: int, s: int) -> None:
        self.clock += 1
        self.stamp[m][s] = self.clock

    def _victim(self, m: int, protected: set) -> int:
        row = self.slot_expert[m]
        for s in range(self.static_slots, self.C):
            if row[s] == EMPTY:
                return s
        best, best_stamp = -1, None
        for s in range(self.static_slots, self.C):
            if row[s] in protected:
                continue
            if best_stamp is None or self.stamp[m][s] < best_stamp:
                best, best_stamp = s, self.stamp[m][s]
        return best

    def _install(self, m: int, s: int, e: int, origin: int) -> int:
        old = self.slot_expert[m][s]
        if old != EMPTY:
            self.stats.evictions += 1
        self.slot_expert[m][s] = e
        self.origin[m][s] = origin
        self._touch(m, s)
        return old

    # -- step protocol ---------------------------------------------------------------------------------------
    def begin_step(self) -> None:
        self._step_start = [set(x for x in row if x != EMPTY) for row in self.slot_expert]
        self._pending_pred = {}

    def _demote_mispredicted(self, m: int, needed: Sequence[int]) -> None:
        for s in range(self.C):
            if self.origin[m][s] == PRED and self.slot_expert[m][s] not in needed:
                self.stamp[m][s] = 0

    def _push_precise_id_order(self, m: int, needed: List[int]) -> PreciseRecord:
        st = self.stats
        rec = PreciseRecord()
        st.accesses += len(needed)
        st.need_experts += len([e for e in needed if e not in self._step_start[m]])
        for i, e in enumerate(needed):
            s = self.slot_of(m, e)
            if s >= 0:
                cls = CLASS_B if self.origin[m][s] == PRED else CLASS_A
                if cls == CLASS_A:
                    st.hits_resident += 1
                else:
                    st.hits_prefetch += 1
                self._touch(m, s)
                rec.expert.append(e); rec.cls.append(cls); rec.slot.append(s); rec.victim.append(-1); rec.dep.append(-1)
                continue
            st.misses += 1
            s = self._victim(m, set())
            old = self.slot_expert[m][s]
            dep = needed.index(old) if old in needed[:i] else -1
            self._install(m, s, e, PRECISE)
            rec.expert.append(e); rec.cls.append(CLASS_C); rec.slot.append(s); rec.victim.append(old); rec.dep.append(dep)
        for s in range(self.C):
            self.origin[m][s] = RESIDENT
        return rec

    def push_precise(self, m: int, needed: Sequence[int]) -> PreciseRecord:
        needed = sorted(set(int(e) for e in needed))
        st = self.stats
        if m in self._pending_pred:
            pred = self._pending_pred.pop(m)
            st.predicted += len(pred)
            st.predicted_correct += len([e for e in pred if e in needed])
        if self.demote:
            self._demote_mispredicted(m, needed)
        if not self.reorder:
            return self._push_precise_id_order(m, needed)
        A = [e for e in needed if self.slot_of(m, e) >= 0 and self.origin[m][self.slot_of(m, e)] != PRED]
        B = [e for e in needed if self.slot_of(m, e) >= 0 and self.origin[m][self.slot_of(m, e)] == PRED]
        Cs = [e for e in needed if self.slot_of(m, e) < 0]
        order = A + B + Cs
        rec = PreciseRecord()
        st.accesses += len(needed)
        st.hits_resident += len(A)
        st.hits_prefetch += len(B)
        st.misses += len(Cs)
        st.need_experts += len([e for e in needed if e not in self._step_start[m]])
        for e in A + B:
            s = self.slot_of(m, e)
            self._touch(m, s)
            rec.expert.append(e); rec.cls.append(CLASS_A if e in A else CLASS_B)
            rec.slot.append(s); rec.victim.append(-1); rec.dep.append(-1)
        unfinished = set(needed)          # pinned while in a slot and not yet computed (G2)
        fin = 0                           # launch-order index of the next expert to finish
        for e in Cs:
            dep = -1
            s = self._victim(m, unfinished)
            while s < 0:                  # every slot pinned: wait for the next finish in launch order
                unfinished.discard(order[fin])
                dep = fin
                fin += 1
                s = self._victim(m, unfinished)
            old = self._install(m, s, e, PRECISE)
            rec.expert.append(e); rec.cls.append(CLASS_C); rec.slot.append(s); rec.victim.append(old); rec.dep.append(dep)
        for s in range(self.C):
            self.origin[m][s] = RESIDENT
        return rec

    def push_predicted(self, m: int, preds: Sequence[int], max_spec: Optional[int] = None) -> PredRecord:
        rec = PredRecord()
        preds = [int(e) for e in preds]
        protected = set(preds)
        self._pending_pred[m] = list(preds)
        allocs = 0
        for e in preds:
            s = self.slot_of(m, e)
            if s >= 0:
                self._touch(m, s)
                rec.expert.append(e); rec.action.append(ACT_TOUCH); rec.slot.append(s); rec.victim.append(-1)
                continue
            s = self._victim(m, protected) if (max_spec is None or allocs < max_spec) else -1
            if s < 0:
                rec.expert.append(e); rec.action.append(ACT_SKIP); rec.slot.append(-1); rec.victim.append(-1)
                continue
            old = self._install(m, s, e, PRED)
            allocs += 1
            self.stats.pred_allocs += 1
            rec.expert.append(e); rec.action.append(ACT_ALLOC); rec.slot.append(s); rec.victim.append(old)
        return rec

    def run_step(self, needed_per_layer: Sequence[Sequence[int]],
                 pred_per_layer: Sequence[Optional[Sequence[int]]], stride: int, max_spec: Optional[int] = None):
        """One prefill/decode step.  needed_per_layer[m] = experts the gate of MoE layer m selected (any token);
        pred_per_layer[m] = list predicted BY the predictor at MoE layer m FOR layer m+stride, or None.
        Order inside a layer: push_precise(m) then push_predicted(m+stride) (SURVEY O3 step 2 then 4; G5: no
        prediction past the last layer, none across steps)."""
        self.begin_step()
        out = []
        for m in range(self.L):
            prec = self.push_precise(m, needed_per_layer[m])
            pr = None
            if pred_per_layer[m] is not None and m + stride < self.L:
                pr = self.push_predicted(m + stride, pred_per_layer[m], max_spec)
            out.append((prec, pr))
        return out
