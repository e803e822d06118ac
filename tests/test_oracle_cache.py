"""Pins for oracle/cache_sim.py (O3) and oracle/accounting.py — CPU only."""
import os
import random
from collections import OrderedDict

import pytest

from oracle.cache_sim import (ACT_ALLOC, ACT_SKIP, ACT_TOUCH, CLASS_A, CLASS_B, CLASS_C, EMPTY, ProMoECacheSim)
from oracle import accounting

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read_gold(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        k, *v = line.split()
        out[k] = v
    return out


def test_fig9_worked_example():
    """PAPER.md Fig. 9, §5.3: prefetched {1,3,4,5}, gate {1,2,4,5} → order 1,4,5,2; 2 is the miss;
    with a 4-slot layer the only evictable expert is 3 (the mispredicted one)."""
    g = _read_gold("fig9_example.txt")
    pref = [int(x) for x in g["prefetched"]]
    gate = [int(x) for x in g["gate"]]
    sim = ProMoECacheSim(1, 8, 4, warm=False)
    sim.begin_step()
    pr = sim.push_predicted(0, pref)
    assert pr.action == [ACT_ALLOC] * 4
    rec = sim.push_precise(0, gate)
    assert rec.expert == [int(x) for x in g["order"]]
    miss = [e for e, c in zip(rec.expert, rec.cls) if c == CLASS_C]
    assert miss == [int(x) for x in g["high_priority"]]
    assert rec.cls == [CLASS_B, CLASS_B, CLASS_B, CLASS_C]
    assert rec.victim[-1] == 3
    assert sim.stats.predicted == 4 and sim.stats.predicted_correct == 3


def test_p85_byte_accounting():
    g = {k: float(v[0]) for k, v in _read_gold("p85_bytes.txt").items()}
    per_tok = accounting.decode_expert_bytes_per_token(int(g["moe_layers"]), int(g["top_k"]), int(g["hidden"]),
                                                       int(g["inter"]), int(g["wbytes"]))
    mib = per_tok / 2 ** 20
    assert round(mib) == 2673                      # the paper prints MiB/1000 as "GiB"
    assert abs(mib / 1000 - g["needed_gib_as_printed"]) < 0.006
    assert abs(mib / 2000 - g["pcie_gib_as_printed"]) < 0.007
    # 1336 MiB in 58.1 ms ≈ 24.1 GB/s, consistent with the printed 23.9 GB/s bandwidth test
    gbs = (per_tok / 2) / (g["fetch_ms"] * 1e-3) / 1e9
    assert abs(gbs - g["bandwidth_test_gbs"]) < 0.5
    assert accounting.expert_bytes(2048, 1408, 2) == 17301504


class TextbookLRU:
    """Independent 10-line LRU (one per layer)."""

    def __init__(self, cap, warm):
        self.cap, self.d = cap, OrderedDict((e, None) for e in warm)

    def access(self, e):
        if e in self.d:
            self.d.move_to_end(e)
            return True, None
        victim = None
        if len(self.d) >= self.cap:
            victim, _ = self.d.popitem(last=False)
        self.d[e] = None
        return False, victim


@pytest.mark.parametrize("warm", [True, False])
def test_reactive_decode_is_textbook_lru(warm):
    """Predictor off + decode (|needed| = k ≤ C): ProMoE's table degenerates to a per-layer LRU accessed in
    the order hits (ascending id) then misses (ascending id)."""
    rng = random.Random(1)
    L, E, C, k = 3, 16, 6, 3
    sim = ProMoECacheSim(L, E, C, warm=warm)
    ref = [TextbookLRU(C, range(C) if warm else []) for _ in range(L)]
    for step in range(300):
        needed = [sorted(rng.sample(range(E), k)) for _ in range(L)]
        out = sim.run_step(needed, [None] * L, stride=1)
        for m in range(L):
            hits = [e for e in needed[m] if e in ref[m].d]
            misses = [e for e in needed[m] if e not in ref[m].d]
            rec = out[m][0]
            assert rec.expert == hits + misses
            victims = []
            for e in hits + misses:
                h, v = ref[m].access(e)
                if not h:
                    victims.append(-1 if v is None else v)
            assert [v for v, c in zip(rec.victim, rec.cls) if c == CLASS_C] == victims
            assert sorted(x for x in sim.slot_expert[m] if x != EMPTY) == sorted(ref[m].d)
    st = sim.stats
    assert st.hits + st.misses == st.accesses == 300 * L * k
    assert st.hits_prefetch == 0


def _check_invariants(sim):
    for m in range(sim.L):
        occ = [e for e in sim.slot_expert[m] if e != EMPTY]
        assert len(occ) == len(set(occ)) <= sim.C
        st = [sim.stamp[m][s] for s in range(sim.C) if sim.slot_expert[m][s] != EMPTY]
        assert len(st) == len(set(st))


def test_full_cache_never_misses_and_counts_add_up():
    rng = random.Random(2)
    L, E, k = 2, 8, 2
    sim = ProMoECacheSim(L, E, E, warm=True)
    for _ in range(100):
        needed = [rng.sample(range(E), k) for _ in range(L)]
        preds = [rng.sample(range(E), k) for _ in range(L)]
        sim.run_step(needed, preds, 1)
        _check_invariants(sim)
    assert sim.stats.misses == 0 and sim.stats.evictions == 0
    assert sim.stats.hits == sim.stats.accesses


@pytest.mark.parametrize("stride", [1, 2, 3])
def test_perfect_prediction_leaves_only_unpredicted_layers_missing(stride):
    """Predictor = the true routing of layer m+stride and C ≥ 2k ⇒ no class-C miss for layers ≥ stride (G5)."""
    rng = random.Random(3)
    L, E, C, k = 6, 32, 8, 4
    sim = ProMoECacheSim(L, E, C, warm=True)
    for _ in range(200):
        needed = [sorted(rng.sample(range(E), k)) for _ in range(L)]
        preds = [needed[m + stride] if m + stride < L else None for m in range(L)]
        out = sim.run_step(needed, preds, stride)
        for m in range(stride, L):
            assert CLASS_C not in out[m][0].cls
        _check_invariants(sim)
    assert sim.stats.predicted == sim.stats.predicted_correct > 0


def test_misses_at_least_compulsory_and_need_accounting():
    rng = random.Random(4)
    L, E, C, k = 4, 16, 4, 3
    sim = ProMoECacheSim(L, E, C, warm=True)
    for _ in range(100):
        start = [set(x for x in row if x != EMPTY) for row in sim.slot_expert]
        needed = [sorted(rng.sample(range(E), k)) for _ in range(L)]
        preds = [rng.sample(range(E), k) for _ in range(L)]
        before = sim.stats.need_experts
        out = sim.run_step(needed, preds, 1)
        comp = sum(len(set(needed[m]) - start[m]) for m in range(L))
        assert sim.stats.need_experts - before == comp
        hb = sum(r.cls.count(CLASS_B) for r, _ in out)
        mc = sum(r.cls.count(CLASS_C) for r, _ in out)
        assert mc + hb >= comp            # everything not resident at step start arrives by prefetch or demand


def test_prediction_never_evicts_its_own_list_and_skips_when_full():
    sim = ProMoECacheSim(1, 8, 2, warm=True)      # slots hold {0,1}
    sim.begin_step()
    rec = sim.push_predicted(0, [5, 6, 7])
    assert rec.action == [ACT_ALLOC, ACT_ALLOC, ACT_SKIP]
    assert sorted(sim.slot_expert[0]) == [5, 6]
    rec = sim.push_predicted(0, [6, 0])
    assert rec.action == [ACT_TOUCH, ACT_ALLOC] and rec.victim[1] == 5


def _replay_plan(sim_before_slots, rec, C):
    """Execute a PreciseRecord physically: copies of deferred allocs wait for `dep`; returns True if every expert is
    present in its slot when it is computed and no slot is overwritten before its occupant was computed."""
    slots = list(sim_before_slots)
    order = rec.expert
    pending = [(i, rec.slot[i], rec.dep[i]) for i in range(len(order)) if rec.cls[i] == CLASS_C]
    done = -1
    for i, e in enumerate(order):
        # perform every copy whose dependency is satisfied (dep <= done), in order
        for (ci, s, dep) in list(pending):
            if dep <= done:
                occupant = slots[s]
                if occupant in order and order.index(occupant) > done:
                    return False          # would overwrite an expert that still has to be computed
                slots[s] = order[ci]
                pending.remove((ci, s, dep))
        if slots[rec.slot[i]] != e:
            return False
        done = i
    return not pending


def test_prefill_slot_recycling_in_launch_order():
    """|needed| > C (prefill): residents first, slots recycled in launch order."""
    rng = random.Random(5)
    E, C = 16, 4
    for trial in range(50):
        sim = ProMoECacheSim(1, E, C, warm=True)
        sim.begin_step()
        if trial % 2:
            sim.push_predicted(0, rng.sample(range(E), 3))
        before = list(sim.slot_expert[0])
        n = rng.randint(C + 1, E)
        needed = sorted(rng.sample(range(E), n))
        rec = sim.push_precise(0, needed)
        assert sorted(rec.expert) == needed
        cls = rec.cls
        assert cls == sorted(cls)                       # A..., B..., C...
        for c in (CLASS_A, CLASS_B, CLASS_C):
            ids = [e for e, x in zip(rec.expert, cls) if x == c]
            assert ids == sorted(ids)
        deps = [d for d in rec.dep if d >= 0]
        assert deps == list(range(len(deps)))           # recycled strictly in launch order
        assert _replay_plan(before, rec, C)
        _check_invariants(sim)
        # the last C experts in launch order are what stays resident
        assert sorted(sim.slot_expert[0]) == sorted(rec.expert[-C:])


def test_cancelled_prediction_keeps_slot_until_lru_evicts_it():
    """an unneeded predicted expert stays logically assigned with the stamp of its prediction."""
    sim = ProMoECacheSim(1, 8, 3, warm=True)      # {0,1,2}, stamps 1,2,3
    sim.begin_step()
    sim.push_predicted(0, [7])                    # evicts 0 (oldest)
    assert sim.slot_of(0, 7) == 0
    rec = sim.push_precise(0, [1, 2])             # 7 not needed
    assert rec.cls == [CLASS_A, CLASS_A]
    assert sim.slot_of(0, 7) == 0 and sim.origin[0] == [0, 0, 0]
    sim.begin_step()
    rec = sim.push_precise(0, [3])                # 7 is now the LRU victim
    assert rec.victim == [7]


# ---- max_spec knob (SURVEY G3 / DESIGN G7): allocations allowed per PushPredicted --------------------------------
def test_max_spec_zero_only_touches():
    """max_spec = 0: a push never allocates; cached predictions are touched (Alg. 2 l.3-5), the rest SKIP, and the
    slot set is unchanged — so demand misses follow the textbook LRU with extra touches."""
    from oracle.cache_sim import ACT_SKIP, ACT_TOUCH, ProMoECacheSim
    sim = ProMoECacheSim(1, 8, 4, warm=True)          # slots: experts 0,1,2,3 ; 0 oldest
    rec = sim.push_predicted(0, [5, 1, 6, 0], max_spec=0)
    assert rec.action == [ACT_SKIP, ACT_TOUCH, ACT_SKIP, ACT_TOUCH]
    assert sorted(sim.slot_expert[0]) == [0, 1, 2, 3] and sim.stats.pred_allocs == 0
    # LRU order is now 2, 3, 1, 0 (oldest first): a demand miss evicts 2
    out = sim.push_precise(0, [7])
    assert out.victim == [2]


def test_max_spec_limits_allocations_in_listed_order():
    from oracle.cache_sim import ACT_ALLOC, ACT_SKIP, ACT_TOUCH, ProMoECacheSim
    sim = ProMoECacheSim(1, 8, 4, warm=True)
    rec = sim.push_predicted(0, [5, 6, 1, 7], max_spec=1)
    assert rec.action == [ACT_ALLOC, ACT_SKIP, ACT_TOUCH, ACT_SKIP]
    assert rec.victim[0] == 0 and sim.stats.pred_allocs == 1
    a = ProMoECacheSim(1, 8, 4, warm=True); b = ProMoECacheSim(1, 8, 4, warm=True)
    ra = a.push_predicted(0, [5, 6, 1, 7]); rb = b.push_predicted(0, [5, 6, 1, 7], max_spec=4)
    assert ra.as_tuples() == rb.as_tuples() and a.slot_expert == b.slot_expert    # None ≡ no limit
