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


# ---- reorder = False: the ID-order ablation baseline (Fig. 12 "Base") ------------------------------------
@pytest.mark.parametrize("warm", [True, False])
@pytest.mark.parametrize("T_experts", [3, 9])
def test_id_order_is_textbook_lru_in_ascending_id(warm, T_experts):
    """Without reordered inference the table is a standard per-layer LRU accessed in ascending expert id — also
    in prefill, where |needed| > C and a needed expert may be evicted before its turn and fetched again."""
    rng = random.Random(7)
    L, E, C = 2, 16, 6
    sim = ProMoECacheSim(L, E, C, warm=warm, reorder=False)
    ref = [TextbookLRU(C, range(C) if warm else []) for _ in range(L)]
    for step in range(200):
        needed = [sorted(rng.sample(range(E), T_experts)) for _ in range(L)]
        out = sim.run_step(needed, [None] * L, stride=1)
        for m in range(L):
            rec = out[m][0]
            assert rec.expert == needed[m]                      # launch order = ascending id
            for i, e in enumerate(needed[m]):
                hit, v = ref[m].access(e)
                assert (rec.cls[i] == CLASS_A) == hit
                if not hit:
                    assert rec.victim[i] == (-1 if v is None else v)
                    # the victim was launched earlier in this layer → its compute must finish first
                    assert rec.dep[i] == (needed[m].index(v) if v in needed[m][:i] else -1)
            assert sorted(x for x in sim.slot_expert[m] if x != EMPTY) == sorted(ref[m].d)
    assert sim.stats.hits + sim.stats.misses == sim.stats.accesses == 200 * L * T_experts


def test_id_order_thrashes_where_reorder_does_not():
    """§5.3: slots {5,6,7,8} hold 5 (oldest) .. 8, the gate needs {1,5,6}.  Reordered: 5, 6 first (touched), then
    1 evicts 7 → one miss.  ID order: 1 comes first and evicts 5 (the LRU entry, needed later), 5 then misses and evicts 6,
    6 misses and evicts 7 → three misses for the same access set."""
    def build(reorder):
        sim = ProMoECacheSim(1, 16, 4, warm=False, reorder=reorder)
        sim.begin_step()
        sim.push_precise(0, [5]); sim.push_precise(0, [6]); sim.push_precise(0, [7]); sim.push_precise(0, [8])
        sim.begin_step()
        return sim
    a = build(True)
    ra = a.push_precise(0, [1, 5, 6])
    assert ra.as_tuples() == [(5, CLASS_A, 0, -1, -1), (6, CLASS_A, 1, -1, -1), (1, CLASS_C, 2, 7, -1)]
    b = build(False)
    rb = b.push_precise(0, [1, 5, 6])
    assert rb.as_tuples() == [(1, CLASS_C, 0, 5, -1), (5, CLASS_C, 1, 6, -1), (6, CLASS_C, 2, 7, -1)]
    assert b.stats.misses - 4 == 3 and a.stats.misses - 4 == 1
    assert b.stats.need_experts == a.stats.need_experts            # B_need = the reorder-achievable minimum either way


# ---- demote = True: a mispredicted prefetch becomes the next victim (G17) ----------------------------------
def test_demoted_misprediction_is_the_next_victim():
    """4 slots hold 0 (oldest), 1, 2, 3.  Prediction {9} for the layer allocates over 0.  The gate then needs {1, 7}:
    9 was NOT selected.  Paper behaviour (demote off): 9 stays most recently used, the miss 7 evicts 2 (1 was just
    touched) — two useful experts lost to one wrong guess.  With demotion 9's slot is the victim of 7: only expert 0,
    the LRU entry the next miss would have taken anyway, is lost."""
    for demote, want_victim, want_set in ((False, 2, [1, 3, 7, 9]), (True, 9, [1, 2, 3, 7])):
        sim = ProMoECacheSim(1, 16, 4, warm=True, demote=demote)
        sim.begin_step()
        pr = sim.push_predicted(0, [9], max_spec=1)
        assert pr.as_tuples() == [(9, ACT_ALLOC, 0, 0)]
        rec = sim.push_precise(0, [1, 7])
        assert rec.as_tuples() == [(1, CLASS_A, 1, -1, -1), (7, CLASS_C, 0 if demote else 2, want_victim, -1)]
        assert sorted(sim.slot_expert[0]) == want_set
        assert sim.stats.predicted == 1 and sim.stats.predicted_correct == 0


def test_demotion_leaves_correct_predictions_and_other_layers_alone():
    """A correct prediction is class B (touched, kept); demotion happens at the slot's OWN gate only; two demoted slots
    are taken in slot order (equal stamps → lowest slot index)."""
    sim = ProMoECacheSim(2, 16, 4, warm=True, demote=True)
    sim.begin_step()
    sim.push_predicted(1, [9, 10, 11], max_spec=3)                 # layer 1: slots 0,1,2 ← 9,10,11 (PRED)
    r0 = sim.push_precise(0, [0, 1])                                # the gate of layer 0 does not touch layer 1
    assert [c for c in r0.cls] == [CLASS_A, CLASS_A]
    assert sim.slot_expert[1][:3] == [9, 10, 11] and all(sim.stamp[1][s] > 0 for s in range(3))
    r1 = sim.push_precise(1, [10, 12, 13])                          # 10 was right; 9 and 11 were not
    assert r1.as_tuples() == [(10, CLASS_B, 1, -1, -1), (12, CLASS_C, 0, 9, -1), (13, CLASS_C, 2, 11, -1)]
    assert sim.slot_expert[1] == [12, 10, 13, 3]
    _check_invariants(sim)


def test_demotion_never_changes_outputs_of_a_reactive_run():
    """No predictions → no PRED slots → demotion is a no-op (same records, same tables)."""
    rng = random.Random(3)
    a, b = ProMoECacheSim(2, 12, 5), ProMoECacheSim(2, 12, 5, demote=True)
    for _ in range(100):
        needed = [sorted(rng.sample(range(12), 3)) for _ in range(2)]
        ra, rb = a.run_step(needed, [None, None], 1), b.run_step(needed, [None, None], 1)
        assert [x[0].as_tuples() for x in ra] == [x[0].as_tuples() for x in rb]
    assert a.slot_expert == b.slot_expert and a.stamp == b.stamp


# ---- static_slots: the "static" baseline (a fixed set + two staging buffers) -------------------------------------
def test_static_cache_keeps_its_fixed_set_and_cycles_two_buffers():
    """C = 6, 4 static slots (experts 0..3 for good) + 2 staging buffers.  Misses alternate between the two buffers by LRU;
    an expert of the fixed set always hits; nothing ever lands in slots 0..3."""
    rng = random.Random(4)
    L, E, C, k = 2, 16, 6, 3
    sim = ProMoECacheSim(L, E, C, warm=True, static_slots=C - 2)
    staging = [TextbookLRU(2, [4, 5]) for _ in range(L)]          # the warm start put experts 4, 5 into the two buffers
    for step in range(200):
        needed = [sorted(rng.sample(range(E), k)) for _ in range(L)]
        out = sim.run_step(needed, [None] * L, stride=1)
        for m in range(L):
            rec = out[m][0]
            assert sim.slot_expert[m][:4] == [0, 1, 2, 3]
            hits = [e for e in needed[m] if e < 4 or e in staging[m].d]
            misses = [e for e in needed[m] if e >= 4 and e not in staging[m].d]
            assert rec.expert == hits + misses and [c for c in rec.cls] == [CLASS_A] * len(hits) + [CLASS_C] * len(misses)
            assert all(s >= 4 for s, c in zip(rec.slot, rec.cls) if c == CLASS_C)
            for e in hits + misses:
                if e >= 4:
                    staging[m].access(e)
            # a buffer that holds a needed expert is pinned until that expert has been computed (G2): more buffer users
            # (hits in a buffer + misses) than buffers → the last miss waits for a finish (dep)
            if len([e for e in hits if e >= 4]) + len(misses) <= 2:
                assert all(d == -1 for d in rec.dep)
            else:
                assert rec.dep[-1] >= 0
            assert sorted(sim.slot_expert[m][4:]) == sorted(staging[m].d)
    # against the LRU cache of the same size on the same stream: the static cache never evicts its fixed set
    assert sim.stats.hits + sim.stats.misses == sim.stats.accesses


def test_static_cache_three_misses_wait_for_a_buffer():
    """Hand-worked: buffers hold 4 (older), 5.  Gate needs {1, 7, 8, 9}: 1 hits; 7 -> buffer of 4, 8 -> buffer of 5, 9 has no
    unpinned buffer left (7 and 8 are needed and not yet computed) and waits for launch position 0 ... the first finish
    that frees a BUFFER is position 1 (expert 7): dep = 1."""
    sim = ProMoECacheSim(1, 16, 6, warm=True, static_slots=4)
    sim.begin_step()
    rec = sim.push_precise(0, [1, 7, 8, 9])
    assert rec.as_tuples() == [(1, CLASS_A, 1, -1, -1), (7, CLASS_C, 4, 4, -1), (8, CLASS_C, 5, 5, -1), (9, CLASS_C, 4, 7, 1)]
