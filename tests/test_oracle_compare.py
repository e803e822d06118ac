"""Pins for oracle/compare.py (parity protocol P1-P4) and the forced-selection branch of OracleModel._moe — CPU only.

These functions decide whether a GPU/oracle disagreement is "a counted near tie" or a failure, so each is tied to
constructed cases with hand values: a selection swap with an exact logit gap of 5e-4 must be accepted, counted and
forced (gates recomputed); the same swap at 2e-3 must raise; duplicates / out-of-range ids must raise; vote
intervals and predicted-list acceptance are checked against brute-force enumeration of every margin-consistent
per-token top-k.
"""
import itertools
import math
import random

import numpy as np
import pytest
import torch

import synth
from oracle import compare as Cmp
from oracle import forward as O
from oracle.predictor import predict_experts, topk_desc

F64 = torch.float64


def tiny_cfg(**shape_over):
    base = dict(n_layers=2, hidden=64, n_q_heads=4, n_kv_heads=2, head_dim=16, vocab=50, max_seq=32,
                n_experts=8, top_k=2, expert_inter=32, pred_hidden=32, wdtype=0, router_bias=1)
    base.update(shape_over)
    shape = synth.Shape(**base)
    return synth.RunConfig("tiny", shape, seed=11, cache_slots=4 * shape.n_moe_layers, stride=1, prompt_len=6,
                           decode_steps=2, zipf_s=0.3)


# ---- _consistent ---------------------------------------------------------------------------------------------------
def test_consistent_hand_cases():
    z = torch.tensor([3.0, 2.0, 2.0 - 5e-4, 1.0, 2.0 - 2e-3], dtype=F64)
    assert Cmp._consistent([0, 1], z, 2)                 # the exact top-2
    assert Cmp._consistent([0, 2], z, 2)                 # k-th swapped with a neighbour 5e-4 below: near tie
    assert not Cmp._consistent([0, 4], z, 2)             # 2e-3 below: a real mismatch
    assert not Cmp._consistent([1, 0], z, 2)             # order inside the list matters (descending logit), gap 1.0
    assert Cmp._consistent([0, 2, 1], z, 3)              # 1 and 2 listed in the other order, 5e-4 apart
    assert not Cmp._consistent([0, 1, 4], z, 3)          # leaves out expert 2 for one 1.5e-3 weaker
    assert not Cmp._consistent([0, 0], z, 2)             # duplicate
    assert not Cmp._consistent([0, 5], z, 2)             # out of range
    assert not Cmp._consistent([0, -1], z, 2)            # negative ids must not wrap around
    assert not Cmp._consistent([0], z, 2)                # wrong length
    assert Cmp._consistent([0, 1, 2, 4, 3], z, 5)        # k = E: only the internal order is checked
    assert not Cmp._consistent([0, 1, 2, 3, 4], z, 5)    # 3 (1.0) listed before 4 (1.998)


def test_consistent_agrees_with_bruteforce_on_random_near_ties():
    """Brute force: a list is margin-consistent iff a perturbation of z by at most MARGIN/2 per entry makes it the exact
    descending top-k — for two values a, b that is a >= b - MARGIN.  Enumerate every ordered k-subset of small cases."""
    rng = random.Random(3)
    for _ in range(60):
        E, k = rng.randint(3, 5), rng.randint(1, 3)
        vals = [rng.choice([0.0, 4e-4, 9e-4, 1.4e-3, 5e-3, 1.0]) + rng.choice([0.0, 1.0]) for _ in range(E)]
        z = torch.tensor(vals, dtype=F64)
        for order in itertools.permutations(range(E), k):
            zs = [vals[e] for e in order]
            rest = [vals[e] for e in range(E) if e not in order]
            want = all(a >= b - Cmp.MARGIN for a, b in zip(zs, zs[1:])) and (not rest or min(zs) >= max(rest) - Cmp.MARGIN)
            assert Cmp._consistent(list(order), z, k) == want


# ---- oracle_step_matching + the override branch of OracleModel._moe ---------------------------------------------------
def _model_with_gap(gap: float, t: int = 2):
    """Tiny 2-layer MoE whose layer-0 router logits of token t have z_(k) - z_(k+1) == gap exactly (set through the
    per-expert router bias, which adds to the logits)."""
    cfg = tiny_cfg()
    w = synth.make_weights(cfg, pin=False)
    E, k = cfg.shape.n_experts, cfg.shape.top_k
    ids = synth.make_prompt(cfg, 5)
    w.dense["l0.router_bias"] = torch.zeros(E, dtype=torch.float64)
    z = O.OracleModel(w, use_predictor=False).forward(ids).layers[0].logits[t]
    order = sorted(range(E), key=lambda i: (-z[i].item(), i))
    ek, en = order[k - 1], order[k]
    b = torch.zeros(E, dtype=torch.float64)
    b[en] = (z[ek] - gap) - z[en]                       # z[en] + b = z[ek] - gap
    w.dense["l0.router_bias"] = b
    return cfg, w, ids, t, ek, en


def test_near_tie_swap_is_accepted_counted_and_forced():
    cfg, w, ids, t, ek, en = _model_with_gap(5e-4)
    k = cfg.shape.top_k
    plain = O.OracleModel(w, use_predictor=False).forward(ids)
    assert plain.layers[0].sel[t][-1] == ek and abs(plain.layers[0].margin[t] - 5e-4) < 1e-12
    # the "GPU" took the runner-up instead of the k-th at (layer 0, token t); its later layers saw that input
    swapped = list(plain.layers[0].sel[t][:-1]) + [en]
    gpu_model = O.OracleModel(w, use_predictor=False)
    gpu_model.overrides[(0, 0, t)] = swapped
    gpu_sel = np.array([[row for row in lt.sel] for lt in gpu_model.forward(ids).layers], dtype=np.int32)
    assert gpu_sel[0, t].tolist() == swapped
    o = O.OracleModel(w, use_predictor=False)
    rep = Cmp.ParityReport()
    st = Cmp.oracle_step_matching(o, ids, gpu_sel, rep)
    assert rep.sel_near_tie == 1 and rep.reruns == 1
    assert o.overrides == {(0, 0, t): [int(x) for x in gpu_sel[0, t]]}
    assert st.layers[0].sel[t] == [int(x) for x in gpu_sel[0, t]]
    # gates recomputed over the FORCED experts' logits: hand value
    z = st.layers[0].logits[t]
    zs = [z[int(e)].item() for e in gpu_sel[0, t]]
    ex = [math.exp(v - max(zs)) for v in zs]
    assert st.layers[0].gates[t] == pytest.approx([v / sum(ex) for v in ex], abs=1e-15)
    assert abs(sum(st.layers[0].gates[t]) - 1.0) < 1e-15
    # the step was re-run from a snapshot, not appended: one step's worth of state
    assert o.pos == len(ids) and o.step_idx == 1 and o.kcache[0].shape[0] == len(ids)
    # the forced expert really is the one computed: layer 0 changes only token t, so by causality rows < t keep
    # their values through the whole stack and row t moves
    assert torch.allclose(st.hidden[:t], plain.hidden[:t], atol=1e-13)
    assert (st.hidden[t] - plain.hidden[t]).abs().max() > 1e-6
    # hand recomputation of the forced MoE output of (layer 0, token t)
    u_probe = O.OracleModel(w, use_predictor=False)
    x = w.dense["emb"][torch.as_tensor(ids, dtype=torch.long)].to(F64)
    h = x + u_probe._attention(0, O.rmsnorm(x, w.dense["l0.ln1"], cfg.shape.rms_eps))
    u = O.rmsnorm(h, w.dense["l0.ln2"], cfg.shape.rms_eps)
    y = sum(g * O.swiglu_ffn(u[t:t + 1], *w.expert_views(0, int(e)))[0] for g, e in zip(st.layers[0].gates[t], gpu_sel[0, t]))
    forced = O.OracleModel(w, use_predictor=False)
    forced.overrides[(0, 0, t)] = [int(e) for e in gpu_sel[0, t]]
    y_model, _ = forced._moe(0, 0, u)
    assert torch.allclose(y_model[t], y, atol=1e-13)


def test_override_with_the_oracles_own_selection_is_a_no_op():
    cfg, w, ids, t, _, _ = _model_with_gap(5e-4)
    plain = O.OracleModel(w, use_predictor=False).forward(ids)
    o = O.OracleModel(w, use_predictor=False)
    o.overrides[(0, 0, t)] = list(plain.layers[0].sel[t])
    st = o.forward(ids)
    assert torch.equal(st.hidden, plain.hidden) and st.layers[0].gates == plain.layers[0].gates


def test_swap_outside_the_margin_raises():
    cfg, w, ids, t, ek, en = _model_with_gap(2e-3)
    k = cfg.shape.top_k
    plain = O.OracleModel(w, use_predictor=False).forward(ids)
    gpu_sel = np.array([[row for row in lt.sel] for lt in plain.layers], dtype=np.int32)
    gpu_sel[0, t, k - 1] = en
    rep = Cmp.ParityReport()
    with pytest.raises(AssertionError, match="outside"):
        Cmp.oracle_step_matching(O.OracleModel(w, use_predictor=False), ids, gpu_sel, rep)
    assert rep.sel_near_tie == 0


@pytest.mark.parametrize("bad", ["duplicate", "out_of_range", "negative"])
def test_malformed_gpu_selection_raises(bad):
    cfg, w, ids, t, ek, en = _model_with_gap(5e-4)
    plain = O.OracleModel(w, use_predictor=False).forward(ids)
    gpu_sel = np.array([[row for row in lt.sel] for lt in plain.layers], dtype=np.int32)
    gpu_sel[0, t, 1] = {"duplicate": gpu_sel[0, t, 0], "out_of_range": cfg.shape.n_experts, "negative": -1}[bad]
    with pytest.raises(AssertionError):
        Cmp.oracle_step_matching(O.OracleModel(w, use_predictor=False), ids, gpu_sel, Cmp.ParityReport())


def test_matching_selection_needs_no_rerun_and_decode_steps_key_on_step_index():
    cfg, w, ids, t, ek, en = _model_with_gap(5e-4)
    o = O.OracleModel(w, use_predictor=False)
    ref = O.OracleModel(w, use_predictor=False)
    rep = Cmp.ParityReport()
    plain = ref.forward(ids)
    gpu_sel = np.array([[row for row in lt.sel] for lt in plain.layers], dtype=np.int32)
    st = Cmp.oracle_step_matching(o, ids, gpu_sel, rep)
    assert rep.reruns == 0 and rep.sel_near_tie == 0 and torch.equal(st.hidden, plain.hidden)
    # second step (decode): an override recorded for step 1 must not leak into a later step
    d = ref.decode(7)
    sel1 = np.array([[row for row in lt.sel] for lt in d.layers], dtype=np.int32)
    st1 = Cmp.oracle_step_matching(o, [7], sel1, rep)
    assert torch.equal(st1.logits, d.logits) and o.step_idx == 2 and not o.overrides


# ---- predicted lists: vote intervals and per-decision acceptance -------------------------------------------------------
def _all_consistent_topk(row, k):
    """Every margin-consistent top-k SET of one token (brute force over subsets)."""
    E = len(row)
    out = []
    for sub in itertools.combinations(range(E), k):
        rest = [row[e] for e in range(E) if e not in sub]
        if not rest or min(row[e] for e in sub) >= max(rest) - Cmp.MARGIN:
            out.append(sub)
    return out


def _list_from_votes(votes, cap):
    order = sorted((e for e in range(len(votes)) if votes[e] > 0), key=lambda e: (-votes[e], e))
    return order[:cap]


def test_vote_bounds_hand_case():
    sc = torch.tensor([[1.0, 0.0, 0.0, 0.0],
                       [0.0, 1.0, 0.0, 0.0],
                       [1.0, 1.0 - 5e-4, 0.0, 0.0],        # near tie between experts 0 and 1
                       [0.0, 0.0, 1.0, 1.0 - 2e-3]], dtype=F64)   # 2e-3: not a near tie
    lo, hi = Cmp.vote_bounds(sc, 1)
    assert lo == [1, 1, 1, 0] and hi == [2, 2, 1, 0]
    assert predict_experts(sc, 1, 4) == [0, 1, 2]
    assert Cmp.pred_list_acceptable([1, 0, 2], sc, 1, 4)         # token 2 flipped: votes 1/2/1
    assert Cmp.pred_list_acceptable([0, 1, 2], sc, 1, 4)
    assert not Cmp.pred_list_acceptable([0, 2, 1], sc, 1, 4)     # expert 2 (1 vote) can never precede expert 1 (>= 1, lower id)
    assert not Cmp.pred_list_acceptable([0, 1, 3], sc, 1, 4)     # expert 3 never gets a vote
    assert not Cmp.pred_list_acceptable([0, 1], sc, 1, 4)        # expert 2 certainly has a vote: list too short
    assert not Cmp.pred_list_acceptable([0, 0, 2], sc, 1, 4)     # duplicate
    assert not Cmp.pred_list_acceptable([0, 1, 4], sc, 1, 4)     # out of range
    assert Cmp.pred_list_acceptable([1], sc, 1, 1) and Cmp.pred_list_acceptable([0], sc, 1, 1)   # cap 1
    assert not Cmp.pred_list_acceptable([2], sc, 1, 1)
    wide = sc.clone(); wide[2, 1] = 1.0 - 2e-3                  # same construction, gap 2e-3: nothing may flip
    assert Cmp.vote_bounds(wide, 1) == ([2, 1, 1, 0], [2, 1, 1, 0])
    assert not Cmp.pred_list_acceptable([1, 0, 2], wide, 1, 4)
    # decode (T = 1): the list is the token's top-k in descending order up to the margin
    one = torch.tensor([[0.5, 0.9, 0.9 - 5e-4, 0.1]], dtype=F64)
    assert Cmp.pred_list_acceptable([2, 1], one, 2, 4) and not Cmp.pred_list_acceptable([1, 0], one, 2, 4)


def test_pred_list_acceptance_against_bruteforce_enumeration():
    """Soundness: every list reachable by flipping near-tie tokens is accepted (no false failures), and the oracle's own
    list is one of them.  Sharpness: with no near tie at all, ONLY the oracle's list is accepted."""
    rng = random.Random(5)
    for trial in range(40):
        T, E, k, cap = rng.randint(2, 5), rng.randint(3, 5), rng.randint(1, 2), rng.randint(1, 5)
        near = trial % 2 == 0
        rows = []
        for _ in range(T):
            base = rng.sample([0.0, 0.3, 0.6, 0.9, 1.2, 1.5], E) if E <= 6 else None
            if near and rng.random() < 0.7:
                i, j = rng.sample(range(E), 2)
                base[j] = base[i] - rng.choice([2e-4, 6e-4])
            rows.append(base)
        sc = torch.tensor(rows, dtype=F64)
        reachable = set()
        for choice in itertools.product(*[_all_consistent_topk(r, k) for r in rows]):
            votes = [0] * E
            for sub in choice:
                for e in sub:
                    votes[e] += 1
            reachable.add(tuple(_list_from_votes(votes, cap)))
        want = tuple(predict_experts(sc, k, cap))
        assert want in reachable
        for lst in reachable:
            assert Cmp.pred_list_acceptable(list(lst), sc, k, cap), (rows, k, cap, lst)
        if not near:
            assert reachable == {want}
            for lst in itertools.permutations(range(E), len(want)):
                assert Cmp.pred_list_acceptable(list(lst), sc, k, cap) == (lst == want)


def test_compare_step_rejects_a_wrong_vote_list_at_realistic_T():
    """The round-1 escape (one global minimum gap over all T tokens) accepted ANY list once T was large; the
    per-decision check must reject a wrong list even when some unrelated token has a near tie."""
    torch.manual_seed(0)
    T, E, k, cap = 512, 16, 2, 8
    sc = torch.randn(T, E, dtype=F64)
    sc[7, 1] = sc[7].max() + 1.0; sc[7, 2] = sc[7, 1] - 1e-5          # token 7: near tie INSIDE its top-2 (no vote moves)
    want = predict_experts(sc, k, cap)
    wrong = list(reversed(want))
    assert Cmp.pred_list_acceptable(want, sc, k, cap)
    assert not Cmp.pred_list_acceptable(wrong, sc, k, cap)
    assert not Cmp.pred_list_acceptable(want[:-1] + [[e for e in range(E) if e not in want][0]], sc, k, cap)
