"""Pins for oracle/forward.py (O1), oracle/predictor.py (O2), oracle/permute.py — CPU only.

Each pin ties a function to something other than itself: closed forms, brute force, torch library routines
(fp64 rms_norm / scaled_dot_product_attention), special cases, and an independently written compact model."""
import math
import random
from dataclasses import replace

import pytest
import torch
import torch.nn.functional as F

import synth
from oracle import forward as O
from oracle.permute import permutation
from oracle.predictor import predict_experts, predictor_scores, topk_desc

F64 = torch.float64


def tiny_cfg(**shape_over):
    base = dict(n_layers=2, hidden=64, n_q_heads=4, n_kv_heads=2, head_dim=16, vocab=50, max_seq=32,
                n_experts=8, top_k=2, expert_inter=32, pred_hidden=32, wdtype=0)
    base.update(shape_over)
    shape = synth.Shape(**base)
    return synth.RunConfig("tiny", shape, seed=7, cache_slots=4 * shape.n_moe_layers, stride=1, prompt_len=9,
                           decode_steps=3, zipf_s=0.3)


# ---- building blocks ----------------------------------------------------------------------------------------
def test_rmsnorm_matches_library_and_closed_form():
    torch.manual_seed(0)
    x = torch.randn(5, 48, dtype=F64)
    w = torch.randn(48)
    got = O.rmsnorm(x, w, 1e-6)
    assert torch.allclose(got, F.rms_norm(x, (48,), w.double(), 1e-6), atol=1e-14)
    c = torch.full((1, 48), 3.0, dtype=F64)        # constant vector → every entry = w·3/sqrt(9+eps)
    assert torch.allclose(O.rmsnorm(c, torch.ones(48), 0.0), torch.ones(1, 48, dtype=F64))


def test_rope_closed_forms():
    torch.manual_seed(1)
    q = torch.randn(6, 3, 16, dtype=F64)
    k = torch.randn(6, 3, 16, dtype=F64)
    pos = torch.arange(6)
    assert torch.allclose(O.rope(q, torch.zeros(6, dtype=torch.long), 10000.0), q)           # position 0 = identity
    assert torch.allclose(O.rope(q, pos, 10000.0).norm(dim=-1), q.norm(dim=-1))              # rotations keep norms
    # <R_m q, R_n k> depends on m - n only
    a = (O.rope(q[:1], torch.tensor([7]), 1e4) * O.rope(k[:1], torch.tensor([3]), 1e4)).sum()
    b = (O.rope(q[:1], torch.tensor([14]), 1e4) * O.rope(k[:1], torch.tensor([10]), 1e4)).sum()
    assert abs(a - b) < 1e-12
    # explicit pair (i, i+d/2), angle pos·θ^(−2i/d): d = 4, pos = 2, i = 1
    x = torch.tensor([[[1.0, 2.0, 3.0, 4.0]]], dtype=F64)
    ang = 2 * 100.0 ** (-2 * 1 / 4)
    y = O.rope(x, torch.tensor([2]), 100.0)[0, 0]
    assert abs(y[1] - (2 * math.cos(ang) - 4 * math.sin(ang))) < 1e-14
    assert abs(y[3] - (4 * math.cos(ang) + 2 * math.sin(ang))) < 1e-14


def test_swiglu_matches_library():
    torch.manual_seed(2)
    u = torch.randn(4, 16, dtype=F64)
    wg, wu, wd = torch.randn(24, 16), torch.randn(24, 16), torch.randn(16, 24)
    ref = F.linear(F.silu(F.linear(u, wg.double())) * F.linear(u, wu.double()), wd.double())
    assert torch.allclose(O.swiglu_ffn(u, wg, wu, wd), ref, atol=1e-13)


def test_route_bruteforce_ties_and_special_cases():
    rng = random.Random(0)
    for _ in range(200):
        E = rng.randint(2, 9)
        k = rng.randint(1, E)
        z = torch.tensor([rng.choice([-1.0, 0.0, 0.5, 1.0, 2.0]) for _ in range(E)], dtype=F64)   # many exact ties
        sel, g, margin = O.route(z, k)
        brute = sorted(range(E), key=lambda i: (-z[i].item(), i))[:k]
        assert sel == brute
        assert abs(sum(g) - 1.0) < 1e-15 * 8
        if k == E:
            assert torch.allclose(torch.tensor(g, dtype=F64), torch.softmax(z[sel], 0))
            assert margin == float("inf")
        else:
            rest = sorted(range(E), key=lambda i: (-z[i].item(), i))[k]
            assert margin == z[sel[-1]].item() - z[rest].item() >= 0
        if k == 1:
            assert g == [1.0]
    # constructed tie: lower index wins and is listed first
    sel, _, margin = O.route(torch.tensor([0.3, 0.9, 0.9, 0.1], dtype=F64), 1)
    assert sel == [1] and margin == 0.0


def test_attention_matches_sdpa_gqa_causal_and_kv_cache():
    cfg = tiny_cfg()
    w = synth.make_weights(cfg, pin=False)
    s = cfg.shape
    m = O.OracleModel(w, use_predictor=False)
    torch.manual_seed(3)
    u1 = torch.randn(7, s.hidden, dtype=F64)
    got = m._attention(0, u1)
    D = w.dense
    qkv = u1 @ D["l0.wqkv"].double().T
    nq, nkv, d = s.n_q_heads, s.n_kv_heads, s.head_dim
    q = qkv[:, :nq * d].view(7, nq, d)
    k = qkv[:, nq * d:(nq + nkv) * d].view(7, nkv, d)
    v = qkv[:, (nq + nkv) * d:].view(7, nkv, d)
    pos = torch.arange(7)
    q, k = O.rope(q, pos, s.rope_theta), O.rope(k, pos, s.rope_theta)
    ref = F.scaled_dot_product_attention(q.transpose(0, 1)[None], k.transpose(0, 1)[None], v.transpose(0, 1)[None],
                                         is_causal=True, enable_gqa=True)[0].transpose(0, 1).reshape(7, nq * d)
    assert torch.allclose(got, ref @ D["l0.wo"].double().T, atol=1e-12)
    # T = 1 from an empty cache: attention output = v of the (repeated) kv head
    m.reset()
    one = m._attention(0, u1[:1])
    v0 = (u1[:1] @ D["l0.wqkv"].double().T)[:, (nq + nkv) * d:].view(1, nkv, d).repeat_interleave(nq // nkv, 1)
    assert torch.allclose(one, v0.reshape(1, nq * d) @ D["l0.wo"].double().T, atol=1e-13)


@pytest.mark.parametrize("variant", ["plain", "shared_gate", "dense0_bias"])
def test_prefill_equals_prefill_plus_decode_and_causality(variant):
    over = {}
    if variant == "shared_gate":
        over = dict(n_shared_inter=48, shared_gate=1)
    if variant == "dense0_bias":
        over = dict(n_layers=3, n_dense_layers=1, dense_inter=40, router_bias=1, n_shared_inter=24)
    cfg = tiny_cfg(**over)
    w = synth.make_weights(cfg, pin=False)
    ids = synth.make_prompt(cfg)
    a = O.OracleModel(w)
    full = a.prefill(ids)
    b = O.OracleModel(w)
    part = b.prefill(ids[:-1])
    last = b.decode(int(ids[-1]))
    assert torch.allclose(full.logits, last.logits, atol=1e-11)
    assert torch.allclose(full.hidden[-1], last.hidden[0], atol=1e-11)
    assert torch.allclose(full.hidden[:-1], part.hidden, atol=1e-11)         # causality: prefix unaffected
    assert full.layers[0].sel[-1] == last.layers[0].sel[0]
    for t in range(len(ids)):                                                # invariants from BASELINE.json
        for lt in full.layers:
            assert len(set(lt.sel[t])) == cfg.shape.top_k
            assert abs(sum(lt.gates[t]) - 1) < 1e-12
    c = O.OracleModel(w)
    ids2 = ids.clone(); ids2[-1] = (ids2[-1] + 1) % cfg.shape.vocab
    assert torch.allclose(c.prefill(ids2).hidden[:-1], full.hidden[:-1], atol=1e-12)


def test_identical_experts_collapse_to_one_dense_ffn():
    """BASELINE.json invariant: if all experts are identical the MoE layer equals one dense FFN (gates sum to 1)."""
    cfg = tiny_cfg()
    w = synth.make_weights(cfg, pin=False)
    w.experts[:] = w.experts[:, :1]
    m = O.OracleModel(w, use_predictor=False)
    u = torch.randn(5, cfg.shape.hidden, dtype=F64)
    y, _ = m._moe(1, 1, u)
    wg, wu, wd = w.expert_views(1, 0)
    assert torch.allclose(y, O.swiglu_ffn(u, wg, wu, wd), atol=1e-12)


# ---- an independently written compact model (third opinion) ----------------------------------------------------
def compact_model_logits(w, ids):
    """Whole-sequence, no KV cache, library ops (F.rms_norm, SDPA, F.linear, torch.topk-free routing by argsort)."""
    s, D = w.shape, w.dense
    T = len(ids)
    nq, nkv, d = s.n_q_heads, s.n_kv_heads, s.head_dim
    x = D["emb"].double()[ids.long()]
    half = d // 2
    inv = s.rope_theta ** (-torch.arange(half, dtype=F64) * 2 / d)
    ang = torch.arange(T, dtype=F64)[:, None] * inv[None]
    cos, sin = torch.cos(ang), torch.sin(ang)

    def rot(t):     # [T, n, d]
        a, b = t[..., :half], t[..., half:]
        return torch.cat([a * cos[:, None] - b * sin[:, None], b * cos[:, None] + a * sin[:, None]], -1)

    mi = 0
    for l in range(s.n_layers):
        p = f"l{l}."
        u1 = F.rms_norm(x, (s.hidden,), D[p + "ln1"].double(), s.rms_eps)
        qkv = F.linear(u1, D[p + "wqkv"].double())
        q, k, v = qkv.split([nq * d, nkv * d, nkv * d], dim=-1)
        q, k, v = rot(q.view(T, nq, d)), rot(k.view(T, nkv, d)), v.view(T, nkv, d)
        o = F.scaled_dot_product_attention(q.transpose(0, 1)[None], k.transpose(0, 1)[None], v.transpose(0, 1)[None],
                                           is_causal=True, enable_gqa=True)[0].transpose(0, 1).reshape(T, nq * d)
        h = x + F.linear(o, D[p + "wo"].double())
        u = F.rms_norm(h, (s.hidden,), D[p + "ln2"].double(), s.rms_eps)

        def ffn(t, g, uu, dd):
            return F.linear(F.silu(F.linear(t, g.double())) * F.linear(t, uu.double()), dd.double())

        if l < s.n_dense_layers:
            y = ffn(u, D[p + "ffn_gate"], D[p + "ffn_up"], D[p + "ffn_down"])
        else:
            z = F.linear(u, D[p + "router"].double())
            if s.router_bias:
                z = z + D[p + "router_bias"].double()
            idx = torch.argsort(z, dim=-1, descending=True, stable=True)[:, :s.top_k]
            gate = torch.softmax(torch.gather(z, 1, idx), dim=-1)
            y = torch.zeros_like(u)
            for t in range(T):
                for j in range(s.top_k):
                    y[t] += gate[t, j] * ffn(u[t:t + 1], *w.expert_views(mi, int(idx[t, j])))[0]
            if s.n_shared_inter:
                sh = ffn(u, D[p + "ffn_gate"], D[p + "ffn_up"], D[p + "ffn_down"])
                if s.shared_gate:
                    sh = torch.sigmoid(F.linear(u, D[p + "shared_gate_w"].double())) * sh
                y = y + sh
            mi += 1
        x = h + y
    return F.linear(F.rms_norm(x[-1], (s.hidden,), D["final_norm"].double(), s.rms_eps), D["lm_head"].double()), x


@pytest.mark.parametrize("name", ["c1", "tiny_c2like", "tiny_c3like"])
def test_whole_model_against_compact_reimplementation(name):
    if name == "c1":
        cfg = synth.get_config("c1")
    elif name == "tiny_c2like":
        cfg = tiny_cfg(n_shared_inter=48, shared_gate=1)
    else:
        cfg = tiny_cfg(n_layers=3, n_dense_layers=1, dense_inter=40, router_bias=1, n_shared_inter=24)
    w = synth.make_weights(cfg, pin=False)
    ids = synth.make_prompt(cfg)
    st = O.OracleModel(w).prefill(ids)
    logits, x = compact_model_logits(w, ids)
    assert torch.allclose(st.logits, logits, atol=1e-10)
    assert torch.allclose(st.hidden, x, atol=1e-10)
    assert st.next_token == int(torch.argmax(logits))


# ---- permutation ------------------------------------------------------------------------------------------------
def test_permutation_invariants_and_bruteforce():
    rng = random.Random(0)
    for _ in range(30):
        E, k, T = rng.randint(2, 12), 0, rng.randint(1, 40)
        k = rng.randint(1, min(4, E))
        sel = [rng.sample(range(E), k) for _ in range(T)]
        count, offset, perm, inv = permutation(sel, E)
        assert sum(count) == T * k == offset[E]
        assert sorted(perm) == list(range(T * k))                      # bijection
        assert all(inv[perm[p]] == p for p in range(T * k))            # inv∘perm = id
        flat = sorted(range(T * k), key=lambda i: (sel[i // k][i % k], i // k))   # brute force: stable sort by expert
        assert perm == flat
        for e in range(E):
            grp = perm[offset[e]:offset[e + 1]]
            assert all(sel[i // k][i % k] == e for i in grp)
            assert [i // k for i in grp] == sorted(i // k for i in grp)  # token-ascending
            assert len(grp) == count[e]


# ---- predictor ---------------------------------------------------------------------------------------------------
def test_predictor_bruteforce_and_votes():
    torch.manual_seed(5)
    u = torch.randn(6, 10, dtype=F64)
    w1, w2 = torch.randn(7, 10), torch.randn(5, 7)
    sc = predictor_scores(u, w1, w2)
    for t in range(6):
        for e in range(5):
            v = sum(w2[e, j].item() * max(0.0, sum(w1[j, i].item() * u[t, i].item() for i in range(10))) for j in range(7))
            assert abs(sc[t, e].item() - v) < 1e-12
    assert predict_experts(sc[:1], 2, 5) == topk_desc(sc[0], 2)
    votes = [0] * 5
    for t in range(6):
        for e in topk_desc(sc[t], 2):
            votes[e] += 1
    want = sorted([e for e in range(5) if votes[e]], key=lambda e: (-votes[e], e))
    assert predict_experts(sc, 2, 3) == want[:3]
    assert topk_desc(torch.tensor([1.0, 2.0, 2.0, 0.0]), 2) == [1, 2]


def test_skip_predictor_construction_is_exact_router_of_target_layer():
    """W1 = [R; −R; 0], W2 = [I, −I, 0] ⇒ W2·ReLU(W1·u) = R·u exactly (skip-based predictor).  Fed the TARGET
    layer's own input it must reproduce that layer's routing: accuracy 100 %."""
    cfg = tiny_cfg(pred_hidden=16)
    w = synth.make_weights(cfg, predictor="skip", pin=False)
    D = w.dense
    u = torch.randn(4, cfg.shape.hidden, dtype=F64)
    sc = predictor_scores(u, D["l0.pred_w1"], D["l0.pred_w2"])
    z = u @ D["l1.router"].double().T
    assert torch.allclose(sc, z, atol=1e-13)
    for t in range(4):
        assert topk_desc(sc[t], 2) == O.route(z[t], 2)[0]
    # last layer has no target: all-zero predictor
    assert D["l1.pred_w1"].abs().sum() == 0


def test_random_predictor_accuracy_near_chance_and_skip_beats_it():
    from oracle.cache_sim import ProMoECacheSim
    cfg = tiny_cfg(n_layers=4, pred_hidden=16)
    acc = {}
    for variant in ("random", "skip"):
        w = synth.make_weights(cfg, predictor=variant, pin=False)
        m = O.OracleModel(w, stride=1, slots_per_layer=4)
        sim = ProMoECacheSim(4, 8, 4)
        g = torch.Generator().manual_seed(0)
        for _ in range(150):
            m.reset()
            st = m.prefill(torch.randint(0, 50, (1,), generator=g))
            sim.run_step(O.needed_sets(st), O.pred_lists(st), 1)
        acc[variant] = sim.stats.predicted_correct / sim.stats.predicted
    assert abs(acc["random"] - 2 / 8) < 0.12        # ≈ k/E
    assert acc["skip"] > acc["random"] + 0.15


def test_fit_predictor_improves_on_its_start_point_cpu():
    """paper_2410_22134_b200/fit_predictor.py (P:159-161, 9:1 split): on synthetic traces whose target routing is a FIXED
    linear map of u that differs from the start point's, the fitted MLP must beat the start point on the held-out split,
    and the weights it returns must reproduce the accuracy it reports (rounded to bf16, as the GPU sees them)."""
    from paper_2410_22134_b200.fit_predictor import fit_layer, topk_accuracy
    g = torch.Generator().manual_seed(5)
    N, H, E, k, ph = 3000, 64, 16, 2, 64
    u = torch.randn(N, H, generator=g)
    R = torch.randn(E, H, generator=g) * H ** -0.5              # what the start point ("skip") assumes
    M = torch.eye(H) + 0.8 * torch.randn(H, H, generator=g) * H ** -0.5
    z = (u @ M.T) @ R.T                                          # what the target layer really computes
    sel = z.topk(k, dim=1).indices
    w1 = torch.zeros(ph, H); w1[:E] = R; w1[E:2 * E] = -R
    w2 = torch.zeros(E, ph); w2[:, :E] = torch.eye(E); w2[:, E:2 * E] = -torch.eye(E)
    r = fit_layer(u, sel, w1, w2, E, k, 1, seed=1, steps=200, lr=2e-3)
    assert r["kept"] == "fitted" and r["acc_test_fitted"] > r["acc_test_skip"] + 0.05
    assert r["n_train"] == 2700 and r["n_test"] == 300
    tgt = torch.zeros(N, E); tgt.scatter_(1, sel, 1.0)
    assert abs(topk_accuracy(u, w1, w2, tgt, k) - (0.9 * r["acc_train_skip"] + 0.1 * r["acc_test_skip"])) < 1e-6
    # returned weights are already bf16-representable
    assert torch.equal(r["w1"], r["w1"].to(torch.bfloat16).float())
    # a start point that is already exact cannot be beaten: the layer keeps it
    sel0 = (u @ R.T).topk(k, dim=1).indices
    r0 = fit_layer(u, sel0, w1, w2, E, k, 0, seed=2, steps=40, lr=1e-4)
    assert r0["acc_test_skip"] == 1.0 and r0["kept"] == "skip" and torch.equal(r0["w1"], w1)


# ---- batched decode: oracle/batch.py ----------------------------------------------------------
def test_batch_of_one_is_the_single_sequence_model():
    from oracle.batch import OracleBatch
    cfg = synth.get_config("c1")
    w = synth.make_weights(cfg, pin=False)
    ids = synth.make_prompt(cfg, 7).tolist()
    a = O.OracleModel(w, stride=1, slots_per_layer=4)
    b = OracleBatch(w, 1, stride=1, slots_per_layer=4)
    a.forward(ids); b.prefill_seq(0, ids)
    for tok in (3, 11, 5):
        sa, sb = a.forward([tok]), b.forward([tok])
        assert torch.equal(sa.hidden, sb.hidden) and torch.equal(sa.logits, sb.logits)
        assert [lt.sel for lt in sa.layers] == [lt.sel for lt in sb.layers]
        assert [lt.pred for lt in sa.layers] == [lt.pred for lt in sb.layers]


def test_batch_rows_are_independent_sequences_and_predictions_vote():
    """Row b of a batched step equals sequence b run alone (its own KV cache and position — here the sequences have
    DIFFERENT lengths); the predicted list of a layer is the G7 vote over the B rows; permuting the batch permutes the rows."""
    from oracle.batch import OracleBatch
    from oracle.predictor import predict_experts
    cfg = synth.get_config("c1")
    w = synth.make_weights(cfg, pin=False)
    prompts = [synth.make_prompt(cfg, n).tolist() for n in (5, 9, 3)]
    toks = [[2, 7], [9, 1], [4, 4]]
    bat = OracleBatch(w, 3, stride=1, slots_per_layer=4)
    solo = [O.OracleModel(w, stride=1, slots_per_layer=4) for _ in range(3)]
    for b in range(3):
        bat.prefill_seq(b, prompts[b]); solo[b].forward(prompts[b])
    for step in range(2):
        st = bat.forward([toks[b][step] for b in range(3)])
        ref = [solo[b].forward([toks[b][step]]) for b in range(3)]
        assert st.hidden.shape == (3, cfg.shape.hidden)
        for b in range(3):
            assert torch.equal(st.hidden[b], ref[b].hidden[0]) and torch.equal(st.seq_logits[b], ref[b].logits)
            for m in range(len(st.layers)):
                assert st.layers[m].sel[b] == ref[b].layers[m].sel[0]
                assert torch.equal(st.layers[m].logits[b], ref[b].layers[m].logits[0])
        for m in range(len(st.layers)):
            scores = torch.cat([ref[b].layers[m].pred_scores for b in range(3)], 0)
            assert st.layers[m].pred == predict_experts(scores, cfg.shape.top_k, 4)
    # permutation of the batch = permutation of the rows
    p = OracleBatch(w, 3, stride=1, slots_per_layer=4)
    order = [2, 0, 1]
    for i, b in enumerate(order):
        p.prefill_seq(i, prompts[b])
    sp = p.forward([toks[b][0] for b in order])
    q = OracleBatch(w, 3, stride=1, slots_per_layer=4)
    for b in range(3):
        q.prefill_seq(b, prompts[b])
    sq = q.forward([toks[b][0] for b in range(3)])
    for i, b in enumerate(order):
        assert torch.equal(sp.hidden[i], sq.hidden[b])
    assert sorted(sp.layers[0].pred) == sorted(sq.layers[0].pred)      # votes do not depend on the row order


def test_batch_near_tie_protocol_forces_one_row():
    """compare.oracle_step_matching on a batch: a forced selection of row b goes to sequence b's own step, the other rows
    are untouched, and snapshot / restore rewind every sequence."""
    from oracle.batch import OracleBatch
    from oracle.compare import ParityReport, oracle_step_matching, restore, snapshot
    import numpy as np
    cfg = synth.get_config("c1")
    w = synth.make_weights(cfg, pin=False)
    bat = OracleBatch(w, 2, stride=1, slots_per_layer=4)
    bat.prefill_seq(0, [1, 2, 3]); bat.prefill_seq(1, [4, 5])
    snap = snapshot(bat)
    st = bat.forward([6, 7])
    restore(bat, snap)
    bat.step_idx = 0
    assert [o.pos for o in bat.seqs] == [3, 2]
    st2 = bat.forward([6, 7])
    assert torch.equal(st.hidden, st2.hidden)
    restore(bat, snap); bat.step_idx = 0
    sel = np.array([[row for row in lt.sel] for lt in st.layers], dtype=np.int32)       # [Lm, B, k]
    rep = ParityReport()
    st3 = oracle_step_matching(bat, [6, 7], sel, rep)
    assert rep.sel_near_tie == 0 and torch.equal(st3.hidden, st.hidden)
