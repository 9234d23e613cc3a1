"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Every test here checks oracle/ against something other than itself: the layer definition
 evaluated independently, closed forms, invariants, brute force on tiny inputs, library
matmuls, hand-derived values.  The paper prints no worked numeric example of a forward pass
(SURVEY.md 4), so there are no printed values to match; the printed group maps / group counts are
under tests/golden/.
"""
import math
import os

import numpy as np
import pytest
import torch
from hypothesis import given, settings, strategies as st

import oracle
from bm_inputs import bf16_bits, CONFIGS, make_layer
from helpers import bf16_tensor, definition_form, f64, oracle_layer, rand_layer, silu

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _read_golden(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as fh:
        for line in fh:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


# --------------------------------------------------------------------------------------------
# A1: canonical fp32 dot product -- closed-form cases in which the summation order decides the value
# --------------------------------------------------------------------------------------------
def _dot(xv, wv):
    return oracle.canon_dot(bf16_bits(bf16_tensor(xv)), bf16_bits(bf16_tensor(wv)))


def test_canon_dot_is_exact_on_small_integers():
    rng = np.random.default_rng(0)
    for D in (8, 16, 256, 264, 1024):
        xv = rng.integers(-8, 9, D).astype(np.float64)
        wv = rng.integers(-8, 9, D).astype(np.float64)
        assert _dot(xv, wv) == float(xv @ wv)      # every partial sum is an exact small integer


def test_canon_dot_partial_assignment_is_j_div_8_mod_32():
    # 2^30 + 1 == 2^30 in fp32 (ulp 128).  x[0] and x[256] both fall in partial 0 (chunks 0 and 32),
    # x[8] in partial 1:  partial0 = 2^30 - 2^30 = 0, partial1 = 1  ->  1.
    # A plain left-to-right sum would give (2^30 + 1) - 2^30 = 0.
    D = 512
    xv = np.zeros(D); wv = np.ones(D)
    xv[0], xv[8], xv[256] = 2.0 ** 30, 1.0, -(2.0 ** 30)
    assert _dot(xv, wv) == 1.0
    # all three inside one 8-element chunk (same partial, ascending j): 2^30 - 2^30 + 1 = 1;
    # an assignment "j mod 32" would put them in three partials and lose the 1 in the butterfly.
    xv = np.zeros(D); xv[0], xv[1], xv[2] = 2.0 ** 30, -(2.0 ** 30), 1.0
    assert _dot(xv, wv) == 1.0
    # ascending order inside a partial: 2^30 + 1 - 2^30 = 0 (the 1 is absorbed first)
    xv = np.zeros(D); xv[0], xv[1], xv[2] = 2.0 ** 30, 1.0, -(2.0 ** 30)
    assert _dot(xv, wv) == 0.0


def test_canon_dot_butterfly_pairs_l_with_l_xor_16_first():
    # partials: p0 = 2^30, p16 = -2^30, p8 = 1.  Butterfly o=16 first: p0+p16 = 0, p8+p24 = 1; then
    # o=8: 0 + 1 = 1.  Summing partials in lane order would absorb the 1: (2^30 + 1) - 2^30 = 0.
    D = 256
    xv = np.zeros(D); wv = np.ones(D)
    xv[0 * 8], xv[16 * 8], xv[8 * 8] = 2.0 ** 30, -(2.0 ** 30), 1.0
    assert _dot(xv, wv) == 1.0
    # o=16 pairs p0 with p16, not with p1: p0 = 2^30, p1 = -2^30, p16 = 1 -> (2^30 + 1) + (-2^30 + 0) = 0
    xv = np.zeros(D); xv[0], xv[8], xv[16 * 8] = 2.0 ** 30, -(2.0 ** 30), 1.0
    assert _dot(xv, wv) == 0.0


def test_canon_logits_close_to_fp64_and_same_selection_off_ties():
    L = make_layer(CONFIGS["tiny"].with_(T=256, zipf_s=1.0), seed=3, weights=False)
    r = oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), L.router_bias.numpy(), 2,
                     L.group_map.numpy(), 4, want_logits=True)
    x, Wr = f64(L.x), f64(L.W_router)
    l64 = x @ Wr.T + L.router_bias.double().numpy()
    bound = 1e-6 * (np.abs(x) @ np.abs(Wr).T + 1.0)
    assert (np.abs(r.logits - l64) <= bound).all()
    srt = np.sort(l64, axis=1)[:, ::-1]
    margin = srt[:, 1] - srt[:, 2]
    ids64 = np.argsort(-l64, axis=1, kind="stable")[:, :2]
    ok = margin > 1e-4
    assert ok.mean() > 0.95
    assert (ids64[ok] == r.expert_ids[ok]).all()


# --------------------------------------------------------------------------------------------
# R2: top-K with lower-index tie-break -- brute force on tiny inputs
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("E,K", [(2, 1), (3, 2), (4, 3), (6, 3), (6, 6), (5, 1)])
def test_topk_brute_force(E, K):
    rng = np.random.default_rng(E * 10 + K)
    T, D = 200, 16
    # coarse values so that exact ties are frequent
    x = bf16_tensor(rng.integers(-2, 3, (T, D)))
    Wr = bf16_tensor(rng.integers(-1, 2, (E, D)))
    r = oracle.route(bf16_bits(x), bf16_bits(Wr), None, K, np.zeros(E, np.int32), 1, want_logits=True)
    l = r.logits
    assert (l == f64(x) @ f64(Wr).T).all()          # integers: the canonical dot is exact
    n_ties = 0
    for t in range(T):
        sel = list(r.expert_ids[t])
        assert len(set(sel)) == K and all(0 <= e < E for e in sel)
        # ranked: descending logit, ascending index among equals
        for a, b in zip(sel[:-1], sel[1:]):
            assert l[t, a] > l[t, b] or (l[t, a] == l[t, b] and a < b)
        for e in sel:
            for e2 in range(E):
                if e2 in sel:
                    continue
                assert l[t, e] > l[t, e2] or (l[t, e] == l[t, e2] and e < e2)
                n_ties += l[t, e] == l[t, e2]
    if K < E:
        assert n_ties > 0                             # the tie-break rule was really exercised


def test_topk_degenerate_rows():
    E, K, D = 6, 3, 8
    x = bf16_tensor(np.ones((4, D)))
    Wr = bf16_tensor(np.zeros((E, D)))               # all logits equal (+0)
    r = oracle.route(bf16_bits(x), bf16_bits(Wr), None, K, np.arange(E, dtype=np.int32), E)
    assert (r.expert_ids == np.arange(K)).all()
    assert np.allclose(r.gate_w, 1.0 / K, atol=1e-7)
    # +0 == -0 is a tie: expert 0 has logit -0 (x * -0 summed), still wins by index
    Wr = bf16_tensor(np.zeros((E, D))); Wr[0] = -0.0
    r = oracle.route(bf16_bits(x), bf16_bits(Wr), None, 1, np.arange(E, dtype=np.int32), E)
    assert (r.expert_ids[:, 0] == 0).all()
    # two identical router rows -> equal logits -> lower index first
    rng = np.random.default_rng(1)
    Wn = rng.standard_normal((E, D)); Wn[4] = Wn[1]
    xr = bf16_tensor(rng.standard_normal((64, D)))
    r = oracle.route(bf16_bits(xr), bf16_bits(bf16_tensor(Wn)), None, E, np.arange(E, dtype=np.int32), E)
    for t in range(64):
        sel = list(r.expert_ids[t])
        assert sorted(sel) == list(range(E))          # K = E selects everything
        assert sel.index(1) + 1 == sel.index(4)       # 1 directly before 4


# --------------------------------------------------------------------------------------------
# R3-R5: gate weights, remap, dedup
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("E,K,G", [(8, 2, 4), (60, 4, 15), (64, 6, 16), (60, 4, 60), (16, 8, 3)])
def test_gate_and_dedup_invariants(E, K, G):
    rng = np.random.default_rng(E + K + G)
    T, D = 300, 64
    x = bf16_tensor(rng.standard_normal((T, D)))
    Wr = bf16_tensor(rng.standard_normal((E, D)) * 0.3)
    gmap = rng.integers(0, G, E).astype(np.int32) if G < E else np.arange(E, dtype=np.int32)
    r = oracle.route(bf16_bits(x), bf16_bits(Wr), None, K, gmap, G, want_logits=True)
    assert np.abs(r.gate_w.astype(np.float64).sum(1) - 1.0).max() <= 1e-6   # BJ:north_star check 3
    for t in range(T):
        n = r.n_slots[t]
        assert 1 <= n <= K
        g = r.group_ids[t]
        assert (g[:n] >= 0).all() and (g[:n] < G).all() and len(set(g[:n])) == n
        assert (g[n:] == -1).all() and (r.gate_w[t, n:] == 0).all() and (r.gate_w[t, :n] > 0).all()
        # brute force of R3-R5 in fp64 from the oracle's own selected logits
        l = r.logits[t, r.expert_ids[t]].astype(np.float64)
        p = np.exp(l - l[0]); w = p / p.sum()
        first, merged = [], {}
        for i, e in enumerate(r.expert_ids[t]):
            u = int(gmap[e])
            if u not in merged:
                first.append(u); merged[u] = 0.0
            merged[u] += w[i]
        assert list(g[:n]) == first                                      # A6: first-occurrence order
        assert np.allclose(r.gate_w[t, :n], [merged[u] for u in first], atol=2e-7)
    if G < E:
        assert (r.n_slots < K).any()                                     # dedup really happened


def test_k1_weight_is_exactly_one():
    rng = np.random.default_rng(5)
    x = bf16_tensor(rng.standard_normal((100, 32)))
    Wr = bf16_tensor(rng.standard_normal((7, 32)))
    r = oracle.route(bf16_bits(x), bf16_bits(Wr), None, 1, np.arange(7, dtype=np.int32) % 3, 3)
    assert (r.gate_w[:, 0] == np.float32(1.0)).all() and (r.n_slots == 1).all()


def test_softmax_subtracts_the_maximum():
    # logits (+96, -96): exp(l - max) = (1, e^-192 -> 0 in fp32); subtracting anything but the
    # maximum overflows to inf/nan.  The weights must come out finite: (1, 0).
    D = 8
    x = np.zeros((1, D)); x[0, 0] = 64.0
    Wr = np.zeros((2, D)); Wr[0, 0], Wr[1, 0] = 1.5, -1.5
    r = oracle.route(bf16_bits(bf16_tensor(x)), bf16_bits(bf16_tensor(Wr)), None, 2,
                     np.array([0, 1], np.int32), 2, want_logits=True)
    assert r.logits.tolist() == [[96.0, -96.0]]
    assert r.expert_ids.tolist() == [[0, 1]] and r.gate_w.tolist() == [[1.0, 0.0]]


def test_constant_logit_shift_changes_nothing():
    # softmax and top-K are shift invariant; a bias equal for every expert must not change the routing
    # (ids exactly, on tokens whose K/K+1 margin is far above fp32 rounding; weights to 1e-5)
    rng = np.random.default_rng(6)
    T, D, E, K = 200, 64, 12, 3
    x = bf16_tensor(rng.standard_normal((T, D)))
    Wr = bf16_tensor(rng.standard_normal((E, D)) * 0.3)
    gmap = (np.arange(E) % 4).astype(np.int32)
    r0 = oracle.route(bf16_bits(x), bf16_bits(Wr), None, K, gmap, 4, want_logits=True)
    r1 = oracle.route(bf16_bits(x), bf16_bits(Wr), np.full(E, 3.0, np.float32), K, gmap, 4)
    srt = np.sort(r0.logits, axis=1)[:, ::-1]
    gaps = np.abs(np.diff(srt[:, :K + 1], axis=1)).min(1)
    ok = gaps > 1e-4
    assert ok.mean() > 0.9
    assert (r0.expert_ids[ok] == r1.expert_ids[ok]).all()
    assert (r0.group_ids[ok] == r1.group_ids[ok]).all()
    assert np.abs(r0.gate_w[ok] - r1.gate_w[ok]).max() < 1e-5


def test_hand_worked_example():
    # D = 8, one-hot tokens, so logit[t,e] = Wr[e, hot(t)].  Token 0: logits (1, .5, .25) ->
    # top-2 = (e0, e1), w = (1, e^-.5)/(1 + e^-.5).  gmap = [0,1,1]: two groups.
    # Token 1: logits (.25, .5, 1) -> top-2 = (e2, e1), both in group 1 -> one slot, weight 1.
    # Experts: W1 = c_u*I, W3 = I, W2 = I  =>  FFN_u(x) = SiLU(c_u x) * x  elementwise.
    D = F = 8
    x = np.zeros((2, D)); x[0, 0] = 1.0; x[1, 3] = 2.0
    Wr = np.zeros((3, D)); Wr[:, 0] = (1.0, 0.5, 0.25); Wr[:, 3] = (0.125, 0.25, 0.5)
    c = (0.5, 2.0)
    I = np.eye(D)
    W1 = np.stack([c[0] * I, c[1] * I]); W3 = np.stack([I, I]); W2 = np.stack([I, I])
    r = oracle.route(bf16_bits(bf16_tensor(x)), bf16_bits(bf16_tensor(Wr)), None, 2,
                     np.array([0, 1, 1], np.int32), 2)
    out = oracle.moe_forward(bf16_bits(bf16_tensor(x)), r, bf16_bits(bf16_tensor(W1)),
                             bf16_bits(bf16_tensor(W3)), bf16_bits(bf16_tensor(W2)))
    assert r.expert_ids.tolist() == [[0, 1], [2, 1]]
    assert r.group_ids.tolist() == [[0, 1], [1, -1]]
    assert r.n_slots.tolist() == [2, 1]
    w0 = 1.0 / (1.0 + math.exp(-0.5))
    assert abs(r.gate_w[0, 0] - w0) < 1e-7 and abs(r.gate_w[0, 1] - (1 - w0)) < 1e-7
    assert abs(r.gate_w[1, 0] - 1.0) < 1e-7 and r.gate_w[1, 1] == 0.0
    assert r.counts.tolist() == [1, 2] and r.offsets.tolist() == [0, 1, 3]
    assert r.row_token.tolist() == [0, 0, 1, -1] and r.row_slot.tolist() == [0, 1, 0, -1]
    assert r.slot_row.tolist() == [[0, 1], [2, -1]]
    sl = lambda a: a / (1.0 + math.exp(-a))
    exp0 = np.zeros(D); exp0[0] = float(r.gate_w[0, 0]) * sl(0.5) + float(r.gate_w[0, 1]) * sl(2.0)
    exp1 = np.zeros(D); exp1[3] = float(r.gate_w[1, 0]) * sl(4.0) * 2.0
    assert np.allclose(out[0], exp0, rtol=0, atol=1e-12) and np.allclose(out[1], exp1, rtol=0, atol=1e-12)


# --------------------------------------------------------------------------------------------
# R6-R7: histogram, scan, permutation
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("T,E,K,G", [(1, 8, 2, 4), (257, 60, 4, 8), (1000, 64, 6, 16), (64, 8, 2, 16)])
def test_permutation_properties(T, E, K, G):
    rng = np.random.default_rng(T + G)
    x = bf16_tensor(rng.standard_normal((T, 32)))
    Wr = bf16_tensor(rng.standard_normal((E, 32)))
    gmap = rng.integers(0, G, E).astype(np.int32)
    if G == 16 and E == 8:
        gmap = (np.arange(E) * 2).astype(np.int32)           # half of the groups stay empty (A10)
    r = oracle.route(bf16_bits(x), bf16_bits(Wr), None, K, gmap, G)
    A = r.A
    assert r.counts.sum() == r.n_slots.sum() == A == r.offsets[G]
    valid = r.group_ids >= 0
    assert (r.counts == np.bincount(r.group_ids[valid], minlength=G)).all()
    assert (r.offsets == np.concatenate([[0], np.cumsum(r.counts)])).all()
    assert (r.row_token[A:] == -1).all() and (r.row_slot[A:] == -1).all()
    # brute force: stable sort of the (group, token) pairs
    tt, ss = np.nonzero(valid)
    order = np.lexsort((tt, r.group_ids[tt, ss]))
    assert (r.row_token[:A] == tt[order]).all() and (r.row_slot[:A] == ss[order]).all()
    # mutual inverses
    assert (r.slot_row[r.row_token[:A], r.row_slot[:A]] == np.arange(A)).all()
    assert (r.slot_row[~valid] == -1).all()
    for u in range(G):
        seg = r.row_token[r.offsets[u]:r.offsets[u + 1]]
        assert (np.diff(seg) > 0).all()                       # A7: token ascending inside a group
        assert (r.group_ids[seg, r.row_slot[r.offsets[u]:r.offsets[u + 1]]] == u).all()
    if G == 16 and E == 8:
        assert (r.counts[1::2] == 0).all()


# --------------------------------------------------------------------------------------------
# F1-F2: the whole layer against the definition, and structural special cases
# --------------------------------------------------------------------------------------------
def _check_against_definition(L, K, G, S, rtol=2e-6):
    r, out = oracle_layer(L, want_logits=True)
    bias = None if L.router_bias is None else L.router_bias.double().numpy()
    ref, ids, margin = definition_form(f64(L.x), f64(L.W_router), bias, K, L.group_map.numpy(),
                                       f64(L.W1), f64(L.W3), f64(L.W2), S)
    ok = margin > 1e-4
    assert ok.mean() > 0.9
    assert (ids[ok] == r.expert_ids[ok]).all()
    scale = np.abs(ref[ok]).max()
    assert np.abs(out[ok] - ref[ok]).max() <= rtol * scale
    return r, out


def test_identity_map_is_standard_topk_moe():
    # BJ:north_star check 1; zero brownout
    rng = np.random.default_rng(11)
    E = 6
    L = rand_layer(rng, T=40, D=32, F=48, E=E, K=2, G=E, gmap=np.arange(E), bias=True)
    r, _ = _check_against_definition(L, 2, E, 0)
    assert (r.n_slots == 2).all() and (r.group_ids == r.expert_ids).all()


@pytest.mark.parametrize("K,G,S", [(2, 3, 0), (4, 2, 0), (3, 4, 2)])
def test_grouped_layer_equals_definition_without_dedup(K, G, S):
    # the definition visits a group once per selected member; the oracle visits it once with summed
    # weights (A5) -- the same real number
    rng = np.random.default_rng(12 + K)
    L = rand_layer(rng, T=48, D=32, F=40, E=8, K=K, G=G, S=S, bias=True)
    _check_against_definition(L, K, G, S)


def test_fig1a_group_maps_and_replicated_weights():
    # PAPER.md:48-52 maps as fixtures.  BJ:north_star check 2: give every expert e the weights of
    # its group; the ungrouped E-expert layer must reproduce the grouped G-group layer.
    rng = np.random.default_rng(13)
    for name, *gm in _read_golden("fig1a_group_maps.txt"):
        gmap = np.array(gm, dtype=np.int32)
        assert gmap.shape == (6,) and sorted(np.bincount(gmap)) == [2, 2, 2]
        L = rand_layer(rng, T=64, D=32, F=40, E=6, K=3, G=3, gmap=gmap)
        r, out = oracle_layer(L)
        from types import SimpleNamespace
        U = SimpleNamespace(**vars(L))
        U.G = 6
        U.group_map = torch.arange(6, dtype=torch.int32)
        idx = torch.as_tensor(gmap, dtype=torch.long)
        U.W1, U.W3, U.W2 = L.W1[idx], L.W3[idx], L.W2[idx]
        ru, outu = oracle_layer(U)
        assert (ru.expert_ids == r.expert_ids).all()
        assert np.abs(out - outu).max() <= 1e-6 * np.abs(out).max()
        assert (r.n_slots < 3).any()


def test_g1_is_a_dense_ffn_library_matmul():
    # G = 1: every token goes through FFN_0 with weight 1 whatever the router says
    rng = np.random.default_rng(14)
    L = rand_layer(rng, T=33, D=64, F=96, E=5, K=3, G=1)
    r, out = oracle_layer(L)
    assert (r.n_slots == 1).all() and np.abs(r.gate_w[:, 0] - 1).max() < 2e-7
    x = L.x.double()
    ref = (torch.nn.functional.silu(x @ L.W1[0].double().T) * (x @ L.W3[0].double().T)) @ L.W2[0].double().T
    gw = r.gate_w[:, :1].astype(np.float64)
    assert np.abs(out - gw * ref.numpy()).max() <= 1e-12 * np.abs(out).max() + 1e-15


def test_closed_forms_and_orientation():
    rng = np.random.default_rng(15)
    D, F, E, K, G, T = 16, 24, 4, 2, 2, 20
    L = rand_layer(rng, T=T, D=D, F=F, E=E, K=K, G=G)
    Z = SimpleNamespaceCopy(L); Z.W2 = torch.zeros_like(L.W2)
    assert (oracle_layer(Z)[1] == 0).all()                                # W2 = 0 => out = 0
    Z = SimpleNamespaceCopy(L); Z.x = torch.zeros_like(L.x)
    assert (oracle_layer(Z)[1] == 0).all()                                # x = 0 => out = 0
    # rectangular identities (F > D): W1 = c*[I;0] ([F,D]), W3 = [I;0], W2 = [I 0] ([D,F])
    # => out = SiLU(c x) * x elementwise for every group; a [D,F]/[F,D] mix-up cannot produce this
    c = 0.5
    I_fd = np.zeros((F, D)); I_fd[:D] = np.eye(D)
    Z = SimpleNamespaceCopy(L)
    Z.W1 = bf16_tensor(np.stack([c * I_fd] * G)); Z.W3 = bf16_tensor(np.stack([I_fd] * G))
    Z.W2 = bf16_tensor(np.stack([I_fd.T] * G))
    r, out = oracle_layer(Z)
    xs = f64(L.x)
    wsum = r.gate_w.astype(np.float64).sum(1, keepdims=True)
    assert np.abs(out - wsum * silu(c * xs) * xs).max() < 1e-12
    # and with F < D the extra input coordinates are dropped
    F2 = 8
    I_fd = np.zeros((F2, D)); I_fd[:, :F2] = np.eye(F2)
    Z.W1 = bf16_tensor(np.stack([c * I_fd] * G)); Z.W3 = bf16_tensor(np.stack([I_fd] * G))
    Z.W2 = bf16_tensor(np.stack([I_fd.T] * G)); Z.F = F2
    r, out = oracle_layer(Z)
    exp = np.zeros_like(xs); exp[:, :F2] = (silu(c * xs) * xs)[:, :F2]
    assert np.abs(out - wsum * exp).max() < 1e-12


def SimpleNamespaceCopy(L):
    from types import SimpleNamespace
    return SimpleNamespace(**vars(L))


def test_sel_tokens_subset_matches_full():
    rng = np.random.default_rng(16)
    L = rand_layer(rng, T=50, D=32, F=40, E=8, K=3, G=4, S=1)
    r, full = oracle_layer(L)
    sel = np.array([0, 7, 8, 31, 49], np.int32)
    _, sub = oracle_layer(L, sel_tokens=sel)
    assert (sub == full[sel]).all()


# --------------------------------------------------------------------------------------------
# Equivariances (hypothesis)
# --------------------------------------------------------------------------------------------
@settings(max_examples=15, deadline=None)
@given(seed=st.integers(0, 10_000), T=st.integers(1, 24), K=st.integers(1, 4), G=st.integers(1, 5))
def test_equivariances(seed, T, K, G):
    rng = np.random.default_rng(seed)
    E = 6
    L = rand_layer(rng, T=T, D=16, F=24, E=E, K=K, G=G)
    r, out = oracle_layer(L)
    # (a) permuting tokens permutes the output rows bit-identically (tokens are independent)
    perm = rng.permutation(T)
    P = SimpleNamespaceCopy(L); P.x = L.x[torch.as_tensor(perm)]
    rp, outp = oracle_layer(P)
    assert (outp == out[perm]).all() and (rp.expert_ids == r.expert_ids[perm]).all()
    # (b) relabelling groups together with their weights leaves out unchanged, permutes counts
    sigma = rng.permutation(G)                       # new label of old group u is sigma[u]
    Q = SimpleNamespaceCopy(L)
    Q.group_map = torch.as_tensor(sigma[L.group_map.numpy()].astype(np.int32))
    inv = torch.as_tensor(np.argsort(sigma))         # new group v holds old group inv[v]
    Q.W1, Q.W3, Q.W2 = L.W1[inv], L.W3[inv], L.W2[inv]
    rq, outq = oracle_layer(Q)
    assert (outq == out).all() and (rq.counts[sigma] == r.counts).all()
    # (c) duplicate input rows give duplicate outputs
    Dd = SimpleNamespaceCopy(L); Dd.x = torch.cat([L.x, L.x[:1]]); Dd.T = T + 1
    _, outd = oracle_layer(Dd)
    assert (outd[-1] == outd[0]).all() and (outd[:T] == out).all()


# --------------------------------------------------------------------------------------------
# Group-count fixture (Eq. 1) and the generator's maps
# --------------------------------------------------------------------------------------------
def test_eq1_group_counts_and_generated_maps_respect_the_cap():
    from bm_inputs import make_group_map, sweep_points, LayerConfig
    rows = [(int(a), int(b), int(c)) for a, b, c in _read_golden("eq1_group_counts.txt")]
    assert rows == [(60, 2, 30), (60, 4, 15), (60, 8, 8)]
    for E, k, G in rows:
        assert G == math.ceil(E / k)                                         # PAPER.md:116 Eq. 1
        cfg = LayerConfig("t", T=1, D=8, F=8, E=E, K=4, G=G)
        for seed in range(3):
            gm = make_group_map(cfg, seed).numpy()
            sizes = np.bincount(gm, minlength=G)
            assert sizes.sum() == E and sizes.max() <= math.ceil(E / G)       # cap
            assert sizes.max() - sizes.min() <= 1
    assert {c.G for c in sweep_points()} == {60, 30, 15, 8}
    fg = CONFIGS["finegrained"]
    sizes = np.bincount(make_group_map(fg, 0).numpy(), minlength=fg.G)
    assert sizes.sum() == 64 and sizes.min() >= 2 and sizes.max() <= 8       # BJ:configs[3]
