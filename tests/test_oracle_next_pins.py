"""Pins (-m "not gpu") for the oracle functions of SURVEY.md 8(f): partial brownout (NEXT-1) and the
united-weight parameter average (NEXT-3).

Partial brownout ("partial-brownout delegates only cold expert tokens to united experts";
P:172): the pins are the two modes the paper names as its limits (zero brownout = every expert
hot, full brownout = every expert cold), an independent definition-form evaluator of P:42 with the
mixed substitution, and the invariants the dedup must keep.
United weights ("initialized as the parameter average of member experts"): closed forms, numpy
mean, linearity.
"""
import numpy as np
import pytest
import torch

import oracle
from bm_inputs import bf16_bits
from helpers import bf16_tensor, f64, ffn_def, rand_layer


def _stack(L, Wo):
    """Weight sets of a partial-brownout layer: [united (G) ; originals (E) ; shared (S)]."""
    G, S = L.G, L.S
    cat = lambda u, o: torch.cat([u[:G], o, u[G:G + S]], dim=0)
    return cat(L.W1, Wo[0]), cat(L.W3, Wo[1]), cat(L.W2, Wo[2])


def _orig_weights(rng, E, F, D, wstd=0.05):
    return (bf16_tensor(rng.standard_normal((E, F, D)) * wstd), bf16_tensor(rng.standard_normal((E, F, D)) * wstd),
            bf16_tensor(rng.standard_normal((E, D, F)) * wstd))


def _route(L, cold=None):
    bias = None if L.router_bias is None else L.router_bias.numpy()
    return oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), bias, L.K, L.group_map.numpy(), L.G, cold_mask=cold)


def _definition_partial(L, Wo, cold):
    """h_t = sum_i g_i FFN_{set(e_i)}(x_t), set(e) = united[gmap[e]] if cold[e] else original[e]."""
    x, Wr = f64(L.x), f64(L.W_router)
    bias = None if L.router_bias is None else L.router_bias.double().numpy()
    U = [f64(L.W1), f64(L.W3), f64(L.W2)]
    O = [f64(w) for w in Wo]
    gmap = L.group_map.numpy()
    outs, ids, margins = [], [], []
    for t in range(x.shape[0]):
        l = Wr @ x[t] + (0 if bias is None else bias)
        order = sorted(range(L.E), key=lambda e: (-l[e], e))
        sel = order[:L.K]
        margins.append(l[order[L.K - 1]] - l[order[L.K]] if L.K < L.E else np.inf)
        p = np.exp(l[sel] - l[sel[0]])
        w = p / p.sum()
        o = np.zeros(x.shape[1])
        for i, e in enumerate(sel):
            if cold[e]:
                u = int(gmap[e])
                o += w[i] * ffn_def(x[t], U[0][u], U[1][u], U[2][u])
            else:
                o += w[i] * ffn_def(x[t], O[0][e], O[1][e], O[2][e])
        for j in range(L.S):
            o += ffn_def(x[t], U[0][L.G + j], U[1][L.G + j], U[2][L.G + j])
        outs.append(o)
        ids.append(sel)
    return np.array(outs), np.array(ids, dtype=np.int32), np.array(margins)


@pytest.mark.parametrize("K,G,S", [(2, 3, 0), (4, 2, 1)])
def test_partial_brownout_equals_definition(K, G, S):
    rng = np.random.default_rng(40 + K)
    E = 8
    L = rand_layer(rng, T=48, D=32, F=40, E=E, K=K, G=G, S=S, bias=True)
    Wo = _orig_weights(rng, E, 40, 32)
    cold = (rng.random(E) < 0.5).astype(np.int32)
    cold[0], cold[1] = 0, 1                                  # both kinds present
    r = _route(L, cold)
    W1, W3, W2 = _stack(L, Wo)
    out = oracle.moe_forward(bf16_bits(L.x), r, bf16_bits(W1), bf16_bits(W3), bf16_bits(W2), S)
    ref, ids, margin = _definition_partial(L, Wo, cold)
    ok = margin > 1e-4
    assert ok.mean() > 0.9 and (ids[ok] == r.expert_ids[ok]).all()
    assert np.abs(out[ok] - ref[ok]).max() <= 2e-6 * np.abs(ref[ok]).max()


def test_all_cold_is_full_brownout_and_all_hot_is_zero_brownout():
    # threshold 0 = "all cold tokens to united experts", threshold 1.0 = "no merging"
    rng = np.random.default_rng(41)
    E, K, G = 8, 3, 3
    L = rand_layer(rng, T=64, D=32, F=24, E=E, K=K, G=G, bias=True)
    full = _route(L)
    cold = _route(L, np.ones(E, np.int32))
    for k in ("expert_ids", "group_ids", "n_slots", "row_token", "row_slot", "slot_row"):
        assert (getattr(full, k) == getattr(cold, k)).all(), k
    assert (cold.counts[:G] == full.counts).all() and (cold.counts[G:] == 0).all()
    assert (cold.gate_w == full.gate_w).all()
    hot = _route(L, np.zeros(E, np.int32))
    assert (hot.group_ids == G + hot.expert_ids).all() and (hot.n_slots == K).all()
    assert (hot.counts[:G] == 0).all()
    assert (hot.counts[G:] == np.bincount(hot.expert_ids.ravel(), minlength=E)).all()
    # zero brownout reproduces the plain top-K layer on the original experts (identity map, G = E)
    Wo = _orig_weights(rng, E, 24, 32)
    W1, W3, W2 = _stack(L, Wo)
    out = oracle.moe_forward(bf16_bits(L.x), hot, bf16_bits(W1), bf16_bits(W3), bf16_bits(W2), 0)
    ident = oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), L.router_bias.numpy(), K,
                         np.arange(E, dtype=np.int32), E)
    out_id = oracle.moe_forward(bf16_bits(L.x), ident, bf16_bits(Wo[0]), bf16_bits(Wo[1]), bf16_bits(Wo[2]), 0)
    assert np.abs(out - out_id).max() <= 1e-12 * (1 + np.abs(out_id).max())


def test_partial_brownout_invariants():
    rng = np.random.default_rng(42)
    E, K, G = 12, 4, 3
    L = rand_layer(rng, T=200, D=16, F=8, E=E, K=K, G=G, bias=True)
    cold = (np.arange(E) % 3 != 0).astype(np.int32)
    r = _route(L, cold)
    gmap = L.group_map.numpy()
    assert r.G == G + E and r.counts.shape == (G + E,) and r.offsets[-1] == r.n_slots.sum() == r.counts.sum()
    assert np.abs(r.gate_w.sum(1) - 1).max() <= 1e-6 and (r.n_slots >= 1).all() and (r.n_slots <= K).all()
    for t in range(200):
        n = r.n_slots[t]
        ids = r.group_ids[t, :n]
        assert len(set(ids.tolist())) == n and (r.group_ids[t, n:] == -1).all()
        # brute force of R4-R5: first-occurrence order of the substituted sets
        seen = []
        for e in r.expert_ids[t]:
            u = int(gmap[e]) if cold[e] else G + int(e)
            if u not in seen:
                seen.append(u)
        assert seen == ids.tolist()
    # a hot expert is never merged with anything: its set receives exactly the tokens that selected it
    sel = np.bincount(r.expert_ids.ravel(), minlength=E)
    for e in range(E):
        if not cold[e]:
            assert r.counts[G + e] == sel[e]
        else:
            assert r.counts[G + e] == 0
    assert (r.counts[:G] > 0).any()


# --------------------------------------------------------------------------------------------
# united-weight parameter average
# --------------------------------------------------------------------------------------------
def test_unite_weights_is_the_member_mean():
    rng = np.random.default_rng(43)
    E, G = 10, 4
    W = bf16_tensor(rng.standard_normal((E, 6, 5)))
    gmap = np.array([0, 1, 1, 3, 0, 1, 3, 3, 3, 0], dtype=np.int32)      # group 2 is empty
    U = oracle.unite_weights(bf16_bits(W), gmap, G)
    Wf = f64(W)
    for u in range(G):
        m = np.nonzero(gmap == u)[0]
        want = Wf[m].mean(0) if len(m) else np.zeros((6, 5))
        assert np.abs(U[u] - want).max() <= 1e-15
    # closed forms: a singleton group returns its member; equal members return themselves
    ident = oracle.unite_weights(bf16_bits(W), np.arange(E, dtype=np.int32), E)
    assert (ident == Wf).all()
    same = bf16_tensor(np.broadcast_to(Wf[0], (4, 6, 5)).copy())
    assert (oracle.unite_weights(bf16_bits(same), np.zeros(4, np.int32), 1)[0] == Wf[0]).all()
    # hand-worked: members 1, 2, 6 -> 3;  -1, 0.5 -> -0.25
    hw = bf16_tensor(np.array([[1.0], [2.0], [6.0], [-1.0], [0.5]]))
    got = oracle.unite_weights(bf16_bits(hw), np.array([0, 0, 0, 1, 1], np.int32), 2)
    assert got.ravel().tolist() == [3.0, -0.25]


def test_united_expert_of_identical_members_reproduces_the_ungrouped_layer():
    # if all members of a group are the same expert, the parameter average is that expert, so the grouped
    # layer built from the average must equal the ungrouped layer (BJ:north_star check 2, via P:245)
    rng = np.random.default_rng(44)
    E, G, K = 6, 3, 2
    gmap = np.array([0, 0, 1, 1, 2, 2], dtype=np.int32)
    L = rand_layer(rng, T=32, D=16, F=24, E=E, K=K, G=G, gmap=gmap)
    idx = torch.as_tensor(gmap, dtype=torch.long)
    Wo = (L.W1[idx], L.W3[idx], L.W2[idx])                      # expert e carries its group's weights
    U = [oracle.unite_weights(bf16_bits(w), gmap, G) for w in Wo]
    for u_avg, w in zip(U, (L.W1, L.W3, L.W2)):
        assert (u_avg == f64(w)).all()


# --------------------------------------------------------------------------------------------
# calibration forward (NEXT-2): routing frequency, expert outputs, cosine matrix, Eq. 5 / Eq. 6
# --------------------------------------------------------------------------------------------
def test_expert_histogram_counts_selections():
    rng = np.random.default_rng(50)
    L = rand_layer(rng, T=300, D=16, F=8, E=10, K=3, G=10, gmap=np.arange(10), bias=True)
    r = _route(L)
    w = oracle.expert_histogram(r.expert_ids, 10)
    assert w.sum() == 300 * 3
    # identity map: selecting expert e == visiting group e, whose rows R6 counted independently
    assert (w == r.counts).all()
    assert (oracle.expert_histogram(np.array([[2, 0], [2, 1]]), 4) == [1, 1, 2, 0]).all()


def test_expert_outputs_match_library_matmuls_and_the_layer():
    rng = np.random.default_rng(51)
    E, T, D, F = 5, 12, 16, 24
    L = rand_layer(rng, T=T, D=D, F=F, E=E, K=1, G=E, gmap=np.arange(E))
    Y = oracle.expert_outputs(bf16_bits(L.x), bf16_bits(L.W1), bf16_bits(L.W3), bf16_bits(L.W2))
    x, W1, W3, W2 = f64(L.x), f64(L.W1), f64(L.W3), f64(L.W2)
    for e in range(E):
        for t in range(T):
            assert np.abs(Y[e, t] - ffn_def(x[t], W1[e], W3[e], W2[e])).max() <= 1e-12 * (1 + np.abs(Y[e, t]).max())
    # top-1 layer (gate weight exactly 1): the layer output of token t is the output of the expert it chose
    r = _route(L)
    out = oracle.moe_forward(bf16_bits(L.x), r, bf16_bits(L.W1), bf16_bits(L.W3), bf16_bits(L.W2), 0)
    for t in range(T):
        assert np.abs(out[t] - Y[r.expert_ids[t, 0], t]).max() <= 1e-12 * (1 + np.abs(out[t]).max())


def test_cosine_matrix_closed_forms():
    rng = np.random.default_rng(52)
    a = rng.standard_normal((7, 5))
    b = rng.standard_normal((7, 5))
    b_perp = b - a * (np.sum(a * b) / np.sum(a * a))            # orthogonal to a as a flattened vector
    Y = np.stack([a, 3.0 * a, -2.0 * a, b_perp, a + b_perp])
    gram, cos = oracle.cosine_matrix(Y)
    assert np.allclose(np.diag(cos), 1.0, atol=1e-12) and np.allclose(cos, cos.T, atol=1e-15)
    assert abs(cos[0, 1] - 1) <= 1e-12 and abs(cos[0, 2] + 1) <= 1e-12 and abs(cos[0, 3]) <= 1e-12
    na, nb = np.sqrt(np.sum(a * a)), np.sqrt(np.sum(b_perp * b_perp))
    assert abs(cos[0, 4] - na / np.sqrt(na * na + nb * nb)) <= 1e-12      # angle of a sum of orthogonal vectors
    assert abs(gram[1, 2] + 6.0 * na * na) <= 1e-9
    assert np.abs(cos).max() <= 1 + 1e-12
    assert np.allclose(gram, np.einsum("etd,ftd->ef", Y, Y), rtol=1e-12, atol=1e-12)   # library contraction


def test_group_mse_hand_worked_and_special_cases():
    # Eq. 5 by hand: members with outputs 1 and 3, selected 1 and 3 times -> alpha = 1/4, 3/4 -> target 2.5;
    # united output 2 -> MSE_0 = 0.25.  Second group: a single member (7), united output 7 -> MSE_1 = 0.
    # w = [1, 3, 4] -> frequencies 1/8, 3/8, 4/8 -> beta = [1/2, 1/2] -> MSE_total = 0.125   (Eq. 6)
    Y = np.array([[[1.0]], [[3.0]], [[7.0]]])
    U = np.array([[[2.0]], [[7.0]]])
    mse, total, target = oracle.group_mse(Y, U, [1, 3, 4], [0, 0, 1], 2)
    assert target.ravel().tolist() == [2.5, 7.0] and mse.tolist() == [0.25, 0.0] and total == 0.125
    # mean over tokens of the squared L2 norm over features (Eq. 9): T = 2, D = 2, differences (1, 2) and (0, 2)
    Y = np.zeros((1, 2, 2))
    U = np.array([[[1.0, 2.0], [0.0, 2.0]]])
    mse, total, _ = oracle.group_mse(Y, U, [5], [0], 1)
    assert mse.tolist() == [(1 + 4 + 0 + 4) / 2] and total == mse[0]
    # identical members: any alpha gives the member itself; a united expert equal to it has zero error
    rng = np.random.default_rng(53)
    a = rng.standard_normal((6, 4))
    Y = np.stack([a, a, rng.standard_normal((6, 4))])
    U = np.stack([a, Y[2]])
    mse, total, _ = oracle.group_mse(Y, U, [2, 9, 1], [0, 0, 1], 2)
    assert np.abs(mse).max() <= 1e-28 and total <= 1e-28
    # a never-selected group carries no weight (beta = 0); an empty group contributes nothing
    Y = np.array([[[1.0]], [[5.0]]])
    U = np.array([[[0.0]], [[0.0]], [[9.0]]])
    mse, total, target = oracle.group_mse(Y, U, [4, 0], [0, 1, ][:2], 3)
    assert mse.tolist() == [1.0, 25.0, 0.0] and total == 1.0
    # the convex target lies between the member outputs (Eq. 5 is a convex combination)
    Y = rng.standard_normal((4, 3, 2))
    _, _, target = oracle.group_mse(Y, np.zeros((1, 3, 2)), [1, 2, 3, 4], [0, 0, 0, 0], 1)
    assert (target[0] <= Y.max(0) + 1e-12).all() and (target[0] >= Y.min(0) - 1e-12).all()
    assert np.allclose(target[0], np.tensordot(np.array([1, 2, 3, 4]) / 10.0, Y, axes=1), atol=1e-14)
