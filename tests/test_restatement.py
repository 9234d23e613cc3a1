"""The all-T matmul restatement (tests/restatement.py) against the plain oracle, on shapes the oracle finishes in
seconds (-m "not gpu").  SURVEY.md 8(c) "Large shapes": the restatement covers all T at full size only because it
agrees with the step-by-step oracle here and on the sampled subset of every full-size GPU test."""
import numpy as np
import pytest
import torch

from helpers import oracle_layer, rand_layer
from restatement import chunk_boundary_tokens, layer_restatement


@pytest.mark.parametrize("T,D,F,E,K,G,S", [
    (300, 512, 1000, 8, 2, 3, 1),
    (257, 264, 328, 60, 4, 15, 0),
    (40, 64, 72, 9, 3, 9, 2),
    (1, 128, 64, 4, 2, 2, 0),
])
def test_restatement_matches_oracle(T, D, F, E, K, G, S):
    rng = np.random.default_rng(T + 13 * F)
    L = rand_layer(rng, T=T, D=D, F=F, E=E, K=K, G=G, S=S, bias=True)
    r, want = oracle_layer(L)
    got64 = layer_restatement(L.x, r, L.W1, L.W3, L.W2, S, dtype=torch.float64, row_block=97)
    scale = np.abs(want).max() + 1e-30
    assert np.abs(got64 - want).max() <= 1e-11 * scale            # same real numbers, fp64 both sides
    got32 = layer_restatement(L.x, r, L.W1, L.W3, L.W2, S, dtype=torch.float32)
    assert np.abs(got32 - want).max() <= 2e-5 * scale             # fp32 matmuls: ~sqrt(F) * 2^-24 relative


def test_restatement_catches_a_dropped_gate_weight_and_a_wrong_group():
    # the comparison above is discriminating: perturbing one routing entry moves the restatement off the oracle
    rng = np.random.default_rng(3)
    L = rand_layer(rng, T=64, D=128, F=192, E=8, K=2, G=4, S=0, bias=True)
    r, want = oracle_layer(L)
    from types import SimpleNamespace
    bad = SimpleNamespace(group_ids=r.group_ids.copy(), gate_w=r.gate_w.copy(), n_slots=r.n_slots.copy())
    bad.gate_w[5, 0] = 1.0 - bad.gate_w[5, 0]
    got = layer_restatement(L.x, bad, L.W1, L.W3, L.W2, 0, dtype=torch.float64)
    assert np.abs(got[5] - want[5]).max() > 1e-3 * np.abs(want).max()
    bad.gate_w[:] = r.gate_w
    bad.group_ids[7, 0] = (bad.group_ids[7, 0] + 1) % 4
    if bad.n_slots[7] == 2 and bad.group_ids[7, 1] == bad.group_ids[7, 0]:
        bad.group_ids[7, 0] = (bad.group_ids[7, 0] + 1) % 4
    got = layer_restatement(L.x, bad, L.W1, L.W3, L.W2, 0, dtype=torch.float64)
    assert np.abs(got[7] - want[7]).max() > 1e-3 * np.abs(want).max()


def test_rounding_switches_model_bf16_and_stay_close():
    rng = np.random.default_rng(4)
    L = rand_layer(rng, T=100, D=256, F=320, E=8, K=2, G=4, S=1)
    r, want = oracle_layer(L)
    got = layer_restatement(L.x, r, L.W1, L.W3, L.W2, 1, dtype=torch.float64, round_h=True, round_y=True)
    err = np.abs(got - want)
    assert err.max() > 0                                          # the roundings do something
    rms = lambda a: float(np.sqrt(np.mean(np.square(a))))
    assert rms(err) <= 4e-3 * rms(want)                           # two bf16 roundings: ~2 * 2^-9 / sqrt(3) relative


def test_chunk_boundary_tokens_hits_every_chunk_edge():
    rng = np.random.default_rng(5)
    L = rand_layer(rng, T=700, D=64, F=64, E=6, K=2, G=3, S=1)
    r, _ = oracle_layer(L)
    sel = chunk_boundary_tokens(r, 700, S=1)
    for u in range(3):
        lo, hi = int(r.offsets[u]), int(r.offsets[u + 1])
        for c0 in range(lo, hi, 128):
            assert int(r.row_token[c0]) in sel and int(r.row_token[min(c0 + 128, hi) - 1]) in sel
    assert {0, 127, 128, 699} <= sel
