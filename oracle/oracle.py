"""ctypes binding of the CPU oracle (oracle/bm_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  It never imports paper_2607_04164_b200 and shares no code with it.

Arrays are numpy: bf16 tensors travel as uint16 storage (`bm_inputs.bf16_bits`).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from types import SimpleNamespace

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bm_oracle.c")
_LIB = os.path.join(_HERE, "libbm_oracle.so")
_lib = None

# x86-64-v3 (AVX2 + FMA) rather than -march=native: the .so may be built on one host and run on
# another.  fmaf() is correctly rounded either way (hardware FMA or glibc's software fma).
# -ffp-contract=off: the only fused multiply-adds are the explicit fmaf() calls of the canonical dot.
CFLAGS = ["-O2", "-std=c11", "-march=x86-64-v3", "-fno-fast-math", "-ffp-contract=off", "-fopenmp",
          "-fPIC", "-shared"]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc if the .so is missing or older than its source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.oracle_canon_dot.restype = ctypes.c_float
        _lib.oracle_route.restype = ctypes.c_int
        _lib.oracle_route_partial.restype = ctypes.c_int
        _lib.oracle_unite_weights.restype = ctypes.c_int
        _lib.oracle_moe_forward.restype = ctypes.c_int
        _lib.oracle_expert_outputs.restype = ctypes.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _u16(a) -> np.ndarray:
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16, a.dtype
    return a


def canon_dot(x_bits: np.ndarray, w_bits: np.ndarray) -> float:
    """Reading A1: canonical fp32 dot product of two bf16 vectors (uint16 storage)."""
    x_bits, w_bits = _u16(x_bits), _u16(w_bits)
    assert x_bits.shape == w_bits.shape and x_bits.ndim == 1
    return float(_load().oracle_canon_dot(_p(x_bits), _p(w_bits), ctypes.c_int(x_bits.shape[0])))


def route(x, W_router, router_bias, K: int, group_map, G: int, want_logits: bool = False,
          cold_mask=None) -> SimpleNamespace:
    """R1-R7 (PAPER.md:42 gate + top-K; Eq. 2 group map; readings A1-A7).

    x [T,D] uint16, W_router [E,D] uint16, router_bias [E] float32 or None, group_map [E] int32.
    cold_mask [E] (non-zero = cold) switches to partial brownout: hot experts keep
    their own weights, numbered as weight sets G + e, and the routing arrays range over G + E sets
    (returned as r.G).  Returns the routing arrays of SURVEY.md 8(b) as numpy arrays.
    """
    x, W_router = _u16(x), _u16(W_router)
    T, D = x.shape
    E = W_router.shape[0]
    assert W_router.shape[1] == D
    gmap = np.ascontiguousarray(group_map, dtype=np.int32)
    assert gmap.shape == (E,)
    bias = None if router_bias is None else np.ascontiguousarray(router_bias, dtype=np.float32)
    cold = None if cold_mask is None else np.ascontiguousarray(cold_mask, dtype=np.int32)
    NS = G if cold is None else G + E
    r = SimpleNamespace(T=T, E=E, K=K, G=NS, G_united=G)
    r.expert_ids = np.empty((T, K), np.int32)
    r.group_ids = np.empty((T, K), np.int32)
    r.gate_w = np.empty((T, K), np.float32)
    r.n_slots = np.empty((T,), np.int32)
    r.counts = np.empty((NS,), np.int32)
    r.offsets = np.empty((NS + 1,), np.int32)
    r.row_token = np.empty((T * K,), np.int32)
    r.row_slot = np.empty((T * K,), np.int32)
    r.slot_row = np.empty((T, K), np.int32)
    r.logits = np.empty((T, E), np.float32) if want_logits else None
    args = [_p(x), T, D, _p(W_router), _p(bias), E, K, _p(gmap), G]
    outs = [_p(r.expert_ids), _p(r.group_ids), _p(r.gate_w), _p(r.n_slots), _p(r.counts), _p(r.offsets),
            _p(r.row_token), _p(r.row_slot), _p(r.slot_row), _p(r.logits)]
    if cold is None:
        rc = _load().oracle_route(*args, *outs)
    else:
        assert cold.shape == (E,)
        rc = _load().oracle_route_partial(*args, _p(cold), *outs)
    if rc != 0:
        raise ValueError("oracle_route: bad shape or group_map entry outside [0,G)")
    r.A = int(r.offsets[NS])
    return r


def unite_weights(W, group_map, G: int) -> np.ndarray:
    """Parameter average of the member experts of every group, fp64.
    W [E, ...] uint16 (bf16 storage) -> [G, ...] float64."""
    W = _u16(W)
    E = W.shape[0]
    n = int(np.prod(W.shape[1:]))
    gmap = np.ascontiguousarray(group_map, dtype=np.int32)
    out = np.empty((G,) + W.shape[1:], np.float64)
    rc = _load().oracle_unite_weights(_p(W), E, ctypes.c_longlong(n), _p(gmap), G, _p(out))
    if rc != 0:
        raise ValueError("oracle_unite_weights: bad arguments")
    return out


def moe_forward(x, routing, W1, W3, W2, S: int = 0, sel_tokens=None) -> np.ndarray:
    """F1-F2 in fp64 (PAPER.md:42 h_t = sum g_i FFN_i(x_t) with united experts; SwiGLU: A3).

    W1, W3 [G+S,F,D] uint16; W2 [G+S,D,F] uint16.  sel_tokens: ascending token indices to evaluate
    (None = all).  Returns out [n_sel, D] float64.
    """
    x, W1, W3, W2 = _u16(x), _u16(W1), _u16(W3), _u16(W2)
    T, D = x.shape
    G, K = routing.G, routing.K
    F = W1.shape[1]
    assert W1.shape == (G + S, F, D) and W3.shape == (G + S, F, D) and W2.shape == (G + S, D, F)
    sel = None
    n_sel = T
    if sel_tokens is not None:
        sel = np.ascontiguousarray(sel_tokens, dtype=np.int32)
        assert sel.ndim == 1 and (np.diff(sel) > 0).all()
        n_sel = sel.shape[0]
    out = np.empty((n_sel, D), np.float64)
    rc = _load().oracle_moe_forward(_p(x), T, D, K, G, _p(routing.group_ids), _p(routing.gate_w),
                                    _p(routing.n_slots), _p(routing.offsets), _p(routing.row_token),
                                    _p(routing.slot_row), _p(W1), _p(W3), _p(W2), F, S,
                                    _p(sel), n_sel, _p(out))
    if rc != 0:
        raise ValueError("oracle_moe_forward: bad arguments")
    return out


# ---------------------------------------------------------------------------------------------------
# Calibration forward: the forward half of the reward evaluation of PAPER.md 4.3
# ---------------------------------------------------------------------------------------------------
def expert_histogram(expert_ids, E: int) -> np.ndarray:
    """Routing frequency w_e, "how often expert e is selected by the gating function on the calibration
    dataset", as integer counts over the ranked top-K ids [T, K]."""
    w = np.zeros(E, np.int64)
    for e in np.asarray(expert_ids).ravel():
        w[int(e)] += 1
    return w


def expert_outputs(x, W1, W3, W2) -> np.ndarray:
    """f_e(x_t) for every original expert e and token t, fp64 [E, T, D] (Eq. 5's f_e)."""
    x, W1, W3, W2 = _u16(x), _u16(W1), _u16(W3), _u16(W2)
    T, D = x.shape
    E, F = W1.shape[0], W1.shape[1]
    assert W1.shape == (E, F, D) and W3.shape == (E, F, D) and W2.shape == (E, D, F)
    out = np.empty((E, T, D), np.float64)
    rc = _load().oracle_expert_outputs(_p(x), T, D, _p(W1), _p(W3), _p(W2), E, F, _p(out))
    if rc != 0:
        raise ValueError("oracle_expert_outputs: bad arguments")
    return out


def cosine_matrix(Y) -> tuple:
    """Pairwise cosine similarity matrix of expert outputs from calibration data.  Reading A19:
    expert e is the vector of all its outputs, Y[e] flattened over tokens and features;
    gram[e, e'] = <Y_e, Y_e'>,  cos[e, e'] = gram[e, e'] / (|Y_e| |Y_e'|).  Returns (gram, cos), fp64 [E, E]."""
    Y = np.asarray(Y, np.float64)
    E = Y.shape[0]
    gram = np.zeros((E, E))
    for a in range(E):
        for b in range(E):
            gram[a, b] = float(np.sum(Y[a] * Y[b]))
    norm = np.sqrt(np.diag(gram))
    cos = np.zeros((E, E))
    for a in range(E):
        for b in range(E):
            cos[a, b] = gram[a, b] / (norm[a] * norm[b]) if norm[a] > 0 and norm[b] > 0 else 0.0
    return gram, cos


def group_mse(Y, U, w, group_map, G: int) -> tuple:
    """Eq. 5 and Eq. 6 for a given united-expert output U [G, T, D]:
        alpha_e = w_e / sum_{e' in G_k} w_e',   t_k(x) = sum_{e in G_k} alpha_e f_e(x)          (5)
        MSE_r = E_x || f_{u_r}(x) - t_r(x) ||_2^2   (mean over calibration tokens of the squared L2 norm, Eq. 9)
        beta_r = sum_{e in G_r} w_e,  MSE_total = sum_r beta_r MSE_r                             (6)
    Reading A20: w_e are the routing counts normalised to sum 1 (frequencies); a group none of whose members
    was ever selected has beta_r = 0 and takes uniform alpha (its term vanishes); an empty group has MSE_r = 0.
    Returns (mse [G], mse_total, target [G, T, D])."""
    Y, U = np.asarray(Y, np.float64), np.asarray(U, np.float64)
    w = np.asarray(w, np.float64)
    gmap = np.asarray(group_map)
    wn = w / w.sum() if w.sum() > 0 else np.zeros_like(w)
    T = Y.shape[1]
    mse = np.zeros(G)
    target = np.zeros_like(U)
    total = 0.0
    for r in range(G):
        members = [e for e in range(len(gmap)) if gmap[e] == r]
        if not members:
            continue
        beta = sum(wn[e] for e in members)
        t = np.zeros_like(U[r])
        for e in members:
            alpha = wn[e] / beta if beta > 0 else 1.0 / len(members)
            t = t + alpha * Y[e]
        target[r] = t
        diff = U[r] - t
        mse[r] = float(np.sum(diff * diff)) / T if T > 0 else 0.0
        total += beta * mse[r]
    return mse, total, target


def num_threads() -> int:
    """Threads the OpenMP loops actually use (OMP_NUM_THREADS, else the affinity mask)."""
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else len(os.sched_getaffinity(0))
