"""Thin ctypes binding of include/bm.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of libbm.so; PyTorch is used for device memory and
streams.  There is no fallback: if the library is missing it is built with nvcc, and if that fails or
no sm_100 device is present the calls raise.
"""
from __future__ import annotations

import ctypes
from ctypes import POINTER, c_float, c_int, c_int32, c_longlong, c_size_t, c_void_p

import torch

from . import build as _build

BM_OK = 0
BM_PATH_AUTO, BM_PATH_DECODE, BM_PATH_PREFILL, BM_PATH_SIMT, BM_PATH_GEMV = 0, 1, 2, 3, 4
BM_DEV_BAD_GROUP_MAP, BM_DEV_NONFINITE_LOGIT, BM_DEV_BAD_ROUTING = 1, 2, 4
BM_MAX_E, BM_MAX_K, BM_MAX_G, BM_MAX_S = 512, 16, 512, 16
BM_DECODE_MAX_T = 320
BM_ERR_LIMIT = -7
BM_STATIC_ROUTE_BYTES, BM_STATIC_ROUTE_MAX_T = 2 * 1024 * 1024, 8192

EXPORTS = ["bm_moe_layer", "bm_expert_outputs_workspace_bytes", "bm_workspace_bytes", "bm_workspace_init", "bm_forward_info", "bm_host_chunks", "bm_set_option", "bm_get_option", "bm_route", "bm_route_static", "bm_route_static_status", "bm_route_partial", "bm_unite_weights", "bm_expert_histogram",
           "bm_expert_outputs", "bm_gram_workspace_bytes", "bm_cosine_gram", "bm_mse_workspace_bytes", "bm_group_mse",
           "bm_moe_forward", "bm_moe_forward_path", "bm_moe_forward_f32", "bm_round_bf16", "bm_moe_layer_host",
           "bm_device_status", "bm_launch_count", "bm_status_string", "bm_profile_enable", "bm_profile_read", "bm_profile_read_kinds",
           "bm_salc_init", "bm_salc_observe", "bm_salc_p90", "bm_salc_cold_mask"]
KERNELS = {"router": 1, "permute": 2, "prep": 3, "gemm1": 4, "gemm2": 5, "finalize": 6, "all": 7}


BM_SALC_MAX_WINDOW = 256


class BmSalc(ctypes.Structure):
    """include/bm.h: bm_salc (host-side SLO-aware latency controller, PAPER.md 4.5)."""
    _fields_ = [("slo", ctypes.c_double), ("warn_frac", ctypes.c_double), ("decrease", ctypes.c_double),
                ("increase", ctypes.c_double), ("threshold", ctypes.c_double), ("window", c_int32),
                ("count", c_int32), ("head", c_int32), ("lat", ctypes.c_double * BM_SALC_MAX_WINDOW)]


class BmRouting(ctypes.Structure):
    _fields_ = [("T", c_int32), ("E", c_int32), ("K", c_int32), ("G", c_int32),
                ("expert_ids", c_void_p), ("group_ids", c_void_p), ("gate_w", c_void_p),
                ("n_slots", c_void_p), ("counts", c_void_p), ("offsets", c_void_p),
                ("row_token", c_void_p), ("row_slot", c_void_p), ("slot_row", c_void_p)]


class BmError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {status_string(code)} ({code})")


_lib = None


def lib() -> ctypes.CDLL:
    """Load libbm.so (building it in-tree with nvcc if it is missing or stale)."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        L.bm_workspace_bytes.restype = c_size_t
        L.bm_workspace_bytes.argtypes = [c_int] * 7
        L.bm_workspace_init.restype = c_int
        L.bm_workspace_init.argtypes = [c_void_p, c_size_t, c_void_p]
        L.bm_forward_info.restype = c_int
        L.bm_forward_info.argtypes = [c_int] * 6 + [POINTER(c_int), POINTER(c_int)]
        L.bm_host_chunks.restype = c_int
        L.bm_host_chunks.argtypes = [c_int] * 4 + [POINTER(c_int), c_int]
        L.bm_set_option.restype = c_int
        L.bm_set_option.argtypes = [ctypes.c_char_p, c_int]
        L.bm_get_option.restype = c_int
        L.bm_get_option.argtypes = [ctypes.c_char_p, POINTER(c_int)]
        L.bm_route.restype = c_int
        L.bm_route.argtypes = [c_void_p, c_int, c_int, c_void_p, c_void_p, c_int, c_int, c_void_p, c_int,
                               POINTER(BmRouting), c_void_p, c_size_t, c_void_p]
        L.bm_route_static.restype = c_int
        L.bm_route_static.argtypes = [c_void_p, c_int, c_int, c_void_p, c_void_p, c_int, c_int, c_void_p, c_int,
                                      POINTER(BmRouting), c_void_p]
        L.bm_route_static_status.restype = c_int
        L.bm_route_static_status.argtypes = [POINTER(c_int32), c_void_p]
        L.bm_route_partial.restype = c_int
        L.bm_route_partial.argtypes = [c_void_p, c_int, c_int, c_void_p, c_void_p, c_int, c_int, c_void_p, c_int,
                                       c_void_p, POINTER(BmRouting), c_void_p, c_size_t, c_void_p]
        L.bm_unite_weights.restype = c_int
        L.bm_unite_weights.argtypes = [c_void_p, c_int, c_size_t, c_void_p, c_int, c_void_p, c_void_p]
        L.bm_expert_histogram.restype = c_int
        L.bm_expert_histogram.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_void_p]
        L.bm_expert_outputs_workspace_bytes.restype = c_size_t
        L.bm_expert_outputs_workspace_bytes.argtypes = [c_int] * 4
        L.bm_expert_outputs.restype = c_int
        L.bm_expert_outputs.argtypes = [c_void_p, c_int, c_int, c_void_p, c_void_p, c_void_p, c_int, c_int, c_void_p,
                                        c_void_p, c_size_t, c_void_p]
        L.bm_gram_workspace_bytes.restype = c_size_t
        L.bm_gram_workspace_bytes.argtypes = [c_int]
        L.bm_cosine_gram.restype = c_int
        L.bm_cosine_gram.argtypes = [c_void_p, c_int, c_int, c_int, c_void_p, c_void_p, c_void_p, c_size_t, c_void_p]
        L.bm_mse_workspace_bytes.restype = c_size_t
        L.bm_mse_workspace_bytes.argtypes = [c_int]
        L.bm_group_mse.restype = c_int
        L.bm_group_mse.argtypes = [c_void_p, c_void_p, c_int, c_int, c_void_p, c_void_p, c_int, c_int, c_void_p,
                                   c_void_p, c_void_p, c_size_t, c_void_p]
        L.bm_moe_forward.restype = c_int
        L.bm_moe_forward.argtypes = [c_void_p, c_int, c_int, POINTER(BmRouting), c_void_p, c_void_p, c_void_p,
                                     c_int, c_int, c_void_p, c_void_p, c_size_t, c_void_p]
        L.bm_moe_forward_f32.restype = c_int
        L.bm_moe_forward_f32.argtypes = L.bm_moe_forward.argtypes
        L.bm_round_bf16.restype = c_int
        L.bm_round_bf16.argtypes = [c_void_p, c_size_t, c_void_p, c_void_p]
        L.bm_salc_init.restype = c_int
        L.bm_salc_init.argtypes = [POINTER(BmSalc), ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double, c_int]
        L.bm_salc_observe.restype = ctypes.c_double
        L.bm_salc_observe.argtypes = [POINTER(BmSalc), ctypes.c_double]
        L.bm_salc_p90.restype = ctypes.c_double
        L.bm_salc_p90.argtypes = [POINTER(BmSalc)]
        L.bm_salc_cold_mask.restype = c_int
        L.bm_salc_cold_mask.argtypes = [c_void_p, c_int, ctypes.c_double, c_void_p]
        L.bm_moe_forward_path.restype = c_int
        L.bm_moe_forward_path.argtypes = L.bm_moe_forward.argtypes + [c_int]
        L.bm_moe_layer.restype = c_int
        L.bm_moe_layer.argtypes = [c_void_p, c_int, c_int, c_void_p, c_void_p, c_int, c_int, c_void_p, c_int,
                                   c_void_p, c_void_p, c_void_p, c_int, c_int, c_void_p, POINTER(BmRouting), c_void_p, c_size_t, c_void_p]
        L.bm_moe_layer_host.restype = c_int
        L.bm_moe_layer_host.argtypes = [c_void_p, c_int, c_int, c_void_p, c_void_p, c_int, c_int, c_void_p, c_int,
                                        c_void_p, c_void_p, c_void_p, c_int, c_int, c_void_p, c_void_p, c_void_p,
                                        POINTER(BmRouting), c_void_p, c_size_t, c_void_p]
        L.bm_device_status.restype = c_int
        L.bm_device_status.argtypes = [c_void_p, POINTER(c_int32), c_void_p]
        L.bm_launch_count.restype = c_longlong
        L.bm_launch_count.argtypes = []
        L.bm_profile_enable.restype = c_int
        L.bm_profile_enable.argtypes = [c_int, c_int]
        L.bm_profile_read.restype = c_int
        L.bm_profile_read.argtypes = [POINTER(c_float), POINTER(c_int)]
        L.bm_profile_read_kinds.restype = c_int
        L.bm_profile_read_kinds.argtypes = [POINTER(c_float), POINTER(c_int)]
        L.bm_status_string.restype = ctypes.c_char_p
        L.bm_status_string.argtypes = [c_int]
        _lib = L
    return _lib


def status_string(code: int) -> str:
    return lib().bm_status_string(code).decode()


def launch_count() -> int:
    return int(lib().bm_launch_count())


def workspace_bytes(T_max: int, D: int, F: int, E: int, K: int, G: int, S: int = 0) -> int:
    return int(lib().bm_workspace_bytes(T_max, D, F, E, K, G, S))


def _ptr(t):
    return None if t is None else c_void_p(t.data_ptr())


def _dev(name, t, dtype, shape=None, optional=False):
    """Marshalling guard: the C ABI takes raw pointers, so a strided, mistyped or host tensor would be read out of
    bounds on the device.  Checks dtype, contiguity, CUDA residency (and the shape when given)."""
    if t is None:
        if optional:
            return
        raise ValueError(f"{name} is required")
    if t.dtype != dtype:
        raise TypeError(f"{name}: expected {dtype}, got {t.dtype}")
    if not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return c_void_p(s.cuda_stream)


def set_option(name: str, value: int) -> None:
    """include/bm.h: bm_set_option (process-global tuning / test switch)."""
    rc = lib().bm_set_option(name.encode(), int(value))
    if rc != BM_OK:
        raise BmError(rc, f"bm_set_option({name})")


def get_option(name: str) -> int:
    v = c_int(0)
    rc = lib().bm_get_option(name.encode(), ctypes.byref(v))
    if rc != BM_OK:
        raise BmError(rc, f"bm_get_option({name})")
    return int(v.value)


class options:
    """Context manager: set options for the duration of a block, then restore the previous values."""

    def __init__(self, **kw):
        self.kw = kw

    def __enter__(self):
        self.old = {k: get_option(k) for k in self.kw}
        for k, v in self.kw.items():
            set_option(k, v)
        return self

    def __exit__(self, *a):
        for k, v in self.old.items():
            set_option(k, v)
        return False


def bm_forward_info(T: int, K: int, G: int, S: int, D: int, F: int):
    """(path, deterministic) of bm_moe_forward for a batch of these sizes (include/bm.h: bm_forward_info)."""
    pth, det = c_int(0), c_int(0)
    rc = lib().bm_forward_info(T, K, G, S, D, F, ctypes.byref(pth), ctypes.byref(det))
    if rc != BM_OK:
        raise BmError(rc, "bm_forward_info")
    return int(pth.value), bool(det.value)


def bm_host_chunks(T: int, F: int, K: int, S: int):
    """Token chunk sizes bm_moe_layer_host processes a batch of T tokens in (include/bm.h: bm_host_chunks)."""
    sizes = (c_int * 16)()
    n = lib().bm_host_chunks(T, F, K, S, sizes, 16)
    if n < 0:
        raise BmError(n, "bm_host_chunks")
    return [int(sizes[i]) for i in range(n)]


class Routing:
    """Device arrays of one batch's routing (bm_routing), allocated at their maximum size."""

    def __init__(self, T_max: int, K: int, G: int, device="cuda"):
        i32 = dict(dtype=torch.int32, device=device)
        n = max(T_max * K, 1)
        self.T_max, self.K, self.G = T_max, K, G
        self.expert_ids = torch.empty(n, **i32)
        self.group_ids = torch.empty(n, **i32)
        self.gate_w = torch.empty(n, dtype=torch.float32, device=device)
        self.n_slots = torch.empty(max(T_max, 1), **i32)
        self.counts = torch.empty(G, **i32)
        self.offsets = torch.empty(G + 1, **i32)
        self.row_token = torch.empty(n, **i32)
        self.row_slot = torch.empty(n, **i32)
        self.slot_row = torch.empty(n, **i32)
        self.c = BmRouting(0, 0, K, G, *[t.data_ptr() for t in (
            self.expert_ids, self.group_ids, self.gate_w, self.n_slots, self.counts, self.offsets,
            self.row_token, self.row_slot, self.slot_row)])

    def view(self, T: int):
        """The routing arrays trimmed/reshaped for a batch of T tokens (no copy)."""
        K = self.K
        return dict(expert_ids=self.expert_ids[:T * K].view(T, K), group_ids=self.group_ids[:T * K].view(T, K),
                    gate_w=self.gate_w[:T * K].view(T, K), n_slots=self.n_slots[:T], counts=self.counts,
                    offsets=self.offsets, row_token=self.row_token[:T * K], row_slot=self.row_slot[:T * K],
                    slot_row=self.slot_row[:T * K].view(T, K))


def alloc_workspace(T_max: int, D: int, F: int, E: int, K: int, G: int, S: int = 0, device="cuda") -> torch.Tensor:
    """Workspace for shapes up to T_max, initialised (zeroed) with bm_workspace_init."""
    n = workspace_bytes(T_max, D, F, E, K, G, S)
    if n == 0:
        raise BmError(-2, "bm_workspace_bytes")
    ws = torch.empty(n, dtype=torch.uint8, device=device)
    rc = lib().bm_workspace_init(_ptr(ws), n, _stream())
    if rc != BM_OK:
        raise BmError(rc, "bm_workspace_init")
    return ws


def _check_route_args(x, W_router, router_bias, group_map, routing, workspace, T, D, E, K, n_sets):
    _dev("x", x, torch.bfloat16)
    _dev("W_router", W_router, torch.bfloat16, (E, D))
    _dev("router_bias", router_bias, torch.float32, (E,), optional=True)
    _dev("group_map", group_map, torch.int32, (E,))
    _dev("workspace", workspace, torch.uint8)
    if T > routing.T_max or K != routing.K or n_sets != routing.G:
        raise ValueError(f"routing arrays were allocated for T <= {routing.T_max}, K = {routing.K}, {routing.G} sets; "
                         f"got T = {T}, K = {K}, {n_sets} sets")


def _check_forward_args(x, routing, W1, W3, W2, out, out_dtype, workspace, S):
    T, D = x.shape
    n_sets, F = W1.shape[0], W1.shape[1]
    _dev("x", x, torch.bfloat16)
    _dev("W1", W1, torch.bfloat16, (n_sets, F, D))
    _dev("W3", W3, torch.bfloat16, (n_sets, F, D))
    _dev("W2", W2, torch.bfloat16, (n_sets, D, F))
    _dev("out", out, out_dtype, (T, D))
    _dev("workspace", workspace, torch.uint8)
    if T > routing.T_max or n_sets != routing.G + S:
        raise ValueError(f"routing arrays hold T <= {routing.T_max} and {routing.G} sets (+ S = {S}); got T = {T}, "
                         f"{n_sets} weight sets")
    return T, D, F


def bm_route(x, W_router, router_bias, K: int, group_map, G: int, routing: Routing, workspace, stream=None):
    """R1-R7 (include/bm.h: bm_route).  x [T,D] bf16, W_router [E,D] bf16, router_bias [E] f32 | None,
    group_map [E] i32; fills `routing` asynchronously on the current stream."""
    T, D = x.shape
    E = W_router.shape[0]
    _check_route_args(x, W_router, router_bias, group_map, routing, workspace, T, D, E, K, G)
    rc = lib().bm_route(_ptr(x), T, D, _ptr(W_router), _ptr(router_bias), E, K, _ptr(group_map), G,
                        ctypes.byref(routing.c), _ptr(workspace), workspace.numel(), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_route")
    return routing


def bm_route_static(x, W_router, router_bias, K: int, group_map, G: int, routing: Routing, stream=None):
    """bm_route without a workspace: its scratch is a fixed 2 MiB device array inside the library, nothing is allocated
    (include/bm.h: bm_route_static).  T <= BM_STATIC_ROUTE_MAX_T, else BmError(BM_ERR_LIMIT); calls that overlap on the
    GPU race on the shared array."""
    T, D = x.shape
    E = W_router.shape[0]
    _dev("x", x, torch.bfloat16)
    _dev("W_router", W_router, torch.bfloat16, (E, D))
    _dev("router_bias", router_bias, torch.float32, (E,), optional=True)
    _dev("group_map", group_map, torch.int32, (E,))
    if T > routing.T_max or K != routing.K or G != routing.G:
        raise ValueError(f"routing arrays were allocated for T <= {routing.T_max}, K = {routing.K}, {routing.G} sets; "
                         f"got T = {T}, K = {K}, {G} sets")
    rc = lib().bm_route_static(_ptr(x), T, D, _ptr(W_router), _ptr(router_bias), E, K, _ptr(group_map), G,
                               ctypes.byref(routing.c), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_route_static")
    return routing


def bm_route_static_status(stream=None) -> int:
    """Device status bits of the last bm_route_static call on this device; synchronises the stream."""
    v = c_int32(0)
    rc = lib().bm_route_static_status(ctypes.byref(v), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_route_static_status")
    return int(v.value)


def bm_route_partial(x, W_router, router_bias, K: int, group_map, G: int, cold_mask, routing: Routing, workspace,
                     stream=None):
    """Partial brownout routing (include/bm.h: bm_route_partial).  cold_mask [E] i32; `routing` must have been
    allocated for G + E weight sets (Routing(T, K, G + E)) and the workspace sized for G + E."""
    T, D = x.shape
    E = W_router.shape[0]
    _check_route_args(x, W_router, router_bias, group_map, routing, workspace, T, D, E, K, G + E)
    _dev("cold_mask", cold_mask, torch.int32, (E,), optional=True)     # None: the C ABI reports BM_ERR_NULL
    rc = lib().bm_route_partial(_ptr(x), T, D, _ptr(W_router), _ptr(router_bias), E, K, _ptr(group_map), G,
                                _ptr(cold_mask), ctypes.byref(routing.c), _ptr(workspace), workspace.numel(),
                                _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_route_partial")
    return routing


def bm_unite_weights(W, group_map, G: int, out=None, stream=None):
    """Parameter average of member experts (include/bm.h: bm_unite_weights).  W [E, ...] bf16 -> [G, ...] bf16."""
    E = W.shape[0]
    n = W[0].numel()
    if out is None:
        out = torch.empty((G,) + tuple(W.shape[1:]), dtype=W.dtype, device=W.device)
    rc = lib().bm_unite_weights(_ptr(W), E, n, _ptr(group_map), G, _ptr(out), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_unite_weights")
    return out


def bm_expert_histogram(expert_ids, E: int, stream=None):
    """w[e] = how often expert e was selected (include/bm.h: bm_expert_histogram).  expert_ids [T,K] i32 -> [E] i32."""
    T, K = expert_ids.shape
    w = torch.empty(E, dtype=torch.int32, device=expert_ids.device)
    rc = lib().bm_expert_histogram(_ptr(expert_ids), T, K, E, _ptr(w), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_expert_histogram")
    return w


def bm_expert_outputs(x, W1, W3, W2, y=None, workspace=None, stream=None):
    """y[t,e,:] = FFN_e(x_t) for every expert and token (include/bm.h: bm_expert_outputs) -> token-major [T,E,D] bf16."""
    T, D = x.shape
    E, F = W1.shape[0], W1.shape[1]
    if y is None:
        y = torch.empty((T, E, D), dtype=torch.bfloat16, device=x.device)
    if workspace is None:
        workspace = torch.empty(int(lib().bm_expert_outputs_workspace_bytes(T, D, F, E)), dtype=torch.uint8, device=x.device)
    rc = lib().bm_expert_outputs(_ptr(x), T, D, _ptr(W1), _ptr(W3), _ptr(W2), E, F, _ptr(y), _ptr(workspace),
                                 workspace.numel(), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_expert_outputs")
    return y


def bm_cosine_gram(Y, stream=None):
    """(gram, cosine) [E,E] f32 of the expert outputs Y [T,E,D] bf16, token-major (include/bm.h: bm_cosine_gram)."""
    _dev("Y", Y, torch.bfloat16)
    T, E, D = Y.shape
    gram = torch.empty((E, E), dtype=torch.float32, device=Y.device)
    cos = torch.empty((E, E), dtype=torch.float32, device=Y.device)
    ws = torch.empty(int(lib().bm_gram_workspace_bytes(E)), dtype=torch.uint8, device=Y.device)
    rc = lib().bm_cosine_gram(_ptr(Y), E, T, D, _ptr(gram), _ptr(cos), _ptr(ws), ws.numel(), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_cosine_gram")
    return gram, cos


def bm_group_mse(Y, U, w, group_map, stream=None):
    """(mse [G] f32, mse_total [1] f32) of Eq. 5-6 (include/bm.h: bm_group_mse).  Y [T,E,D], U [T,G,D] bf16, token-major."""
    _dev("Y", Y, torch.bfloat16)
    _dev("U", U, torch.bfloat16)
    T, E, D = Y.shape
    G = U.shape[1]
    mse = torch.empty(G, dtype=torch.float32, device=Y.device)
    tot = torch.empty(1, dtype=torch.float32, device=Y.device)
    ws = torch.empty(int(lib().bm_mse_workspace_bytes(G)), dtype=torch.uint8, device=Y.device)
    rc = lib().bm_group_mse(_ptr(Y), _ptr(U), T, D, _ptr(w), _ptr(group_map), E, G, _ptr(mse), _ptr(tot), _ptr(ws),
                            ws.numel(), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_group_mse")
    return mse, tot


def bm_moe_forward(x, routing: Routing, W1, W3, W2, out, workspace, S: int = 0, path: int = BM_PATH_AUTO,
                   stream=None):
    """Steps 9-13 (include/bm.h: bm_moe_forward / bm_moe_forward_path).  W1, W3 [G+S,F,D], W2 [G+S,D,F] bf16;
    out [T,D] bf16 is overwritten."""
    T, D, F = _check_forward_args(x, routing, W1, W3, W2, out, torch.bfloat16, workspace, S)
    rc = lib().bm_moe_forward_path(_ptr(x), T, D, ctypes.byref(routing.c), _ptr(W1), _ptr(W3), _ptr(W2), F, S,
                                   _ptr(out), _ptr(workspace), workspace.numel(), _stream(stream), path)
    if rc != BM_OK:
        raise BmError(rc, "bm_moe_forward")
    return out


def bm_moe_forward_f32(x, routing: Routing, W1, W3, W2, out_f32, workspace, S: int = 0, stream=None):
    """One rank's fp32 partial of a layer whose F dimension is sharded (include/bm.h: bm_moe_forward_f32)."""
    T, D, F = _check_forward_args(x, routing, W1, W3, W2, out_f32, torch.float32, workspace, S)
    rc = lib().bm_moe_forward_f32(_ptr(x), T, D, ctypes.byref(routing.c), _ptr(W1), _ptr(W3), _ptr(W2), F, S,
                                  _ptr(out_f32), _ptr(workspace), workspace.numel(), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_moe_forward_f32")
    return out_f32


def bm_round_bf16(src, out=None, stream=None):
    """bf16(fp32), round to nearest even (include/bm.h: bm_round_bf16)."""
    if out is None:
        out = torch.empty(src.shape, dtype=torch.bfloat16, device=src.device)
    rc = lib().bm_round_bf16(_ptr(src), src.numel(), _ptr(out), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_round_bf16")
    return out


class Salc:
    """SLO-aware latency controller (include/bm.h: bm_salc_*; host logic, no GPU)."""

    def __init__(self, slo, warn_frac=0.8, decrease=0.7, increase=0.05, window=32):
        self.c = BmSalc()
        rc = lib().bm_salc_init(ctypes.byref(self.c), slo, warn_frac, decrease, increase, window)
        if rc != BM_OK:
            raise BmError(rc, "bm_salc_init")

    def observe(self, latency) -> float:
        return lib().bm_salc_observe(ctypes.byref(self.c), float(latency))

    def p90(self) -> float:
        return lib().bm_salc_p90(ctypes.byref(self.c))

    @property
    def threshold(self) -> float:
        return self.c.threshold


def bm_salc_cold_mask(w, threshold):
    """cold_mask [E] int32 (host tensor) for bm_route_partial from routing frequencies w [E] (host int32)."""
    w = w.to(dtype=torch.int32, device="cpu").contiguous()
    mask = torch.zeros_like(w)
    rc = lib().bm_salc_cold_mask(w.data_ptr(), w.numel(), float(threshold), mask.data_ptr())
    if rc != BM_OK:
        raise BmError(rc, "bm_salc_cold_mask")
    return mask


def bm_moe_layer(x, W_router, router_bias, K: int, group_map, G: int, W1, W3, W2, out, routing: Routing, workspace,
                 S: int = 0, stream=None):
    """bm_route + bm_moe_forward as one call (include/bm.h: bm_moe_layer); single-token decode runs as one kernel."""
    T, D = x.shape
    E = W_router.shape[0]
    _check_route_args(x, W_router, router_bias, group_map, routing, workspace, T, D, E, K, G)
    _, _, F = _check_forward_args(x, routing, W1, W3, W2, out, torch.bfloat16, workspace, S)
    rc = lib().bm_moe_layer(_ptr(x), T, D, _ptr(W_router), _ptr(router_bias), E, K, _ptr(group_map), G, _ptr(W1), _ptr(W3),
                            _ptr(W2), F, S, _ptr(out), ctypes.byref(routing.c), _ptr(workspace), workspace.numel(), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_moe_layer")
    return out


def bm_moe_layer_host(x_host, W_router, router_bias, K, group_map, G, W1, W3, W2, S, out_host, x_dev, out_dev,
                      routing: Routing, workspace, stream=None):
    """Whole layer for a batch in (pinned) host memory; returns after the device->host copy has finished."""
    T, D = x_host.shape
    E = W_router.shape[0]
    F = W1.shape[1]
    rc = lib().bm_moe_layer_host(_ptr(x_host), T, D, _ptr(W_router), _ptr(router_bias), E, K, _ptr(group_map), G,
                                 _ptr(W1), _ptr(W3), _ptr(W2), F, S, _ptr(out_host), _ptr(x_dev), _ptr(out_dev),
                                 ctypes.byref(routing.c), _ptr(workspace), workspace.numel(), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_moe_layer_host")
    return out_host


def bm_device_status(workspace, stream=None) -> int:
    v = c_int32(0)
    rc = lib().bm_device_status(_ptr(workspace), ctypes.byref(v), _stream(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_device_status")
    return int(v.value)


def profile_enable(kernel: str | None, max_records: int = 0) -> None:
    """Record CUDA-event pairs around the launches of one kernel kind (KERNELS), None = off."""
    rc = lib().bm_profile_enable(0 if kernel is None else KERNELS[kernel], max_records)
    if rc != BM_OK:
        raise BmError(rc, "bm_profile_enable")


def profile_read():
    """(summed milliseconds, number of event pairs) since the last read; synchronises on the events."""
    ms, n = c_float(0), c_int(0)
    rc = lib().bm_profile_read(ctypes.byref(ms), ctypes.byref(n))
    if rc != BM_OK:
        raise BmError(rc, "bm_profile_read")
    return float(ms.value), int(n.value)


def profile_read_kinds():
    """{kind: (summed milliseconds, launches)} since the last read, for every kernel kind that was recorded."""
    n_kinds = KERNELS["all"]
    ms, n = (c_float * n_kinds)(), (c_int * n_kinds)()
    rc = lib().bm_profile_read_kinds(ms, n)
    if rc != BM_OK:
        raise BmError(rc, "bm_profile_read_kinds")
    return {name: (float(ms[k]), int(n[k])) for name, k in KERNELS.items() if k < n_kinds}
