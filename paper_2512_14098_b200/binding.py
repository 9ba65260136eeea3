"""Thin Python binding of libcf_b200.so (include/cf.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI. PyTorch is used for device
memory and streams, nothing else. There is no CPU fallback: if the shared library is missing the
import of this module raises, and without a CUDA device every compute call raises.
"""
from __future__ import annotations

import ctypes as C
import functools
import os
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcf_b200.so")

CF_OK, CF_ERR_ARG, CF_ERR_RANGE, CF_ERR_PLAN, CF_ERR_TABLE, CF_ERR_CUDA, CF_ERR_WORKSPACE = \
    0, -1, -2, -3, -4, -5, -6

# include/cf.h (the product ABI) and include/cf_debug.h (test / tuning / bench hooks)
EXPORTS = ["cf_workspace_bytes", "cf_eval_plans", "cf_goodput_bisect", "cf_stream_bytes",
           "cf_materialize_workspace_bytes", "cf_materialize_stream", "cf_eval_plans_stream",
           "cf_goodput_bisect_stream", "cf_trace_sim", "cf_workspace_status", "cf_strerror",
           "cf_workspace_wide_count", "cf_bisect_probes", "cf_aux_workspace_bytes",
           "cf_pareto_workspace_bytes", "cf_flow_bound", "cf_mc_latency", "cf_pareto_select", "cf_cache_clear",
           "cf_pareto_select_static", "cf_pareto_static_max_plans"]
DEBUG_EXPORTS = ["cf_eval_plans_opt", "cf_eval_plans_stream_opt", "cf_goodput_bisect_opt",
                 "cf_goodput_bisect_stream_opt", "cf_trace_sim_opt", "cf_last_launch_count",
                 "cf_bench_int32_peak"]
CF_KERNEL_AUTO, CF_KERNEL_WIDE64, CF_KERNEL_FAST32, CF_KERNEL_SCAN = 0, 1, 2, 3


class CfError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {strerror(status)} ({status})")


class cf_qtab(C.Structure):
    _fields_ = [("levels", C.c_uint32), ("log2_cells", C.c_uint32), ("q", C.POINTER(C.c_int32))]


class cf_graph(C.Structure):
    _fields_ = [("n_comp", C.c_uint32), ("n_types", C.c_uint32), ("n_req", C.c_uint32),
                ("n_trials", C.c_uint32), ("type_mask", C.POINTER(C.c_uint8)),
                ("type_thresh", C.POINTER(C.c_uint32)), ("svc_tab", C.POINTER(C.c_uint16)),
                ("tabs", C.POINTER(cf_qtab)), ("n_tabs", C.c_uint32), ("arr_tab", cf_qtab),
                ("edges", C.POINTER(C.c_uint8)), ("n_edges", C.c_uint32),
                ("edge_delay_us", C.c_int64), ("cpu_tab", C.POINTER(C.c_uint16)),
                ("join_mode", C.c_uint32), ("order_mode", C.c_uint32)]


class cf_plans(C.Structure):
    _fields_ = [("n_plans", C.c_uint32), ("max_stages", C.c_uint32),
                ("n_stages", C.POINTER(C.c_uint8)), ("stage_mask", C.POINTER(C.c_uint8)),
                ("stage_c", C.POINTER(C.c_uint16)), ("max_routes", C.c_uint32),
                ("route_mask", C.POINTER(C.c_uint8)), ("route_cum", C.POINTER(C.c_uint32))]


class cf_options(C.Structure):
    _fields_ = [("kernel_mode", C.c_uint32), ("bisect_depth", C.c_uint32), ("bisect_predict", C.c_uint32),
                ("reserved", C.c_uint32 * 5)]


class cf_slo(C.Structure):
    _fields_ = [("L_us", C.POINTER(C.c_int64)), ("att_num", C.POINTER(C.c_uint32)),
                ("att_den", C.POINTER(C.c_uint32))]


if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2512_14098_b200.build` "
                      "(there is no CPU fallback)")
_lib = C.CDLL(LIB_PATH)
_lib.cf_workspace_bytes.restype = C.c_size_t
_lib.cf_stream_bytes.restype = C.c_size_t
_lib.cf_materialize_workspace_bytes.restype = C.c_size_t
_lib.cf_strerror.restype = C.c_char_p
_lib.cf_last_launch_count.restype = C.c_uint32
_lib.cf_workspace_wide_count.restype = C.c_int64
_lib.cf_bisect_probes.restype = C.c_int32
_lib.cf_aux_workspace_bytes.restype = C.c_size_t
_lib.cf_pareto_workspace_bytes.restype = C.c_size_t
for _n in ("cf_flow_bound", "cf_mc_latency", "cf_pareto_select", "cf_pareto_select_static"):
    getattr(_lib, _n).restype = C.c_int32
_lib.cf_pareto_static_max_plans.restype = C.c_uint32
for _n in ("cf_eval_plans", "cf_goodput_bisect", "cf_materialize_stream", "cf_eval_plans_stream",
           "cf_goodput_bisect_stream", "cf_trace_sim", "cf_workspace_status", "cf_bench_int32_peak",
           "cf_eval_plans_opt", "cf_eval_plans_stream_opt", "cf_goodput_bisect_opt",
           "cf_goodput_bisect_stream_opt", "cf_trace_sim_opt"):
    getattr(_lib, _n).restype = C.c_int32

# Test / tuning options (include/cf_debug.h). The library itself has no knobs: this module-level
# record belongs to the Python binding; while it holds defaults, calls go through the product entry
# points of cf.h, otherwise through their *_opt twins with the record as the per-call argument.
_OPT = cf_options()


def _opt_active() -> bool:
    return bool(_OPT.kernel_mode or _OPT.bisect_depth or _OPT.bisect_predict)


_lib.cf_cache_clear.restype = None


def cf_cache_clear() -> None:
    _lib.cf_cache_clear()


def strerror(status: int) -> str:
    return _lib.cf_strerror(C.c_int32(status)).decode()


def _hp(a: Optional[np.ndarray], ctype):
    if a is None:
        return C.cast(None, C.POINTER(ctype))
    return a.ctypes.data_as(C.POINTER(ctype))


def _dp(t: Optional[torch.Tensor]):
    if t is None:
        return C.c_void_p(0)
    assert t.is_cuda and t.is_contiguous()
    return C.c_void_p(t.data_ptr())


def _stream_ptr(stream: Optional[torch.cuda.Stream]):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


class Marshalled:
    """Host structs of a (graph, plans, slo) triple; keeps the numpy buffers alive."""

    def __init__(self, graph, plans=None, slo=None):
        self.keep = []
        g = graph
        tabs = (cf_qtab * len(g.tabs))()
        for j, t in enumerate(g.tabs):
            tabs[j] = cf_qtab(t.levels, t.log2_cells, _hp(t.q, C.c_int32))
        edges = np.ascontiguousarray(g.edges, dtype=np.uint8).reshape(-1)
        self.keep += [tabs, edges]
        self.g = cf_graph(g.n_comp, g.n_types, g.n_req, g.n_trials, _hp(g.type_mask, C.c_uint8),
                          _hp(g.type_thresh, C.c_uint32), _hp(g.svc_tab, C.c_uint16), tabs,
                          len(g.tabs), cf_qtab(g.arr_tab.levels, g.arr_tab.log2_cells,
                                               _hp(g.arr_tab.q, C.c_int32)),
                          _hp(edges if edges.size else None, C.c_uint8), edges.size // 2,
                          int(g.edge_delay_us), _hp(getattr(g, "cpu_tab", None), C.c_uint16),
                          int(getattr(g, "join_mode", 0)), int(getattr(g, "order_mode", 0)))
        self.pl = None
        if plans is not None:
            sm = np.ascontiguousarray(plans.stage_mask).reshape(-1)
            sc = np.ascontiguousarray(plans.stage_c).reshape(-1)
            self.keep += [sm, sc]
            rm = getattr(plans, "route_mask", None)
            rcum = getattr(plans, "route_cum", None)
            if rm is not None:
                rm = np.ascontiguousarray(rm, dtype=np.uint8).reshape(-1)
                rcum = np.ascontiguousarray(rcum, dtype=np.uint32).reshape(-1)
                self.keep += [rm, rcum]
            self.pl = cf_plans(plans.n_plans, plans.max_stages, _hp(plans.n_stages, C.c_uint8),
                               _hp(sm, C.c_uint8), _hp(sc, C.c_uint16), int(getattr(plans, "max_routes", 0)),
                               _hp(rm, C.c_uint8), _hp(rcum, C.c_uint32))
        self.slo = None
        if slo is not None:
            self.slo = cf_slo(_hp(slo.L_us, C.c_int64), _hp(slo.att_num, C.c_uint32),
                              _hp(slo.att_den, C.c_uint32))


def _on_stream(fn):
    """Runs the wrapped call with `stream` (keyword) as torch's current stream: the temporaries the
    binding makes (rate arrays copied to the device, outputs, workspaces) are then allocated and
    filled on the stream the library launches on, so there is no cross-stream race and the caching
    allocator cannot hand them out again while the kernels still use them."""
    @functools.wraps(fn)
    def wrapped(*args, **kw):
        stream = kw.get("stream")
        if stream is None or not torch.cuda.is_available():
            return fn(*args, **kw)
        with torch.cuda.stream(stream):
            return fn(*args, **kw)
    return wrapped


def _require_cuda():
    if not torch.cuda.is_available():
        raise RuntimeError("libcf_b200 needs a CUDA device (no CPU fallback)")


def cf_workspace_bytes(graph, plans, R: int) -> int:
    m = Marshalled(graph, plans)
    return int(_lib.cf_workspace_bytes(C.byref(m.g), C.byref(m.pl), C.c_uint32(R)))


def alloc_workspace(graph, plans, R: int, device="cuda") -> torch.Tensor:
    return torch.empty(cf_workspace_bytes(graph, plans, R), dtype=torch.uint8, device=device)


def _as_dev_u32(x, device) -> torch.Tensor:
    """uint32 values as an int32-typed CUDA tensor (bit pattern preserved)."""
    if isinstance(x, torch.Tensor):
        assert x.dtype in (torch.int32, torch.uint32)
        return x.contiguous().to(device)
    a = np.ascontiguousarray(x, dtype=np.uint32)
    return torch.from_numpy(a.view(np.int32)).to(device)


def cf_workspace_status(workspace: torch.Tensor, stream=None) -> int:
    return int(_lib.cf_workspace_status(_dp(workspace), _stream_ptr(stream)))


def cf_workspace_wide_count(workspace: torch.Tensor, stream=None) -> int:
    """Simulations of the last call on `workspace` that the 64-bit kernel had to redo."""
    return int(_lib.cf_workspace_wide_count(_dp(workspace), _stream_ptr(stream)))


def cf_debug_kernel_mode(mode: int) -> None:
    """Kernel choice of later calls made through this binding (cf_debug.h CF_KERNEL_*): 0 = automatic
    (32-bit fast kernel + 64-bit fixup, or the scan kernel), 1 = 64-bit kernel only, 2 = fast kernel
    (never the scan kernel; traces run on it), 3 = max-plus scan kernel."""
    if not 0 <= mode <= 3:
        raise CfError(CF_ERR_ARG, "cf_debug_kernel_mode")
    _OPT.kernel_mode = mode


def cf_bisect_probes(workspace: torch.Tensor, n_plans: int, stream=None) -> np.ndarray:
    """Probes on the bisection path of each plan in the last cf_goodput_bisect call on `workspace`."""
    out = np.zeros(n_plans, dtype=np.uint32)
    rc = int(_lib.cf_bisect_probes(_dp(workspace), C.c_uint32(n_plans), _hp(out, C.c_uint32), _stream_ptr(stream)))
    if rc != CF_OK:
        raise CfError(rc, "cf_bisect_probes")
    return out


def cf_debug_bisect_depth(depth: int) -> None:
    """Bisection steps simulated per pass by later calls: 0 = automatic, 1..4 = fixed (tests, tuning)."""
    if not 0 <= depth <= 4:
        raise CfError(CF_ERR_ARG, "cf_debug_bisect_depth")
    _OPT.bisect_depth = depth


def cf_debug_bisect_predict(mode: int) -> None:
    """0 = default, 1 = always the full decision tree, 2 = always node + predicted child (cf_debug.h)."""
    if not 0 <= mode <= 2:
        raise CfError(CF_ERR_ARG, "cf_debug_bisect_predict")
    _OPT.bisect_predict = mode


def cf_last_launch_count() -> int:
    return int(_lib.cf_last_launch_count())


@_on_stream
def cf_eval_plans(graph, plans, rate_mrps, slo, seed: int, variant: int = 0, *, out_counts=None,
                  out_dep_sum=None, out_makespan=None, workspace=None, stream=None, aux=True,
                  stream_records=None, n_variants: int = 1, plan_variant=None, check=True):
    """cf_eval_plans / cf_eval_plans_stream (if stream_records is given). rate_mrps: [P,R] CUDA int32
    tensor (uint32 bit pattern) or anything numpy can convert. Returns dict of CUDA tensors:
    counts int32 [P,R,K,T,2], dep_sum int64 [P,R,K] (uint64 bit pattern), makespan int64 [P,R,K]."""
    _require_cuda()
    dev = torch.device("cuda")
    m = Marshalled(graph, plans, slo)
    rates = _as_dev_u32(rate_mrps, dev).reshape(plans.n_plans, -1)
    P, R = rates.shape
    K, T = graph.n_trials, graph.n_types
    if out_counts is None:
        out_counts = torch.empty((P, R, K, T, 2), dtype=torch.int32, device=dev)
    if aux and out_dep_sum is None:
        out_dep_sum = torch.empty((P, R, K), dtype=torch.int64, device=dev)
    if aux and out_makespan is None:
        out_makespan = torch.empty((P, R, K), dtype=torch.int64, device=dev)
    if workspace is None:
        workspace = alloc_workspace(graph, plans, R)
    opt = (C.byref(_OPT),) if _opt_active() else ()
    if stream_records is None:
        fn = _lib.cf_eval_plans_opt if opt else _lib.cf_eval_plans
        rc = fn(*opt, C.byref(m.g), C.byref(m.pl), _dp(rates), C.c_uint32(R), C.byref(m.slo),
                C.c_uint64(seed), C.c_uint32(variant), _dp(out_counts), _dp(out_dep_sum),
                _dp(out_makespan), _dp(workspace), C.c_size_t(workspace.numel()), _stream_ptr(stream))
    else:
        pv = None if plan_variant is None else np.ascontiguousarray(plan_variant, dtype=np.uint32)
        fn = _lib.cf_eval_plans_stream_opt if opt else _lib.cf_eval_plans_stream
        rc = fn(*opt, C.byref(m.g), C.byref(m.pl), _dp(rates), C.c_uint32(R), C.byref(m.slo),
                _dp(stream_records), C.c_uint32(n_variants), _hp(pv, C.c_uint32), _dp(out_counts),
                _dp(out_dep_sum), _dp(out_makespan), _dp(workspace), C.c_size_t(workspace.numel()),
                _stream_ptr(stream))
    if check and rc != CF_OK:
        raise CfError(rc, "cf_eval_plans")
    return dict(counts=out_counts, dep_sum=out_dep_sum, makespan=out_makespan, workspace=workspace,
                rc=int(rc))


@_on_stream
def cf_goodput_bisect(graph, plans, rate_hi_mrps, n_steps: int, slo, seed: int, variant: int = 0, *,
                      workspace=None, stream=None, stream_records=None, n_variants: int = 1,
                      plan_variant=None, want_counts=True, check=True):
    """cf_goodput_bisect / cf_goodput_bisect_stream. Returns dict of CUDA tensors: rate_mrps int32 [P],
    goodput_mrps int32 [P,T], counts int32 [P,K,T,2]."""
    _require_cuda()
    dev = torch.device("cuda")
    m = Marshalled(graph, plans, slo)
    hi = _as_dev_u32(rate_hi_mrps, dev).reshape(-1)
    P, K, T = plans.n_plans, graph.n_trials, graph.n_types
    assert hi.numel() == P
    rate = torch.empty(P, dtype=torch.int32, device=dev)
    good = torch.empty((P, T), dtype=torch.int32, device=dev)
    counts = torch.empty((P, K, T, 2), dtype=torch.int32, device=dev) if want_counts else None
    if workspace is None:
        workspace = alloc_workspace(graph, plans, 1)
    opt = (C.byref(_OPT),) if _opt_active() else ()
    if stream_records is None:
        fn = _lib.cf_goodput_bisect_opt if opt else _lib.cf_goodput_bisect
        rc = fn(*opt, C.byref(m.g), C.byref(m.pl), _dp(hi), C.c_uint32(n_steps), C.byref(m.slo),
                C.c_uint64(seed), C.c_uint32(variant), _dp(rate), _dp(good), _dp(counts), _dp(workspace),
                C.c_size_t(workspace.numel()), _stream_ptr(stream))
    else:
        pv = None if plan_variant is None else np.ascontiguousarray(plan_variant, dtype=np.uint32)
        fn = _lib.cf_goodput_bisect_stream_opt if opt else _lib.cf_goodput_bisect_stream
        rc = fn(*opt, C.byref(m.g), C.byref(m.pl), _dp(hi), C.c_uint32(n_steps), C.byref(m.slo),
                _dp(stream_records), C.c_uint32(n_variants), _hp(pv, C.c_uint32), _dp(rate), _dp(good),
                _dp(counts), _dp(workspace), C.c_size_t(workspace.numel()), _stream_ptr(stream))
    if check and rc != CF_OK:
        raise CfError(rc, "cf_goodput_bisect")
    return dict(rate_mrps=rate, goodput_mrps=good, counts=counts, workspace=workspace, rc=int(rc))


def cf_stream_bytes(graph, n_variants: int) -> int:
    m = Marshalled(graph)
    return int(_lib.cf_stream_bytes(C.byref(m.g), C.c_uint32(n_variants)))


@_on_stream
def cf_materialize_stream(graph, seed: int, variant_lo: int, n_variants: int, *, out=None,
                          stream=None, check=True):
    """Returns a CUDA uint8 tensor [n_variants, K, N, 32] of stream records."""
    _require_cuda()
    m = Marshalled(graph)
    if out is None:
        out = torch.empty((n_variants, graph.n_trials, graph.n_req, 32), dtype=torch.uint8, device="cuda")
    wsb = int(_lib.cf_materialize_workspace_bytes(C.byref(m.g), C.c_uint32(n_variants)))
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda")
    rc = _lib.cf_materialize_stream(C.byref(m.g), C.c_uint64(seed), C.c_uint32(variant_lo),
                                    C.c_uint32(n_variants), _dp(out), _dp(ws), C.c_size_t(wsb),
                                    _stream_ptr(stream))
    if check and rc != CF_OK:
        raise CfError(rc, "cf_materialize_stream")
    torch.cuda.current_stream().synchronize() if stream is None else stream.synchronize()  # ws lifetime
    return out


@_on_stream
def cf_trace_sim(graph, plans, plan: int, rate_mrps: int, trial: int, seed: int, variant: int = 0, *,
                 stream=None, check=True):
    _require_cuda()
    m = Marshalled(graph, plans)
    N = graph.n_req
    arr = torch.empty(N, dtype=torch.int64, device="cuda")
    dep = torch.empty(N, dtype=torch.int64, device="cuda")
    typ = torch.empty(N, dtype=torch.uint8, device="cuda")
    ws = alloc_workspace(graph, plans, 1)
    opt = (C.byref(_OPT),) if _opt_active() else ()
    fn = _lib.cf_trace_sim_opt if opt else _lib.cf_trace_sim
    rc = fn(*opt, C.byref(m.g), C.byref(m.pl), C.c_uint32(plan), C.c_uint32(rate_mrps),
            C.c_uint32(trial), C.c_uint64(seed), C.c_uint32(variant), _dp(arr), _dp(dep),
            _dp(typ), _dp(ws), C.c_size_t(ws.numel()), _stream_ptr(stream))
    if check and rc != CF_OK:
        raise CfError(rc, "cf_trace_sim")
    status = cf_workspace_status(ws, stream)
    wide = cf_workspace_wide_count(ws, stream) if rc == CF_OK else -1
    return dict(arrival=arr, departure=dep, type=typ, rc=int(rc), status=status, wide=wide)


def _aux_workspace(m, stream_dev="cuda") -> torch.Tensor:
    n = int(_lib.cf_aux_workspace_bytes(C.byref(m.g), C.byref(m.pl) if m.pl is not None else None))
    return torch.empty(n, dtype=torch.uint8, device=stream_dev)


@_on_stream
def cf_flow_bound(graph, plans, alpha_num: int = 1, alpha_den: int = 1, *, stream=None, check=True):
    """Phase 1 on the device. Returns dict of CUDA tensors: rate_mrps int32 [P] (alpha R_d),
    bound_mrps int32 [P] (R_d), bottleneck uint8 [P], redundant uint8 [P]."""
    _require_cuda()
    m = Marshalled(graph, plans)
    P = plans.n_plans
    rate = torch.empty(P, dtype=torch.int32, device="cuda")
    bound = torch.empty(P, dtype=torch.int32, device="cuda")
    bott = torch.empty(P, dtype=torch.uint8, device="cuda")
    red = torch.empty(P, dtype=torch.uint8, device="cuda")
    ws = _aux_workspace(m)
    rc = _lib.cf_flow_bound(C.byref(m.g), C.byref(m.pl), C.c_uint32(alpha_num), C.c_uint32(alpha_den), _dp(rate),
                            _dp(bound), _dp(bott), _dp(red), _dp(ws), C.c_size_t(ws.numel()), _stream_ptr(stream))
    if check and rc != CF_OK:
        raise CfError(rc, "cf_flow_bound")
    return dict(rate_mrps=rate, bound_mrps=bound, bottleneck=bott, redundant=red, workspace=ws, rc=int(rc))


@_on_stream
def cf_mc_latency(graph, plans, rate_mrps, slo, seed: int, variant: int = 0, *, want_counts=True, stream=None,
                  check=True):
    """Phase 2 on the device. rate_mrps: [P] CUDA int32 tensor or array-like. Returns dict of CUDA
    tensors: counts int32 [P,K,T,2] (or None), goodput_mrps int32 [P,T]."""
    _require_cuda()
    m = Marshalled(graph, plans, slo)
    P, K, T = plans.n_plans, graph.n_trials, graph.n_types
    rates = _as_dev_u32(rate_mrps, torch.device("cuda")).reshape(-1)
    assert rates.numel() == P
    counts = torch.empty((P, K, T, 2), dtype=torch.int32, device="cuda") if want_counts else None
    good = torch.empty((P, T), dtype=torch.int32, device="cuda")
    ws = _aux_workspace(m)
    rc = _lib.cf_mc_latency(C.byref(m.g), C.byref(m.pl), _dp(rates), C.byref(m.slo), C.c_uint64(seed),
                            C.c_uint32(variant), _dp(counts), _dp(good), _dp(ws), C.c_size_t(ws.numel()),
                            _stream_ptr(stream))
    if check and rc != CF_OK:
        raise CfError(rc, "cf_mc_latency")
    return dict(counts=counts, goodput_mrps=good, workspace=ws, rc=int(rc))


@_on_stream
def cf_pareto_select(goodput_mrps, alive=None, *, stream=None, check=True):
    """Pruning + policy on the device. goodput_mrps: [P,T] CUDA int32 tensor or array-like; alive: [P]
    CUDA uint8 tensor, array-like or None. Returns dict of CUDA tensors: pruned uint8 [P], best int32
    [1] (uint32 bit pattern), n_survivors int32 [1]."""
    _require_cuda()
    dev = torch.device("cuda")
    gp = goodput_mrps if isinstance(goodput_mrps, torch.Tensor) else \
        torch.from_numpy(np.ascontiguousarray(goodput_mrps, dtype=np.uint32).view(np.int32)).to(dev)
    gp = gp.contiguous()
    P, T = gp.shape
    al = None
    if alive is not None:
        al = alive if isinstance(alive, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(alive, dtype=np.uint8)).to(dev)
        al = al.contiguous()
    pruned = torch.empty(P, dtype=torch.uint8, device=dev)
    best = torch.empty(1, dtype=torch.int32, device=dev)
    ns = torch.empty(1, dtype=torch.int32, device=dev)
    ws = torch.empty(int(_lib.cf_pareto_workspace_bytes()), dtype=torch.uint8, device=dev)
    rc = _lib.cf_pareto_select(_dp(gp), C.c_uint32(P), C.c_uint32(T), _dp(al), _dp(pruned), _dp(best), _dp(ns),
                               _dp(ws), C.c_size_t(ws.numel()), _stream_ptr(stream))
    if check and rc != CF_OK:
        raise CfError(rc, "cf_pareto_select")
    return dict(pruned=pruned, best=best, n_survivors=ns, workspace=ws, rc=int(rc))


def cf_bench_int32_peak(mix: int, iters: int = 2000, stream=None):
    """Returns (lane_ops, microseconds) of the integer-issue micro-benchmark."""
    _require_cuda()
    ops, usec = C.c_uint64(0), C.c_uint64(0)
    rc = _lib.cf_bench_int32_peak(C.c_uint32(mix), C.c_uint32(iters), C.byref(ops), C.byref(usec),
                                  _stream_ptr(stream))
    if rc != CF_OK:
        raise CfError(rc, "cf_bench_int32_peak")
    return int(ops.value), int(usec.value)


def to_numpy_u32(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().numpy().view(np.uint32)


def to_numpy_u64(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().numpy().view(np.uint64)


def cf_pareto_static_max_plans() -> int:
    return int(_lib.cf_pareto_static_max_plans())


@_on_stream
def cf_pareto_select_static(goodput_mrps, alive, pruned, best, n_survivors, *, stream=None, check=True):
    """cf_pareto_select without a workspace (scratch = a fixed array inside the library; at most
    cf_pareto_static_max_plans() plans). Allocates nothing: every argument is a CUDA tensor the caller
    made beforehand (goodput_mrps int32 [P,T] contiguous, alive uint8 [P] or None, outputs pruned uint8
    [P], best int32 [1] or None, n_survivors int32 [1] or None). Returns the status code."""
    _require_cuda()
    P, T = goodput_mrps.shape
    rc = int(_lib.cf_pareto_select_static(_dp(goodput_mrps), C.c_uint32(P), C.c_uint32(T), _dp(alive), _dp(pruned),
                                          _dp(best), _dp(n_survivors), _stream_ptr(stream)))
    if check and rc != CF_OK:
        raise CfError(rc, "cf_pareto_select_static")
    return rc
