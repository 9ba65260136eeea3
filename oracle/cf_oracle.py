"""ctypes wrapper of the CPU oracle (oracle/cf_oracle.cpp) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this. It marshals the neutral containers of paper_2512_14098_b200.workloads into the oracle's own
C structs; it imports nothing from the CUDA binding.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libcf_oracle.so")
_SRC = os.path.join(_HERE, "cf_oracle.cpp")
_SRC2 = os.path.join(_HERE, "cf_oracle_phases.cpp")
_HDR = os.path.join(_HERE, "cf_oracle.h")

ORC_OK, ORC_ERR_ARG, ORC_ERR_RANGE, ORC_ERR_PLAN, ORC_ERR_TABLE = 0, -1, -2, -3, -4


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O2 (plain, untuned)."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC2), os.path.getmtime(_HDR))
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < newest:
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-pthread", "-Wall", "-o", _SO, _SRC, _SRC2]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


class _QTab(C.Structure):
    _fields_ = [("levels", C.c_uint32), ("log2_cells", C.c_uint32), ("q", C.POINTER(C.c_int32))]


class _Graph(C.Structure):
    _fields_ = [("n_comp", C.c_uint32), ("n_types", C.c_uint32), ("n_req", C.c_uint32),
                ("n_trials", C.c_uint32), ("type_mask", C.POINTER(C.c_uint8)),
                ("type_thresh", C.POINTER(C.c_uint32)), ("svc_tab", C.POINTER(C.c_uint16)),
                ("tabs", C.POINTER(_QTab)), ("n_tabs", C.c_uint32), ("arr_tab", _QTab),
                ("edges", C.POINTER(C.c_uint8)), ("n_edges", C.c_uint32),
                ("edge_delay_us", C.c_int64), ("cpu_tab", C.POINTER(C.c_uint16)),
                ("join_mode", C.c_uint32), ("order_mode", C.c_uint32)]


class _Plans(C.Structure):
    _fields_ = [("n_plans", C.c_uint32), ("max_stages", C.c_uint32),
                ("n_stages", C.POINTER(C.c_uint8)), ("stage_mask", C.POINTER(C.c_uint8)),
                ("stage_c", C.POINTER(C.c_uint16)), ("max_routes", C.c_uint32),
                ("route_mask", C.POINTER(C.c_uint8)), ("route_cum", C.POINTER(C.c_uint32))]


class _Slo(C.Structure):
    _fields_ = [("L_us", C.POINTER(C.c_int64)), ("att_num", C.POINTER(C.c_uint32)),
                ("att_den", C.POINTER(C.c_uint32))]


def _ptr(a: Optional[np.ndarray], ctype):
    if a is None:
        return C.cast(None, C.POINTER(ctype))
    return a.ctypes.data_as(C.POINTER(ctype))


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        _lib.orc_qtab_sample.restype = C.c_int64
        _lib.orc_qtab_sample.argtypes = [C.POINTER(_QTab), C.c_uint32]
        _lib.orc_philox4x32_10.restype = None
        for name in ("orc_validate", "orc_eval_plans", "orc_goodput_bisect", "orc_trace_sim",
                     "orc_materialize_stream", "orc_flow_bound", "orc_mc_latency", "orc_pareto_select"):
            getattr(_lib, name).restype = C.c_int32
        _lib.orc_qtab_mean_q16.restype = C.c_uint64
    return _lib


class _Marshalled:
    """Keeps the numpy buffers alive for the duration of a call."""

    def __init__(self, graph, plans=None, slo=None):
        self.keep = []
        g = graph
        tabs = (_QTab * len(g.tabs))()
        for j, t in enumerate(g.tabs):
            tabs[j] = _QTab(t.levels, t.log2_cells, _ptr(t.q, C.c_int32))
        self.keep.append(tabs)
        edges = np.ascontiguousarray(g.edges, dtype=np.uint8).reshape(-1)
        self.keep.append(edges)
        self.g = _Graph(g.n_comp, g.n_types, g.n_req, g.n_trials, _ptr(g.type_mask, C.c_uint8),
                        _ptr(g.type_thresh, C.c_uint32), _ptr(g.svc_tab, C.c_uint16), tabs,
                        len(g.tabs), _QTab(g.arr_tab.levels, g.arr_tab.log2_cells,
                                           _ptr(g.arr_tab.q, C.c_int32)),
                        _ptr(edges if edges.size else None, C.c_uint8), edges.size // 2,
                        int(g.edge_delay_us), _ptr(getattr(g, "cpu_tab", None), C.c_uint16),
                        int(getattr(g, "join_mode", 0)), int(getattr(g, "order_mode", 0)))
        self.pl = None
        if plans is not None:
            sm = np.ascontiguousarray(plans.stage_mask).reshape(-1)
            sc = np.ascontiguousarray(plans.stage_c).reshape(-1)
            self.keep += [sm, sc]
            rm = getattr(plans, "route_mask", None)
            rc = getattr(plans, "route_cum", None)
            if rm is not None:
                rm = np.ascontiguousarray(rm, dtype=np.uint8).reshape(-1)
                rc = np.ascontiguousarray(rc, dtype=np.uint32).reshape(-1)
                self.keep += [rm, rc]
            self.pl = _Plans(plans.n_plans, plans.max_stages, _ptr(plans.n_stages, C.c_uint8),
                             _ptr(sm, C.c_uint8), _ptr(sc, C.c_uint16), int(getattr(plans, "max_routes", 0)),
                             _ptr(rm, C.c_uint8), _ptr(rc, C.c_uint32))
        self.slo = None
        if slo is not None:
            self.slo = _Slo(_ptr(slo.L_us, C.c_int64), _ptr(slo.att_num, C.c_uint32),
                            _ptr(slo.att_den, C.c_uint32))


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def qtab_sample(tab, u: int) -> int:
    t = _QTab(tab.levels, tab.log2_cells, _ptr(tab.q, C.c_int32))
    return int(lib().orc_qtab_sample(C.byref(t), C.c_uint32(int(u) & 0xFFFFFFFF)))


def validate(graph, plans) -> int:
    m = _Marshalled(graph, plans)
    return int(lib().orc_validate(C.byref(m.g), C.byref(m.pl)))


def eval_plans(graph, plans, rate_mrps, slo, seed: int, variant: int = 0, n_threads: int = 1,
               return_status: bool = False):
    """Returns dict(counts [P,R,K,T,2] u32, dep_sum [P,R,K] u64, makespan [P,R,K] i64,
    sim_status [P,R,K] i32, rc)."""
    m = _Marshalled(graph, plans, slo)
    rates = np.ascontiguousarray(rate_mrps, dtype=np.uint32).reshape(plans.n_plans, -1)
    P, R = rates.shape
    K, T = graph.n_trials, graph.n_types
    counts = np.zeros((P, R, K, T, 2), dtype=np.uint32)
    dep = np.zeros((P, R, K), dtype=np.uint64)
    mk = np.zeros((P, R, K), dtype=np.int64)
    st = np.zeros((P, R, K), dtype=np.int32)
    rc = lib().orc_eval_plans(C.byref(m.g), C.byref(m.pl), _ptr(rates, C.c_uint32), C.c_uint32(R),
                              C.byref(m.slo), C.c_uint64(seed), C.c_uint32(variant),
                              _ptr(counts, C.c_uint32), _ptr(dep, C.c_uint64), _ptr(mk, C.c_int64),
                              _ptr(st, C.c_int32), C.c_int32(n_threads))
    return dict(counts=counts, dep_sum=dep, makespan=mk, sim_status=st, rc=int(rc))


def goodput_bisect(graph, plans, rate_hi_mrps, n_steps: int, slo, seed: int, variant: int = 0,
                   n_threads: int = 1):
    m = _Marshalled(graph, plans, slo)
    hi = np.ascontiguousarray(rate_hi_mrps, dtype=np.uint32).reshape(-1)
    P, K, T = plans.n_plans, graph.n_trials, graph.n_types
    assert hi.size == P
    rate = np.zeros(P, dtype=np.uint32)
    good = np.zeros((P, T), dtype=np.uint32)
    counts = np.zeros((P, K, T, 2), dtype=np.uint32)
    rc = lib().orc_goodput_bisect(C.byref(m.g), C.byref(m.pl), _ptr(hi, C.c_uint32),
                                  C.c_uint32(n_steps), C.byref(m.slo), C.c_uint64(seed),
                                  C.c_uint32(variant), _ptr(rate, C.c_uint32),
                                  _ptr(good, C.c_uint32), _ptr(counts, C.c_uint32),
                                  C.c_int32(n_threads))
    return dict(rate_mrps=rate, goodput_mrps=good, counts=counts, rc=int(rc))


def trace_sim(graph, plans, plan: int, rate_mrps: int, trial: int, seed: int, variant: int = 0):
    m = _Marshalled(graph, plans)
    N = graph.n_req
    arr = np.zeros(N, dtype=np.int64)
    dep = np.zeros(N, dtype=np.int64)
    typ = np.zeros(N, dtype=np.uint8)
    rc = lib().orc_trace_sim(C.byref(m.g), C.byref(m.pl), C.c_uint32(plan), C.c_uint32(rate_mrps),
                             C.c_uint32(trial), C.c_uint64(seed), C.c_uint32(variant),
                             _ptr(arr, C.c_int64), _ptr(dep, C.c_int64), _ptr(typ, C.c_uint8))
    return dict(arrival=arr, departure=dep, type=typ, rc=int(rc))


STREAM_DTYPE = np.dtype([("head", "<u8"), ("svc", "<i4", (6,))])


def materialize_stream(graph, seed: int, variant_lo: int, n_variants: int):
    """Returns a structured array [n_variants, K, N] of 32-byte records."""
    m = _Marshalled(graph)
    out = np.zeros((n_variants, graph.n_trials, graph.n_req), dtype=STREAM_DTYPE)
    rc = lib().orc_materialize_stream(C.byref(m.g), C.c_uint64(seed), C.c_uint32(variant_lo),
                                      C.c_uint32(n_variants), out.ctypes.data_as(C.c_void_p))
    assert rc == 0, rc
    return out


# ---- the cheap phases around the simulation (cf_oracle_phases.cpp) ----------------------------------
def qtab_mean_q16(tab) -> int:
    t = _QTab(tab.levels, tab.log2_cells, _ptr(tab.q, C.c_int32))
    return int(lib().orc_qtab_mean_q16(C.byref(t)))


def flow_bound(graph, plans, alpha_num: int = 1, alpha_den: int = 1):
    """Returns dict(rate_mrps [P] u32, bound_mrps [P] u32, bottleneck [P] u8, redundant [P] u8, rc)."""
    m = _Marshalled(graph, plans)
    P = plans.n_plans
    rate = np.zeros(P, dtype=np.uint32)
    bound = np.zeros(P, dtype=np.uint32)
    bott = np.zeros(P, dtype=np.uint8)
    red = np.zeros(P, dtype=np.uint8)
    rc = lib().orc_flow_bound(C.byref(m.g), C.byref(m.pl), C.c_uint32(alpha_num), C.c_uint32(alpha_den),
                              _ptr(rate, C.c_uint32), _ptr(bound, C.c_uint32), _ptr(bott, C.c_uint8),
                              _ptr(red, C.c_uint8))
    return dict(rate_mrps=rate, bound_mrps=bound, bottleneck=bott, redundant=red, rc=int(rc))


def mc_latency(graph, plans, rate_mrps, slo, seed: int, variant: int = 0):
    """Returns dict(counts [P,K,T,2] u32, goodput_mrps [P,T] u32, rc)."""
    m = _Marshalled(graph, plans, slo)
    P, K, T = plans.n_plans, graph.n_trials, graph.n_types
    rates = np.ascontiguousarray(rate_mrps, dtype=np.uint32).reshape(-1)
    assert rates.size == P
    counts = np.zeros((P, K, T, 2), dtype=np.uint32)
    good = np.zeros((P, T), dtype=np.uint32)
    rc = lib().orc_mc_latency(C.byref(m.g), C.byref(m.pl), _ptr(rates, C.c_uint32), C.byref(m.slo),
                              C.c_uint64(seed), C.c_uint32(variant), _ptr(counts, C.c_uint32),
                              _ptr(good, C.c_uint32))
    return dict(counts=counts, goodput_mrps=good, rc=int(rc))


def pareto_select(goodput, alive=None):
    """goodput [P,T] u32; alive [P] u8 or None. Returns dict(pruned [P] u8, best, n_survivors, rc)."""
    gp = np.ascontiguousarray(goodput, dtype=np.uint32)
    P, T = gp.shape
    al = None if alive is None else np.ascontiguousarray(alive, dtype=np.uint8)
    pruned = np.zeros(P, dtype=np.uint8)
    best, ns = C.c_uint32(0), C.c_uint32(0)
    rc = lib().orc_pareto_select(_ptr(gp, C.c_uint32), C.c_uint32(P), C.c_uint32(T), _ptr(al, C.c_uint8),
                                 _ptr(pruned, C.c_uint8), C.byref(best), C.byref(ns))
    return dict(pruned=pruned, best=int(best.value), n_survivors=int(ns.value), rc=int(rc))
