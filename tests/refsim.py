"""Independent pure-Python checkers used to PIN the oracle (tiny inputs only).

Nothing here is shared with oracle/ or with the CUDA path: the Philox generator and the table
sampler are restated from their definitions (Salmon et al. SC'11; R3), and the queueing
checkers are *different algorithms* from the oracle's recursion:
  - lindley_bruteforce: O(n^2) closed form D_n = max_{i<=n}(A_i + sum_{j=i..n} S_j)
  - tandem_last_passage: max over monotone paths (last-passage percolation) for c=1 tandems
  - event_sim: a discrete-event simulator with an explicit event heap, explicit per-server busy
    state and per-stage ticket queues (index-order service, R2)
"""
from __future__ import annotations

import heapq
from typing import List

M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
MASK = 0xFFFFFFFF


def philox4x32_10(ctr, key):
    c0, c1, c2, c3 = [int(x) & MASK for x in ctr]
    k0, k1 = [int(x) & MASK for x in key]
    for _ in range(10):
        p0 = M0 * c0
        p1 = M1 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & MASK, p1 & MASK, ((p0 >> 32) ^ c3 ^ k1) & MASK, p0 & MASK
        k0 = (k0 + W0) & MASK
        k1 = (k1 + W1) & MASK
    return [c0, c1, c2, c3]


def qtab_sample(levels: int, log2_cells: int, q, u: int) -> int:
    """Written from the table's *geometric* definition rather than from the bit recipe: find the
    level from the binary expansion of u/2^32, then the position inside the level as an exact
    rational, then floor the linear interpolation."""
    u &= MASK
    L, B = levels, log2_cells
    # level k: u/2^32 in [1-2^-k, 1-2^-(k+1)) for k<L-1, cap level [1-2^-(L-1), 1)
    k = 0
    while k < L - 1 and u >= (1 << 32) - (1 << (31 - k)):
        k += 1
    left = (1 << 32) - (1 << (32 - k)) if k > 0 else 0   # left edge of level k, as a 32-bit integer
    width_bits = (31 - k) if k < L - 1 else (32 - (L - 1))  # level width = 2^width_bits
    pos = u - left                                           # in [0, 2^width_bits)
    # position scaled to B+16 bits (cell index . 16-bit fraction); bits below are truncated
    if width_bits >= B + 16:
        scaled = pos >> (width_bits - B - 16)
    else:
        scaled = pos << (B + 16 - width_bits)
    m, f = scaled >> 16, scaled & 0xFFFF
    i = (k << B) + m
    return int(q[i]) + (((int(q[i + 1]) - int(q[i])) * f) >> 16)


def gen_requests(graph, seed: int, variant: int, trial: int, rate_mrps: int):
    """Per-request inputs of one trial: system arrivals A, types, per-component services (list of
    dicts), following DESIGN.md "Algorithm" (draw layout, R4, R5)."""
    key = (seed & MASK, (seed >> 32) & MASK)
    period = (10**9 + rate_mrps // 2) // rate_mrps
    C, T = graph.n_comp, graph.n_types
    cu = 0
    A, types, svc = [], [], []
    for n in range(graph.n_req):
        b0 = philox4x32_10((n, trial, 0, variant), key)
        at = graph.arr_tab
        cu += qtab_sample(at.levels, at.log2_cells, at.q, b0[0])
        A.append((cu * period + 32768) >> 16)
        t = T - 1
        for tt in range(T):
            if b0[1] < int(graph.type_thresh[tt]):
                t = tt
                break
        types.append(t)
        s = {}
        for i in range(C):
            if (int(graph.type_mask[t]) >> i) & 1:
                b = philox4x32_10((n, trial, 1 + i // 4, variant), key)
                tb = graph.tabs[int(graph.svc_tab[i * T + t])]
                s[i] = qtab_sample(tb.levels, tb.log2_cells, tb.q, b[i % 4])
        svc.append(s)
    return A, types, svc


def stage_services(graph, plans, p: int, types, svc):
    """For plan p: per request the ordered list of (stage, S) it visits (R6: one visit per stage,
    service = sum of the request's component services colocated there)."""
    out = []
    for n, t in enumerate(types):
        tm = int(graph.type_mask[t])
        route = []
        for s in range(int(plans.n_stages[p])):
            m = int(plans.stage_mask[p, s]) & tm
            if m:
                route.append((s, sum(svc[n][i] for i in range(graph.n_comp) if (m >> i) & 1)))
        out.append(route)
    return out


def lindley_bruteforce(A: List[int], S: List[int]) -> List[int]:
    return [max(A[i] + sum(S[i:n + 1]) for i in range(n + 1)) for n in range(len(A))]


def tandem_last_passage(A: List[int], S: List[List[int]]) -> List[int]:
    """All c=1, every request visits every stage, no edge delay: D^V_n = max over
    0<=i_1<=...<=i_V<=n of A_{i_1} + sum_s sum_{j=i_s..i_{s+1}} S[s][j] (i_{V+1}=n). Evaluated by
    explicit enumeration of the monotone index paths."""
    V = len(S)
    n_req = len(A)

    def best(stage: int, start: int, n: int) -> int:
        # max over i_{stage+1..V} given i_stage = start
        if stage == V - 1:
            return sum(S[stage][start:n + 1])
        return max(sum(S[stage][start:nxt + 1]) + best(stage + 1, nxt, n) for nxt in range(start, n + 1))

    return [max(A[i] + best(0, i, n) for i in range(n + 1)) for n in range(n_req)]


def event_sim(A: List[int], routes, stage_c: List[int], edge_delay: int = 0) -> List[int]:
    """Discrete-event simulation with an event heap. Each stage has c servers with explicit busy
    flags and a ticket queue: it serves its visiting requests in request-index order (R2), a server
    starting the next ticket as soon as that request has arrived at the stage and a server is idle.
    Returns the final departure of every request (A_n for an empty route, R14)."""
    n_req = len(A)
    V = len(stage_c)
    tickets = [[n for n in range(n_req) if any(s == st for st, _ in routes[n])] for s in range(V)]
    nxt = [0] * V
    idle = [stage_c[s] for s in range(V)]
    arrived = [dict() for _ in range(V)]
    hop = [0] * n_req
    done = [None] * n_req
    ev = []
    seq = 0
    for n in range(n_req):
        if routes[n]:
            heapq.heappush(ev, (A[n], seq, 0, n)); seq += 1  # kind 0: arrival at routes[n][hop]
        else:
            done[n] = A[n]

    def dispatch(s, now):
        nonlocal seq
        while nxt[s] < len(tickets[s]) and idle[s] > 0:
            n = tickets[s][nxt[s]]
            if n not in arrived[s]:
                break
            service = routes[n][hop[n]][1]
            idle[s] -= 1
            nxt[s] += 1
            heapq.heappush(ev, (now + service, seq, 1, n)); seq += 1  # kind 1: service completion

    while ev:
        now, _, kind, n = heapq.heappop(ev)
        s = routes[n][hop[n]][0]
        if kind == 0:
            arrived[s][n] = now
            dispatch(s, now)
        else:
            idle[s] += 1
            hop[n] += 1
            if hop[n] == len(routes[n]):
                done[n] = now
            else:
                heapq.heappush(ev, (now + edge_delay, seq, 0, n)); seq += 1
            dispatch(s, now)
    return done


def per_server_sim(A: List[int], routes, stage_c: List[int], edge_delay: int = 0) -> List[int]:
    """Explicit per-server state, no sorting: every stage keeps an UNSORTED list busy_until[j];
    requests are bound in index order to the server with the smallest busy_until (argmin scan).
    Same semantics as the oracle's sorted-vector recursion (R2/R13) through a different data
    structure; used where a causal event simulation does not coincide with the recursion."""
    busy = [[0] * c for c in stage_c]
    out = []
    for n, a in enumerate(A):
        x = a
        for hop, (s, service) in enumerate(routes[n]):
            if hop > 0:
                x += edge_delay
            j = min(range(len(busy[s])), key=lambda jj: busy[s][jj])
            x = max(x, busy[s][j]) + service
            busy[s][j] = x
        out.append(x)
    return out


def erlang_c(c: int, a: float) -> float:
    """Erlang-C probability of waiting, offered load a = lambda/mu < c."""
    term, s = 1.0, 1.0
    for k in range(1, c):
        term *= a / k
        s += term
    last = term * a / c / (1.0 - a / c)
    return last / (s + last)


def fcfs_event_sim(A: List[int], routes, stage_c: List[int], edge_delay: int = 0) -> List[int]:
    """Textbook FCFS at every stage: a stage serves its visitors in the order in which they REACH
    the stage (ties by request index), on the server that frees first. This is the discipline
    index-order service (R2) departs from when stage arrivals are not monotone in the
    request index: it measures that gap, and it pins the oracle's arrival-order mode (DESIGN.md
    R27), which reaches the same result stage by stage with a sort instead of an event queue.
    A hop may carry a third entry, the CPU pre-processing time paid only when the request finds
    a server idle on arrival (R24)."""
    n_stage = len(stage_c)
    free = [[0] * c for c in stage_c]
    queue = [[] for _ in range(n_stage)]          # heap of (arrival at the stage, request)
    pos = [0] * len(A)
    dep = [None] * len(A)
    ev = []                                        # (time, kind, request/stage): 0 = arrival, 1 = a server frees
    for n in range(len(A)):
        if routes[n]:
            heapq.heappush(ev, (A[n], 0, n))
        else:
            dep[n] = A[n]

    def dispatch(st, now):
        while queue[st]:
            k = min(range(stage_c[st]), key=lambda j: free[st][j])
            if free[st][k] > now:
                break
            at, r = heapq.heappop(queue[st])
            hop = routes[r][pos[r]]
            if free[st][k] <= at:                    # idle on arrival: CPU + GPU time
                done = at + (hop[2] if len(hop) > 2 else 0) + hop[1]
            else:                                    # the request queued: GPU time alone
                done = free[st][k] + hop[1]
            free[st][k] = done
            heapq.heappush(ev, (done, 1, st))
            pos[r] += 1
            if pos[r] == len(routes[r]):
                dep[r] = done
            else:
                heapq.heappush(ev, (done + edge_delay, 0, r))

    while ev:
        now, kind, x = heapq.heappop(ev)
        if kind == 0:
            st = routes[x][pos[x]][0]
            heapq.heappush(queue[st], (now, x))
            dispatch(st, now)
        else:
            dispatch(x, now)
    return dep
