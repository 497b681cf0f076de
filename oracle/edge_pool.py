"""Runs the UNCHANGED oracle (oracle/sim3_gn_oracle.py) edge-parallel on the host cores.

TEST INFRASTRUCTURE ONLY (same rule as sim3_gn_oracle.py): imported by ``tests/`` and by ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs, never by the product path.

No arithmetic of the method lives here.  The normal-equation assembly of PAPER.md:118 is a sum over edges, and every
edge touches only the two diagonal and one off-diagonal 7x7 blocks of its endpoints; a worker process therefore calls
``sim3_gn_oracle.build_system(..., edge_subset=[e])`` -- the oracle as it stands, one edge at a time -- and hands back
that edge's 14 x 14 corner of the returned H (rows/columns of keyframes i and j), its 14 entries of g and g_abs and the
per-edge outputs.  The parent adds the corners into the 7N system in ascending edge order, which is the order the
serial oracle adds them in, so the result is bit-identical to ``build_system`` over all edges (checked in
tests/test_oracle_system.py).  The graph arrays are shared with the workers through fork (copy-on-write, never
written).
"""
from __future__ import annotations

import multiprocessing as mp
import os
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

from oracle import sim3_gn_oracle as orc

_SHARED: Dict[str, object] = {}


def host_cores() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:  # pragma: no cover
        return max(1, os.cpu_count() or 1)


def _edge_chunk(chunk: Sequence[int]) -> List[Tuple]:
    from threadpoolctl import threadpool_limits
    poses, points, conf, edges, match, prm = (_SHARED[k] for k in ("poses", "points", "conf", "edges", "match", "prm"))
    out = []
    with threadpool_limits(limits=1):                       # one core per worker: the pool is the parallelism
        for e in chunk:
            i, j = int(edges[e, 0]), int(edges[e, 1])
            sysm = orc.build_system(poses, points, conf, edges, match, prm, edge_subset=[e])
            idx = np.r_[7 * i:7 * i + 7, 7 * j:7 * j + 7]
            out.append((e, sysm.H[np.ix_(idx, idx)].copy(), sysm.g[idx].copy(), sysm.g_abs[idx].copy(), int(sysm.n_valid[e]),
                        int(sysm.checksum[e]), sysm.edge_A[e].copy(), sysm.edge_b[e].copy(), float(sysm.edge_cost[e]),
                        sysm.edge_b_abs[e].copy()))
    return out


def build_system_parallel(poses: np.ndarray, points: np.ndarray, conf: np.ndarray, edges: np.ndarray, match: np.ndarray,
                          prm: orc.Params, edge_subset: Optional[Sequence[int]] = None, n_workers: Optional[int] = None,
                          dense: bool = True) -> orc.System:
    """``orc.build_system`` with the edges spread over ``n_workers`` processes (default: every core).  ``dense=False``
    skips the 7N x 7N H (returned as None) when only the per-edge outputs are wanted."""
    N, E = points.shape[0], edges.shape[0]
    todo = list(range(E)) if edge_subset is None else [int(e) for e in edge_subset]
    n_workers = max(1, min(n_workers or host_cores(), max(1, len(todo))))
    # small chunks, dealt round-robin in edge order: every worker sees a mix of cheap and expensive edges
    per = max(1, min(16, len(todo) // (4 * n_workers) or 1))
    chunks = [todo[k:k + per] for k in range(0, len(todo), per)]
    _SHARED.update(poses=np.ascontiguousarray(poses), points=points, conf=conf, edges=edges, match=match, prm=prm)
    try:
        if n_workers == 1:
            parts = [_edge_chunk(c) for c in chunks]
        else:
            with mp.get_context("fork").Pool(n_workers) as pool:
                parts = pool.map(_edge_chunk, chunks, chunksize=1)
    finally:
        _SHARED.clear()
    H = np.zeros((7 * N, 7 * N)) if dense else None
    g, g_abs = np.zeros(7 * N), np.zeros(7 * N)
    n_valid = np.zeros(E, dtype=np.int64)
    checksum = np.zeros(E, dtype=np.uint64)
    edge_A, edge_b, edge_cost, edge_b_abs = np.zeros((E, 7, 7)), np.zeros((E, 7)), np.zeros(E), np.zeros((E, 7))
    cost = 0.0
    for rec in sorted((r for p in parts for r in p), key=lambda r: r[0]):   # ascending edge order = the serial oracle's
        e, Hc, gc, gac, nv, chk, A, b, c, ba = rec
        i, j = int(edges[e, 0]), int(edges[e, 1])
        si, sj = slice(7 * i, 7 * i + 7), slice(7 * j, 7 * j + 7)
        if dense:
            H[si, si] += Hc[:7, :7]
            H[si, sj] += Hc[:7, 7:]
            H[sj, si] += Hc[7:, :7]
            H[sj, sj] += Hc[7:, 7:]
        g[si] += gc[:7]
        g[sj] += gc[7:]
        g_abs[si] += gac[:7]
        g_abs[sj] += gac[7:]
        n_valid[e], checksum[e] = nv, np.uint64(chk)
        edge_A[e], edge_b[e], edge_cost[e], edge_b_abs[e] = A, b, c, ba
        cost += c
    return orc.System(H, g, g_abs, cost, n_valid, checksum, edge_A, edge_b, edge_cost, edge_b_abs)
