"""Sharding ONE assembly problem across ranks ("no data dependencies between
... any two element stiffness matrices").  Host-side index logic only -- no arithmetic of the method.

Row-owner partition with redundant halo work and NO data-path exchange:

  * rank r owns the block rows (nodes) [N r / W, N (r+1) / W): contiguous id ranges, i.e. spatial slabs for a
    spatially coherent numbering;
  * it takes every quadrature point within `halo` of the bounding box of its owned nodes -- in whole groups of 8
    consecutive global ids, see below -- and every node within `halo` of the farthest taken point's distance
    from that box (2 * `halo` when no group sticks out).  If `halo` bounds the support radius (distance from a
    point to its k-th nearest node) of every point, then (a) every point whose support touches an owned row is
    taken, and (b) the k nearest nodes of a taken point among the taken nodes are its k nearest nodes among ALL
    nodes.  The owned rows of the rank's sub-problem are then complete; the rows of halo nodes are partial and
    are discarded;
  * rounding: with supports ascending and points in ascending order the row-owner kernel (and the oracle) add
    a row's contributions point by point in the same order as on the undivided problem: owned rows are
    bit-identical.  The panel kernel first sums the points of a group of 8 consecutive LOCAL ids in registers;
    because points are taken in whole global groups (`make_shard(group=8)`), local groups are the undivided
    problem's groups and its owned rows are bit-identical too (tests/test_gpu_sharded.py runs both kernels).
    With `group=1` that kernel's owned rows agree only to rounding;
  * the bound has to be VERIFIED after the support search, and `verify_shard` does it (the tests and
    `bench.py --shard` call it and refuse to go on otherwise): on the sub-cloud the k-th neighbour distance can
    only be larger than the true one, so `max <= halo` on every rank (`support_radius_ok`) proves the premise
    for every point that some rank has taken -- and that every point IS taken by at least one rank is checked
    too, since a point farther than `halo` from every slab's box would otherwise be dropped silently;
  * the only collective of the path is allreduce(max) of one double: alpha = penalty * max_i K_ii.  A halo row's
    partial diagonal never exceeds its complete value (every contribution to a diagonal entry is >= 0), which
    the owning rank holds, so max over ranks of the local maxima is the global maximum.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class Shard:
    rank: int
    world: int
    row_lo: int                # owned global rows [row_lo, row_hi)
    row_hi: int
    node_ids: np.ndarray       # global ids of the taken nodes, ascending (local id = position)
    point_ids: np.ndarray      # global ids of the taken points, ascending
    own_lo: int                # owned rows in LOCAL numbering [own_lo, own_hi) (contiguous: ids are ascending)
    own_hi: int
    halo: float


def owned_rows(N: int, rank: int, world: int):
    return (N * rank) // world, (N * (rank + 1)) // world


def halo_estimate(nodes: np.ndarray, k: int, safety: float = 2.2) -> float:
    """A support-radius bound from the mean node density: radius of the ball holding k nodes, times `safety`
    (a point in a corner of the domain sees one octant: factor 2; the rest covers jitter).  It is an estimate;
    `support_radius_ok` is what validates it."""
    ext = nodes.max(axis=0) - nodes.min(axis=0)
    vol = float(np.prod(np.maximum(ext, 1e-9 * ext.max())))
    h = (vol / nodes.shape[0]) ** (1.0 / 3.0)
    return safety * (3.0 * k / (4.0 * np.pi)) ** (1.0 / 3.0) * h


POINT_GROUP = 8   # the panel reduction sums the points of a group of 8 consecutive ids in registers first


def _box_distance(x: np.ndarray, blo: np.ndarray, bhi: np.ndarray) -> np.ndarray:
    """Chebyshev distance of every row of x to the axis-aligned box [blo, bhi] (0 inside)."""
    return np.maximum(np.maximum(blo - x, x - bhi), 0.0).max(axis=1)


def make_shard(nodes: np.ndarray, qpts: np.ndarray, k: int, rank: int, world: int, halo: float | None = None,
               group: int = POINT_GROUP) -> Shard:
    """`group`: points are taken in whole groups of `group` consecutive global ids (a group with one point within
    `halo` of the box is taken entirely).  The shard's local groups of `group` consecutive points are then the
    undivided problem's groups, so a reduction that sums group-wise (the panel kernel) rounds the owned rows exactly
    as it does on the undivided problem.  The node halo grows accordingly: `halo` beyond the farthest taken point."""
    N, Nq = nodes.shape[0], qpts.shape[0]
    lo, hi = owned_rows(N, rank, world)
    if halo is None:
        halo = halo_estimate(nodes, k)
    own = nodes[lo:hi]
    blo, bhi = own.min(axis=0), own.max(axis=0)
    dist_p = _box_distance(qpts, blo, bhi)
    take_p = dist_p <= halo
    if group > 1:
        G = -(-Nq // group)
        pad = np.zeros(G * group, dtype=bool)
        pad[:Nq] = take_p
        take_p = np.repeat(pad.reshape(G, group).any(axis=1), group)[:Nq]
    reach = max(float(halo), float(dist_p[take_p].max())) if take_p.any() else float(halo)
    take_n = _box_distance(nodes, blo, bhi) <= reach + halo      # every taken point's support (radius <= halo)
    take_n[lo:hi] = True
    node_ids = np.nonzero(take_n)[0].astype(np.int64)
    point_ids = np.nonzero(take_p)[0].astype(np.int64)
    own_lo = int(np.searchsorted(node_ids, lo))
    own_hi = int(np.searchsorted(node_ids, hi))
    assert own_hi - own_lo == hi - lo
    return Shard(rank, world, lo, hi, node_ids, point_ids, own_lo, own_hi, float(halo))


def support_radius_ok(sub_nodes: np.ndarray, sub_pts: np.ndarray, support_local: np.ndarray, halo: float) -> bool:
    """max over the taken points of the distance to the farthest node of the support found on the sub-cloud."""
    d = sub_nodes[support_local] - sub_pts[:, None, :]
    return bool(np.sqrt((d * d).sum(axis=2)).max() <= halo)


def verify_shard(shard: Shard, sub_nodes: np.ndarray, sub_pts: np.ndarray, support_local: np.ndarray, nq_total: int,
                 allreduce=None):
    """The two premises of the docstring above, checked after the support search of every rank: (1) `halo` bounds
    the support radius found on the sub-cloud (`support_radius_ok`) on EVERY rank, (2) every quadrature point of
    the domain is taken by at least one rank.  `allreduce(array, op)` with op in {"min", "max"} reduces a float64
    / uint8 numpy array over the ranks and returns the result (None: single rank).  Returns
    (all ranks' halo bound holds, number of points no rank has taken); a caller must not use the owned rows
    unless the result is (True, 0)."""
    ok = np.array([1.0 if support_radius_ok(sub_nodes, sub_pts, support_local, shard.halo) else 0.0])
    taken = np.zeros(nq_total, dtype=np.uint8)
    taken[shard.point_ids] = 1
    if allreduce is not None:
        ok = allreduce(ok, "min")
        taken = allreduce(taken, "max")
    return bool(ok[0] == 1.0), int(nq_total - int(taken.sum(dtype=np.int64)))


def local_bc(shard: Shard, bc_nodes: np.ndarray, bc_mask: np.ndarray, bc_ubar: np.ndarray):
    """The boundary conditions of the owned rows, in local numbering."""
    sel = (bc_nodes >= shard.row_lo) & (bc_nodes < shard.row_hi)
    loc = np.searchsorted(shard.node_ids, bc_nodes[sel]).astype(np.int64)
    return np.ascontiguousarray(loc), np.ascontiguousarray(bc_mask[sel]), np.ascontiguousarray(bc_ubar[sel])


def owned_csr_rows(shard: Shard, row_ptr: np.ndarray, col_idx: np.ndarray, vals: np.ndarray, f: np.ndarray):
    """The owned scalar rows of a rank's local CSR, columns mapped back to GLOBAL DOF ids."""
    a, b = int(row_ptr[3 * shard.own_lo]), int(row_ptr[3 * shard.own_hi])
    ci = col_idx[a:b].astype(np.int64)
    gcol = 3 * shard.node_ids[ci // 3] + ci % 3
    return (row_ptr[3 * shard.own_lo:3 * shard.own_hi + 1].astype(np.int64) - a, gcol, vals[a:b],
            f[3 * shard.own_lo:3 * shard.own_hi])
