"""CPU tests (gloo, world_size 2) of the SHARDED N > 1 path (paper_1802_04256_b200/partition.py):
one domain cut into row slabs with a halo of points and nodes, no data-path exchange, allreduce(max) of one
double for the penalty alpha.  The ranks' engine here is the CPU oracle (no GPU in this container); the same
partition logic drives the CUDA path in tests/test_gpu_sharded.py and `bench.py --shard`.

Checked: the owned row ranges tile [0, N); every point whose (true) support touches a rank's rows is taken by
that rank and the supports of the taken points lie inside the taken nodes (the halos are supersets); the
sub-cloud search finds the true supports; the owned rows of every rank are BIT-identical to the same rows of the
undivided problem; alpha is identical on every rank and equals the undivided alpha."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _problem():
    import workloads
    return workloads.make_block("shard", 12, 9, 8, 1.0, 2, 30, 5e9, 0.3, jitter=0.3, seed=21,
                                body=(0.0, 0.0, -2.5e4), bc="bottom+roller")


def _rank_assemble(w, sh):
    """Sub-problem of one rank with the oracle: local supports, pattern, K, f; penalty-free."""
    import oracle
    nodes, pts, qw = np.ascontiguousarray(w.nodes[sh.node_ids]), np.ascontiguousarray(w.qpts[sh.point_ids]), \
        np.ascontiguousarray(w.qw[sh.point_ids])
    s = oracle.knn(nodes, pts, w.k, "grid")
    rp, ci = oracle.pattern(s, nodes.shape[0])
    vals, f, ns = oracle.assemble(nodes, pts, qw, s, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, rp, ci)
    return nodes, pts, s, rp, ci, vals, f


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    from paper_1802_04256_b200 import partition as pt

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _problem()
        sh = pt.make_shard(w.nodes, w.qpts, w.k, rank, world)
        nodes, pts, s, rp, ci, vals, f = _rank_assemble(w, sh)
        import bench
        ok, missing = pt.verify_shard(sh, nodes, pts, s, w.Nq, bench.rank_allreduce(world))   # as bench.py --shard does
        assert missing == 0
        flag = torch.tensor([1.0 if ok else 0.0], dtype=torch.float64)
        # points that no rank takes (here: every rank forgets every other one of its own; on this small block the
        # halos make both ranks take all points, so the odd ones are lost) are seen by EVERY rank
        cut = pt.Shard(sh.rank, sh.world, sh.row_lo, sh.row_hi, sh.node_ids, sh.point_ids[::2], sh.own_lo, sh.own_hi,
                       sh.halo)
        ok2, missing2 = pt.verify_shard(cut, nodes, pts[::2], s[::2], w.Nq, bench.rank_allreduce(world))
        assert ok2 and missing2 > 0
        rows = np.repeat(np.arange(len(rp) - 1), np.diff(rp))
        local_max = float(vals[rows == ci].max())             # over ALL local rows, partial halo rows included
        t = torch.tensor([local_max], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        alpha = w.penalty_alpha * float(t.item())
        orp, gcol, ovals, of = pt.owned_csr_rows(sh, rp, ci, vals, f)
        bn, bm, bu = pt.local_bc(sh, w.bc_nodes, w.bc_mask, w.bc_ubar)
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), lo=sh.row_lo, hi=sh.row_hi, node_ids=sh.node_ids,
                 point_ids=sh.point_ids, support=s, halo_ok=float(flag.item()), alpha=alpha, local_max=local_max,
                 orp=orp, gcol=gcol, ovals=ovals, of=of, bc_local=bn, bc_global=sh.node_ids[bn])
    finally:
        dist.destroy_process_group()


def test_two_ranks_shard_one_domain_and_stitch_back_to_the_undivided_matrix(tmp_path):
    import torch.multiprocessing as mp
    import oracle

    world, port = 2, 31000 + os.getpid() % 2000
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    R = [np.load(tmp_path / f"r{r}.npz") for r in range(world)]
    w = _problem()
    S = oracle.knn(w.nodes, w.qpts, w.k, "brute")
    rp, ci = oracle.pattern(S, w.N)
    vals, f, _ = oracle.assemble(w.nodes, w.qpts, w.qw, S, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, rp, ci)
    rows = np.repeat(np.arange(len(rp) - 1), np.diff(rp))
    kmax = vals[rows == ci].max()
    # the owned ranges tile the rows
    assert int(R[0]["lo"]) == 0 and int(R[-1]["hi"]) == w.N
    assert all(int(R[i]["hi"]) == int(R[i + 1]["lo"]) for i in range(world - 1))
    for r in R:
        lo, hi = int(r["lo"]), int(r["hi"])
        touching = np.nonzero(((S >= lo) & (S < hi)).any(axis=1))[0]
        assert np.isin(touching, r["point_ids"]).all()                       # halo of points is a superset
        assert np.isin(S[r["point_ids"]].ravel(), r["node_ids"]).all()       # halo of nodes is a superset
        assert np.array_equal(r["node_ids"][r["support"]], S[r["point_ids"]])  # sub-cloud search = true supports
        assert float(r["halo_ok"]) == 1.0
        gid, cnt = np.unique(r["point_ids"] // 8, return_counts=True)          # points come in whole groups of 8
        assert np.all(cnt[gid < w.Nq // 8] == 8)
        a, b = int(rp[3 * lo]), int(rp[3 * hi])
        assert np.array_equal(r["orp"], rp[3 * lo:3 * hi + 1] - a)            # owned rows: pattern bit-exact
        assert np.array_equal(r["gcol"], ci[a:b])
        assert np.array_equal(r["ovals"], vals[a:b])                          # and values BIT-identical
        assert np.array_equal(r["of"], f[3 * lo:3 * hi])
        assert float(r["alpha"]) == w.penalty_alpha * kmax                    # identical alpha on every rank
        sel = (w.bc_nodes >= lo) & (w.bc_nodes < hi)
        assert np.array_equal(r["bc_global"], w.bc_nodes[sel])
    assert float(R[0]["alpha"]) == float(R[1]["alpha"])
    assert max(float(r["local_max"]) for r in R) == kmax


def test_partition_degenerates_gracefully():
    from paper_1802_04256_b200 import partition as pt
    w = _problem()
    one = pt.make_shard(w.nodes, w.qpts, w.k, 0, 1)
    assert one.row_lo == 0 and one.row_hi == w.N and one.own_lo == 0 and one.own_hi == w.N
    assert one.node_ids.size == w.N and one.point_ids.size == w.Nq
    lo_hi = [pt.owned_rows(10, r, 4) for r in range(4)]
    assert lo_hi == [(0, 2), (2, 5), (5, 7), (7, 10)]
    # a halo that is too small is caught by the check, not silently accepted
    import oracle
    sh = pt.make_shard(w.nodes, w.qpts, w.k, 1, 2, halo=0.5)
    nodes, pts = w.nodes[sh.node_ids], w.qpts[sh.point_ids]
    s = oracle.knn(np.ascontiguousarray(nodes), np.ascontiguousarray(pts), w.k, "grid")
    assert not pt.support_radius_ok(nodes, pts, s, sh.halo)
    # bench.py --shard refuses to time such a partition: the halo bound fails, and with so small a halo the two
    # ranks together do not even take every point
    import bench
    ok, missing = pt.verify_shard(sh, nodes, pts, s, w.Nq)
    assert not ok and missing > 0
    import pytest
    with pytest.raises(RuntimeError, match="halo"):
        import dataclasses
        bench.check_shard(sh, dataclasses.replace(w, nodes=nodes, qpts=pts), s, w.Nq, 1)
    good = pt.make_shard(w.nodes, w.qpts, w.k, 0, 1)
    s_all = oracle.knn(w.nodes, w.qpts, w.k, "grid")
    assert pt.verify_shard(good, w.nodes, w.qpts, s_all, w.Nq) == (True, 0)


def test_bench_shard_workload_covers_the_domain_once():
    """bench.py --shard: the ranks' sub-problems own every block row and every boundary condition exactly once, and
    take every quadrature point at least once (halo points more than once)."""
    import bench
    import workloads
    world = 3
    w = workloads.config("cantilever")
    rows, bcs, pts = [], [], np.zeros(w.Nq, dtype=np.int64)
    for r in range(world):
        wl, sh, nq = bench.shard_workload("cantilever", r, world)
        assert nq == w.Nq and wl.N == sh.node_ids.size and wl.Nq == sh.point_ids.size
        rows.append((sh.row_lo, sh.row_hi))
        bcs.append(sh.node_ids[wl.bc_nodes])                     # local -> global ids of the rank's boundary nodes
        assert np.all((bcs[-1] >= sh.row_lo) & (bcs[-1] < sh.row_hi))
        pts[sh.point_ids] += 1
        assert np.array_equal(wl.nodes, w.nodes[sh.node_ids]) and np.array_equal(wl.qw, w.qw[sh.point_ids])
    assert rows[0][0] == 0 and rows[-1][1] == w.N and all(a[1] == b[0] for a, b in zip(rows[:-1], rows[1:]))
    assert np.array_equal(np.sort(np.concatenate(bcs)), w.bc_nodes)
    assert pts.min() >= 1 and pts.max() > 1
