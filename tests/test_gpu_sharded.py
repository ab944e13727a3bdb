"""-m gpu: ONE domain sharded into row slabs with halos (paper_1802_04256_b200/partition.py), the
shards run one after the other on this GPU through the C ABI (no rank waits on another: each shard is a complete,
independent problem; the only exchange of the path, allreduce(max) of a double, is a host max here).  The
stitched matrix must equal the undivided CUDA result bit for bit, alpha included, with either reduction kernel
(the panel kernel sums groups of 8 points first: shards take whole groups, partition.py), and -- the check that
does not compare the CUDA path with itself -- every rank's owned rows must match the ORACLE's undivided matrix:
pattern bit-exact, values within 1e-10 * max|K_ii| (BASELINE.json north_star)."""
import numpy as np
import pytest

import workloads
from gpu_harness import kmax_diag, run_cuda, run_oracle

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("world,reduction", [(2, 1), (3, 1), (2, 2), (3, 2)])
def test_sharded_assembly_stitches_to_the_undivided_result(world, reduction):
    from paper_1802_04256_b200 import partition as pt
    w = workloads.make_block("shard", 8, 7, 26, 1.0, 2, 30, 5e9, 0.3, jitter=0.3, seed=22,
                             body=(0.0, 0.0, -2.5e4), bc="bottom+roller")
    full = run_cuda(w, index_bits=64, want_shape=False, reduction=reduction)
    assert full["reduction_used"] == reduction
    o = run_oracle(w)
    km = kmax_diag(o)
    shards = [pt.make_shard(w.nodes, w.qpts, w.k, r, world) for r in range(world)]
    assert shards[0].row_lo == 0 and shards[-1].row_hi == w.N
    assert any(s.point_ids.size < w.Nq for s in shards)                       # the halo really cuts work
    # each shard is run to completion on its own; closures keep the device state until alpha is known
    import torch
    parts = []
    for sh in shards:
        parts.append(_run_shard_keep(w, sh, reduction))
    alpha = w.penalty_alpha * max(p["local_max"] for p in parts)              # = allreduce(max) across ranks
    assert alpha == full["alpha"]
    rp_f, ci_f = full["row_ptr"], full["col_idx"]
    for sh, p in zip(shards, parts):
        orp, gcol, ovals, of = p["finish"](alpha)
        a, b = int(rp_f[3 * sh.row_lo]), int(rp_f[3 * sh.row_hi])
        assert np.array_equal(orp, rp_f[3 * sh.row_lo:3 * sh.row_hi + 1] - a)
        assert np.array_equal(gcol, ci_f[a:b])
        assert np.array_equal(ovals, full["vals"][a:b])                       # penalised values, bit for bit
        assert np.array_equal(of, full["f"][3 * sh.row_lo:3 * sh.row_hi])
        # against the oracle's undivided, penalised matrix (its alpha is the oracle's own max_i K_ii)
        assert np.array_equal(orp, o["row_ptr"][3 * sh.row_lo:3 * sh.row_hi + 1] - a) and np.array_equal(gcol, o["col_idx"][a:b])
        assert abs(alpha - o["alpha"]) <= 1e-12 * o["alpha"]
        pen = np.abs(o["vals"][a:b] - o["vals0"][a:b]) > 0                    # the constrained diagonals
        assert np.array_equal(pen, np.abs(ovals - full["vals0"][a:b]) > 0)
        assert np.abs(ovals - o["vals"][a:b])[~pen].max() <= 1e-10 * km
        assert np.abs(ovals - o["vals"][a:b])[pen].max() <= 1e-10 * o["alpha"]
        assert np.abs(of - o["f"][3 * sh.row_lo:3 * sh.row_hi]).max() <= 1e-10 * np.abs(o["f"]).max()
        p["close"]()
    torch.cuda.empty_cache()


def _run_shard_keep(w, sh, reduction):
    """Like _run_shard but the context stays open until the caller has applied the penalty."""
    import torch
    import paper_1802_04256_b200 as rp
    from paper_1802_04256_b200 import partition as pt
    dev = torch.device("cuda:0")
    nodes = np.ascontiguousarray(w.nodes[sh.node_ids])
    pts = np.ascontiguousarray(w.qpts[sh.point_ids])
    qw = np.ascontiguousarray(w.qw[sh.point_ids])
    ctx = rp.Context(0)
    ctx.set_reduction(reduction)
    keep = {}
    keep["d_n"], keep["d_q"] = torch.from_numpy(nodes).to(dev), torch.from_numpy(pts).to(dev)
    nnz, bits = ctx.build_pattern(keep["d_n"], keep["d_q"], w.k, 64)
    d_rp = torch.empty(3 * nodes.shape[0] + 1, dtype=torch.int64, device=dev)
    d_ci = torch.empty(nnz, dtype=torch.int64, device=dev)
    d_sup = torch.empty((pts.shape[0], w.k), dtype=torch.int32, device=dev)
    ctx.get_pattern(d_rp, d_ci, d_sup)
    d_vals = torch.empty(nnz, dtype=torch.float64, device=dev)
    d_f = torch.empty(3 * nodes.shape[0], dtype=torch.float64, device=dev)
    ns = ctx.assemble(torch.from_numpy(qw).to(dev), w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, d_vals, d_f)
    assert ns == 0
    assert pt.verify_shard(sh, nodes, pts, d_sup.cpu().numpy(), w.Nq)[0]
    assert ctx.reduction_used() == reduction
    local_max = ctx.apply_penalty(None, None, None, 1.0, True, d_vals, d_f)          # m = 0: max_d K_dd, nothing applied

    def finish(alpha_abs):
        bn, bm, bu = pt.local_bc(sh, w.bc_nodes, w.bc_mask, w.bc_ubar)
        if bn.size:
            ctx.apply_penalty(torch.from_numpy(bn).to(dev), torch.from_numpy(bm).to(dev), torch.from_numpy(bu).to(dev),
                              alpha_abs, False, d_vals, d_f)
        return pt.owned_csr_rows(sh, d_rp.cpu().numpy(), d_ci.cpu().numpy(), d_vals.cpu().numpy(), d_f.cpu().numpy())

    return dict(local_max=local_max, finish=finish, close=ctx.close, keep=keep)
