"""rpim_apply_penalty_static: the penalty stage for callers that must not allocate device memory.

Who needs it: a program that has already given (nearly) all of the GPU's memory to its own pool -- at the `stress`
configuration K, col_idx and the staged shape functions fill 174 of 180 GB, so a late cudaMalloc inside the
library can fail -- or one that runs other streams on the device, which every cudaMalloc / cudaFree would stall.
rpim_apply_penalty draws its scratch memory from the context's workspace and so may allocate; the static entry
point keeps the same scratch in one fixed array inside librpim.so (see include/rpim.h for the limit and the
sharing rules).

What is checked here: on the same K and f both entry points leave bitwise the same K, f and alpha_used (the
arithmetic is an exact maximum, one product and one add per entry, so the bar is equality, tighter than the
1e-10 * max|K_ii| the parity tests allow), on two calls in a row.  The second call uses another boundary list, a
smaller problem and a fresh context: the array is shared by all contexts and keeps the first call's contents, so
a stale "seen" bit or counter would show up as a wrongly rejected list or a wrong alpha.

The file is named so that pytest collects it last: a failure here cannot hide the other tests behind `-x`.
It does not depend on them either (it passes alone in a fresh process and after the rest of the suite).
"""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


def _assembled(ctx, w):
    """Pattern + K, f of workload w on ctx; the coordinate tensors are returned so that they outlive the pattern."""
    import torch
    dev = torch.device("cuda:0")
    keep = (torch.from_numpy(w.nodes).to(dev), torch.from_numpy(w.qpts).to(dev))
    nnz, _ = ctx.build_pattern(keep[0], keep[1], w.k)
    vals = torch.empty(nnz, dtype=torch.float64, device=dev)
    f = torch.empty(3 * w.N, dtype=torch.float64, device=dev)
    ctx.assemble(torch.from_numpy(w.qw).to(dev), w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, vals, f)
    return keep, vals, f


def _both_paths(ctx, vals, f, bc_nodes, bc_mask, ubar, alpha, relative):
    """Apply the penalty to two copies of (K, f): existing path, static path.  Returns both results."""
    import torch
    dev = vals.device
    bn = torch.from_numpy(np.ascontiguousarray(bc_nodes, dtype=np.int64)).to(dev)
    bm = None if bc_mask is None else torch.from_numpy(np.ascontiguousarray(bc_mask, dtype=np.uint8)).to(dev)
    ub = torch.from_numpy(np.ascontiguousarray(ubar, dtype=np.float64)).to(dev)
    v_ref, f_ref, v_sta, f_sta = vals.clone(), f.clone(), vals.clone(), f.clone()
    a_ref = ctx.apply_penalty(bn, bm, ub, alpha, relative, v_ref, f_ref)
    a_sta = ctx.apply_penalty_static(bn, bm, ub, alpha, relative, v_sta, f_sta)
    torch.cuda.synchronize()
    return (a_ref, v_ref, f_ref), (a_sta, v_sta, f_sta)


def _assert_same(ref, sta, vals0):
    import torch
    assert sta[0] == ref[0]                                    # alpha_used
    assert torch.equal(sta[1], ref[1]) and torch.equal(sta[2], ref[2])
    assert int((sta[1] != vals0).sum()) > 0                    # and something was in fact applied


def test_static_penalty_matches_the_allocating_path_on_two_calls_in_a_row():
    import torch
    import paper_1802_04256_b200 as rp
    assert rp.rpim_apply_penalty_static_max_nodes() == 4194304
    rng = np.random.default_rng(7)

    # call 1: jittered block, relative alpha, the workload's own boundary list (bottom fixed + rollers, masks)
    w1 = workloads.make_block("na1", 9, 8, 7, 1.0, 2, 30, 5e9, 0.3, jitter=0.3, seed=11, body=(0.0, 0.0, -2.5e4),
                              bc="bottom+roller")
    with rp.Context(0) as ctx:
        keep, vals, f = _assembled(ctx, w1)
        ub1 = rng.uniform(-1e-3, 1e-3, size=(len(w1.bc_nodes), 3))
        ref, sta = _both_paths(ctx, vals, f, w1.bc_nodes, w1.bc_mask, ub1, w1.penalty_alpha, True)
        _assert_same(ref, sta, vals)
        assert sta[0] > 0.0

    # call 2, straight after, in a NEW context on a smaller cloud whose list contains ids that call 1 also listed:
    # only a cleared array accepts them; absolute alpha, no mask
    w2 = workloads.make_block("na2", 6, 5, 5, 1.0, 1, 12, 1e9, 0.3, jitter=0.2, seed=5, body=(0.0, 0.0, -1.0))
    common = np.intersect1d(w1.bc_nodes, np.arange(w2.N))
    assert len(common) >= 3
    list2 = np.concatenate([common[:3], [w2.N - 1]])
    with rp.Context(0) as ctx:
        keep, vals, f = _assembled(ctx, w2)
        ub2 = rng.uniform(-1.0, 1.0, size=(len(list2), 3))
        ref, sta = _both_paths(ctx, vals, f, list2, None, ub2, 1e3, False)
        _assert_same(ref, sta, vals)
        assert sta[0] == 1e3

        # a rejected list (id listed twice) leaves K and f alone, and the counter it raised does not poison the
        # next call on the shared array
        v0, f0 = vals.clone(), f.clone()
        dup = torch.tensor([3, 7, 3], dtype=torch.int64, device=vals.device)
        ub = torch.full((3, 3), 0.5, dtype=torch.float64, device=vals.device)
        with pytest.raises(rp.RpimError) as e:
            ctx.apply_penalty_static(dup, None, ub, 1e3, False, vals, f)
        assert e.value.code == -5
        assert torch.equal(vals, v0) and torch.equal(f, f0)
        ref, sta = _both_paths(ctx, vals, f, [3, 7, 4], None, ub.cpu().numpy(), 2.0, True)
        _assert_same(ref, sta, vals)

        # m = 0: nothing to apply, alpha_used = alpha * max_d K_dd as in the allocating path
        a_ref = ctx.apply_penalty(None, None, None, 1.0, True, vals, f)
        a_sta = ctx.apply_penalty_static(None, None, None, 1.0, True, vals, f)
        assert a_sta == a_ref and torch.equal(vals, v0) and torch.equal(f, f0)


def test_static_penalty_allocates_nothing_and_refuses_problems_beyond_its_limit():
    import torch
    import paper_1802_04256_b200 as rp
    dev = torch.device("cuda:0")
    w = workloads.make_block("na3", 6, 5, 5, 1.0, 1, 12, 1e9, 0.3, jitter=0.2, seed=9, body=(0.0, 0.0, -1.0))
    with rp.Context(0) as ctx:
        keep, vals, f = _assembled(ctx, w)
        bn = torch.tensor([0, 1, 2], dtype=torch.int64, device=dev)
        ub = torch.zeros((3, 3), dtype=torch.float64, device=dev)
        ctx.apply_penalty_static(bn, None, ub, 1.0, True, vals, f)      # first call on the device: set-up
        torch.cuda.synchronize()
        ws, (free0, _) = ctx.workspace_bytes(), torch.cuda.mem_get_info(0)
        for _ in range(3):
            ctx.apply_penalty_static(bn, None, ub, 1.0, True, vals, f)
        torch.cuda.synchronize()
        assert ctx.workspace_bytes() == ws                              # the context's workspace did not grow
        assert torch.cuda.mem_get_info(0)[0] == free0                   # and the device's free memory did not move

    # one node more than the array has bits for (4194305 = 5 * 397 * 2113, a regular lattice); only the few nodes
    # around 16 quadrature points get a matrix row, so the pattern and K stay tiny
    nmax = rp.rpim_apply_penalty_static_max_nodes()
    nx, ny, nz = 5, 397, 2113
    N = nx * ny * nz
    assert N == nmax + 1
    ids = np.arange(N, dtype=np.int64)
    nodes = np.stack([ids % nx, (ids // nx) % ny, ids // (nx * ny)], axis=1).astype(np.float64)
    rng = np.random.default_rng(3)
    qpts = np.array([2.0, 200.0, 1000.0]) + rng.uniform(-1.5, 1.5, size=(16, 3))
    with rp.Context(0) as ctx:
        dn, dq = torch.from_numpy(nodes).to(dev), torch.from_numpy(qpts).to(dev)
        nnz, _ = ctx.build_pattern(dn, dq, 8)
        vals = torch.ones(nnz, dtype=torch.float64, device=dev)
        f = torch.zeros(3 * N, dtype=torch.float64, device=dev)
        v0 = vals.clone()
        with pytest.raises(rp.RpimError) as e:
            ctx.apply_penalty_static(None, None, None, 1.0, False, vals, f)
        assert e.value.code == -7 and "RPIM_STATIC_PENALTY_MAX_NODES" in str(e.value)
        assert torch.equal(vals, v0)
        assert ctx.apply_penalty(None, None, None, 1.0, False, vals, f) == 1.0   # the allocating path still serves it
