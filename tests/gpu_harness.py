"""Helpers shared by the -m gpu parity tests: run the CUDA path through the C ABI binding and the
CPU oracle on the same seeded inputs."""
from __future__ import annotations

import numpy as np


def run_cuda(w, *, penalty=True, loads=True, index_bits=None, want_shape=True, ctx=None):
    import torch
    import paper_1802_04256_b200 as rp

    dev = torch.device("cuda:0")
    own = ctx is None
    if own:
        ctx = rp.Context(0)
    out = {}
    try:
        d_nodes = torch.from_numpy(w.nodes).to(dev)
        d_qpts = torch.from_numpy(w.qpts).to(dev)
        d_qw = torch.from_numpy(w.qw).to(dev)
        bits_req = w.index_bits if index_bits is None else index_bits
        nnz, bits = ctx.build_pattern(d_nodes, d_qpts, w.k, bits_req)
        idt = torch.int32 if bits == 32 else torch.int64
        d_rp = torch.empty(3 * w.N + 1, dtype=idt, device=dev)
        d_ci = torch.empty(nnz, dtype=idt, device=dev)
        d_sup = torch.empty((w.Nq, w.k), dtype=torch.int32, device=dev)
        ctx.get_pattern(d_rp, d_ci, d_sup)
        d_vals = torch.full((nnz,), float("nan"), dtype=torch.float64, device=dev)
        d_f = torch.full((3 * w.N,), float("nan"), dtype=torch.float64, device=dev)
        nsing = ctx.assemble(d_qw, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, d_vals, d_f)
        out.update(nnz=nnz, bits=bits, nsing=nsing, phase_ms=ctx.phase_ms())
        if want_shape:
            d_phi = torch.empty((w.Nq, w.k), dtype=torch.float64, device=dev)
            d_dphi = torch.empty((w.Nq, 3, w.k), dtype=torch.float64, device=dev)
            d_sing = torch.empty(w.Nq, dtype=torch.uint8, device=dev)
            ctx.get_shape(d_phi, d_dphi, d_sing)
            out.update(phi=d_phi.cpu().numpy(), dphi=d_dphi.cpu().numpy(), singular=d_sing.cpu().numpy())
        out.update(vals0=d_vals.cpu().numpy(), f0=d_f.cpu().numpy())
        if loads and w.load_pts is not None:
            ctx.add_point_loads(torch.from_numpy(w.load_pts).to(dev), torch.from_numpy(w.load_w).to(dev),
                                torch.from_numpy(w.load_t).to(dev), d_f)
        out["f_loaded"] = d_f.cpu().numpy()
        if penalty:
            alpha = ctx.apply_penalty(torch.from_numpy(w.bc_nodes).to(dev), torch.from_numpy(w.bc_mask).to(dev),
                                      torch.from_numpy(w.bc_ubar).to(dev), w.penalty_alpha, True, d_vals, d_f)
            out["alpha"] = alpha
        torch.cuda.synchronize()
        out.update(row_ptr=d_rp.cpu().numpy(), col_idx=d_ci.cpu().numpy(), support=d_sup.cpu().numpy(),
                   vals=d_vals.cpu().numpy(), f=d_f.cpu().numpy(), launches=ctx.launch_count())
    finally:
        if own:
            ctx.close()
    return out


def run_oracle(w, *, penalty=True, loads=True):
    import oracle

    s = oracle.knn(w.nodes, w.qpts, w.k, "grid")
    rp_, ci = oracle.pattern(s, w.N)
    phi, dphi, sing = oracle.shape(w.nodes, w.qpts, s, w.alpha_c, w.d_c, w.q)
    vals, f, ns = oracle.assemble(w.nodes, w.qpts, w.qw, s, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, rp_, ci)
    out = dict(support=s, row_ptr=rp_, col_idx=ci, phi=phi, dphi=dphi, singular=sing, vals0=vals.copy(),
               f0=f.copy(), nsing=ns)
    if loads and w.load_pts is not None:
        ls = oracle.knn(w.nodes, w.load_pts, w.k, "grid")
        oracle.point_loads(w.nodes, w.load_pts, w.load_w, w.load_t, ls, w.alpha_c, w.d_c, w.q, f)
    out["f_loaded"] = f.copy()
    if penalty:
        out["alpha"] = oracle.penalty(w.bc_nodes, w.bc_mask, w.bc_ubar, w.penalty_alpha, True, w.N, rp_, ci, vals, f)
    out.update(vals=vals, f=f)
    return out


def kmax_diag(o):
    """max_i |K_ii| before penalty (the scale of the 1e-10 tolerance, BASELINE.json north_star)."""
    rp_, ci, v = o["row_ptr"], o["col_idx"], o["vals0"]
    rows = np.repeat(np.arange(len(rp_) - 1), np.diff(rp_))
    return np.abs(v[rows == ci]).max()


def run_cuda_rows(w, slabs, *, want_shape=True):
    """Full-size run of the CUDA path in the launch configuration bench.py times; brings back only
    what the sampled checks need: for every node slab [lo, hi) the CSR rows, values (before and after
    the penalty) and load entries, plus the ids, supports and shape functions of the quadrature points
    incident to the slab."""
    import torch
    import paper_1802_04256_b200 as rp

    dev = torch.device("cuda:0")
    out = {"slabs": []}
    with rp.Context(0) as ctx:
        d_nodes = torch.from_numpy(w.nodes).to(dev)
        d_qpts = torch.from_numpy(w.qpts).to(dev)
        d_qw = torch.from_numpy(w.qw).to(dev)
        nnz, bits = ctx.build_pattern(d_nodes, d_qpts, w.k, w.index_bits)
        idt = torch.int32 if bits == 32 else torch.int64
        d_rp = torch.empty(3 * w.N + 1, dtype=idt, device=dev)
        d_ci = torch.empty(nnz, dtype=idt, device=dev)
        d_sup = torch.empty((w.Nq, w.k), dtype=torch.int32, device=dev)
        ctx.get_pattern(d_rp, d_ci, d_sup)
        d_vals = torch.full((nnz,), float("nan"), dtype=torch.float64, device=dev)
        d_f = torch.full((3 * w.N,), float("nan"), dtype=torch.float64, device=dev)
        nsing = ctx.assemble(d_qw, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, d_vals, d_f)
        out.update(nnz=nnz, bits=bits, nsing=nsing)
        # pattern-wide properties that hold at any size (cheap on the device)
        rp64 = d_rp.to(torch.int64)
        out["row_ptr_monotone"] = bool((rp64[1:] >= rp64[:-1]).all().item()) and int(rp64[0]) == 0 and int(rp64[-1]) == nnz
        out["support_sorted"] = bool((d_sup[:, 1:] > d_sup[:, :-1]).all().item())
        del rp64
        pts_of = []
        for lo, hi in slabs:
            parts = []   # in chunks of points: the temporaries stay small next to a 170 GB problem
            for c0 in range(0, w.Nq, 1 << 20):
                blk = d_sup[c0:c0 + (1 << 20)]
                parts.append(torch.nonzero(((blk >= lo) & (blk < hi)).any(dim=1)).flatten() + c0)
            ids = torch.cat(parts)
            pts_of.append(ids)
            a, b = int(d_rp[3 * lo]), int(d_rp[3 * hi])
            out["slabs"].append(dict(lo=lo, hi=hi, q=ids.cpu().numpy(), support=d_sup[ids].cpu().numpy(),
                                     row_ptr=(d_rp[3 * lo:3 * hi + 1].to(torch.int64) - a).cpu().numpy(),
                                     col_idx=d_ci[a:b].to(torch.int64).cpu().numpy(),
                                     vals0=d_vals[a:b].cpu().numpy(), f0=d_f[3 * lo:3 * hi].cpu().numpy(), a=a, b=b))
        if want_shape:
            d_phi = torch.empty((w.Nq, w.k), dtype=torch.float64, device=dev)
            d_dphi = torch.empty((w.Nq, 3, w.k), dtype=torch.float64, device=dev)
            ctx.get_shape(d_phi, d_dphi, None)
            for s, ids in zip(out["slabs"], pts_of):
                s["phi"] = d_phi[ids].cpu().numpy()
                s["dphi"] = d_dphi[ids].cpu().numpy()
            del d_phi, d_dphi
        out["alpha"] = ctx.apply_penalty(torch.from_numpy(w.bc_nodes).to(dev), torch.from_numpy(w.bc_mask).to(dev),
                                         torch.from_numpy(w.bc_ubar).to(dev), w.penalty_alpha, True, d_vals, d_f)
        for s in out["slabs"]:
            s["vals"] = d_vals[s["a"]:s["b"]].cpu().numpy()
            s["f"] = d_f[3 * s["lo"]:3 * s["hi"]].cpu().numpy()
        out["launches"] = ctx.launch_count()
        del d_vals, d_ci, d_rp, d_sup, d_f
    torch.cuda.empty_cache()
    return out


def oracle_rows(w, slab):
    """The oracle on the same slab: supports of the incident points (its own grid search over ALL nodes),
    the CSR rows of the slab's nodes, their values and load entries (row-slab mode of the oracle)."""
    import oracle

    lo, hi = slab["lo"], slab["hi"]
    q = slab["q"]
    pts, qw = np.ascontiguousarray(w.qpts[q]), np.ascontiguousarray(w.qw[q])
    s = oracle.knn(w.nodes, pts, w.k, "grid")
    rp_, ci = oracle.pattern(s, w.N)               # complete for the slab's rows: every incident point is in q
    a, b = rp_[3 * lo], rp_[3 * hi]
    rows_rp = rp_[3 * lo:3 * hi + 1] - a
    rows_ci = ci[a:b]
    phi, dphi, sing = oracle.shape(w.nodes, pts, s, w.alpha_c, w.d_c, w.q)
    vals, f, ns = oracle.assemble(w.nodes, pts, qw, s, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, rows_rp, rows_ci,
                                  node_lo=lo, node_hi=hi)
    return dict(support=s, row_ptr=rows_rp, col_idx=rows_ci, phi=phi, dphi=dphi, vals0=vals, f0=f, nsing=ns)
