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
