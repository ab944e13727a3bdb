"""Helpers shared by the -m gpu parity tests: run the CUDA path through the C ABI binding and the
CPU oracle on the same seeded inputs."""
from __future__ import annotations

import numpy as np


def run_cuda(w, *, penalty=True, loads=True, index_bits=None, want_shape=True, ctx=None, reduction=0, panel_shape=None):
    import torch
    import paper_1802_04256_b200 as rp

    dev = torch.device("cuda:0")
    own = ctx is None
    if own:
        ctx = rp.Context(0)
    out = {}
    try:
        ctx.set_reduction(reduction)
        ctx.set_panel_shape(**(panel_shape or {}))
        d_nodes = torch.from_numpy(w.nodes).to(dev)
        d_qpts = torch.from_numpy(w.qpts).to(dev)
        d_qw = torch.from_numpy(w.qw).to(dev)
        bits_req = w.index_bits if index_bits is None else index_bits
        nnz, bits = ctx.build_pattern(d_nodes, d_qpts, w.k, bits_req)
        idt = torch.int32 if bits == 32 else torch.int64
        cdt = torch.int64 if bits == 64 else torch.int32           # RPIM_INDEX_MIXED (6432): int64 offsets, int32 ids
        d_rp = torch.empty(3 * w.N + 1, dtype=idt, device=dev)
        d_ci = torch.empty(nnz, dtype=cdt, device=dev)
        d_sup = torch.empty((w.Nq, w.k), dtype=torch.int32, device=dev)
        ctx.get_pattern(d_rp, d_ci, d_sup)
        d_vals = torch.full((nnz,), float("nan"), dtype=torch.float64, device=dev)
        d_f = torch.full((3 * w.N,), float("nan"), dtype=torch.float64, device=dev)
        nsing = ctx.assemble(d_qw, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, d_vals, d_f)
        out.update(nnz=nnz, bits=bits, nsing=nsing, phase_ms=ctx.phase_ms(), reduction_used=ctx.reduction_used(),
                   reduction_params=ctx.reduction_params())
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


# ---------------------------------------------------------------------------------------------------
# Full-size parity (BASELINE.json configs 3-5).  The oracle NEVER sees anything computed by the CUDA
# path: it searches the supports of ALL quadrature points itself (in parallel over forked workers),
# the whole support table is compared bit for bit, and the points incident to a row slab are then
# taken from the ORACLE's table.  Every block row of `slope` and `large` is compared (slabs of
# consecutive node ids spread over the workers); `stress` compares sampled slabs.
# ---------------------------------------------------------------------------------------------------
_G = {}   # state inherited (copy-on-write) by the forked oracle workers


def _pool(nproc=None):
    import multiprocessing as mp
    import os
    return mp.get_context("fork").Pool(nproc or max(1, min(os.cpu_count() or 1, 32)))


def _knn_chunk(c):
    import oracle
    w = _G["w"]
    return oracle.knn(w.nodes, w.qpts[c[0]:c[1]], w.k, "grid")


def oracle_support_table(w, pool, chunk=32768):
    """The oracle's supports of all points (its own cell-grid search over all nodes); _G["w"] = w must
    have been set before the pool was forked."""
    cs = [(a, min(a + chunk, w.Nq)) for a in range(0, w.Nq, chunk)]
    return np.concatenate(pool.map(_knn_chunk, cs), axis=0)


def _shape_chunk(c):
    import oracle
    w, S = _G["w"], _G["S"]
    phi, dphi, sing = oracle.shape(w.nodes, w.qpts[c[0]:c[1]], S[c[0]:c[1]], w.alpha_c, w.d_c, w.q)
    return (bool(np.array_equal(phi, _G["phi"][c[0]:c[1]])), bool(np.array_equal(dphi, _G["dphi"][c[0]:c[1]])),
            int(sing.sum()))


def _slab_check(slab):
    """One node slab [lo, hi): the oracle's CSR rows, values and loads against the CUDA path's."""
    import oracle
    w, S = _G["w"], _G["S"]
    lo, hi = slab
    q = np.nonzero(((S >= lo) & (S < hi)).any(axis=1))[0]          # incident points, from the ORACLE's table
    pts, qw, s = np.ascontiguousarray(w.qpts[q]), np.ascontiguousarray(w.qw[q]), np.ascontiguousarray(S[q])
    rp_, ci = oracle.pattern(s, w.N)                                # complete for the slab's rows
    a, b = int(rp_[3 * lo]), int(rp_[3 * hi])
    rows_rp = rp_[3 * lo:3 * hi + 1] - a
    rows_ci = ci[a:b]
    del rp_, ci
    g = _G["rows"](lo, hi)                                          # the CUDA path's rows of this slab (host arrays)
    out = dict(lo=lo, hi=hi, npts=int(q.size), nnz=int(rows_ci.size))
    out["pattern_ok"] = bool(np.array_equal(g["row_ptr"], rows_rp) and np.array_equal(g["col_idx"], rows_ci))
    if not out["pattern_ok"]:
        return out
    vals, f, ns = oracle.assemble(w.nodes, pts, qw, s, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, rows_rp, rows_ci,
                                  node_lo=lo, node_hi=hi)
    rows = np.repeat(np.arange(len(rows_rp) - 1), np.diff(rows_rp))
    diag = rows_ci == rows + 3 * lo
    out.update(nsing=ns, ndiag=int(diag.sum()), km=float(np.abs(vals[diag]).max()),
               err_K=float(np.abs(g["vals0"] - vals).max()), err_f=float(np.abs(g["f0"] - f).max()),
               fmax=float(np.abs(f).max()))
    if "phi" in g:                                                  # sampled mode: shape functions of the slab's points
        phi, dphi, _ = oracle.shape(w.nodes, pts, s, w.alpha_c, w.d_c, w.q)
        out["shape_ok"] = bool(np.array_equal(phi, g["phi"]) and np.array_equal(dphi, g["dphi"]))
    if "Kx" in g:                                                   # product y[rows] = K[rows, :] x from the ORACLE's rows
        import scipy.sparse as sp
        y = sp.csr_matrix((vals, rows_ci, rows_rp), shape=(len(rows_rp) - 1, 3 * w.N)) @ _G["x"]
        out["err_Kx"] = float(np.abs(g["Kx"] - y).max())
    # penalty: exactly the constrained diagonals moved, each by alpha (u_bar = 0 on these configs: f untouched)
    if "vals" in g:
        changed = g["vals"] != g["vals0"]
        expect = np.zeros_like(changed)
        bc = _G["bc"]
        dpos = np.nonzero(diag)[0]
        for r, p in zip(rows[dpos], dpos):
            node, c = divmod(int(r), 3)
            if (bc.get(node + lo, 0) >> c) & 1:
                expect[p] = True
        out["penalty_ok"] = bool(np.array_equal(changed, expect) and np.array_equal(g["f"], g["f0"]) and
                                 (not expect.any() or np.allclose(g["vals"][expect] - g["vals0"][expect],
                                                                  _G["alpha"], rtol=1e-12, atol=0)))
    return out


def gpu_invariants(ctx, w, d_nodes, d_vals, d_f):
    """Whole-matrix properties of the (unpenalised) CUDA result at any size, through rpim_matvec:
    x^T (K y) = y^T (K x), K r = 0 for the six rigid-body modes, sum_I f_I = b * Vol (SURVEY.md 8(c) pins).
    Returns the raw numbers; the caller scales them by max|K_ii|."""
    import torch
    dev = d_vals.device
    n3 = 3 * w.N
    gen = torch.Generator(device="cpu").manual_seed(20240611)
    x = (torch.rand(n3, generator=gen, dtype=torch.float64) * 2 - 1).to(dev)
    y = (torch.rand(n3, generator=gen, dtype=torch.float64) * 2 - 1).to(dev)
    Kx, Ky = torch.empty_like(x), torch.empty_like(y)
    ctx.matvec(d_vals, x, Kx)
    ctx.matvec(d_vals, y, Ky)
    out = dict(x=x.cpu().numpy(), Kx=Kx)
    out["sym"] = float((torch.dot(x, Ky) - torch.dot(y, Kx)).abs() / (x.norm() * Ky.norm()))
    r = d_nodes - d_nodes.mean(dim=0, keepdim=True)
    worst = 0.0
    Km = torch.empty_like(x)
    for c in range(3):
        t = torch.zeros((w.N, 3), dtype=torch.float64, device=dev)
        t[:, c] = 1.0
        e = torch.zeros(3, dtype=torch.float64, device=dev)
        e[c] = 1.0
        for m in (t, torch.linalg.cross(e.expand_as(r), r)):
            m = m.contiguous().view(-1)
            ctx.matvec(d_vals, m, Km)
            worst = max(worst, float(Km.abs().max() / m.abs().max()))
    out["rigid"] = worst                                   # max |K r| / max |r|, to be compared with max|K_ii|
    fs = d_f.view(-1, 3).sum(dim=0).cpu().numpy()
    expect = np.asarray(w.body) * w.volume
    out["fsum_err"] = float(np.abs(fs - expect).max() / max(np.abs(expect).max(), 1e-300))
    # moment resultant about the centroid: sum_I r_I x f_I = sum_q w (r_q x b)  (linear reproduction)
    tq = torch.linalg.cross(r, d_f.view(-1, 3)).sum(dim=0).cpu().numpy()
    xc = d_nodes.mean(dim=0).cpu().numpy()
    texp = np.cross(((w.qpts - xc) * w.qw[:, None]).sum(axis=0), np.asarray(w.body))
    lever = float(np.abs(w.nodes - xc).max()) * max(np.abs(expect).max(), 1e-300)
    out["torque_err"] = float(np.abs(tq - texp).max() / lever)
    out["qw_err"] = float(abs(w.qw.sum() - w.volume) / w.volume)
    # energy identity for linear fields (the oracle's own pin in test_oracle_pins.py):
    # v^T K u = Vol * eps_v^T D eps_u.  Unlike symmetry and the rigid-body modes -- which every single point's
    # w B^T D B satisfies on its own -- this one moves when a point (1 / Nq of the energy) is dropped or doubled.
    lam, mu = w.E * w.nu / ((1 + w.nu) * (1 - 2 * w.nu)), w.E / (2 * (1 + w.nu))
    D = np.zeros((6, 6))
    D[:3, :3] = lam
    D[np.arange(3), np.arange(3)] += 2 * mu
    D[np.arange(3, 6), np.arange(3, 6)] = mu

    def voigt(H):
        e = 0.5 * (H + H.T)
        return np.array([e[0, 0], e[1, 1], e[2, 2], 2 * e[0, 1], 2 * e[1, 2], 2 * e[2, 0]])
    rng = np.random.default_rng(3)
    worst = 0.0
    Ku = torch.empty_like(x)
    for _ in range(6):
        Hu, Hv = rng.standard_normal((3, 3)), rng.standard_normal((3, 3))
        u = (r @ torch.from_numpy(Hu.T).to(dev)).contiguous().view(-1)      # (centred coordinates: a rigid shift of u)
        v = (r @ torch.from_numpy(Hv.T).to(dev)).contiguous().view(-1)
        ctx.matvec(d_vals, u, Ku)
        got = float(torch.dot(v, Ku))
        expect = w.volume * voigt(Hv) @ D @ voigt(Hu)
        scale = w.volume * np.abs(D).max() * np.abs(Hu).max() * np.abs(Hv).max()
        worst = max(worst, abs(got - expect) / scale)
    out["energy_err"] = float(worst)
    return out


def run_full_config(w, *, whole, slabs, want_shape, nproc=None, reduction=0):
    """Full-size run of the CUDA path in the launch configuration bench.py times, compared with the oracle.

    whole=True : every block row (slabs = list of (lo, hi) covering [0, N)), whole matrix brought to the host.
    whole=False: only the given slabs are brought back (config 5 does not fit host-side comparisons of 62 GB).
    Returns a dict of the findings; the test asserts on them."""
    import torch
    import paper_1802_04256_b200 as rp

    dev = torch.device("cuda:0")
    res = {}
    _G["w"] = w                  # the workers are forked by _pool(): everything they read must be set before
    pool = _pool(nproc)
    try:
        S = oracle_support_table(w, pool)
    finally:
        pool.close()
        pool.join()
    with rp.Context(0) as ctx:
        ctx.set_reduction(reduction)
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
        res.update(nnz=nnz, bits=bits, nsing=nsing, reduction_used=ctx.reduction_used())
        # a1 over the WHOLE table, bit for bit
        sup = d_sup.cpu().numpy()
        res["support_equal"] = bool(np.array_equal(sup, S))
        del sup, d_sup
        rp64 = d_rp.to(torch.int64)
        res["row_ptr_monotone"] = bool((rp64[1:] >= rp64[:-1]).all().item()) and int(rp64[0]) == 0 and int(rp64[-1]) == nnz
        del rp64
        inv = gpu_invariants(ctx, w, d_nodes, d_vals, d_f)
        d_Kx = inv.pop("Kx")
        res["invariants"] = {k: v for k, v in inv.items() if k != "x"}
        host = {}
        if whole:
            host["row_ptr"] = d_rp.to(torch.int64).cpu().numpy()
            host["col_idx"] = d_ci.cpu().numpy()
            host["vals0"] = d_vals.cpu().numpy()
            host["f0"] = d_f.cpu().numpy()
            host["Kx"] = d_Kx.cpu().numpy()
            if want_shape:
                d_phi = torch.empty((w.Nq, w.k), dtype=torch.float64, device=dev)
                d_dphi = torch.empty((w.Nq, 3, w.k), dtype=torch.float64, device=dev)
                ctx.get_shape(d_phi, d_dphi, None)
                host["phi"], host["dphi"] = d_phi.cpu().numpy(), d_dphi.cpu().numpy()
                del d_phi, d_dphi
            d_vals0 = d_vals.clone()
        else:
            per = []
            for lo, hi in slabs:
                a, b = int(d_rp[3 * lo]), int(d_rp[3 * hi])
                per.append(dict(a=a, b=b, row_ptr=(d_rp[3 * lo:3 * hi + 1].to(torch.int64) - a).cpu().numpy(),
                                col_idx=d_ci[a:b].to(torch.int64).cpu().numpy(), vals0=d_vals[a:b].cpu().numpy(),
                                f0=d_f[3 * lo:3 * hi].cpu().numpy(), Kx=d_Kx[3 * lo:3 * hi].cpu().numpy()))
            if want_shape:
                d_phi = torch.empty((w.Nq, w.k), dtype=torch.float64, device=dev)
                d_dphi = torch.empty((w.Nq, 3, w.k), dtype=torch.float64, device=dev)
                ctx.get_shape(d_phi, d_dphi, None)
                for (lo, hi), g in zip(slabs, per):
                    q = torch.from_numpy(np.nonzero(((S >= lo) & (S < hi)).any(axis=1))[0]).to(dev)
                    g["phi"], g["dphi"] = d_phi[q].cpu().numpy(), d_dphi[q].cpu().numpy()
                del d_phi, d_dphi
        del d_Kx
        alpha = ctx.apply_penalty(torch.from_numpy(w.bc_nodes).to(dev), torch.from_numpy(w.bc_mask).to(dev),
                                  torch.from_numpy(w.bc_ubar).to(dev), w.penalty_alpha, True, d_vals, d_f)
        res["alpha"] = alpha
        res["launches"] = ctx.launch_count()
        if whole:
            # a7 over the whole matrix, on the device: exactly the constrained diagonals moved, each by alpha
            ch = torch.nonzero(d_vals != d_vals0).flatten()
            res["penalty_changed"] = ch.cpu().numpy()
            res["penalty_delta"] = (d_vals[ch] - d_vals0[ch]).cpu().numpy()
            res["f_untouched"] = bool(torch.equal(d_f.cpu(), torch.from_numpy(host["f0"])))
            del d_vals0
        else:
            for g in per:
                g["vals"] = d_vals[g["a"]:g["b"]].cpu().numpy()
                g["f"] = None
            for (lo, hi), g in zip(slabs, per):
                g["f"] = d_f[3 * lo:3 * hi].cpu().numpy()
        del d_vals, d_ci, d_rp, d_f
    torch.cuda.empty_cache()

    if whole:
        rp_h, ci_h = host["row_ptr"], host["col_idx"]

        def rows(lo, hi):
            a, b = int(rp_h[3 * lo]), int(rp_h[3 * hi])
            return dict(row_ptr=rp_h[3 * lo:3 * hi + 1] - a, col_idx=ci_h[a:b].astype(np.int64, copy=False),
                        vals0=host["vals0"][a:b], f0=host["f0"][3 * lo:3 * hi], Kx=host["Kx"][3 * lo:3 * hi])
    else:
        by = {s: g for s, g in zip(slabs, per)}

        def rows(lo, hi):
            return by[(lo, hi)]
    _G.update(w=w, S=S, rows=rows, x=inv["x"], alpha=alpha,
              bc={int(n): int(m) for n, m in zip(w.bc_nodes, w.bc_mask)})
    if whole and want_shape:
        _G.update(phi=host["phi"], dphi=host["dphi"])
    pool = _pool(nproc)
    try:
        res["slabs"] = pool.map(_slab_check, list(slabs), chunksize=1)
        if whole and want_shape:
            cs = [(a, min(a + 16384, w.Nq)) for a in range(0, w.Nq, 16384)]
            sh = pool.map(_shape_chunk, cs)
            res["phi_equal"] = all(t[0] for t in sh)
            res["dphi_equal"] = all(t[1] for t in sh)
            res["oracle_nsing"] = sum(t[2] for t in sh)
    finally:
        pool.close()
        pool.join()
    if whole:
        # expected positions of the penalty: diagonal entries of the constrained DOFs in the (validated) pattern
        exp = []
        for n, m in zip(w.bc_nodes, w.bc_mask):
            for c in range(3):
                if (int(m) >> c) & 1:
                    d = 3 * int(n) + c
                    a, b = int(rp_h[d]), int(rp_h[d + 1])
                    exp.append(a + int(np.searchsorted(ci_h[a:b], d)))
        res["penalty_expected"] = np.sort(np.asarray(exp, dtype=np.int64))
    _G.clear()
    return res
