"""-m gpu parity of stage 3: rpim_matvec, rpim_solve_pcg (block-Jacobi PCG) and
rpim_recover_stress against oracle/stage3.py (sparse direct solve, literal B and D) on the oracle's own K.

Tolerances: the product is compared at 1e-12 of max|K x|; the solution at 1e-6 of
max|u| (PCG stops at a relative residual of 1e-12, the Jacobi-scaled penalised matrices of these cases
have condition numbers of 1e4..1e5); stresses at 1e-6 of max|sigma|."""
import json
import os

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


def _gpu(w, with_loads=False):
    import torch
    import paper_1802_04256_b200 as rp

    dev = torch.device("cuda:0")
    out = {}
    with rp.Context(0) as ctx:
        d_nodes, d_qpts, d_qw = (torch.from_numpy(a).to(dev) for a in (w.nodes, w.qpts, w.qw))
        nnz, bits = ctx.build_pattern(d_nodes, d_qpts, w.k, w.index_bits)
        d_vals = torch.empty(nnz, dtype=torch.float64, device=dev)
        d_f = torch.empty(3 * w.N, dtype=torch.float64, device=dev)
        ctx.assemble(d_qw, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, d_vals, d_f)
        if with_loads:
            ctx.add_point_loads(torch.from_numpy(w.load_pts).to(dev), torch.from_numpy(w.load_w).to(dev),
                                torch.from_numpy(w.load_t).to(dev), d_f)
        ctx.apply_penalty(torch.from_numpy(w.bc_nodes).to(dev), torch.from_numpy(w.bc_mask).to(dev),
                          torch.from_numpy(w.bc_ubar).to(dev), w.penalty_alpha, True, d_vals, d_f)
        rng = np.random.default_rng(1)
        x = rng.standard_normal(3 * w.N)
        d_y = torch.empty(3 * w.N, dtype=torch.float64, device=dev)
        ctx.matvec(d_vals, torch.from_numpy(x).to(dev), d_y)
        out["x"], out["y"] = x, d_y.cpu().numpy()
        d_u = torch.zeros(3 * w.N, dtype=torch.float64, device=dev)
        out["iters"], out["relres"] = ctx.solve_pcg(d_vals, d_f, d_u, 1e-12, 50000)
        u1 = d_u.cpu().numpy()
        d_u.zero_()
        ctx.solve_pcg(d_vals, d_f, d_u, 1e-12, 50000)
        out["u"], out["u_again"] = u1, d_u.cpu().numpy()
        d_sig = torch.empty((w.Nq, 6), dtype=torch.float64, device=dev)
        ctx.recover_stress(d_u, w.E, w.nu, d_sig)
        out["sigma"] = d_sig.cpu().numpy()
    return out


def _oracle(w, with_loads=False):
    import oracle
    from oracle import stage3

    s = oracle.knn(w.nodes, w.qpts, w.k, "grid")
    rp_, ci = oracle.pattern(s, w.N)
    vals, f, _ = oracle.assemble(w.nodes, w.qpts, w.qw, s, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, rp_, ci)
    if with_loads:
        ls = oracle.knn(w.nodes, w.load_pts, w.k, "grid")
        oracle.point_loads(w.nodes, w.load_pts, w.load_w, w.load_t, ls, w.alpha_c, w.d_c, w.q, f)
    oracle.penalty(w.bc_nodes, w.bc_mask, w.bc_ubar, w.penalty_alpha, True, w.N, rp_, ci, vals, f)
    u = stage3.solve(rp_, ci, vals, f)
    _, dphi, _ = oracle.shape(w.nodes, w.qpts, s, w.alpha_c, w.d_c, w.q)
    return dict(rp=rp_, ci=ci, vals=vals, f=f, u=u, sigma=stage3.stress(s, dphi, u, w.E, w.nu))


def _compare(w, g, o):
    from oracle import stage3
    y = stage3.matvec(o["rp"], o["ci"], o["vals"], g["x"])
    assert np.abs(g["y"] - y).max() <= 1e-12 * np.abs(y).max()
    # the loop stops on the residual RECURRENCE (1e-12 asked for); what is reported is the TRUE ||f - K u|| / ||f||
    # of the returned iterate, which a penalty-stiffened K (alpha = 1e8 max K_ii) holds at ~1e-10 (measured 1.6e-10)
    assert g["relres"] <= 1e-9 and g["iters"] > 0
    assert np.array_equal(g["u"], g["u_again"])                               # fixed-order reductions
    assert np.abs(g["u"] - o["u"]).max() <= 1e-6 * np.abs(o["u"]).max()
    assert np.abs(g["sigma"] - o["sigma"]).max() <= 1e-6 * np.abs(o["sigma"]).max()


def test_patch_solve_and_stress():
    w = workloads.config("patch")
    _compare(w, _gpu(w), _oracle(w))


def test_cantilever_solve_stress_and_tip_deflection():
    w = workloads.config("cantilever")
    g, o = _gpu(w, True), _oracle(w, True)
    _compare(w, g, o)
    tip = g["u"].reshape(-1, 3)[np.isclose(w.nodes[:, 0], 10.0), 2].mean()
    euler = -1e6 * 10.0 ** 3 / (3 * w.E / 12.0)
    timo = euler - 1e6 * 10.0 / ((5.0 / 6.0) * w.E / (2 * (1 + w.nu)))
    assert min(abs(tip - euler) / abs(euler), abs(tip - timo) / abs(timo)) < 0.01


def test_gravity_column_bottom_stress_of_the_paper():
    g0 = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_example1.json")))
    rho, grav, H, n = g0["density_kg_m3"], g0["inferred"]["g"], g0["inferred"]["height_m"], 9
    w = workloads.make_block("cube", n, n, n, H / (n - 1), 2, 27, 20e9, 0.25, jitter=0.2, seed=4,
                             body=(0.0, 0.0, -rho * grav), bc="bottom+roller")
    g, o = _gpu(w), _oracle(w)
    _compare(w, g, o)
    low = w.qpts[:, 2] < 0.5 * H / (n - 1)
    est = -(g["sigma"][low, 2].mean() + rho * grav * (H - w.qpts[low, 2]).mean()) + rho * grav * H
    assert abs(est / 1e6 - g0["theoretical_bottom_stress_MPa"]) / g0["theoretical_bottom_stress_MPa"] < 0.03


def test_pcg_reports_the_true_residual_handles_zero_load_and_flags_breakdown():
    import torch
    import paper_1802_04256_b200 as rp
    w = workloads.make_block("pcg", 8, 7, 6, 1.0, 2, 30, 5e9, 0.3, jitter=0.3, seed=12, body=(0.0, 0.0, -2.5e4),
                             bc="bottom")
    dev = torch.device("cuda:0")
    with rp.Context(0) as ctx:
        d_nodes, d_qpts = torch.from_numpy(w.nodes).to(dev), torch.from_numpy(w.qpts).to(dev)   # must outlive the pattern
        nnz, _ = ctx.build_pattern(d_nodes, d_qpts, w.k)
        vals = torch.empty(nnz, dtype=torch.float64, device=dev)
        f = torch.empty(3 * w.N, dtype=torch.float64, device=dev)
        ctx.assemble(torch.from_numpy(w.qw).to(dev), w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, vals, f)
        ctx.apply_penalty(torch.from_numpy(w.bc_nodes).to(dev), torch.from_numpy(w.bc_mask).to(dev),
                          torch.from_numpy(w.bc_ubar).to(dev), w.penalty_alpha, True, vals, f)
        # stopped early on purpose: the reported number must be ||f - K u|| / ||f|| of the returned iterate
        u = torch.zeros_like(f)
        iters, rel = ctx.solve_pcg(vals, f, u, 1e-30, 50)
        assert iters == 50
        Ku = torch.empty_like(f)
        ctx.matvec(vals, u, Ku)
        true_rel = float((f - Ku).norm() / f.norm())
        assert abs(rel - true_rel) <= 1e-10 * true_rel
        # f = 0: u = 0 whatever the initial guess
        u = torch.ones_like(f)
        iters, rel = ctx.solve_pcg(vals, torch.zeros_like(f), u, 1e-10, 100)
        assert iters == 0 and rel == 0.0 and not u.any()
        # a matrix that is not positive definite (here -K): breakdown is detected and reported, no spinning
        u = torch.zeros_like(f)
        with pytest.raises(rp.RpimError) as e:
            ctx.solve_pcg(-vals, f, u, 1e-10, 10000)
        assert e.value.code == -8
        # a load vector with a NaN is not "f = 0": no converged solve is reported, and the guess is left alone
        fn = f.clone()
        fn[5] = float("nan")
        u = torch.full_like(f, 3.0)
        with pytest.raises(rp.RpimError) as e:
            ctx.solve_pcg(vals, fn, u, 1e-10, 100)
        assert e.value.code == -8 and "finite" in str(e.value)
        assert bool((u == 3.0).all())
