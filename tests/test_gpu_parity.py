"""-m gpu parity tests: the CUDA path (through the C ABI binding) against the CPU oracle on the same
seeded inputs.  Bars (BASELINE.json north_star): supports and CSR pattern bit-exact; K and f within
1e-10 relative, per entry, scaled by max|K_ii| (of the matrix compared).  Shape functions are
compared BITWISE: DESIGN.md section 2 specifies the per-point stage at the operation level."""
import numpy as np
import pytest

import workloads
from gpu_harness import kmax_diag, run_cuda, run_oracle

pytestmark = pytest.mark.gpu

TOL = 1e-10


def _compare(w, g, o, check_penalty=True):
    assert np.array_equal(g["support"], o["support"])                     # a1 bit-exact
    assert g["row_ptr"].dtype == (np.int32 if g["bits"] == 32 else np.int64)
    assert np.array_equal(g["row_ptr"].astype(np.int64), o["row_ptr"])    # a2 bit-exact
    assert np.array_equal(g["col_idx"].astype(np.int64), o["col_idx"])
    assert g["nsing"] == o["nsing"]
    assert np.array_equal(g["singular"], o["singular"])
    assert np.array_equal(g["phi"], o["phi"])                             # a3+a4 bitwise
    assert np.array_equal(g["dphi"], o["dphi"])
    km = kmax_diag(o)
    assert np.abs(g["vals0"] - o["vals0"]).max() <= TOL * km              # a5+a6
    fs = max(np.abs(o["f_loaded"]).max(), 1e-300)
    assert np.abs(g["f0"] - o["f0"]).max() <= TOL * max(np.abs(o["f0"]).max(), 1e-300)
    assert np.abs(g["f_loaded"] - o["f_loaded"]).max() <= TOL * fs        # a5b
    if check_penalty:                                                      # a7
        assert abs(g["alpha"] - o["alpha"]) <= 1e-13 * o["alpha"]
        km_pen = max(km, np.abs(o["vals"]).max())
        assert np.abs(g["vals"] - o["vals"]).max() <= TOL * km_pen
        changed = g["vals"] != g["vals0"]
        ochanged = o["vals"] != o["vals0"]
        assert np.array_equal(changed, ochanged)                           # exactly the constrained diagonals
        assert np.allclose(g["vals"][changed] - g["vals0"][changed], g["alpha"], rtol=1e-12, atol=0)
        assert np.abs(g["f"] - o["f"]).max() <= TOL * max(np.abs(o["f"]).max(), 1e-300)


def test_config1_patch_full_parity():
    w = workloads.config("patch")
    _compare(w, run_cuda(w), run_oracle(w))


def test_config2_cantilever_full_parity_with_traction_and_penalty():
    w = workloads.config("cantilever")
    g, o = run_cuda(w), run_oracle(w)
    _compare(w, g, o)
    assert abs(g["f_loaded"].reshape(-1, 3).sum(0)[2] + 1e6) < 1e-6       # total end shear = -1e6 N


@pytest.mark.parametrize("k,dims,jit,gauss", [
    (4, (5, 4, 4), 0.3, 1),        # smallest k: n = 8, only the four 2x2 pivots
    (8, (6, 5, 5), 0.2, 1),
    (27, (7, 7, 6), 0.25, 2),
    (33, (8, 7, 7), 0.3, 2),       # k just over one warp
    (40, (9, 8, 7), 0.3, 2),
    (60, (10, 9, 8), 0.3, 2),
    (64, (9, 9, 8), 0.3, 1),
    (124, (9, 8, 8), 0.3, 1),      # maximum k: 128 x 128 moment systems
])
def test_jittered_blocks_span_tiles_and_ragged_tails(k, dims, jit, gauss):
    # with k = 4 some boundary nodes belong to no support (no matrix row): use an empty BC list there,
    # which also covers the m = 0 edge case of rpim_apply_penalty
    w = workloads.make_block(f"j{k}", *dims, 1.0, gauss, k, 5e9, 0.3, jitter=jit, seed=100 + k,
                             body=(10.0, -20.0, -2.5e4), bc="none" if k == 4 else "bottom+roller")
    _compare(w, run_cuda(w), run_oracle(w))


@pytest.mark.parametrize("k,dims,gauss", [
    (27, (7, 7, 6), 2),            # union of a cell's 8 supports: 2 chunks of 32; odd k
    (40, (9, 8, 7), 2),            # 3 chunks
    (60, (10, 9, 8), 2),           # 4 chunks, rows of ~400 block columns
    (30, (9, 5, 5), 3),            # 27 points per cell: groups of 8 straddle cells
    (124, (9, 8, 8), 2),           # unions beyond the 128-node limit: the row-owner kernel takes over
    (64, (9, 9, 8), 2),
    (12, (6, 6, 5), 1),            # one point per cell: sparse groups, still correct
])
def test_panel_reduction_matches_the_oracle_and_the_row_owner_kernel(k, dims, gauss):
    # rpim_set_reduction(ctx, 2): groups of 8 points, tiles of rows, accumulators in shared memory, group panels
    # through a bulk-copy ring (reduce_panels.cu).  Same bars as the default path; run twice for bitwise reproducibility.
    w = workloads.make_block(f"t{k}", *dims, 1.0, gauss, k, 5e9, 0.3, jitter=0.3, seed=300 + k,
                             body=(10.0, -20.0, -2.5e4), bc="bottom+roller")
    g, o = run_cuda(w, reduction=2), run_oracle(w)
    assert g["reduction_used"] == (1 if k == 124 else 2)
    _compare(w, g, o)
    g2 = run_cuda(w, reduction=2)
    assert np.array_equal(g["vals"], g2["vals"]) and np.array_equal(g["f"], g2["f"])
    g1 = run_cuda(w, reduction=1)
    assert g1["reduction_used"] == 1
    km = kmax_diag(o)
    assert np.abs(g["vals0"] - g1["vals0"]).max() <= 1e-13 * km


def test_nonunit_spacing_other_exponent_and_absolute_penalty():
    w = workloads.make_block("q", 8, 7, 6, 0.37, 2, 30, 7e9, 0.33, jitter=0.25, seed=3, q=1.5, alpha_c=3.0,
                             body=(0.0, 0.0, -1.0), bc="x0")
    _compare(w, run_cuda(w), run_oracle(w))


def test_run_to_run_bitwise_determinism_and_index_width():
    w = workloads.make_block("det", 10, 9, 8, 1.0, 2, 40, 5e9, 0.3, jitter=0.3, seed=8,
                             body=(0.0, 0.0, -2.5e4), bc="bottom")
    a = run_cuda(w, index_bits=32)
    b = run_cuda(w, index_bits=64)
    c = run_cuda(w, index_bits=0)
    assert a["bits"] == 32 and b["bits"] == 64 and c["bits"] == 32
    assert a["row_ptr"].dtype == np.int32 and b["row_ptr"].dtype == np.int64
    assert np.array_equal(a["row_ptr"], b["row_ptr"]) and np.array_equal(a["col_idx"], b["col_idx"])
    for key in ("vals", "f", "vals0", "phi", "dphi"):
        assert np.array_equal(a[key], b[key]) and np.array_equal(a[key], c[key])
    assert a["launches"] > 0
    # mixed widths (RPIM_INDEX_MIXED): 64-bit row offsets, 32-bit column ids, same pattern and values; also through
    # the host-buffer entry points
    import paper_1802_04256_b200 as rp
    m = run_cuda(w, index_bits=rp.RPIM_INDEX_MIXED)
    assert m["bits"] == rp.RPIM_INDEX_MIXED and m["row_ptr"].dtype == np.int64 and m["col_idx"].dtype == np.int32
    assert np.array_equal(m["row_ptr"], b["row_ptr"]) and np.array_equal(m["col_idx"], b["col_idx"])
    assert np.array_equal(m["vals"], b["vals"]) and np.array_equal(m["f"], b["f"])
    with rp.Context(0) as ctx:
        nnz, bits = ctx.host_pattern(w.nodes, w.qpts, w.k, rp.RPIM_INDEX_MIXED)
        assert bits == rp.RPIM_INDEX_MIXED and nnz == b["nnz"]
        rpa, cia = np.full(3 * w.N + 1, -1, np.int64), np.full(nnz, -1, np.int32)
        vals, f = np.empty(nnz), np.empty(3 * w.N)
        ctx.host_assemble(w.qw, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, w.bc_nodes, w.bc_mask, w.bc_ubar,
                          w.penalty_alpha, True, rpa, cia, vals, f)
        assert np.array_equal(rpa, b["row_ptr"]) and np.array_equal(cia, b["col_idx"])
        assert np.array_equal(vals, b["vals"]) and np.array_equal(f, b["f"])
        with pytest.raises(rp.RpimError) as e:
            ctx.host_pattern(w.nodes, w.qpts, w.k, 48)
        assert e.value.code == -1


def test_shuffled_node_numbering():
    # 69,120 nodes numbered at random (no spatial coherence of the ids: hash tables, incidence lists and
    # the cell grid must not rely on it; also the largest parity case the oracle finishes in seconds).
    # Same bars as everywhere else.
    w = workloads.make_block("shuf", 48, 40, 36, 1.0, 1, 8, 5e9, 0.3, jitter=0.3, seed=77,
                             body=(0.0, 0.0, -2.5e4), bc="bottom")
    rng = np.random.default_rng(5)
    perm = rng.permutation(w.N)                 # new id i holds old node perm[i]
    inv = np.empty_like(perm)
    inv[perm] = np.arange(w.N)
    w.nodes = np.ascontiguousarray(w.nodes[perm])
    nb = inv[w.bc_nodes]
    order = np.argsort(nb)
    w.bc_nodes = np.ascontiguousarray(nb[order]).astype(np.int64)
    w.bc_mask = np.ascontiguousarray(w.bc_mask[order])
    w.bc_ubar = np.ascontiguousarray(w.bc_ubar[order])
    _compare(w, run_cuda(w), run_oracle(w))


def test_degenerate_sizes_single_point_and_k_equal_N():
    # one quadrature point only; and every node in every support (k = N): one dense block row per node
    w = workloads.make_block("one", 5, 4, 4, 1.0, 1, 20, 3e9, 0.3, jitter=0.2, seed=9, body=(1.0, 2.0, -3.0), bc="none")
    w.qpts = np.ascontiguousarray(w.qpts[7:8])
    w.qw = np.ascontiguousarray(w.qw[7:8])
    _compare(w, run_cuda(w, penalty=False), run_oracle(w, penalty=False), check_penalty=False)
    w = workloads.make_block("kN", 4, 3, 3, 1.0, 2, 36, 3e9, 0.3, jitter=0.25, seed=10, body=(0.0, 0.0, -1e4), bc="bottom")
    assert w.N == w.k
    g, o = run_cuda(w), run_oracle(w)
    _compare(w, g, o)
    assert g["nnz"] == 9 * w.N * w.N


def test_one_context_serves_problems_of_changing_size():
    # the workspace cache hands blocks from earlier, differently sized problems back out: results must not
    # depend on what the context did before
    import paper_1802_04256_b200 as rp
    cases = [workloads.make_block("c1", 9, 8, 7, 1.0, 2, 30, 5e9, 0.3, jitter=0.3, seed=31, body=(0.0, 0.0, -2.5e4), bc="bottom"),
             workloads.make_block("c2", 5, 5, 4, 0.5, 1, 12, 2e9, 0.2, jitter=0.2, seed=32, body=(1.0, 0.0, -1e4), bc="x0"),
             workloads.make_block("c3", 10, 9, 9, 1.0, 2, 40, 5e9, 0.3, jitter=0.3, seed=33, body=(0.0, 0.0, -2.5e4), bc="bottom+roller"),
             workloads.make_block("c1", 9, 8, 7, 1.0, 2, 30, 5e9, 0.3, jitter=0.3, seed=31, body=(0.0, 0.0, -2.5e4), bc="bottom")]
    with rp.Context(0) as ctx:
        outs = [run_cuda(w, ctx=ctx) for w in cases]
    for w, g in zip(cases[:3], outs[:3]):
        _compare(w, g, run_oracle(w))
    for key in ("vals", "f", "col_idx", "phi", "dphi"):
        assert np.array_equal(outs[0][key], outs[3][key]), key       # same problem again: same bits


def test_planar_cloud_every_point_is_singular():
    nodes = np.array([[i, j, 0.0] for j in range(6) for i in range(6)], dtype=np.float64)
    w = workloads.make_block("flat", 6, 6, 2, 1.0, 1, 12, 1e9, 0.3)
    w.nodes = nodes
    w.qpts = np.ascontiguousarray(w.qpts[:25] * np.array([1.0, 1.0, 0.0]))
    w.qw = np.ascontiguousarray(w.qw[:25])
    w.bc_nodes = np.array([0, 1], dtype=np.int64)
    w.bc_mask = np.array([7, 7], dtype=np.uint8)
    w.bc_ubar = np.zeros((2, 3))
    g, o = run_cuda(w, penalty=False), run_oracle(w, penalty=False)
    assert g["nsing"] == o["nsing"] == 25
    assert np.array_equal(g["support"], o["support"])
    assert not g["vals"].any() and not g["phi"].any()


def test_error_codes():
    import torch
    import paper_1802_04256_b200 as rp
    w = workloads.make_block("e", 4, 4, 4, 1.0, 1, 8, 1e9, 0.3)
    dev = torch.device("cuda:0")
    dn, dq = torch.from_numpy(w.nodes).to(dev), torch.from_numpy(w.qpts).to(dev)
    with rp.Context(0) as ctx:
        with pytest.raises(rp.RpimError) as e:
            ctx.build_pattern(dn, dq, 3)
        assert e.value.code == -1
        with pytest.raises(rp.RpimError) as e:
            ctx.build_pattern(dn, dq, 65)          # k > N = 64
        assert e.value.code == -1
        with pytest.raises(rp.RpimError) as e:
            ctx.assemble(torch.from_numpy(w.qw).to(dev), 1e9, 0.3, 4.0, 1.0, 1.03, (0, 0, 0),
                         torch.empty(1, dtype=torch.float64, device=dev),
                         torch.empty(1, dtype=torch.float64, device=dev))
        assert e.value.code == -4                  # state: no pattern yet
        nnz, bits = ctx.build_pattern(dn, dq, 8)
        vals = torch.empty(nnz, dtype=torch.float64, device=dev)
        f = torch.empty(3 * w.N, dtype=torch.float64, device=dev)
        ctx.assemble(torch.from_numpy(w.qw).to(dev), 1e9, 0.3, 4.0, 1.0, 1.03, (0, 0, 0), vals, f)
        bad = torch.tensor([1, 64], dtype=torch.int64, device=dev)
        with pytest.raises(rp.RpimError) as e:
            ctx.apply_penalty(bad, None, torch.zeros((2, 3), dtype=torch.float64, device=dev), 1.0, False, vals, f)
        assert e.value.code == -5
        assert ctx.workspace_bytes() > 0
        # rpim_set_panel_shape: out-of-range values are refused and change nothing
        for bad_shape in (dict(rows_per_tile=3), dict(rows_per_tile=10), dict(warps_per_group=5), dict(rows_per_group=3),
                          dict(ring_stages=1), dict(ring_stages=9), dict(staging=3), dict(tile_desc=-1)):
            with pytest.raises(rp.RpimError) as e:
                ctx.set_panel_shape(**bad_shape)
            assert e.value.code == -1
        ctx.set_panel_shape()                      # all automatic


def test_host_buffer_entry_points_match_device_path():
    import paper_1802_04256_b200 as rp
    w = workloads.make_block("h", 9, 8, 7, 1.0, 2, 30, 5e9, 0.3, jitter=0.3, seed=21, body=(0.0, 0.0, -2.5e4),
                             bc="bottom+roller")
    g = run_cuda(w)
    with rp.Context(0) as ctx:
        nnz, bits = ctx.host_pattern(w.nodes, w.qpts, w.k, 0)
        idt = np.int32 if bits == 32 else np.int64
        rpa, cia = np.empty(3 * w.N + 1, idt), np.empty(nnz, idt)
        vals, f = np.empty(nnz), np.empty(3 * w.N)
        ns, alpha = ctx.host_assemble(w.qw, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, w.bc_nodes, w.bc_mask,
                                      w.bc_ubar, w.penalty_alpha, True, rpa, cia, vals, f)
    assert ns == 0 and alpha == g["alpha"]
    assert np.array_equal(rpa, g["row_ptr"]) and np.array_equal(cia, g["col_idx"])
    assert np.array_equal(vals, g["vals"]) and np.array_equal(f, g["f"])


def test_long_row_kernel_matches_the_oracle():
    # accumulate_generic_kernel (rows of more than 1024 block columns take it automatically) forced on a small
    # case through rpim_set_reduction(ctx, 3): same bars as the default kernels
    w = workloads.make_block("gen", 9, 8, 7, 1.0, 2, 33, 5e9, 0.3, jitter=0.3, seed=41, body=(3.0, -2.0, -2.5e4),
                             bc="bottom+roller")
    g = run_cuda(w, reduction=3)
    assert g["reduction_used"] == 1
    _compare(w, g, run_oracle(w))


def test_boundary_list_is_validated_before_anything_is_applied():
    import torch
    import paper_1802_04256_b200 as rp
    w = workloads.make_block("dup", 6, 5, 5, 1.0, 1, 12, 1e9, 0.3, jitter=0.2, seed=5, body=(0.0, 0.0, -1.0))
    dev = torch.device("cuda:0")
    with rp.Context(0) as ctx:
        d_nodes, d_qpts = torch.from_numpy(w.nodes).to(dev), torch.from_numpy(w.qpts).to(dev)   # must outlive the pattern
        nnz, _ = ctx.build_pattern(d_nodes, d_qpts, w.k)
        vals = torch.empty(nnz, dtype=torch.float64, device=dev)
        f = torch.empty(3 * w.N, dtype=torch.float64, device=dev)
        ctx.assemble(torch.from_numpy(w.qw).to(dev), w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, vals, f)
        v0, f0 = vals.clone(), f.clone()
        ub = torch.full((3, 3), 0.5, dtype=torch.float64, device=dev)
        for bad in ([3, 7, 3], [3, -1, 4], [3, w.N, 4]):       # listed twice, negative, out of range
            with pytest.raises(rp.RpimError) as e:
                ctx.apply_penalty(torch.tensor(bad, dtype=torch.int64, device=dev), None, ub, 1e3, False, vals, f)
            assert e.value.code == -5
            assert torch.equal(vals, v0) and torch.equal(f, f0)    # nothing applied
        a = ctx.apply_penalty(torch.tensor([3, 7, 4], dtype=torch.int64, device=dev), None, ub, 1e3, False, vals, f)
        assert a == 1e3 and int((vals != v0).sum()) == 9 and int((f != f0).sum()) == 9


def test_point_loads_report_singular_load_points():
    import torch
    import paper_1802_04256_b200 as rp
    # two far-apart node planes (z = 0 and z = 10): the 12 nearest nodes of a point ON the plane z = 0 are coplanar
    w = workloads.make_block("face", 6, 6, 2, 1.0, 1, 12, 1e9, 0.3, body=(0.0, 0.0, -1.0))
    w.nodes[:, 2] *= 10.0
    w.qpts[:, 2] *= 10.0
    dev = torch.device("cuda:0")
    with rp.Context(0) as ctx:
        d_nodes, d_qpts = torch.from_numpy(w.nodes).to(dev), torch.from_numpy(w.qpts).to(dev)   # must outlive the pattern
        nnz, _ = ctx.build_pattern(d_nodes, d_qpts, w.k)
        vals = torch.empty(nnz, dtype=torch.float64, device=dev)
        f = torch.empty(3 * w.N, dtype=torch.float64, device=dev)
        ctx.assemble(torch.from_numpy(w.qw).to(dev), w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, vals, f)
        f0 = f.clone()
        pts = torch.tensor([[2.5, 2.5, 0.0]], dtype=torch.float64, device=dev)       # on the face z = 0
        one = torch.ones(1, dtype=torch.float64, device=dev)
        t = torch.tensor([[0.0, 0.0, -1.0]], dtype=torch.float64, device=dev)
        with pytest.raises(rp.RpimError) as e:
            ctx.add_point_loads(pts, one, t, f)
        assert e.value.code == -9 and torch.equal(f, f0)
        pts_ok = torch.tensor([[2.5, 2.5, 5.0]], dtype=torch.float64, device=dev)    # between the planes: regular
        ctx.add_point_loads(pts_ok, one, t, f)                                       # the flags were cleared
        assert abs(float((f - f0).view(-1, 3).sum(0)[2]) + 1.0) < 1e-12


@pytest.mark.parametrize("idx", range(4))
@pytest.mark.parametrize("reduction", [1, 2])
def test_cuda_K_against_the_plain_definition(idx, reduction):
    """The CUDA K and f against the DEFINITION (oracle.assemble_dense_ref: plain moment matrix in global
    coordinates, powl, partial-pivoting LU, literal B and D, long double throughout), not the operation-level
    recipe both sides transcribe: configs 1 and 2 and jittered k = 40 / k = 60 blocks, both reduction kernels.
    Bar: the definition-level tolerance of tests/test_oracle_definition.py (about 10x the measured error, under
    the a-priori bound 2 cond(G) eps of the moment systems)."""
    from test_oracle_definition import DEF_TOL, definition_K, definition_cases
    w = definition_cases()[idx]
    s, rp, ci, vr, fr, km = definition_K(w)
    g = run_cuda(w, penalty=False, loads=False, reduction=reduction)
    assert np.array_equal(g["support"], s)
    assert np.array_equal(g["row_ptr"].astype(np.int64), rp) and np.array_equal(g["col_idx"].astype(np.int64), ci)
    err = np.abs(g["vals0"] - vr).max() / km
    ferr = np.abs(g["f0"] - fr).max() / max(np.abs(fr).max(), 1e-300)
    print(f"{w.name}: k={w.k} reduction={g['reduction_used']} CUDA vs definition: max|dK|/max|K_ii| = {err:.3e}, f {ferr:.3e}")
    assert err <= DEF_TOL[w.k] and (ferr <= DEF_TOL[w.k] or np.abs(fr).max() == 0.0)


@pytest.mark.parametrize("shape", [
    dict(rows_per_group=2, warps_per_group=3),                       # row pairs sharing the gradient loads
    dict(rows_per_group=2, warps_per_group=1, rows_per_tile=2),      # one warp takes all chunks of its pair
    dict(rows_per_group=1, warps_per_group=1, ring_stages=2),
    dict(rows_per_group=1, warps_per_group=3, rows_per_tile=4),
    dict(tile_desc=2),     # the descriptor kernel large problems take (one thread per tile)
    dict(staging=1),       # gradient rows by the 2-D tensor copy
    dict(staging=2),       # whole staged rows by a plain bulk copy
])
def test_panel_reduction_launch_shapes(shape):
    """The other launch shapes of reduce_panels_kernel (rows per warp group, warps per group, rows per tile, ring
    depth, staging; forced through rpim_set_panel_shape): same bars, and bitwise the same K as the default
    shape (the order of summation per entry does not depend on the launch shape)."""
    w = workloads.make_block("shape60", 10, 9, 8, 1.0, 2, 60, 5e9, 0.3, jitter=0.3, seed=360,
                             body=(10.0, -20.0, -2.5e4), bc="bottom+roller")
    g0, o = run_cuda(w, reduction=2), run_oracle(w)
    g = run_cuda(w, reduction=2, panel_shape=shape)
    assert g["reduction_used"] == 2
    used = g["reduction_params"]
    for key, name in (("rows_per_tile", "rows_per_tile"), ("warps_per_group", "warps_per_row_group"),
                      ("rows_per_group", "rows_per_warp_group"), ("ring_stages", "ring_stages")):
        assert key not in shape or used[name] == shape[key], (key, used)
    assert "staging" not in shape or used["tensor_copy_staging"] == (1 if shape["staging"] == 1 else 0)
    _compare(w, g, o)
    assert np.array_equal(g["vals"], g0["vals"]) and np.array_equal(g["f"], g0["f"])


@pytest.mark.parametrize("q,alpha_c", [(0.5, 4.0), (0.5, 1.5), (-0.5, 4.0)])
def test_classic_and_inverse_multiquadric(q, alpha_c):
    """the other members of the radial family R = (r^2 + c^2)^q go through the same
    kernels (classic multiquadric q = 1/2, inverse multiquadric q = -1/2); same bars, shape functions bitwise."""
    w = workloads.make_block(f"mq{q}", 9, 8, 7, 1.0, 2, 30, 5e9, 0.3, jitter=0.3, seed=77, q=q, alpha_c=alpha_c,
                             body=(10.0, -20.0, -2.5e4), bc="bottom+roller")
    _compare(w, run_cuda(w), run_oracle(w))


def test_graded_density_supports_and_pattern():
    """A cloud whose local density is hundreds of times the mean (a 16^3 cluster of spacing 0.05 inside a unit-spaced
    block): the 5 x 5 x 5 ring of grid cells around a query holds more nodes than the largest on-chip candidate
    buffer, so the queries fall through to the last tier of the support search (own cell outwards, streaming
    selection without a capacity limit).  Supports and CSR pattern must still equal the oracle's bit for bit."""
    import torch
    import oracle
    import paper_1802_04256_b200 as rp
    rng = np.random.default_rng(5)
    w = workloads.make_block("graded", 8, 8, 6, 1.0, 1, 30, 5e9, 0.3, jitter=0.3, seed=9)
    g = (np.stack(np.meshgrid(*[np.arange(16)] * 3, indexing="ij"), -1).reshape(-1, 3) * 0.05 + np.array([3.1, 3.2, 2.1])
         + rng.uniform(-0.01, 0.01, (4096, 3)))
    nodes = np.ascontiguousarray(np.concatenate([w.nodes, g]))
    pts = np.ascontiguousarray(np.concatenate([w.qpts, g[::7] + 0.013, rng.uniform([2.5, 2.6, 1.5], [4.5, 4.6, 3.5], (300, 3))]))
    k = 30
    s = oracle.knn(nodes, pts, k, "brute")
    rp_o, ci_o = oracle.pattern(s, nodes.shape[0])
    dev = torch.device("cuda:0")
    ctx = rp.Context(0)
    try:
        d_n, d_q = torch.from_numpy(nodes).to(dev), torch.from_numpy(pts).to(dev)
        nnz, bits = ctx.build_pattern(d_n, d_q, k, 64)
        d_rp = torch.empty(3 * nodes.shape[0] + 1, dtype=torch.int64, device=dev)
        d_ci = torch.empty(nnz, dtype=torch.int64, device=dev)
        d_sup = torch.empty((pts.shape[0], k), dtype=torch.int32, device=dev)
        ctx.get_pattern(d_rp, d_ci, d_sup)
        assert np.array_equal(d_sup.cpu().numpy(), s)
        assert np.array_equal(d_rp.cpu().numpy(), rp_o) and np.array_equal(d_ci.cpu().numpy(), ci_o)
    finally:
        ctx.close()


@pytest.mark.parametrize("reduction", [1, 2])
def test_strata_modulus_scale(reduction):
    """DESIGN.md R8b (part): per-point modulus scale E_q = E s_q with one Poisson ratio, both
    reduction kernels, against the oracle; the loads do not change; rpim_recover_stress scales with s_q; switching
    the scale off restores the unscaled matrix bit for bit."""
    import torch
    import oracle
    import paper_1802_04256_b200 as rp
    w = workloads.make_block("strata", 9, 8, 7, 1.0, 2, 30, 5e9, 0.3, jitter=0.3, seed=41, body=(10.0, -20.0, -2.5e4))
    rng = np.random.default_rng(8)
    esc = np.where(w.qpts[:, 2] < 3.0, 4.0, 0.5) * rng.uniform(0.9, 1.1, w.Nq)
    s = oracle.knn(w.nodes, w.qpts, w.k, "grid")
    rpo, cio = oracle.pattern(s, w.N)
    vo, fo, _ = oracle.assemble(w.nodes, w.qpts, w.qw, s, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, rpo, cio, escale=esc)
    rows = np.repeat(np.arange(3 * w.N), np.diff(rpo))
    km = np.abs(vo[rows == cio]).max()
    dev = torch.device("cuda:0")
    ctx = rp.Context(0)
    try:
        ctx.set_reduction(reduction)
        d_n, d_q, d_w = (torch.from_numpy(a).to(dev) for a in (w.nodes, w.qpts, w.qw))
        nnz, bits = ctx.build_pattern(d_n, d_q, w.k, 64)
        assert ctx.reduction_used() == reduction and nnz == rpo[-1]
        d_vals = torch.empty(nnz, dtype=torch.float64, device=dev)
        d_f = torch.empty(3 * w.N, dtype=torch.float64, device=dev)
        ctx.assemble(d_w, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, d_vals, d_f)
        v_plain, f_plain = d_vals.cpu().numpy().copy(), d_f.cpu().numpy().copy()
        d_e = torch.from_numpy(esc).to(dev)
        ctx.set_modulus_scale(d_e)
        ctx.assemble(d_w, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, d_vals, d_f)
        assert np.abs(d_vals.cpu().numpy() - vo).max() <= TOL * km
        assert np.array_equal(d_f.cpu().numpy(), f_plain) and np.abs(f_plain - fo).max() <= TOL * np.abs(fo).max()
        # stresses: sigma(s) = s_q * sigma(1) for the same displacement field
        d_u = torch.from_numpy(rng.uniform(-1e-3, 1e-3, 3 * w.N)).to(dev)
        d_s1 = torch.empty((w.Nq, 6), dtype=torch.float64, device=dev)
        d_s0 = torch.empty_like(d_s1)
        ctx.recover_stress(d_u, w.E, w.nu, d_s1)
        ctx.set_modulus_scale(None)
        ctx.recover_stress(d_u, w.E, w.nu, d_s0)
        s0, s1 = d_s0.cpu().numpy(), d_s1.cpu().numpy()
        assert np.abs(s1 - esc[:, None] * s0).max() <= 1e-12 * np.abs(s1).max()
        ctx.assemble(d_w, w.E, w.nu, w.alpha_c, w.d_c, w.q, w.body, d_vals, d_f)
        assert np.array_equal(d_vals.cpu().numpy(), v_plain)
    finally:
        ctx.close()
