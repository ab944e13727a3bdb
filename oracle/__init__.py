"""CPU oracle for the RPIM hot path -- TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports the CUDA package
(``paper_1802_04256_b200``) and the CUDA package never imports it.

Thin ctypes wrappers (argument marshalling only) around ``oracle/rpim_oracle.cpp``; see
that file's header for what each function computes and which DESIGN.md reading it follows.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.orc_pow_qm1.restype = C.c_double
        _lib.orc_pow_qm1.argtypes = [C.c_double, C.c_double]
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def pow_qm1(t: float, q: float) -> float:
    return float(lib().orc_pow_qm1(float(t), float(q)))


def knn(nodes, qpts, k: int, method: str = "grid") -> np.ndarray:
    nodes = _f64(nodes)
    qpts = _f64(qpts)
    out = np.empty((qpts.shape[0], k), dtype=np.int32)
    rc = lib().orc_knn(_p(nodes, C.c_double), C.c_int64(nodes.shape[0]), _p(qpts, C.c_double),
                       C.c_int64(qpts.shape[0]), C.c_int(k), C.c_int(0 if method == "brute" else 1),
                       _p(out, C.c_int32))
    if rc:
        raise ValueError(f"orc_knn failed ({rc})")
    return out


def pattern(support: np.ndarray, N: int):
    """Scalar CSR pattern (row_ptr int64 [3N+1], col_idx int64 [nnz])."""
    support = np.ascontiguousarray(support, dtype=np.int32)
    Nq, k = support.shape
    row_ptr = np.empty(3 * N + 1, dtype=np.int64)
    lib().orc_pattern_count(_p(support, C.c_int32), C.c_int64(Nq), C.c_int(k), C.c_int64(N),
                            _p(row_ptr, C.c_int64))
    col_idx = np.empty(int(row_ptr[-1]), dtype=np.int64)
    rc = lib().orc_pattern_fill(_p(support, C.c_int32), C.c_int64(Nq), C.c_int(k), C.c_int64(N),
                                _p(row_ptr, C.c_int64), _p(col_idx, C.c_int64))
    if rc:
        raise RuntimeError(f"orc_pattern_fill failed ({rc})")
    return row_ptr, col_idx


def shape(nodes, pts, support, alpha_c: float, d_c: float, q: float):
    """phi (M,k), dphi (M,3,k), singular (M,) for M points with given supports."""
    nodes = _f64(nodes)
    pts = _f64(pts)
    support = np.ascontiguousarray(support, dtype=np.int32)
    M, k = support.shape
    phi = np.empty((M, k))
    dphi = np.empty((M, 3, k))
    sing = np.empty(M, dtype=np.uint8)
    lib().orc_shape(_p(nodes, C.c_double), _p(pts, C.c_double), _p(support, C.c_int32), C.c_int64(M),
                    C.c_int(k), C.c_double(alpha_c), C.c_double(d_c), C.c_double(q),
                    _p(phi, C.c_double), _p(dphi, C.c_double), _p(sing, C.c_uint8))
    return phi, dphi, sing


def shape_dense_ref(nodes, pts, support, alpha_c: float, d_c: float, q: float):
    """The definition in long double (plain G, textbook LU); pin for ``shape``."""
    nodes = _f64(nodes)
    pts = _f64(pts)
    support = np.ascontiguousarray(support, dtype=np.int32)
    M, k = support.shape
    phi = np.empty((M, k))
    dphi = np.empty((M, 3, k))
    lib().orc_shape_dense_ref(_p(nodes, C.c_double), _p(pts, C.c_double), _p(support, C.c_int32),
                              C.c_int64(M), C.c_int(k), C.c_double(alpha_c), C.c_double(d_c),
                              C.c_double(q), _p(phi, C.c_double), _p(dphi, C.c_double))
    return phi, dphi


def assemble(nodes, pts, w, support, E, nu, alpha_c, d_c, q, body, row_ptr, col_idx,
             node_lo: int = 0, node_hi: int | None = None, escale=None):
    """K values and f for rows of nodes [node_lo, node_hi).

    ``row_ptr`` / ``col_idx`` describe exactly those rows (row_ptr starts at 0).
    ``escale`` (optional, one value per point): strata with one Poisson ratio, E_q = E * escale[q]
    (R8b); the loads are not scaled.
    Returns (vals, f, n_singular).
    """
    nodes = _f64(nodes)
    pts = _f64(pts)
    w = _f64(w)
    body = _f64(body)
    support = np.ascontiguousarray(support, dtype=np.int32)
    row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
    col_idx = np.ascontiguousarray(col_idx, dtype=np.int64)
    M, k = support.shape
    if node_hi is None:
        node_hi = nodes.shape[0]
    nrows = 3 * (node_hi - node_lo)
    assert row_ptr.shape[0] == nrows + 1 and row_ptr[0] == 0
    vals = np.empty(int(row_ptr[-1]))
    f = np.empty(nrows)
    nsing = C.c_int64(0)
    if escale is not None:
        escale = _f64(escale)
        assert escale.shape == (M,)
        rc = lib().orc_assemble_strata(_p(nodes, C.c_double), _p(pts, C.c_double), _p(w, C.c_double), _p(escale, C.c_double),
                                       _p(support, C.c_int32), C.c_int64(M), C.c_int(k), C.c_double(E),
                                       C.c_double(nu), C.c_double(alpha_c), C.c_double(d_c), C.c_double(q),
                                       _p(body, C.c_double), C.c_int64(node_lo), C.c_int64(node_hi),
                                       _p(row_ptr, C.c_int64), _p(col_idx, C.c_int64), _p(vals, C.c_double),
                                       _p(f, C.c_double), C.byref(nsing))
        if rc:
            raise RuntimeError(f"orc_assemble_strata failed ({rc})")
        return vals, f, int(nsing.value)
    rc = lib().orc_assemble(_p(nodes, C.c_double), _p(pts, C.c_double), _p(w, C.c_double),
                            _p(support, C.c_int32), C.c_int64(M), C.c_int(k), C.c_double(E),
                            C.c_double(nu), C.c_double(alpha_c), C.c_double(d_c), C.c_double(q),
                            _p(body, C.c_double), C.c_int64(node_lo), C.c_int64(node_hi),
                            _p(row_ptr, C.c_int64), _p(col_idx, C.c_int64), _p(vals, C.c_double),
                            _p(f, C.c_double), C.byref(nsing))
    if rc:
        raise RuntimeError(f"orc_assemble failed ({rc})")
    return vals, f, int(nsing.value)


def assemble_dense_ref(nodes, pts, w, support, E, nu, alpha_c, d_c, q, body, row_ptr, col_idx,
                       node_lo: int = 0, node_hi: int | None = None):
    """K values and f from the definition end to end in long double (pin for ``assemble``)."""
    nodes = _f64(nodes)
    pts = _f64(pts)
    w = _f64(w)
    body = _f64(body)
    support = np.ascontiguousarray(support, dtype=np.int32)
    row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
    col_idx = np.ascontiguousarray(col_idx, dtype=np.int64)
    M, k = support.shape
    if node_hi is None:
        node_hi = nodes.shape[0]
    nrows = 3 * (node_hi - node_lo)
    assert row_ptr.shape[0] == nrows + 1 and row_ptr[0] == 0
    vals = np.empty(int(row_ptr[-1]))
    f = np.empty(nrows)
    rc = lib().orc_assemble_dense_ref(_p(nodes, C.c_double), _p(pts, C.c_double), _p(w, C.c_double),
                                      _p(support, C.c_int32), C.c_int64(M), C.c_int(k), C.c_double(E),
                                      C.c_double(nu), C.c_double(alpha_c), C.c_double(d_c), C.c_double(q),
                                      _p(body, C.c_double), C.c_int64(node_lo), C.c_int64(node_hi),
                                      _p(row_ptr, C.c_int64), _p(col_idx, C.c_int64), _p(vals, C.c_double),
                                      _p(f, C.c_double))
    if rc:
        raise RuntimeError(f"orc_assemble_dense_ref failed ({rc})")
    return vals, f


def point_loads(nodes, pts, w, t, support, alpha_c, d_c, q, f):
    """f (3N, modified in place) += (w * phi_I) * t at the given points."""
    nodes = _f64(nodes)
    pts = _f64(pts)
    w = _f64(w)
    t = _f64(t)
    support = np.ascontiguousarray(support, dtype=np.int32)
    M, k = support.shape
    assert f.dtype == np.float64 and f.flags.c_contiguous
    lib().orc_point_loads(_p(nodes, C.c_double), _p(pts, C.c_double), _p(w, C.c_double),
                          _p(t, C.c_double), _p(support, C.c_int32), C.c_int64(M), C.c_int(k),
                          C.c_double(alpha_c), C.c_double(d_c), C.c_double(q), _p(f, C.c_double))
    return f


def penalty(bc_nodes, bc_mask, ubar, alpha, relative, N, row_ptr, col_idx, vals, f):
    """In-place penalty on (vals, f); returns alpha_used."""
    bc_nodes = np.ascontiguousarray(bc_nodes, dtype=np.int64)
    ubar = _f64(ubar)
    row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
    col_idx = np.ascontiguousarray(col_idx, dtype=np.int64)
    mask_p = None
    if bc_mask is not None:
        bc_mask = np.ascontiguousarray(bc_mask, dtype=np.uint8)
        mask_p = _p(bc_mask, C.c_uint8)
    used = C.c_double(0.0)
    rc = lib().orc_penalty(_p(bc_nodes, C.c_int64), mask_p, _p(ubar, C.c_double),
                           C.c_int64(bc_nodes.shape[0]), C.c_double(alpha), C.c_int(int(relative)),
                           C.c_int64(N), _p(row_ptr, C.c_int64), _p(col_idx, C.c_int64),
                           _p(vals, C.c_double), _p(f, C.c_double), C.byref(used))
    if rc:
        raise RuntimeError(f"orc_penalty failed ({rc})")
    return float(used.value)
