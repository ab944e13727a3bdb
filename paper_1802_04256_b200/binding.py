"""ctypes binding of librpim.so: same names as include/rpim.h, argument marshalling only.

Device arrays are torch CUDA tensors (their ``data_ptr()`` is passed down), host arrays are
numpy arrays.  Every step of the path runs in the library's CUDA kernels; nothing here computes.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "librpim.so")

EXPORTED_SYMBOLS = (
    "rpim_create", "rpim_destroy", "rpim_last_error", "rpim_workspace_bytes", "rpim_build_pattern",
    "rpim_get_pattern", "rpim_assemble", "rpim_add_point_loads", "rpim_apply_penalty", "rpim_get_shape",
    "rpim_host_pattern", "rpim_host_assemble", "rpim_last_phase_ms", "rpim_phase_totals", "rpim_launch_count",
    "rpim_matvec", "rpim_solve_pcg", "rpim_recover_stress", "rpim_set_reduction", "rpim_reduction_used",
    "rpim_probe_fp64", "rpim_update_nodes", "rpim_reduction_params", "rpim_set_modulus_scale",
    "rpim_apply_penalty_static", "rpim_apply_penalty_static_max_nodes", "rpim_set_panel_shape",
    "rpim_probe_fp64_dmma",
)


RPIM_INDEX_MIXED = 6432   # index_bits: row_ptr int64, col_idx int32 (include/rpim.h)


class RpimError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"librpim error {code}: {msg}")
        self.code = code


def library_path() -> str:
    return _LIB_PATH


_lib = None


def _load():
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_1802_04256_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(_LIB_PATH)
    vp, i64, dbl = C.c_void_p, C.c_int64, C.c_double
    lib.rpim_create.argtypes = [C.POINTER(vp), C.c_int, vp]
    lib.rpim_destroy.argtypes = [vp]
    lib.rpim_last_error.argtypes = [vp]
    lib.rpim_last_error.restype = C.c_char_p
    lib.rpim_workspace_bytes.argtypes = [vp]
    lib.rpim_workspace_bytes.restype = i64
    lib.rpim_launch_count.argtypes = [vp]
    lib.rpim_launch_count.restype = i64
    lib.rpim_build_pattern.argtypes = [vp, vp, i64, vp, i64, C.c_int, C.c_int, C.POINTER(i64), C.POINTER(C.c_int)]
    lib.rpim_get_pattern.argtypes = [vp, vp, vp, vp]
    lib.rpim_update_nodes.argtypes = [vp, vp, vp, C.POINTER(i64), C.POINTER(C.c_int), C.POINTER(i64)]
    lib.rpim_assemble.argtypes = [vp, vp, dbl, dbl, dbl, dbl, dbl, C.POINTER(dbl), vp, vp, C.POINTER(i64)]
    lib.rpim_add_point_loads.argtypes = [vp, vp, vp, vp, i64, vp]
    lib.rpim_apply_penalty.argtypes = [vp, vp, vp, vp, i64, dbl, C.c_int, vp, vp, C.POINTER(dbl)]
    lib.rpim_apply_penalty_static.argtypes = [vp, vp, vp, vp, i64, dbl, C.c_int, vp, vp, C.POINTER(dbl)]
    lib.rpim_apply_penalty_static_max_nodes.argtypes = []
    lib.rpim_apply_penalty_static_max_nodes.restype = i64
    lib.rpim_get_shape.argtypes = [vp, vp, vp, vp]
    lib.rpim_host_pattern.argtypes = [vp, vp, i64, vp, i64, C.c_int, C.c_int, C.POINTER(i64), C.POINTER(C.c_int)]
    lib.rpim_host_assemble.argtypes = [vp, vp, dbl, dbl, dbl, dbl, dbl, C.POINTER(dbl), vp, vp, vp, i64, dbl,
                                       C.c_int, vp, vp, vp, vp, C.POINTER(i64), C.POINTER(dbl)]
    lib.rpim_last_phase_ms.argtypes = [vp, C.POINTER(C.c_float)]
    lib.rpim_phase_totals.argtypes = [vp, C.POINTER(dbl), C.POINTER(i64), C.c_int]
    lib.rpim_matvec.argtypes = [vp, vp, vp, vp]
    lib.rpim_solve_pcg.argtypes = [vp, vp, vp, vp, dbl, C.c_int, C.POINTER(C.c_int), C.POINTER(dbl)]
    lib.rpim_recover_stress.argtypes = [vp, vp, dbl, dbl, vp]
    lib.rpim_probe_fp64.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl)]
    lib.rpim_probe_fp64_dmma.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl)]
    lib.rpim_set_reduction.argtypes = [vp, C.c_int]
    lib.rpim_reduction_used.argtypes = [vp]
    lib.rpim_reduction_params.argtypes = [vp, C.POINTER(C.c_int)]
    lib.rpim_set_modulus_scale.argtypes = [vp, vp]
    lib.rpim_set_panel_shape.argtypes = [vp] + [C.c_int] * 6
    _lib = lib
    return lib


def _check(ctx, rc):
    if rc != 0:
        raise RpimError(rc, (_load().rpim_last_error(ctx) or b"").decode())


def _dptr(t, dtype=None):
    """Device pointer of a contiguous CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError(f"expected dtype {dtype}, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _hptr(a, dtype):
    if a is None:
        return None
    if not isinstance(a, np.ndarray) or a.dtype != dtype or not a.flags.c_contiguous:
        raise ValueError(f"expected a C-contiguous numpy array of {dtype}")
    return C.c_void_p(a.ctypes.data)


# ---------------------------------------------------------------- functions named as in include/rpim.h
def rpim_create(device: int = 0, cuda_stream: int = 0):
    ctx = C.c_void_p()
    rc = _load().rpim_create(C.byref(ctx), int(device), C.c_void_p(int(cuda_stream)))
    if rc != 0:
        raise RpimError(rc, "rpim_create failed (no CUDA device?)")
    return ctx


def rpim_destroy(ctx):
    _load().rpim_destroy(ctx)


def rpim_last_error(ctx) -> str:
    return (_load().rpim_last_error(ctx) or b"").decode()


def rpim_matvec(ctx, d_vals, d_x, d_y):
    import torch
    _check(ctx, _load().rpim_matvec(ctx, _dptr(d_vals, torch.float64), _dptr(d_x, torch.float64),
                                    _dptr(d_y, torch.float64)))


def rpim_solve_pcg(ctx, d_vals, d_f, d_u, rel_tol=1e-10, max_iter=10000):
    """Returns (iterations, relative residual reached)."""
    import torch
    it, rel = C.c_int(0), C.c_double(0.0)
    _check(ctx, _load().rpim_solve_pcg(ctx, _dptr(d_vals, torch.float64), _dptr(d_f, torch.float64),
                                       _dptr(d_u, torch.float64), float(rel_tol), int(max_iter), C.byref(it),
                                       C.byref(rel)))
    return it.value, rel.value


def rpim_recover_stress(ctx, d_u, E, nu, d_sigma):
    import torch
    _check(ctx, _load().rpim_recover_stress(ctx, _dptr(d_u, torch.float64), float(E), float(nu),
                                            _dptr(d_sigma, torch.float64)))


def rpim_probe_fp64(ctx):
    """{"tflops": sustained FP64 fma rate, "ms": duration of the best launch}."""
    tf, ms = C.c_double(0.0), C.c_double(0.0)
    _check(ctx, _load().rpim_probe_fp64(ctx, C.byref(tf), C.byref(ms)))
    return {"tflops": float(tf.value), "ms": float(ms.value)}


def rpim_probe_fp64_dmma(ctx):
    """{"tflops": sustained FP64 mma.sync m8n8k4 rate, "ms": duration of the best launch}."""
    tf, ms = C.c_double(0.0), C.c_double(0.0)
    _check(ctx, _load().rpim_probe_fp64_dmma(ctx, C.byref(tf), C.byref(ms)))
    return {"tflops": float(tf.value), "ms": float(ms.value)}


def rpim_set_reduction(ctx, mode: int):
    _check(ctx, _load().rpim_set_reduction(ctx, int(mode)))


def rpim_set_panel_shape(ctx, rows_per_tile=0, warps_per_group=0, rows_per_group=0, ring_stages=0, staging=0,
                         tile_desc=0):
    """Force parts of the panel kernel's launch shape (0 = automatic); see include/rpim.h."""
    _check(ctx, _load().rpim_set_panel_shape(ctx, int(rows_per_tile), int(warps_per_group), int(rows_per_group),
                                             int(ring_stages), int(staging), int(tile_desc)))


def rpim_reduction_used(ctx) -> int:
    return int(_load().rpim_reduction_used(ctx))


def rpim_set_modulus_scale(ctx, d_escale):
    """d_escale: CUDA float64 tensor of Nq values (kept alive by the caller) or None."""
    _check(ctx, _load().rpim_set_modulus_scale(ctx, C.c_void_p(0 if d_escale is None else d_escale.data_ptr())))


def rpim_reduction_params(ctx) -> dict:
    out = (C.c_int * 10)()
    rc = _load().rpim_reduction_params(ctx, out)
    if rc != 0:
        raise RpimError(rc, "rpim_reduction_params failed")
    keys = ("kernel", "union_chunks", "rows_per_tile", "warps_per_row_group", "ring_stages", "max_upper_columns",
            "max_block_row", "mean_union_x100", "rows_per_warp_group", "tensor_copy_staging")
    return dict(zip(keys, [int(v) for v in out]))


def rpim_workspace_bytes(ctx) -> int:
    return int(_load().rpim_workspace_bytes(ctx))


def rpim_launch_count(ctx) -> int:
    return int(_load().rpim_launch_count(ctx))


def rpim_build_pattern(ctx, d_nodes, d_qpts, k: int, index_bits: int = 0):
    import torch
    nnz, bits = C.c_int64(0), C.c_int(0)
    rc = _load().rpim_build_pattern(ctx, _dptr(d_nodes, torch.float64), d_nodes.shape[0], _dptr(d_qpts, torch.float64),
                                    d_qpts.shape[0], int(k), int(index_bits), C.byref(nnz), C.byref(bits))
    _check(ctx, rc)
    return int(nnz.value), int(bits.value)


def rpim_update_nodes(ctx, d_nodes, d_qpts=None):
    """Returns (changed points, pattern rebuilt?, nnz)."""
    import torch
    ch, rb, nnz = C.c_int64(0), C.c_int(0), C.c_int64(0)
    _check(ctx, _load().rpim_update_nodes(ctx, _dptr(d_nodes, torch.float64), _dptr(d_qpts, torch.float64),
                                          C.byref(ch), C.byref(rb), C.byref(nnz)))
    return int(ch.value), bool(rb.value), int(nnz.value)


def rpim_get_pattern(ctx, d_row_ptr=None, d_col_idx=None, d_support=None):
    _check(ctx, _load().rpim_get_pattern(ctx, _dptr(d_row_ptr), _dptr(d_col_idx), _dptr(d_support)))


def rpim_assemble(ctx, d_qw, E, nu, alpha_c, d_c, q, body, d_vals, d_f, want_singular: bool = True):
    import torch
    b = (C.c_double * 3)(*[float(x) for x in body])
    ns = C.c_int64(0)
    rc = _load().rpim_assemble(ctx, _dptr(d_qw, torch.float64), float(E), float(nu), float(alpha_c), float(d_c),
                               float(q), b, _dptr(d_vals, torch.float64), _dptr(d_f, torch.float64),
                               C.byref(ns) if want_singular else None)
    _check(ctx, rc)
    return int(ns.value) if want_singular else None


def rpim_add_point_loads(ctx, d_pts, d_w, d_t, d_f):
    import torch
    rc = _load().rpim_add_point_loads(ctx, _dptr(d_pts, torch.float64), _dptr(d_w, torch.float64),
                                      _dptr(d_t, torch.float64), d_pts.shape[0], _dptr(d_f, torch.float64))
    _check(ctx, rc)


def rpim_apply_penalty(ctx, d_bc_nodes, d_bc_mask, d_u_bar, alpha, alpha_is_relative, d_vals, d_f):
    import torch
    used = C.c_double(0.0)
    m = 0 if d_bc_nodes is None else d_bc_nodes.shape[0]
    rc = _load().rpim_apply_penalty(ctx, _dptr(d_bc_nodes, torch.int64), _dptr(d_bc_mask, torch.uint8),
                                    _dptr(d_u_bar, torch.float64), m, float(alpha), int(bool(alpha_is_relative)),
                                    _dptr(d_vals, torch.float64), _dptr(d_f, torch.float64), C.byref(used))
    _check(ctx, rc)
    return float(used.value)


def rpim_apply_penalty_static(ctx, d_bc_nodes, d_bc_mask, d_u_bar, alpha, alpha_is_relative, d_vals, d_f):
    """rpim_apply_penalty for callers that must not allocate device memory (see include/rpim.h): same arguments
    and results, scratch memory in a fixed array inside the library, at most
    ``rpim_apply_penalty_static_max_nodes()`` nodes.  Returns alpha_used."""
    import torch
    used = C.c_double(0.0)
    m = 0 if d_bc_nodes is None else d_bc_nodes.shape[0]
    rc = _load().rpim_apply_penalty_static(ctx, _dptr(d_bc_nodes, torch.int64), _dptr(d_bc_mask, torch.uint8),
                                           _dptr(d_u_bar, torch.float64), m, float(alpha),
                                           int(bool(alpha_is_relative)), _dptr(d_vals, torch.float64),
                                           _dptr(d_f, torch.float64), C.byref(used))
    _check(ctx, rc)
    return float(used.value)


def rpim_apply_penalty_static_max_nodes() -> int:
    return int(_load().rpim_apply_penalty_static_max_nodes())


def rpim_get_shape(ctx, d_phi=None, d_dphi=None, d_singular=None):
    _check(ctx, _load().rpim_get_shape(ctx, _dptr(d_phi), _dptr(d_dphi), _dptr(d_singular)))


def rpim_host_pattern(ctx, h_nodes, h_qpts, k: int, index_bits: int = 0):
    nnz, bits = C.c_int64(0), C.c_int(0)
    rc = _load().rpim_host_pattern(ctx, _hptr(h_nodes, np.float64), h_nodes.shape[0], _hptr(h_qpts, np.float64),
                                   h_qpts.shape[0], int(k), int(index_bits), C.byref(nnz), C.byref(bits))
    _check(ctx, rc)
    return int(nnz.value), int(bits.value)


def rpim_host_assemble(ctx, h_qw, E, nu, alpha_c, d_c, q, body, h_bc_nodes, h_bc_mask, h_u_bar, alpha,
                       alpha_is_relative, h_row_ptr, h_col_idx, h_vals, h_f):
    b = (C.c_double * 3)(*[float(x) for x in body])
    ns, used = C.c_int64(0), C.c_double(0.0)
    m = 0 if h_bc_nodes is None else h_bc_nodes.shape[0]
    idt = None if h_row_ptr is None else h_row_ptr.dtype
    cdt = None if h_col_idx is None else h_col_idx.dtype     # RPIM_INDEX_MIXED: int64 offsets, int32 column ids
    rc = _load().rpim_host_assemble(ctx, _hptr(h_qw, np.float64), float(E), float(nu), float(alpha_c), float(d_c),
                                    float(q), b, _hptr(h_bc_nodes, np.int64), _hptr(h_bc_mask, np.uint8),
                                    _hptr(h_u_bar, np.float64), m, float(alpha), int(bool(alpha_is_relative)),
                                    _hptr(h_row_ptr, idt), _hptr(h_col_idx, cdt), _hptr(h_vals, np.float64),
                                    _hptr(h_f, np.float64), C.byref(ns), C.byref(used))
    _check(ctx, rc)
    return int(ns.value), float(used.value)


def rpim_last_phase_ms(ctx):
    out = (C.c_float * 5)()
    _check(ctx, _load().rpim_last_phase_ms(ctx, out))
    return [float(x) for x in out]


def rpim_phase_totals(ctx, reset: bool = False):
    out = (C.c_double * 5)()
    calls = (C.c_int64 * 2)()
    _check(ctx, _load().rpim_phase_totals(ctx, out, calls, int(reset)))
    return [float(x) for x in out], [int(c) for c in calls]


class Context:
    """Owns one ``rpim_ctx`` on the current torch stream; methods forward to the functions above."""

    def __init__(self, device: int = 0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("librpim needs a CUDA device (there is no CPU fallback)")
        s = torch.cuda.current_stream(device) if stream is None else stream
        self._stream = s
        self.device = device
        self.ctx = rpim_create(device, s.cuda_stream)

    def close(self):
        if self.ctx is not None:
            rpim_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def build_pattern(self, d_nodes, d_qpts, k, index_bits=0):
        return rpim_build_pattern(self.ctx, d_nodes, d_qpts, k, index_bits)

    def update_nodes(self, d_nodes, d_qpts=None):
        return rpim_update_nodes(self.ctx, d_nodes, d_qpts)

    def get_pattern(self, d_row_ptr=None, d_col_idx=None, d_support=None):
        return rpim_get_pattern(self.ctx, d_row_ptr, d_col_idx, d_support)

    def assemble(self, d_qw, E, nu, alpha_c, d_c, q, body, d_vals, d_f, want_singular=True):
        return rpim_assemble(self.ctx, d_qw, E, nu, alpha_c, d_c, q, body, d_vals, d_f, want_singular)

    def add_point_loads(self, d_pts, d_w, d_t, d_f):
        return rpim_add_point_loads(self.ctx, d_pts, d_w, d_t, d_f)

    def apply_penalty(self, d_bc_nodes, d_bc_mask, d_u_bar, alpha, relative, d_vals, d_f):
        return rpim_apply_penalty(self.ctx, d_bc_nodes, d_bc_mask, d_u_bar, alpha, relative, d_vals, d_f)

    def apply_penalty_static(self, d_bc_nodes, d_bc_mask, d_u_bar, alpha, relative, d_vals, d_f):
        return rpim_apply_penalty_static(self.ctx, d_bc_nodes, d_bc_mask, d_u_bar, alpha, relative, d_vals, d_f)

    def get_shape(self, d_phi=None, d_dphi=None, d_singular=None):
        return rpim_get_shape(self.ctx, d_phi, d_dphi, d_singular)

    def host_pattern(self, h_nodes, h_qpts, k, index_bits=0):
        return rpim_host_pattern(self.ctx, h_nodes, h_qpts, k, index_bits)

    def host_assemble(self, *args):
        return rpim_host_assemble(self.ctx, *args)

    def phase_ms(self):
        return rpim_last_phase_ms(self.ctx)

    def phase_totals(self, reset=False):
        return rpim_phase_totals(self.ctx, reset)

    def matvec(self, d_vals, d_x, d_y):
        return rpim_matvec(self.ctx, d_vals, d_x, d_y)

    def solve_pcg(self, d_vals, d_f, d_u, rel_tol=1e-10, max_iter=10000):
        return rpim_solve_pcg(self.ctx, d_vals, d_f, d_u, rel_tol, max_iter)

    def recover_stress(self, d_u, E, nu, d_sigma):
        return rpim_recover_stress(self.ctx, d_u, E, nu, d_sigma)

    def probe_fp64(self):
        return rpim_probe_fp64(self.ctx)

    def probe_fp64_dmma(self):
        return rpim_probe_fp64_dmma(self.ctx)

    def set_reduction(self, mode):
        return rpim_set_reduction(self.ctx, mode)

    def set_panel_shape(self, **shape):
        return rpim_set_panel_shape(self.ctx, **shape)

    def reduction_used(self):
        return rpim_reduction_used(self.ctx)

    def reduction_params(self):
        return rpim_reduction_params(self.ctx)

    def set_modulus_scale(self, d_escale):
        self._escale = d_escale          # keeps the tensor alive while the library points at it
        return rpim_set_modulus_scale(self.ctx, d_escale)

    def launch_count(self):
        return rpim_launch_count(self.ctx)

    def workspace_bytes(self):
        return rpim_workspace_bytes(self.ctx)
