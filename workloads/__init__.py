"""Seeded synthetic input generators for the five BASELINE.json configs.

This module holds NONE of the method's arithmetic (no kNN, no RBF, no shape
functions, no assembly).  It only produces the plain input arrays that both the
CPU oracle (``oracle/``) and the CUDA library (``paper_1802_04256_b200``) consume:
node coordinates, quadrature points and weights, material constants, body force,
boundary-condition node lists and (config 2) face-traction points.

Conventions (BASELINE.json ``configs``):
  * node id = ix + nx*(iy + ny*iz)
  * quadrature points are ordered cell-major (cx fastest, then cy, cz) and, inside a
    cell, Gauss index a fastest, then b, then c
  * Gauss-Legendre rules on [-1, 1] with 1, 2 or 3 points per axis
  * jitter is a counter-based hash of (seed, node, axis) -> uniform in +-amp*h; the
    component normal to a face is zeroed for nodes on that face (faces stay planar)
"""
from .generators import (  # noqa: F401
    Workload,
    make_block,
    config,
    CONFIG_NAMES,
    gauss_rule,
    jitter_uniform,
)
