from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

CONFIG_NAMES = ("patch", "cantilever", "slope", "large", "stress")


@dataclass
class Workload:
    """Plain input arrays of one RPIM assembly problem (all float64 / int64, C-contiguous)."""

    name: str
    nodes: np.ndarray          # (N, 3)
    qpts: np.ndarray           # (Nq, 3)
    qw: np.ndarray             # (Nq,)
    k: int
    E: float
    nu: float
    alpha_c: float
    d_c: float
    q: float
    body: np.ndarray           # (3,)
    bc_nodes: np.ndarray       # (m,) int64, unique, ascending
    bc_mask: np.ndarray        # (m,) uint8, bit c set = constrain DOF c
    bc_ubar: np.ndarray        # (m, 3)
    penalty_alpha: float       # relative: alpha = penalty_alpha * max_i K_ii
    index_bits: int            # 0 = auto, 32, 64
    grid: tuple                # (nx, ny, nz)
    h: float
    volume: float
    load_pts: Optional[np.ndarray] = None   # (M, 3) face Gauss points (config 2)
    load_w: Optional[np.ndarray] = None     # (M,)
    load_t: Optional[np.ndarray] = None     # (M, 3) traction vectors
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.nodes.shape[0])

    @property
    def Nq(self) -> int:
        return int(self.qpts.shape[0])


def gauss_rule(n: int):
    """Gauss-Legendre abscissae and weights on [-1, 1], n in {1, 2, 3}."""
    if n == 1:
        return np.array([0.0]), np.array([2.0])
    if n == 2:
        a = 1.0 / np.sqrt(3.0)
        return np.array([-a, a]), np.array([1.0, 1.0])
    if n == 3:
        a = np.sqrt(3.0 / 5.0)
        return np.array([-a, 0.0, a]), np.array([5.0 / 9.0, 8.0 / 9.0, 5.0 / 9.0])
    raise ValueError("gauss_rule: n must be 1, 2 or 3")


def _splitmix64(x: np.ndarray) -> np.ndarray:
    x = x.astype(np.uint64, copy=True)
    with np.errstate(over="ignore"):
        x += np.uint64(0x9E3779B97F4A7C15)
        z = x
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def jitter_uniform(seed: int, n_nodes: int) -> np.ndarray:
    """Counter-based uniform numbers in [-1, 1): one per (node, axis); shape (n_nodes, 3)."""
    ctr = np.arange(n_nodes * 3, dtype=np.uint64)
    with np.errstate(over="ignore"):
        key = _splitmix64(np.uint64(seed) * np.uint64(0xD1342543DE82EF95) + ctr)
    u = (key >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
    return (2.0 * u - 1.0).reshape(n_nodes, 3)


def _grid_index(nx, ny, nz):
    iz, iy, ix = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return ix.reshape(-1), iy.reshape(-1), iz.reshape(-1)


def make_block(
    name: str,
    nx: int,
    ny: int,
    nz: int,
    h: float,
    gauss: int,
    k: int,
    E: float,
    nu: float,
    *,
    jitter: float = 0.0,
    seed: int = 0,
    body=(0.0, 0.0, 0.0),
    bc: str = "bottom",            # "all" | "x0" | "bottom" | "bottom+roller"
    ubar_linear: Optional[float] = None,
    alpha_c: float = 4.0,
    q: float = 1.03,
    penalty_alpha: float = 1e8,
    index_bits: int = 0,
    end_traction=None,             # (tx, ty, tz) on the x = max face, 3x3 face Gauss points
) -> Workload:
    """A regular nx*ny*nz node block (spacing h) with optional seeded jitter."""
    ix, iy, iz = _grid_index(nx, ny, nz)
    N = nx * ny * nz
    nodes = np.stack([ix, iy, iz], axis=1).astype(np.float64) * h
    if jitter > 0.0:
        u = jitter_uniform(seed, N) * (jitter * h)
        u[(ix == 0) | (ix == nx - 1), 0] = 0.0
        u[(iy == 0) | (iy == ny - 1), 1] = 0.0
        u[(iz == 0) | (iz == nz - 1), 2] = 0.0
        nodes = nodes + u
    nodes = np.ascontiguousarray(nodes)

    # background cells + Gauss points
    xi, wi = gauss_rule(gauss)
    ncx, ncy, ncz = nx - 1, ny - 1, nz - 1
    cz, cy, cx = np.meshgrid(np.arange(ncz), np.arange(ncy), np.arange(ncx), indexing="ij")
    cx = cx.reshape(-1, 1)
    cy = cy.reshape(-1, 1)
    cz = cz.reshape(-1, 1)
    gc, gb, ga = np.meshgrid(np.arange(gauss), np.arange(gauss), np.arange(gauss), indexing="ij")
    ga = ga.reshape(1, -1)
    gb = gb.reshape(1, -1)
    gc = gc.reshape(1, -1)
    qx = (cx + 0.5 + 0.5 * xi[ga]) * h
    qy = (cy + 0.5 + 0.5 * xi[gb]) * h
    qz = (cz + 0.5 + 0.5 * xi[gc]) * h
    qpts = np.ascontiguousarray(np.stack([qx.reshape(-1), qy.reshape(-1), qz.reshape(-1)], axis=1))
    wcell = (wi[ga] * wi[gb] * wi[gc]) * (h * h * h / 8.0)
    qw = np.ascontiguousarray(np.broadcast_to(wcell, (ncx * ncy * ncz, gauss ** 3)).reshape(-1))

    # boundary conditions
    ids = np.arange(N, dtype=np.int64)
    mask = np.zeros(N, dtype=np.uint8)
    if bc == "all":
        on = (ix == 0) | (ix == nx - 1) | (iy == 0) | (iy == ny - 1) | (iz == 0) | (iz == nz - 1)
        mask[on] = 7
    elif bc == "x0":
        mask[ix == 0] = 7
    elif bc == "bottom":
        mask[iz == 0] = 7
    elif bc == "bottom+roller":
        mask[(ix == 0) | (ix == nx - 1)] |= 1
        mask[(iy == 0) | (iy == ny - 1)] |= 2
        mask[iz == 0] = 7
    elif bc == "none":
        pass
    else:
        raise ValueError(bc)
    sel = mask != 0
    bc_nodes = np.ascontiguousarray(ids[sel])
    bc_mask = np.ascontiguousarray(mask[sel])
    ubar = np.zeros((bc_nodes.size, 3))
    if ubar_linear is not None:
        p = nodes[bc_nodes]
        val = ubar_linear * (p[:, 0] + 2.0 * p[:, 1] + 3.0 * p[:, 2])
        ubar[:] = val[:, None]

    load_pts = load_w = load_t = None
    if end_traction is not None:
        xf, wf = gauss_rule(3)
        fz, fy = np.meshgrid(np.arange(ncz), np.arange(ncy), indexing="ij")
        fy = fy.reshape(-1, 1)
        fz = fz.reshape(-1, 1)
        gb2, ga2 = np.meshgrid(np.arange(3), np.arange(3), indexing="ij")
        ga2 = ga2.reshape(1, -1)
        gb2 = gb2.reshape(1, -1)
        py = (fy + 0.5 + 0.5 * xf[ga2]) * h
        pz = (fz + 0.5 + 0.5 * xf[gb2]) * h
        px = np.full_like(py, (nx - 1) * h)
        load_pts = np.ascontiguousarray(np.stack([px.reshape(-1), py.reshape(-1), pz.reshape(-1)], axis=1))
        wface = (wf[ga2] * wf[gb2]) * (h * h / 4.0)
        load_w = np.ascontiguousarray(np.broadcast_to(wface, (ncy * ncz, 9)).reshape(-1))
        load_t = np.ascontiguousarray(np.broadcast_to(np.asarray(end_traction, dtype=np.float64), (load_w.size, 3)))

    return Workload(
        name=name, nodes=nodes, qpts=qpts, qw=qw, k=k, E=E, nu=nu, alpha_c=alpha_c, d_c=h, q=q,
        body=np.asarray(body, dtype=np.float64), bc_nodes=bc_nodes, bc_mask=bc_mask,
        bc_ubar=np.ascontiguousarray(ubar), penalty_alpha=penalty_alpha, index_bits=index_bits,
        grid=(nx, ny, nz), h=h, volume=float(ncx * ncy * ncz) * h ** 3,
        load_pts=load_pts, load_w=load_w, load_t=load_t,
        meta={"gauss": gauss, "jitter": jitter, "seed": seed, "bc": bc},
    )


def config(which) -> Workload:
    """The five BASELINE.json configs, by index 0..4 or name (see CONFIG_NAMES)."""
    if isinstance(which, int):
        which = CONFIG_NAMES[which]
    if which == "patch":          # BASELINE.json configs[0]
        return make_block("patch", 5, 5, 5, 0.25, 2, 27, 20e9, 0.25, bc="all", ubar_linear=1e-3)
    if which == "cantilever":     # configs[1]; A8: end shear t = (0, 0, -1e6) Pa
        return make_block("cantilever", 41, 5, 5, 0.25, 3, 30, 30e9, 0.2, bc="x0",
                          end_traction=(0.0, 0.0, -1e6))
    if which == "slope":          # configs[2]
        return make_block("slope", 50, 50, 25, 1.0, 2, 40, 5e9, 0.3, jitter=0.3, seed=3,
                          body=(0.0, 0.0, -2500.0 * 9.81), bc="bottom+roller")
    if which == "large":          # configs[3]; A7: rho = 2500; A9: int64 forced
        return make_block("large", 100, 100, 100, 1.0, 1, 30, 10e9, 0.25, jitter=0.25, seed=4,
                          body=(0.0, 0.0, -2500.0 * 9.81), bc="bottom", index_bits=64)
    if which == "stress":         # configs[4]
        return make_block("stress", 160, 160, 80, 1.0, 2, 60, 20e9, 0.25, jitter=0.3, seed=5,
                          body=(0.0, 0.0, -2500.0 * 9.81), bc="bottom+roller", index_bits=64)
    raise KeyError(which)
