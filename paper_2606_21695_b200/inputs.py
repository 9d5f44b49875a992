"""Seeded synthetic inputs for the five BASELINE.json configs ("Input recipe").

This module serves BOTH the CPU oracle (tests, bench cpu_baseline) and the CUDA library.
It holds none of the method's arithmetic: it only places nodes, samples the wave speed
c(x) and the source f(x) AT the global GLL nodes, and names the partition / solver options
of each config.  No RNG is re-implemented on either side: the random draws happen here
(numpy.random.default_rng(seed)) and reach both sides as plain arrays.

The paper's workloads are synthetic too (constant / piecewise-constant coefficients on a
square with uniform elements; the Y-waveguide picture of Fig. 1,
PAPER.md:27), so nothing here stands in for a public dataset.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

# Gauss-Lobatto-Legendre points on [-1,1] in closed form (p <= 4); only used to PLACE the
# nodes at which c and f are sampled.  The oracle and the CUDA library each compute their
# own nodes, weights and differentiation matrices.
_GLL_CLOSED_FORM = {
    1: (-1.0, 1.0),
    2: (-1.0, 0.0, 1.0),
    3: (-1.0, -1.0 / math.sqrt(5.0), 1.0 / math.sqrt(5.0), 1.0),
    4: (-1.0, -math.sqrt(3.0 / 7.0), 0.0, math.sqrt(3.0 / 7.0), 1.0),
}


def node_coords_1d(n: int, p: int, a: float = 0.0, b: float = 1.0) -> np.ndarray:
    """The n*p+1 node abscissae of n uniform degree-p elements on [a,b]."""
    xi = np.asarray(_GLL_CLOSED_FORM[p])
    h = (b - a) / n
    x = np.empty(n * p + 1)
    for e in range(n):
        x[e * p:e * p + p] = a + h * (e + (xi[:-1] + 1.0) / 2.0)
    x[-1] = b
    return x


@dataclass
class HzInputs:
    """Everything hz_mesh_setup / hz_partition / hz_ddm_solve (and the oracle) need."""
    name: str
    nx: int
    ny: int
    p: int
    x0: float
    y0: float
    x1: float
    y1: float
    omega: float
    c_nodes: np.ndarray            # (ny*p+1, nx*p+1) float64, x fastest
    f_re: np.ndarray               # (ny*p+1, nx*p+1) float64
    f_im: np.ndarray | None
    sx: int
    sy: int
    cfl_frac: float = 0.5
    relax: float = 0.5
    n_wh: int = 5
    warm_start: bool = True
    seed: int = 0
    meta: dict = field(default_factory=dict)
    vx: np.ndarray | None = None   # general quads (F3): (ny+1, nx+1) vertex coordinates; None = uniform rectangles
    vy: np.ndarray | None = None

    @property
    def npx(self):
        return self.nx * self.p + 1

    @property
    def npy(self):
        return self.ny * self.p + 1


def omega_for_ppw(n: int, p: int, ppw: float, c_ref: float = 1.0, length: float = 1.0) -> float:
    """omega such that the wavelength 2 pi c_ref / omega spans `ppw` node spacings h/p
    (reading R18)."""
    return 2.0 * math.pi * c_ref * p * n / (ppw * length)


def _seg_dist(X, Y, ax, ay, bx, by):
    dx, dy = bx - ax, by - ay
    t = ((X - ax) * dx + (Y - ay) * dy) / (dx * dx + dy * dy)
    t = np.clip(t, 0.0, 1.0)
    return np.hypot(X - (ax + t * dx), Y - (ay + t * dy))


def y_waveguide_speed(X, Y, c_in: float = 3.0, c_out: float = 1.0, width: float = 0.1):
    """c = c_in where the distance to any of the three centre-line segments of the Y is
    <= width/2 (closed set), else c_out (reading R16)."""
    d = np.minimum(_seg_dist(X, Y, 0.5, 0.0, 0.5, 0.5),
                   np.minimum(_seg_dist(X, Y, 0.5, 0.5, 0.2, 1.0),
                              _seg_dist(X, Y, 0.5, 0.5, 0.8, 1.0)))
    return np.where(d <= 0.5 * width, c_in, c_out)


def random_block_speed(X, Y, rng, nb: int = 8, lo: float = 1.0, hi: float = 3.0):
    """Piecewise-constant c on an nb x nb grid of blocks with i.i.d. U[lo,hi] values; a node
    on a block line belongs to block min(floor(nb*x), nb-1) (reading R14)."""
    vals = rng.uniform(lo, hi, size=(nb, nb))
    bi = np.minimum(np.floor(nb * X).astype(int), nb - 1)
    bj = np.minimum(np.floor(nb * Y).astype(int), nb - 1)
    return vals[bj, bi], vals


def draw_source_points(rng, count: int):
    """x_s ~ U([0.15,0.85]^2), rejecting |x_s - (1/2,1/2)|_inf < 0.05 (reading R17)."""
    pts = []
    while len(pts) < count:
        xs, ys = rng.uniform(0.15, 0.85, size=2)
        if max(abs(xs - 0.5), abs(ys - 0.5)) < 0.05:
            continue
        pts.append((float(xs), float(ys)))
    return pts


def gaussian_sources(X, Y, pts, sigma: float):
    f = np.zeros_like(X)
    for xs, ys in pts:
        f += np.exp(-((X - xs) ** 2 + (Y - ys) ** 2) / (2.0 * sigma ** 2))
    return f


def distorted_vertices(nx: int, ny: int, rng, amp: float, x0=0.0, y0=0.0, x1=1.0, y1=1.0):
    """Vertices of a logically rectangular mesh of straight-sided convex quads: the uniform grid with every
    INTERIOR vertex moved by amp * (hx, hy) * U(-1,1)^2 (amp <= 0.25 keeps all elements convex); the boundary
    vertices stay, so the domain is still the rectangle."""
    gx, gy = np.linspace(x0, x1, nx + 1), np.linspace(y0, y1, ny + 1)
    VX, VY = np.meshgrid(gx, gy, indexing="xy")
    VX, VY = VX.copy(), VY.copy()
    hx, hy = (x1 - x0) / nx, (y1 - y0) / ny
    VX[1:-1, 1:-1] += amp * hx * rng.uniform(-1, 1, size=(ny - 1, nx - 1))
    VY[1:-1, 1:-1] += amp * hy * rng.uniform(-1, 1, size=(ny - 1, nx - 1))
    return VX, VY


def mapped_node_coords(p: int, VX: np.ndarray, VY: np.ndarray):
    """(npy, npx) positions of the GLL nodes of the bilinearly mapped elements (node placement only)."""
    xi = np.asarray(_GLL_CLOSED_FORM[p])
    ny, nx = VX.shape[0] - 1, VX.shape[1] - 1
    XI, ETA = np.meshgrid(xi, xi, indexing="xy")
    X = np.zeros((ny * p + 1, nx * p + 1))
    Y = np.zeros_like(X)
    for b in range(p + 1):          # local node (a,b) of every element at once
        for a in range(p + 1):
            n00, n10 = (1 - xi[a]) * (1 - xi[b]) / 4.0, (1 + xi[a]) * (1 - xi[b]) / 4.0
            n01, n11 = (1 - xi[a]) * (1 + xi[b]) / 4.0, (1 + xi[a]) * (1 + xi[b]) / 4.0
            for Z, V in ((X, VX), (Y, VY)):
                Z[b:b + (ny - 1) * p + 1:p, a:a + (nx - 1) * p + 1:p] = (
                    n00 * V[:-1, :-1] + n10 * V[:-1, 1:] + n01 * V[1:, :-1] + n11 * V[1:, 1:])
    return X, Y


def make_config(cfg: int, n: int | None = None, p: int | None = None, sub_elems: int | None = None,
                seed: int | None = None, distort: float = 0.0) -> HzInputs:
    """Config `cfg` in 1..5 of BASELINE.json.  `n` (elements per side), `p` and `sub_elems`
    (elements per subdomain side) override the full-size values to get a SMALLER problem of
    the same structure for the parity tests; the full-size values are the defaults.
    `distort` > 0: the same config on general convex quads: interior vertices moved by
    distort * h * U(-1,1), c and f sampled at the mapped nodes."""
    defaults = {1: (16, 2, 8, 8.0), 2: (128, 3, 8, 10.0), 3: (512, 3, 8, 10.0),
                4: (1024, 3, 32, 10.0), 5: (2048, 3, 8, 10.0)}
    n0, p0, s0, ppw = defaults[cfg]
    n = n0 if n is None else n
    p = p0 if p is None else p
    s = s0 if sub_elems is None else sub_elems
    if n % s:
        raise ValueError("sub_elems must divide n")
    seed = 1000 + cfg if seed is None else seed
    rng = np.random.default_rng(seed)
    x = node_coords_1d(n, p)
    X, Y = np.meshgrid(x, x, indexing="xy")            # [J, I]: x fastest
    h = 1.0 / n
    omega = omega_for_ppw(n, p, ppw)
    meta = {"ppw": ppw}
    VX = VY = None
    if distort > 0.0:
        VX, VY = distorted_vertices(n, n, np.random.default_rng(seed + 7919), distort)
        X, Y = mapped_node_coords(p, VX, VY)
        meta["distort"] = distort
    if cfg == 1:
        c = np.ones_like(X)
        pts = draw_source_points(rng, 1)
        sigma = 0.03 * (16.0 / n)                          # = 0.03 at n = 16
    elif cfg in (2, 4):
        c = y_waveguide_speed(X, Y)
        pts = draw_source_points(rng, 1)
        sigma = 1.28 * h                                   # = 0.01 at n = 128
    else:
        c, vals = random_block_speed(X, Y, rng)
        meta["block_speeds"] = vals
        pts = draw_source_points(rng, 3)
        sigma = 1.28 * h
    f = gaussian_sources(X, Y, pts, sigma)
    meta.update(sources=pts, sigma=sigma)
    return HzInputs(name=f"cfg{cfg}_n{n}_p{p}_s{s}" + ("_quads" if VX is not None else ""), nx=n, ny=n, p=p,
                    x0=0.0, y0=0.0, x1=1.0, y1=1.0,
                    omega=omega, c_nodes=np.ascontiguousarray(c, dtype=np.float64),
                    f_re=np.ascontiguousarray(f, dtype=np.float64), f_im=None,
                    sx=n // s, sy=n // s, seed=seed, meta=meta, vx=VX, vy=VY)


def random_lambda(rng, n_sub: int, edge_nodes: int):
    """A random complex interface vector lambda[l, side, node] (the paper's benchmark applies
    the DDM cycle to a random input vector)."""
    return rng.standard_normal((n_sub, 4, edge_nodes)) + 1j * rng.standard_normal((n_sub, 4, edge_nodes))


# ---------------------------------------------------------------------------------------------------------
# 3-D hexahedral variant (uniform elements on a box, constant or blockwise
# coefficients, random input)
# ---------------------------------------------------------------------------------------------------------
@dataclass
class Hz3Inputs:
    name: str
    nx: int
    ny: int
    nz: int
    p: int
    box: tuple
    omega: float
    c_nodes: np.ndarray            # (npz, npy, npx)
    f_re: np.ndarray
    f_im: np.ndarray | None
    sx: int
    sy: int
    sz: int
    cfl_frac: float = 0.5
    seed: int = 0

    @property
    def shape(self):
        return self.nz * self.p + 1, self.ny * self.p + 1, self.nx * self.p + 1


def make_config_3d(n, p: int, sub_elems, seed: int = 3000, ppw: float = 8.0, random_c: bool = True,
                   box=(0.0, 0.0, 0.0, 1.0, 1.0, 1.0)) -> Hz3Inputs:
    """n (int or 3-tuple) elements per side of a box, subdomains of sub_elems (int or 3-tuple) elements per side;
    omega for `ppw` node spacings per wavelength; nodal c ~ 1 + U(0,1) (or 1); Gaussian source at a random point."""
    nx, ny, nz = (n, n, n) if isinstance(n, int) else n
    ex, ey, ez = (sub_elems,) * 3 if isinstance(sub_elems, int) else sub_elems
    if nx % ex or ny % ey or nz % ez:
        raise ValueError("sub_elems must divide n")
    rng = np.random.default_rng(seed)
    xs = [node_coords_1d(m, p, box[d], box[d + 3]) for d, m in enumerate((nx, ny, nz))]
    Z, Y, X = np.meshgrid(xs[2], xs[1], xs[0], indexing="ij")
    c = 1.0 + rng.uniform(0, 1, size=X.shape) if random_c else np.ones_like(X)
    omega = omega_for_ppw(nx, p, ppw, length=box[3] - box[0])
    x0 = np.array([rng.uniform(box[d] + 0.25 * (box[d + 3] - box[d]), box[d] + 0.75 * (box[d + 3] - box[d])) for d in range(3)])
    sig = 1.5 * (box[3] - box[0]) / nx
    f = np.exp(-((X - x0[0]) ** 2 + (Y - x0[1]) ** 2 + (Z - x0[2]) ** 2) / (2 * sig ** 2))
    return Hz3Inputs(name=f"box_{nx}x{ny}x{nz}_p{p}_s{ex}x{ey}x{ez}", nx=nx, ny=ny, nz=nz, p=p, box=tuple(box),
                     omega=omega, c_nodes=np.ascontiguousarray(c), f_re=np.ascontiguousarray(f), f_im=None,
                     sx=nx // ex, sy=ny // ey, sz=nz // ez, seed=seed)
