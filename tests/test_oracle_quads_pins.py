"""Pins of the oracle's general-quadrilateral operators (oracle/hz_oracle.py, section F3)
against what the mathematics fixes.  CPU only."""
import math

import numpy as np
import pytest

from oracle import hz_oracle as O
from paper_2606_21695_b200.inputs import distorted_vertices, make_config


def random_mesh(nx, ny, seed, amp=0.22, move_boundary=True):
    """Every vertex moved (boundary too): the domain is a general polygon."""
    rng = np.random.default_rng(seed)
    VX, VY = np.meshgrid(np.linspace(0.0, 1.3, nx + 1), np.linspace(0.0, 0.7, ny + 1), indexing="xy")
    VX = VX + amp * (1.3 / nx) * rng.uniform(-1, 1, VX.shape)
    VY = VY + amp * (0.7 / ny) * rng.uniform(-1, 1, VY.shape)
    return VX, VY


def polygon_area_and_moment(px, py):
    """Shoelace area and first x-moment (int x dA) of a closed polygon, counter-clockwise."""
    x0, y0, x1, y1 = px, py, np.roll(px, -1), np.roll(py, -1)
    cr = x0 * y1 - x1 * y0
    return 0.5 * cr.sum(), ((x0 + x1) * cr).sum() / 6.0


def boundary_polygon(VX, VY):
    px = np.concatenate([VX[0, :-1], VX[:-1, -1], VX[-1, :0:-1], VX[:0:-1, 0]])
    py = np.concatenate([VY[0, :-1], VY[:-1, -1], VY[-1, :0:-1], VY[:0:-1, 0]])
    return px, py


@pytest.mark.parametrize("p", [1, 2, 3, 4])
def test_rectangles_reduce_to_the_rectangular_operators(p):
    ex, ey, hx, hy = 3, 2, 0.37, 0.21
    VX, VY = np.meshgrid(0.4 + hx * np.arange(ex + 1), -0.2 + hy * np.arange(ey + 1), indexing="xy")
    A, m, s = O.region_operators_quads(p, VX, VY)
    A0, m0, s0 = O._region_operators(p, ex, ey, hx, hy)
    assert abs(A - A0).max() < 1e-12 * abs(A0).max()
    assert np.allclose(m, m0, rtol=1e-13, atol=0)
    for a, b in zip(s, s0):
        assert np.allclose(a, b, rtol=1e-13, atol=0)
    c = 1.0 + np.random.default_rng(3).uniform(0, 1, size=m.shape)
    assert O.choose_nt_quads(p, VX, VY, c, 31.0, 0.5) == O.choose_nt(p, hx, hy, float(c.max()), 31.0, 0.5)


def test_rotated_rectangle_has_the_same_stiffness():
    # the Laplacian is invariant under rotation: a rotated rectangular element has the matrix of the unrotated one
    th = 0.7
    R = np.array([[math.cos(th), -math.sin(th)], [math.sin(th), math.cos(th)]])
    X4, Y4 = np.array([[0.0, 0.5], [0.0, 0.5]]), np.array([[0.0, 0.0], [0.3, 0.3]])
    XR, YR = R[0, 0] * X4 + R[0, 1] * Y4, R[1, 0] * X4 + R[1, 1] * Y4
    assert np.allclose(O.element_stiffness_quad(3, XR, YR), O.element_stiffness(3, 0.5, 0.3), atol=1e-12)


@pytest.mark.parametrize("p", [1, 2, 3, 4])
def test_patch_test_area_moment_and_side_lengths(p):
    VX, VY = random_mesh(4, 3, seed=10 + p)
    A, m, s = O.region_operators_quads(p, VX, VY)
    X, Y = O.node_coords_quads(p, VX, VY)
    assert abs(A - A.T).max() < 1e-12
    assert np.abs(A @ np.ones(A.shape[0])).max() < 1e-11                 # constants in the kernel
    npy, npx = X.shape
    interior = np.zeros((npy, npx), bool)
    interior[1:-1, 1:-1] = True
    u = 0.7 * X - 1.9 * Y + 0.3                                           # a linear field: A u = boundary flux only
    assert np.abs((A @ u.reshape(-1))[interior.reshape(-1)]).max() < 1e-11
    px, py = boundary_polygon(VX, VY)
    area, mom = polygon_area_and_moment(px, py)
    assert abs(m.sum() - area) < 1e-13                                    # detJ is bilinear: GLL exact
    assert abs(u.reshape(-1) @ (A @ u.reshape(-1)) - (0.7 ** 2 + 1.9 ** 2) * area) < 1e-11   # |grad u|^2 area
    if p >= 2:                                                            # x^2 is in the mapped space for p >= 2
        assert abs((X ** 2).reshape(-1) @ (A @ X.reshape(-1)) - 2.0 * mom) < 1e-11           # int grad(x^2).grad(x)
    sides = [(VX[:, 0], VY[:, 0]), (VX[:, -1], VY[:, -1]), (VX[0, :], VY[0, :]), (VX[-1, :], VY[-1, :])]
    for w_, (qx, qy) in zip(s, sides):
        assert abs(w_.sum() - np.hypot(np.diff(qx), np.diff(qy)).sum()) < 1e-13
    # transposing the mesh (x <-> y, xi <-> eta) transposes the operators
    At, mt, _ = O.region_operators_quads(p, VY.T, VX.T)
    perm = np.arange(npx * npy).reshape(npy, npx).T.reshape(-1)
    assert abs(At - A[perm][:, perm]).max() < 1e-11 and np.allclose(mt, m.T)


def test_geometric_factors_by_finite_differences():
    # J and g from a central difference of the returned node positions of a FINE GLL grid of the same element
    X4, Y4 = np.array([[0.0, 1.1], [-0.1, 1.4]]), np.array([[0.0, 0.2], [0.9, 1.3]])
    p = 4
    xi = O.gll(p)[0]
    x, y, det, gxx, gxy, gyy = O.quad_geometry(p, X4, Y4)

    def pos(s, t):
        n = [(1 - s) * (1 - t), (1 + s) * (1 - t), (1 - s) * (1 + t), (1 + s) * (1 + t)]
        return (sum(a * b for a, b in zip(n, [X4[0, 0], X4[0, 1], X4[1, 0], X4[1, 1]])) / 4,
                sum(a * b for a, b in zip(n, [Y4[0, 0], Y4[0, 1], Y4[1, 0], Y4[1, 1]])) / 4)
    h = 1e-6
    for b in range(p + 1):
        for a in range(p + 1):
            assert np.allclose(pos(xi[a], xi[b]), (x[b, a], y[b, a]))
            xp, yp = pos(xi[a] + h, xi[b]); xm, ym = pos(xi[a] - h, xi[b])
            xq, yq = pos(xi[a], xi[b] + h); xn, yn = pos(xi[a], xi[b] - h)
            J = np.array([[(xp - xm), (xq - xn)], [(yp - ym), (yq - yn)]]) / (2 * h)
            G = np.linalg.det(J) * np.linalg.inv(J) @ np.linalg.inv(J).T
            assert abs(det[b, a] - np.linalg.det(J)) < 1e-8
            assert np.allclose([gxx[b, a], gxy[b, a], gyy[b, a]], [G[0, 0], G[0, 1], G[1, 1]], atol=1e-7)


@pytest.mark.parametrize("p", [1, 2, 3, 4])
def test_nt_bound_bounds_the_spectrum(p):
    VX, VY = random_mesh(4, 4, seed=40 + p, amp=0.24)
    rng = np.random.default_rng(p)
    A, m, _ = O.region_operators_quads(p, VX, VY)
    c = 1.0 + rng.uniform(0, 1.0, size=m.shape)
    M = (m / c ** 2).reshape(-1)
    lmax = np.max(np.linalg.eigvalsh(A.toarray() / np.sqrt(np.outer(M, M))))
    omega, cfl = 25.0, 1.0
    nt = O.choose_nt_quads(p, VX, VY, c, omega, cfl)
    dt = 2 * math.pi / omega / nt
    assert dt * dt * lmax <= 4.0                       # leapfrog stability of the undamped problem
    assert dt * dt * lmax > 0.8                        # and the bound is not wildly pessimistic


def refine(VX, VY):
    """Split every quad into 4 by its edge midpoints and centroid (keeps the mesh family shape-regular)."""
    ny, nx = VX.shape[0] - 1, VX.shape[1] - 1
    out = []
    for V in (VX, VY):
        R = np.zeros((2 * ny + 1, 2 * nx + 1))
        R[::2, ::2] = V
        R[::2, 1::2] = 0.5 * (V[:, :-1] + V[:, 1:])
        R[1::2, ::2] = 0.5 * (V[:-1, :] + V[1:, :])
        R[1::2, 1::2] = 0.25 * (V[:-1, :-1] + V[:-1, 1:] + V[1:, :-1] + V[1:, 1:])
        out.append(R)
    return out


def test_plane_wave_recovered_on_a_distorted_mesh_family():
    # eq. (1) with impedance data of a plane wave, on a distorted 8x8 mesh and its two uniform refinements:
    # the error falls at high order (it would stall at O(1) with a wrong metric, sign or edge weight)
    p = 2
    omega = 2 * math.pi * p * 8 / 10
    d = np.array([math.cos(0.3), math.sin(0.3)])
    VX, VY = distorted_vertices(8, 8, np.random.default_rng(5), 0.2)
    errs = []
    for _ in range(3):
        n = VX.shape[0] - 1
        X, Y = O.node_coords_quads(p, VX, VY)
        uex = np.exp(1j * omega * (d[0] * X + d[1] * Y))
        normals = [(-1, 0), (1, 0), (0, -1), (0, 1)]
        edges = [uex[:, 0], uex[:, -1], uex[0, :], uex[-1, :]]
        lam = [1j * omega * (d[0] * nx + d[1] * ny - 1.0) * e for (nx, ny), e in zip(normals, edges)]
        pr = O.Problem(n, n, p, 0, 0, 1, 1, np.ones_like(X), omega, np.zeros_like(X, dtype=complex),
                       bc_lambda=lam, vx=VX, vy=VY)
        u = O.direct_solve(pr)
        errs.append(np.linalg.norm(u - uex) / np.linalg.norm(uex))
        VX, VY = refine(VX, VY)
    assert errs[0] / errs[1] > 6 and errs[1] / errs[2] > 6 and errs[2] < 2e-3, errs


def test_ddm_on_quads_converges_to_the_direct_solve():
    inp = make_config(1, n=8, p=2, sub_elems=4, distort=0.2)
    pr = O.Problem(inp.nx, inp.ny, inp.p, 0, 0, 1, 1, inp.c_nodes, inp.omega, inp.f_re.astype(complex),
                   vx=inp.vx, vy=inp.vy)
    uref = O.direct_solve(pr)
    st = O.ddm_solve(pr, inp.sx, inp.sy, 500, 5)
    u = O.ddm_gather(st)
    assert np.linalg.norm(u - uref) / np.linalg.norm(uref) < 2e-9     # linear convergence, 1e-13 after 800 sweeps
    assert O.residual(pr, u) < 5e-8


# ---------------------------------------------------------------- ragged partitions (reading R25)
def test_split_elements_is_the_even_split():
    for n in range(1, 40):
        for s in range(1, n + 1):
            sizes, offs = O.split_elements(n, s)
            assert sum(sizes) == n and max(sizes) - min(sizes) <= 1 and sorted(sizes, reverse=True) == sizes
            assert offs == [sum(sizes[:k]) for k in range(s)]


@pytest.mark.parametrize("quads", [False, True])
def test_ragged_ddm_converges_to_the_same_direct_solve(quads):
    # the converged answer does not depend on the partition: 7x5 elements in 3x2 subdomains (3,2,2 x 3,2 elements)
    rng = np.random.default_rng(3)
    nx, ny, p = 7, 5, 2
    VX = VY = None
    if quads:
        VX, VY = distorted_vertices(nx, ny, rng, 0.2)
    shape = (ny * p + 1, nx * p + 1)
    c = 1.0 + 0.5 * rng.uniform(0, 1, shape)
    f = rng.standard_normal(shape) + 0j
    pr = O.Problem(nx, ny, p, 0, 0, 1, 1, c, 9.0, f, vx=VX, vy=VY)
    uref = O.direct_solve(pr)
    st = O.ddm_setup(pr, 3, 2)
    assert [(sd.npx, sd.npy) for sd in st.subs] == [(7, 7), (5, 7), (5, 7), (7, 5), (5, 5), (5, 5)]
    errs = []
    for _ in range(3):                                  # linear convergence towards the partition-independent answer
        st = O.ddm_solve(pr, 3, 2, 200, 5, state=st)
        errs.append(np.linalg.norm(O.ddm_gather(st) - uref) / np.linalg.norm(uref))
    assert errs[2] < 1e-5 and errs[1] < 0.3 * errs[0] and errs[2] < 0.3 * errs[1], errs
