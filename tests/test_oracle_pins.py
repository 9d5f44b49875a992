"""Pins of the CPU oracle (oracle/hz_oracle.py) against what the paper and the mathematics
fix -- none of them re-types a formula of the oracle or re-calls its own routine as the
expected value.  CPU only (`-m "not gpu"`).

T-numbers are those of SURVEY.md section 4; citations are PAPER.md lines.
"""
import math
import os

import numpy as np
import pytest

from oracle import hz_oracle as O
from paper_2606_21695_b200.inputs import make_config

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "survey_probe_values.txt")


def golden():
    out = {}
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()[:2]
        out[k] = float(v)
    return out


def problem_from(inp):
    f = inp.f_re.astype(complex)
    if inp.f_im is not None:
        f = f + 1j * inp.f_im
    return O.Problem(inp.nx, inp.ny, inp.p, inp.x0, inp.y0, inp.x1, inp.y1, inp.c_nodes, inp.omega, f)


# ---------------------------------------------------------------- GLL / D / K (closed forms)
@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 7])
def test_gll_quadrature_and_derivative_exactness(p):
    xi, w, D = O.gll(p)
    assert abs(w.sum() - 2.0) < 1e-14
    assert np.allclose(xi, -xi[::-1], atol=1e-15) and np.all(np.diff(xi) > 0)
    # GLL with p+1 points integrates x^k exactly for k <= 2p-1  (int_-1^1 x^k = 2/(k+1), k even)
    for k in range(2 * p):
        exact = 0.0 if k % 2 else 2.0 / (k + 1)
        assert abs(np.dot(w, xi ** k) - exact) < 1e-13
    # ... and NOT for k = 2p (so the rule really is the (p+1)-point Lobatto rule)
    assert abs(np.dot(w, xi ** (2 * p)) - 2.0 / (2 * p + 1)) > 1e-6
    # D differentiates every polynomial of degree <= p exactly at the nodes
    for k in range(p + 1):
        dk = k * xi ** (k - 1) if k > 0 else np.zeros_like(xi)
        assert np.allclose(D @ xi ** k, dk, atol=1e-12)


def test_gll_nodes_closed_form():
    assert np.allclose(O.gll(2)[0], [-1, 0, 1])
    assert np.allclose(O.gll(3)[0], [-1, -1 / math.sqrt(5), 1 / math.sqrt(5), 1])
    assert np.allclose(O.gll(4)[0], [-1, -math.sqrt(3 / 7), 0, math.sqrt(3 / 7), 1])
    assert np.allclose(O.gll(3)[1], [1 / 6, 5 / 6, 5 / 6, 1 / 6])


def test_lambda_p_values():
    g = golden()
    assert abs(O.lambda_p(1) - 4.0) < 1e-12      # 2x2 pencil [[.5,-.5],[-.5,.5]]*2, W=diag(.5,.5)
    assert abs(O.lambda_p(2) - 24.0) < 1e-11
    assert abs(O.lambda_p(3) - g["lambda_p_3"]) < 5e-6
    assert abs(O.lambda_p(4) - g["lambda_p_4"]) < 5e-6


def test_element_stiffness_p1_literal():
    # Q1 element, unit square, trapezoid (=2-point GLL) quadrature: written out by hand.
    lit = np.array([[1, -.5, -.5, 0], [-.5, 1, 0, -.5], [-.5, 0, 1, -.5], [0, -.5, -.5, 1]])
    assert np.allclose(O.element_stiffness(1, 1.0, 1.0), lit)
    # anisotropic: d/dx part scales with hy/hx, d/dy part with hx/hy
    hx, hy = 0.5, 2.0
    lit2 = (hy / hx) * np.array([[.5, -.5, 0, 0], [-.5, .5, 0, 0], [0, 0, .5, -.5], [0, 0, -.5, .5]]) \
        + (hx / hy) * np.array([[.5, 0, -.5, 0], [0, .5, 0, -.5], [-.5, 0, .5, 0], [0, -.5, 0, .5]])
    assert np.allclose(O.element_stiffness(1, hx, hy), lit2)


@pytest.mark.parametrize("p", [1, 2, 3, 4])
def test_element_stiffness_kernel_symmetry_energy(p):
    hx, hy = 0.3, 0.7
    Ae = O.element_stiffness(p, hx, hy)
    assert np.allclose(Ae, Ae.T, atol=1e-13)
    assert np.allclose(Ae @ np.ones((p + 1) ** 2), 0, atol=1e-12)     # constants in the kernel (T3)
    ev = np.linalg.eigvalsh(Ae)
    assert ev.min() > -1e-12
    # energy of u = 2x - 3y (exactly representable): int |grad u|^2 = (4+9) hx hy
    xi = O.gll(p)[0]
    x = hx * (xi + 1) / 2
    y = hy * (xi + 1) / 2
    u = (2 * x[None, :] - 3 * y[:, None]).reshape(-1)
    assert abs(u @ Ae @ u - 13 * hx * hy) < 1e-12
    if p >= 2:   # u = x*y: |grad u|^2 = x^2 + y^2, degree 2 <= 2p-1 -> exact
        u = (x[None, :] * y[:, None]).reshape(-1)
        assert abs(u @ Ae @ u - (hx ** 3 * hy / 3 + hx * hy ** 3 / 3)) < 1e-12


def test_global_operators_measure_and_symmetry():
    # sum of lumped mass = area, sum of edge weights = side lengths, A symmetric, A 1 = 0 (T3)
    c = np.ones((3 * 3 + 1, 4 * 3 + 1))
    pr = O.Problem(4, 3, 3, 0.0, 0.0, 2.0, 0.6, c, 5.0, np.zeros_like(c, dtype=complex))
    A, M, H, b = O.assemble_global(pr)
    assert abs(M.sum() - 2.0 * 0.6) < 1e-13
    assert abs(H.sum() - 2 * (2.0 + 0.6)) < 1e-13
    assert abs(A - A.T).max() < 1e-13
    assert np.abs(A @ np.ones(A.shape[0])).max() < 1e-12
    # c scaling: M ~ c^-2, H ~ c^-1
    pr2 = O.Problem(4, 3, 3, 0.0, 0.0, 2.0, 0.6, 2 * c, 5.0, np.zeros_like(c, dtype=complex))
    _, M2, H2, _ = O.assemble_global(pr2)
    assert np.allclose(M2, M / 4) and np.allclose(H2, H / 2)


# ---------------------------------------------------------------- T6 plane wave (eq. (1))
def planewave_error(p, n):
    omega = 2 * math.pi * p * 16 / 10
    d = np.array([math.cos(0.3), math.sin(0.3)])
    inp = make_config(1, n=n, p=p, sub_elems=n)
    pr0 = O.Problem(n, n, p, 0, 0, 1, 1, np.ones_like(inp.c_nodes), omega, np.zeros_like(inp.c_nodes, dtype=complex))
    xs, ys = pr0.node_coords()
    X, Y = np.meshgrid(xs, ys, indexing="xy")
    uex = np.exp(1j * omega * (d[0] * X + d[1] * Y))
    k = omega
    # lambda = (d_n - ik) u = ik (d.n - 1) u on each side (W,E,S,N)
    normals = [(-1, 0), (1, 0), (0, -1), (0, 1)]
    edges = [uex[:, 0], uex[:, -1], uex[0, :], uex[-1, :]]
    lam = [1j * k * (d[0] * nx + d[1] * ny - 1.0) * e for (nx, ny), e in zip(normals, edges)]
    pr = O.Problem(n, n, p, 0, 0, 1, 1, np.ones_like(inp.c_nodes), omega,
                   np.zeros_like(inp.c_nodes, dtype=complex), bc_lambda=lam)
    u = O.direct_solve(pr)
    return np.linalg.norm(u - uex) / np.linalg.norm(uex)


def test_plane_wave_recovered_at_discretisation_order():
    g = golden()
    e2 = [planewave_error(2, n) for n in (16, 32, 64)]
    e3 = [planewave_error(3, n) for n in (16, 32)]
    # order ~ h^(2p) (T6): each halving of h divides the error by ~2^(2p)
    assert 10 < e2[0] / e2[1] < 24 and 10 < e2[1] / e2[2] < 24
    assert 30 < e3[0] / e3[1] < 90
    # same digits as the survey's independent probe (2 significant digits printed there)
    for got, key in zip(e2 + e3, ["planewave_err_p2_n16", "planewave_err_p2_n32", "planewave_err_p2_n64",
                                  "planewave_err_p3_n16", "planewave_err_p3_n32"]):
        assert abs(got / g[key] - 1) < 0.08, (key, got)


# ---------------------------------------------------------------- T7/T8 tables
@pytest.mark.parametrize("nt", [3, 4, 5, 28, 122])
def test_filter_orthogonality(nt):
    tab = O.wh_tables(nt, 7.3)
    th = 2 * np.pi * np.arange(nt) / nt
    thh = 2 * np.pi * (np.arange(nt) + 0.5) / nt
    # against a pure-omega harmonic: (2/N) sum kappa_nu cos = 1, (2/N) sum kappa_nu sin = 0, and the
    # same at the half steps; the constant -1/4 + 1/4 tan^2 sums to 0 against it
    assert abs(2 / nt * np.sum(tab.kappa * np.cos(th)) - 1) < 1e-12
    assert abs(2 / nt * np.sum(tab.kappa * np.sin(th))) < 1e-12
    assert abs(2 / nt * np.sum(tab.kappa_half * np.cos(thh)) - 1) < 1e-12
    assert abs(2 / nt * np.sum(tab.kappa_half * np.sin(thh))) < 1e-12
    const = -0.25 + 0.25 * math.tan(math.pi / nt) ** 2
    assert np.allclose(tab.kappa - np.cos(th), const) and np.allclose(tab.kappa_half - np.cos(thh), const)
    # the pair reconstructs u exactly from p = Re{u e^{-i th}}, pdot = Re{-i w u e^{-i thh}}:
    u = 0.3 - 1.7j
    om = 7.3
    p = np.real(u * np.exp(-1j * th))
    pd = np.real(-1j * om * u * np.exp(-1j * thh))
    rec = 2 / nt * np.sum(tab.kappa * p - (1 / (1j * om)) * tab.kappa_half * pd)
    assert abs(rec - u) < 1e-12


def test_theta_sigma_limits():
    om = 11.0
    tab = O.wh_tables(4000, om)
    assert abs(tab.theta / (tab.dt / 2) - 1) < 1e-5 and abs(tab.sigma / tab.dt - 1) < 1e-5   # T8
    tab = O.wh_tables(12, om)
    # exactness relations behind PAPER.md:144: sigma = 2 sin(w dt/2)/w, sigma/theta = 2 cos(w dt/2)
    assert abs(tab.sigma * om / 2 - math.sin(om * tab.dt / 2)) < 1e-15
    assert abs(tab.sigma / tab.theta - 2 * math.cos(om * tab.dt / 2)) < 1e-13


def test_nt_rule_matches_survey_table_and_paper_formula_is_unstable():
    g = golden()
    om1 = 2 * math.pi * 2 * 16 / 8          # config 1: n=16, p=2, 8 points per wavelength
    om2 = 2 * math.pi * 3 * 128 / 10        # config 2: n=128, p=3, 10 points per wavelength
    assert O.choose_nt(2, 1 / 16, 1 / 16, 1.0, om1, 0.5) == int(g["nt_config1"])
    assert O.choose_nt(3, 1 / 128, 1 / 128, 3.0, om2, 0.5) == int(g["nt_config2"])
    # reading R9: the printed bound dt <= 2h/(p^2 c) is not a stability bound in 2-D (p=1)
    inp = make_config(1, n=8, p=1, sub_elems=8)
    pr = problem_from(inp)
    A, M, H, b = O.assemble_global(pr)
    T = 2 * math.pi / pr.omega
    nt_paper = max(4, math.ceil(T / (0.99 * 2 * pr.hx / 1.0)))      # 0.99 x the printed bound
    u = np.zeros_like(b)
    for _ in range(30):
        u = O.waveholtz_iteration(A, M, H, b, u, pr.omega, O.wh_tables(nt_paper, pr.omega))
    assert not np.all(np.isfinite(u)) or np.linalg.norm(u) > 1e20
    nt_ok = O.choose_nt(1, pr.hx, pr.hy, 1.0, pr.omega, 0.99)
    u = np.zeros_like(b)
    for _ in range(30):
        u = O.waveholtz_iteration(A, M, H, b, u, pr.omega, O.wh_tables(nt_ok, pr.omega))
    assert np.linalg.norm(u) < 1e3 * np.linalg.norm(b)
