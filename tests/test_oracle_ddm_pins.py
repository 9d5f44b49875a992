"""Pins of the oracle's WaveHoltz and DDM parts (oracle/hz_oracle.py) against what the paper
and the mathematics fix.  CPU only.  T-numbers: SURVEY.md section 4; citations: PAPER.md lines.

None of the expected values below is produced by the function under test: they come from a
dense direct solve (numpy.linalg.solve on matrices assembled in the test or by the pinned
`assemble_global`), from closed forms, or from hand-written element matrices.
"""
import math

import numpy as np
import pytest

from oracle import hz_oracle as O
from paper_2606_21695_b200.inputs import make_config


def problem_from(inp):
    f = inp.f_re.astype(complex)
    if inp.f_im is not None:
        f = f + 1j * inp.f_im
    return O.Problem(inp.nx, inp.ny, inp.p, inp.x0, inp.y0, inp.x1, inp.y1, inp.c_nodes, inp.omega, f)


def small_hetero_problem(nx=6, ny=4, p=3, seed=5, omega=9.0, complex_f=True):
    """Non-square mesh (hx != hy, nx != ny), variable c, complex f: transposition or
    anisotropy mistakes cannot cancel."""
    rng = np.random.default_rng(seed)
    shape = (ny * p + 1, nx * p + 1)
    c = 1.0 + rng.uniform(0, 1.5, size=shape)
    f = rng.standard_normal(shape) + (1j * rng.standard_normal(shape) if complex_f else 0)
    return O.Problem(nx, ny, p, 0.0, 0.0, 1.5, 0.8, c, omega, f.astype(complex))


def dense_solve(A, M, H, b, omega):
    Z = A.toarray().astype(complex) - np.diag(1j * omega * H + omega ** 2 * M)
    return np.linalg.solve(Z, b)


# ---------------------------------------------------------------- T1: fixed point of Pi
@pytest.mark.parametrize("p,nt", [(1, 9), (2, 28), (3, 40), (4, 61)])
def test_direct_solution_is_fixed_point_of_waveholtz(p, nt):
    # PAPER.md:144 "guarantee that the WaveHoltz iteration exactly converges to u".
    pr = small_hetero_problem(4, 3, p, seed=p, omega=6.0 + p)
    A, M, H, b = O.assemble_global(pr)
    ustar = dense_solve(A, M, H, b, pr.omega)
    nt_stable = O.choose_nt(p, pr.hx, pr.hy, float(pr.c_nodes.max()), pr.omega, 0.5)
    tab = O.wh_tables(max(nt, nt_stable), pr.omega)
    u1 = O.waveholtz_iteration(A, M, H, b, ustar, pr.omega, tab)
    assert np.linalg.norm(u1 - ustar) / np.linalg.norm(ustar) < 1e-12
    # the conjugate (what the Algorithm-1 sign of the pdot term would converge to, reading R2)
    # is NOT a fixed point
    u2 = O.waveholtz_iteration(A, M, H, b, np.conj(ustar), pr.omega, tab)
    assert np.linalg.norm(u2 - np.conj(ustar)) / np.linalg.norm(ustar) > 1e-3


def test_leapfrog_evolves_time_harmonic_solution_exactly():
    # T2: with u the solution of (4), p^nu = Re{u e^{-i nu w dt}} and
    # pdot^{nu+1/2} = Re{-i w u e^{-i (nu+1/2) w dt}} at EVERY step.
    pr = small_hetero_problem(5, 3, 2, seed=11, omega=7.5)
    A, M, H, b = O.assemble_global(pr)
    ustar = dense_solve(A, M, H, b, pr.omega)
    nt = O.choose_nt(2, pr.hx, pr.hy, float(pr.c_nodes.max()), pr.omega, 0.5)
    tab = O.wh_tables(nt, pr.omega)
    trace = []
    O.waveholtz_iteration(A, M, H, b, ustar, pr.omega, tab, trace=trace)
    assert len(trace) == nt
    scale = np.abs(ustar).max()
    for nu, (p_nu, pd_nu) in enumerate(trace):
        ph = np.exp(-1j * pr.omega * tab.dt * nu)
        phh = np.exp(-1j * pr.omega * tab.dt * (nu + 0.5))
        assert np.abs(p_nu - np.real(ustar * ph)).max() < 1e-11 * scale
        assert np.abs(pd_nu - np.real(-1j * pr.omega * ustar * phh)).max() < 1e-11 * scale * pr.omega


def test_waveholtz_from_zero_converges_to_direct_solution():
    inp = make_config(1, n=8, p=2, sub_elems=8)
    pr = problem_from(inp)
    A, M, H, b = O.assemble_global(pr)
    ustar = dense_solve(A, M, H, b, pr.omega)
    tab = O.wh_tables(O.choose_nt(2, pr.hx, pr.hy, 1.0, pr.omega, 0.5), pr.omega)
    u = np.zeros_like(b)
    errs = []
    for _ in range(120):
        u = O.waveholtz_iteration(A, M, H, b, u, pr.omega, tab)
        errs.append(np.linalg.norm(u - ustar) / np.linalg.norm(ustar))
    assert errs[-1] < 1e-9 and errs[-1] < errs[10] < errs[0]


# ---------------------------------------------------------------- hand-sized 2x1 split
def test_ddm_cycle_two_q1_elements_by_hand():
    """2x1 Q1 elements on [0,2]x[0,1], split into two one-element subdomains.  Every matrix
    of subdomain 0 is written out by hand (trapezoid quadrature): one sweep of the oracle with
    (numerically) exact inner solves must give u_0 = Z_0^-1 b_0 and g = -lam - 2 i k u."""
    omega = 1.3
    c = np.array([[1.0, 2.0, 1.5], [1.2, 1.0, 2.5]])          # [J, I]
    f = np.array([[0.3, -1.0, 0.2], [0.7, 0.1, -0.4]]) + 1j * np.array([[0.0, 0.5, 0.1], [-0.2, 0.3, 0.0]])
    pr = O.Problem(2, 1, 1, 0.0, 0.0, 2.0, 1.0, c, omega, f)
    st = O.ddm_setup(pr, 2, 1, n_t=16)
    lam_E = np.array([0.4 - 0.3j, -0.2 + 0.9j])               # incoming data on subdomain 0's E side
    st.lam[0][O.E_] = lam_E.copy()
    u0, g = O.ddm_cycle(st, 0, n_wh=300, warm_start=False)
    # --- by hand: unit-square Q1 element, local order (0,0),(1,0),(0,1),(1,1)
    Ae = np.array([[1, -.5, -.5, 0], [-.5, 1, 0, -.5], [-.5, 0, 1, -.5], [0, -.5, -.5, 1.0]])
    cl = np.array([1.0, 2.0, 1.2, 1.0])                       # c at those four nodes
    fl = np.array([f[0, 0], f[0, 1], f[1, 0], f[1, 1]])
    m = np.full(4, 0.25)                                      # lumped mass: area/4
    M = m / cl ** 2
    H = (0.5 + 0.5) / cl                                      # every node lies on two sides, weight 1/2 each
    b = fl * m
    b[1] += 0.5 * lam_E[0]                                    # E side: nodes (1,0) and (1,1)
    b[3] += 0.5 * lam_E[1]
    uh = np.linalg.solve(Ae - np.diag(1j * omega * H + omega ** 2 * M), b)
    assert np.linalg.norm(u0 - uh) / np.linalg.norm(uh) < 1e-10
    assert g[O.W_] is None and g[O.S_] is None and g[O.N_] is None
    k = omega / np.array([cl[1], cl[3]])
    assert np.allclose(g[O.E_], -lam_E - 2j * k * np.array([uh[1], uh[3]]), atol=1e-10)
    # exchange with relaxation lands in subdomain 1's W slot only (reading R12)
    st.lam[1][O.W_] = np.array([1.0 + 1.0j, -2.0j])
    old = st.lam[1][O.W_].copy()
    O.ddm_sweep(st, n_wh=300, warm_start=False, relax=0.25)
    assert np.allclose(st.lam[1][O.W_], 0.75 * old + 0.25 * g[O.E_], atol=1e-10)


# ---------------------------------------------------------------- T4 / T5 / R3
def test_ddm_converges_to_direct_solve_config1():
    # T4 and the north_star bar: converged DDM == direct solve of (4), relative L2 <= 1e-8.
    pr = problem_from(make_config(1))
    ud = O.direct_solve(pr)
    A, M, H, b = O.assemble_global(pr)
    assert np.allclose(ud.reshape(-1), dense_solve(A, M, H, b, pr.omega), atol=1e-12 * np.abs(ud).max())
    st = O.ddm_solve(pr, 2, 2, n_outer=300, n_wh=2, warm_start=True, relax=0.5)
    assert st.tab.n_t == 28
    u = O.ddm_gather(st)
    assert np.linalg.norm(u - ud) / np.linalg.norm(ud) < 1e-8
    assert O.residual(pr, u) < 1e-6
    # at the fixed point: continuity of u and discrete flux balance lam_lr + lam_rl + 2ik u = 0
    for l, sd in enumerate(st.subs):
        for side in range(4):
            r = sd.neighbour[side]
            if r < 0:
                assert not np.any(st.lam[l][side])
                continue
            o = O.OPPOSITE[side]
            ul = st.u[l][sd.edge_idx[side]]
            ur = st.u[r][st.subs[r].edge_idx[o]]
            assert np.abs(ul - ur).max() < 1e-6 * np.abs(ud).max()
            bal = st.lam[l][side] + st.lam[r][o] + 2j * sd.k_edge[side] * ul
            assert np.abs(bal).max() < 1e-5 * np.abs(st.lam[l][side]).max()


def test_ddm_converges_heterogeneous_rectangular_partition():
    # 3x2 subdomains of 2x2 elements, hx != hy, variable c, complex f, p=3 (cross-points, R13)
    pr = small_hetero_problem(6, 4, 3, seed=3, omega=30.0)
    ud = O.direct_solve(pr)
    st = O.ddm_solve(pr, 3, 2, n_outer=360, n_wh=2, warm_start=True, relax=0.5)
    u = O.ddm_gather(st)
    assert np.linalg.norm(u - ud) / np.linalg.norm(ud) < 1e-8


def test_single_subdomain_ddm_is_plain_waveholtz():
    # T5: L = 1 -> the DDM cycle is WaveHoltz on the whole domain.
    pr = small_hetero_problem(4, 3, 2, seed=8, omega=5.0)
    A, M, H, b = O.assemble_global(pr)
    st = O.ddm_setup(pr, 1, 1)
    u = np.zeros_like(b)
    for sweep in range(3):
        O.ddm_sweep(st, n_wh=2, warm_start=True, relax=0.5)
        for _ in range(2):
            u = O.waveholtz_iteration(A, M, H, b, u, pr.omega, st.tab)
        assert np.abs(st.u[0] - u).max() <= 1e-14 * np.abs(u).max()
    assert np.array_equal(O.ddm_gather(st).reshape(-1), st.u[0])


def test_printed_sign_of_eq2_diverges_and_unrelaxed_stagnates():
    # reading R3: with B = d_n - ik the update is -lam - 2ik u; the printed +2ik diverges.
    pr = problem_from(make_config(1, n=8, p=2, sub_elems=4))
    ud = O.direct_solve(pr)

    def err(**kw):
        st = O.ddm_solve(pr, 2, 2, n_outer=40, n_wh=25, warm_start=True, **kw)
        return np.linalg.norm(O.ddm_gather(st) - ud) / np.linalg.norm(ud)

    good = err(relax=0.5)
    bad = err(relax=0.5, sign_2ik=+1.0)
    assert good < 1e-3 and bad > 1e2


def test_cold_start_is_literal_algorithm1_and_warm_start_differs():
    # reading R11: warm_start=False restarts every cycle from u=0
    pr = problem_from(make_config(1, n=8, p=2, sub_elems=4))
    st_c = O.ddm_solve(pr, 2, 2, n_outer=2, n_wh=3, warm_start=False)
    st_w = O.ddm_solve(pr, 2, 2, n_outer=2, n_wh=3, warm_start=True)
    # first sweep identical (both start from zero), second differs
    st_1c = O.ddm_solve(pr, 2, 2, n_outer=1, n_wh=3, warm_start=False)
    st_1w = O.ddm_solve(pr, 2, 2, n_outer=1, n_wh=3, warm_start=True)
    assert all(np.array_equal(a, b) for a, b in zip(st_1c.u, st_1w.u))
    assert any(np.abs(a - b).max() > 1e-6 * np.abs(a).max() for a, b in zip(st_c.u, st_w.u))
