"""Pins of the oracle's Krylov-accelerated outer iteration (oracle.hz_oracle.ddm_gmres).
None of the expected values comes from the function under test: dense direct solves, an explicit Krylov
basis with numpy.linalg.lstsq (brute force on a tiny case) and the plain fixed-point iteration."""
import numpy as np

from oracle import hz_oracle as O
from paper_2606_21695_b200.inputs import make_config


def problem_from(inp):
    return O.Problem(inp.nx, inp.ny, inp.p, inp.x0, inp.y0, inp.x1, inp.y1, inp.c_nodes, inp.omega,
                     inp.f_re.astype(complex))


def tiny_problem():
    rng = np.random.default_rng(3)
    nx, ny, p = 4, 2, 2
    shape = (ny * p + 1, nx * p + 1)
    c = 1.0 + rng.uniform(0, 1.0, size=shape)
    f = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    return O.Problem(nx, ny, p, 0.0, 0.0, 1.0, 0.6, c, 7.0, f)


def affine_map(pr, sx, sy, n_wh, relax):
    st = O.ddm_setup(pr, sx, sy)

    def F(x):
        O.ddm_unpack(st, x)
        O.ddm_sweep(st, n_wh, True, relax)
        return O.ddm_pack(st)
    x0 = np.zeros_like(O.ddm_pack(st))
    return st, F, x0


def test_sweep_is_affine_and_real_linear_but_not_complex_linear():
    pr = tiny_problem()
    st, F, x0 = affine_map(pr, 2, 1, 2, 0.5)
    c = F(x0)
    rng = np.random.default_rng(0)
    a, b = rng.standard_normal(len(x0)), rng.standard_normal(len(x0))
    T = lambda v: F(v) - c
    assert np.linalg.norm(T(2.0 * a - 3.0 * b) - (2.0 * T(a) - 3.0 * T(b))) < 1e-10 * np.linalg.norm(T(a))
    # multiplication by i (swap of the re/im halves with a sign) does NOT commute with T: WaveHoltz takes real parts
    h = len(a) // 2
    ia = np.concatenate([-a[h:], a[:h]])
    Ta = T(a)
    iTa = np.concatenate([-Ta[h:], Ta[:h]])
    assert np.linalg.norm(T(ia) - iTa) > 1e-3 * np.linalg.norm(Ta)


def test_gmres_iterate_is_the_krylov_least_squares_minimiser_brute_force():
    pr = tiny_problem()
    st, F, x0 = affine_map(pr, 2, 1, 2, 0.5)
    c = F(x0)
    A = lambda v: v - (F(v) - c)
    k = 6
    K = [c]
    for _ in range(k - 1):
        K.append(A(K[-1]))
    K = np.stack(K, axis=1)
    AK = np.stack([A(K[:, i]) for i in range(k)], axis=1)
    y, *_ = np.linalg.lstsq(AK, c, rcond=None)
    x_ref = K @ y
    st_g, hist = O.ddm_gmres(pr, 2, 1, 2, 0.5, restart=10, n_steps=k)
    x_g = O.ddm_pack(st_g)
    assert np.linalg.norm(x_g - x_ref) < 1e-8 * np.linalg.norm(x_ref)
    assert abs(hist[-1] - np.linalg.norm(c - AK @ y) / np.linalg.norm(c)) < 1e-9
    assert all(hist[i + 1] <= hist[i] * (1 + 1e-12) for i in range(len(hist) - 1)), "GMRES residuals are monotone"


def test_gmres_converges_to_the_direct_solution_and_beats_the_plain_iteration():
    inp = make_config(1)
    pr = problem_from(inp)
    ustar = O.direct_solve(pr)
    st, hist = O.ddm_gmres(pr, inp.sx, inp.sy, 2, 0.5, restart=40, n_steps=120, tol=1e-11)
    err = np.linalg.norm(O.ddm_gather(st) - ustar) / np.linalg.norm(ustar)
    assert err < 1e-8, err
    n_gmres = len(hist) - 1
    # the relaxed fixed-point iteration needs 320 sweeps for a 1e-8 residual on this config (bench extras)
    st_j = O.ddm_solve(pr, inp.sx, inp.sy, n_gmres, 2, warm_start=True, relax=0.5)
    err_j = np.linalg.norm(O.ddm_gather(st_j) - ustar) / np.linalg.norm(ustar)
    assert n_gmres < 120 and err_j > 100 * err


def test_restart_continues_from_the_current_iterate():
    pr = tiny_problem()
    st_a, hist_a = O.ddm_gmres(pr, 2, 1, 2, 0.5, restart=4, n_steps=12)
    st_b, hist_b = O.ddm_gmres(pr, 2, 1, 2, 0.5, restart=12, n_steps=12)
    assert hist_a[4] == hist_b[4]                      # identical until the first restart
    assert hist_a[-1] >= hist_b[-1] * (1 - 1e-9)       # restarting cannot beat full GMRES
    assert hist_a[-1] < hist_a[4]                      # but keeps converging
