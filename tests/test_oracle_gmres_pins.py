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


# ---------------------------------------------------------------- Krylov iteration on lambda alone (cold-started sweeps)
def lambda_map(pr, sx, sy, n_wh, relax):
    st = O.ddm_setup(pr, sx, sy)

    def G(x):
        O.ddm_unpack(st, x, with_u=False)
        O.ddm_sweep(st, n_wh, False, relax)
        return O.ddm_pack(st, with_u=False)
    x0 = np.zeros_like(O.ddm_pack(st, with_u=False))
    return st, G, x0


def test_cold_started_sweep_is_an_affine_map_of_lambda_alone():
    """PAPER.md:164 (u^(0) <- 0): the sweep then has no memory of u_l, so lambda -> G lambda + d is a map of the interface
    data alone (a stale u_l in the state does not change it) and it is affine and real-linear."""
    pr = tiny_problem()
    st, G, x0 = lambda_map(pr, 2, 1, 3, 0.5)
    assert len(x0) < len(O.ddm_pack(st)) // 4          # interfaces only: far smaller than the joint state
    d = G(x0)
    rng = np.random.default_rng(1)
    a, b = rng.standard_normal(len(x0)), rng.standard_normal(len(x0))
    Ga = G(a)
    for l in range(len(st.u)):                           # scramble the stale subdomain fields
        st.u[l] = rng.standard_normal(len(st.u[l])) + 1j * rng.standard_normal(len(st.u[l]))
    assert np.array_equal(G(a), Ga)
    T = lambda v: G(v) - d
    assert np.linalg.norm(T(2.0 * a - 3.0 * b) - (2.0 * T(a) - 3.0 * T(b))) < 1e-10 * np.linalg.norm(T(a))


def test_lambda_gmres_iterate_is_the_krylov_least_squares_minimiser_brute_force():
    pr = tiny_problem()
    st, G, x0 = lambda_map(pr, 2, 1, 3, 0.5)
    d = G(x0)
    A = lambda v: v - (G(v) - d)
    k = 5
    K = [d]
    for _ in range(k - 1):
        K.append(A(K[-1]))
    K = np.stack(K, axis=1)
    AK = np.stack([A(K[:, i]) for i in range(k)], axis=1)
    y, *_ = np.linalg.lstsq(AK, d, rcond=None)
    x_ref = K @ y
    st_g, hist = O.ddm_gmres(pr, 2, 1, 3, 0.5, restart=10, n_steps=k, lambda_only=True)
    x_g = O.ddm_pack(st_g, with_u=False)
    assert np.linalg.norm(x_g - x_ref) < 1e-8 * np.linalg.norm(x_ref)
    assert abs(hist[-1] - np.linalg.norm(d - AK @ y) / np.linalg.norm(d)) < 1e-9
    # the returned u_l is the cold-started n_wh-iteration WaveHoltz field of that lambda (lambda itself not advanced)
    st_c = O.ddm_setup(pr, 2, 1)
    O.ddm_unpack(st_c, x_ref, with_u=False)
    for l in range(len(st_c.subs)):
        u_l, _ = O.ddm_cycle(st_c, l, 3, False)
        assert np.linalg.norm(st_g.u[l] - u_l) < 1e-8 * np.linalg.norm(u_l)


def test_lambda_gmres_tends_to_the_direct_solution_as_the_subdomain_solves_tighten():
    """The fixed point of the lambda-only map is the DDM fixed point of the INEXACT subdomain solver (n_wh WaveHoltz
    iterations from zero): its distance to the dense direct solve falls with n_wh and reaches 1e-8 (config 1, rho = 1 =
    eq. (2) literally)."""
    inp = make_config(1)
    pr = problem_from(inp)
    ustar = O.direct_solve(pr)
    errs = []
    for n_wh in (10, 20, 40):
        st, hist = O.ddm_gmres(pr, inp.sx, inp.sy, n_wh, 1.0, restart=60, n_steps=60, tol=1e-11, lambda_only=True)
        assert hist[-1] <= 1e-8
        errs.append(np.linalg.norm(O.ddm_gather(st) - ustar) / np.linalg.norm(ustar))
    assert errs[0] > 20 * errs[1] > 400 * errs[2], errs
    assert errs[2] < 1e-8, errs
