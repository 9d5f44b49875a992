"""Pins of the oracle's MINRES comparator (oracle.hz_oracle.minres / block_system; SURVEY.md 8(f) F1,
PAPER.md:113-117, 271-277) against dense algebra, brute force and scipy's own MINRES."""
import numpy as np
import scipy.sparse.linalg as spla

from oracle import hz_oracle as O
from paper_2606_21695_b200.inputs import make_config


def small_system(seed=2, p=2, nx=3, ny=2, omega=6.5):
    rng = np.random.default_rng(seed)
    shape = (ny * p + 1, nx * p + 1)
    c = 1.0 + rng.uniform(0, 1.0, size=shape)
    f = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    pr = O.Problem(nx, ny, p, 0.0, 0.0, 1.0, 0.7, c, omega, f)
    A, M, H, b = O.assemble_global(pr)
    return A, M, H, b, omega


def test_block_system_is_symmetric_and_equivalent_to_the_complex_system():
    A, M, H, b, omega = small_system()
    K, rhs = O.block_system(A, M, H, b, omega)
    assert abs(K - K.T).max() < 1e-14                      # PAPER.md:117 "symmetric"
    ev = np.linalg.eigvalsh(K.toarray())
    assert ev.min() < 0 < ev.max()                          # "indefinite"
    u = np.linalg.solve(O.helmholtz_matrix(A, M, H, omega).toarray(), b)
    assert np.linalg.norm(K @ np.concatenate([u.real, u.imag]) - rhs) < 1e-10 * np.linalg.norm(rhs)


def test_minres_iterate_minimises_the_residual_over_the_krylov_space_brute_force():
    A, M, H, b, omega = small_system()
    K, rhs = O.block_system(A, M, H, b, omega)
    k = 7
    basis = [rhs]
    for _ in range(k - 1):
        basis.append(K @ basis[-1])
    Kr = np.stack(basis, axis=1)
    Q, _ = np.linalg.qr(Kr)                                 # well-conditioned basis of the same space
    y, *_ = np.linalg.lstsq(K @ Q, rhs, rcond=None)
    x_ref = Q @ y
    hist = []
    x, its = O.minres(K, rhs, tol=0.0, max_iters=k, history=hist)
    assert its == k
    assert np.linalg.norm(x - x_ref) < 1e-9 * np.linalg.norm(x_ref)
    # the recurrence's residual norm is the true residual norm
    assert abs(hist[-1] - np.linalg.norm(rhs - K @ x) / np.linalg.norm(rhs)) < 1e-10
    assert all(hist[i + 1] <= hist[i] * (1 + 1e-12) for i in range(len(hist) - 1))


def test_minres_converges_to_the_direct_solution_and_agrees_with_scipy():
    inp = make_config(1, n=8, sub_elems=8)
    pr = O.Problem(inp.nx, inp.ny, inp.p, inp.x0, inp.y0, inp.x1, inp.y1, inp.c_nodes, inp.omega,
                   inp.f_re.astype(complex))
    A, M, H, b = O.assemble_global(pr)
    K, rhs = O.block_system(A, M, H, b, pr.omega)
    x, its = O.minres(K, rhs, tol=1e-12, max_iters=5000)
    n = len(b)
    u = x[:n] + 1j * x[n:]
    ustar = O.direct_solve(pr).reshape(-1)
    assert np.linalg.norm(u - ustar) < 1e-9 * np.linalg.norm(ustar)
    assert np.linalg.norm(rhs - K @ x) <= 2e-12 * np.linalg.norm(rhs)
    xs, info = spla.minres(K, rhs, rtol=1e-12, maxiter=5000)
    assert info == 0 and np.linalg.norm(xs - x) < 1e-8 * np.linalg.norm(x)
    # the same number of Lanczos steps as scipy's implementation needs, within a few
    cnt = [0]
    spla.minres(K, rhs, rtol=1e-12, maxiter=5000, callback=lambda xk: cnt.__setitem__(0, cnt[0] + 1))
    assert abs(cnt[0] - its) <= max(5, its // 20)


def test_ddm_with_minres_subdomain_solves_reaches_the_direct_solution():
    inp = make_config(1)
    pr = O.Problem(inp.nx, inp.ny, inp.p, inp.x0, inp.y0, inp.x1, inp.y1, inp.c_nodes, inp.omega,
                   inp.f_re.astype(complex))
    st = O.ddm_setup(pr, inp.sx, inp.sy)
    for _ in range(60):
        O.ddm_sweep_minres(st, 1e-12, 5000, True, 0.5)
    ustar = O.direct_solve(pr)
    err = np.linalg.norm(O.ddm_gather(st) - ustar) / np.linalg.norm(ustar)
    assert err < 1e-5, err       # exact subdomain solves + relaxed iteration: 2.6e-8 after 100 sweeps [SURVEY R12 probe]
