"""GPU parity of the Krylov-accelerated outer iteration (hz_ddm_solve_gmres) against the oracle's
ddm_gmres after IDENTICAL Arnoldi step counts, and its convergence to the direct solve.

Tolerance: the GMRES iterate is the unique minimiser of ||c - (I-T)x|| over the Krylov space, but the two
sides orthogonalise differently (oracle: modified Gram-Schmidt; library: classical Gram-Schmidt twice) and
sum the inner products in different orders, so fp64 agreement is limited by the conditioning of the small
least-squares problem rather than by 1e-10 per sweep: the bound used is 1e-9 on the state and on the
residual history (measured ~1e-12); fp32 1e-4 as everywhere."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import hz_oracle as O  # noqa: E402
from paper_2606_21695_b200 import hz  # noqa: E402
from paper_2606_21695_b200.inputs import make_config  # noqa: E402
from test_gpu_parity import oracle_state_arrays, problem_from, rel  # noqa: E402  (tests/ is on sys.path)


def gpu_gmres(inp, prec, k, **kw):
    ctx, info = hz.setup_from_inputs(inp, prec, k)
    try:
        dt = torch.float64 if prec == hz.HZ_F64 else torch.float32
        u = torch.zeros(2 * inp.npx * inp.npy, dtype=dt, device="cuda")
        ginfo, hist = hz.hz_ddm_solve_gmres(ctx, u_out_ptr=u.data_ptr(), want_history=True, **kw)
        usub = torch.zeros(info.blocks * 2 * info.dofs_per_sub, dtype=torch.float64, device="cuda")
        lam = torch.zeros(info.blocks * 8 * info.edge_stride, dtype=torch.float64, device="cuda")
        hz.hz_get_subdomain_state(ctx, usub.data_ptr(), lam.data_ptr())
        ug = u.double().cpu().numpy().reshape(2, inp.npy, inp.npx)
        return dict(ginfo=ginfo, hist=hist, u=ug[0] + 1j * ug[1],
                    usub=usub.cpu().numpy().reshape(info.blocks, 2, info.dofs_per_sub),
                    lam=lam.cpu().numpy().reshape(info.blocks, 4, 2, info.edge_stride))
    finally:
        hz.hz_destroy(ctx)


@pytest.mark.parametrize("prec,k,tol", [(hz.HZ_F64, 0, 1e-9), (hz.HZ_F64, 1, 1e-9), (hz.HZ_F32, 0, 1e-4)])
def test_gmres_iterates_match_the_oracle(prec, k, tol):
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    inp = make_config(2, n=24)           # 3x3 subdomains of 8x8 elements, Y-guide
    steps, restart = 14, 6                # two restarts inside the run
    st, hist_o = O.ddm_gmres(problem_from(inp), inp.sx, inp.sy, 2, 0.5, restart=restart, n_steps=steps)
    g = gpu_gmres(inp, prec, k, max_steps=steps, n_wh=2, relax=0.5, restart=restart)
    assert g["ginfo"].steps_done == steps and g["ginfo"].cycles == 3
    u_o, lam_o = oracle_state_arrays(st)
    assert rel(g["usub"], u_o) <= tol, rel(g["usub"], u_o)
    assert rel(g["lam"], lam_o) <= tol, rel(g["lam"], lam_o)
    assert np.allclose(g["hist"], hist_o[1:], rtol=max(tol, 1e-9) * 100, atol=0)
    # the reported Helmholtz residual is the oracle's residual of the oracle's iterate
    r_o = O.residual(problem_from(inp), O.ddm_gather(st))
    assert abs(g["ginfo"].rel_residual - r_o) <= (1e-6 if prec == hz.HZ_F64 else 1e-2) * r_o


def test_gmres_reaches_the_direct_solution_with_far_fewer_sweeps_than_the_plain_iteration():
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    inp = make_config(1)
    ustar = O.direct_solve(problem_from(inp))
    g = gpu_gmres(inp, hz.HZ_F64, 0, max_steps=300, n_wh=2, relax=0.5, restart=60, tol=1e-9)
    assert g["ginfo"].rel_residual <= 1e-9
    assert rel(g["u"], ustar) < 1e-8
    assert g["ginfo"].sweeps_done < 150       # the relaxed fixed-point iteration needs 320 sweeps for 1e-8


def test_gmres_continues_from_the_current_state():
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    inp = make_config(1)
    ctx, info = hz.setup_from_inputs(inp, hz.HZ_F64, 0)
    try:
        a = hz.hz_ddm_solve_gmres(ctx, 20, restart=20, reset_state=True)
        b = hz.hz_ddm_solve_gmres(ctx, 20, restart=20, reset_state=False)
        assert b.rel_residual < a.rel_residual
    finally:
        hz.hz_destroy(ctx)


# ---------------------------------------------------------------- Krylov iteration on lambda alone (lambda_only = 1)
@pytest.mark.parametrize("prec,k,tol", [(hz.HZ_F64, 0, 1e-9), (hz.HZ_F64, 1, 1e-9), (hz.HZ_F32, 0, 1e-4)])
def test_lambda_only_gmres_iterates_match_the_oracle(prec, k, tol):
    """Same Arnoldi step counts (two restarts inside the run), cold-started sweeps of 3 WaveHoltz iterations, the field
    polished by 2 more at the final lambda: lambda, u_l and the residual history against oracle.ddm_gmres(lambda_only)."""
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    inp = make_config(2, n=24)           # 3x3 subdomains of 8x8 elements, Y-guide
    steps, restart = 14, 6
    st, hist_o = O.ddm_gmres(problem_from(inp), inp.sx, inp.sy, 3, 0.5, restart=restart, n_steps=steps, lambda_only=True,
                             n_polish=2)
    g = gpu_gmres(inp, prec, k, max_steps=steps, n_wh=3, relax=0.5, restart=restart, lambda_only=True, n_polish=2)
    assert g["ginfo"].steps_done == steps and g["ginfo"].cycles == 3
    u_o, lam_o = oracle_state_arrays(st)
    assert rel(g["lam"], lam_o) <= tol, rel(g["lam"], lam_o)
    assert rel(g["usub"], u_o) <= tol, rel(g["usub"], u_o)
    assert np.allclose(g["hist"], hist_o[1:], rtol=max(tol, 1e-9) * 100, atol=0)
    r_o = O.residual(problem_from(inp), O.ddm_gather(st))
    assert abs(g["ginfo"].rel_residual - r_o) <= (1e-6 if prec == hz.HZ_F64 else 1e-2) * r_o
    # the basis vectors have the size of the interface data, not of the joint state
    assert g["ginfo"].krylov_bytes * 5 < (restart + 3) * g["usub"].size * (8 if prec == hz.HZ_F64 else 4)


def test_lambda_only_gmres_reaches_the_direct_solution_with_tight_subdomain_solves():
    """Config 1, rho = 1 (eq. (2) literally), 40 cold-started WaveHoltz iterations per sweep: the fixed point of the
    lambda-only map is then the discrete solution to 1e-8 (oracle pin of the same statement)."""
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required")
    inp = make_config(1)
    ustar = O.direct_solve(problem_from(inp))
    g = gpu_gmres(inp, hz.HZ_F64, 0, max_steps=60, n_wh=40, relax=1.0, restart=60, lambda_only=True)
    assert g["ginfo"].lin_residual <= 1e-8        # (the oracle's history stagnates at 3.5e-9: the Krylov space is exhausted)
    assert rel(g["u"], ustar) < 1e-8
    assert g["ginfo"].rel_residual < 1e-7
