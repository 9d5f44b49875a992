"""GPU parity of the 3-D hexahedral variant (include/hz3.h) against oracle/hz_oracle3d.py, element by
element after identical iteration counts: fp64 <= 1e-10, fp32 <= 1e-4 (north_star's bar)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import hz_oracle3d as O  # noqa: E402
from paper_2606_21695_b200 import hz, hz3  # noqa: E402
from paper_2606_21695_b200.inputs import Hz3Inputs, make_config_3d  # noqa: E402

TOL = {hz.HZ_F64: 1e-10, hz.HZ_F32: 1e-4}


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(np.asarray(b)), 1e-300))


def problem_from(inp, bc=None):
    f = inp.f_re.astype(complex)
    if inp.f_im is not None:
        f = f + 1j * inp.f_im
    return O.Problem3D(inp.nx, inp.ny, inp.nz, inp.p, inp.box, inp.c_nodes, inp.omega, f, bc)


def pack_bc(inp, bc):
    if bc is None:
        return None
    npz, npy, npx = inp.shape
    FB = max(npy * npz, npx * npz, npx * npy)
    out = np.zeros((6, 2, FB))
    for f in range(6):
        a = np.asarray(bc[f]).reshape(-1)
        out[f, 0, :a.size], out[f, 1, :a.size] = a.real, a.imag
    return out


def check_case(inp, prec, n_outer=2, n_wh=2, warm=True, relax=0.5, bc=None, nodes_per_thread=0):
    assert torch.cuda.is_available(), "CUDA device required (there is no CPU fallback)"
    pr = problem_from(inp, bc)
    st = O.ddm_setup(pr, inp.sx, inp.sy, inp.sz, inp.cfl_frac)
    for _ in range(n_outer):
        O.ddm_sweep(st, n_wh, warm, relax)
    ug = O.ddm_gather(st)
    ctx = hz3.hz3_mesh_setup(inp.nx, inp.ny, inp.nz, inp.box, inp.p, inp.c_nodes, inp.omega, inp.f_re, inp.f_im,
                             pack_bc(inp, bc))
    try:
        info = hz3.hz3_partition(ctx, inp.sx, inp.sy, inp.sz, prec, inp.cfl_frac, nodes_per_thread)
        assert info.n_t == st.tab.n_t, "N_t must be reproduced independently"
        dt = torch.float64 if prec == hz.HZ_F64 else torch.float32
        nn = int(np.prod(inp.shape))
        u_out = torch.zeros(2 * nn, dtype=dt, device="cuda")
        s = hz3.hz3_ddm_solve(ctx, n_outer, n_wh=n_wh, warm_start=warm, relax=relax, reset_state=True,
                              u_out_ptr=u_out.data_ptr(), stream=torch.cuda.current_stream().cuda_stream)
        assert s.n_outer_done == n_outer and s.launches == 2 * n_outer + 1
        L, N, F = info.blocks, info.dofs_per_sub, info.face_stride
        usub = torch.zeros(L * 2 * N, dtype=torch.float64, device="cuda")
        lam = torch.zeros(L * 12 * F, dtype=torch.float64, device="cuda")
        hz3.hz3_get_subdomain_state(ctx, usub.data_ptr(), lam.data_ptr())
        usub = usub.cpu().numpy().reshape(L, 2, N)
        lam = lam.cpu().numpy().reshape(L, 6, 2, F)
        u_o = np.stack([np.stack([st.u[l].real, st.u[l].imag]) for l in range(L)])
        lam_o = np.zeros_like(lam)
        for l in range(L):
            for f in range(6):
                a = st.lam[l][f].reshape(-1)
                lam_o[l, f, 0, :a.size], lam_o[l, f, 1, :a.size] = a.real, a.imag
        tol = TOL[prec]
        assert rel(usub, u_o) <= tol, f"u_l: {rel(usub, u_o):.3e}"
        assert rel(lam, lam_o) <= tol, f"lambda: {rel(lam, lam_o):.3e}"
        u = u_out.double().cpu().numpy().reshape((2,) + inp.shape)
        assert rel(u[0] + 1j * u[1], ug) <= tol
        # the residual kernel applied to the ORACLE's field against the oracle's residual of it
        t = torch.from_numpy(np.concatenate([ug.real.ravel(), ug.imag.ravel()])).cuda()
        r_o = O.residual(pr, ug)
        assert abs(hz3.hz3_residual(ctx, t.data_ptr(), hz.HZ_F64) - r_o) <= 1e-9 * r_o
        return info
    finally:
        hz3.hz3_destroy(ctx)


@pytest.mark.parametrize("prec", [hz.HZ_F64, hz.HZ_F32])
@pytest.mark.parametrize("p,n,s", [(1, 8, 4), (2, 4, 2), (3, 4, 2), (4, 2, 1)])
@pytest.mark.parametrize("col", [True, False])
def test_cube_all_degrees(prec, p, n, s, col):
    # col: one thread per node column along z (k3_sweep_col); else one thread per node (k3_sweep_dof)
    info = check_case(make_config_3d(n, p, s, seed=3000 + p), prec, n_outer=3, n_wh=2, nodes_per_thread=0 if col else 1)
    assert info.dofs_per_sub == (s * p + 1) ** 3 and info.blocks == (n // s) ** 3
    assert info.nodes_per_thread == (s * p + 1 if col else 1)


def test_column_kernel_falls_back_when_the_column_length_is_not_compiled():
    # 3 elements of degree 2 along z: lnz = 7 is not an instantiated column length for p = 2 -> one node per thread
    info = check_case(make_config_3d((2, 2, 3), 2, (2, 2, 3), seed=8), hz.HZ_F64, n_outer=2, n_wh=2)
    assert info.nodes_per_thread == 1


def test_anisotropic_box_boundary_data_complex_source_cold_start():
    # hx != hy != hz, ex != ey != ez, complex f, non-zero datum on all six faces, unequal subdomain grid 2x3x1
    inp = make_config_3d((4, 6, 2), 2, (2, 2, 2), seed=11, box=(0.0, 0.0, 0.0, 1.3, 0.9, 0.5))
    rng = np.random.default_rng(4)
    f_im = rng.standard_normal(inp.shape)
    inp = Hz3Inputs(**{**inp.__dict__, "f_im": f_im})
    npz, npy, npx = inp.shape
    shapes = [(npz, npy), (npz, npy), (npz, npx), (npz, npx), (npy, npx), (npy, npx)]
    bc = [rng.standard_normal(sh) + 1j * rng.standard_normal(sh) for sh in shapes]
    check_case(inp, hz.HZ_F64, n_outer=3, n_wh=2, warm=False, bc=bc)
    check_case(inp, hz.HZ_F64, n_outer=2, n_wh=3, warm=True, relax=1.0, bc=bc)


def test_paper_block_shapes():
    # P=3 with 4 elements per subdomain... here the cubic shapes that fit 1024 threads: P=1 8^3 elements
    # (729 nodes), P=3 2^3 elements (343 nodes), P=1 with 2x2x1 subdomains of 8x8x8
    check_case(make_config_3d((16, 16, 8), 1, 8, seed=21), hz.HZ_F32, n_outer=2, n_wh=2)
    check_case(make_config_3d(6, 3, 3, seed=22), hz.HZ_F64, n_outer=2, n_wh=1)     # 10^3 = 1000 nodes per subdomain


def test_converges_to_the_direct_solve():
    inp = make_config_3d(4, 2, 2, seed=5, ppw=10.0)
    uref = O.direct_solve(problem_from(inp))
    ctx = hz3.hz3_mesh_setup(inp.nx, inp.ny, inp.nz, inp.box, inp.p, inp.c_nodes, inp.omega, inp.f_re)
    try:
        hz3.hz3_partition(ctx, inp.sx, inp.sy, inp.sz, hz.HZ_F64)
        u_out = torch.zeros(2 * int(np.prod(inp.shape)), dtype=torch.float64, device="cuda")
        # residual-based stop outside the sweep (hz3_solve_opts.tol / check_every)
        r = hz3.hz3_ddm_solve(ctx, 20000, n_wh=5, reset_state=True, u_out_ptr=u_out.data_ptr(), tol=1e-7, check_every=100)
        u = u_out.cpu().numpy().reshape((2,) + inp.shape)
        assert r.rel_residual <= 1e-7 and r.n_outer_done < 20000 and r.n_outer_done % 100 == 0
        assert abs(hz3.hz3_residual(ctx, u_out.data_ptr(), hz.HZ_F64) - r.rel_residual) <= 1e-9 * r.rel_residual
        assert rel(u[0] + 1j * u[1], uref) < 1e-6
    finally:
        hz3.hz3_destroy(ctx)


def test_errors():
    inp = make_config_3d(4, 3, 2)
    with pytest.raises(hz.HzError) as e:
        hz3.hz3_mesh_setup(4, 4, 4, inp.box, 7, inp.c_nodes, inp.omega, inp.f_re)
    assert e.value.status == hz.HZ_EUNSUPPORTED
    ctx = hz3.hz3_mesh_setup(inp.nx, inp.ny, inp.nz, inp.box, inp.p, inp.c_nodes, inp.omega, inp.f_re)
    try:
        with pytest.raises(hz.HzError) as e:
            hz3.hz3_partition(ctx, 3, 1, 1, hz.HZ_F64)            # does not divide
        assert e.value.status == hz.HZ_EINVAL
        with pytest.raises(hz.HzError) as e:
            hz3.hz3_partition(ctx, 1, 1, 1, hz.HZ_F64)            # 13^3 nodes > 1024 threads
        assert e.value.status == hz.HZ_EUNSUPPORTED
        with pytest.raises(hz.HzError) as e:
            hz3.hz3_ddm_solve(ctx, 1)                             # not partitioned
        assert e.value.status == hz.HZ_ESTATE
    finally:
        hz3.hz3_destroy(ctx)
