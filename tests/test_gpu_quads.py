"""GPU parity of the general-quadrilateral path (hz_mesh_setup_quads, hz_sweep_quad.cuh) against
the oracle's general-geometry operators, element by element, same bar as tests/test_gpu_parity.py."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import hz_oracle as O  # noqa: E402
from paper_2606_21695_b200 import hz  # noqa: E402
from paper_2606_21695_b200.inputs import HzInputs, distorted_vertices, make_config, mapped_node_coords  # noqa: E402
from test_gpu_parity import check_case, problem_from, rel, run_gpu, TOL  # noqa: E402


def quad_inputs(nx, ny, p, sx, sy, seed, amp=0.2, complex_f=False, move_boundary=False):
    """Non-square distorted mesh, smoothly random c, random f."""
    rng = np.random.default_rng(seed)
    VX, VY = distorted_vertices(nx, ny, rng, amp, 0.0, 0.0, 1.5, 0.8)
    if move_boundary:   # a general polygonal domain: boundary vertices move too
        VX = VX + 0.1 * (1.5 / nx) * rng.uniform(-1, 1, VX.shape)
        VY = VY + 0.1 * (0.8 / ny) * rng.uniform(-1, 1, VY.shape)
    shape = (ny * p + 1, nx * p + 1)
    c = 1.0 + rng.uniform(0, 1.5, size=shape)
    f_re = rng.standard_normal(shape)
    f_im = rng.standard_normal(shape) if complex_f else None
    omega = 2.0 * np.pi * p * nx / 10.0 / 1.5
    return HzInputs(name=f"quads_{nx}x{ny}_p{p}", nx=nx, ny=ny, p=p, x0=0.0, y0=0.0, x1=1.5, y1=0.8, omega=omega,
                    c_nodes=c, f_re=f_re, f_im=f_im, sx=sx, sy=sy, seed=seed, vx=VX, vy=VY)


@pytest.mark.parametrize("p", [1, 2, 3, 4])
def test_quads_all_degrees_fp64(p):
    g = check_case(quad_inputs(8, 6, p, 2, 2, seed=200 + p), hz.HZ_F64, 0, n_outer=3, n_wh=2)
    assert g["info"].dofs_per_thread == (p + 1) ** 2 and g["info"].threads_per_block == 32


@pytest.mark.parametrize("p", [1, 2, 3, 4])
def test_quads_all_degrees_fp32(p):
    check_case(quad_inputs(8, 8, p, 2, 2, seed=300 + p), hz.HZ_F32, 0, n_outer=3, n_wh=2)


def test_quads_boundary_data_complex_source_cold_start_polygonal_domain():
    inp = quad_inputs(9, 6, 3, 3, 2, seed=77, complex_f=True, move_boundary=True)
    rng = np.random.default_rng(5)
    bc = [rng.standard_normal(n) + 1j * rng.standard_normal(n) for n in (inp.npy, inp.npy, inp.npx, inp.npx)]
    check_case(inp, hz.HZ_F64, 0, n_outer=3, n_wh=2, warm=False, bc=bc)
    check_case(inp, hz.HZ_F64, 0, n_outer=2, n_wh=3, warm=True, relax=1.0, bc=bc)


def test_quads_single_subdomain_and_strip_partitions():
    check_case(quad_inputs(6, 4, 2, 1, 1, seed=31), hz.HZ_F64, 0, n_outer=2, n_wh=2)
    check_case(quad_inputs(6, 4, 3, 6, 1, seed=32), hz.HZ_F64, 0, n_outer=3, n_wh=2)   # one element wide
    check_case(quad_inputs(4, 6, 3, 1, 6, seed=33), hz.HZ_F64, 0, n_outer=3, n_wh=2)


@pytest.mark.parametrize("prec", [hz.HZ_F64, hz.HZ_F32])
def test_quads_config3_block_shape_several_warps(prec):
    # config-3 block shape (8x8 elements, p=3: 64 element threads = 2 warps) on a distorted mesh, 3x3 subdomains
    check_case(make_config(3, n=24, distort=0.2), prec, 0, n_outer=2, n_wh=2)


def test_quads_large_subdomain_more_than_256_elements():
    # 18x18 = 324 elements per subdomain: the 1024-thread instantiation (fp32: the fp64 strips exceed one SM)
    check_case(make_config(2, n=18, p=2, sub_elems=18, distort=0.15), hz.HZ_F32, 0, n_outer=1, n_wh=1)


def test_rectangles_through_the_quad_path_match_the_rectangular_oracle():
    # uniform rectangles given as vertices: the general-geometry kernels against the oracle's RECTANGULAR operators
    inp = make_config(2, n=16)
    gx = np.linspace(0.0, 1.0, inp.nx + 1)
    VX, VY = np.meshgrid(gx, gx, indexing="xy")
    pr = problem_from(inp)                                        # no vertices: rectangular oracle path
    st = O.ddm_solve(pr, inp.sx, inp.sy, 3, 2)
    inp_q = HzInputs(**{**inp.__dict__, "vx": VX, "vy": VY})
    g = run_gpu(inp_q, hz.HZ_F64, 0, 3, 2, True, 0.5)
    assert g["info"].n_t == st.tab.n_t
    assert rel(g["u"], O.ddm_gather(st)) <= TOL[hz.HZ_F64]


def test_quads_converge_to_the_direct_solve_and_replicated_nodes_stay_consistent():
    inp = make_config(1, n=8, p=2, sub_elems=4, distort=0.2)
    pr = problem_from(inp)
    uref = O.direct_solve(pr)
    ctx, info = hz.setup_from_inputs(inp, hz.HZ_F64, 0)
    try:
        u_out = torch.zeros(2 * inp.npx * inp.npy, dtype=torch.float64, device="cuda")
        r = hz.hz_ddm_solve(ctx, 900, n_wh=5, tol=1e-11, check_every=50, reset_state=True, use_graph=True,
                            u_out_ptr=u_out.data_ptr())
        u = u_out.cpu().numpy().reshape(2, inp.npy, inp.npx)
        assert r.rel_residual <= 1e-11
        assert rel(u[0] + 1j * u[1], uref) < 1e-10
        # GMRES on (lambda, u) drives the same kernel
        r2 = hz.hz_ddm_solve_gmres(ctx, 400, n_wh=2, restart=40, tol=1e-10, reset_state=True,
                                   u_out_ptr=u_out.data_ptr())
        u = u_out.cpu().numpy().reshape(2, inp.npy, inp.npx)
        assert rel(u[0] + 1j * u[1], uref) < 1e-8, r2.rel_residual
    finally:
        hz.hz_destroy(ctx)


@pytest.mark.parametrize("prec", [hz.HZ_F64, hz.HZ_F32])
def test_ragged_partitions(prec):
    # 11x7 elements in 3x2 subdomains: 4,4,3 x 4,3 elements; blocks sized for 4x4, the smaller ones idle threads
    inp = quad_inputs(11, 7, 3, 3, 2, seed=91)
    rng = np.random.default_rng(6)
    bc = [rng.standard_normal(n) + 1j * rng.standard_normal(n) for n in (inp.npy, inp.npy, inp.npx, inp.npx)]
    g = check_case(inp, prec, 0, n_outer=3, n_wh=2, bc=bc)
    assert g["info"].dofs_per_sub == 13 * 13 and g["info"].blocks == 6
    # 7x5 in 3x2 (3,2,2 x 3,2), p = 2, and a partition into single elements and pairs (5 in 3: 2,2,1)
    check_case(quad_inputs(7, 5, 2, 3, 2, seed=92), prec, 0, n_outer=3, n_wh=2)
    check_case(quad_inputs(5, 5, 4, 3, 3, seed=93), prec, 0, n_outer=2, n_wh=2)


def test_ragged_rectangles_converge_to_the_direct_solve():
    # uniform rectangles as vertices, 10x10 elements in 3x3 subdomains (4,3,3): converged field == direct solve
    inp = make_config(1, n=10, p=2, sub_elems=10)
    gx = np.linspace(0.0, 1.0, inp.nx + 1)
    VX, VY = np.meshgrid(gx, gx, indexing="xy")
    inp = HzInputs(**{**inp.__dict__, "vx": VX, "vy": VY, "sx": 3, "sy": 3})
    uref = O.direct_solve(O.Problem(inp.nx, inp.ny, inp.p, 0, 0, 1, 1, inp.c_nodes, inp.omega, inp.f_re.astype(complex)))
    ctx, info = hz.setup_from_inputs(inp, hz.HZ_F64, 0)
    try:
        u_out = torch.zeros(2 * inp.npx * inp.npy, dtype=torch.float64, device="cuda")
        r = hz.hz_ddm_solve(ctx, 2000, n_wh=5, tol=1e-11, check_every=50, reset_state=True, use_graph=True,
                            u_out_ptr=u_out.data_ptr())
        u = u_out.cpu().numpy().reshape(2, inp.npy, inp.npx)
        assert r.rel_residual <= 1e-11 and rel(u[0] + 1j * u[1], uref) < 1e-9
    finally:
        hz.hz_destroy(ctx)


def test_quads_errors():
    inp = quad_inputs(4, 4, 2, 2, 2, seed=1)
    bad = inp.vx.copy()
    bad[2, 2] += 1.0                                              # folds an element over
    with pytest.raises(hz.HzError) as e:
        hz.hz_mesh_setup_quads(inp.nx, inp.ny, inp.p, bad, inp.vy, inp.c_nodes, inp.omega, inp.f_re)
    assert e.value.status == hz.HZ_EINVAL
    ctx = hz.hz_mesh_setup_quads(inp.nx, inp.ny, inp.p, inp.vx, inp.vy, inp.c_nodes, inp.omega, inp.f_re)
    try:
        with pytest.raises(hz.HzError) as e:
            hz.hz_partition(ctx, 2, 2, prec=hz.HZ_F64, dofs_per_thread=1)
        assert e.value.status == hz.HZ_EUNSUPPORTED
        with pytest.raises(hz.HzError) as e:
            hz.hz_partition(ctx, 5, 2, prec=hz.HZ_F64, dofs_per_thread=0)      # more subdomain columns than elements
        assert e.value.status == hz.HZ_EINVAL
        hz.hz_partition(ctx, 2, 2, prec=hz.HZ_F64, dofs_per_thread=0)
        with pytest.raises(hz.HzError) as e:
            hz.hz_minres_cycle(ctx, 4, 1e-6, 10, False, 0.5)
        assert e.value.status == hz.HZ_EUNSUPPORTED
    finally:
        hz.hz_destroy(ctx)


def test_sources_stream_and_set_source_on_a_quad_context():
    # hz_set_source rebuilds the load with the general-geometry mass; hz_ddm_solve_sources does the same from its
    # staging buffers: both against the oracle with the new source
    inp = quad_inputs(8, 6, 2, 2, 2, seed=55)
    rng = np.random.default_rng(2)
    f2 = rng.standard_normal(inp.f_re.shape)
    inp2 = HzInputs(**{**inp.__dict__, "f_re": f2})
    st = O.ddm_solve(problem_from(inp2), inp.sx, inp.sy, 2, 2)
    ref = O.ddm_gather(st)
    nn = inp.npx * inp.npy
    ctx, info = hz.setup_from_inputs(inp, hz.HZ_F64, 0)           # set up with the OLD source
    try:
        u = torch.zeros(2 * nn, dtype=torch.float64, device="cuda")
        hz.hz_set_source(ctx, f2)
        hz.hz_ddm_solve(ctx, 2, n_wh=2, reset_state=True, u_out_ptr=u.data_ptr())
        a = u.cpu().numpy().reshape(2, inp.npy, inp.npx)
        assert rel(a[0] + 1j * a[1], ref) <= 1e-10
        f_pin = [torch.from_numpy(np.ascontiguousarray(f)).pin_memory() for f in (inp.f_re, f2)]
        u_pin = [torch.empty(2 * nn, dtype=torch.float64).pin_memory() for _ in range(2)]
        hz.hz_ddm_solve_sources(ctx, [t.data_ptr() for t in f_pin], [t.data_ptr() for t in u_pin], n_outer=2, n_wh=2,
                                reset_state=True)
        b = u_pin[1].numpy().reshape(2, inp.npy, inp.npx)
        assert rel(b[0] + 1j * b[1], ref) <= 1e-10
    finally:
        hz.hz_destroy(ctx)
