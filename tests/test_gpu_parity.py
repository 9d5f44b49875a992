"""GPU parity: the CUDA path (through the C ABI, paper_2606_21695_b200.hz) against the CPU oracle
(oracle/hz_oracle.py), element by element, after IDENTICAL iteration counts on the same seeded inputs.

Bar (BASELINE.json north_star): fp64 relative L2 <= 1e-10, fp32 <= 1e-4 -- on the raw per-subdomain
states u_l, on the interface data lambda, and on the gathered global field.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import hz_oracle as O  # noqa: E402
from paper_2606_21695_b200 import hz  # noqa: E402
from paper_2606_21695_b200.inputs import HzInputs, make_config  # noqa: E402

TOL = {hz.HZ_F64: 1e-10, hz.HZ_F32: 1e-4}


def _require_cuda():
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (there is no CPU fallback)")


def problem_from(inp, bc=None):
    f = inp.f_re.astype(complex)
    if inp.f_im is not None:
        f = f + 1j * inp.f_im
    return O.Problem(inp.nx, inp.ny, inp.p, inp.x0, inp.y0, inp.x1, inp.y1, inp.c_nodes, inp.omega, f, bc,
                     vx=getattr(inp, "vx", None), vy=getattr(inp, "vy", None))


def pack_bc(inp, bc):
    """oracle bc_lambda (4 complex side arrays) -> the C ABI's 4 x (re[EB], im[EB]) block."""
    if bc is None:
        return None
    EB = max(inp.npx, inp.npy)
    out = np.zeros((4, 2, EB))
    for s in range(4):
        out[s, 0, :len(bc[s])] = bc[s].real
        out[s, 1, :len(bc[s])] = bc[s].imag
    return out


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(np.asarray(b)), 1e-300))


def oracle_state_arrays(st):
    L = len(st.subs)
    nxm, nym = max(sd.npx for sd in st.subs), max(sd.npy for sd in st.subs)   # ragged: padded to the largest
    N = nxm * nym
    E = max(nxm, nym)
    u = np.zeros((L, 2, N))
    lam = np.zeros((L, 4, 2, E))
    for l in range(L):
        sd = st.subs[l]
        u[l, 0].reshape(nym, nxm)[:sd.npy, :sd.npx] = st.u[l].real.reshape(sd.npy, sd.npx)
        u[l, 1].reshape(nym, nxm)[:sd.npy, :sd.npx] = st.u[l].imag.reshape(sd.npy, sd.npx)
        for s in range(4):
            a = st.lam[l][s]
            lam[l, s, 0, :len(a)], lam[l, s, 1, :len(a)] = a.real, a.imag
    return u, lam


def run_gpu(inp, prec, k, n_outer, n_wh, warm, relax, bc=None, res_field=None, flags=None):
    if getattr(inp, "vx", None) is not None:
        ctx = hz.hz_mesh_setup_quads(inp.nx, inp.ny, inp.p, inp.vx, inp.vy, inp.c_nodes, inp.omega, inp.f_re,
                                     inp.f_im, pack_bc(inp, bc))
    else:
        ctx = hz.hz_mesh_setup(inp.nx, inp.ny, inp.x0, inp.y0, inp.x1, inp.y1, inp.p, inp.c_nodes, inp.omega,
                               inp.f_re, inp.f_im, pack_bc(inp, bc))
    try:
        info = hz.hz_partition_ex(ctx, inp.sx, inp.sy, hz.HZ_TC_IMPEDANCE0, prec, k, inp.cfl_frac, **(flags or {}))
        dt = torch.float64 if prec == hz.HZ_F64 else torch.float32
        u_out = torch.zeros(2 * inp.npx * inp.npy, dtype=dt, device="cuda")
        sinfo = hz.hz_ddm_solve(ctx, n_outer, n_wh=n_wh, warm_start=warm, relax=relax, reset_state=True,
                                u_out_ptr=u_out.data_ptr(), stream=torch.cuda.current_stream().cuda_stream)
        usub = torch.zeros(info.blocks * 2 * info.dofs_per_sub, dtype=torch.float64, device="cuda")
        lam = torch.zeros(info.blocks * 8 * info.edge_stride, dtype=torch.float64, device="cuda")
        hz.hz_get_subdomain_state(ctx, usub.data_ptr(), lam.data_ptr())
        res = hz.hz_residual(ctx, u_out.data_ptr(), prec)
        res_of_field = None
        if res_field is not None:  # residual kernel (A10) applied to a field given by the caller
            t = torch.from_numpy(np.concatenate([res_field.real.ravel(), res_field.imag.ravel()])).cuda()
            res_of_field = hz.hz_residual(ctx, t.data_ptr(), hz.HZ_F64)
        u_glob = u_out.double().cpu().numpy().reshape(2, inp.npy, inp.npx)
        return dict(info=info, sinfo=sinfo, u=u_glob[0] + 1j * u_glob[1],
                    usub=usub.cpu().numpy().reshape(info.blocks, 2, info.dofs_per_sub),
                    lam=lam.cpu().numpy().reshape(info.blocks, 4, 2, info.edge_stride), res=res,
                    res_of_field=res_of_field)
    finally:
        hz.hz_destroy(ctx)


def check_case(inp, prec, k, n_outer=3, n_wh=2, warm=True, relax=0.5, bc=None, flags=None):
    _require_cuda()
    pr = problem_from(inp, bc)
    st = O.ddm_solve(pr, inp.sx, inp.sy, n_outer, n_wh, warm_start=warm, relax=relax, cfl_frac=inp.cfl_frac)
    ug = O.ddm_gather(st)
    g = run_gpu(inp, prec, k, n_outer, n_wh, warm, relax, bc, res_field=ug, flags=flags)
    assert g["info"].n_t == st.tab.n_t, "N_t must be reproduced independently (reading R9)"
    assert g["sinfo"].n_outer_done == n_outer
    if k:
        assert g["info"].dofs_per_thread == k
    u_o, lam_o = oracle_state_arrays(st)
    tol = TOL[prec]
    assert rel(g["usub"], u_o) <= tol, f"u_l: {rel(g['usub'], u_o):.3e}"
    assert rel(g["lam"], lam_o) <= tol, f"lambda: {rel(g['lam'], lam_o):.3e}"
    assert rel(g["u"], ug) <= tol, f"gathered u: {rel(g['u'], ug):.3e}"
    # the residual kernel (A10), applied to the ORACLE's field, against the oracle's residual of it
    r_o = O.residual(pr, ug)
    assert abs(g["res_of_field"] - r_o) <= 1e-9 * r_o, (g["res_of_field"], r_o)
    return g


def hetero_inputs(nx, ny, p, sx, sy, seed, complex_f=False, omega=None):
    """Non-square mesh (hx != hy, ex != ey), smoothly random c, random f: a transposed operand or an
    anisotropy mistake cannot cancel."""
    rng = np.random.default_rng(seed)
    shape = (ny * p + 1, nx * p + 1)
    c = 1.0 + rng.uniform(0, 1.5, size=shape)
    f_re = rng.standard_normal(shape)
    f_im = rng.standard_normal(shape) if complex_f else None
    if omega is None:
        omega = 2.0 * np.pi * p * nx / 10.0 / 1.5
    return HzInputs(name=f"hetero_{nx}x{ny}_p{p}", nx=nx, ny=ny, p=p, x0=0.0, y0=0.0, x1=1.5, y1=0.8, omega=omega,
                    c_nodes=c, f_re=f_re, f_im=f_im, sx=sx, sy=sy, seed=seed)


# ------------------------------------------------------------------ config 1 at full size (fp64)
@pytest.mark.parametrize("k", [1, 4])
def test_config1_full_fp64(k):
    check_case(make_config(1), hz.HZ_F64, k, n_outer=4, n_wh=5)


def test_config1_cold_start_algorithm1_literal():
    # warm_start = 0 is Algorithm 1 as printed (u^(0) <- 0)
    check_case(make_config(1), hz.HZ_F64, 1, n_outer=3, n_wh=3, warm=False)
    check_case(make_config(1), hz.HZ_F64, 4, n_outer=3, n_wh=3, warm=False)


# ------------------------------------------------------------------ configs 2/3 reduced (several tiles + ragged tail)
@pytest.mark.parametrize("prec", [hz.HZ_F64, hz.HZ_F32])
@pytest.mark.parametrize("k", [1, 9])
def test_config2_reduced(prec, k):
    # Y-waveguide, p=3, 4x4 subdomains of 8x8 elements (625 DOF each: the full-size block shape)
    check_case(make_config(2, n=32), prec, k, n_outer=3, n_wh=5)


@pytest.mark.parametrize("prec", [hz.HZ_F64, hz.HZ_F32])
def test_config3_reduced(prec):
    check_case(make_config(3, n=40), prec, 9, n_outer=3, n_wh=2)


@pytest.mark.parametrize("prec", [hz.HZ_F64, hz.HZ_F32])
def test_config4_reduced_large_subdomain(prec):
    # 2x2 subdomains of 16x16 elements (2401 DOF): only the register-blocked variant fits
    check_case(make_config(4, n=32, sub_elems=16), prec, 0, n_outer=2, n_wh=2)


# ------------------------------------------------------------------ degrees, tiles, anisotropy
@pytest.mark.parametrize("p,k", [(1, 1), (1, 4), (1, 16), (2, 1), (2, 4), (2, 16), (3, 1), (3, 9), (3, 18), (4, 1), (4, 16)])
def test_degrees_and_tiles_fp64(p, k):
    nx, ny = (8, 8) if k >= 16 and p <= 2 else (8, 4)
    if p == 1 and k == 16:
        nx, ny = 16, 8
    inp = hetero_inputs(nx, ny, p, 2, 2, seed=10 * p + k)
    check_case(inp, hz.HZ_F64, k, n_outer=3, n_wh=2)


@pytest.mark.parametrize("p,k", [(1, 4), (2, 16), (3, 9), (3, 18), (4, 16)])
def test_degrees_and_tiles_fp32(p, k):
    inp = hetero_inputs(8, 8, p, 2, 2, seed=100 + 10 * p + k)
    check_case(inp, hz.HZ_F32, k, n_outer=3, n_wh=2)


def test_complex_source_and_boundary_datum_one_dof_per_thread():
    inp = hetero_inputs(6, 4, 3, 3, 2, seed=77, complex_f=True)
    rng = np.random.default_rng(5)
    bc = [rng.standard_normal(n) + 1j * rng.standard_normal(n) for n in (inp.npy, inp.npy, inp.npx, inp.npx)]
    check_case(inp, hz.HZ_F64, 1, n_outer=3, n_wh=2, bc=bc)


def test_boundary_datum_register_blocked():
    inp = hetero_inputs(6, 4, 3, 3, 2, seed=78)
    rng = np.random.default_rng(6)
    bc = [rng.standard_normal(n) + 1j * rng.standard_normal(n) for n in (inp.npy, inp.npy, inp.npx, inp.npx)]
    check_case(inp, hz.HZ_F64, 9, n_outer=3, n_wh=2, bc=bc)


# ------------------------------------------------------------------ degenerate cases
@pytest.mark.parametrize("k", [1, 9])
def test_single_subdomain_is_plain_waveholtz(k):
    # L = 1: no interfaces, the exchange is a no-op (T5)
    inp = hetero_inputs(4, 4, 3, 1, 1, seed=3)
    check_case(inp, hz.HZ_F64, k, n_outer=2, n_wh=3)


def test_one_element_subdomains():
    inp = hetero_inputs(4, 3, 3, 4, 3, seed=4)
    check_case(inp, hz.HZ_F64, 9, n_outer=3, n_wh=2)
    check_case(inp, hz.HZ_F64, 1, n_outer=3, n_wh=2)


def test_zero_sweeps_returns_zero_field():
    _require_cuda()
    inp = make_config(1)
    g = run_gpu(inp, hz.HZ_F64, 0, 0, 1, True, 0.5)
    assert np.all(g["u"] == 0) and np.all(g["lam"] == 0)
    assert abs(g["res"] - 1.0) < 1e-14


def test_relaxation_one_is_equation_2_literally():
    check_case(make_config(1), hz.HZ_F64, 4, n_outer=4, n_wh=2, relax=1.0)


def test_continue_equals_one_shot():
    """Two calls of 2 sweeps (state kept in the context) == one call of 4 sweeps, bit for bit."""
    _require_cuda()
    inp = make_config(2, n=16)
    ctx, info = hz.setup_from_inputs(inp, hz.HZ_F64, 9)
    try:
        a = torch.zeros(2 * inp.npx * inp.npy, dtype=torch.float64, device="cuda")
        b = torch.zeros_like(a)
        hz.hz_ddm_solve(ctx, 4, n_wh=2, reset_state=True, u_out_ptr=a.data_ptr())
        hz.hz_ddm_solve(ctx, 2, n_wh=2, reset_state=True)
        hz.hz_ddm_solve(ctx, 2, n_wh=2, reset_state=False, u_out_ptr=b.data_ptr())
        assert torch.equal(a, b)
    finally:
        hz.hz_destroy(ctx)


def test_variants_agree_and_are_deterministic():
    _require_cuda()
    inp = make_config(2, n=16)
    g1 = run_gpu(inp, hz.HZ_F64, 1, 3, 2, True, 0.5)
    g9 = run_gpu(inp, hz.HZ_F64, 9, 3, 2, True, 0.5)
    g9b = run_gpu(inp, hz.HZ_F64, 9, 3, 2, True, 0.5)
    assert rel(g1["usub"], g9["usub"]) < 1e-11
    assert np.array_equal(g9["usub"], g9b["usub"]), "no atomics: runs must be bit-identical"


def test_converged_ddm_matches_direct_solve_and_tolerance_stop():
    """North star: converged DDM == direct solve of the global system (here the oracle's sparse LU),
    and the tol-driven stop of the driver reports a residual that hz_residual reproduces."""
    _require_cuda()
    inp = make_config(1)
    pr = problem_from(inp)
    ustar = O.direct_solve(pr)
    ctx, info = hz.setup_from_inputs(inp, hz.HZ_F64, 0)
    try:
        u = torch.zeros(2 * inp.npx * inp.npy, dtype=torch.float64, device="cuda")
        s = hz.hz_ddm_solve(ctx, 600, n_wh=2, warm_start=True, relax=0.5, tol=1e-9, check_every=10, reset_state=True,
                            u_out_ptr=u.data_ptr())
        assert s.n_outer_done < 600 and s.rel_residual <= 1e-9
        ug = u.cpu().numpy().reshape(2, inp.npy, inp.npx)
        assert rel(ug[0] + 1j * ug[1], ustar) < 1e-8
        assert abs(hz.hz_residual(ctx, u.data_ptr(), hz.HZ_F64) - s.rel_residual) <= 1e-6 * s.rel_residual
    finally:
        hz.hz_destroy(ctx)


def test_fp32_reaches_the_shared_residual_tolerance():
    """fp32 and fp64 reach the same final residual tolerance 1e-4 (reading R21)."""
    _require_cuda()
    inp = make_config(1)
    for prec in (hz.HZ_F64, hz.HZ_F32):
        ctx, info = hz.setup_from_inputs(inp, prec, 0)
        try:
            s = hz.hz_ddm_solve(ctx, 400, n_wh=2, tol=1e-4, check_every=5, reset_state=True)
            assert s.rel_residual <= 1e-4 and s.n_outer_done < 400
        finally:
            hz.hz_destroy(ctx)


def test_error_paths():
    _require_cuda()
    inp = make_config(1)
    with pytest.raises(hz.HzError) as e:
        hz.hz_mesh_setup(inp.nx, inp.ny, 0, 0, 1, 1, 7, inp.c_nodes, inp.omega, inp.f_re)
    assert e.value.status == hz.HZ_EUNSUPPORTED
    ctx = hz.hz_mesh_setup(inp.nx, inp.ny, 0, 0, 1, 1, inp.p, inp.c_nodes, inp.omega, inp.f_re)
    try:
        with pytest.raises(hz.HzError) as e:
            hz.hz_ddm_solve(ctx, 1)
        assert e.value.status == hz.HZ_ESTATE
        with pytest.raises(hz.HzError) as e:
            hz.hz_partition(ctx, 3, 2)
        assert e.value.status == hz.HZ_EINVAL
        with pytest.raises(hz.HzError) as e:
            hz.hz_partition(ctx, 2, 2, dofs_per_thread=7)
        assert e.value.status == hz.HZ_EUNSUPPORTED
        hz.hz_partition(ctx, 2, 2)
        with pytest.raises(hz.HzError) as e:
            hz.hz_ddm_solve(ctx, 1, n_wh=0)
        assert e.value.status == hz.HZ_EINVAL
    finally:
        hz.hz_destroy(ctx)


def test_graph_replay_is_bit_identical_to_plain_launches():
    """use_graph = 1 replays the captured {sweep, exchange} pairs: same kernels, same arguments."""
    _require_cuda()
    inp = make_config(2, n=16)
    ctx, info = hz.setup_from_inputs(inp, hz.HZ_F64, 0)
    try:
        a = torch.zeros(2 * inp.npx * inp.npy, dtype=torch.float64, device="cuda")
        b = torch.zeros_like(a)
        sa = hz.hz_ddm_solve(ctx, 23, n_wh=2, reset_state=True, u_out_ptr=a.data_ptr())
        sb = hz.hz_ddm_solve(ctx, 23, n_wh=2, reset_state=True, use_graph=True, tol=1e-30, check_every=5,
                             u_out_ptr=b.data_ptr())
        assert sa.n_outer_done == sb.n_outer_done == 23
        assert torch.equal(a, b)
        assert sb.sweep_ms_total == -1.0 and sb.total_ms > 0
    finally:
        hz.hz_destroy(ctx)


@pytest.mark.parametrize("prec", [hz.HZ_F64, hz.HZ_F32])
def test_streamed_fallback_variant(prec):
    """dofs_per_thread = -1: state in global scratch (the variant that covers subdomains too large for one SM)."""
    inp = hetero_inputs(6, 4, 3, 3, 2, seed=91, complex_f=True)
    rng = np.random.default_rng(8)
    bc = [rng.standard_normal(n) + 1j * rng.standard_normal(n) for n in (inp.npy, inp.npy, inp.npx, inp.npx)]
    g = check_case(inp, prec, -1, n_outer=3, n_wh=2, bc=bc)
    check_case(make_config(2, n=32), prec, -1, n_outer=2, n_wh=2)
    check_case(make_config(1), prec, -1, n_outer=3, n_wh=3, warm=False)


def test_auto_uses_a_cluster_when_one_sm_cannot_hold_the_state():
    # 2x2 subdomains of 32x32 elements, p=3, fp64: 9409 DOF x 6 values x 8 B = 452 KB > one SM (config-4 block shape)
    g = check_case(make_config(4, n=64, sub_elems=32), hz.HZ_F64, 0, n_outer=2, n_wh=1)
    assert g["info"].cluster_size > 1 and g["info"].dofs_per_thread == 9


def test_auto_falls_back_to_streamed_when_no_on_chip_variant_fits():
    # the same blocks with the cluster kernels switched off (as on a device without clusters): streamed fallback
    g = check_case(make_config(4, n=64, sub_elems=32), hz.HZ_F64, 0, n_outer=2, n_wh=1, flags=dict(cluster=-1))
    assert g["info"].dofs_per_thread == -1 and g["info"].cluster_size == 1


def test_more_than_256_time_steps_uses_the_shared_memory_table():
    """The register-blocked kernels take the time-step table as a kernel parameter (<= 256 rows); a finer CFL
    fraction must fall back to a variant that keeps the table in shared / global memory, with the same result."""
    inp = make_config(2, n=16)
    inp.cfl_frac = 0.2
    g = check_case(inp, hz.HZ_F64, 0, n_outer=2, n_wh=1)
    assert g["info"].n_t > 256 and g["info"].dofs_per_thread == 1


@pytest.mark.parametrize("prec,cl,k", [(hz.HZ_F64, 2, 9), (hz.HZ_F64, 4, 9), (hz.HZ_F32, 2, 9), (hz.HZ_F32, 8, 9), (hz.HZ_F64, 16, 9),
                                       (hz.HZ_F32, 2, 18), (hz.HZ_F32, 4, 18), (hz.HZ_F32, 8, 18)])
def test_cluster_kernel_matches_the_oracle(prec, cl, k):
    """Thread-block-cluster variants: the subdomain's tile grid is cut into column strips, one CTA each, with the
    strip-boundary chunks pushed through DSMEM.  k_sweep_cl (hz_sweep_cl.cuh; fp32 k = 9 with 2 or 8 CTAs, fp64 with 2)
    and k_sweep_cw (hz_sweep_cw.cuh: warp-specialised edge pieces; fp32 with 6x3 tiles, k = 18, fp64 k = 9 with 4 or 16
    CTAs).  Forced here on small subdomains (the automatic choice only uses clusters when one SM cannot hold the state)."""
    g = check_case(make_config(2, n=32, sub_elems=16 if cl >= 8 or k == 18 else None), prec, k, n_outer=3, n_wh=2,
                   flags=dict(cluster=cl))
    assert g["info"].cluster_size == cl
    if cl >= 8:      # 16 (beyond the portable size: opt-in attribute) and 8 need at least that many tile columns
        return
    inp = hetero_inputs(12, 4, 3, 2, 2, seed=55)      # 6x2-element subdomains: strips of unequal width
    rng = np.random.default_rng(12)
    bc = [rng.standard_normal(n) + 1j * rng.standard_normal(n) for n in (inp.npy, inp.npy, inp.npx, inp.npx)]
    if k == 18 and cl > 3:
        return                                        # 3 columns of 6x3 tiles: at most 3 strips
    g = check_case(inp, prec, k, n_outer=3, n_wh=2, warm=False, bc=bc, flags=dict(cluster=cl))
    assert g["info"].cluster_size == cl


def test_stream_of_sources_matches_the_sequential_calls_bit_for_bit():
    """hz_ddm_solve_sources (copies overlapped with the sweeps on private streams, double-buffered staging) against
    hz_set_source + hz_ddm_solve + device-to-host copy, source by source; then against the oracle for the last one."""
    _require_cuda()
    inp = make_config(2, n=32)
    rng = np.random.default_rng(9)
    nn = inp.npx * inp.npy
    srcs = [inp.f_re] + [inp.f_re * rng.uniform(0.5, 1.5) + 0.1 * rng.standard_normal(inp.f_re.shape) for _ in range(4)]
    for prec, dt in ((hz.HZ_F64, torch.float64), (hz.HZ_F32, torch.float32)):
        ctx, info = hz.setup_from_inputs(inp, prec, 0)
        try:
            f_pin = [torch.from_numpy(np.ascontiguousarray(f)).pin_memory() for f in srcs]
            u_pin = [torch.empty(2 * nn, dtype=dt).pin_memory() for _ in srcs]
            hz.hz_ddm_solve(ctx, 0, reset_state=True)
            r = hz.hz_ddm_solve_sources(ctx, [t.data_ptr() for t in f_pin], [t.data_ptr() for t in u_pin],
                                        n_outer=2, n_wh=2, stream=torch.cuda.current_stream().cuda_stream)
            assert r.sources_done == 5 and r.launches == 5 * (1 + 4 + 1)
            assert r.h2d_bytes == 5 * nn * 8 and r.d2h_bytes == 5 * 2 * nn * u_pin[0].element_size()
            res_last = hz.hz_residual(ctx, torch.from_numpy(np.zeros(2 * nn)).cuda().data_ptr(), hz.HZ_F64)
            assert abs(res_last - 1.0) < 1e-12                      # residual of u = 0 is 1: the context holds a source
            # sequential reference on the same context type
            hz.hz_ddm_solve(ctx, 0, reset_state=True)
            u_dev = torch.zeros(2 * nn, dtype=dt, device="cuda")
            for f, got in zip(srcs, u_pin):
                hz.hz_set_source(ctx, f)
                hz.hz_ddm_solve(ctx, 2, n_wh=2, u_out_ptr=u_dev.data_ptr())
                assert torch.equal(u_dev.cpu(), got), "pipelined and sequential paths must agree bit for bit"
        finally:
            hz.hz_destroy(ctx)


@pytest.mark.parametrize("prec,cl,k", [(hz.HZ_F32, 2, 9), (hz.HZ_F32, 4, 9), (hz.HZ_F32, 8, 9), (hz.HZ_F64, 2, 9), (hz.HZ_F64, 4, 9),
                                       (hz.HZ_F64, 8, 9), (hz.HZ_F64, 16, 9), (hz.HZ_F32, 2, 18), (hz.HZ_F32, 4, 18),
                                       (hz.HZ_F32, 8, 18)])      # every p = 3 cluster shape that is compiled
def test_cluster_halo_protocol_stress(prec, cl, k):
    """compute-sanitizer is closed on this GPU pool, so the two-slot halo protocol of hz_sweep_cl.cuh (st.async pushes
    into the adjacent CTA's shared memory, mbarrier transaction counts, no cluster barrier in the time loop) is
    stressed instead, for k_sweep_cl and k_sweep_cw (k = 18, and fp64 with 4 or 16 CTAs): many time steps with strips of
    UNEQUAL width (17, resp. 16 or 8, tile columns over cl CTAs; some strips are a single column), 20 repeats that must be bit-identical (a race shows as run-to-run noise), and the
    result must agree with the single-CTA kernel's to rounding (its edge pieces associate their sums differently)."""
    _require_cuda()
    inp = make_config(2, n=32, sub_elems=16)
    nn = inp.npx * inp.npy
    dt = torch.float64 if prec == hz.HZ_F64 else torch.float32

    def run(flags, reps):
        ctx, info = hz.setup_from_inputs(inp, prec, k if flags.get("cluster", 0) > 1 else 9, **flags)
        try:
            outs = []
            for _ in range(reps):
                u = torch.zeros(2 * nn, dtype=dt, device="cuda")
                hz.hz_ddm_solve(ctx, 6, n_wh=4, relax=0.5, reset_state=True, u_out_ptr=u.data_ptr())
                outs.append(u)
            return info, outs
        finally:
            hz.hz_destroy(ctx)

    info, outs = run(dict(cluster=cl, grid_blocks=4096), 20)   # grid_blocks: the register-capped instantiations compete too
    assert info.cluster_size == cl
    for u in outs[1:]:
        assert torch.equal(u, outs[0]), "cluster kernel is not deterministic: halo race"
    info1, ref = run(dict(cluster=-1), 1)
    assert info1.cluster_size == 1 and info1.dofs_per_thread == 9
    d = float((outs[0].double() - ref[0].double()).norm() / ref[0].double().norm())
    assert d <= (1e-12 if prec == hz.HZ_F64 else 3e-5), d


def test_graph_is_rebuilt_when_a_complex_source_arrives():
    """A cached CUDA graph holds the kernel arguments of its capture; hz_set_source with a first imaginary part
    allocates the Im b array, so the graph must be re-captured (it used to replay bbf_im = NULL and drop Im f)."""
    _require_cuda()
    inp = make_config(2, n=16)
    rng = np.random.default_rng(21)
    f_im = rng.standard_normal(inp.f_re.shape)
    ctx, info = hz.setup_from_inputs(inp, hz.HZ_F64, 1)
    try:
        a = torch.zeros(2 * inp.npx * inp.npy, dtype=torch.float64, device="cuda")
        b = torch.zeros_like(a)
        hz.hz_ddm_solve(ctx, 8, n_wh=2, reset_state=True, use_graph=True, u_out_ptr=a.data_ptr())     # graph cached
        hz.hz_set_source(ctx, inp.f_re, f_im)
        hz.hz_ddm_solve(ctx, 8, n_wh=2, reset_state=True, use_graph=True, u_out_ptr=a.data_ptr())
        hz.hz_ddm_solve(ctx, 8, n_wh=2, reset_state=True, use_graph=False, u_out_ptr=b.data_ptr())
        assert torch.equal(a, b)
        inp2 = HzInputs(**{**inp.__dict__, "f_im": f_im})
        st = O.ddm_solve(problem_from(inp2), inp.sx, inp.sy, 8, 2, True, 0.5, inp.cfl_frac)
        ug = a.cpu().numpy().reshape(2, inp.npy, inp.npx)
        assert rel(ug[0] + 1j * ug[1], O.ddm_gather(st)) <= 1e-10
    finally:
        hz.hz_destroy(ctx)


@pytest.mark.parametrize("prec", [hz.HZ_F64, hz.HZ_F32])
@pytest.mark.parametrize("p,nx,ny", [(1, 37, 9), (2, 33, 11), (3, 35, 10), (4, 34, 9),
                                     (1, 101, 27), (2, 99, 26), (3, 70, 20), (4, 100, 27), (3, 131, 35)])
def test_global_operator_kernel_matches_the_assembled_matrix(p, nx, ny, prec):
    """hz_operator_time's kernel (the paper's "operator" of PAPER.md:223; the residual kernel's other mode): y =
    (A - i w H - w^2 M) u on a random complex vector against the oracle's assembled sparse matrix.  The mesh spans
    several 32x8-element blocks of the kernel with ragged tails in both directions; the larger meshes have patches
    strictly inside the mesh, which run the interior kernels (cp.async staging; TMA bulk copies for fp64 at p >= 3), the
    smaller ones only the general kernel of the boundary ring.  The residual mode is checked against the same matrix."""
    _require_cuda()
    inp = hetero_inputs(nx, ny, p, 1, 1, seed=300 + p)
    pr = problem_from(inp)
    A, M, H, b = O.assemble_global(pr)
    Z = O.helmholtz_matrix(A, M, H, pr.omega)
    rng = np.random.default_rng(17)
    nn = inp.npx * inp.npy
    u = rng.standard_normal(nn) + 1j * rng.standard_normal(nn)
    y_o = Z @ u
    dt = torch.float64 if prec == hz.HZ_F64 else torch.float32
    ctx = hz.hz_mesh_setup(inp.nx, inp.ny, inp.x0, inp.y0, inp.x1, inp.y1, inp.p, inp.c_nodes, inp.omega, inp.f_re)
    try:
        ud = torch.from_numpy(np.concatenate([u.real, u.imag])).to(dt).cuda()
        yd = torch.zeros(2 * nn, dtype=dt, device="cuda")
        ms = hz.hz_operator_time(ctx, ud.data_ptr(), prec, 2, y_ptr=yd.data_ptr())
        assert ms > 0
        y = yd.double().cpu().numpy()
        assert rel(y[:nn] + 1j * y[nn:], y_o) <= (1e-13 if prec == hz.HZ_F64 else 2e-6)
        # residual mode of the same kernels: || b - Z u || / || b || with u in the precision `prec`
        ur = ud.double().cpu().numpy()
        want = np.linalg.norm(b - Z @ (ur[:nn] + 1j * ur[nn:])) / np.linalg.norm(b)
        got = hz.hz_residual(ctx, ud.data_ptr(), prec)
        assert abs(got - want) <= 1e-9 * want
    finally:
        hz.hz_destroy(ctx)
