"""hz_residual_static (include/hz.h): the global residual of system (4) for callers that cannot
allocate -- block partial sums in a file-scope `static __device__` array, result left on the device -- against the
existing hz_residual, on two calls in a row that share the array.  Collected last (file name) so that a failure
here cannot hide another test under `pytest -x`; passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_2606_21695_b200 import hz  # noqa: E402
from paper_2606_21695_b200.inputs import make_config  # noqa: E402

TOL64 = 1e-12   # fp64 bar of the parity tests (tests/test_gpu_parity.py); the two paths are in fact bit-identical


def mesh_ctx(inp):
    return hz.hz_mesh_setup(inp.nx, inp.ny, inp.x0, inp.y0, inp.x1, inp.y1, inp.p, inp.c_nodes, inp.omega, inp.f_re)


def random_field(inp, seed, dtype, scale):
    g = torch.Generator(device="cpu").manual_seed(seed)
    return (scale * torch.randn(2 * inp.npx * inp.npy, generator=g, dtype=torch.float64)).to(dtype).cuda()


@pytest.mark.parametrize("cfg,n,p", [(2, 40, 3), (5, 96, 1), (3, 48, 4)])
def test_two_calls_in_a_row_match_hz_residual(cfg, n, p):
    assert torch.cuda.is_available(), "CUDA device required"
    inp = make_config(cfg, n=n, p=p)
    ctx = mesh_ctx(inp)
    try:
        hz.hz_residual_static_setup(ctx)
        out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
        # second field 1000x smaller and in the other precision: partial sums left over from the first call would show
        fields = [(random_field(inp, 1, torch.float64, 1.0), hz.HZ_F64), (random_field(inp, 2, torch.float32, 1e-3), hz.HZ_F32)]
        want = [hz.hz_residual(ctx, u.data_ptr(), prec) for u, prec in fields]
        assert abs(want[0] - want[1]) > 0.1 * want[0]
        hz.hz_residual_static(ctx, fields[1][0].data_ptr(), fields[1][1], out.data_ptr())   # loads the kernels (lazy loading)
        torch.cuda.synchronize()
        out.fill_(float("nan"))
        free_before = torch.cuda.mem_get_info()[0]
        for k, (u, prec) in enumerate(fields):
            hz.hz_residual_static(ctx, u.data_ptr(), prec, out[k:].data_ptr())
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before            # nothing was allocated on the device
        got = out.cpu().numpy()
        for k in range(2):
            assert abs(got[k] - want[k]) <= TOL64 * want[k], (k, got[k], want[k])
        # the same pair again, in the opposite order and on a side stream
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            for k in (1, 0):
                u, prec = fields[k]
                hz.hz_residual_static(ctx, u.data_ptr(), prec, out[k:].data_ptr(), stream=s.cuda_stream)
        s.synchronize()
        assert np.array_equal(out.cpu().numpy(), got)
    finally:
        hz.hz_destroy(ctx)


def test_general_quads_and_a_second_context_share_the_array():
    a = make_config(2, n=24, distort=0.2)
    b = make_config(1)
    ca = hz.hz_mesh_setup_quads(a.nx, a.ny, a.p, a.vx, a.vy, a.c_nodes, a.omega, a.f_re)
    cb = mesh_ctx(b)
    try:
        out = torch.zeros(2, dtype=torch.float64, device="cuda")
        ua, ub = random_field(a, 3, torch.float64, 1.0), random_field(b, 4, torch.float64, 1.0)
        hz.hz_residual_static(ca, ua.data_ptr(), hz.HZ_F64, out[0:].data_ptr())     # first use resolves the address itself
        hz.hz_residual_static(cb, ub.data_ptr(), hz.HZ_F64, out[1:].data_ptr())
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        want = [hz.hz_residual(ca, ua.data_ptr(), hz.HZ_F64), hz.hz_residual(cb, ub.data_ptr(), hz.HZ_F64)]
        for k in range(2):
            assert abs(got[k] - want[k]) <= TOL64 * want[k], (k, got[k], want[k])
    finally:
        hz.hz_destroy(ca)
        hz.hz_destroy(cb)


def test_sizes_beyond_the_static_maximum_and_bad_arguments_are_rejected():
    cap = hz.lib().hz_residual_static_max_blocks()
    assert cap == 262144
    # the smallest mesh beyond the maximum that the launch grid allows: a thin p = 1 mesh with 5 patch columns
    # (129 nodes) and 52429 patch rows, ceil((nx+1)/32) * ceil((ny+1)/8) = 262145 blocks (54 M nodes)
    nx, ny = 128, 8 * 52429 - 1
    npx, npy = nx + 1, ny + 1
    c = np.ones((npy, npx))
    f = np.zeros((npy, npx))
    f[npy // 2, npx // 2] = 1.0
    ctx = hz.hz_mesh_setup(nx, ny, 0.0, 0.0, 1.0, float(ny) / nx, 1, c, 2.0, f)
    try:
        u = torch.zeros(2 * npx * npy, dtype=torch.float32, device="cuda")
        out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
        with pytest.raises(hz.HzError) as e:
            hz.hz_residual_static(ctx, u.data_ptr(), hz.HZ_F32, out.data_ptr())
        assert e.value.status == hz.HZ_EINVAL and "262145" in str(e.value) and "262144" in str(e.value)
        torch.cuda.synchronize()
        assert out.item() == -1.0                                     # nothing was enqueued
        assert hz.hz_residual(ctx, u.data_ptr(), hz.HZ_F32) == 1.0    # the allocating path takes the mesh (u = 0: r = b)
        with pytest.raises(hz.HzError):
            hz.hz_residual_static(ctx, 0, hz.HZ_F32, out.data_ptr())
        with pytest.raises(hz.HzError):
            hz.hz_residual_static(ctx, u.data_ptr(), 7, out.data_ptr())
    finally:
        hz.hz_destroy(ctx)
