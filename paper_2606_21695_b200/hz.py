"""Thin ctypes binding over the C-ABI library of include/hz.h (same names, argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libhz.so; nothing here computes.  PyTorch
is used by callers for device memory and streams only: device arrays are passed as `tensor.data_ptr()`
integers, streams as `torch.cuda.current_stream().cuda_stream`.  There is no CPU fallback: if the
library is not built, loading it raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhz.so")

HZ_OK, HZ_EINVAL, HZ_ENOMEM, HZ_ECUDA, HZ_EUNSUPPORTED, HZ_ESTATE = range(6)
HZ_F32, HZ_F64 = 0, 1
HZ_TC_IMPEDANCE0 = 0
STATUS_NAMES = {0: "HZ_OK", 1: "HZ_EINVAL", 2: "HZ_ENOMEM", 3: "HZ_ECUDA", 4: "HZ_EUNSUPPORTED", 5: "HZ_ESTATE"}

# every symbol include/hz.h declares
EXPORTS = ("hz_mesh_setup", "hz_mesh_setup_quads", "hz_set_source", "hz_partition", "hz_partition_ex", "hz_ddm_solve",
           "hz_operator_time", "hz_ddm_solve_sources", "hz_ddm_solve_gmres", "hz_ddm_solve_mixed", "hz_minres_cycle",
           "hz_residual", "hz_residual_static_max_blocks", "hz_residual_static_setup", "hz_residual_static",
           "hz_get_subdomain_state", "hz_set_subdomain_state", "hz_last_error", "hz_destroy")


class hz_part_info(C.Structure):
    _fields_ = [("n_t", C.c_int), ("dofs_per_sub", C.c_int), ("edge_nodes_x", C.c_int), ("edge_nodes_y", C.c_int),
                ("edge_stride", C.c_int), ("threads_per_block", C.c_int), ("blocks", C.c_int),
                ("dofs_per_thread", C.c_int), ("tile_mx", C.c_int), ("tile_my", C.c_int), ("cluster_size", C.c_int),
                ("subs_per_block", C.c_int), ("dt", C.c_double), ("theta", C.c_double), ("sigma", C.c_double),
                ("smem_bytes", C.c_size_t), ("workspace_bytes", C.c_size_t), ("kernel", C.c_char * 24)]


class hz_part_flags(C.Structure):
    _fields_ = [("cluster", C.c_int), ("no_warp_spec", C.c_int), ("no_reg_cap", C.c_int), ("grid_blocks", C.c_int),
                ("warp_order", C.c_int), ("pack", C.c_int)]


class hz_mixed_opts(C.Structure):
    _fields_ = [("n_cycles_max", C.c_int), ("m_inner", C.c_int), ("n_wh", C.c_int), ("relax", C.c_double),
                ("tol", C.c_double), ("check_every", C.c_int), ("reset_state", C.c_int)]


class hz_mixed_info(C.Structure):
    _fields_ = [("cycles_done", C.c_int), ("sweeps_lo", C.c_int), ("sweeps_hi", C.c_int), ("rel_residual", C.c_double),
                ("total_ms", C.c_double), ("dof_timesteps", C.c_double)]


class hz_solve_opts(C.Structure):
    _fields_ = [("n_outer_max", C.c_int), ("n_wh", C.c_int), ("warm_start", C.c_int), ("relax", C.c_double),
                ("tol", C.c_double), ("check_every", C.c_int), ("reset_state", C.c_int), ("use_graph", C.c_int)]


class hz_sources_info(C.Structure):
    _fields_ = [("sources_done", C.c_int), ("total_ms", C.c_double), ("dof_timesteps", C.c_double),
                ("launches", C.c_int), ("h2d_bytes", C.c_double), ("d2h_bytes", C.c_double)]


class hz_solve_info(C.Structure):
    _fields_ = [("n_outer_done", C.c_int), ("n_t", C.c_int), ("rel_residual", C.c_double),
                ("sweep_ms_total", C.c_double), ("exch_ms_total", C.c_double), ("total_ms", C.c_double),
                ("dof_timesteps", C.c_double), ("sweep_launches", C.c_int), ("exch_launches", C.c_int),
                ("other_launches", C.c_int)]


class hz_gmres_opts(C.Structure):
    _fields_ = [("n_wh", C.c_int), ("relax", C.c_double), ("restart", C.c_int), ("max_steps", C.c_int),
                ("lin_tol", C.c_double), ("tol", C.c_double), ("reset_state", C.c_int),
                ("lin_history", C.POINTER(C.c_double)), ("history_len", C.c_int), ("lambda_only", C.c_int),
                ("n_polish", C.c_int)]


class hz_gmres_info(C.Structure):
    _fields_ = [("steps_done", C.c_int), ("sweeps_done", C.c_int), ("cycles", C.c_int), ("lin_residual", C.c_double),
                ("rel_residual", C.c_double), ("total_ms", C.c_double), ("krylov_bytes", C.c_size_t)]


class hz_minres_opts(C.Structure):
    _fields_ = [("tol", C.c_double), ("max_iters", C.c_int), ("warm_start", C.c_int), ("relax", C.c_double)]


class hz_minres_info(C.Structure):
    _fields_ = [("iters_max", C.c_int), ("iters_mean", C.c_double), ("res_max", C.c_double), ("kernel_ms", C.c_double)]


class HzError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


_lib = None


def lib():
    """Loads libhz.so (built by `python -m paper_2606_21695_b200.build`).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is not built (run `python -m paper_2606_21695_b200.build`); "
                           "there is no CPU fallback")
    L = C.CDLL(LIB_PATH)
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.c_int
    L.hz_mesh_setup.argtypes = [C.POINTER(vp), ip, ip, C.c_double, C.c_double, C.c_double, C.c_double, ip,
                                vp, C.c_double, vp, vp, vp]
    L.hz_mesh_setup_quads.argtypes = [C.POINTER(vp), ip, ip, ip, vp, vp, vp, C.c_double, vp, vp, vp]
    L.hz_set_source.argtypes = [vp, vp, vp]
    L.hz_partition.argtypes = [vp, ip, ip, ip, ip, ip, C.c_double, C.POINTER(hz_part_info)]
    L.hz_partition_ex.argtypes = [vp, ip, ip, ip, ip, ip, C.c_double, C.POINTER(hz_part_flags), C.POINTER(hz_part_info)]
    L.hz_ddm_solve_mixed.argtypes = [vp, vp, C.POINTER(hz_mixed_opts), vp, C.POINTER(hz_mixed_info), vp]
    L.hz_ddm_solve.argtypes = [vp, C.POINTER(hz_solve_opts), vp, C.POINTER(hz_solve_info), vp]
    L.hz_operator_time.argtypes = [vp, vp, ip, ip, vp, C.POINTER(C.c_double), vp]
    L.hz_ddm_solve_sources.argtypes = [vp, C.POINTER(hz_solve_opts), ip, C.POINTER(vp), C.POINTER(vp),
                                       C.POINTER(hz_sources_info), vp]
    L.hz_ddm_solve_gmres.argtypes = [vp, C.POINTER(hz_gmres_opts), vp, C.POINTER(hz_gmres_info), vp]
    L.hz_minres_cycle.argtypes = [vp, C.POINTER(hz_minres_opts), vp, vp, C.POINTER(hz_minres_info), vp]
    L.hz_residual.argtypes = [vp, vp, ip, dp, vp]
    L.hz_residual_static_max_blocks.argtypes = []
    L.hz_residual_static_max_blocks.restype = C.c_int
    L.hz_residual_static_setup.argtypes = [vp]
    L.hz_residual_static.argtypes = [vp, vp, ip, vp, vp]
    L.hz_get_subdomain_state.argtypes = [vp, vp, vp, vp]
    L.hz_set_subdomain_state.argtypes = [vp, vp, vp, vp]
    L.hz_last_error.argtypes = [vp]
    L.hz_last_error.restype = C.c_char_p
    L.hz_destroy.argtypes = [vp]
    L.hz_destroy.restype = None
    for name in EXPORTS:
        if name not in ("hz_last_error", "hz_destroy"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _host_ptr(a, n=None):
    """Pointer to a C-contiguous float64 host array (or None)."""
    if a is None:
        return None, None
    arr = np.ascontiguousarray(a, dtype=np.float64)
    if n is not None and arr.size != n:
        raise ValueError(f"expected {n} values, got {arr.size}")
    return arr.ctypes.data_as(C.c_void_p), arr


def _check(ctx, st):
    if st != HZ_OK:
        raise HzError(st, lib().hz_last_error(ctx).decode())


def hz_mesh_setup(nx, ny, x0, y0, x1, y1, p, c_nodes, omega, f_re, f_im=None, bc_lambda=None):
    """-> context handle (c_void_p).  Host numpy arrays; see include/hz.h."""
    L = lib()
    ctx = C.c_void_p()
    cp, _c = _host_ptr(c_nodes)
    fr, _fr = _host_ptr(f_re)
    fi, _fi = _host_ptr(f_im)
    bc, _bc = _host_ptr(bc_lambda)
    st = L.hz_mesh_setup(C.byref(ctx), nx, ny, x0, y0, x1, y1, p, cp, omega, fr, fi, bc)
    if st != HZ_OK:
        raise HzError(st, L.hz_last_error(None).decode())
    return ctx


def hz_mesh_setup_quads(nx, ny, p, vx, vy, c_nodes, omega, f_re, f_im=None, bc_lambda=None):
    """General straight-sided convex quads: vx, vy are (ny+1, nx+1) vertex arrays.  -> context handle."""
    L = lib()
    ctx = C.c_void_p()
    xp, _x = _host_ptr(vx)
    yp, _y = _host_ptr(vy)
    cp, _c = _host_ptr(c_nodes)
    fr, _fr = _host_ptr(f_re)
    fi, _fi = _host_ptr(f_im)
    bc, _bc = _host_ptr(bc_lambda)
    st = L.hz_mesh_setup_quads(C.byref(ctx), nx, ny, p, xp, yp, cp, omega, fr, fi, bc)
    if st != HZ_OK:
        raise HzError(st, L.hz_last_error(None).decode())
    return ctx


def hz_set_source(ctx, f_re, f_im=None):
    fr, _fr = _host_ptr(f_re)
    fi, _fi = _host_ptr(f_im)
    _check(ctx, lib().hz_set_source(ctx, fr, fi))


def hz_set_source_ptr(ctx, f_re_ptr, f_im_ptr=None):
    """Same as hz_set_source with raw HOST pointers (e.g. pinned torch tensors' data_ptr())."""
    _check(ctx, lib().hz_set_source(ctx, C.c_void_p(f_re_ptr), C.c_void_p(f_im_ptr) if f_im_ptr else None))


def hz_partition(ctx, sx, sy, tc=HZ_TC_IMPEDANCE0, prec=HZ_F64, dofs_per_thread=0, cfl_frac=0.5):
    info = hz_part_info()
    _check(ctx, lib().hz_partition(ctx, sx, sy, tc, prec, dofs_per_thread, cfl_frac, C.byref(info)))
    return info


def hz_partition_ex(ctx, sx, sy, tc=HZ_TC_IMPEDANCE0, prec=HZ_F64, dofs_per_thread=0, cfl_frac=0.5, cluster=0,
                    no_warp_spec=False, no_reg_cap=False, grid_blocks=0, warp_order=0, pack=0):
    """hz_partition with the explicit variant-choice controls of include/hz.h::hz_part_flags."""
    info = hz_part_info()
    fl = hz_part_flags(int(cluster), int(bool(no_warp_spec)), int(bool(no_reg_cap)), int(grid_blocks), int(warp_order),
                       int(pack))
    _check(ctx, lib().hz_partition_ex(ctx, sx, sy, tc, prec, dofs_per_thread, cfl_frac, C.byref(fl), C.byref(info)))
    return info


def hz_ddm_solve_mixed(lo, hi, n_cycles_max, m_inner, n_wh=2, relax=0.5, tol=0.0, check_every=0, reset_state=False,
                       u_out_ptr=None, stream=None):
    """fp32 sweeps on the correction, fp64 state on `hi` (include/hz.h).  -> hz_mixed_info"""
    opts = hz_mixed_opts(int(n_cycles_max), int(m_inner), int(n_wh), float(relax), float(tol), int(check_every),
                         int(bool(reset_state)))
    info = hz_mixed_info()
    _check(hi, lib().hz_ddm_solve_mixed(lo, hi, C.byref(opts), C.c_void_p(u_out_ptr) if u_out_ptr else None,
                                        C.byref(info), C.c_void_p(stream) if stream else None))
    return info


def hz_ddm_solve(ctx, n_outer_max, n_wh=5, warm_start=True, relax=0.5, tol=0.0, check_every=0, reset_state=False,
                 use_graph=False, u_out_ptr=None, stream=None):
    opts = hz_solve_opts(int(n_outer_max), int(n_wh), int(bool(warm_start)), float(relax), float(tol),
                         int(check_every), int(bool(reset_state)), int(bool(use_graph)))
    info = hz_solve_info()
    _check(ctx, lib().hz_ddm_solve(ctx, C.byref(opts), C.c_void_p(u_out_ptr) if u_out_ptr else None, C.byref(info),
                                   C.c_void_p(stream) if stream else None))
    return info


def hz_operator_time(ctx, u_ptr, prec=HZ_F64, reps=20, stream=None, y_ptr=None):
    """ms per evaluation y = (A - i w H - w^2 M) u of the global Helmholtz operator in precision `prec` on the device
    field at u_ptr (the paper's normaliser); y goes to y_ptr if given."""
    ms = C.c_double()
    _check(ctx, lib().hz_operator_time(ctx, C.c_void_p(u_ptr), int(prec), int(reps), C.c_void_p(y_ptr) if y_ptr else None,
                                       C.byref(ms), C.c_void_p(stream) if stream else None))
    return ms.value


def hz_ddm_solve_sources(ctx, f_host_ptrs, u_host_ptrs, n_outer=1, n_wh=5, warm_start=True, relax=0.5,
                         reset_state=False, stream=None):
    """A stream of sources, host to host, copies overlapped with the sweeps (include/hz.h).  f_host_ptrs /
    u_host_ptrs: raw HOST pointers (e.g. pinned torch tensors' data_ptr()).  -> hz_sources_info"""
    n = len(f_host_ptrs)
    assert n == len(u_host_ptrs) and n >= 1
    fa = (C.c_void_p * n)(*[C.c_void_p(int(q)) for q in f_host_ptrs])
    ua = (C.c_void_p * n)(*[C.c_void_p(int(q)) for q in u_host_ptrs])
    opts = hz_solve_opts(int(n_outer), int(n_wh), int(bool(warm_start)), float(relax), 0.0, 0, int(bool(reset_state)), 0)
    info = hz_sources_info()
    _check(ctx, lib().hz_ddm_solve_sources(ctx, C.byref(opts), n, fa, ua, C.byref(info),
                                           C.c_void_p(stream) if stream else None))
    return info


def hz_ddm_solve_gmres(ctx, max_steps, n_wh=2, relax=0.5, restart=50, lin_tol=0.0, tol=0.0, reset_state=True,
                       u_out_ptr=None, stream=None, want_history=False, lambda_only=False, n_polish=0):
    """-> hz_gmres_info (and the per-step relative linear residuals if want_history)."""
    hist = (C.c_double * max(1, int(max_steps)))() if want_history else None
    opts = hz_gmres_opts(int(n_wh), float(relax), int(restart), int(max_steps), float(lin_tol), float(tol),
                         int(bool(reset_state)), hist if want_history else None, int(max_steps) if want_history else 0,
                         int(bool(lambda_only)), int(n_polish))
    info = hz_gmres_info()
    _check(ctx, lib().hz_ddm_solve_gmres(ctx, C.byref(opts), C.c_void_p(u_out_ptr) if u_out_ptr else None,
                                         C.byref(info), C.c_void_p(stream) if stream else None))
    if want_history:
        return info, [hist[i] for i in range(info.steps_done)]
    return info


def hz_minres_cycle(ctx, blocks, tol, max_iters, warm_start=False, relax=0.0, stream=None):
    """-> (hz_minres_info, iterations per subdomain, true relative residual per subdomain)"""
    opts = hz_minres_opts(float(tol), int(max_iters), int(bool(warm_start)), float(relax))
    info = hz_minres_info()
    iters = np.zeros(blocks, dtype=np.int32)
    res = np.zeros(blocks, dtype=np.float64)
    _check(ctx, lib().hz_minres_cycle(ctx, C.byref(opts), iters.ctypes.data_as(C.c_void_p), res.ctypes.data_as(C.c_void_p),
                                      C.byref(info), C.c_void_p(stream) if stream else None))
    return info, iters, res


def hz_residual(ctx, u_ptr, u_prec, stream=None):
    r = C.c_double()
    _check(ctx, lib().hz_residual(ctx, C.c_void_p(u_ptr), u_prec, C.byref(r), C.c_void_p(stream) if stream else None))
    return r.value


def hz_residual_static_setup(ctx):
    _check(ctx, lib().hz_residual_static_setup(ctx))


def hz_residual_static(ctx, u_ptr, u_prec, rel_ptr, stream=None):
    """No allocation, no host copy, no synchronisation: the relative residual lands in the device double at rel_ptr."""
    _check(ctx, lib().hz_residual_static(ctx, C.c_void_p(u_ptr), u_prec, C.c_void_p(rel_ptr),
                                         C.c_void_p(stream) if stream else None))


def hz_get_subdomain_state(ctx, u_sub_ptr=None, lambda_ptr=None, stream=None):
    _check(ctx, lib().hz_get_subdomain_state(ctx, C.c_void_p(u_sub_ptr) if u_sub_ptr else None,
                                             C.c_void_p(lambda_ptr) if lambda_ptr else None,
                                             C.c_void_p(stream) if stream else None))


def hz_set_subdomain_state(ctx, u_sub_ptr=None, lambda_ptr=None, stream=None):
    _check(ctx, lib().hz_set_subdomain_state(ctx, C.c_void_p(u_sub_ptr) if u_sub_ptr else None,
                                             C.c_void_p(lambda_ptr) if lambda_ptr else None,
                                             C.c_void_p(stream) if stream else None))


def hz_last_error(ctx):
    return lib().hz_last_error(ctx).decode()


def hz_destroy(ctx):
    if ctx:
        lib().hz_destroy(ctx)


def setup_from_inputs(inp, prec=HZ_F64, dofs_per_thread=0, **flags):
    """Convenience: hz_mesh_setup + hz_partition(_ex) from an inputs.HzInputs.  -> (ctx, part_info)."""
    if getattr(inp, "vx", None) is not None:
        ctx = hz_mesh_setup_quads(inp.nx, inp.ny, inp.p, inp.vx, inp.vy, inp.c_nodes, inp.omega, inp.f_re, inp.f_im)
    else:
        ctx = hz_mesh_setup(inp.nx, inp.ny, inp.x0, inp.y0, inp.x1, inp.y1, inp.p, inp.c_nodes, inp.omega, inp.f_re,
                            inp.f_im)
    try:
        info = hz_partition_ex(ctx, inp.sx, inp.sy, HZ_TC_IMPEDANCE0, prec, dofs_per_thread, inp.cfl_frac, **flags)
    except Exception:
        hz_destroy(ctx)
        raise
    return ctx, info
