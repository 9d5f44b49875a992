"""ctypes binding of include/hz3.h (3-D hexahedral variant): argument marshalling only."""
from __future__ import annotations

import ctypes as C

import numpy as np

from .hz import HZ_F32, HZ_F64, HZ_OK, HzError, _host_ptr, lib

EXPORTS = ("hz3_mesh_setup", "hz3_partition", "hz3_ddm_solve", "hz3_residual", "hz3_operator_time", "hz3_get_subdomain_state",
           "hz3_last_error", "hz3_destroy")


class hz3_part_info(C.Structure):
    _fields_ = [("n_t", C.c_int), ("dofs_per_sub", C.c_int), ("lnx", C.c_int), ("lny", C.c_int), ("lnz", C.c_int),
                ("face_stride", C.c_int), ("threads_per_block", C.c_int), ("nodes_per_thread", C.c_int), ("blocks", C.c_int),
                ("dt", C.c_double), ("theta", C.c_double), ("sigma", C.c_double),
                ("smem_bytes", C.c_size_t), ("workspace_bytes", C.c_size_t)]


class hz3_solve_opts(C.Structure):
    _fields_ = [("n_outer", C.c_int), ("n_wh", C.c_int), ("warm_start", C.c_int), ("relax", C.c_double),
                ("reset_state", C.c_int), ("tol", C.c_double), ("check_every", C.c_int)]


class hz3_solve_info(C.Structure):
    _fields_ = [("n_outer_done", C.c_int), ("n_t", C.c_int), ("rel_residual", C.c_double), ("total_ms", C.c_double),
                ("sweep_ms_total", C.c_double),
                ("exch_ms_total", C.c_double), ("dof_timesteps", C.c_double), ("launches", C.c_int)]


_ready = False


def lib3():
    global _ready
    L = lib()
    if not _ready:
        vp, ip = C.c_void_p, C.c_int
        L.hz3_mesh_setup.argtypes = [C.POINTER(vp), ip, ip, ip, vp, ip, vp, C.c_double, vp, vp, vp]
        L.hz3_partition.argtypes = [vp, ip, ip, ip, ip, C.c_double, ip, C.POINTER(hz3_part_info)]
        L.hz3_ddm_solve.argtypes = [vp, C.POINTER(hz3_solve_opts), vp, C.POINTER(hz3_solve_info), vp]
        L.hz3_residual.argtypes = [vp, vp, ip, C.POINTER(C.c_double), vp]
        L.hz3_operator_time.argtypes = [vp, vp, ip, C.POINTER(C.c_double), vp]
        L.hz3_get_subdomain_state.argtypes = [vp, vp, vp]
        L.hz3_last_error.argtypes = [vp]
        L.hz3_last_error.restype = C.c_char_p
        L.hz3_destroy.argtypes = [vp]
        L.hz3_destroy.restype = None
        _ready = True
    return L


def _check(ctx, st):
    if st != HZ_OK:
        raise HzError(st, lib3().hz3_last_error(ctx).decode())


def hz3_mesh_setup(nx, ny, nz, box, p, c_nodes, omega, f_re, f_im=None, bc_lambda=None):
    L = lib3()
    ctx = C.c_void_p()
    bx, _b = _host_ptr(np.asarray(box, dtype=np.float64), 6)
    cp, _c = _host_ptr(c_nodes)
    fr, _fr = _host_ptr(f_re)
    fi, _fi = _host_ptr(f_im)
    bc, _bc = _host_ptr(bc_lambda)
    st = L.hz3_mesh_setup(C.byref(ctx), nx, ny, nz, bx, p, cp, omega, fr, fi, bc)
    if st != HZ_OK:
        raise HzError(st, L.hz3_last_error(None).decode())
    return ctx


def hz3_partition(ctx, sx, sy, sz, prec=HZ_F64, cfl_frac=0.5, nodes_per_thread=0):
    info = hz3_part_info()
    _check(ctx, lib3().hz3_partition(ctx, sx, sy, sz, prec, cfl_frac, int(nodes_per_thread), C.byref(info)))
    return info


def hz3_ddm_solve(ctx, n_outer, n_wh=5, warm_start=True, relax=0.5, reset_state=False, u_out_ptr=None, stream=None,
                  tol=0.0, check_every=0):
    opts = hz3_solve_opts(int(n_outer), int(n_wh), int(bool(warm_start)), float(relax), int(bool(reset_state)),
                          float(tol), int(check_every))
    info = hz3_solve_info()
    _check(ctx, lib3().hz3_ddm_solve(ctx, C.byref(opts), C.c_void_p(u_out_ptr) if u_out_ptr else None, C.byref(info),
                                     C.c_void_p(stream) if stream else None))
    return info


def hz3_residual(ctx, u_ptr, prec, stream=None):
    rel = C.c_double()
    _check(ctx, lib3().hz3_residual(ctx, C.c_void_p(u_ptr), prec, C.byref(rel), C.c_void_p(stream) if stream else None))
    return rel.value


def hz3_operator_time(ctx, u_ptr, reps=20, stream=None):
    """ms per evaluation of the global Helmholtz operator (fp64) on the device field at u_ptr."""
    ms = C.c_double()
    _check(ctx, lib3().hz3_operator_time(ctx, C.c_void_p(u_ptr), int(reps), C.byref(ms), C.c_void_p(stream) if stream else None))
    return ms.value


def hz3_get_subdomain_state(ctx, u_sub_ptr, lam_ptr):
    _check(ctx, lib3().hz3_get_subdomain_state(ctx, C.c_void_p(u_sub_ptr) if u_sub_ptr else None,
                                               C.c_void_p(lam_ptr) if lam_ptr else None))


def hz3_destroy(ctx):
    lib3().hz3_destroy(ctx)
