/* hz3.h — C ABI of the 3-D hexahedral variant of the block-level DDM / WaveHoltz sweep (
 * PAPER.md:263-269, Section VII.B: "(P+1)^3 degrees of freedom per element ... small subdomains").
 *
 * Same method as include/hz.h on a uniform mesh of nx*ny*nz hexahedra of degree p on a box: spectral elements with
 * GLL quadrature, sx*sy*sz box subdomains with the impedance transmission condition on all six
 * faces, one thread block per subdomain and one thread per subdomain node or per column of nodes
 * (at most 1024 nodes per subdomain), WaveHoltz as the subdomain solver (Algorithm 1,
 * PAPER.md:160-183).
 *
 * Plain pointers, no torch types.  HOST = host memory read during the call; DEVICE = device memory owned by the caller.
 * Node (I,J,K) of the global mesh has the flat index (K*npy + J)*npx + I (npx = nx*p+1, ...).  Faces are ordered
 * W (I=0), E (I=max), S (J=0), N (J=max), B (K=0), T (K=max); a face array is indexed K*npy+J on W/E, K*npx+I on S/N,
 * J*npx+I on B/T (per subdomain: with the subdomain's own node counts).  Status codes and hz_prec are those of hz.h;
 * every call returns HZ_OK or an error whose message hz3_last_error gives.  Not thread-safe per context. */
#ifndef HZ3_H
#define HZ3_H

#include "hz.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hz3_ctx hz3_ctx;

/* The Helmholtz problem (eq. (1a,b)) on the box [box[0],box[3]] x [box[1],box[4]] x [box[2],box[5]].
 *   c_nodes, f_re, f_im   HOST, npx*npy*npz doubles: wave speed (> 0) and source at the nodes; f_im may be NULL.
 *   bc_lambda             HOST or NULL: boundary datum of eq. (1b) on the six outer faces, six consecutive blocks of
 *                         2*FB doubles (re[FB], im[FB]), FB = max(npy*npz, npx*npz, npx*npy), indexed as above.
 *   p                     1..4 (else HZ_EUNSUPPORTED). */
hz_status hz3_mesh_setup(hz3_ctx **out, int nx, int ny, int nz, const double *box, int p, const double *c_nodes,
                         double omega, const double *f_re, const double *f_im, const double *bc_lambda);

typedef struct {
  int n_t;               /* time steps per period (reading R9 with 1/hx^2 + 1/hy^2 + 1/hz^2) */
  int dofs_per_sub;      /* lnx*lny*lnz */
  int lnx, lny, lnz;     /* nodes per subdomain side */
  int face_stride;       /* F = max(lny*lnz, lnx*lnz, lnx*lny): stride of one face in lambda arrays */
  int threads_per_block; /* nodes (one-node-per-thread kernel) or (i,j) node columns (column kernel), rounded to a warp */
  int nodes_per_thread;  /* 1, or lnz: one thread per node column along z with its nodes in registers */
  int blocks;            /* sx*sy*sz */
  double dt, theta, sigma;
  size_t smem_bytes, workspace_bytes;
} hz3_part_info;

/* sx*sy*sz subdomains (must divide nx, ny, nz: HZ_EINVAL otherwise), one thread block each
 * (HZ_EUNSUPPORTED if a subdomain has more than 1024 nodes).  prec: arithmetic of the sweep.
 * nodes_per_thread: 0 = automatic (one thread per node column along z where that column length is compiled, else one
 * node per thread); 1 = one node per thread (PAPER.md:191-207 in three dimensions); other values HZ_EINVAL. */
hz_status hz3_partition(hz3_ctx *ctx, int sx, int sy, int sz, hz_prec prec, double cfl_frac, int nodes_per_thread,
                        hz3_part_info *info);

typedef struct {
  int n_outer;     /* sweeps (each followed by the exchange with relaxation) */
  int n_wh;        /* WaveHoltz iterations per sweep (the paper's benchmark uses 5) */
  int warm_start;  /* 0: u^(0) = 0 (Algorithm 1 as printed); 1: previous u_l (reading R11) */
  double relax;    /* rho in (0,1] (reading R12) */
  int reset_state; /* 1: lambda = 0, u_l = 0 first */
  double tol;      /* > 0 with check_every > 0: stop when the global relative residual (hz3_residual of the gathered
                      field, fp64) is <= tol; the check runs outside the sweep, every check_every sweeps */
  int check_every;
} hz3_solve_opts;

typedef struct {
  int n_outer_done, n_t;
  double rel_residual;                  /* last residual check, or -1 */
  double total_ms;                      /* CUDA-event time of the whole call */
  double sweep_ms_total, exch_ms_total; /* CUDA-event times of the sweep / exchange kernels */
  double dof_timesteps;                 /* sweeps * blocks * dofs_per_sub * n_wh * (n_t - 1) */
  int launches;
} hz3_solve_info;

/* n_outer x {sweep kernel (Algorithm 1 on every subdomain), exchange kernel (eq. (2) with relaxation)} on `stream`;
 * u_out: DEVICE or NULL, 2*npx*npy*npz values of the partition's precision (re then im): the gathered field (mean of
 * the copies at shared nodes, reading R19). */
hz_status hz3_ddm_solve(hz3_ctx *ctx, const hz3_solve_opts *opts, void *u_out, hz3_solve_info *info, void *stream);

/* || b - (A - i w H - w^2 M) u || / || b || of the unpartitioned system (eq. (4)) in fp64;
 * u_dev: DEVICE, 2*npx*npy*npz values of precision `prec`. */
hz_status hz3_residual(hz3_ctx *ctx, const void *u_dev, hz_prec prec, double *rel, void *stream);

/* The paper's "operator time" normaliser ("the time it takes to evaluate the Helmholtz operator
 * A - i w H - w^2 M on the entire domain"): `reps` back-to-back evaluations of the global operator (the kernel of
 * hz3_residual, fp64) on u_dev (DEVICE, 2*npx*npy*npz doubles); *ms_per_eval = CUDA-event time / reps. */
hz_status hz3_operator_time(hz3_ctx *ctx, const double *u_dev, int reps, double *ms_per_eval, void *stream);

/* Raw per-subdomain state in fp64 (parity tests): u_sub DEVICE [L][2][N] (N = dofs_per_sub, node (i,j,k) at
 * (k*lny+j)*lnx+i), lam DEVICE [L][6][2][F]; either may be NULL. */
hz_status hz3_get_subdomain_state(hz3_ctx *ctx, double *u_sub, double *lam);

const char *hz3_last_error(hz3_ctx *ctx);
void hz3_destroy(hz3_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif
