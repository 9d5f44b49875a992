/* hz.h — C ABI of the B200-native block-level DDM / WaveHoltz Helmholtz sweep.
 *
 * Implements the hot path of arxiv/paper_2606_21695 ("Efficient Domain Decomposition for the
 * Helmholtz Equation on GPUs").  Citations are PAPER.md:<line> (section / equation / algorithm);
 * "reading Rn" refers to the list of readings in DESIGN.md.
 *
 * Every entry point returns an hz_status and never throws or aborts across the ABI.  Output
 * parameters are left untouched on error.  A NULL required pointer gives HZ_EINVAL.  CUDA runtime
 * failures give HZ_ECUDA with the runtime's message in hz_last_error().  There is no CPU fallback:
 * without a CUDA device every compute call fails with HZ_ECUDA.
 *
 * Pointer kinds are stated per argument: HOST (plain host memory, copied during the call, the caller
 * keeps ownership) or DEVICE (device memory owned by the caller, e.g. a torch tensor; must stay
 * valid until the stream work that uses it has finished).  Everything the library allocates on
 * the device is owned by the context and released by hz_destroy().
 *
 * Node numbering (all arrays): nx*ny rectangular elements of degree p on [x0,x1]x[y0,y1];
 * global node (I,J), I in 0..nx*p, J in 0..ny*p, flat index J*(nx*p+1)+I (x fastest); nodes sit at
 * the Gauss-Lobatto-Legendre points of each element.
 * Sides: 0=W (I=0), 1=E (I=max), 2=S (J=0), 3=N (J=max); an edge array runs along increasing J (W,E)
 * or increasing I (S,N) and includes both end nodes.
 */
#ifndef HZ_H
#define HZ_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hz_ctx hz_ctx; /* opaque; owns every device buffer it creates */

typedef enum {
  HZ_OK = 0,
  HZ_EINVAL = 1,       /* bad argument (NULL, non-positive size, partition does not divide the mesh) */
  HZ_ENOMEM = 2,       /* host or device allocation failed */
  HZ_ECUDA = 3,        /* CUDA runtime error; see hz_last_error */
  HZ_EUNSUPPORTED = 4, /* degree, subdomain size or variant has no compiled kernel */
  HZ_ESTATE = 5        /* call order violated (e.g. hz_ddm_solve before hz_partition) */
} hz_status;

typedef enum { HZ_F32 = 0, HZ_F64 = 1 } hz_prec;

/* Transmission operator on interfaces.  B = d/dn - i k is the only one in the paper
 * (Section III). */
typedef enum { HZ_TC_IMPEDANCE0 = 0 } hz_transmission;

/* ---------------------------------------------------------------------------------------------
 * hz_mesh_setup — the Helmholtz problem (eq. (1a,b)) on a uniform quad mesh with
 * the spectral-element discretisation of PAPER.md:94-117 (Section IV, eq. (3)-(4)).
 *
 *   out        receives a new context.
 *   nx, ny     elements per direction (>= 1);  [x0,x1]x[y0,y1] the domain (x1>x0, y1>y0).
 *   p          polynomial degree, 1..4 (else HZ_EUNSUPPORTED).
 *   c_nodes    HOST, (nx*p+1)*(ny*p+1) doubles: wave speed c(x_j) > 0 AT the global nodes (reading R14).
 *   omega      angular frequency > 0;  k_j = omega / c_j.
 *   f_re,f_im  HOST, same shape: source f(x_j) at the nodes.  f_im may be NULL (= 0).
 *   bc_lambda  HOST or NULL (= 0): boundary datum lambda of eq. (1b) on the outer boundary, as
 *              4 consecutive side blocks W,E,S,N, each 2*EB doubles (re[EB] then im[EB]) with
 *              EB = max(nx*p+1, ny*p+1); side arrays are indexed by J (W,E) or I (S,N).
 * ------------------------------------------------------------------------------------------- */
hz_status hz_mesh_setup(hz_ctx **out, int nx, int ny, double x0, double y0, double x1, double y1, int p,
                        const double *c_nodes, double omega, const double *f_re, const double *f_im,
                        const double *bc_lambda);

/* ---------------------------------------------------------------------------------------------
 * hz_mesh_setup_quads — the same problem on a logically rectangular mesh of GENERAL straight-sided convex
 * quadrilaterals ("quadrilateral ... elements"; gradient through D, geometric
 * factors at the quadrature points, D^T).  Element (gx,gy) is the bilinear image of
 * the reference square with the vertices (vx,vy)[gy..gy+1][gx..gx+1].
 *
 *   vx, vy     HOST, (ny+1)*(nx+1) doubles each, row-major (x index fastest): vertex coordinates.  Every element
 *              must be convex and counter-clockwise (detJ > 0 at all its GLL points), else HZ_EINVAL.
 *   c_nodes, f_re, f_im, bc_lambda, omega, p   as in hz_mesh_setup, sampled at the MAPPED GLL nodes.
 * hz_partition on such a context has one kernel variant (one thread per element, the element's (p+1)^2 nodes in
 * registers; pass dofs_per_thread = 0; at most 1024 elements per subdomain) and takes N_t from the element-wise
 * bound of reading R24; hz_minres_cycle returns HZ_EUNSUPPORTED.  Everything else (hz_ddm_solve,
 * hz_ddm_solve_gmres, hz_residual, state get/set) works as on a uniform mesh.
 * ------------------------------------------------------------------------------------------- */
hz_status hz_mesh_setup_quads(hz_ctx **out, int nx, int ny, int p, const double *vx, const double *vy,
                              const double *c_nodes, double omega, const double *f_re, const double *f_im,
                              const double *bc_lambda);

/* Replace the source f (HOST arrays as in hz_mesh_setup; f_im may be NULL).  After hz_partition
 * the per-subdomain load vectors are rebuilt on the device ("Assemble b from f"). */
hz_status hz_set_source(hz_ctx *ctx, const double *f_re, const double *f_im);

/* What hz_partition chose; all values are also what the oracle must reproduce independently. */
typedef struct {
  int n_t;               /* time steps per period T = 2 pi / omega (reading R9) */
  int dofs_per_sub;      /* (ex*p+1)*(ey*p+1) */
  int edge_nodes_x;      /* ex*p+1: nodes on a S/N side */
  int edge_nodes_y;      /* ey*p+1: nodes on a W/E side */
  int edge_stride;       /* E = max of the two: stride of one side in lambda arrays */
  int threads_per_block; /* block size of the sweep kernel */
  int blocks;            /* = sx*sy subdomains */
  int dofs_per_thread;   /* 1, or (mx*p)*(my*p) of the register-blocked variant, or -1 (streamed); general quads:
                            (p+1)^2 = the nodes of one element, shared ones replicated */
  int tile_mx, tile_my;  /* elements per thread tile (0 for the one-DOF-per-thread variant) */
  int cluster_size;      /* thread blocks (CTAs of one cluster, on as many SMs) per subdomain; 1 unless the state of
                            a subdomain needs the registers of several SMs (hz_sweep_cl.cuh) */
  int subs_per_block;    /* subdomains per thread block; 1 except for the packed small-subdomain kernel */
  double dt, theta, sigma; /* dt = T/n_t; theta = tan(w dt/2)/w; sigma = 2 sin(w dt/2)/w */
  size_t smem_bytes;       /* dynamic shared memory per block */
  size_t workspace_bytes;  /* device bytes the context allocated for this partition */
  char kernel[24];         /* name of the sweep kernel the partition launches, e.g. "k_sweep_ws" (NUL-terminated) */
} hz_part_info;

/* ---------------------------------------------------------------------------------------------
 * hz_partition — non-overlapping decomposition into sx*sy rectangular subdomains of
 * (nx/sx)*(ny/sy) elements, one thread block per subdomain, and the
 * per-subdomain operator data of the modified leapfrog (alpha_j, beta_j).
 *
 *   sx, sy           subdomain grid; must divide nx, ny on a uniform-mesh context (else HZ_EINVAL; reading R23).
 *                    On a hz_mesh_setup_quads context any 1 <= sx <= nx, 1 <= sy <= ny is accepted (ragged
 *                    partitions, reading R25; "at most K elements"): the first nx mod sx subdomain
 *                    columns have floor(nx/sx)+1 elements, the others floor(nx/sx); same in y.  All per-subdomain
 *                    arrays (and hz_part_info) are then sized for the largest subdomain, the padding is zero, and
 *                    the excess threads of a smaller subdomain's block idle (PAPER.md fn. at 203).
 *   tc               transmission condition (only HZ_TC_IMPEDANCE0).
 *   prec             arithmetic of the sweep (fp32 or fp64 build of the subdomain solve).
 *   dofs_per_thread  1 = one DOF per thread (needs dofs_per_sub <= 1024);
 *                    k > 1 = register-blocked variant with k = (mx*p)*(my*p) DOFs per thread
 *                    (PAPER.md:209-217), HZ_EUNSUPPORTED if no tile of that size is compiled or fits;
 *                    0 = choose automatically (falls back to the streamed variant when the subdomain's
 *                    state does not fit one SM's registers + shared memory);
 *                    -1 = streamed variant: state in an L2-resident global scratch (PAPER.md:209-217's
 *                    pGlobal idea), any subdomain size, slow.
 *   cfl_frac         fraction of the stable leapfrog step, in (0,1] (0.5 in all configs).
 *   info_out         may be NULL.
 * Re-partitioning an existing context is allowed; it discards lambda and the subdomain states.
 * ------------------------------------------------------------------------------------------- */
hz_status hz_partition(hz_ctx *ctx, int sx, int sy, hz_transmission tc, hz_prec prec, int dofs_per_thread,
                       double cfl_frac, hz_part_info *info_out);

/* hz_partition with explicit control of the variant choice (the (P, B, T) sweep of block layouts).
 * All fields zero (or flags == NULL) is hz_partition.  Used to time and to parity-test one particular launch shape,
 * e.g. the launch shape of a full-size config on a reduced mesh. */
typedef struct {
  int cluster;       /* 0: automatic; -1: never a thread-block-cluster kernel (streamed fallback instead);
                        c > 1: only cluster kernels with exactly c CTAs per subdomain compete */
  int no_warp_spec;  /* 1: never the warp-specialised kernel (the uniform register-blocked kernel instead) */
  int no_reg_cap;    /* 1: never a register-capped (higher-occupancy) instantiation */
  int grid_blocks;   /* > 0: choose the variant as if the partition had this many subdomains (the register-capped
                        instantiations are only picked when the grid fills the GPU) */
  int warp_order;    /* 0: automatic; 1, 2, 3: warp-role order 0, 1, 2 of the warp-specialised kernel */
  int pack;          /* 0: automatic; g >= 1: g subdomains per thread block (small-subdomain kernel), HZ_EUNSUPPORTED
                        if no such instantiation fits */
} hz_part_flags;
hz_status hz_partition_ex(hz_ctx *ctx, int sx, int sy, hz_transmission tc, hz_prec prec, int dofs_per_thread,
                          double cfl_frac, const hz_part_flags *flags, hz_part_info *info_out);

typedef struct {
  int n_outer_max;  /* sweeps to run (>= 0) */
  int n_wh;         /* WaveHoltz iterations per sweep (>= 1; reading R10; the paper times 5) */
  int warm_start;   /* 0: u^(0) = 0 every sweep (Algorithm 1); 1: previous u_l (reading R11) */
  double relax;     /* rho in (0,1]; 1 = eq. (2) literally; configs use 0.5 (reading R12) */
  double tol;       /* > 0: stop when the global relative residual <= tol (checked every check_every sweeps) */
  int check_every;  /* residual check period in sweeps; <= 0 = never (run exactly n_outer_max) */
  int reset_state;  /* 1: zero lambda and u_l before the first sweep; 0: continue from the current state */
  int use_graph;    /* 1: the {sweep, exchange} pairs between two residual checks are captured once into a CUDA
                       graph and replayed (removes the per-launch overhead that dominates tiny configs); the
                       per-kernel timings of hz_solve_info are then not measured (-1), total_ms still is */
} hz_solve_opts;

typedef struct {
  int n_outer_done;
  int n_t;
  double rel_residual;   /* last residual computed, or -1 if none was */
  double sweep_ms_total; /* device time of all sweep launches (CUDA events on `stream`); -1 with use_graph */
  double exch_ms_total;  /* device time of all exchange launches */
  double total_ms;       /* device time of the whole call on `stream` */
  double dof_timesteps;  /* sum_l N_l * n_wh * (n_t-1) * n_outer_done  (WaveHoltz DOF-timestep updates) */
  int sweep_launches, exch_launches, other_launches; /* kernels launched by this call */
} hz_solve_info;

/* ---------------------------------------------------------------------------------------------
 * hz_ddm_solve — the outer iteration on the interface data lambda (eq. (2) with the
 * sign of reading R3): each sweep applies the DDM cycle of Algorithm 1 to all
 * subdomains concurrently in ONE kernel launch, then exchanges the outgoing
 * interface data with relaxation.
 *
 *   u_out   DEVICE or NULL: 2*(nx*p+1)*(ny*p+1) reals of the partition's precision, re plane then
 *           im plane; nodes shared by several subdomains hold the mean of their copies (reading R19).
 *   info    may be NULL.
 *   stream  a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); 0 = default stream.
 * The call enqueues all work on `stream` and synchronises the stream before returning (timings
 * in `info` are then valid).
 * ------------------------------------------------------------------------------------------- */
hz_status hz_ddm_solve(hz_ctx *ctx, const hz_solve_opts *opts, void *u_out, hz_solve_info *info, void *stream);

/* The paper's "operator time" normaliser (the DDM cycle is compared "to the time it takes to evaluate
 * the Helmholtz operator A - i w H - w^2 M on the entire domain"): `reps` back-to-back evaluations y = (A - i w H -
 * w^2 M) u of the global operator in the arithmetic `prec` (that of the DDM cycle it normalises).
 *   u_dev  DEVICE, 2*(nx*p+1)*(ny*p+1) values of precision prec (re plane, im plane).
 *   y_dev  DEVICE or NULL: receives y (same layout and precision); NULL = a vector owned by the context.
 *   *ms_per_eval = CUDA-event time / reps.
 * General-quadrilateral contexts: HZ_F64 and y_dev = NULL only (the residual kernel is timed). */
hz_status hz_operator_time(hz_ctx *ctx, const void *u_dev, hz_prec prec, int reps, void *y_dev, double *ms_per_eval,
                           void *stream);

/* ---------------------------------------------------------------------------------------------
 * hz_ddm_solve_sources — a stream of right-hand sides on one mesh and partition, end to end from HOST to HOST:
 * for s = 0..n_src-1: copy source f_s to the device, rebuild the load ("Assemble b from f"), run
 * opts->n_outer_max {sweep, exchange} pairs (continuing from the current lambda / u_l unless opts->reset_state),
 * gather the field and copy it to u_host[s].  The copies run on two private streams with double-buffered staging, so
 * the upload of source s+1 and the download of field s-1 overlap the sweeps of source s; the results are bit-identical
 * to hz_set_source + hz_ddm_solve + a device-to-host copy, source by source.
 *
 *   f_re_host  n_src HOST pointers, (nx*p+1)*(ny*p+1) doubles each (pinned memory for the copies to overlap);
 *              real sources only (HZ_EUNSUPPORTED if the context has an imaginary source).
 *   u_host     n_src HOST pointers, 2*(nx*p+1)*(ny*p+1) values of the PARTITION's precision each (re, then im).
 *   opts       n_outer_max (>= 1), n_wh, warm_start, relax, reset_state are used; no tolerance check.
 *   info       optional; total_ms = CUDA-event time from the first upload to the last download.
 * On return all copies have completed and the context holds the last source.
 * ------------------------------------------------------------------------------------------- */
typedef struct {
  int sources_done;
  double total_ms;
  double dof_timesteps;        /* all sources together */
  int launches;                /* kernels launched (build + sweeps + exchanges + gather per source) */
  double h2d_bytes, d2h_bytes; /* copied in total */
} hz_sources_info;
hz_status hz_ddm_solve_sources(hz_ctx *ctx, const hz_solve_opts *opts, int n_src, const double *const *f_re_host,
                               void *const *u_host, hz_sources_info *info, void *stream);

/* ---------------------------------------------------------------------------------------------
 * hz_ddm_solve_gmres — Krylov acceleration of the outer iteration (the fixed-point iteration on
 * lambda "can be accelerated with a Krylov space method").  One warm-started sweep (sweep kernel + exchange
 * kernel, exactly as in hz_ddm_solve) is an affine, real-linear map x -> T x + c of the joint state
 * x = (lambda, u_l); restarted GMRES(restart) solves (I - T) x = c, one sweep per Arnoldi step (classical
 * Gram-Schmidt applied twice, Givens rotations on the host).  The fixed point is the DDM fixed point.
 *
 * lambda_only = 1: the Krylov iteration on lambda ALONE.  With cold-started sweeps (u^(0) = 0, Algorithm 1 as printed,
 * PAPER.md:164) and a fixed n_wh, lambda -> G lambda + d is an affine map of the interface data alone, so the basis
 * vectors have the size of the interfaces (about 1/25 of the joint state at 625 DOFs per subdomain) and a large
 * `restart` is cheap.  Its fixed point is the DDM fixed point of the INEXACT subdomain solver (n_wh WaveHoltz
 * iterations from zero): n_wh sets the attainable Helmholtz residual (about 0.55^n_wh on 8x8-element subdomains).
 * The field returned is u_l(lambda) from one more sweep kernel at the final lambda (lambda not advanced), followed by
 * n_polish warm-started WaveHoltz iterations at that lambda.
 * ------------------------------------------------------------------------------------------- */
typedef struct {
  int n_wh;        /* WaveHoltz iterations per sweep (>= 1) */
  double relax;    /* rho in (0,1] of the exchange */
  int restart;     /* Krylov vectors per cycle (>= 1) */
  int max_steps;   /* Arnoldi steps (= sweeps, besides one per cycle start) to run at most */
  double lin_tol;  /* > 0: stop when the relative linear residual ||c - (I-T)x|| / ||c|| <= lin_tol */
  double tol;      /* > 0: stop when the global Helmholtz residual (hz_residual) <= tol.  It is evaluated at the end of
                      a cycle; a cycle is ended early once the linear residual estimate reaches tol/2 (a target
                      that is tightened whenever the true residual is still above tol) */
  int reset_state; /* 1: start from x = 0; 0: start from the context's current (lambda, u_l) */
  double *lin_history; /* HOST or NULL: receives the relative linear residual after each Arnoldi step */
  int history_len;     /* capacity of lin_history */
  int lambda_only;     /* 0: x = (lambda, u_l), warm-started sweeps; 1: x = lambda, cold-started sweeps (see above) */
  int n_polish;        /* lambda_only: WaveHoltz iterations added to u_l at the final lambda (>= 0) */
} hz_gmres_opts;

typedef struct {
  int steps_done;      /* Arnoldi steps */
  int sweeps_done;     /* sweep launches (steps + one per cycle start + one for c) */
  int cycles;
  double lin_residual; /* last relative linear residual estimate */
  double rel_residual; /* global Helmholtz residual of the final iterate (always computed) */
  double total_ms;     /* device time of the call */
  size_t krylov_bytes; /* device memory held by the Krylov basis */
} hz_gmres_info;

hz_status hz_ddm_solve_gmres(hz_ctx *ctx, const hz_gmres_opts *opts, void *u_out, hz_gmres_info *info, void *stream);

/* ---------------------------------------------------------------------------------------------
 * hz_ddm_solve_mixed — the fp32 path to the fp64 path's residual tolerance ("Since the DDM is a
 * preconditioner, we can gain significant speedups simply by evaluating the preconditioner in a lower precision";
 * reading R27).  Defect correction in the DDM state space X = (lambda, u_l), X held in fp64 by `hi`:
 *     D = F(X) - X                              one fp64 sweep + exchange on `hi` (F = the warm-started sweep map)
 *     delta_1 = D,  delta_{k+1} = T delta_k + D  m_inner - 1 fp32 sweeps + exchanges on `lo` with the load removed
 *     X <- X + delta_m
 * Without rounding a cycle is exactly m_inner plain sweeps; the fp32 sweeps only ever see the correction, so the
 * iteration converges to the fixed point of the fp64 map at the fp64 rate, at close to fp32 cost.
 *
 *   lo, hi   two contexts of the SAME mesh, source and subdomain grid (else HZ_EINVAL), partitioned with
 *            HZ_F32 and HZ_F64 respectively (else HZ_ESTATE); uniform-mesh contexts with a real source.
 *            `hi` holds X (continue / reset as in hz_ddm_solve); the state of `lo` is scratch.
 *   u_out    DEVICE or NULL: 2*(nx*p+1)*(ny*p+1) DOUBLES, the gathered fp64 field.
 * The global residual (hz_residual of the gathered X, fp64) is checked after every check_every cycles.
 * ------------------------------------------------------------------------------------------- */
typedef struct {
  int n_cycles_max; /* defect-correction cycles (>= 0); one cycle advances the iteration by m_inner sweeps */
  int m_inner;      /* >= 1 */
  int n_wh;         /* WaveHoltz iterations per sweep */
  double relax;     /* rho in (0,1] */
  double tol;       /* > 0: stop when the global relative residual <= tol */
  int check_every;  /* in cycles; <= 0 = never */
  int reset_state;  /* 1: X = 0 first */
} hz_mixed_opts;
typedef struct {
  int cycles_done;
  int sweeps_lo, sweeps_hi; /* fp32 / fp64 sweep launches */
  double rel_residual;      /* last residual computed, or -1 */
  double total_ms;          /* device time of the call */
  double dof_timesteps;     /* of all sweeps, both precisions */
} hz_mixed_info;
hz_status hz_ddm_solve_mixed(hz_ctx *lo, hz_ctx *hi, const hz_mixed_opts *opts, double *u_out, hz_mixed_info *info,
                             void *stream);

/* ---------------------------------------------------------------------------------------------
 * hz_minres_cycle — the paper's comparator: one DDM cycle on every subdomain (one thread
 * block per subdomain, one launch) with unpreconditioned MINRES on the real symmetric block system (5)
 * as the subdomain solver instead of WaveHoltz.  Assembles b from f and the current lambda^n,
 * iterates until the recurrence's relative residual <= tol (the paper: 1e-6 in single, 1e-12 in double precision) or
 * max_iters, stores u_l and the outgoing interface data, then (relax > 0) runs the exchange kernel.
 * Runs in the layout of the partition: one DOF per thread (hz_partition(..., dofs_per_thread = 1)), or register-blocked
 * with the WaveHoltz kernels' square thread tiles of at most 16 DOFs (k = 4, 9, 16; one thread block per subdomain
 * even where the WaveHoltz sweep packs several or uses a cluster: those give HZ_EUNSUPPORTED, like larger tiles).
 * max_iters = 0 with warm_start = 1 only evaluates the subdomain residuals of the current u_l.
 *   iters_out  HOST or NULL: `blocks` ints, MINRES iterations of each subdomain.
 *   res_out    HOST or NULL: `blocks` doubles, true relative residual ||rhs - K x|| / ||rhs|| of each subdomain.
 * ------------------------------------------------------------------------------------------- */
typedef struct {
  double tol;
  int max_iters;
  int warm_start;  /* 0: x0 = 0; 1: x0 = current u_l */
  double relax;    /* > 0: run the exchange with this rho afterwards; 0: leave lambda untouched */
} hz_minres_opts;

typedef struct {
  int iters_max;
  double iters_mean;
  double res_max;    /* largest true relative subdomain residual */
  double kernel_ms;  /* device time of the MINRES kernel */
} hz_minres_info;

hz_status hz_minres_cycle(hz_ctx *ctx, const hz_minres_opts *opts, int *iters_out, double *res_out,
                          hz_minres_info *info, void *stream);

/* Relative residual || b - (A - i w H - w^2 M) u ||_2 / || b ||_2 of a global nodal vector on the
 * UNPARTITIONED system (4) (the operator is the "Operator time" kernel of PAPER.md:223),
 * accumulated in fp64.  u_dev: DEVICE, layout as u_out, of precision u_prec.  Synchronises `stream`. */
hz_status hz_residual(hz_ctx *ctx, const void *u_dev, hz_prec u_prec, double *rel_residual, void *stream);

/* ---------------------------------------------------------------------------------------------
 * hz_residual_static — hz_residual for callers that cannot allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the same kernels (k_helm / k_residual_quad block partial sums, fp64
 * reduction), but the partial sums live in a file-scope `static __device__` array of the library
 * instead of the context's lazily allocated buffers, the result stays on the DEVICE, and the call neither allocates,
 * frees, copies to the host nor synchronises: it only enqueues work on `stream`.
 *
 *   ctx               a context of hz_mesh_setup / hz_mesh_setup_quads (its device arrays c, f, bc are the inputs);
 *                     hz_partition is not needed.  The context's device must be current.
 *   u_dev             DEVICE, layout as u_out (re plane then im plane), of precision u_prec.
 *   rel_residual_dev  DEVICE, 1 double, owned by the caller: receives ||b - (A - i w H - w^2 M) u|| / ||b||
 *                     (bit-identical to hz_residual) once the work enqueued on `stream` has run.
 * Limit: the mesh may need at most HZ_RESIDUAL_STATIC_MAX_BLOCKS partial-sum blocks (uniform meshes: one per patch
 * of 32 x 8 elements, ceil((nx+1)/32) * ceil((ny+1)/8); general quads: one per 256 nodes), i.e. 4 MiB + 256 bytes of
 * device memory, which EVERY GPU that loads the library holds until the process exits.  That covers all BASELINE.json
 * configs (config 5 at p = 1: 148 417 blocks).  Larger meshes: HZ_EINVAL with a message (use hz_residual).
 * The array is shared by all contexts and calls of the process on one device and keeps the last call's contents
 * (the slots a call reads are cleared first, on `stream`): calls that overlap on the GPU (different streams, or
 * several host threads without stream ordering) RACE on it; calls ordered on one stream are safe, as are different devices.
 * hz_residual_static_setup resolves the array's device address for the CURRENT device (cudaGetSymbolAddress; cached per
 * device).  Call it once per device at set-up, e.g. before stream capture begins; hz_residual_static does the same
 * on first use otherwise.  Errors: HZ_ECUDA with the CUDA message.
 * ------------------------------------------------------------------------------------------- */
#define HZ_RESIDUAL_STATIC_MAX_BLOCKS 262144
int hz_residual_static_max_blocks(void);
hz_status hz_residual_static_setup(hz_ctx *ctx);
hz_status hz_residual_static(hz_ctx *ctx, const void *u_dev, hz_prec u_prec, double *rel_residual_dev, void *stream);

/* Raw state for parity tests.  u_sub_dev: DEVICE or NULL, doubles [blocks][2][dofs_per_sub]
 * (re then im, local node (I,J) at J*edge_nodes_x+I).  lambda_dev: DEVICE or NULL, doubles
 * [blocks][4][2][edge_stride] (current lambda^n; zeros on physical sides). */
hz_status hz_get_subdomain_state(hz_ctx *ctx, double *u_sub_dev, double *lambda_dev, void *stream);

/* Overwrite the state (same layouts; either may be NULL = keep).  Used by the paper-style benchmark
 * that applies one DDM cycle to a random interface vector. */
hz_status hz_set_subdomain_state(hz_ctx *ctx, const double *u_sub_dev, const double *lambda_dev, void *stream);

/* Message of the last failure on this context ("" if none).  Valid until the next call on ctx.
 * Not thread-safe.  ctx == NULL returns the message of the last failed hz_mesh_setup. */
const char *hz_last_error(const hz_ctx *ctx);

/* Frees the context and all its device memory.  NULL-safe. */
void hz_destroy(hz_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* HZ_H */
