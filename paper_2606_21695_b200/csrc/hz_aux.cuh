// hz_aux.cuh — the kernels around the sweep: per-subdomain operator builder (A0), interface exchange (A8),
// gather of the global field (A7/R19), global residual (A10), state import/export and the peak probes.
#pragma once
#include "hz_internal.h"

namespace hz {

// Mesh / partition description used by the auxiliary kernels (all fp64).
struct Geo {
  int nx, ny, p, npx, npy;  // global elements, degree, global nodes per side
  int sx, sy, ex, ey;       // subdomain grid, elements per subdomain side (the maximum, for ragged partitions)
  int exq, exr, eyq, eyr;   // nx = sx*exq + exr, ny = sy*eyq + eyr: the first exr (eyr) subdomain columns (rows)
                            // have exq+1 (eyq+1) elements, the others exq (eyq) (reading R25); uniform: exr = eyr = 0
  int E, EB;                // edge stride of lambda arrays; of the bc_lambda side blocks
  double hx, hy, omega, theta, sigma;
};

// even split of n = s*q + r elements into s groups: size, offset of group k, group of element e
__host__ __device__ inline int sub_size(int q, int r, int k) { return q + (k < r ? 1 : 0); }
__host__ __device__ inline int sub_off(int q, int r, int k) { return k * q + (k < r ? k : r); }
__host__ __device__ inline int sub_of_elem(int q, int r, int e) {
  return e < r * (q + 1) ? e / (q + 1) : r + (e - r * (q + 1)) / q;
}

// ---------------------------------------------------------------------------------------------
// A0: per-subdomain operator data (PAPER.md:107-113 for M, H; PAPER.md:144 for alpha, beta).
// One thread per (subdomain, local node).  wxl/wyl: assembled reference GLL weights of the ex (ey)
// elements of a subdomain side.  Everything is computed in fp64 and rounded once.
// ---------------------------------------------------------------------------------------------
// Index arithmetic without divisions: gid -> (subdomain, row, column) by multiplication with host-computed
// reciprocals (floor(x / d) = umul64hi(x, ceil(2^64 / d)) exactly for x, d < 2^32), the slot from the separable
// tables sxp[i] + syp[j] of Layout::slot; one reciprocal of c and one of the denominator instead of six divisions.
struct BuildIdx {
  unsigned long long magN, magLnx, magSx;   // ceil(2^64 / N), ceil(2^64 / lnx), ceil(2^64 / sx)
  const int *sxp, *syp;              // [lnx], [lny]: x and y part of Layout::slot
};
template <typename real>
__global__ void k_build(Geo g, Layout lay, BuildIdx bi, const double *__restrict__ c, const double *__restrict__ f_re,
                        const double *__restrict__ f_im, const double *__restrict__ bc, const double *__restrict__ wxl,
                        const double *__restrict__ wyl, real *gamma, real *alpha, real *bbf_re, real *bbf_im,
                        real *k2edge, real *bs, int only_source) {
  const int N = lay.lnx * lay.lny;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long total = (long long)g.sx * g.sy * N;
  if (gid >= total) return;
  const int l = (int)__umul64hi((unsigned long long)gid, bi.magN), q = (int)(gid - (long long)l * N);
  const int j = (int)__umul64hi((unsigned long long)q, bi.magLnx), i = q - j * lay.lnx;
  const int siy = g.sx == 1 ? l : (int)__umul64hi((unsigned long long)l, bi.magSx), six = l - siy * g.sx;
  const int I = six * g.ex * g.p + i, J = siy * g.ey * g.p + j;
  const size_t gn = (size_t)J * g.npx + I;
  const double cj = c[gn], rc = 1.0 / cj;
  const double m = 0.25 * g.hx * g.hy * wxl[i] * wyl[j];  // local lumped mass (geometric)
  const double M = m * rc * rc;
  // impedance weight on the WHOLE subdomain boundary: interfaces carry the same operator as the
  // outer boundary
  const bool onW = i == 0, onE = i == lay.lnx - 1, onS = j == 0, onN = j == lay.lny - 1;
  const double sWE = 0.5 * g.hy * wyl[j], sSN = 0.5 * g.hx * wxl[i];
  double H = 0.0;
  if (onW) H += sWE * rc;
  if (onE) H += sWE * rc;
  if (onS) H += sSN * rc;
  if (onN) H += sSN * rc;
  const double den = M + g.theta * H, rden = 1.0 / den;
  const double beta = g.sigma * rden;
  // load: f(x_j) m_j (+ the outer-boundary datum lambda of eq. (1b) on physical sides)
  double bre = f_re[gn] * m, bim = f_im ? f_im[gn] * m : 0.0;
  if (bc) {
    if (onW && six == 0) { bre += sWE * bc[(0 * 2 + 0) * g.EB + J]; bim += sWE * bc[(0 * 2 + 1) * g.EB + J]; }
    if (onE && six == g.sx - 1) { bre += sWE * bc[(1 * 2 + 0) * g.EB + J]; bim += sWE * bc[(1 * 2 + 1) * g.EB + J]; }
    if (onS && siy == 0) { bre += sSN * bc[(2 * 2 + 0) * g.EB + I]; bim += sSN * bc[(2 * 2 + 1) * g.EB + I]; }
    if (onN && siy == g.sy - 1) { bre += sSN * bc[(3 * 2 + 0) * g.EB + I]; bim += sSN * bc[(3 * 2 + 1) * g.EB + I]; }
  }
  const size_t o = (size_t)l * lay.NS + bi.sxp[i] + bi.syp[j];
  bbf_re[o] = (real)(beta * bre);
  if (bbf_im) bbf_im[o] = (real)(beta * bim);
  if (only_source) return;
  gamma[o] = (real)(beta * m);
  alpha[o] = (real)((M - g.theta * H) * rden);
  const size_t eb = (size_t)l * 4 * g.E;
  const double k2 = 2.0 * g.omega * rc;
  if (onW) { k2edge[eb + 0 * g.E + j] = (real)k2; bs[eb + 0 * g.E + j] = (real)(beta * sWE); }
  if (onE) { k2edge[eb + 1 * g.E + j] = (real)k2; bs[eb + 1 * g.E + j] = (real)(beta * sWE); }
  if (onS) { k2edge[eb + 2 * g.E + i] = (real)k2; bs[eb + 2 * g.E + i] = (real)(beta * sSN); }
  if (onN) { k2edge[eb + 3 * g.E + i] = (real)k2; bs[eb + 3 * g.E + i] = (real)(beta * sSN); }
}

// ---------------------------------------------------------------------------------------------
// Operator data of the MINRES comparator (block system (5)), natural slot layout:
// m_j, w^2 M_j, w H_j, the load f m (+ outer-boundary datum) and the geometric edge weights s_j^{side}.
// ---------------------------------------------------------------------------------------------
template <typename real>
__global__ void k_build_minres(Geo g, Layout lay, const double *__restrict__ c, const double *__restrict__ f_re,
                               const double *__restrict__ f_im, const double *__restrict__ bc,
                               const double *__restrict__ wxl, const double *__restrict__ wyl, real *mloc, real *w2M,
                               real *wH, real *bf_re, real *bf_im, real *sedge) {
  const int N = lay.lnx * lay.lny;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= (long long)g.sx * g.sy * N) return;
  const int l = (int)(gid / N), q = (int)(gid - (long long)l * N);
  const int i = q % lay.lnx, j = q / lay.lnx;
  const int six = l % g.sx, siy = l / g.sx;
  const int I = six * g.ex * g.p + i, J = siy * g.ey * g.p + j;
  const size_t gn = (size_t)J * g.npx + I;
  const double cj = c[gn];
  const double m = 0.25 * g.hx * g.hy * wxl[i] * wyl[j];
  const bool onW = i == 0, onE = i == lay.lnx - 1, onS = j == 0, onN = j == lay.lny - 1;
  const double sWE = 0.5 * g.hy * wyl[j], sSN = 0.5 * g.hx * wxl[i];
  double H = 0.0;
  if (onW) H += sWE / cj;
  if (onE) H += sWE / cj;
  if (onS) H += sSN / cj;
  if (onN) H += sSN / cj;
  double bre = f_re[gn] * m, bim = f_im ? f_im[gn] * m : 0.0;
  if (bc) {
    if (onW && six == 0) { bre += sWE * bc[(0 * 2 + 0) * g.EB + J]; bim += sWE * bc[(0 * 2 + 1) * g.EB + J]; }
    if (onE && six == g.sx - 1) { bre += sWE * bc[(1 * 2 + 0) * g.EB + J]; bim += sWE * bc[(1 * 2 + 1) * g.EB + J]; }
    if (onS && siy == 0) { bre += sSN * bc[(2 * 2 + 0) * g.EB + I]; bim += sSN * bc[(2 * 2 + 1) * g.EB + I]; }
    if (onN && siy == g.sy - 1) { bre += sSN * bc[(3 * 2 + 0) * g.EB + I]; bim += sSN * bc[(3 * 2 + 1) * g.EB + I]; }
  }
  const size_t o = (size_t)l * lay.NS + lay.slot(i, j);
  mloc[o] = (real)m;
  w2M[o] = (real)(g.omega * g.omega * m / (cj * cj));
  wH[o] = (real)(g.omega * H);
  bf_re[o] = (real)bre;
  if (bf_im) bf_im[o] = (real)bim;
  const size_t eb = (size_t)l * 4 * g.E;
  if (onW) sedge[eb + 0 * g.E + j] = (real)sWE;
  if (onE) sedge[eb + 1 * g.E + j] = (real)sWE;
  if (onS) sedge[eb + 2 * g.E + i] = (real)sSN;
  if (onN) sedge[eb + 3 * g.E + i] = (real)sSN;
}

// ---------------------------------------------------------------------------------------------
// A8: exchange with relaxation (eq. (2); readings R3, R12):
//   lambda^{n+1}_{r,o} = (1-rho) lambda^n_{r,o} + rho g_{nb(r,o), opp(o)}      on interface sides.
// One thread per (subdomain r, side o, re/im, edge node); in place on lambda (each entry is read and
// written by one thread only; g is a separate array).
// ---------------------------------------------------------------------------------------------
template <typename real>
__global__ void k_exchange(int sx, int sy, int E, int ex_nodes, int ey_nodes, real rho, real *__restrict__ lam,
                           const real *__restrict__ g) {
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long total = (long long)sx * sy * 8 * E;
  if (gid >= total) return;
  const int e = (int)(gid % E);
  const int c = (int)((gid / E) % 2);
  const int o = (int)((gid / (2 * E)) % 4);
  const int r = (int)(gid / (8 * E));
  const int rx = r % sx, ry = r / sx;
  int nb = -1;
  if (o == kSideW && rx > 0) nb = r - 1;
  if (o == kSideE && rx < sx - 1) nb = r + 1;
  if (o == kSideS && ry > 0) nb = r - sx;
  if (o == kSideN && ry < sy - 1) nb = r + sx;
  if (nb < 0) return;
  const int len = (o < 2) ? ey_nodes : ex_nodes;
  if (e >= len) return;
  const int opp = o ^ 1;
  const real gv = g[(((size_t)nb * 4 + opp) * 2 + c) * E + e];
  lam[gid] = (real(1) - rho) * lam[gid] + rho * gv;
}

// ---------------------------------------------------------------------------------------------
// A7 / R19: global nodal field, mean of the copies at nodes shared by several subdomains, summed in
// the fixed order (iy ascending, ix ascending).
// ---------------------------------------------------------------------------------------------
// Layout::slot is separable: slot(i, j) = sx(i) + sy(j).  The host tabulates, for every GLOBAL node column I (row J),
// the subdomain column (row) that owns the element having it as a lower node, the x (y) part of the slot there and, at a
// node shared with the subdomain column (row) before, the part there: no divisions in the kernel, and the mean over
// 1, 2 or 4 copies is a multiplication by an exact power of two.
struct GatherLine {
  int s1;     // subdomain column ix1 (x table) / iy1 * sx (y table): the last subdomain that holds the line
  int p1;     // slot part of the line in that subdomain
  int p0;     // slot part in the subdomain before (valid if n == 2)
  int n;      // 1 or 2 copies along this direction
};
template <typename real, typename outT>
__global__ void __launch_bounds__(256) k_gather(int npx, int npy, int sxg, size_t NS, const GatherLine *__restrict__ colx,
                                                const GatherLine *__restrict__ rowy, const real *__restrict__ u_sub,
                                                outT *__restrict__ u_out) {
  const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y;
  if (I >= npx) return;
  const GatherLine cx = colx[I], ry = rowy[J];
  const size_t total = (size_t)npx * npy, gid = (size_t)J * npx + I;
  double sr = 0.0, si = 0.0;
  // fixed order: iy ascending, ix ascending (reading R19)
  for (int ky = ry.n - 1; ky >= 0; --ky) {
    const int ly = ry.s1 - ky * sxg, py = ky ? ry.p0 : ry.p1;
    for (int kx = cx.n - 1; kx >= 0; --kx) {
      const size_t o = (size_t)(ly + cx.s1 - kx) * 2 * NS + (size_t)(py + (kx ? cx.p0 : cx.p1));
      sr += (double)u_sub[o];
      si += (double)u_sub[o + NS];
    }
  }
  const double w = 1.0 / (double)(cx.n * ry.n);   // 1, 1/2, 1/4: exact
  u_out[gid] = (outT)(sr * w);
  u_out[total + gid] = (outT)(si * w);
}

// ---------------------------------------------------------------------------------------------
// A10: r = b - (A - i w H - w^2 M) u on the unpartitioned system (4), fp64.
// One thread per global node; the stiffness is applied matrix-free from the 1-D element matrix
// K1 = D^T W D in constant memory.  Block partial sums of |r|^2 and |b|^2 are
// written to part[2*blockIdx] and reduced in a fixed order by k_reduce2 (deterministic).
// ---------------------------------------------------------------------------------------------
struct Ref1D {
  double K[kMaxP + 1][kMaxP + 1];
  double w[kMaxP + 1];
};

// 1-D reference data of the global operator kernel in its own arithmetic (filled on the host once per launch):
// the element stiffness rows already carry the metric factor of their direction, so the kernel has no divisions.
template <typename acc>
struct HelmC {
  acc kx[kMaxP + 1][kMaxP + 1];  // (hy / hx) K1[a][c],  K1 = D^T W D
  acc ky[kMaxP + 1][kMaxP + 1];  // (hx / hy) K1[a][c]
  acc w[kMaxP + 1];              // GLL weights
  acc wa[kMaxP + 1];             // assembled weights of an interior node line: wa[0] = w[0] + w[P], wa[a] = w[a]
  acc mh;                        // hx hy / 4
  // interior blocks: the assembled row of a node shared by two elements (index c + P, c = -P..P) and the lumped mass
  // mh wa[a] wa[b] of tile node (a, b)
  acc kx0[2 * kMaxP + 1], ky0[2 * kMaxP + 1];
  acc wm[kMaxP][kMaxP];
};
__device__ __forceinline__ float hfma(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double hfma(double a, double b, double c) { return fma(a, b, c); }

// Launch shape of k_helm: a block of HB_X x HB_Y threads, one thread per ELEMENT (its P x P lower-left nodes, as in the
// sweep kernels; the phantom elements nx / ny own the last node column / row), and its shared-memory patch.
constexpr int kHelmBX = 32, kHelmBY = 8;
// shared memory: the u patch (re, im) of the input type; MODE 1 adds the w^2/c^2 values of the block's own nodes
inline size_t helm_smem(int P, size_t elem_in, size_t elem_k2) {
  return 2 * (size_t)((kHelmBX + 1) * P + 1) * ((kHelmBY + 1) * P + 1) * elem_in + (size_t)kHelmBX * P * kHelmBY * P * elem_k2;
}
// The gx x gy grid of patches and the range [1, bxh) x [1, byh) of patches strictly inside the mesh (interior kernel);
// the other patches (a ring) go to the general kernel.  bxh = byh = 1: no interior patch.
struct HelmGrid {
  int gx, gy, bxh, byh;
};
inline HelmGrid helm_grid(int nx, int ny, int P) {
  HelmGrid h;
  h.gx = (nx + 1 + kHelmBX - 1) / kHelmBX;
  h.gy = (ny + 1 + kHelmBY - 1) / kHelmBY;
  const int PW = (kHelmBX + 1) * P + 1, PH = (kHelmBY + 1) * P + 1, npx = nx * P + 1, npy = ny * P + 1;
  // patch b is interior iff b >= 1 and b * B * P - P + PW <= np - 1
  const int lx = npx - 1 - PW + P, ly = npy - 1 - PH + P;
  h.bxh = lx < 0 ? 1 : lx / (kHelmBX * P) + 1;
  h.byh = ly < 0 ? 1 : ly / (kHelmBY * P) + 1;
  if (h.bxh < 1) h.bxh = 1;
  if (h.byh < 1) h.byh = 1;
  if (h.bxh > h.gx) h.bxh = h.gx;
  if (h.byh > h.gy) h.byh = h.gy;
  if (h.bxh == 1 || h.byh == 1) h.bxh = h.byh = 1;
  return h;
}
// resident blocks per SM the kernel is compiled for (register cap 64K / (256 * n)): several blocks per SM are what
// overlaps the cp.async staging of one block with the arithmetic of another
template <typename acc, int P, int MODE, bool TMA = false>
constexpr int helm_minb() {
  if (MODE == 0) return 2;
  if (sizeof(acc) == 4) return P <= 2 ? 6 : (P == 3 ? 4 : 3);
  return P == 1 ? 6 : (P == 2 ? 3 : (P == 3 ? (TMA ? 3 : 2) : 2));
}

// asynchronous global -> shared copy of one 4- or 8-byte element (cp.async, no register staging: the whole patch of a
// block is in flight at once); pred = false writes zeros (src-size 0)
template <int BYTES>
__device__ __forceinline__ void cp_async_elem(void *dst_smem, const void *src, bool pred) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
  const int sz = pred ? BYTES : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2, %3;" ::"r"(d), "l"(src), "n"(BYTES), "r"(sz) : "memory");
}
template <int BYTES>
__device__ __forceinline__ void cp_async_elem(void *dst_smem, const void *src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(d), "l"(src), "n"(BYTES) : "memory");
}

// One thread's P x P nodes of k_helm from the staged patch, anywhere in the mesh (one-sided weights, missing
// neighbours, the impedance term and the datum of eq. (1b) on the outer boundary).
template <typename inT, typename acc, int P, int MODE>
__device__ __forceinline__ void helm_tile(const Geo &g, const HelmC<acc> &hc, const double *__restrict__ c,
                                          const double *__restrict__ f_re, const double *__restrict__ f_im,
                                          const double *__restrict__ bc, const inT *sr, const inT *si, const acc *sk, int PW,
                                          int OW, int tx, int ty, int ex, int ey, double &r2, double &b2,
                                          acc (&outr)[MODE == 1 ? P : 1][MODE == 1 ? P : 1],
                                          acc (&outi)[MODE == 1 ? P : 1][MODE == 1 ? P : 1]) {
  const bool hasL = ex > 0, hasR = ex < g.nx, hasD = ey > 0, hasU = ey < g.ny;
  const int bx = (tx + 1) * P, by = (ty + 1) * P;   // patch coordinates of the tile's first node
#pragma unroll
  for (int b = 0; b < P; ++b) {
    if (b > 0 && !hasU) break;
    const acc wy = b == 0 ? (hasD ? hc.w[P] : acc(0)) + (hasU ? hc.w[0] : acc(0)) : hc.w[b];
#pragma unroll
    for (int a = 0; a < P; ++a) {
      if (a > 0 && !hasR) break;
      const acc wx = a == 0 ? (hasL ? hc.w[P] : acc(0)) + (hasR ? hc.w[0] : acc(0)) : hc.w[a];
      const inT *rr = sr + (by + b) * PW + bx, *ri = si + (by + b) * PW + bx;   // row of this node, at the tile's x origin
      const inT *cr = sr + by * PW + bx + a, *ci = si + by * PW + bx + a;       // column of this node, at the tile's y origin
      acc kxr = 0, kxi = 0, kyr = 0, kyi = 0;
      if (a == 0) {   // node shared by the element on the left (its row P) and this one (row 0), where they exist
#pragma unroll
        for (int cc = 0; cc <= P; ++cc) {
          const acc kl = hasL ? hc.kx[P][cc] : acc(0), kr = hasR ? hc.kx[0][cc] : acc(0);
          kxr += kl * (acc)rr[cc - P] + kr * (acc)rr[cc];
          kxi += kl * (acc)ri[cc - P] + kr * (acc)ri[cc];
        }
      } else {
#pragma unroll
        for (int cc = 0; cc <= P; ++cc) {
          kxr += hc.kx[a][cc] * (acc)rr[cc];
          kxi += hc.kx[a][cc] * (acc)ri[cc];
        }
      }
      if (b == 0) {
#pragma unroll
        for (int cc = 0; cc <= P; ++cc) {
          const acc kd = hasD ? hc.ky[P][cc] : acc(0), ku = hasU ? hc.ky[0][cc] : acc(0);
          kyr += kd * (acc)cr[(cc - P) * PW] + ku * (acc)cr[cc * PW];
          kyi += kd * (acc)ci[(cc - P) * PW] + ku * (acc)ci[cc * PW];
        }
      } else {
#pragma unroll
        for (int cc = 0; cc <= P; ++cc) {
          kyr += hc.ky[b][cc] * (acc)cr[cc * PW];
          kyi += hc.ky[b][cc] * (acc)ci[cc * PW];
        }
      }
      const int I = ex * P + a, J = ey * P + b;
      const size_t n = (size_t)J * g.npx + I;
      const acc u_r = (acc)rr[a], u_i = (acc)ri[a];
      const acc Aur = wy * kxr + wx * kyr, Aui = wy * kxi + wx * kyi;
      const acc m = hc.mh * wx * wy;
      acc kk;   // w^2 / c^2
      double cj = 0.0;
      if (MODE == 1) kk = sk[(ty * P + b) * OW + tx * P + a];
      else { cj = c[n]; kk = (acc)(g.omega * g.omega / (cj * cj)); }
      acc wH = 0;
      double bre = 0.0, bim = 0.0;
      if (MODE == 0) { bre = f_re[n] * (double)m; bim = f_im ? f_im[n] * (double)m : 0.0; }
      {
        const bool onb = I == 0 || I == g.npx - 1 || J == 0 || J == g.npy - 1;
        if (onb) {   // impedance term and datum of eq. (1b) on the outer boundary only
          if (MODE == 1) cj = c[n];
          const double sWE = 0.5 * g.hy * (double)wy, sSN = 0.5 * g.hx * (double)wx;
          double H = 0.0;
          if (I == 0) { H += sWE / cj; if (MODE == 0 && bc) { bre += sWE * bc[(0 * 2 + 0) * g.EB + J]; bim += sWE * bc[(0 * 2 + 1) * g.EB + J]; } }
          if (I == g.npx - 1) { H += sWE / cj; if (MODE == 0 && bc) { bre += sWE * bc[(1 * 2 + 0) * g.EB + J]; bim += sWE * bc[(1 * 2 + 1) * g.EB + J]; } }
          if (J == 0) { H += sSN / cj; if (MODE == 0 && bc) { bre += sSN * bc[(2 * 2 + 0) * g.EB + I]; bim += sSN * bc[(2 * 2 + 1) * g.EB + I]; } }
          if (J == g.npy - 1) { H += sSN / cj; if (MODE == 0 && bc) { bre += sSN * bc[(3 * 2 + 0) * g.EB + I]; bim += sSN * bc[(3 * 2 + 1) * g.EB + I]; } }
          wH = (acc)(g.omega * H);
        }
      }
      // (A - i w H - w^2 M) u = (A u_r - w2M u_r + wH u_i) + i (A u_i - w2M u_i - wH u_r)
      const acc w2M = kk * m;
      const acc yr = Aur - w2M * u_r + wH * u_i, yi = Aui - w2M * u_i - wH * u_r;
      if (MODE == 1) {   // kept in registers until every thread has read the patch, then staged for coalesced stores
        outr[b][a] = yr;
        outi[b][a] = yi;
      } else {
        const double rr_ = bre - (double)yr, ri_ = bim - (double)yi;
        r2 += rr_ * rr_ + ri_ * ri_;
        b2 += bre * bre + bim * bim;
      }
    }
  }
}

// helm_tile for a block strictly inside the mesh: every weight is a table entry, every sum an FMA chain.
template <typename inT, typename acc, int P, int MODE>
__device__ __forceinline__ void helm_tile_int(const Geo &g, const HelmC<acc> &hc, const double *__restrict__ c,
                                              const double *__restrict__ f_re, const double *__restrict__ f_im,
                                              const inT *sr, const inT *si, const acc *sk, int PW, int OW, int tx, int ty,
                                              int ex, int ey, double &r2, double &b2,
                                              acc (&outr)[MODE == 1 ? P : 1][MODE == 1 ? P : 1],
                                              acc (&outi)[MODE == 1 ? P : 1][MODE == 1 ? P : 1]) {
  const int bx = (tx + 1) * P, by = (ty + 1) * P;
  const inT *or_ = sr + by * PW + bx, *oi_ = si + by * PW + bx;   // the tile's first node
#pragma unroll
  for (int b = 0; b < P; ++b) {
#pragma unroll
    for (int a = 0; a < P; ++a) {
      const inT *rr = or_ + b * PW, *ri = oi_ + b * PW;   // row of this node, at the tile's x origin
      const inT *cr = or_ + a, *ci = oi_ + a;             // column of this node, at the tile's y origin
      acc kxr, kxi, kyr, kyi;
      if (a == 0) {
        kxr = hc.kx0[0] * (acc)rr[-P];
        kxi = hc.kx0[0] * (acc)ri[-P];
#pragma unroll
        for (int cc = 1 - P; cc <= P; ++cc) {
          kxr = hfma(hc.kx0[cc + P], (acc)rr[cc], kxr);
          kxi = hfma(hc.kx0[cc + P], (acc)ri[cc], kxi);
        }
      } else {
        kxr = hc.kx[a][0] * (acc)rr[0];
        kxi = hc.kx[a][0] * (acc)ri[0];
#pragma unroll
        for (int cc = 1; cc <= P; ++cc) {
          kxr = hfma(hc.kx[a][cc], (acc)rr[cc], kxr);
          kxi = hfma(hc.kx[a][cc], (acc)ri[cc], kxi);
        }
      }
      if (b == 0) {
        kyr = hc.ky0[0] * (acc)cr[-P * PW];
        kyi = hc.ky0[0] * (acc)ci[-P * PW];
#pragma unroll
        for (int cc = 1 - P; cc <= P; ++cc) {
          kyr = hfma(hc.ky0[cc + P], (acc)cr[cc * PW], kyr);
          kyi = hfma(hc.ky0[cc + P], (acc)ci[cc * PW], kyi);
        }
      } else {
        kyr = hc.ky[b][0] * (acc)cr[0];
        kyi = hc.ky[b][0] * (acc)ci[0];
#pragma unroll
        for (int cc = 1; cc <= P; ++cc) {
          kyr = hfma(hc.ky[b][cc], (acc)cr[cc * PW], kyr);
          kyi = hfma(hc.ky[b][cc], (acc)ci[cc * PW], kyi);
        }
      }
      const acc u_r = (acc)rr[a], u_i = (acc)ri[a];
      const acc m = hc.wm[b][a];
      acc kk;   // w^2 / c^2
      const size_t n = (size_t)(ey * P + b) * g.npx + ex * P + a;
      if (MODE == 1) kk = sk[(ty * P + b) * OW + tx * P + a];
      else { const double cj = c[n]; kk = (acc)(g.omega * g.omega / (cj * cj)); }
      const acc w2M = kk * m;
      const acc yr = hfma(-w2M, u_r, hfma(hc.wa[b], kxr, hc.wa[a] * kyr));
      const acc yi = hfma(-w2M, u_i, hfma(hc.wa[b], kxi, hc.wa[a] * kyi));
      if (MODE == 1) {
        outr[b][a] = yr;
        outi[b][a] = yi;
      } else {
        const double bre = f_re[n] * (double)m, bim = f_im ? f_im[n] * (double)m : 0.0;
        const double rr_ = bre - (double)yr, ri_ = bim - (double)yi;
        r2 += rr_ * rr_ + ri_ * ri_;
        b2 += bre * bre + bim * bim;
      }
    }
  }
}

// MODE 0: residual of (4): block partial sums of |b - (A - i w H - w^2 M) u|^2 and |b|^2 -> part (hz_residual)
// MODE 1: operator evaluation y = (A - i w H - w^2 M) u written to y (re | im planes) -- the paper's "operator time"
//         kernel, in the arithmetic `acc` of the DDM cycle it normalises
// u: re | im planes of type inT.  k2: w^2 / c^2 per node in `acc` precision (MODE 1) or NULL (then c, fp64, is read).
// The block stages the u patch ((32+1)P+1) x ((8+1)P+1) into shared memory with cp.async, one patch row per warp and
// pass (element data staged asynchronously, north_star (b): this is the one kernel of the path that streams per-element
// data from HBM); every thread then applies the two 1-D element operators to its P x P nodes from shared memory
// (3P^2 + 2P reads per plane for P^2 nodes instead of 2(2P+1) P^2), compile-time P, coefficients in the constant bank.
// Blocks strictly inside the mesh (all but the outermost ring) take a path without bounds checks, one-sided weights or
// boundary terms.  Several blocks per SM (helm_minb) overlap one block's staging with another's arithmetic.
template <typename inT, typename acc, int P, int MODE, bool EDGE>
__global__ void __launch_bounds__(kHelmBX *kHelmBY, EDGE ? (MODE == 1 && P <= 3 ? 3 : 2) : helm_minb<acc, P, MODE>())
    k_helm(Geo g, const HelmGrid hg, const __grid_constant__ HelmC<acc> hc, const double *__restrict__ c, const acc *__restrict__ k2,
           const double *__restrict__ f_re, const double *__restrict__ f_im, const double *__restrict__ bc,
           const inT *__restrict__ u, double *__restrict__ part, acc *__restrict__ y) {
  constexpr int PW = (kHelmBX + 1) * P + 1, PH = (kHelmBY + 1) * P + 1;
  constexpr int OW = kHelmBX * P, OH = kHelmBY * P;   // the block's own nodes (patch coordinates [P, P+OW) x [P, P+OH))
  constexpr int NW = kHelmBX * kHelmBY / 32;
  extern __shared__ __align__(16) unsigned char helm_raw[];
  inT *sr = reinterpret_cast<inT *>(helm_raw), *si = sr + PW * PH;
  acc *sk = reinterpret_cast<acc *>(si + PW * PH);    // MODE 1: w^2/c^2 of the own nodes, staged like the patch
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * kHelmBX + tx;
  const int wrp = tid >> 5, ln = tid & 31;
  int bxi, byi;   // block coordinates in the gx x gy grid of 32 x 8-element patches
  if (!EDGE) { bxi = 1 + blockIdx.x; byi = 1 + blockIdx.y; }
  else {          // the ring around the interior range [1, bxh) x [1, byh): bottom row, top rows, then the two sides
    int q = blockIdx.x;
    const int top = (hg.gy - hg.byh) * hg.gx, per = 1 + hg.gx - hg.bxh;
    if (q < hg.gx) { bxi = q; byi = 0; }
    else if (q - hg.gx < top) { q -= hg.gx; byi = hg.byh + q / hg.gx; bxi = q - (byi - hg.byh) * hg.gx; }
    else { q -= hg.gx + top; byi = 1 + q / per; const int j = q - (byi - 1) * per; bxi = j == 0 ? 0 : hg.bxh + j - 1; }
  }
  const int ex = bxi * kHelmBX + tx, ey = byi * kHelmBY + ty;
  const int I0 = bxi * kHelmBX * P - P, J0 = byi * kHelmBY * P - P;  // patch origin
  const long long total = (long long)g.npx * g.npy;
  // !EDGE: strictly inside -- the patch and the own nodes lie in the mesh, no own node on the boundary, every element
  // has 4 neighbours (HelmGrid holds that range)
  constexpr bool interior = !EDGE;
  if (interior) {
    // one patch row (both planes) per warp and pass, 32 consecutive elements per copy instruction, running pointers
    constexpr int NCH = (PW + 31) / 32, NIT = (PH + NW - 1) / NW;
    const inT *s_re = u + (size_t)(J0 + wrp) * g.npx + I0 + ln;
    const inT *s_im = s_re + total;
    inT *d_re = sr + wrp * PW + ln;
    const size_t sstep = (size_t)NW * g.npx;
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
      if ((it + 1) * NW <= PH || wrp + it * NW < PH) {
#pragma unroll
        for (int k = 0; k < NCH; ++k)
          if ((k + 1) * 32 <= PW || ln < PW - k * 32) {
            cp_async_elem<sizeof(inT)>(d_re + it * NW * PW + k * 32, s_re + k * 32);
            cp_async_elem<sizeof(inT)>(d_re + PW * PH + it * NW * PW + k * 32, s_im + k * 32);
          }
      }
      s_re += sstep;
      s_im += sstep;
    }
    if (MODE == 1) {   // OH = NW * P rows of OW = 32 * P values
      const acc *s_k = k2 + (size_t)(J0 + P + wrp) * g.npx + I0 + P + ln;
#pragma unroll
      for (int it = 0; it < P; ++it) {
#pragma unroll
        for (int k = 0; k < P; ++k) cp_async_elem<sizeof(acc)>(sk + (wrp + it * NW) * OW + k * 32 + ln, s_k + k * 32);
        s_k += sstep;
      }
    }
  } else {
    for (int q = tid; q < PW * PH; q += kHelmBX * kHelmBY) {
      const int px = q % PW, py = q / PW;
      const int I = I0 + px, J = J0 + py;
      const bool in = I >= 0 && I < g.npx && J >= 0 && J < g.npy;
      const size_t n = (size_t)(in ? J : 0) * g.npx + (in ? I : 0);
      cp_async_elem<sizeof(inT)>(sr + q, u + n, in);
      cp_async_elem<sizeof(inT)>(si + q, u + total + n, in);
    }
    if (MODE == 1) {
      for (int q = tid; q < OW * OH; q += kHelmBX * kHelmBY) {
        const int I = I0 + P + q % OW, J = J0 + P + q / OW;
        const bool in = I < g.npx && J < g.npy;
        cp_async_elem<sizeof(acc)>(sk + q, k2 + (in ? (size_t)J * g.npx + I : 0), in);
      }
    }
  }
  asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
  __syncthreads();
  double r2 = 0.0, b2 = 0.0;
  acc outr[MODE == 1 ? P : 1][MODE == 1 ? P : 1], outi[MODE == 1 ? P : 1][MODE == 1 ? P : 1];
  if (MODE == 1) {
#pragma unroll
    for (int b = 0; b < P; ++b)
#pragma unroll
      for (int a = 0; a < P; ++a) outr[b][a] = outi[b][a] = acc(0);
  }
  if constexpr (interior) helm_tile_int<inT, acc, P, MODE>(g, hc, c, f_re, f_im, sr, si, sk, PW, OW, tx, ty, ex, ey, r2, b2, outr, outi);
  else if (ex <= g.nx && ey <= g.ny)
    helm_tile<inT, acc, P, MODE>(g, hc, c, f_re, f_im, bc, sr, si, sk, PW, OW, tx, ty, ex, ey, r2, b2, outr, outi);
  if (MODE == 1) {
    // y of the own nodes goes through shared memory (the patch is dead now) so that the global stores are whole rows
    acc *yo_r = reinterpret_cast<acc *>(helm_raw), *yo_i = yo_r + OW * OH;
    __syncthreads();
#pragma unroll
    for (int b = 0; b < P; ++b)
#pragma unroll
      for (int a = 0; a < P; ++a) {
        yo_r[(ty * P + b) * OW + tx * P + a] = outr[b][a];
        yo_i[(ty * P + b) * OW + tx * P + a] = outi[b][a];
      }
    __syncthreads();
    if (interior) {   // one output row (both planes) per warp and pass
      acc *d_r = y + (size_t)(J0 + P + wrp) * g.npx + I0 + P + ln;
      acc *d_i = d_r + total;
      const size_t sstep = (size_t)NW * g.npx;
#pragma unroll
      for (int it = 0; it < P; ++it) {
        const acc *srow = yo_r + (wrp + it * NW) * OW + ln;
#pragma unroll
        for (int k = 0; k < P; ++k) {
          d_r[k * 32] = srow[k * 32];
          d_i[k * 32] = srow[OW * OH + k * 32];
        }
        d_r += sstep;
        d_i += sstep;
      }
    } else {
      for (int q = tid; q < OW * OH; q += kHelmBX * kHelmBY) {
        const int I = I0 + P + q % OW, J = J0 + P + q / OW;
        if (I < g.npx && J < g.npy) {
          const size_t n = (size_t)J * g.npx + I;
          y[n] = yo_r[q];
          y[total + n] = yo_i[q];
        }
      }
    }
  }
  if (MODE == 0) {
    __shared__ double red[2][32];
    for (int o = 16; o > 0; o >>= 1) {
      r2 += __shfl_down_sync(0xffffffffu, r2, o);
      b2 += __shfl_down_sync(0xffffffffu, b2, o);
    }
    const int w = tid >> 5;
    if (ln == 0) { red[0][w] = r2; red[1][w] = b2; }
    __syncthreads();
    if (w == 0) {
      r2 = ln < NW ? red[0][ln] : 0.0;
      b2 = ln < NW ? red[1][ln] : 0.0;
      for (int o = 16; o > 0; o >>= 1) {
        r2 += __shfl_down_sync(0xffffffffu, r2, o);
        b2 += __shfl_down_sync(0xffffffffu, b2, o);
      }
      const size_t bid = (size_t)byi * hg.gx + bxi;
      if (ln == 0) { part[2 * bid] = r2; part[2 * bid + 1] = b2; }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// k_helm_tma: the patches strictly inside the mesh (all but the outermost ring; HelmGrid) where a patch row is long
// enough for the TMA unit to pay off (fp64, P >= 3: rows of 800 bytes and more).  Same arithmetic as helm_tile_int, but
// the patch is staged by ONE 1-D bulk copy (cp.async.bulk, completion bytes on an mbarrier) per patch row and plane,
// issued by the lanes of warp 0: 80 copy instructions per block at P = 3 instead of 31 cp.async per THREAD.  A bulk copy
// needs 16-byte aligned addresses and sizes, and a patch row starts at an arbitrary element (rows are npx = nx P + 1
// elements long; a 2-D tensor map is ruled out for the same reason, its row stride must be a multiple of 16 bytes): each
// copy fetches the aligned superset of its row, so row r's data begin `shift(r)` elements (0 .. 16/size - 1) into its
// shared-memory row, and the threads carry one base pointer per patch row they read.  Measured on the config-5 mesh
// (fp64 operator, P = 3): 0.275 ms against 0.316 ms with 8-byte cp.async; in fp32 the 400-byte copies of a block
// serialise in the TMA unit (half of the warp time waits on the mbarrier): 0.207 ms against 0.191 ms, so fp32 and
// P <= 2 keep the cp.async kernel.  (Also tried: 16-byte cp.async of the same aligned supersets: no faster than 4-byte.)
// ---------------------------------------------------------------------------------------------
template <int BYTES> __host__ __device__ constexpr int helm_pitch(int w) { return (w + 2 * (16 / BYTES) - 2) / (16 / BYTES) * (16 / BYTES); }
inline size_t helm_tma_smem(int P, size_t elem_in, size_t elem_k2) {
  const int PW = (kHelmBX + 1) * P + 1, PH = (kHelmBY + 1) * P + 1, OW = kHelmBX * P, OH = kHelmBY * P;
  const int ei = (int)(16 / elem_in);
  const size_t pws = (size_t)(PW + 2 * ei - 2) / ei * ei;
  size_t b = 16 + 2 * (size_t)PH * pws * elem_in;   // 16 bytes: the mbarrier
  if (elem_k2) { const int ea = (int)(16 / elem_k2); b += (size_t)OH * ((size_t)(OW + 2 * ea - 2) / ea * ea) * elem_k2; }
  return b;
}
__device__ __forceinline__ void helm_bulk_row(unsigned dst, const void *src, unsigned bytes, unsigned mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
               "r"(bytes), "r"(mbar)
               : "memory");
}

template <typename inT, typename acc, int P, int MODE>
__global__ void __launch_bounds__(kHelmBX *kHelmBY, helm_minb<acc, P, MODE, true>())
    k_helm_tma(Geo g, const HelmGrid hg, const __grid_constant__ HelmC<acc> hc, const double *__restrict__ c,
               const acc *__restrict__ k2, const double *__restrict__ f_re, const double *__restrict__ f_im,
               const inT *__restrict__ u, double *__restrict__ part, acc *__restrict__ y) {
  constexpr int PW = (kHelmBX + 1) * P + 1, PH = (kHelmBY + 1) * P + 1;
  constexpr int OW = kHelmBX * P, OH = kHelmBY * P;
  constexpr int NW = kHelmBX * kHelmBY / 32;
  constexpr int EI = 16 / (int)sizeof(inT), EA = 16 / (int)sizeof(acc);
  constexpr int PWS = helm_pitch<sizeof(inT)>(PW), OWS = helm_pitch<sizeof(acc)>(OW);
  constexpr int NR = 2 * PH + (MODE == 1 ? OH : 0);   // bulk copies per block
  extern __shared__ __align__(16) unsigned char helm_raw[];
  inT *sr = reinterpret_cast<inT *>(helm_raw + 16), *si = sr + PH * PWS;
  acc *sk = reinterpret_cast<acc *>(si + PH * PWS);
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * kHelmBX + tx;
  const int wrp = tid >> 5, ln = tid & 31;
  const int bxi = 1 + blockIdx.x, byi = 1 + blockIdx.y;
  const int ex = bxi * kHelmBX + tx, ey = byi * kHelmBY + ty;
  const int I0 = bxi * kHelmBX * P - P, J0 = byi * kHelmBY * P - P;  // patch origin
  const long long total = (long long)g.npx * g.npy;
  // element index of the patch origin, modulo the elements per 16 bytes (unsigned wrap-around keeps the residue)
  const unsigned ua = (unsigned)(reinterpret_cast<size_t>(u) / sizeof(inT)), ka = (unsigned)(reinterpret_cast<size_t>(k2) / sizeof(acc));
  const unsigned npxu = (unsigned)g.npx;
  const unsigned o_re = ua + (unsigned)J0 * npxu + (unsigned)I0, o_im = o_re + (unsigned)total;
  const unsigned o_k = ka + (unsigned)(J0 + P) * npxu + (unsigned)(I0 + P);
  const unsigned mbar = (unsigned)__cvta_generic_to_shared(helm_raw);
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 32;" ::"r"(mbar) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (wrp == 0) {   // lane l issues the copies of rows l, l + 32, ...; it first announces their bytes on the mbarrier
    unsigned bytes = 0;
#pragma unroll
    for (int r0 = 0; r0 < NR; r0 += 32) {
      const int r = r0 + ln;
      if (r < 2 * PH) {
        const int pl = r >= PH ? 1 : 0, pr = r - pl * PH;
        const unsigned sh = ((pl ? o_im : o_re) + (unsigned)pr * npxu) & (EI - 1);
        bytes += (sh + PW + EI - 1) / EI * 16u;
      } else if (r < NR) {
        const unsigned sh = (o_k + (unsigned)(r - 2 * PH) * npxu) & (EA - 1);
        bytes += (sh + OW + EA - 1) / EA * 16u;
      }
    }
    asm volatile("{ .reg .b64 st; mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1; }" ::"r"(mbar), "r"(bytes) : "memory");
#pragma unroll
    for (int r0 = 0; r0 < NR; r0 += 32) {
      const int r = r0 + ln;
      if (r < 2 * PH) {
        const int pl = r >= PH ? 1 : 0, pr = r - pl * PH;
        const unsigned sh = ((pl ? o_im : o_re) + (unsigned)pr * npxu) & (EI - 1);
        const inT *src = u + (pl ? total : 0) + (size_t)(J0 + pr) * g.npx + I0 - sh;
        helm_bulk_row((unsigned)__cvta_generic_to_shared((pl ? si : sr) + pr * PWS), src, (sh + PW + EI - 1) / EI * 16u, mbar);
      } else if (r < NR) {
        const int kr = r - 2 * PH;
        const unsigned sh = (o_k + (unsigned)kr * npxu) & (EA - 1);
        const acc *src = k2 + (size_t)(J0 + P + kr) * g.npx + I0 + P - sh;
        helm_bulk_row((unsigned)__cvta_generic_to_shared(sk + kr * OWS), src, (sh + OW + EA - 1) / EA * 16u, mbar);
      }
    }
  }
  // base pointers of the 3P patch rows this thread reads (rows ty P .. ty P + 3P - 1), at its tile's x origin
  const inT *rowr[3 * P], *rowi[3 * P];
  const acc *skr[MODE == 1 ? P : 1];
#pragma unroll
  for (int k = 0; k < 3 * P; ++k) {
    const int pr = ty * P + k;
    rowr[k] = sr + pr * PWS + ((o_re + (unsigned)pr * npxu) & (EI - 1)) + (tx + 1) * P;
    rowi[k] = si + pr * PWS + ((o_im + (unsigned)pr * npxu) & (EI - 1)) + (tx + 1) * P;
  }
  if (MODE == 1) {
#pragma unroll
    for (int b = 0; b < P; ++b) skr[b] = sk + (ty * P + b) * OWS + ((o_k + (unsigned)(ty * P + b) * npxu) & (EA - 1)) + tx * P;
  }
  {   // all bytes have landed (single phase: parity 0)
    asm volatile(
        "{\n\t.reg .pred P1;\n\t"
        "HZ_HW_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], 0;\n\t"
        "@P1 bra HZ_HD_%=;\n\t"
        "bra HZ_HW_%=;\n\t"
        "HZ_HD_%=:\n\t}" ::"r"(mbar) : "memory");
  }
  double r2 = 0.0, b2 = 0.0;
  acc outr[MODE == 1 ? P : 1][MODE == 1 ? P : 1], outi[MODE == 1 ? P : 1][MODE == 1 ? P : 1];
#pragma unroll
  for (int b = 0; b < P; ++b) {
#pragma unroll
    for (int a = 0; a < P; ++a) {
      const inT *rr = rowr[P + b], *ri = rowi[P + b];
      acc kxr, kxi, kyr, kyi;
      if (a == 0) {
        kxr = hc.kx0[0] * (acc)rr[-P];
        kxi = hc.kx0[0] * (acc)ri[-P];
#pragma unroll
        for (int cc = 1 - P; cc <= P; ++cc) {
          kxr = hfma(hc.kx0[cc + P], (acc)rr[cc], kxr);
          kxi = hfma(hc.kx0[cc + P], (acc)ri[cc], kxi);
        }
      } else {
        kxr = hc.kx[a][0] * (acc)rr[0];
        kxi = hc.kx[a][0] * (acc)ri[0];
#pragma unroll
        for (int cc = 1; cc <= P; ++cc) {
          kxr = hfma(hc.kx[a][cc], (acc)rr[cc], kxr);
          kxi = hfma(hc.kx[a][cc], (acc)ri[cc], kxi);
        }
      }
      if (b == 0) {
        kyr = hc.ky0[0] * (acc)rowr[0][a];
        kyi = hc.ky0[0] * (acc)rowi[0][a];
#pragma unroll
        for (int cc = 1 - P; cc <= P; ++cc) {
          kyr = hfma(hc.ky0[cc + P], (acc)rowr[P + cc][a], kyr);
          kyi = hfma(hc.ky0[cc + P], (acc)rowi[P + cc][a], kyi);
        }
      } else {
        kyr = hc.ky[b][0] * (acc)rowr[P][a];
        kyi = hc.ky[b][0] * (acc)rowi[P][a];
#pragma unroll
        for (int cc = 1; cc <= P; ++cc) {
          kyr = hfma(hc.ky[b][cc], (acc)rowr[P + cc][a], kyr);
          kyi = hfma(hc.ky[b][cc], (acc)rowi[P + cc][a], kyi);
        }
      }
      const acc u_r = (acc)rr[a], u_i = (acc)ri[a];
      const acc m = hc.wm[b][a];
      acc kk;   // w^2 / c^2
      const size_t n = (size_t)(ey * P + b) * g.npx + ex * P + a;
      if (MODE == 1) kk = skr[b][a];
      else { const double cj = c[n]; kk = (acc)(g.omega * g.omega / (cj * cj)); }
      const acc w2M = kk * m;
      const acc yr = hfma(-w2M, u_r, hfma(hc.wa[b], kxr, hc.wa[a] * kyr));
      const acc yi = hfma(-w2M, u_i, hfma(hc.wa[b], kxi, hc.wa[a] * kyi));
      if (MODE == 1) {
        outr[b][a] = yr;
        outi[b][a] = yi;
      } else {
        const double bre = f_re[n] * (double)m, bim = f_im ? f_im[n] * (double)m : 0.0;
        const double rr_ = bre - (double)yr, ri_ = bim - (double)yi;
        r2 += rr_ * rr_ + ri_ * ri_;
        b2 += bre * bre + bim * bim;
      }
    }
  }
  if (MODE == 1) {
    // y of the own nodes goes through shared memory (the patch is dead now) so that the global stores are whole rows
    acc *yo_r = reinterpret_cast<acc *>(helm_raw + 16), *yo_i = yo_r + OW * OH;
    __syncthreads();
#pragma unroll
    for (int b = 0; b < P; ++b)
#pragma unroll
      for (int a = 0; a < P; ++a) {
        yo_r[(ty * P + b) * OW + tx * P + a] = outr[b][a];
        yo_i[(ty * P + b) * OW + tx * P + a] = outi[b][a];
      }
    __syncthreads();
    acc *d_r = y + (size_t)(J0 + P + wrp) * g.npx + I0 + P + ln;   // one output row (both planes) per warp and pass
    acc *d_i = d_r + total;
    const size_t sstep = (size_t)NW * g.npx;
#pragma unroll
    for (int it = 0; it < P; ++it) {
      const acc *srow = yo_r + (wrp + it * NW) * OW + ln;
#pragma unroll
      for (int k = 0; k < P; ++k) {
        d_r[k * 32] = srow[k * 32];
        d_i[k * 32] = srow[OW * OH + k * 32];
      }
      d_r += sstep;
      d_i += sstep;
    }
  }
  if (MODE == 0) {
    __shared__ double red[2][32];
    for (int o = 16; o > 0; o >>= 1) {
      r2 += __shfl_down_sync(0xffffffffu, r2, o);
      b2 += __shfl_down_sync(0xffffffffu, b2, o);
    }
    if (ln == 0) { red[0][wrp] = r2; red[1][wrp] = b2; }
    __syncthreads();
    if (wrp == 0) {
      r2 = ln < NW ? red[0][ln] : 0.0;
      b2 = ln < NW ? red[1][ln] : 0.0;
      for (int o = 16; o > 0; o >>= 1) {
        r2 += __shfl_down_sync(0xffffffffu, r2, o);
        b2 += __shfl_down_sync(0xffffffffu, b2, o);
      }
      const size_t bid = (size_t)byi * hg.gx + bxi;
      if (ln == 0) { part[2 * bid] = r2; part[2 * bid + 1] = b2; }
    }
  }
}

// k2[n] = w^2 / c_n^2 in the operator's precision (built once per context and precision)
template <typename acc>
__global__ void k_helm_k2(long long n, double omega, const double *__restrict__ c, acc *__restrict__ k2) {
  const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (q < n) k2[q] = (acc)(omega * omega / (c[q] * c[q]));
}

static __global__ void k_reduce2(const double *__restrict__ part, int n, double *__restrict__ out) {
  __shared__ double red[2][32];
  double a = 0.0, b = 0.0;
  for (int q = threadIdx.x; q < n; q += blockDim.x) { a += part[2 * (size_t)q]; b += part[2 * (size_t)q + 1]; }
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_down_sync(0xffffffffu, a, o);
    b += __shfl_down_sync(0xffffffffu, b, o);
  }
  const int w = threadIdx.x >> 5, ln = threadIdx.x & 31;
  if (ln == 0) { red[0][w] = a; red[1][w] = b; }
  __syncthreads();
  if (w == 0) {
    const int nw = blockDim.x >> 5;
    a = ln < nw ? red[0][ln] : 0.0;
    b = ln < nw ? red[1][ln] : 0.0;
    for (int o = 16; o > 0; o >>= 1) {
      a += __shfl_down_sync(0xffffffffu, a, o);
      b += __shfl_down_sync(0xffffffffu, b, o);
    }
    if (ln == 0) { out[0] = a; out[1] = b; }
  }
}

// ---------------------------------------------------------------------------------------------
// State export / import in canonical fp64 layout (parity tests, random-lambda benchmark)
// ---------------------------------------------------------------------------------------------
template <typename real>
__global__ void k_state_get(Layout lay, int L, const real *__restrict__ u_sub, double *__restrict__ out) {
  const int N = lay.lnx * lay.lny;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= (long long)L * 2 * N) return;
  const int q = (int)(gid % N), c = (int)((gid / N) % 2), l = (int)(gid / (2 * N));
  out[gid] = (double)u_sub[(size_t)l * 2 * lay.NS + (size_t)c * lay.NS + lay.slot(q % lay.lnx, q / lay.lnx)];
}
template <typename real>
__global__ void k_state_set(Layout lay, int L, real *__restrict__ u_sub, const double *__restrict__ in) {
  const int N = lay.lnx * lay.lny;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= (long long)L * 2 * N) return;
  const int q = (int)(gid % N), c = (int)((gid / N) % 2), l = (int)(gid / (2 * N));
  u_sub[(size_t)l * 2 * lay.NS + (size_t)c * lay.NS + lay.slot(q % lay.lnx, q / lay.lnx)] = (real)in[gid];
}
template <typename A, typename B>
__global__ void k_convert(long long n, const A *__restrict__ in, B *__restrict__ out) {
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid < n) out[gid] = (B)in[gid];
}

// ---------------------------------------------------------------------------------------------
// State transfer of the mixed-precision defect correction (hz_ddm_solve_mixed; reading R27).
// The joint state (lambda | u_l) of the fp64 context `hi` and of the fp32 context `lo` share the lambda layout
// [L][4][2][E] but not the node slot map (each precision picks its own thread tile).  One thread per canonical
// element: q < nlam is a lambda entry, q >= nlam is (l, re/im, node).
//   k_mixed_defect :  D = hi_new - hi_old (fp64)  ->  lo_state = lo_D = (float) D          (delta_1 = D)
//   k_mixed_update :  hi_state = hi_old + (double) lo_state                                  (X <- X + delta_m)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void mixed_index(long long q, long long nlam, Layout lh, Layout ll, size_t *ih, size_t *il) {
  if (q < nlam) { *ih = (size_t)q; *il = (size_t)q; return; }
  const long long r = q - nlam;
  const int N = lh.lnx * lh.lny;
  const int node = (int)(r % N), c = (int)((r / N) % 2);
  const long long l = r / (2 * N);
  const int i = node % lh.lnx, j = node / lh.lnx;
  *ih = (size_t)nlam + (size_t)l * 2 * lh.NS + (size_t)c * lh.NS + lh.slot(i, j);
  *il = (size_t)nlam + (size_t)l * 2 * ll.NS + (size_t)c * ll.NS + ll.slot(i, j);
}
static __global__ void k_mixed_defect(long long total, long long nlam, Layout lh, Layout ll, const double *__restrict__ hi_new,
                                      const double *__restrict__ hi_old, float *__restrict__ lo_state, float *__restrict__ lo_D) {
  const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= total) return;
  size_t ih, il;
  mixed_index(q, nlam, lh, ll, &ih, &il);
  const float d = (float)(hi_new[ih] - hi_old[ih]);
  lo_state[il] = d;
  lo_D[il] = d;
}
static __global__ void k_mixed_update(long long total, long long nlam, Layout lh, Layout ll, double *__restrict__ hi_state,
                                      const double *__restrict__ hi_old, const float *__restrict__ lo_state) {
  const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= total) return;
  size_t ih, il;
  mixed_index(q, nlam, lh, ll, &ih, &il);
  hi_state[ih] = hi_old[ih] + (double)lo_state[il];
}
// x += y over the whole flat state
static __global__ void k_add_f32(long long n, float *__restrict__ x, const float *__restrict__ y) {
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) x[e] += y[e];
}

}  // namespace hz

namespace hz {

// ---------------------------------------------------------------------------------------------
// Vector kernels of the Krylov-accelerated outer iteration.  The joint
// state x = (lambda | u_l) is one flat array of `real`; Krylov vectors V_i are rows of a [nv][n] array.
// Inner products are accumulated in fp64 and reduced in a fixed order (deterministic).
// ---------------------------------------------------------------------------------------------
template <typename real>
__global__ void k_dots(long long n, const real *__restrict__ V, long long ld, const real *__restrict__ w,
                       double *__restrict__ part) {
  // grid (nblk, nv): block (bx, i) -> partial sum of V_i . w over its grid-stride slice
  __shared__ double red[32];
  const real *v = V + (size_t)blockIdx.y * ld;
  double s = 0.0;
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x)
    s += (double)v[e] * (double)w[e];
  for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
  const int wp = threadIdx.x >> 5, ln = threadIdx.x & 31;
  if (ln == 0) red[wp] = s;
  __syncthreads();
  if (wp == 0) {
    s = ln < (blockDim.x >> 5) ? red[ln] : 0.0;
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if (ln == 0) part[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = s;
  }
}

static __global__ void k_reduce_rows(const double *__restrict__ part, int nblk, double *__restrict__ out) {
  // one block per row: out[row] = sum of part[row][0..nblk)
  __shared__ double red[32];
  double s = 0.0;
  for (int q = threadIdx.x; q < nblk; q += blockDim.x) s += part[(size_t)blockIdx.x * nblk + q];
  for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
  const int wp = threadIdx.x >> 5, ln = threadIdx.x & 31;
  if (ln == 0) red[wp] = s;
  __syncthreads();
  if (wp == 0) {
    s = ln < (blockDim.x >> 5) ? red[ln] : 0.0;
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if (ln == 0) out[blockIdx.x] = s;
  }
}

// w[e] += sum_i coef[i] V_i[e]   (coef on the device, already signed)
template <typename real>
__global__ void k_axpys(long long n, real *__restrict__ w, const real *__restrict__ V, long long ld, int nv,
                        const double *__restrict__ coef) {
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
    double s = (double)w[e];
    for (int i = 0; i < nv; ++i) s += coef[i] * (double)V[(size_t)i * ld + e];
    w[e] = (real)s;
  }
}

// out = a*x + b*y + c*z  (z may be NULL)
template <typename real>
__global__ void k_lincomb(long long n, real *__restrict__ out, double a, const real *__restrict__ x, double b,
                          const real *__restrict__ y, double c, const real *__restrict__ z) {
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
    double s = a * (double)x[e] + b * (double)y[e];
    if (z) s += c * (double)z[e];
    out[e] = (real)s;
  }
}

}  // namespace hz
