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
template <typename real>
__global__ void k_build(Geo g, Layout lay, const double *__restrict__ c, const double *__restrict__ f_re,
                        const double *__restrict__ f_im, const double *__restrict__ bc, const double *__restrict__ wxl,
                        const double *__restrict__ wyl, real *gamma, real *alpha, real *bbf_re, real *bbf_im,
                        real *k2edge, real *bs, int only_source) {
  const int N = lay.lnx * lay.lny;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long total = (long long)g.sx * g.sy * N;
  if (gid >= total) return;
  const int l = (int)(gid / N), q = (int)(gid - (long long)l * N);
  const int i = q % lay.lnx, j = q / lay.lnx;
  const int six = l % g.sx, siy = l / g.sx;
  const int I = six * g.ex * g.p + i, J = siy * g.ey * g.p + j;
  const size_t gn = (size_t)J * g.npx + I;
  const double cj = c[gn];
  const double m = 0.25 * g.hx * g.hy * wxl[i] * wyl[j];  // local lumped mass (geometric)
  const double M = m / (cj * cj);
  // impedance weight on the WHOLE subdomain boundary: interfaces carry the same operator as the
  // outer boundary
  const bool onW = i == 0, onE = i == lay.lnx - 1, onS = j == 0, onN = j == lay.lny - 1;
  const double sWE = 0.5 * g.hy * wyl[j], sSN = 0.5 * g.hx * wxl[i];
  double H = 0.0;
  if (onW) H += sWE / cj;
  if (onE) H += sWE / cj;
  if (onS) H += sSN / cj;
  if (onN) H += sSN / cj;
  const double den = M + g.theta * H;
  const double beta = g.sigma / den;
  // load: f(x_j) m_j (+ the outer-boundary datum lambda of eq. (1b) on physical sides)
  double bre = f_re[gn] * m, bim = f_im ? f_im[gn] * m : 0.0;
  if (bc) {
    if (onW && six == 0) { bre += sWE * bc[(0 * 2 + 0) * g.EB + J]; bim += sWE * bc[(0 * 2 + 1) * g.EB + J]; }
    if (onE && six == g.sx - 1) { bre += sWE * bc[(1 * 2 + 0) * g.EB + J]; bim += sWE * bc[(1 * 2 + 1) * g.EB + J]; }
    if (onS && siy == 0) { bre += sSN * bc[(2 * 2 + 0) * g.EB + I]; bim += sSN * bc[(2 * 2 + 1) * g.EB + I]; }
    if (onN && siy == g.sy - 1) { bre += sSN * bc[(3 * 2 + 0) * g.EB + I]; bim += sSN * bc[(3 * 2 + 1) * g.EB + I]; }
  }
  const size_t o = (size_t)l * lay.NS + lay.slot(i, j);
  bbf_re[o] = (real)(beta * bre);
  if (bbf_im) bbf_im[o] = (real)(beta * bim);
  if (only_source) return;
  gamma[o] = (real)(beta * m);
  alpha[o] = (real)((M - g.theta * H) / den);
  const size_t eb = (size_t)l * 4 * g.E;
  const double k2 = 2.0 * g.omega / cj;
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
template <typename real, typename outT>
__global__ void k_gather(Geo g, Layout lay, const real *__restrict__ u_sub, outT *__restrict__ u_out) {
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long total = (long long)g.npx * g.npy;
  if (gid >= total) return;
  const int I = (int)(gid % g.npx), J = (int)(gid / g.npx);
  // the subdomain column (row) of the element that has this node as a lower node, and the one before at a shared node
  const int ehx = I / g.p > g.nx - 1 ? g.nx - 1 : I / g.p, ehy = J / g.p > g.ny - 1 ? g.ny - 1 : J / g.p;
  const int ix1 = sub_of_elem(g.exq, g.exr, ehx), iy1 = sub_of_elem(g.eyq, g.eyr, ehy);
  const int ix0 = (I == sub_off(g.exq, g.exr, ix1) * g.p && ix1 > 0) ? ix1 - 1 : ix1;
  const int iy0 = (J == sub_off(g.eyq, g.eyr, iy1) * g.p && iy1 > 0) ? iy1 - 1 : iy1;
  double sr = 0.0, si = 0.0;
  int cnt = 0;
  for (int iy = iy0; iy <= iy1; ++iy)
    for (int ix = ix0; ix <= ix1; ++ix) {
      const int l = iy * g.sx + ix;
      const int s = lay.slot(I - sub_off(g.exq, g.exr, ix) * g.p, J - sub_off(g.eyq, g.eyr, iy) * g.p);
      sr += (double)u_sub[(size_t)l * 2 * lay.NS + s];
      si += (double)u_sub[(size_t)l * 2 * lay.NS + lay.NS + s];
      ++cnt;
    }
  u_out[gid] = (outT)(sr / cnt);
  u_out[total + gid] = (outT)(si / cnt);
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

// Launch shape of k_helm: a block of HB_X x HB_Y threads, one thread per ELEMENT (its P x P lower-left nodes, as in the
// sweep kernels; the phantom elements nx / ny own the last node column / row), and its shared-memory patch.
constexpr int kHelmBX = 32, kHelmBY = 8;
// shared memory: the u patch (re, im) of the input type; MODE 1 adds the w^2/c^2 values of the block's own nodes
inline size_t helm_smem(int P, size_t elem_in, size_t elem_k2) {
  return 2 * (size_t)((kHelmBX + 1) * P + 1) * ((kHelmBY + 1) * P + 1) * elem_in + (size_t)kHelmBX * P * kHelmBY * P * elem_k2;
}

// asynchronous global -> shared copy of one 4- or 8-byte element (cp.async, no register staging: the whole patch of a
// block is in flight at once); pred = false writes zeros (src-size 0)
template <int BYTES>
__device__ __forceinline__ void cp_async_elem(void *dst_smem, const void *src, bool pred) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
  const int sz = pred ? BYTES : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2, %3;" ::"r"(d), "l"(src), "n"(BYTES), "r"(sz) : "memory");
}

// MODE 0: residual of (4): block partial sums of |b - (A - i w H - w^2 M) u|^2 and |b|^2 -> part (hz_residual)
// MODE 1: operator evaluation y = (A - i w H - w^2 M) u written to y (re | im planes) -- the paper's "operator time"
//         kernel, in the arithmetic `acc` of the DDM cycle it normalises
// u: re | im planes of type inT.  k2: w^2 / c^2 per node in `acc` precision (MODE 1) or NULL (then c, fp64, is read).
// The block stages the u patch ((32+1)P+1) x ((8+1)P+1) into shared memory with cp.async (element data staged
// asynchronously, north_star (b): this is the one kernel of the path that streams per-element data from HBM); every
// thread then applies the two 1-D element operators to its P x P nodes from shared memory (3P^2 + 2P reads per plane
// for P^2 nodes instead of 2(2P+1) P^2), compile-time P, coefficients in the constant bank.
template <typename inT, typename acc, int P, int MODE>
__global__ void __launch_bounds__(kHelmBX *kHelmBY, 2) k_helm(Geo g, Ref1D ref, const double *__restrict__ c,
                                                               const acc *__restrict__ k2, const double *__restrict__ f_re,
                                                               const double *__restrict__ f_im, const double *__restrict__ bc,
                                                               const inT *__restrict__ u, double *__restrict__ part,
                                                               acc *__restrict__ y) {
  constexpr int PW = (kHelmBX + 1) * P + 1, PH = (kHelmBY + 1) * P + 1;
  constexpr int OW = kHelmBX * P, OH = kHelmBY * P;   // the block's own nodes (patch coordinates [P, P+OW) x [P, P+OH))
  extern __shared__ __align__(16) unsigned char helm_raw[];
  inT *sr = reinterpret_cast<inT *>(helm_raw), *si = sr + PW * PH;
  acc *sk = reinterpret_cast<acc *>(si + PW * PH);    // MODE 1: w^2/c^2 of the own nodes, staged like the patch
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * kHelmBX + tx;
  const int ex = blockIdx.x * kHelmBX + tx, ey = blockIdx.y * kHelmBY + ty;
  const int I0 = blockIdx.x * kHelmBX * P - P, J0 = blockIdx.y * kHelmBY * P - P;  // patch origin
  const long long total = (long long)g.npx * g.npy;
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
  if (ex <= g.nx && ey <= g.ny) {
    const bool hasL = ex > 0, hasR = ex < g.nx, hasD = ey > 0, hasU = ey < g.ny;
    const acc ax_ = (acc)(g.hy / g.hx), ay_ = (acc)(g.hx / g.hy);
    const acc mh = (acc)(0.25 * g.hx * g.hy);
    // patch coordinates of the tile's first node
    const int bx = (tx + 1) * P, by = (ty + 1) * P;
#pragma unroll
    for (int b = 0; b < P; ++b) {
      if (b > 0 && !hasU) break;
      const acc wy = b == 0 ? (acc)((hasD ? ref.w[P] : 0.0) + (hasU ? ref.w[0] : 0.0)) : (acc)ref.w[b];
#pragma unroll
      for (int a = 0; a < P; ++a) {
        if (a > 0 && !hasR) break;
        const acc wx = a == 0 ? (acc)((hasL ? ref.w[P] : 0.0) + (hasR ? ref.w[0] : 0.0)) : (acc)ref.w[a];
        const inT *rr = sr + (by + b) * PW + bx, *ri = si + (by + b) * PW + bx;   // row of this node, at the tile's x origin
        const inT *cr = sr + by * PW + bx + a, *ci = si + by * PW + bx + a;       // column of this node, at the tile's y origin
        acc kxr = 0, kxi = 0, kyr = 0, kyi = 0;
        if (a == 0) {   // node shared by the element on the left (its row P) and this one (row 0), where they exist
#pragma unroll
          for (int cc = 0; cc <= P; ++cc) {
            const acc kl = hasL ? (acc)ref.K[P][cc] : acc(0), kr = hasR ? (acc)ref.K[0][cc] : acc(0);
            kxr += kl * (acc)rr[cc - P] + kr * (acc)rr[cc];
            kxi += kl * (acc)ri[cc - P] + kr * (acc)ri[cc];
          }
        } else {
#pragma unroll
          for (int cc = 0; cc <= P; ++cc) {
            kxr += (acc)ref.K[a][cc] * (acc)rr[cc];
            kxi += (acc)ref.K[a][cc] * (acc)ri[cc];
          }
        }
        if (b == 0) {
#pragma unroll
          for (int cc = 0; cc <= P; ++cc) {
            const acc kd = hasD ? (acc)ref.K[P][cc] : acc(0), ku = hasU ? (acc)ref.K[0][cc] : acc(0);
            kyr += kd * (acc)cr[(cc - P) * PW] + ku * (acc)cr[cc * PW];
            kyi += kd * (acc)ci[(cc - P) * PW] + ku * (acc)ci[cc * PW];
          }
        } else {
#pragma unroll
          for (int cc = 0; cc <= P; ++cc) {
            kyr += (acc)ref.K[b][cc] * (acc)cr[cc * PW];
            kyi += (acc)ref.K[b][cc] * (acc)ci[cc * PW];
          }
        }
        const int I = ex * P + a, J = ey * P + b;
        const size_t n = (size_t)J * g.npx + I;
        const acc u_r = (acc)rr[a], u_i = (acc)ri[a];
        const acc Aur = ax_ * wy * kxr + ay_ * wx * kyr, Aui = ax_ * wy * kxi + ay_ * wx * kyi;
        const acc m = mh * wx * wy;
        acc kk;   // w^2 / c^2
        double cj = 0.0;
        if (MODE == 1) kk = sk[(ty * P + b) * OW + tx * P + a];
        else { cj = c[n]; kk = (acc)(g.omega * g.omega / (cj * cj)); }
        const bool onb = I == 0 || I == g.npx - 1 || J == 0 || J == g.npy - 1;
        acc wH = 0;
        double bre = 0.0, bim = 0.0;
        if (MODE == 0) { bre = f_re[n] * (double)m; bim = f_im ? f_im[n] * (double)m : 0.0; }
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
    for (int q = tid; q < OW * OH; q += kHelmBX * kHelmBY) {
      const int I = I0 + P + q % OW, J = J0 + P + q / OW;
      if (I < g.npx && J < g.npy) {
        const size_t n = (size_t)J * g.npx + I;
        y[n] = yo_r[q];
        y[total + n] = yo_i[q];
      }
    }
  }
  if (MODE == 0) {
    __shared__ double red[2][32];
    for (int o = 16; o > 0; o >>= 1) {
      r2 += __shfl_down_sync(0xffffffffu, r2, o);
      b2 += __shfl_down_sync(0xffffffffu, b2, o);
    }
    const int w = tid >> 5, ln = tid & 31;
    if (ln == 0) { red[0][w] = r2; red[1][w] = b2; }
    __syncthreads();
    if (w == 0) {
      constexpr int nw = kHelmBX * kHelmBY / 32;
      r2 = ln < nw ? red[0][ln] : 0.0;
      b2 = ln < nw ? red[1][ln] : 0.0;
      for (int o = 16; o > 0; o >>= 1) {
        r2 += __shfl_down_sync(0xffffffffu, r2, o);
        b2 += __shfl_down_sync(0xffffffffu, b2, o);
      }
      const size_t bid = (size_t)blockIdx.y * gridDim.x + blockIdx.x;
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
