// hz_minres.cuh — block-level MINRES subdomain solve, the paper's comparator.
// Same one-block-per-subdomain, one-DOF-per-thread layout as k_sweep_dof: every subdomain's real symmetric
// indefinite block system (5)
//     [[A - w^2 M, w H], [w H, w^2 M - A]] [Re u; Im u] = [Re b; -Im b]
// is solved by unpreconditioned MINRES (Paige & Saunders; Lanczos + Givens, "five vectors and two inner
// products per iteration") until the recurrence's residual norm <= tol ||rhs|| or
// max_iters.  Each thread holds the (re, im) entries of its node for x, v_{j-1}, v_j, w_{j-1}, w_j and the
// work vector; the stiffness is applied as in k_sweep_dof (A z = m (Lx z + Ly z), rows of the assembled 1-D
// operators in registers, z in two shared-memory planes with a halo); the two inner products per iteration
// are block reductions (warp shuffles + shared memory, fp64 accumulation, fixed order).
#pragma once
#include "hz_line.cuh"

namespace hz {

template <typename real>
struct MinresArgs {
  Layout lay;
  int sx, sy, E;
  int warm, max_iters;
  real tol;
  const real *mloc, *w2M, *wH, *bf_re, *bf_im;  // [L][NS]: m_j, w^2 M_j, w H_j, (f m + bc)_j re / im (im may be NULL)
  const real *sedge;                             // [L][4][E] geometric edge weights s_j^{side}
  const real *bandx, *bandy;                     // rows of Lx, Ly
  real *u_sub;                                   // [L][2][NS]
  const real *lam;                               // [L][4][2][E]
  real *gout;                                    // [L][4][2][E]
  const real *k2edge;                            // [L][4][E]
  int *iters;                                    // [L]
  double *res;                                   // [L] true relative residual of the returned x
};

// sum over the block of (a, b); every thread gets the result.  red: 66 doubles of shared memory.
__device__ __forceinline__ void block_sum2(double &a, double &b, double *red) {
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_down_sync(0xffffffffu, a, o);
    b += __shfl_down_sync(0xffffffffu, b, o);
  }
  const int w = threadIdx.x >> 5, ln = threadIdx.x & 31, nw = blockDim.x >> 5;
  if (ln == 0) { red[w] = a; red[32 + w] = b; }
  __syncthreads();
  if (w == 0) {
    a = ln < nw ? red[ln] : 0.0;
    b = ln < nw ? red[32 + ln] : 0.0;
    for (int o = 16; o > 0; o >>= 1) {
      a += __shfl_down_sync(0xffffffffu, a, o);
      b += __shfl_down_sync(0xffffffffu, b, o);
    }
    if (ln == 0) { red[64] = a; red[65] = b; }
  }
  __syncthreads();
  a = red[64];
  b = red[65];
  __syncthreads();  // red is reused by the next reduction
}

template <typename real, int P>
__global__ void __launch_bounds__(1024, 1) k_minres_dof(const MinresArgs<real> A) {
  constexpr int B = 2 * P + 1;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double *red = reinterpret_cast<double *>(smem_raw);  // 66 doubles (padded to 72)
  const int lnx = A.lay.lnx, lny = A.lay.lny, N = lnx * lny, NS = A.lay.NS;
  const int W = lnx + 2 * P, H = lny + 2 * P;
  real *zr = reinterpret_cast<real *>(red + 72), *zi = zr + W * H;
  const int t = threadIdx.x, NT = blockDim.x, l = blockIdx.x;
  const bool act = t < N;
  const int i = act ? t % lnx : 0, j = act ? t / lnx : 0;
  for (int q = t; q < 2 * W * H; q += NT) zr[q] = real(0);
  real cx[B], cy[B];
#pragma unroll
  for (int d = 0; d < B; ++d) {
    cx[d] = act ? A.bandx[i * B + d] : real(0);
    cy[d] = act ? A.bandy[j * B + d] : real(0);
  }
  const size_t base = (size_t)l * NS + t;
  const real m = act ? A.mloc[base] : real(0), w2M = act ? A.w2M[base] : real(0), wH = act ? A.wH[base] : real(0);
  // rhs = [Re b; -Im b],  b = f m (+ bc) + sum_sides s lambda^n
  real br = act ? A.bf_re[base] : real(0), bi = (act && A.bf_im) ? A.bf_im[base] : real(0);
  const int six = l % A.sx, siy = l / A.sx;
  const size_t lbase = (size_t)l * 4 * 2 * A.E, ebase = (size_t)l * 4 * A.E;
  const bool onW = act && i == 0 && six > 0, onE = act && i == lnx - 1 && six < A.sx - 1;
  const bool onS = act && j == 0 && siy > 0, onN = act && j == lny - 1 && siy < A.sy - 1;
  if (onW) { const real s = A.sedge[ebase + kSideW * A.E + j];
    br = fmaT(s, A.lam[lbase + (kSideW * 2 + 0) * A.E + j], br); bi = fmaT(s, A.lam[lbase + (kSideW * 2 + 1) * A.E + j], bi); }
  if (onE) { const real s = A.sedge[ebase + kSideE * A.E + j];
    br = fmaT(s, A.lam[lbase + (kSideE * 2 + 0) * A.E + j], br); bi = fmaT(s, A.lam[lbase + (kSideE * 2 + 1) * A.E + j], bi); }
  if (onS) { const real s = A.sedge[ebase + kSideS * A.E + i];
    br = fmaT(s, A.lam[lbase + (kSideS * 2 + 0) * A.E + i], br); bi = fmaT(s, A.lam[lbase + (kSideS * 2 + 1) * A.E + i], bi); }
  if (onN) { const real s = A.sedge[ebase + kSideN * A.E + i];
    br = fmaT(s, A.lam[lbase + (kSideN * 2 + 0) * A.E + i], br); bi = fmaT(s, A.lam[lbase + (kSideN * 2 + 1) * A.E + i], bi); }
  const real rr = br, ri = -bi;
  const int center = (j + P) * W + (i + P);
  __syncthreads();

  // (K z)_r = (A - w^2 M) z_r + w H z_i,   (K z)_i = w H z_r + (w^2 M - A) z_i,   A z = m (Lx z + Ly z)
  auto applyK = [&](real ar, real ai, real &kr, real &ki) {
    if (act) { zr[center] = ar; zi[center] = ai; }
    __syncthreads();
    real Sr = real(0), Si = real(0);
#pragma unroll
    for (int d = 0; d < B; ++d) {
      Sr = fmaT(cx[d], zr[center + (d - P)], Sr);
      Sr = fmaT(cy[d], zr[center + (d - P) * W], Sr);
      Si = fmaT(cx[d], zi[center + (d - P)], Si);
      Si = fmaT(cy[d], zi[center + (d - P) * W], Si);
    }
    __syncthreads();
    kr = fmaT(m, Sr, fmaT(-w2M, ar, wH * ai));
    ki = fmaT(-m, Si, fmaT(w2M, ai, wH * ar));
  };

  real xr = real(0), xi = real(0);
  if (act && A.warm) { xr = A.u_sub[(size_t)l * 2 * NS + t]; xi = A.u_sub[(size_t)l * 2 * NS + NS + t]; }
  real vr = rr, vi = ri;
  if (A.warm) {
    real kr, ki;
    applyK(xr, xi, kr, ki);
    vr = rr - kr; vi = ri - ki;
  }
  double s0 = act ? (double)rr * rr + (double)ri * ri : 0.0, s1 = act ? (double)vr * vr + (double)vi * vi : 0.0;
  block_sum2(s0, s1, red);
  const double bnorm = sqrt(s0);
  double gamma = sqrt(s1), eta = gamma;
  real vor = 0, voi = 0, wor = 0, woi = 0, wr = 0, wi = 0;
  double s_old = 0.0, s = 0.0, c_old = 1.0, c = 1.0;
  int it = 0;
  const double thr = (double)A.tol * bnorm;
  // a right-hand side below the underflow guard is treated as zero (x = x0): 1/gamma would overflow in `real`
  const double tiny = sizeof(real) == 4 ? 1e-30 : 1e-140;
  if (bnorm > tiny && gamma > thr) {
    for (it = 1; it <= A.max_iters; ++it) {
      const real ig = (real)(1.0 / gamma);
      vr *= ig; vi *= ig;
      real kr, ki;
      applyK(vr, vi, kr, ki);
      double d0 = act ? (double)vr * kr + (double)vi * ki : 0.0, dz = 0.0;
      block_sum2(d0, dz, red);
      const double delta = d0;
      real nr = fmaT((real)(-delta), vr, fmaT((real)(-gamma), vor, kr));
      real ni = fmaT((real)(-delta), vi, fmaT((real)(-gamma), voi, ki));
      double g2 = act ? (double)nr * nr + (double)ni * ni : 0.0;
      dz = 0.0;
      block_sum2(g2, dz, red);
      const double gamma_new = sqrt(g2);
      const double a0 = c * delta - c_old * s * gamma;
      const double a1 = sqrt(a0 * a0 + gamma_new * gamma_new);
      const double a2 = s * delta + c_old * c * gamma;
      const double a3 = s_old * gamma;
      const double c_new = a0 / a1, s_new = gamma_new / a1;
      const real ia1 = (real)(1.0 / a1);
      const real wnr = (vr - (real)a3 * wor - (real)a2 * wr) * ia1;
      const real wni = (vi - (real)a3 * woi - (real)a2 * wi) * ia1;
      xr = fmaT((real)(c_new * eta), wnr, xr);
      xi = fmaT((real)(c_new * eta), wni, xi);
      eta = -s_new * eta;
      vor = vr; voi = vi; vr = nr; vi = ni; gamma = gamma_new;
      wor = wr; woi = wi; wr = wnr; wi = wni;
      s_old = s; s = s_new; c_old = c; c = c_new;
      if (fabs(eta) <= thr || gamma == 0.0) break;
    }
    if (it > A.max_iters) it = A.max_iters;
  }
  // true relative residual of the returned x
  {
    real kr, ki;
    applyK(xr, xi, kr, ki);
    const real er = rr - kr, ei = ri - ki;
    double e2 = act ? (double)er * er + (double)ei * ei : 0.0, dz = 0.0;
    block_sum2(e2, dz, red);
    if (t == 0) {
      A.iters[l] = it;
      A.res[l] = bnorm > tiny ? sqrt(e2) / bnorm : 0.0;
    }
  }
  if (act) {
    A.u_sub[(size_t)l * 2 * NS + t] = xr;
    A.u_sub[(size_t)l * 2 * NS + NS + t] = xi;
    // outgoing interface data g = -lambda^n - 2 i k u  (eq. (2); sign per reading R3)
    if (onW) { const real k2 = A.k2edge[ebase + kSideW * A.E + j];
      A.gout[lbase + (kSideW * 2 + 0) * A.E + j] = fmaT(k2, xi, -A.lam[lbase + (kSideW * 2 + 0) * A.E + j]);
      A.gout[lbase + (kSideW * 2 + 1) * A.E + j] = fmaT(-k2, xr, -A.lam[lbase + (kSideW * 2 + 1) * A.E + j]); }
    if (onE) { const real k2 = A.k2edge[ebase + kSideE * A.E + j];
      A.gout[lbase + (kSideE * 2 + 0) * A.E + j] = fmaT(k2, xi, -A.lam[lbase + (kSideE * 2 + 0) * A.E + j]);
      A.gout[lbase + (kSideE * 2 + 1) * A.E + j] = fmaT(-k2, xr, -A.lam[lbase + (kSideE * 2 + 1) * A.E + j]); }
    if (onS) { const real k2 = A.k2edge[ebase + kSideS * A.E + i];
      A.gout[lbase + (kSideS * 2 + 0) * A.E + i] = fmaT(k2, xi, -A.lam[lbase + (kSideS * 2 + 0) * A.E + i]);
      A.gout[lbase + (kSideS * 2 + 1) * A.E + i] = fmaT(-k2, xr, -A.lam[lbase + (kSideS * 2 + 1) * A.E + i]); }
    if (onN) { const real k2 = A.k2edge[ebase + kSideN * A.E + i];
      A.gout[lbase + (kSideN * 2 + 0) * A.E + i] = fmaT(k2, xi, -A.lam[lbase + (kSideN * 2 + 0) * A.E + i]);
      A.gout[lbase + (kSideN * 2 + 1) * A.E + i] = fmaT(-k2, xr, -A.lam[lbase + (kSideN * 2 + 1) * A.E + i]); }
  }
}

}  // namespace hz

namespace hz {

// ------------------------------------------------------------------------------------------------------------------
// k_minres_tile: the same MINRES in the REGISTER-BLOCKED layout of the WaveHoltz kernels (PAPER.md:271-277 compares
// the two subdomain solvers "in the same layouts", Table I at 291-306): a thread owns the P x P lower-left nodes of
// M x M elements, all MINRES vectors of its nodes live in its registers (x, v_{j-1}, v_j, w_{j-1}, w_j, complex: ten
// values per node, which is what the paper means by "arrays that spill into L1" for large tiles), and the stiffness is
// applied with the line operators and the partial-sum / raw-value exchange records of hz_sweep_tile.cuh, once per
// plane (re, im).  Two block reductions per iteration as before.  One subdomain per block, uniform code (the ragged
// last node column / row is an extra tile column / row; its padding nodes have zero coefficients and stay zero).
// ------------------------------------------------------------------------------------------------------------------
template <typename real, int P, int M>
__global__ void __launch_bounds__(256, 1) k_minres_tile(const MinresArgs<real> A, const Elem1D<real> ex1, const Elem1D<real> ey1) {
  constexpr int T = M * P;
  constexpr int V16 = 16 / (int)sizeof(real);
  constexpr int CH = (T + V16 - 1) / V16 * V16;
  constexpr int RS = 4 * CH + V16;   // PX | RX | PY | RY + 16 bytes: odd number of 16-byte units
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double *red = reinterpret_cast<double *>(smem_raw);  // 66 doubles (padded to 72)
  const int t = threadIdx.x, NTH = blockDim.x, l = blockIdx.x;
  const int ntx = A.lay.ntx, nty = A.lay.nty, NS = A.lay.NS, NTV = A.lay.NT;
  const int lnx = A.lay.lnx, lny = A.lay.lny;
  const int PLW = (NTH + 2) * RS;   // one plane of records: NTH tiles + zero record + scratch record
  real *xb = reinterpret_cast<real *>(red + 72);
  const bool act = t < ntx * nty;
  const int tx = act ? t % ntx : 0, ty = act ? t / ntx : 0;
  const int ZR = NTH, SCR = NTH + 1;
  for (int q = t; q < 2 * PLW; q += NTH) xb[q] = real(0);
  const bool hasL = act && tx > 0, hasR = act && tx < ntx - 1, hasD = act && ty > 0, hasU = act && ty < nty - 1;
  const real *pL = xb + (hasL ? t - 1 : ZR) * RS, *pR = xb + (hasR ? t + 1 : ZR) * RS + CH;
  const real *pD = xb + (hasD ? t - ntx : ZR) * RS + 2 * CH, *pU = xb + (hasU ? t + ntx : ZR) * RS + 3 * CH;
  real *pMy = xb + (act ? t : SCR) * RS;
  const real d0x = (hasR ? ex1.k0[0] : real(0)) + (hasL ? ex1.kp[P] : real(0));
  const real d0y = (hasU ? ey1.k0[0] : real(0)) + (hasD ? ey1.kp[P] : real(0));
  const real s0x = (hasL && hasR) ? real(1) : real(2), s0y = (hasD && hasU) ? real(1) : real(2);

  real mm[T][T], w2M[T][T], rr[T][T], ri[T][T];
  real wHc[T], wHr[T];   // w H is non-zero on the subdomain boundary only: column 0 / row 0 of the outer tiles
  const size_t base = (size_t)l * NS + t;
#pragma unroll
  for (int b = 0; b < T; ++b)
#pragma unroll
    for (int a = 0; a < T; ++a) {
      const size_t o = base + (size_t)(b * T + a) * NTV;
      mm[b][a] = act ? A.mloc[o] : real(0);
      w2M[b][a] = act ? A.w2M[o] : real(0);
      rr[b][a] = act ? A.bf_re[o] : real(0);
      ri[b][a] = (act && A.bf_im) ? A.bf_im[o] : real(0);
    }
#pragma unroll
  for (int n = 0; n < T; ++n) {
    wHc[n] = act ? A.wH[base + (size_t)(n * T) * NTV] : real(0);
    wHr[n] = act ? A.wH[base + (size_t)n * NTV] : real(0);
  }
  // rhs = [Re b; -Im b],  b = f m (+ bc) + sum_sides s lambda^n
  const int six = l % A.sx, siy = l / A.sx;
  const size_t lbase = (size_t)l * 4 * 2 * A.E, ebase = (size_t)l * 4 * A.E;
  int sideX = -1, sideY = -1;
  if (act && tx == 0 && six > 0) sideX = kSideW;
  if (act && tx == ntx - 1 && six < A.sx - 1) sideX = kSideE;
  if (act && ty == 0 && siy > 0) sideY = kSideS;
  if (act && ty == nty - 1 && siy < A.sy - 1) sideY = kSideN;
  if (sideX >= 0) {
#pragma unroll
    for (int b = 0; b < T; ++b) {
      const int j = ty * T + b;
      if (j < lny) {
        const real s = A.sedge[ebase + sideX * A.E + j];
        rr[b][0] = fmaT(s, A.lam[lbase + (sideX * 2 + 0) * A.E + j], rr[b][0]);
        ri[b][0] = fmaT(s, A.lam[lbase + (sideX * 2 + 1) * A.E + j], ri[b][0]);
      }
    }
  }
  if (sideY >= 0) {
#pragma unroll
    for (int a = 0; a < T; ++a) {
      const int i = tx * T + a;
      if (i < lnx) {
        const real s = A.sedge[ebase + sideY * A.E + i];
        rr[0][a] = fmaT(s, A.lam[lbase + (sideY * 2 + 0) * A.E + i], rr[0][a]);
        ri[0][a] = fmaT(s, A.lam[lbase + (sideY * 2 + 1) * A.E + i], ri[0][a]);
      }
    }
  }
#pragma unroll
  for (int b = 0; b < T; ++b)
#pragma unroll
    for (int a = 0; a < T; ++a) ri[b][a] = -ri[b][a];
  __syncthreads();

  // S = Lx z + Ly z of one plane z (values in registers), through record plane `pl`
  auto stiff = [&](const real (&z)[T][T], int pl) {
    real *my = pMy + pl * PLW;
    {
      real vPX[T], vRX[T], vPY[T], vRY[T];
#pragma unroll
      for (int b = 0; b < T; ++b) {
        real q[T + 1];
#pragma unroll
        for (int a = 0; a < T; ++a) q[a] = z[b][a];
        q[T] = real(0);
        vPX[b] = line_partial<real, P, M>(q, ex1);
        vRX[b] = z[b][0];
      }
#pragma unroll
      for (int a = 0; a < T; ++a) {
        real q[T + 1];
#pragma unroll
        for (int b = 0; b < T; ++b) q[b] = z[b][a];
        q[T] = real(0);
        vPY[a] = line_partial<real, P, M>(q, ey1);
        vRY[a] = z[0][a];
      }
      st_chunk<T>(my, vPX);
      st_chunk<T>(my + CH, vRX);
      st_chunk<T>(my + 2 * CH, vPY);
      st_chunk<T>(my + 3 * CH, vRY);
    }
  };
  auto stiff_finish = [&](const real (&z)[T][T], real (&S)[T][T], int pl) {
    real qR[T], piL[T], qU[T], piD[T], X0[T], Y0[T];
    ld_chunk<T>(pL + pl * PLW, piL);
    ld_chunk<T>(pR + pl * PLW, qR);
    ld_chunk<T>(pD + pl * PLW, piD);
    ld_chunk<T>(pU + pl * PLW, qU);
#pragma unroll
    for (int b = 0; b < T; ++b) {
      real q[T + 1];
#pragma unroll
      for (int a = 0; a < T; ++a) q[a] = z[b][a];
      q[T] = real(0);
      X0[b] = line_own<real, P, M, false>(q, d0x, ex1, S[b]);
    }
#pragma unroll
    for (int a = 0; a < T; ++a) {
      real q[T + 1], Sc[T];
#pragma unroll
      for (int b = 0; b < T; ++b) { q[b] = z[b][a]; Sc[b] = S[b][a]; }
      q[T] = real(0);
      if (a == 0) Y0[a] = line_own<real, P, M, false>(q, d0y, ey1, Sc);
      else Y0[a] = line_own<real, P, M, true>(q, d0y, ey1, Sc);
#pragma unroll
      for (int b = 1; b < T; ++b) S[b][a] = Sc[b];
    }
#pragma unroll
    for (int b = 0; b < T; ++b) {
      if (b == 0) line_finish<real, P, M, false>(qR[b], piL[b], s0x, X0[b], ex1, S[b]);
      else line_finish<real, P, M, true>(qR[b], piL[b], s0x, X0[b], ex1, S[b]);
    }
#pragma unroll
    for (int a = 0; a < T; ++a) {
      real Sc[T];
#pragma unroll
      for (int b = 0; b < T; ++b) Sc[b] = S[b][a];
      line_finish<real, P, M, true>(qU[a], piD[a], s0y, Y0[a], ey1, Sc);
#pragma unroll
      for (int b = 0; b < T; ++b) S[b][a] = Sc[b];
    }
  };
  // (K z)_r = (A - w^2 M) z_r + w H z_i,   (K z)_i = w H z_r + (w^2 M - A) z_i,   A z = m (Lx z + Ly z)
  auto applyK = [&](const real (&ar)[T][T], const real (&ai)[T][T], real (&kr)[T][T], real (&ki)[T][T]) {
    stiff(ar, 0);
    stiff(ai, 1);
    __syncthreads();
    stiff_finish(ar, kr, 0);
    stiff_finish(ai, ki, 1);
    __syncthreads();
#pragma unroll
    for (int b = 0; b < T; ++b)
#pragma unroll
      for (int a = 0; a < T; ++a) {
        const real wh = a == 0 ? wHc[b] : (b == 0 ? wHr[a] : real(0));
        const real Sr = kr[b][a], Si = ki[b][a];
        kr[b][a] = fmaT(mm[b][a], Sr, fmaT(-w2M[b][a], ar[b][a], wh * ai[b][a]));
        ki[b][a] = fmaT(-mm[b][a], Si, fmaT(w2M[b][a], ai[b][a], wh * ar[b][a]));
      }
  };
  auto dot2 = [&](const real (&a1)[T][T], const real (&a2)[T][T], const real (&b1)[T][T], const real (&b2)[T][T]) {
    double s = 0.0;
#pragma unroll
    for (int b = 0; b < T; ++b)
#pragma unroll
      for (int a = 0; a < T; ++a) s += (double)a1[b][a] * b1[b][a] + (double)a2[b][a] * b2[b][a];
    return s;
  };

  real xr[T][T], xi[T][T], vr[T][T], vi[T][T], kr[T][T], ki[T][T];
#pragma unroll
  for (int b = 0; b < T; ++b)
#pragma unroll
    for (int a = 0; a < T; ++a) {
      const size_t o = (size_t)(b * T + a) * NTV + t;
      xr[b][a] = (act && A.warm) ? A.u_sub[(size_t)l * 2 * NS + o] : real(0);
      xi[b][a] = (act && A.warm) ? A.u_sub[(size_t)l * 2 * NS + NS + o] : real(0);
      vr[b][a] = rr[b][a];
      vi[b][a] = ri[b][a];
    }
  if (A.warm) {
    applyK(xr, xi, kr, ki);
#pragma unroll
    for (int b = 0; b < T; ++b)
#pragma unroll
      for (int a = 0; a < T; ++a) { vr[b][a] = rr[b][a] - kr[b][a]; vi[b][a] = ri[b][a] - ki[b][a]; }
  }
  double s0 = dot2(rr, ri, rr, ri), s1 = dot2(vr, vi, vr, vi);
  block_sum2(s0, s1, red);
  const double bnorm = sqrt(s0);
  double gamma = sqrt(s1), eta = gamma;
  real vor[T][T], voi[T][T], wor[T][T], woi[T][T], wr[T][T], wi[T][T];
#pragma unroll
  for (int b = 0; b < T; ++b)
#pragma unroll
    for (int a = 0; a < T; ++a) vor[b][a] = voi[b][a] = wor[b][a] = woi[b][a] = wr[b][a] = wi[b][a] = real(0);
  double s_old = 0.0, s = 0.0, c_old = 1.0, c = 1.0;
  int it = 0;
  const double thr = (double)A.tol * bnorm;
  const double tiny = sizeof(real) == 4 ? 1e-30 : 1e-140;
  if (bnorm > tiny && gamma > thr) {
#pragma unroll 1
    for (it = 1; it <= A.max_iters; ++it) {
      const real ig = (real)(1.0 / gamma);
#pragma unroll
      for (int b = 0; b < T; ++b)
#pragma unroll
        for (int a = 0; a < T; ++a) { vr[b][a] *= ig; vi[b][a] *= ig; }
      applyK(vr, vi, kr, ki);
      double d0 = dot2(vr, vi, kr, ki), dz = 0.0;
      block_sum2(d0, dz, red);
      const double delta = d0;
      double g2 = 0.0;
#pragma unroll
      for (int b = 0; b < T; ++b)
#pragma unroll
        for (int a = 0; a < T; ++a) {   // kr, ki become the next Lanczos vector
          kr[b][a] = fmaT((real)(-delta), vr[b][a], fmaT((real)(-gamma), vor[b][a], kr[b][a]));
          ki[b][a] = fmaT((real)(-delta), vi[b][a], fmaT((real)(-gamma), voi[b][a], ki[b][a]));
          g2 += (double)kr[b][a] * kr[b][a] + (double)ki[b][a] * ki[b][a];
        }
      dz = 0.0;
      block_sum2(g2, dz, red);
      const double gamma_new = sqrt(g2);
      const double a0 = c * delta - c_old * s * gamma;
      const double a1 = sqrt(a0 * a0 + gamma_new * gamma_new);
      const double a2 = s * delta + c_old * c * gamma;
      const double a3 = s_old * gamma;
      const double c_new = a0 / a1, s_new = gamma_new / a1;
      const real ia1 = (real)(1.0 / a1), ce = (real)(c_new * eta);
#pragma unroll
      for (int b = 0; b < T; ++b)
#pragma unroll
        for (int a = 0; a < T; ++a) {
          const real wnr = (vr[b][a] - (real)a3 * wor[b][a] - (real)a2 * wr[b][a]) * ia1;
          const real wni = (vi[b][a] - (real)a3 * woi[b][a] - (real)a2 * wi[b][a]) * ia1;
          xr[b][a] = fmaT(ce, wnr, xr[b][a]);
          xi[b][a] = fmaT(ce, wni, xi[b][a]);
          vor[b][a] = vr[b][a]; voi[b][a] = vi[b][a];
          vr[b][a] = kr[b][a]; vi[b][a] = ki[b][a];
          wor[b][a] = wr[b][a]; woi[b][a] = wi[b][a];
          wr[b][a] = wnr; wi[b][a] = wni;
        }
      eta = -s_new * eta;
      gamma = gamma_new;
      s_old = s; s = s_new; c_old = c; c = c_new;
      if (fabs(eta) <= thr || gamma == 0.0) break;
    }
    if (it > A.max_iters) it = A.max_iters;
  }
  {  // true relative residual of the returned x
    applyK(xr, xi, kr, ki);
    double e2 = 0.0, dz = 0.0;
#pragma unroll
    for (int b = 0; b < T; ++b)
#pragma unroll
      for (int a = 0; a < T; ++a) {
        const real er = rr[b][a] - kr[b][a], ei = ri[b][a] - ki[b][a];
        e2 += (double)er * er + (double)ei * ei;
      }
    block_sum2(e2, dz, red);
    if (t == 0) {
      A.iters[l] = it;
      A.res[l] = bnorm > tiny ? sqrt(e2) / bnorm : 0.0;
    }
  }
  if (act) {
#pragma unroll
    for (int b = 0; b < T; ++b)
#pragma unroll
      for (int a = 0; a < T; ++a) {
        const size_t o = (size_t)(b * T + a) * NTV + t;
        A.u_sub[(size_t)l * 2 * NS + o] = xr[b][a];
        A.u_sub[(size_t)l * 2 * NS + NS + o] = xi[b][a];
      }
  }
  // outgoing interface data g = -lambda^n - 2 i k u  (eq. (2); sign per reading R3)
  if (sideX >= 0) {
#pragma unroll
    for (int b = 0; b < T; ++b) {
      const int j = ty * T + b;
      if (j < lny) {
        const real k2 = A.k2edge[ebase + sideX * A.E + j];
        A.gout[lbase + (sideX * 2 + 0) * A.E + j] = fmaT(k2, xi[b][0], -A.lam[lbase + (sideX * 2 + 0) * A.E + j]);
        A.gout[lbase + (sideX * 2 + 1) * A.E + j] = fmaT(-k2, xr[b][0], -A.lam[lbase + (sideX * 2 + 1) * A.E + j]);
      }
    }
  }
  if (sideY >= 0) {
#pragma unroll
    for (int a = 0; a < T; ++a) {
      const int i = tx * T + a;
      if (i < lnx) {
        const real k2 = A.k2edge[ebase + sideY * A.E + i];
        A.gout[lbase + (sideY * 2 + 0) * A.E + i] = fmaT(k2, xi[0][a], -A.lam[lbase + (sideY * 2 + 0) * A.E + i]);
        A.gout[lbase + (sideY * 2 + 1) * A.E + i] = fmaT(-k2, xr[0][a], -A.lam[lbase + (sideY * 2 + 1) * A.E + i]);
      }
    }
  }
}

}  // namespace hz
