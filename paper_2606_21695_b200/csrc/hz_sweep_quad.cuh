// hz_sweep_quad.cuh — sweep kernel for general straight-sided convex quadrilaterals (
// D, geometric factors, D^T).  One thread block per subdomain, ONE THREAD PER ELEMENT.
//
// A thread keeps the (P+1)^2 local nodes of its element in registers — p, pdot, v_r, v_i of ALL of them, so a node
// shared by 2 (4) elements has 2 (4) replicated copies that are updated identically — and applies the element
// operator  out = Dxi^T (Gxx Dxi p + Gxy Deta p) + Deta^T (Gxy Dxi p + Gyy Deta p)  entirely in registers.
// What crosses threads per time step is only the partial sum `out` on the element's boundary nodes: four chunks
// (W, E, S, N edge, P+1 values each, 128-bit stores) per element, read by the 4 edge neighbours (128-bit loads) and,
// one value each, by the 4 diagonal neighbours; ping-pong buffers, ONE barrier per step.  The copies of a shared
// node stay bit-identical because every copy adds the same partial sums in the same association:
// edge nodes  (west/south element) + (east/north element);  corners  (DL + DR) + (UL + UR).
// (The paper's layout — one thread per element-local node, every operand through shared memory, 3 barriers per
// step — is the prior art this replaces.)
// Per-thread strip in shared memory: for each node row b the (beta, alpha, beta Re b, beta Im b) of its P+1 nodes,
// then the 3 geometric factors (weights folded in) of its P+1 points.
#pragma once
#include "hz_line.cuh"

namespace hz {

template <typename real, int P, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB)
    k_sweep_quad(const SweepArgs<real> A, const __grid_constant__ QuadArgs<real> Q, const __grid_constant__ TabC<real> TC) {
  constexpr int N1 = P + 1, NQ = N1 * N1;
  constexpr int V16 = 16 / (int)sizeof(real);
  constexpr int CH = (N1 + V16 - 1) / V16 * V16;
  constexpr int RS0 = 4 * CH;
  constexpr int RS = ((RS0 / V16) % 2 == 0) ? RS0 + V16 : RS0;  // odd number of 16-byte units
  constexpr int GR = (3 * N1 + V16 - 1) / V16 * V16;            // geometric factors of one node row
  constexpr int ROWW = 4 * N1 + GR;
  constexpr int CS0 = N1 * ROWW;
  constexpr int CST = ((CS0 / V16) % 2 == 0) ? CS0 + V16 : CS0;
  constexpr int oW = 0, oE = CH, oS = 2 * CH, oN = 3 * CH;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int t = threadIdx.x, NT = blockDim.x, l = blockIdx.x;
  const int BUFW = (NT + 2) * RS;  // + one all-zero record (missing neighbours; a broadcast read) + one scratch record
  real *xb = reinterpret_cast<real *>(smem_raw);
  real *csm = xb + 2 * BUFW + (size_t)t * CST;
  // ex = element stride of the thread grid (the widest subdomain); exl x eyl = this subdomain's elements (ragged
  // partitions, reading R25); lnx = node stride of the per-DOF arrays, lnxl x lnyl = this subdomain's nodes
  const int ex = A.lay.ntx, NS = A.lay.NS, lnx = A.lay.lnx;
  const int six = l % A.sx, siy = l / A.sx;
  const int exl = A.exq + (six < A.exr ? 1 : 0), eyl = A.eyq + (siy < A.eyr ? 1 : 0);
  const int lnxl = exl * P + 1, lnyl = eyl * P + 1;
  const bool act = t < ex * A.lay.nty && t % ex < exl && t / ex < eyl;
  const int fx = act ? t % ex : 0, fy = act ? t / ex : 0;
  const int ZR = NT, SCR = NT + 1;

  for (int q = t; q < 2 * BUFW; q += NT) xb[q] = real(0);

  const bool hasL = act && fx > 0, hasR = act && fx < exl - 1, hasD = act && fy > 0, hasU = act && fy < eyl - 1;
  auto rec = [&](bool has, int nb) { return xb + (has ? nb : ZR) * RS; };
  const real *pL = rec(hasL, t - 1) + oE, *pR = rec(hasR, t + 1) + oW;
  const real *pD = rec(hasD, t - ex) + oN, *pU = rec(hasU, t + ex) + oS;
  const real *pDL = rec(hasD && hasL, t - ex - 1) + oE + P, *pDR = rec(hasD && hasR, t - ex + 1) + oW + P;
  const real *pUL = rec(hasU && hasL, t + ex - 1) + oE, *pUR = rec(hasU && hasR, t + ex + 1) + oW;
  real *pMy = xb + (act ? t : SCR) * RS;

  real p[N1][N1], pd[N1][N1], vr[N1][N1], vi[N1][N1], ur[N1][N1], ui[N1][N1];
  const size_t lbase = (size_t)l * 4 * 2 * A.E, ebase = (size_t)l * 4 * A.E;
  if (act) {
#pragma unroll
    for (int b = 0; b < N1; ++b)
#pragma unroll
      for (int a = 0; a < N1; ++a) {
        const int i = fx * P + a, j = fy * P + b;
        const size_t o = (size_t)l * NS + (size_t)j * lnx + i;
        real br = A.bbf_re[o], bi = A.bbf_im ? A.bbf_im[o] : real(0);
        // b from lambda^n on the interface sides; a subdomain-corner node gets both sides
        if (i == 0 && six > 0) {
          const real s = A.bs[ebase + kSideW * A.E + j];
          br = fmaT(s, A.lam[lbase + (kSideW * 2 + 0) * A.E + j], br);
          bi = fmaT(s, A.lam[lbase + (kSideW * 2 + 1) * A.E + j], bi);
        }
        if (i == lnxl - 1 && six < A.sx - 1) {
          const real s = A.bs[ebase + kSideE * A.E + j];
          br = fmaT(s, A.lam[lbase + (kSideE * 2 + 0) * A.E + j], br);
          bi = fmaT(s, A.lam[lbase + (kSideE * 2 + 1) * A.E + j], bi);
        }
        if (j == 0 && siy > 0) {
          const real s = A.bs[ebase + kSideS * A.E + i];
          br = fmaT(s, A.lam[lbase + (kSideS * 2 + 0) * A.E + i], br);
          bi = fmaT(s, A.lam[lbase + (kSideS * 2 + 1) * A.E + i], bi);
        }
        if (j == lnyl - 1 && siy < A.sy - 1) {
          const real s = A.bs[ebase + kSideN * A.E + i];
          br = fmaT(s, A.lam[lbase + (kSideN * 2 + 0) * A.E + i], br);
          bi = fmaT(s, A.lam[lbase + (kSideN * 2 + 1) * A.E + i], bi);
        }
        real *cr = csm + b * ROWW;
        cr[4 * a + 0] = A.gamma[o];  // beta_j
        cr[4 * a + 1] = A.alpha[o];
        cr[4 * a + 2] = br;
        cr[4 * a + 3] = bi;
#pragma unroll
        for (int k = 0; k < 3; ++k)
          cr[4 * N1 + 3 * a + k] = Q.G[((size_t)l * 3 * NQ + 3 * (b * N1 + a) + k) * Q.nep + t];
        ur[b][a] = A.warm ? A.u_sub[(size_t)l * 2 * NS + (size_t)j * lnx + i] : real(0);
        ui[b][a] = A.warm ? A.u_sub[(size_t)l * 2 * NS + NS + (size_t)j * lnx + i] : real(0);
      }
  } else {
#pragma unroll
    for (int b = 0; b < N1; ++b)
#pragma unroll
      for (int a = 0; a < N1; ++a) ur[b][a] = ui[b][a] = real(0);
  }
  __syncthreads();

  const real sigma = A.sigma;
  int cur = 0;
  for (int m = 0; m < A.n_wh; ++m) {
    const Tab4<real> t0 = A.n_t <= kTabCMax ? TC.t[0] : A.tab[0];
#pragma unroll
    for (int b = 0; b < N1; ++b)
#pragma unroll
      for (int a = 0; a < N1; ++a) {  // WaveHoltz init (readings R2, R8)
        p[b][a] = ur[b][a];
        pd[b][a] = A.omega * (ui[b][a] * A.cos_h - ur[b][a] * A.sin_h);
        vr[b][a] = t0.k * p[b][a];
        vi[b][a] = t0.kh * pd[b][a];
      }
#pragma unroll 1
    for (int nu = 1; nu < A.n_t; ++nu) {
      const Tab4<real> tn = A.n_t <= kTabCMax ? TC.t[nu] : A.tab[nu];
      real out[N1][N1];
      if (act) {
#pragma unroll
        for (int b = 0; b < N1; ++b)
#pragma unroll
          for (int a = 0; a < N1; ++a) p[b][a] = fmaT(sigma, pd[b][a], p[b][a]);
        real fr[N1][N1], fs[N1][N1];
#pragma unroll
        for (int b = 0; b < N1; ++b) {
          real g[GR];
          ld_chunk<GR>(csm + b * ROWW + 4 * N1, g);
#pragma unroll
          for (int a = 0; a < N1; ++a) {  // gradient on the reference element, then the geometric factors
            real ux = Q.D[a][0] * p[b][0], uy = Q.D[b][0] * p[0][a];
#pragma unroll
            for (int c = 1; c < N1; ++c) {
              ux = fmaT(Q.D[a][c], p[b][c], ux);
              uy = fmaT(Q.D[b][c], p[c][a], uy);
            }
            fr[b][a] = fmaT(g[3 * a], ux, g[3 * a + 1] * uy);
            fs[b][a] = fmaT(g[3 * a + 1], ux, g[3 * a + 2] * uy);
          }
        }
#pragma unroll
        for (int b = 0; b < N1; ++b)
#pragma unroll
          for (int a = 0; a < N1; ++a) {  // D^T
            real o = Q.D[0][a] * fr[b][0];
#pragma unroll
            for (int c = 1; c < N1; ++c) o = fmaT(Q.D[c][a], fr[b][c], o);
#pragma unroll
            for (int c = 0; c < N1; ++c) o = fmaT(Q.D[c][b], fs[c][a], o);
            out[b][a] = o;
          }
        {  // publish the partial sums of the element's boundary nodes
          real *my = pMy + cur;
          real vW[N1], vE[N1], vS[N1], vN[N1];
#pragma unroll
          for (int k = 0; k < N1; ++k) {
            vW[k] = out[k][0]; vE[k] = out[k][P]; vS[k] = out[0][k]; vN[k] = out[P][k];
          }
          st_chunk<N1>(my + oW, vW);
          st_chunk<N1>(my + oE, vE);
          st_chunk<N1>(my + oS, vS);
          st_chunk<N1>(my + oN, vN);
        }
#pragma unroll
        for (int b = 0; b < N1; ++b)
#pragma unroll
          for (int a = 0; a < N1; ++a) vr[b][a] = fmaT(tn.k, p[b][a], vr[b][a]);
      }
      __syncthreads();
      if (act) {
        real inL[N1], inR[N1], inD[N1], inU[N1];
        ld_chunk<N1>(pL + cur, inL);
        ld_chunk<N1>(pR + cur, inR);
        ld_chunk<N1>(pD + cur, inD);
        ld_chunk<N1>(pU + cur, inU);
        const real dDL = pDL[cur], dDR = pDR[cur], dUL = pUL[cur], dUR = pUR[cur];
        // assemble: same values, same association in every copy of a shared node
        const real c00 = (dDL + inD[0]) + (inL[0] + out[0][0]);
        const real cP0 = (inD[P] + dDR) + (out[0][P] + inR[0]);
        const real c0P = (inL[P] + out[P][0]) + (dUL + inU[0]);
        const real cPP = (out[P][P] + inR[P]) + (inU[P] + dUR);
#pragma unroll
        for (int k = 1; k < P; ++k) {
          out[k][0] = inL[k] + out[k][0];
          out[k][P] = out[k][P] + inR[k];
          out[0][k] = inD[k] + out[0][k];
          out[P][k] = out[P][k] + inU[k];
        }
        out[0][0] = c00; out[0][P] = cP0; out[P][0] = c0P; out[P][P] = cPP;
#pragma unroll
        for (int b = 0; b < N1; ++b) {
          real cf[4 * N1];
          ld_chunk<4 * N1>(csm + b * ROWW, cf);
#pragma unroll
          for (int a = 0; a < N1; ++a) {  // pdot, filter
            const real x = fmaT(cf[4 * a + 3], tn.s, fmaT(-cf[4 * a], out[b][a], cf[4 * a + 2] * tn.c));
            pd[b][a] = fmaT(cf[4 * a + 1], pd[b][a], x);
            vi[b][a] = fmaT(tn.kh, pd[b][a], vi[b][a]);
          }
        }
      }
      cur = BUFW - cur;
    }
#pragma unroll
    for (int b = 0; b < N1; ++b)
#pragma unroll
      for (int a = 0; a < N1; ++a) {  // eq. (7) prefactor (reading R4)
        ur[b][a] = A.two_over_nt * vr[b][a];
        ui[b][a] = A.two_over_nt * vi[b][a];
      }
  }
  if (!act) return;
  // store u_l (A7) — each node by the element that has it as a lower-left node (or the last element of the row /
  // column) — and g = -lambda^n - 2 i k u on the interface sides (A6; eq. (2), sign per reading R3)
#pragma unroll
  for (int b = 0; b < N1; ++b)
#pragma unroll
    for (int a = 0; a < N1; ++a) {
      if ((a == P && fx != exl - 1) || (b == P && fy != eyl - 1)) continue;
      const int i = fx * P + a, j = fy * P + b;
      A.u_sub[(size_t)l * 2 * NS + (size_t)j * lnx + i] = ur[b][a];
      A.u_sub[(size_t)l * 2 * NS + NS + (size_t)j * lnx + i] = ui[b][a];
      int side[2], idx[2], ns = 0;
      if (i == 0 && six > 0) { side[ns] = kSideW; idx[ns++] = j; }
      if (i == lnxl - 1 && six < A.sx - 1) { side[ns] = kSideE; idx[ns++] = j; }
      if (j == 0 && siy > 0) { side[ns] = kSideS; idx[ns++] = i; }
      if (j == lnyl - 1 && siy < A.sy - 1) { side[ns] = kSideN; idx[ns++] = i; }
      for (int k = 0; k < ns; ++k) {
        const real k2 = A.k2edge[ebase + side[k] * A.E + idx[k]];
        const size_t o = lbase + (size_t)(side[k] * 2) * A.E + idx[k];
        A.gout[o] = fmaT(k2, ui[b][a], -A.lam[o]);
        A.gout[o + A.E] = fmaT(-k2, ur[b][a], -A.lam[o + A.E]);
      }
    }
}

}  // namespace hz
