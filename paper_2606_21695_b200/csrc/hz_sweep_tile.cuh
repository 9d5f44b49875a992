// hz_sweep_tile.cuh — register-blocked sweep kernel with rectangular thread tiles, uniform code
// (no warp specialisation): k = (MX*P)*(MY*P) DOFs per thread (PAPER.md:209-217 re-designed).
//
// A thread owns the "lower-left" P x P nodes of MX x MY elements; p, pdot, v_r, v_i stay in registers for
// the whole sweep, gamma_j and beta_j Re b_j too unless CSM (then they sit in shared memory, one 16-byte
// aligned strip per thread read with 128-bit loads: large subdomains whose state alone fills the register
// file).  Per time step and tile line the thread publishes one raw value and one partial sum and reads one
// of each from its 4 neighbours (see hz_sweep_ws.cuh for the protocol); the ragged last node column / row
// is an extra tile column / row whose tiles own one line (padding has gamma = 0).
// Exchange record of thread t: chunks PX[TY] | RX[TY] | PY[TX] | RY[TX], each padded to 16 bytes, the record
// padded to an odd number of 16-byte units; records NT..NT+31 are always zero, NT+32 is scratch.  CSM strip: (gamma_n, beta b_r,n) pairs.
// Used where the warp-specialised kernel (square tiles only) has no instantiation, e.g. the 6 x 3 tiles
// (k = 18) of config 4.
#pragma once
#include "hz_line.cuh"

namespace hz {

template <typename real, int P, int MX, int MY, bool CSM, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_sweep_tile(const SweepArgs<real> A, const __grid_constant__ TabC<real> TC) {
  constexpr int TX = MX * P, TY = MY * P, KT = TX * TY;
  constexpr int V16 = 16 / (int)sizeof(real);
  constexpr int CHX = (TX + V16 - 1) / V16 * V16, CHY = (TY + V16 - 1) / V16 * V16;
  constexpr int RS0 = 2 * CHX + 2 * CHY;
  constexpr int RS = ((RS0 / V16) % 2 == 0) ? RS0 + V16 : RS0;  // odd number of 16-byte units
  constexpr int CS0 = (2 * KT + V16 - 1) / V16 * V16;            // CSM strip: (gamma_n, beta b_r,n) pairs
  constexpr int CST = ((CS0 / V16) % 2 == 0) ? CS0 + V16 : CS0;  // stride per thread, odd number of 16-byte units
  constexpr int GRP = V16 / 2;                                   // nodes per 16-byte load of the strip
  constexpr int oPX = 0, oRX = CHY, oPY = 2 * CHY, oRY = 2 * CHY + CHX;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int t = threadIdx.x, NT = blockDim.x, l = blockIdx.x;
  const int BUFW = (NT + 33) * RS;
  real *xb = reinterpret_cast<real *>(smem_raw);
  real *csm = xb + 2 * BUFW + (size_t)t * CST;  // this thread's strip
  const int ntx = A.lay.ntx, nty = A.lay.nty, NS = A.lay.NS;
  const int lnx = A.lay.lnx, lny = A.lay.lny;
  const bool act = t < ntx * nty;
  const int tx = act ? t % ntx : 0, ty = act ? t / ntx : 0;
  const int ZR = NT, SCR = NT + 32;

  for (int q = t; q < 2 * BUFW; q += NT) xb[q] = real(0);

  const bool hasL = act && tx > 0, hasR = act && tx < ntx - 1, hasD = act && ty > 0, hasU = act && ty < nty - 1;
  const real *pL = xb + (hasL ? t - 1 : ZR + ((t - 1) & 31)) * RS + oPX;
  const real *pR = xb + (hasR ? t + 1 : ZR + ((t + 1) & 31)) * RS + oRX;
  const real *pD = xb + (hasD ? t - ntx : ZR + ((t - ntx) & 31)) * RS + oPY;
  const real *pU = xb + (hasU ? t + ntx : ZR + ((t + ntx) & 31)) * RS + oRY;
  real *pMy = xb + (act ? t : SCR) * RS;
  // first node of the tile: one-sided at the subdomain ends (assembled weight w_0 instead of 2 w_0)
  const real d0x = (hasR ? A.ex1.k0[0] : real(0)) + (hasL ? A.ex1.kp[P] : real(0));
  const real d0y = (hasU ? A.ey1.k0[0] : real(0)) + (hasD ? A.ey1.kp[P] : real(0));
  const real s0x = (hasL && hasR) ? real(1) : real(2);
  const real s0y = (hasD && hasU) ? real(1) : real(2);

  real p[TY][TX], pd[TY][TX], vr[TY][TX], vi[TY][TX], ur[TY][TX], ui[TY][TX];
  real gam[CSM ? 1 : TY][CSM ? 1 : TX], bbr[CSM ? 1 : TY][CSM ? 1 : TX];
  real alc[TY], bic[TY], alr[TX], bir[TX];  // boundary-only data: column 0 and row 0 of the tile
  const size_t base = (size_t)l * NS + t;
#pragma unroll
  for (int b = 0; b < TY; ++b)
#pragma unroll
    for (int a = 0; a < TX; ++a) {
      const size_t o = base + (size_t)(b * TX + a) * NT;
      const real g_ = A.gamma[o], r_ = A.bbf_re[o];
      if (CSM) {
        csm[2 * (b * TX + a)] = g_;
        csm[2 * (b * TX + a) + 1] = r_;
      } else {
        gam[CSM ? 0 : b][CSM ? 0 : a] = g_;
        bbr[CSM ? 0 : b][CSM ? 0 : a] = r_;
      }
      ur[b][a] = A.warm ? A.u_sub[(size_t)l * 2 * NS + (size_t)(b * TX + a) * NT + t] : real(0);
      ui[b][a] = A.warm ? A.u_sub[(size_t)l * 2 * NS + NS + (size_t)(b * TX + a) * NT + t] : real(0);
    }
#pragma unroll
  for (int b = 0; b < TY; ++b) {
    const size_t o = base + (size_t)(b * TX) * NT;
    alc[b] = A.alpha[o];
    bic[b] = A.bbf_im ? A.bbf_im[o] : real(0);
  }
#pragma unroll
  for (int a = 0; a < TX; ++a) {
    const size_t o = base + (size_t)a * NT;
    alr[a] = A.alpha[o];
    bir[a] = A.bbf_im ? A.bbf_im[o] : real(0);
  }
  // Assemble b from lambda^n.  Boundary nodes are column 0 of the first/last tile column and
  // row 0 of the first/last tile row; lambda^n is re-read in the epilogue instead of being held in registers.
  const int six = l % A.sx, siy = l / A.sx;
  const size_t lbase = (size_t)l * 4 * 2 * A.E, ebase = (size_t)l * 4 * A.E;
  int sideX = -1, sideY = -1;
  if (act && tx == 0 && six > 0) sideX = kSideW;
  if (act && tx == ntx - 1 && six < A.sx - 1) sideX = kSideE;
  if (act && ty == 0 && siy > 0) sideY = kSideS;
  if (act && ty == nty - 1 && siy < A.sy - 1) sideY = kSideN;
  if (sideX >= 0) {
#pragma unroll
    for (int b = 0; b < TY; ++b) {
      const int j = ty * TY + b;
      if (j < lny) {
        const real lr_ = A.lam[lbase + (sideX * 2 + 0) * A.E + j], li_ = A.lam[lbase + (sideX * 2 + 1) * A.E + j];
        const real s = A.bs[ebase + sideX * A.E + j];
        if (CSM) csm[2 * (b * TX) + 1] = fmaT(s, lr_, csm[2 * (b * TX) + 1]);
        else bbr[CSM ? 0 : b][0] = fmaT(s, lr_, bbr[CSM ? 0 : b][0]);
        bic[b] = fmaT(s, li_, bic[b]);
      }
    }
  }
  if (sideY >= 0) {
#pragma unroll
    for (int a = 0; a < TX; ++a) {
      const int i = tx * TX + a;
      if (i < lnx) {
        const real lr_ = A.lam[lbase + (sideY * 2 + 0) * A.E + i], li_ = A.lam[lbase + (sideY * 2 + 1) * A.E + i];
        const real s = A.bs[ebase + sideY * A.E + i];
        if (CSM) csm[2 * a + 1] = fmaT(s, lr_, csm[2 * a + 1]);
        else bbr[0][CSM ? 0 : a] = fmaT(s, lr_, bbr[0][CSM ? 0 : a]);
        if (a == 0) bic[0] = fmaT(s, li_, bic[0]);
        else bir[a] = fmaT(s, li_, bir[a]);
      }
    }
  }
  __syncthreads();

  const real sigma = A.sigma;
  int cur = 0;
  for (int m = 0; m < A.n_wh; ++m) {
    const Tab4<real> t0 = TC.t[0];
#pragma unroll
    for (int b = 0; b < TY; ++b)
#pragma unroll
      for (int a = 0; a < TX; ++a) {  // WaveHoltz init (readings R2, R8)
        p[b][a] = ur[b][a];
        pd[b][a] = A.omega * (ui[b][a] * A.cos_h - ur[b][a] * A.sin_h);
        vr[b][a] = t0.k * p[b][a];
        vi[b][a] = t0.kh * pd[b][a];
      }
#pragma unroll 1
    for (int nu = 1; nu < A.n_t; ++nu) {
#pragma unroll
      for (int b = 0; b < TY; ++b)
#pragma unroll
        for (int a = 0; a < TX; ++a) p[b][a] = fmaT(sigma, pd[b][a], p[b][a]);
      {  // publish what the neighbours need
        real *my = pMy + cur;
        real vPX[TY], vRX[TY], vPY[TX], vRY[TX];
#pragma unroll
        for (int b = 0; b < TY; ++b) {
          real q[TX + 1];
#pragma unroll
          for (int a = 0; a < TX; ++a) q[a] = p[b][a];
          q[TX] = real(0);
          vPX[b] = line_partial<real, P, MX>(q, A.ex1);
          vRX[b] = p[b][0];
        }
#pragma unroll
        for (int a = 0; a < TX; ++a) {
          real q[TY + 1];
#pragma unroll
          for (int b = 0; b < TY; ++b) q[b] = p[b][a];
          q[TY] = real(0);
          vPY[a] = line_partial<real, P, MY>(q, A.ey1);
          vRY[a] = p[0][a];
        }
        st_chunk<TY>(my + oPX, vPX);
        st_chunk<TY>(my + oRX, vRX);
        st_chunk<TX>(my + oPY, vPY);
        st_chunk<TX>(my + oRY, vRY);
      }
      __syncthreads();
      // neighbour loads first, then the part of the step that needs none of them
      real qR[TY], piL[TY], qU[TX], piD[TX];
      ld_chunk<TY>(pL + cur, piL);
      ld_chunk<TY>(pR + cur, qR);
      ld_chunk<TX>(pD + cur, piD);
      ld_chunk<TX>(pU + cur, qU);
      cur = BUFW - cur;
      const Tab4<real> tn = TC.t[nu];
      real S[TY][TX], X0[TY], Y0[TX];
#pragma unroll
      for (int b = 0; b < TY; ++b) {
        real q[TX + 1];
#pragma unroll
        for (int a = 0; a < TX; ++a) q[a] = p[b][a];
        q[TX] = real(0);
        X0[b] = line_own<real, P, MX, false>(q, d0x, A.ex1, S[b]);
      }
#pragma unroll
      for (int a = 0; a < TX; ++a) {
        real q[TY + 1], Sc[TY];
#pragma unroll
        for (int b = 0; b < TY; ++b) { q[b] = p[b][a]; Sc[b] = S[b][a]; }
        q[TY] = real(0);
        if (a == 0) Y0[a] = line_own<real, P, MY, false>(q, d0y, A.ey1, Sc);
        else Y0[a] = line_own<real, P, MY, true>(q, d0y, A.ey1, Sc);
#pragma unroll
        for (int b = 1; b < TY; ++b) S[b][a] = Sc[b];
      }
#pragma unroll
      for (int b = 0; b < TY; ++b)
#pragma unroll
        for (int a = 0; a < TX; ++a) vr[b][a] = fmaT(tn.k, p[b][a], vr[b][a]);
#pragma unroll
      for (int b = 0; b < TY; ++b) {
        if (b == 0) line_finish<real, P, MX, false>(qR[b], piL[b], s0x, X0[b], A.ex1, S[b]);
        else line_finish<real, P, MX, true>(qR[b], piL[b], s0x, X0[b], A.ex1, S[b]);
      }
#pragma unroll
      for (int a = 0; a < TX; ++a) {
        real Sc[TY];
#pragma unroll
        for (int b = 0; b < TY; ++b) Sc[b] = S[b][a];
        line_finish<real, P, MY, true>(qU[a], piD[a], s0y, Y0[a], A.ey1, Sc);
#pragma unroll
        for (int b = 0; b < TY; ++b) S[b][a] = Sc[b];
      }
      // pdot, filter; CSM: gamma / beta b_r come in 16-byte groups from this thread's strip
      real gr[V16];
#pragma unroll
      for (int n = 0; n < KT; ++n) {
        const int b = n / TX, a = n % TX;
        if (CSM && n % GRP == 0) ld_chunk<V16>(csm + 2 * n, gr);
        const real g_ = CSM ? gr[2 * (n % GRP)] : gam[CSM ? 0 : b][CSM ? 0 : a];
        const real r_ = CSM ? gr[2 * (n % GRP) + 1] : bbr[CSM ? 0 : b][CSM ? 0 : a];
        if (a == 0) {
          const real x = fmaT(bic[b], tn.s, fmaT(-g_, S[b][a], r_ * tn.c));
          pd[b][a] = fmaT(alc[b], pd[b][a], x);
        } else if (b == 0) {
          const real x = fmaT(bir[a], tn.s, fmaT(-g_, S[b][a], r_ * tn.c));
          pd[b][a] = fmaT(alr[a], pd[b][a], x);
        } else {  // interior of the subdomain: alpha = 1, Im b = 0
          pd[b][a] = fmaT(r_, tn.c, fmaT(-g_, S[b][a], pd[b][a]));
        }
        vi[b][a] = fmaT(tn.kh, pd[b][a], vi[b][a]);
      }
    }
#pragma unroll
    for (int b = 0; b < TY; ++b)
#pragma unroll
      for (int a = 0; a < TX; ++a) {  // eq. (7) prefactor (reading R4)
        ur[b][a] = A.two_over_nt * vr[b][a];
        ui[b][a] = A.two_over_nt * vi[b][a];
      }
  }
  // store u_l (A7) and the outgoing interface data g = -lambda^n - 2 i k u (A6; eq. (2), sign per reading R3)
#pragma unroll
  for (int b = 0; b < TY; ++b)
#pragma unroll
    for (int a = 0; a < TX; ++a) {
      A.u_sub[(size_t)l * 2 * NS + (size_t)(b * TX + a) * NT + t] = ur[b][a];
      A.u_sub[(size_t)l * 2 * NS + NS + (size_t)(b * TX + a) * NT + t] = ui[b][a];
    }
  if (sideX >= 0) {
#pragma unroll
    for (int b = 0; b < TY; ++b) {
      const int j = ty * TY + b;
      if (j < lny) {
        const real k2 = A.k2edge[ebase + sideX * A.E + j];
        A.gout[lbase + (sideX * 2 + 0) * A.E + j] = fmaT(k2, ui[b][0], -A.lam[lbase + (sideX * 2 + 0) * A.E + j]);
        A.gout[lbase + (sideX * 2 + 1) * A.E + j] = fmaT(-k2, ur[b][0], -A.lam[lbase + (sideX * 2 + 1) * A.E + j]);
      }
    }
  }
  if (sideY >= 0) {
#pragma unroll
    for (int a = 0; a < TX; ++a) {
      const int i = tx * TX + a;
      if (i < lnx) {
        const real k2 = A.k2edge[ebase + sideY * A.E + i];
        A.gout[lbase + (sideY * 2 + 0) * A.E + i] = fmaT(k2, ui[0][a], -A.lam[lbase + (sideY * 2 + 0) * A.E + i]);
        A.gout[lbase + (sideY * 2 + 1) * A.E + i] = fmaT(-k2, ur[0][a], -A.lam[lbase + (sideY * 2 + 1) * A.E + i]);
      }
    }
  }
}

}  // namespace hz
