// hz_sweep_stream.cuh — streamed fallback of the sweep kernel for subdomains whose state does not fit one
// SM's registers + shared memory (e.g. config 4 in fp64: 9409 DOF x 6 values x 8 B = 452 KB; config-5
// subdomains of 64x64 elements).  Still one thread block per subdomain, one launch per sweep, no atomics and
// no device-wide synchronisation, but p, pdot, v_r, v_i live in a per-subdomain global scratch that stays
// L2-resident (the paper's pGlobal idea, applied to the whole state).  Each thread walks the
// nodes j = t, t+NT, ... of the subdomain; per time step:
//   phase A   p_new[j] = p[j] + sigma pdot[j];  v_r[j] += kappa p_new[j]            (own nodes only)
//   __syncthreads()                                                               (one barrier per step)
//   phase B   S = (Lx p_new + Ly p_new)_j from the 2(2P+1) neighbours;  pdot, v_i update
// p is double-buffered, which makes the single barrier sufficient.  Bound by L1/L2 bandwidth
// (about 26 words per DOF-step), a few per cent of the FMA peak: it exists for coverage, not for speed.
#pragma once
#include "hz_sweep.cuh"

namespace hz {

template <typename real, int P>
__global__ void __launch_bounds__(1024, 1) k_sweep_stream(const SweepArgs<real> A, real *__restrict__ scr) {
  constexpr int B = 2 * P + 1;
  const int lnx = A.lay.lnx, lny = A.lay.lny, N = lnx * lny, NS = A.lay.NS;
  const int t = threadIdx.x, NT = blockDim.x, l = blockIdx.x;
  // scratch of this subdomain: p0 | p1 | pdot | v_r | v_i | beta b_r | beta b_i
  real *p0 = scr + (size_t)l * 7 * NS, *p1 = p0 + NS, *pd = p1 + NS, *vr = pd + NS, *vi = vr + NS;
  real *bbr = vi + NS, *bbi = bbr + NS;
  real *ur = A.u_sub + (size_t)l * 2 * NS, *ui = ur + NS;
  const real *gam = A.gamma + (size_t)l * NS, *al = A.alpha + (size_t)l * NS;
  const int six = l % A.sx, siy = l / A.sx;
  const bool nbW = six > 0, nbE = six < A.sx - 1, nbS = siy > 0, nbN = siy < A.sy - 1;
  const size_t lbase = (size_t)l * 4 * 2 * A.E, ebase = (size_t)l * 4 * A.E;

  // Assemble beta b from f and lambda^n
  for (int j = t; j < N; j += NT) {
    const int i = j % lnx, jj = j / lnx;
    real br = A.bbf_re[(size_t)l * NS + j], bi = A.bbf_im ? A.bbf_im[(size_t)l * NS + j] : real(0);
    if (i == 0 && nbW) { const real s = A.bs[ebase + kSideW * A.E + jj];
      br = fmaT(s, A.lam[lbase + (kSideW * 2 + 0) * A.E + jj], br); bi = fmaT(s, A.lam[lbase + (kSideW * 2 + 1) * A.E + jj], bi); }
    if (i == lnx - 1 && nbE) { const real s = A.bs[ebase + kSideE * A.E + jj];
      br = fmaT(s, A.lam[lbase + (kSideE * 2 + 0) * A.E + jj], br); bi = fmaT(s, A.lam[lbase + (kSideE * 2 + 1) * A.E + jj], bi); }
    if (jj == 0 && nbS) { const real s = A.bs[ebase + kSideS * A.E + i];
      br = fmaT(s, A.lam[lbase + (kSideS * 2 + 0) * A.E + i], br); bi = fmaT(s, A.lam[lbase + (kSideS * 2 + 1) * A.E + i], bi); }
    if (jj == lny - 1 && nbN) { const real s = A.bs[ebase + kSideN * A.E + i];
      br = fmaT(s, A.lam[lbase + (kSideN * 2 + 0) * A.E + i], br); bi = fmaT(s, A.lam[lbase + (kSideN * 2 + 1) * A.E + i], bi); }
    bbr[j] = br;
    bbi[j] = bi;
    if (!A.warm) { ur[j] = real(0); ui[j] = real(0); }
  }
  const real sigma = A.sigma;
  real *pc = p0, *pn = p1;
  for (int m = 0; m < A.n_wh; ++m) {
    const Tab4<real> t0 = A.tab[0];
    for (int j = t; j < N; j += NT) {  // WaveHoltz init (readings R2, R8)
      const real u_r = ur[j], u_i = ui[j];
      const real pj = u_r, pdj = A.omega * (u_i * A.cos_h - u_r * A.sin_h);
      pc[j] = pj; pd[j] = pdj; vr[j] = t0.k * pj; vi[j] = t0.kh * pdj;
    }
    for (int nu = 1; nu < A.n_t; ++nu) {
      const Tab4<real> tn = A.tab[nu];
      for (int j = t; j < N; j += NT) {  // phase A
        const real pj = fmaT(sigma, pd[j], pc[j]);
        pn[j] = pj;
        vr[j] = fmaT(tn.k, pj, vr[j]);
      }
      __syncthreads();
      for (int j = t; j < N; j += NT) {  // phase B
        const int i = j % lnx, jj = j / lnx;
        real S = real(0);
#pragma unroll
        for (int d = 0; d < B; ++d) {
          const int ii = i + d - P, j2 = jj + d - P;
          if (ii >= 0 && ii < lnx) S = fmaT(A.bandx[i * B + d], pn[jj * lnx + ii], S);
          if (j2 >= 0 && j2 < lny) S = fmaT(A.bandy[jj * B + d], pn[j2 * lnx + i], S);
        }
        const real src = fmaT(bbr[j], tn.c, bbi[j] * tn.s);
        const real pdj = fmaT(al[j], pd[j], fmaT(-gam[j], S, src));
        pd[j] = pdj;
        vi[j] = fmaT(tn.kh, pdj, vi[j]);
      }
      real *sw = pc; pc = pn; pn = sw;
    }
    for (int j = t; j < N; j += NT) {  // eq. (7) prefactor (reading R4)
      ur[j] = A.two_over_nt * vr[j];
      ui[j] = A.two_over_nt * vi[j];
    }
    // the next WaveHoltz iteration's init reads only the thread's own nodes: no barrier needed here, but the
    // first phase B of that iteration must not read a pn that a slow thread still uses in this iteration's
    // last phase B: the barrier of its first step orders that.
    __syncthreads();
  }
  // outgoing interface data g = -lambda^n - 2 i k u (eq. (2); sign per reading R3)
  for (int j = t; j < N; j += NT) {
    const int i = j % lnx, jj = j / lnx;
    const real u_r = ur[j], u_i = ui[j];
    if (i == 0 && nbW) { const real k2 = A.k2edge[ebase + kSideW * A.E + jj];
      A.gout[lbase + (kSideW * 2 + 0) * A.E + jj] = fmaT(k2, u_i, -A.lam[lbase + (kSideW * 2 + 0) * A.E + jj]);
      A.gout[lbase + (kSideW * 2 + 1) * A.E + jj] = fmaT(-k2, u_r, -A.lam[lbase + (kSideW * 2 + 1) * A.E + jj]); }
    if (i == lnx - 1 && nbE) { const real k2 = A.k2edge[ebase + kSideE * A.E + jj];
      A.gout[lbase + (kSideE * 2 + 0) * A.E + jj] = fmaT(k2, u_i, -A.lam[lbase + (kSideE * 2 + 0) * A.E + jj]);
      A.gout[lbase + (kSideE * 2 + 1) * A.E + jj] = fmaT(-k2, u_r, -A.lam[lbase + (kSideE * 2 + 1) * A.E + jj]); }
    if (jj == 0 && nbS) { const real k2 = A.k2edge[ebase + kSideS * A.E + i];
      A.gout[lbase + (kSideS * 2 + 0) * A.E + i] = fmaT(k2, u_i, -A.lam[lbase + (kSideS * 2 + 0) * A.E + i]);
      A.gout[lbase + (kSideS * 2 + 1) * A.E + i] = fmaT(-k2, u_r, -A.lam[lbase + (kSideS * 2 + 1) * A.E + i]); }
    if (jj == lny - 1 && nbN) { const real k2 = A.k2edge[ebase + kSideN * A.E + i];
      A.gout[lbase + (kSideN * 2 + 0) * A.E + i] = fmaT(k2, u_i, -A.lam[lbase + (kSideN * 2 + 0) * A.E + i]);
      A.gout[lbase + (kSideN * 2 + 1) * A.E + i] = fmaT(-k2, u_r, -A.lam[lbase + (kSideN * 2 + 1) * A.E + i]); }
  }
}

}  // namespace hz
