// hz_sweep_ws.cuh — warp-specialised register-blocked sweep kernel (square thread tiles, MX = MY = M).
//
// Same arithmetic and the same shared-memory exchange protocol as k_sweep_tile (hz_sweep.cuh), but the
// (ntx-1) x (nty-1) "bulk" tiles, which own full (M*P)^2 node tiles, run in their own warps, and the
// ntx + nty - 1 ragged tiles on the far edges (last node column / last node row of the subdomain, which
// own only one line of M*P nodes) are packed one per lane into separate "edge" warps that run a
// line-only code path.  In k_sweep_tile the ragged tiles execute the full-tile instruction stream on
// padding (28 % of the issue slots at 8x8 elements, p = 3); here they cost a fraction of a warp.
//
// Exchange records: virtual tile v = ty*ntx + tx owns record v = four 16-byte-aligned chunks PX[b] | RX[b] |
// PY[a] | RY[a] plus 16 bytes of padding (an odd number of 16-byte units, so 8 lane-consecutive records are
// conflict-free for the 128-bit accesses used: one LDS.128 / STS.128 per chunk).
//   PX[b]  partial sum  sum_{c<P} kp_x[c] p[b][last element, c]   (what the right neighbour's first column needs)
//   RX[b]  raw p[b][0]                                           (what the left neighbour's last element needs)
//   PY[a], RY[a] the same along y.  An edge piece uses element 0 of the chunks of its "along" direction.
// Records NTV..NTV+31 are always zero (missing neighbours, same bank group as the record they stand in for),
// NTV+32..NTV+63 are write-only scratch for idle lanes.  Two buffers (ping-pong), one named barrier per step.
#pragma once
#include <type_traits>
#include "hz_line.cuh"

#ifndef HZ_WS_PACK
#define HZ_WS_PACK 1
#endif

namespace hz {

template <typename real, int P, int M, bool CSM, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_sweep_ws(const SweepArgs<real> A, const __grid_constant__ TabC<real> TC) {
  constexpr int T = M * P, KT = T * T;
  // fp32, register-capped instantiation (MINB > 1: the one hz_partition picks when the grid fills the GPU, i.e. the
  // issue-bound case): the element-wise updates p += sigma p-dot, v_r += kappa p, v_i += kappa' p-dot of the node
  // columns (2j, 2j+1) of a bulk tile run as packed pairs (FFMA2: one issue slot, two round-to-nearest FMAs, each
  // half bit-identical to the scalar FFMA); an odd last column stays scalar.  Measured: config 3
  // 1.279 -> 1.259 ms per sweep; on the latency-bound config 2 (256 blocks) packing is 6 % slower, and packing the
  // y-direction lines or the p-dot update as well is slower everywhere, hence this scope.
  constexpr bool PK = HZ_WS_PACK && std::is_same<real, float>::value && !CSM && MINB > 1 && T >= 2;
  constexpr int NP = PK ? T / 2 : 0;
  constexpr bool PRE = MINB > 1;  // own-only work before the barrier (see the time loop)
  // record = 4 chunks PX | RX | PY | RY of CH values each (T padded to 16 bytes) + 16 bytes of padding, so the
  // stride is an odd number of 16-byte units: lane-consecutive records are conflict-free for 128-bit accesses
  constexpr int V16 = 16 / (int)sizeof(real);
  constexpr int CH = (T + V16 - 1) / V16 * V16;
  constexpr int RS = 4 * CH + V16;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int NTH = blockDim.x, l = blockIdx.x;
  // Warp-role order.  Roles are a function of the VIRTUAL thread index h; worder permutes the physical warps
  // so that the bulk warps of consecutive blocks spread evenly over the 4 SM sub-partitions (hardware warp slot
  // mod 4): 1 = the first edge warp sits at physical warp 1, 2 = at physical warp 0.
  int wv_ = threadIdx.x >> 5;
  {
    const int nw_ = NTH >> 5;
    if (A.worder == 1 && nw_ >= 3) wv_ = (wv_ == 1) ? nw_ - 1 : (wv_ == nw_ - 1 ? 1 : wv_);
    else if (A.worder == 2) wv_ = (wv_ == 0) ? nw_ - 1 : wv_ - 1;
  }
  const int h = (wv_ << 5) | (threadIdx.x & 31);
  const int ntx = A.lay.ntx, nty = A.lay.nty, NTV = A.lay.NT, NS = A.lay.NS;
  const int lnx = A.lay.lnx, lny = A.lay.lny;
  const int w = ntx - 1, nbulk = (ntx - 1) * (nty - 1), nedge = ntx + nty - 1;
  const int bulk_warps = (nbulk + 31) >> 5;
  const int ZR = NTV, SCR = NTV + 32;  // zero records, scratch records
  const int NE32 = (nedge + 31) & ~31;
  const int EAO = (NTV + 64) * RS;     // per buffer, after the records: PA[NE32] | RA[NE32], the edge pieces'
  const int BUFW = EAO + 2 * NE32;     // along-the-edge partial sums and raw values, indexed by edge lane
  real *xb = reinterpret_cast<real *>(smem_raw);
  real *csm = xb + 2 * BUFW;  // CSM: [2][KT][NTH] gamma | beta b_r of the bulk tiles
  const int warp = h >> 5, lane = h & 31;

  for (int q = h; q < 2 * BUFW; q += NTH) xb[q] = real(0);

  const int six = l % A.sx, siy = l / A.sx;
  const size_t lbase = (size_t)l * 4 * 2 * A.E, ebase = (size_t)l * 4 * A.E;
  const real sigma = A.sigma;

  if (warp < bulk_warps) {
    // ============================ bulk tiles: full T x T node tiles ============================
    const bool act = h < nbulk;
    const int tx = act ? h % (ntx - 1) : 0, ty = act ? h / (ntx - 1) : 0;
    const int v = ty * ntx + tx;
    const int rMy = act ? v : SCR;
    const int rL = (act && tx > 0) ? v - 1 : ZR + ((v - 1) & 31);
    const int rR = act ? v + 1 : ZR + ((v + 1) & 31);
    const int rD = (act && ty > 0) ? v - ntx : ZR + ((v - ntx) & 31);
    const int rU = act ? v + ntx : ZR + ((v + ntx) & 31);
    const real *pL = xb + rL * RS, *pR = xb + rR * RS, *pD = xb + rD * RS, *pU = xb + rU * RS;
    real *pMy = xb + rMy * RS;
    real *pMyRX = pMy + CH;
    const bool hasL = tx > 0, hasD = ty > 0;
    const real d0x = A.ex1.k0[0] + (hasL ? A.ex1.kp[P] : real(0));
    const real d0y = A.ey1.k0[0] + (hasD ? A.ey1.kp[P] : real(0));
    const real s0x = hasL ? real(1) : real(2), s0y = hasD ? real(1) : real(2);

    real p[T][T], pd[T][T], vr[T][T], vi[T][T], ur[T][T], ui[T][T];
    real gam[CSM ? 1 : T][CSM ? 1 : T], bbr[CSM ? 1 : T][CSM ? 1 : T];
    real alc[T], bic[T], alr[T], bir[T];
    const size_t base = (size_t)l * NS + v;
#pragma unroll
    for (int b = 0; b < T; ++b)
#pragma unroll
      for (int a = 0; a < T; ++a) {
        const size_t o = base + (size_t)(b * T + a) * NTV;
        const real g_ = act ? A.gamma[o] : real(0), r_ = act ? A.bbf_re[o] : real(0);
        if (CSM) {
          csm[(b * T + a) * NTH + h] = g_;
          csm[(KT + b * T + a) * NTH + h] = r_;
        } else {
          gam[CSM ? 0 : b][CSM ? 0 : a] = g_;
          bbr[CSM ? 0 : b][CSM ? 0 : a] = r_;
        }
        ur[b][a] = (act && A.warm) ? A.u_sub[(size_t)l * 2 * NS + (size_t)(b * T + a) * NTV + v] : real(0);
        ui[b][a] = (act && A.warm) ? A.u_sub[(size_t)l * 2 * NS + NS + (size_t)(b * T + a) * NTV + v] : real(0);
      }
#pragma unroll
    for (int b = 0; b < T; ++b) {
      const size_t o = base + (size_t)(b * T) * NTV;
      alc[b] = act ? A.alpha[o] : real(0);
      bic[b] = (act && A.bbf_im) ? A.bbf_im[o] : real(0);
    }
#pragma unroll
    for (int a = 0; a < T; ++a) {
      const size_t o = base + (size_t)a * NTV;
      alr[a] = act ? A.alpha[o] : real(0);
      bir[a] = (act && A.bbf_im) ? A.bbf_im[o] : real(0);
    }
    // Assemble b from lambda^n: bulk tiles touch only the W side (tx = 0) and the S side (ty = 0)
    const bool onW = act && tx == 0 && six > 0, onS = act && ty == 0 && siy > 0;
    // (lambda^n is re-read from global memory in the epilogue instead of being held in registers)
    if (onW) {
#pragma unroll
      for (int b = 0; b < T; ++b) {
        const int j = ty * T + b;
        const real lr_ = A.lam[lbase + (kSideW * 2 + 0) * A.E + j];
        const real li_ = A.lam[lbase + (kSideW * 2 + 1) * A.E + j];
        const real s = A.bs[ebase + kSideW * A.E + j];
        if (CSM) csm[(KT + b * T) * NTH + h] = fmaT(s, lr_, csm[(KT + b * T) * NTH + h]);
        else bbr[CSM ? 0 : b][0] = fmaT(s, lr_, bbr[CSM ? 0 : b][0]);
        bic[b] = fmaT(s, li_, bic[b]);
      }
    }
    if (onS) {
#pragma unroll
      for (int a = 0; a < T; ++a) {
        const int i = tx * T + a;
        const real lr_ = A.lam[lbase + (kSideS * 2 + 0) * A.E + i];
        const real li_ = A.lam[lbase + (kSideS * 2 + 1) * A.E + i];
        const real s = A.bs[ebase + kSideS * A.E + i];
        if (CSM) csm[(KT + a) * NTH + h] = fmaT(s, lr_, csm[(KT + a) * NTH + h]);
        else bbr[0][CSM ? 0 : a] = fmaT(s, lr_, bbr[0][CSM ? 0 : a]);
        if (a == 0) bic[0] = fmaT(s, li_, bic[0]);
        else bir[a] = fmaT(s, li_, bir[a]);
      }
    }
    bar_sync_all(NTH);

    int cur = 0;
    for (int m = 0; m < A.n_wh; ++m) {
      const Tab4<real> t0 = TC.t[0];
#pragma unroll
      for (int b = 0; b < T; ++b)
#pragma unroll
        for (int a = 0; a < T; ++a) {
          p[b][a] = ur[b][a];
          pd[b][a] = A.omega * (ui[b][a] * A.cos_h - ur[b][a] * A.sin_h);
          vr[b][a] = t0.k * p[b][a];
          vi[b][a] = t0.kh * pd[b][a];
        }
#pragma unroll 1
      for (int nu = 1; nu < A.n_t; ++nu) {
#pragma unroll
        for (int b = 0; b < T; ++b) {
          if constexpr (PK) {
#pragma unroll
            for (int j = 0; j < NP; ++j) {
              const int a = 2 * j;
              un2(fmaT(mk2(sigma, sigma), mk2(pd[b][a], pd[b][a + 1]), mk2(p[b][a], p[b][a + 1])), p[b][a], p[b][a + 1]);
            }
          }
#pragma unroll
          for (int a = 0; a < T; ++a)
            if (a >= 2 * NP) p[b][a] = fmaT(sigma, pd[b][a], p[b][a]);
        }
        real *my = pMy + cur, *myRX = pMyRX + cur;
        {
          real oPX[T], oRX[T], oPY[T], oRY[T];
#pragma unroll
          for (int b = 0; b < T; ++b) {
            real q[T + 1];
#pragma unroll
            for (int a = 0; a < T; ++a) q[a] = p[b][a];
            q[T] = real(0);
            oPX[b] = line_partial<real, P, M>(q, A.ex1);
            oRX[b] = p[b][0];
          }
#pragma unroll
          for (int a = 0; a < T; ++a) {
            real q[T + 1];
#pragma unroll
            for (int b = 0; b < T; ++b) q[b] = p[b][a];
            q[T] = real(0);
            oPY[a] = line_partial<real, P, M>(q, A.ey1);
            oRY[a] = p[0][a];
          }
          st_chunk<T>(my, oPX);
          st_chunk<T>(myRX, oRX);
          st_chunk<T>(my + 2 * CH, oPY);
          st_chunk<T>(my + 3 * CH, oRY);
        }
        const Tab4<real> tn = TC.t[nu];
        real S[T][T], X0[T], Y0[T];
        // the part of the step that needs no neighbour data (own terms of the line operators, v_r update).  PRE: run it
        // before the barrier, so that the skew between the warps of a block is absorbed by work instead of by waiting
        // (grid-filling instantiations: config 3 fp32 1.257 -> 1.224 ms, fp64 2.498 -> 2.415 ms); otherwise after the
        // neighbour loads are issued, where it covers their latency (config 2, one bulk warp per scheduler: 0.114 ms
        // against 0.124 ms with PRE)
        auto own_part = [&]() {
#pragma unroll
        for (int b = 0; b < T; ++b) {
          real q[T + 1];
#pragma unroll
          for (int a = 0; a < T; ++a) q[a] = p[b][a];
          q[T] = real(0);
          X0[b] = line_own<real, P, M, false>(q, d0x, A.ex1, S[b]);
        }
#pragma unroll
        for (int a = 0; a < T; ++a) {
          real q[T + 1], Sc[T];
#pragma unroll
          for (int b = 0; b < T; ++b) { q[b] = p[b][a]; Sc[b] = S[b][a]; }
          q[T] = real(0);
          if (a == 0) Y0[a] = line_own<real, P, M, false>(q, d0y, A.ey1, Sc);
          else Y0[a] = line_own<real, P, M, true>(q, d0y, A.ey1, Sc);
#pragma unroll
          for (int b = 1; b < T; ++b) S[b][a] = Sc[b];
        }
#pragma unroll
        for (int b = 0; b < T; ++b) {
          if constexpr (PK) {
#pragma unroll
            for (int j = 0; j < NP; ++j) {
              const int a = 2 * j;
              un2(fmaT(mk2(tn.k, tn.k), mk2(p[b][a], p[b][a + 1]), mk2(vr[b][a], vr[b][a + 1])), vr[b][a], vr[b][a + 1]);
            }
          }
#pragma unroll
          for (int a = 0; a < T; ++a)
            if (a >= 2 * NP) vr[b][a] = fmaT(tn.k, p[b][a], vr[b][a]);
        }
        };
        if constexpr (PRE) own_part();
        bar_sync_all(NTH);
        // issue the neighbour loads first, then do the part of the step that needs none of them
        const real *nL = pL + cur, *nR = pR + cur, *nD = pD + cur, *nU = pU + cur;
        cur = BUFW - cur;
        real qR[T], piL[T], qU[T], piD[T];
        ld_chunk<T>(nL, piL);
        ld_chunk<T>(nR + CH, qR);
        ld_chunk<T>(nD + 2 * CH, piD);
        ld_chunk<T>(nU + 3 * CH, qU);
        if constexpr (!PRE) own_part();
#pragma unroll
        for (int b = 0; b < T; ++b) {
          if (b == 0) line_finish<real, P, M, false>(qR[b], piL[b], s0x, X0[b], A.ex1, S[b]);
          else line_finish<real, P, M, true>(qR[b], piL[b], s0x, X0[b], A.ex1, S[b]);
        }
#pragma unroll
        for (int a = 0; a < T; ++a) {
          real Sc[T];
#pragma unroll
          for (int b = 0; b < T; ++b) Sc[b] = S[b][a];
          line_finish<real, P, M, true>(qU[a], piD[a], s0y, Y0[a], A.ey1, Sc);
#pragma unroll
          for (int b = 0; b < T; ++b) S[b][a] = Sc[b];
        }
#pragma unroll
        for (int b = 0; b < T; ++b)
#pragma unroll
          for (int a = 0; a < T; ++a) {
            const real g_ = CSM ? csm[(b * T + a) * NTH + h] : gam[CSM ? 0 : b][CSM ? 0 : a];
            const real r_ = CSM ? csm[(KT + b * T + a) * NTH + h] : bbr[CSM ? 0 : b][CSM ? 0 : a];
            if (a == 0) {
              const real x = fmaT(bic[b], tn.s, fmaT(-g_, S[b][a], r_ * tn.c));
              pd[b][a] = fmaT(alc[b], pd[b][a], x);
            } else if (b == 0) {
              const real x = fmaT(bir[a], tn.s, fmaT(-g_, S[b][a], r_ * tn.c));
              pd[b][a] = fmaT(alr[a], pd[b][a], x);
            } else {  // interior of the subdomain: alpha = 1, Im b = 0
              pd[b][a] = fmaT(r_, tn.c, fmaT(-g_, S[b][a], pd[b][a]));
            }
            if (a >= 2 * NP) vi[b][a] = fmaT(tn.kh, pd[b][a], vi[b][a]);
          }
        if constexpr (PK) {
#pragma unroll
          for (int b = 0; b < T; ++b)
#pragma unroll
            for (int j = 0; j < NP; ++j) {
              const int a = 2 * j;
              un2(fmaT(mk2(tn.kh, tn.kh), mk2(pd[b][a], pd[b][a + 1]), mk2(vi[b][a], vi[b][a + 1])), vi[b][a], vi[b][a + 1]);
            }
        }
      }
#pragma unroll
      for (int b = 0; b < T; ++b)
#pragma unroll
        for (int a = 0; a < T; ++a) {
          ur[b][a] = A.two_over_nt * vr[b][a];
          ui[b][a] = A.two_over_nt * vi[b][a];
        }
    }
    if (act) {
#pragma unroll
      for (int b = 0; b < T; ++b)
#pragma unroll
        for (int a = 0; a < T; ++a) {
          A.u_sub[(size_t)l * 2 * NS + (size_t)(b * T + a) * NTV + v] = ur[b][a];
          A.u_sub[(size_t)l * 2 * NS + NS + (size_t)(b * T + a) * NTV + v] = ui[b][a];
        }
    }
    if (onW) {
#pragma unroll
      for (int b = 0; b < T; ++b) {
        const int j = ty * T + b;
        const real k2 = A.k2edge[ebase + kSideW * A.E + j];
        A.gout[lbase + (kSideW * 2 + 0) * A.E + j] = fmaT(k2, ui[b][0], -A.lam[lbase + (kSideW * 2 + 0) * A.E + j]);
        A.gout[lbase + (kSideW * 2 + 1) * A.E + j] = fmaT(-k2, ur[b][0], -A.lam[lbase + (kSideW * 2 + 1) * A.E + j]);
      }
    }
    if (onS) {
#pragma unroll
      for (int a = 0; a < T; ++a) {
        const int i = tx * T + a;
        const real k2 = A.k2edge[ebase + kSideS * A.E + i];
        A.gout[lbase + (kSideS * 2 + 0) * A.E + i] = fmaT(k2, ui[0][a], -A.lam[lbase + (kSideS * 2 + 0) * A.E + i]);
        A.gout[lbase + (kSideS * 2 + 1) * A.E + i] = fmaT(-k2, ur[0][a], -A.lam[lbase + (kSideS * 2 + 1) * A.E + i]);
      }
    }
  } else {
    // ============================ edge pieces: one line of T nodes per lane ============================
    // lane e < nty-1: right piece, virtual tile (ntx-1, e), nodes (lnx-1, e*T + n), "along" = y.
    // lane e >= nty-1: top piece, virtual tile (e-(nty-1), nty-1), nodes (tx*T + n, lny-1), "along" = x;
    //                  the last one (tx = ntx-1) is the corner and owns node 0 only.
    const int e = h - 32 * bulk_warps;
    const bool act = e < (nty - 1) + ntx;
    const bool top = act && e >= nty - 1;
    const int tx = !act ? 0 : (top ? e - (nty - 1) : ntx - 1);
    const int ty = !act ? 0 : (top ? nty - 1 : e);
    const int v = ty * ntx + tx;
    const int ta = top ? tx : ty, nta = top ? ntx : nty;  // position / count along the line direction
    const int sa = top ? 1 : ntx;                         // virtual-tile stride along
    const int sc = top ? ntx : 1;                         // virtual-tile stride across
    // record field offsets: along partial / along raw / across partial (read from the bulk tile) / across raw
    const int oPA = top ? 0 : 2 * CH, oRA = top ? CH : 3 * CH, oPC = top ? 2 * CH : 0, oRC = top ? 3 * CH : CH;
    const bool hasP = act && ta > 0, hasN = act && ta < nta - 1;
    // raw values for the bulk tile across: own record (virtual tile v), chunk RX (right piece) / RY (top piece)
    real *pRaw = xb + (act ? v : SCR) * RS + oRC;
    // along-the-edge exchange through the compact arrays PA[e], RA[e] (conflict-free).  The last right piece's
    // partial sum has one reader, the corner, which reads it as a chunk: it goes to element 0 of that piece's
    // own PY chunk (whose other elements stay zero).
    real *pPAout = !act ? xb + SCR * RS : ((!top && ty == nty - 2) ? xb + v * RS + 2 * CH : xb + EAO + e);
    real *pRAout = !act ? xb + SCR * RS + 1 : xb + EAO + NE32 + e;
    const real *pP = hasP ? xb + EAO + e - 1 : xb + ZR * RS;
    const real *pN = hasN ? xb + EAO + NE32 + ((!top && ty == nty - 2) ? nedge - 1 : e + 1) : xb + ZR * RS;
    // the partial sums from the tile across: bulk tile below / left; for the corner the last right piece
    const real *pC = xb + (act ? v - sc : ZR) * RS + oPC;
    Elem1D<real> ka;  // coefficients along
#pragma unroll
    for (int c = 0; c <= P; ++c) {
      ka.k0[c] = top ? A.ex1.k0[c] : A.ey1.k0[c];
      ka.kp[c] = top ? A.ex1.kp[c] : A.ey1.kp[c];
#pragma unroll
      for (int a = 1; a < P; ++a) ka.kin[a][c] = top ? A.ex1.kin[a][c] : A.ey1.kin[a][c];
    }
    const real d0a = (hasN ? ka.k0[0] : real(0)) + (hasP ? ka.kp[P] : real(0));
    const real s0a = (hasP && hasN) ? real(1) : real(2);
    // across: the piece sits on the last node line, only the element before it exists
    const real d0c = top ? A.ey1.kp[P] : A.ex1.kp[P];
    const real s0c = real(2);

    real p[T], pd[T], vr[T], vi[T], ur[T], ui[T], gam[T], bbr[T], al[T], bbi[T];
    const size_t base = (size_t)l * NS + v;
#pragma unroll
    for (int n = 0; n < T; ++n) {
      const size_t o = base + (size_t)(top ? n : n * T) * NTV;  // tile node (a=n,b=0) or (a=0,b=n)
      gam[n] = act ? A.gamma[o] : real(0);
      bbr[n] = act ? A.bbf_re[o] : real(0);
      al[n] = act ? A.alpha[o] : real(0);
      bbi[n] = (act && A.bbf_im) ? A.bbf_im[o] : real(0);
      ur[n] = (act && A.warm) ? A.u_sub[(size_t)l * 2 * NS + (o - (size_t)l * NS)] : real(0);
      ui[n] = (act && A.warm) ? A.u_sub[(size_t)l * 2 * NS + NS + (o - (size_t)l * NS)] : real(0);
    }
    // interface sides: the whole piece lies on N (top) or E (right); node 0 may also lie on a second side
    const int side1 = top ? kSideN : kSideE;
    const bool on1 = act && (top ? siy < A.sy - 1 : six < A.sx - 1);
    const int len1 = top ? lnx : lny;
    int side2 = -1, idx2 = 0;
    if (act && top && tx == 0 && six > 0) { side2 = kSideW; idx2 = lny - 1; }
    if (act && top && tx == ntx - 1 && six < A.sx - 1) { side2 = kSideE; idx2 = lny - 1; }
    if (act && !top && ty == 0 && siy > 0) { side2 = kSideS; idx2 = lnx - 1; }
#pragma unroll
    for (int n = 0; n < T; ++n) {
      const int idx = ta * T + n;
      if (on1 && idx < len1) {
        const real lr_ = A.lam[lbase + (side1 * 2 + 0) * A.E + idx];
        const real li_ = A.lam[lbase + (side1 * 2 + 1) * A.E + idx];
        const real s = A.bs[ebase + side1 * A.E + idx];
        bbr[n] = fmaT(s, lr_, bbr[n]);
        bbi[n] = fmaT(s, li_, bbi[n]);
      }
    }
    if (side2 >= 0) {
      const real l2r = A.lam[lbase + (side2 * 2 + 0) * A.E + idx2];
      const real l2i = A.lam[lbase + (side2 * 2 + 1) * A.E + idx2];
      const real s = A.bs[ebase + side2 * A.E + idx2];
      bbr[0] = fmaT(s, l2r, bbr[0]);
      bbi[0] = fmaT(s, l2i, bbi[0]);
    }
    bar_sync_all(NTH);

    int cur = 0;
    for (int m = 0; m < A.n_wh; ++m) {
      const Tab4<real> t0 = TC.t[0];
#pragma unroll
      for (int n = 0; n < T; ++n) {
        p[n] = ur[n];
        pd[n] = A.omega * (ui[n] * A.cos_h - ur[n] * A.sin_h);
        vr[n] = t0.k * p[n];
        vi[n] = t0.kh * pd[n];
      }
#pragma unroll 1
      for (int nu = 1; nu < A.n_t; ++nu) {
        real q[T + 1];
#pragma unroll
        for (int n = 0; n < T; ++n) { p[n] = fmaT(sigma, pd[n], p[n]); q[n] = p[n]; }
        q[T] = real(0);
        real *raw = pRaw + cur;
        pPAout[cur] = line_partial<real, P, M>(q, ka);
        pRAout[cur] = p[0];
        st_chunk<T>(raw, p);
        bar_sync_all(NTH);
        const real qN = pN[cur], piP = pP[cur];
        real piC[T];
        ld_chunk<T>(pC + cur, piC);
        cur = BUFW - cur;
        const Tab4<real> tn = TC.t[nu];
        real S[T];
        const real a0 = line_own<real, P, M, false>(q, d0a, ka, S);
        real cown[T];
#pragma unroll
        for (int n = 0; n < T; ++n) { cown[n] = d0c * p[n]; vr[n] = fmaT(tn.k, p[n], vr[n]); }
        line_finish<real, P, M, false>(qN, piP, s0a, a0, ka, S);
#pragma unroll
        for (int n = 0; n < T; ++n) S[n] = fmaT(s0c, cown[n] + piC[n], S[n]);
#pragma unroll
        for (int n = 0; n < T; ++n) {
          real x = fmaT(-gam[n], S[n], bbr[n] * tn.c);
          x = fmaT(bbi[n], tn.s, x);
          pd[n] = fmaT(al[n], pd[n], x);
          vi[n] = fmaT(tn.kh, pd[n], vi[n]);
        }
      }
#pragma unroll
      for (int n = 0; n < T; ++n) {
        ur[n] = A.two_over_nt * vr[n];
        ui[n] = A.two_over_nt * vi[n];
      }
    }
    if (act) {
#pragma unroll
      for (int n = 0; n < T; ++n) {
        const size_t o = (size_t)(top ? n : n * T) * NTV + v;
        A.u_sub[(size_t)l * 2 * NS + o] = ur[n];
        A.u_sub[(size_t)l * 2 * NS + NS + o] = ui[n];
        const int idx = ta * T + n;
        if (on1 && idx < len1) {
          const real k2 = A.k2edge[ebase + side1 * A.E + idx];
          A.gout[lbase + (side1 * 2 + 0) * A.E + idx] = fmaT(k2, ui[n], -A.lam[lbase + (side1 * 2 + 0) * A.E + idx]);
          A.gout[lbase + (side1 * 2 + 1) * A.E + idx] = fmaT(-k2, ur[n], -A.lam[lbase + (side1 * 2 + 1) * A.E + idx]);
        }
      }
      if (side2 >= 0) {
        const real k2 = A.k2edge[ebase + side2 * A.E + idx2];
        A.gout[lbase + (side2 * 2 + 0) * A.E + idx2] = fmaT(k2, ui[0], -A.lam[lbase + (side2 * 2 + 0) * A.E + idx2]);
        A.gout[lbase + (side2 * 2 + 1) * A.E + idx2] = fmaT(-k2, ur[0], -A.lam[lbase + (side2 * 2 + 1) * A.E + idx2]);
      }
    }
  }
}

}  // namespace hz
