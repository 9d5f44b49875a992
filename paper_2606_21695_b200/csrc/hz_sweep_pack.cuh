// hz_sweep_pack.cuh — SEVERAL SMALL SUBDOMAINS PER THREAD BLOCK (config 5: 25 .. 289-DOF subdomains, PAPER.md:231,
// the B = 256, T = 1 corner of the paper's sweep; "several subdomains per warp/block needed").
//
// A 25-DOF subdomain is 1 full thread tile + 3 edge pieces at p = 1: one block per subdomain leaves most lanes of its
// two warps idle and pays the block's fixed costs 2.4 million times.  Here a block holds G subdomains: the full
// tiles of ALL of them fill the "bulk" warps (lane h -> subdomain h / NB, tile h % NB), the one-line edge pieces of
// all of them fill the "edge" warps, so the roles stay warp-uniform as in k_sweep_ws (hz_sweep_ws.cuh) and the
// lanes are dense.  Same arithmetic, same exchange-record protocol, same association of every sum as k_sweep_ws
// (bit-identical results); what changes is the indexing: every subdomain has its own compact slice of shared
// memory (ntx*nty records + one zero record + the along-the-edge arrays) and the per-node global arrays use the
// unrounded tile count as their stride (Layout::NT = ntx*nty), so a 25-DOF subdomain occupies 36 slots, not 128.
// One named barrier per time step for the whole block: all subdomains share N_t and run in lockstep.
#pragma once
#include <type_traits>
#include "hz_line.cuh"

namespace hz {

// a product that the compiler may not contract into a following addition (keeps the corner node's sums in the
// association the piece code uses: mul, then add)
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }

// (a register cap for two blocks of 256 threads per SM gains 5-10 % on the 4-tile subdomains and loses 10-45 % on the
// 16-tile ones and in fp64: not used)
// PRE: the neighbour-independent part of a step (own-tile line sums, the cos-filter sum of Re u) runs BEFORE the block
// barrier, as in k_sweep_cw, so the wait overlaps arithmetic: faster where a subdomain has fewer than 16 full tiles
// (one or two bulk warps per block), at M = 1 and in fp64 at p = 1; slower for the 16-tile M > 1 shapes, which keep
// the order of k_sweep_ws (profiles/r02_config_sweep.md).  Same sums, same association: results are bit-identical.
// MINB > 1: register-capped instantiation for TWO 64-tile subdomains per block (4 bulk warps + ONE edge warp of 2 x 16
// pieces, instead of two blocks of 2 bulk warps + 1 half-empty edge warp each): the edge warp's instruction stream is
// then paid once per two subdomains.  In fp32 it also issues the element-wise updates as packed pairs (FFMA2), as
// k_sweep_ws does.
// Records live on a PADDED grid of (ntx + 1) x (nty + 1) per subdomain: virtual tile (tx, ty) at index (ty + 1)(ntx + 1) +
// tx + 1, column -1 and row -1 never written (zero).  Every full tile then finds its four neighbours at the same offsets
// from its own record (-1, +1, -(ntx+1), +(ntx+1) records), so the time loop keeps ONE pointer per thread (own record in
// the current buffer) instead of five; NTX > 0 fixes ntx = nty = NTX at compile time and the offsets become immediates
// of the load instructions (17 of 181 instructions per step were address arithmetic).
template <typename real, int P, int M, int MAXT, bool PRE, int MINB = 1, int NTX = 0>
__global__ void __launch_bounds__(MAXT, MINB) k_sweep_pack(const SweepArgs<real> A, const __grid_constant__ TabC<real> TC) {
  constexpr int T = M * P;
  constexpr bool PK = std::is_same<real, float>::value && MINB > 1 && T >= 2;
  constexpr int NP = PK ? T / 2 : 0;
  constexpr int V16 = 16 / (int)sizeof(real);
  constexpr int CH = (T + V16 - 1) / V16 * V16;
  constexpr int RS = 4 * CH + V16;  // record: PX | RX | PY | RY + 16 bytes (odd number of 16-byte units)
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int NTH = blockDim.x, h = threadIdx.x, G = A.pack;
  const int ntx = NTX > 0 ? NTX : A.lay.ntx, nty = NTX > 0 ? NTX : A.lay.nty, NTV = A.lay.NT, NS = A.lay.NS;
  const int lnx = A.lay.lnx, lny = A.lay.lny;
  // edge pieces per subdomain: cmerge = 1: the last top piece also owns the corner node; 0: the corner is a piece of its own
  // (which of the two is faster depends on the shape: hz_partition decides from the config-5 measurements)
  const bool cm = A.cmerge != 0;
  const int NB = (ntx - 1) * (nty - 1), NE = ntx + nty - (cm ? 2 : 1);
  // PAD (the compile-time tile grids): padded record grid; otherwise the compact grid ntx x nty with one zero record per
  // slice standing in for the missing neighbours (a 25-DOF subdomain has 4 records: padding would double its slice and
  // halve the blocks per SM)
  constexpr bool PAD = NTX > 0;
  const int NXP = PAD ? ntx + 1 : ntx, NREC = PAD ? NXP * (nty + 1) : ntx * nty;
  const int bulkW = (G * NB + 31) & ~31;         // lanes of the bulk warps
  const int NEP = (NE + 1 + V16 - 1) / V16 * V16;   // PA / RA entries: one per piece + the corner node's raw value
  const int ZR = NREC;                           // the zero record of a slice (edge pieces without a neighbour along)
  const int EAO = (NREC + 1) * RS;               // in a slice, after the records: PA[NEP] | RA[NEP]
  const int SW = EAO + 2 * NEP;                  // words per subdomain slice
  const int BUFW = G * SW + (PAD ? 2 * NXP + 3 : 1) * RS;  // per buffer: G slices + a scratch region for idle lanes
  real *xb = reinterpret_cast<real *>(smem_raw);
  const int SCRo = G * SW + (PAD ? NXP + 1 : 0) * RS;   // the scratch record: the middle of that region (its neighbour offsets stay inside)

  for (int q = h; q < 2 * BUFW; q += NTH) xb[q] = real(0);
  const real sigma = A.sigma;

  if (h < bulkW) {
    // ============================ bulk tiles: full T x T node tiles ============================
    const int g = h / NB, t = h - g * NB;
    const int l = blockIdx.x * G + g;
    const bool act = h < G * NB && l < A.L;
    const int tx = act ? t % (ntx - 1) : 0, ty = act ? t / (ntx - 1) : 0;
    const int v = ty * ntx + tx;
    real *sl = xb + (act ? g : 0) * SW;          // this subdomain's slice (buffer 0)
    const int vq = PAD ? (ty + 1) * NXP + tx + 1 : v;   // record index
    real *pMy = act ? sl + vq * RS : xb + SCRo;
    // word offsets of the four neighbour records from the own one: constants on the padded grid; on the compact grid the
    // slice's zero record stands in for a missing neighbour (idle lanes read their own scratch record)
    const int oL = PAD ? -RS : (!act ? 0 : (tx > 0 ? -RS : (ZR - vq) * RS));
    const int oR = PAD ? RS : (!act ? 0 : RS);
    const int oDn = PAD ? -NXP * RS : (!act ? 0 : (ty > 0 ? -NXP * RS : (ZR - vq) * RS));
    const int oUp = PAD ? NXP * RS : (!act ? 0 : NXP * RS);
    const bool hasL = tx > 0, hasD = ty > 0;
    const real d0x = A.ex1.k0[0] + (hasL ? A.ex1.kp[P] : real(0));
    const real d0y = A.ey1.k0[0] + (hasD ? A.ey1.kp[P] : real(0));
    const real s0x = hasL ? real(1) : real(2), s0y = hasD ? real(1) : real(2);
    const int lc = act ? l : 0;
    const int six = lc % A.sx, siy = lc / A.sx;
    const size_t lbase = (size_t)lc * 4 * 2 * A.E, ebase = (size_t)lc * 4 * A.E;

    real p[T][T], pd[T][T], vr[T][T], vi[T][T], ur[T][T], ui[T][T], gam[T][T], bbr[T][T];
    real alc[T], bic[T], alr[T], bir[T];
    const size_t base = (size_t)lc * NS + v;
#pragma unroll
    for (int b = 0; b < T; ++b)
#pragma unroll
      for (int a = 0; a < T; ++a) {
        const size_t o = base + (size_t)(b * T + a) * NTV;
        gam[b][a] = act ? A.gamma[o] : real(0);
        bbr[b][a] = act ? A.bbf_re[o] : real(0);
        ur[b][a] = (act && A.warm) ? A.u_sub[(size_t)lc * 2 * NS + (size_t)(b * T + a) * NTV + v] : real(0);
        ui[b][a] = (act && A.warm) ? A.u_sub[(size_t)lc * 2 * NS + NS + (size_t)(b * T + a) * NTV + v] : real(0);
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
    if (onW) {
#pragma unroll
      for (int b = 0; b < T; ++b) {
        const int j = ty * T + b;
        const real s = A.bs[ebase + kSideW * A.E + j];
        bbr[b][0] = fmaT(s, A.lam[lbase + (kSideW * 2 + 0) * A.E + j], bbr[b][0]);
        bic[b] = fmaT(s, A.lam[lbase + (kSideW * 2 + 1) * A.E + j], bic[b]);
      }
    }
    if (onS) {
#pragma unroll
      for (int a = 0; a < T; ++a) {
        const int i = tx * T + a;
        const real s = A.bs[ebase + kSideS * A.E + i];
        const real li_ = A.lam[lbase + (kSideS * 2 + 1) * A.E + i];
        bbr[0][a] = fmaT(s, A.lam[lbase + (kSideS * 2 + 0) * A.E + i], bbr[0][a]);
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
        for (int a = 0; a < T; ++a) {  // WaveHoltz init (readings R2, R8)
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
        {
          real *my = pMy + cur;
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
          st_chunk<T>(my + CH, oRX);
          st_chunk<T>(my + 2 * CH, oPY);
          st_chunk<T>(my + 3 * CH, oRY);
        }
        const real *mr = pMy + cur;
        const Tab4<real> tn = TC.t[nu];
        real S[T][T], X0[T], Y0[T];
        real qR[T], piL[T], qU[T], piD[T];
        if (!PRE) {
          bar_sync_all(NTH);
          ld_chunk<T>(mr + oL, piL);
          ld_chunk<T>(mr + oR + CH, qR);
          ld_chunk<T>(mr + oDn + 2 * CH, piD);
          ld_chunk<T>(mr + oUp + 3 * CH, qU);
        }
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
        if (PRE) {
          bar_sync_all(NTH);
          ld_chunk<T>(mr + oL, piL);
          ld_chunk<T>(mr + oR + CH, qR);
          ld_chunk<T>(mr + oDn + 2 * CH, piD);
          ld_chunk<T>(mr + oUp + 3 * CH, qU);
        }
        cur = BUFW - cur;
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
            const real g_ = gam[b][a], r_ = bbr[b][a];
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
        for (int a = 0; a < T; ++a) {  // eq. (7) prefactor (reading R4)
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
    // piece e < nty-1: right piece, virtual tile (ntx-1, e), nodes (lnx-1, e*T + n), "along" = y.
    // piece e >= nty-1: top piece, virtual tile (e-(nty-1), nty-1), nodes (tx*T + n, lny-1), "along" = x.
    // The corner node (lnx-1, lny-1) -- node 0 of virtual tile (ntx-1, nty-1) -- has no lane of its own: the lane of the
    // LAST top piece (tx = ntx-2) carries it as one extra node (same operations, same association as a piece of its
    // own would apply), so that a subdomain has ntx + nty - 2 pieces: 16 at 8x8 tiles, two subdomains per edge warp.
    const int eh = h - bulkW;
    const int g = eh / NE, e = eh - g * NE;
    const int l = blockIdx.x * G + g;
    const bool act = eh < G * NE && l < A.L;
    const bool top = act && e >= nty - 1;
    const int tx = !act ? 0 : (top ? e - (nty - 1) : ntx - 1);
    const int ty = !act ? 0 : (top ? nty - 1 : e);
    const int v = ty * ntx + tx;                          // slot in the per-node global arrays
    const int vq = PAD ? (ty + 1) * NXP + tx + 1 : v;     // record index
    const int ta = top ? tx : ty, nta = top ? ntx : nty;  // position / count along the line direction
    const int sc = top ? NXP : 1;                         // record stride across
    const int oRC = top ? 3 * CH : CH, oPC = top ? 2 * CH : 0;
    const bool hasP = act && ta > 0, hasN = act && ta < nta - 1;
    real *sl = xb + (act ? g : 0) * SW;
    real *scr = xb + SCRo;
    real *pRaw = act ? sl + vq * RS + oRC : scr;
    // along-the-edge exchange through the compact arrays PA[e], RA[e].  The last right piece's partial sum has one
    // reader, the corner, which reads it as a chunk: it goes to element 0 of that piece's own PY chunk.
    real *pPAout = !act ? scr : ((!top && ty == nty - 2) ? sl + vq * RS + 2 * CH : sl + EAO + e);
    real *pRAout = !act ? scr + 1 : sl + EAO + NEP + e;
    const real *pP = hasP ? sl + EAO + e - 1 : sl + ZR * RS;
    const real *pN = hasN ? sl + EAO + NEP + ((!top && ty == nty - 2) ? ntx + nty - 2 : e + 1) : sl + ZR * RS;   // RA[ntx+nty-2]: the corner node
    const real *pC = sl + (act ? vq - sc : ZR) * RS + oPC;
    const bool isLT = cm && act && top && tx == ntx - 2;  // carries the corner node
    const int vC = (nty - 1) * ntx + ntx - 1;            // the corner's virtual tile
    real *pRAc = isLT ? sl + EAO + NEP + ntx + nty - 2 : scr + 2;   // its raw value, read by the last right piece and by this lane
    const real *pCc = sl + (isLT ? (PAD ? (nty - 1) * NXP + ntx : vC - ntx) : ZR) * RS + 2 * CH;   // the last right piece's partial (element 0 of its PY chunk)
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
    const real d0c = top ? A.ey1.kp[P] : A.ex1.kp[P];
    const real s0c = real(2);
    const int lc = act ? l : 0;
    const int six = lc % A.sx, siy = lc / A.sx;
    const size_t lbase = (size_t)lc * 4 * 2 * A.E, ebase = (size_t)lc * 4 * A.E;

    real p[T], pd[T], vr[T], vi[T], ur[T], ui[T], gam[T], bbr[T], al[T], bbi[T];
    const size_t base = (size_t)lc * NS + v;
#pragma unroll
    for (int n = 0; n < T; ++n) {
      const size_t o = base + (size_t)(top ? n : n * T) * NTV;  // tile node (a=n,b=0) or (a=0,b=n)
      gam[n] = act ? A.gamma[o] : real(0);
      bbr[n] = act ? A.bbf_re[o] : real(0);
      al[n] = act ? A.alpha[o] : real(0);
      bbi[n] = (act && A.bbf_im) ? A.bbf_im[o] : real(0);
      ur[n] = (act && A.warm) ? A.u_sub[(size_t)lc * 2 * NS + (o - (size_t)lc * NS)] : real(0);
      ui[n] = (act && A.warm) ? A.u_sub[(size_t)lc * 2 * NS + NS + (o - (size_t)lc * NS)] : real(0);
    }
    const int side1 = top ? kSideN : kSideE;
    const bool on1 = act && (top ? siy < A.sy - 1 : six < A.sx - 1);
    const int len1 = top ? lnx : lny;
    int side2 = -1, idx2 = 0;
    if (act && top && tx == 0 && six > 0) { side2 = kSideW; idx2 = lny - 1; }
    if (act && top && tx == ntx - 1 && six < A.sx - 1) { side2 = kSideE; idx2 = lny - 1; }   // (the corner as a piece of its own)
    if (act && !top && ty == 0 && siy > 0) { side2 = kSideS; idx2 = lnx - 1; }
#pragma unroll
    for (int n = 0; n < T; ++n) {
      const int idx = ta * T + n;
      if (on1 && idx < len1) {
        const real s = A.bs[ebase + side1 * A.E + idx];
        bbr[n] = fmaT(s, A.lam[lbase + (side1 * 2 + 0) * A.E + idx], bbr[n]);
        bbi[n] = fmaT(s, A.lam[lbase + (side1 * 2 + 1) * A.E + idx], bbi[n]);
      }
    }
    if (side2 >= 0) {
      const real s = A.bs[ebase + side2 * A.E + idx2];
      bbr[0] = fmaT(s, A.lam[lbase + (side2 * 2 + 0) * A.E + idx2], bbr[0]);
      bbi[0] = fmaT(s, A.lam[lbase + (side2 * 2 + 1) * A.E + idx2], bbi[0]);
    }
    // the corner node: on side N (if that is an interface) at index lnx-1 and on side E at index lny-1
    real pc = 0, pdc = 0, vrc = 0, vic = 0, urc = 0, uic = 0, gamc = 0, bbrc = 0, alc_ = 0, bbic = 0;
    const size_t oC = (size_t)lc * NS + vC;
    const bool cN = isLT && siy < A.sy - 1, cE = isLT && six < A.sx - 1;
    if (isLT) {
      gamc = A.gamma[oC]; bbrc = A.bbf_re[oC]; alc_ = A.alpha[oC];
      bbic = A.bbf_im ? A.bbf_im[oC] : real(0);
      urc = A.warm ? A.u_sub[(size_t)lc * 2 * NS + vC] : real(0);
      uic = A.warm ? A.u_sub[(size_t)lc * 2 * NS + NS + vC] : real(0);
      if (cN) {
        const real s = A.bs[ebase + kSideN * A.E + lnx - 1];
        bbrc = fmaT(s, A.lam[lbase + (kSideN * 2 + 0) * A.E + lnx - 1], bbrc);
        bbic = fmaT(s, A.lam[lbase + (kSideN * 2 + 1) * A.E + lnx - 1], bbic);
      }
      if (cE) {
        const real s = A.bs[ebase + kSideE * A.E + lny - 1];
        bbrc = fmaT(s, A.lam[lbase + (kSideE * 2 + 0) * A.E + lny - 1], bbrc);
        bbic = fmaT(s, A.lam[lbase + (kSideE * 2 + 1) * A.E + lny - 1], bbic);
      }
    }
    const real d0ac = real(0) + A.ex1.kp[P];   // along x: only the element before the corner exists
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
      pc = urc;
      pdc = A.omega * (uic * A.cos_h - urc * A.sin_h);
      vrc = t0.k * pc;
      vic = t0.kh * pdc;
#pragma unroll 1
      for (int nu = 1; nu < A.n_t; ++nu) {
        real q[T + 1];
#pragma unroll
        for (int n = 0; n < T; ++n) { p[n] = fmaT(sigma, pd[n], p[n]); q[n] = p[n]; }
        q[T] = real(0);
        const real pa = line_partial<real, P, M>(q, ka);
        pPAout[cur] = pa;
        pRAout[cur] = p[0];
        st_chunk<T>(pRaw + cur, p);
        pc = fmaT(sigma, pdc, pc);
        pRAc[cur] = pc;
        bar_sync_all(NTH);
        const real qN = pN[cur], piP = pP[cur];
        real piC[T];
        ld_chunk<T>(pC + cur, piC);
        const real piCc = pCc[cur];
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
        if (isLT) {   // the corner node: along x after the last top piece (its partial `pa`), across y after the last right piece
          const real cownc = d0c * pc;
          vrc = fmaT(tn.k, pc, vrc);
          real Sc = real(2) * (mul_rn(d0ac, pc) + pa);
          Sc = fmaT(s0c, cownc + piCc, Sc);
          real x = fmaT(-gamc, Sc, bbrc * tn.c);
          x = fmaT(bbic, tn.s, x);
          pdc = fmaT(alc_, pdc, x);
          vic = fmaT(tn.kh, pdc, vic);
        }
      }
#pragma unroll
      for (int n = 0; n < T; ++n) {
        ur[n] = A.two_over_nt * vr[n];
        ui[n] = A.two_over_nt * vi[n];
      }
      urc = A.two_over_nt * vrc;
      uic = A.two_over_nt * vic;
    }
    if (isLT) {
      A.u_sub[(size_t)l * 2 * NS + vC] = urc;
      A.u_sub[(size_t)l * 2 * NS + NS + vC] = uic;
      if (cN) {
        const real k2 = A.k2edge[ebase + kSideN * A.E + lnx - 1];
        A.gout[lbase + (kSideN * 2 + 0) * A.E + lnx - 1] = fmaT(k2, uic, -A.lam[lbase + (kSideN * 2 + 0) * A.E + lnx - 1]);
        A.gout[lbase + (kSideN * 2 + 1) * A.E + lnx - 1] = fmaT(-k2, urc, -A.lam[lbase + (kSideN * 2 + 1) * A.E + lnx - 1]);
      }
      if (cE) {
        const real k2 = A.k2edge[ebase + kSideE * A.E + lny - 1];
        A.gout[lbase + (kSideE * 2 + 0) * A.E + lny - 1] = fmaT(k2, uic, -A.lam[lbase + (kSideE * 2 + 0) * A.E + lny - 1]);
        A.gout[lbase + (kSideE * 2 + 1) * A.E + lny - 1] = fmaT(-k2, urc, -A.lam[lbase + (kSideE * 2 + 1) * A.E + lny - 1]);
      }
    }
    if (act) {
#pragma unroll
      for (int n = 0; n < T; ++n) {
        const size_t o = (size_t)(top ? n : n * T) * NTV + v;
        const int idx = ta * T + n;
        if (idx < len1) {
          A.u_sub[(size_t)l * 2 * NS + o] = ur[n];
          A.u_sub[(size_t)l * 2 * NS + NS + o] = ui[n];
        }
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
