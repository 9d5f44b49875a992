// hz_sweep_cw.cuh — thread-block-CLUSTER sweep kernel with WARP-SPECIALISED edge pieces and rectangular thread tiles:
// the successor of k_sweep_cl (hz_sweep_cl.cuh) for subdomains whose state needs the registers of several SMs
// (config 4: 9409 DOF; config-5 subdomains of 32..64 elements per side).
//
// k_sweep_cl runs the 65 ragged tiles of a 33x33 tile grid through the full-tile instruction stream, leaves 5 % of its
// threads idle and spends 100 of 278 instructions per tile and time step on addressing (profiles/r01_e_*): 30.5
// thread-instructions per DOF-timestep against 22 in the single-CTA warp-specialised kernel.  Here
//   * the full TX x TY tiles of a strip of tile columns are the "bulk" lanes of a CTA, numbered column by column;
//   * the one-line pieces on the far edges are separate "edge" lanes with a line-only code path: every CTA owns the
//     "top" pieces (TX nodes along x, last node row) of its columns, the last CTA of the cluster also the "right" pieces
//     (TY nodes along y, last node column) and the corner node;
//   * tiles may be rectangular (6 x 3 nodes at p = 3, fp32: 18 DOFs per thread halve the exchange and addressing work
//     per DOF);
//   * the neighbour-independent part of a step runs in front of the CTA barrier.
// Across a strip boundary: the x-direction chunk of the boundary tile column (partial sums to the right, raw values to
// the left) and one scalar per direction between the adjacent top pieces are pushed into halo slots of the neighbour
// CTA's shared memory with st.async (DSMEM), completing transaction bytes on one of that CTA's two mbarriers; the
// readers of a halo slot wait on the mbarrier's phase.  Two halo slot sets and two mbarriers alternate (a push for
// step nu+1 cannot land in a slot step nu still reads: a CTA pushes nu+1 only after its own barrier of step nu, which
// its neighbour's halo readers of step nu-1 have passed).  barrier.cluster only at start and end.  Same arithmetic
// and association of all sums as the other register-blocked kernels; one launch per sweep, no global memory in the
// time loop, no atomics.
// Virtual tiles are numbered column by column (Layout::cm = 1): v = tx*nty + ty.
#pragma once
#include <type_traits>
#include "hz_sweep_cl.cuh"

namespace hz {

// push one value (in a 16-byte packet, the rest zero) to a shared::cluster address, completing 16 bytes on a remote mbarrier
__device__ __forceinline__ void push_scalar(unsigned raddr, unsigned rmbar, float v) {
  const float a[1] = {v};
  push_chunk<1>(raddr, rmbar, a);
}
__device__ __forceinline__ void push_scalar(unsigned raddr, unsigned rmbar, double v) {
  const double a[1] = {v};
  push_chunk<1>(raddr, rmbar, a);
}

template <typename real, int P, int MX, int MY, int CL, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_sweep_cw(const SweepArgs<real> A, const __grid_constant__ TabC<real> TC) {
  constexpr int TX = MX * P, TY = MY * P;
  constexpr int V16 = 16 / (int)sizeof(real);
  constexpr int CHX = (TX + V16 - 1) / V16 * V16, CHY = (TY + V16 - 1) / V16 * V16;
  constexpr int RS0 = 2 * CHX + 2 * CHY;
  constexpr int RS = ((RS0 / V16) % 2 == 0) ? RS0 + V16 : RS0;
  constexpr int oPX = 0, oRX = CHY, oPY = 2 * CHY, oRY = 2 * CHY + CHX;
  constexpr unsigned RB = (unsigned)sizeof(real);
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int NTH = blockDim.x, h = threadIdx.x;
  const int l = blockIdx.x / CL, rk = blockIdx.x % CL;
  const int ntx = A.lay.ntx, nty = A.lay.nty, NTV = A.lay.NT, NS = A.lay.NS;
  const int lnx = A.lay.lnx, lny = A.lay.lny;
  const int NBC = ntx - 1, NBR = nty - 1;            // columns / rows of full tiles
  const int wq = NBC / CL, wrem = NBC % CL, wmax = wq + (wrem ? 1 : 0);
  const int c0 = rk * wq + (rk < wrem ? rk : wrem), wloc = wq + (rk < wrem ? 1 : 0);
  const bool lastc = rk == CL - 1;
  const int bulkW = (wmax * NBR + 31) & ~31;          // bulk lanes (uniform over the cluster)
  const int NEL = NBR + wmax + 1;                     // edge lanes of the last CTA: right pieces | top pieces | corner
  const int NEP = (NEL + V16 - 1) / V16 * V16;
  // Records on a PADDED grid of (wmax + 2) columns x (nty + 1) rows: local tile column c at grid column c + 1, tile row t at
  // grid row t + 1; grid row 0 is never written (zero: no tile below), grid column 0 and the column after the strip are the
  // HALO columns the adjacent CTAs push into (zero where the subdomain ends; in the last CTA the column after the strip is the
  // right pieces' own).  Every full tile finds its four neighbours at the same offsets from its own record, so the time loop
  // keeps one pointer per thread (own record, current buffer) instead of five and no per-source buffer stride.
  const int NYP = nty + 1;
  const int NREC = (wmax + 2) * NYP;
  // idle lanes own the middle record of a scratch region behind the grid (their neighbour offsets stay inside it); grid record
  // (column 0, row 0) is never written and serves as the zero record
  const int SCR = NREC + NYP, ZR = 0;
  const int EAO = (NREC + 2 * NYP + 1) * RS;          // after the records: PA[NEP] | RA[NEP] of the edge lanes
  const int BUFW = EAO + 2 * NEP;
  const int HS = 2 * V16;                             // halo scalars per buffer (top pieces across a cut): PAh | RAh
  real *xb = reinterpret_cast<real *>(smem_raw);
  real *halo = xb + 2 * BUFW;
  const unsigned mbar0 = (unsigned)__cvta_generic_to_shared(halo + 2 * HS);
  const unsigned hbase = (unsigned)__cvta_generic_to_shared(halo);
  const unsigned xbase = (unsigned)__cvta_generic_to_shared(xb);
  const int oPAh = 0, oRAh = V16;
  const int wlocP = wq + (rk - 1 < wrem ? 1 : 0);    // strip width of the previous CTA
  auto recq = [&](int c, int t) { return (c + 1) * NYP + t + 1; };   // record of local tile column c, tile row t

  for (int q = h; q < 2 * BUFW + 2 * HS; q += NTH) xb[q] = real(0);
  if (h == 0) {
    mbar_init1(mbar0);
    mbar_init1(mbar0 + 8);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // bytes this CTA receives per step: one x chunk per tile row and one scalar from each adjacent CTA
  const unsigned tx_bytes = (unsigned)((rk > 0 ? 1 : 0) + (lastc ? 0 : 1)) * ((unsigned)(NBR * CHY) * RB + 16u);
  const int six = l % A.sx, siy = l / A.sx;
  const size_t lbase = (size_t)l * 4 * 2 * A.E, ebase = (size_t)l * 4 * A.E;
  const real sigma = A.sigma;

  if (h < bulkW) {
    // ============================ bulk tiles: full TX x TY node tiles of this CTA's column strip ============================
    const bool act = h < wloc * NBR;
    const int txl = act ? h / NBR : 0, ty = act ? h - txl * NBR : 0;
    const int tx = c0 + txl;
    const int v = tx * nty + ty;                      // slot in the per-node global arrays
    const int rec = recq(txl, ty);
    const bool remL = act && txl == 0 && rk > 0, remR = act && txl == wloc - 1 && !lastc;
    const bool hasL = tx > 0, hasD = ty > 0;
    real *pMy = xb + (act ? rec : SCR) * RS;
    const int oX = NYP * RS;                          // record offset of the tile column to the right / left
    const bool wwait = __any_sync(0xffffffffu, remL || remR);
    // what the tile across the cut needs goes into the adjacent CTA's halo column, at the chunk its reader loads
    const unsigned pushR = remR ? mapa_cluster(xbase + (unsigned)(recq(-1, ty) * RS + oPX) * RB, rk + 1) : 0u;
    const unsigned pushL = remL ? mapa_cluster(xbase + (unsigned)(recq(wlocP, ty) * RS + oRX) * RB, rk - 1) : 0u;
    const unsigned mbR = remR ? mapa_cluster(mbar0, rk + 1) : 0u, mbL = remL ? mapa_cluster(mbar0, rk - 1) : 0u;
    const real d0x = A.ex1.k0[0] + (hasL ? A.ex1.kp[P] : real(0));
    const real d0y = A.ey1.k0[0] + (hasD ? A.ey1.kp[P] : real(0));
    const real s0x = hasL ? real(1) : real(2), s0y = hasD ? real(1) : real(2);

    real p[TY][TX], pd[TY][TX], vr[TY][TX], vi[TY][TX], ur[TY][TX], ui[TY][TX], gam[TY][TX], bbr[TY][TX];
    real alc[TY], bic[TY], alr[TX], bir[TX];
    const size_t base = (size_t)l * NS + v;
#pragma unroll
    for (int b = 0; b < TY; ++b)
#pragma unroll
      for (int a = 0; a < TX; ++a) {
        const size_t o = base + (size_t)(b * TX + a) * NTV;
        gam[b][a] = act ? A.gamma[o] : real(0);
        bbr[b][a] = act ? A.bbf_re[o] : real(0);
        ur[b][a] = (act && A.warm) ? A.u_sub[(size_t)l * 2 * NS + (size_t)(b * TX + a) * NTV + v] : real(0);
        ui[b][a] = (act && A.warm) ? A.u_sub[(size_t)l * 2 * NS + NS + (size_t)(b * TX + a) * NTV + v] : real(0);
      }
#pragma unroll
    for (int b = 0; b < TY; ++b) {
      const size_t o = base + (size_t)(b * TX) * NTV;
      alc[b] = act ? A.alpha[o] : real(0);
      bic[b] = (act && A.bbf_im) ? A.bbf_im[o] : real(0);
    }
#pragma unroll
    for (int a = 0; a < TX; ++a) {
      const size_t o = base + (size_t)a * NTV;
      alr[a] = act ? A.alpha[o] : real(0);
      bir[a] = (act && A.bbf_im) ? A.bbf_im[o] : real(0);
    }
    // Assemble b from lambda^n: bulk tiles touch only the W side (tx = 0) and the S side (ty = 0)
    const bool onW = act && tx == 0 && six > 0, onS = act && ty == 0 && siy > 0;
    if (onW) {
#pragma unroll
      for (int b = 0; b < TY; ++b) {
        const int j = ty * TY + b;
        const real s = A.bs[ebase + kSideW * A.E + j];
        bbr[b][0] = fmaT(s, A.lam[lbase + (kSideW * 2 + 0) * A.E + j], bbr[b][0]);
        bic[b] = fmaT(s, A.lam[lbase + (kSideW * 2 + 1) * A.E + j], bic[b]);
      }
    }
    if (onS) {
#pragma unroll
      for (int a = 0; a < TX; ++a) {
        const int i = tx * TX + a;
        const real s = A.bs[ebase + kSideS * A.E + i];
        const real li_ = A.lam[lbase + (kSideS * 2 + 1) * A.E + i];
        bbr[0][a] = fmaT(s, A.lam[lbase + (kSideS * 2 + 0) * A.E + i], bbr[0][a]);
        if (a == 0) bic[0] = fmaT(s, li_, bic[0]);
        else bir[a] = fmaT(s, li_, bir[a]);
      }
    }
    __syncthreads();
    cluster_sync_all();  // every CTA's mbarriers and zeroed buffers exist before anyone pushes

    int cur = 0, bsel = 0;
    unsigned nstep = 0;   // time steps done: barrier nstep & 1 is in its phase (nstep >> 1)
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
        {
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
          // strip boundary: push what the tile across the cut needs into the adjacent CTA's halo column (same buffer)
          if (h == 0) mbar_arm(mbar0 + 8u * bsel, tx_bytes);   // (arming from the edge warp instead measured 4 % slower in fp32)
          if (remR || remL) {
            if (remR) push_chunk<TY>(pushR + (unsigned)cur * RB, mbR + 8u * bsel, vPX);
            if (remL) push_chunk<TY>(pushL + (unsigned)cur * RB, mbL + 8u * bsel, vRX);
          }
        }
        const Tab4<real> tn = TC.t[nu];
        real S[TY][TX], X0[TY], Y0[TX];
        // the neighbour-independent part of the step, in front of the barrier
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
        __syncthreads();
        if (wwait) mbar_wait_parity(mbar0 + 8u * bsel, (nstep >> 1) & 1u);
        ++nstep;
        real qR[TY], piL[TY], qU[TX], piD[TX];
        const real *mr = pMy + cur;
        ld_chunk<TY>(mr - oX + oPX, piL);
        ld_chunk<TY>(mr + oX + oRX, qR);
        ld_chunk<TX>(mr - RS + oPY, piD);
        ld_chunk<TX>(mr + RS + oRY, qU);
        cur = BUFW - cur;
        bsel ^= 1;
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
#pragma unroll
        for (int b = 0; b < TY; ++b)
#pragma unroll
          for (int a = 0; a < TX; ++a) {
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
    cluster_sync_all();  // no CTA may leave while a neighbour can still push into its halo slots
    if (act) {
#pragma unroll
      for (int b = 0; b < TY; ++b)
#pragma unroll
        for (int a = 0; a < TX; ++a) {
          A.u_sub[(size_t)l * 2 * NS + (size_t)(b * TX + a) * NTV + v] = ur[b][a];
          A.u_sub[(size_t)l * 2 * NS + NS + (size_t)(b * TX + a) * NTV + v] = ui[b][a];
        }
    }
    if (onW) {
#pragma unroll
      for (int b = 0; b < TY; ++b) {
        const int j = ty * TY + b;
        const real k2 = A.k2edge[ebase + kSideW * A.E + j];
        A.gout[lbase + (kSideW * 2 + 0) * A.E + j] = fmaT(k2, ui[b][0], -A.lam[lbase + (kSideW * 2 + 0) * A.E + j]);
        A.gout[lbase + (kSideW * 2 + 1) * A.E + j] = fmaT(-k2, ur[b][0], -A.lam[lbase + (kSideW * 2 + 1) * A.E + j]);
      }
    }
    if (onS) {
#pragma unroll
      for (int a = 0; a < TX; ++a) {
        const int i = tx * TX + a;
        const real k2 = A.k2edge[ebase + kSideS * A.E + i];
        A.gout[lbase + (kSideS * 2 + 0) * A.E + i] = fmaT(k2, ui[0][a], -A.lam[lbase + (kSideS * 2 + 0) * A.E + i]);
        A.gout[lbase + (kSideS * 2 + 1) * A.E + i] = fmaT(-k2, ur[0][a], -A.lam[lbase + (kSideS * 2 + 1) * A.E + i]);
      }
    }
  } else {
    // ============================ edge pieces ============================
    // edge lane e:  e < NBR (last CTA only): right piece r = e, tile (ntx-1, r), nodes (lnx-1, r*TY + n), along y;
    //               NBR <= e < NBR + wloc: top piece of local column e - NBR, tile (tx, nty-1), nodes (tx*TX + n, lny-1), along x;
    //               e == NBR + wloc (last CTA only): the corner, tile (ntx-1, nty-1), node 0 only, handled as a top piece.
    constexpr int TE = TX > TY ? TX : TY;
    const int e = h - bulkW;
    const bool isR = lastc && e < NBR;
    const bool isT = e >= NBR && e < NBR + wloc;
    const bool isC = lastc && e == NBR + wloc;
    const bool act = isR || isT || isC;
    const bool top = isT || isC;
    const int txl = top ? e - NBR : wloc;              // local tile column (wloc = the right pieces' column)
    const int tx = top ? c0 + txl : ntx - 1;           // (the corner: c0 + wloc = ntx - 1 in the last CTA)
    const int ty = top ? nty - 1 : (isR ? e : 0);
    const int v = tx * nty + ty;
    const int rec = recq(txl, ty);
    const int ta = top ? tx : ty, nta = top ? ntx : nty;
    const bool hasP = act && ta > 0, hasN = act && ta < nta - 1;
    // along-the-edge neighbours across a strip cut (top pieces only)
    const bool remP = isT && txl == 0 && rk > 0, remN = isT && txl == wloc - 1 && !lastc;
    real *scr = xb + SCR * RS;
    real *pRaw = act ? xb + rec * RS + (top ? oRY : oRX) : scr;
    const bool lastR = isR && ty == nty - 2;           // its along-partial has one reader, the corner, as element 0 of a PY chunk
    real *pPAout = !act ? scr : (lastR ? xb + rec * RS + oPY : xb + EAO + e);
    real *pRAout = !act ? scr + 1 : xb + EAO + NEP + e;
    const real *pP = remP ? halo + oPAh : (hasP ? xb + EAO + e - 1 : xb + ZR * RS);
    const real *pN = remN ? halo + oRAh : (hasN ? xb + EAO + NEP + (lastR ? NBR + wloc : e + 1) : xb + ZR * RS);
    const int strP = remP ? HS : BUFW, strN = remN ? HS : BUFW;
    // partial sums from the tile across: bulk tile below (its PY) / to the left (its PX); for the corner the last right piece
    const real *pC = xb + (act ? (top ? rec - 1 : rec - NYP) : ZR) * RS + (top ? oPY : oPX);
    const bool wwait = __any_sync(0xffffffffu, remP || remN);
    const unsigned pushPA = remN ? mapa_cluster(hbase + (unsigned)oPAh * RB, rk + 1) : 0u;   // my partial -> next CTA's first top piece
    const unsigned pushRA = remP ? mapa_cluster(hbase + (unsigned)oRAh * RB, rk - 1) : 0u;   // my raw p[0] -> previous CTA's last top piece
    const unsigned mbN = remN ? mapa_cluster(mbar0, rk + 1) : 0u, mbP = remP ? mapa_cluster(mbar0, rk - 1) : 0u;
    const int side1 = top ? kSideN : kSideE;
    const bool on1 = act && (top ? siy < A.sy - 1 : six < A.sx - 1);
    const int len1 = top ? lnx : lny;
    int side2 = -1, idx2 = 0;
    if (act && top && tx == 0 && six > 0) { side2 = kSideW; idx2 = lny - 1; }
    if (act && top && tx == ntx - 1 && six < A.sx - 1) { side2 = kSideE; idx2 = lny - 1; }
    if (act && !top && ty == 0 && siy > 0) { side2 = kSideS; idx2 = lnx - 1; }

    real p[TE], pd[TE], vr[TE], vi[TE], ur[TE], ui[TE], gam[TE], bbr[TE], al[TE], bbi[TE];
    const size_t base = (size_t)l * NS + v;
    const int tlen = top ? TX : TY, tstr = top ? 1 : TX;   // nodes of the piece, tile-node stride along it
#pragma unroll
    for (int n = 0; n < TE; ++n) {
      const bool in = act && n < tlen;
      const size_t o = base + (size_t)(n * tstr) * NTV;    // tile node (a=n,b=0) or (a=0,b=n)
      gam[n] = in ? A.gamma[o] : real(0);
      bbr[n] = in ? A.bbf_re[o] : real(0);
      al[n] = in ? A.alpha[o] : real(0);
      bbi[n] = (in && A.bbf_im) ? A.bbf_im[o] : real(0);
      ur[n] = (in && A.warm) ? A.u_sub[(size_t)l * 2 * NS + (o - (size_t)l * NS)] : real(0);
      ui[n] = (in && A.warm) ? A.u_sub[(size_t)l * 2 * NS + NS + (o - (size_t)l * NS)] : real(0);
      const int idx = ta * tlen + n;
      if (in && on1 && idx < len1) {
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
    const real k00 = top ? A.ex1.k0[0] : A.ey1.k0[0], kpP = top ? A.ex1.kp[P] : A.ey1.kp[P];
    const real d0a = (hasN ? k00 : real(0)) + (hasP ? kpP : real(0));
    const real s0a = (hasP && hasN) ? real(1) : real(2);
    const real d0c = top ? A.ey1.kp[P] : A.ex1.kp[P];
    const real s0c = real(2);
    __syncthreads();
    cluster_sync_all();

    // one piece of T_ nodes = ME_ elements along direction `k`: publish (before the barrier) / finish (after it)
    auto publish = [&](auto tag, const auto &k, int cur, int bsel) {
      constexpr int ME_ = decltype(tag)::value, T_ = ME_ * P;
      real q[T_ + 1];
#pragma unroll
      for (int n = 0; n < T_; ++n) { p[n] = fmaT(sigma, pd[n], p[n]); q[n] = p[n]; }
      q[T_] = real(0);
      const real pa = line_partial<real, P, ME_>(q, k);
      pPAout[cur] = pa;
      pRAout[cur] = p[0];
      real pr_[T_];
#pragma unroll
      for (int n = 0; n < T_; ++n) pr_[n] = p[n];
      st_chunk<T_>(pRaw + cur, pr_);
      if (remN) push_scalar(pushPA + (unsigned)(bsel * HS) * RB, mbN + 8u * bsel, pa);
      if (remP) push_scalar(pushRA + (unsigned)(bsel * HS) * RB, mbP + 8u * bsel, p[0]);
    };
    auto finish = [&](auto tag, const auto &k, int cur, int bsel, const Tab4<real> &tn) {
      constexpr int ME_ = decltype(tag)::value, T_ = ME_ * P;
      const real qN = pN[remN ? bsel * strN : cur], piP = pP[remP ? bsel * strP : cur];
      real piC[T_], q[T_ + 1], S[T_];
      ld_chunk<T_>(pC + cur, piC);
#pragma unroll
      for (int n = 0; n < T_; ++n) q[n] = p[n];
      q[T_] = real(0);
      const real a0 = line_own<real, P, ME_, false>(q, d0a, k, S);
      real cown[T_];
#pragma unroll
      for (int n = 0; n < T_; ++n) { cown[n] = d0c * p[n]; vr[n] = fmaT(tn.k, p[n], vr[n]); }
      line_finish<real, P, ME_, false>(qN, piP, s0a, a0, k, S);
#pragma unroll
      for (int n = 0; n < T_; ++n) S[n] = fmaT(s0c, cown[n] + piC[n], S[n]);
#pragma unroll
      for (int n = 0; n < T_; ++n) {
        real x = fmaT(-gam[n], S[n], bbr[n] * tn.c);
        x = fmaT(bbi[n], tn.s, x);
        pd[n] = fmaT(al[n], pd[n], x);
        vi[n] = fmaT(tn.kh, pd[n], vi[n]);
      }
    };
    using MXt = std::integral_constant<int, MX>;
    using MYt = std::integral_constant<int, MY>;

    int cur = 0, bsel = 0;
    unsigned nstep = 0;   // time steps done: barrier nstep & 1 is in its phase (nstep >> 1)
    for (int m = 0; m < A.n_wh; ++m) {
      const Tab4<real> t0 = TC.t[0];
#pragma unroll
      for (int n = 0; n < TE; ++n) {
        p[n] = ur[n];
        pd[n] = A.omega * (ui[n] * A.cos_h - ur[n] * A.sin_h);
        vr[n] = t0.k * p[n];
        vi[n] = t0.kh * pd[n];
      }
#pragma unroll 1
      for (int nu = 1; nu < A.n_t; ++nu) {
        if (top) publish(MXt{}, A.ex1, cur, bsel);
        else publish(MYt{}, A.ey1, cur, bsel);
        __syncwarp();   // the two piece kinds reconverge before the (aligned) block barrier
        __syncthreads();
        if (wwait) mbar_wait_parity(mbar0 + 8u * bsel, (nstep >> 1) & 1u);
        ++nstep;
        const Tab4<real> tn = TC.t[nu];
        if (top) finish(MXt{}, A.ex1, cur, bsel, tn);
        else finish(MYt{}, A.ey1, cur, bsel, tn);
        cur = BUFW - cur;
        bsel ^= 1;
      }
#pragma unroll
      for (int n = 0; n < TE; ++n) {
        ur[n] = A.two_over_nt * vr[n];
        ui[n] = A.two_over_nt * vi[n];
      }
    }
    cluster_sync_all();
    if (act) {
#pragma unroll
      for (int n = 0; n < TE; ++n) {
        const int idx = ta * tlen + n;
        if (n < tlen && idx < len1) {   // (the corner piece owns node 0 only)
          const size_t o = (size_t)(n * tstr) * NTV + v;
          A.u_sub[(size_t)l * 2 * NS + o] = ur[n];
          A.u_sub[(size_t)l * 2 * NS + NS + o] = ui[n];
          if (on1) {
            const real k2 = A.k2edge[ebase + side1 * A.E + idx];
            A.gout[lbase + (side1 * 2 + 0) * A.E + idx] = fmaT(k2, ui[n], -A.lam[lbase + (side1 * 2 + 0) * A.E + idx]);
            A.gout[lbase + (side1 * 2 + 1) * A.E + idx] = fmaT(-k2, ur[n], -A.lam[lbase + (side1 * 2 + 1) * A.E + idx]);
          }
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
