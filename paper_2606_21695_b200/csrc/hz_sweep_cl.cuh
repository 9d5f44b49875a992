// hz_sweep_cl.cuh — thread-block-CLUSTER version of the uniform register-blocked sweep kernel, for subdomains whose
// state does not fit one SM (config 4: 9409 DOF; config-5 subdomains of 32..64 elements per side).
//
// The paper keeps one subdomain on one thread block and declines to go further ("distribute each subdomain over
// several thread blocks ... we do not explore this").  On sm_90+/sm_100 a cluster of CL thread blocks on
// CL SMs with distributed shared memory is the natural unit past one block: the subdomain's thread-tile grid is cut
// into CL column strips, one per CTA; every CTA keeps its strip's p, pdot, v_r, v_i, gamma, beta b_r in REGISTERS (no
// shared-memory coefficients), publishes its exchange records in its own shared memory, and the tiles on a strip
// boundary PUSH the chunk their neighbour across the cut needs into a halo slot of the adjacent CTA's shared memory
// with st.async (DSMEM), completing transaction bytes on an mbarrier of that CTA.  Per time step a CTA therefore
// synchronises with __syncthreads (its own records) plus a wait on its own mbarrier (the halo pushes of its one or
// two neighbour CTAs): no cluster-wide barrier in the time loop (barrier.cluster with release/acquire costs a
// MEMBAR.ALL.GPU + L1 invalidate per thread per step: measured 2-3x slower), one at start and one at the end.
// Still one kernel launch per sweep, no global memory in the time loop, no atomics, no device-wide synchronisation;
// same arithmetic and record protocol as k_sweep_tile (hz_sweep_tile.cuh).
#pragma once
#include "hz_line.cuh"

namespace hz {

__device__ __forceinline__ unsigned mapa_cluster(unsigned addr, unsigned rank) {
  unsigned r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// push N values (padded to 16 bytes with zeros) to a shared::cluster address, completing bytes on a remote mbarrier
template <int N>
__device__ __forceinline__ void push_chunk(unsigned raddr, unsigned rmbar, const float (&v)[N]) {
#pragma unroll
  for (int i = 0; i < (N + 3) / 4; ++i) {
    const unsigned a = __float_as_uint(v[4 * i]);
    const unsigned b = 4 * i + 1 < N ? __float_as_uint(v[4 * i + 1 < N ? 4 * i + 1 : 0]) : 0u;
    const unsigned c = 4 * i + 2 < N ? __float_as_uint(v[4 * i + 2 < N ? 4 * i + 2 : 0]) : 0u;
    const unsigned d = 4 * i + 3 < N ? __float_as_uint(v[4 * i + 3 < N ? 4 * i + 3 : 0]) : 0u;
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.b32 [%0], {%1,%2,%3,%4}, [%5];" ::"r"(raddr + 16u * i),
                 "r"(a), "r"(b), "r"(c), "r"(d), "r"(rmbar)
                 : "memory");
  }
}
template <int N>
__device__ __forceinline__ void push_chunk(unsigned raddr, unsigned rmbar, const double (&v)[N]) {
#pragma unroll
  for (int i = 0; i < (N + 1) / 2; ++i) {
    const long long a = __double_as_longlong(v[2 * i]);
    const long long b = 2 * i + 1 < N ? __double_as_longlong(v[2 * i + 1 < N ? 2 * i + 1 : 0]) : 0ll;
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1,%2}, [%3];" ::"r"(raddr + 16u * i),
                 "l"(a), "l"(b), "r"(rmbar)
                 : "memory");
  }
}
__device__ __forceinline__ void mbar_init1(unsigned bar) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arm(unsigned bar, unsigned tx_bytes) {
  asm volatile("{ .reg .b64 st; mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1; }" ::"r"(bar), "r"(tx_bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait_parity(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n\t.reg .pred P1;\n\t"
      "HZ_MBW_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
      "@P1 bra HZ_MBD_%=;\n\t"
      "bra HZ_MBW_%=;\n\t"
      "HZ_MBD_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}

template <typename real, int P, int MX, int MY, int CL, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) k_sweep_cl(const SweepArgs<real> A, const __grid_constant__ TabC<real> TC) {
  constexpr bool CSM = false;
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
  const int t = threadIdx.x, NT = blockDim.x;
  const int l = blockIdx.x / CL, rk = blockIdx.x % CL;  // subdomain, rank of this CTA in its cluster (cluster = CL x 1 x 1)
  const int BUFW = (NT + 33) * RS;
  real *xb = reinterpret_cast<real *>(smem_raw);
  real *csm = xb;  // unused (coefficients are registers)
  // after the two record buffers: per buffer the halo slots haloL[nty][CHY] | haloR[nty][CHY] that the adjacent CTAs
  // push into, then the two mbarriers (one per buffer)
  const int HS = 2 * A.lay.nty * CHY;
  real *halo = xb + 2 * BUFW;
  const unsigned mbar0 = (unsigned)__cvta_generic_to_shared(halo + 2 * HS);
  const int ntx = A.lay.ntx, nty = A.lay.nty, NS = A.lay.NS, NTV = A.lay.NT;
  const int lnx = A.lay.lnx, lny = A.lay.lny;
  // column strip of this CTA: tile columns [c0, c0 + wloc)
  const int wq = ntx / CL, wrem = ntx % CL;
  const int c0 = rk * wq + (rk < wrem ? rk : wrem), wloc = wq + (rk < wrem ? 1 : 0);
  const int wleft = wq + (rk - 1 < wrem ? 1 : 0), wright = wq + (rk + 1 < wrem ? 1 : 0);
  const bool act = t < wloc * nty;
  // threads number the strip's tiles column by column: the tiles on a strip boundary (first / last column) then sit
  // in the first / last two warps, and only those warps ever wait for the adjacent CTA's pushes
  // ... and those columns come LAST in thread order (position q of column c below): the arbiter favours the
  // highest warp index, and the boundary warps are the critical path of a step (they start it late, after the wait,
  // and their pushes release the adjacent CTA)
  const int ord = (CL == 1 || wloc < 2) ? 0 : (rk == 0 ? 0 : (rk == CL - 1 ? 1 : 2));  // 0 natural, 1 reversed, 2 column 0 moved to wloc-2
  auto pos_of = [&](int c) { return ord == 0 ? c : (ord == 1 ? wloc - 1 - c : (c == 0 ? wloc - 2 : (c == wloc - 1 ? c : c - 1))); };
  auto col_of = [&](int q) { return ord == 0 ? q : (ord == 1 ? wloc - 1 - q : (q == wloc - 2 ? 0 : (q == wloc - 1 ? q : q + 1))); };
  const int txl = act ? col_of(t / nty) : 0, ty = act ? t % nty : 0;
  const int tLn = pos_of(txl > 0 ? txl - 1 : 0) * nty + ty, tRn = pos_of(txl < wloc - 1 ? txl + 1 : txl) * nty + ty;  // records of the x neighbours
  const int tx = c0 + txl;
  const int v = tx * nty + ty;  // virtual tile index = slot in the per-node global arrays (Layout::cm = 1)
  const int ZR = NT, SCR = NT + 32;

  for (int q = t; q < 2 * BUFW + 2 * HS; q += NT) xb[q] = real(0);
  if (t == 0) {
    mbar_init1(mbar0);
    mbar_init1(mbar0 + 8);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }

  const bool hasL = act && tx > 0, hasR = act && tx < ntx - 1, hasD = act && ty > 0, hasU = act && ty < nty - 1;
  // neighbour records: own CTA's records, a halo slot fed by the adjacent CTA (strip boundary), or a zero record
  const bool remL = hasL && txl == 0, remR = hasR && txl == wloc - 1;
  const real *pL = remL ? halo + ty * CHY : xb + (hasL ? tLn : ZR + ((t - nty) & 31)) * RS + oPX;
  const real *pR = remR ? halo + (nty + ty) * CHY : xb + (hasR ? tRn : ZR + ((t + nty) & 31)) * RS + oRX;
  const real *pD = xb + (hasD ? t - 1 : ZR + ((t - 1) & 31)) * RS + oPY;
  const real *pU = xb + (hasU ? t + 1 : ZR + ((t + 1) & 31)) * RS + oRY;
  const bool wwait = __any_sync(0xffffffffu, remL || remR);  // warp-uniform: this warp reads a halo slot
  const int strL = remL ? HS : BUFW, strR = remR ? HS : BUFW;  // distance between the two buffers of that source
  // where this tile pushes for the CTA across the cut: its PX chunk to the right CTA's haloL[ty], its RX chunk to the
  // left CTA's haloR[ty]; and that CTA's mbarriers
  const unsigned hbase = (unsigned)__cvta_generic_to_shared(halo), RB = (unsigned)sizeof(real);
  const unsigned pushR = remR ? mapa_cluster(hbase + (unsigned)(ty * CHY) * RB, rk + 1) : 0u;
  const unsigned pushL = remL ? mapa_cluster(hbase + (unsigned)((nty + ty) * CHY) * RB, rk - 1) : 0u;
  const unsigned mbR = remR ? mapa_cluster(mbar0, rk + 1) : 0u, mbL = remL ? mapa_cluster(mbar0, rk - 1) : 0u;
  // bytes this CTA receives per step
  const unsigned tx_bytes = (unsigned)(((rk > 0) ? 1 : 0) + ((rk < CL - 1) ? 1 : 0)) * (unsigned)(nty * CHY) * RB;
  real *pMy = xb + (act ? t : SCR) * RS;
  // first node of the tile: one-sided at the subdomain ends (assembled weight w_0 instead of 2 w_0)
  const real d0x = (hasR ? A.ex1.k0[0] : real(0)) + (hasL ? A.ex1.kp[P] : real(0));
  const real d0y = (hasU ? A.ey1.k0[0] : real(0)) + (hasD ? A.ey1.kp[P] : real(0));
  const real s0x = (hasL && hasR) ? real(1) : real(2);
  const real s0y = (hasD && hasU) ? real(1) : real(2);

  real p[TY][TX], pd[TY][TX], vr[TY][TX], vi[TY][TX], ur[TY][TX], ui[TY][TX];
  real gam[CSM ? 1 : TY][CSM ? 1 : TX], bbr[CSM ? 1 : TY][CSM ? 1 : TX];
  real alc[TY], bic[TY], alr[TX], bir[TX];  // boundary-only data: column 0 and row 0 of the tile
  const size_t base = (size_t)l * NS + v;
#pragma unroll
  for (int b = 0; b < TY; ++b)
#pragma unroll
    for (int a = 0; a < TX; ++a) {
      const size_t o = base + (size_t)(b * TX + a) * NTV;
      const real g_ = act ? A.gamma[o] : real(0), r_ = act ? A.bbf_re[o] : real(0);
      if (CSM) {
        csm[2 * (b * TX + a)] = g_;
        csm[2 * (b * TX + a) + 1] = r_;
      } else {
        gam[CSM ? 0 : b][CSM ? 0 : a] = g_;
        bbr[CSM ? 0 : b][CSM ? 0 : a] = r_;
      }
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
  cluster_sync_all();  // every CTA's mbarriers and zeroed buffers exist before anyone pushes

  const real sigma = A.sigma;
  int cur = 0, bsel = 0;
  unsigned ph0 = 0, ph1 = 0;  // phase parities of the two mbarriers
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
        // strip boundary: push what the tile across the cut needs into the adjacent CTA's halo slot
        if (remR) push_chunk<TY>(pushR + (unsigned)(bsel * HS) * RB, mbR + 8u * bsel, vPX);
        if (remL) push_chunk<TY>(pushL + (unsigned)(bsel * HS) * RB, mbL + 8u * bsel, vRX);
      }
      if (t == 0) mbar_arm(mbar0 + 8u * bsel, tx_bytes);
      __syncthreads();
      if (wwait) mbar_wait_parity(mbar0 + 8u * bsel, bsel ? ph1 : ph0);
      if (bsel) ph1 ^= 1u;
      else ph0 ^= 1u;
      // neighbour loads first, then the part of the step that needs none of them
      real qR[TY], piL[TY], qU[TX], piD[TX];
      ld_chunk<TY>(pL + bsel * strL, piL);
      ld_chunk<TY>(pR + bsel * strR, qR);
      ld_chunk<TX>(pD + cur, piD);
      ld_chunk<TX>(pU + cur, qU);
      cur = BUFW - cur;
      bsel ^= 1;
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
  cluster_sync_all();  // no CTA may leave while a neighbour can still read its records
  // store u_l (A7) and the outgoing interface data g = -lambda^n - 2 i k u (A6; eq. (2), sign per reading R3)
#pragma unroll
  for (int b = 0; b < TY; ++b)
#pragma unroll
    for (int a = 0; a < TX; ++a) {
      if (act) {
        A.u_sub[(size_t)l * 2 * NS + (size_t)(b * TX + a) * NTV + v] = ur[b][a];
        A.u_sub[(size_t)l * 2 * NS + NS + (size_t)(b * TX + a) * NTV + v] = ui[b][a];
      }
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
