// hz_line.cuh — device helpers shared by the sweep kernels: FMA wrapper, the named barrier, the 1-D line
// operators of the register-blocked kernels (own part / neighbour part / outgoing partial sum) and the
// 128-bit access to 16-byte-aligned record chunks.
#pragma once
#include "hz_internal.h"

namespace hz {

template <typename real>
__device__ __forceinline__ real fmaT(real a, real b, real c);
template <>
__device__ __forceinline__ float fmaT<float>(float a, float b, float c) { return fmaf(a, b, c); }
template <>
__device__ __forceinline__ double fmaT<double>(double a, double b, double c) { return fma(a, b, c); }

// Two fp32 values in one aligned register pair, operated on by the packed sm_100 instruction FFMA2 (one issue slot
// for two IEEE round-to-nearest FMAs, each half bit-identical to the scalar FFMA).  mk2 / un2 are register
// renamings; mk2(x, x) becomes a broadcast operand of the instruction (no copy).
struct f2 {
  unsigned long long v;
};
__device__ __forceinline__ f2 mk2(float lo, float hi) {
  f2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void un2(f2 a, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v)); }
template <>
__device__ __forceinline__ f2 fmaT<f2>(f2 a, f2 b, f2 c) {
  f2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v));
  return r;
}
__device__ __forceinline__ f2 operator*(f2 a, f2 b) {
  f2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
  return r;
}

__device__ __forceinline__ void bar_sync_all(int nthreads) {
  asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory");
}

// One line of T = M*P owned nodes q[0..T-1] plus q[T] (first node of the next tile along the line):
// S[n] (+)= (assembled 1-D operator row n) . q, using the incoming partial `pin` for node 0.
// k: Elem1D coefficients of this direction.  d0/s0: diagonal and scale of node 0 (one-sided at the ends).
template <typename real, int P, int M, bool ACC, typename KT>
__device__ __forceinline__ void line_apply(const real (&q)[M * P + 1], real pin, real d0, real s0, const KT &k,
                                           real (&S)[M * P]) {
  {
    real T = fmaT(d0, q[0], pin);
#pragma unroll
    for (int c = 1; c <= P; ++c) T = fmaT(k.k0[c], q[c], T);
    S[0] = ACC ? fmaT(s0, T, S[0]) : s0 * T;
  }
#pragma unroll
  for (int e = 0; e < M; ++e) {
#pragma unroll
    for (int a = 1; a < P; ++a) {
      real T = ACC ? fmaT(k.kin[a][0], q[e * P], S[e * P + a]) : k.kin[a][0] * q[e * P];
#pragma unroll
      for (int c = 1; c <= P; ++c) T = fmaT(k.kin[a][c], q[e * P + c], T);
      S[e * P + a] = T;
    }
    if (e > 0) {
      real T = ACC ? fmaT(k.k0[0] + k.kp[P], q[e * P], S[e * P]) : (k.k0[0] + k.kp[P]) * q[e * P];
#pragma unroll
      for (int c = 0; c < P; ++c) T = fmaT(k.kp[c], q[(e - 1) * P + c], T);
#pragma unroll
      for (int c = 1; c <= P; ++c) T = fmaT(k.k0[c], q[e * P + c], T);
      S[e * P] = T;
    }
  }
}

// Own-only part of one tile line (no neighbour data): S[n] (+)= terms over q[0..T-1] for n >= 1; returns the
// unscaled own part of node 0.
template <typename real, int P, int M, bool ACC, typename KT>
__device__ __forceinline__ real line_own(const real (&q)[M * P + 1], real d0, const KT &k, real (&S)[M * P]) {
  constexpr int T = M * P;
  real t0 = d0 * q[0];
#pragma unroll
  for (int c = 1; c <= P; ++c)
    if (c < T) t0 = fmaT(k.k0[c], q[c], t0);
#pragma unroll
  for (int e = 0; e < M; ++e) {
#pragma unroll
    for (int a = 1; a < P; ++a) {
      real t = ACC ? fmaT(k.kin[a][0], q[e * P], S[e * P + a]) : k.kin[a][0] * q[e * P];
#pragma unroll
      for (int c = 1; c <= P; ++c)
        if (e * P + c < T) t = fmaT(k.kin[a][c], q[e * P + c], t);
      S[e * P + a] = t;
    }
    if (e > 0) {
      real t = ACC ? fmaT(k.k0[0] + k.kp[P], q[e * P], S[e * P]) : (k.k0[0] + k.kp[P]) * q[e * P];
#pragma unroll
      for (int c = 0; c < P; ++c) t = fmaT(k.kp[c], q[(e - 1) * P + c], t);
#pragma unroll
      for (int c = 1; c <= P; ++c)
        if (e * P + c < T) t = fmaT(k.k0[c], q[e * P + c], t);
      S[e * P] = t;
    }
  }
  return t0;
}
// Neighbour part: qT = first node of the next tile along the line, pin = partial sum from the previous tile.
template <typename real, int P, int M, bool ACC0, typename KT>
__device__ __forceinline__ void line_finish(real qT, real pin, real s0, real t0, const KT &k, real (&S)[M * P]) {
#pragma unroll
  for (int a = 1; a < P; ++a) S[(M - 1) * P + a] = fmaT(k.kin[a][P], qT, S[(M - 1) * P + a]);
  if (M == 1) t0 = fmaT(k.k0[P], qT, t0);
  else S[(M - 1) * P] = fmaT(k.k0[P], qT, S[(M - 1) * P]);
  t0 += pin;
  S[0] = ACC0 ? fmaT(s0, t0, S[0]) : s0 * t0;
}

// Vectorised access to one record chunk of N values (16-byte aligned, padded to a multiple of 16 bytes).
template <int N>
__device__ __forceinline__ void st_chunk(float *dst, const float (&v)[N]) {
#pragma unroll
  for (int i = 0; i < (N + 3) / 4; ++i) {
    float4 x;
    x.x = v[4 * i];
    x.y = 4 * i + 1 < N ? v[4 * i + 1 < N ? 4 * i + 1 : 0] : 0.f;
    x.z = 4 * i + 2 < N ? v[4 * i + 2 < N ? 4 * i + 2 : 0] : 0.f;
    x.w = 4 * i + 3 < N ? v[4 * i + 3 < N ? 4 * i + 3 : 0] : 0.f;
    reinterpret_cast<float4 *>(dst)[i] = x;
  }
}
template <int N>
__device__ __forceinline__ void ld_chunk(const float *src, float (&v)[N]) {
#pragma unroll
  for (int i = 0; i < (N + 3) / 4; ++i) {
    const float4 x = reinterpret_cast<const float4 *>(src)[i];
    v[4 * i] = x.x;
    if (4 * i + 1 < N) v[4 * i + 1 < N ? 4 * i + 1 : 0] = x.y;
    if (4 * i + 2 < N) v[4 * i + 2 < N ? 4 * i + 2 : 0] = x.z;
    if (4 * i + 3 < N) v[4 * i + 3 < N ? 4 * i + 3 : 0] = x.w;
  }
}
template <int N>
__device__ __forceinline__ void st_chunk(double *dst, const double (&v)[N]) {
#pragma unroll
  for (int i = 0; i < (N + 1) / 2; ++i) {
    double2 x;
    x.x = v[2 * i];
    x.y = 2 * i + 1 < N ? v[2 * i + 1 < N ? 2 * i + 1 : 0] : 0.0;
    reinterpret_cast<double2 *>(dst)[i] = x;
  }
}
template <int N>
__device__ __forceinline__ void ld_chunk(const double *src, double (&v)[N]) {
#pragma unroll
  for (int i = 0; i < (N + 1) / 2; ++i) {
    const double2 x = reinterpret_cast<const double2 *>(src)[i];
    v[2 * i] = x.x;
    if (2 * i + 1 < N) v[2 * i + 1 < N ? 2 * i + 1 : 0] = x.y;
  }
}

template <typename real, int P, int M, typename KT>
__device__ __forceinline__ real line_partial(const real (&q)[M * P + 1], const KT &k) {
  real s = k.kp[0] * q[(M - 1) * P];
#pragma unroll
  for (int c = 1; c < P; ++c) s = fmaT(k.kp[c], q[(M - 1) * P + c], s);
  return s;
}

}  // namespace hz
