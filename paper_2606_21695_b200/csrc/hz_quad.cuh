// hz_quad.cuh — general straight-sided convex quadrilaterals on a logically rectangular mesh (
// gradient through D, geometric factors at the quadrature points, then D^T).
// Geometry of the bilinear element map, the per-subdomain operator builder for this geometry (A0), the
// per-quadrature-point geometric factors the sweep kernel keeps on chip, and the global residual (A10).
#pragma once
#include "hz_aux.cuh"

namespace hz {

struct RefQ {  // reference GLL data (fp64)
  double xi[kMaxP + 1], w[kMaxP + 1], D[kMaxP + 1][kMaxP + 1];
};

// Bilinear map of [-1,1]^2 onto the quad with vertices (x00,y00) (xi=-1,eta=-1), (x10,..) (xi=+1,eta=-1),
// (x01,..) (xi=-1,eta=+1), (x11,..).  J = d(x,y)/d(xi,eta);  g = detJ J^-1 J^-T.
struct QuadPt {
  double det, gxx, gxy, gyy;
};
__host__ __device__ inline QuadPt quad_point(const double X[4], const double Y[4], double xi, double eta) {
  const double x_xi = 0.25 * ((1.0 - eta) * (X[1] - X[0]) + (1.0 + eta) * (X[3] - X[2]));
  const double y_xi = 0.25 * ((1.0 - eta) * (Y[1] - Y[0]) + (1.0 + eta) * (Y[3] - Y[2]));
  const double x_et = 0.25 * ((1.0 - xi) * (X[2] - X[0]) + (1.0 + xi) * (X[3] - X[1]));
  const double y_et = 0.25 * ((1.0 - xi) * (Y[2] - Y[0]) + (1.0 + xi) * (Y[3] - Y[1]));
  QuadPt q;
  q.det = x_xi * y_et - x_et * y_xi;
  q.gxx = (x_et * x_et + y_et * y_et) / q.det;
  q.gxy = -(x_xi * x_et + y_xi * y_et) / q.det;
  q.gyy = (x_xi * x_xi + y_xi * y_xi) / q.det;
  return q;
}
// vertices of global element (gx, gy): index 0..3 = (0,0), (1,0), (0,1), (1,1)
__host__ __device__ inline void quad_vertices(const double *vx, const double *vy, int nx, int gx, int gy, double X[4],
                                              double Y[4]) {
  const size_t o = (size_t)gy * (nx + 1) + gx;
  X[0] = vx[o]; X[1] = vx[o + 1]; X[2] = vx[o + nx + 1]; X[3] = vx[o + nx + 2];
  Y[0] = vy[o]; Y[1] = vy[o + 1]; Y[2] = vy[o + nx + 1]; Y[3] = vy[o + nx + 2];
}

// Local lumped mass and the edge weights of node (i,j) of the region of elements [gx0, gx0+ex) x [gy0, gy0+ey)
// (a subdomain, or the whole mesh): m = sum_e w_a w_b detJ;  s[side] = sum_e w_a |edge_e| / 2 on the region's sides.
__device__ inline void quad_node_weights(const RefQ &ref, const double *vx, const double *vy, int nx, int P, int gx0,
                                         int gy0, int ex, int ey, int i, int j, double *m, double s[4]) {
  const int fx_hi = (i == ex * P) ? ex - 1 : i / P, fx_lo = (i % P == 0 && i > 0) ? i / P - 1 : fx_hi;
  const int fy_hi = (j == ey * P) ? ey - 1 : j / P, fy_lo = (j % P == 0 && j > 0) ? j / P - 1 : fy_hi;
  double mm = 0.0;
  s[0] = s[1] = s[2] = s[3] = 0.0;
  for (int fy = fy_lo; fy <= fy_hi; ++fy)
    for (int fx = fx_lo; fx <= fx_hi; ++fx) {
      double X[4], Y[4];
      quad_vertices(vx, vy, nx, gx0 + fx, gy0 + fy, X, Y);
      const int a = i - fx * P, b = j - fy * P;
      mm += ref.w[a] * ref.w[b] * quad_point(X, Y, ref.xi[a], ref.xi[b]).det;
      if (i == 0 && fx == 0) s[kSideW] += ref.w[b] * 0.5 * hypot(X[2] - X[0], Y[2] - Y[0]);
      if (i == ex * P && fx == ex - 1) s[kSideE] += ref.w[b] * 0.5 * hypot(X[3] - X[1], Y[3] - Y[1]);
      if (j == 0 && fy == 0) s[kSideS] += ref.w[a] * 0.5 * hypot(X[1] - X[0], Y[1] - Y[0]);
      if (j == ey * P && fy == ey - 1) s[kSideN] += ref.w[a] * 0.5 * hypot(X[3] - X[2], Y[3] - Y[2]);
    }
  *m = mm;
}

// ---------------------------------------------------------------------------------------------
// A0 for general quads: as k_build, with the local lumped mass and the edge weights from the geometry.
// `gamma` holds beta_j (the sweep kernel of this geometry applies the assembled stiffness itself).
// ---------------------------------------------------------------------------------------------
template <typename real>
__global__ void k_build_quad(Geo g, Layout lay, RefQ ref, const double *__restrict__ vx, const double *__restrict__ vy,
                             const double *__restrict__ c, const double *__restrict__ f_re,
                             const double *__restrict__ f_im, const double *__restrict__ bc, real *gamma, real *alpha,
                             real *bbf_re, real *bbf_im, real *k2edge, real *bs, int only_source) {
  const int N = lay.lnx * lay.lny;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= (long long)g.sx * g.sy * N) return;
  const int l = (int)(gid / N), q = (int)(gid - (long long)l * N);
  const int i = q % lay.lnx, j = q / lay.lnx;
  const int six = l % g.sx, siy = l / g.sx;
  const int exl = sub_size(g.exq, g.exr, six), eyl = sub_size(g.eyq, g.eyr, siy);  // this subdomain's elements
  const int gx0 = sub_off(g.exq, g.exr, six), gy0 = sub_off(g.eyq, g.eyr, siy);
  const int lnxl = exl * g.p + 1, lnyl = eyl * g.p + 1;
  if (i >= lnxl || j >= lnyl) return;  // padding of a ragged subdomain: stays zero
  const int I = gx0 * g.p + i, J = gy0 * g.p + j;
  const size_t gn = (size_t)J * g.npx + I;
  const double cj = c[gn];
  double m, s[4];
  quad_node_weights(ref, vx, vy, g.nx, g.p, gx0, gy0, exl, eyl, i, j, &m, s);
  const double M = m / (cj * cj);
  const double H = (s[0] + s[1] + s[2] + s[3]) / cj;  // impedance on the whole subdomain boundary
  const double den = M + g.theta * H;
  const double beta = g.sigma / den;
  double bre = f_re[gn] * m, bim = f_im ? f_im[gn] * m : 0.0;
  if (bc) {
    if (i == 0 && six == 0) { bre += s[0] * bc[(0 * 2 + 0) * g.EB + J]; bim += s[0] * bc[(0 * 2 + 1) * g.EB + J]; }
    if (i == lnxl - 1 && six == g.sx - 1) { bre += s[1] * bc[(1 * 2 + 0) * g.EB + J]; bim += s[1] * bc[(1 * 2 + 1) * g.EB + J]; }
    if (j == 0 && siy == 0) { bre += s[2] * bc[(2 * 2 + 0) * g.EB + I]; bim += s[2] * bc[(2 * 2 + 1) * g.EB + I]; }
    if (j == lnyl - 1 && siy == g.sy - 1) { bre += s[3] * bc[(3 * 2 + 0) * g.EB + I]; bim += s[3] * bc[(3 * 2 + 1) * g.EB + I]; }
  }
  const size_t o = (size_t)l * lay.NS + lay.slot(i, j);
  bbf_re[o] = (real)(beta * bre);
  if (bbf_im) bbf_im[o] = (real)(beta * bim);
  if (only_source) return;
  gamma[o] = (real)beta;
  alpha[o] = (real)((M - g.theta * H) / den);
  const size_t eb = (size_t)l * 4 * g.E;
  const double k2 = 2.0 * g.omega / cj;
  if (i == 0) { k2edge[eb + 0 * g.E + j] = (real)k2; bs[eb + 0 * g.E + j] = (real)(beta * s[0]); }
  if (i == lnxl - 1) { k2edge[eb + 1 * g.E + j] = (real)k2; bs[eb + 1 * g.E + j] = (real)(beta * s[1]); }
  if (j == 0) { k2edge[eb + 2 * g.E + i] = (real)k2; bs[eb + 2 * g.E + i] = (real)(beta * s[2]); }
  if (j == lnyl - 1) { k2edge[eb + 3 * g.E + i] = (real)k2; bs[eb + 3 * g.E + i] = (real)(beta * s[3]); }
}

// Geometric factors of every quadrature point, weights folded in: G[l][3 n + {0,1,2}][t] = w_a w_b {gxx, gxy, gyy}
// for element t = fy*ex + fx of subdomain l (ex = the maximal width: ragged subdomains leave gaps) and point
// n = b (P+1) + a; nep = element stride (threads per block).
template <typename real>
__global__ void k_build_quad_metric(Geo g, RefQ ref, const double *__restrict__ vx, const double *__restrict__ vy,
                                    int nep, real *G) {
  const int P = g.p, NQ = (P + 1) * (P + 1), ne = g.ex * g.ey;
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= (long long)g.sx * g.sy * ne * NQ) return;
  const int t = (int)(gid % ne), n = (int)((gid / ne) % NQ), l = (int)(gid / ((long long)ne * NQ));
  const int fx = t % g.ex, fy = t / g.ex, a = n % (P + 1), b = n / (P + 1);
  const int six = l % g.sx, siy = l / g.sx;
  if (fx >= sub_size(g.exq, g.exr, six) || fy >= sub_size(g.eyq, g.eyr, siy)) return;
  double X[4], Y[4];
  quad_vertices(vx, vy, g.nx, sub_off(g.exq, g.exr, six) + fx, sub_off(g.eyq, g.eyr, siy) + fy, X, Y);
  const QuadPt q = quad_point(X, Y, ref.xi[a], ref.xi[b]);
  const double ww = ref.w[a] * ref.w[b];
  real *o = G + ((size_t)l * 3 * NQ + 3 * n) * nep + t;
  o[0] = (real)(ww * q.gxx);
  o[nep] = (real)(ww * q.gxy);
  o[2 * (size_t)nep] = (real)(ww * q.gyy);
}

// ---------------------------------------------------------------------------------------------
// A10 for general quads: r = b - (A - i w H - w^2 M) u on the unpartitioned system, fp64, one thread per global
// node gathering its row of A_e u from the (up to four) elements around it.  Same reduction as k_residual.
// ---------------------------------------------------------------------------------------------
template <typename inT>
__global__ void k_residual_quad(Geo g, RefQ ref, const double *__restrict__ vx, const double *__restrict__ vy,
                                const double *__restrict__ c, const double *__restrict__ f_re,
                                const double *__restrict__ f_im, const double *__restrict__ bc,
                                const inT *__restrict__ u, double *__restrict__ part) {
  __shared__ double red[2][32];
  const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long total = (long long)g.npx * g.npy;
  double r2 = 0.0, b2 = 0.0;
  if (gid < total) {
    const int I = (int)(gid % g.npx), J = (int)(gid / g.npx);
    const int P = g.p;
    const inT *ur = u, *ui = u + total;
    const int fx_hi = (I == g.nx * P) ? g.nx - 1 : I / P, fx_lo = (I % P == 0 && I > 0) ? I / P - 1 : fx_hi;
    const int fy_hi = (J == g.ny * P) ? g.ny - 1 : J / P, fy_lo = (J % P == 0 && J > 0) ? J / P - 1 : fy_hi;
    double Ar = 0.0, Ai = 0.0;
    for (int fy = fy_lo; fy <= fy_hi; ++fy)
      for (int fx = fx_lo; fx <= fx_hi; ++fx) {
        double X[4], Y[4];
        quad_vertices(vx, vy, g.nx, fx, fy, X, Y);
        const int a = I - fx * P, b = J - fy * P;
        const size_t n0 = (size_t)(fy * P) * g.npx + fx * P;  // element node (0,0)
        // row b: sum_c D[c][a] fr(c,b);  column a: sum_c D[c][b] fs(a,c)
        for (int cc = 0; cc <= P; ++cc) {
          {  // point (cc, b)
            double uxr = 0, uxi = 0, uyr = 0, uyi = 0;
            for (int d = 0; d <= P; ++d) {
              const size_t nx_ = n0 + (size_t)b * g.npx + d, ny_ = n0 + (size_t)d * g.npx + cc;
              uxr += ref.D[cc][d] * (double)ur[nx_]; uxi += ref.D[cc][d] * (double)ui[nx_];
              uyr += ref.D[b][d] * (double)ur[ny_]; uyi += ref.D[b][d] * (double)ui[ny_];
            }
            const QuadPt q = quad_point(X, Y, ref.xi[cc], ref.xi[b]);
            const double ww = ref.w[cc] * ref.w[b] * ref.D[cc][a];
            Ar += ww * (q.gxx * uxr + q.gxy * uyr);
            Ai += ww * (q.gxx * uxi + q.gxy * uyi);
          }
          {  // point (a, cc)
            double uxr = 0, uxi = 0, uyr = 0, uyi = 0;
            for (int d = 0; d <= P; ++d) {
              const size_t nx_ = n0 + (size_t)cc * g.npx + d, ny_ = n0 + (size_t)d * g.npx + a;
              uxr += ref.D[a][d] * (double)ur[nx_]; uxi += ref.D[a][d] * (double)ui[nx_];
              uyr += ref.D[cc][d] * (double)ur[ny_]; uyi += ref.D[cc][d] * (double)ui[ny_];
            }
            const QuadPt q = quad_point(X, Y, ref.xi[a], ref.xi[cc]);
            const double ww = ref.w[a] * ref.w[cc] * ref.D[cc][b];
            Ar += ww * (q.gxy * uxr + q.gyy * uyr);
            Ai += ww * (q.gxy * uxi + q.gyy * uyi);
          }
        }
      }
    double m, s[4];
    quad_node_weights(ref, vx, vy, g.nx, P, 0, 0, g.nx, g.ny, I, J, &m, s);
    const double cj = c[gid];
    const double M = m / (cj * cj);
    const double H = (s[0] + s[1] + s[2] + s[3]) / cj;
    double bre = f_re[gid] * m, bim = f_im ? f_im[gid] * m : 0.0;
    if (bc) {
      if (I == 0) { bre += s[0] * bc[(0 * 2 + 0) * g.EB + J]; bim += s[0] * bc[(0 * 2 + 1) * g.EB + J]; }
      if (I == g.npx - 1) { bre += s[1] * bc[(1 * 2 + 0) * g.EB + J]; bim += s[1] * bc[(1 * 2 + 1) * g.EB + J]; }
      if (J == 0) { bre += s[2] * bc[(2 * 2 + 0) * g.EB + I]; bim += s[2] * bc[(2 * 2 + 1) * g.EB + I]; }
      if (J == g.npy - 1) { bre += s[3] * bc[(3 * 2 + 0) * g.EB + I]; bim += s[3] * bc[(3 * 2 + 1) * g.EB + I]; }
    }
    const double u_r = (double)ur[gid], u_i = (double)ui[gid];
    const double w2M = g.omega * g.omega * M, wH = g.omega * H;
    const double rr = bre - Ar + (w2M * u_r - wH * u_i);
    const double ri = bim - Ai + (w2M * u_i + wH * u_r);
    r2 = rr * rr + ri * ri;
    b2 = bre * bre + bim * bim;
  }
  for (int o = 16; o > 0; o >>= 1) {
    r2 += __shfl_down_sync(0xffffffffu, r2, o);
    b2 += __shfl_down_sync(0xffffffffu, b2, o);
  }
  const int w = threadIdx.x >> 5, ln = threadIdx.x & 31;
  if (ln == 0) { red[0][w] = r2; red[1][w] = b2; }
  __syncthreads();
  if (w == 0) {
    const int nw = blockDim.x >> 5;
    r2 = ln < nw ? red[0][ln] : 0.0;
    b2 = ln < nw ? red[1][ln] : 0.0;
    for (int o = 16; o > 0; o >>= 1) {
      r2 += __shfl_down_sync(0xffffffffu, r2, o);
      b2 += __shfl_down_sync(0xffffffffu, b2, o);
    }
    if (ln == 0) { part[2 * blockIdx.x] = r2; part[2 * blockIdx.x + 1] = b2; }
  }
}

}  // namespace hz
