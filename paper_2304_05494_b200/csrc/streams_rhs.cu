// a4-a8: the fused right-hand side + RK update.  One pass over the primitives produces, per
// interior node, the convective terms in x, y, z (central split form, O1), the viscous
// terms (O4) and the low-storage RK3 update (O5), so R is written once and w is updated in place
// (stencils read the primitive copy q, never w, so no ping-pong buffer is needed).
//
//   weno_kernel      : runs first.  Each block takes a chunk of interfaces of one direction, compacts the flagged
//                      ones (hybrid: the flag bits of flags_kernel; full-WENO: all) into a block-local list and
//                      evaluates them with full warps: WENO characteristic flux (O3) minus, in hybrid mode, the
//                      central flux that rhs_main_kernel will use there -> dF at the left node's index.
//   rhs_main_kernel  : every node: central scheme + viscous terms, adds -(dF_{n+1/2} - dF_{n-1/2}) metric at nodes
//                      next to a flagged interface, then the RK update.  R and w are written once.
// Every flagged interface is evaluated exactly once, by a warp whose lanes all do WENO work.
#include "streams_dev.cuh"
#include "streams_launch.h"

namespace streams {

struct VAcc {          // velocity / temperature / viscosity / dilatation derivatives at a node
  double g[3][3];      // g[a][b] = d u_a / d x_b
  double gT[3], gmu[3], gdiv[3];
  double lap[3], lapT;
};

template <int D>
__device__ __forceinline__ double pick(double a, double b, double c) { return D == 0 ? a : (D == 1 ? b : c); }

// ---------------------------------------------------------------------------------------------
// One direction at one node.  Convective part in pair-difference form: with
//   Pq(a,b) = (rho_a+rho_b)(ud_a+ud_b)(phi_a+phi_b)  the flux difference telescopes to
//   f_{n+1/2} - f_{n-1/2} = 1/4 sum_l a_l [P(n, n+l) - P(n-l, n)]   (+ sum_l a_l (p_{n+l} - p_{n-l}))
// which is the same sum as the oracle's interface-flux form (O1) in another order.
// Viscous part: first derivatives of u, v, w, T, mu, div and second derivatives of u, v, w, T.
// c0 = (rho, u, v, w, H, p) at the node.
// ---------------------------------------------------------------------------------------------
template <int D, int L, int LV, bool CONV, bool VISC>
__device__ __forceinline__ void dir_terms(const DevP& P, long long n, long long s, double met_c, double met_v,
                                          double eyy, const double c0[6], double T0, double r[5], VAcc& V) {
  const double* __restrict__ RHO = P.q + Q_RHO * P.fs + n;
  const double* __restrict__ U = P.q + Q_U * P.fs + n;
  const double* __restrict__ Vv = P.q + Q_V * P.fs + n;
  const double* __restrict__ W = P.q + Q_W * P.fs + n;
  const double* __restrict__ Hh = P.q + Q_H * P.fs + n;
  const double* __restrict__ Pp = P.q + Q_P * P.fs + n;
  const double* __restrict__ Tt = P.q + Q_T * P.fs + n;
  const double* __restrict__ Mu = P.q + Q_MU * P.fs + n;
  const double* __restrict__ Dv = P.div + n;
  constexpr int LC = CONV ? L : 0;
  constexpr int LVV = VISC ? LV : 0;
  constexpr int LM = LC > LVV ? LC : LVV;
  double S[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, SP = 0.0;
  double d1[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};   // u v w T mu div
  double d2[4] = {0.0, 0.0, 0.0, 0.0};             // u v w T
  const double ud0 = pick<D>(c0[1], c0[2], c0[3]);
#pragma unroll
  for (int l = 1; l <= LM; ++l) {
    const long long off = l * s;
    const double ub = U[off], ua = U[-off];
    const double vb = Vv[off], va = Vv[-off];
    const double wb = W[off], wa = W[-off];
    if (l <= LC) {
      const double rb = RHO[off], ra = RHO[-off];
      const double hb = Hh[off], ha = Hh[-off];
      const double pb = Pp[off], pa = Pp[-off];
      const double mb = (c0[0] + rb) * (ud0 + pick<D>(ub, vb, wb));
      const double ma = (ra + c0[0]) * (pick<D>(ua, va, wa) + ud0);
      const double al = P.a1[l - 1];
      S[0] += al * (mb - ma);
      S[1] += al * (mb * (c0[1] + ub) - ma * (ua + c0[1]));
      S[2] += al * (mb * (c0[2] + vb) - ma * (va + c0[2]));
      S[3] += al * (mb * (c0[3] + wb) - ma * (wa + c0[3]));
      S[4] += al * (mb * (c0[4] + hb) - ma * (ha + c0[4]));
      SP += al * (pb - pa);
    }
    if (l <= LVV) {
      const double tb = Tt[off], ta = Tt[-off];
      const double a = P.a1v[l - 1], b = P.b2v[l - 1];
      d1[0] += a * (ub - ua);  d2[0] += b * ((ub - 2.0 * c0[1]) + ua);
      d1[1] += a * (vb - va);  d2[1] += b * ((vb - 2.0 * c0[2]) + va);
      d1[2] += a * (wb - wa);  d2[2] += b * ((wb - 2.0 * c0[3]) + wa);
      d1[3] += a * (tb - ta);  d2[3] += b * ((tb - 2.0 * T0) + ta);
      d1[4] += a * (Mu[off] - Mu[-off]);
      d1[5] += a * (Dv[off] - Dv[-off]);
    }
  }
  if (CONV) {
    r[0] -= met_c * (0.5 * S[0]);
    r[1] -= met_c * (0.25 * S[1]);
    r[2] -= met_c * (0.25 * S[2]);
    r[3] -= met_c * (0.25 * S[3]);
    r[4] -= met_c * (0.25 * S[4]);
    r[1 + D] -= met_c * SP;
  }
  if (VISC) {
    const double m2 = met_v * met_v;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      V.g[a][D] = d1[a] * met_v;
      double sec = d2[a] * m2;
      if (D == 1) sec += eyy * d1[a];
      V.lap[a] += sec;
    }
    V.gT[D] = d1[3] * met_v;
    double secT = d2[3] * m2;
    if (D == 1) secT += eyy * d1[3];
    V.lapT += secT;
    V.gmu[D] = d1[4] * met_v;
    V.gdiv[D] = d1[5] * met_v;
  }
}

// ---------------------------------------------------------------------------------------------
// Viscous combination (O4), R store and RK update (O5) for one node.
// ---------------------------------------------------------------------------------------------
template <bool VISC, bool WENO, bool DENSE>
__device__ __forceinline__ void finish(const DevP& P, const StageArgs& sa, long long n, long long o, double met_y,
                                       const double c0[6], double mu0, double r[5], const VAcc& V) {
  if (VISC) {
    const double dv = (V.g[0][0] + V.g[1][1]) + V.g[2][2];
    double vm[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      double cross = 0.0;
#pragma unroll
      for (int b = 0; b < 3; ++b) cross += V.gmu[b] * (V.g[a][b] + V.g[b][a]);
      vm[a] = mu0 * V.lap[a] + cross - (2.0 / 3.0) * V.gmu[a] * dv + mu0 * V.gdiv[a] * (1.0 / 3.0);
    }
    const double s01 = V.g[0][1] + V.g[1][0], s02 = V.g[0][2] + V.g[2][0], s12 = V.g[1][2] + V.g[2][1];
    const double phi = mu0 * (2.0 * (V.g[0][0] * V.g[0][0] + V.g[1][1] * V.g[1][1] + V.g[2][2] * V.g[2][2]) +
                              s01 * s01 + s02 * s02 + s12 * s12 - (2.0 / 3.0) * dv * dv);
    const double cond = P.kfac * (mu0 * V.lapT + (V.gmu[0] * V.gT[0] + V.gmu[1] * V.gT[1] + V.gmu[2] * V.gT[2]));
    r[1] += vm[0];
    r[2] += vm[1];
    r[3] += vm[2];
    r[4] += (c0[1] * vm[0] + c0[2] * vm[1] + c0[3] * vm[2]) + phi + cond;
  }
  if (WENO) {
    // flux corrections of the flagged interfaces around this node (written by weno_kernel)
    const unsigned fl = DENSE ? 0x3fu : (unsigned)P.nflag[n];
    if (fl) {
      const long long st[3] = {1, P.sy, P.sz};
      const double met[3] = {P.inv_dx, met_y, P.inv_dz};
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const unsigned b = (fl >> (2 * d)) & 3u;
        if (b == 0) continue;
        const double* __restrict__ f = P.dF + (long long)(d * 5) * P.fs + n;
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          const double fp = (b & 2u) ? f[q * P.fs] : 0.0;
          const double fm = (b & 1u) ? f[q * P.fs - st[d]] : 0.0;
          r[q] -= (fp - fm) * met[d];
        }
      }
    }
  }
  if (sa.update_w) {
    const double dt = P.scal[S_DT];
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      double inc = sa.gam * r[q];
      if (sa.read_prev) inc += sa.rhk * P.R[q * P.N + o];
      double* wp = P.w + q * P.fs + n;
      *wp = *wp + dt * inc;
    }
  }
  if (sa.write_r) {
#pragma unroll
    for (int q = 0; q < 5; ++q) sa.r_out[q * P.N + o] = r[q];
  }
}

__device__ __forceinline__ void load_centre(const DevP& P, long long n, double c0[6]) {
  c0[0] = P.q[Q_RHO * P.fs + n];
  c0[1] = P.q[Q_U * P.fs + n];
  c0[2] = P.q[Q_V * P.fs + n];
  c0[3] = P.q[Q_W * P.fs + n];
  c0[4] = P.q[Q_H * P.fs + n];
  c0[5] = P.q[Q_P * P.fs + n];
}

__device__ __forceinline__ void zero_vacc(VAcc& V) {
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    V.lap[a] = 0.0; V.gT[a] = 0.0; V.gmu[a] = 0.0; V.gdiv[a] = 0.0;
#pragma unroll
    for (int b = 0; b < 3; ++b) V.g[a][b] = 0.0;
  }
  V.lapT = 0.0;
}

// ---------------------------------------------------------------------------------------------
// rhs_main_kernel: BX x BY x BZ nodes per block.  Blocks are numbered so that a slab of `slab`
// block-rows in y is swept through all of z before the next slab starts: the 2 ng z-neighbour
// planes of a slab then stay in L2.
// ---------------------------------------------------------------------------------------------
template <int L, int LV, bool VISC, bool CONV, bool WENO, int BX, int BY, int BZ>
__global__ void __launch_bounds__(BX * BY * BZ) rhs_main_kernel(const DevP P, const StageArgs sa, int nbx, int nby,
                                                               int nbz, int slab) {
  // decode block id -> (bx, by, bz), slab-major
  long long bid = blockIdx.x;
  const long long per_slab = (long long)nbx * slab * nbz;
  const int sl = (int)(bid / per_slab);
  const int rows = min(slab, nby - sl * slab);
  bid -= (long long)sl * per_slab;
  // inside a slab: x fastest, then y (rows of this slab), then z
  const int bx = (int)(bid % nbx);
  const long long t = bid / nbx;
  const int byl = (int)(t % rows);
  const int bz = (int)(t / rows);
  if (bz >= nbz) return;
  const int tx = threadIdx.x % BX, ty = (threadIdx.x / BX) % BY, tz = threadIdx.x / (BX * BY);
  const int i = bx * BX + tx, j = (sl * slab + byl) * BY + ty, k = bz * BZ + tz;
  if (i >= P.nx || j >= P.ny || k >= P.nz) return;
  const long long o = iidx(P, i, j, k);
  const long long n = pidx(P, i, j, k);
  double c0[6];
  load_centre(P, n, c0);
  double T0 = 0.0, mu0 = 0.0, eyv = 0.0, eyy = 0.0;
  if (VISC) { T0 = P.q[Q_T * P.fs + n]; mu0 = P.q[Q_MU * P.fs + n]; eyv = P.eta_y_v[j]; eyy = P.eta_yy_v[j]; }
  double r[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  VAcc V;
  zero_vacc(V);
  dir_terms<0, L, LV, CONV, VISC>(P, n, 1, P.inv_dx, P.inv_dx, 0.0, c0, T0, r, V);
  const double eyc = P.eta_y_c[j];
  dir_terms<1, L, LV, CONV, VISC>(P, n, P.sy, eyc, eyv, eyy, c0, T0, r, V);
  dir_terms<2, L, LV, CONV, VISC>(P, n, P.sz, P.inv_dz, P.inv_dz, 0.0, c0, T0, r, V);
  finish<VISC, WENO, !CONV>(P, sa, n, o, eyc, c0, mu0, r, V);
}

// ---------------------------------------------------------------------------------------------
// WENO reconstruction of order 2R-1 with Jiang-Shu weights (O3 step 4); v[0..2R-2] upwind->downwind,
// value at the interface between v[R-1] and v[R].
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double sq(double x) { return x * x; }

// 1/x for positive, normal x (sums of smoothness weights, sound speeds, 1 + sqrt(density ratio)): hardware
// seed + two Newton steps, ~1 ulp, no special-case branches (an IEEE divide is ~3x the instructions).
__device__ __forceinline__ double rcp_pos(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  r = fma(r, e, r);
  e = fma(-x, r, 1.0);
  return fma(r, e, r);
}

template <int R>
__device__ __forceinline__ double weno_rec(const double* v, double eps);

template <>
__device__ __forceinline__ double weno_rec<1>(const double* v, double) { return v[0]; }

// The Jiang-Shu weights alpha_k = d_k / (eps + beta_k)^2 are scaled by prod_j (eps + beta_j)^2, which leaves
// omega_k = alpha_k / sum(alpha) unchanged and needs one division per reconstruction instead of R + 1.
template <>
__device__ __forceinline__ double weno_rec<2>(const double* v, double eps) {
  const double q0 = 0.5 * (3.0 * v[1] - v[0]), q1 = 0.5 * (v[1] + v[2]);
  const double s0 = eps + sq(v[1] - v[0]), s1 = eps + sq(v[2] - v[1]);
  const double a0 = (1.0 / 3.0) * sq(s1), a1 = (2.0 / 3.0) * sq(s0);
  return (a0 * q0 + a1 * q1) * rcp_pos(a0 + a1);
}

template <>
__device__ __forceinline__ double weno_rec<3>(const double* v, double eps) {
  const double q0 = (2.0 * v[0] - 7.0 * v[1] + 11.0 * v[2]) * (1.0 / 6.0);
  const double q1 = (-v[1] + 5.0 * v[2] + 2.0 * v[3]) * (1.0 / 6.0);
  const double q2 = (2.0 * v[2] + 5.0 * v[3] - v[4]) * (1.0 / 6.0);
  const double s0 = eps + ((13.0 / 12.0) * sq(v[0] - 2.0 * v[1] + v[2]) + 0.25 * sq(v[0] - 4.0 * v[1] + 3.0 * v[2]));
  const double s1 = eps + ((13.0 / 12.0) * sq(v[1] - 2.0 * v[2] + v[3]) + 0.25 * sq(v[1] - v[3]));
  const double s2 = eps + ((13.0 / 12.0) * sq(v[2] - 2.0 * v[3] + v[4]) + 0.25 * sq(3.0 * v[2] - 4.0 * v[3] + v[4]));
  const double a0 = 0.1 * sq(s1 * s2), a1 = 0.6 * sq(s0 * s2), a2 = 0.3 * sq(s0 * s1);
  return (a0 * q0 + a1 * q1 + a2 * q2) * rcp_pos((a0 + a1) + a2);
}

template <>
__device__ __forceinline__ double weno_rec<4>(const double* v, double eps) {
  const double q0 = (-3.0 * v[0] + 13.0 * v[1] - 23.0 * v[2] + 25.0 * v[3]) * (1.0 / 12.0);
  const double q1 = (v[1] - 5.0 * v[2] + 13.0 * v[3] + 3.0 * v[4]) * (1.0 / 12.0);
  const double q2 = (-v[2] + 7.0 * v[3] + 7.0 * v[4] - v[5]) * (1.0 / 12.0);
  const double q3 = (3.0 * v[3] + 13.0 * v[4] - 5.0 * v[5] + v[6]) * (1.0 / 12.0);
  const double k = 1.0 / 240.0;
  const double s0 = eps + k * (v[0] * (547.0 * v[0] - 3882.0 * v[1] + 4642.0 * v[2] - 1854.0 * v[3]) +
                               v[1] * (7043.0 * v[1] - 17246.0 * v[2] + 7042.0 * v[3]) +
                               v[2] * (11003.0 * v[2] - 9402.0 * v[3]) + 2107.0 * v[3] * v[3]);
  const double s1 = eps + k * (v[1] * (267.0 * v[1] - 1642.0 * v[2] + 1602.0 * v[3] - 494.0 * v[4]) +
                               v[2] * (2843.0 * v[2] - 5966.0 * v[3] + 1922.0 * v[4]) +
                               v[3] * (3443.0 * v[3] - 2522.0 * v[4]) + 547.0 * v[4] * v[4]);
  const double s2 = eps + k * (v[2] * (547.0 * v[2] - 2522.0 * v[3] + 1922.0 * v[4] - 494.0 * v[5]) +
                               v[3] * (3443.0 * v[3] - 5966.0 * v[4] + 1602.0 * v[5]) +
                               v[4] * (2843.0 * v[4] - 1642.0 * v[5]) + 267.0 * v[5] * v[5]);
  const double s3 = eps + k * (v[3] * (2107.0 * v[3] - 9402.0 * v[4] + 7042.0 * v[5] - 1854.0 * v[6]) +
                               v[4] * (11003.0 * v[4] - 17246.0 * v[5] + 4642.0 * v[6]) +
                               v[5] * (7043.0 * v[5] - 3882.0 * v[6]) + 547.0 * v[6] * v[6]);
  const double p01 = s0 * s1, p23 = s2 * s3;
  const double a0 = (1.0 / 35.0) * sq(s1 * p23), a1 = (12.0 / 35.0) * sq(s0 * p23);
  const double a2 = (18.0 / 35.0) * sq(p01 * s3), a3 = (4.0 / 35.0) * sq(p01 * s2);
  return (a0 * q0 + a1 * q1 + a2 * q2 + a3 * q3) * rcp_pos(((a0 + a1) + a2) + a3);
}

// ---------------------------------------------------------------------------------------------
// WENO characteristic flux at interface n+1/2 along D (O3).  Characteristic projections are formed
// from primitives: l.W = rho (l0 + l1 u + l2 v + l3 w + l4 H) - l4 p and
// l.F = u_D (l.W) + p (l_{1+D} + l4 u_D), since F = u_D W + p (0, e_D, u_D); for the two shear fields
// (l = (-vbar_t, e_t, 0)) this collapses to l.W = rho (v_t - vbar_t), l.F = u_D (l.W).
// One characteristic field at a time (5 x 2 reconstructions).  The 2R-node stencil of (rho, u, v, w, H, p)
// lives in a per-thread column of shared memory (st[(f * 2R + m) * WTH], conflict-free), not in registers:
// the kernel then fits 4 blocks of 128 threads per SM instead of 2.
// ---------------------------------------------------------------------------------------------
constexpr int WTH = 128;       // threads per block of weno_kernel
constexpr int WCH = 2048;      // interface slots per block

template <int D, int R>
__device__ __forceinline__ void weno_flux(const DevP& P, long long n, long long s, double f[5], double* __restrict__ st) {
  constexpr int NS = 2 * R;
  enum { F_RHO = 0, F_U = 1, F_V = 2, F_W = 3, F_H = 4, F_P = 5 };
#define ST(fld, m) (((volatile double*)st)[((fld) * NS + (m)) * WTH])
  double lam_m = 0.0, lam_0 = 0.0, lam_p = 0.0;
#pragma unroll
  for (int m = 0; m < NS; ++m) {
    const long long a = n + (long long)(m - R + 1) * s;
    const double u = P.q[Q_U * P.fs + a], v = P.q[Q_V * P.fs + a], w = P.q[Q_W * P.fs + a];
    const double c = P.q[Q_C * P.fs + a];
    ST(F_RHO, m) = P.q[Q_RHO * P.fs + a];
    ST(F_U, m) = u;
    ST(F_V, m) = v;
    ST(F_W, m) = w;
    ST(F_H, m) = P.q[Q_H * P.fs + a];
    ST(F_P, m) = P.q[Q_P * P.fs + a];
    const double ud = D == 0 ? u : (D == 1 ? v : w);
    lam_m = fmax(lam_m, fabs(ud - c));
    lam_0 = fmax(lam_0, fabs(ud));
    lam_p = fmax(lam_p, fabs(ud + c));
  }
  // Roe average of nodes n (slot R-1) and n+1 (slot R)
  const double rw = sqrt(ST(F_RHO, R) * rcp_pos(ST(F_RHO, R - 1)));
  const double iden = rcp_pos(1.0 + rw);
  double vb[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) vb[a] = (ST(F_U + a, R - 1) + rw * ST(F_U + a, R)) * iden;
  const double Hb = (ST(F_H, R - 1) + rw * ST(F_H, R)) * iden;
  const double qq = 0.5 * (vb[0] * vb[0] + vb[1] * vb[1] + vb[2] * vb[2]);
  const double c2 = P.gm1 * (Hb - qq);
  const double cb = sqrt(c2);
  const double ic = rcp_pos(cb);
  const double b1 = P.gm1 * (ic * ic), b2 = qq * b1;
  const double un = vb[D];
  constexpr int T1 = (D == 0) ? 1 : 0;
  constexpr int T2 = (D == 2) ? 1 : 2;
#pragma unroll
  for (int q = 0; q < 5; ++q) f[q] = 0.0;
  // One characteristic field after the other.  The stencil is read through volatile shared-memory loads so
  // that the compiler cannot hoist all 36 values of every field into registers (it then needs > 200).
#pragma unroll
  for (int sc = 0; sc < 5; ++sc) {
    double gp[NS], gm[NS];
    double rv[5];                                   // right eigenvector of this field
    if (sc == 2 || sc == 3) {
      const int t = (sc == 2) ? T1 : T2;
      const double vbt = t == 0 ? vb[0] : (t == 1 ? vb[1] : vb[2]);
      const volatile double* stt = st + (F_U + t) * NS * WTH;
#pragma unroll
      for (int m = 0; m < NS; ++m) {
        const double lw = (0.5 * ST(F_RHO, m)) * (stt[m * WTH] - vbt);   // (l.W) / 2
        const double lf = ST(F_U + D, m) * lw;                           // (l.F) / 2
        gp[m] = fma(lam_0, lw, lf);
        gm[NS - 1 - m] = fma(-lam_0, lw, lf);        // mirrored: gm[0] is node n+R
      }
      rv[0] = 0.0;
#pragma unroll
      for (int a = 0; a < 3; ++a) rv[1 + a] = (a == t) ? 1.0 : 0.0;
      rv[4] = vbt;
    } else {
      double l0, lv[3], l4, lam;
      if (sc == 1) {
        l0 = 0.5 * (1.0 - b2);                      // the 1/2 of the flux splitting is folded into l
#pragma unroll
        for (int a = 0; a < 3; ++a) lv[a] = 0.5 * (b1 * vb[a]);
        l4 = -0.5 * b1;
        lam = lam_0;
        rv[0] = 1.0;
#pragma unroll
        for (int a = 0; a < 3; ++a) rv[1 + a] = vb[a];
        rv[4] = qq;
      } else {
        const double sg = (sc == 0) ? 1.0 : -1.0;
        l0 = 0.25 * (b2 + sg * un * ic);
#pragma unroll
        for (int a = 0; a < 3; ++a) lv[a] = 0.25 * (-b1 * vb[a] - (a == D ? sg * ic : 0.0));
        l4 = 0.25 * b1;
        lam = (sc == 0) ? lam_m : lam_p;
        rv[0] = 1.0;
#pragma unroll
        for (int a = 0; a < 3; ++a) rv[1 + a] = vb[a] - (a == D ? sg * cb : 0.0);
        rv[4] = Hb - sg * un * cb;
      }
#pragma unroll
      for (int m = 0; m < NS; ++m) {
        const double um = ST(F_U, m), vm = ST(F_V, m), wm = ST(F_W, m), pm = ST(F_P, m);
        const double ud = D == 0 ? um : (D == 1 ? vm : wm);
        const double lw = ST(F_RHO, m) * (l0 + lv[0] * um + lv[1] * vm + lv[2] * wm + l4 * ST(F_H, m)) - l4 * pm;
        const double lf = ud * lw + pm * (lv[D] + l4 * ud);
        gp[m] = fma(lam, lw, lf);
        gm[NS - 1 - m] = fma(-lam, lw, lf);
      }
    }
    const double gh = weno_rec<R>(gp, P.weno_eps) + weno_rec<R>(gm, P.weno_eps);
#pragma unroll
    for (int q = 0; q < 5; ++q) f[q] += gh * rv[q];
  }
#undef ST
}

// Central interface flux (O1) from the same shared-memory stencil (needs L <= R): the flux that
// rhs_main_kernel's pair-difference form implies at this interface, subtracted in hybrid mode.
template <int D, int L, int R>
__device__ __forceinline__ void central_flux_st(const DevP& P, double f[5], const double* st) {
  static_assert(L <= R, "the central stencil must fit in the WENO stencil");
  constexpr int NS = 2 * R;
  enum { F_RHO = 0, F_U = 1, F_V = 2, F_W = 3, F_H = 4, F_P = 5 };
#define ST(fld, m) (((const volatile double*)st)[((fld) * NS + (m)) * WTH])
  double fs[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, ps = 0.0;
#pragma unroll
  for (int l = 1; l <= L; ++l) {
    double in[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, pin = 0.0;
#pragma unroll
    for (int m = 0; m < l; ++m) {
      const int a = R - 1 - m, b = a + l;          // slots of nodes n - m and n - m + l
      const double ua = ST(F_U, a), va = ST(F_V, a), wa = ST(F_W, a);
      const double ub = ST(F_U, b), vb = ST(F_V, b), wb = ST(F_W, b);
      const double uda = D == 0 ? ua : (D == 1 ? va : wa), udb = D == 0 ? ub : (D == 1 ? vb : wb);
      const double ru = (ST(F_RHO, a) + ST(F_RHO, b)) * (uda + udb);
      in[0] += ru * 2.0;
      in[1] += ru * (ua + ub);
      in[2] += ru * (va + vb);
      in[3] += ru * (wa + wb);
      in[4] += ru * (ST(F_H, a) + ST(F_H, b));
      pin += ST(F_P, a) + ST(F_P, b);
    }
#pragma unroll
    for (int q = 0; q < 5; ++q) fs[q] += P.a1[l - 1] * in[q];
    ps += P.a1[l - 1] * pin;
  }
#pragma unroll
  for (int q = 0; q < 5; ++q) f[q] = 0.25 * fs[q];
  f[1 + D] += ps;
#undef ST
}

// ---------------------------------------------------------------------------------------------
// weno_kernel: blocks [0, nb0) work on x interfaces, [nb0, nb0 + nb1) on y, the rest on z.  A block owns
// WCH consecutive interface slots of its direction (slot = interior extents with the D extent enlarged by
// one; slot s along D is the interface between nodes s - 1 and s).  Hybrid mode: the flagged slots are
// compacted into a shared-memory list (flag bits of flags_kernel: plus side of the left node, or minus side
// of node 0 for the first interface of a pencil), then walked by all threads, so lanes stay converged on
// WENO work whatever the activation pattern.  DENSE (full-WENO mode): every slot, WENO flux itself stored.
// ---------------------------------------------------------------------------------------------
template <int D, int L, int R, bool DENSE>
__device__ __forceinline__ void weno_block(const DevP& P, long long chunk, int* s_list, int* s_count, double* s_st) {
  const long long s = D == 0 ? 1 : (D == 1 ? P.sy : P.sz);
  const int e0 = P.nx + (D == 0), e1 = P.ny + (D == 1), e2 = P.nz + (D == 2);
  const int lane = threadIdx.x & 31;
  if (threadIdx.x == 0) *s_count = 0;
  __syncthreads();
  // slot of this thread in round 0, decoded once; later rounds advance it by WTH
  const long long t0 = chunk * WCH + threadIdx.x;
  int i = (int)(t0 % e0);
  const long long t1 = t0 / e0;
  int j = (int)(t1 % e1), k = (int)(t1 / e1);
  for (int rr = 0; rr < WCH / WTH; ++rr) {
    bool want = false;
    int n = 0;
    if (k < e2) {
      n = (int)pidx(P, i - (D == 0), j - (D == 1), k - (D == 2));       // left node of the interface
      if (DENSE) want = true;
      else {
        const int a = D == 0 ? i : (D == 1 ? j : k);
        want = a > 0 ? ((P.nflag[n] >> (2 * D + 1)) & 1) : ((P.nflag[n + s] >> (2 * D)) & 1);
      }
    }
    const unsigned bal = __ballot_sync(0xffffffffu, want);
    int pos = 0;
    if (lane == 0 && bal) pos = atomicAdd(s_count, __popc(bal));
    pos = __shfl_sync(0xffffffffu, pos, 0);
    if (want) s_list[pos + __popc(bal & ((1u << lane) - 1u))] = n;
    i += WTH;
    while (i >= e0) { i -= e0; if (++j >= e1) { j = 0; ++k; } }
  }
  __syncthreads();
  const int count = *s_count;
  double* __restrict__ out = P.dF + (long long)(D * 5) * P.fs;
  for (int e = threadIdx.x; e < count; e += WTH) {
    const long long n = s_list[e];
    double fw[5];
    weno_flux<D, R>(P, n, s, fw, s_st + threadIdx.x);
    if (!DENSE) {
      double fc[5];
      central_flux_st<D, L, R>(P, fc, s_st + threadIdx.x);
#pragma unroll
      for (int q = 0; q < 5; ++q) fw[q] -= fc[q];
    }
#pragma unroll
    for (int q = 0; q < 5; ++q) out[q * P.fs + n] = fw[q];
  }
}

#ifndef STREAMS_WENO_MINB
#define STREAMS_WENO_MINB 4
#endif
template <int L, int R, bool DENSE>
__global__ void __launch_bounds__(WTH, STREAMS_WENO_MINB) weno_kernel(const DevP P, int nb0, int nb1) {
  __shared__ int s_list[WCH];
  __shared__ int s_count;
  __shared__ double s_st[6 * 2 * R * WTH];
  const int b = blockIdx.x;
  if (b < nb0) weno_block<0, L, R, DENSE>(P, b, s_list, &s_count, s_st);
  else if (b < nb0 + nb1) weno_block<1, L, R, DENSE>(P, b - nb0, s_list, &s_count, s_st);
  else weno_block<2, L, R, DENSE>(P, b - nb0 - nb1, s_list, &s_count, s_st);
}

// -------------------------------------------------------------------------- launch
constexpr int MBX = 32, MBY = 4, MBZ = 4;

template <int L, int LV, int R>
static int launch_main_T(const DevP& P, const StageArgs& sa, cudaStream_t st) {
  const bool visc = P.visc_law != VISC_NONE;
  const bool conv = P.flux_mode != FLUX_WENO;
  const bool weno = P.flux_mode != FLUX_CENTRAL;
  const int nbx = (P.nx + MBX - 1) / MBX, nby = (P.ny + MBY - 1) / MBY, nbz = (P.nz + MBZ - 1) / MBZ;
  int slab = 8;                                  // 8 block rows = 32 grid rows per slab
  if (slab > nby) slab = nby;
  const int nslab = (nby + slab - 1) / slab;
  const long long nblocks = (long long)nslab * nbx * slab * nbz;
  dim3 b(MBX * MBY * MBZ), g((unsigned)nblocks);
#define STREAMS_MAIN(V, C, W) rhs_main_kernel<L, LV, V, C, W, MBX, MBY, MBZ><<<g, b, 0, st>>>(P, sa, nbx, nby, nbz, slab)
  if (visc && conv && weno) STREAMS_MAIN(true, true, true);
  else if (visc && conv) STREAMS_MAIN(true, true, false);
  else if (visc) STREAMS_MAIN(true, false, true);
  else if (conv && weno) STREAMS_MAIN(false, true, true);
  else if (conv) STREAMS_MAIN(false, true, false);
  else STREAMS_MAIN(false, false, true);
#undef STREAMS_MAIN
  return 1;
}

template <int L, int R>
static int launch_weno_T(const DevP& P, cudaStream_t st) {
  if (P.flux_mode == FLUX_CENTRAL) return 0;
  const long long a = (long long)P.nx * P.ny * P.nz;
  auto blocks = [&](long long extra) { return (int)((a + extra + WCH - 1) / WCH); };
  const int nb0 = blocks((long long)P.ny * P.nz), nb1 = blocks((long long)P.nx * P.nz), nb2 = blocks((long long)P.nx * P.ny);
  dim3 b(WTH), g((unsigned)(nb0 + nb1 + nb2));
  if (P.flux_mode == FLUX_HYBRID) weno_kernel<L, R, false><<<g, b, 0, st>>>(P, nb0, nb1);
  else weno_kernel<L, R, true><<<g, b, 0, st>>>(P, nb0, nb1);
  return 1;
}

bool rhs_supported(int L, int Lv, int r, int flux_mode, int visc_law) {
  const int lv = visc_law == VISC_NONE ? 3 : Lv;
  const int rr = flux_mode == FLUX_CENTRAL ? 3 : r;
  return L == 3 && lv == 3 && rr == 3;
}

int launch_rhs_main(const DevP& P, int L, int Lv, int r, const StageArgs& sa, cudaStream_t st) {
  if (!rhs_supported(L, Lv, r, P.flux_mode, P.visc_law)) return -1;
  return launch_main_T<3, 3, 3>(P, sa, st);
}
int launch_weno(const DevP& P, int L, int Lv, int r, cudaStream_t st) {
  if (!rhs_supported(L, Lv, r, P.flux_mode, P.visc_law)) return -1;
  return launch_weno_T<3, 3>(P, st);
}

}  // namespace streams
