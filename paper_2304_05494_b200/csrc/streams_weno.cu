// a4-a6 at the interfaces that take the WENO branch, and the net correction they leave at the nodes.
//
//   weno_list_kernel   : hybrid mode.  The flagged interfaces of each direction were compacted into work lists by
//                        flags_kernel; persistent blocks evaluate them with full warps: WENO characteristic flux (O3)
//                        minus the central flux that rhs_march_kernel implies there -> dF at the left node's index.
//   weno_kernel        : full-WENO mode: every interface, the WENO flux itself.
//   corr_gather_kernel : per node next to a flagged interface, corr_q = sum_d metric_d (dF_d(n) - dF_d(n - e_d)) over its
//                        flagged interfaces in the fixed order x, y, z (bit-reproducible, no atomics): the five values
//                        rhs_march_kernel subtracts from the node's right-hand side.
// Every flagged interface is evaluated exactly once, by a warp whose lanes all do WENO work.
#include "streams_dev.cuh"
#include "streams_launch.h"
#include "streams_tma.cuh"

namespace streams {

// ---------------------------------------------------------------------------------------------
// WENO reconstruction of order 2R-1 with Jiang-Shu weights (O3 step 4); v[0..2R-2] upwind->downwind,
// value at the interface between v[R-1] and v[R].
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double sq(double x) { return x * x; }

// Z: WENO-Z weights (S19) alpha_k = d_k (1 + (tau / s_k)^2) with s_k = eps + beta_k and the global indicator
// tau of the whole stencil; scaled by prod_j s_j^2 like the Jiang-Shu ones: a_k = d_k (s_k^2 + tau^2) prod_{j != k} s_j^2.
template <int R, bool Z>
__device__ __forceinline__ double weno_rec(const double* v, double eps);

template <>
__device__ __forceinline__ double weno_rec<1, false>(const double* v, double) { return v[0]; }
template <>
__device__ __forceinline__ double weno_rec<1, true>(const double* v, double) { return v[0]; }

// The Jiang-Shu weights alpha_k = d_k / (eps + beta_k)^2 are scaled by prod_j (eps + beta_j)^2, which leaves
// omega_k = alpha_k / sum(alpha) unchanged and needs one division per reconstruction instead of R + 1.
template <bool Z>
__device__ __forceinline__ double weno_rec2(const double* v, double eps) {
  const double q0 = 0.5 * (3.0 * v[1] - v[0]), q1 = 0.5 * (v[1] + v[2]);
  const double s0 = eps + sq(v[1] - v[0]), s1 = eps + sq(v[2] - v[1]);
  const double t2 = Z ? sq(s0 - s1) : 0.0;            // tau^2, tau = |beta_0 - beta_1|
  const double a0 = (1.0 / 3.0) * (Z ? (sq(s0) + t2) * sq(s1) : sq(s1)), a1 = (2.0 / 3.0) * (Z ? (sq(s1) + t2) * sq(s0) : sq(s0));
  return (a0 * q0 + a1 * q1) * rcp_pos(a0 + a1);
}
template <> __device__ __forceinline__ double weno_rec<2, false>(const double* v, double eps) { return weno_rec2<false>(v, eps); }
template <> __device__ __forceinline__ double weno_rec<2, true>(const double* v, double eps) { return weno_rec2<true>(v, eps); }

// Fifth order, written on the undivided differences d_m = v[m+1] - v[m], which the candidate values and the smoothness
// indicators share (the same real-number function as the textbook form, 49 instead of 59 operations):
//   q0 = v2 + (5 d1 - 2 d0)/6, q1 = v2 + (d1 + 2 d2)/6, q2 = v2 + (4 d2 - d3)/6,
//   beta0 = 13/12 (d1 - d0)^2 + 1/4 (3 d1 - d0)^2, beta1 = 13/12 (d2 - d1)^2 + 1/4 (d1 + d2)^2,
//   beta2 = 13/12 (d3 - d2)^2 + 1/4 (d3 - 3 d2)^2;  result = v2 + sum_k a_k (q_k - v2) / sum_k a_k.
template <bool Z>
__device__ __forceinline__ double weno_rec3(const double* v, double eps) {
  const double d0 = v[1] - v[0], d1 = v[2] - v[1], d2 = v[3] - v[2], d3 = v[4] - v[3];
  const double e0 = fma(5.0 / 6.0, d1, (-2.0 / 6.0) * d0);
  const double e1 = fma(2.0 / 6.0, d2, (1.0 / 6.0) * d1);
  const double e2 = fma(4.0 / 6.0, d2, (-1.0 / 6.0) * d3);
  const double s0 = fma(13.0 / 12.0, sq(d1 - d0), fma(0.25, sq(fma(3.0, d1, -d0)), eps));
  const double s1 = fma(13.0 / 12.0, sq(d2 - d1), fma(0.25, sq(d1 + d2), eps));
  const double s2 = fma(13.0 / 12.0, sq(d3 - d2), fma(0.25, sq(fma(-3.0, d2, d3)), eps));
  double a0 = 0.1 * sq(s1 * s2), a1 = 0.6 * sq(s0 * s2), a2 = 0.3 * sq(s0 * s1);
  if (Z) {
    const double t2 = sq(s0 - s2);                    // tau^2, tau = |beta_0 - beta_2|
    a0 *= sq(s0) + t2; a1 *= sq(s1) + t2; a2 *= sq(s2) + t2;
  }
  return fma(fma(a0, e0, fma(a1, e1, a2 * e2)), rcp_pos((a0 + a1) + a2), v[2]);
}
template <> __device__ __forceinline__ double weno_rec<3, false>(const double* v, double eps) { return weno_rec3<false>(v, eps); }
template <> __device__ __forceinline__ double weno_rec<3, true>(const double* v, double eps) { return weno_rec3<true>(v, eps); }

template <bool Z>
__device__ __forceinline__ double weno_rec4(const double* v, double eps) {
  const double q0 = (-3.0 * v[0] + 13.0 * v[1] - 23.0 * v[2] + 25.0 * v[3]) * (1.0 / 12.0);
  const double q1 = (v[1] - 5.0 * v[2] + 13.0 * v[3] + 3.0 * v[4]) * (1.0 / 12.0);
  const double q2 = (-v[2] + 7.0 * v[3] + 7.0 * v[4] - v[5]) * (1.0 / 12.0);
  const double q3 = (3.0 * v[3] + 13.0 * v[4] - 5.0 * v[5] + v[6]) * (1.0 / 12.0);
  // smoothness indicators as the sums of squares they are: beta = U^2/36 + (13/12) S^2 + (781/720) T^2 with U, S, T the
  // undivided-difference forms of c1 + c3/4, c2, c3 of the sub-stencil's cubic (the expanded polynomial with the
  // coefficients 547, -3882, ... is the same quadratic form and loses ~8 digits to cancellation on smooth data)
  const double U0 = ((2.0 * v[0] - 9.0 * v[1]) + 18.0 * v[2]) - 11.0 * v[3], S0 = ((v[0] - 4.0 * v[1]) + 5.0 * v[2]) - 2.0 * v[3];
  const double T0 = ((v[0] - 3.0 * v[1]) + 3.0 * v[2]) - v[3];
  const double U1 = ((v[1] - 6.0 * v[2]) + 3.0 * v[3]) + 2.0 * v[4], S1 = (v[2] - 2.0 * v[3]) + v[4];
  const double T1 = ((v[1] - 3.0 * v[2]) + 3.0 * v[3]) - v[4];
  const double U2 = ((2.0 * v[2] + 3.0 * v[3]) - 6.0 * v[4]) + v[5];
  const double T2 = ((v[2] - 3.0 * v[3]) + 3.0 * v[4]) - v[5];
  const double U3 = ((11.0 * v[3] - 18.0 * v[4]) + 9.0 * v[5]) - 2.0 * v[6], S3 = ((2.0 * v[3] - 5.0 * v[4]) + 4.0 * v[5]) - v[6];
  const double T3 = ((v[3] - 3.0 * v[4]) + 3.0 * v[5]) - v[6];
  constexpr double cU = 1.0 / 36.0, cS = 13.0 / 12.0, cT = 781.0 / 720.0;
  const double s0 = eps + (cU * sq(U0) + cS * sq(S0) + cT * sq(T0));
  const double s1 = eps + (cU * sq(U1) + cS * sq(S1) + cT * sq(T1));
  const double s2 = eps + (cU * sq(U2) + cS * sq(S1) + cT * sq(T2));
  const double s3 = eps + (cU * sq(U3) + cS * sq(S3) + cT * sq(T3));
  const double p01 = s0 * s1, p23 = s2 * s3;
  double a0 = (1.0 / 35.0) * sq(s1 * p23), a1 = (12.0 / 35.0) * sq(s0 * p23);
  double a2 = (18.0 / 35.0) * sq(p01 * s3), a3 = (4.0 / 35.0) * sq(p01 * s2);
  if (Z) {
    const double t2 = sq(((s0 - s1) - s2) + s3);      // tau^2, tau = |beta_0 - beta_1 - beta_2 + beta_3|
    a0 *= sq(s0) + t2; a1 *= sq(s1) + t2; a2 *= sq(s2) + t2; a3 *= sq(s3) + t2;
  }
  return (a0 * q0 + a1 * q1 + a2 * q2 + a3 * q3) * rcp_pos(((a0 + a1) + a2) + a3);
}
template <> __device__ __forceinline__ double weno_rec<4, false>(const double* v, double eps) { return weno_rec4<false>(v, eps); }
template <> __device__ __forceinline__ double weno_rec<4, true>(const double* v, double eps) { return weno_rec4<true>(v, eps); }

// Both reconstructions of a characteristic field (upwind and mirrored stencil) as ONE call with the arguments by
// value, in registers: the five fields of an interface then share one copy of the code instead of ten inlined
// reconstructions (instruction-cache footprint: the list kernel's straight-line code shrinks by 30 %), while the two
// reconstructions of a field still interleave.
template <int R, bool Z>
__device__ __forceinline__ double weno_rec_pair(const double* gp, const double* gm, double eps) {
  return weno_rec<R, Z>(gp, eps) + weno_rec<R, Z>(gm, eps);
}
__device__ __noinline__ double weno_rec5_pair_call(double p0, double p1, double p2, double p3, double p4, double m0, double m1,
                                                  double m2, double m3, double m4, double eps) {
  const double gp[5] = {p0, p1, p2, p3, p4}, gm[5] = {m0, m1, m2, m3, m4};
  return weno_rec<3, false>(gp, eps) + weno_rec<3, false>(gm, eps);
}
template <>
__device__ __forceinline__ double weno_rec_pair<3, false>(const double* gp, const double* gm, double eps) {
  return weno_rec5_pair_call(gp[0], gp[1], gp[2], gp[3], gp[4], gm[0], gm[1], gm[2], gm[3], gm[4], eps);
}

// ---------------------------------------------------------------------------------------------
// WENO characteristic flux at interface n+1/2 along D (O3), and the central flux (O1) it replaces.
// Characteristic projections are formed from primitives: with W the conserved state and
// F = u_D W + p (0, e_D, u_D), l.W = rho (l0 + l1 u + l2 v + l3 w + l4 H) - l4 p and
// l.F = u_D (l.W) + p (l_{1+D} + l4 u_D).  With b1 = (gamma-1)/c^2, b2 = b1 q^2/2 and the 1/2 of the
// Lax-Friedrichs splitting folded into l, the three non-shear rows share per node
//   A  = [rho (b2 - b1 vbar.v + b1 H) - b1 p] / 4        B  = rho (un - u_D) / (4 c)
//   FA = u_D A + b1 p (u_D - un) / 4                     FB = u_D B - p / (4 c)
// as  u-c: (l.W, l.F) = (A + B, FA + FB);  u+c: (A - B, FA - FB);  entropy: (rho/2 - 2A, rho u_D/2 - 2FA);
// the two shear rows (l = (-vbar_t, e_t, 0)) collapse to l.W = rho (v_t - vbar_t)/2, l.F = u_D (l.W).
// The stencil of (rho, u, v, w, H, p) lives in a per-thread column of shared memory (st[(f * 2M + m) * WTH],
// conflict-free) so that the kernel fits 4 blocks of 128 threads per SM; M = max(L, R) nodes each side of the
// interface: the central flux of order 2L uses all 2M of them (coefficients beyond L are zero), the WENO
// reconstruction of order 2R-1 and its Lax-Friedrichs speeds the inner 2R (slots M-R .. M+R-1).
// ---------------------------------------------------------------------------------------------
constexpr int WTH = 128;       // threads per block of the WENO kernels

#define ST(fld, m) (((volatile double*)st)[((fld) * NS + (m)) * WTH])
enum { SF_RHO = 0, SF_U = 1, SF_V = 2, SF_W = 3, SF_H = 4, SF_P = 5 };

// Central interface flux (O1) from the shared-memory stencil: the flux that rhs_march_kernel's pair-difference form
// implies at this interface.  f = 1/4 sum_l a_l sum_{m<l} (rho_a+rho_b)(ud_a+ud_b)(phi_a+phi_b),
// pairs (a, b) = (n-m, n-m+l).  The M left nodes stay in registers, the right nodes stream past them.
template <int D, int M>
__device__ __forceinline__ void central_flux_st(const DevP& P, double f[5], const double* st) {
  constexpr int NS = 2 * M;
  double lf[M][6];                                 // left nodes n, n-1, .., n-M+1: rho, u, v, w, H, p
#pragma unroll
  for (int m = 0; m < M; ++m) {
#pragma unroll
    for (int q = 0; q < 6; ++q) lf[m][q] = ST(q, M - 1 - m);
  }
  double fs[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, ps = 0.0;
#pragma unroll
  for (int j = 0; j < M; ++j) {                    // right node n+1+j pairs with left node n-m at distance l = j+1+m
    double rt[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) rt[q] = ST(q, M + j);
#pragma unroll
    for (int m = 0; m + j < M; ++m) {
      const double al = P.a1[j + m];
      const double ru = (al * (lf[m][SF_RHO] + rt[SF_RHO])) * (lf[m][SF_U + D] + rt[SF_U + D]);
      fs[0] += ru;
#pragma unroll
      for (int q = 1; q < 5; ++q) fs[q] = fma(ru, lf[m][q] + rt[q], fs[q]);
      ps = fma(al, lf[m][SF_P] + rt[SF_P], ps);
    }
  }
  f[0] = 0.5 * fs[0];
#pragma unroll
  for (int q = 1; q < 5; ++q) f[q] = 0.25 * fs[q];
  f[1 + D] += ps;
}

// Fills the stencil column of interface n+1/2 (left node index n, stride s along D) and returns the local
// Lax-Friedrichs speeds max |u_D - c|, |u_D|, |u_D + c| over the 2R nodes of the WENO stencil.
// The 12 M values of the column go from global to shared memory by cp.async, all in flight at once (through registers
// the loads went in batches of what the register budget holds, each batch exposing a memory latency: the kernel's
// stall samples on config 4 were 23 % long scoreboard + 27 % MIO queue behind the waiting shared-memory stores); the
// sound speeds of the 2R inner nodes are loaded into registers meanwhile.
template <int D, int M, int R>
__device__ __forceinline__ void weno_stencil(const DevP& P, long long n, long long s, double* __restrict__ st, double lam[3]) {
  constexpr int NS = 2 * M;
  const double* __restrict__ q0 = P.q + n - (long long)(M - 1) * s;
#pragma unroll
  for (int m = 0; m < NS; ++m) {
    const double* __restrict__ qa = q0 + (long long)m * s;
    cp_async8(st + (SF_RHO * NS + m) * WTH, qa + Q_RHO * P.fs);
    cp_async8(st + (SF_U * NS + m) * WTH, qa + Q_U * P.fs);
    cp_async8(st + (SF_V * NS + m) * WTH, qa + Q_V * P.fs);
    cp_async8(st + (SF_W * NS + m) * WTH, qa + Q_W * P.fs);
    cp_async8(st + (SF_H * NS + m) * WTH, qa + Q_H * P.fs);
    cp_async8(st + (SF_P * NS + m) * WTH, qa + Q_P * P.fs);
  }
  double c[2 * R];
#pragma unroll
  for (int m = 0; m < 2 * R; ++m) c[m] = q0[Q_C * P.fs + (long long)(M - R + m) * s];
  cp_async_wait_all();
  lam[0] = lam[1] = lam[2] = 0.0;
#pragma unroll
  for (int m = 0; m < 2 * R; ++m) {
    const double ud = ST(SF_U + D, M - R + m);
    lam[0] = fmax(lam[0], fabs(ud - c[m]));
    lam[1] = fmax(lam[1], fabs(ud));
    lam[2] = fmax(lam[2], fabs(ud + c[m]));
  }
}

template <int D, int M, int R, bool Z>
__device__ __forceinline__ void weno_flux(const DevP& P, const double lam[3], double f[5], const double* __restrict__ st) {
  constexpr int NS = 2 * M;                        // column pitch (the ST macro)
  constexpr int NW = 2 * R;                        // WENO stencil nodes, column slots O .. O + NW - 1
  constexpr int O = M - R;
  // Roe average of nodes n (slot M-1) and n+1 (slot M)
  const double rw = sqrt(ST(SF_RHO, M) * rcp_pos(ST(SF_RHO, M - 1)));
  const double iden = rcp_pos(1.0 + rw);
  double vb[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) vb[a] = (ST(SF_U + a, M - 1) + rw * ST(SF_U + a, M)) * iden;
  const double Hb = (ST(SF_H, M - 1) + rw * ST(SF_H, M)) * iden;
  const double qq = 0.5 * (vb[0] * vb[0] + vb[1] * vb[1] + vb[2] * vb[2]);
  const double cb = sqrt(P.gm1 * (Hb - qq));
  const double ic = rcp_pos(cb);
  const double un = vb[D];
  const double k1 = 0.25 * (P.gm1 * (ic * ic)), k2 = qq * k1, ki = 0.25 * ic;
  constexpr int T1 = (D == 0) ? 1 : 0;
  constexpr int T2 = (D == 2) ? 1 : 2;
  double gp[NW], gm[NW];

  // shared rows of the two acoustic fields and the entropy field, one pass over the nodes
  double A[NW], B[NW], FA[NW], FB[NW];
#pragma unroll
  for (int m = 0; m < NW; ++m) {
    const double rho = ST(SF_RHO, O + m), um = ST(SF_U, O + m), vm = ST(SF_V, O + m), wm = ST(SF_W, O + m),
                 hm = ST(SF_H, O + m), pm = ST(SF_P, O + m);
    const double ud = D == 0 ? um : (D == 1 ? vm : wm);
    const double dot = fma(vb[2], wm, fma(vb[1], vm, vb[0] * um));
    const double kp = k1 * pm, du = ud - un;
    A[m] = fma(rho, fma(k1, hm - dot, k2), -kp);
    B[m] = -((rho * ki) * du);
    FA[m] = fma(ud, A[m], kp * du);
    FB[m] = fma(ud, B[m], -(ki * pm));
  }
  // u - c
#pragma unroll
  for (int m = 0; m < NW; ++m) {
    const double lw = A[m] + B[m], lf = FA[m] + FB[m];
    gp[m] = fma(lam[0], lw, lf);
    gm[NW - 1 - m] = fma(-lam[0], lw, lf);          // mirrored: gm[0] is node n+R
  }
  const double g0 = weno_rec_pair<R, Z>(gp, gm, P.weno_eps);
  // u + c
#pragma unroll
  for (int m = 0; m < NW; ++m) {
    const double lw = A[m] - B[m], lf = FA[m] - FB[m];
    gp[m] = fma(lam[2], lw, lf);
    gm[NW - 1 - m] = fma(-lam[2], lw, lf);
  }
  const double g4 = weno_rec_pair<R, Z>(gp, gm, P.weno_eps);
  // entropy
#pragma unroll
  for (int m = 0; m < NW; ++m) {
    const double hr = 0.5 * ST(SF_RHO, O + m);
    const double lw = fma(-2.0, A[m], hr), lf = fma(-2.0, FA[m], hr * ST(SF_U + D, O + m));
    gp[m] = fma(lam[1], lw, lf);
    gm[NW - 1 - m] = fma(-lam[1], lw, lf);
  }
  const double g1 = weno_rec_pair<R, Z>(gp, gm, P.weno_eps);
  // the two shear fields
  double gs[2];
#pragma unroll
  for (int e = 0; e < 2; ++e) {
    const int t = e == 0 ? T1 : T2;
#pragma unroll
    for (int m = 0; m < NW; ++m) {
      const double lw = (0.5 * ST(SF_RHO, O + m)) * (ST(SF_U + t, O + m) - vb[t]);
      const double lf = ST(SF_U + D, O + m) * lw;
      gp[m] = fma(lam[1], lw, lf);
      gm[NW - 1 - m] = fma(-lam[1], lw, lf);
    }
    gs[e] = weno_rec_pair<R, Z>(gp, gm, P.weno_eps);
  }
  // f = sum over the fields of g r: r(u-+c) = (1, vbar -+ c e_D, H -+ un c), r(entropy) = (1, vbar, q^2/2), r(shear t) = (0, e_t, vbar_t)
  const double gsum = (g0 + g4) + g1, gdc = (g4 - g0) * cb;
  f[0] = gsum;
#pragma unroll
  for (int a = 0; a < 3; ++a) f[1 + a] = vb[a] * gsum;
  f[1 + D] += gdc;
  f[1 + T1] += gs[0];
  f[1 + T2] += gs[1];
  f[4] = fma(Hb, g0 + g4, fma(un, gdc, fma(qq, g1, fma(vb[T1], gs[0], vb[T2] * gs[1]))));
}
#undef ST

#ifndef STREAMS_WENO_MINB
#define STREAMS_WENO_MINB 4
#endif
// resident blocks per SM: the seventh-order reconstructions need more registers than 124
template <int R> struct WenoOcc { static constexpr int MINB = R >= 4 ? 2 : STREAMS_WENO_MINB; };

// ---------------------------------------------------------------------------------------------
// weno_kernel (full-WENO mode): every interface of every direction, the WENO flux itself stored at the left
// node's index.  Flat index over the interface slots of the three directions (slot = interior extents with the D
// extent enlarged by one; slot s along D is the interface between nodes s - 1 and s), grid-stride.
// ---------------------------------------------------------------------------------------------
template <int D, int M, int R, bool Z>
__device__ __forceinline__ void weno_dense_item(const DevP& P, long long t, double* s_st) {
  const long long s = D == 0 ? 1 : (D == 1 ? P.sy : P.sz);
  const int e0 = P.nx + (D == 0), e1 = P.ny + (D == 1);
  const int i = (int)(t % e0);
  const long long t1 = t / e0;
  const int j = (int)(t1 % e1), k = (int)(t1 / e1);
  const long long n = pidx(P, i - (D == 0), j - (D == 1), k - (D == 2));       // left node of the interface
  double fw[5], lam[3];
  weno_stencil<D, M, R>(P, n, s, s_st + threadIdx.x, lam);
  weno_flux<D, M, R, Z>(P, lam, fw, s_st + threadIdx.x);
  double* __restrict__ out = P.dF + ((long long)D * P.fs + n) * 5;      // record of the interface: five consecutive values
#pragma unroll
  for (int q = 0; q < 5; ++q) out[q] = fw[q];
}

template <int M, int R, bool Z>
__global__ void __launch_bounds__(WTH, WenoOcc<R>::MINB) weno_kernel(const DevP P) {
  __shared__ double s_st[6 * 2 * M * WTH];
  const long long a = (long long)P.nx * P.ny * P.nz;
  const long long n0 = a + (long long)P.ny * P.nz, n1 = a + (long long)P.nx * P.nz, n2 = a + (long long)P.nx * P.ny;
  const long long stride = (long long)gridDim.x * WTH;
  for (long long t = (long long)blockIdx.x * WTH + threadIdx.x; t < n0; t += stride) weno_dense_item<0, M, R, Z>(P, t, s_st);
  for (long long t = (long long)blockIdx.x * WTH + threadIdx.x; t < n1; t += stride) weno_dense_item<1, M, R, Z>(P, t, s_st);
  for (long long t = (long long)blockIdx.x * WTH + threadIdx.x; t < n2; t += stride) weno_dense_item<2, M, R, Z>(P, t, s_st);
}

// ---------------------------------------------------------------------------------------------
// weno_list_kernel (hybrid mode): the flagged interfaces of each direction were compacted into global work
// lists by flags_kernel (DevP::ilist, counts in DevP::counters), so every warp here is full of WENO work
// whatever the activation pattern.  Persistent blocks walk groups of WTH consecutive list entries
// (consecutive entries are mostly consecutive nodes: coalesced stencil loads), directions one after the other.
// ---------------------------------------------------------------------------------------------
template <int D, int M, int R, bool Z>
__device__ __forceinline__ void weno_list_item(const DevP& P, long long n, double* s_st) {
  const long long s = D == 0 ? 1 : (D == 1 ? P.sy : P.sz);
  double fw[5], fc[5], lam[3];
  weno_stencil<D, M, R>(P, n, s, s_st + threadIdx.x, lam);
  central_flux_st<D, M>(P, fc, s_st + threadIdx.x);        // first: its registers are free before the WENO rows are live
  weno_flux<D, M, R, Z>(P, lam, fw, s_st + threadIdx.x);
  double* __restrict__ out = P.dF + ((long long)D * P.fs + n) * 5;      // record of the interface: five consecutive values
#pragma unroll
  for (int q = 0; q < 5; ++q) out[q] = fw[q] - fc[q];
}

template <int M, int R, bool Z>
__global__ void __launch_bounds__(WTH, WenoOcc<R>::MINB) weno_list_kernel(const DevP P) {
  __shared__ double s_st[6 * 2 * M * WTH];
  const int c0 = P.counters[C_NIFACE], c1 = P.counters[C_NIFACE + 1], c2 = P.counters[C_NIFACE + 2];
  const int g0 = (c0 + WTH - 1) / WTH, g1 = (c1 + WTH - 1) / WTH, g2 = (c2 + WTH - 1) / WTH;
#ifndef STREAMS_WENO_CHUNK
#define STREAMS_WENO_CHUNK 4
#endif
  // blocks take chunks of consecutive groups round-robin: list neighbours are grid neighbours, so the stencil rows
  // of a group are still in this SM's L1 when the next rows' interfaces need them, while all blocks advance through
  // the lists together (one direction's code in the instruction cache at a time).  The list entry of the next item
  // is fetched before the current item is evaluated, which takes one dependent memory latency off every item.
  constexpr int CH = STREAMS_WENO_CHUNK;
  const int gt = g0 + g1 + g2;
  auto group_of = [&](int it) { return ((int)blockIdx.x + (it / CH) * (int)gridDim.x) * CH + (it % CH); };
  auto fetch = [&](int g, int& d) {                    // padded index of the left node of this thread's item, or -1
    d = 0;
    if (g >= gt) return -1;
    int e, cd;
    if (g < g0) { e = g * WTH + threadIdx.x; cd = c0; }
    else if (g < g0 + g1) { d = 1; e = (g - g0) * WTH + threadIdx.x; cd = c1; }
    else { d = 2; e = (g - g0 - g1) * WTH + threadIdx.x; cd = c2; }
    return e < cd ? P.ilist[(long long)d * P.lcap + e] : -1;
  };
  int d_cur, d_nxt;
  int n_cur = fetch(group_of(0), d_cur);
#pragma unroll 1
  for (int it = 0; group_of(it) < gt; ++it) {
    const int n_nxt = fetch(group_of(it + 1), d_nxt);
    if (n_cur >= 0) {
      if (d_cur == 0) weno_list_item<0, M, R, Z>(P, n_cur, s_st);
      else if (d_cur == 1) weno_list_item<1, M, R, Z>(P, n_cur, s_st);
      else weno_list_item<2, M, R, Z>(P, n_cur, s_st);
    }
    n_cur = n_nxt; d_cur = d_nxt;
  }
}

// ---------------------------------------------------------------------------------------------
// corr_gather_kernel: the net correction of a node, corr_q(n) = sum_d metric_d (dF_d,q(n) - dF_d,q(n - e_d)) over the
// flagged interfaces around it (hybrid: the bits of DevP::nflag, bit 2d = minus side, 2d+1 = plus side; full WENO:
// all six), directions in the order x, y, z.  dF holds stale values at interfaces that are not flagged: they are
// never read.  HBM: 1 B per node + (<= 30 R + 5 W) x 8 B per flagged node.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void corr_node(const DevP& P, long long n, unsigned fl, const double met[3]) {
  const long long st[3] = {1, P.sy, P.sz};
  // all (up to 30) gathers first, then the sums: the loads of a node are independent and scattered, their latency is
  // the kernel's time
  double fp[3][5], fm[3][5];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const double* __restrict__ f = P.dF + ((long long)d * P.fs + n) * 5;
    const bool hp = (fl >> (2 * d + 1)) & 1u, hm = (fl >> (2 * d)) & 1u;
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      fp[d][q] = hp ? __ldg(f + q) : 0.0;
      fm[d][q] = hm ? __ldg(f + q - 5 * st[d]) : 0.0;
    }
  }
  double c[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
#pragma unroll
    for (int q = 0; q < 5; ++q) c[q] = fma(met[d], fp[d][q] - fm[d][q], c[q]);
  }
#pragma unroll
  for (int q = 0; q < 5; ++q) P.corr[n * 5 + q] = c[q];                  // record of the node: five consecutive values
}

// full-WENO mode: every node, one thread each
__global__ void __launch_bounds__(128) corr_gather_dense_kernel(const DevP P) {
  const int i = blockIdx.x * 128 + threadIdx.x, j = blockIdx.y, k = blockIdx.z;
  if (i >= P.nx) return;
  const double met[3] = {P.inv_dx, P.eta_y_c[j], P.inv_dz};
  corr_node(P, pidx(P, i, j, k), 0x3fu, met);
}

// hybrid mode: flags_kernel has compacted the nodes next to a flagged interface into a fourth work list (DevP::ilist
// [3], count in DevP::counters[C_NIFACE + 3]); persistent blocks walk it, one thread per listed node, so every lane
// has a gather to do (a scan of the flag bytes of the whole grid by one thread per node took 1.4 ms on config 4, of
// which most was threads finding nothing to do).  Consecutive entries are mostly consecutive nodes: coalesced.
__global__ void __launch_bounds__(256) corr_gather_kernel(const DevP P) {
  const int count = P.counters[C_NIFACE + 3];
  const int* __restrict__ list = P.ilist + 3 * P.lcap;
  const int rowlen = (int)P.sy;
  for (int e = blockIdx.x * 256 + threadIdx.x; e < count; e += gridDim.x * 256) {
    const int n = list[e];
    const unsigned fl = P.nflag[n];
    const int j = (n / rowlen) % P.py - P.ng;        // row of the node (y metric)
    const double met[3] = {P.inv_dx, P.eta_y_c[j], P.inv_dz};
    corr_node(P, n, fl, met);
  }
}

// -------------------------------------------------------------------------- launch
template <int M, int R, bool Z>
static int launch_weno_Z(const DevP& P, cudaStream_t st) {
  if (P.flux_mode == FLUX_HYBRID) weno_list_kernel<M, R, Z><<<P.nsm * WenoOcc<R>::MINB, WTH, 0, st>>>(P);
  else weno_kernel<M, R, Z><<<P.nsm * WenoOcc<R>::MINB * 4, WTH, 0, st>>>(P);
  return 1;
}
template <int M, int R>
static int launch_weno_T(const DevP& P, cudaStream_t st) {
  if (P.weno_z && R > 1) return launch_weno_Z<M, R, true>(P, st);     // (first order has no weights)
  return launch_weno_Z<M, R, false>(P, st);
}

int launch_corr(const DevP& P, cudaStream_t st) {
  if (P.flux_mode == FLUX_CENTRAL) return 0;
  if (P.flux_mode == FLUX_HYBRID) {
    corr_gather_kernel<<<P.nsm * 8, 256, 0, st>>>(P);
  } else {
    dim3 b(128), g((unsigned)((P.nx + 127) / 128), (unsigned)P.ny, (unsigned)P.nz);
    corr_gather_dense_kernel<<<g, b, 0, st>>>(P);
  }
  return 1;
}

// (M, R): M = max(L, R) stencil nodes each side of the interface (hybrid: the central flux of order 2L is subtracted;
// full WENO: M = R), R = (weno_order + 1) / 2.  All ten pairs R <= M <= 4 are instantiated.
int launch_weno(const DevP& P, int L, int r, cudaStream_t st) {
  if (P.flux_mode == FLUX_CENTRAL) return 0;
  const int M = P.flux_mode == FLUX_HYBRID ? (L > r ? L : r) : r;
  if (r < 1 || r > 4 || M > 4 || M > P.ng) return -1;
#define STREAMS_WENO_CASE(MM, RR) if (M == MM && r == RR) return launch_weno_T<MM, RR>(P, st)
  STREAMS_WENO_CASE(1, 1);
  STREAMS_WENO_CASE(2, 1); STREAMS_WENO_CASE(2, 2);
  STREAMS_WENO_CASE(3, 1); STREAMS_WENO_CASE(3, 2); STREAMS_WENO_CASE(3, 3);
  STREAMS_WENO_CASE(4, 1); STREAMS_WENO_CASE(4, 2); STREAMS_WENO_CASE(4, 3); STREAMS_WENO_CASE(4, 4);
#undef STREAMS_WENO_CASE
  return -1;
}

}  // namespace streams
