// a4-a8 (+ a2, a1 and a9 of the next stage): the fused right-hand side, RK update and primitives.
//
//   weno_list_kernel : hybrid mode, runs first.  The flagged interfaces of each direction were compacted into work lists by
//                      flags_kernel; persistent blocks evaluate them with full warps: WENO characteristic flux (O3) minus
//                      the central flux that rhs_march_kernel implies there -> dF at the left node's index.
//   weno_kernel      : full-WENO mode: every interface, the WENO flux itself.
//   rhs_march_kernel : every node, one pass (2.5-D z-march, TMA + mbarrier pipeline): central split convective terms in
//                      x, y, z (O1), viscous terms (O4), -(dF_{n+1/2} - dF_{n-1/2}) metric at nodes next to a
//                      flagged interface, body force (S17), low-storage RK3 update (O5); then the primitives of the updated
//                      node into the OTHER primitive buffer (stencils of this stage still read the current one), also at
//                      its periodic images in the ghost layers, and in the last stage the time-step rate (a9).
// R, w and the primitives are written once per stage; every flagged interface is evaluated exactly once, by a warp
// whose lanes all do WENO work.
#include "streams_dev.cuh"
#include "streams_launch.h"
#include "streams_tma.cuh"

namespace streams {

template <int D>
__device__ __forceinline__ double pick(double a, double b, double c) { return D == 0 ? a : (D == 1 ? b : c); }

// fields of the marching kernel = the first nine slots of DevP::q
enum { F_U = Q_U, F_V = Q_V, F_W = Q_W, F_H = Q_H, F_P = Q_P, F_RHO = Q_RHO, F_T = Q_T, F_MU = Q_MU, F_DIV = Q_DIV };

// ------------------------------------------------------------------ arithmetic of one node
// Stencil coefficients of direction D.  x and z: the uniform metric is folded in on the host (DevP::avx ...);
// y: raw coefficients, the row's metrics are applied to the sums.
template <int D> __device__ __forceinline__ double coef_a(const DevP& P, int l) { return D == 0 ? P.avx[l] : (D == 1 ? P.a1v[l] : P.avz[l]); }
template <int D> __device__ __forceinline__ double coef_b(const DevP& P, int l) { return D == 0 ? P.bvx[l] : (D == 1 ? P.b2v[l] : P.bvz[l]); }

struct YMet { double eyc, eyv, eyv2, eyy; };   // d eta/dy (central order, viscous order), its square, d2 eta/dy2

// Viscous accumulators of a node (O4), folded as the derivatives arrive so that few values stay live:
//   vm_a  = mu (lap u_a + (d_a div)/3) + sum_b d_b mu (d_b u_a + d_a u_b) - 2/3 d_a mu div u
//   Phi   = mu [2 sum_a (d_a u_a)^2 + sum_{a<b} (d_b u_a + d_a u_b)^2 - 2/3 (div u)^2]
//   cond  = (cp/Pr) (mu lap T + grad mu . grad T)
struct Visc {
  double gmu[3];
  double vm[3];          // cross terms sum_b d_b mu (d_b u_a + d_a u_b)
  double lap[3];         // second-derivative sums of u_a + (d_a div)/3 (centre term applied at the end)
  double dv, ph, cond;
  double k10, k20, k21;  // d_x v, d_x w, d_y w kept for the symmetric strain terms
};

// grad mu, grad T, lap T, grad div along D; G(f, o) = field f at offset o along D.
template <int D, int LV, class G>
__device__ __forceinline__ void scalar_terms(const DevP& P, const G& g, const YMet& ym, double gT[3], double& lapT, Visc& V) {
  double dm = 0.0, dd = 0.0, dT = 0.0, sT = 0.0;
#pragma unroll
  for (int l = 1; l <= LV; ++l) {
    const double a = coef_a<D>(P, l - 1), b = coef_b<D>(P, l - 1);
    const double tb = g(F_T, l), ta = g(F_T, -l);
    dm = fma(a, g(F_MU, l) - g(F_MU, -l), dm);
    dd = fma(a, g(F_DIV, l) - g(F_DIV, -l), dd);
    dT = fma(a, tb - ta, dT);
    sT = fma(b, tb + ta, sT);
  }
  if (D == 1) {
    sT = fma(ym.eyy, dT, ym.eyv2 * sT);
    dm *= ym.eyv; dd *= ym.eyv; dT *= ym.eyv;
  }
  V.gmu[D] = dm;
  V.lap[D] = dd * (1.0 / 3.0);
  gT[D] = dT;
  lapT += sT;
}

// Convective terms (O1) and the velocity derivatives along D.
// Convective part in pair-difference form: with m(a,b) = (a_l/4)(rho_a+rho_b)(ud_a+ud_b),
//   f_{n+1/2} - f_{n-1/2} = sum_l [ m(n,n+l)(phi_n+phi_{n+l}) - m(n-l,n)(phi_{n-l}+phi_n) ]
//                         = phi_n S0 + sum_l [ m(n,n+l) phi_{n+l} - m(n-l,n) phi_{n-l} ],  S0 = sum_l [m(n,n+l) - m(n-l,n)]
// (the oracle's interface-flux sum, regrouped), plus sum_l a_l (p_{n+l} - p_{n-l}) on the D-momentum.
// c0 = (u, v, w, H, p, rho) at the node, alr[l] = (a_l/4) rho_0.
template <int D, int L, int LV, bool CONV, bool VISC, class G>
__device__ __forceinline__ void dir_terms(const DevP& P, const G& g, const YMet& ym, const double c0[6],
                                          const double alr[3], double r[5], Visc& V) {
  constexpr int LC = CONV ? L : 0;
  constexpr int LVV = VISC ? LV : 0;
  constexpr int LM = LC > LVV ? LC : LVV;
  double S0 = 0.0, S[4] = {0.0, 0.0, 0.0, 0.0}, SP = 0.0;
  double d1[3] = {0.0, 0.0, 0.0}, d2[3] = {0.0, 0.0, 0.0};
  const double ud0 = pick<D>(c0[0], c0[1], c0[2]);
#pragma unroll
  for (int l = 1; l <= LM; ++l) {
    const double ub = g(F_U, l), ua = g(F_U, -l);
    const double vb = g(F_V, l), va = g(F_V, -l);
    const double wb = g(F_W, l), wa = g(F_W, -l);
    if constexpr (CONV) if (l <= LC) {
      const double rb = g(F_RHO, l), ra = g(F_RHO, -l);
      const double hb = g(F_H, l), ha = g(F_H, -l);
      const double pb = g(F_P, l), pa = g(F_P, -l);
      const double mb = fma(P.kc[l - 1], rb, alr[l - 1]) * (ud0 + pick<D>(ub, vb, wb));
      const double ma = fma(P.kc[l - 1], ra, alr[l - 1]) * (pick<D>(ua, va, wa) + ud0);
      S0 += mb - ma;
      S[0] = fma(mb, ub, S[0]); S[0] = fma(-ma, ua, S[0]);
      S[1] = fma(mb, vb, S[1]); S[1] = fma(-ma, va, S[1]);
      S[2] = fma(mb, wb, S[2]); S[2] = fma(-ma, wa, S[2]);
      S[3] = fma(mb, hb, S[3]); S[3] = fma(-ma, ha, S[3]);
      SP = fma(P.a1[l - 1], pb - pa, SP);
    }
    if constexpr (VISC) if (l <= LVV) {
      const double a = coef_a<D>(P, l - 1), b = coef_b<D>(P, l - 1);
      d1[0] = fma(a, ub - ua, d1[0]);  d2[0] = fma(b, ub + ua, d2[0]);
      d1[1] = fma(a, vb - va, d1[1]);  d2[1] = fma(b, vb + va, d2[1]);
      d1[2] = fma(a, wb - wa, d1[2]);  d2[2] = fma(b, wb + wa, d2[2]);
    }
  }
  if (CONV) {
    const double met = D == 0 ? P.inv_dx : (D == 1 ? ym.eyc : P.inv_dz);
    r[0] = fma(-2.0 * met, S0, r[0]);
#pragma unroll
    for (int q = 0; q < 4; ++q) r[1 + q] = fma(-met, fma(c0[q], S0, S[q]), r[1 + q]);
    r[1 + D] = fma(-met, SP, r[1 + D]);
  }
  if (VISC) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      if (D == 1) {
        d2[a] = fma(ym.eyy, d1[a], ym.eyv2 * d2[a]);
        d1[a] *= ym.eyv;
      }
      V.lap[a] += d2[a];
      V.vm[a] = fma(V.gmu[D], d1[a], V.vm[a]);          // d_D mu d_D u_a
    }
    double t = V.gmu[0] * d1[0];                          // sum_a d_a mu d_D u_a -> vm_D
    t = fma(V.gmu[1], d1[1], t);
    t = fma(V.gmu[2], d1[2], t);
    V.vm[D] += t;
    V.dv += d1[D];
    V.ph = fma(d1[D], d1[D], V.ph);                       // doubled at the end
    if (D == 0) { V.k10 = d1[1]; V.k20 = d1[2]; }
    if (D == 1) { const double s01 = d1[0] + V.k10; V.k10 = s01 * s01; V.k21 = d1[2]; }
    if (D == 2) {
      const double s02 = d1[0] + V.k20, s12 = d1[1] + V.k21;
      V.k20 = fma(s02, s02, V.k10);
      V.k20 = fma(s12, s12, V.k20);                       // sum of the squared off-diagonal strains
    }
  }
}

// closes the viscous terms of a node: c0 = (u, v, w, ...), T0, mu0 at the node, sb2 = -2 sum_d sum_l b_l metric_d^2
__device__ __forceinline__ void viscous_close(const DevP& P, const double c0[6], double mu0, double sb2, double r[5], Visc& V) {
  const double tdv = (2.0 / 3.0) * V.dv;
  double e = fma(mu0, fma(-tdv, V.dv, fma(2.0, V.ph, V.k20)), P.kfac * V.cond);
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double lap = fma(sb2, c0[a], V.lap[a]);
    const double vm = fma(mu0, lap, fma(-V.gmu[a], tdv, V.vm[a]));
    r[1 + a] += vm;
    e = fma(c0[a], vm, e);
  }
  r[4] += e;
}

// ---------------------------------------------------------------------------------------------
// rhs_march_kernel (a4-a8 in one pass).  A block owns a 32 x TY tile of (x, y) and marches through a chunk
// of z planes (2.5-D blocking):
//   - z neighbours: every thread keeps the 7-plane column (k-3 .. k+3) of its node for all fields in
//     registers; plane k+4 arrives by TMA in a shared-memory slot and enters the ring at the shift;
//   - x / y neighbours: the centre plane of all fields with its 3-wide halo is ONE 4-D TMA box
//     (x, y, z, field) = (40, TY+6, 1, 9) into one of two shared-memory buffers, issued two planes ahead;
//     every stencil offset is a compile-time immediate;
//   - RK operands (w, previous-stage R) of the plane arrive by TMA one plane ahead;
//   - flux corrections of flagged interfaces (hybrid / WENO): cp.async with zero fill, by the warps that
//     have a flagged node only.
// One thread issues the TMA copies after a split barrier (bar.arrive by the other warps, bar.sync by
// its warp), so no warp but that one waits for the slowest.  Completion is tracked by mbarriers.
// ---------------------------------------------------------------------------------------------
template <int TY, bool VISC, bool WENO>
struct MarchSmem {
  using G = MarchGeom<TY>;
  static constexpr int NF = VISC ? 9 : 6;
  static constexpr size_t BUF = (size_t)NF * G::PLANE * 8;     // one centre-plane buffer
  static constexpr size_t RING = (size_t)NF * G::NT * 8;       // one ring-plane slot
  static constexpr size_t EPI = (size_t)10 * G::NT * 8;        // one RK-operand slot: R[5], w[5]
  static constexpr size_t DFS = WENO ? (size_t)30 * G::NT * 8 : 0;
  static constexpr size_t OFF_RING = 2 * BUF, OFF_EPI = OFF_RING + 2 * RING, OFF_DFS = OFF_EPI + 2 * EPI,
                          OFF_BAR = OFF_DFS + DFS, TOTAL = OFF_BAR + 32 + 8 * 32;   // 4 mbarriers, rate scratch
  static_assert(BUF % 128 == 0 && RING % 128 == 0 && EPI % 128 == 0, "TMA destinations are 128-byte aligned");
};

template <int L, int LV, bool VISC, bool CONV, bool WENO, int TY>
#ifndef STREAMS_MARCH_MINB
#define STREAMS_MARCH_MINB 1
#endif
__global__ void __launch_bounds__(MTX * TY, STREAMS_MARCH_MINB)
rhs_march_kernel(const __grid_constant__ CUtensorMap tm_centre, const __grid_constant__ CUtensorMap tm_ring,
                 const __grid_constant__ CUtensorMap tm_w, const __grid_constant__ CUtensorMap tm_r, const DevP P,
                 const StageArgs sa, int nbx, int nby, int kz) {
  using G = MarchGeom<TY>;
  using SM = MarchSmem<TY, VISC, WENO>;
  constexpr int NF = SM::NF;
  constexpr int NG = 3;
  static_assert(L <= NG && LV <= NG, "ring depth");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double* const buf = reinterpret_cast<double*>(smem_raw);                  // [2][NF][PLANE]
  double* const ring = reinterpret_cast<double*>(smem_raw + SM::OFF_RING);  // [2][NF][NT]
  double* const epi = reinterpret_cast<double*>(smem_raw + SM::OFF_EPI);    // [2][10][NT]
  double* const dfs = reinterpret_cast<double*>(smem_raw + SM::OFF_DFS);    // [30][NT]
  unsigned long long* const bars = reinterpret_cast<unsigned long long*>(smem_raw + SM::OFF_BAR);
  unsigned long long* const full_c = bars;        // [2] centre plane landed
  unsigned long long* const full_e = bars + 2;    // [2] ring plane + RK operands landed

  const int tid = threadIdx.x;
  const int tx = tid & 31, ty = tid >> 5;
  int bid = blockIdx.x;
  const int bx = bid % nbx; bid /= nbx;
  const int by = bid % nby;
  const int bc = bid / nby;
  const int i0 = bx * MTX, j0 = by * TY;
  const int kb = bc * kz, ke = min(P.nz, kb + kz);
  if (kb >= ke) return;
  const int i = i0 + tx, j = j0 + ty;
  const bool active = i < P.nx && j < P.ny;
  const int ic = min(i, P.nx + P.ng - 1), jc = min(j, P.ny + P.ng - 1);
  const int isz = (int)P.sz;
  const int ncol = (int)pidx(P, ic, jc, 0);            // this thread's column at k = 0 (padded index < 2^31)
  const int s0 = (ty + 3) * G::ROW + tx + 4;           // this node in a shared-memory plane

  const unsigned bytes_c = (unsigned)SM::BUF;
  const unsigned bytes_e = (unsigned)SM::RING + (sa.update_w ? 5u * G::NT * 8u : 0u) + (sa.read_prev ? 5u * G::NT * 8u : 0u);
  const int cx0 = i0 + P.ox, cy0 = j0 + P.ng;          // tile origin in padded coordinates

  auto issue_centre = [&](int k, int b) {              // thread 0 only
    mbar_expect_tx(&full_c[b], bytes_c);
    tma_load_4d(buf + (size_t)b * NF * G::PLANE, &tm_centre, &full_c[b], cx0 - 4, cy0 - 3, k + P.ng, 0);
  };
  auto issue_ring_epi = [&](int k, int b) {            // ring plane k+4 and the RK operands of plane k into slot b
    mbar_expect_tx(&full_e[b], bytes_e);
    tma_load_4d(ring + (size_t)b * NF * G::NT, &tm_ring, &full_e[b], cx0, cy0, k + NG + 1 + P.ng, 0);
    if (sa.read_prev) tma_load_4d(epi + (size_t)b * 10 * G::NT, &tm_r, &full_e[b], cx0, cy0, k + P.ng, 0);
    if (sa.update_w) tma_load_4d(epi + (size_t)b * 10 * G::NT + 5 * G::NT, &tm_w, &full_e[b], cx0, cy0, k + P.ng, 0);
  };

#ifndef STREAMS_MARCH_PF
#define STREAMS_MARCH_PF 2
#endif
  // The streams that miss L2 (the new ring plane and the RK operands) are needed one plane after they are
  // issued, which keeps too few bytes in flight to cover the DRAM latency: PF planes further ahead the same
  // boxes are requested into L2 only.
  constexpr int PF = (VISC || WENO) ? 0 : STREAMS_MARCH_PF;   // measured: helps the lean variant only
  auto prefetch_ring_epi = [&](int k) {                // thread 0 only
    if (PF > 0 && k < ke) {
      tma_prefetch_4d(&tm_ring, cx0, cy0, k + NG + 1 + P.ng, 0);
      if (sa.read_prev) tma_prefetch_4d(&tm_r, cx0, cy0, k + P.ng, 0);
      if (sa.update_w) tma_prefetch_4d(&tm_w, cx0, cy0, k + P.ng, 0);
    }
  };
  if (tid == 0) {
    mbar_init(&full_c[0], 1); mbar_init(&full_c[1], 1);
    mbar_init(&full_e[0], 1); mbar_init(&full_e[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) {
    issue_centre(kb, 0);
    if (kb + 1 < ke) issue_centre(kb + 1, 1);
    issue_ring_epi(kb, 0);
#pragma unroll
    for (int a = 1; a <= PF; ++a) prefetch_ring_epi(kb + a);
  }

  // metrics of this row (constant along the march)
  YMet ym;
  ym.eyc = P.eta_y_c[min(j, P.ny - 1)];
  ym.eyv = ym.eyv2 = ym.eyy = 0.0;
  if (VISC) {
    ym.eyv = P.eta_y_v[min(j, P.ny - 1)];
    ym.eyv2 = ym.eyv * ym.eyv;
    ym.eyy = P.eta_yy_v[min(j, P.ny - 1)];
  }
  const double sb2 = fma(-2.0 * P.sbv, ym.eyv2, P.sb2xz);
  const double dt = sa.update_w ? P.scal[S_DT] : 0.0;

  // ring = planes kb-3 .. kb+3 of this thread's column
  double zr[NF][2 * NG + 1];
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    const double* __restrict__ fp = P.q + (long long)f * P.fs + ncol + (long long)(kb - NG) * P.sz;
#pragma unroll
    for (int m = 0; m < 2 * NG + 1; ++m) zr[f][m] = fp[(long long)m * P.sz];
  }
  // offsets (doubles) of this node's periodic images in the ghost layers, 0 = none (DevP::own_*)
  const int xoff = !P.own_x ? 0 : (i < NG ? P.nx : (i >= P.nx - NG ? -P.nx : 0));
  const int yoff = !P.own_y ? 0 : (j < NG ? P.ny * (int)P.sy : (j >= P.ny - NG ? -P.ny * (int)P.sy : 0));
  double rate = 0.0;                                  // a9 of the next step (last stage only)
  bool rate_nan = false;
  unsigned fl_next = 0;
  if (WENO && CONV && active) fl_next = ld_u8_now(P.nflag + ncol + (long long)kb * P.sz);

  for (int k = kb; k < ke; ++k) {
    const int it = k - kb, b = it & 1;
    const unsigned par = (unsigned)(it >> 1) & 1u;
    const int n = ncol + k * isz;
    if (tid == G::NT - 32) prefetch_ring_epi(k + 1 + PF);   // no shared-memory hazard: any thread, off the issuing warp's path
    // flags of this plane (prefetched), of the next one, and this plane's flux corrections
    unsigned fl = 0;
    bool any_fl = false;
    if (WENO) {
      fl = CONV ? fl_next : (active ? 0x3fu : 0u);
      if (CONV && active && k + 1 < ke) fl_next = ld_u8_now(P.nflag + n + isz);
      any_fl = __any_sync(0xffffffffu, fl != 0);
      if (any_fl) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
          const int sd = d == 0 ? 1 : (d == 1 ? (int)P.sy : isz);
          const double* __restrict__ f = P.dF + (long long)(d * 5) * P.fs + n;
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            cp_async8_zfill(dfs + ((d * 5 + q) * 2 + 0) * G::NT + tid, f + (long long)q * P.fs, (fl >> (2 * d + 1)) & 1u);
            cp_async8_zfill(dfs + ((d * 5 + q) * 2 + 1) * G::NT + tid, f + (long long)q * P.fs - sd, (fl >> (2 * d)) & 1u);
          }
        }
      }
    }

    // (C) the right-hand side of this node
    mbar_wait(&full_c[b], par);
    const double* __restrict__ sc = buf + (size_t)b * NF * G::PLANE + s0;
    auto gx = [&](int f, int o2) { return sc[f * G::PLANE + o2]; };
    auto gy = [&](int f, int o2) { return sc[f * G::PLANE + o2 * G::ROW]; };
    auto gz = [&](int f, int o2) { return zr[f][NG + o2]; };
    double c0[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) c0[q] = zr[q][NG];
    double alr[3];
#pragma unroll
    for (int l = 0; l < 3; ++l) alr[l] = P.kc[l] * c0[F_RHO];
    double r[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    Visc V;
    if (VISC) {
      double gT[3], lapT = 0.0;
      scalar_terms<0, LV>(P, gx, ym, gT, lapT, V);
      scalar_terms<1, LV>(P, gy, ym, gT, lapT, V);
      scalar_terms<2, LV>(P, gz, ym, gT, lapT, V);
      const double mu0 = zr[VISC ? F_MU : 0][NG];
      double cond = mu0 * fma(sb2, zr[VISC ? F_T : 0][NG], lapT);
      cond = fma(V.gmu[0], gT[0], cond);
      cond = fma(V.gmu[1], gT[1], cond);
      V.cond = fma(V.gmu[2], gT[2], cond);
      V.vm[0] = V.vm[1] = V.vm[2] = 0.0;
      V.dv = 0.0; V.ph = 0.0;
    }
    dir_terms<0, L, LV, CONV, VISC>(P, gx, ym, c0, alr, r, V);
    dir_terms<1, L, LV, CONV, VISC>(P, gy, ym, c0, alr, r, V);
    dir_terms<2, L, LV, CONV, VISC>(P, gz, ym, c0, alr, r, V);
    if (VISC) viscous_close(P, c0, zr[VISC ? F_MU : 0][NG], sb2, r, V);

    // every warp is done with buf[b], ring[b^1], epi[b^1]: the issuing thread refills them
    // (two alternating barrier ids: a warp may run one iteration ahead of the slowest)
    if (tid >> 5) {
      if (b) asm volatile("bar.arrive 2, %0;" ::"n"(G::NT) : "memory");
      else asm volatile("bar.arrive 1, %0;" ::"n"(G::NT) : "memory");
    } else {
      if (b) asm volatile("bar.sync 2, %0;" ::"n"(G::NT) : "memory");
      else asm volatile("bar.sync 1, %0;" ::"n"(G::NT) : "memory");
      if (tid == 0) {
        if (k + 1 < ke) issue_ring_epi(k + 1, b ^ 1);   // needed one plane from now: ahead of the larger centre box
        if (k + 2 < ke) issue_centre(k + 2, b);
      }
    }

    // (D) flux corrections of flagged interfaces, RK update, stores
    mbar_wait(&full_e[b], par);
    const double* __restrict__ ep = epi + (size_t)b * 10 * G::NT + tid;
    if (WENO && any_fl) {
      cp_async_wait_all();
      const double met[3] = {P.inv_dx, ym.eyc, P.inv_dz};
#pragma unroll
      for (int d = 0; d < 3; ++d) {
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          const double fp = dfs[((d * 5 + q) * 2 + 0) * G::NT + tid];
          const double fm = dfs[((d * 5 + q) * 2 + 1) * G::NT + tid];
          r[q] = fma(-met[d], fp - fm, r[q]);
        }
      }
    }
    if (P.has_accel) {                               // S17: uniform body acceleration and its work
      const double rho0 = c0[F_RHO];
#pragma unroll
      for (int a = 0; a < 3; ++a) r[1 + a] = fma(rho0, P.accel[a], r[1 + a]);
      r[4] = fma(rho0, fma(c0[F_U], P.accel[0], fma(c0[F_V], P.accel[1], c0[F_W] * P.accel[2])), r[4]);
    }
    if (active) {
      if (sa.update_w) {
        double wn[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          double inc = sa.gam * r[q];
          if (sa.read_prev) inc = fma(sa.rhk, ep[q * G::NT], inc);
          wn[q] = fma(dt, inc, ep[(5 + q) * G::NT]);
          P.w[(long long)q * P.fs + n] = wn[q];
        }
        // a2 of the next stage: the primitives of the updated node go to the other q buffer (stencils of this
        // stage still read the current one); the next stage only fills the ghost shell
        double mu, cc, vel[3], o[NQ];
        prims_from_state<VISC, WENO>(P, wn, sa.want_rate != 0, o, mu, cc, vel);
        double* __restrict__ qo = sa.q_out + n;
        store_prims<VISC, WENO>(P, qo, o);
        // a1 of the next stage for the periodic directions: the owner also writes its images in the ghost layers
        const int zoff = !P.own_z ? 0 : (k < NG ? P.nz * isz : (k >= P.nz - NG ? -P.nz * isz : 0));
        if (xoff) store_prims<VISC, WENO>(P, qo + xoff, o);
        if (yoff) store_prims<VISC, WENO>(P, qo + yoff, o);
        if (zoff) store_prims<VISC, WENO>(P, qo + zoff, o);
        if (sa.want_rate) rate = fmax(rate, dt_rate<VISC>(P, vel, cc, mu, wn[0], ym.eyc));
        if (sa.want_rate && !(rate == rate)) rate_nan = true;   // fmax would drop a NaN on the next plane
      }
      if (sa.write_r) {
#pragma unroll
        for (int q = 0; q < 5; ++q) P.R[(long long)q * P.fs + n] = r[q];
      }
      if (sa.r_dense) {
        const long long o = ((long long)k * P.ny + j) * P.nx + i;
#pragma unroll
        for (int q = 0; q < 5; ++q) sa.r_dense[q * P.N + o] = r[q];
      }
    }

    // (E) shift the ring
    const double* __restrict__ rn = ring + (size_t)b * NF * G::NT + tid;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
#pragma unroll
      for (int m = 0; m < 2 * NG; ++m) zr[f][m] = zr[f][m + 1];
      zr[f][2 * NG] = rn[f * G::NT];
    }
  }
  // a9 of the next step: one atomicMax per block on the bit pattern of the largest rate (a NaN wins)
  if (sa.want_rate) {
    if (rate_nan) rate = __longlong_as_double(0x7ff8000000000000LL);
    block_rate_max(P, rate, bars + 4);
  }
}

// ---------------------------------------------------------------------------------------------
// WENO reconstruction of order 2R-1 with Jiang-Shu weights (O3 step 4); v[0..2R-2] upwind->downwind,
// value at the interface between v[R-1] and v[R].
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double sq(double x) { return x * x; }

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

// Both reconstructions of a characteristic field (upwind and mirrored stencil) as ONE call with the arguments by
// value, in registers: the five fields of an interface then share one copy of the code instead of ten inlined
// reconstructions (instruction-cache footprint: the list kernel's straight-line code shrinks by 30 %), while the two
// reconstructions of a field still interleave.  STREAMS_WENO_REC_INLINE restores the inlined form.
template <int R>
__device__ __forceinline__ double weno_rec_pair(const double* gp, const double* gm, double eps) {
  return weno_rec<R>(gp, eps) + weno_rec<R>(gm, eps);
}
#ifndef STREAMS_WENO_REC_INLINE
__device__ __noinline__ double weno_rec5_pair_call(double p0, double p1, double p2, double p3, double p4, double m0, double m1,
                                                  double m2, double m3, double m4, double eps) {
  const double gp[5] = {p0, p1, p2, p3, p4}, gm[5] = {m0, m1, m2, m3, m4};
  return weno_rec<3>(gp, eps) + weno_rec<3>(gm, eps);
}
template <>
__device__ __forceinline__ double weno_rec_pair<3>(const double* gp, const double* gm, double eps) {
  return weno_rec5_pair_call(gp[0], gp[1], gp[2], gp[3], gp[4], gm[0], gm[1], gm[2], gm[3], gm[4], eps);
}
#endif

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
// The 2R-node stencil of (rho, u, v, w, H, p) lives in a per-thread column of shared memory
// (st[(f * 2R + m) * WTH], conflict-free) so that the kernel fits 4 blocks of 128 threads per SM; every node is
// read once per pass (central pairs, shared rows, entropy row, shear rows): ~120 loads per interface.
// ---------------------------------------------------------------------------------------------
constexpr int WTH = 128;       // threads per block of weno_kernel
constexpr int WCH = 2048;      // interface slots per block

#define ST(fld, m) (((volatile double*)st)[((fld) * NS + (m)) * WTH])
enum { SF_RHO = 0, SF_U = 1, SF_V = 2, SF_W = 3, SF_H = 4, SF_P = 5 };

// Central interface flux (O1) from the shared-memory stencil (needs L <= R): the flux that rhs_march_kernel's
// pair-difference form implies at this interface.  f = 1/4 sum_l a_l sum_{m<l} (rho_a+rho_b)(ud_a+ud_b)(phi_a+phi_b),
// pairs (a, b) = (n-m, n-m+l).  The L left nodes stay in registers, the right nodes stream past them.
template <int D, int L, int R>
__device__ __forceinline__ void central_flux_st(const DevP& P, double f[5], const double* st) {
  static_assert(L <= R, "the central stencil must fit in the WENO stencil");
  constexpr int NS = 2 * R;
  double lf[L][6];                                 // left nodes n, n-1, .., n-L+1: rho, u, v, w, H, p
#pragma unroll
  for (int m = 0; m < L; ++m) {
#pragma unroll
    for (int q = 0; q < 6; ++q) lf[m][q] = ST(q, R - 1 - m);
  }
  double fs[5] = {0.0, 0.0, 0.0, 0.0, 0.0}, ps = 0.0;
#pragma unroll
  for (int j = 0; j < L; ++j) {                    // right node n+1+j pairs with left node n-m at distance l = j+1+m
    double rt[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) rt[q] = ST(q, R + j);
#pragma unroll
    for (int m = 0; m + j < L; ++m) {
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
// Lax-Friedrichs speeds max |u_D - c|, |u_D|, |u_D + c| over its 2R nodes.
template <int D, int R>
__device__ __forceinline__ void weno_stencil(const DevP& P, long long n, long long s, double* __restrict__ st, double lam[3]) {
  constexpr int NS = 2 * R;
  lam[0] = lam[1] = lam[2] = 0.0;
#pragma unroll
  for (int m = 0; m < NS; ++m) {
    const long long a = n + (long long)(m - R + 1) * s;
    const double u = P.q[Q_U * P.fs + a], v = P.q[Q_V * P.fs + a], w = P.q[Q_W * P.fs + a];
    const double c = P.q[Q_C * P.fs + a];
    ST(SF_RHO, m) = P.q[Q_RHO * P.fs + a];
    ST(SF_U, m) = u;
    ST(SF_V, m) = v;
    ST(SF_W, m) = w;
    ST(SF_H, m) = P.q[Q_H * P.fs + a];
    ST(SF_P, m) = P.q[Q_P * P.fs + a];
    const double ud = D == 0 ? u : (D == 1 ? v : w);
    lam[0] = fmax(lam[0], fabs(ud - c));
    lam[1] = fmax(lam[1], fabs(ud));
    lam[2] = fmax(lam[2], fabs(ud + c));
  }
}

template <int D, int R>
__device__ __forceinline__ void weno_flux(const DevP& P, const double lam[3], double f[5], const double* __restrict__ st) {
  constexpr int NS = 2 * R;
  // Roe average of nodes n (slot R-1) and n+1 (slot R)
  const double rw = sqrt(ST(SF_RHO, R) * rcp_pos(ST(SF_RHO, R - 1)));
  const double iden = rcp_pos(1.0 + rw);
  double vb[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) vb[a] = (ST(SF_U + a, R - 1) + rw * ST(SF_U + a, R)) * iden;
  const double Hb = (ST(SF_H, R - 1) + rw * ST(SF_H, R)) * iden;
  const double qq = 0.5 * (vb[0] * vb[0] + vb[1] * vb[1] + vb[2] * vb[2]);
  const double cb = sqrt(P.gm1 * (Hb - qq));
  const double ic = rcp_pos(cb);
  const double un = vb[D];
  const double k1 = 0.25 * (P.gm1 * (ic * ic)), k2 = qq * k1, ki = 0.25 * ic;
  constexpr int T1 = (D == 0) ? 1 : 0;
  constexpr int T2 = (D == 2) ? 1 : 2;
  double gp[NS], gm[NS];

  // shared rows of the two acoustic fields and the entropy field, one pass over the nodes
  double A[NS], B[NS], FA[NS], FB[NS];
#pragma unroll
  for (int m = 0; m < NS; ++m) {
    const double rho = ST(SF_RHO, m), um = ST(SF_U, m), vm = ST(SF_V, m), wm = ST(SF_W, m), hm = ST(SF_H, m), pm = ST(SF_P, m);
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
  for (int m = 0; m < NS; ++m) {
    const double lw = A[m] + B[m], lf = FA[m] + FB[m];
    gp[m] = fma(lam[0], lw, lf);
    gm[NS - 1 - m] = fma(-lam[0], lw, lf);          // mirrored: gm[0] is node n+R
  }
  const double g0 = weno_rec_pair<R>(gp, gm, P.weno_eps);
  // u + c
#pragma unroll
  for (int m = 0; m < NS; ++m) {
    const double lw = A[m] - B[m], lf = FA[m] - FB[m];
    gp[m] = fma(lam[2], lw, lf);
    gm[NS - 1 - m] = fma(-lam[2], lw, lf);
  }
  const double g4 = weno_rec_pair<R>(gp, gm, P.weno_eps);
  // entropy
#pragma unroll
  for (int m = 0; m < NS; ++m) {
    const double hr = 0.5 * ST(SF_RHO, m);
    const double lw = fma(-2.0, A[m], hr), lf = fma(-2.0, FA[m], hr * ST(SF_U + D, m));
    gp[m] = fma(lam[1], lw, lf);
    gm[NS - 1 - m] = fma(-lam[1], lw, lf);
  }
  const double g1 = weno_rec_pair<R>(gp, gm, P.weno_eps);
  // the two shear fields
  double gs[2];
#pragma unroll
  for (int e = 0; e < 2; ++e) {
    const int t = e == 0 ? T1 : T2;
#pragma unroll
    for (int m = 0; m < NS; ++m) {
      const double lw = (0.5 * ST(SF_RHO, m)) * (ST(SF_U + t, m) - vb[t]);
      const double lf = ST(SF_U + D, m) * lw;
      gp[m] = fma(lam[1], lw, lf);
      gm[NS - 1 - m] = fma(-lam[1], lw, lf);
    }
    gs[e] = weno_rec_pair<R>(gp, gm, P.weno_eps);
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
    double fw[5], lam[3];
    weno_stencil<D, R>(P, n, s, s_st + threadIdx.x, lam);
    weno_flux<D, R>(P, lam, fw, s_st + threadIdx.x);
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

// ---------------------------------------------------------------------------------------------
// weno_list_kernel (hybrid mode): the flagged interfaces of each direction were compacted into global work
// lists by flags_kernel (DevP::ilist, counts in DevP::counters), so every warp here is full of WENO work
// whatever the activation pattern.  Persistent blocks walk groups of WTH consecutive list entries
// (consecutive entries are mostly consecutive nodes: coalesced stencil loads), directions one after the other.
// ---------------------------------------------------------------------------------------------
template <int D, int L, int R>
__device__ __forceinline__ void weno_list_item(const DevP& P, long long n, double* s_st) {
  const long long s = D == 0 ? 1 : (D == 1 ? P.sy : P.sz);
  double fw[5], fc[5], lam[3];
  weno_stencil<D, R>(P, n, s, s_st + threadIdx.x, lam);
  central_flux_st<D, L, R>(P, fc, s_st + threadIdx.x);     // first: its registers are free before the WENO rows are live
  weno_flux<D, R>(P, lam, fw, s_st + threadIdx.x);
  double* __restrict__ out = P.dF + (long long)(D * 5) * P.fs + n;
#pragma unroll
  for (int q = 0; q < 5; ++q) out[q * P.fs] = fw[q] - fc[q];
}

template <int L, int R>
__global__ void __launch_bounds__(WTH, STREAMS_WENO_MINB) weno_list_kernel(const DevP P) {
  __shared__ double s_st[6 * 2 * R * WTH];
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
      if (d_cur == 0) weno_list_item<0, L, R>(P, n_cur, s_st);
      else if (d_cur == 1) weno_list_item<1, L, R>(P, n_cur, s_st);
      else weno_list_item<2, L, R>(P, n_cur, s_st);
    }
    n_cur = n_nxt; d_cur = d_nxt;
  }
}

// -------------------------------------------------------------------------- launch
template <int L, int LV, bool VISC, bool CONV, bool WENO, int TY>
static int launch_march(const DevP& P, const MarchMaps& mp, const StageArgs& sa, cudaStream_t st) {
  using G = MarchGeom<TY>;
  using SM = MarchSmem<TY, VISC, WENO>;
  auto kern = rhs_march_kernel<L, LV, VISC, CONV, WENO, TY>;
  static int attr_dev = -1;                          // the opt-in is per device: redo it when the current device changes
  int dev = 0;
  cudaGetDevice(&dev);
  if (attr_dev != dev) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM::TOTAL) != cudaSuccess) return -2;
    attr_dev = dev;
  }
  const int nbx = (P.nx + MTX - 1) / MTX, nby = (P.ny + TY - 1) / TY;
  const int tiles = nbx * nby;
  const int chunks = pick_chunks(tiles, P.nz, P.nsm * STREAMS_MARCH_MINB);
  const int kz = (P.nz + chunks - 1) / chunks;
  kern<<<(unsigned)(tiles * chunks), G::NT, SM::TOTAL, st>>>(mp.centre, mp.ring, mp.w, mp.r, P, sa, nbx, nby, kz);
  return 1;
}

template <int L, int LV, int R>
static int launch_main_T(const DevP& P, const MarchMaps& mp, const StageArgs& sa, cudaStream_t st) {
  const bool visc = P.visc_law != VISC_NONE;
  const bool conv = P.flux_mode != FLUX_WENO;
  const bool weno = P.flux_mode != FLUX_CENTRAL;
  constexpr int TY = STREAMS_MARCH_TY;
#define STREAMS_MAIN(V, C, W) return launch_march<L, LV, V, C, W, TY>(P, mp, sa, st)
  if (visc && conv && weno) STREAMS_MAIN(true, true, true);
  else if (visc && conv) STREAMS_MAIN(true, true, false);
  else if (visc) STREAMS_MAIN(true, false, true);
  else if (conv && weno) STREAMS_MAIN(false, true, true);
  else if (conv) STREAMS_MAIN(false, true, false);
  else STREAMS_MAIN(false, false, true);
#undef STREAMS_MAIN
}

// TMA descriptors (cuTensorMapEncodeTiled through the runtime's driver entry point: libstreams does not link
// libcuda).  All four tensors are 4-D (x, y, z, field) views of padded fields: the primitives + dilatation
// (DevP::q, NF fields), w and R (5 fields each).
int make_march_maps(const DevP& P, MarchMaps* maps) {
  typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess)
    return -1;
  const encode_fn encode = (encode_fn)fn;
  constexpr int TY = STREAMS_MARCH_TY;
  const cuuint32_t nf = P.visc_law != VISC_NONE ? 9 : 6;
  const cuuint64_t strides[3] = {(cuuint64_t)P.px * 8, (cuuint64_t)P.sz * 8, (cuuint64_t)P.fs * 8};
  const cuuint32_t ones[4] = {1, 1, 1, 1};
  auto make = [&](CUtensorMap* m, void* base, cuuint64_t nfields, cuuint32_t bx, cuuint32_t by, cuuint32_t bf) {
    const cuuint64_t dims[4] = {(cuuint64_t)P.px, (cuuint64_t)P.py, (cuuint64_t)P.pz, nfields};
    const cuuint32_t box[4] = {bx, by, 1, bf};
    return encode(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  };
  if (make(&maps->centre, P.q, nf, MarchGeom<TY>::ROW, MarchGeom<TY>::ROWS, nf) != CUDA_SUCCESS) return -2;
  if (make(&maps->ring, P.q, nf, MTX, TY, nf) != CUDA_SUCCESS) return -2;
  if (make(&maps->w, P.w, 5, MTX, TY, 5) != CUDA_SUCCESS) return -2;
  if (make(&maps->r, P.R, 5, MTX, TY, 5) != CUDA_SUCCESS) return -2;
  constexpr int STY = STREAMS_SENSOR_TY;
  if (make(&maps->s_centre, P.q, nf, MarchGeom<STY>::ROW, MarchGeom<STY>::ROWS, 3) != CUDA_SUCCESS) return -2;
  if (make(&maps->s_ring, P.q, nf, MTX, STY, 3) != CUDA_SUCCESS) return -2;
  return 0;
}

template <int L, int R>
static int launch_weno_T(const DevP& P, cudaStream_t st) {
  if (P.flux_mode == FLUX_CENTRAL) return 0;
  const long long a = (long long)P.nx * P.ny * P.nz;
  auto blocks = [&](long long extra) { return (int)((a + extra + WCH - 1) / WCH); };
  const int nb0 = blocks((long long)P.ny * P.nz), nb1 = blocks((long long)P.nx * P.nz), nb2 = blocks((long long)P.nx * P.ny);
  dim3 b(WTH), g((unsigned)(nb0 + nb1 + nb2));
  if (P.flux_mode == FLUX_HYBRID) weno_list_kernel<L, R><<<P.nsm * STREAMS_WENO_MINB, b, 0, st>>>(P);
  else weno_kernel<L, R, true><<<g, b, 0, st>>>(P, nb0, nb1);
  return 1;
}

// Instantiated scheme families: m = 1, 2, 3 with central order 2m, viscous order 2m and WENO order 2m - 1
// (2/1/2, 4/3/4, 6/5/6); orders a mode does not use are ignored.  The layout always carries ng = 3 ghost layers.
bool rhs_supported(int L, int Lv, int r, int flux_mode, int visc_law) {
  return L >= 1 && L <= 3 && (visc_law == VISC_NONE || Lv == L) && (flux_mode == FLUX_CENTRAL || r == L);
}

int launch_rhs_main(const DevP& P, const MarchMaps& mp, int L, int Lv, int r, const StageArgs& sa, cudaStream_t st) {
  if (!rhs_supported(L, Lv, r, P.flux_mode, P.visc_law)) return -1;
  if (L == 1) return launch_main_T<1, 1, 1>(P, mp, sa, st);
  if (L == 2) return launch_main_T<2, 2, 2>(P, mp, sa, st);
  return launch_main_T<3, 3, 3>(P, mp, sa, st);
}
int launch_weno(const DevP& P, int L, int Lv, int r, cudaStream_t st) {
  if (!rhs_supported(L, Lv, r, P.flux_mode, P.visc_law)) return -1;
  if (L == 1) return launch_weno_T<1, 1>(P, st);
  if (L == 2) return launch_weno_T<2, 2>(P, st);
  return launch_weno_T<3, 3>(P, st);
}

}  // namespace streams
