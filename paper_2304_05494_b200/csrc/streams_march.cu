// a4-a8 (+ a2, a1 and a9 of the next stage): the fused right-hand side, RK update and primitives.
//
//   rhs_march_kernel : every node, one pass (2.5-D z-march, TMA + mbarrier pipeline): central split convective terms in
//                      x, y, z (O1), viscous terms (O4), the net WENO correction of the node where an adjacent
//                      interface is flagged (DevP::corr, gathered by corr_gather_kernel, streams_weno.cu), body force
//                      (S17), low-storage RK3 update (O5); then the primitives of the updated node into the OTHER
//                      primitive buffer (stencils of this stage still read the current one), also at its periodic images
//                      in the ghost layers, and in the last stage the time-step rate (a9) and a finiteness check.
// R, w and the primitives are written once per stage.
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
// c0 = (u, v, w, H, p, rho) at the node, alr[l] = (a_l/4) rho_0.  Orders below the instantiated one run on
// zero-padded coefficient tables (DevP::a1 ...): the extra terms are exact zeros.
template <int D, int L, int LV, bool CONV, bool VISC, class G>
__device__ __forceinline__ void dir_terms(const DevP& P, const G& g, const YMet& ym, const double c0[6],
                                          const double alr[4], double r[5], Visc& V) {
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
// of z planes (2.5-D blocking); NG = DevP::ng (3, or 4 for the order-8 / WENO-7 layouts):
//   - z neighbours: every thread keeps the (2 NG + 1)-plane column (k-NG .. k+NG) of its node for all fields in
//     registers; plane k+NG+1 arrives by TMA in a shared-memory slot and enters the ring at the shift;
//   - x / y neighbours: the centre plane of all fields with its NG-wide halo is ONE 4-D TMA box
//     (x, y, z, field) = (40, TY+2NG, 1, NF) into one of two shared-memory buffers, issued two planes ahead;
//     every stencil offset is a compile-time immediate;
//   - RK operands (w, previous-stage R) of the plane arrive by TMA one plane ahead;
//   - the net WENO correction of nodes next to a flagged interface (hybrid / WENO; 5 values per node, already
//     multiplied by the metrics): cp.async with zero fill, by the warps that have such a node only.
// One thread issues the TMA copies after a split barrier (bar.arrive by the other warps, bar.sync by
// its warp), so no warp but that one waits for the slowest.  Completion is tracked by mbarriers.
// ---------------------------------------------------------------------------------------------
#ifndef STREAMS_MARCH_NSLOT
#define STREAMS_MARCH_NSLOT 2
#endif
template <int TY, int NG, bool VISC, bool WENO>
struct MarchSmem {
  using G = MarchGeom<TY, NG>;
  static constexpr int NF = VISC ? 9 : 6;
  static constexpr size_t BUF = (size_t)NF * G::PLANE * 8;     // one centre-plane buffer
  static constexpr size_t RING = (size_t)NF * G::NT * 8;       // one ring-plane slot
  static constexpr size_t EPI = (size_t)10 * G::NT * 8;        // one RK-operand slot: R[5], w[1..4] (+ one spare field)
  static constexpr size_t DFS = WENO ? (size_t)5 * G::NT * 8 : 0;
  static constexpr int NSLOT = STREAMS_MARCH_NSLOT;            // ring-plane / RK-operand slots: loads run NSLOT - 1 planes ahead
  static constexpr size_t FLG = WENO ? 2 * (((size_t)G::NT + 127) / 128 * 128) : 0;   // interface-flag bytes of the centre planes
  static constexpr size_t OFF_RING = 2 * BUF, OFF_EPI = OFF_RING + NSLOT * RING, OFF_DFS = OFF_EPI + NSLOT * EPI,
                          OFF_FLG = OFF_DFS + DFS, OFF_BAR = OFF_FLG + FLG,
                          TOTAL = OFF_BAR + 64 + 8 * 32;                               // 2 + NSLOT mbarriers, rate scratch
  static_assert(BUF % 128 == 0 && RING % 128 == 0 && EPI % 128 == 0, "TMA destinations are 128-byte aligned");
  static_assert(TOTAL <= 227 * 1024, "shared memory of one block");
};

constexpr int MARCH_MINB = 1;                        // one block of 8 warps per SM (253 registers per thread)
template <int L, int LV, bool VISC, bool CONV, bool WENO, bool UPD, int TY, int NG>
__global__ void __launch_bounds__(MTX * TY, MARCH_MINB)
rhs_march_kernel(const __grid_constant__ CUtensorMap tm_centre, const __grid_constant__ CUtensorMap tm_ring,
                 const __grid_constant__ CUtensorMap tm_w, const __grid_constant__ CUtensorMap tm_r,
                 const __grid_constant__ CUtensorMap tm_flag, const DevP P,
                 const StageArgs sa, int nbx, int nby, int kz) {
  using G = MarchGeom<TY, NG>;
  using SM = MarchSmem<TY, NG, VISC, WENO>;
  constexpr int NF = SM::NF;
  static_assert(L <= NG && LV <= NG, "ring depth");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double* const buf = reinterpret_cast<double*>(smem_raw);                  // [2][NF][PLANE]
  constexpr int NSLOT = SM::NSLOT;
  double* const ring = reinterpret_cast<double*>(smem_raw + SM::OFF_RING);  // [NSLOT][NF][NT]
  double* const epi = reinterpret_cast<double*>(smem_raw + SM::OFF_EPI);    // [NSLOT][10][NT]
  double* const dfs = reinterpret_cast<double*>(smem_raw + SM::OFF_DFS);    // [5][NT]
  unsigned char* const flg = smem_raw + SM::OFF_FLG;                        // [2][NT] (hybrid)
  constexpr bool FLAGS = WENO && CONV;                                      // hybrid: per-node interface flags decide
  constexpr int FLGB = (int)(SM::FLG / 2);
  unsigned long long* const bars = reinterpret_cast<unsigned long long*>(smem_raw + SM::OFF_BAR);
  unsigned long long* const full_c = bars;        // [2] centre plane landed
  unsigned long long* const full_e = bars + 2;    // [NSLOT] ring plane + RK operands landed

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
  const int ic = min(i, P.nx + NG - 1), jc = min(j, P.ny + NG - 1);
  const int isz = (int)P.sz;
  const int ncol = (int)pidx(P, ic, jc, 0);            // this thread's column at k = 0 (padded index < 2^31)
  const int s0 = (ty + NG) * G::ROW + tx + 4;          // this node in a shared-memory plane

  const unsigned bytes_c = (unsigned)SM::BUF + (FLAGS ? (unsigned)G::NT : 0u);
  // (the density of the old state is not fetched with the other four conserved variables: the ring's centre value of
  // the rho slot is the same number, q[Q_RHO] being a copy of w[0])
  const unsigned bytes_e = (unsigned)SM::RING + (UPD ? 4u * G::NT * 8u : 0u) + (sa.read_prev ? 5u * G::NT * 8u : 0u);
  const int cx0 = i0 + P.ox, cy0 = j0 + NG;            // tile origin in padded coordinates

  auto issue_centre = [&](int k, int b) {              // thread 0 only
    mbar_expect_tx(&full_c[b], bytes_c);
    tma_load_4d(buf + (size_t)b * NF * G::PLANE, &tm_centre, &full_c[b], cx0 - 4, cy0 - NG, k + NG, 0);
    // the flag bytes of the plane's nodes ride with it (a byte loaded by its thread one plane ahead stalled every plane:
    // the compiler tests the byte where it is requested and carries the predicate; 11 % of the kernel's samples)
    if (FLAGS) tma_load_4d(flg + b * FLGB, &tm_flag, &full_c[b], cx0, cy0, k + NG, 0);
  };
  auto issue_ring_epi = [&](int k, int b) {            // ring plane k+NG+1 and the RK operands of plane k into slot b
    mbar_expect_tx(&full_e[b], bytes_e);
    tma_load_4d(ring + (size_t)b * NF * G::NT, &tm_ring, &full_e[b], cx0, cy0, k + NG + 1 + NG, 0);
    if (sa.read_prev) tma_load_4d(epi + (size_t)b * 10 * G::NT, &tm_r, &full_e[b], cx0, cy0, k + NG, 0);
    if (UPD) tma_load_4d(epi + (size_t)b * 10 * G::NT + 5 * G::NT, &tm_w, &full_e[b], cx0, cy0, k + NG, 0);
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
      tma_prefetch_4d(&tm_ring, cx0, cy0, k + NG + 1 + NG, 0);
      if (sa.read_prev) tma_prefetch_4d(&tm_r, cx0, cy0, k + NG, 0);
      if (UPD) tma_prefetch_4d(&tm_w, cx0, cy0, k + NG, 0);
    }
  };
  if (tid == 0) {
    mbar_init(&full_c[0], 1); mbar_init(&full_c[1], 1);
#pragma unroll
    for (int a = 0; a < NSLOT; ++a) mbar_init(&full_e[a], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) {
    issue_centre(kb, 0);
    if (kb + 1 < ke) issue_centre(kb + 1, 1);
#pragma unroll
    for (int a = 0; a < NSLOT - 1; ++a)
      if (kb + a < ke) issue_ring_epi(kb + a, a);
#pragma unroll
    for (int a = 1; a <= PF; ++a) prefetch_ring_epi(kb + NSLOT - 2 + a);
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
  const double dt = UPD ? P.scal[S_DT] : 0.0;
  double acc[3] = {P.accel[0], P.accel[1], P.accel[2]};   // S17; owned by the device-side controller when has_accel == 2
  if (P.has_accel == 2) { acc[0] = P.scal[S_ACC]; acc[1] = P.scal[S_ACC + 1]; acc[2] = P.scal[S_ACC + 2]; }

  // ring = planes kb-NG .. kb+NG of this thread's column
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
  bool bad = false;                                   // a NaN rate, or a non-finite updated state

  // a2 / a1 / a9 of the next stage for the node just updated (state wn of plane kk): its primitives go to the other q
  // buffer (stencils of this stage still read the current one), also at the node's periodic images in the ghost layers
  // (the owner writes them; the next stage only fills the non-periodic ghost shell), then the time-step rate and the
  // finiteness check of the last stage.  DEFER: evaluated one plane late, inside the stencil phase of the next plane,
  // so that its long dependent chain (reciprocal, square roots, Newton steps) overlaps the wide stencil arithmetic
  // instead of running alone between two barriers.
  constexpr bool DEFER = true;
  double wn[5] = {1.0, 0.0, 0.0, 0.0, 1.0};
  // (no branch around the arithmetic: `ok` only predicates the stores, so the chain sits in the stencil phase's block)
  auto finish_node = [&](int kk, bool ok) {
    double mu, cc, vel[3], o[NQ];
    prims_from_state<VISC, WENO>(P, wn, sa.want_rate != 0, o, mu, cc, vel);
    double* __restrict__ qo = sa.q_out + (ncol + kk * isz);
    if (ok) store_prims<VISC, WENO>(P, qo, o);
    const int zoff = !P.own_z ? 0 : (kk < NG ? P.nz * isz : (kk >= P.nz - NG ? -P.nz * isz : 0));
    if (ok && xoff) store_prims<VISC, WENO>(P, qo + xoff, o);
    if (ok && yoff) store_prims<VISC, WENO>(P, qo + yoff, o);
    if (ok && zoff) store_prims<VISC, WENO>(P, qo + zoff, o);
    if (ok && sa.want_rate) {                                // fmax drops a NaN operand: test the rate before the max
      const double rr = dt_rate<VISC>(P, vel, cc, mu, wn[0], ym.eyc);
      bad |= !(rr == rr);
      rate = fmax(rate, rr);
    }
    if (ok && sa.check_state)                          // the step's last stage: Inf or NaN anywhere in the new state
      bad |= !(fabs((wn[0] + wn[1]) + (wn[2] + wn[3]) + wn[4]) <= 1.7976931348623157e308);
  };

  for (int k = kb; k < ke; ++k) {
    const int it = k - kb, b = it & 1;
    const unsigned par = (unsigned)(it >> 1) & 1u;
    const int se = it % NSLOT;                            // ring / RK-operand slot of this plane
    const unsigned par_e = (unsigned)(it / NSLOT) & 1u;
    const int n = ncol + k * isz;
    if (tid == G::NT - 32) prefetch_ring_epi(k + NSLOT - 1 + PF);   // no shared-memory hazard: any thread, off the issuing warp's path
    // (C) the right-hand side of this node
    mbar_wait(&full_c[b], par);
    // does this node have a net WENO correction (an adjacent flagged interface)?  The five values are staged while
    // the stencils run
    bool fl = false, any_fl = false;
    if (WENO) {
      fl = active && (!FLAGS || flg[b * FLGB + tid] != 0);
      any_fl = __any_sync(0xffffffffu, fl);
      if (any_fl) {
#pragma unroll
        for (int q = 0; q < 5; ++q) cp_async8_zfill(dfs + q * G::NT + tid, P.corr + (long long)n * 5 + q, fl);   // the node's record
      }
    }
    if (DEFER && UPD) finish_node(k - 1, active && it > 0);
    const double* __restrict__ sc = buf + (size_t)b * NF * G::PLANE + s0;
    auto gx = [&](int f, int o2) { return sc[f * G::PLANE + o2]; };
    auto gy = [&](int f, int o2) { return sc[f * G::PLANE + o2 * G::ROW]; };
    auto gz = [&](int f, int o2) { return zr[f][NG + o2]; };
    double c0[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) c0[q] = zr[q][NG];
    double alr[4];
#pragma unroll
    for (int l = 0; l < 4; ++l) alr[l] = P.kc[l] * c0[F_RHO];
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

    // every warp is done with buf[b] and with the ring / RK-operand slot of the previous plane: the issuing thread
    // refills them
    // (two alternating barrier ids: a warp may run one iteration ahead of the slowest)
    if (tid >> 5) {
      if (b) asm volatile("bar.arrive 2, %0;" ::"n"(G::NT) : "memory");
      else asm volatile("bar.arrive 1, %0;" ::"n"(G::NT) : "memory");
    } else {
      if (b) asm volatile("bar.sync 2, %0;" ::"n"(G::NT) : "memory");
      else asm volatile("bar.sync 1, %0;" ::"n"(G::NT) : "memory");
      if (tid == 0) {
        if (k + NSLOT - 1 < ke) issue_ring_epi(k + NSLOT - 1, (it + NSLOT - 1) % NSLOT);   // ahead of the larger centre box
        if (k + 2 < ke) issue_centre(k + 2, b);
      }
    }

    // (D) net correction of the flagged interfaces around the node, body force, RK update, stores
    mbar_wait(&full_e[se], par_e);
    const double* __restrict__ ep = epi + (size_t)se * 10 * G::NT + tid;
    if (WENO && any_fl) {
      cp_async_wait_all();
#pragma unroll
      for (int q = 0; q < 5; ++q) r[q] -= dfs[q * G::NT + tid];     // each thread reads what it staged itself
    }
    if (P.has_accel) {                               // S17: uniform body acceleration and its work
      const double rho0 = c0[F_RHO];
#pragma unroll
      for (int a = 0; a < 3; ++a) r[1 + a] = fma(rho0, acc[a], r[1 + a]);
      r[4] = fma(rho0, fma(c0[F_U], acc[0], fma(c0[F_V], acc[1], c0[F_W] * acc[2])), r[4]);
    }
    if (UPD) {
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        double inc = sa.gam * r[q];
        if (sa.read_prev) inc = fma(sa.rhk, ep[q * G::NT], inc);
        wn[q] = fma(dt, inc, q == 0 ? c0[F_RHO] : ep[(4 + q) * G::NT]);
        if (active) st_out(P.w + (long long)q * P.fs + n, wn[q]);
      }
      if (!DEFER) finish_node(k, active);
    }
    if (active) {
      if (sa.write_r) {
#pragma unroll
        for (int q = 0; q < 5; ++q) st_out(P.R + (long long)q * P.fs + n, r[q]);
      }
      if (sa.r_dense) {
        const long long o = ((long long)k * P.ny + j) * P.nx + i;
#pragma unroll
        for (int q = 0; q < 5; ++q) sa.r_dense[q * P.N + o] = r[q];
      }
    }

    // (E) shift the ring
    const double* __restrict__ rn = ring + (size_t)se * NF * G::NT + tid;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
#pragma unroll
      for (int m = 0; m < 2 * NG; ++m) zr[f][m] = zr[f][m + 1];
      zr[f][2 * NG] = rn[f * G::NT];
    }
  }
  if (DEFER && UPD) finish_node(ke - 1, active);
  if (bad) P.scal[S_NAN] = 1.0;                       // streams_step returns STREAMS_ENAN
  // a9 of the next step: one atomicMax per block on the bit pattern of the largest rate (a NaN wins)
  if (sa.want_rate) {
    if (bad) rate = __longlong_as_double(0x7ff8000000000000LL);
    block_rate_max(P, rate, bars + 8);
  }
}

// -------------------------------------------------------------------------- launch
// configure: only opt the instantiation in to its dynamic shared memory on the current device (streams_init).
template <int L, int LV, bool VISC, bool CONV, bool WENO, bool UPD, int TY, int NG>
static int launch_march(const DevP& P, const MarchMaps& mp, const StageArgs& sa, cudaStream_t st, bool configure) {
  using G = MarchGeom<TY, NG>;
  using SM = MarchSmem<TY, NG, VISC, WENO>;
  auto kern = rhs_march_kernel<L, LV, VISC, CONV, WENO, UPD, TY, NG>;
  if (configure)
    return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM::TOTAL) == cudaSuccess ? 0 : -2;
  const int nbx = (P.nx + MTX - 1) / MTX, nby = (P.ny + TY - 1) / TY;
  const int tiles = nbx * nby;
  const int chunks = pick_chunks(tiles, P.nz, P.nsm * MARCH_MINB);
  const int kz = (P.nz + chunks - 1) / chunks;
  kern<<<(unsigned)(tiles * chunks), G::NT, SM::TOTAL, st>>>(mp.centre, mp.ring, mp.w, mp.r, mp.flag, P, sa, nbx, nby, kz);
  return 1;
}

template <int M, int NG>
static int launch_main_T(const DevP& P, const MarchMaps& mp, const StageArgs& sa, cudaStream_t st, bool configure) {
  const bool visc = P.visc_law != VISC_NONE;
  const bool conv = P.flux_mode != FLUX_WENO;
  const bool weno = P.flux_mode != FLUX_CENTRAL;
  constexpr int TY = STREAMS_MARCH_TY;
#define STREAMS_MAIN(V, C, W)                                                                              \
  do {                                                                                                     \
    if (configure) {                                                                                       \
      const int a = launch_march<M, M, V, C, W, true, TY, NG>(P, mp, sa, st, true);                        \
      const int b = launch_march<M, M, V, C, W, false, TY, NG>(P, mp, sa, st, true);                       \
      return (a | b) ? -2 : 0;                                                                             \
    }                                                                                                      \
    if (sa.update_w) return launch_march<M, M, V, C, W, true, TY, NG>(P, mp, sa, st, false);               \
    return launch_march<M, M, V, C, W, false, TY, NG>(P, mp, sa, st, false);                               \
  } while (0)
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
#ifndef STREAMS_TMA_L2_PROMOTION
#define STREAMS_TMA_L2_PROMOTION CU_TENSOR_MAP_L2_PROMOTION_L2_128B
#endif
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
  constexpr int TY = STREAMS_MARCH_TY, STY = STREAMS_SENSOR_TY;
  const cuuint32_t nf = P.visc_law != VISC_NONE ? 9 : 6;
  const cuuint64_t strides[3] = {(cuuint64_t)P.px * 8, (cuuint64_t)P.sz * 8, (cuuint64_t)P.fs * 8};
  const cuuint32_t ones[4] = {1, 1, 1, 1};
  auto make = [&](CUtensorMap* m, void* base, cuuint64_t nfields, cuuint32_t bx, cuuint32_t by, cuuint32_t bf, cuuint32_t bz = 1) {
    const cuuint64_t dims[4] = {(cuuint64_t)P.px, (cuuint64_t)P.py, (cuuint64_t)P.pz, nfields};
    const cuuint32_t box[4] = {bx, by, bz, bf};
    return encode(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_NONE, STREAMS_TMA_L2_PROMOTION, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  };
  const cuuint32_t halo = 2 * (cuuint32_t)P.ng;        // MarchGeom<TY, NG>::ROW / ROWS with NG = DevP::ng
  if (make(&maps->centre, P.q, nf, MTX + 8, TY + halo, nf) != CUDA_SUCCESS) return -2;
  if (make(&maps->ring, P.q, nf, MTX, TY, nf) != CUDA_SUCCESS) return -2;
  if (make(&maps->w, P.w + P.fs, 4, MTX, TY, 4) != CUDA_SUCCESS) return -2;     // rho u, rho v, rho w, rho E
  if (make(&maps->r, P.R, 5, MTX, TY, 5) != CUDA_SUCCESS) return -2;
  maps->flag = maps->r;                                // (never read outside hybrid mode)
  if (P.flux_mode == FLUX_HYBRID) {                    // the interface-flag bytes, one per node of the padded box
    const cuuint64_t dims[4] = {(cuuint64_t)P.px, (cuuint64_t)P.py, (cuuint64_t)P.pz, 1};
    const cuuint64_t bstr[3] = {(cuuint64_t)P.px, (cuuint64_t)P.sz, (cuuint64_t)P.fs};
    const cuuint32_t box[4] = {MTX, TY, 1, 1};
    if (encode(&maps->flag, CU_TENSOR_MAP_DATA_TYPE_UINT8, 4, P.nflag, dims, bstr, box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return -2;
  }
  if (make(&maps->s_centre, P.q, nf, MTX + 8, STY + halo, 3, 2) != CUDA_SUCCESS) return -2;   // two planes per box:
  if (make(&maps->s_ring, P.q, nf, MTX, STY, 3, 2) != CUDA_SUCCESS) return -2;                // SKU of sensor_march_kernel
  return 0;
}

// Instantiated families: m = 1, 2, 3 on the three-layer layout, m = 4 (central 8 / viscous 8) on the four-layer
// one.  A scheme runs on the smallest family that covers its central and viscous orders (and on m = 4 whenever the
// layout has four ghost layers, e.g. for WENO 7 with a lower central order); the coefficient tables of DevP are
// zero-padded, so the terms beyond the requested order are exact zeros (x + 0 = x): mixed orders give the same
// numbers as an instantiation of their own would.
int march_family(int L, int Lv, int ng) { return ng == 4 ? 4 : (L > Lv ? L : Lv); }

int launch_rhs_main(const DevP& P, const MarchMaps& mp, int L, int Lv, const StageArgs& sa, cudaStream_t st, bool configure) {
  const int m = march_family(P.flux_mode != FLUX_WENO ? L : 1, P.visc_law != VISC_NONE ? Lv : 1, P.ng);
  if (m < 1 || m > 4 || (P.ng != 3 && P.ng != 4)) return -1;
  if (m == 1) return launch_main_T<1, 3>(P, mp, sa, st, configure);
  if (m == 2) return launch_main_T<2, 3>(P, mp, sa, st, configure);
  if (m == 3) return launch_main_T<3, 3>(P, mp, sa, st, configure);
  return launch_main_T<4, 4>(P, mp, sa, st, configure);
}

}  // namespace streams
