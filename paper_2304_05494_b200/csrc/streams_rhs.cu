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
  double lap[3], lapT; // sum over directions of the second-derivative stencils, centre term applied at the end
};

template <int D>
__device__ __forceinline__ double pick(double a, double b, double c) { return D == 0 ? a : (D == 1 ? b : c); }

// fields of the marching kernel, in the order of DevP::q (F_DIV is DevP::div)
enum { F_U = 0, F_V = 1, F_W = 2, F_H = 3, F_P = 4, F_RHO = 5, F_T = 6, F_MU = 7, F_DIV = 8 };

__device__ __forceinline__ const double* field_ptr(const DevP& P, int f) { return f < 8 ? P.q + f * P.fs : P.div; }

__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gsrc) : "memory");
}
// copies 8 bytes when `take`, writes zeros (and reads nothing) otherwise
__device__ __forceinline__ void cp_async8_zfill(void* smem_dst, const void* gsrc, bool take) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
  const unsigned n = take ? 8u : 0u;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(s), "l"(gsrc), "r"(n) : "memory");
}
// a load the compiler may not sink to its first use
__device__ __forceinline__ unsigned ld_u8_now(const unsigned char* p) {
  unsigned v;
  asm volatile("ld.global.u8 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// per-direction stencil coefficients with the metric folded in
struct DirCoef {
  double kc[3];        // convective: a_l / 4            (mass flux pairs; the metric multiplies the sums)
  double ap[3];        // pressure:   a_l
  double met_c;        // convective metric
  double av[3];        // viscous first derivative:  a_l * metric
  double bv[3];        // viscous second derivative: b_l * metric^2
};

// ---------------------------------------------------------------------------------------------
// One direction at one node; G(f, o) returns field f at offset o (-3..3) along the direction.
// Convective part (O1) in pair-difference form: with m(a,b) = (a_l/4)(rho_a+rho_b)(ud_a+ud_b),
//   f_{n+1/2} - f_{n-1/2} = sum_l [ m(n,n+l)(phi_n+phi_{n+l}) - m(n-l,n)(phi_{n-l}+phi_n) ]
//                         = phi_n S0 + sum_l [ m(n,n+l) phi_{n+l} - m(n-l,n) phi_{n-l} ],  S0 = sum_l [m(n,n+l) - m(n-l,n)]
// (the same sum as the oracle's interface-flux form, regrouped), plus sum_l a_l (p_{n+l} - p_{n-l}) on the
// D-momentum.  Viscous part (O4): first derivatives of u, v, w, T, mu, div; second-derivative sums
// sum_l b_l (f_{+l} + f_{-l}) of u, v, w, T (the centre term -2 f_0 sum b_l is applied once by the caller).
// c0 = (u, v, w, H, p, rho) at the node, alr[l] = kc[l] * rho_0.
// ---------------------------------------------------------------------------------------------
template <int D, int L, int LV, bool CONV, bool VISC, class G>
__device__ __forceinline__ void dir_terms(const G& g, const DirCoef& c, const double c0[6], const double alr[3],
                                          double eyr, double r[5], VAcc& V) {
  constexpr int LC = CONV ? L : 0;
  constexpr int LVV = VISC ? LV : 0;
  constexpr int LM = LC > LVV ? LC : LVV;
  double S0 = 0.0, S[4] = {0.0, 0.0, 0.0, 0.0}, SP = 0.0;
  double d1[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};   // u v w T mu div
  double d2[4] = {0.0, 0.0, 0.0, 0.0};             // u v w T
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
      const double mb = fma(c.kc[l - 1], rb, alr[l - 1]) * (ud0 + pick<D>(ub, vb, wb));
      const double ma = fma(c.kc[l - 1], ra, alr[l - 1]) * (pick<D>(ua, va, wa) + ud0);
      S0 += mb - ma;
      S[0] = fma(mb, ub, S[0]); S[0] = fma(-ma, ua, S[0]);
      S[1] = fma(mb, vb, S[1]); S[1] = fma(-ma, va, S[1]);
      S[2] = fma(mb, wb, S[2]); S[2] = fma(-ma, wa, S[2]);
      S[3] = fma(mb, hb, S[3]); S[3] = fma(-ma, ha, S[3]);
      SP = fma(c.ap[l - 1], pb - pa, SP);
    }
    if constexpr (VISC) if (l <= LVV) {
      const double tb = g(F_T, l), ta = g(F_T, -l);
      const double a = c.av[l - 1], b = c.bv[l - 1];
      d1[0] = fma(a, ub - ua, d1[0]);  d2[0] = fma(b, ub + ua, d2[0]);
      d1[1] = fma(a, vb - va, d1[1]);  d2[1] = fma(b, vb + va, d2[1]);
      d1[2] = fma(a, wb - wa, d1[2]);  d2[2] = fma(b, wb + wa, d2[2]);
      d1[3] = fma(a, tb - ta, d1[3]);  d2[3] = fma(b, tb + ta, d2[3]);
      d1[4] = fma(a, g(F_MU, l) - g(F_MU, -l), d1[4]);
      d1[5] = fma(a, g(F_DIV, l) - g(F_DIV, -l), d1[5]);
    }
  }
  if (CONV) {
    r[0] = fma(-2.0 * c.met_c, S0, r[0]);
#pragma unroll
    for (int q = 0; q < 4; ++q) r[1 + q] = fma(-c.met_c, fma(c0[q], S0, S[q]), r[1 + q]);
    r[1 + D] = fma(-c.met_c, SP, r[1 + D]);
  }
  if (VISC) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      V.g[a][D] = d1[a];
      V.lap[a] += (D == 1) ? fma(eyr, d1[a], d2[a]) : d2[a];
    }
    V.gT[D] = d1[3];
    V.lapT += (D == 1) ? fma(eyr, d1[3], d2[3]) : d2[3];
    V.gmu[D] = d1[4];
    V.gdiv[D] = d1[5];
  }
}

// ---------------------------------------------------------------------------------------------
// Viscous combination (O4) for one node; c0 = (u, v, w, ...).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void viscous_combine(const DevP& P, const double c0[6], double mu0, double r[5], const VAcc& V) {
  const double dv = (V.g[0][0] + V.g[1][1]) + V.g[2][2];
  const double s01 = V.g[0][1] + V.g[1][0], s02 = V.g[0][2] + V.g[2][0], s12 = V.g[1][2] + V.g[2][1];
  const double s[3][3] = {{2.0 * V.g[0][0], s01, s02}, {s01, 2.0 * V.g[1][1], s12}, {s02, s12, 2.0 * V.g[2][2]}};
  const double tdv = (2.0 / 3.0) * dv;
  double vm[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double cross = V.gmu[0] * s[a][0];
    cross = fma(V.gmu[1], s[a][1], cross);
    cross = fma(V.gmu[2], s[a][2], cross);
    cross = fma(-V.gmu[a], tdv, cross);
    vm[a] = fma(mu0, fma(V.gdiv[a], 1.0 / 3.0, V.lap[a]), cross);
  }
  double ph = V.g[0][0] * V.g[0][0];
  ph = fma(V.g[1][1], V.g[1][1], ph);
  ph = fma(V.g[2][2], V.g[2][2], ph);
  ph = ph + ph;
  ph = fma(s01, s01, ph);
  ph = fma(s02, s02, ph);
  ph = fma(s12, s12, ph);
  ph = fma(-tdv, dv, ph);
  double cond = mu0 * V.lapT;
  cond = fma(V.gmu[0], V.gT[0], cond);
  cond = fma(V.gmu[1], V.gT[1], cond);
  cond = fma(V.gmu[2], V.gT[2], cond);
  r[1] += vm[0];
  r[2] += vm[1];
  r[3] += vm[2];
  double e = fma(mu0, ph, P.kfac * cond);
  e = fma(c0[0], vm[0], e);
  e = fma(c0[1], vm[1], e);
  e = fma(c0[2], vm[2], e);
  r[4] += e;
}

// ---------------------------------------------------------------------------------------------
// rhs_march_kernel (a4-a8 in one pass).  A block owns a 32 x TY tile of (x, y) and marches through a chunk
// of z planes (2.5-D blocking):
//   - z neighbours: every thread keeps the 7-plane column (k-3 .. k+3) of its node for all fields in
//     registers; plane k+4 is fetched one iteration ahead (plain coalesced loads, consumed at the ring shift);
//   - x / y neighbours: the centre plane of every field sits in shared memory with its 3-wide halo
//     (interior written from the registers, halo copied with cp.async one iteration ahead, two buffers, one
//     barrier per plane); all stencil offsets are compile-time immediates;
//   - RK operands (previous-stage R, w) are staged with cp.async at the start of the iteration and consumed
//     at its end, so no global-memory latency is exposed in the loop.
// Threads of a ragged tile beyond the interior load (clamped) ghost nodes, so the tile's shared-memory
// plane is correct wherever an interior thread reads it; they do not store.
// ---------------------------------------------------------------------------------------------
constexpr int MTX = 32;

template <int TY>
struct MarchGeom {
  static constexpr int ROW = MTX + 8;            // row pitch: 4 halo columns each side (3 used), rows stay 16 B aligned
  static constexpr int ROWS = TY + 6;
  static constexpr int PLANE = ROW * ROWS;       // doubles per field per buffer
  static constexpr int NT = MTX * TY;
  static constexpr int NH = 6 * TY + 6 * MTX;    // halo nodes of a plane (corners are never read)
  static constexpr int HE = (NH + NT - 1) / NT;  // halo nodes per thread
};

template <int L, int LV, bool VISC, bool CONV, bool WENO, int TY>
__global__ void __launch_bounds__(MTX * TY, (TY >= 8 ? 1 : 2))
rhs_march_kernel(const DevP P, const StageArgs sa, int nbx, int nby, int kz) {
  using G = MarchGeom<TY>;
  constexpr int NF = VISC ? 9 : 6;
  constexpr int NG = 3;
  static_assert(L <= NG && LV <= NG, "ring depth");
  extern __shared__ double smem[];
  double* buf = smem;                              // [2][NF][PLANE]  centre planes with halo
  double* epi = buf + 2 * NF * G::PLANE;           // [10][NT]         previous-stage R, w of this plane
  double* nxs = epi + 10 * G::NT;                  // [NF][NT]         plane k+4 of this thread's column
  double* dfs = nxs + NF * G::NT;                  // [30][NT]         flux corrections around this node (WENO)

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
  const long long ncol = pidx(P, ic, jc, 0);       // this thread's column at k = 0
  const long long ocol = (long long)j * P.nx + i;  // interior index at k = 0 (active threads only)
  const int s0 = (ty + 3) * G::ROW + tx + 4;       // this node in a shared-memory plane

  // halo nodes handled by this thread: offset in a padded plane, offset in a shared-memory plane
  int hsrc[G::HE], hdst[G::HE];
#pragma unroll
  for (int h = 0; h < G::HE; ++h) {
    const int e = tid + h * G::NT;
    int xo, yo;
    if (e < 6 * TY) { const int rr = e / 6, c = e % 6; yo = rr; xo = c < 3 ? c - 3 : MTX + c - 3; }
    else { const int e2 = e - 6 * TY, hr = e2 / MTX; xo = e2 % MTX; yo = hr < 3 ? hr - 3 : TY + hr - 3; }
    const int ih = min(i0 + xo, P.nx + P.ng - 1), jh = min(j0 + yo, P.ny + P.ng - 1);
    hsrc[h] = e < G::NH ? (int)((long long)(jh + P.ng) * P.sy + ih + P.ox) : -1;
    hdst[h] = (yo + 3) * G::ROW + 4 + xo;
  }

  // y metrics of this row (constant along the march)
  DirCoef cx, cy, cz;
  const double eyc = P.eta_y_c[min(j, P.ny - 1)];
  double eyv = 0.0, eyr = 0.0;
  if (VISC) { eyv = P.eta_y_v[min(j, P.ny - 1)]; eyr = P.eta_yy_v[min(j, P.ny - 1)] / eyv; }
#pragma unroll
  for (int l = 0; l < 3; ++l) {
    cx.kc[l] = cy.kc[l] = cz.kc[l] = 0.25 * P.a1[l];
    cx.ap[l] = cy.ap[l] = cz.ap[l] = P.a1[l];
    cx.av[l] = P.a1v[l] * P.inv_dx; cx.bv[l] = P.b2v[l] * (P.inv_dx * P.inv_dx);
    cy.av[l] = P.a1v[l] * eyv;      cy.bv[l] = P.b2v[l] * (eyv * eyv);
    cz.av[l] = P.a1v[l] * P.inv_dz; cz.bv[l] = P.b2v[l] * (P.inv_dz * P.inv_dz);
  }
  cx.met_c = P.inv_dx; cy.met_c = eyc; cz.met_c = P.inv_dz;
  const double sb2 = -2.0 * (((cx.bv[0] + cx.bv[1]) + cx.bv[2]) + ((cy.bv[0] + cy.bv[1]) + cy.bv[2]) +
                             ((cz.bv[0] + cz.bv[1]) + cz.bv[2]));
  const double dt = sa.update_w ? P.scal[S_DT] : 0.0;

  // ---- prologue: ring = planes kb-3 .. kb+3, halo of plane kb
  double zr[NF][2 * NG + 1];
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    const double* __restrict__ fp = field_ptr(P, f) + ncol + (long long)(kb - NG) * P.sz;
#pragma unroll
    for (int m = 0; m < 2 * NG + 1; ++m) zr[f][m] = fp[(long long)m * P.sz];
  }
  {
    const long long pl = (long long)(kb + P.ng) * P.sz;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const double* __restrict__ fp = field_ptr(P, f) + pl;
#pragma unroll
      for (int h = 0; h < G::HE; ++h)
        if (hsrc[h] >= 0) cp_async8(buf + f * G::PLANE + hdst[h], fp + hsrc[h]);
    }
    cp_async_commit();
  }

  for (int k = kb; k < ke; ++k) {
    const int b = (k - kb) & 1;
    double* __restrict__ sm = buf + b * NF * G::PLANE;
    // (A) centre plane -> shared memory; halo of plane k has been in flight for one iteration
#pragma unroll
    for (int f = 0; f < NF; ++f) sm[f * G::PLANE + s0] = zr[f][NG];
    cp_async_wait<0>();
    __syncthreads();
    // (B) start what the next iteration and this iteration's epilogue need
    const long long n = ncol + (long long)k * P.sz;
    const long long o = ocol + (long long)k * P.ny * P.nx;
    unsigned fl = 0;
    if (WENO) {
      fl = CONV ? (active ? ld_u8_now(P.nflag + n) : 0u) : 0x3fu;
    }
    if (active) {
      if (sa.read_prev) {
#pragma unroll
        for (int q = 0; q < 5; ++q) cp_async8(epi + q * G::NT + tid, P.R + q * P.N + o);
      }
      if (sa.update_w) {
#pragma unroll
        for (int q = 0; q < 5; ++q) cp_async8(epi + (5 + q) * G::NT + tid, P.w + q * P.fs + n);
      }
    }
    {
      // plane k+4 (clamped to the last ghost plane: the value is unused when it is beyond)
      const int kn = min(k + NG + 1, P.nz + P.ng - 1);
      const long long nn = ncol + (long long)kn * P.sz;
#pragma unroll
      for (int f = 0; f < NF; ++f) cp_async8(nxs + f * G::NT + tid, field_ptr(P, f) + nn);
    }
    cp_async_commit();
    if (k + 1 < ke) {
      double* __restrict__ smn = buf + (b ^ 1) * NF * G::PLANE;
      const long long pl = (long long)(k + 1 + P.ng) * P.sz;
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        const double* __restrict__ fp = field_ptr(P, f) + pl;
#pragma unroll
        for (int h = 0; h < G::HE; ++h)
          if (hsrc[h] >= 0) cp_async8(smn + f * G::PLANE + hdst[h], fp + hsrc[h]);
      }
    }
    cp_async_commit();
    // flux corrections of the flagged interfaces around the nodes of this warp (third group: waited with
    // the first at the epilogue; zero-filled where an interface is not flagged)
    bool any_fl = false;
    if (WENO) {
      any_fl = __any_sync(0xffffffffu, fl != 0);
      if (any_fl) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
          const long long sd = d == 0 ? 1 : (d == 1 ? P.sy : P.sz);
          const double* __restrict__ f = P.dF + (long long)(d * 5) * P.fs + n;
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            cp_async8_zfill(dfs + ((d * 5 + q) * 2 + 0) * G::NT + tid, f + q * P.fs, (fl >> (2 * d + 1)) & 1u);
            cp_async8_zfill(dfs + ((d * 5 + q) * 2 + 1) * G::NT + tid, f + q * P.fs - sd, (fl >> (2 * d)) & 1u);
          }
        }
      }
    }
    cp_async_commit();

    // (C) the right-hand side of this node
    double c0[6];
#pragma unroll
    for (int q = 0; q < 6; ++q) c0[q] = zr[q][NG];
    double alr[3];
#pragma unroll
    for (int l = 0; l < 3; ++l) alr[l] = cx.kc[l] * c0[F_RHO];
    double r[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    VAcc V;
#pragma unroll
    for (int a = 0; a < 3; ++a) { V.lap[a] = 0.0; }
    V.lapT = 0.0;
    {
      const double* __restrict__ sc = sm + s0;
      auto gx = [&](int f, int o2) { return sc[f * G::PLANE + o2]; };
      dir_terms<0, L, LV, CONV, VISC>(gx, cx, c0, alr, 0.0, r, V);
      auto gy = [&](int f, int o2) { return sc[f * G::PLANE + o2 * G::ROW]; };
      dir_terms<1, L, LV, CONV, VISC>(gy, cy, c0, alr, eyr, r, V);
      auto gz = [&](int f, int o2) { return zr[f][NG + o2]; };
      dir_terms<2, L, LV, CONV, VISC>(gz, cz, c0, alr, 0.0, r, V);
    }
    if (VISC) {
#pragma unroll
      for (int a = 0; a < 3; ++a) V.lap[a] = fma(sb2, c0[a], V.lap[a]);
      V.lapT = fma(sb2, zr[VISC ? F_T : 0][NG], V.lapT);
      viscous_combine(P, c0, zr[VISC ? F_MU : 0][NG], r, V);
    }

    // (D) flux corrections of flagged interfaces, RK update, stores
    cp_async_wait<0>();
    if (active) {
      if (WENO && any_fl) {
        const double met[3] = {P.inv_dx, eyc, P.inv_dz};
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
      if (sa.update_w) {
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          double inc = sa.gam * r[q];
          if (sa.read_prev) inc = fma(sa.rhk, epi[q * G::NT + tid], inc);
          P.w[q * P.fs + n] = fma(dt, inc, epi[(5 + q) * G::NT + tid]);
        }
      }
      if (sa.write_r) {
#pragma unroll
        for (int q = 0; q < 5; ++q) sa.r_out[q * P.N + o] = r[q];
      }
    }

    // (E) shift the ring
#pragma unroll
    for (int f = 0; f < NF; ++f) {
#pragma unroll
      for (int m = 0; m < 2 * NG; ++m) zr[f][m] = zr[f][m + 1];
      zr[f][2 * NG] = nxs[f * G::NT + tid];
    }
  }
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
// z chunks per tile: enough blocks to fill every SM slot in whole waves, long enough that the ring fill
// (6 planes of loads, no arithmetic) stays a small part of a chunk.
static int pick_chunks(int tiles, int nz, int slots) {
  int best_c = 1;
  double best = 1e300;
  for (int c = 1; c <= (nz + 3) / 4; ++c) {
    const int kz = (nz + c - 1) / c, ce = (nz + kz - 1) / kz;
    const long long waves = ((long long)tiles * ce + slots - 1) / slots;
    const double cost = (double)waves * (kz + 1.0);
    if (cost < best - 1e-9) { best = cost; best_c = ce; }
  }
  return best_c;
}

#ifndef STREAMS_MARCH_TY
#define STREAMS_MARCH_TY 8
#endif

template <int L, int LV, bool VISC, bool CONV, bool WENO, int TY>
static int launch_march(const DevP& P, const StageArgs& sa, cudaStream_t st) {
  using G = MarchGeom<TY>;
  constexpr int NF = VISC ? 9 : 6;
  const size_t smem = (size_t)(2 * NF * G::PLANE + (10 + NF + (WENO ? 30 : 0)) * G::NT) * sizeof(double);
  auto kern = rhs_march_kernel<L, LV, VISC, CONV, WENO, TY>;
  static bool attr_set = false;
  if (!attr_set) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -2;
    attr_set = true;
  }
  const int nbx = (P.nx + MTX - 1) / MTX, nby = (P.ny + TY - 1) / TY;
  const int tiles = nbx * nby;
  const int slots = P.nsm * (TY >= 8 ? 1 : 2);
  const int chunks = pick_chunks(tiles, P.nz, slots);
  const int kz = (P.nz + chunks - 1) / chunks;
  kern<<<(unsigned)(tiles * chunks), G::NT, smem, st>>>(P, sa, nbx, nby, kz);
  return 1;
}

template <int L, int LV, int R>
static int launch_main_T(const DevP& P, const StageArgs& sa, cudaStream_t st) {
  const bool visc = P.visc_law != VISC_NONE;
  const bool conv = P.flux_mode != FLUX_WENO;
  const bool weno = P.flux_mode != FLUX_CENTRAL;
  constexpr int TY = STREAMS_MARCH_TY;
#define STREAMS_MAIN(V, C, W) return launch_march<L, LV, V, C, W, TY>(P, sa, st)
  if (visc && conv && weno) STREAMS_MAIN(true, true, true);
  else if (visc && conv) STREAMS_MAIN(true, true, false);
  else if (visc) STREAMS_MAIN(true, false, true);
  else if (conv && weno) STREAMS_MAIN(false, true, true);
  else if (conv) STREAMS_MAIN(false, true, false);
  else STREAMS_MAIN(false, false, true);
#undef STREAMS_MAIN
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
