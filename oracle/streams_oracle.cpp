// =============================================================================
// streams_oracle.cpp -- TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct CPU statement of the STREAmS-2 hot path as the
// paper (arXiv 2304.05494, /root/reference/PAPER.md) describes it: one right-hand
// side of the 3-D compressible Navier-Stokes equations on a structured Cartesian
// grid + the low-storage RK3 update + the CFL time step.  fp64 throughout
// ("All benchmarks ... refer to the double precision real64 type").
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may load this library.  It shares no code, header, table or
// helper with the CUDA path (paper_2304_05494_b200/csrc) and includes nothing
// from include/.  Build: g++ -std=c++17 -O2 -ffp-contract=off [-fopenmp].
//
// PAPER.md prints no equations (the method is seven sentences).
// Every formula below is the reading fixed in SURVEY.md section 8(c) and listed
// in DESIGN.md "Readings"; tags O1..O6 / S1..S16 refer to those.  The code walks
// the algorithm in the paper's order with no blocking, fusion or reordering.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"):
//   O1 central flux    : brute-force 7-term split form, telescoping, KE identity,
//                        pressure stencil (1,-8,37,37,-8,1)/60, free stream == 0.0
//   O2 sensor / mask   : closed forms (rotation, compression, expansion), dilation
//   O3 WENO            : L.R = I, linear-weight limit, polynomial exactness,
//                        Jiang-Shu beta from the definition, Sod tube, order
//   O4 viscous         : manufactured solution vs symbolic derivatives, zero on
//                        uniform state, stretched-y order
//   O5 RK3 / dt        : exp(z) Taylor polynomial, sum of coefficients, order 3
//   O6 ghost fill      : wall at rest => R = 0 to round-off, Poiseuille balance, odd reflection, the
//                        T_ghost >= 0.1 T_w clamp read back from the conserved ghosts
//   S6 scalar ghosts   : flags next to non-periodic faces vs a clamped brute-force dilation; div ghosts at
//                        a wall via (mu/3) grad(div) of a 1-D flow (clamped, not mirrored or wrapped)
//   O4 power law       : mu_ref (T/T_ref)^n closed form (n = 0.5, 0.76, 1, 2; T_ref != 1) and the
//                        manufactured Navier-Stokes terms with n = 0.76 at design order
//   S17 body force     : uniform state => R = (0, rho g, rho u.g) exactly; momentum budget of a periodic box;
//                        Poiseuille flow driven by g instead of a pressure gradient
//   S19 WENO-Z         : design order 2r-1 at a first-order critical point (Jiang-Shu: lower), weights within
//                        O(dx^4) of the linear ones on smooth data, the smooth side at a jump
//   S18 flow control   : deadbeat on a frictionless uniform flow (P reaches its target in one step and stays), holds
//                        a laminar channel against its wall friction
// Unpinned against the real STREAmS code (not in the container): S1, S2, S4, S5,
// S6, S7, S8, S9, S10, S12, S13, S15, S16 -- "parity unpinned vs STREAmS"; the
// oracle's reading is the definition for this build.
// =============================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum { BC_PERIODIC = 0, BC_WALL = 1, BC_FREESTREAM = 2 };
enum { VISC_NONE = 0, VISC_POWER = 1, VISC_SUTHERLAND = 2 };
enum { FLUX_CENTRAL = 0, FLUX_WENO = 1, FLUX_HYBRID = 2 };
enum { DBG_WENO_LINEAR = 1, DBG_NO_PRESSURE = 2 };
enum { PART_X = 1, PART_Y = 2, PART_Z = 4, PART_VISC = 8, PART_FORCE = 16, PART_ALL = 31 };

}  // namespace

// Flat parameter block (mirrored field by field in oracle/oracle.py).
extern "C" struct oracle_params {
  int nx, ny, nz;
  int bc_x, bc_y_lo, bc_y_hi, bc_z;
  int visc_law;
  int central_order, weno_order, visc_order, flux_mode;
  int dt_every;
  int dbg_flags;
  double lx, ly, lz;
  double y_lo, y_hi;            // boundary planes in y (wall / free-stream sides)
  double t_wall_lo, t_wall_hi;
  double gamma, rgas, prandtl;
  double mu_ref, t_ref, suth_s, pow_exp;
  double u_ref, l_ref;
  double freestream[5];
  double sensor_threshold, weno_eps;
  double cfl, dt_fixed;
  double accel[3];              // uniform body acceleration g (S17)
  int weno_variant;             // 0: Jiang-Shu weights, 1: WENO-Z (S19)
};

namespace {

// -----------------------------------------------------------------------------
// Central finite-difference coefficients (O1, O4).  First derivative of order 2L:
// f'_i ~ (1/h) sum_l a_l (f_{i+l} - f_{i-l});  second derivative, difference form:
// f''_i ~ (1/h^2) sum_l b_l (f_{i+l} - 2 f_i + f_{i-l}).
// Rationals as listed in SURVEY 8(c) O1 / O4; a_l = (double)p / (double)q.
// -----------------------------------------------------------------------------
void fd1_coeffs(int L, double* a) {
  switch (L) {
    case 1: a[0] = 1.0 / 2.0; break;
    case 2: a[0] = 2.0 / 3.0; a[1] = -1.0 / 12.0; break;
    case 3: a[0] = 3.0 / 4.0; a[1] = -3.0 / 20.0; a[2] = 1.0 / 60.0; break;
    case 4: a[0] = 4.0 / 5.0; a[1] = -1.0 / 5.0; a[2] = 4.0 / 105.0; a[3] = -1.0 / 280.0; break;
    default: break;
  }
}
void fd2_coeffs(int L, double* b) {
  switch (L) {
    case 1: b[0] = 1.0; break;
    case 2: b[0] = 4.0 / 3.0; b[1] = -1.0 / 12.0; break;
    case 3: b[0] = 3.0 / 2.0; b[1] = -3.0 / 20.0; b[2] = 1.0 / 90.0; break;
    case 4: b[0] = 8.0 / 5.0; b[1] = -1.0 / 5.0; b[2] = 8.0 / 315.0; b[3] = -1.0 / 560.0; break;
    default: break;
  }
}

// -----------------------------------------------------------------------------
// WENO reconstruction of order 2r-1 (O3 step 4), Jiang-Shu weights.
// v[0 .. 2r-2] are point values ordered upwind -> downwind; the value returned is
// the reconstruction at the interface between v[r-1] and v[r].
// r=3 formulas are the ones printed in SURVEY 8(c) O3.4; r=1,2,4 are the same
// construction at other orders (beta from the Jiang-Shu definition, pinned in
// tests/test_oracle_weno.py by exact rational derivation).
// beta_out (optional) receives the r smoothness indicators.
// -----------------------------------------------------------------------------
double weno_reconstruct(const double* v, int r, double eps, bool linear, double* beta_out, int variant = 0) {
  double q[4], beta[4], d[4];
  if (r == 1) {
    if (beta_out) beta_out[0] = 0.0;
    return v[0];
  } else if (r == 2) {
    const double vm1 = v[0], v0 = v[1], vp1 = v[2];
    q[0] = (-vm1 + 3.0 * v0) / 2.0;
    q[1] = (v0 + vp1) / 2.0;
    beta[0] = (v0 - vm1) * (v0 - vm1);
    beta[1] = (vp1 - v0) * (vp1 - v0);
    d[0] = 1.0 / 3.0; d[1] = 2.0 / 3.0;
  } else if (r == 3) {
    const double vm2 = v[0], vm1 = v[1], v0 = v[2], vp1 = v[3], vp2 = v[4];
    q[0] = (2.0 * vm2 - 7.0 * vm1 + 11.0 * v0) / 6.0;
    q[1] = (-vm1 + 5.0 * v0 + 2.0 * vp1) / 6.0;
    q[2] = (2.0 * v0 + 5.0 * vp1 - vp2) / 6.0;
    double t1, t2;
    t1 = vm2 - 2.0 * vm1 + v0;  t2 = vm2 - 4.0 * vm1 + 3.0 * v0;
    beta[0] = 13.0 / 12.0 * t1 * t1 + 0.25 * t2 * t2;
    t1 = vm1 - 2.0 * v0 + vp1;  t2 = vm1 - vp1;
    beta[1] = 13.0 / 12.0 * t1 * t1 + 0.25 * t2 * t2;
    t1 = v0 - 2.0 * vp1 + vp2;  t2 = 3.0 * v0 - 4.0 * vp1 + vp2;
    beta[2] = 13.0 / 12.0 * t1 * t1 + 0.25 * t2 * t2;
    d[0] = 0.1; d[1] = 0.6; d[2] = 0.3;
  } else {  // r == 4, seventh order
    const double a = v[0], b = v[1], c = v[2], e = v[3], f = v[4], g = v[5], h = v[6];
    q[0] = (-3.0 * a + 13.0 * b - 23.0 * c + 25.0 * e) / 12.0;
    q[1] = (b - 5.0 * c + 13.0 * e + 3.0 * f) / 12.0;
    q[2] = (-c + 7.0 * e + 7.0 * f - g) / 12.0;
    q[3] = (3.0 * e + 13.0 * f - 5.0 * g + h) / 12.0;
    // beta_k = sum_{m=1..3} int (d^m p_k / dx^m)^2 dx of the cubic p_k = c0 + c1 x + c2 x^2 + c3 x^3 through the four
    // cell averages: = (c1 + c3/4)^2 + (13/3) c2^2 + (781/20) c3^2 = U^2/36 + (13/12) S^2 + (781/720) T^2 with
    // U = 6 (c1 + c3/4), S = 2 c2, T = 6 c3 (undivided difference combinations; derived in exact rationals by
    // tests/test_oracle_weno.py).  This is the Jiang-Shu definition written as the sum of squares it is; the
    // expanded polynomial of Balsara & Shu (coefficients 547, -3882, ...) is the same quadratic form but loses
    // ~8 digits to cancellation on smooth data (S8).
    {
      const double U0 = ((2.0 * a - 9.0 * b) + 18.0 * c) - 11.0 * e, S0 = ((a - 4.0 * b) + 5.0 * c) - 2.0 * e, T0 = ((a - 3.0 * b) + 3.0 * c) - e;
      const double U1 = ((b - 6.0 * c) + 3.0 * e) + 2.0 * f, S1 = (c - 2.0 * e) + f, T1 = ((b - 3.0 * c) + 3.0 * e) - f;
      const double U2 = ((2.0 * c + 3.0 * e) - 6.0 * f) + g, S2 = (c - 2.0 * e) + f, T2 = ((c - 3.0 * e) + 3.0 * f) - g;
      const double U3 = ((11.0 * e - 18.0 * f) + 9.0 * g) - 2.0 * h, S3 = ((2.0 * e - 5.0 * f) + 4.0 * g) - h, T3 = ((e - 3.0 * f) + 3.0 * g) - h;
      beta[0] = (U0 * U0) / 36.0 + (13.0 / 12.0) * (S0 * S0) + (781.0 / 720.0) * (T0 * T0);
      beta[1] = (U1 * U1) / 36.0 + (13.0 / 12.0) * (S1 * S1) + (781.0 / 720.0) * (T1 * T1);
      beta[2] = (U2 * U2) / 36.0 + (13.0 / 12.0) * (S2 * S2) + (781.0 / 720.0) * (T2 * T2);
      beta[3] = (U3 * U3) / 36.0 + (13.0 / 12.0) * (S3 * S3) + (781.0 / 720.0) * (T3 * T3);
    }
    d[0] = 1.0 / 35.0; d[1] = 12.0 / 35.0; d[2] = 18.0 / 35.0; d[3] = 4.0 / 35.0;
  }
  if (beta_out) for (int k = 0; k < r; ++k) beta_out[k] = beta[k];
  double alpha[4], asum = 0.0;
  // S19 (variant 1, WENO-Z of Borges et al. 2008 / Castro et al. 2011): the global indicator
  // tau = |beta_0 - beta_{r-1}| (r = 2, 3), |beta_0 - beta_1 - beta_2 + beta_3| (r = 4) measures the smoothness of the
  // whole stencil; alpha_k = d_k (1 + (tau / (eps + beta_k))^2) keeps the weights within O(dx^(2r-2))... of the linear
  // ones wherever the data are smooth, critical points included (Jiang-Shu weights drop to order r there).
  double tau = 0.0;
  if (variant == 1 && r >= 2) tau = std::fabs(r == 4 ? ((beta[0] - beta[1]) - beta[2]) + beta[3] : beta[0] - beta[r - 1]);
  for (int k = 0; k < r; ++k) {
    // Jiang-Shu: alpha_k = d_k / (eps + beta_k)^2 ; debug switch: omega_k = d_k (linear limit, O3 pin ii)
    if (linear) alpha[k] = d[k];
    else if (variant == 1) { const double t = tau / (eps + beta[k]); alpha[k] = d[k] * (1.0 + t * t); }
    else alpha[k] = d[k] / ((eps + beta[k]) * (eps + beta[k]));
    asum += alpha[k];
  }
  double res = 0.0;
  for (int k = 0; k < r; ++k) res += (alpha[k] / asum) * q[k];
  return res;
}

// -----------------------------------------------------------------------------
// Left / right eigenvectors of the Euler flux Jacobian in direction d (O3 step 2)
// at the state (vel[3], H) with c^2 = (gamma-1)(H - q^2/2).  Lm is row-major 5x5
// (rows = characteristic fields, acting on conserved (rho, rho u, rho v, rho w, rho E)),
// Rm is row-major 5x5 with the right eigenvectors as COLUMNS.
// Field order: u_d - c, entropy, shear (lower tangential index), shear, u_d + c.
// -----------------------------------------------------------------------------
void euler_eigenvectors(int d, const double vel[3], double H, double gamma, double* Lm, double* Rm) {
  const double qq = 0.5 * (vel[0] * vel[0] + vel[1] * vel[1] + vel[2] * vel[2]);
  const double c2 = (gamma - 1.0) * (H - qq);
  const double c = std::sqrt(c2);
  const double b1 = (gamma - 1.0) / c2;
  const double b2 = qq * b1;
  const double un = vel[d];
  const int t1 = (d == 0) ? 1 : 0;
  const int t2 = (d == 2) ? 1 : 2;
  for (int n = 0; n < 25; ++n) { Lm[n] = 0.0; Rm[n] = 0.0; }
  // --- left eigenvectors (rows)
  Lm[0 * 5 + 0] = 0.5 * (b2 + un / c);
  Lm[4 * 5 + 0] = 0.5 * (b2 - un / c);
  for (int m = 0; m < 3; ++m) {
    const double nd = (m == d) ? 1.0 : 0.0;
    Lm[0 * 5 + 1 + m] = 0.5 * (-b1 * vel[m] - nd / c);
    Lm[4 * 5 + 1 + m] = 0.5 * (-b1 * vel[m] + nd / c);
    Lm[1 * 5 + 1 + m] = b1 * vel[m];
  }
  Lm[0 * 5 + 4] = 0.5 * b1;
  Lm[4 * 5 + 4] = 0.5 * b1;
  Lm[1 * 5 + 0] = 1.0 - b2;
  Lm[1 * 5 + 4] = -b1;
  Lm[2 * 5 + 0] = -vel[t1];  Lm[2 * 5 + 1 + t1] = 1.0;
  Lm[3 * 5 + 0] = -vel[t2];  Lm[3 * 5 + 1 + t2] = 1.0;
  // --- right eigenvectors (columns)
  Rm[0 * 5 + 0] = 1.0;  Rm[0 * 5 + 1] = 1.0;  Rm[0 * 5 + 4] = 1.0;
  for (int m = 0; m < 3; ++m) {
    const double nd = (m == d) ? 1.0 : 0.0;
    Rm[(1 + m) * 5 + 0] = vel[m] - c * nd;
    Rm[(1 + m) * 5 + 1] = vel[m];
    Rm[(1 + m) * 5 + 4] = vel[m] + c * nd;
  }
  Rm[4 * 5 + 0] = H - un * c;
  Rm[4 * 5 + 1] = qq;
  Rm[4 * 5 + 4] = H + un * c;
  Rm[(1 + t1) * 5 + 2] = 1.0;  Rm[4 * 5 + 2] = vel[t1];
  Rm[(1 + t2) * 5 + 3] = 1.0;  Rm[4 * 5 + 3] = vel[t2];
}

// -----------------------------------------------------------------------------
// The solver state.  Arrays are SoA, C order [k][j][i] with ng ghost layers on
// every side (w_gpu(1-ng:nx+ng, 1-ng:ny+ng, 1-ng:nz+ng, nv),
// x unit-stride, variable index slowest).
// -----------------------------------------------------------------------------
struct Solver {
  oracle_params P;
  int nx, ny, nz, ng, L, Lv, r;
  int px, py, pz;
  size_t np;                      // padded points per field
  double a1[4], a1v[4], b2v[4];   // a_l (central order), a_l and b_l (viscous order)
  double inv_dx, inv_dz;
  std::vector<double> ynode;      // ny + 2 ng node coordinates incl. reflected ghosts
  std::vector<double> eta_y_c;    // d eta / dy, central-order stencil        [ny]
  std::vector<double> eta_y_v;    // d eta / dy, viscous-order stencil        [ny]
  std::vector<double> eta_yy_v;   // d2 eta / dy2, viscous-order stencil      [ny]
  bool uniform_y;
  std::vector<double> w[5];       // conserved rho, rho u, rho v, rho w, rho E  (padded)
  std::vector<double> u, v, ww, H, p, T, mu, c;   // primitives (padded)
  std::vector<double> theta, divu;                // sensor and dilatation (padded)
  std::vector<uint8_t> mask;                      // node flag (padded)
  std::vector<uint8_t> mask_override;             // optional externally imposed mask (interior)
  bool have_override = false;
  std::vector<double> R[5], Rprev[5];             // interior only (PAPER:156 fln_gpu(1:nx,1:ny,1:nz,nv))
  bool have_fields = false;
  long step_count = 0;
  double time = 0.0, dt = 0.0;

  size_t idx(int i, int j, int k) const {
    return (size_t)(k + ng) * py * px + (size_t)(j + ng) * px + (size_t)(i + ng);
  }
  size_t iidx(int i, int j, int k) const { return ((size_t)k * ny + j) * nx + i; }

  explicit Solver(const oracle_params& p_, const double* y_nodes) : P(p_) {
    nx = P.nx; ny = P.ny; nz = P.nz;
    L = P.central_order / 2;
    Lv = (P.visc_law == VISC_NONE) ? 0 : P.visc_order / 2;
    r = (P.flux_mode == FLUX_CENTRAL) ? 0 : (P.weno_order + 1) / 2;
    ng = std::max(L, std::max(Lv, r));
    px = nx + 2 * ng; py = ny + 2 * ng; pz = nz + 2 * ng;
    np = (size_t)px * py * pz;
    fd1_coeffs(L, a1);
    if (Lv > 0) { fd1_coeffs(Lv, a1v); fd2_coeffs(Lv, b2v); }
    inv_dx = (double)nx / P.lx;
    inv_dz = (double)nz / P.lz;
    for (int m = 0; m < 5; ++m) { w[m].assign(np, 0.0); R[m].assign((size_t)nx * ny * nz, 0.0); Rprev[m].assign((size_t)nx * ny * nz, 0.0); }
    for (auto* f : {&u, &v, &ww, &H, &p, &T, &mu, &c, &theta, &divu}) f->assign(np, 0.0);
    mask.assign(np, 0);
    build_metrics(y_nodes);
  }

  // ---------------------------------------------------------------------------
  // y metrics (O4 / S3): computational coordinate eta has unit spacing, eta_j = j.
  // d/dy = eta_y d/deta,  d2/dy2 = eta_y^2 d2/deta2 + eta_yy d/deta,
  // eta_y = 1 / (D_eta y),  eta_yy = -(D_etaeta y) eta_y^3, with the same central
  // stencils applied to the node array, extended by odd reflection about the
  // boundary planes (wall / free-stream sides) or by the period (periodic).
  // Uniform y (no node array): constants, eta_y = 1/dy exactly, eta_yy = 0.
  // ---------------------------------------------------------------------------
  void build_metrics(const double* y_nodes) {
    uniform_y = (y_nodes == nullptr);
    eta_y_c.assign(ny, 0.0); eta_y_v.assign(ny, 0.0); eta_yy_v.assign(ny, 0.0);
    ynode.assign(ny + 2 * ng, 0.0);
    const bool per = (P.bc_y_lo == BC_PERIODIC);
    if (uniform_y) {
      const double inv_dy = per ? (double)ny / P.ly : (double)ny / (P.y_hi - P.y_lo);
      for (int j = 0; j < ny; ++j) { eta_y_c[j] = inv_dy; eta_y_v[j] = inv_dy; eta_yy_v[j] = 0.0; }
      const double dy = 1.0 / inv_dy;
      for (int j = -ng; j < ny + ng; ++j) ynode[j + ng] = per ? j * dy : P.y_lo + (j + 0.5) * dy;
      return;
    }
    for (int j = 0; j < ny; ++j) ynode[j + ng] = y_nodes[j];
    for (int m = 0; m < ng; ++m) {
      if (per) {
        ynode[ng - 1 - m] = y_nodes[ny - 1 - m] - P.ly;
        ynode[ng + ny + m] = y_nodes[m] + P.ly;
      } else {
        ynode[ng - 1 - m] = 2.0 * P.y_lo - y_nodes[m];
        ynode[ng + ny + m] = 2.0 * P.y_hi - y_nodes[ny - 1 - m];
      }
    }
    for (int j = 0; j < ny; ++j) {
      const double* y = &ynode[j + ng];
      double acc = a1[0] * (y[1] - y[-1]);
      for (int l = 2; l <= L; ++l) acc = acc + a1[l - 1] * (y[l] - y[-l]);
      eta_y_c[j] = 1.0 / acc;
      if (Lv > 0) {
        double d1 = a1v[0] * (y[1] - y[-1]);
        for (int l = 2; l <= Lv; ++l) d1 = d1 + a1v[l - 1] * (y[l] - y[-l]);
        double d2 = b2v[0] * ((y[1] - 2.0 * y[0]) + y[-1]);
        for (int l = 2; l <= Lv; ++l) d2 = d2 + b2v[l - 1] * ((y[l] - 2.0 * y[0]) + y[-l]);
        const double ey = 1.0 / d1;
        eta_y_v[j] = ey;
        eta_yy_v[j] = -d2 * ((ey * ey) * ey);
      }
    }
  }

  // ---------------------------------------------------------------------------
  // O6 ghost fill (BASELINE north_star "periodic and isothermal wall").
  // Periodic: w(-1-m) = w(n-1-m), w(n+m) = w(m).
  // Isothermal no-slip wall, staggered (wall plane midway between j=-1 and j=0):
  //   u_i(-1-m) = -u_i(m), T(-1-m) = 2 T_w - T(m), p(-1-m) = p(m), rho = p/(R T),
  //   then the conserved state is rebuilt.  T_ghost is clamped to >= 0.1 T_w (S15).
  // Free stream: ghosts = freestream[5].
  // Order x, then y over all (padded) i, then z over all (padded) i, j.
  // ---------------------------------------------------------------------------
  void wall_image(const double src[5], double t_wall, double dst[5]) const {
    const double rho = src[0];
    const double uu = src[1] / rho, vv = src[2] / rho, wv = src[3] / rho;
    const double ke = 0.5 * ((uu * uu + vv * vv) + wv * wv);
    const double pp = (P.gamma - 1.0) * (src[4] - rho * ke);
    const double TT = pp / (rho * P.rgas);
    double Tg = 2.0 * t_wall - TT;
    const double Tmin = 0.1 * t_wall;
    if (Tg < Tmin) Tg = Tmin;
    const double rg = pp / (P.rgas * Tg);
    dst[0] = rg;
    dst[1] = -(rg * uu);
    dst[2] = -(rg * vv);
    dst[3] = -(rg * wv);
    dst[4] = pp / (P.gamma - 1.0) + rg * ke;
  }

  void fill_ghosts() {
    // x faces
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int m = 0; m < ng; ++m)
          for (int q = 0; q < 5; ++q) {
            if (P.bc_x == BC_PERIODIC) {
              w[q][idx(-1 - m, j, k)] = w[q][idx(nx - 1 - m, j, k)];
              w[q][idx(nx + m, j, k)] = w[q][idx(m, j, k)];
            } else {
              w[q][idx(-1 - m, j, k)] = P.freestream[q];
              w[q][idx(nx + m, j, k)] = P.freestream[q];
            }
          }
    // y faces (all padded i)
    for (int k = 0; k < nz; ++k)
      for (int m = 0; m < ng; ++m)
        for (int i = -ng; i < nx + ng; ++i) {
          double s[5], g[5];
          // low side
          if (P.bc_y_lo == BC_PERIODIC) {
            for (int q = 0; q < 5; ++q) w[q][idx(i, -1 - m, k)] = w[q][idx(i, ny - 1 - m, k)];
          } else if (P.bc_y_lo == BC_WALL) {
            for (int q = 0; q < 5; ++q) s[q] = w[q][idx(i, m, k)];
            wall_image(s, P.t_wall_lo, g);
            for (int q = 0; q < 5; ++q) w[q][idx(i, -1 - m, k)] = g[q];
          } else {
            for (int q = 0; q < 5; ++q) w[q][idx(i, -1 - m, k)] = P.freestream[q];
          }
          // high side
          if (P.bc_y_hi == BC_PERIODIC) {
            for (int q = 0; q < 5; ++q) w[q][idx(i, ny + m, k)] = w[q][idx(i, m, k)];
          } else if (P.bc_y_hi == BC_WALL) {
            for (int q = 0; q < 5; ++q) s[q] = w[q][idx(i, ny - 1 - m, k)];
            wall_image(s, P.t_wall_hi, g);
            for (int q = 0; q < 5; ++q) w[q][idx(i, ny + m, k)] = g[q];
          } else {
            for (int q = 0; q < 5; ++q) w[q][idx(i, ny + m, k)] = P.freestream[q];
          }
        }
    // z faces (all padded i, j)
    for (int m = 0; m < ng; ++m)
      for (int j = -ng; j < ny + ng; ++j)
        for (int i = -ng; i < nx + ng; ++i)
          for (int q = 0; q < 5; ++q) {
            if (P.bc_z == BC_PERIODIC) {
              w[q][idx(i, j, -1 - m)] = w[q][idx(i, j, nz - 1 - m)];
              w[q][idx(i, j, nz + m)] = w[q][idx(i, j, m)];
            } else {
              w[q][idx(i, j, -1 - m)] = P.freestream[q];
              w[q][idx(i, j, nz + m)] = P.freestream[q];
            }
          }
  }

  // ---------------------------------------------------------------------------
  // a2 conservative -> primitive on every padded node (ideal gas):
  // u_i = rho u_i / rho; p = (gamma-1)(rho E - rho q^2/2); T = p/(rho R);
  // H = (rho E + p)/rho; c = sqrt(gamma p / rho); mu(T).
  // Sutherland: mu = mu_ref t sqrt(t) (1+s)/(t+s), t = T/T_ref (O4: t*sqrt(t), never pow).
  // ---------------------------------------------------------------------------
  double viscosity(double TT) const {
    if (P.visc_law == VISC_NONE) return 0.0;
    const double t = TT / P.t_ref;
    if (P.visc_law == VISC_SUTHERLAND) return ((P.mu_ref * (t * std::sqrt(t))) * (1.0 + P.suth_s)) / (t + P.suth_s);
    return P.mu_ref * std::pow(t, P.pow_exp);
  }

  void cons_to_prim() {
#pragma omp parallel for
    for (long n = 0; n < (long)np; ++n) {
      const double rho = w[0][n];
      const double uu = w[1][n] / rho, vv = w[2][n] / rho, wv = w[3][n] / rho;
      const double ke = 0.5 * ((uu * uu + vv * vv) + wv * wv);
      const double pp = (P.gamma - 1.0) * (w[4][n] - rho * ke);
      u[n] = uu; v[n] = vv; ww[n] = wv; p[n] = pp;
      T[n] = pp / (rho * P.rgas);
      H[n] = (w[4][n] + pp) / rho;
      c[n] = std::sqrt(P.gamma * pp / rho);
      mu[n] = viscosity(T[n]);
    }
  }

  double metric1(int d, int j) const { return d == 0 ? inv_dx : (d == 1 ? eta_y_c[j] : inv_dz); }

  // ---------------------------------------------------------------------------
  // O2 sensor and node mask ("modified version of the classical Ducros
  // shock sensor"): theta = max(-div / sqrt(div^2 + |curl|^2 + eps_s), 0),
  // eps_s = (u_ref/l_ref)^2, flagged iff theta > threshold (strict).
  // Velocity derivatives: 2L-order central, canonical evaluation order
  // (no contraction; this file is built with -ffp-contract=off):
  //   delta_l = f_{+l} - f_{-l}; acc = a_1 delta_1; acc = acc + a_l delta_l (l = 2..L);
  //   derivative = acc * metric.
  // Ghost nodes of theta/div/mask (S6): periodic wrap copy; otherwise constant
  // extrapolation of the nearest interior value.
  // ---------------------------------------------------------------------------
  double ddx(const std::vector<double>& f, size_t n, size_t stride, double metric) const {
    double acc = a1[0] * (f[n + stride] - f[n - stride]);
    for (int l = 2; l <= L; ++l) acc = acc + a1[l - 1] * (f[n + l * stride] - f[n - l * stride]);
    return acc * metric;
  }

  void sensor() {
    const double rr = P.u_ref / P.l_ref;
    const double eps_s = rr * rr;
    const size_t sx = 1, sy = px, sz = (size_t)px * py;
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          const size_t n = idx(i, j, k);
          const double my = eta_y_c[j];
          const double ux = ddx(u, n, sx, inv_dx), uy = ddx(u, n, sy, my), uz = ddx(u, n, sz, inv_dz);
          const double vx = ddx(v, n, sx, inv_dx), vy = ddx(v, n, sy, my), vz = ddx(v, n, sz, inv_dz);
          const double wx = ddx(ww, n, sx, inv_dx), wy = ddx(ww, n, sy, my), wz = ddx(ww, n, sz, inv_dz);
          const double dv = (ux + vy) + wz;
          const double ox = wy - vz, oy = uz - wx, oz = vx - uy;
          const double s = (((dv * dv + ox * ox) + oy * oy) + oz * oz) + eps_s;
          double th = -dv / std::sqrt(s);
          if (!(th > 0.0)) th = 0.0;
          divu[n] = dv;
          theta[n] = th;
          mask[n] = (th > P.sensor_threshold) ? 1 : 0;
          if (have_override) mask[n] = mask_override[iidx(i, j, k)];
        }
    fill_scalar_ghosts(divu); fill_scalar_ghosts(theta); fill_scalar_ghosts(mask);
  }

  template <class V>
  void fill_scalar_ghosts(V& f) const {
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int m = 0; m < ng; ++m) {
          const bool per = P.bc_x == BC_PERIODIC;
          f[idx(-1 - m, j, k)] = f[idx(per ? nx - 1 - m : 0, j, k)];
          f[idx(nx + m, j, k)] = f[idx(per ? m : nx - 1, j, k)];
        }
    for (int k = 0; k < nz; ++k)
      for (int m = 0; m < ng; ++m)
        for (int i = -ng; i < nx + ng; ++i) {
          f[idx(i, -1 - m, k)] = f[idx(i, P.bc_y_lo == BC_PERIODIC ? ny - 1 - m : 0, k)];
          f[idx(i, ny + m, k)] = f[idx(i, P.bc_y_hi == BC_PERIODIC ? m : ny - 1, k)];
        }
    for (int m = 0; m < ng; ++m)
      for (int j = -ng; j < ny + ng; ++j)
        for (int i = -ng; i < nx + ng; ++i) {
          const bool per = P.bc_z == BC_PERIODIC;
          f[idx(i, j, -1 - m)] = f[idx(i, j, per ? nz - 1 - m : 0)];
          f[idx(i, j, nz + m)] = f[idx(i, j, per ? m : nz - 1)];
        }
  }

  // Interface flag (O2 / S5): interface n+1/2 along stride uses WENO iff any node of
  // its 2r-node WENO stencil {n-r+1, ..., n+r} is flagged.  Binary switch.
  bool interface_flag(size_t n, size_t stride) const {
    if (P.flux_mode == FLUX_CENTRAL) return false;
    if (P.flux_mode == FLUX_WENO) return true;
    for (int m = -r + 1; m <= r; ++m)
      if (mask[n + m * stride]) return true;
    return false;
  }

  // ---------------------------------------------------------------------------
  // O1 central flux of order 2L at interface n+1/2 along direction d
  // (PAPER:36 skew-symmetric split form cast as numerical fluxes, ref [27]):
  //   f^phi = 1/4 sum_{l=1..L} a_l sum_{m=0..l-1}
  //             (rho_a + rho_b)(u_d,a + u_d,b)(phi_a + phi_b),  a = n-m, b = n-m+l,
  //   phi in {1, u, v, w, H};  pressure p^ = sum_l a_l sum_m (p_a + p_b) added to the
  //   d-momentum flux only (S1: cubic split; S2: energy variable H).
  // ---------------------------------------------------------------------------
  void central_flux(int d, size_t n, size_t stride, double f[5]) const {
    const std::vector<double>& rho = w[0];
    const std::vector<double>& ud = (d == 0) ? u : (d == 1 ? v : ww);
    double fs[5] = {0, 0, 0, 0, 0}, ps = 0.0;
    for (int l = 1; l <= L; ++l) {
      double in[5] = {0, 0, 0, 0, 0}, pin = 0.0;
      for (int m = 0; m < l; ++m) {
        const size_t a = n - m * stride, b = a + l * stride;
        const double ru = (rho[a] + rho[b]) * (ud[a] + ud[b]);
        in[0] += ru * 2.0;
        in[1] += ru * (u[a] + u[b]);
        in[2] += ru * (v[a] + v[b]);
        in[3] += ru * (ww[a] + ww[b]);
        in[4] += ru * (H[a] + H[b]);
        pin += p[a] + p[b];
      }
      for (int q = 0; q < 5; ++q) fs[q] += a1[l - 1] * in[q];
      ps += a1[l - 1] * pin;
    }
    for (int q = 0; q < 5; ++q) f[q] = 0.25 * fs[q];
    if (!(P.dbg_flags & DBG_NO_PRESSURE)) f[1 + d] += ps;
  }

  // ---------------------------------------------------------------------------
  // O3 WENO characteristic flux at interface n+1/2 along direction d.
  // 1. Roe average of nodes n, n+1.  2. Eigenvectors at that state.
  // 3. Local Lax-Friedrichs split per characteristic field s over the 2r stencil
  //    nodes: lambda_s = max |u_d - c|, |u_d|, |u_d + c|;
  //    g+-_{s,node} = 1/2 l_s . (F_d(w_node) +- lambda_s w_node).
  // 4. g^+ from nodes n-r+1..n+r-1 (left-biased), g^- from the mirror set
  //    n+r..n-r+2, order 2r-1, Jiang-Shu weights.
  // 5. f^ = sum_s (g^+_s + g^-_s) r_s   (pressure is inside F_d).
  // ---------------------------------------------------------------------------
  void weno_flux(int d, size_t n, size_t stride, double f[5]) const {
    const std::vector<double>& rho = w[0];
    const std::vector<double>& ud = (d == 0) ? u : (d == 1 ? v : ww);
    // 1. Roe average
    const size_t nl = n, nr = n + stride;
    const double rw = std::sqrt(rho[nr] / rho[nl]);
    const double den = 1.0 + rw;
    double vel[3];
    vel[0] = (u[nl] + rw * u[nr]) / den;
    vel[1] = (v[nl] + rw * v[nr]) / den;
    vel[2] = (ww[nl] + rw * ww[nr]) / den;
    const double Hb = (H[nl] + rw * H[nr]) / den;
    // 2. eigenvectors
    double Lm[25], Rm[25];
    euler_eigenvectors(d, vel, Hb, P.gamma, Lm, Rm);
    // 3. wave-speed bounds over the 2r stencil nodes
    double lam[5] = {0, 0, 0, 0, 0};
    for (int m = -r + 1; m <= r; ++m) {
      const size_t q = n + m * stride;
      lam[0] = std::max(lam[0], std::fabs(ud[q] - c[q]));
      lam[1] = std::max(lam[1], std::fabs(ud[q]));
      lam[4] = std::max(lam[4], std::fabs(ud[q] + c[q]));
    }
    lam[2] = lam[1]; lam[3] = lam[1];
    // nodal fluxes and states on the stencil, index m + r - 1 for m = -r+1 .. r
    double Fn[8][5], Wn[8][5];
    for (int m = -r + 1; m <= r; ++m) {
      const size_t q = n + m * stride;
      double* F = Fn[m + r - 1];
      double* W = Wn[m + r - 1];
      W[0] = w[0][q]; W[1] = w[1][q]; W[2] = w[2][q]; W[3] = w[3][q]; W[4] = w[4][q];
      const double un = ud[q];
      F[0] = W[0] * un;
      F[1] = W[1] * un;
      F[2] = W[2] * un;
      F[3] = W[3] * un;
      F[1 + d] += p[q];
      F[4] = (W[4] + p[q]) * un;
    }
    const bool linear = (P.dbg_flags & DBG_WENO_LINEAR) != 0;
    double ghat[5];
    for (int s = 0; s < 5; ++s) {
      double gp[7], gm[7];
      for (int m = 0; m < 2 * r - 1; ++m) {
        // left-biased stencil n-r+1 .. n+r-1  -> stencil slots 0 .. 2r-2
        // mirror stencil      n+r   .. n-r+2  -> stencil slots 2r-1 .. 1
        const double* Fp = Fn[m];          const double* Wp = Wn[m];
        const double* Fm = Fn[2 * r - 1 - m]; const double* Wm = Wn[2 * r - 1 - m];
        double sp = 0.0, sm = 0.0;
        for (int q = 0; q < 5; ++q) {
          sp += Lm[s * 5 + q] * (Fp[q] + lam[s] * Wp[q]);
          sm += Lm[s * 5 + q] * (Fm[q] - lam[s] * Wm[q]);
        }
        gp[m] = 0.5 * sp;
        gm[m] = 0.5 * sm;
      }
      ghat[s] = weno_reconstruct(gp, r, P.weno_eps, linear, nullptr, P.weno_variant) +
                weno_reconstruct(gm, r, P.weno_eps, linear, nullptr, P.weno_variant);
    }
    // 5. project back on the right eigenvectors
    for (int q = 0; q < 5; ++q) {
      double acc = 0.0;
      for (int s = 0; s < 5; ++s) acc += ghat[s] * Rm[q * 5 + s];
      f[q] = acc;
    }
  }

  // a4-a6: R -= (f_{n+1/2} - f_{n-1/2}) * metric along each pencil of direction d.
  void convective(int d) {
    const size_t stride = (d == 0) ? 1 : (d == 1 ? (size_t)px : (size_t)px * py);
    const int nd = (d == 0) ? nx : (d == 1 ? ny : nz);
    const int n1 = (d == 0) ? ny : nx;                 // faster of the two remaining loops
    const int n2 = (d == 2) ? ny : nz;                 // slower
#pragma omp parallel for
    for (int b = 0; b < n2; ++b) {
      std::vector<double> fl((size_t)(nd + 1) * 5);
      for (int a = 0; a < n1; ++a) {
        for (int s = -1; s < nd; ++s) {
          int i, j, k;
          if (d == 0) { i = s; j = a; k = b; }
          else if (d == 1) { i = a; j = s; k = b; }
          else { i = a; j = b; k = s; }
          const size_t n = idx(i, j, k);
          double* f = &fl[(size_t)(s + 1) * 5];
          if (interface_flag(n, stride)) weno_flux(d, n, stride, f);
          else central_flux(d, n, stride, f);
        }
        for (int s = 0; s < nd; ++s) {
          int i, j, k;
          if (d == 0) { i = s; j = a; k = b; }
          else if (d == 1) { i = a; j = s; k = b; }
          else { i = a; j = b; k = s; }
          const double met = metric1(d, j);
          const size_t o = iidx(i, j, k);
          for (int q = 0; q < 5; ++q)
            R[q][o] -= (fl[(size_t)(s + 1) * 5 + q] - fl[(size_t)s * 5 + q]) * met;
        }
      }
    }
  }

  // ---------------------------------------------------------------------------
  // O4 viscous terms, "expanded in Laplacian form", order 2Lv:
  //  momentum_i += mu lap(u_i) + d_j mu (d_j u_i + d_i u_j) - 2/3 d_i mu div u
  //                + mu d_i(div u)/3            (last: first derivative of stored nodal div)
  //  energy     += u_i (viscous momentum)_i + Phi + lambda lap(T) + grad lambda . grad T,
  //  Phi = mu [2(u_x^2+v_y^2+w_z^2) + (u_y+v_x)^2 + (u_z+w_x)^2 + (v_z+w_y)^2 - 2/3 (div u)^2],
  //  lambda = cp mu / Pr, cp = gamma R/(gamma-1); grad mu by differencing nodal mu.
  // Second derivatives in difference form sum_l b_l (f_{+l} - 2 f_0 + f_{-l}) so a
  // uniform state gives exactly 0.  Stretched y: d_yy = eta_y^2 d_etaeta + eta_yy d_eta.
  // The local div in Phi and the -2/3 term is the sum of this routine's own
  // u_x, v_y, w_z; the stored div (from sensor(), 2L-order) is used for grad(div) only.
  // ---------------------------------------------------------------------------
  double d1v(const std::vector<double>& f, size_t n, size_t stride) const {
    double acc = a1v[0] * (f[n + stride] - f[n - stride]);
    for (int l = 2; l <= Lv; ++l) acc = acc + a1v[l - 1] * (f[n + l * stride] - f[n - l * stride]);
    return acc;
  }
  double d2v(const std::vector<double>& f, size_t n, size_t stride) const {
    double acc = b2v[0] * ((f[n + stride] - 2.0 * f[n]) + f[n - stride]);
    for (int l = 2; l <= Lv; ++l) acc = acc + b2v[l - 1] * ((f[n + l * stride] - 2.0 * f[n]) + f[n - l * stride]);
    return acc;
  }

  void viscous() {
    const double cp = P.gamma * P.rgas / (P.gamma - 1.0);
    const double kfac = cp / P.prandtl;     // lambda = kfac * mu
    const size_t st[3] = {1, (size_t)px, (size_t)px * py};
#pragma omp parallel for
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          const size_t n = idx(i, j, k);
          const double m1[3] = {inv_dx, eta_y_v[j], inv_dz};
          const std::vector<double>* vel[3] = {&u, &v, &ww};
          double g[3][3];        // g[a][b] = d u_a / d x_b
          double lap[3] = {0, 0, 0}, lapT = 0.0;
          double gT[3], gmu[3], gdiv[3];
          for (int b = 0; b < 3; ++b) {
            const double met = m1[b];
            for (int a = 0; a < 3; ++a) {
              const double de = d1v(*vel[a], n, st[b]);
              g[a][b] = de * met;
              double sec = d2v(*vel[a], n, st[b]) * (met * met);
              if (b == 1) sec += eta_yy_v[j] * de;
              lap[a] += sec;
            }
            const double dT = d1v(T, n, st[b]);
            gT[b] = dT * met;
            double secT = d2v(T, n, st[b]) * (met * met);
            if (b == 1) secT += eta_yy_v[j] * dT;
            lapT += secT;
            gmu[b] = d1v(mu, n, st[b]) * met;
            gdiv[b] = d1v(divu, n, st[b]) * met;
          }
          const double dv = (g[0][0] + g[1][1]) + g[2][2];
          const double m = mu[n];
          double vm[3];
          for (int a = 0; a < 3; ++a) {
            double cross = 0.0;
            for (int b = 0; b < 3; ++b) cross += gmu[b] * (g[a][b] + g[b][a]);
            vm[a] = m * lap[a] + cross - (2.0 / 3.0) * gmu[a] * dv + m * gdiv[a] / 3.0;
          }
          const double s01 = g[0][1] + g[1][0], s02 = g[0][2] + g[2][0], s12 = g[1][2] + g[2][1];
          const double phi = m * (2.0 * (g[0][0] * g[0][0] + g[1][1] * g[1][1] + g[2][2] * g[2][2]) +
                                  s01 * s01 + s02 * s02 + s12 * s12 - (2.0 / 3.0) * dv * dv);
          const double cond = kfac * (m * lapT + (gmu[0] * gT[0] + gmu[1] * gT[1] + gmu[2] * gT[2]));
          const size_t o = iidx(i, j, k);
          R[1][o] += vm[0];
          R[2][o] += vm[1];
          R[3][o] += vm[2];
          R[4][o] += (u[n] * vm[0] + v[n] * vm[1] + ww[n] * vm[2]) + phi + cond;
        }
  }

  // ---------------------------------------------------------------------------
  // S17 forcing ("Forcing term evaluations"; Table 2): a uniform body acceleration g drives the flow
  // (the streamwise pressure gradient of a channel): rho g on the momentum equations and its work (rho u) . g on
  // the total energy.  The paper's controller, which adjusts g to hold the bulk flow rate, is host logic on top
  // of the bulk sums and not part of the right-hand side.
  // ---------------------------------------------------------------------------
  void body_force() {
    const double* g = P.accel;
    if (g[0] == 0.0 && g[1] == 0.0 && g[2] == 0.0) return;
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          const size_t n = idx(i, j, k), o = iidx(i, j, k);
          R[1][o] += w[0][n] * g[0];
          R[2][o] += w[0][n] * g[1];
          R[3][o] += w[0][n] * g[2];
          R[4][o] += (w[1][n] * g[0] + w[2][n] * g[1]) + w[3][n] * g[2];
        }
  }

  // Per RK stage (O5): fill ghosts -> prims -> sensor/div (+ghosts) -> R.
  void rhs(int parts) {
    fill_ghosts();
    cons_to_prim();
    if (P.flux_mode == FLUX_HYBRID || P.visc_law != VISC_NONE) sensor();
    for (int q = 0; q < 5; ++q) std::fill(R[q].begin(), R[q].end(), 0.0);
    if (parts & PART_X) convective(0);
    if (parts & PART_Y) convective(1);
    if (parts & PART_Z) convective(2);
    if ((parts & PART_VISC) && P.visc_law != VISC_NONE) viscous();
    if (parts & PART_FORCE) body_force();
  }

  // ---------------------------------------------------------------------------
  // a9 / O5 time step ("Time step evaluation (max reduction)"; S13):
  // dt = CFL / max over interior points and the three directions of
  //   (|u_d| + c) m_d,  (mu/rho) m_d^2,  (gamma mu / (rho Pr)) m_d^2,
  // m_d = 1/dx, eta_y(j), 1/dz.  Uses the state at the start of the step.
  // ---------------------------------------------------------------------------
  double compute_dt() {
    fill_ghosts();
    cons_to_prim();
    double rmax = 0.0;
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          const size_t n = idx(i, j, k);
          const double md[3] = {inv_dx, eta_y_c[j], inv_dz};
          const double vel[3] = {u[n], v[n], ww[n]};
          const double nu = mu[n] / w[0][n];
          for (int d = 0; d < 3; ++d) {
            rmax = std::max(rmax, (std::fabs(vel[d]) + c[n]) * md[d]);
            rmax = std::max(rmax, nu * (md[d] * md[d]));
            rmax = std::max(rmax, (P.gamma * nu / P.prandtl) * (md[d] * md[d]));
          }
        }
    return P.cfl / rmax;
  }

  // ---------------------------------------------------------------------------
  // O5 third-order low-storage Runge-Kutta (S12: Wray's coefficients):
  // w^(l) = w^(l-1) + dt [gamma_l R(w^(l-1)) + rho_l R(w^(l-2))],
  // gamma = (8/15, 5/12, 3/4), rho = (0, -17/60, -5/12); time += dt per step.
  // The paper splits the update into update_flux + update_field.
  // ---------------------------------------------------------------------------
  int step(int nsteps) {
    const double gam[3] = {8.0 / 15.0, 5.0 / 12.0, 3.0 / 4.0};
    const double rhk[3] = {0.0, -17.0 / 60.0, -5.0 / 12.0};
    for (int s = 0; s < nsteps; ++s) {
      if (P.dt_fixed > 0.0) dt = P.dt_fixed;
      else if (step_count % std::max(P.dt_every, 1) == 0) dt = compute_dt();
      if (!std::isfinite(dt)) return -5;
      for (int l = 0; l < 3; ++l) {
        rhs(PART_ALL);
#pragma omp parallel for
        for (int k = 0; k < nz; ++k)
          for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
              const size_t o = iidx(i, j, k), n = idx(i, j, k);
              for (int q = 0; q < 5; ++q)
                w[q][n] = w[q][n] + dt * (gam[l] * R[q][o] + rhk[l] * Rprev[q][o]);
            }
        for (int q = 0; q < 5; ++q) R[q].swap(Rprev[q]);
      }
      time += dt;
      step_count += 1;
    }
    return 0;
  }

  // ---------------------------------------------------------------------------
  // S18 bulk-flow control of a forced channel ("forcing term evaluations (sum reduction)"
  // force_rhs): after every step the volume integrals M = sum rho dV and P = sum (rho u_d) dV are taken
  // (dV = dx dz / eta_y(j), nodes in index order) and the uniform acceleration along d is reset so that P returns to
  // its target over the next step: a force g acting for dt changes P by g M dt, hence
  //   g <- [g - (P - P_prev) / (M dt)] + (P_target - P) / (M dt),
  // the first bracket being the force that would have kept P constant over the step just taken (the running estimate
  // of the wall friction).  The paper prints no controller formula: this reading is pinned by its defining property
  // (deadbeat on a frictionless uniform flow, tests/test_oracle_force.py), not against STREAmS.
  // ---------------------------------------------------------------------------
  bool ctrl_started = false;
  double ctrl_prev = 0.0, ctrl_target = 0.0;
  void bulk_sums(int d, double& mass, double& mom) const {
    mass = 0.0; mom = 0.0;
    const double dxdz = 1.0 / (inv_dx * inv_dz);
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          const size_t n = idx(i, j, k);
          const double dV = dxdz / eta_y_c[j];
          mass += w[0][n] * dV;
          mom += w[1 + d][n] * dV;
        }
  }
  int step_forced(int nsteps, int d, double target) {
    double mass, mom;
    if (!ctrl_started) {
      bulk_sums(d, mass, mom);
      ctrl_prev = mom;
      ctrl_target = std::isnan(target) ? mom : target;
      ctrl_started = true;
    } else if (!std::isnan(target)) {
      ctrl_target = target;
    }
    for (int s = 0; s < nsteps; ++s) {
      const int rc = step(1);
      if (rc) return rc;
      bulk_sums(d, mass, mom);
      const double g_balance = P.accel[d] - (mom - ctrl_prev) / (mass * dt);
      P.accel[d] = g_balance + (ctrl_target - mom) / (mass * dt);
      ctrl_prev = mom;
    }
    return 0;
  }
};

}  // namespace

// =============================================================================
// C entry points used by oracle/oracle.py (ctypes).  Interior arrays are
// [5][nz][ny][nx] (conserved) or [nz][ny][nx] (scalars), C order, host memory.
// =============================================================================
extern "C" {

void* oracle_create(const oracle_params* p, const double* y_nodes) {
  if (!p || p->nx < 1 || p->ny < 1 || p->nz < 1) return nullptr;
  const int L = p->central_order / 2;
  if (p->central_order % 2 || L < 1 || L > 4) return nullptr;
  if (p->flux_mode != FLUX_CENTRAL && (p->weno_order % 2 == 0 || p->weno_order < 1 || p->weno_order > 7)) return nullptr;
  if (p->weno_variant < 0 || p->weno_variant > 1) return nullptr;
  if (p->visc_law != VISC_NONE && (p->visc_order % 2 || p->visc_order < 2 || p->visc_order > 8)) return nullptr;
  return new Solver(*p, y_nodes);
}
void oracle_destroy(void* h) { delete static_cast<Solver*>(h); }
int oracle_ng(void* h) { return static_cast<Solver*>(h)->ng; }

int oracle_set_fields(void* h, const double* win) {
  Solver* s = static_cast<Solver*>(h);
  const size_t N = (size_t)s->nx * s->ny * s->nz;
  for (int q = 0; q < 5; ++q)
    for (int k = 0; k < s->nz; ++k)
      for (int j = 0; j < s->ny; ++j)
        for (int i = 0; i < s->nx; ++i) s->w[q][s->idx(i, j, k)] = win[q * N + s->iidx(i, j, k)];
  for (int q = 0; q < 5; ++q) std::fill(s->Rprev[q].begin(), s->Rprev[q].end(), 0.0);
  s->have_fields = true; s->step_count = 0; s->time = 0.0;
  return 0;
}
int oracle_get_fields(void* h, double* wout) {
  Solver* s = static_cast<Solver*>(h);
  const size_t N = (size_t)s->nx * s->ny * s->nz;
  for (int q = 0; q < 5; ++q)
    for (int k = 0; k < s->nz; ++k)
      for (int j = 0; j < s->ny; ++j)
        for (int i = 0; i < s->nx; ++i) wout[q * N + s->iidx(i, j, k)] = s->w[q][s->idx(i, j, k)];
  return 0;
}
// parts: bit0 x-convective, bit1 y, bit2 z, bit3 viscous, bit4 body force (PART_ALL = 31 = the full RHS).
int oracle_rhs(void* h, int parts, double* rhs_out) {
  Solver* s = static_cast<Solver*>(h);
  if (!s->have_fields) return -4;
  s->rhs(parts);
  const size_t N = (size_t)s->nx * s->ny * s->nz;
  if (rhs_out) for (int q = 0; q < 5; ++q) std::memcpy(rhs_out + q * N, s->R[q].data(), N * sizeof(double));
  return 0;
}
int oracle_step(void* h, int nsteps, double* dt_last, double* time) {
  Solver* s = static_cast<Solver*>(h);
  if (!s->have_fields) return -4;
  const int rc = s->step(nsteps);
  if (dt_last) *dt_last = s->dt;
  if (time) *time = s->time;
  return rc;
}
double oracle_compute_dt(void* h) { return static_cast<Solver*>(h)->compute_dt(); }
// S18: nsteps steps under the bulk-flow controller along direction d; target NaN = hold the current bulk momentum.
// accel3_out (nullable) receives the acceleration after the last update.
int oracle_step_forced(void* h, int nsteps, int d, double target, double* dt_last, double* time, double* accel3_out) {
  Solver* s = static_cast<Solver*>(h);
  if (!s->have_fields) return -4;
  if (d < 0 || d > 2) return -1;
  const int rc = s->step_forced(nsteps, d, target);
  if (dt_last) *dt_last = s->dt;
  if (time) *time = s->time;
  if (accel3_out) for (int a = 0; a < 3; ++a) accel3_out[a] = s->P.accel[a];
  return rc;
}
void oracle_bulk_sums(void* h, int d, double* mass, double* mom) { static_cast<Solver*>(h)->bulk_sums(d, *mass, *mom); }

// theta / mask / div of the last rhs() (interior, [nz][ny][nx]).
int oracle_get_sensor(void* h, double* theta_out, unsigned char* mask_out, double* div_out) {
  Solver* s = static_cast<Solver*>(h);
  for (int k = 0; k < s->nz; ++k)
    for (int j = 0; j < s->ny; ++j)
      for (int i = 0; i < s->nx; ++i) {
        const size_t n = s->idx(i, j, k), o = s->iidx(i, j, k);
        if (theta_out) theta_out[o] = s->theta[n];
        if (mask_out) mask_out[o] = s->mask[n];
        if (div_out) div_out[o] = s->divu[n];
      }
  return 0;
}
// Impose a node mask instead of the sensor's (activation sweeps, dilation pin). NULL clears it.
int oracle_set_mask_override(void* h, const unsigned char* m) {
  Solver* s = static_cast<Solver*>(h);
  if (!m) { s->have_override = false; return 0; }
  s->mask_override.assign(m, m + (size_t)s->nx * s->ny * s->nz);
  s->have_override = true;
  return 0;
}
// Interface flags of the last rhs() along direction d: out[(nd+1) * n1 * n2] laid out as the
// interior array with the d extent enlarged by one (entry s <-> interface s - 1/2).
int oracle_interface_flags(void* h, int d, unsigned char* out) {
  Solver* s = static_cast<Solver*>(h);
  const size_t stride = (d == 0) ? 1 : (d == 1 ? (size_t)s->px : (size_t)s->px * s->py);
  const int ex = s->nx + (d == 0), ey = s->ny + (d == 1), ez = s->nz + (d == 2);
  for (int k = 0; k < ez; ++k)
    for (int j = 0; j < ey; ++j)
      for (int i = 0; i < ex; ++i) {
        const int ii = i - (d == 0), jj = j - (d == 1), kk = k - (d == 2);
        out[((size_t)k * ey + j) * ex + i] = s->interface_flag(s->idx(ii, jj, kk), stride) ? 1 : 0;
      }
  return 0;
}
// Primitive fields of the last rhs(): which = 0 u, 1 v, 2 w, 3 H, 4 p, 5 T, 6 mu, 7 c (interior).
int oracle_get_prim(void* h, int which, double* out) {
  Solver* s = static_cast<Solver*>(h);
  const std::vector<double>* f[8] = {&s->u, &s->v, &s->ww, &s->H, &s->p, &s->T, &s->mu, &s->c};
  for (int k = 0; k < s->nz; ++k)
    for (int j = 0; j < s->ny; ++j)
      for (int i = 0; i < s->nx; ++i) out[s->iidx(i, j, k)] = (*f[which])[s->idx(i, j, k)];
  return 0;
}
// Padded conserved field q after the last ghost fill: out[(nz+2ng)(ny+2ng)(nx+2ng)].
int oracle_get_padded(void* h, int q, double* out) {
  Solver* s = static_cast<Solver*>(h);
  std::memcpy(out, s->w[q].data(), s->np * sizeof(double));
  return 0;
}
int oracle_get_metrics(void* h, double* eta_y_c, double* eta_y_v, double* eta_yy_v, double* ynode_padded) {
  Solver* s = static_cast<Solver*>(h);
  for (int j = 0; j < s->ny; ++j) {
    if (eta_y_c) eta_y_c[j] = s->eta_y_c[j];
    if (eta_y_v) eta_y_v[j] = s->eta_y_v[j];
    if (eta_yy_v) eta_yy_v[j] = s->eta_yy_v[j];
  }
  if (ynode_padded) for (int j = 0; j < s->ny + 2 * s->ng; ++j) ynode_padded[j] = s->ynode[j];
  return 0;
}

// ---- building blocks exposed for the pins ----
void oracle_fd_coeffs(int order, double* a, double* b) { fd1_coeffs(order / 2, a); fd2_coeffs(order / 2, b); }
double oracle_weno_reconstruct(const double* v, int r, double eps, int linear, double* beta_out) {
  return weno_reconstruct(v, r, eps, linear != 0, beta_out);
}
double oracle_weno_reconstruct_variant(const double* v, int r, double eps, int variant) {
  return weno_reconstruct(v, r, eps, false, nullptr, variant);
}
void oracle_eigenvectors(int d, const double* vel, double H, double gamma, double* Lm, double* Rm) {
  euler_eigenvectors(d, vel, H, gamma, Lm, Rm);
}
// Threads the OpenMP build will use (1 for the serial build).
int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
