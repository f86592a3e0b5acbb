// a1 + a2 outside the fused RHS pass: ghost / boundary fill and conservative -> primitive
//   fill_prim_kernel  : the whole padded box, first evaluation after streams_set_fields (optionally with the
//                       time-step rate of every interior node, a9)
//   fill_ghost_kernel : the ghost shell of the non-periodic directions, every other stage
// Built with the default FMA contraction like streams_march.cu, whose epilogue writes the same primitives through the same
// prims_from_state (streams_dev.cuh): both translation units then compile its library calls (pow of the power-law
// viscosity) identically and a state gets the same primitive bits whichever kernel produced them.  The arithmetic that
// reaches the sensor mask (ghost velocities: wall image, u = rho u / rho) is written with explicit single-rounded
// intrinsics.
#include "streams_dev.cuh"
#include "streams_launch.h"

namespace streams {

// ---------------------------------------------------------------------------------------------
// a1 + a2: ghost / boundary fill and conservative -> primitive in one pass over the padded box.
// Each padded node finds the interior node it images (periodic wrap, wall mirror) or takes the
// free-stream state, rebuilds the conserved ghost state (isothermal no-slip wall: u -> -u,
// T -> 2 T_w - T, p -> p, rho = p/(R T); O6) and then the primitives.
// HBM: 40 B read (interior) + 8 B x (#primitive fields) write per padded node.
// ---------------------------------------------------------------------------------------------
// With DT the same pass takes the time-step rate of every interior node (a9) and reduces it (block_rate_max).
// fill_node: one padded node (i, j, k in interior coordinates, ghosts negative or beyond the extents).
template <bool VISC, bool STORE_C, bool DT>
__device__ __forceinline__ double fill_node(const DevP& P, int i, int j, int k) {
  int is = i, js = j, ks = k;
  bool fsx = false, fsy = false, fsz = false;
  double t_wall = 0.0;
  bool wall = false;
  if (i < 0) { if (P.bc_x == BC_PERIODIC) is = i + P.nx; else { fsx = true; is = 0; } }
  else if (i >= P.nx) { if (P.bc_x == BC_PERIODIC) is = i - P.nx; else { fsx = true; is = P.nx - 1; } }
  if (j < 0) {
    if (P.bc_y_lo == BC_PERIODIC) js = j + P.ny;
    else if (P.bc_y_lo == BC_WALL) { js = -1 - j; wall = true; t_wall = P.t_wall_lo; }
    else { fsy = true; js = 0; }
  } else if (j >= P.ny) {
    if (P.bc_y_hi == BC_PERIODIC) js = j - P.ny;
    else if (P.bc_y_hi == BC_WALL) { js = 2 * P.ny - 1 - j; wall = true; t_wall = P.t_wall_hi; }
    else { fsy = true; js = P.ny - 1; }
  }
  if (k < 0) { if (P.bc_z == BC_PERIODIC) ks = k + P.nz; else { fsz = true; ks = 0; } }
  else if (k >= P.nz) { if (P.bc_z == BC_PERIODIC) ks = k - P.nz; else { fsz = true; ks = P.nz - 1; } }

  const long long ns = pidx(P, is, js, ks);
  double s[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) s[q] = P.w[q * P.fs + ns];
  if (fsx) {
#pragma unroll
    for (int q = 0; q < 5; ++q) s[q] = P.fsw[q];
  }
  if (fsy) {
#pragma unroll
    for (int q = 0; q < 5; ++q) s[q] = P.fsw[q];
  } else if (wall) {
    // every operation a single IEEE operation in the order of DESIGN.md O6 (the ghost velocities feed the sensor's
    // stencils next to the wall, hence the mask): explicit intrinsics, independent of the contraction mode
    const double rho = s[0];
    const double uu = __ddiv_rn(s[1], rho), vv = __ddiv_rn(s[2], rho), wv = __ddiv_rn(s[3], rho);
    const double ke = __dmul_rn(0.5, __dadd_rn(__dadd_rn(__dmul_rn(uu, uu), __dmul_rn(vv, vv)), __dmul_rn(wv, wv)));
    const double pp = __dmul_rn(P.gm1, __dsub_rn(s[4], __dmul_rn(rho, ke)));
    const double TT = __ddiv_rn(pp, __dmul_rn(rho, P.rgas));
    double Tg = __dsub_rn(__dmul_rn(2.0, t_wall), TT);
    const double Tmin = __dmul_rn(0.1, t_wall);
    if (Tg < Tmin) Tg = Tmin;
    const double rg = __ddiv_rn(pp, __dmul_rn(P.rgas, Tg));
    s[0] = rg;
    s[1] = -__dmul_rn(rg, uu);
    s[2] = -__dmul_rn(rg, vv);
    s[3] = -__dmul_rn(rg, wv);
    s[4] = __dadd_rn(__ddiv_rn(pp, P.gm1), __dmul_rn(rg, ke));
  }
  if (fsz) {
#pragma unroll
    for (int q = 0; q < 5; ++q) s[q] = P.fsw[q];
  }
  const long long n = pidx(P, i, j, k);
  const bool ghost = (is != i) || (js != j) || (ks != k) || fsx || fsy || fsz;
  if (ghost) {
#pragma unroll
    for (int q = 0; q < 5; ++q) P.w[q * P.fs + n] = s[q];
  }
  double mu, cc, vel[3], o[NQ];
  prims_from_state<VISC, STORE_C>(P, s, DT, o, mu, cc, vel);
  store_prims<VISC, STORE_C>(P, P.q + n, o);
  double rmax = 0.0;
  if (DT && !ghost) rmax = dt_rate<VISC>(P, vel, cc, mu, s[0], P.eta_y_c[j]);
  return rmax;
}

template <bool VISC, bool STORE_C, bool DT>
__global__ void __launch_bounds__(128) fill_prim_kernel(const DevP P) {
  const int ip = blockIdx.x * blockDim.x + threadIdx.x;
  const int i = ip - P.ox, j = (int)blockIdx.y - P.ng, k = (int)blockIdx.z - P.ng;
  double rmax = 0.0;
  const bool halo_plane = P.bc_z == BC_HALO && (k < 0 || k >= P.nz);      // a neighbour's planes: not ours to fill
  if (i >= -P.ng && i < P.nx + P.ng && !halo_plane) rmax = fill_node<VISC, STORE_C, DT>(P, i, j, k);
  if (DT) {
    __shared__ unsigned long long sm[4];
    block_rate_max(P, rmax, sm);
  }
}

// The ghost shell only (every stage but the first after streams_set_fields: the fused RHS kernel has already
// written the primitives of the updated interior nodes and of their periodic images, DevP::own_*).  Up to three
// segments of a flat index (directions the RHS kernel owns are skipped): the z slabs (whole padded
// planes), the y slabs of the interior planes, the x columns of the interior rows.
template <bool VISC, bool STORE_C>
__global__ void __launch_bounds__(128) fill_ghost_kernel(const DevP P) {
  const int g = P.ng, wx = P.nx + 2 * g;
  const long long nZ = (P.own_z || P.bc_z == BC_HALO) ? 0 : 2LL * g * P.py * wx, nY = P.own_y ? 0 : (long long)P.nz * 2 * g * wx,
                  nX = P.own_x ? 0 : (long long)P.nz * P.ny * 2 * g;
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int i, j, k;
  if (t < nZ) {
    i = (int)(t % wx) - g;
    const long long t2 = t / wx;
    j = (int)(t2 % P.py) - g;
    const int m = (int)(t2 / P.py);
    k = m < g ? m - g : P.nz + (m - g);
  } else if ((t -= nZ) < nY) {
    i = (int)(t % wx) - g;
    const long long t2 = t / wx;
    const int m = (int)(t2 % (2 * g));
    k = (int)(t2 / (2 * g));
    j = m < g ? m - g : P.ny + (m - g);
  } else if ((t -= nY) < nX) {
    const int m = (int)(t % (2 * g));
    const long long t2 = t / (2 * g);
    j = (int)(t2 % P.ny);
    k = (int)(t2 / P.ny);
    i = m < g ? m - g : P.nx + (m - g);
  } else {
    return;
  }
  fill_node<VISC, STORE_C, false>(P, i, j, k);
}

// -------------------------------------------------------------------------- launch wrappers
int launch_fill_prim(const DevP& P, bool with_dt, cudaStream_t st) {
  dim3 b(128), g((P.px + 127) / 128, P.py, P.pz);
  const bool visc = P.visc_law != VISC_NONE, sc = P.flux_mode != FLUX_CENTRAL;
#define STREAMS_FILL(V, C)                                            \
  do {                                                                \
    if (with_dt) fill_prim_kernel<V, C, true><<<g, b, 0, st>>>(P);    \
    else fill_prim_kernel<V, C, false><<<g, b, 0, st>>>(P);           \
  } while (0)
  if (visc && sc) STREAMS_FILL(true, true);
  else if (visc) STREAMS_FILL(true, false);
  else if (sc) STREAMS_FILL(false, true);
  else STREAMS_FILL(false, false);
#undef STREAMS_FILL
  return 1;
}

int launch_fill_ghosts(const DevP& P, cudaStream_t st) {
  const int g = P.ng;
  const long long wx = P.nx + 2 * g;
  const long long total = ((P.own_z || P.bc_z == BC_HALO) ? 0 : 2LL * g * P.py * wx) + (P.own_y ? 0 : (long long)P.nz * 2 * g * wx) +
                          (P.own_x ? 0 : (long long)P.nz * P.ny * 2 * g);
  if (total == 0) return 0;
  dim3 b(128), gr((unsigned)((total + 127) / 128));
  const bool visc = P.visc_law != VISC_NONE, sc = P.flux_mode != FLUX_CENTRAL;
  if (visc && sc) fill_ghost_kernel<true, true><<<gr, b, 0, st>>>(P);
  else if (visc) fill_ghost_kernel<true, false><<<gr, b, 0, st>>>(P);
  else if (sc) fill_ghost_kernel<false, true><<<gr, b, 0, st>>>(P);
  else fill_ghost_kernel<false, false><<<gr, b, 0, st>>>(P);
  return 1;
}

}  // namespace streams
