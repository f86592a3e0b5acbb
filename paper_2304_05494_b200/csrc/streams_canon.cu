// Kernels whose arithmetic decides an integer (the shock-sensor mask) or feeds it:
// ghost fill + conservative->primitive, sensor/mask, interface flags, time-step reduction.
// This translation unit is compiled with -fmad=false so that every operation is a single
// IEEE fp64 operation in source order: the
// mask is then bit-identical to any IEEE evaluation of the same formulas on the same state.
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
__device__ __forceinline__ double viscosity(const DevP& P, double T) {
  const double t = T / P.t_ref;
  if (P.visc_law == VISC_SUTHERLAND) return ((P.mu_ref * (t * sqrt(t))) * (1.0 + P.suth_s)) / (t + P.suth_s);
  return P.mu_ref * pow(t, P.pow_exp);
}

template <bool VISC, bool STORE_C>
__global__ void __launch_bounds__(128) fill_prim_kernel(const DevP P) {
  const int ip = blockIdx.x * blockDim.x + threadIdx.x;
  const int i = ip - P.ox, j = (int)blockIdx.y - P.ng, k = (int)blockIdx.z - P.ng;
  if (i < -P.ng || i >= P.nx + P.ng) return;
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
    const double rho = s[0];
    const double uu = s[1] / rho, vv = s[2] / rho, wv = s[3] / rho;
    const double ke = 0.5 * ((uu * uu + vv * vv) + wv * wv);
    const double pp = P.gm1 * (s[4] - rho * ke);
    const double TT = pp / (rho * P.rgas);
    double Tg = 2.0 * t_wall - TT;
    const double Tmin = 0.1 * t_wall;
    if (Tg < Tmin) Tg = Tmin;
    const double rg = pp / (P.rgas * Tg);
    s[0] = rg;
    s[1] = -(rg * uu);
    s[2] = -(rg * vv);
    s[3] = -(rg * wv);
    s[4] = pp / P.gm1 + rg * ke;
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
  const double rho = s[0];
  const double uu = s[1] / rho, vv = s[2] / rho, wv = s[3] / rho;
  const double ke = 0.5 * ((uu * uu + vv * vv) + wv * wv);
  const double pp = P.gm1 * (s[4] - rho * ke);
  P.q[Q_U * P.fs + n] = uu;
  P.q[Q_V * P.fs + n] = vv;
  P.q[Q_W * P.fs + n] = wv;
  P.q[Q_H * P.fs + n] = (s[4] + pp) / rho;
  P.q[Q_P * P.fs + n] = pp;
  P.q[Q_RHO * P.fs + n] = rho;
  if (VISC) {
    const double TT = pp / (rho * P.rgas);
    P.q[Q_T * P.fs + n] = TT;
    P.q[Q_MU * P.fs + n] = viscosity(P, TT);
  }
  if (STORE_C) P.q[Q_C * P.fs + n] = sqrt(P.gamma * pp / rho);
}

// ---------------------------------------------------------------------------------------------
// a3: Ducros-type sensor, node mask and dilatation (O2).  One thread per interior node.
// Canonical order: delta_l = f(+l) - f(-l); acc = a_1 delta_1; acc = acc + a_l delta_l; d = acc * metric;
// div = (u_x + v_y) + w_z; s = (((div^2 + ox^2) + oy^2) + oz^2) + eps_s; theta = max(-div/sqrt(s), 0).
// The face ghosts of div / mask are filled by scalar_ghost_kernel right after.
// HBM: 24 B read + 8 B (div) + 1 B (mask) write per node.
// ---------------------------------------------------------------------------------------------
template <int L>
__device__ __forceinline__ double ddc(const DevP& P, const double* __restrict__ f, long long n, long long s, double metric) {
  double acc = P.a1[0] * (f[n + s] - f[n - s]);
#pragma unroll
  for (int l = 2; l <= L; ++l) acc = acc + P.a1[l - 1] * (f[n + l * s] - f[n - l * s]);
  return acc * metric;
}

// Face ghosts of the nodal scalars div and mask (S6): periodic wrap, else constant extrapolation of the
// nearest interior value.  One thread per face-ghost node (edges and corners are never read: every
// consumer is a star stencil).  Segments of the flat index: x faces, y faces, z faces.
template <bool MASK>
__global__ void __launch_bounds__(256) scalar_ghost_kernel(const DevP P) {
  const int g = P.ng;
  const long long nX = 2LL * g * P.ny * P.nz, nY = 2LL * g * P.nx * P.nz, nZ = 2LL * g * P.nx * P.ny;
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int i, j, k, is, js, ks;
  if (t < nX) {
    const int m = (int)(t % (2 * g));
    const long long t2 = t / (2 * g);
    j = js = (int)(t2 % P.ny); k = ks = (int)(t2 / P.ny);
    i = m < g ? m - g : P.nx + (m - g);
    is = P.bc_x == BC_PERIODIC ? (i < 0 ? i + P.nx : i - P.nx) : (i < 0 ? 0 : P.nx - 1);
  } else if ((t -= nX) < nY) {
    i = is = (int)(t % P.nx);
    const long long t2 = t / P.nx;
    const int m = (int)(t2 % (2 * g));
    k = ks = (int)(t2 / (2 * g));
    j = m < g ? m - g : P.ny + (m - g);
    if (j < 0) js = P.bc_y_lo == BC_PERIODIC ? j + P.ny : 0;
    else js = P.bc_y_hi == BC_PERIODIC ? j - P.ny : P.ny - 1;
  } else if ((t -= nY) < nZ) {
    i = is = (int)(t % P.nx);
    const long long t2 = t / P.nx;
    j = js = (int)(t2 % P.ny);
    const int m = (int)(t2 / P.ny);
    k = m < g ? m - g : P.nz + (m - g);
    ks = P.bc_z == BC_PERIODIC ? (k < 0 ? k + P.nz : k - P.nz) : (k < 0 ? 0 : P.nz - 1);
  } else {
    return;
  }
  const long long n = pidx(P, i, j, k), ns = pidx(P, is, js, ks);
  P.div[n] = P.div[ns];
  if (MASK) P.mask[n] = P.mask[ns];
}

template <int L, bool MASK, bool THETA>
__global__ void __launch_bounds__(256) sensor_kernel(const DevP P) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  if (i >= P.nx || j >= P.ny) return;
  const long long n = pidx(P, i, j, k);
  const double* __restrict__ u = P.q + Q_U * P.fs;
  const double* __restrict__ v = P.q + Q_V * P.fs;
  const double* __restrict__ w = P.q + Q_W * P.fs;
  const double my = P.eta_y_c[j];
  const double ux = ddc<L>(P, u, n, 1, P.inv_dx), uy = ddc<L>(P, u, n, P.sy, my), uz = ddc<L>(P, u, n, P.sz, P.inv_dz);
  const double vx = ddc<L>(P, v, n, 1, P.inv_dx), vy = ddc<L>(P, v, n, P.sy, my), vz = ddc<L>(P, v, n, P.sz, P.inv_dz);
  const double wx = ddc<L>(P, w, n, 1, P.inv_dx), wy = ddc<L>(P, w, n, P.sy, my), wz = ddc<L>(P, w, n, P.sz, P.inv_dz);
  const double dv = (ux + vy) + wz;
  P.div[n] = dv;
  if (MASK || THETA) {
    const double ox = wy - vz, oy = uz - wx, oz = vx - uy;
    const double s = (((dv * dv + ox * ox) + oy * oy) + oz * oz) + P.eps_s;
    double th = -dv / sqrt(s);
    if (!(th > 0.0)) th = 0.0;
    if (THETA) P.theta[iidx(P, i, j, k)] = th;
    if (MASK) {
      const unsigned char m = (th > P.thr) ? 1 : 0;
      P.mask[n] = m;
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Interface flags (O2 / S5): interface n+1/2 along d uses WENO iff any node of its 2r-node
// stencil {n-r+1..n+r} is flagged.  Per interior node the six adjacent interfaces are packed in a
// byte (bit 2d: minus side, bit 2d+1: plus side).  Three kinds of work lists are built from it:
//   list      nodes with any bit set (consumed by rhs_apply_kernel),
//   ilist[d]  flagged interfaces of direction d, each named by the padded index of its left node and
//             owned by exactly one thread: the node on its left, or - for the interface below the first
//             node of a pencil - that first node (consumed by weno_kernel).
// Appends are aggregated per block (one atomic per list per block); the order inside a list is
// irrelevant, every entry is processed independently and writes its own slot.
// ---------------------------------------------------------------------------------------------
template <int R>
__global__ void __launch_bounds__(256) flags_kernel(const DevP P) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  const bool in = (i < P.nx && j < P.ny);
  unsigned f = 0, own = 0;
  long long o = 0, n = 0;
  const long long st[3] = {1, P.sy, P.sz};
  if (in) {
    n = pidx(P, i, j, k);
    o = iidx(P, i, j, k);
    own = P.mask[n];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      unsigned mid = 0;
#pragma unroll
      for (int m = -R + 1; m <= R - 1; ++m) mid |= P.mask[n + m * st[d]];
      const unsigned lo = mid | P.mask[n - R * st[d]];
      const unsigned hi = mid | P.mask[n + R * st[d]];
      f |= (lo ? 1u : 0u) << (2 * d);
      f |= (hi ? 1u : 0u) << (2 * d + 1);
    }
    P.nflag[o] = (unsigned char)f;
  }
  // categories: 0 node list; 1..3 plus-side interface of x, y, z; 4..6 minus-side interface of the first
  // node of a pencil in x, y, z; 7 flagged nodes (count only)
  const bool want[8] = {f != 0, (f & 2u) != 0, (f & 8u) != 0, (f & 32u) != 0,
                        i == 0 && (f & 1u) != 0, j == 0 && (f & 4u) != 0, k == 0 && (f & 16u) != 0, own != 0};
  __shared__ int s_cnt[8][8];
  __shared__ int s_base[8];
  const int tid = threadIdx.y * blockDim.x + threadIdx.x;
  const int lane = tid & 31, wid = tid >> 5;
  unsigned bal[8];
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    bal[c] = __ballot_sync(0xffffffffu, want[c]);
    if (lane == 0) s_cnt[c][wid] = __popc(bal[c]);
  }
  __syncthreads();
  if (tid < 8) {
    int tot = 0;
    for (int w = 0; w < 8; ++w) { const int c = s_cnt[tid][w]; s_cnt[tid][w] = tot; tot += c; }
    int base = 0;
    if (tot) {
      unsigned long long* cum = reinterpret_cast<unsigned long long*>(P.counters + C_TOTALS);
      const int d = (tid - 1) % 3;
      if (tid == 0) { base = atomicAdd(&P.counters[C_NSHOCK], tot); atomicAdd(&cum[0], (unsigned long long)tot); }
      else if (tid == 7) { atomicAdd(&P.counters[C_NFLAGGED], tot); atomicAdd(&cum[1], (unsigned long long)tot); }
      else { base = atomicAdd(&P.counters[C_NIFACE + d], tot); atomicAdd(&cum[3 + d], (unsigned long long)tot); }
    }
    s_base[tid] = base;
  }
  __syncthreads();
  const unsigned lt = (1u << lane) - 1u;
  if (want[0]) P.list[s_base[0] + s_cnt[0][wid] + __popc(bal[0] & lt)] = (int)o;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (want[1 + d]) P.ilist[d][s_base[1 + d] + s_cnt[1 + d][wid] + __popc(bal[1 + d] & lt)] = (int)n;
    if (want[4 + d]) P.ilist[d][s_base[4 + d] + s_cnt[4 + d][wid] + __popc(bal[4 + d] & lt)] = (int)(n - st[d]);
  }
}

// ---------------------------------------------------------------------------------------------
// a9: time-step reduction (O5 / S13): max over interior nodes and directions of
// (|u_d| + c) m_d, nu m_d^2, gamma nu m_d^2 / Pr.  Warp-shuffle max on the bit patterns (rates are
// non-negative, so unsigned order = numeric order, and a NaN wins and is detected), one atomicMax
// per block.  HBM: ~56 B read per node.
// ---------------------------------------------------------------------------------------------
template <bool VISC>
__global__ void __launch_bounds__(256) dt_kernel(const DevP P) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  double rmax = 0.0;
  if (i < P.nx && j < P.ny) {
    const long long n = pidx(P, i, j, k);
    const double rho = P.q[Q_RHO * P.fs + n];
    const double pp = P.q[Q_P * P.fs + n];
    const double c = sqrt(P.gamma * pp / rho);
    const double md[3] = {P.inv_dx, P.eta_y_c[j], P.inv_dz};
    const double vel[3] = {P.q[Q_U * P.fs + n], P.q[Q_V * P.fs + n], P.q[Q_W * P.fs + n]};
    double nu = 0.0;
    if (VISC) nu = P.q[Q_MU * P.fs + n] / rho;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      rmax = fmax(rmax, (fabs(vel[d]) + c) * md[d]);
      if (VISC) {
        rmax = fmax(rmax, nu * (md[d] * md[d]));
        rmax = fmax(rmax, (P.gamma * nu / P.prandtl) * (md[d] * md[d]));
      }
    }
    if (!(rmax == rmax) || !(c == c)) rmax = __longlong_as_double(0x7ff8000000000000LL);
  }
  unsigned long long bits = (unsigned long long)__double_as_longlong(rmax);
#pragma unroll
  for (int s = 16; s > 0; s >>= 1) {
    const unsigned long long o = __shfl_xor_sync(0xffffffffu, bits, s);
    bits = o > bits ? o : bits;
  }
  __shared__ unsigned long long sm[8];
  const int tid = threadIdx.y * blockDim.x + threadIdx.x;
  if ((tid & 31) == 0) sm[tid >> 5] = bits;
  __syncthreads();
  if (tid < 32) {
    bits = tid < (int)((blockDim.x * blockDim.y + 31) >> 5) ? sm[tid] : 0ull;
#pragma unroll
    for (int s = 4; s > 0; s >>= 1) {
      const unsigned long long o = __shfl_xor_sync(0xffffffffu, bits, s);
      bits = o > bits ? o : bits;
    }
    if (tid == 0) atomicMax(reinterpret_cast<unsigned long long*>(P.scal + S_RATE), bits);
  }
}

__global__ void dt_finalize_kernel(const DevP P, double dt_fixed) {
  const double rate = P.scal[S_RATE];
  const double dt = dt_fixed > 0.0 ? dt_fixed : P.cfl / rate;
  P.scal[S_DT] = dt;
  P.scal[S_RATE] = 0.0;
  if (!isfinite(dt)) P.scal[S_NAN] = 1.0;
}

__global__ void step_end_kernel(const DevP P) {
  P.scal[S_TIME] = P.scal[S_TIME] + P.scal[S_DT];
  P.scal[S_NSTEP] = P.scal[S_NSTEP] + 1.0;
}

__global__ void reset_counters_kernel(const DevP P) {
  P.counters[C_NSHOCK] = 0;
  P.counters[C_NFLAGGED] = 0;
  P.counters[C_NIFACE] = 0; P.counters[C_NIFACE + 1] = 0; P.counters[C_NIFACE + 2] = 0;
  reinterpret_cast<unsigned long long*>(P.counters + C_TOTALS)[2] += 1ull;   // sensor evaluations since set_fields
}

// -------------------------------------------------------------------------- launch wrappers
static inline dim3 grid2d(const DevP& P, dim3 b) { return dim3((P.nx + b.x - 1) / b.x, (P.ny + b.y - 1) / b.y, P.nz); }

int launch_fill_prim(const DevP& P, cudaStream_t st) {
  dim3 b(128), g((P.px + 127) / 128, P.py, P.pz);
  const bool visc = P.visc_law != VISC_NONE, sc = P.flux_mode != FLUX_CENTRAL;
  if (visc && sc) fill_prim_kernel<true, true><<<g, b, 0, st>>>(P);
  else if (visc) fill_prim_kernel<true, false><<<g, b, 0, st>>>(P);
  else if (sc) fill_prim_kernel<false, true><<<g, b, 0, st>>>(P);
  else fill_prim_kernel<false, false><<<g, b, 0, st>>>(P);
  return 1;
}

template <int L>
static int launch_sensor_L(const DevP& P, bool mask, bool theta, cudaStream_t st) {
  dim3 b(64, 4), g = grid2d(P, b);
  if (theta) sensor_kernel<L, true, true><<<g, b, 0, st>>>(P);
  else if (mask) sensor_kernel<L, true, false><<<g, b, 0, st>>>(P);
  else sensor_kernel<L, false, false><<<g, b, 0, st>>>(P);
  const long long ghosts = 2LL * P.ng * ((long long)P.ny * P.nz + (long long)P.nx * P.nz + (long long)P.nx * P.ny);
  dim3 gg((unsigned)((ghosts + 255) / 256));
  if (mask || theta) scalar_ghost_kernel<true><<<gg, 256, 0, st>>>(P);
  else scalar_ghost_kernel<false><<<gg, 256, 0, st>>>(P);
  return 2;
}
int launch_sensor(const DevP& P, int L, bool mask, bool theta, cudaStream_t st) {
  switch (L) {
    case 1: return launch_sensor_L<1>(P, mask, theta, st);
    case 2: return launch_sensor_L<2>(P, mask, theta, st);
    case 3: return launch_sensor_L<3>(P, mask, theta, st);
    default: return launch_sensor_L<4>(P, mask, theta, st);
  }
}

int launch_flags(const DevP& P, int r, cudaStream_t st) {
  dim3 b(64, 4), g = grid2d(P, b);
  reset_counters_kernel<<<1, 1, 0, st>>>(P);
  switch (r) {
    case 1: flags_kernel<1><<<g, b, 0, st>>>(P); break;
    case 2: flags_kernel<2><<<g, b, 0, st>>>(P); break;
    case 3: flags_kernel<3><<<g, b, 0, st>>>(P); break;
    default: flags_kernel<4><<<g, b, 0, st>>>(P); break;
  }
  return 2;
}

int launch_dt(const DevP& P, double dt_fixed, cudaStream_t st) {
  int n = 0;
  if (!(dt_fixed > 0.0)) {
    dim3 b(64, 4), g = grid2d(P, b);
    if (P.visc_law != VISC_NONE) dt_kernel<true><<<g, b, 0, st>>>(P);
    else dt_kernel<false><<<g, b, 0, st>>>(P);
    ++n;
  }
  dt_finalize_kernel<<<1, 1, 0, st>>>(P, dt_fixed);
  return n + 1;
}

int launch_step_end(const DevP& P, cudaStream_t st) {
  step_end_kernel<<<1, 1, 0, st>>>(P);
  return 1;
}

}  // namespace streams
