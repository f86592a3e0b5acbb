// Kernels whose arithmetic decides an integer (the shock-sensor mask): sensor/mask, interface flags and work lists;
// plus the one-thread step scalars, the fixed-order sum reductions and the fp64 probe.
// This translation unit is compiled with -fmad=false so that every operation is a single
// IEEE fp64 operation in source order: the
// mask is then bit-identical to any IEEE evaluation of the same formulas on the same state.
#include "streams_dev.cuh"
#include "streams_launch.h"
#include "streams_tma.cuh"

namespace streams {

// ---------------------------------------------------------------------------------------------
// a3: Ducros-type sensor, node mask and dilatation (O2): sensor_march_kernel below.
// Canonical order: delta_l = f(+l) - f(-l); acc = a_1 delta_1; acc = acc + a_l delta_l; d = acc * metric;
// div = (u_x + v_y) + w_z; s = (((div^2 + ox^2) + oy^2) + oz^2) + eps_s; theta = max(-div/sqrt(s), 0).
// ---------------------------------------------------------------------------------------------
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
  } else if ((t -= nY) < nZ && P.bc_z != BC_HALO) {
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

// ---------------------------------------------------------------------------------------------
// sensor_march_kernel: the same sensor (identical operations in identical order, so identical bits) as a
// z-marching kernel like rhs_march_kernel (streams_march.cu): a block owns a 32 x TY tile and a chunk of z
// planes; the centre plane of (u, v, w) with its halo is one 4-D TMA box per plane (two buffers, issued two
// planes ahead), the z neighbours live in a 7-plane register ring fed by a second TMA box per plane.
// HBM: 24 B read + 8 B (div) + 1 B (mask) write per node; every stencil offset is an immediate.
// ---------------------------------------------------------------------------------------------
constexpr int SKU = 2;            // planes per iteration of sensor_march_kernel
template <int TY, int NG>
struct SensorSmem {
  using G = MarchGeom<TY, NG>;
  static constexpr size_t BUF = (size_t)3 * SKU * G::PLANE * 8, RING = (size_t)3 * SKU * G::NT * 8;
  static constexpr size_t OFF_RING = 2 * BUF, OFF_BAR = OFF_RING + 2 * RING, TOTAL = OFF_BAR + 64;
  static_assert(BUF % 128 == 0 && RING % 128 == 0, "TMA destinations are 128-byte aligned");
};

// acc = a_1 d_1; acc = acc + a_l d_l; derivative = acc * metric (canonical order), G(o) = value at offset o
template <int L, class G>
__device__ __forceinline__ double ddc_g(const DevP& P, const G& g, double metric) {
  double acc = P.a1[0] * (g(1) - g(-1));
#pragma unroll
  for (int l = 2; l <= L; ++l) acc = acc + P.a1[l - 1] * (g(l) - g(-l));
  return acc * metric;
}

#ifndef STREAMS_SENSOR_MINB
#define STREAMS_SENSOR_MINB 2
#endif
// An iteration handles the SKU = 2 planes k, k + 1 of the tile: the boxes are two planes deep, the ring holds
// 2 NG + 2 planes (k - NG .. k + NG + 1) and shifts by two, so the register moves of the shift, the barrier, the
// mbarrier waits and the loop bookkeeping are paid once per two nodes, and the two nodes' derivative chains interleave.
template <int L, bool MASK, bool THETA, int TY, int NG>
__global__ void __launch_bounds__(MTX * TY, STREAMS_SENSOR_MINB)
sensor_march_kernel(const __grid_constant__ CUtensorMap tm_centre, const __grid_constant__ CUtensorMap tm_ring, const DevP P,
                    int nbx, int nby, int kz) {
  using G = MarchGeom<TY, NG>;             // NG = DevP::ng: ghost width / ring depth of the layout
  using SM = SensorSmem<TY, NG>;
  static_assert(L <= NG, "ring depth");
  constexpr int NR = 2 * NG + SKU;         // ring planes
  extern __shared__ __align__(128) unsigned char smem_raw[];
  double* const buf = reinterpret_cast<double*>(smem_raw);                  // [2][3][SKU][PLANE]
  double* const ring = reinterpret_cast<double*>(smem_raw + SM::OFF_RING);  // [2][3][SKU][NT]
  unsigned long long* const full_c = reinterpret_cast<unsigned long long*>(smem_raw + SM::OFF_BAR);
  unsigned long long* const full_r = full_c + 2;

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
  const int ncol = (int)pidx(P, ic, jc, 0);
  const int s0 = (ty + NG) * G::ROW + tx + 4;
  const int cx0 = i0 + P.ox, cy0 = j0 + NG;

  // (planes beyond the padded box -- the second plane of an odd tail, the ring planes of the last iterations -- are
  // filled with zeros by the TMA unit and never used)
  auto issue_centre = [&](int k, int b) {            // planes k, k + 1
    mbar_expect_tx(&full_c[b], (unsigned)SM::BUF);
    tma_load_4d(buf + (size_t)b * 3 * SKU * G::PLANE, &tm_centre, &full_c[b], cx0 - 4, cy0 - NG, k + NG, 0);
  };
  auto issue_ring = [&](int k, int b) {              // ring planes k + NG + 2, k + NG + 3 into slot b
    mbar_expect_tx(&full_r[b], (unsigned)SM::RING);
    tma_load_4d(ring + (size_t)b * 3 * SKU * G::NT, &tm_ring, &full_r[b], cx0, cy0, k + NG + SKU + NG, 0);
  };
  if (MASK && tid == 0 && blockIdx.x == 0 && P.flux_mode == FLUX_HYBRID) {
    // per-evaluation counters of flags_kernel (which runs after this kernel; their last readers ran before it)
    P.counters[C_NSHOCK] = 0;
    P.counters[C_NFLAGGED] = 0;
    P.counters[C_NIFACE] = 0; P.counters[C_NIFACE + 1] = 0; P.counters[C_NIFACE + 2] = 0; P.counters[C_NIFACE + 3] = 0;
    reinterpret_cast<unsigned long long*>(P.counters + C_TOTALS)[2] += 1ull;   // sensor evaluations since set_fields
  }
  if (tid == 0) {
    mbar_init(&full_c[0], 1); mbar_init(&full_c[1], 1);
    mbar_init(&full_r[0], 1); mbar_init(&full_r[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) {
    issue_centre(kb, 0);
    if (kb + SKU < ke) issue_centre(kb + SKU, 1);
    issue_ring(kb, 0);
  }
  const double my = P.eta_y_c[min(j, P.ny - 1)];
  double zr[3][NR];                                   // planes kb - NG .. kb + NG + 1 (the last one clamped into the box)
#pragma unroll
  for (int f = 0; f < 3; ++f) {
    const double* __restrict__ fp = P.q + (long long)f * P.fs + ncol;
#pragma unroll
    for (int m = 0; m < NR; ++m) zr[f][m] = fp[(long long)(min(kb + m, P.pz - 1) - NG) * P.sz];
  }

  // this thread's column in the outputs, advanced plane by plane
  double* __restrict__ div_p = P.div + ncol + (long long)kb * isz;
  unsigned char* __restrict__ mask_p = P.mask + ncol + (long long)kb * isz;
  const unsigned char* __restrict__ ovr_p = P.mask_ovr ? P.mask_ovr + ncol : nullptr;
  // does this thread own x / y face ghosts (DevP::sown: the kernel writes them itself)?
  const bool per_z = P.bc_z == BC_PERIODIC;
  const bool zface = P.sown != 0 && P.bc_z != BC_HALO;    // (halo planes in z come from the neighbouring slab)
  const bool gplan = P.sown && active &&
                     ((P.bc_x == BC_PERIODIC ? (i < NG || i >= P.nx - NG) : (i == 0 || i == P.nx - 1)) ||
                      (j < NG && P.bc_y_lo == BC_PERIODIC) || (j >= P.ny - NG && P.bc_y_hi == BC_PERIODIC) ||
                      (j == 0 && P.bc_y_lo != BC_PERIODIC) || (j == P.ny - 1 && P.bc_y_hi != BC_PERIODIC));

  for (int k = kb, it = 0; k < ke; k += SKU, ++it) {
    const int b = it & 1;
    const unsigned par = (unsigned)(it >> 1) & 1u;
    mbar_wait(&full_c[b], par);
    const double* __restrict__ sc = buf + (size_t)b * 3 * SKU * G::PLANE + s0;
    double gx[SKU][3], gy[SKU][3], gz[SKU][3];
#pragma unroll
    for (int z = 0; z < SKU; ++z) {
#pragma unroll
      for (int f = 0; f < 3; ++f) {
        gx[z][f] = ddc_g<L>(P, [&](int o) { return sc[(f * SKU + z) * G::PLANE + o]; }, P.inv_dx);
        gy[z][f] = ddc_g<L>(P, [&](int o) { return sc[(f * SKU + z) * G::PLANE + o * G::ROW]; }, my);
        gz[z][f] = ddc_g<L>(P, [&](int o) { return zr[f][NG + z + o]; }, P.inv_dz);
      }
    }
    if (tid >> 5) {
      if (b) asm volatile("bar.arrive 2, %0;" ::"n"(G::NT) : "memory");
      else asm volatile("bar.arrive 1, %0;" ::"n"(G::NT) : "memory");
    } else {
      if (b) asm volatile("bar.sync 2, %0;" ::"n"(G::NT) : "memory");
      else asm volatile("bar.sync 1, %0;" ::"n"(G::NT) : "memory");
      if (tid == 0) {
        if (k + SKU < ke) issue_ring(k + SKU, b ^ 1);     // needed first
        if (k + 2 * SKU < ke) issue_centre(k + 2 * SKU, b);
      }
    }
#pragma unroll
    for (int z = 0; z < SKU; ++z) {
      const int kk = k + z;
      const double dv = (gx[z][0] + gy[z][1]) + gz[z][2];
      if (active && (z == 0 || kk < ke)) {
        div_p[z * isz] = dv;
        unsigned char mk = 0;
        if (MASK || THETA) {
          const double ox = gy[z][2] - gz[z][1], oy = gz[z][0] - gx[z][2], oz = gx[z][1] - gy[z][0];
          const double s = (((dv * dv + ox * ox) + oy * oy) + oz * oz) + P.eps_s;
          // mask = theta > thr with theta = max(-dv / sqrt(s), 0).  Without the theta output the decision is taken on
          // the squares wherever it is clear by a margin far above the rounding of either form (1e-12 relative, the
          // quotient is good to 2 ulp); only a node within that margin of the threshold evaluates the square root and
          // the division -- the same operations as the definition, so the mask carries the bits of the definition.
          const double a = -dv, a2 = a * a, t2 = P.thr2 * s;
          bool clear_hi = a > 0.0 && a2 > t2 * (1.0 + 1e-12), clear_lo = !(a > 0.0) || a2 < t2 * (1.0 - 1e-12);
          if (P.thr < 0.0) { clear_hi = true; clear_lo = false; }       // theta >= 0 > thr at every node
          if (a != a) { clear_hi = false; clear_lo = true; }              // NaN: theta = 0, not above a threshold >= 0
          if (THETA || !(clear_hi || clear_lo)) {
            double th = -dv / sqrt(s);
            if (!(th > 0.0)) th = 0.0;
            if (THETA) P.theta[iidx(P, i, j, kk)] = th;
            mk = (th > P.thr) ? 1 : 0;
          } else {
            mk = clear_hi ? 1 : 0;
          }
          if (MASK && ovr_p) mk = ovr_p[(long long)kk * isz];   // imposed mask (activation sweeps)
          if (MASK) mask_p[z * isz] = mk;
        }
        // face ghosts of div / mask (S6), written by the node they copy: its periodic image, or the NG ghost nodes
        // beyond a non-periodic face (constant extrapolation).  Which x / y ghosts a thread owns is fixed along the
        // march (gplan), the z faces are a property of the plane.
        if (gplan | (zface && (per_z ? (kk < NG || kk >= P.nz - NG) : (kk == 0 || kk == P.nz - 1)))) {
          auto put = [&](long long m) { div_p[z * isz + m] = dv; if (MASK) mask_p[z * isz + m] = mk; };
          auto face = [&](int a, int na, bool per, long long st) {      // a: index along the direction, st: its stride
            if (per) {
              if (a < NG) put(na * st);
              else if (a >= na - NG) put(-na * st);
            } else {
              if (a == 0) { for (int m = 1; m <= NG; ++m) put(-m * st); }
              if (a == na - 1) { for (int m = 1; m <= NG; ++m) put(m * st); }
            }
          };
          face(i, P.nx, P.bc_x == BC_PERIODIC, 1);
          if (j < NG || j >= P.ny - NG) {
            if (j < NG && P.bc_y_lo == BC_PERIODIC) put(P.ny * P.sy);
            if (j >= P.ny - NG && P.bc_y_hi == BC_PERIODIC) put(-P.ny * P.sy);
            if (j == 0 && P.bc_y_lo != BC_PERIODIC) { for (int m = 1; m <= NG; ++m) put(-m * P.sy); }
            if (j == P.ny - 1 && P.bc_y_hi != BC_PERIODIC) { for (int m = 1; m <= NG; ++m) put(m * P.sy); }
          }
          if (P.bc_z != BC_HALO) face(kk, P.nz, per_z, P.sz);     // halo planes belong to the caller's exchange (streams.h)
        }
      }
    }
    div_p += SKU * isz;
    mask_p += SKU * isz;
    mbar_wait(&full_r[b], par);
    const double* __restrict__ rn = ring + (size_t)b * 3 * SKU * G::NT + tid;
    // (register moves: renaming the ring through a phase switch measured slower, here and in rhs_march_kernel)
#pragma unroll
    for (int f = 0; f < 3; ++f) {
#pragma unroll
      for (int m = 0; m < 2 * NG; ++m) zr[f][m] = zr[f][m + SKU];
#pragma unroll
      for (int z = 0; z < SKU; ++z) zr[f][2 * NG + z] = rn[(f * SKU + z) * G::NT];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Interface flags (O2 / S5): interface n+1/2 along d uses WENO iff any node of its 2r-node
// stencil {n-r+1..n+r} is flagged.  Per interior node the six adjacent interfaces are packed in a byte
// (bit 2d: minus side, bit 2d+1: plus side), stored at the node's padded index.
// One thread handles 8 consecutive x nodes as one 64-bit word of 0/1 mask bytes: the y / z windows are
// ORs of 64-bit loads, the x window is an OR of byte-shifted words (SWAR), so the whole kernel is ~15
// 8-byte loads per 8 nodes and no per-node atomics.  It also counts, per evaluation, flagged nodes,
// nodes next to a flagged interface and flagged interfaces per direction (the paper's "WENO
// activation"): warp-shuffle sums, one atomic per counter per block.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long ldw(const unsigned char* p) {
  return *reinterpret_cast<const unsigned long long*>(p);
}
// bytes of `cur` shifted so that byte b holds the mask of node b + m (|m| < 8); prev / next are the
// neighbouring words along x
__device__ __forceinline__ unsigned long long xshift(unsigned long long prev, unsigned long long cur,
                                                     unsigned long long next, int m) {
  if (m == 0) return cur;
  if (m > 0) return (cur >> (8 * m)) | (next << (64 - 8 * m));
  return (cur << (-8 * m)) | (prev >> (64 + 8 * m));
}

#ifndef STREAMS_FLAGS_MINB
#define STREAMS_FLAGS_MINB 8
#endif
template <int R>
__global__ void __launch_bounds__(256, STREAMS_FLAGS_MINB) flags_kernel(const DevP P, int nwx) {
  // one block row per plane (blockIdx.y = k): a thread finds its word of the plane with one 32-bit division
  const unsigned t = blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned nwords = (unsigned)nwx * (unsigned)P.ny;             // words of a plane
  int cnt[6] = {0, 0, 0, 0, 0, 0};   // flagged nodes, shock nodes, interfaces x, y, z, nodes next to a flagged interface
  unsigned long long hiw[4] = {0ull, 0ull, 0ull, 0ull}, first[4] = {0ull, 0ull, 0ull, 0ull};   // flagged interfaces named by their
  int n0w = 0;                                                                    // left node: plus sides, pencil starts
  if (t < nwords) {
    const int j = (int)(t / (unsigned)nwx), iw = (int)(t - (unsigned)j * (unsigned)nwx), k = (int)blockIdx.y;
    const int i0 = iw * 8;
    const long long n0 = pidx(P, i0, j, k);
    const unsigned char* m = P.mask + n0;
    const int nvalid = min(8, P.nx - i0);
    const unsigned long long valid = nvalid == 8 ? ~0ull : ((1ull << (8 * nvalid)) - 1ull);
    const unsigned long long cur = ldw(m), prev = ldw(m - 8);
    const unsigned long long next = (i0 + 8 < P.nx + P.ng) ? ldw(m + 8) : 0ull;
    unsigned long long lo[3], hi[3];
    {
      unsigned long long mid = cur;
#pragma unroll
      for (int q = 1; q <= R - 1; ++q) mid |= xshift(prev, cur, next, q) | xshift(prev, cur, next, -q);
      lo[0] = mid | xshift(prev, cur, next, -R);
      hi[0] = mid | xshift(prev, cur, next, R);
    }
    const long long st[3] = {1, P.sy, P.sz};
#pragma unroll
    for (int d = 1; d < 3; ++d) {
      unsigned long long mid = cur;
#pragma unroll
      for (int q = 1; q <= R - 1; ++q) mid |= ldw(m + q * st[d]) | ldw(m - q * st[d]);
      lo[d] = mid | ldw(m - R * st[d]);
      hi[d] = mid | ldw(m + R * st[d]);
    }
    unsigned long long nf = 0ull, any = 0ull;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      lo[d] &= valid & 0x0101010101010101ull;
      hi[d] &= valid & 0x0101010101010101ull;
      nf |= (lo[d] << (2 * d)) | (hi[d] << (2 * d + 1));
      any |= lo[d] | hi[d];
    }
    *reinterpret_cast<unsigned long long*>(P.nflag + n0) = nf;
    cnt[0] = __popcll(cur & valid & 0x0101010101010101ull);
    cnt[1] = __popcll(any);
    // every interface is counted by its left node; the one below the first node of a pencil by that node
    n0w = (int)n0;
    first[0] = i0 == 0 ? (lo[0] & 1ull) : 0ull;
    first[1] = j == 0 ? lo[1] : 0ull;
    first[2] = k == 0 ? lo[2] : 0ull;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      hiw[d] = hi[d];
      cnt[2 + d] = __popcll(hi[d]) + __popcll(first[d]);
    }
    hiw[3] = any;                                    // list 3: the nodes that receive a net correction (corr_gather_kernel)
    cnt[5] = cnt[1];
  }
  // counters 0, 1: warp-shuffle sums, one atomic per block
  __shared__ int s_cnt[2];
  __shared__ int s_wsum[4][8], s_base[4];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (threadIdx.x < 2) s_cnt[threadIdx.x] = 0;
  // most blocks see no flagged node at all: nothing to count or to append (the barrier also publishes s_cnt)
  if (!__syncthreads_or(cnt[0] | cnt[1])) return;
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    int v = cnt[c];
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) v += __shfl_xor_sync(0xffffffffu, v, s);
    if (lane == 0 && v) atomicAdd(&s_cnt[c], v);
  }
  // flagged interfaces: exclusive scan over the block, one atomic per direction per block reserves the
  // block's range of the direction's work list (DevP::ilist), every thread writes its own entries
  int off[4];
#pragma unroll
  for (int d = 0; d < 4; ++d) {
    int v = cnt[2 + d];
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
      const int t2 = __shfl_up_sync(0xffffffffu, v, s);
      if (lane >= s) v += t2;
    }
    if (lane == 31) s_wsum[d][wid] = v;
    off[d] = v - cnt[2 + d];
  }
  __syncthreads();
  if (threadIdx.x < 4) {
    const int d = threadIdx.x;
    int run = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) { const int t2 = s_wsum[d][w]; s_wsum[d][w] = run; run += t2; }
    int base = 0;
    if (run) {
      base = atomicAdd(&P.counters[C_NIFACE + d], run);
      if (d < 3) atomicAdd(&reinterpret_cast<unsigned long long*>(P.counters + C_TOTALS)[3 + d], (unsigned long long)run);
    }
    s_base[d] = base;
  } else if (threadIdx.x >= 32 && threadIdx.x < 34 && s_cnt[threadIdx.x - 32]) {
    // counters: C_NFLAGGED, C_NSHOCK; totals: [0] shock, [1] flagged
    const int c = threadIdx.x - 32, v = s_cnt[c];
    atomicAdd(&P.counters[c == 0 ? C_NFLAGGED : C_NSHOCK], v);
    atomicAdd(&reinterpret_cast<unsigned long long*>(P.counters + C_TOTALS)[c == 0 ? 1 : 0], (unsigned long long)v);
  }
  __syncthreads();
  if (t < nwords) {
#pragma unroll
    for (int d = 0; d < 4; ++d) {
      if (cnt[2 + d] == 0) continue;
      int* __restrict__ Lst = P.ilist + (long long)d * P.lcap + s_base[d] + s_wsum[d][wid] + off[d];
      unsigned long long wl = first[d], wh = hiw[d];
      const int nl = n0w - (int)(d == 0 ? 1 : (d == 1 ? P.sy : P.sz));
      while (wl) { *Lst++ = nl + ((__ffsll((long long)wl) - 1) >> 3); wl &= wl - 1; }
      while (wh) { *Lst++ = n0w + ((__ffsll((long long)wh) - 1) >> 3); wh &= wh - 1; }
    }
  }
}

// Step scalars, one thread at the start of every step.  recompute: a9, second half: dt = CFL / (the rate reduced by
// fill_prim_kernel<.., DT> or by the last stage's RHS epilogue), or the fixed step.  Always: the time and the step count
// the step will have reached when its three stages are done (read by streams_step after them).
__global__ void dt_finalize_kernel(const DevP P, double dt_fixed, int recompute) {
  if (recompute) {
    const double rate = P.scal[S_RATE];
    const double dt = dt_fixed > 0.0 ? dt_fixed : P.cfl / rate;
    P.scal[S_DT] = dt;
    P.scal[S_RATE] = 0.0;
    if (!isfinite(dt)) P.scal[S_NAN] = 1.0;
  }
  P.scal[S_TIME] = P.scal[S_TIME] + P.scal[S_DT];
  P.scal[S_NSTEP] = P.scal[S_NSTEP] + 1.0;
}

// ---------------------------------------------------------------------------------------------
// fp64 pipe probe (streams_measure_fp64): 16 independent chains per thread, ITERS trips; KIND 0 chains are
// x = fma(x, a, b), KIND 1 alternate x = x + b and x = x * a (this unit is built without contraction, so they
// stay separate instructions).  The result is stored so that nothing is optimised away.
// ---------------------------------------------------------------------------------------------
template <int KIND>
__global__ void __launch_bounds__(256) fp64_probe_kernel(double* out, double a, double b, int iters) {
  double x[16];
#pragma unroll
  for (int c = 0; c < 16; ++c) x[c] = 1.0 + 1e-3 * (threadIdx.x + 16 * c);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int c = 0; c < 16; ++c) {
      if (KIND == 0) x[c] = fma(x[c], a, b);
      else { x[c] = x[c] + b; x[c] = x[c] * a; }
    }
  }
  double s = 0.0;
#pragma unroll
  for (int c = 0; c < 16; ++c) s += x[c];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// Returns thread-level fp64 instructions per second (best of `repeats`), or a negative value on a CUDA error.
// scratch: caller's device buffer of measure_fp64_scratch_bytes() (the library allocates no device memory).
size_t measure_fp64_scratch_bytes() {
  int dev = 0, nsm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return 0;
  return (size_t)nsm * 8 * 256 * sizeof(double);
}
double measure_fp64(cudaStream_t st, int kind, int repeats, double* scratch, size_t scratch_bytes) {
  int dev = 0, nsm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return -1.0;
  const int blocks = nsm * 8, threads = 256, iters = 4096;
  if (!scratch || scratch_bytes < (size_t)blocks * threads * sizeof(double)) return -2.0;
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess) return -1.0;
  if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); return -1.0; }
  double best = -1.0;
  for (int r = 0; r < repeats + 1; ++r) {            // the first launch warms up
    cudaEventRecord(e0, st);
    if (kind == 0) fp64_probe_kernel<0><<<blocks, threads, 0, st>>>(scratch, 0.999999, 1e-6, iters);
    else fp64_probe_kernel<1><<<blocks, threads, 0, st>>>(scratch, 0.999999, 1e-6, iters);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0; break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double inst = (double)blocks * threads * 16.0 * iters * (kind == 0 ? 1.0 : 2.0);
    if (r > 0 && ms > 0.f) best = fmax(best, inst / (ms * 1e-3));
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return cudaGetLastError() == cudaSuccess ? best : -1.0;
}

// ---------------------------------------------------------------------------------------------
// Sum reductions ("compute_residual", Table 2 "forcing term evaluations"): five sums over the interior
// nodes in a FIXED order, so the result is reproducible bit for bit: block b owns the rows b, b + gridDim.x, ... and
// sums them in that order (threads stride the row, shuffle tree, warps in index order), a second one-block launch adds
// the per-block partials in index order.  KIND 0: sum_q of w_q dV with dV = dx dz / eta_y(j) (volume integrals of the
// conserved variables: the discretely conserved quantities); KIND 1: sum of R_q^2 (the paper's residual of the
// right-hand side held in DevP::R).
// ---------------------------------------------------------------------------------------------
constexpr int SUM_BLOCKS = 592, SUM_THREADS = 256;

template <int KIND>
__global__ void __launch_bounds__(SUM_THREADS) sum_partial_kernel(const DevP P, double* __restrict__ partial) {
  double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
  const long long rows = (long long)P.ny * P.nz;
  const double dxdz = 1.0 / (P.inv_dx * P.inv_dz);
  for (long long row = blockIdx.x; row < rows; row += gridDim.x) {
    const int k = (int)(row / P.ny), j = (int)(row - (long long)k * P.ny);
    const double wgt = KIND == 0 ? dxdz / P.eta_y_c[j] : 1.0;
    const long long n0 = pidx(P, 0, j, k);
    for (int i = threadIdx.x; i < P.nx; i += SUM_THREADS) {
#pragma unroll
      for (int q = 0; q < 5; ++q) {
        const double v = (KIND == 0 ? P.w : P.R)[q * P.fs + n0 + i];
        acc[q] += KIND == 0 ? v * wgt : v * v;
      }
    }
  }
  __shared__ double sm[5][SUM_THREADS / 32];
#pragma unroll
  for (int q = 0; q < 5; ++q) {
    double v = acc[q];
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) v += __shfl_xor_sync(0xffffffffu, v, s);
    if ((threadIdx.x & 31) == 0) sm[q][threadIdx.x >> 5] = v;
  }
  __syncthreads();
  if (threadIdx.x < 5) {
    double v = 0.0;
    for (int w = 0; w < SUM_THREADS / 32; ++w) v += sm[threadIdx.x][w];
    partial[threadIdx.x * SUM_BLOCKS + blockIdx.x] = v;
  }
}

__global__ void sum_final_kernel(const double* __restrict__ partial, double* __restrict__ out) {
  if (threadIdx.x < 5) {
    double v = 0.0;
    for (int b = 0; b < SUM_BLOCKS; ++b) v += partial[threadIdx.x * SUM_BLOCKS + b];
    out[threadIdx.x] = v;
  }
}

// S18: bulk-flow controller, one thread after the state sums of a step.  A force g acting for dt changes
// the bulk momentum P = sums[1 + d] by g M dt (M = sums[0]): g <- [g - (P - P_prev) / (M dt)] + (P_target - P) / (M dt).
// init: the first call records P (and takes it as the target when none was given, target = NaN) and leaves g alone.
__global__ void controller_kernel(const DevP P, const double* __restrict__ sums, int d, double target, int init) {
  const double mass = sums[0], mom = sums[1 + d];
  if (init) {
    P.scal[S_PPREV] = mom;
    P.scal[S_PTARGET] = (target != target) ? mom : target;
    return;
  }
  if (target == target) P.scal[S_PTARGET] = target;
  const double dt = P.scal[S_DT];
  const double g_balance = P.scal[S_ACC + d] - (mom - P.scal[S_PPREV]) / (mass * dt);
  P.scal[S_ACC + d] = g_balance + (P.scal[S_PTARGET] - mom) / (mass * dt);
  P.scal[S_PPREV] = mom;
}
int launch_controller(const DevP& P, const double* sums, int d, double target, bool init, cudaStream_t st) {
  controller_kernel<<<1, 1, 0, st>>>(P, sums, d, target, init ? 1 : 0);
  return 1;
}

// partial: 5 * SUM_BLOCKS doubles of scratch, out: 5 doubles (device)
int launch_sums(const DevP& P, int kind, double* partial, double* out, cudaStream_t st) {
  if (kind == 0) sum_partial_kernel<0><<<SUM_BLOCKS, SUM_THREADS, 0, st>>>(P, partial);
  else sum_partial_kernel<1><<<SUM_BLOCKS, SUM_THREADS, 0, st>>>(P, partial);
  sum_final_kernel<<<1, 32, 0, st>>>(partial, out);
  return 2;
}
int sums_scratch_doubles() { return 5 * SUM_BLOCKS + 8; }

// -------------------------------------------------------------------------- launch wrappers
// configure: only opt the instantiation in to its dynamic shared memory on the current device (streams_init).
template <int L, bool MASK, bool THETA, int NG>
static int launch_sensor_march(const DevP& P, const MarchMaps& mp, cudaStream_t st, bool configure) {
  constexpr int TY = STREAMS_SENSOR_TY;
  using SM = SensorSmem<TY, NG>;
  auto kern = sensor_march_kernel<L, MASK, THETA, TY, NG>;
  if (configure)
    return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM::TOTAL) == cudaSuccess ? 0 : -2;
  const int nbx = (P.nx + MTX - 1) / MTX, nby = (P.ny + TY - 1) / TY;
  const int chunks = pick_chunks(nbx * nby, P.nz, P.nsm * STREAMS_SENSOR_MINB);
  const int kz = (P.nz + chunks - 1) / chunks;
  kern<<<(unsigned)(nbx * nby * chunks), MTX * TY, SM::TOTAL, st>>>(mp.s_centre, mp.s_ring, P, nbx, nby, kz);
  if (P.sown) return 1;                              // the kernel wrote the face ghosts itself
  const long long ghosts = 2LL * P.ng * ((long long)P.ny * P.nz + (long long)P.nx * P.nz + (long long)P.nx * P.ny);
  dim3 gg((unsigned)((ghosts + 255) / 256));
  if (MASK) scalar_ghost_kernel<true><<<gg, 256, 0, st>>>(P);
  else scalar_ghost_kernel<false><<<gg, 256, 0, st>>>(P);
  return 2;
}

// L = central_order / 2 on the three-layer layout; the four-layer layout runs the L = 4 instance on the zero-padded
// coefficient table (acc + 0 * delta = acc exactly: the canonical order and its bits are those of order 2L).
// variant: 0 dilatation only, 1 + mask, 2 + mask + theta; bit 2 set = configure all three variants.
int launch_sensor(const DevP& P, const MarchMaps& mp, int L, bool mask, bool theta, cudaStream_t st, bool configure) {
  if (L < 1 || L > P.ng || (P.ng != 3 && P.ng != 4)) return -1;
#define STREAMS_SENSOR(LL, GG)                                                                  \
  do {                                                                                          \
    if (configure) {                                                                            \
      const int a = launch_sensor_march<LL, true, true, GG>(P, mp, st, true);                   \
      const int b = launch_sensor_march<LL, true, false, GG>(P, mp, st, true);                  \
      const int c = launch_sensor_march<LL, false, false, GG>(P, mp, st, true);                 \
      return (a | b | c) ? -2 : 0;                                                              \
    }                                                                                           \
    if (theta) return launch_sensor_march<LL, true, true, GG>(P, mp, st, false);                \
    if (mask) return launch_sensor_march<LL, true, false, GG>(P, mp, st, false);                \
    return launch_sensor_march<LL, false, false, GG>(P, mp, st, false);                         \
  } while (0)
  if (P.ng == 4) STREAMS_SENSOR(4, 4);
  if (L == 1) STREAMS_SENSOR(1, 3);
  if (L == 2) STREAMS_SENSOR(2, 3);
  STREAMS_SENSOR(3, 3);
#undef STREAMS_SENSOR
}

int launch_flags(const DevP& P, int r, cudaStream_t st) {
  const int nwx = (P.nx + 7) / 8;
  const long long nwords = (long long)nwx * P.ny;        // per plane
  dim3 b(256), g((unsigned)((nwords + 255) / 256), (unsigned)P.nz);   // (sensor_march_kernel has reset the per-evaluation counters)
  switch (r) {
    case 1: flags_kernel<1><<<g, b, 0, st>>>(P, nwx); break;
    case 2: flags_kernel<2><<<g, b, 0, st>>>(P, nwx); break;
    case 3: flags_kernel<3><<<g, b, 0, st>>>(P, nwx); break;
    case 4: flags_kernel<4><<<g, b, 0, st>>>(P, nwx); break;
    default: return -1;
  }
  return 1;
}

int launch_dt(const DevP& P, double dt_fixed, bool recompute, cudaStream_t st) {
  dt_finalize_kernel<<<1, 1, 0, st>>>(P, dt_fixed, recompute ? 1 : 0);
  return 1;
}

}  // namespace streams
