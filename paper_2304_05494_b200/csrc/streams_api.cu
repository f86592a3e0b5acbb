// C ABI of libstreams (include/streams.h): context, workspace carving, y metrics, and the host
// driver that sequences the kernels of one RK3 step.  No compute happens on the host.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/streams.h"
#include "streams_dev.cuh"
#include "streams_launch.h"

using namespace streams;

namespace {

thread_local char g_init_error[256] = "";

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Sizes {
  int L, Lv, r, ng, ox, px, py, pz;
  size_t fs;            // doubles per padded field
  size_t N, lcap;
  size_t off_w, off_q, off_q2, off_theta, off_mask, off_movr, off_nflag, off_ilist, off_dF, off_corr, off_counters, off_R,
      off_metrics, off_scal, off_sums, total;
  int nq;
};

void fd1(int L, double* a) {
  const double t[4][4] = {{1.0 / 2.0, 0, 0, 0},
                          {2.0 / 3.0, -1.0 / 12.0, 0, 0},
                          {3.0 / 4.0, -3.0 / 20.0, 1.0 / 60.0, 0},
                          {4.0 / 5.0, -1.0 / 5.0, 4.0 / 105.0, -1.0 / 280.0}};
  for (int l = 0; l < 4; ++l) a[l] = (L >= 1 && L <= 4) ? t[L - 1][l] : 0.0;
}
void fd2(int L, double* b) {
  const double t[4][4] = {{1.0, 0, 0, 0},
                          {4.0 / 3.0, -1.0 / 12.0, 0, 0},
                          {3.0 / 2.0, -3.0 / 20.0, 1.0 / 90.0, 0},
                          {8.0 / 5.0, -1.0 / 5.0, 8.0 / 315.0, -1.0 / 560.0}};
  for (int l = 0; l < 4; ++l) b[l] = (L >= 1 && L <= 4) ? t[L - 1][l] : 0.0;
}

bool valid_bc(int b) { return b == STREAMS_BC_PERIODIC || b == STREAMS_BC_WALL_ISOTHERMAL || b == STREAMS_BC_FREESTREAM; }
bool valid_bc_z(int b) { return valid_bc(b) || b == STREAMS_BC_HALO; }

// Validates the problem and lays out the workspace.  Returns NULL on success, else a message.
const char* plan(const streams_grid* g, const streams_gas* gas, const streams_scheme* sc, Sizes& S) {
  if (!g || !gas || !sc) return "null argument";
  if (g->nx < 1 || g->ny < 1 || g->nz < 1) return "grid extents must be positive";
  if (((long long)g->nx + 48) * ((long long)g->ny + 8) * ((long long)g->nz + 8) > 2000000000LL)
    return "grid too large for 32-bit node indices";
  if (!(g->lx > 0) || !(g->lz > 0)) return "lx, lz must be positive";
  if (!valid_bc(g->bc_x) || !valid_bc(g->bc_y_lo) || !valid_bc(g->bc_y_hi) || !valid_bc_z(g->bc_z)) return "bad bc code";
  if (g->bc_x == STREAMS_BC_WALL_ISOTHERMAL || g->bc_z == STREAMS_BC_WALL_ISOTHERMAL) return "walls are supported in y only";
  if ((g->bc_y_lo == STREAMS_BC_PERIODIC) != (g->bc_y_hi == STREAMS_BC_PERIODIC)) return "y periodic on one side only";
  if (g->bc_y_lo == STREAMS_BC_PERIODIC && !(g->ly > 0)) return "ly must be positive";
  if (g->bc_y_lo != STREAMS_BC_PERIODIC && !(g->y_wall_hi > g->y_wall_lo)) return "y_wall_hi must exceed y_wall_lo";
  if (sc->central_order < 2 || sc->central_order > 8 || sc->central_order % 2) return "central_order must be 2, 4, 6 or 8";
  if (sc->flux_mode < 0 || sc->flux_mode > 2) return "bad flux_mode";
  if (sc->weno_variant != STREAMS_WENO_JS && sc->weno_variant != STREAMS_WENO_Z) return "bad weno_variant";
  if (gas->visc_law < 0 || gas->visc_law > 2) return "bad visc_law";
  if (sc->flux_mode != STREAMS_FLUX_CENTRAL && (sc->weno_order < 1 || sc->weno_order > 7 || sc->weno_order % 2 == 0))
    return "weno_order must be 1, 3, 5 or 7";
  if (gas->visc_law != STREAMS_VISC_NONE && (sc->visc_order < 2 || sc->visc_order > 8 || sc->visc_order % 2))
    return "visc_order must be 2, 4, 6 or 8";
  if (!(gas->gamma > 1) || !(gas->rgas > 0)) return "gamma must exceed 1 and rgas be positive";
  if (gas->visc_law != STREAMS_VISC_NONE && (!(gas->prandtl > 0) || !(gas->t_ref > 0))) return "prandtl, t_ref must be positive";
  if (sc->flux_mode == STREAMS_FLUX_HYBRID && !(gas->l_ref > 0)) return "l_ref must be positive";
  if (!(sc->dt_fixed > 0) && !(sc->cfl > 0)) return "cfl must be positive when dt_fixed is not set";
  S.L = sc->central_order / 2;
  S.Lv = gas->visc_law == STREAMS_VISC_NONE ? 0 : sc->visc_order / 2;
  S.r = sc->flux_mode == STREAMS_FLUX_CENTRAL ? 0 : (sc->weno_order + 1) / 2;
  // three ghost layers, four when an order of the scheme reaches further (central / viscous 8, WENO 7)
  S.ng = std::max(3, std::max(S.L, std::max(S.Lv, S.r)));
  if (g->nx < S.ng || g->ny < S.ng || g->nz < S.ng) return "each extent must be at least the ghost width";
  if (g->bc_z == STREAMS_BC_HALO && g->nz_global != 0 && g->nz_global < g->nz) return "nz_global must be at least nz";
  if (g->ny + 2 * S.ng > 65535 || g->nz + 2 * S.ng > 65535) return "ny and nz (with ghosts) must not exceed 65535";
  S.ox = 16;                                              // interior i = 0 starts a 128-byte line
  S.px = (int)align_up((size_t)S.ox + g->nx + S.ng, 16);
  S.py = g->ny + 2 * S.ng;
  S.pz = g->nz + 2 * S.ng;
  S.fs = align_up((size_t)S.px * S.py * S.pz, 32);
  S.N = (size_t)g->nx * g->ny * g->nz;
  S.nq = NQ;
  const bool hyb = sc->flux_mode == STREAMS_FLUX_HYBRID;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
  S.off_w = take(5 * S.fs * 8);
  S.off_q = take((size_t)S.nq * S.fs * 8);       // two primitive buffers: a stage reads one while the fused RHS kernel
  S.off_q2 = take((size_t)S.nq * S.fs * 8);      // writes the primitives of the updated state into the other
  S.off_theta = take(S.N * 8);
  S.off_mask = take(S.fs);
  S.off_movr = take(hyb ? S.fs : 256);                    // imposed mask (streams_set_mask_override)
  S.off_nflag = take(hyb ? S.fs : 256);
  {
    const size_t face = std::max(std::max((size_t)g->ny * g->nz, (size_t)g->nx * g->nz), (size_t)g->nx * g->ny);
    S.lcap = align_up(S.N + face, 64);
    S.off_ilist = take(hyb ? 4 * S.lcap * 4 : 256);     // interfaces x, y, z and the nodes next to one
  }
  S.off_dF = take(sc->flux_mode != STREAMS_FLUX_CENTRAL ? 15 * S.fs * 8 : 256);
  S.off_corr = take(sc->flux_mode != STREAMS_FLUX_CENTRAL ? 5 * S.fs * 8 : 256);
  S.off_counters = take(C_COUNT * 4);
  S.off_R = take(5 * S.fs * 8);
  S.off_metrics = take(3 * (size_t)g->ny * 8);
  S.off_scal = take(S_COUNT * 8);
  S.off_sums = take((size_t)sums_scratch_doubles() * 8);
  S.total = off;
  return nullptr;
}

}  // namespace

struct streams_ctx {
  streams_grid grid;
  streams_gas gas;
  streams_scheme scheme;
  Sizes S;
  DevP P;                   // P.q / P.div point at the CURRENT primitive buffer (qbuf[cur])
  MarchMaps maps[2];        // TMA views of each primitive buffer
  double* qbuf[2];
  int cur;                  // index of the buffer that holds (or will receive) the primitives of the current state
  bool prims_interior;      // qbuf[cur] already holds the primitives of every interior node (written by the last stage)
  bool r_valid;             // DevP::R holds the right-hand side of the current state (after streams_rhs)
  bool rate_ready;          // scal[S_RATE] already holds the rate of the current state (reduced by the last stage)
  cudaStream_t stream;
  char* base;
  bool have_fields;
  long long step_count;     // steps since set_fields (host mirror; decides when dt is recomputed)
  long long launches;
  char err[256];
  // per-kernel device timing (streams_profile): event pairs recorded on the stream around each launch
  bool prof_on;
  std::vector<cudaEvent_t> prof_pool;             // 2 events per record
  std::vector<int> prof_kind;                     // kernel class of record i
  size_t prof_used;                               // records in flight
  double prof_ms[STREAMS_K_COUNT];
  long long prof_n[STREAMS_K_COUNT];
  long long prof_dropped;
  // CUDA graphs of one RK3 step (streams_step): the launches of a step are captured once per variant
  // (primitive buffer the step starts from, dt recomputed at its start, rate reduced at its end) and replayed
  bool graphs_on;
  cudaGraphExec_t step_graph[8];
  int step_graph_launches[8];
  long long graph_launches;
};

namespace {

int fail(streams_ctx* c, int code, const char* msg) {
  if (c) std::snprintf(c->err, sizeof c->err, "%s", msg);
  else std::snprintf(g_init_error, sizeof g_init_error, "%s", msg);
  return code;
}
int cuda_fail(streams_ctx* c, cudaError_t e, const char* where) {
  char buf[256];
  std::snprintf(buf, sizeof buf, "%s: %s", where, cudaGetErrorString(e));
  return fail(c, STREAMS_ECUDA, buf);
}
#define CU(call)                                                   \
  do {                                                             \
    cudaError_t e__ = (call);                                      \
    if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call);     \
  } while (0)

// y metrics on the host (O4 / S3), same evaluation order as the definition:
// D = a_1 (y_{+1} - y_{-1}); D = D + a_l (y_{+l} - y_{-l}); eta_y = 1 / D;
// eta_yy = -(D2) eta_y^3 with D2 = sum_l b_l ((y_{+l} - 2 y_0) + y_{-l}).
void build_metrics(const streams_ctx* c, const double* y_nodes, std::vector<double>& eyc, std::vector<double>& eyv,
                   std::vector<double>& eyyv) {
  const streams_grid& g = c->grid;
  const int ny = g.ny, ng = c->S.ng, L = c->S.L, Lv = c->S.Lv;
  eyc.assign(ny, 0.0); eyv.assign(ny, 0.0); eyyv.assign(ny, 0.0);
  const bool per = g.bc_y_lo == STREAMS_BC_PERIODIC;
  if (!y_nodes) {
    const double inv_dy = per ? (double)ny / g.ly : (double)ny / (g.y_wall_hi - g.y_wall_lo);
    for (int j = 0; j < ny; ++j) { eyc[j] = inv_dy; eyv[j] = inv_dy; }
    return;
  }
  std::vector<double> yn(ny + 2 * ng);
  for (int j = 0; j < ny; ++j) yn[j + ng] = y_nodes[j];
  for (int m = 0; m < ng; ++m) {
    if (per) {
      yn[ng - 1 - m] = y_nodes[ny - 1 - m] - g.ly;
      yn[ng + ny + m] = y_nodes[m] + g.ly;
    } else {
      yn[ng - 1 - m] = 2.0 * g.y_wall_lo - y_nodes[m];
      yn[ng + ny + m] = 2.0 * g.y_wall_hi - y_nodes[ny - 1 - m];
    }
  }
  for (int j = 0; j < ny; ++j) {
    const double* y = &yn[j + ng];
    double acc = c->P.a1[0] * (y[1] - y[-1]);
    for (int l = 2; l <= L; ++l) acc = acc + c->P.a1[l - 1] * (y[l] - y[-l]);
    eyc[j] = 1.0 / acc;
    if (Lv > 0) {
      double d1 = c->P.a1v[0] * (y[1] - y[-1]);
      for (int l = 2; l <= Lv; ++l) d1 = d1 + c->P.a1v[l - 1] * (y[l] - y[-l]);
      double d2 = c->P.b2v[0] * ((y[1] - 2.0 * y[0]) + y[-1]);
      for (int l = 2; l <= Lv; ++l) d2 = d2 + c->P.b2v[l - 1] * ((y[l] - 2.0 * y[0]) + y[-l]);
      const double ey = 1.0 / d1;
      eyv[j] = ey;
      eyyv[j] = -d2 * ((ey * ey) * ey);
    }
  }
}

// Runs one launch wrapper; with profiling on, brackets it with an event pair on the stream.
template <class F>
int timed(streams_ctx* ctx, int kind, F&& launch) {
  const bool rec = ctx->prof_on && 2 * (ctx->prof_used + 1) <= ctx->prof_pool.size();
  if (ctx->prof_on && !rec) ctx->prof_dropped += 1;
  if (rec) cudaEventRecord(ctx->prof_pool[2 * ctx->prof_used], ctx->stream);
  const int n = launch();
  if (rec && n > 0) {                                 // a wrapper that launched nothing leaves no record
    cudaEventRecord(ctx->prof_pool[2 * ctx->prof_used + 1], ctx->stream);
    ctx->prof_kind[ctx->prof_used] = kind;
    ctx->prof_used += 1;
  }
  if (n > 0) ctx->launches += n;
  return n;
}

// Folds the finished event pairs into the per-class totals (synchronises the stream).
cudaError_t prof_drain(streams_ctx* ctx) {
  if (ctx->prof_used == 0) return cudaSuccess;
  cudaError_t e = cudaStreamSynchronize(ctx->stream);
  if (e != cudaSuccess) return e;
  for (size_t i = 0; i < ctx->prof_used; ++i) {
    float ms = 0.f;
    e = cudaEventElapsedTime(&ms, ctx->prof_pool[2 * i], ctx->prof_pool[2 * i + 1]);
    if (e != cudaSuccess) return e;
    ctx->prof_ms[ctx->prof_kind[i]] += ms;
    ctx->prof_n[ctx->prof_kind[i]] += 1;
  }
  ctx->prof_used = 0;
  return cudaSuccess;
}

// ghost fill + primitives (+ dt) + sensor + flags: everything a stage needs before the RHS kernels.
// After an updating stage the fused RHS kernel has already written the primitives of every interior node of the
// new state (and, on request, reduced its time-step rate): only the ghost shell is left.  Otherwise (first
// evaluation after streams_set_fields, or a dt wanted that no stage prepared) the full pass runs.
// The three parts of what a stage needs before its RHS kernels (a sharded run exchanges halo planes between them,
// streams_shard_*): (1) ghost fill + primitives (+ the local time-step rate when no stage prepared it) ...
int prepare_fill(streams_ctx* ctx, bool want_dt) {
  const DevP& P = ctx->P;
  cudaStream_t st = ctx->stream;
  const bool reduce_dt = want_dt && !(ctx->scheme.dt_fixed > 0.0) && !ctx->rate_ready;
  int n;
  if (ctx->prims_interior && !reduce_dt) n = timed(ctx, STREAMS_K_FILL_PRIM, [&] { return launch_fill_ghosts(P, st); });
  else n = timed(ctx, STREAMS_K_FILL_PRIM, [&] { return launch_fill_prim(P, reduce_dt, st); });
  ctx->prims_interior = true;
  return n < 0 ? n : 0;
}
// ... (2) the step scalars at the start of a step (dt = CFL / rate, time, step count), then sensor / dilatation ...
int prepare_sensor(streams_ctx* ctx, bool want_dt, bool theta, bool step_start) {
  const DevP& P = ctx->P;
  cudaStream_t st = ctx->stream;
  int rc = 0;
  auto run = [&](int kind, auto&& launch) { const int n = timed(ctx, kind, launch); if (n < 0 && rc == 0) rc = n; };
  if (step_start) run(STREAMS_K_DT, [&] { return launch_dt(P, ctx->scheme.dt_fixed, want_dt, st); });
  if (want_dt) ctx->rate_ready = false;             // dt_finalize consumed (and zeroed) the rate
  const bool hyb = ctx->scheme.flux_mode == STREAMS_FLUX_HYBRID;
  const bool visc = ctx->gas.visc_law != STREAMS_VISC_NONE;
  if (hyb || visc || theta)
    run(STREAMS_K_SENSOR, [&] { return launch_sensor(P, ctx->maps[ctx->cur], ctx->S.L, hyb || theta, theta, st, false); });
  return rc;
}
// ... (3) interface flags and work lists from the node mask.
int prepare_flags(streams_ctx* ctx) {
  if (ctx->scheme.flux_mode != STREAMS_FLUX_HYBRID) return 0;
  const int n = timed(ctx, STREAMS_K_FLAGS, [&] { return launch_flags(ctx->P, ctx->S.r, ctx->stream); });
  return n < 0 ? n : 0;
}
int enqueue_prepare(streams_ctx* ctx, bool want_dt, bool theta, bool step_start = false) {
  int rc = prepare_fill(ctx, want_dt);
  if (rc == 0) rc = prepare_sensor(ctx, want_dt, theta, step_start);
  if (rc == 0) rc = prepare_flags(ctx);
  return rc;
}

// error of a negative launch code (streams_launch.h)
int launch_fail(streams_ctx* ctx, int rc) {
  if (rc == -2) return fail(ctx, STREAMS_ECUDA, "cudaFuncSetAttribute: cannot opt a kernel in to its dynamic shared memory");
  return fail(ctx, STREAMS_EINVAL, "order combination outside the instantiated kernels");
}

// points DevP::q / div at primitive buffer b
void use_qbuf(streams_ctx* ctx, int b) {
  ctx->cur = b;
  ctx->P.q = ctx->qbuf[b];
  ctx->P.div = ctx->qbuf[b] + (size_t)Q_DIV * ctx->S.fs;
}

void drop_step_graphs(streams_ctx* ctx) {            // kernel arguments baked into the graphs have changed
  for (int g = 0; g < 8; ++g) {
    if (ctx->step_graph[g]) cudaGraphExecDestroy(ctx->step_graph[g]);
    ctx->step_graph[g] = nullptr;
  }
}

// the RHS (+ update) of one stage: the WENO flux corrections of the flagged interfaces first (they read the
// primitives only), then the fused central / viscous / correction / update pass over all nodes
int enqueue_rhs(streams_ctx* ctx, const StageArgs& sa) {
  const DevP& P = ctx->P;
  cudaStream_t st = ctx->stream;
  int b = 0, c = 0;
  if (ctx->scheme.flux_mode != STREAMS_FLUX_CENTRAL) {
    b = timed(ctx, STREAMS_K_WENO, [&] { return launch_weno(P, ctx->S.L, ctx->S.r, st); });
    c = timed(ctx, STREAMS_K_CORR, [&] { return launch_corr(P, st); });
  }
  const int a = timed(ctx, STREAMS_K_RHS_MAIN, [&] { return launch_rhs_main(P, ctx->maps[ctx->cur], ctx->S.L, ctx->S.Lv, sa, st, false); });
  return a < 0 ? a : (b < 0 ? b : (c < 0 ? c : a + b + c));
}

// the RHS kernels and the update of stage l (0, 1, 2); the primitive buffers swap
int enqueue_stage_rhs(streams_ctx* ctx, int l, bool want_rate) {
  // Wray's low-storage RK3 (O5 / S12)
  const double gam[3] = {8.0 / 15.0, 5.0 / 12.0, 3.0 / 4.0};
  const double rhk[3] = {0.0, -17.0 / 60.0, -5.0 / 12.0};
  StageArgs sa;
  sa.gam = gam[l]; sa.rhk = rhk[l]; sa.update_w = 1; sa.read_prev = (l > 0); sa.write_r = (l < 2);
  sa.r_dense = nullptr;
  sa.q_out = ctx->qbuf[ctx->cur ^ 1];
  sa.want_rate = (l == 2 && want_rate) ? 1 : 0;
  sa.check_state = (l == 2);
  const int rc = enqueue_rhs(ctx, sa);
  if (rc < 0) return rc;
  use_qbuf(ctx, ctx->cur ^ 1);                       // the updated state's primitives are in the other buffer
  ctx->prims_interior = true;
  if (sa.want_rate) ctx->rate_ready = true;
  return 0;
}

// the launches of one RK3 step: three stages of (ghost fill, step scalars, sensor, flags, WENO, gather, fused RHS + update)
int enqueue_step(streams_ctx* ctx, bool want_dt, bool want_rate) {
  for (int l = 0; l < 3; ++l) {
    int rc = enqueue_prepare(ctx, want_dt && l == 0, false, l == 0);
    if (rc < 0) return rc;
    if ((rc = enqueue_stage_rhs(ctx, l, want_rate)) < 0) return rc;
  }
  return 0;
}

}  // namespace

extern "C" {

size_t streams_workspace_bytes(const streams_grid* grid, const streams_gas* gas, const streams_scheme* scheme) {
  Sizes S;
  const char* msg = plan(grid, gas, scheme, S);
  if (msg) { fail(nullptr, STREAMS_EINVAL, msg); return 0; }
  return S.total;
}

int streams_init(streams_ctx** out, const streams_grid* grid, const streams_gas* gas, const streams_scheme* scheme,
                 void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
  if (!out) return fail(nullptr, STREAMS_EINVAL, "out is null");
  *out = nullptr;
  Sizes S;
  const char* msg = plan(grid, gas, scheme, S);
  if (msg) return fail(nullptr, STREAMS_EINVAL, msg);
  if (!workspace_dev || workspace_bytes < S.total) return fail(nullptr, STREAMS_ENOMEM, "workspace too small");
  if (((uintptr_t)workspace_dev) % 256) return fail(nullptr, STREAMS_EINVAL, "workspace must be 256-byte aligned");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return fail(nullptr, STREAMS_ECUDA, "no CUDA device");
  streams_ctx* ctx = new (std::nothrow) streams_ctx();
  if (!ctx) return fail(nullptr, STREAMS_ENOMEM, "host allocation failed");
  ctx->grid = *grid; ctx->gas = *gas; ctx->scheme = *scheme; ctx->S = S;
  ctx->grid.y_nodes = nullptr;
  ctx->stream = (cudaStream_t)cuda_stream;
  ctx->base = (char*)workspace_dev;
  ctx->have_fields = false; ctx->step_count = 0; ctx->launches = 0; ctx->err[0] = 0;
  ctx->prof_on = false; ctx->prof_used = 0; ctx->prof_dropped = 0;
  {
    const char* ng = std::getenv("STREAMS_NO_GRAPH");   // debugging aid: launch every kernel of a step individually
    ctx->graphs_on = !(ng && ng[0] && ng[0] != '0');
  }
  for (int g = 0; g < 8; ++g) { ctx->step_graph[g] = nullptr; ctx->step_graph_launches[g] = 0; }
  ctx->graph_launches = 0;
  for (int k = 0; k < STREAMS_K_COUNT; ++k) { ctx->prof_ms[k] = 0.0; ctx->prof_n[k] = 0; }
  if (ctx->scheme.dt_every < 1) ctx->scheme.dt_every = 1;
  DevP& P = ctx->P;
  std::memset(&P, 0, sizeof P);
  P.nx = grid->nx; P.ny = grid->ny; P.nz = grid->nz; P.ng = S.ng; P.ox = S.ox;
  P.px = S.px; P.py = S.py; P.pz = S.pz;
  P.sy = S.px; P.sz = (long long)S.px * S.py; P.fs = (long long)S.fs; P.N = (long long)S.N;
  P.w = (double*)(ctx->base + S.off_w);
  ctx->qbuf[0] = (double*)(ctx->base + S.off_q);
  ctx->qbuf[1] = (double*)(ctx->base + S.off_q2);
  ctx->prims_interior = false; ctx->rate_ready = false; ctx->r_valid = false;
  P.theta = (double*)(ctx->base + S.off_theta);
  P.mask = (unsigned char*)(ctx->base + S.off_mask);
  P.mask_ovr = nullptr;
  P.nflag = (unsigned char*)(ctx->base + S.off_nflag);
  P.ilist = (int*)(ctx->base + S.off_ilist);
  P.lcap = (long long)S.lcap;
  P.dF = (double*)(ctx->base + S.off_dF);
  P.corr = (double*)(ctx->base + S.off_corr);
  P.counters = (int*)(ctx->base + S.off_counters);
  P.R = (double*)(ctx->base + S.off_R);
  double* met = (double*)(ctx->base + S.off_metrics);
  P.eta_y_c = met; P.eta_y_v = met + grid->ny; P.eta_yy_v = met + 2 * (size_t)grid->ny;
  P.scal = (double*)(ctx->base + S.off_scal);
  P.inv_dx = (double)grid->nx / grid->lx;
  P.inv_dz = (double)(grid->bc_z == STREAMS_BC_HALO && grid->nz_global > 0 ? grid->nz_global : grid->nz) / grid->lz;
  fd1(S.L, P.a1); fd1(S.Lv, P.a1v); fd2(S.Lv, P.b2v);
  P.sbv = 0.0;
  for (int l = 0; l < 4; ++l) {
    P.kc[l] = 0.25 * P.a1[l];
    P.avx[l] = P.a1v[l] * P.inv_dx; P.bvx[l] = P.b2v[l] * (P.inv_dx * P.inv_dx);
    P.avz[l] = P.a1v[l] * P.inv_dz; P.bvz[l] = P.b2v[l] * (P.inv_dz * P.inv_dz);
    P.sbv += P.b2v[l];
  }
  P.sb2xz = -2.0 * P.sbv * (P.inv_dx * P.inv_dx + P.inv_dz * P.inv_dz);
  P.gamma = gas->gamma; P.gm1 = gas->gamma - 1.0; P.rgas = gas->rgas; P.prandtl = gas->prandtl;
  P.kfac = (gas->gamma * gas->rgas / (gas->gamma - 1.0)) / gas->prandtl;
  P.inv_rgas = 1.0 / gas->rgas; P.inv_tref = gas->t_ref > 0.0 ? 1.0 / gas->t_ref : 0.0;
  P.mu_ref = gas->mu_ref; P.t_ref = gas->t_ref; P.suth_s = gas->suth_s_over_tref; P.pow_exp = gas->pow_exp;
  const double rr = gas->u_ref / gas->l_ref;
  P.eps_s = rr * rr;
  P.thr = scheme->sensor_threshold; P.thr2 = P.thr * P.thr; P.weno_eps = scheme->weno_eps; P.cfl = scheme->cfl;
  for (int q = 0; q < 5; ++q) P.fsw[q] = gas->freestream[q];
  for (int d = 0; d < 3; ++d) P.accel[d] = gas->accel[d];
  P.has_accel = (gas->accel[0] != 0.0 || gas->accel[1] != 0.0 || gas->accel[2] != 0.0) ? 1 : 0;
  P.t_wall_lo = grid->t_wall_lo; P.t_wall_hi = grid->t_wall_hi;
  P.bc_x = grid->bc_x; P.bc_y_lo = grid->bc_y_lo; P.bc_y_hi = grid->bc_y_hi; P.bc_z = grid->bc_z;
  P.visc_law = gas->visc_law; P.flux_mode = scheme->flux_mode;
  P.weno_z = scheme->weno_variant == STREAMS_WENO_Z;
  P.own_x = grid->bc_x == STREAMS_BC_PERIODIC && grid->nx >= 2 * S.ng;
  P.own_y = grid->bc_y_lo == STREAMS_BC_PERIODIC && grid->ny >= 2 * S.ng;
  P.own_z = grid->bc_z == STREAMS_BC_PERIODIC && grid->nz >= 2 * S.ng;
  P.sown = (P.own_x || grid->bc_x != STREAMS_BC_PERIODIC) && (P.own_y || grid->bc_y_lo != STREAMS_BC_PERIODIC) &&
           (P.own_z || grid->bc_z != STREAMS_BC_PERIODIC);
  {
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || nsm < 1) {
      delete ctx;
      return fail(nullptr, STREAMS_ECUDA, "cannot query the device");
    }
    P.nsm = nsm;
  }
  int maps_rc = 0;
  for (int b = 1; b >= 0; --b) {                    // ends on buffer 0, the first current one
    P.q = ctx->qbuf[b];
    P.div = P.q + (size_t)Q_DIV * S.fs;
    ctx->cur = b;
    if (make_march_maps(P, &ctx->maps[b]) != 0) maps_rc = -1;
  }
  if (maps_rc != 0) {
    delete ctx;
    return fail(nullptr, STREAMS_ECUDA, "cannot build the TMA descriptors (cuTensorMapEncodeTiled)");
  }

  {
    // opt the z-marching kernels this context launches in to their dynamic shared memory on this device, once
    StageArgs sa0{};
    int rc = launch_rhs_main(P, ctx->maps[0], S.L, S.Lv, sa0, ctx->stream, true);
    if (rc == 0)                                     // (streams_get_sensor may run the sensor in any mode)
      rc = launch_sensor(P, ctx->maps[0], S.L, true, true, ctx->stream, true);
    if (rc != 0) {
      delete ctx;
      return rc == -2 ? fail(nullptr, STREAMS_ECUDA, "cudaFuncSetAttribute: cannot opt a kernel in to its dynamic shared memory")
                      : fail(nullptr, STREAMS_EINVAL, "order combination outside the instantiated kernels");
    }
  }

  std::vector<double> eyc, eyv, eyyv;
  build_metrics(ctx, grid->y_nodes, eyc, eyv, eyyv);
  cudaError_t e = cudaMemsetAsync(ctx->base, 0, S.total, ctx->stream);   // defined ghosts / scalars from the start
  if (e == cudaSuccess) e = cudaMemcpyAsync(met, eyc.data(), grid->ny * 8, cudaMemcpyHostToDevice, ctx->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(met + grid->ny, eyv.data(), grid->ny * 8, cudaMemcpyHostToDevice, ctx->stream);
  if (e == cudaSuccess) e = cudaMemcpyAsync(met + 2 * (size_t)grid->ny, eyyv.data(), grid->ny * 8, cudaMemcpyHostToDevice, ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);          // host vectors go out of scope
  if (e != cudaSuccess) {
    cuda_fail(nullptr, e, "streams_init");
    delete ctx;
    return STREAMS_ECUDA;
  }
  *out = ctx;
  return STREAMS_OK;
}

int streams_set_fields(streams_ctx* ctx, const double* w, int src_is_device) {
  if (!ctx || !w) return fail(ctx, STREAMS_EINVAL, "null argument");
  const DevP& P = ctx->P;
  const cudaMemcpyKind kind = src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  for (int q = 0; q < 5; ++q) {
    cudaMemcpy3DParms p;
    std::memset(&p, 0, sizeof p);
    p.srcPtr = make_cudaPitchedPtr((void*)(w + (size_t)q * P.N), (size_t)P.nx * 8, P.nx, P.ny);
    p.dstPtr = make_cudaPitchedPtr((void*)(P.w + q * P.fs), (size_t)P.px * 8, P.px, P.py);
    p.dstPos = make_cudaPos((size_t)P.ox * 8, P.ng, P.ng);
    p.extent = make_cudaExtent((size_t)P.nx * 8, P.ny, P.nz);
    p.kind = kind;
    CU(cudaMemcpy3DAsync(&p, ctx->stream));
  }
  CU(cudaMemsetAsync(P.scal, 0, S_ACC * 8, ctx->stream));   // step scalars; the controller's (S_ACC ..) are kept
  CU(cudaMemsetAsync(P.counters, 0, C_COUNT * 4, ctx->stream));
  if (!src_is_device) CU(cudaStreamSynchronize(ctx->stream));   // the host buffer may be reused on return
  ctx->have_fields = true;
  ctx->step_count = 0;
  ctx->prims_interior = false;                       // the next evaluation runs the full ghost + primitive pass
  ctx->rate_ready = false;
  ctx->r_valid = false;
  return STREAMS_OK;
}

int streams_get_fields(streams_ctx* ctx, double* w_out, int dst_is_device) {
  if (!ctx || !w_out) return fail(ctx, STREAMS_EINVAL, "null argument");
  if (!ctx->have_fields) return fail(ctx, STREAMS_ESTATE, "no fields set");
  const DevP& P = ctx->P;
  const cudaMemcpyKind kind = dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  for (int q = 0; q < 5; ++q) {
    cudaMemcpy3DParms p;
    std::memset(&p, 0, sizeof p);
    p.srcPtr = make_cudaPitchedPtr((void*)(P.w + q * P.fs), (size_t)P.px * 8, P.px, P.py);
    p.srcPos = make_cudaPos((size_t)P.ox * 8, P.ng, P.ng);
    p.dstPtr = make_cudaPitchedPtr((void*)(w_out + (size_t)q * P.N), (size_t)P.nx * 8, P.nx, P.ny);
    p.extent = make_cudaExtent((size_t)P.nx * 8, P.ny, P.nz);
    p.kind = kind;
    CU(cudaMemcpy3DAsync(&p, ctx->stream));
  }
  if (!dst_is_device) CU(cudaStreamSynchronize(ctx->stream));
  return STREAMS_OK;
}

int streams_rhs(streams_ctx* ctx, double* rhs_out_dev) {
  if (!ctx) return fail(ctx, STREAMS_EINVAL, "null context");
  if (!ctx->have_fields) return fail(ctx, STREAMS_ESTATE, "streams_rhs before streams_set_fields");
  int rc = enqueue_prepare(ctx, false, false);
  if (rc < 0) return launch_fail(ctx, rc);
  StageArgs sa;
  sa.gam = 0.0; sa.rhk = 0.0; sa.update_w = 0; sa.read_prev = 0; sa.write_r = 1;
  sa.r_dense = rhs_out_dev; sa.q_out = nullptr; sa.want_rate = 0; sa.check_state = 0;
  if ((rc = enqueue_rhs(ctx, sa)) < 0) return launch_fail(ctx, rc);
  CU(cudaGetLastError());
  ctx->r_valid = true;
  return STREAMS_OK;
}

// One RK3 step on the stream: replayed from its CUDA graph when its launch sequence is the steady one, launched kernel
// by kernel otherwise.  Returns STREAMS_OK or an error code (message set).
static int run_one_step(streams_ctx* ctx) {
  const bool want_dt = (ctx->step_count % ctx->scheme.dt_every) == 0;
  // the last stage also reduces the time-step rate of the state it produces if the next step recomputes dt
  const bool want_rate = !(ctx->scheme.dt_fixed > 0.0) && ((ctx->step_count + 1) % ctx->scheme.dt_every) == 0;
  // A step whose launch sequence is the steady one (primitives of the state already in place, the rate for its dt
  // already reduced) is replayed from a CUDA graph: the 10-16 launches of a step become one submission, which is
  // what a small grid needs (grids below ~2 M points cannot hide the launch latency).
  const bool steady = ctx->prims_interior && (!want_dt || ctx->scheme.dt_fixed > 0.0 || ctx->rate_ready);
  if (ctx->graphs_on && !ctx->prof_on && steady) {
    const int key = ctx->cur | (want_dt ? 2 : 0) | (want_rate ? 4 : 0);
    if (!ctx->step_graph[key]) {
      const long long l0 = ctx->launches;
      const int cur0 = ctx->cur;
      const bool rr0 = ctx->rate_ready;
      if (cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();                          // e.g. the legacy default stream cannot be captured: launch directly
        ctx->graphs_on = false;
        const int rd = enqueue_step(ctx, want_dt, want_rate);
        if (rd < 0) return launch_fail(ctx, rd);
        ctx->step_count += 1;
        return STREAMS_OK;
      }
      const int rc = enqueue_step(ctx, want_dt, want_rate);
      cudaGraph_t graph = nullptr;
      const cudaError_t ee = cudaStreamEndCapture(ctx->stream, &graph);
      // nothing ran during the capture, whether it succeeded or not: rewind the host state it advanced (the replay
      // below advances it again; on an error return the context still describes the state on the device)
      const int captured = (int)(ctx->launches - l0);
      ctx->launches = l0;
      use_qbuf(ctx, cur0);
      ctx->rate_ready = rr0;
      if (rc < 0) { if (graph) cudaGraphDestroy(graph); return launch_fail(ctx, rc); }
      if (ee != cudaSuccess) return cuda_fail(ctx, ee, "cudaStreamEndCapture");
      const cudaError_t ei = cudaGraphInstantiate(&ctx->step_graph[key], graph, 0);
      cudaGraphDestroy(graph);
      if (ei != cudaSuccess) { ctx->step_graph[key] = nullptr; return cuda_fail(ctx, ei, "cudaGraphInstantiate"); }
      ctx->step_graph_launches[key] = captured;
    }
    CU(cudaGraphLaunch(ctx->step_graph[key], ctx->stream));
    ctx->graph_launches += 1;
    ctx->launches += ctx->step_graph_launches[key];
    use_qbuf(ctx, ctx->cur ^ 1);                   // three stages, three swaps of the primitive buffers
    if (want_dt) ctx->rate_ready = false;
    if (want_rate) ctx->rate_ready = true;
  } else {
    const int rc = enqueue_step(ctx, want_dt, want_rate);
    if (rc < 0) return launch_fail(ctx, rc);
  }
  ctx->step_count += 1;
  return STREAMS_OK;
}

// reads the step scalars back (synchronises the stream) and maps a non-finite state or time step to STREAMS_ENAN
static int finish_steps(streams_ctx* ctx, double* dt_last, double* time, double* accel3_out) {
  CU(cudaGetLastError());
  double h[S_COUNT];
  CU(cudaMemcpyAsync(h, ctx->P.scal, sizeof h, cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  if (dt_last) *dt_last = h[S_DT];
  if (time) *time = h[S_TIME];
  if (accel3_out) for (int a = 0; a < 3; ++a) accel3_out[a] = ctx->P.has_accel == 2 ? h[S_ACC + a] : ctx->P.accel[a];
  if (h[S_NAN] != 0.0 || !std::isfinite(h[S_DT]) || !std::isfinite(h[S_TIME]) || !std::isfinite(h[S_RATE]))
    return fail(ctx, STREAMS_ENAN, "the state or the time step became non-finite");
  return STREAMS_OK;
}

int streams_step(streams_ctx* ctx, int nsteps, double* dt_last, double* time) {
  if (!ctx) return fail(ctx, STREAMS_EINVAL, "null context");
  if (!ctx->have_fields) return fail(ctx, STREAMS_ESTATE, "streams_step before streams_set_fields");
  if (nsteps < 0) return fail(ctx, STREAMS_EINVAL, "nsteps must be non-negative");
  if (nsteps > 0) ctx->r_valid = false;              // R becomes the low-storage scheme's previous-stage register
  for (int s = 0; s < nsteps; ++s) {
    const int rc = run_one_step(ctx);
    if (rc != STREAMS_OK) return rc;
  }
  return finish_steps(ctx, dt_last, time, nullptr);
}

int streams_step_forced(streams_ctx* ctx, int nsteps, int direction, double target, double* dt_last, double* time,
                        double* accel3_out) {
  if (!ctx) return fail(ctx, STREAMS_EINVAL, "null context");
  if (!ctx->have_fields) return fail(ctx, STREAMS_ESTATE, "streams_step_forced before streams_set_fields");
  if (nsteps < 0 || direction < 0 || direction > 2) return fail(ctx, STREAMS_EINVAL, "bad nsteps or direction");
  double* scratch = (double*)(ctx->base + ctx->S.off_sums);
  double* sums_dev = scratch + (sums_scratch_doubles() - 8);
  cudaStream_t st = ctx->stream;
  if (ctx->P.has_accel != 2) {
    // the controller takes the acceleration over: its current value moves to the device scalars, the kernels read it
    // there from now on (until streams_set_body_force hands it back to the host)
    CU(cudaMemcpyAsync(ctx->P.scal + S_ACC, ctx->P.accel, 3 * sizeof(double), cudaMemcpyHostToDevice, st));
    CU(cudaStreamSynchronize(st));                   // P.accel is host memory of the context
    ctx->P.has_accel = 2;
    drop_step_graphs(ctx);
    timed(ctx, STREAMS_K_MISC, [&] { return launch_sums(ctx->P, STREAMS_SUM_STATE, scratch, sums_dev, st); });
    timed(ctx, STREAMS_K_MISC, [&] { return launch_controller(ctx->P, sums_dev, direction, target, true, st); });
    target = std::nan("");                           // recorded; later updates keep it
  }
  if (nsteps > 0) ctx->r_valid = false;
  for (int s = 0; s < nsteps; ++s) {
    const int rc = run_one_step(ctx);
    if (rc != STREAMS_OK) return rc;
    timed(ctx, STREAMS_K_MISC, [&] { return launch_sums(ctx->P, STREAMS_SUM_STATE, scratch, sums_dev, st); });
    timed(ctx, STREAMS_K_MISC, [&] { return launch_controller(ctx->P, sums_dev, direction, target, false, st); });
    target = std::nan("");
  }
  return finish_steps(ctx, dt_last, time, accel3_out);
}

// ---- sharded stepping: one context per z slab, the caller exchanges halo planes between the phases
static bool shard_want_dt(const streams_ctx* ctx) { return (ctx->step_count % ctx->scheme.dt_every) == 0; }
static bool shard_want_rate(const streams_ctx* ctx) {
  return !(ctx->scheme.dt_fixed > 0.0) && ((ctx->step_count + 1) % ctx->scheme.dt_every) == 0;
}
static int shard_check(streams_ctx* ctx, int stage) {
  if (!ctx) return fail(ctx, STREAMS_EINVAL, "null context");
  if (!ctx->have_fields) return fail(ctx, STREAMS_ESTATE, "no fields set");
  if (stage < 0 || stage > 2) return fail(ctx, STREAMS_EINVAL, "stage must be 0, 1 or 2");
  return STREAMS_OK;
}

int streams_shard_fill(streams_ctx* ctx, int stage, int* rate_is_local) {
  int rc = shard_check(ctx, stage);
  if (rc != STREAMS_OK) return rc;
  if (stage == 0) ctx->r_valid = false;
  const bool want_dt = stage == 0 && shard_want_dt(ctx);
  if (rate_is_local) *rate_is_local = (want_dt && !(ctx->scheme.dt_fixed > 0.0)) ? 1 : 0;
  if ((rc = prepare_fill(ctx, want_dt)) < 0) return launch_fail(ctx, rc);
  CU(cudaGetLastError());
  return STREAMS_OK;
}

int streams_shard_sensor(streams_ctx* ctx, int stage) {
  int rc = shard_check(ctx, stage);
  if (rc != STREAMS_OK) return rc;
  if ((rc = prepare_sensor(ctx, stage == 0 && shard_want_dt(ctx), false, stage == 0)) < 0) return launch_fail(ctx, rc);
  CU(cudaGetLastError());
  return STREAMS_OK;
}

int streams_shard_rhs(streams_ctx* ctx, int stage) {
  int rc = shard_check(ctx, stage);
  if (rc != STREAMS_OK) return rc;
  if ((rc = prepare_flags(ctx)) < 0) return launch_fail(ctx, rc);
  if ((rc = enqueue_stage_rhs(ctx, stage, shard_want_rate(ctx))) < 0) return launch_fail(ctx, rc);
  if (stage == 2) ctx->step_count += 1;
  CU(cudaGetLastError());
  return STREAMS_OK;
}

int streams_shard_finish(streams_ctx* ctx, double* dt_last, double* time) {
  if (!ctx) return fail(ctx, STREAMS_EINVAL, "null context");
  return finish_steps(ctx, dt_last, time, nullptr);
}

int streams_halo_slabs(streams_ctx* ctx, int what, void** lo_send, void** lo_recv, void** hi_send, void** hi_recv,
                       size_t* slab_bytes, int* nfields, size_t* field_stride_bytes) {
  if (!ctx) return fail(ctx, STREAMS_EINVAL, "null context");
  if (what != STREAMS_HALO_PRIMS && what != STREAMS_HALO_DIV && what != STREAMS_HALO_MASK && what != STREAMS_HALO_RATE)
    return fail(ctx, STREAMS_EINVAL, "bad halo selector");
  const DevP& P = ctx->P;
  char* base;
  size_t elem = 8, fstride = (size_t)P.fs * 8;
  int nf = 1;
  if (what == STREAMS_HALO_RATE) {                   // the local time-step rate (one double): max-reduce it over the ranks
    if (lo_send) *lo_send = P.scal + S_RATE;
    if (lo_recv) *lo_recv = nullptr;
    if (hi_send) *hi_send = nullptr;
    if (hi_recv) *hi_recv = nullptr;
    if (slab_bytes) *slab_bytes = 8;
    if (nfields) *nfields = 1;
    if (field_stride_bytes) *field_stride_bytes = 0;
    return STREAMS_OK;
  }
  if (what == STREAMS_HALO_PRIMS) { base = (char*)P.q; nf = NQ; }
  else if (what == STREAMS_HALO_DIV) { base = (char*)P.div; }
  else { base = (char*)P.mask; elem = 1; fstride = 0; }
  const size_t plane = (size_t)P.sz * elem, slab = (size_t)P.ng * plane;
  if (lo_recv) *lo_recv = base;                                        // ghost planes k = -ng .. -1
  if (lo_send) *lo_send = base + slab;                                 // interior planes 0 .. ng-1
  if (hi_send) *hi_send = base + (size_t)P.nz * plane;                 // interior planes nz-ng .. nz-1
  if (hi_recv) *hi_recv = base + (size_t)(P.nz + P.ng) * plane;        // ghost planes nz .. nz+ng-1
  if (slab_bytes) *slab_bytes = slab;
  if (nfields) *nfields = nf;
  if (field_stride_bytes) *field_stride_bytes = fstride;
  return STREAMS_OK;
}

int streams_get_sensor(streams_ctx* ctx, double* theta_out, unsigned char* mask_out, int dst_is_device) {
  if (!ctx) return fail(ctx, STREAMS_EINVAL, "null context");
  if (!ctx->have_fields) return fail(ctx, STREAMS_ESTATE, "no fields set");
  const DevP& P = ctx->P;
  const int prc = enqueue_prepare(ctx, false, true);
  if (prc < 0) return launch_fail(ctx, prc);
  CU(cudaGetLastError());
  const cudaMemcpyKind kind = dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
  if (theta_out) CU(cudaMemcpyAsync(theta_out, P.theta, (size_t)P.N * 8, kind, ctx->stream));
  if (mask_out) {
    cudaMemcpy3DParms p;
    std::memset(&p, 0, sizeof p);
    p.srcPtr = make_cudaPitchedPtr((void*)P.mask, (size_t)P.px, P.px, P.py);
    p.srcPos = make_cudaPos((size_t)P.ox, P.ng, P.ng);
    p.dstPtr = make_cudaPitchedPtr((void*)mask_out, (size_t)P.nx, P.nx, P.ny);
    p.extent = make_cudaExtent((size_t)P.nx, P.ny, P.nz);
    p.kind = kind;
    CU(cudaMemcpy3DAsync(&p, ctx->stream));
  }
  if (!dst_is_device) CU(cudaStreamSynchronize(ctx->stream));
  return STREAMS_OK;
}

int streams_get_activation(streams_ctx* ctx, long long* flagged_nodes, long long* shock_nodes, long long* interfaces) {
  if (!ctx) return fail(ctx, STREAMS_EINVAL, "null context");
  const DevP& P = ctx->P;
  int h[C_COUNT] = {0};
  if (ctx->scheme.flux_mode == STREAMS_FLUX_HYBRID) {
    CU(cudaMemcpyAsync(h, P.counters, sizeof h, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
  } else if (ctx->scheme.flux_mode == STREAMS_FLUX_WENO) {
    h[C_NSHOCK] = (int)P.N; h[C_NFLAGGED] = (int)P.N;
    h[C_NIFACE] = (P.nx + 1) * P.ny * P.nz; h[C_NIFACE + 1] = P.nx * (P.ny + 1) * P.nz; h[C_NIFACE + 2] = P.nx * P.ny * (P.nz + 1);
  }
  if (shock_nodes) *shock_nodes = h[C_NSHOCK];
  if (flagged_nodes) *flagged_nodes = h[C_NFLAGGED];
  if (interfaces) for (int d = 0; d < 3; ++d) interfaces[d] = h[C_NIFACE + d];
  return STREAMS_OK;
}

int streams_get_activation_totals(streams_ctx* ctx, long long* flagged_sum, long long* shock_sum, long long* interfaces_sum,
                                  long long* evaluations) {
  if (!ctx) return fail(ctx, STREAMS_EINVAL, "null context");
  unsigned long long h[6] = {0, 0, 0, 0, 0, 0};
  if (ctx->scheme.flux_mode == STREAMS_FLUX_HYBRID) {
    CU(cudaMemcpyAsync(h, ctx->P.counters + C_TOTALS, sizeof h, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
  }
  if (shock_sum) *shock_sum = (long long)h[0];
  if (flagged_sum) *flagged_sum = (long long)h[1];
  if (evaluations) *evaluations = (long long)h[2];
  if (interfaces_sum) for (int d = 0; d < 3; ++d) interfaces_sum[d] = (long long)h[3 + d];
  return STREAMS_OK;
}

int streams_set_mask_override(streams_ctx* ctx, const unsigned char* mask, int src_is_device) {
  if (!ctx) return fail(ctx, STREAMS_EINVAL, "null context");
  if (ctx->scheme.flux_mode != STREAMS_FLUX_HYBRID) return fail(ctx, STREAMS_EINVAL, "a node mask exists in hybrid mode only");
  DevP& P = ctx->P;
  drop_step_graphs(ctx);
  if (!mask) { P.mask_ovr = nullptr; return STREAMS_OK; }
  unsigned char* dst = (unsigned char*)(ctx->base + ctx->S.off_movr);
  cudaMemcpy3DParms p;
  std::memset(&p, 0, sizeof p);
  p.srcPtr = make_cudaPitchedPtr((void*)mask, (size_t)P.nx, P.nx, P.ny);
  p.dstPtr = make_cudaPitchedPtr((void*)dst, (size_t)P.px, P.px, P.py);
  p.dstPos = make_cudaPos((size_t)P.ox, P.ng, P.ng);
  p.extent = make_cudaExtent((size_t)P.nx, P.ny, P.nz);
  p.kind = src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  CU(cudaMemcpy3DAsync(&p, ctx->stream));
  if (!src_is_device) CU(cudaStreamSynchronize(ctx->stream));
  P.mask_ovr = dst;
  return STREAMS_OK;
}

int streams_set_body_force(streams_ctx* ctx, const double* accel3) {
  if (!ctx || !accel3) return fail(ctx, STREAMS_EINVAL, "null argument");
  for (int d = 0; d < 3; ++d) {
    if (!std::isfinite(accel3[d])) return fail(ctx, STREAMS_EINVAL, "accel must be finite");
    ctx->P.accel[d] = accel3[d];
    ctx->gas.accel[d] = accel3[d];
  }
  ctx->P.has_accel = (accel3[0] != 0.0 || accel3[1] != 0.0 || accel3[2] != 0.0) ? 1 : 0;   // host-owned again
  drop_step_graphs(ctx);
  ctx->r_valid = false;                              // R no longer is the right-hand side under the new force
  return STREAMS_OK;
}

int streams_get_sums(streams_ctx* ctx, int kind, double* out5) {
  if (!ctx || !out5) return fail(ctx, STREAMS_EINVAL, "null argument");
  if (kind != STREAMS_SUM_STATE && kind != STREAMS_SUM_RESIDUAL) return fail(ctx, STREAMS_EINVAL, "bad kind");
  if (!ctx->have_fields) return fail(ctx, STREAMS_ESTATE, "no fields set");
  if (kind == STREAMS_SUM_RESIDUAL && !ctx->r_valid)
    return fail(ctx, STREAMS_ESTATE, "the residual needs a streams_rhs of the current state");
  double* scratch = (double*)(ctx->base + ctx->S.off_sums);
  double* out_dev = scratch + (sums_scratch_doubles() - 8);
  timed(ctx, STREAMS_K_MISC, [&] { return launch_sums(ctx->P, kind, scratch, out_dev, ctx->stream); });
  CU(cudaGetLastError());
  CU(cudaMemcpyAsync(out5, out_dev, 5 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  return STREAMS_OK;
}

long long streams_kernel_launches(const streams_ctx* ctx) { return ctx ? ctx->launches : 0; }
long long streams_graph_launches(const streams_ctx* ctx) { return ctx ? ctx->graph_launches : 0; }

int streams_profile(streams_ctx* ctx, int enable, int max_records) {
  if (!ctx) return fail(ctx, STREAMS_EINVAL, "null context");
  CU(prof_drain(ctx));
  for (int k = 0; k < STREAMS_K_COUNT; ++k) { ctx->prof_ms[k] = 0.0; ctx->prof_n[k] = 0; }
  ctx->prof_dropped = 0;
  ctx->prof_on = enable != 0;
  if (enable) {
    const size_t want = 2 * (size_t)(max_records > 0 ? max_records : 4096);
    while (ctx->prof_pool.size() < want) {
      cudaEvent_t ev;
      CU(cudaEventCreate(&ev));
      ctx->prof_pool.push_back(ev);
    }
    ctx->prof_kind.resize(ctx->prof_pool.size() / 2);
  }
  return STREAMS_OK;
}

int streams_get_profile(streams_ctx* ctx, double* ms, long long* count, long long* dropped) {
  if (!ctx) return fail(ctx, STREAMS_EINVAL, "null context");
  CU(prof_drain(ctx));
  for (int k = 0; k < STREAMS_K_COUNT; ++k) {
    if (ms) ms[k] = ctx->prof_ms[k];
    if (count) count[k] = ctx->prof_n[k];
  }
  if (dropped) *dropped = ctx->prof_dropped;
  return STREAMS_OK;
}

size_t streams_measure_fp64_scratch_bytes(void) { return measure_fp64_scratch_bytes(); }

int streams_measure_fp64(void* cuda_stream, int kind, int repeats, void* scratch_dev, size_t scratch_bytes, double* ginst_per_s) {
  if (!ginst_per_s || kind < 0 || kind > 1) return fail(nullptr, STREAMS_EINVAL, "streams_measure_fp64: bad argument");
  const double v = measure_fp64((cudaStream_t)cuda_stream, kind, repeats < 1 ? 1 : repeats, (double*)scratch_dev, scratch_bytes);
  if (v == -2.0) return fail(nullptr, STREAMS_ENOMEM, "streams_measure_fp64: scratch buffer missing or too small");
  if (v < 0.0) return fail(nullptr, STREAMS_ECUDA, "streams_measure_fp64: CUDA error");
  *ginst_per_s = v * 1e-9;
  return STREAMS_OK;
}

const char* streams_kernel_name(int kind) {
  static const char* names[STREAMS_K_COUNT] = {"fill_prim", "dt", "sensor", "flags", "rhs_main", "weno", "corr_gather", "misc"};
  return (kind >= 0 && kind < STREAMS_K_COUNT) ? names[kind] : "";
}

const char* streams_last_error(const streams_ctx* ctx) { return ctx ? ctx->err : g_init_error; }

int streams_destroy(streams_ctx* ctx) {
  if (!ctx) return STREAMS_EINVAL;
  cudaStreamSynchronize(ctx->stream);
  drop_step_graphs(ctx);
  for (cudaEvent_t ev : ctx->prof_pool) cudaEventDestroy(ev);
  delete ctx;
  return STREAMS_OK;
}

}  // extern "C"
