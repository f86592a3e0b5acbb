/* =============================================================================
 * streams.h -- C ABI of the B200-native STREAmS-2 hot path.
 *
 * One library, libstreams.so (sm_100a), exposing the per-time-step right-hand side
 * of the 3-D compressible Navier-Stokes equations on a structured Cartesian grid
 * and the low-storage RK3 update that applies it, as the paper describes the
 * method (arXiv 2304.05494; section 2):
 *   - central energy-preserving split convective flux of order 2L
 *   - WENO characteristic reconstruction where a Ducros-type sensor fires
 *   - viscous terms in Laplacian form, central differences, stretched y
 *   - third-order low-storage Runge-Kutta
 *   - time-step max-reduction
 *   - conserved array w(x,y,z,v) with ghost layers, x unit-stride
 * The paper prints no formulas; the exact reading of each operation is listed in
 * DESIGN.md ("Readings", tags O1..O6 / S1..S16 of SURVEY.md section 8(c)).
 *
 * Conventions
 *   - fp64 everywhere.  Interior arrays are C order [v][k][j][i]
 *     = [5][nz][ny][nx] (conserved rho, rho u, rho v, rho w, rho E) or [nz][ny][nx].
 *   - Every pointer argument says whether it is HOST or DEVICE memory.
 *   - The caller owns the workspace and the CUDA stream and keeps both alive until
 *     streams_destroy.  The library never allocates device memory itself (the fp64 probe
 *     streams_measure_fp64 takes its scratch buffer from the caller as well).
 *   - Host arrays passed in (y_nodes, the structs) are copied before the call returns.
 *   - Calls enqueue work on the caller's stream.  Calls that return host scalars or
 *     copy to host memory synchronise that stream before returning.
 *   - Errors: negative return code, text via streams_last_error(); nothing aborts or
 *     throws across this boundary.  There is no CPU fallback: without a CUDA device
 *     every compute entry point fails with STREAMS_ECUDA.
 * ============================================================================= */
#ifndef STREAMS_H
#define STREAMS_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct streams_ctx streams_ctx; /* opaque, owned by the library */

enum { STREAMS_OK = 0, STREAMS_EINVAL = -1, STREAMS_ENOMEM = -2, STREAMS_ECUDA = -3,
       STREAMS_ESTATE = -4, STREAMS_ENAN = -5 };
enum { STREAMS_BC_PERIODIC = 0, STREAMS_BC_WALL_ISOTHERMAL = 1, STREAMS_BC_FREESTREAM = 2,
       STREAMS_BC_HALO = 3 /* bc_z only: ghost planes delivered by the caller's halo exchange (sharded stepping) */ };
enum { STREAMS_VISC_NONE = 0, STREAMS_VISC_POWER = 1, STREAMS_VISC_SUTHERLAND = 2 };
enum { STREAMS_FLUX_CENTRAL = 0, STREAMS_FLUX_WENO = 1, STREAMS_FLUX_HYBRID = 2 };
enum { STREAMS_WENO_JS = 0, STREAMS_WENO_Z = 1 };

/* Grid ("Cartesian coordinates", "evaluation of grid metrics").
 * Uniform directions: spacing l/n, node i at i*l/n.  y is stretched when y_nodes != NULL. */
typedef struct {
  int nx, ny, nz;
  double lx, ly, lz;          /* domain lengths; ly is the period when y is periodic            */
  const double* y_nodes;      /* HOST, ny node coordinates, NULL = uniform; copied at init      */
  double y_wall_lo, y_wall_hi;/* boundary planes in y for wall / free-stream sides (staggered:  */
                              /* the plane lies midway between the last node and the first ghost)*/
  int bc_x, bc_y_lo, bc_y_hi, bc_z; /* STREAMS_BC_*; walls are supported in y only              */
  double t_wall_lo, t_wall_hi;/* isothermal wall temperatures                                   */
  int nz_global;              /* bc_z == STREAMS_BC_HALO: z nodes of the whole domain, of which this context holds  */
                              /* nz planes (lz is the whole domain's length: dz = lz / nz_global); else 0 (= nz)    */
} streams_grid;

/* Gas and flow parameters (PAPER:36 ideal gas; PAPER:40 calorically perfect branch). */
typedef struct {
  double gamma, rgas, prandtl;
  int visc_law;               /* STREAMS_VISC_*                                                 */
  double mu_ref, t_ref;       /* mu(t_ref) = mu_ref                                             */
  double suth_s_over_tref;    /* Sutherland: mu = mu_ref t^1.5 (1+s)/(t+s), t = T/t_ref         */
  double pow_exp;             /* power law:  mu = mu_ref t^pow_exp                              */
  double u_ref, l_ref;        /* sensor regulariser eps_s = (u_ref/l_ref)^2                     */
  double freestream[5];       /* conserved free-stream state for STREAMS_BC_FREESTREAM ghosts   */
  double accel[3];            /* uniform body acceleration g (PAPER:377 forcing; e.g. the driving  */
                              /* force of a channel): rho g on momentum, (rho u).g on total energy */
} streams_gas;

/* Scheme (PAPER:38 orders "up to 8th and 7th"; production pair 6/5; the paper's order sweep runs the
 * families 2/1/2, 4/3/4, 6/5/6, 8/7/8).  Every combination of central order 2..8, WENO order 1..7 and
 * viscous order 2..8 is accepted; an order the chosen mode does not use is ignored.  The four families above are
 * template instances of their own; a mixed combination runs on the smallest instance that covers it with zero-padded
 * coefficient tables (same numbers, the speed of the covering instance).  The layout carries three ghost layers, four
 * when an order reaches further (central / viscous 8, WENO 7).  Invalid orders make streams_workspace_bytes return 0
 * and streams_init return STREAMS_EINVAL (never later). */
typedef struct {
  int central_order;          /* 2L: 2, 4, 6, 8                                                 */
  int weno_order;             /* 2r-1: 1, 3, 5, 7; ignored when flux_mode == CENTRAL            */
  int visc_order;             /* 2, 4, 6, 8; ignored when visc_law == NONE                      */
  int flux_mode;              /* STREAMS_FLUX_*                                                 */
  double sensor_threshold;    /* node flagged iff theta > threshold (strict)                    */
  double weno_eps;            /* epsilon of the Jiang-Shu weights                               */
  double cfl;                 /* dt = cfl / max rate                                            */
  double dt_fixed;            /* > 0 overrides the CFL time step                                */
  int dt_every;               /* recompute dt every dt_every steps (10 in production)*/
  int weno_variant;           /* STREAMS_WENO_JS (Jiang-Shu weights) or STREAMS_WENO_Z (WENO-Z, S19) */
} streams_scheme;

/* Bytes of DEVICE workspace streams_init needs for this grid/gas/scheme; 0 on invalid input. */
size_t streams_workspace_bytes(const streams_grid* grid, const streams_gas* gas,
                               const streams_scheme* scheme);

/* Create a context.  workspace_dev: DEVICE buffer of at least streams_workspace_bytes(), 256-byte
 * aligned, owned by the caller.  cuda_stream: a cudaStream_t (NULL = default stream).
 * Unsupported order / boundary combinations fail here with STREAMS_EINVAL, not later. */
int streams_init(streams_ctx** out, const streams_grid* grid, const streams_gas* gas,
                 const streams_scheme* scheme, void* workspace_dev, size_t workspace_bytes,
                 void* cuda_stream);

/* Load the conserved state w[5][nz][ny][nx] (interior).  src_is_device: 0 = HOST, 1 = DEVICE.
 * Resets time and the step counter. */
int streams_set_fields(streams_ctx* ctx, const double* w, int src_is_device);

/* One right-hand-side evaluation R(w) of the current state (ghost fill, primitives, sensor,
 * convective x/y/z, viscous).  rhs_out_dev: DEVICE [5][nz][ny][nx], may be NULL.
 * Never changes the interior of w.  STREAMS_ESTATE before streams_set_fields. */
int streams_rhs(streams_ctx* ctx, double* rhs_out_dev);

/* nsteps full RK3 steps (3 RHS + 3 updates each, dt per scheme).  dt_last, time: HOST, nullable.
 * Returns STREAMS_ENAN if the time step or the state became non-finite: the last stage of every step checks the
 * updated state for Inf / NaN, and the time-step rate of every node keeps a NaN (a negative pressure); the error
 * is reported when the call returns (the remaining steps of the call still run). */
int streams_step(streams_ctx* ctx, int nsteps, double* dt_last, double* time);

/* Sharded stepping (PAPER:85 GPU-aware halo communication, PAPER:507 synchronous mode): the domain is cut
 * into z slabs, one context per slab (one process per GPU), each created with bc_z = STREAMS_BC_HALO and its own nz.
 * A slab's z ghost planes then hold its neighbours' first / last `ng` interior planes and are written by the CALLER
 * (a peer copy or an NCCL send / receive of the slabs below), never by the library.  One RK3 step of a slab is, for
 * stage = 0, 1, 2:
 *     streams_shard_fill(ctx, stage, &rate_is_local)   ghost fill of the other directions, primitives
 *       [stage 0, *rate_is_local != 0: max-reduce the double at STREAMS_HALO_RATE over all slabs, in place]
 *       [exchange STREAMS_HALO_PRIMS]
 *     streams_shard_sensor(ctx, stage)                 step scalars (stage 0), sensor, dilatation
 *       [exchange STREAMS_HALO_DIV and STREAMS_HALO_MASK]
 *     streams_shard_rhs(ctx, stage)                    flags, WENO fluxes, fused RHS + update; primitive buffers swap
 * and streams_shard_finish after the last step of a batch (synchronises; dt, time, STREAMS_ENAN as streams_step).
 * Every node is computed by the same arithmetic as in a single context, so a sharded run reproduces the single-GPU
 * run bit for bit (tests/test_gpu_sharded.py).  Only z is cut; x and y keep their boundary conditions.
 * streams_halo_slabs(what): DEVICE pointers of the slabs to exchange for the CURRENT state (call it after every
 * streams_shard_rhs: the primitive buffers swap): *lo_send = this slab's first ng interior planes (they become the
 * upper ghosts of the slab below), *lo_recv = its lower ghost planes, *hi_send / *hi_recv likewise at the upper end;
 * each is `nfields` pieces of `slab_bytes` contiguous bytes, `field_stride_bytes` apart (whole padded planes: the x / y
 * ghosts travel with them).  STREAMS_HALO_RATE: *lo_send = the local time-step rate (8 bytes), nothing else. */
enum { STREAMS_HALO_PRIMS = 0, STREAMS_HALO_DIV = 1, STREAMS_HALO_MASK = 2, STREAMS_HALO_RATE = 3 };
int streams_shard_fill(streams_ctx* ctx, int stage, int* rate_is_local);
int streams_shard_sensor(streams_ctx* ctx, int stage);
int streams_shard_rhs(streams_ctx* ctx, int stage);
int streams_shard_finish(streams_ctx* ctx, double* dt_last, double* time);
int streams_halo_slabs(streams_ctx* ctx, int what, void** lo_send, void** lo_recv, void** hi_send, void** hi_recv,
                       size_t* slab_bytes, int* nfields, size_t* field_stride_bytes);

/* Copy the conserved state out, w_out[5][nz][ny][nx].  dst_is_device: 0 = HOST, 1 = DEVICE. */
int streams_get_fields(streams_ctx* ctx, double* w_out, int dst_is_device);

/* Sensor of the current state: theta_out [nz][ny][nx] doubles and/or mask_out [nz][ny][nx] bytes
 * (1 = node flagged), either may be NULL.  Evaluates ghost fill + primitives + sensor. */
int streams_get_sensor(streams_ctx* ctx, double* theta_out, unsigned char* mask_out,
                       int dst_is_device);

/* Diagnostics of the last RHS evaluation, HOST outputs, nullable: number of flagged nodes, number of
 * nodes next to a flagged interface, and interfaces[3] = flagged interfaces per direction (the paper's
 * "WENO activation"). */
int streams_get_activation(streams_ctx* ctx, long long* flagged_nodes, long long* shock_nodes,
                           long long* interfaces);

/* The same counts summed over every sensor evaluation since streams_set_fields (hybrid mode; zeros
 * otherwise), and the number of evaluations: the activation "is not known a priori and may even vary"
 * (PAPER:497).  HOST outputs, nullable; interfaces_sum has 3 entries.  Synchronises the stream. */
int streams_get_activation_totals(streams_ctx* ctx, long long* flagged_sum, long long* shock_sum,
                                  long long* interfaces_sum, long long* evaluations);

/* Imposes the node mask of the shock sensor (hybrid mode): from the next evaluation on, the sensor still
 * computes theta and the dilatation but flags exactly the nodes with mask[n] != 0 (values must be 0 or 1),
 * mask = [nz][ny][nx] bytes, HOST or DEVICE (copied before return; synchronises the stream for a host source).
 * NULL restores the sensor's own decision.  This is the hook of the paper's activation sweep (PAPER:497-501:
 * WENO forced on a chosen fraction of the points).  STREAMS_EINVAL unless flux_mode == STREAMS_FLUX_HYBRID. */
int streams_set_mask_override(streams_ctx* ctx, const unsigned char* mask, int src_is_device);

/* Replaces the uniform body acceleration streams_gas.accel (3 HOST doubles, copied) from the next evaluation on, and
 * takes it back from the bulk-flow controller if streams_step_forced had been used. */
int streams_set_body_force(streams_ctx* ctx, const double* accel3);

/* nsteps RK3 steps of a forced flow under the bulk-flow controller ("forcing term evaluations (sum
 * reduction)", PAPER:386 force_rhs; reading S18 of DESIGN.md): after every step the volume integrals of mass M and of
 * the momentum P along `direction` (0, 1, 2) are reduced on the device in a fixed order and a one-thread kernel resets
 * the acceleration along `direction`,  g <- [g - (P - P_prev) / (M dt)] + (P_target - P) / (M dt):  the force that would
 * have kept P constant over the step just taken plus what returns P to its target over the next one.  The kernels of
 * the following step read g from device memory; nothing is synchronised with the host between the steps.
 * target: the bulk momentum integral to hold, NaN = keep the one in force (at the first call: the current P).
 * dt_last, time, accel3_out (the acceleration after the last update): HOST, nullable.  Errors as streams_step.
 * A later streams_step keeps the last g; streams_set_body_force returns the acceleration to the host. */
int streams_step_forced(streams_ctx* ctx, int nsteps, int direction, double target, double* dt_last,
                        double* time, double* accel3_out);

/* Sum reductions over the interior nodes (PAPER:218-236 compute_residual; Table 2 "forcing term evaluations (sum
 * reduction)"), in a fixed order: the five doubles of out5 (HOST) are reproducible bit for bit.
 *   STREAMS_SUM_STATE:    out5[q] = sum of w_q dV, dV = dx dz / (d eta/dy)(j): the volume integrals of mass, momentum
 *                         and total energy, i.e. the quantities the scheme conserves discretely in a periodic box;
 *   STREAMS_SUM_RESIDUAL: out5[q] = sum of R_q^2 with R the right-hand side (per unit time) of the CURRENT state as
 *                         evaluated by the last streams_rhs (the paper's residual is entry 1, rho u);
 *                         STREAMS_ESTATE if the state changed since (or no streams_rhs was called).
 * Synchronises the stream. */
enum { STREAMS_SUM_STATE = 0, STREAMS_SUM_RESIDUAL = 1 };
int streams_get_sums(streams_ctx* ctx, int kind, double* out5);

/* The same sum reductions (PAPER:218-236 compute_residual; Table 2 "forcing term evaluations (sum reduction)") for a
 * caller that cannot provide device scratch memory -- no context, no workspace, and the call allocates nothing.
 * Who needs it: everything else in this header runs inside a context whose workspace the caller allocated, and the
 * per-block partial sums of streams_get_sums live there.  That does not suit a program that took all the device memory
 * it may use into its own arena at start-up, a hook that another solver calls in the middle of its time step with
 * borrowed device pointers (cudaMalloc / cudaFree there would synchronise the device and undo the overlap the host
 * application arranged, and a failed allocation would stop the run for the sake of a diagnostic), or a tool that only
 * wants the integrals of a field it already holds.  Here the partial sums go to an array that is part of the library's
 * own device image instead: STREAMS_SUMS_STATIC_MAX_FIELDS x 592 doubles = 75 776 bytes, held on every GPU on which the
 * library's device code is loaded until the process exits.  No cudaMalloc, cudaFree or allocating library routine is
 * called, now or later.
 *   f_dev          DEVICE, nfields arrays [nz][ny][nx] one after the other (C order, no ghost layers): e.g. the w that
 *                  streams_get_fields(.., dst_is_device = 1) wrote, or the rhs_out_dev of streams_rhs.  Read only.
 *   nfields        1 .. STREAMS_SUMS_STATIC_MAX_FIELDS.  The limit is what the static array holds; more fields in one
 *                  call fail with STREAMS_ENOMEM (split the call).  nx, ny, nz are not limited by the scratch.
 *   row_weight_dev DEVICE, ny doubles, or NULL (= 1): the weight of a node of row j for STREAMS_SUM_STATE, i.e. the cell
 *                  volume dx dz / (d eta/dy)(j) if the sums are to be volume integrals.  Ignored by STREAMS_SUM_RESIDUAL.
 *   kind           STREAMS_SUM_STATE: out[q] = sum of f_q * row_weight(j);  STREAMS_SUM_RESIDUAL: out[q] = sum of f_q^2.
 *   out_dev        DEVICE, nfields doubles, written by the last kernel of the call (the call itself does not
 *                  synchronise: read it in stream order).  Owned by the caller like every other argument.
 *   cuda_stream    a cudaStream_t (NULL = default stream) of the CURRENT device; f_dev, row_weight_dev and out_dev must
 *                  be memory of that device.
 *   err, err_len   HOST buffer for the error text, nullable: set to "" on success, to a message on failure (this call
 *                  has no context to keep it in; streams_last_error does not report it).
 * The summation order is that of streams_get_sums, so for the same numbers and weights the results are bit-identical
 * to it and from call to call.  Returns STREAMS_OK once the two kernels are enqueued, STREAMS_EINVAL (null pointer, bad
 * kind, non-positive extent or nfields), STREAMS_ENOMEM (nfields above the maximum), STREAMS_ECUDA.
 * Set-up: the first call on each device looks up the device address of the static array (cudaGetSymbolAddress, with
 * that device current; this may load the library's device code there) and keeps it; make that first call outside any
 * stream capture.  Later calls on that device only launch the two kernels.
 * Sharing: there is ONE such array per device and process, every call uses it and finds the previous call's partials
 * in it.  No call relies on them: each slot is written before it is read within the call, so nothing needs clearing.
 * Calls issued to the same stream are ordered and safe.  Two calls whose kernels may run on the GPU at the same time
 * (different streams without an event between them, different host threads) race on the array and return garbage:
 * order them with an event, or serialise them on one stream. */
#define STREAMS_SUMS_STATIC_MAX_FIELDS 16
int streams_sums_static(const double* f_dev, int nfields, int nx, int ny, int nz, const double* row_weight_dev,
                        int kind, double* out_dev, void* cuda_stream, char* err, size_t err_len);

/* Number of kernels the library has launched on this context since streams_init (kernels replayed from a CUDA graph
 * count one by one), and the number of graph submissions among them: streams_step captures the launches of one RK3
 * step once per variant of its launch sequence and replays them afterwards (small grids cannot hide the
 * launch latency).  Profiling (streams_profile) and the environment variable STREAMS_NO_GRAPH=1 switch the graphs off. */
long long streams_kernel_launches(const streams_ctx* ctx);
long long streams_graph_launches(const streams_ctx* ctx);

/* Per-kernel device timing, the measurement of BASELINE metric part 2 ("per-kernel % of roofline";
 * the paper's analogue is its per-kernel table).  Kernel classes: */
enum { STREAMS_K_FILL_PRIM = 0, STREAMS_K_DT = 1, STREAMS_K_SENSOR = 2, STREAMS_K_FLAGS = 3,
       STREAMS_K_RHS_MAIN = 4, STREAMS_K_WENO = 5, STREAMS_K_CORR = 6, STREAMS_K_MISC = 7,
       STREAMS_K_COUNT = 8 };

/* enable != 0: from now on every launch is bracketed by a CUDA event pair on the context's stream
 * (at most max_records launches between two streams_get_profile calls are recorded, the rest are
 * counted as dropped; max_records <= 0 means 4096).  enable == 0: stop.  Either way the totals are
 * reset.  Synchronises the stream. */
int streams_profile(streams_ctx* ctx, int enable, int max_records);

/* Totals since streams_profile: ms[STREAMS_K_COUNT] device milliseconds and count[STREAMS_K_COUNT]
 * recorded launch groups per class, *dropped = launches not recorded.  HOST outputs, each nullable.
 * Synchronises the stream. */
int streams_get_profile(streams_ctx* ctx, double* ms, long long* count, long long* dropped);

/* Measures the fp64 pipe of the current device, the "alu" roof of SURVEY 8(d): kind 0 = independent DFMA chains,
 * kind 1 = DADD and DMUL alternating.  *ginst_per_s (HOST) receives thread-level fp64 instructions per second in
 * units of 1e9, the best of `repeats` launches timed with CUDA events on `cuda_stream` (each launch runs
 * 8 x 256-thread blocks per SM, 16 chains per thread).  scratch_dev: DEVICE buffer of at least
 * streams_measure_fp64_scratch_bytes() bytes, owned by the caller (the probe stores one double per thread there).
 * Needs no context; synchronises the stream.  Returns STREAMS_EINVAL for a bad kind / null output, STREAMS_ENOMEM for
 * a missing or short scratch buffer, STREAMS_ECUDA on a CUDA error. */
size_t streams_measure_fp64_scratch_bytes(void);
int streams_measure_fp64(void* cuda_stream, int kind, int repeats, void* scratch_dev, size_t scratch_bytes,
                         double* ginst_per_s);

/* Name of a kernel class ("" if out of range); static storage. */
const char* streams_kernel_name(int kind);

/* Text of the last error on this context ("" if none); ctx may be NULL for init failures. */
const char* streams_last_error(const streams_ctx* ctx);

int streams_destroy(streams_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* STREAMS_H */
