// Host-side launch wrappers implemented by the kernel translation units.
// Each returns the number of kernels it launched.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include "streams_dev.cuh"

namespace streams {

// RK stage description for the fused RHS + update kernel.
struct StageArgs {
  double gam, rhk;      // w += dt (gam R + rhk R_prev)            (O5)
  int update_w;         // 0: RHS only (streams_rhs)
  int read_prev;        // stage uses the previous-stage RHS
  int write_r;          // keep R (padded layout, DevP::R) for the next stage
  double* r_dense;      // if not null: also write R here, interior [5][N] (streams_rhs output)
  double* q_out;        // update_w: the primitives of the updated state go here (the other DevP::q buffer)
  int want_rate;        // update_w: also reduce the time-step rate of the updated state into scal[S_RATE]
  int check_state;      // update_w: raise scal[S_NAN] if the updated state holds an Inf or a NaN (last stage of a step)
};

// TMA descriptors of the z-marching kernels (built once per context and primitive buffer by make_march_maps):
// centre planes with halo and ring planes of the primitives, RK operands w and R, the interface-flag bytes of a tile
// plane (hybrid mode); s_*: (u, v, w) boxes of the sensor.
struct MarchMaps { CUtensorMap centre, ring, w, r, flag, s_centre, s_ring; };
// Returns 0, or a negative code: -1 driver entry point missing, -2 encode failed.
int make_march_maps(const DevP& P, MarchMaps* maps);

// Launch wrappers.  Each returns the number of kernels it launched (0 when the mode does not need it), -1 if the
// order combination is outside what is instantiated, -2 if a kernel could not be opted in to its shared memory.
// `configure` = true: launch nothing, only opt the kernels this context will use in to their dynamic shared memory on
// the current device (streams_init); returns 0 or -2.
int launch_fill_prim(const DevP& P, bool with_dt, cudaStream_t st);   // with_dt: also reduce the time-step rate (a9)
int launch_fill_ghosts(const DevP& P, cudaStream_t st);                // ghost shell only (interior primitives already current)
int launch_sensor(const DevP& P, const MarchMaps& maps, int L, bool mask, bool theta, cudaStream_t st, bool configure);
int launch_flags(const DevP& P, int r, cudaStream_t st);
int launch_dt(const DevP& P, double dt_fixed, bool recompute, cudaStream_t st);   // step scalars (dt, time, step count)
// WENO fluxes of the flagged (or all) interfaces, then the per-node gather of their net correction; both run before
int launch_weno(const DevP& P, int L, int r, cudaStream_t st);
int launch_corr(const DevP& P, cudaStream_t st);
// the fused RHS + update over all nodes
int launch_rhs_main(const DevP& P, const MarchMaps& maps, int L, int Lv, const StageArgs& sa, cudaStream_t st, bool configure);
int march_family(int L, int Lv, int ng);
int launch_sums(const DevP& P, int kind, double* partial, double* out, cudaStream_t st);   // streams_get_sums
int sums_scratch_doubles();
int launch_controller(const DevP& P, const double* sums, int d, double target, bool init, cudaStream_t st);   // S18
size_t measure_fp64_scratch_bytes();
double measure_fp64(cudaStream_t st, int kind, int repeats, double* scratch, size_t scratch_bytes);   // streams_measure_fp64

}  // namespace streams
