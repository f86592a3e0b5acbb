// Host-side launch wrappers implemented by the kernel translation units.
// Each returns the number of kernels it launched.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include "streams_dev.cuh"

namespace streams {

// RK stage description for the fused RHS + update kernels.
struct StageArgs {
  double gam, rhk;      // w += dt (gam R + rhk R_prev)            (O5)
  int update_w;         // 0: RHS only (streams_rhs)
  int read_prev;        // stage uses the previous-stage RHS
  int write_r;          // keep R (padded layout, DevP::R) for the next stage
  double* r_dense;      // if not null: also write R here, interior [5][N] (streams_rhs output)
  double* q_out;        // update_w: the primitives of the updated state go here (the other DevP::q buffer)
  int want_rate;        // update_w: also reduce the time-step rate of the updated state into scal[S_RATE]
};




// TMA descriptors of the fused RHS kernel (built once per context by make_march_maps):
// centre planes with halo and ring planes of the primitives, RK operands w and R.
struct MarchMaps { CUtensorMap centre, ring, w, r, s_centre, s_ring; };   // centre / ring / s_*: views of ONE q buffer   // s_*: (u, v, w) boxes of the sensor kernel
// Returns 0, or a negative code: -1 driver entry point missing, -2 encode failed.
int make_march_maps(const DevP& P, MarchMaps* maps);

int launch_fill_prim(const DevP& P, bool with_dt, cudaStream_t st);   // with_dt: also reduce the time-step rate (a9)
int launch_fill_ghosts(const DevP& P, cudaStream_t st);                // ghost shell only (interior primitives already current)
int launch_sensor(const DevP& P, const MarchMaps& maps, int L, bool mask, bool theta, cudaStream_t st);
int launch_flags(const DevP& P, int L, int r, cudaStream_t st);
int launch_dt(const DevP& P, double dt_fixed, bool recompute, cudaStream_t st);   // step scalars (dt, time, step count)
// The per-interface WENO flux corrections (run first) and the fused RHS + update over all nodes; each
// returns the number of launches (0 when the flux mode does not need it) or < 0 if the (L, Lv, r)
// combination is not instantiated.
int launch_weno(const DevP& P, int L, int Lv, int r, cudaStream_t st);
int launch_rhs_main(const DevP& P, const MarchMaps& maps, int L, int Lv, int r, const StageArgs& sa, cudaStream_t st);
int launch_sums(const DevP& P, int kind, double* partial, double* out, cudaStream_t st);   // streams_get_sums
int sums_scratch_doubles();
double measure_fp64(cudaStream_t st, int kind, int repeats);   // streams_measure_fp64
bool rhs_supported(int L, int Lv, int r, int flux_mode, int visc_law);

}  // namespace streams
