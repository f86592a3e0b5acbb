// streams_sums_static (include/streams.h): the fixed-order field sums of streams_get_sums (PAPER:218-236
// "compute_residual"; Table 2 "forcing term evaluations (sum reduction)") for a caller that has no device memory to give.
//
// Why this exists.  Every other compute call of the library works inside a context whose workspace the caller sized with
// streams_workspace_bytes and allocated itself; the per-block partial sums of the reduction live in that workspace.  Some
// users of the sums cannot do that:
//   - a code that grabbed the device memory it is allowed to use at start-up (an arena, a memory pool with a hard
//     budget) and has no allocation left to hand out for somebody else's scratch;
//   - a hook that runs in the middle of another solver's time step (a residual monitor, a coupling layer) on borrowed
//     device pointers: cudaMalloc / cudaFree there would synchronise the whole device and serialise streams that the
//     host application overlaps on purpose, and a failed allocation would take the run down for a diagnostic;
//   - a post-processing tool that only wants the integrals of a field it already holds and has no reason to build a
//     solver context (several hundred bytes per node) to get them.
// For them the partials live in the file-scope device array below: 75 776 bytes that every GPU on which this library's
// device code gets loaded keeps until the process exits.  The entry point calls no cudaMalloc, cudaFree, cudaMallocAsync
// nor any library routine that allocates; the caller passes the field, the optional weights and the result buffer.
//
// Same summation order as sum_partial_kernel / sum_final_kernel of streams_canon.cu (block b owns the rows b, b + 592,
// ...; a thread strides its row; xor shuffle tree; warps in index order; blocks in index order), written with explicit
// round-to-nearest multiplies and adds so that no contraction setting can change it: on the same numbers the two paths
// return the same bits (tests/test_zz_no_alloc.py).  This unit shares no code with streams_canon.cu: the two constants
// below restate its SUM_BLOCKS / SUM_THREADS and the test fails if they drift apart.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../include/streams.h"

namespace {

constexpr int SUM_BLOCKS = 592, SUM_THREADS = 256;
constexpr int MAX_FIELDS = STREAMS_SUMS_STATIC_MAX_FIELDS;

// The scratch: partial[q * SUM_BLOCKS + b] = sum of field q over the rows of block b.  Every slot a call reads is
// written earlier in the same call (all 592 blocks store their partial of each of the nfields fields, rows or no rows),
// so nothing here has to start at zero and nothing is cleared; what a previous call left is overwritten or never read.
// One array per device and process: two calls whose kernels can be on the GPU at the same time (different streams,
// different host threads) would write the same slots -- see the header for the rule.
static __device__ __align__(256) double g_sums_scratch[MAX_FIELDS * SUM_BLOCKS];

// In host code `g_sums_scratch` is only a handle for the runtime, not a device address: the address a kernel can use
// comes from cudaGetSymbolAddress, per device, with that device current.  Looked up once per device and kept here.
constexpr int MAX_DEVICES = 64;
std::mutex g_setup_mutex;
double* g_scratch_addr[MAX_DEVICES] = {};

cudaError_t scratch_of_current_device(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> hold(g_setup_mutex);
  if (dev >= 0 && dev < MAX_DEVICES && g_scratch_addr[dev]) {
    *out = g_scratch_addr[dev];
    return cudaSuccess;
  }
  double* p = nullptr;
  e = cudaGetSymbolAddress((void**)&p, g_sums_scratch);      // set-up: loads this unit's device code on `dev` if needed
  if (e != cudaSuccess) return e;
  if (!p) return cudaErrorInvalidSymbol;
  if (dev >= 0 && dev < MAX_DEVICES) g_scratch_addr[dev] = p; // (a device index past the table is looked up every call)
  *out = p;
  return cudaSuccess;
}

// KIND 0: sum of f * weight(j) (weight 1 when wy is null), KIND 1: sum of f^2.  One field after the other, each in the
// order described at the top of the file.
template <int KIND>
__global__ void __launch_bounds__(SUM_THREADS)
sums_static_partial_kernel(const double* __restrict__ f, int nfields, int nx, int ny, int nz,
                           const double* __restrict__ wy, double* __restrict__ partial) {
  __shared__ double sm[SUM_THREADS / 32];
  const long long rows = (long long)ny * nz;
  const size_t field = (size_t)rows * (size_t)nx;
  for (int q = 0; q < nfields; ++q) {
    double acc = 0.0;
    for (long long row = blockIdx.x; row < rows; row += gridDim.x) {
      const int j = (int)(row % ny);
      const double wgt = (KIND == 0 && wy) ? wy[j] : 1.0;
      const double* __restrict__ p = f + (size_t)q * field + (size_t)row * (size_t)nx;
      for (int i = threadIdx.x; i < nx; i += SUM_THREADS) {
        const double v = p[i];
        acc = __dadd_rn(acc, KIND == 0 ? __dmul_rn(v, wgt) : __dmul_rn(v, v));
      }
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) acc = __dadd_rn(acc, __shfl_xor_sync(0xffffffffu, acc, s));
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
      double v = 0.0;
      for (int w = 0; w < SUM_THREADS / 32; ++w) v = __dadd_rn(v, sm[w]);
      partial[q * SUM_BLOCKS + blockIdx.x] = v;
    }
    __syncthreads();                                          // sm is reused by the next field
  }
}

__global__ void sums_static_final_kernel(const double* __restrict__ partial, int nfields, double* __restrict__ out) {
  if ((int)threadIdx.x < nfields) {
    double v = 0.0;
    for (int b = 0; b < SUM_BLOCKS; ++b) v = __dadd_rn(v, partial[threadIdx.x * SUM_BLOCKS + b]);
    out[threadIdx.x] = v;
  }
}

int refuse(char* err, size_t err_len, int code, const char* msg, const char* detail = "") {
  if (err && err_len) std::snprintf(err, err_len, "streams_sums_static: %s%s", msg, detail);
  return code;
}

}  // namespace

extern "C" int streams_sums_static(const double* f_dev, int nfields, int nx, int ny, int nz, const double* row_weight_dev,
                                   int kind, double* out_dev, void* cuda_stream, char* err, size_t err_len) {
  if (err && err_len) err[0] = '\0';
  if (!f_dev || !out_dev) return refuse(err, err_len, STREAMS_EINVAL, "f_dev and out_dev must not be null");
  if (kind != STREAMS_SUM_STATE && kind != STREAMS_SUM_RESIDUAL)
    return refuse(err, err_len, STREAMS_EINVAL, "kind must be STREAMS_SUM_STATE or STREAMS_SUM_RESIDUAL");
  if (nfields < 1) return refuse(err, err_len, STREAMS_EINVAL, "nfields must be at least 1");
  if (nfields > MAX_FIELDS) {
    char detail[96];
    std::snprintf(detail, sizeof detail, " (asked for %d, the static scratch array holds the partial sums of %d)", nfields,
                  MAX_FIELDS);
    return refuse(err, err_len, STREAMS_ENOMEM, "more than STREAMS_SUMS_STATIC_MAX_FIELDS fields in one call", detail);
  }
  if (nx < 1 || ny < 1 || nz < 1) return refuse(err, err_len, STREAMS_EINVAL, "grid extents must be positive");

  double* scratch = nullptr;
  cudaError_t e = scratch_of_current_device(&scratch);
  if (e != cudaSuccess) return refuse(err, err_len, STREAMS_ECUDA, "cudaGetSymbolAddress of the scratch array: ", cudaGetErrorString(e));

  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (kind == STREAMS_SUM_STATE)
    sums_static_partial_kernel<0><<<SUM_BLOCKS, SUM_THREADS, 0, st>>>(f_dev, nfields, nx, ny, nz, row_weight_dev, scratch);
  else
    sums_static_partial_kernel<1><<<SUM_BLOCKS, SUM_THREADS, 0, st>>>(f_dev, nfields, nx, ny, nz, nullptr, scratch);
  sums_static_final_kernel<<<1, 32, 0, st>>>(scratch, nfields, out_dev);
  e = cudaGetLastError();
  if (e != cudaSuccess) return refuse(err, err_len, STREAMS_ECUDA, "kernel launch: ", cudaGetErrorString(e));
  return STREAMS_OK;
}
