// idg_power_norm_average_static: the power-normalisation average (§3.3, R22) for callers that
// must not allocate device memory.
//
// Who that is.  An imager that runs this library next to its own work usually hands the whole device to one
// pool at start-up (the master grids of a 32k^2 IQUV image alone fill a 40 GB card), so a
// raw cudaMalloc from inside a library call fails although the pool has room; and cudaMalloc / cudaFree
// synchronise the whole device, which stalls gridding batches in flight on the caller's other streams --
// exactly what happens when the correction image of one major cycle is prepared while the next cycle's
// batches already run.  idg_power_norm_average allocates three buffers per call and frees them after a
// stream synchronise; this entry point allocates nothing and frees nothing.
//
// How.  The kernels are the ones idg_power_norm_average runs (direct_f64.cu: one fp64 partial sum per pixel
// and per slice of the (p, q, interval) list, then a sum over the slices in fixed order).  Their scratch -- the
// kPowerNormSlices x L x L partial sums -- lives in the file-scope device array below instead of a per-call
// allocation; the (p, q, interval) list and its weights, which the allocating call builds and uploads itself,
// are inputs here (idg_plan_power_norm_terms lists them on the host).
//
// The array's name is only a handle in host code; the kernels need its device address, which
// cudaGetSymbolAddress gives per device.  That lookup is the one-time set-up of a device's first call.
#include <cuda_runtime.h>

#include <mutex>
#include <string>

#include "idg_b200.h"
#include "idg_internal.h"
#include "kernels.h"

namespace idg {
namespace {

constexpr int kStaticMaxL = IDG_STATIC_MAX_SUBGRID_SIZE;
constexpr size_t kStaticScratchDoubles = static_cast<size_t>(kPowerNormSlices) * kStaticMaxL * kStaticMaxL;

// 64 slices x 96 x 96 pixels x 8 B = 4.5 MiB, held by every device that loads the library until the process
// exits.  Every call writes the entries it later reads, so nothing here has to start at zero; what a call
// leaves behind is overwritten by the next one.  Calls that overlap on one device share it and race.
static __device__ __align__(256) double g_power_norm_scratch[kStaticScratchDoubles];

constexpr int kMaxDevices = 64;
std::mutex g_scratch_mu;
double* g_scratch_addr[kMaxDevices] = {};   // device address of the array, per device ordinal

// Device address of g_power_norm_scratch on the current device, looked up once per device.
cudaError_t scratch_address(double** out, std::string* why) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { *why = "cudaGetDevice"; return e; }
  if (dev < 0 || dev >= kMaxDevices) { *why = "device ordinal beyond the table of 64 devices"; return cudaErrorInvalidDevice; }
  std::lock_guard<std::mutex> lock(g_scratch_mu);
  if (g_scratch_addr[dev] == nullptr) {
    double* p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_power_norm_scratch);
    if (e != cudaSuccess) { *why = "cudaGetSymbolAddress(g_power_norm_scratch)"; return e; }
    if (p == nullptr) { *why = "cudaGetSymbolAddress returned a null address"; return cudaErrorInvalidSymbol; }
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return cudaSuccess;
}

}  // namespace
}  // namespace idg

using namespace idg;

extern "C" {

int idg_plan_power_norm_terms(const idg_plan* plan, int32_t* pairs_host, double* weights_host, int64_t capacity,
                              int64_t* n_terms, double* weight_sum) {
  if (!plan || capacity < 0 || (capacity > 0 && (!pairs_host || !weights_host))) {
    set_error("idg_plan_power_norm_terms: bad argument");
    return IDG_EINVAL;
  }
  // planned visibilities per (baseline, interval): the weights of PAPER.md:257's average (R22); the factor is
  // the same for every subgrid of a (baseline, interval), conjugated or not
  const int32_t n_int = plan->n_intervals;
  std::vector<double> w(static_cast<size_t>(plan->par.n_baselines) * n_int, 0.0);
  for (int64_t s = 0; s < plan->n_subgrids; ++s) {
    const int32_t* e = &plan->sub[static_cast<size_t>(s) * 8];
    w[static_cast<size_t>(e[0]) * n_int + e[1] / plan->par.aterm_period] += static_cast<double>(e[2]) * e[4];
  }
  int64_t n = 0;
  double wsum = 0.0;
  for (size_t i = 0; i < w.size(); ++i) {
    if (w[i] == 0.0) continue;
    if (n < capacity) {
      const size_t b = i / n_int;
      pairs_host[n * 3] = plan->baselines[b * 2];
      pairs_host[n * 3 + 1] = plan->baselines[b * 2 + 1];
      pairs_host[n * 3 + 2] = static_cast<int32_t>(i % n_int);
      weights_host[n] = w[i];
    }
    wsum += w[i];
    ++n;
  }
  if (n_terms) *n_terms = n;
  if (weight_sum) *weight_sum = wsum;
  if (capacity > 0 && n > capacity) {
    set_error("idg_plan_power_norm_terms: " + std::to_string(n) + " terms, room for " + std::to_string(capacity));
    return IDG_ENOMEM;
  }
  return IDG_OK;
}

int idg_power_norm_average_static(const void* aterms_dev, int32_t subgrid_size, int32_t n_intervals,
                                  const int32_t* pairs_dev, const double* weights_dev, int64_t n_terms,
                                  double weight_sum, double* avg_dev, void* cuda_stream) {
  if (!aterms_dev || !pairs_dev || !weights_dev || !avg_dev) {
    set_error("idg_power_norm_average_static: null argument");
    return IDG_EINVAL;
  }
  if (subgrid_size < 2 || (subgrid_size & 1) || n_intervals < 1 || n_terms < 1 || !(weight_sum > 0.0)) {
    set_error("idg_power_norm_average_static: subgrid_size must be even and >= 2, n_intervals >= 1, n_terms >= 1, weight_sum > 0");
    return IDG_EINVAL;
  }
  if (subgrid_size > kStaticMaxL) {
    set_error("idg_power_norm_average_static: subgrid_size " + std::to_string(subgrid_size) +
              " is beyond the built-in scratch (IDG_STATIC_MAX_SUBGRID_SIZE = " + std::to_string(kStaticMaxL) +
              "); use idg_power_norm_average, which allocates its own");
    return IDG_EUNSUPPORTED;
  }
  double* scratch = nullptr;
  std::string why;
  cudaError_t e = scratch_address(&scratch, &why);
  if (e != cudaSuccess) {
    set_error("idg_power_norm_average_static: " + why + ": " + cudaGetErrorString(e));
    return IDG_ECUDA;
  }
  e = launch_power_norm_average(static_cast<const float4*>(aterms_dev), subgrid_size, n_intervals, pairs_dev,
                                weights_dev, n_terms, weight_sum, scratch, avg_dev,
                                static_cast<cudaStream_t>(cuda_stream));
  if (e != cudaSuccess) {
    set_error(std::string("idg_power_norm_average_static: kernel launch: ") + cudaGetErrorString(e));
    return IDG_ECUDA;
  }
  return IDG_OK;
}

}  // extern "C"
