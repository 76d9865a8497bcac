// Launcher interface between the C-ABI layer (api.cu) and the kernels.  Plain structs of device
// pointers and sizes; every launcher enqueues on `stream` and returns the cudaError_t of the
// launch.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "idg_internal.h"

namespace idg {

struct SubgridJob {
  const int32_t* meta;      // [n_subgrids, kMetaStride] device
  const double* uvw;        // [n_rows, 3] metres
  const double* kappa;      // [n_chan]
  const float* nprime;      // [L, L] n'(l, m) at the subgrid pixels
  const float4* aterms;     // [n_st, n_int, L, L, 2] rows of the 2x2 Jones matrices
  const float* taper;       // [L, L]
  const float* weights;     // [n_rows, n_chan] imaging weights applied at load, or nullptr
  int64_t first;            // first subgrid (global index) of the range the launch belongs to
  int64_t count;            // blocks' worth of subgrids in this launch
  const int32_t* index;     // nullptr: block i handles subgrid first + i; else first + index[i] (kernel choice
                            // per subgrid, PAPER.md:247 fn 7); the subgrid's slot in the stack is the same offset
  int32_t subgrid_size, grid_size, n_times, n_chan, n_intervals;
  int32_t max_nt;           // upper bound of nt over subgrids = min(n_times, aterm_period)
  double image_size;        // S
  double w_step;
  double dkappa;            // kappa[c + 1] - kappa[c] when the channels are uniformly spaced, else 0
  float dkappa_f;           // the same rounded to fp32 (a constant-bank operand of the rotating gridder)
  int32_t power_norm;       // imaging: divide the sandwich by || M_p M_q^H ||_F per pixel (R22)
};

// offset of a block's subgrid within the launch's range
__device__ __forceinline__ int64_t job_slot(const SubgridJob& job, unsigned block) {
  return job.index != nullptr ? static_cast<int64_t>(job.index[block]) : static_cast<int64_t>(block);
}

// steps a1-a3: stage visibilities, direct sum (Eq. 10), A-term sandwich and taper.
// out [count, 4, L, L] complex64.
cudaError_t launch_gridder(const SubgridJob& job, const float4* vis, float2* out, cudaStream_t stream);

// the same with the 2x2 complex MACs on the tensor cores (tcgen05, A operand generated into TMEM)
cudaError_t launch_gridder_tc(const SubgridJob& job, const float4* vis, float2* out, cudaStream_t stream);

// steps a8-a9: taper + A-term on image-domain subgrids, then the per-visibility sum (Eq. 13).
// in [count, 4, L, L] complex64; vis [n_rows, n_chan, 4] complex64.
cudaError_t launch_degridder(const SubgridJob& job, const float2* in, float4* vis, cudaStream_t stream);

// the same with the MACs on the tensor cores (thread = visibility, pixels streamed through shared memory)
cudaError_t launch_degridder_tc(const SubgridJob& job, const float2* in, float4* vis, cudaStream_t stream);

// steps a4 / a7: centred L x L DFT of n_planes planes in place, scaled by 1/L^2.
cudaError_t launch_subgrid_fft(int L, int64_t n_planes, float2* planes, int direction, cudaStream_t stream);

// steps a6 + a7 in one pass: the inverse transform reads the master grid patch under each subgrid
// (the splitter's gather) instead of the stack, and writes the image-domain subgrid to the stack.
cudaError_t launch_split_ifft(const int32_t* meta, int64_t first, int64_t count, int L, int Ng, const float2* grid,
                              float2* subgrids, cudaStream_t stream);

// step a5: tile-owner adder.  csr lists, per non-empty tile, the subgrids overlapping it.
// subgrids: the stack of subgrids [first, first + count)
cudaError_t launch_adder(const int32_t* meta, const DeviceCsr& csr, int64_t first, int64_t count, int L, int Ng,
                         int tiles_x, int tiles_y, const float2* subgrids, float2* grid,
                         cudaStream_t stream);

// dst[i] += src[i] over n complex samples
cudaError_t launch_grid_add(const float2* src, float2* dst, int64_t n, cudaStream_t stream);

// step a6: splitter (gather).
cudaError_t launch_splitter(const int32_t* meta, int64_t first, int64_t count, int L, int Ng,
                            const float2* grid, float2* subgrids, cudaStream_t stream);

// w-stacking closure (closure.cu; outside the hot path, master-grid FFT by cuFFT).  `fft_plan` comes from
// closure_plan_create (one per idg_plan).  tmp: [4, Ng, Ng] complex64 scratch.
int  closure_plan_create(int Ng, void** out);
void closure_plan_destroy(void* fft_plan);
cudaError_t launch_grid_to_image(void* fft_plan, const float2* grid, const float* corr, float2* image, float2* tmp,
                                 int Ng, int n_layers, int wl_min, double w_step, double S, cudaStream_t stream);
cudaError_t launch_image_to_grid(void* fft_plan, const float2* image, const float* corr, float2* grid, int Ng,
                                 int n_layers, int wl_min, double w_step, double S, cudaStream_t stream);

// fp64 SIMT variants of the two direct sums with their A-term / taper step (direct_f64.cu).
// OUT / IN = double2 keeps fp64 end to end (stage calls), float2 rounds to the complex64 stack / table.
cudaError_t launch_gridder_f64(const SubgridJob& job, const float4* vis, float2* out32, double2* out64, cudaStream_t stream);
cudaError_t launch_degridder_f64(const SubgridJob& job, const float2* in32, const double2* in64, float4* vis32,
                                 double2* vis64, cudaStream_t stream);

// weighted average of 1 / || M_p M_q^H ||_F over (baseline, interval) pairs (R22):
// pairs [n_pairs, 3] int32 (p, q, it), weights [n_pairs] double, avg [L*L] double = sum w f / sum w
cudaError_t launch_power_norm_average(const float4* aterms, int L, int n_intervals, const int32_t* pairs,
                                      const double* weights, int64_t n_pairs, double wsum, double* scratch,
                                      double* avg, cudaStream_t stream);

constexpr int kPowerNormSlices = 64;   // slices of the (p, q, it) list, each one partial sum per pixel

// records which direct-sum kernel ran (idg_kernel_config_mask)
void note_kernel(int kind, int bit);

// Empirical FFMA / FFMA2 / MUFU rates per SM clock (peaks.cu); synchronous.
cudaError_t measure_alu_peaks(double* out5);

void count_launch(int n = 1);

}  // namespace idg
