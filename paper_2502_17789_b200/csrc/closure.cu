// w-stacking closure either side of the hot path: master uv grid <-> image.
//
//   imaging    (Eq. 11 :145-148):  I[j] = corr[j] * sum_layers e^{+2 pi i w0 n'(l_j, m_j)} F^-1{grid[layer]}[j]
//   prediction (Eq. 12 :164-166):  grid[layer] = F{ corr[j] * e^{-2 pi i w0 n'(l_j, m_j)} * I[j] }
//
// with F the CENTRED unnormalised DFT over the Ng x Ng master grid (DC at Ng/2 in both domains, as R1),
// w0 = (wl + 1/2) w_step the layer's w offset (R9), l_j = (j - Ng/2) S / Ng, and corr an optional real
// per-pixel factor the caller supplies (1 / (T_full n_vis) for a dirty image in Jy, 1 / T_full for a model:
// R4 leaves the image-level taper correction to the caller).  Not on the measured hot path; the master-grid
// FFT is cuFFT's (north_star permits it there).  Centred DFT = checkerboard * DFT * checkerboard for even Ng.
#include <cufft.h>

#include <algorithm>

#include "kernels.h"

namespace idg {

namespace {

// e^{sign 2 pi i w0 n'(l, m)} at master-grid pixel (y, x); the phase is reduced to one cycle in fp64
__device__ __forceinline__ float2 w_screen(int x, int y, int Ng, double S, double w0, float sign) {
  if (w0 == 0.0) return make_float2(1.f, 0.f);
  const double l = (x - Ng / 2) * S / Ng, m = (y - Ng / 2) * S / Ng;
  const double r2 = l * l + m * m;
  const double np = -r2 / (1.0 + sqrt(1.0 - r2));      // n' = sqrt(1 - r2) - 1, cancellation-free (R13)
  double ph = w0 * np;
  ph -= rint(ph);
  float s, c;
  sincospif(2.0f * static_cast<float>(ph), &s, &c);
  return make_float2(c, sign * s);
}

__device__ __forceinline__ float2 cmul_(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

// tmp[p, y, x] = (-1)^(x+y) * layer[p, y, x]
__global__ void __launch_bounds__(256) checker_copy(const float2* in, float2* out, int Ng,   // in == out allowed
                                                    int64_t n) {
  for (int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; i < n;
       i += static_cast<int64_t>(gridDim.x) * blockDim.x) {
    const int x = static_cast<int>(i % Ng), y = static_cast<int>((i / Ng) % Ng);
    const float2 v = in[i];
    out[i] = ((x + y) & 1) ? make_float2(-v.x, -v.y) : v;
  }
}

// image[p, y, x] (+)= corr[y, x] * screen(+) * (-1)^(x+y) * tmp[p, y, x]
__global__ void __launch_bounds__(256) accumulate_layer(const float2* __restrict__ tmp, float2* __restrict__ image,
                                                        const float* __restrict__ corr, int Ng, double S, double w0,
                                                        int first) {
  const int64_t plane = static_cast<int64_t>(Ng) * Ng;
  for (int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; i < plane;
       i += static_cast<int64_t>(gridDim.x) * blockDim.x) {
    const int x = static_cast<int>(i % Ng), y = static_cast<int>(i / Ng);
    float2 f = w_screen(x, y, Ng, S, w0, +1.f);
    float k = ((x + y) & 1) ? -1.f : 1.f;
    if (corr) k *= corr[i];
    f = make_float2(f.x * k, f.y * k);
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      const float2 v = cmul_(tmp[p * plane + i], f);
      if (first) image[p * plane + i] = v;
      else image[p * plane + i] = make_float2(image[p * plane + i].x + v.x, image[p * plane + i].y + v.y);
    }
  }
}

// layer[p, y, x] = (-1)^(x+y) * corr[y, x] * screen(-) * image[p, y, x]     (before the forward FFT)
__global__ void __launch_bounds__(256) screen_image(const float2* __restrict__ image, float2* __restrict__ layer,
                                                    const float* __restrict__ corr, int Ng, double S, double w0) {
  const int64_t plane = static_cast<int64_t>(Ng) * Ng;
  for (int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; i < plane;
       i += static_cast<int64_t>(gridDim.x) * blockDim.x) {
    const int x = static_cast<int>(i % Ng), y = static_cast<int>(i / Ng);
    float2 f = w_screen(x, y, Ng, S, w0, -1.f);
    float k = ((x + y) & 1) ? -1.f : 1.f;
    if (corr) k *= corr[i];
    f = make_float2(f.x * k, f.y * k);
#pragma unroll
    for (int p = 0; p < 4; ++p) layer[p * plane + i] = cmul_(image[p * plane + i], f);
  }
}

unsigned blocks_for(int64_t n) { return static_cast<unsigned>(std::min<int64_t>((n + 255) / 256, 148 * 32)); }

}  // namespace

// cuFFT plan of 4 planes of Ng x Ng, created once per idg_plan (closure_plan_destroy frees it).
int closure_plan_create(int Ng, void** out) {
  cufftHandle h;
  int n[2] = {Ng, Ng};
  if (cufftPlanMany(&h, 2, n, nullptr, 1, Ng * Ng, nullptr, 1, Ng * Ng, CUFFT_C2C, 4) != CUFFT_SUCCESS) return -1;
  *out = new cufftHandle(h);
  return 0;
}
void closure_plan_destroy(void* p) {
  if (!p) return;
  cufftDestroy(*static_cast<cufftHandle*>(p));
  delete static_cast<cufftHandle*>(p);
}

cudaError_t launch_grid_to_image(void* fft_plan, const float2* grid, const float* corr, float2* image, float2* tmp,
                                 int Ng, int n_layers, int wl_min, double w_step, double S, cudaStream_t stream) {
  cufftHandle h = *static_cast<cufftHandle*>(fft_plan);
  if (cufftSetStream(h, stream) != CUFFT_SUCCESS) return cudaErrorUnknown;
  const int64_t plane = static_cast<int64_t>(Ng) * Ng;
  for (int k = 0; k < n_layers; ++k) {
    const double w0 = w_step > 0.0 ? (wl_min + k + 0.5) * w_step : 0.0;
    checker_copy<<<blocks_for(4 * plane), 256, 0, stream>>>(grid + k * 4 * plane, tmp, Ng, 4 * plane);
    if (cufftExecC2C(h, reinterpret_cast<cufftComplex*>(tmp), reinterpret_cast<cufftComplex*>(tmp), CUFFT_INVERSE) !=
        CUFFT_SUCCESS)
      return cudaErrorUnknown;
    accumulate_layer<<<blocks_for(plane), 256, 0, stream>>>(tmp, image, corr, Ng, S, w0, k == 0);
    count_launch(2);
  }
  return cudaGetLastError();
}

cudaError_t launch_image_to_grid(void* fft_plan, const float2* image, const float* corr, float2* grid, int Ng,
                                 int n_layers, int wl_min, double w_step, double S, cudaStream_t stream) {
  cufftHandle h = *static_cast<cufftHandle*>(fft_plan);
  if (cufftSetStream(h, stream) != CUFFT_SUCCESS) return cudaErrorUnknown;
  const int64_t plane = static_cast<int64_t>(Ng) * Ng;
  for (int k = 0; k < n_layers; ++k) {
    const double w0 = w_step > 0.0 ? (wl_min + k + 0.5) * w_step : 0.0;
    float2* layer = grid + k * 4 * plane;
    screen_image<<<blocks_for(plane), 256, 0, stream>>>(image, layer, corr, Ng, S, w0);
    if (cufftExecC2C(h, reinterpret_cast<cufftComplex*>(layer), reinterpret_cast<cufftComplex*>(layer),
                     CUFFT_FORWARD) != CUFFT_SUCCESS)
      return cudaErrorUnknown;
    checker_copy<<<blocks_for(4 * plane), 256, 0, stream>>>(layer, layer, Ng, 4 * plane);
    count_launch(2);
  }
  return cudaGetLastError();
}

}  // namespace idg
