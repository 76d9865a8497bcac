// Empirical ALU peaks of the device, the way the paper measures its Table 1 (§5.1 :339-351
// "empirical peak" by micro-benchmark): register-only loops of independent FFMA / FFMA2 / MUFU
// chains, one resident wave of full blocks, timed with clock64() inside the kernel (per SM: last warp
// out minus first warp in, since the warp arbiter does not serve warps evenly), so the result is in
// lane-operations per SM clock and does not depend on the clock the run happened to get.
// These numbers are the denominators of the ALU roofline in DESIGN.md and bench.py.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <vector>

#include "kernels.h"

namespace idg {
namespace {

constexpr int kThreads = 256;
constexpr int kChains = 8;

// MODE 0: FFMA   (kChains independent chains, 1 FMA per lane per instruction)
// MODE 1: FFMA2  (packed fp32x2: 2 FMA per lane per instruction)
// MODE 2: MUFU.EX2
// MODE 3: sin.approx + cos.approx  (FMUL.RZ + MUFU.SIN, FMUL.RZ + MUFU.COS)
// MODE 4: the gridder's mix per pixel pair: 2 x (FFMA, sincos) + 16 FFMA2
// MODE 5: the same with 32 scalar FFMA;  MODE 6: sincos + head/remainder split only
__device__ __forceinline__ float ex2(float x) {
  float y;
  asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

template <int MODE>
__global__ void __launch_bounds__(kThreads) peak_kernel(int iters, float seed, float* sink, long long* stamps) {
  float2 a[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) a[i] = make_float2(seed + i + threadIdx.x * 1e-3f, seed - i);
  const float2 m = make_float2(1.0f - seed * 1e-6f, 1.0f + seed * 1e-6f);
  const float2 c = make_float2(seed * 1e-7f, -seed * 1e-7f);
  __syncthreads();
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
    if (MODE == 0) {
#pragma unroll
      for (int i = 0; i < kChains; ++i) { a[i].x = fmaf(a[i].x, m.x, c.x); a[i].y = fmaf(a[i].y, m.y, c.y); }
    } else if (MODE == 1) {
#pragma unroll
      for (int i = 0; i < kChains; ++i) { a[i] = __ffma2_rn(a[i], m, c); a[i] = __ffma2_rn(a[i], m, c); }
    } else if (MODE == 2) {
#pragma unroll
      for (int i = 0; i < kChains; ++i) { a[i].x = ex2(a[i].x); a[i].y = ex2(a[i].y); }
    } else if (MODE == 3) {
#pragma unroll
      for (int i = 0; i < kChains; ++i) { float s, co; __sincosf(a[i].x, &s, &co); a[i].x = s; a[i].y += co; }
    } else if (MODE == 5) {
      // the same mix with scalar FFMA instead of FFMA2 (32 FFMA per pixel pair)
      float s0, c0, s1, c1;
      __sincosf(fmaf(a[0].x, m.x, c.x), &s0, &c0);
      __sincosf(fmaf(a[0].y, m.y, c.y), &s1, &c1);
#pragma unroll
      for (int i = 0; i < kChains; ++i) {
        a[i].x = fmaf(m.x, c0, a[i].x); a[i].y = fmaf(m.y, c1, a[i].y);
        a[i].x = fmaf(c.x, s0, a[i].x); a[i].y = fmaf(c.y, s1, a[i].y);
      }
    } else if (MODE == 6) {
      // operand generation only (a tensor-core formulation would take the MACs): per pixel
      // phase FFMA + sincos + split of cos and sin into a 19-bit head and an exact remainder
#pragma unroll
      for (int i = 0; i < kChains; ++i) {
        float s0, c0;
        __sincosf(fmaf(a[i].x, m.x, c.x), &s0, &c0);
        const float ch = __uint_as_float(__float_as_uint(c0) & 0xffffe000u);
        const float sh = __uint_as_float(__float_as_uint(s0) & 0xffffe000u);
        a[i].x = (c0 - ch) + sh;
        a[i].y += (s0 - sh) + ch;
      }
    } else {
      // one pixel pair: phases for two pixels, two sincos, 16 FFMA2 into 8 float2 accumulators
      float s0, c0, s1, c1;
      __sincosf(fmaf(a[0].x, m.x, c.x), &s0, &c0);
      __sincosf(fmaf(a[0].y, m.y, c.y), &s1, &c1);
      const float2 cc = make_float2(c0, c1), ss = make_float2(s0, s1);
#pragma unroll
      for (int i = 0; i < kChains; ++i) { a[i] = __ffma2_rn(m, cc, a[i]); a[i] = __ffma2_rn(c, ss, a[i]); }
    }
  }
  const long long t1 = clock64();
  float acc = 0.f;
#pragma unroll
  for (int i = 0; i < kChains; ++i) acc += a[i].x + a[i].y;
  if (acc == 123.456f) sink[0] = acc;
  if (threadIdx.x % 32 == 0) {
    unsigned smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    long long* o = stamps + (static_cast<long long>(blockIdx.x) * (kThreads / 32) + threadIdx.x / 32) * 3;
    o[0] = smid; o[1] = t0; o[2] = t1;
  }
}

constexpr int kMaxSm = 256;

template <int MODE>
cudaError_t run(int blocks_per_sm, int n_sm, int iters, float* sink, long long* stamps_dev, double* mean_cycles) {
  const int blocks = blocks_per_sm * n_sm;
  const int n_warps = blocks * (kThreads / 32);
  peak_kernel<MODE><<<blocks, kThreads>>>(iters, 1.0f, sink, stamps_dev);   // warm-up
  peak_kernel<MODE><<<blocks, kThreads>>>(iters, 1.0f, sink, stamps_dev);
  cudaError_t e = cudaDeviceSynchronize();
  if (e != cudaSuccess) return e;
  std::vector<long long> host(static_cast<size_t>(n_warps) * 3);
  e = cudaMemcpy(host.data(), stamps_dev, sizeof(long long) * host.size(), cudaMemcpyDeviceToHost);
  if (e != cudaSuccess) return e;
  // per SM: busy window = last warp out - first warp in; work = warps that ran there
  long long lo[kMaxSm], hi[kMaxSm];
  int cnt[kMaxSm];
  for (int i = 0; i < kMaxSm; ++i) { lo[i] = INT64_MAX; hi[i] = INT64_MIN; cnt[i] = 0; }
  for (int w = 0; w < n_warps; ++w) {
    const int sm = static_cast<int>(host[w * 3]) % kMaxSm;
    lo[sm] = std::min(lo[sm], host[w * 3 + 1]);
    hi[sm] = std::max(hi[sm], host[w * 3 + 2]);
    ++cnt[sm];
  }
  // cycles per warp-slot, averaged over SMs, scaled to the nominal warps per SM
  double s = 0;
  int used = 0;
  const double nominal = static_cast<double>(blocks_per_sm) * (kThreads / 32);
  for (int i = 0; i < kMaxSm; ++i)
    if (cnt[i] > 0) { s += static_cast<double>(hi[i] - lo[i]) * nominal / cnt[i]; ++used; }
  *mean_cycles = s / used;
  return cudaSuccess;
}

}  // namespace

// out[0..6]: lane-operations per clock per SM for FFMA, FFMA2 (counted as 2 FMA per lane), MUFU.EX2,
// sincos pairs (one sin + one cos = 1), and (vis,pixel) pairs per clock per SM for the gridder mix.
cudaError_t measure_alu_peaks(double* out) {
  int dev = 0, n_sm = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  const int bps = 4, iters = 4096;                     // 4 x 256 threads per SM = 8 warps per SMSP
  float* sink = nullptr;
  long long* cyc = nullptr;
  if ((e = cudaMalloc(&sink, 16)) != cudaSuccess) return e;
  if ((e = cudaMalloc(&cyc, sizeof(long long) * 3 * bps * n_sm * (kThreads / 32))) != cudaSuccess) { cudaFree(sink); return e; }
  double mc[7] = {0, 0, 0, 0, 0, 0, 0};
  e = run<0>(bps, n_sm, iters, sink, cyc, &mc[0]);
  if (e == cudaSuccess) e = run<1>(bps, n_sm, iters, sink, cyc, &mc[1]);
  if (e == cudaSuccess) e = run<2>(bps, n_sm, iters, sink, cyc, &mc[2]);
  if (e == cudaSuccess) e = run<3>(bps, n_sm, iters, sink, cyc, &mc[3]);
  if (e == cudaSuccess) e = run<4>(bps, n_sm, iters, sink, cyc, &mc[4]);
  if (e == cudaSuccess) e = run<5>(bps, n_sm, iters, sink, cyc, &mc[5]);
  if (e == cudaSuccess) e = run<6>(bps, n_sm, iters, sink, cyc, &mc[6]);
  cudaFree(sink);
  cudaFree(cyc);
  if (e != cudaSuccess) return e;
  const double lanes = static_cast<double>(bps) * kThreads * iters;   // lane-iterations per SM
  out[0] = lanes * kChains * 2 / mc[0];          // FFMA: 2 per chain per iteration
  out[1] = lanes * kChains * 4 / mc[1];          // FFMA2: 2 instructions x 2 FMA
  out[2] = lanes * kChains * 2 / mc[2];          // MUFU.EX2
  out[3] = lanes * kChains / mc[3];              // sincos pairs
  out[4] = lanes * 2 / mc[4];                    // (vis,pixel) pairs: two per iteration
  out[5] = lanes * 2 / mc[5];
  out[6] = lanes * kChains / mc[6];
  count_launch(14);
  return cudaSuccess;
}

}  // namespace idg
