// fp64 variants of the two direct sums with their A-term / taper step.
//
//   gridder  : S[y,x]  = sum_k V_k exp(+2 pi i phi_k(y,x)),  S' = taper * M_p S M_q^H   (Eq. 10 :133-137, :156)
//   degridder: S'      = M_p (taper S) M_q^H,  V_k = sum_{y,x} S'[y,x] exp(-2 pi i phi_k(y,x))   (Eq. 13 :171-174)
//
// The paper runs its accuracy experiments with double-precision kernels (§4.1 :289-293) and reports them
// about 4.5x slower than single precision (§5.3 :371).  These are plain SIMT kernels for accuracy work at
// sizes the CPU oracle cannot reach: the phase is formed in fp64 from the fp64 uvw table exactly as written
// in Eq. 10 (no slope / offset split, no fixed-point reduction: fp64 has the digits), sincospi() gives
// sin and cos, and the 2x2 complex MACs accumulate in fp64 registers.  Inputs are the path's own (complex64
// visibilities and A-terms, float32 taper); outputs are complex128 (stage calls) or rounded once to the
// complex64 stack / visibility table (IDG_VARIANT_FP64 inside idg_grid / idg_degrid).
#include "kernels.h"

namespace idg {

namespace {

constexpr int kT = 256;          // threads per block
constexpr int kPixStage = 128;   // degridder: pixels staged per step

struct cd { double x, y; };
__device__ __forceinline__ cd cmul(cd a, cd b) { return {a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x}; }
__device__ __forceinline__ cd cmulc(cd a, cd b) { return {a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y}; }   // a conj(b)
__device__ __forceinline__ cd cadd(cd a, cd b) { return {a.x + b.x, a.y + b.y}; }

// z = t * Mp x Mq^H (row-major 2x2 complex); norm != 0 divides by || Mp Mq^H ||_F (R22)
__device__ __forceinline__ void sandwich64(const cd x[4], const float4 mp0, const float4 mp1, const float4 mq0,
                                           const float4 mq1, double t, bool norm, cd z[4]) {
  const cd a{mp0.x, mp0.y}, b{mp0.z, mp0.w}, c{mp1.x, mp1.y}, d{mp1.z, mp1.w};
  const cd q00{mq0.x, mq0.y}, q01{mq0.z, mq0.w}, q10{mq1.x, mq1.y}, q11{mq1.z, mq1.w};
  if (norm) {
    const cd p00 = cadd(cmulc(a, q00), cmulc(b, q01)), p01 = cadd(cmulc(a, q10), cmulc(b, q11));
    const cd p10 = cadd(cmulc(c, q00), cmulc(d, q01)), p11 = cadd(cmulc(c, q10), cmulc(d, q11));
    t /= sqrt(p00.x * p00.x + p00.y * p00.y + p01.x * p01.x + p01.y * p01.y + p10.x * p10.x + p10.y * p10.y +
              p11.x * p11.x + p11.y * p11.y);
  }
  const cd y00 = cadd(cmul(a, x[0]), cmul(b, x[2])), y01 = cadd(cmul(a, x[1]), cmul(b, x[3]));
  const cd y10 = cadd(cmul(c, x[0]), cmul(d, x[2])), y11 = cadd(cmul(c, x[1]), cmul(d, x[3]));
  cd r;
  r = cadd(cmulc(y00, q00), cmulc(y01, q01)); z[0] = {t * r.x, t * r.y};
  r = cadd(cmulc(y00, q10), cmulc(y01, q11)); z[1] = {t * r.x, t * r.y};
  r = cadd(cmulc(y10, q00), cmulc(y11, q01)); z[2] = {t * r.x, t * r.y};
  r = cadd(cmulc(y10, q10), cmulc(y11, q11)); z[3] = {t * r.x, t * r.y};
}

struct Sub {
  int b, t0, nt, c0, nc, sp, sq, it;
  bool conj;
  double u0, v0, w0;
  int64_t row0;
};

__device__ __forceinline__ Sub read_sub(const SubgridJob& job, int64_t sg) {
  const int32_t* m = job.meta + (job.first + sg) * kMetaStride;
  const int L = job.subgrid_size;
  Sub s;
  s.b = m[0]; s.t0 = m[1]; s.nt = m[2]; s.c0 = m[3]; s.nc = m[4];
  s.sp = m[8]; s.sq = m[9]; s.it = m[10];
  s.conj = (m[12] & kMetaConj) != 0;
  s.u0 = (m[5] + L / 2 - job.grid_size / 2) / job.image_size;
  s.v0 = (m[6] + L / 2 - job.grid_size / 2) / job.image_size;
  s.w0 = job.w_step > 0.0 ? (m[7] + 0.5) * job.w_step : 0.0;
  s.row0 = static_cast<int64_t>(s.b) * job.n_times + s.t0;
  return s;
}

// direction cosines of subgrid pixel (y, x): R3, R13
__device__ __forceinline__ void pixel_lmn(const SubgridJob& job, int pix, double* l, double* m, double* n1) {
  const int L = job.subgrid_size;
  *l = (pix % L - L / 2) * job.image_size / L;
  *m = (pix / L - L / 2) * job.image_size / L;
  const double r2 = *l * *l + *m * *m;
  *n1 = -r2 / (1.0 + sqrt(1.0 - r2));
}

__global__ void __launch_bounds__(kT) gridder_f64_kernel(const SubgridJob job, const float4* __restrict__ vis,
                                                         float2* __restrict__ out32, double2* __restrict__ out64) {
  const int64_t sg = job_slot(job, blockIdx.x);
  const Sub s = read_sub(job, sg);
  const int L = job.subgrid_size;
  const double sgn = s.conj ? -1.0 : 1.0;
  const float4* __restrict__ ap = job.aterms + (static_cast<int64_t>(s.sp) * job.n_intervals + s.it) * (L * L * 2);
  const float4* __restrict__ aq = job.aterms + (static_cast<int64_t>(s.sq) * job.n_intervals + s.it) * (L * L * 2);
  for (int pix = threadIdx.x; pix < L * L; pix += kT) {
    double l, m, n1;
    pixel_lmn(job, pix, &l, &m, &n1);
    cd acc[4] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
    for (int r = 0; r < s.nt; ++r) {
      const double* uvw = job.uvw + (s.row0 + r) * 3;
      const double um = sgn * uvw[0], vm = sgn * uvw[1], wm = sgn * uvw[2];
      for (int c = 0; c < s.nc; ++c) {
        const double kap = job.kappa[s.c0 + c];
        const double phi = (um * kap - s.u0) * l + (vm * kap - s.v0) * m + (wm * kap - s.w0) * n1;   // cycles
        double sn, cs;
        sincospi(2.0 * phi, &sn, &cs);
        const float4* v = vis + ((s.row0 + r) * job.n_chan + s.c0 + c) * 2;
        const float4 v01 = __ldg(&v[0]), v23 = __ldg(&v[1]);
        double wgt = 1.0;
        if (job.weights != nullptr) wgt = __ldg(&job.weights[(s.row0 + r) * job.n_chan + s.c0 + c]);
        cd x[4] = {{v01.x, v01.y}, {v01.z, v01.w}, {v23.x, v23.y}, {v23.z, v23.w}};
        if (s.conj) {                                   // V^dagger = conj of (XX, YX, XY, YY)
          const cd t1 = x[1];
          x[0].y = -x[0].y; x[3].y = -x[3].y;
          x[1] = {x[2].x, -x[2].y};
          x[2] = {t1.x, -t1.y};
        }
#pragma unroll
        for (int p = 0; p < 4; ++p) {
          // weight 0 = flagged: an exact zero whatever the sample holds
          const double re = wgt == 0.0 ? 0.0 : x[p].x * wgt, im = wgt == 0.0 ? 0.0 : x[p].y * wgt;
          acc[p].x += re * cs - im * sn;
          acc[p].y += re * sn + im * cs;
        }
      }
    }
    cd z[4];
    sandwich64(acc, __ldg(&ap[pix * 2]), __ldg(&ap[pix * 2 + 1]), __ldg(&aq[pix * 2]), __ldg(&aq[pix * 2 + 1]),
               static_cast<double>(__ldg(&job.taper[pix])), job.power_norm != 0, z);
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      const int64_t o = (sg * 4 + p) * L * L + pix;
      if (out64 != nullptr) out64[o] = make_double2(z[p].x, z[p].y);
      else out32[o] = make_float2(static_cast<float>(z[p].x), static_cast<float>(z[p].y));
    }
  }
}

__global__ void __launch_bounds__(kT) degridder_f64_kernel(const SubgridJob job, const float2* __restrict__ in32,
                                                           const double2* __restrict__ in64,
                                                           float4* __restrict__ vis32, double2* __restrict__ vis64) {
  __shared__ cd spix[kPixStage][4];
  __shared__ double slmn[kPixStage][3];
  const int64_t sg = job_slot(job, blockIdx.x);
  const Sub s = read_sub(job, sg);
  const int L = job.subgrid_size;
  const double sgn = s.conj ? -1.0 : 1.0;
  const float4* __restrict__ ap = job.aterms + (static_cast<int64_t>(s.sp) * job.n_intervals + s.it) * (L * L * 2);
  const float4* __restrict__ aq = job.aterms + (static_cast<int64_t>(s.sq) * job.n_intervals + s.it) * (L * L * 2);
  const int K = s.nt * s.nc;
  for (int kb = 0; kb < K; kb += kT) {
    const int k = kb + threadIdx.x;
    const bool on = k < K;
    double du = 0, dv = 0, dw = 0;
    int r = 0, c = 0;
    if (on) {
      r = k / s.nc; c = k - r * s.nc;
      const double* uvw = job.uvw + (s.row0 + r) * 3;
      const double kap = job.kappa[s.c0 + c];
      du = sgn * uvw[0] * kap - s.u0;
      dv = sgn * uvw[1] * kap - s.v0;
      dw = sgn * uvw[2] * kap - s.w0;
    }
    cd acc[4] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
    for (int p0 = 0; p0 < L * L; p0 += kPixStage) {
      __syncthreads();
      if (threadIdx.x < kPixStage) {
        const int pix = p0 + threadIdx.x;
        cd x[4], z[4];
#pragma unroll
        for (int p = 0; p < 4; ++p) {
          const int64_t o = (sg * 4 + p) * L * L + pix;
          if (in64 != nullptr) { const double2 v = in64[o]; x[p] = {v.x, v.y}; }
          else { const float2 v = __ldg(&in32[o]); x[p] = {v.x, v.y}; }
        }
        // M_p (t S) M_q^H == t (M_p S M_q^H); prediction is not power-normalised (R22)
        sandwich64(x, __ldg(&ap[pix * 2]), __ldg(&ap[pix * 2 + 1]), __ldg(&aq[pix * 2]), __ldg(&aq[pix * 2 + 1]),
                   static_cast<double>(__ldg(&job.taper[pix])), false, z);
#pragma unroll
        for (int p = 0; p < 4; ++p) spix[threadIdx.x][p] = z[p];
        pixel_lmn(job, pix, &slmn[threadIdx.x][0], &slmn[threadIdx.x][1], &slmn[threadIdx.x][2]);
      }
      __syncthreads();
      if (on) {
        for (int i = 0; i < kPixStage; ++i) {
          const double phi = du * slmn[i][0] + dv * slmn[i][1] + dw * slmn[i][2];
          double sn, cs;
          sincospi(2.0 * phi, &sn, &cs);
#pragma unroll
          for (int p = 0; p < 4; ++p) {                 // S' (cos - i sin)
            acc[p].x += spix[i][p].x * cs + spix[i][p].y * sn;
            acc[p].y += spix[i][p].y * cs - spix[i][p].x * sn;
          }
        }
      }
    }
    if (on) {
      if (s.conj) {                                     // (XX, XY, YX, YY) <- conj of (XX, YX, XY, YY)
        const cd t1 = acc[1];
        acc[0].y = -acc[0].y; acc[3].y = -acc[3].y;
        acc[1] = {acc[2].x, -acc[2].y};
        acc[2] = {t1.x, -t1.y};
      }
      const int64_t o = ((s.row0 + r) * job.n_chan + s.c0 + c) * 4;
      if (vis64 != nullptr) {
#pragma unroll
        for (int p = 0; p < 4; ++p) vis64[o + p] = make_double2(acc[p].x, acc[p].y);
      } else {
        float4* o4 = vis32 + o / 2;
        o4[0] = make_float4(static_cast<float>(acc[0].x), static_cast<float>(acc[0].y), static_cast<float>(acc[1].x),
                            static_cast<float>(acc[1].y));
        o4[1] = make_float4(static_cast<float>(acc[2].x), static_cast<float>(acc[2].y), static_cast<float>(acc[3].x),
                            static_cast<float>(acc[3].y));
      }
    }
  }
}

// one thread per pixel, one block row per slice of the (p, q, it) list; fp64 partial sums in fixed order
__global__ void __launch_bounds__(kT) power_norm_partial_kernel(const float4* __restrict__ aterms, int L, int n_intervals,
                                                                const int32_t* __restrict__ pairs,
                                                                const double* __restrict__ weights, int64_t n_pairs,
                                                                int n_slices, double* __restrict__ scratch) {
  const int pix = blockIdx.x * kT + threadIdx.x;
  if (pix >= L * L) return;
  const int64_t per = (n_pairs + n_slices - 1) / n_slices;
  const int64_t i0 = blockIdx.y * per, i1 = min(n_pairs, i0 + per);
  double acc = 0.0;
  for (int64_t i = i0; i < i1; ++i) {
    const int p = pairs[i * 3], q = pairs[i * 3 + 1], it = pairs[i * 3 + 2];
    const float4* ap = aterms + (static_cast<int64_t>(p) * n_intervals + it) * (L * L * 2) + pix * 2;
    const float4* aq = aterms + (static_cast<int64_t>(q) * n_intervals + it) * (L * L * 2) + pix * 2;
    const cd one[4] = {{1, 0}, {0, 0}, {0, 0}, {1, 0}};
    cd z[4];
    // || Mp Mq^H ||_F = || Mp I Mq^H ||_F: the sandwich of the identity
    sandwich64(one, __ldg(&ap[0]), __ldg(&ap[1]), __ldg(&aq[0]), __ldg(&aq[1]), 1.0, false, z);
    const double n2 = z[0].x * z[0].x + z[0].y * z[0].y + z[1].x * z[1].x + z[1].y * z[1].y + z[2].x * z[2].x +
                      z[2].y * z[2].y + z[3].x * z[3].x + z[3].y * z[3].y;
    acc += weights[i] / sqrt(n2);
  }
  scratch[static_cast<int64_t>(blockIdx.y) * L * L + pix] = acc;
}

__global__ void power_norm_reduce_kernel(const double* __restrict__ scratch, int n_pix, int n_slices, double wsum,
                                         double* __restrict__ avg) {
  const int pix = blockIdx.x * blockDim.x + threadIdx.x;
  if (pix >= n_pix) return;
  double acc = 0.0;
  for (int s = 0; s < n_slices; ++s) acc += scratch[static_cast<int64_t>(s) * n_pix + pix];
  avg[pix] = acc / wsum;
}

}  // namespace

cudaError_t launch_gridder_f64(const SubgridJob& job, const float4* vis, float2* out32, double2* out64,
                               cudaStream_t stream) {
  if (job.count == 0) return cudaSuccess;
  gridder_f64_kernel<<<static_cast<unsigned>(job.count), kT, 0, stream>>>(job, vis, out32, out64);
  count_launch();
  note_kernel(IDG_K_GRIDDER, IDG_KMASK_FP64);
  return cudaGetLastError();
}

cudaError_t launch_degridder_f64(const SubgridJob& job, const float2* in32, const double2* in64, float4* vis32,
                                 double2* vis64, cudaStream_t stream) {
  if (job.count == 0) return cudaSuccess;
  degridder_f64_kernel<<<static_cast<unsigned>(job.count), kT, 0, stream>>>(job, in32, in64, vis32, vis64);
  count_launch();
  note_kernel(IDG_K_DEGRIDDER, IDG_KMASK_FP64);
  return cudaGetLastError();
}

cudaError_t launch_power_norm_average(const float4* aterms, int L, int n_intervals, const int32_t* pairs,
                                      const double* weights, int64_t n_pairs, double wsum, double* scratch,
                                      double* avg, cudaStream_t stream) {
  const int n_pix = L * L;
  const dim3 grid((n_pix + kT - 1) / kT, kPowerNormSlices);
  power_norm_partial_kernel<<<grid, kT, 0, stream>>>(aterms, L, n_intervals, pairs, weights, n_pairs, kPowerNormSlices,
                                                     scratch);
  power_norm_reduce_kernel<<<(n_pix + kT - 1) / kT, kT, 0, stream>>>(scratch, n_pix, kPowerNormSlices, wsum, avg);
  count_launch(2);
  return cudaGetLastError();
}

}  // namespace idg
