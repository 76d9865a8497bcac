// Gridder: steps a1-a3 of the hot path.
//
//   S[y,x] = sum_{t,c} V[r,c] exp(+2 pi i phi),  phi = (u-u0) l_x + (v-v0) m_y + (w-w0) n'
//                                                    (Eq. 10 :133-137; 2x2 per :253)
//   S'     = taper * M_p S M_q^H                       (PAPER.md :156, §3.3 :251-257)
//
// Launch geometry follows the paper's (§3.2.1 :206-231): one subgrid per block row, threads own
// pixels and keep their accumulators in registers, visibilities are staged through shared
// memory.  What differs on sm_100a:
//   * a thread owns P pixels of one column, and pixel PAIRS share one FFMA2 (packed fp32x2,
//     new on sm_100): the 16 real FMAs of a 2x2 complex MAC become 8 issue slots, so the FP32
//     pipe (not the issue port) is the limit.  The staged visibilities are stored as
//     (re,re,im,im) per polarisation so both halves of an FFMA2 see the same multiplier.
//   * the paper's "phase per row in metres, times 1/lambda in the inner loop" (:231) is kept in
//     a cancellation-free form: per (row, pixel) a slope a = 2 pi (u_m l + v_m m + w_m n') and
//     an offset b = 2 pi phi(kappa_ref) are set up once, the inner loop is one FFMA
//     phi = a * (kappa_c - kappa_ref) + b.  b is reduced modulo one cycle exactly, in 32-bit
//     fixed point (alpha_fix * ix + beta_fix * iy wraps), so |phi| stays a few cycles and
//     __sincosf's own range reduction stays accurate.
#include "device_math.cuh"
#include "kernels.h"

namespace idg {

namespace {

constexpr int kChunk = 64;   // channels staged per chunk (one table row at a time)

struct RowData {
  int32_t alpha_fix, beta_fix;   // (u-u0) S/L and (v-v0) S/L at kappa_ref, cycles/pixel * 2^32 (wrapping)
  float gamma;                   // 2 pi (w kappa_ref - w0)
  float us, vs, ws;              // 2 pi u_m S/L, 2 pi v_m S/L, 2 pi w_m   [rad per unit kappa]
};

template <int L, int T, int P>
__global__ void __launch_bounds__(T) gridder_kernel(const SubgridJob job, const float4* __restrict__ vis,
                                                    float2* __restrict__ out) {
  static_assert(T % L == 0 && (L * L) % (T * P) == 0 && P % 2 == 0 && T >= 2 * kChunk, "launch shape");
  constexpr int PIECES = (L * L) / (T * P);
  constexpr int YSTEP = T / L;

  __shared__ __align__(16) float4 svis[2][kChunk][4];
  __shared__ float sdk[2][kChunk];
  __shared__ RowData srow[2];

  const int tid = threadIdx.x;
  const int64_t sg = job_slot(job, blockIdx.x / PIECES);
  const int piece = blockIdx.x % PIECES;
  const int32_t* __restrict__ m = job.meta + (job.first + sg) * kMetaStride;
  const int b = m[0], t0 = m[1], nt = m[2], c0 = m[3], nc = m[4], x0 = m[5], y0 = m[6], wl = m[7];
  const int sp = m[8], sq = m[9], it = m[10];
  const bool conj = (m[12] & kMetaConj) != 0;          // rows used as (-u,-v,-w) with V^dagger (PAPER.md:178 fn 4, R21)

  const double S = job.image_size;
  const double u0 = (x0 + L / 2 - job.grid_size / 2) / S;
  const double v0 = (y0 + L / 2 - job.grid_size / 2) / S;
  const double w0 = job.w_step > 0.0 ? (wl + 0.5) * job.w_step : 0.0;
  const int cref = c0 + nc / 2;
  const double kref = job.kappa[cref];

  const int ix = tid % L;
  const int iy0 = piece * (T * P / L) + tid / L;
  const float fx = static_cast<float>(ix - L / 2);
  float np[P];
#pragma unroll
  for (int j = 0; j < P; ++j) np[j] = job.nprime[(iy0 + j * YSTEP) * L + ix];

  float2 are[4][P / 2], aim[4][P / 2];
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int j = 0; j < P / 2; ++j) are[p][j] = aim[p][j] = make_float2(0.f, 0.f);

  const int cpr = (nc + kChunk - 1) / kChunk;   // chunks per row
  const int nchunks = nt * cpr;
  const int64_t row0 = static_cast<int64_t>(b) * job.n_times + t0;

  // --- staging (step a1): visibilities of one table row chunk -> smem, plus the row constants.
  float4 pre = make_float4(0.f, 0.f, 0.f, 0.f);
  auto stage_load = [&](int ci) {
    const int r = ci / cpr, cc = (ci % cpr) * kChunk;
    const int cnt = min(kChunk, nc - cc);
    if (tid < 2 * cnt) {
      if (!conj) {
        pre = __ldg(&vis[((row0 + r) * job.n_chan + c0 + cc) * 2 + tid]);
      } else {
        // V^dagger = conj of (XX, YX, XY, YY): this thread's pair is (XX, YX)* or (XY, YY)*
        const float2* v2 = reinterpret_cast<const float2*>(vis) + ((row0 + r) * job.n_chan + c0 + cc + (tid >> 1)) * 4;
        const float2 a = __ldg(&v2[tid & 1]), b2 = __ldg(&v2[2 + (tid & 1)]);
        pre = make_float4(a.x, -a.y, b2.x, -b2.y);
      }
      if (job.weights != nullptr) {                     // weighting at load
        const float wgt = __ldg(&job.weights[(row0 + r) * job.n_chan + c0 + cc + (tid >> 1)]);
        // weight 0 = flagged: an exact zero whatever the sample holds (NaN * 0 would poison the pixel sums)
        pre = wgt == 0.f ? make_float4(0.f, 0.f, 0.f, 0.f) : make_float4(pre.x * wgt, pre.y * wgt, pre.z * wgt, pre.w * wgt);
      }
    }
  };
  auto stage_store = [&](int ci, int buf) {
    const int r = ci / cpr, cc = (ci % cpr) * kChunk;
    const int cnt = min(kChunk, nc - cc);
    if (tid < 2 * cnt) {
      // (re0, im0, re1, im1) of two polarisations -> (re,re,im,im) each
      svis[buf][tid >> 1][(tid & 1) * 2 + 0] = make_float4(pre.x, pre.x, pre.y, pre.y);
      svis[buf][tid >> 1][(tid & 1) * 2 + 1] = make_float4(pre.z, pre.z, pre.w, pre.w);
    }
    if (tid < cnt) sdk[buf][tid] = static_cast<float>(job.kappa[c0 + cc + tid] - kref);
    if (tid == T - 1) {
      const double* uvw = job.uvw + (row0 + r) * 3;
      const double sgn = conj ? -1.0 : 1.0;
      const double um = sgn * uvw[0], vm = sgn * uvw[1], wm = sgn * uvw[2];
      const double two_pi = 6.283185307179586476925286766559;
      const double sl = S / L;
      const double alpha = (um * kref - u0) * sl, beta = (vm * kref - v0) * sl;
      RowData rd;
      rd.alpha_fix = static_cast<int32_t>(static_cast<uint32_t>(static_cast<int64_t>(rint(alpha * 4294967296.0))));
      rd.beta_fix = static_cast<int32_t>(static_cast<uint32_t>(static_cast<int64_t>(rint(beta * 4294967296.0))));
      rd.gamma = static_cast<float>(two_pi * (wm * kref - w0));
      rd.us = static_cast<float>(two_pi * um * sl);
      rd.vs = static_cast<float>(two_pi * vm * sl);
      rd.ws = static_cast<float>(two_pi * wm);
      srow[buf] = rd;
    }
  };

  float pa[P], pb[P];
  if (nchunks > 0) {
    stage_load(0);
    stage_store(0, 0);
  }
  __syncthreads();

  for (int ci = 0; ci < nchunks; ++ci) {
    const int buf = ci & 1;
    const bool has_next = ci + 1 < nchunks;
    if (has_next) stage_load(ci + 1);

    if (ci % cpr == 0) {
      // per-(row, pixel) slope and offset of the phase; amortised over the row's channels
      const RowData rd = srow[buf];
      const float ax = rd.us * fx;
      const uint32_t bx = static_cast<uint32_t>(rd.alpha_fix) * static_cast<uint32_t>(ix - L / 2);   // unsigned: meant to wrap
#pragma unroll
      for (int j = 0; j < P; ++j) {
        const int iy = iy0 + j * YSTEP - L / 2;
        pa[j] = fmaf(rd.vs, static_cast<float>(iy), fmaf(rd.ws, np[j], ax));
        const int32_t bf = static_cast<int32_t>(bx + static_cast<uint32_t>(rd.beta_fix) * static_cast<uint32_t>(iy));   // exact mod 1 cycle
        pb[j] = fmaf(rd.gamma, np[j], static_cast<float>(bf) * 1.4629180792671596e-9f);  // 2 pi / 2^32
      }
    }

    const int cnt = min(kChunk, nc - (ci % cpr) * kChunk);
#pragma unroll 2
    for (int c = 0; c < cnt; ++c) {
      const float dk = sdk[buf][c];
      const float4 v0 = svis[buf][c][0], v1 = svis[buf][c][1], v2 = svis[buf][c][2], v3 = svis[buf][c][3];
#pragma unroll
      for (int j = 0; j < P / 2; ++j) {
        float s0, c0_, s1, c1_;
        __sincosf(fmaf(pa[2 * j], dk, pb[2 * j]), &s0, &c0_);
        __sincosf(fmaf(pa[2 * j + 1], dk, pb[2 * j + 1]), &s1, &c1_);
        const float2 cc2 = make_float2(c0_, c1_), ss2 = make_float2(s0, s1);
#define IDG_MAC(POL, V)                                                        \
        are[POL][j] = ffma2(make_float2(V.x, V.y), cc2, are[POL][j]);           \
        are[POL][j] = ffma2(neg2(make_float2(V.z, V.w)), ss2, are[POL][j]);     \
        aim[POL][j] = ffma2(make_float2(V.x, V.y), ss2, aim[POL][j]);           \
        aim[POL][j] = ffma2(make_float2(V.z, V.w), cc2, aim[POL][j]);
        IDG_MAC(0, v0) IDG_MAC(1, v1) IDG_MAC(2, v2) IDG_MAC(3, v3)
#undef IDG_MAC
      }
    }

    if (has_next) stage_store(ci + 1, buf ^ 1);
    __syncthreads();
  }

  // --- epilogue (step a3): A-term sandwich and taper, once per pixel.
  const float4* __restrict__ ap = job.aterms + (static_cast<int64_t>(sp) * job.n_intervals + it) * (L * L * 2);
  const float4* __restrict__ aq = job.aterms + (static_cast<int64_t>(sq) * job.n_intervals + it) * (L * L * 2);
  float2* __restrict__ o = out + sg * 4 * L * L;
#pragma unroll
  for (int j = 0; j < P; ++j) {
    const int pix = (iy0 + j * YSTEP) * L + ix;
    float2 x[4], z[4];
#pragma unroll
    for (int p = 0; p < 4; ++p)
      x[p] = (j & 1) ? make_float2(are[p][j / 2].y, aim[p][j / 2].y) : make_float2(are[p][j / 2].x, aim[p][j / 2].x);
    const float4 mp0 = __ldg(&ap[pix * 2]), mp1 = __ldg(&ap[pix * 2 + 1]);
    const float4 mq0 = __ldg(&aq[pix * 2]), mq1 = __ldg(&aq[pix * 2 + 1]);
    float t = __ldg(&job.taper[pix]);
    if (job.power_norm) t *= frobenius_inv(mp0, mp1, mq0, mq1);        // PAPER.md:257, R22
    sandwich(x, mp0, mp1, mq0, mq1, t, z);
#pragma unroll
    for (int p = 0; p < 4; ++p) o[p * L * L + pix] = z[p];
  }
}

template <int L, int T, int P>
cudaError_t launch(const SubgridJob& job, const float4* vis, float2* out, cudaStream_t stream) {
  constexpr int PIECES = (L * L) / (T * P);
  const int64_t blocks = job.count * PIECES;
  if (blocks == 0) return cudaSuccess;
  gridder_kernel<L, T, P><<<static_cast<unsigned>(blocks), T, 0, stream>>>(job, vis, out);
  count_launch();
  note_kernel(IDG_K_GRIDDER, IDG_KMASK_SIMT);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_gridder(const SubgridJob& job, const float4* vis, float2* out, cudaStream_t stream) {
  switch (job.subgrid_size) {
    case 32:  return launch<32, 128, 8>(job, vis, out, stream);
    case 48:  return launch<48, 192, 6>(job, vis, out, stream);
    case 64:  return launch<64, 256, 8>(job, vis, out, stream);
    case 96:  return launch<96, 384, 8>(job, vis, out, stream);
    case 128: return launch<128, 256, 8>(job, vis, out, stream);
    case 160: return launch<160, 320, 8>(job, vis, out, stream);
    default:  return cudaErrorInvalidValue;
  }
}

}  // namespace idg
