// Degridder: steps a8-a9 of the hot path.
//
//   S'      = M_p (taper * S) M_q^H                                   (Eq. 13 :173; R4, R5)
//   V[r,c]  = sum_{y,x} S'[y,x] exp(-2 pi i phi),  phi as in the gridder  (Eq. 13 :171-174)
//
// The paper's degridder keeps the gridder's pixel-parallel geometry and pays a warp-level
// reduction per visibility (§3.2.2 :233-249), because a thread-per-visibility kernel starves on
// sparsely occupied subgrids.  Here one block owns one subgrid and BOTH axes are split: the
// lanes of a warp own visibilities (PV each, accumulators in registers, pairs of visibilities
// sharing one FFMA2), and the warps of the block are spread over pixel slices when the subgrid
// has too few visibilities to fill them.  The slices are summed once per visibility through
// shared memory at the end, in a fixed order (deterministic).  Pixels are staged through shared
// memory in chunks, already multiplied by taper and A-terms, stored (re,re,im,im) per
// polarisation so both halves of an FFMA2 see the same multiplier.
#include "device_math.cuh"
#include "kernels.h"

namespace idg {

namespace {

constexpr int kPixChunk = 256;   // pixels staged per chunk
constexpr int kSeg = 16;         // pixels of one subgrid row handled by one warp at a time

template <int L, int T, int PV>
__global__ void __launch_bounds__(T) degridder_kernel(const SubgridJob job, const float2* __restrict__ in,
                                                      float4* __restrict__ vis) {
  static_assert(L % kSeg == 0 && (L * L) % kPixChunk == 0 && PV % 2 == 0, "shape");
  constexpr int NW = T / 32;
  constexpr int NSEG = kPixChunk / kSeg;
  constexpr int NCHUNK = L * L / kPixChunk;

  __shared__ __align__(16) float4 spix[kPixChunk][5];   // 4 x (re,re,im,im) + (n', n', fx, fx), fx within the segment
  __shared__ __align__(16) float4 sred[T][2];

  const int tid = threadIdx.x, warp = tid / 32, lane = tid % 32;
  const int64_t sg = job_slot(job, blockIdx.x);
  const int32_t* __restrict__ m = job.meta + (job.first + sg) * kMetaStride;
  const int b = m[0], t0 = m[1], nt = m[2], c0 = m[3], nc = m[4], x0 = m[5], y0 = m[6], wl = m[7];
  const int sp = m[8], sq = m[9], it = m[10];
  // rows used as (-u,-v,-w) of the swapped baseline: the sum predicts V(-u,-v,-w) of (q,p) and its dagger is
  // written (PAPER.md:178 fn 4, R21)
  const bool conj = (m[12] & kMetaConj) != 0;
  const double sgn = conj ? -1.0 : 1.0;

  const double S = job.image_size;
  const double u0 = (x0 + L / 2 - job.grid_size / 2) / S;
  const double v0 = (y0 + L / 2 - job.grid_size / 2) / S;
  const double w0 = job.w_step > 0.0 ? (wl + 0.5) * job.w_step : 0.0;
  const int64_t row0 = static_cast<int64_t>(b) * job.n_times + t0;

  const float4* __restrict__ ap = job.aterms + (static_cast<int64_t>(sp) * job.n_intervals + it) * (L * L * 2);
  const float4* __restrict__ aq = job.aterms + (static_cast<int64_t>(sq) * job.n_intervals + it) * (L * L * 2);
  const float2* __restrict__ sub = in + sg * 4 * L * L;

  const int K = nt * nc;
  const int n_vt = (K + PV - 1) / PV;        // visibility-threads needed
  const int VW = (n_vt + 31) / 32;           // visibility-warps needed
  const int VWB = min(VW, NW);               // visibility-warps per pass
  const int G = NW / VWB;                    // pixel slices
  const int vw = warp % VWB, g = warp / VWB;
  const bool active = g < G;

  for (int vb = 0; vb < VW; vb += VWB) {
    const int v = (vb + vw) * 32 + lane;
    // my PV visibilities: k_j = j * n_vt + v  (consecutive lanes -> consecutive visibilities)
    // phase [rad] = al fx + be fy + ga n'.  The part linear in the pixel position reaches hundreds of radians at
    // the subgrid's edge, so the first pixel of every 16-pixel segment takes it modulo one cycle EXACTLY in 32-bit
    // fixed point (afix * ix + bfix * iy wraps), as the gridders do; al * (0..15) and ga n' are fp32.
    float2 al[PV / 2], ga[PV / 2];
    int32_t afix[PV], bfix[PV];                  // cycles per pixel * 2^32
#pragma unroll
    for (int j = 0; j < PV; ++j) {
      const int k = j * n_vt + v;
      float a_ = 0.f, g_ = 0.f;
      afix[j] = bfix[j] = 0;
      if (active && v < n_vt && k < K) {
        const int r = k / nc, c = k % nc;
        const double* uvw = job.uvw + (row0 + r) * 3;
        const double kap = job.kappa[c0 + c];
        const double two_pi = 6.283185307179586476925286766559;
        const double alpha = (sgn * uvw[0] * kap - u0) * (S / L), beta = (sgn * uvw[1] * kap - v0) * (S / L);
        a_ = static_cast<float>(two_pi * alpha);
        afix[j] = static_cast<int32_t>(static_cast<uint32_t>(static_cast<int64_t>(rint(alpha * 4294967296.0))));
        bfix[j] = static_cast<int32_t>(static_cast<uint32_t>(static_cast<int64_t>(rint(beta * 4294967296.0))));
        g_ = static_cast<float>(two_pi * (sgn * uvw[2] * kap - w0));
      }
      if (j & 1) { al[j / 2].y = a_; ga[j / 2].y = g_; }
      else       { al[j / 2].x = a_; ga[j / 2].x = g_; }
    }
    float2 vre[4][PV / 2], vim[4][PV / 2];
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
      for (int j = 0; j < PV / 2; ++j) vre[p][j] = vim[p][j] = make_float2(0.f, 0.f);

    for (int chunk = 0; chunk < NCHUNK; ++chunk) {
      __syncthreads();
      // --- staging (step a8): taper and A-term sandwich, once per pixel
      for (int i = tid; i < kPixChunk; i += T) {
        const int pix = chunk * kPixChunk + i;
        float2 x[4], z[4];
        const float t = __ldg(&job.taper[pix]);
#pragma unroll
        for (int p = 0; p < 4; ++p) {
          x[p] = __ldg(&sub[p * L * L + pix]);
        }
        // M_p (t S) M_q^H == t (M_p S M_q^H)
        sandwich(x, __ldg(&ap[pix * 2]), __ldg(&ap[pix * 2 + 1]), __ldg(&aq[pix * 2]), __ldg(&aq[pix * 2 + 1]), t, z);
#pragma unroll
        for (int p = 0; p < 4; ++p) spix[i][p] = make_float4(z[p].x, z[p].x, z[p].y, z[p].y);
        const float np = __ldg(&job.nprime[pix]);
        const float fx = static_cast<float>(i % kSeg);    // offset within the 16-pixel segment
        spix[i][4] = make_float4(np, np, fx, fx);
      }
      __syncthreads();
      if (active) {
        for (int seg = g; seg < NSEG; seg += G) {
          const int q0 = chunk * kPixChunk + seg * kSeg;
          const int ix0 = q0 % L - L / 2, iy = q0 / L - L / 2;
          float2 tt[PV / 2];
#pragma unroll
          for (int j = 0; j < PV / 2; ++j)
            tt[j] = make_float2(static_cast<float>(wrap_dot2(afix[2 * j], ix0, bfix[2 * j], iy)) * 1.4629180792671596e-9f,
                                static_cast<float>(wrap_dot2(afix[2 * j + 1], ix0, bfix[2 * j + 1], iy)) * 1.4629180792671596e-9f);
#pragma unroll 2
          for (int i = 0; i < kSeg; ++i) {
            const float4* rec = spix[seg * kSeg + i];
            const float4 s0 = rec[0], s1 = rec[1], s2 = rec[2], s3 = rec[3], gm = rec[4];
            const float2 n2 = make_float2(gm.x, gm.y), fx2 = make_float2(gm.z, gm.w);
#pragma unroll
            for (int j = 0; j < PV / 2; ++j) {
              const float2 ph = ffma2(al[j], fx2, ffma2(ga[j], n2, tt[j]));
              float sa, ca, sb, cb;
              __sincosf(ph.x, &sa, &ca);
              __sincosf(ph.y, &sb, &cb);
              const float2 cc2 = make_float2(ca, cb), ss2 = make_float2(sa, sb);
#define IDG_MAC(POL, SV)                                                      \
              vre[POL][j] = ffma2(make_float2(SV.x, SV.y), cc2, vre[POL][j]);   \
              vre[POL][j] = ffma2(make_float2(SV.z, SV.w), ss2, vre[POL][j]);   \
              vim[POL][j] = ffma2(make_float2(SV.z, SV.w), cc2, vim[POL][j]);   \
              vim[POL][j] = ffma2(neg2(make_float2(SV.x, SV.y)), ss2, vim[POL][j]);
              IDG_MAC(0, s0) IDG_MAC(1, s1) IDG_MAC(2, s2) IDG_MAC(3, s3)
#undef IDG_MAC
            }
          }
        }
      }
    }

    // --- sum the pixel slices, one visibility of every thread at a time, fixed order
#pragma unroll
    for (int j = 0; j < PV; ++j) {
      __syncthreads();
      if (j & 1) {
        sred[tid][0] = make_float4(vre[0][j / 2].y, vim[0][j / 2].y, vre[1][j / 2].y, vim[1][j / 2].y);
        sred[tid][1] = make_float4(vre[2][j / 2].y, vim[2][j / 2].y, vre[3][j / 2].y, vim[3][j / 2].y);
      } else {
        sred[tid][0] = make_float4(vre[0][j / 2].x, vim[0][j / 2].x, vre[1][j / 2].x, vim[1][j / 2].x);
        sred[tid][1] = make_float4(vre[2][j / 2].x, vim[2][j / 2].x, vre[3][j / 2].x, vim[3][j / 2].x);
      }
      __syncthreads();
      const int k = j * n_vt + v;
      if (g == 0 && v < n_vt && k < K) {
        float4 a0 = sred[tid][0], a1 = sred[tid][1];
        for (int gg = 1; gg < G; ++gg) {
          const float4 b0 = sred[(gg * VWB + vw) * 32 + lane][0], b1 = sred[(gg * VWB + vw) * 32 + lane][1];
          a0.x += b0.x; a0.y += b0.y; a0.z += b0.z; a0.w += b0.w;
          a1.x += b1.x; a1.y += b1.y; a1.z += b1.z; a1.w += b1.w;
        }
        const int r = k / nc, c = k % nc;
        float4* o = vis + ((row0 + r) * job.n_chan + c0 + c) * 2;
        if (conj) {                                     // (XX, XY, YX, YY) <- conj of (XX, YX, XY, YY)
          const float4 d0 = make_float4(a0.x, -a0.y, a1.x, -a1.y), d1 = make_float4(a0.z, -a0.w, a1.z, -a1.w);
          a0 = d0; a1 = d1;
        }
        o[0] = a0;
        o[1] = a1;
      }
    }
  }
}

template <int L, int T, int PV>
cudaError_t launch(const SubgridJob& job, const float2* in, float4* vis, cudaStream_t stream) {
  if (job.count == 0) return cudaSuccess;
  degridder_kernel<L, T, PV><<<static_cast<unsigned>(job.count), T, 0, stream>>>(job, in, vis);
  count_launch();
  note_kernel(IDG_K_DEGRIDDER, IDG_KMASK_SIMT);
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_degridder(const SubgridJob& job, const float2* in, float4* vis, cudaStream_t stream) {
  switch (job.subgrid_size) {
    case 32:  return launch<32, 256, 8>(job, in, vis, stream);
    case 48:  return launch<48, 256, 8>(job, in, vis, stream);
    case 64:  return launch<64, 256, 8>(job, in, vis, stream);
    case 96:  return launch<96, 256, 8>(job, in, vis, stream);
    case 128: return launch<128, 256, 8>(job, in, vis, stream);
    case 160: return launch<160, 256, 8>(job, in, vis, stream);
    default:  return cudaErrorInvalidValue;
  }
}

}  // namespace idg
