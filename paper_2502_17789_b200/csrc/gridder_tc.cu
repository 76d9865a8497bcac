// Tensor-core gridder: steps a1-a3 with the 2x2 complex MACs on tcgen05 (north_star: "tensor cores
// only if a phasor-matrix formulation is shown by ncu to win"; profiles/ has the evidence).
//
//   S[pix, n] = sum_k E[pix, k] B[k, n]                                 (Eq. 10 :133-137)
//
// with k = (visibility v, part in {cos, sin}), n = (polarisation, re/im):
//   E[pix, (v,cos)] = cos 2 pi phi(pix, v),  E[pix, (v,sin)] = sin 2 pi phi(pix, v)
//   B[(v,cos), (p,re)] =  Re V_p   B[(v,cos), (p,im)] = Im V_p
//   B[(v,sin), (p,re)] = -Im V_p   B[(v,sin), (p,im)] = Re V_p
// The SIMT pipes only GENERATE the phasor matrix E (phase FFMA + __sincosf per pair: the SFU-bound
// part, 8 pairs/clk/SM) and hand it to the tensor cores through tensor memory; the 16 FMAs per pair
// that bound a SIMT kernel at 7.11 pairs/clk/SM leave the FP32 pipe.
//
// Precision.  kind::tf32 keeps 11 significant bits, so every operand is split into a tf32-exact head
// and an fp32 remainder: E = Eh + El (mask + exact subtraction), V = Vh + Vl.  One MMA of N = 16
// columns [B(Vh) | B(Vl)] per A part gives Eh Vh + Eh Vl + El Vh + El Vl; the two column halves are
// added when the accumulator is read.  The tensor core's fp32 accumulation truncates, which biases
// long chains (measured 4e-6 after 128 MMAs), so the accumulator is drained into fp32 registers
// (round-to-nearest adds) every DG chunks, alternating two TMEM accumulators so that draining one
// overlaps the MMAs into the other.
//
// Roles per CTA (128 compute threads = 128 pixels = the M rows of the MMA, plus one service warp):
//   compute threads  per chunk of <= KC channels of one table row: sincos -> head/remainder ->
//                    tcgen05.st into A[g & 1]; arrive on full[g & 1]; drain accumulators; epilogue
//                    (A-term sandwich and taper as in gridder.cu).
//   service warp     stages the B operand of the next chunk in shared memory (canonical K-major
//                    core-matrix layout, heads and remainders of the visibilities), and one lane
//                    issues the MMAs of chunk g once full[g & 1] completes: 2 x KC/4 MMAs of
//                    M = 128, N = 16, K = 8; commit -> empty[g & 1] and, at a group's end, dfull[q & 1].
#include "device_math.cuh"
#include "kernels.h"
#include "tc_common.cuh"

namespace idg {

namespace {

#ifndef IDG_TC_KC
#define IDG_TC_KC 8
#endif
#ifndef IDG_TC_G
#define IDG_TC_G 8
#endif
#ifndef IDG_TC_DG
#define IDG_TC_DG 4
#endif
#ifndef IDG_TC_NA
#define IDG_TC_NA 3
#endif

constexpr int kTileM = 128;           // pixels per MMA tile = compute threads
constexpr int kThreadsTc = kTileM + 32;
constexpr int kMaxRowsTc = 128;       // rows of one subgrid whose constants are kept in shared memory
constexpr int kMaxChanTc = 2048;      // channels of one subgrid whose offsets are kept in shared memory

struct RowDataTc {
  int32_t alpha_fix, beta_fix;   // (u-u0) S/L and (v-v0) S/L at kappa_ref, cycles/pixel * 2^32 (wrapping)
  float gamma;                   // 2 pi (w kappa_ref - w0)
  float us, vs, ws;              // 2 pi u_m S/L, 2 pi v_m S/L, 2 pi w_m   [rad per unit kappa]
};

// tf32-exact head of x (the low 13 mantissa bits cleared); x - head is exact in fp32
__device__ __forceinline__ float tf32_head(float x) { return __uint_as_float(__float_as_uint(x) & 0xffffe000u); }
__device__ __forceinline__ float tf32_round(float x) {
  return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
}

// G = tiles per CTA, KC = visibilities per chunk (8 or 16), DG = chunks per accumulator group,
// NA = depth of the (A in TMEM, B in shared memory) operand ring
template <int L, int G, int KC, int DG, int NA>
__global__ void __launch_bounds__(kThreadsTc) gridder_tc_kernel(const SubgridJob job, const float4* __restrict__ vis,
                                                                float2* __restrict__ out) {
  static_assert((L * L) % (kTileM * G) == 0 && (KC == 8 || KC == 16) && NA >= 3 && NA <= 4, "shape");
  constexpr int PIECES = (L * L) / (kTileM * G);
  constexpr int A_COLS = 4 * KC;                       // per buffer: heads [0, 2KC), remainders [2KC, 4KC)
  constexpr int D_COL = NA * A_COLS;                   // two accumulators of 16 columns
  constexpr int TMEM_COLS = (D_COL + 32) <= 128 ? 128 : ((D_COL + 32) <= 256 ? 256 : 512);
  constexpr int B_BYTES = KC * 128;                    // 2 KC k-rows x 16 columns x 4 bytes
  constexpr uint32_t IDESC = tc::make_idesc_tf32(kTileM, 16);

  __shared__ __align__(1024) unsigned char sB[NA][B_BYTES];
  __shared__ __align__(16) float sdk[kMaxChanTc];
  __shared__ RowDataTc srow[kMaxRowsTc];
  __shared__ __align__(8) uint64_t bars[2 * NA + 4];   // full[NA], empty[NA], dfull[2], dempty[2]
  __shared__ uint32_t s_tmem;

  const int tid = threadIdx.x, warp = tid / 32, lane = tid % 32;
  const int sg = blockIdx.x / PIECES;
  const int piece = blockIdx.x % PIECES;
  const int32_t* __restrict__ m = job.meta + (job.first + sg) * kMetaStride;
  const int b = m[0], t0 = m[1], nt = m[2], c0 = m[3], nc = m[4], x0 = m[5], y0 = m[6], wl = m[7];
  const int sp = m[8], sq = m[9], it = m[10];
  const int64_t row0 = static_cast<int64_t>(b) * job.n_times + t0;

  const uint32_t bar_full = tc::smem_u32(&bars[0]), bar_empty = tc::smem_u32(&bars[NA]);
  const uint32_t bar_dfull = tc::smem_u32(&bars[2 * NA]), bar_dempty = tc::smem_u32(&bars[2 * NA + 2]);

  if (tid == 0) {
    for (int i = 0; i < NA; ++i) {
      tc::mbar_init(bar_full + 8 * i, kTileM);
      tc::mbar_init(bar_empty + 8 * i, 1);
    }
    for (int i = 0; i < 2; ++i) {
      tc::mbar_init(bar_dfull + 8 * i, 1);
      tc::mbar_init(bar_dempty + 8 * i, kTileM);
    }
    tc::fence_barrier_init();
  }
  if (warp == 4) tc::tmem_alloc(tc::smem_u32(&s_tmem), TMEM_COLS);

  // --- per-subgrid constants, once per CTA: channel offsets and the row constants (fp64 -> fp32)
  {
    const double S = job.image_size;
    const double kref = job.kappa[c0 + nc / 2];
    for (int c = tid; c < nc; c += kThreadsTc) sdk[c] = static_cast<float>(job.kappa[c0 + c] - kref);
    const int ncpad = (nc + KC - 1) / KC * KC;
    for (int c = nc + tid; c < ncpad; c += kThreadsTc) sdk[c] = 0.f;
    if (tid < nt) {
      const double u0 = (x0 + L / 2 - job.grid_size / 2) / S;
      const double v0 = (y0 + L / 2 - job.grid_size / 2) / S;
      const double w0 = job.w_step > 0.0 ? (wl + 0.5) * job.w_step : 0.0;
      const double* uvw = job.uvw + (row0 + tid) * 3;
      const double um = uvw[0], vm = uvw[1], wm = uvw[2];
      const double two_pi = 6.283185307179586476925286766559;
      const double sl = S / L;
      const double alpha = (um * kref - u0) * sl, beta = (vm * kref - v0) * sl;
      RowDataTc rd;
      rd.alpha_fix = static_cast<int32_t>(static_cast<uint32_t>(static_cast<int64_t>(rint(alpha * 4294967296.0))));
      rd.beta_fix = static_cast<int32_t>(static_cast<uint32_t>(static_cast<int64_t>(rint(beta * 4294967296.0))));
      rd.gamma = static_cast<float>(two_pi * (wm * kref - w0));
      rd.us = static_cast<float>(two_pi * um * sl);
      rd.vs = static_cast<float>(two_pi * vm * sl);
      rd.ws = static_cast<float>(two_pi * wm);
      srow[tid] = rd;
    }
  }
  tc::fence_before_thread_sync();
  __syncthreads();
  tc::fence_after_thread_sync();
  const uint32_t tmem = s_tmem;

  const int cpr = (nc + KC - 1) / KC;                  // chunks per table row
  const int nchunks = nt * cpr;                        // chunks per tile
  const int total = nchunks * G;                       // the CTA's chunk sequence g = 0 .. total-1

  if (warp == 4) {
    // ===== service warp: stage B, issue MMAs =====
    // lane -> items (visibility j, polarisation p) of a chunk; element (n, k) of the N x K operand
    // lives at ((k/4)*2 + n/8)*128 + (n%8)*16 + (k%4)*4 bytes; rows (2j, 2j+1) of one column are adjacent
    constexpr int ITEMS = KC * 4 / 32;
    constexpr int PD = 4;                              // visibility prefetch distance in chunks
    float2 ring[PD][ITEMS];
    int pr = 0, pcc = 0, pn = 0;                       // next chunk to prefetch: row, first channel, index
    auto prefetch = [&](float2 (&dst)[ITEMS]) {
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) {
        const int item = lane + 32 * i, j = item >> 2, p = item & 3;
        dst[i] = make_float2(0.f, 0.f);
        if (pn < total && pcc + j < nc)
          dst[i] = __ldg(reinterpret_cast<const float2*>(vis) + ((row0 + pr) * job.n_chan + c0 + pcc + j) * 4 + p);
      }
      ++pn;
      pcc += KC;
      if (pcc >= nc) { pcc = 0; if (++pr == nt) pr = 0; }
    };
    auto b_store = [&](const float2 (&src)[ITEMS], int slot) {
      float* Bf = reinterpret_cast<float*>(&sB[slot][0]);
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) {
        const int item = lane + 32 * i, j = item >> 2, p = item & 3;
        const float hr = tf32_round(src[i].x), hi = tf32_round(src[i].y);
        const float lr = tf32_round(src[i].x - hr), li = tf32_round(src[i].y - hi);
        auto at2 = [&](int n) -> float2* {
          return reinterpret_cast<float2*>(&Bf[((j >> 1) * 2 + (n >> 3)) * 32 + (n & 7) * 4 + (j & 1) * 2]);
        };
        *at2(2 * p) = make_float2(hr, -hi);           // column (p,re): rows (v,cos) = Re V, (v,sin) = -Im V
        *at2(2 * p + 1) = make_float2(hi, hr);        // column (p,im): rows (v,cos) = Im V, (v,sin) =  Re V
        *at2(2 * p + 8) = make_float2(lr, -li);
        *at2(2 * p + 9) = make_float2(li, lr);
      }
      tc::fence_proxy_async();
    };
    auto shift_ring = [&]() {
#pragma unroll
      for (int d = 0; d + 1 < PD; ++d)
#pragma unroll
        for (int i = 0; i < ITEMS; ++i) ring[d][i] = ring[d + 1][i];
    };

    // ring[d] holds the visibilities of chunk (staged + d).  B is staged S = NA - 2 chunks ahead of the
    // MMAs, so the slot being overwritten was read two chunks ago and the wait below rarely blocks.
    constexpr int S = NA - 2;
#pragma unroll
    for (int d = 0; d < PD; ++d) prefetch(ring[d]);
    int staged = 0, sslot = 0, sphase = 0;             // next chunk to stage, its slot and ring phase
#pragma unroll
    for (int d = 0; d < S; ++d) {
      if (staged < total) b_store(ring[0], sslot);
      shift_ring();
      prefetch(ring[PD - 1]);
      ++staged;
      if (++sslot == NA) { sslot = 0; sphase ^= 1; }
    }
    __syncwarp();

    int slot = 0, phase = 0, ci = 0, cig = 0, q = 0;
    for (int g = 0; g < total; ++g) {
      const bool tile_last = ci == nchunks - 1;
      if (lane == 0) {
        if (cig == 0 && q >= 2) {                      // accumulator q & 1 drained (group q - 2)
          tc::mbar_wait(bar_dempty + 8 * (q & 1), ((q - 2) >> 1) & 1);
          tc::fence_after_thread_sync();
        }
        tc::mbar_wait(bar_full + 8 * slot, phase);
        tc::fence_after_thread_sync();
        const uint32_t a0 = tmem + slot * A_COLS;
        const uint32_t d0 = tmem + D_COL + 16 * (q & 1);
        const uint32_t bbase = tc::smem_u32(&sB[slot][0]);
#pragma unroll
        for (int part = 0; part < 2; ++part)
#pragma unroll
          for (int ks = 0; ks < KC / 4; ++ks) {
            const uint64_t bdesc = tc::make_smem_desc(bbase + ks * 512, 256, 128);
            tc::mma_tf32_ts(d0, a0 + part * 2 * KC + ks * 8, bdesc, IDESC, (cig > 0 || part > 0 || ks > 0) ? 1u : 0u);
          }
        tc::mma_commit(bar_empty + 8 * slot);
        if (cig == DG - 1 || tile_last) tc::mma_commit(bar_dfull + 8 * (q & 1));
        // the slot of chunk `staged` = g + S was last read by the MMAs of chunk staged - NA
        if (staged < total && staged >= NA) tc::mbar_wait(bar_empty + 8 * sslot, sphase ^ 1);
      }
      __syncwarp();
      if (staged < total) b_store(ring[0], sslot);
      shift_ring();
      prefetch(ring[PD - 1]);
      ++staged;
      if (++sslot == NA) { sslot = 0; sphase ^= 1; }
      __syncwarp();
      if (++slot == NA) { slot = 0; phase ^= 1; }
      if (++ci == nchunks) ci = 0;
      if (++cig == DG || tile_last) { cig = 0; ++q; }
    }
  } else {
    // ===== compute threads: one pixel of the current tile each =====
    const uint32_t lane_base = static_cast<uint32_t>(warp * 32) << 16;
    const float4* __restrict__ ap = job.aterms + (static_cast<int64_t>(sp) * job.n_intervals + it) * (L * L * 2);
    const float4* __restrict__ aq = job.aterms + (static_cast<int64_t>(sq) * job.n_intervals + it) * (L * L * 2);
    float2* __restrict__ o = out + static_cast<int64_t>(sg) * 4 * L * L;

    float acc[8];
    // accumulator group p -> registers (fp32 round-to-nearest adds), then hand the TMEM columns back
    auto drain = [&](int p) {
      tc::mbar_wait(bar_dfull + 8 * (p & 1), (p >> 1) & 1);
      tc::fence_after_thread_sync();
      uint32_t d[16];
      tc::tmem_ld16(tmem + lane_base + D_COL + 16 * (p & 1), d);
      tc::tmem_wait_ld();
      tc::fence_before_thread_sync();
      tc::mbar_arrive(bar_dempty + 8 * (p & 1));
#pragma unroll
      for (int n = 0; n < 8; ++n) acc[n] += __uint_as_float(d[n]) + __uint_as_float(d[n + 8]);
    };

    int g = 0, q = 0, slot = 0, phase = 0;             // chunk index, group index, ring slot and ring phase
    for (int tile = 0; tile < G; ++tile) {
      const int pix = (piece * G + tile) * kTileM + tid;
      const int ix = pix % L - L / 2, iy = pix / L - L / 2;
      const float np = job.nprime[pix];
#pragma unroll
      for (int n = 0; n < 8; ++n) acc[n] = 0.f;
      int cig = 0, gin = 0;                            // chunks in the current group, groups done in this tile
      for (int r = 0; r < nt; ++r) {
        // per-(row, pixel) slope and offset of the phase; amortised over the row's channels
        const RowDataTc rd = srow[r];
        const float pa = fmaf(rd.vs, static_cast<float>(iy), fmaf(rd.ws, np, rd.us * static_cast<float>(ix)));
        const int32_t bf = rd.alpha_fix * ix + rd.beta_fix * iy;                    // wraps: exact mod 1 cycle
        const float pb = fmaf(rd.gamma, np, static_cast<float>(bf) * 1.4629180792671596e-9f);   // 2 pi / 2^32
        for (int cc = 0; cc < nc; cc += KC) {
          if (g >= NA) tc::mbar_wait(bar_empty + 8 * slot, phase ^ 1);              // A[slot] read by chunk g - NA
          const uint32_t abuf = tmem + lane_base + slot * A_COLS;
#pragma unroll
          for (int half = 0; half < KC / 8; ++half) {
            uint32_t hi[16], lo[16];
            const float4 dka = *reinterpret_cast<const float4*>(&sdk[cc + half * 8]);
            const float4 dkb = *reinterpret_cast<const float4*>(&sdk[cc + half * 8 + 4]);
            const float dk[8] = {dka.x, dka.y, dka.z, dka.w, dkb.x, dkb.y, dkb.z, dkb.w};
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              float s, c;
              __sincosf(fmaf(pa, dk[j], pb), &s, &c);
              const float ch = tf32_head(c), sh = tf32_head(s);
              hi[2 * j] = __float_as_uint(ch);
              hi[2 * j + 1] = __float_as_uint(sh);
              lo[2 * j] = __float_as_uint(c - ch);
              lo[2 * j + 1] = __float_as_uint(s - sh);
            }
            tc::tmem_st16(abuf + half * 16, hi);
            tc::tmem_st16(abuf + 2 * KC + half * 16, lo);
          }
          tc::tmem_wait_st();
          tc::fence_before_thread_sync();
          tc::mbar_arrive(bar_full + 8 * slot);
          ++g;
          if (++slot == NA) { slot = 0; phase ^= 1; }
          const bool tile_last = (r == nt - 1) && (cc + KC >= nc);
          if (++cig == DG || tile_last) {
            if (gin > 0) drain(q - 1);                 // the previous group: its MMAs finished long ago
            cig = 0; ++q; ++gin;
          }
        }
      }
      drain(q - 1);                                    // the tile's last group
      // --- epilogue (step a3): A-term sandwich and taper, once per pixel
      float2 x[4], z[4];
#pragma unroll
      for (int p = 0; p < 4; ++p) x[p] = make_float2(acc[2 * p], acc[2 * p + 1]);
      sandwich(x, __ldg(&ap[pix * 2]), __ldg(&ap[pix * 2 + 1]), __ldg(&aq[pix * 2]), __ldg(&aq[pix * 2 + 1]),
               __ldg(&job.taper[pix]), z);
#pragma unroll
      for (int p = 0; p < 4; ++p) o[p * L * L + pix] = z[p];
    }
  }

  tc::fence_before_thread_sync();
  __syncthreads();
  if (warp == 4) tc::tmem_dealloc(tmem, TMEM_COLS);
}

// largest divisor of the subgrid's tile count that is <= want
constexpr int tiles_per_cta(int L, int want) {
  const int tiles = L * L / kTileM;
  int g = 1;
  for (int d = 1; d <= want && d <= tiles; ++d)
    if (tiles % d == 0) g = d;
  return g;
}

template <int L, int G, int KC, int DG, int NA>
cudaError_t launch(const SubgridJob& job, const float4* vis, float2* out, cudaStream_t stream) {
  constexpr int PIECES = (L * L) / (kTileM * G);
  const int64_t blocks = job.count * PIECES;
  if (blocks == 0) return cudaSuccess;
  gridder_tc_kernel<L, G, KC, DG, NA><<<static_cast<unsigned>(blocks), kThreadsTc, 0, stream>>>(job, vis, out);
  count_launch();
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_gridder_tc(const SubgridJob& job, const float4* vis, float2* out, cudaStream_t stream) {
  // shapes whose per-subgrid constants do not fit the kernel's shared-memory tables take the SIMT kernel
  if (job.n_chan > kMaxChanTc - 16 || job.max_nt > kMaxRowsTc) return launch_gridder(job, vis, out, stream);
  switch (job.subgrid_size) {
    case 32:  return launch<32, tiles_per_cta(32, IDG_TC_G), IDG_TC_KC, IDG_TC_DG, IDG_TC_NA>(job, vis, out, stream);
    case 64:  return launch<64, tiles_per_cta(64, IDG_TC_G), IDG_TC_KC, IDG_TC_DG, IDG_TC_NA>(job, vis, out, stream);
    case 96:  return launch<96, tiles_per_cta(96, IDG_TC_G), IDG_TC_KC, IDG_TC_DG, IDG_TC_NA>(job, vis, out, stream);
    case 128: return launch<128, tiles_per_cta(128, IDG_TC_G), IDG_TC_KC, IDG_TC_DG, IDG_TC_NA>(job, vis, out, stream);
    default:  return cudaErrorInvalidValue;
  }
}

}  // namespace idg
