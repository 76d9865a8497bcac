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
// Precision.  The tensor core takes 11-bit operands (fp16 and tf32 alike), so every operand is split into a
// head and a remainder: E = Eh + El, V = Vh + Vl.  Default (IDG_TC_FP16): fp16 heads and fp16 remainders.
// |E| <= 1, so (cos, sin) of one visibility pack into ONE 32-bit word of heads and one of remainders, 8 B per
// (visibility, pixel) pair in tensor memory instead of 16, and a chunk of 8 visibilities is one K = 16
// kind::f16 MMA per part instead of two K = 8 kind::tf32 ones; the remainder (<= 2^-12) is kept to 2^-25
// absolute.  The visibilities are brought into fp16's range by one power-of-two scale per segment (the largest
// |component|, found while staging), undone exactly when a tile is finished.  -DIDG_TC_TF32 selects the first
// scheme instead: tf32-exact heads by masking, fp32 remainders, 16 B per pair.  Either way one MMA of N = 16
// columns [B(Vh) | B(Vl)] per A part gives Eh Vh + Eh Vl + El Vh + El Vl, the two column halves being added
// when the accumulator is read.  The tensor core's fp32 accumulation truncates, which biases long chains, so
// the accumulator is drained into fp32 registers (round-to-nearest adds) every DG chunks, alternating two TMEM
// accumulators so that draining one overlaps the MMAs into the other.  Measured against the oracle: 1.1e-6
// per subgrid and 0.8e-6 on a recovered point-source flux (fp16, DG = 12: 24 MMAs per accumulator); 1.7e-6 and
// 1.8e-6 with tf32 operands (48 MMAs).  Halving the bytes stored per pair is also why it is faster (the
// tensor-memory stores cost 20 % of the tf32 kernel's time): 5.45 against 5.19 pairs/clk/SM on config 2.
//
// Phasors by rotation (round 2, template parameter ROT; uniformly spaced channels): the phase is linear in the channel,
// so per 8 channels ONE __sincosf seeds e = (cos, sin) and 7 steps of d += -4 sin^2(delta/2) e, e += d (one packed FFMA2
// and one packed FADD2 each) give the rest; delta = pa * dkappa per (row, pixel), its 1 - cos and sin from Taylor series
// at delta / 4 plus two angle doublings (relative accuracy: a rotor error grows linearly along the chain).  MUFU per pair
// 2 -> 0.25.  Chunks are 16 channels (KC) with fp16 operands: half the per-chunk bookkeeping, one tcgen05.st.x32, four
// K = 16 MMAs, a ring of 2 slots, accumulator groups of 6 chunks.  6.32 pairs/clk/SM on config 2 (0.89 of the ALU
// roofline) against 5.38 for the round-1 kernel.
//
// One CTA per subgrid: NG groups of 128 compute threads plus one service warp per group; NG = 1, 2 or 4
// chosen at launch so that 4 / NG CTAs share an SM (see launch_l).
//   all threads      stage the B operand of the subgrid's visibilities ONCE in shared memory (heads
//                    and remainders, canonical K-major core-matrix layout); every pixel tile reuses it.
//                    Subgrids with more visibilities than fit are processed in segments of whole table
//                    rows; partial sums then pass through the output buffer.
//   compute group    owns one tile of 128 pixels per round (thread = pixel = MMA row = TMEM lane).
//                    Per chunk of <= KC channels of one table row: seed + rotations (or sincos) -> head/remainder ->
//                    tcgen05.st into the group's A ring slot.  The hand-off of chunk g (wait::st,
//                    fence, mbarrier arrive) is issued after the arithmetic of chunk g+1, so the
//                    store latency is hidden.  Accumulators are drained one group of DG chunks late,
//                    and a tile's epilogue (A-term sandwich and taper as in gridder.cu) runs inside
//                    the next tile, so no thread waits for the tensor core.
//   service warp     one lane walks (chunk, group) in lock step: waits for full[group][slot], issues the
//                    2 x KC/4 MMAs (M = 128, N = 16, K = 8), commits to empty[group][slot] and, at an
//                    accumulator group's end, to dfull[group][q & 1].
#include <algorithm>

#include <cuda_fp16.h>

#include "device_math.cuh"
#include "kernels.h"
#include "tc_common.cuh"

namespace idg {

namespace {

#ifndef IDG_TC_TF32
#define IDG_TC_FP16 1                 // operand format: fp16 head + fp16 remainder (default) or split tf32
#endif
// fp16 operands (default): chunks of 16 channels (half the per-chunk ring / barrier bookkeeping of 8-channel chunks:
// 6.32 against 5.82 pairs/clk/SM on config 2), a ring of 2 slots of 32 TMEM columns, accumulator groups of 6 chunks
// (24 MMAs between drains, as with 12 chunks of 8).  Split tf32: chunks of 8, ring of 3, groups of 12.
#ifdef IDG_TC_FP16
#ifndef IDG_TC_KC
#define IDG_TC_KC 16
#endif
#ifndef IDG_TC_DG
#define IDG_TC_DG 6
#endif
#ifndef IDG_TC_NA
#define IDG_TC_NA 2
#endif
#else
#ifndef IDG_TC_KC
#define IDG_TC_KC 8
#endif
#ifndef IDG_TC_DG
#define IDG_TC_DG 12
#endif
#ifndef IDG_TC_NA
#define IDG_TC_NA 3
#endif
#endif

constexpr int kTileM = 128;           // pixels per MMA tile = threads per compute group
constexpr int kMaxRowsTc = 128;       // rows of one subgrid whose constants are kept in shared memory
constexpr int kMaxChanTc = 1280;      // channels of one subgrid whose offsets are kept in shared memory
constexpr int kMaxBBytes = 160 * 1024;   // shared memory for the B operand
#ifdef IDG_TC_FP16
constexpr int kVisBytes = 64;            // B operand bytes per visibility: 2 k-rows x 16 columns x 2 bytes
#else
constexpr int kVisBytes = 128;           // 2 k-rows x 16 columns x 4 bytes
#endif

struct alignas(16) RowDataTc {     // 32 bytes: two 128-bit shared-memory loads
  int32_t alpha_fix, beta_fix;   // (u-u0) S/L and (v-v0) S/L at kappa_ref, cycles/pixel * 2^32 (wrapping)
  float gamma;                   // 2 pi (w kappa_ref - w0)
  float us, vs, ws;              // 2 pi u_m S/L, 2 pi v_m S/L, 2 pi w_m   [rad per unit kappa]
  float dmax;                    // bound of |pa * dkappa| over the subgrid's pixels: the phase step per channel [rad]
};

// tf32-exact head of x (the low 13 mantissa bits cleared); x - head is exact in fp32
[[maybe_unused]] __device__ __forceinline__ float tf32_head(float x) { return __uint_as_float(__float_as_uint(x) & 0xffffe000u); }
[[maybe_unused]] __device__ __forceinline__ float tf32_round(float x) {
  return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
}

// NG = compute groups (tiles in flight) per CTA, KC = visibilities per chunk, DG = chunks per accumulator
// group, NA = depth of a group's A ring in TMEM, ROT = phasors by rotation along the channel axis (uniformly
// spaced channels, job.dkappa != 0) instead of one __sincosf per (visibility, pixel) pair
template <int L, int NG, int KC, int DG, int NA, bool ROT>
__global__ void __launch_bounds__(NG* kTileM + NG * 32, NG == 1 ? 4 : (NG == 2 ? 2 : 1))
    gridder_tc_kernel(const SubgridJob job, const float4* __restrict__ vis, float2* __restrict__ out,
                      const int cap_chunks) {
  constexpr int TILES = (L * L) / kTileM;
  static_assert(TILES % NG == 0 && (KC == 8 || KC == 16) && NA >= 2, "shape");
  constexpr int ROUNDS = TILES / NG;
  constexpr int NTHREADS = NG * kTileM + NG * 32;
#ifdef IDG_TC_FP16
  constexpr int A_COLS = 2 * KC;                       // per slot and 8 visibilities: 8 words of (cos, sin) heads, 8 of remainders
#else
  constexpr int A_COLS = 4 * KC;                       // per slot: heads [0, 2KC), remainders [2KC, 4KC)
#endif
  constexpr int D_COL = NA * A_COLS;                   // then two accumulators of 16 columns
  constexpr int GCOLS = D_COL + 32;                    // TMEM columns per compute group
  constexpr int TMEM_COLS = NG * GCOLS <= 128 ? 128 : (NG * GCOLS <= 256 ? 256 : 512);
  static_assert(NG * GCOLS <= 512, "TMEM");
#ifdef IDG_TC_FP16
  constexpr int CHUNK_BYTES = KC * 64;                 // 2 KC k-rows x 16 columns x 2 bytes
#else
  constexpr int CHUNK_BYTES = KC * 128;                // 2 KC k-rows x 16 columns x 4 bytes
#endif
  static_assert(DG % NA == 0, "an accumulator group is a whole number of ring revolutions");
  constexpr int RPG = DG / NA;                         // revolutions per accumulator group
  constexpr int NBAR = 2 * NA + 4;                     // per group: full[NA], empty[NA], dfull[2], dempty[2]
#ifdef IDG_TC_FP16
  constexpr uint32_t IDESC = tc::make_idesc_f16(kTileM, 16);
#else
  constexpr uint32_t IDESC = tc::make_idesc_tf32(kTileM, 16);
#endif

  extern __shared__ __align__(1024) unsigned char sB[];   // [cap_chunks][CHUNK_BYTES]
  __shared__ __align__(16) float sdk[kMaxChanTc];
  __shared__ RowDataTc srow[kMaxRowsTc];
  __shared__ __align__(8) uint64_t bars[NG * NBAR];
  __shared__ uint32_t s_tmem;
  __shared__ uint32_t s_vmax;                          // fp16 operands: bits of the segment's largest |component|

  const int tid = threadIdx.x, warp = tid / 32;
  const int64_t sg = job_slot(job, blockIdx.x);
  const int32_t* m = job.meta + (job.first + sg) * kMetaStride;
  const int b = m[0], t0 = m[1], nt = m[2], c0 = m[3], nc = m[4], x0 = m[5], y0 = m[6], wl = m[7];
  const int sp = m[8], sq = m[9], it = m[10];
  const bool conj = (m[12] & kMetaConj) != 0;          // rows used as (-u,-v,-w) with V^dagger (PAPER.md:178 fn 4, R21)
  const int64_t row0 = static_cast<int64_t>(b) * job.n_times + t0;

  const uint32_t bar0 = tc::smem_u32(&bars[0]);
  auto bar_full = [&](int gi, int s) { return bar0 + 8 * (gi * NBAR + s); };
  auto bar_empty = [&](int gi, int s) { return bar0 + 8 * (gi * NBAR + NA + s); };
  auto bar_dfull = [&](int gi, int p) { return bar0 + 8 * (gi * NBAR + 2 * NA + p); };
  auto bar_dempty = [&](int gi, int p) { return bar0 + 8 * (gi * NBAR + 2 * NA + 2 + p); };

  if (tid == 0) {
    for (int gi = 0; gi < NG; ++gi) {
      for (int i = 0; i < NA; ++i) {
        tc::mbar_init(bar_full(gi, i), kTileM);
        tc::mbar_init(bar_empty(gi, i), 1);
      }
      for (int i = 0; i < 2; ++i) {
        tc::mbar_init(bar_dfull(gi, i), 1);
        tc::mbar_init(bar_dempty(gi, i), kTileM);
      }
    }
    tc::fence_barrier_init();
  }
  if (warp == NG * 4) tc::tmem_alloc(tc::smem_u32(&s_tmem), TMEM_COLS);

  // --- per-subgrid constants, once per CTA: channel offsets and the row constants (fp64 -> fp32)
  {
    const double S = job.image_size;
    const double kref = job.kappa[c0 + nc / 2];
    for (int c = tid; c < nc; c += NTHREADS) sdk[c] = static_cast<float>(job.kappa[c0 + c] - kref);
    const int ncpad = (nc + KC - 1) / KC * KC;
    for (int c = nc + tid; c < ncpad; c += NTHREADS) sdk[c] = 0.f;
    if (tid < nt) {
      const double u0 = (x0 + L / 2 - job.grid_size / 2) / S;
      const double v0 = (y0 + L / 2 - job.grid_size / 2) / S;
      const double w0 = job.w_step > 0.0 ? (wl + 0.5) * job.w_step : 0.0;
      const double* uvw = job.uvw + (row0 + tid) * 3;
      const double sgn = conj ? -1.0 : 1.0;
      const double um = sgn * uvw[0], vm = sgn * uvw[1], wm = sgn * uvw[2];
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
      // the corner pixel (0, 0) has the largest |l|, |m| and |n'|
      rd.dmax = static_cast<float>(fabs(job.dkappa) * two_pi *
                                   ((fabs(um) + fabs(vm)) * sl * (L / 2) + fabs(wm) * fabs(static_cast<double>(job.nprime[0]))));
      srow[tid] = rd;
    }
  }
  tc::fence_before_thread_sync();
  __syncthreads();
  tc::fence_after_thread_sync();
  const uint32_t tmem = s_tmem;

  const int cpr = (nc + KC - 1) / KC;                  // chunks per table row
  const int rows_per_seg = max(1, min(nt, cap_chunks / cpr));
  const int nseg = (nt + rows_per_seg - 1) / rows_per_seg;

  // warp index as a value the compiler knows to be warp-uniform (service-warp operands then live in
  // uniform registers and every tcgen05.mma is one predicated instruction)
  const int uwarp = __shfl_sync(0xffffffffu, warp, 0);
  const int gi = uwarp >> 2;                           // compute group; service warp NG*4 + k drives group k
  const int mygroup = gi < NG ? gi : uwarp - NG * 4;

  // running positions in the barrier rings; compute threads and service warps step them alike.
  // Barrier addresses of the group: full[s] at gbar + 8 s, empty[s] at + 8 NA, dfull[p] at + 16 NA,
  // dempty[p] at + 16 NA + 16.  `opaque` keeps them in registers.
  const uint32_t gbar = tc::opaque(bar0 + 8 * mygroup * NBAR);
  const uint32_t gtmem = tc::opaque(tmem + mygroup * GCOLS + (static_cast<uint32_t>((warp & 3) * 32) << 16));
  int q = 0;                                           // accumulator groups closed
  uint32_t phase = 0;                                  // parity of the current revolution

  const int tpix = tid & (kTileM - 1);
  const float4* __restrict__ ap = job.aterms + (static_cast<int64_t>(sp) * job.n_intervals + it) * (L * L * 2);
  const float4* __restrict__ aq = job.aterms + (static_cast<int64_t>(sq) * job.n_intervals + it) * (L * L * 2);
  float2* o = out + sg * 4 * L * L;
  const uint32_t sdk_addr = tc::opaque(tc::smem_u32(&sdk[0]));
  const uint32_t srow_addr = tc::opaque(tc::smem_u32(&srow[0]));

  for (int seg = 0; seg < nseg; ++seg) {
    const int r_begin = seg * rows_per_seg, r_end = min(nt, r_begin + rows_per_seg);
    const int nchunks = (r_end - r_begin) * cpr;       // chunks of one tile in this segment
    const bool first_seg = seg == 0, last_seg = seg == nseg - 1;

    // --- step a1: the B operand of the segment's visibilities.  Element (n, k) of a chunk's N x K
    // operand lives at ((k/4)*2 + n/8)*128 + (n%8)*16 + (k%4)*4 bytes; k = 2 j + {cos, sin}.
    if (seg > 0) __syncthreads();                      // every MMA of the previous segment was drained
    // One warp per 8 visibilities x 4 polarisations, so the row / channel split is once per warp.
    constexpr int UPC = KC / 8;
    // polarisation p of visibility (row r, channel c) as the sum uses it: V, or V^dagger = conj of (XX, YX, XY, YY)
    auto load_vis = [&](int r, int c, int p) -> float2 {
      const int ps = conj ? ((p == 1 || p == 2) ? 3 - p : p) : p;
      const float2 v = __ldg(reinterpret_cast<const float2*>(vis) + ((row0 + r) * job.n_chan + c0 + c) * 4 + ps);
      return conj ? make_float2(v.x, -v.y) : v;
    };
    // the chunk count is padded to whole ring revolutions with zero chunks (B = 0 contributes nothing), so
    // neither the compute threads nor the service warp ever test whether a slot is in use
    const int nchunks_pad = (nchunks + NA - 1) / NA * NA;
#ifdef IDG_TC_FP16
    // fp16 operands need the visibilities in range: one power-of-two scale per segment, undone at the drain
    if (tid == 0) s_vmax = 0u;
    __syncthreads();
    {
      float mx = 0.f;
      for (int u = warp; u < nchunks * UPC; u += NTHREADS / 32) {
        const int ci = u / UPC, j = (u % UPC) * 8 + ((tid & 31) >> 2), p = tid & 3;
        const int rr = ci / cpr;
        const int r = r_begin + rr, cc = (ci - rr * cpr) * KC;
        if (cc + j < nc) {
          float2 v = load_vis(r, cc + j, p);
          if (job.weights != nullptr) {
            const float wgt = __ldg(&job.weights[(row0 + r) * job.n_chan + c0 + cc + j]);
            v = wgt == 0.f ? make_float2(0.f, 0.f) : make_float2(v.x * wgt, v.y * wgt);   // flagged: out of the scale too
          }
          mx = fmaxf(mx, fmaxf(fabsf(v.x), fabsf(v.y)));
        }
      }
      for (int o2 = 16; o2 > 0; o2 >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o2));
      if ((tid & 31) == 0) atomicMax(&s_vmax, __float_as_uint(mx));
    }
    __syncthreads();
    // scale = 2^e >= max, so every component / scale lies in [-1, 1]
    const uint32_t ebits = (s_vmax & 0x7f800000u);
    const float vscale = ebits == 0u ? 1.f : __uint_as_float(ebits + 0x00800000u);
    const float vinv = 1.f / vscale;
    for (int u = warp; u < nchunks_pad * UPC; u += NTHREADS / 32) {
      const int ci = u / UPC, j = (u % UPC) * 8 + ((tid & 31) >> 2), p = tid & 3;
      const int rr = ci / cpr;
      const int r = r_begin + rr, cc = (ci - rr * cpr) * KC;
      float2 v = make_float2(0.f, 0.f);
      if (ci < nchunks && cc + j < nc) {
        v = load_vis(r, cc + j, p);
        if (job.weights != nullptr) {
          const float wgt = __ldg(&job.weights[(row0 + r) * job.n_chan + c0 + cc + j]);
          v = wgt == 0.f ? make_float2(0.f, 0.f) : make_float2(v.x * wgt, v.y * wgt);   // weight 0 = flagged: exact zero
        }
        v = make_float2(v.x * vinv, v.y * vinv);
      }
      const __half hr = __float2half_rn(v.x), hi = __float2half_rn(v.y);
      const __half lr = __float2half_rn(v.x - __half2float(hr)), li = __float2half_rn(v.y - __half2float(hi));
      // element (n, k) of the chunk's N x K operand: ((k/8)*2 + n/8)*128 + (n%8)*16 + (k%8)*2 bytes, k = 2 j + part
      unsigned char* Bc = sB + static_cast<size_t>(ci) * CHUNK_BYTES;
      auto at2 = [&](int n) -> __half2* {
        return reinterpret_cast<__half2*>(Bc + ((j >> 2) * 2 + (n >> 3)) * 128 + (n & 7) * 16 + (j & 3) * 4);
      };
      *at2(2 * p) = __halves2half2(hr, __hneg(hi));     // column (p,re): rows (v,cos) = Re V, (v,sin) = -Im V
      *at2(2 * p + 1) = __halves2half2(hi, hr);         // column (p,im): rows (v,cos) = Im V, (v,sin) =  Re V
      *at2(2 * p + 8) = __halves2half2(lr, __hneg(li));
      *at2(2 * p + 9) = __halves2half2(li, lr);
    }
#else
    const float vscale = 1.f;
    for (int u = warp; u < nchunks_pad * UPC; u += NTHREADS / 32) {
      const int ci = u / UPC, j = (u % UPC) * 8 + ((tid & 31) >> 2), p = tid & 3;
      const int rr = ci / cpr;
      const int r = r_begin + rr, cc = (ci - rr * cpr) * KC;
      float2 v = make_float2(0.f, 0.f);
      if (ci < nchunks && cc + j < nc) {
        v = load_vis(r, cc + j, p);
        if (job.weights != nullptr) {                  // weighting at load
          const float wgt = __ldg(&job.weights[(row0 + r) * job.n_chan + c0 + cc + j]);
          v = wgt == 0.f ? make_float2(0.f, 0.f) : make_float2(v.x * wgt, v.y * wgt);   // weight 0 = flagged: exact zero
        }
      }
      const float hr = tf32_round(v.x), hi = tf32_round(v.y);
      const float lr = tf32_round(v.x - hr), li = tf32_round(v.y - hi);
      float* Bf = reinterpret_cast<float*>(sB + static_cast<size_t>(ci) * CHUNK_BYTES);
      auto at2 = [&](int n) -> float2* {
        return reinterpret_cast<float2*>(&Bf[((j >> 1) * 2 + (n >> 3)) * 32 + (n & 7) * 4 + (j & 1) * 2]);
      };
      *at2(2 * p) = make_float2(hr, -hi);              // column (p,re): rows (v,cos) = Re V, (v,sin) = -Im V
      *at2(2 * p + 1) = make_float2(hi, hr);           // column (p,im): rows (v,cos) = Im V, (v,sin) =  Re V
      *at2(2 * p + 8) = make_float2(lr, -li);
      *at2(2 * p + 9) = make_float2(li, lr);
    }
#endif
    tc::fence_proxy_async();
    __syncthreads();

    // The chunk stream of a tile is walked in ring revolutions of NA slots (slot = position in the
    // unrolled body); an accumulator group is RPG revolutions.  Slots past the tile's last chunk still
    // cycle their barriers, without stores or MMAs.
    const int nrev = (nchunks + NA - 1) / NA;
    if (gi >= NG) {
      // ===== service warp of group `mygroup`: warp-uniform control flow, one elected lane issues =====
      // every operand below derives from warp-shuffled values, so it stays in uniform registers
      const uint32_t bbase = __shfl_sync(0xffffffffu, tc::smem_u32(sB), 0);
      const uint32_t gt = __shfl_sync(0xffffffffu, tmem, 0) + mygroup * GCOLS;
      const uint32_t sbar = __shfl_sync(0xffffffffu, bar0, 0) + 8 * mygroup * NBAR;
      const int n_u = __shfl_sync(0xffffffffu, nchunks, 0);
      const int nrev_u = (n_u + NA - 1) / NA;
      for (int round = 0; round < ROUNDS; ++round) {
        int rig = 0;
        for (int rev = 0; rev < nrev_u; ++rev) {
          const bool group_last = rig == RPG - 1 || rev == nrev_u - 1;
          const uint32_t d0 = gt + D_COL + 16 * (q & 1);
          if (rig == 0)                                // accumulator q & 1 drained (group q - 2; fresh barriers pass)
            tc::mbar_wait(sbar + 16 * NA + 16 + 8 * (q & 1), ((q - 2) >> 1) & 1);
#pragma unroll
          for (int s = 0; s < NA; ++s) {
            const int ci = rev * NA + s;
            tc::mbar_wait(sbar + 8 * s, phase);
            tc::fence_after_thread_sync();
            const uint64_t bdesc0 = tc::make_smem_desc(bbase + ci * CHUNK_BYTES, 256, 128);
            if (tc::elect_one()) {
#ifdef IDG_TC_FP16
#pragma unroll
              for (int half = 0; half < KC / 8; ++half)   // 8 visibilities = 16 k-rows of B, 512 bytes on
#pragma unroll
                for (int part = 0; part < 2; ++part)      // heads, remainders: one K = 16 MMA each
                  tc::mma_f16_ts(d0, gt + s * A_COLS + half * 16 + part * 8, bdesc0 + half * (512 >> 4), IDESC,
                                 (rig > 0 || s > 0 || half > 0 || part > 0) ? 1u : 0u);
#else
#pragma unroll
              for (int part = 0; part < 2; ++part)
#pragma unroll
                for (int ks = 0; ks < KC / 4; ++ks)
                  tc::mma_tf32_ts(d0, gt + s * A_COLS + part * 2 * KC + ks * 8, bdesc0 + ks * (512 >> 4), IDESC,
                                  (rig > 0 || s > 0 || part > 0 || ks > 0) ? 1u : 0u);
#endif
              tc::mma_commit(sbar + 8 * NA + 8 * s);
              if (s == NA - 1 && group_last) tc::mma_commit(sbar + 16 * NA + 8 * (q & 1));
            }
            __syncwarp();
          }
          phase ^= 1;
          if (group_last) { rig = 0; ++q; } else { ++rig; }
        }
      }
    } else {
      // ===== compute threads: one pixel of the group's current tile each =====
      float acc[8], pacc[8];
      int ppix = -1;                                   // tile whose last accumulator group is still in flight
      bool pending = false;                            // the ring's last slot is stored but not yet handed over

      auto drain = [&](int qq, float (&dst)[8]) {
        tc::mbar_wait(gbar + 16 * NA + 8 * (qq & 1), (qq >> 1) & 1);
        tc::fence_after_thread_sync();
        uint32_t d[16];
        tc::tmem_ld16(gtmem + D_COL + 16 * (qq & 1), d);
        tc::tmem_wait_ld();
        tc::fence_before_thread_sync();
        tc::mbar_arrive(gbar + 16 * NA + 16 + 8 * (qq & 1));
#pragma unroll
        for (int n = 0; n < 8; ++n) dst[n] += __uint_as_float(d[n]) + __uint_as_float(d[n + 8]);
      };
      // a finished tile: partial sums of earlier segments in, then either the partial sum out or
      // the epilogue (step a3): A-term sandwich and taper, once per pixel
      auto finalize = [&](const float (&a)[8], int pix) {
        float2 x[4], z[4];
#pragma unroll
        for (int p = 0; p < 4; ++p) x[p] = make_float2(a[2 * p] * vscale, a[2 * p + 1] * vscale);
        if (!first_seg) {
#pragma unroll
          for (int p = 0; p < 4; ++p) {
            const float2 prev = o[p * L * L + pix];
            x[p].x += prev.x;
            x[p].y += prev.y;
          }
        }
        if (last_seg) {
          const float4 mp0 = __ldg(&ap[pix * 2]), mp1 = __ldg(&ap[pix * 2 + 1]);
          const float4 mq0 = __ldg(&aq[pix * 2]), mq1 = __ldg(&aq[pix * 2 + 1]);
          float t = __ldg(&job.taper[pix]);
          if (job.power_norm) t *= frobenius_inv(mp0, mp1, mq0, mq1);    // PAPER.md:257, R22
          sandwich(x, mp0, mp1, mq0, mq1, t, z);
#pragma unroll
          for (int p = 0; p < 4; ++p) o[p * L * L + pix] = z[p];
        } else {
#pragma unroll
          for (int p = 0; p < 4; ++p) o[p * L * L + pix] = x[p];
        }
      };
      auto hand_off = [&](uint32_t full_bar) {
        tc::tmem_wait_st();
        tc::fence_before_thread_sync();
        tc::mbar_arrive(full_bar);
      };

      for (int round = 0; round < ROUNDS; ++round) {
        const int pix = (round * NG + gi) * kTileM + tpix;
        const int ix = pix % L - L / 2, iy = pix / L - L / 2;
        const float np = job.nprime[pix];
#pragma unroll
        for (int n = 0; n < 8; ++n) acc[n] = 0.f;
        // per-(row, pixel) slope and offset of the phase; amortised over the row's channels
        float pa, pb;
        // ROT: the phase is linear in the channel, phi(c + 1) = phi(c) + delta with delta = pa * dkappa per (row,
        // pixel), so e(c + 1) = e(c) rot, rot = exp(i delta) (the per-row precomputation, one step
        // further).  Kept as kh = 1 - cos(delta) and sg = sin(delta), both to RELATIVE fp32 accuracy (a rotor error
        // grows linearly along the chain): Taylor series at delta for |delta| < 0.5, at delta / 4 with two angle
        // doublings for |delta| < 3, the accurate sincosf beyond (short rows of long baselines).
        [[maybe_unused]] float2 nk2 = make_float2(0.f, 0.f);     // (-2 kh, -2 kh) = -4 sin^2(delta / 2)
        [[maybe_unused]] float kh = 0.f, sg = 0.f;
        auto row_setup = [&](int r) {
          // the row's 32 bytes as two 128-bit loads from an address kept in a register
          const float4 ra = tc::lds128(srow_addr + r * 32), rb = tc::lds128(srow_addr + r * 32 + 16);
          RowDataTc rd;
          rd.alpha_fix = __float_as_int(ra.x); rd.beta_fix = __float_as_int(ra.y); rd.gamma = ra.z; rd.us = ra.w;
          rd.vs = rb.x; rd.ws = rb.y; rd.dmax = rb.z;
          pa = fmaf(rd.vs, static_cast<float>(iy), fmaf(rd.ws, np, rd.us * static_cast<float>(ix)));
          const int32_t bf = wrap_dot2(rd.alpha_fix, ix, rd.beta_fix, iy);                  // wraps: exact mod 1 cycle
          pb = fmaf(rd.gamma, np, static_cast<float>(bf) * 1.4629180792671596e-9f);   // 2 pi / 2^32
          if constexpr (ROT) {
            const float delta = pa * job.dkappa_f;
            if (rd.dmax < 0.5f) {                        // CTA-uniform: the series at delta itself (error < 5e-9 relative)
              const float t = delta * delta;
              float s1 = fmaf(t, -1.9841270e-4f, 8.3333333e-3f);
              s1 = fmaf(t, s1, -1.6666667e-1f);
              sg = fmaf(delta * t, s1, delta);
              float k1 = fmaf(t, -2.4801587e-5f, 1.3888889e-3f);
              k1 = fmaf(t, k1, -4.1666667e-2f);
              k1 = fmaf(t, k1, 0.5f);
              kh = k1 * t;
            } else if (rd.dmax < 3.0f) {
              const float x = 0.25f * delta, t = x * x;
              // sin x = x (1 - t/6 + t^2/120 - t^3/5040 + t^4/362880), 1 - cos x = t (1/2 - t/24 + t^2/720 - t^3/40320)
              float s1 = fmaf(t, 2.7557319e-6f, -1.9841270e-4f);
              s1 = fmaf(t, s1, 8.3333333e-3f);
              s1 = fmaf(t, s1, -1.6666667e-1f);
              s1 = fmaf(x * t, s1, x);
              float k1 = fmaf(t, -2.4801587e-5f, 1.3888889e-3f);
              k1 = fmaf(t, k1, -4.1666667e-2f);
              k1 = fmaf(t, k1, 0.5f);
              k1 *= t;
              // doubling: sin 2x = 2 s (1 - k), 1 - cos 2x = 2 s^2
              const float s2 = 2.f * s1 * (1.f - k1), k2 = 2.f * s1 * s1;
              sg = 2.f * s2 * (1.f - k2);
              kh = 2.f * s2 * s2;
            } else {
              // from the half angle: 1 - cos(delta) would cancel for the pixels near the subgrid centre, whose delta
              // is small although the row's dmax is not (3e-8 absolute in kh grows as j^2 along the recurrence)
              float sh, ch;
              sincosf(0.5f * delta, &sh, &ch);
              kh = 2.f * sh * sh;
              sg = 2.f * sh * ch;
            }
            nk2 = make_float2(-2.f * kh, -2.f * kh);
          }
        };
        int r = r_begin, cc = 0;
        row_setup(r);
        uint32_t dk_addr = sdk_addr;
        int rig = 0, gin = 0;                          // revolutions in the current group, groups closed in this tile
        for (int rev = 0; rev < nrev; ++rev) {
#pragma unroll
          for (int s = 0; s < NA; ++s) {
            constexpr bool valid = true;                // padding chunks are computed like any other
            // the previous slot goes to the service warp before this one's arithmetic: its stores were
            // issued a whole hand-off / wait / store sequence ago
            if (s > 0) hand_off(gbar + 8 * (s - 1));
            else if (pending) hand_off(gbar + 8 * (NA - 1));
            // the A words of a chunk (channels past the row's last one are generated like any other and meet zero rows
            // of B: skipping a chunk's empty half under a CTA-uniform test cost 6 % on config 2 and on config 3)
            uint32_t hi[KC / 8][16];
            [[maybe_unused]] uint32_t lo[KC / 8][16];
#ifdef IDG_TC_FP16
            if constexpr (ROT) {
              // one __sincosf per 8 channels (which bounds the growth of rounding errors), then 7 rotations:
              // d(c + 1) = d(c) - 4 sin^2(delta / 2) e(c), e(c + 1) = e(c) + d(c + 1), d(1) = e(0) (rot - 1),
              // both components of e = (cos, sin) in one packed instruction each
#pragma unroll
              for (int half = 0; half < KC / 8; ++half) {
                const float ph = fmaf(pa, tc::lds32(dk_addr + half * 32), pb);
                float2 e;
                __sincosf(ph, &e.y, &e.x);
                float2 d = make_float2(fmaf(-kh, e.x, -sg * e.y), fmaf(-kh, e.y, sg * e.x));
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                  if (j == 1) e = __fadd2_rn(e, d);
                  if (j > 1) { d = ffma2(e, nk2, d); e = __fadd2_rn(e, d); }
                  const __half2 q = __floats2half2_rn(e.x, e.y);
                  const uint32_t qw = *reinterpret_cast<const uint32_t*>(&q);
                  const float2 l = tc::sub_half2(e, qw);
                  const __half2 rr = __floats2half2_rn(l.x, l.y);
                  hi[half][j] = qw;
                  hi[half][8 + j] = *reinterpret_cast<const uint32_t*>(&rr);
                }
              }
            } else
#endif
            if (valid) {
#pragma unroll
              for (int half = 0; half < KC / 8; ++half) {
                const float4 dka = tc::lds128(dk_addr + half * 32);
                const float4 dkb = tc::lds128(dk_addr + half * 32 + 16);
                const float2 dk2[4] = {make_float2(dka.x, dka.y), make_float2(dka.z, dka.w),
                                       make_float2(dkb.x, dkb.y), make_float2(dkb.z, dkb.w)};
                const float2 pa2 = make_float2(pa, pa), pb2 = make_float2(pb, pb), m1 = make_float2(-1.f, -1.f);
#pragma unroll
                for (int j2 = 0; j2 < 4; ++j2) {
                  // two visibilities per packed FFMA; (cos, sin) pairs split by one packed FFMA each
                  const float2 ph = ffma2(pa2, dk2[j2], pb2);
                  float2 e0, e1;                        // (cos, sin) of the two phases
                  __sincosf(ph.x, &e0.y, &e0.x);
                  __sincosf(ph.y, &e1.y, &e1.x);
#ifdef IDG_TC_FP16
                  // (cos, sin) -> fp16 head pair and fp16 remainder pair, one 32-bit word each
                  const __half2 q0 = __floats2half2_rn(e0.x, e0.y), q1 = __floats2half2_rn(e1.x, e1.y);
                  const float2 l0 = tc::sub_half2(e0, *reinterpret_cast<const uint32_t*>(&q0));
                  const float2 l1 = tc::sub_half2(e1, *reinterpret_cast<const uint32_t*>(&q1));
                  const __half2 r0 = __floats2half2_rn(l0.x, l0.y), r1 = __floats2half2_rn(l1.x, l1.y);
                  hi[half][2 * j2] = *reinterpret_cast<const uint32_t*>(&q0);
                  hi[half][2 * j2 + 1] = *reinterpret_cast<const uint32_t*>(&q1);
                  hi[half][8 + 2 * j2] = *reinterpret_cast<const uint32_t*>(&r0);
                  hi[half][8 + 2 * j2 + 1] = *reinterpret_cast<const uint32_t*>(&r1);
#else
                  const float2 h0 = make_float2(tf32_head(e0.x), tf32_head(e0.y));
                  const float2 h1 = make_float2(tf32_head(e1.x), tf32_head(e1.y));
                  const float2 l0 = ffma2(h0, m1, e0), l1 = ffma2(h1, m1, e1);      // e - head, exact
                  hi[half][4 * j2] = __float_as_uint(h0.x);
                  hi[half][4 * j2 + 1] = __float_as_uint(h0.y);
                  hi[half][4 * j2 + 2] = __float_as_uint(h1.x);
                  hi[half][4 * j2 + 3] = __float_as_uint(h1.y);
                  lo[half][4 * j2] = __float_as_uint(l0.x);
                  lo[half][4 * j2 + 1] = __float_as_uint(l0.y);
                  lo[half][4 * j2 + 2] = __float_as_uint(l1.x);
                  lo[half][4 * j2 + 3] = __float_as_uint(l1.y);
#endif
                }
              }
            }
            tc::mbar_wait(gbar + 8 * NA + 8 * s, phase ^ 1);          // MMAs of the last revolution (a fresh barrier passes parity 1)
            if (valid) {
#pragma unroll
              for (int half = 0; half < KC / 8; ++half) {
#ifdef IDG_TC_FP16
                // per 8 visibilities: 8 head words, 8 remainder words (16 columns)
                if constexpr (KC == 8) tc::tmem_st16(gtmem + s * A_COLS, hi[half]);
                else if (half == 0) tc::tmem_st32(gtmem + s * A_COLS, hi[0], hi[KC / 8 - 1]);
#else
                if constexpr (KC == 8) {
                  tc::tmem_st32(gtmem + s * A_COLS, hi[half], lo[half]);     // heads and remainders are adjacent
                } else {
                  tc::tmem_st16(gtmem + s * A_COLS + half * 16, hi[half]);
                  tc::tmem_st16(gtmem + s * A_COLS + 2 * KC + half * 16, lo[half]);
                }
#endif
              }
              dk_addr += KC * 4;
              cc += KC;
              if (cc >= nc) {
                cc = 0;
                dk_addr = sdk_addr;
                if (++r < r_end) row_setup(r);
              }
            }
          }
          pending = true;
          phase ^= 1;
          if (++rig == RPG || rev == nrev - 1) {
            // group q closes; group q - 1 was handed over a group ago, so its MMAs are done
            if (ppix >= 0) {
              drain(q - 1, pacc);
              finalize(pacc, ppix);
              ppix = -1;
            } else if (gin > 0) {
              drain(q - 1, acc);
            }
            rig = 0; ++q; ++gin;
          }
        }
        // the tile's last group is drained inside the next tile
#pragma unroll
        for (int n = 0; n < 8; ++n) pacc[n] = acc[n];
        ppix = pix;
      }
      hand_off(gbar + 8 * (NA - 1));
      pending = false;
      drain(q - 1, pacc);
      finalize(pacc, ppix);
    }
  }

  tc::fence_before_thread_sync();
  __syncthreads();
  if (warp == NG * 4) tc::tmem_dealloc(tmem, TMEM_COLS);
}

template <int L, int NG, int KC, int DG, int NA, bool ROT>
cudaError_t launch_rot(const SubgridJob& job, const float4* vis, float2* out, cudaStream_t stream) {
  if (job.count == 0) return cudaSuccess;
#ifdef IDG_TC_FP16
  constexpr int CHUNK_BYTES = KC * 64;
#else
  constexpr int CHUNK_BYTES = KC * 128;
#endif
  const int cpr_max = (job.n_chan + KC - 1) / KC;
  const int cap_chunks = std::min(job.max_nt * cpr_max, kMaxBBytes / CHUNK_BYTES);
  const size_t dyn = static_cast<size_t>(cap_chunks + NA - 1) * CHUNK_BYTES;   // + padding chunks
  auto kernel = gridder_tc_kernel<L, NG, KC, DG, NA, ROT>;
  // per launch (the attribute belongs to the (function, device) pair and the call is cheap), but always the
  // instantiation's MAXIMUM, never this launch's own size: two host threads with plans of different shapes could
  // otherwise interleave set(large), set(small), launch(large) and fail the launch
  constexpr int kDynMax = kMaxBBytes + (NA - 1) * CHUNK_BYTES;
  cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kDynMax);
  if (e != cudaSuccess) return e;
  kernel<<<static_cast<unsigned>(job.count), NG * kTileM + NG * 32, dyn, stream>>>(job, vis, out, cap_chunks);
  count_launch();
  note_kernel(IDG_K_GRIDDER, IDG_KMASK_TC(NG) | (ROT ? IDG_KMASK_ROT : 0));
  return cudaGetLastError();
}

// Rotation along the channel axis needs uniformly spaced channels (job.dkappa != 0, checked by the planner).
template <int L, int NG, int KC, int DG, int NA>
cudaError_t launch(const SubgridJob& job, const float4* vis, float2* out, cudaStream_t stream) {
#if defined(IDG_TC_FP16)
  if (job.dkappa != 0.0) return launch_rot<L, NG, KC, DG, NA, true>(job, vis, out, stream);
#endif
  return launch_rot<L, NG, KC, DG, NA, false>(job, vis, out, stream);
}

// Groups per CTA.  Tensor memory holds four groups per SM whatever the split; with fewer groups per CTA
// several CTAs (different subgrids) share the SM, so one CTA's prologue (B staging, row constants) and
// tail overlap the others' arithmetic: measured 4.73 (1 group x 4 CTAs), 4.65 (2 x 2), 4.53 (4 x 1)
// pairs/clk/SM on config 2.  What decides is whether the CTAs' B operands fit shared memory side by side.
template <int L>
cudaError_t launch_l(const SubgridJob& job, const float4* vis, float2* out, cudaStream_t stream) {
  constexpr int KC = IDG_TC_KC;
  const size_t dyn = static_cast<size_t>(std::min(job.max_nt * ((job.n_chan + KC - 1) / KC), kMaxBBytes / (KC * kVisBytes)) + IDG_TC_NA - 1) *
                     (KC * kVisBytes);
  constexpr size_t kStaticAndReserved = 12 * 1024, kSmemPerSm = 227 * 1024;
  if (4 * (dyn + kStaticAndReserved) <= kSmemPerSm) return launch<L, 1, KC, IDG_TC_DG, IDG_TC_NA>(job, vis, out, stream);
  if (2 * (dyn + kStaticAndReserved) <= kSmemPerSm || ((L * L) / kTileM) % 4 != 0)     // L = 48: 18 tiles
    return launch<L, 2, KC, IDG_TC_DG, IDG_TC_NA>(job, vis, out, stream);
  if constexpr (((L * L) / kTileM) % 4 == 0) return launch<L, 4, KC, IDG_TC_DG, IDG_TC_NA>(job, vis, out, stream);
  return cudaErrorInvalidValue;
}

}  // namespace

bool gridder_tc_fits(int n_chan, int max_nt) {
  constexpr int KC = IDG_TC_KC;
  return n_chan <= kMaxChanTc - KC && max_nt <= kMaxRowsTc && (n_chan + KC - 1) / KC <= kMaxBBytes / (KC * kVisBytes);
}

cudaError_t launch_gridder_tc(const SubgridJob& job, const float4* vis, float2* out, cudaStream_t stream) {
  // shapes whose per-subgrid constants do not fit the kernel's shared-memory tables take the SIMT kernel
  if (!gridder_tc_fits(job.n_chan, job.max_nt)) return launch_gridder(job, vis, out, stream);
  switch (job.subgrid_size) {
    case 32:  return launch_l<32>(job, vis, out, stream);
    case 48:  return launch_l<48>(job, vis, out, stream);
    case 64:  return launch_l<64>(job, vis, out, stream);
    case 96:  return launch_l<96>(job, vis, out, stream);
    case 128: return launch_l<128>(job, vis, out, stream);
    case 160: return launch_l<160>(job, vis, out, stream);
    default:  return cudaErrorInvalidValue;
  }
}

}  // namespace idg
