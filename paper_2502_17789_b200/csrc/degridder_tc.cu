// Tensor-core degridder: steps a8-a9 with the 2x2 complex MACs on tcgen05.
//
//   V[k, n] = sum_pix E[k, (pix, part)] B[(pix, part), n]              (Eq. 13 :171-174)
//
// with k a visibility of the subgrid, part in {cos, sin}, n = (polarisation, re/im):
//   E[k, (pix,cos)] = cos 2 pi phi(pix, k),   E[k, (pix,sin)] = sin 2 pi phi(pix, k)
//   B[(pix,cos), (p,re)] = Re S'_p   B[(pix,cos), (p,im)] =  Im S'_p
//   B[(pix,sin), (p,re)] = Im S'_p   B[(pix,sin), (p,im)] = -Re S'_p       (V = sum S' e^{-i phi})
// S' = M_p (taper S) M_q^H (step a8; R4, R5).  The mirror image of gridder_tc.cu: there a thread owns
// a pixel and the visibilities are the contraction, here a thread owns a visibility (its uvw offsets
// live in registers) and the pixels are the contraction.  Operands are split into tf32 heads and
// fp32 remainders and the accumulators are drained every DG chunks exactly as in the gridder.
//
// One CTA per subgrid: NG groups of 128 compute threads, one service warp per group, two producer warps.
//   producer warps   stream the subgrid through shared memory in stages of 256 pixels: loads the four
//                    polarisation planes, applies taper and A-terms once per pixel and writes the B
//                    operand (heads and remainders, canonical K-major core matrices) plus n'(pixel).
//   compute group    owns a tile of 128 visibilities (thread = visibility = MMA row = TMEM lane) and a
//                    share of every stage's pixels: with T tiles in a round and NG groups, each tile is
//                    served by NG / T groups that split the stage's chunks; their partial sums meet in
//                    shared memory at the end of the round (fixed order, deterministic).
//                    Per chunk of 8 pixels of one subgrid row: two phase FFMAs, sincos, head/remainder,
//                    tcgen05.st into the group's A ring; hand-off pipelined as in the gridder.
//   service warp     waits for the stage and for full[slot], one elected lane issues the 4 MMAs
//                    (M = 128, N = 16, K = 8) per chunk, commits to empty[slot], to dfull at an
//                    accumulator group's end and to the stage's empty barrier after its last chunk.
#include <algorithm>
#include <type_traits>

#include "device_math.cuh"
#include "kernels.h"
#include "tc_common.cuh"

namespace idg {

namespace {

#ifndef IDG_DTC_NG
#define IDG_DTC_NG 2
#endif
#ifndef IDG_DTC_DG
#define IDG_DTC_DG 12
#endif
#ifndef IDG_DTC_NA
#define IDG_DTC_NA 3
#endif
#ifndef IDG_DTC_NS
#define IDG_DTC_NS 4
#endif

constexpr int kTileV = 128;           // visibilities per MMA tile = threads per compute group
constexpr int kKC = 8;                // pixels per chunk
constexpr int kStagePix = 256;        // pixels per shared-memory stage
constexpr int kStageChunks = kStagePix / kKC;
// B operand layout: canonical K-major core matrices (8 n-rows x 16 B), the two n-groups of a k-group 128 B
// apart, k-groups (2 pixels x {cos, sin}) kKgBytes apart: 16 B of padding per k-group spread the
// producer's stores over all banks (without it every lane of a store hits the same two).
constexpr int kKgBytes = 272;
constexpr int kChunkBytes = (kKC / 2) * kKgBytes;          // 1088
constexpr int kStageBBytes = kStageChunks * kChunkBytes;   // 34 KB
constexpr int kProducers = 2;                              // producer warps, each half of every stage

__device__ __forceinline__ float dtc_head(float x) { return __uint_as_float(__float_as_uint(x) & 0xffffe000u); }
__device__ __forceinline__ float dtc_round(float x) {
  return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xffffe000u);
}

template <int L, int NG, int DG, int NA, int NS>
__global__ void __launch_bounds__(NG* kTileV + NG * 32 + kProducers * 32, NG == 2 ? 2 : 1)
    degridder_tc_kernel(const SubgridJob job, const float2* __restrict__ in, float4* __restrict__ vis) {
  static_assert((L * L) % kStagePix == 0 && L % kKC == 0 && (NG == 2 || NG == 4) && (NS & (NS - 1)) == 0, "shape");
  static_assert(DG % NA == 0, "an accumulator group is a whole number of ring revolutions");
  constexpr int NSTAGES = (L * L) / kStagePix;
  constexpr int A_COLS = 4 * kKC;                      // per slot: heads [0, 16), remainders [16, 32)
  constexpr int D_COL = NA * A_COLS;                   // then two accumulators of 16 columns
  constexpr int GCOLS = D_COL + 32;
  constexpr int TMEM_COLS = NG * GCOLS <= 128 ? 128 : (NG * GCOLS <= 256 ? 256 : 512);
  static_assert(NG * GCOLS <= 512, "TMEM");
  constexpr int RPG = DG / NA;
  constexpr int NBAR = 2 * NA + 4;                     // per group: full[NA], empty[NA], dfull[2], dempty[2]
  constexpr uint32_t IDESC = tc::make_idesc_tf32(kTileV, 16);

  // dynamic: B ring [NS][32 KB], n' ring [NS][256] f32, partial sums [(NG-1)][128][8] f32
  extern __shared__ __align__(1024) unsigned char smem[];
  unsigned char* sB = smem;
  float* snp = reinterpret_cast<float*>(smem + NS * kStageBBytes);
  float* sred = snp + NS * kStagePix;
  __shared__ __align__(8) uint64_t bars[NG * NBAR + 2 * NS];
  __shared__ uint32_t s_tmem;

  const int tid = threadIdx.x, warp = tid / 32, lane = tid % 32;
  const int64_t sg = job_slot(job, blockIdx.x);
  const int32_t* m = job.meta + (job.first + sg) * kMetaStride;
  const int b = m[0], t0 = m[1], nt = m[2], c0 = m[3], nc = m[4], x0 = m[5], y0 = m[6], wl = m[7];
  const int sp = m[8], sq = m[9], it = m[10];
  // rows used as (-u,-v,-w) of the swapped baseline: the sum predicts V(-u,-v,-w) of (q,p) and its dagger is
  // written (PAPER.md:178 fn 4, R21)
  const bool conj = (m[12] & kMetaConj) != 0;
  const int64_t row0 = static_cast<int64_t>(b) * job.n_times + t0;
  const int K = nt * nc;                               // visibilities of the subgrid
  const int T = (K + kTileV - 1) / kTileV;             // visibility tiles

  const uint32_t bar0 = tc::smem_u32(&bars[0]);
  const uint32_t bar_sfull = bar0 + 8 * NG * NBAR, bar_sempty = bar_sfull + 8 * NS;
  if (tid == 0) {
    for (int gi = 0; gi < NG; ++gi) {
      const uint32_t gb = bar0 + 8 * gi * NBAR;
      for (int i = 0; i < NA; ++i) {
        tc::mbar_init(gb + 8 * i, kTileV);
        tc::mbar_init(gb + 8 * NA + 8 * i, 1);
      }
      for (int i = 0; i < 2; ++i) {
        tc::mbar_init(gb + 16 * NA + 8 * i, 1);
        tc::mbar_init(gb + 16 * NA + 16 + 8 * i, kTileV);
      }
    }
    for (int i = 0; i < NS; ++i) {
      tc::mbar_init(bar_sfull + 8 * i, kProducers);
      tc::mbar_init(bar_sempty + 8 * i, NG);
    }
    tc::fence_barrier_init();
  }
  if (warp == NG * 4) tc::tmem_alloc(tc::smem_u32(&s_tmem), TMEM_COLS);
  tc::fence_before_thread_sync();
  __syncthreads();
  tc::fence_after_thread_sync();
  const uint32_t tmem = s_tmem;

  const int uwarp = __shfl_sync(0xffffffffu, warp, 0);  // warp-uniform to the compiler
  const bool is_compute = uwarp < NG * 4, is_service = !is_compute && uwarp < NG * 5;
  const int gi = is_compute ? (uwarp >> 2) : (uwarp - NG * 4);   // group of a compute / service warp
  const uint32_t gbar = tc::opaque(bar0 + 8 * gi * NBAR);
  const uint32_t gtmem = tc::opaque(tmem + gi * GCOLS + (static_cast<uint32_t>((warp & 3) * 32) << 16));
  const int tpix = tid & (kTileV - 1);

  int q = 0;                                           // accumulator groups closed
  uint32_t phase = 0;                                  // parity of the current revolution
  int sc0 = 0;                                         // stages streamed before this round

  for (int t_base = 0; t_base < T; t_base += NG, sc0 += NSTAGES) {
    const int t_round = min(NG, T - t_base);           // tiles of this round
    const int lgP = t_round == 1 ? (NG == 4 ? 2 : 1) : ((t_round == 2 && NG == 4) ? 1 : 0);   // groups per tile P = 1 << lgP
    const int tile_l = gi % t_round, part = gi / t_round;
    const bool active = part < (1 << lgP);
    const int lgn = 5 - lgP;                           // a part's chunks per stage: ncs = 1 << lgn
    const int ncs = 1 << lgn;
    const int total = NSTAGES << lgn;                  // chunks of this group in the round
    const int nrev = (total + NA - 1) / NA;

    if (!is_compute && !is_service) {
      // ===== producer warp (step a8): taper and A-term sandwich once per pixel -> B operand =====
      const float4* __restrict__ ap = job.aterms + (static_cast<int64_t>(sp) * job.n_intervals + it) * (L * L * 2);
      const float4* __restrict__ aq = job.aterms + (static_cast<int64_t>(sq) * job.n_intervals + it) * (L * L * 2);
      const float2* __restrict__ sub = in + sg * 4 * L * L;
      const int pw = uwarp - NG * 5;                   // producer warp index
      for (int st = 0; st < NSTAGES; ++st) {
        const int gst = sc0 + st, slot = gst & (NS - 1);
        if (gst >= NS) tc::mbar_wait_backoff(bar_sempty + 8 * slot, ((gst / NS) - 1) & 1, 256);
        float* Bs = reinterpret_cast<float*>(sB + slot * kStageBBytes);
#pragma unroll 2
        for (int i = 0; i < kStagePix / (32 * kProducers); ++i) {
          const int lp = (pw * (kStagePix / (32 * kProducers)) + i) * 32 + lane, pix = st * kStagePix + lp;
          float2 x[4], z[4];
#pragma unroll
          for (int p = 0; p < 4; ++p) x[p] = __ldg(&sub[p * L * L + pix]);
          // M_p (t S) M_q^H == t (M_p S M_q^H)
          sandwich(x, __ldg(&ap[pix * 2]), __ldg(&ap[pix * 2 + 1]), __ldg(&aq[pix * 2]), __ldg(&aq[pix * 2 + 1]),
                   __ldg(&job.taper[pix]), z);
          snp[slot * kStagePix + lp] = __ldg(&job.nprime[pix]);
          // element (n, k) of a chunk's N x K operand lives at (k/4)*kKgBytes + (n/8)*128 + (n%8)*16 + (k%4)*4
          // bytes; k = 2 j + {cos, sin}, j = pixel within the chunk
          const int ci = lp >> 3, j = lp & 7;
          float* Bf = Bs + ci * (kChunkBytes / 4);
          auto at2 = [&](int n) -> float2* {
            return reinterpret_cast<float2*>(&Bf[(j >> 1) * (kKgBytes / 4) + (n >> 3) * 32 + (n & 7) * 4 + (j & 1) * 2]);
          };
#pragma unroll
          for (int p = 0; p < 4; ++p) {
            const float hr = dtc_round(z[p].x), hi = dtc_round(z[p].y);
            const float lr = dtc_round(z[p].x - hr), li = dtc_round(z[p].y - hi);
            *at2(2 * p) = make_float2(hr, hi);          // column (p,re): rows (pix,cos) = Re S', (pix,sin) =  Im S'
            *at2(2 * p + 1) = make_float2(hi, -hr);     // column (p,im): rows (pix,cos) = Im S', (pix,sin) = -Re S'
            *at2(2 * p + 8) = make_float2(lr, li);
            *at2(2 * p + 9) = make_float2(li, -lr);
          }
        }
        tc::fence_proxy_async();
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(bar_sfull + 8 * slot);
      }
    } else if (is_service) {
      // ===== service warp of group gi: warp-uniform control flow, one elected lane issues =====
      const uint32_t bbase = __shfl_sync(0xffffffffu, tc::smem_u32(sB), 0);
      const uint32_t gt = __shfl_sync(0xffffffffu, tmem, 0) + gi * GCOLS;
      const uint32_t sbar = __shfl_sync(0xffffffffu, bar0, 0) + 8 * gi * NBAR;
      const uint32_t sfull = __shfl_sync(0xffffffffu, bar_sfull, 0), sempty = sfull + 8 * NS;
      if (!active) {
        // an idle group still counts on the stage barriers
        for (int st = 0; st < NSTAGES; ++st) {
          const int gst = sc0 + st, slot = gst & (NS - 1);
          tc::mbar_wait(sfull + 8 * slot, (gst / NS) & 1);
          if (tc::elect_one()) tc::mbar_arrive(sempty + 8 * slot);
          __syncwarp();
        }
      } else {
        int rig = 0;
        for (int rev = 0; rev < nrev; ++rev) {
          const bool group_last = rig == RPG - 1 || rev == nrev - 1;
          const uint32_t d0 = gt + D_COL + 16 * (q & 1);
          if (rig == 0)                                // accumulator q & 1 drained (group q - 2; fresh barriers pass)
            tc::mbar_wait(sbar + 16 * NA + 16 + 8 * (q & 1), ((q - 2) >> 1) & 1);
#pragma unroll
          for (int s = 0; s < NA; ++s) {
            const int n = rev * NA + s;                // chunk of this group in the round
            const bool valid = n < total;
            const int st = n >> lgn, cl = n & (ncs - 1);
            const int gst = sc0 + st, slot = gst & (NS - 1);
            if (valid && cl == 0) tc::mbar_wait(sfull + 8 * slot, (gst / NS) & 1);
            tc::mbar_wait(sbar + 8 * s, phase);
            tc::fence_after_thread_sync();
            const uint64_t bdesc0 =
                tc::make_smem_desc(bbase + slot * kStageBBytes + ((part << lgn) + cl) * kChunkBytes, kKgBytes, 128);
            if (tc::elect_one()) {
              if (valid) {
#pragma unroll
                for (int pt = 0; pt < 2; ++pt)
#pragma unroll
                  for (int ks = 0; ks < kKC / 4; ++ks)
                    tc::mma_tf32_ts(d0, gt + s * A_COLS + pt * 2 * kKC + ks * 8, bdesc0 + ks * ((2 * kKgBytes) >> 4), IDESC,
                                    (rig > 0 || s > 0 || pt > 0 || ks > 0) ? 1u : 0u);
              }
              tc::mma_commit(sbar + 8 * NA + 8 * s);
              if (valid && cl == ncs - 1) tc::mma_commit(sempty + 8 * slot);
              if (s == NA - 1 && group_last) tc::mma_commit(sbar + 16 * NA + 8 * (q & 1));
            }
            __syncwarp();
          }
          phase ^= 1;
          if (group_last) { rig = 0; ++q; } else { ++rig; }
        }
      }
    }

    float acc[8];
#pragma unroll
    for (int n = 0; n < 8; ++n) acc[n] = 0.f;
    const int k = (t_base + tile_l) * kTileV + tpix;   // my visibility (compute threads)
    const bool vis_ok = is_compute && active && k < K;
    const int vr = vis_ok ? k / nc : 0, vc = vis_ok ? k - vr * nc : 0;

    if (is_compute && active) {
      // ===== compute threads: one visibility of the group's tile each =====
      // phase [rad] = al fx + be fy + ga n', offsets relative to the subgrid centre from fp64.  The part that is
      // linear in the pixel position reaches hundreds of radians at the subgrid's edge (L = 128, 160), more than
      // fp32 resolves to 1e-6, so a chunk's first pixel takes it modulo one cycle EXACTLY, in 32-bit fixed
      // point (alpha_fix * ix + beta_fix * iy wraps), as the gridders do; only al * j (j < 8) and ga n' are fp32.
      float al = 0.f, ga = 0.f;
      int32_t alpha_fix = 0, beta_fix = 0;             // cycles per pixel * 2^32
      if (vis_ok) {
        const double S = job.image_size;
        const double u0 = (x0 + L / 2 - job.grid_size / 2) / S;
        const double v0 = (y0 + L / 2 - job.grid_size / 2) / S;
        const double w0 = job.w_step > 0.0 ? (wl + 0.5) * job.w_step : 0.0;
        const double* uvw = job.uvw + (row0 + vr) * 3;
        const double kap = job.kappa[c0 + vc];
        const double two_pi = 6.283185307179586476925286766559;
        const double sgn = conj ? -1.0 : 1.0;
        const double alpha = (sgn * uvw[0] * kap - u0) * (S / L), beta = (sgn * uvw[1] * kap - v0) * (S / L);
        al = static_cast<float>(two_pi * alpha);
        alpha_fix = static_cast<int32_t>(static_cast<uint32_t>(static_cast<int64_t>(rint(alpha * 4294967296.0))));
        beta_fix = static_cast<int32_t>(static_cast<uint32_t>(static_cast<int64_t>(rint(beta * 4294967296.0))));
        ga = static_cast<float>(two_pi * (sgn * uvw[2] * kap - w0));
      }
      // A warp none of whose 32 visibilities exists (the ragged tail of the subgrid's last tile) generates no
      // phasors and stores nothing: it only keeps the ring's barriers in step (its tensor-memory rows hold
      // stale finite-or-not values that no thread reads: MMA rows are independent).  The SIMT work is thus
      // padded to 32 visibilities, not 128 (low-occupancy tails).
      const bool warp_on = (t_base + tile_l) * kTileV + (uwarp & 3) * 32 < K;      // from warp-uniform values only
      bool pending = false;                            // the ring's last slot is stored but not yet handed over
      auto drain = [&](int qq) {
        tc::mbar_wait(gbar + 16 * NA + 8 * (qq & 1), (qq >> 1) & 1);
        tc::fence_after_thread_sync();
        uint32_t d[16];
        tc::tmem_ld16(gtmem + D_COL + 16 * (qq & 1), d);
        tc::tmem_wait_ld();
        tc::fence_before_thread_sync();
        tc::mbar_arrive(gbar + 16 * NA + 16 + 8 * (qq & 1));
#pragma unroll
        for (int n = 0; n < 8; ++n) acc[n] += __uint_as_float(d[n]) + __uint_as_float(d[n + 8]);
      };
      auto hand_off = [&](uint32_t full_bar) {
        tc::tmem_wait_st();
        tc::fence_before_thread_sync();
        tc::mbar_arrive(full_bar);
      };

      const uint32_t snp_addr = tc::smem_u32(snp);
      uint32_t np_addr = 0;                            // n' of the next chunk's pixels
      int ix0 = 0, iy = 0;                             // pixel offsets of the next chunk's first pixel
      // cl = chunks left in my share of the current stage; kept in plain registers (`opaque`)
      const int ncs_r = static_cast<int>(tc::opaque(static_cast<uint32_t>(ncs)));
      const int lp0 = static_cast<int>(tc::opaque(static_cast<uint32_t>((part << lgn) * kKC)));
      int cl = 0, st = 0, rig = 0, gin = 0;
      // the round's chunk loop, in two copies: warps with visibilities (ON: no test inside the loop) and the
      // bookkeeping-only copy for the warps of a ragged tail
      auto chunk_loop = [&](auto on_tag) {
      constexpr bool ON = decltype(on_tag)::value;
      for (int rev = 0; rev < nrev; ++rev) {
#pragma unroll
        for (int s = 0; s < NA; ++s) {
          // slots past the round's last chunk are computed and stored like any other (the service warp issues
          // no MMA for them), so the compute threads never test whether a slot is in use
          constexpr bool valid = ON;
          // the previous slot goes to the service warp before this one's arithmetic
          if (s > 0) hand_off(gbar + 8 * (s - 1));
          else if (pending) hand_off(gbar + 8 * (NA - 1));
          uint32_t hi[16], lo[16];
          if (valid) {
            if (cl == 0 && st < NSTAGES) {
              // a new stage: wait for the producer, find my share of its pixels
              const int gst = sc0 + st, slot = gst & (NS - 1);
              tc::mbar_wait(bar_sfull + 8 * slot, (gst / NS) & 1);
              const int pix0 = st * kStagePix + lp0;
              np_addr = snp_addr + (slot * kStagePix + lp0) * 4;
              ix0 = pix0 % L - L / 2;
              iy = pix0 / L - L / 2;
              ++st;
              cl = ncs_r;
            }
            const float4 na = tc::lds128(np_addr), nb = tc::lds128(np_addr + 16);
            const float2 np2[4] = {make_float2(na.x, na.y), make_float2(na.z, na.w),
                                   make_float2(nb.x, nb.y), make_float2(nb.z, nb.w)};
            const float base = static_cast<float>(wrap_dot2(alpha_fix, ix0, beta_fix, iy)) * 1.4629180792671596e-9f;   // 2 pi / 2^32
            const float2 base2 = make_float2(base, base), al2 = make_float2(al, al), ga2 = make_float2(ga, ga);
            const float2 m1 = make_float2(-1.f, -1.f);
#pragma unroll
            for (int j2 = 0; j2 < 4; ++j2) {
              // two pixels per packed FFMA; (cos, sin) pairs split by one packed FFMA each
              const float2 jj = make_float2(static_cast<float>(2 * j2), static_cast<float>(2 * j2 + 1));
              const float2 ph = ffma2(ga2, np2[j2], ffma2(al2, jj, base2));
              float2 e0, e1;                            // (cos, sin) of the two phases
              __sincosf(ph.x, &e0.y, &e0.x);
              __sincosf(ph.y, &e1.y, &e1.x);
              const float2 h0 = make_float2(dtc_head(e0.x), dtc_head(e0.y));
              const float2 h1 = make_float2(dtc_head(e1.x), dtc_head(e1.y));
              const float2 l0 = ffma2(h0, m1, e0), l1 = ffma2(h1, m1, e1);          // e - head, exact
              hi[4 * j2] = __float_as_uint(h0.x);
              hi[4 * j2 + 1] = __float_as_uint(h0.y);
              hi[4 * j2 + 2] = __float_as_uint(h1.x);
              hi[4 * j2 + 3] = __float_as_uint(h1.y);
              lo[4 * j2] = __float_as_uint(l0.x);
              lo[4 * j2 + 1] = __float_as_uint(l0.y);
              lo[4 * j2 + 2] = __float_as_uint(l1.x);
              lo[4 * j2 + 3] = __float_as_uint(l1.y);
            }
          }
          tc::mbar_wait(gbar + 8 * NA + 8 * s, phase ^ 1);            // MMAs of the last revolution (a fresh barrier passes parity 1)
          if (valid) {
            tc::tmem_st16(gtmem + s * A_COLS, hi);
            tc::tmem_st16(gtmem + s * A_COLS + 2 * kKC, lo);
            np_addr += kKC * 4;
            ix0 += kKC;
            if (ix0 >= L / 2) { ix0 = -L / 2; ++iy; }
            --cl;
          }
        }
        pending = true;
        phase ^= 1;
        if (++rig == RPG || rev == nrev - 1) {
          // group q closes; group q - 1 was handed over a group ago, so its MMAs are done
          if (gin > 0) drain(q - 1);
          rig = 0; ++q; ++gin;
        }
      }
      };
      if (warp_on) chunk_loop(std::true_type{}); else chunk_loop(std::false_type{});
      hand_off(gbar + 8 * (NA - 1));
      drain(q - 1);
      // partial sums of the groups that share my tile meet in shared memory
      if (part > 0) {
        float4* r4 = reinterpret_cast<float4*>(sred + ((gi - t_round) * kTileV + tpix) * 8);
        r4[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
        r4[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
      }
    }
    __syncthreads();
    if (vis_ok && part == 0) {
      for (int pp = 1; pp < (1 << lgP); ++pp) {
        const float4* r4 = reinterpret_cast<const float4*>(sred + ((pp * t_round + tile_l - t_round) * kTileV + tpix) * 8);
        const float4 a0 = r4[0], a1 = r4[1];
        acc[0] += a0.x; acc[1] += a0.y; acc[2] += a0.z; acc[3] += a0.w;
        acc[4] += a1.x; acc[5] += a1.y; acc[6] += a1.z; acc[7] += a1.w;
      }
      float4* o = vis + ((row0 + vr) * job.n_chan + c0 + vc) * 2;
      if (conj) {                                       // (XX, XY, YX, YY) <- conj of (XX, YX, XY, YY)
        o[0] = make_float4(acc[0], -acc[1], acc[4], -acc[5]);
        o[1] = make_float4(acc[2], -acc[3], acc[6], -acc[7]);
      } else {
        o[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
        o[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
      }
    }
    __syncthreads();
  }

  tc::fence_before_thread_sync();
  __syncthreads();
  if (warp == NG * 4) tc::tmem_dealloc(tmem, TMEM_COLS);
}

// Two groups per CTA with a two-stage B ring let two CTAs (different subgrids) share an SM, so one CTA's
// prologue and end-of-round reduction overlap the other's arithmetic; four groups and four stages make one
// CTA per SM.  IDG_DTC_NG picks; the default is the measured winner on config 2.
template <int L>
cudaError_t launch(const SubgridJob& job, const float2* in, float4* vis, cudaStream_t stream) {
  if (job.count == 0) return cudaSuccess;
  constexpr int NG = IDG_DTC_NG, NS = NG == 2 ? 2 : IDG_DTC_NS;
  constexpr size_t dyn = NS * kStageBBytes + NS * kStagePix * 4 + (NG - 1) * kTileV * 8 * 4;
  auto kernel = degridder_tc_kernel<L, NG, IDG_DTC_DG, IDG_DTC_NA, NS>;
  // per launch: the attribute belongs to the (function, device) pair and the call is cheap
  cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(dyn));
  if (e != cudaSuccess) return e;
  kernel<<<static_cast<unsigned>(job.count), NG * kTileV + NG * 32 + kProducers * 32, dyn, stream>>>(job, in, vis);
  count_launch();
  note_kernel(IDG_K_DEGRIDDER, IDG_KMASK_TC(NG));
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_degridder_tc(const SubgridJob& job, const float2* in, float4* vis, cudaStream_t stream) {
  switch (job.subgrid_size) {
    case 32:  return launch<32>(job, in, vis, stream);
    case 48:  return launch<48>(job, in, vis, stream);
    case 64:  return launch<64>(job, in, vis, stream);
    case 96:  return launch<96>(job, in, vis, stream);
    case 128: return launch<128>(job, in, vis, stream);
    case 160: return launch<160>(job, in, vis, stream);
    default:  return cudaErrorInvalidValue;
  }
}

}  // namespace idg
