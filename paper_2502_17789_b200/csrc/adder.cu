// Adder (step a5) and splitter (step a6): PAPER.md Eq. 6 :102, :158, :169.
//
//   adder   : grid[layer, pol, y0+gy, x0+gx] += subgrids[s, pol, gy, gx]
//   splitter: subgrids[s, pol, gy, gx]         = grid[layer, pol, y0+gy, x0+gx]
//
// Subgrids overlap, so the adder is organised by the OUTPUT: one block owns one
// tile of 1024 master-grid pixels (64 x 16 or 128 x 8; all four polarisation planes) of one w-layer and walks the plan's list of the
// subgrids that overlap the tile, in ascending subgrid order, accumulating in fp64 registers and
// touching the master grid exactly once.  Long lists are cut into segments of kAdderSegment subgrids, one
// block each, whose fp64 partial sums the tile's last block adds in segment order (plan.cpp).  No atomics; the summation order is fixed by the plan,
// so results are bitwise reproducible (R18).
#include <cuda.h>

#include "kernels.h"
#include "tc_common.cuh"

namespace idg {

namespace {

constexpr int kAdderThreads = 512;   // consumer threads; one more warp issues the copies
constexpr int kAdderStages = 6;      // subgrid patches in flight per block (staging ring in shared memory)
// samples per box row: the box starts on an even sample (16-byte aligned, see below), so it is two samples wider
// than the tile; every stage of the ring must start 128-byte aligned
__host__ __device__ constexpr int box_bytes(int W, int H) { return 4 * H * (W + 2) * static_cast<int>(sizeof(float2)); }   // ~33 KB
static_assert(box_bytes(64, 16) % 128 == 0 && box_bytes(128, 8) % 128 == 0, "stage alignment");

// The subgrid stack as a 3-D tensor of 64-bit elements (complex samples) [planes][L][L] (north_star: staging through
// shared memory via TMA): the patch of one subgrid under one tile is a BOX {W + 2, H, 4} at signed coordinates,
// and whatever part of the box lies outside the subgrid arrives as zeros (the tensor map's out-of-bounds fill), so one
// cp.async.bulk.tensor per (tile, subgrid) replaces 8 predicated 8-byte cp.async per thread, and the consumers add
// the whole box without a single bounds test.  The hardware wants the box to start 16-byte aligned in global memory
// (an odd sample offset is an illegal instruction), hence the box starts at the even sample at or below the tile's
// first column and is two samples wider than the tile.
__device__ __forceinline__ void tma_load_box(uint32_t dst, const CUtensorMap* map, int x, int y, int z, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(dst),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}

// One block owns one SEGMENT of the list of one W x H tile (all four polarisation planes of one
// w-layer).  Consumer thread (tx, ty) owns column tx and rows ty, ty + T / W, ...  A producer warp walks the
// segment's subgrids and keeps kAdderStages boxes in flight (full / empty mbarriers per stage; the consumers release
// a stage with one arrival per warp).  Single-segment tiles go straight to the grid; otherwise the block leaves
// its fp64 partial sum in scratch and the LAST block of the tile to finish (a counter per tile) adds
// the partial sums in segment order and touches the grid once.
template <int T, int W, int H>
__global__ void __launch_bounds__(T + 32) adder_kernel(const __grid_constant__ CUtensorMap stack_map,
                                                       const int32_t* __restrict__ meta,
                                                       const int32_t* __restrict__ tile_ids,
                                                       const int32_t* __restrict__ segs,
                                                       const int32_t* __restrict__ items, int64_t first, int Ng,
                                                       int tiles_x, int tiles_y, float2* __restrict__ grid,
                                                       double* __restrict__ partials, int32_t* __restrict__ counters) {
  constexpr int kTileW = W, kTileH = H, kBoxW = W + 2, kBoxBytes = box_bytes(W, H);
  constexpr int RSTEP = T / kTileW;              // consumer rows per pass
  constexpr int ROWS = kTileH / RSTEP;           // tile rows per thread
  constexpr int PART = 4 * ROWS * 2;             // doubles per thread in a partial sum
  static_assert(T % kTileW == 0 && kTileH % RSTEP == 0 && W * H == kTilePixels, "tile shape");
  extern __shared__ __align__(1024) unsigned char adder_smem[];   // [kAdderStages][4][kTileH][kBoxW] float2
  __shared__ int s_x0[kAdderSegment], s_y0[kAdderSegment], s_sub[kAdderSegment];
  __shared__ __align__(8) uint64_t bars[2 * kAdderStages];        // full[stage], empty[stage]
  __shared__ int s_last;
  const int32_t* sg = segs + static_cast<int64_t>(blockIdx.x) * kSegStride;
  const int tidx = sg[0], beg = sg[1], end = sg[2], k = sg[3], nseg = sg[4], slot = sg[5];
  const int tile = tile_ids[tidx];
  const int tx = tile % tiles_x;
  const int ty = (tile / tiles_x) % tiles_y;
  const int layer = tile / (tiles_x * tiles_y);
  const int n = end - beg;
  const uint32_t bar0 = tc::smem_u32(&bars[0]);
  const uint32_t stg0 = tc::smem_u32(adder_smem);
  if (threadIdx.x == 0) {
    for (int i = 0; i < kAdderStages; ++i) {
      tc::mbar_init(bar0 + 8 * i, 1);                               // full: the producer's expect_tx arrival
      tc::mbar_init(bar0 + 8 * (kAdderStages + i), T / 32);         // empty: one arrival per consumer warp
    }
    tc::fence_barrier_init();
  }
  for (int i = threadIdx.x; i < n; i += T + 32) {
    const int s = items[beg + i];
    s_sub[i] = s;
    s_x0[i] = meta[static_cast<int64_t>(s) * kMetaStride + 5];
    s_y0[i] = meta[static_cast<int64_t>(s) * kMetaStride + 6];
  }
  __syncthreads();

  if (threadIdx.x >= T) {
    // ===== producer warp: one elected lane issues the box copies =====
    if (threadIdx.x == T) {
      for (int i = 0; i < n; ++i) {
        const int st = i % kAdderStages;
        if (i >= kAdderStages) tc::mbar_wait(bar0 + 8 * (kAdderStages + st), ((i / kAdderStages) - 1) & 1);
        mbar_expect_tx(bar0 + 8 * st, kBoxBytes);
        tma_load_box(stg0 + st * kBoxBytes, &stack_map, (tx * kTileW - s_x0[i]) & ~1, ty * kTileH - s_y0[i],
                     static_cast<int>((s_sub[i] - first) * 4), bar0 + 8 * st);
      }
    }
    return;
  }

  const int cx = threadIdx.x % kTileW, cy = threadIdx.x / kTileW;
  const int gx = tx * kTileW + cx;                           // master-grid column of this thread
  const int gy0 = ty * kTileH + cy;                          // first master-grid row
  double acc_re[4][ROWS], acc_im[4][ROWS];
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int j = 0; j < ROWS; ++j) acc_re[p][j] = acc_im[p][j] = 0.0;

  const float2* stg = reinterpret_cast<const float2*>(adder_smem);
  for (int i = 0; i < n; ++i) {
    const int st = i % kAdderStages;
    tc::mbar_wait(bar0 + 8 * st, (i / kAdderStages) & 1);
    // samples outside the subgrid arrived as zeros and are added like any other (testing for them was slower: 40.8
    // against 35.9 ms on config 3)
    const float2* src = stg + static_cast<size_t>(st) * (kBoxBytes / sizeof(float2)) + cy * kBoxW + cx +
                        ((tx * kTileW - s_x0[i]) & 1);               // the box starts on an even sample
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
      for (int j = 0; j < ROWS; ++j) {
        const float2 v = src[(p * kTileH + j * RSTEP) * kBoxW];
        acc_re[p][j] += static_cast<double>(v.x);
        acc_im[p][j] += static_cast<double>(v.y);
      }
    __syncwarp();
    if ((threadIdx.x & 31) == 0) tc::mbar_arrive(bar0 + 8 * (kAdderStages + st));
  }

  // (the producer warp has left: block-wide barriers below are named barriers over the T consumer threads)
  auto consumer_sync = [] { asm volatile("bar.sync 1, %0;" ::"n"(T) : "memory"); };
  if (nseg > 1) {
    // partial sums: [slot][component][thread], coalesced; then find out whether this block is the last
    double* mine = partials + static_cast<int64_t>(slot) * PART * T + threadIdx.x;
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
      for (int j = 0; j < ROWS; ++j) {
        mine[((p * ROWS + j) * 2 + 0) * T] = acc_re[p][j];
        mine[((p * ROWS + j) * 2 + 1) * T] = acc_im[p][j];
      }
    __threadfence();
    consumer_sync();
    if (threadIdx.x == 0) {
      const int done = atomicAdd(&counters[tidx], 1);
      s_last = done == nseg - 1;
      if (s_last) counters[tidx] = 0;                       // ready for the next launch
    }
    consumer_sync();
    if (!s_last) return;
    __threadfence();
    const double* all = partials + static_cast<int64_t>(slot - k) * PART * T + threadIdx.x;
#pragma unroll
    for (int p = 0; p < 4; ++p)
#pragma unroll
      for (int j = 0; j < ROWS; ++j) acc_re[p][j] = acc_im[p][j] = 0.0;
    for (int kk = 0; kk < nseg; ++kk) {                      // fixed order: deterministic
      const double* src = all + static_cast<int64_t>(kk) * PART * T;
#pragma unroll
      for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int j = 0; j < ROWS; ++j) {
          acc_re[p][j] += __ldcg(&src[((p * ROWS + j) * 2 + 0) * T]);
          acc_im[p][j] += __ldcg(&src[((p * ROWS + j) * 2 + 1) * T]);
        }
    }
  }
  if (gx < Ng) {
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      float2* __restrict__ g = grid + (static_cast<int64_t>(layer) * 4 + p) * Ng * static_cast<int64_t>(Ng);
#pragma unroll
      for (int j = 0; j < ROWS; ++j) {
        const int gy = gy0 + j * RSTEP;
        if (gy < Ng) {
          float2 v = g[static_cast<int64_t>(gy) * Ng + gx];
          v.x = static_cast<float>(static_cast<double>(v.x) + acc_re[p][j]);
          v.y = static_cast<float>(static_cast<double>(v.y) + acc_im[p][j]);
          g[static_cast<int64_t>(gy) * Ng + gx] = v;
        }
      }
    }
  }
}

__global__ void __launch_bounds__(256) splitter_kernel(const int32_t* __restrict__ meta, int64_t first, int L, int Ng,
                                                       const float2* __restrict__ grid,
                                                       float2* __restrict__ subgrids) {
  const int64_t sl = blockIdx.x;
  const int pol = blockIdx.y;
  const int32_t* m = meta + (first + sl) * kMetaStride;
  const int x0 = m[5], y0 = m[6], layer = m[11];
  const float2* __restrict__ g = grid + (static_cast<int64_t>(layer) * 4 + pol) * Ng * static_cast<int64_t>(Ng);
  float2* __restrict__ plane = subgrids + (sl * 4 + pol) * static_cast<int64_t>(L) * L;
  for (int i = threadIdx.x; i < L * L; i += blockDim.x) {
    const int y = i / L, x = i % L;
    plane[i] = __ldg(&g[static_cast<int64_t>(y0 + y) * Ng + x0 + x]);
  }
}

// dst += src (the host-buffer imaging call adds the caller's grid after the subgrids, off the critical path)
__global__ void __launch_bounds__(256) grid_add_kernel(const float2* __restrict__ src, float2* __restrict__ dst,
                                                       int64_t n) {
  for (int64_t i = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; i < n;
       i += static_cast<int64_t>(gridDim.x) * blockDim.x) {
    const float2 a = src[i], b = dst[i];
    dst[i] = make_float2(a.x + b.x, a.y + b.y);
  }
}

}  // namespace

cudaError_t launch_grid_add(const float2* src, float2* dst, int64_t n, cudaStream_t stream) {
  if (n == 0) return cudaSuccess;
  grid_add_kernel<<<148 * 8, 256, 0, stream>>>(src, dst, n);
  count_launch();
  return cudaGetLastError();
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

cudaError_t stack_tensor_map(const float2* subgrids, int L, int64_t n_subgrids, int W, int H, CUtensorMap* map) {
  static EncodeTiledFn encode = nullptr;
  if (!encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
    if (e != cudaSuccess) return e;
    if (q != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
    encode = reinterpret_cast<EncodeTiledFn>(fn);
  }
  const cuuint64_t dims[3] = {static_cast<cuuint64_t>(L), static_cast<cuuint64_t>(L), static_cast<cuuint64_t>(n_subgrids * 4)};
  const cuuint64_t strides[2] = {static_cast<cuuint64_t>(L) * sizeof(float2), static_cast<cuuint64_t>(L) * L * sizeof(float2)};
  const cuuint32_t box[3] = {static_cast<cuuint32_t>(W + 2), static_cast<cuuint32_t>(H), 4};
  const cuuint32_t ones[3] = {1, 1, 1};
  const CUresult r = encode(map, CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, const_cast<float2*>(subgrids), dims, strides, box, ones,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);          // out-of-bounds elements read as zero
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int W, int H>
cudaError_t launch_adder_wh(const CUtensorMap& map, const int32_t* meta, const DeviceCsr& csr, int64_t first, int L, int Ng,
                            int tiles_x, int tiles_y, float2* grid, cudaStream_t stream) {
  constexpr size_t smem = static_cast<size_t>(kAdderStages) * box_bytes(W, H);
  auto kernel = adder_kernel<kAdderThreads, W, H>;
  // per launch: the attribute belongs to the (function, device) pair and the call is cheap
  cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
  if (e != cudaSuccess) return e;
  kernel<<<static_cast<unsigned>(csr.n_segs), kAdderThreads + 32, smem, stream>>>(map, meta, csr.tile_ids, csr.segs, csr.items,
                                                                                first, Ng, tiles_x, tiles_y, grid,
                                                                                csr.partials, csr.counters);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_adder(const int32_t* meta, const DeviceCsr& csr, int64_t first, int64_t count, int L, int Ng, int tiles_x,
                         int tiles_y, const float2* subgrids, float2* grid, cudaStream_t stream) {
  if (csr.n_segs == 0) return cudaSuccess;
  if (csr.n_slots > 0 && (!csr.partials || !csr.counters)) return cudaErrorInvalidValue;
  // the tensor map wants a 16-byte aligned base (include/idg_b200.h asks that of every device pointer)
  if (reinterpret_cast<uintptr_t>(subgrids) & 15) return cudaErrorMisalignedAddress;
  const int W = tile_width(L), H = tile_height(L);
  CUtensorMap map;
  cudaError_t e = stack_tensor_map(subgrids, L, count, W, H, &map);
  if (e != cudaSuccess) return e;
  if (W == 64) return launch_adder_wh<64, 16>(map, meta, csr, first, L, Ng, tiles_x, tiles_y, grid, stream);
  return launch_adder_wh<128, 8>(map, meta, csr, first, L, Ng, tiles_x, tiles_y, grid, stream);
}

cudaError_t launch_splitter(const int32_t* meta, int64_t first, int64_t count, int L, int Ng, const float2* grid,
                            float2* subgrids, cudaStream_t stream) {
  if (count == 0) return cudaSuccess;
  dim3 grid_dim(static_cast<unsigned>(count), 4, 1);
  splitter_kernel<<<grid_dim, 256, 0, stream>>>(meta, first, L, Ng, grid, subgrids);
  count_launch();
  return cudaGetLastError();
}

}  // namespace idg
