// Adder (step a5) and splitter (step a6): PAPER.md Eq. 6 :102, :158, :169.
//
//   adder   : grid[layer, pol, y0+gy, x0+gx] += subgrids[s, pol, gy, gx]
//   splitter: subgrids[s, pol, gy, gx]         = grid[layer, pol, y0+gy, x0+gx]
//
// Subgrids overlap, so the adder is organised by the OUTPUT: one block owns one
// kTile x kTile tile (all four polarisation planes) of one w-layer and walks the plan's list of the
// subgrids that overlap the tile, in ascending subgrid order, accumulating in fp64 registers and
// touching the master grid exactly once.  Long lists are cut into segments of kAdderSegment subgrids, one
// block each, whose fp64 partial sums the tile's last block adds in segment order (plan.cpp).  No atomics; the summation order is fixed by the plan,
// so results are bitwise reproducible (R18).
#include "kernels.h"

namespace idg {

namespace {

constexpr int kAdderThreads = 512;
constexpr int kAdderStages = 6;      // subgrid patches in flight per block (staging ring in shared memory)

// One block owns one SEGMENT of the list of one kTile x kTile tile (all four polarisation planes of one
// w-layer).  Thread (tx, ty) owns column tx and rows ty, ty + T/kTile, ...; the (x0, y0) of the
// segment's subgrids are staged through shared memory so the loads of one item do not wait on a
// dependent metadata load.  Single-segment tiles go straight to the grid; otherwise the block leaves
// its fp64 partial sum in scratch and the LAST block of the tile to finish (a counter per tile) adds
// the partial sums in segment order and touches the grid once.
template <int T>
__global__ void __launch_bounds__(T) adder_kernel(const int32_t* __restrict__ meta, const int32_t* __restrict__ tile_ids,
                                                  const int32_t* __restrict__ segs,
                                                  const int32_t* __restrict__ items, int64_t first, int L, int Ng,
                                                  int tiles_x, int tiles_y, const float2* __restrict__ subgrids,
                                                  float2* __restrict__ grid, double* __restrict__ partials,
                                                  int32_t* __restrict__ counters) {
  constexpr int ROWS = kTile * kTile / T;        // tile rows per thread
  constexpr int RSTEP = T / kTile;
  constexpr int PART = 4 * ROWS * 2;             // doubles per thread in a partial sum
  __shared__ int s_x0[kAdderSegment], s_y0[kAdderSegment], s_sub[kAdderSegment];
  __shared__ int s_last;
  const int32_t* sg = segs + static_cast<int64_t>(blockIdx.x) * kSegStride;
  const int tidx = sg[0], beg = sg[1], end = sg[2], k = sg[3], nseg = sg[4], slot = sg[5];
  const int tile = tile_ids[tidx];
  const int tx = tile % tiles_x;
  const int ty = (tile / tiles_x) % tiles_y;
  const int layer = tile / (tiles_x * tiles_y);
  const int gx = tx * kTile + threadIdx.x % kTile;          // master-grid column of this thread
  const int gy0 = ty * kTile + threadIdx.x / kTile;         // first master-grid row
  double acc_re[4][ROWS], acc_im[4][ROWS];
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int j = 0; j < ROWS; ++j) acc_re[p][j] = acc_im[p][j] = 0.0;

  const int64_t plane_px = static_cast<int64_t>(L) * L;
  const int n = end - beg;
  for (int i = threadIdx.x; i < n; i += T) {
    const int s = items[beg + i];
    s_sub[i] = s;
    s_x0[i] = meta[static_cast<int64_t>(s) * kMetaStride + 5];
    s_y0[i] = meta[static_cast<int64_t>(s) * kMetaStride + 6];
  }
  __syncthreads();
  // The patches of the next kAdderStages - 1 subgrids are in flight while one is accumulated: every
  // thread copies its own 4 x ROWS samples with 8-byte cp.async into its private slots of a staging
  // ring (no registers held by loads in flight, no block-level synchronisation).
  extern __shared__ __align__(16) unsigned char adder_smem[];
  float2* stg = reinterpret_cast<float2*>(adder_smem);       // [kAdderStages][4 * ROWS][T]
  auto issue = [&](int i) {
    if (i < n) {
      const int sx = gx - s_x0[i];
      if (sx >= 0 && sx < L) {
        const int sy0 = gy0 - s_y0[i];
        const float2* base = subgrids + (s_sub[i] - first) * 4 * plane_px + sx;
        float2* dst = stg + (static_cast<size_t>(i % kAdderStages) * 4 * ROWS) * T + threadIdx.x;
#pragma unroll
        for (int j = 0; j < ROWS; ++j) {
          const int sy = sy0 + j * RSTEP;
          if (sy >= 0 && sy < L) {
#pragma unroll
            for (int p = 0; p < 4; ++p) {
              const uint32_t d = static_cast<uint32_t>(__cvta_generic_to_shared(dst + (p * ROWS + j) * T));
              asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(base + p * plane_px + sy * L)
                           : "memory");
            }
          }
        }
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  for (int i = 0; i < kAdderStages - 1; ++i) issue(i);
  for (int i = 0; i < n; ++i) {
    issue(i + kAdderStages - 1);
    asm volatile("cp.async.wait_group %0;" ::"n"(kAdderStages - 1) : "memory");
    const int sx = gx - s_x0[i];
    if (sx < 0 || sx >= L) continue;
    const int sy0 = gy0 - s_y0[i];
    const float2* src = stg + (static_cast<size_t>(i % kAdderStages) * 4 * ROWS) * T + threadIdx.x;
#pragma unroll
    for (int j = 0; j < ROWS; ++j) {
      const int sy = sy0 + j * RSTEP;
      if (sy >= 0 && sy < L) {
#pragma unroll
        for (int p = 0; p < 4; ++p) {
          const float2 v = src[(p * ROWS + j) * T];
          acc_re[p][j] += static_cast<double>(v.x);
          acc_im[p][j] += static_cast<double>(v.y);
        }
      }
    }
  }

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
    __syncthreads();
    if (threadIdx.x == 0) {
      const int done = atomicAdd(&counters[tidx], 1);
      s_last = done == nseg - 1;
      if (s_last) counters[tidx] = 0;                       // ready for the next launch
    }
    __syncthreads();
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

cudaError_t launch_adder(const int32_t* meta, const DeviceCsr& csr, int64_t first, int L, int Ng, int tiles_x,
                         int tiles_y, const float2* subgrids, float2* grid, cudaStream_t stream) {
  if (csr.n_segs == 0) return cudaSuccess;
  if (csr.n_slots > 0 && (!csr.partials || !csr.counters)) return cudaErrorInvalidValue;
  dim3 grid_dim(static_cast<unsigned>(csr.n_segs), 1, 1);
  constexpr size_t smem = static_cast<size_t>(kAdderStages) * 4 * (kTile * kTile / kAdderThreads) * kAdderThreads * sizeof(float2);
  // per launch: the attribute belongs to the (function, device) pair and the call is cheap
  cudaError_t e = cudaFuncSetAttribute(adder_kernel<kAdderThreads>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       static_cast<int>(smem));
  if (e != cudaSuccess) return e;
  adder_kernel<kAdderThreads><<<grid_dim, kAdderThreads, smem, stream>>>(meta, csr.tile_ids, csr.segs, csr.items, first, L,
                                                                      Ng, tiles_x, tiles_y, subgrids, grid,
                                                                      csr.partials, csr.counters);
  count_launch();
  return cudaGetLastError();
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
