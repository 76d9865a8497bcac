// Adder (step a5) and splitter (step a6): PAPER.md Eq. 6 :102, :158, :169.
//
//   adder   : grid[layer, pol, y0+gy, x0+gx] += subgrids[s, pol, gy, gx]
//   splitter: subgrids[s, pol, gy, gx]         = grid[layer, pol, y0+gy, x0+gx]
//
// Subgrids overlap, so the adder is organised by the OUTPUT: one block owns one
// kTile x kTile tile (all four polarisation planes) of one w-layer and walks the plan's list of the
// subgrids that overlap the tile, in ascending subgrid order, accumulating in fp64 registers and
// touching the master grid exactly once.  Tiles are launched heaviest first (plan.cpp).  No atomics; the summation order is fixed by the plan,
// so results are bitwise reproducible (R18).
#include "kernels.h"

namespace idg {

namespace {

constexpr int kAdderThreads = 512;
constexpr int kItemChunk = 256;     // subgrid origins staged through shared memory per chunk

// One block owns one kTile x kTile tile of all four polarisation planes of one w-layer.  Thread
// (tx, ty) owns column tx and rows ty, ty + T/kTile, ...; the (x0, y0) of the listed subgrids are
// staged through shared memory so the loads of one item do not wait on a dependent metadata load.
template <int T>
__global__ void __launch_bounds__(T) adder_kernel(const int32_t* __restrict__ meta, const int32_t* __restrict__ tile_ids,
                                                  const int32_t* __restrict__ offsets,
                                                  const int32_t* __restrict__ items, int64_t first, int L, int Ng,
                                                  int tiles_x, int tiles_y, const float2* __restrict__ subgrids,
                                                  float2* __restrict__ grid) {
  constexpr int ROWS = kTile * kTile / T;        // tile rows per thread
  constexpr int RSTEP = T / kTile;
  __shared__ int s_x0[kItemChunk], s_y0[kItemChunk], s_sub[kItemChunk];
  const int tile = tile_ids[blockIdx.x];
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
  const int beg = offsets[blockIdx.x], end = offsets[blockIdx.x + 1];
  for (int c0 = beg; c0 < end; c0 += kItemChunk) {
    const int n = min(kItemChunk, end - c0);
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += T) {
      const int s = items[c0 + i];
      s_sub[i] = s;
      s_x0[i] = meta[static_cast<int64_t>(s) * kMetaStride + 5];
      s_y0[i] = meta[static_cast<int64_t>(s) * kMetaStride + 6];
    }
    __syncthreads();
    for (int i = 0; i < n; ++i) {
      const int sx = gx - s_x0[i];
      if (sx < 0 || sx >= L) continue;
      const int sy0 = gy0 - s_y0[i];
      const float2* __restrict__ base = subgrids + (s_sub[i] - first) * 4 * plane_px + sx;
      float2 v[4][ROWS];
#pragma unroll
      for (int j = 0; j < ROWS; ++j) {
        const int sy = sy0 + j * RSTEP;
        const bool in = sy >= 0 && sy < L;
#pragma unroll
        for (int p = 0; p < 4; ++p)
          v[p][j] = in ? __ldcs(&base[p * plane_px + sy * L]) : make_float2(0.f, 0.f);
      }
#pragma unroll
      for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int j = 0; j < ROWS; ++j) {
          acc_re[p][j] += static_cast<double>(v[p][j].x);
          acc_im[p][j] += static_cast<double>(v[p][j].y);
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

}  // namespace

cudaError_t launch_adder(const int32_t* meta, const DeviceCsr& csr, int64_t first, int L, int Ng, int tiles_x,
                         int tiles_y, const float2* subgrids, float2* grid, cudaStream_t stream) {
  if (csr.n_tiles == 0) return cudaSuccess;
  dim3 grid_dim(static_cast<unsigned>(csr.n_tiles), 1, 1);
  adder_kernel<kAdderThreads><<<grid_dim, kAdderThreads, 0, stream>>>(meta, csr.tile_ids, csr.offsets, csr.items, first,
                                                                      L, Ng, tiles_x, tiles_y, subgrids, grid);
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
