// Adder (step a5) and splitter (step a6): PAPER.md Eq. 6 :102, :158, :169.
//
//   adder   : grid[layer, pol, y0+gy, x0+gx] += subgrids[s, pol, gy, gx]
//   splitter: subgrids[s, pol, gy, gx]         = grid[layer, pol, y0+gy, x0+gx]
//
// Subgrids overlap, so the adder is organised by the OUTPUT: one block owns one
// kTile x kTile tile of one polarisation plane of one w-layer and walks the plan's list of the
// subgrids that overlap the tile, in ascending subgrid order, accumulating in fp64 registers and
// touching the master grid exactly once.  No atomics; the summation order is fixed by the plan,
// so results are bitwise reproducible (R18).
#include "kernels.h"

namespace idg {

namespace {

constexpr int kAdderThreads = 256;

template <int T>
__global__ void __launch_bounds__(T) adder_kernel(const int32_t* __restrict__ meta, const int32_t* __restrict__ tile_ids,
                                                  const int32_t* __restrict__ offsets,
                                                  const int32_t* __restrict__ items, int64_t first, int L, int Ng,
                                                  int tiles_x, int tiles_y, const float2* __restrict__ subgrids,
                                                  float2* __restrict__ grid) {
  constexpr int ROWS = kTile * kTile / T;        // tile rows per thread
  constexpr int RSTEP = T / kTile;
  const int tile = tile_ids[blockIdx.x];
  const int pol = blockIdx.y;
  const int tx = tile % tiles_x;
  const int ty = (tile / tiles_x) % tiles_y;
  const int layer = tile / (tiles_x * tiles_y);
  const int gx = tx * kTile + threadIdx.x % kTile;          // master-grid column of this thread
  const int gy0 = ty * kTile + threadIdx.x / kTile;         // first master-grid row
  double acc_re[ROWS], acc_im[ROWS];
#pragma unroll
  for (int j = 0; j < ROWS; ++j) acc_re[j] = acc_im[j] = 0.0;

  const int beg = offsets[blockIdx.x], end = offsets[blockIdx.x + 1];
  for (int i = beg; i < end; ++i) {
    const int s = items[i];
    const int x0 = meta[static_cast<int64_t>(s) * kMetaStride + 5];
    const int y0 = meta[static_cast<int64_t>(s) * kMetaStride + 6];
    const int sx = gx - x0;
    if (sx < 0 || sx >= L) continue;
    const float2* __restrict__ plane = subgrids + ((s - first) * 4 + pol) * static_cast<int64_t>(L) * L;
#pragma unroll
    for (int j = 0; j < ROWS; ++j) {
      const int sy = gy0 + j * RSTEP - y0;
      if (sy >= 0 && sy < L) {
        const float2 v = __ldg(&plane[sy * L + sx]);
        acc_re[j] += static_cast<double>(v.x);
        acc_im[j] += static_cast<double>(v.y);
      }
    }
  }
  if (gx < Ng) {
    float2* __restrict__ g = grid + (static_cast<int64_t>(layer) * 4 + pol) * Ng * static_cast<int64_t>(Ng);
#pragma unroll
    for (int j = 0; j < ROWS; ++j) {
      const int gy = gy0 + j * RSTEP;
      if (gy < Ng) {
        float2 v = g[static_cast<int64_t>(gy) * Ng + gx];
        v.x = static_cast<float>(static_cast<double>(v.x) + acc_re[j]);
        v.y = static_cast<float>(static_cast<double>(v.y) + acc_im[j]);
        g[static_cast<int64_t>(gy) * Ng + gx] = v;
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
  dim3 grid_dim(static_cast<unsigned>(csr.n_tiles), 4, 1);
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
