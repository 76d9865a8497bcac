// Internal declarations shared by the host planner, the C-ABI layer and the kernel launchers.
// Nothing here is visible through include/idg_b200.h.
#pragma once
#include <cstdint>
#include <mutex>
#include <string>
#include <utility>
#include <vector>

#include "../../include/idg_b200.h"

namespace idg {

constexpr double kSpeedOfLight = 299792458.0;
constexpr int kMetaStride = 16;   // int32 per subgrid on the device: b,t0,nt,c0,nc,x0,y0,wl,p,q,it,layer,flags,-,-,-
constexpr int kMetaConj = 1;      // flags bit 0: rows are used conjugated, (u,v,w) -> -(u,v,w), V -> V^dagger (R21); p,q already swapped
// Adder tile: 1024 master-grid pixels, WIDE and flat (64 x 16 for L <= 64, 128 x 8 above).  A subgrid row (L samples,
// contiguous in the stack) then falls into one or two tiles instead of three, so fewer DRAM sectors straddle a tile
// boundary and are fetched twice, while a tile is not much wider than the subgrids it collects.
constexpr int kTilePixels = 1024;
inline int tile_width(int L) { return L <= 64 ? 64 : 128; }
inline int tile_height(int L) { return kTilePixels / tile_width(L); }
constexpr int kAdderSegment = 128;   // subgrids one adder block walks; longer tile lists are split
// Visibilities from which a subgrid takes the tensor-core degridder under AUTO.  Measured on config 3 (occupancy
// 1 ... 1536): sending the subgrids below 48 visibilities to the SIMT kernel cost 8 % of the launch (its lanes own 8
// visibilities each, so a handful of visibilities leaves the block idle), while the tensor-core kernel's idle warps
// cost nothing, so every subgrid takes the tensor-core kernel.
constexpr int kDegridTensorMin = 1;
constexpr int kSegStride = 6;     // int32 per adder segment: tile index, begin, end, k, n_seg, partial slot

// tile -> subgrid lists for the atomic-free adder (one CSR per batch of subgrids).
struct TileCsr {
  std::vector<int32_t> tile_ids;   // (layer*tiles_y + ty)*tiles_x + tx of every non-empty tile
  std::vector<int32_t> offsets;    // [n_tiles + 1] into items
  std::vector<int32_t> items;      // subgrid indices (global), ascending within a tile
  // Work units of the adder: segment k of n_seg of a tile's list, items [begin, end).  A tile with one
  // segment is added to the grid directly; otherwise every segment leaves an fp64 partial sum in
  // `slot` and the tile's last block to finish adds them up in the order k = 0, 1, ... (fixed order).
  std::vector<int32_t> segs;       // [n_segs, kSegStride], longest first
  int32_t n_slots = 0;
};

struct DeviceCsr {
  int32_t* tile_ids = nullptr;
  int32_t* offsets = nullptr;
  int32_t* items = nullptr;
  int32_t* segs = nullptr;
  int32_t n_tiles = 0, n_segs = 0, n_slots = 0;
  double* partials = nullptr;      // [n_slots, 4, tile, 2] scratch (not owned: DeviceState / caller)
  int32_t* counters = nullptr;     // [n_tiles] segments finished per tile, zero between launches
};

// Which subgrids of a range go to which direct-sum kernel (IDG_VARIANT_AUTO decides per subgrid,
// PAPER.md:247 fn 7).  Indices are relative to the range's first subgrid; an empty `tensor` AND empty
// `simt` list never occurs for a non-empty range.  When one list is empty the other launch needs no
// indirection.
struct KernelSplit {
  std::vector<int32_t> tensor, simt;
  int variant = 0;                 // the plan's IDG_VARIANT_* for this step (FP64 and forced variants: no lists)
};

struct Batch {
  int64_t first = 0, count = 0;
  TileCsr csr;
  KernelSplit grid_split, degrid_split;
};

struct DeviceSplit {
  int32_t* tensor = nullptr;       // device copies of KernelSplit's lists (nullptr when not mixed)
  int32_t* simt = nullptr;
  int32_t n_tensor = 0, n_simt = 0;
  int variant = 0;
};

struct DeviceState {
  double* uvw = nullptr;        // [n_rows, 3] metres
  double* kappa = nullptr;      // [n_chan] nu/c
  int32_t* meta = nullptr;      // [n_subgrids, kMetaStride]
  float* nprime = nullptr;      // [L, L] n'(l, m) at the subgrid pixels
  std::vector<DeviceCsr> batch_csr;
  std::vector<DeviceSplit> batch_grid_split, batch_degrid_split;
  double* adder_partials = nullptr;   // shared by the batches: sized for the largest
  int32_t* adder_counters = nullptr;
  void* closure_fft = nullptr;        // cuFFT plan of the master-grid transform, created on first use
  int device = -1;
};

}  // namespace idg

struct idg_plan {
  idg_params par{};
  int64_t n_rows = 0;
  int32_t n_intervals = 0;
  double image_size = 0.0;                // S = Ng * cell
  std::vector<double> uvw;                // host copy [n_rows*3]
  std::vector<double> kappa;              // nu_c / c
  double dkappa = 0.0;                    // channel spacing in kappa when uniform (to 1e-9 of the band), else 0
  std::vector<int32_t> baselines;         // [n_bl*2]
  std::vector<int32_t> sub;               // [n_subgrids*8]
  int64_t n_subgrids = 0, n_vis_planned = 0, n_vis_dropped = 0;
  int32_t wl_min = 0, n_wlayers = 1;
  int32_t tiles_x = 0, tiles_y = 0, tile_w = 0, tile_h = 0;   // adder tiles
  int64_t batch_capacity = 0;             // subgrids per batch
  std::vector<idg::Batch> batches;
  // rows of the visibility table grouped by the first / last batch that touches them (host-buffer calls)
  mutable std::vector<std::vector<std::pair<int64_t, int64_t>>> rows_first, rows_last;
  // per w-layer, the master-grid rows [first, last) under any subgrid: all the host-buffer calls move
  mutable std::vector<std::pair<int32_t, int32_t>> grid_rows;
  mutable std::mutex mu;
  mutable idg::DeviceState* dev = nullptr;   // uploaded on first device call
};

namespace idg {

void set_error(const std::string& msg);

// host planner (plan.cpp)
int  plan_build(idg_plan* plan);
void build_tile_csr(const idg_plan* plan, int64_t first, int64_t count, TileCsr* out);
void fill_meta(const idg_plan* plan, std::vector<int32_t>* meta);
bool subgrid_conjugated(const idg_plan* plan, const int32_t* sub8);
void split_kernels(const idg_plan* plan, int64_t first, int64_t count, int direction, KernelSplit* out);
// whether the tensor-core gridder's shared-memory tables hold a plan of this shape (gridder_tc.cu); if not, a
// launch handed to it runs the SIMT kernel, and split_kernels reports it so
bool gridder_tc_fits(int n_chan, int max_nt);

}  // namespace idg
