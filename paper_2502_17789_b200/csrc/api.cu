// C-ABI layer: argument validation, plan lifetime, lazy upload of the plan metadata, and the
// orchestration of the kernels per batch.  See include/idg_b200.h for the contract.
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <mutex>
#include <vector>

#include "kernels.h"

namespace idg {

static thread_local std::string g_last_error;
static std::atomic<int64_t> g_launches{0};
static std::atomic<int> g_variant[IDG_K_COUNT] = {IDG_VARIANT_AUTO, 0, 0, 0, 0, IDG_VARIANT_AUTO};

void set_error(const std::string& msg) { g_last_error = msg; }
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

namespace {

// ---- optional per-kernel timing with CUDA events on the caller's stream -----------------------
struct ProfRecord { int kind; cudaEvent_t a, b; };
std::mutex g_prof_mu;
bool g_prof_on = false;
std::vector<ProfRecord> g_prof_pending;

struct ProfScope {
  cudaStream_t stream;
  int kind;
  cudaEvent_t a = nullptr, b = nullptr;
  bool on = false;
  ProfScope(int kind_, cudaStream_t s) : stream(s), kind(kind_) {
    std::lock_guard<std::mutex> lock(g_prof_mu);
    on = g_prof_on;
    if (on) {
      if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { on = false; return; }
      cudaEventRecord(a, stream);
    }
  }
  ~ProfScope() {
    if (!on) return;
    cudaEventRecord(b, stream);
    std::lock_guard<std::mutex> lock(g_prof_mu);
    g_prof_pending.push_back({kind, a, b});
  }
};

int cuda_fail(cudaError_t e, const char* what) {
  set_error(std::string(what) + ": " + cudaGetErrorString(e));
  return IDG_ECUDA;
}

#define IDG_CUDA(call)                                      \
  do {                                                      \
    cudaError_t e_ = (call);                                \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call);     \
  } while (0)

template <typename T>
cudaError_t upload(const std::vector<T>& host, T** dev) {
  *dev = nullptr;
  if (host.empty()) return cudaSuccess;
  cudaError_t e = cudaMalloc(reinterpret_cast<void**>(dev), host.size() * sizeof(T));
  if (e != cudaSuccess) return e;
  return cudaMemcpy(*dev, host.data(), host.size() * sizeof(T), cudaMemcpyHostToDevice);
}

cudaError_t upload_csr(const TileCsr& csr, DeviceCsr* out) {
  out->n_tiles = static_cast<int32_t>(csr.tile_ids.size());
  cudaError_t e;
  if ((e = upload(csr.tile_ids, &out->tile_ids)) != cudaSuccess) return e;
  if ((e = upload(csr.offsets, &out->offsets)) != cudaSuccess) return e;
  if ((e = upload(csr.items, &out->items)) != cudaSuccess) return e;
  out->n_segs = static_cast<int32_t>(csr.segs.size() / kSegStride);
  out->n_slots = csr.n_slots;
  return upload(csr.segs, &out->segs);
}

// fp64 partial sums [n_slots][4 pol][kTile][kTile][re, im] and one zeroed counter per tile
constexpr size_t kPartialBytes = static_cast<size_t>(4) * kTile * kTile * 2 * sizeof(double);
cudaError_t alloc_adder_scratch(int32_t n_slots, int32_t n_tiles, double** partials, int32_t** counters) {
  *partials = nullptr; *counters = nullptr;
  if (n_slots == 0) return cudaSuccess;
  cudaError_t e = cudaMalloc(reinterpret_cast<void**>(partials), kPartialBytes * n_slots);
  if (e != cudaSuccess) return e;
  e = cudaMalloc(reinterpret_cast<void**>(counters), sizeof(int32_t) * n_tiles);
  if (e != cudaSuccess) return e;
  return cudaMemset(*counters, 0, sizeof(int32_t) * n_tiles);
}

void free_csr(DeviceCsr* c) {
  cudaFree(c->tile_ids); cudaFree(c->offsets); cudaFree(c->items); cudaFree(c->segs);
  *c = DeviceCsr{};
}

void free_device_state(DeviceState* d) {
  if (!d) return;
  cudaFree(d->uvw); cudaFree(d->kappa); cudaFree(d->meta); cudaFree(d->nprime);
  for (auto& c : d->batch_csr) free_csr(&c);
  cudaFree(d->adder_partials); cudaFree(d->adder_counters);
  delete d;
}

// Uploads the plan metadata on first use (the only device memory the library owns).
int ensure_device(const idg_plan* plan, const DeviceState** out) {
  std::lock_guard<std::mutex> lock(plan->mu);
  if (plan->dev) { *out = plan->dev; return IDG_OK; }
  int dev = 0;
  IDG_CUDA(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  IDG_CUDA(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10) {
    set_error("idg_b200 needs an sm_100 (Blackwell B200) device; found compute capability " +
              std::to_string(prop.major) + "." + std::to_string(prop.minor));
    return IDG_ECUDA;
  }
  DeviceState* d = new (std::nothrow) DeviceState();
  if (!d) { set_error("host allocation failed"); return IDG_ENOMEM; }
  d->device = dev;
  std::vector<int32_t> meta;
  fill_meta(plan, &meta);
  // n'(l, m) at the subgrid pixels, rounded once from fp64 (R13: cancellation-free form)
  const int L = plan->par.subgrid_size;
  std::vector<float> np(static_cast<size_t>(L) * L);
  for (int y = 0; y < L; ++y)
    for (int x = 0; x < L; ++x) {
      const double l = (x - L / 2) * plan->image_size / L, mm = (y - L / 2) * plan->image_size / L;
      const double r2 = l * l + mm * mm;
      np[static_cast<size_t>(y) * L + x] = static_cast<float>(-r2 / (1.0 + std::sqrt(1.0 - r2)));
    }
  cudaError_t e;
  if ((e = upload(plan->uvw, &d->uvw)) != cudaSuccess || (e = upload(plan->kappa, &d->kappa)) != cudaSuccess ||
      (e = upload(meta, &d->meta)) != cudaSuccess || (e = upload(np, &d->nprime)) != cudaSuccess) {
    free_device_state(d);
    return cuda_fail(e, "plan upload");
  }
  d->batch_csr.resize(plan->batches.size());
  for (size_t i = 0; i < plan->batches.size(); ++i) {
    if ((e = upload_csr(plan->batches[i].csr, &d->batch_csr[i])) != cudaSuccess) {
      free_device_state(d);
      return cuda_fail(e, "plan upload (tile lists)");
    }
  }
  // the adder's scratch is shared by the batches (they run one after another on one stream)
  int32_t max_slots = 0, max_tiles = 0;
  for (const auto& c : d->batch_csr) { max_slots = std::max(max_slots, c.n_slots); max_tiles = std::max(max_tiles, c.n_tiles); }
  if ((e = alloc_adder_scratch(max_slots, max_tiles, &d->adder_partials, &d->adder_counters)) != cudaSuccess) {
    free_device_state(d);
    return cuda_fail(e, "plan upload (adder scratch)");
  }
  for (auto& c : d->batch_csr) { c.partials = d->adder_partials; c.counters = d->adder_counters; }
  plan->dev = d;
  *out = d;
  return IDG_OK;
}

SubgridJob make_job(const idg_plan* plan, const DeviceState* d, int64_t first, int64_t count, const void* aterms,
                    const float* taper) {
  SubgridJob j{};
  j.meta = d->meta; j.uvw = d->uvw; j.kappa = d->kappa; j.nprime = d->nprime;
  j.aterms = static_cast<const float4*>(aterms);
  j.taper = taper;
  j.first = first; j.count = count;
  j.subgrid_size = plan->par.subgrid_size; j.grid_size = plan->par.grid_size;
  j.n_times = plan->par.n_times; j.n_chan = plan->par.n_chan; j.n_intervals = plan->n_intervals;
  j.max_nt = plan->par.n_times < plan->par.aterm_period ? plan->par.n_times : plan->par.aterm_period;
  j.image_size = plan->image_size; j.w_step = plan->par.w_step;
  return j;
}

// Fraction of the tensor-core gridder's 8-channel chunks that carry visibilities, over a subgrid range:
// rows of few channels leave most of a chunk empty, and the SIMT kernel, which has no padding, wins.
double tensor_fill(const idg_plan* plan, int64_t first, int64_t count) {
  double used = 0.0, padded = 0.0;
  for (int64_t s = first; s < first + count; ++s) {
    const int32_t* m = &plan->sub[s * 8];
    used += static_cast<double>(m[2]) * m[4];
    padded += static_cast<double>(m[2]) * ((m[4] + 7) / 8 * 8);
  }
  return padded > 0.0 ? used / padded : 0.0;
}

// The same for the tensor-core degridder, whose MMA rows are tiles of 128 visibilities.
double tensor_fill_degrid(const idg_plan* plan, int64_t first, int64_t count) {
  double used = 0.0, padded = 0.0;
  for (int64_t s = first; s < first + count; ++s) {
    const int32_t* m = &plan->sub[s * 8];
    const int64_t k = static_cast<int64_t>(m[2]) * m[4];
    used += static_cast<double>(k);
    padded += static_cast<double>((k + 127) / 128 * 128);
  }
  return padded > 0.0 ? used / padded : 0.0;
}

constexpr double kTensorFillMin = 0.8;

cudaError_t run_degridder(const idg_plan* plan, const SubgridJob& job, const float2* in, float4* vis,
                          cudaStream_t stream) {
  int v = g_variant[IDG_K_DEGRIDDER].load();
  if (v == IDG_VARIANT_AUTO)
    v = tensor_fill_degrid(plan, job.first, job.count) >= kTensorFillMin ? IDG_VARIANT_TENSOR : IDG_VARIANT_SIMT;
  return v == IDG_VARIANT_TENSOR ? launch_degridder_tc(job, in, vis, stream) : launch_degridder(job, in, vis, stream);
}

cudaError_t run_gridder(const idg_plan* plan, const SubgridJob& job, const float4* vis, float2* out,
                        cudaStream_t stream) {
  int v = g_variant[IDG_K_GRIDDER].load();
  if (v == IDG_VARIANT_AUTO)
    v = tensor_fill(plan, job.first, job.count) >= kTensorFillMin ? IDG_VARIANT_TENSOR : IDG_VARIANT_SIMT;
  return v == IDG_VARIANT_TENSOR ? launch_gridder_tc(job, vis, out, stream) : launch_gridder(job, vis, out, stream);
}

bool range_ok(const idg_plan* plan, int64_t first, int64_t count) {
  return first >= 0 && count >= 0 && first + count <= plan->n_subgrids;
}

size_t stack_bytes(const idg_plan* plan, int64_t count) {
  const size_t L = plan->par.subgrid_size;
  return static_cast<size_t>(count) * 4 * L * L * sizeof(float2);
}

}  // namespace
}  // namespace idg

using namespace idg;

extern "C" {

int idg_plan_create(const idg_params* params, const double* uvw_m_host, const double* freqs_host,
                    const int32_t* baselines_host, idg_plan** out) {
  if (!params || !uvw_m_host || !freqs_host || !baselines_host || !out) {
    set_error("idg_plan_create: null argument");
    return IDG_EINVAL;
  }
  *out = nullptr;
  const idg_params& p = *params;
  if (p.subgrid_size != 32 && p.subgrid_size != 64 && p.subgrid_size != 96 && p.subgrid_size != 128) {
    set_error("idg_plan_create: subgrid_size must be 32, 64, 96 or 128");
    return IDG_EUNSUPPORTED;
  }
  if (p.grid_size < p.subgrid_size || (p.grid_size & 1) || p.padding < 0 || p.padding >= p.subgrid_size - 1 ||
      p.n_stations < 1 || p.n_baselines < 0 || p.n_times < 1 || p.n_chan < 1 || p.aterm_period < 1 ||
      !(p.cell_size > 0.0) || !(p.w_step >= 0.0) || !(p.comfort > 0.0 && p.comfort <= 1.0) ||
      p.max_batch_subgrids < 0) {
    set_error("idg_plan_create: invalid parameter");
    return IDG_EINVAL;
  }
  if (!(p.grid_size * p.cell_size < 1.4)) {   // l^2 + m^2 < 1 at the subgrid corners
    set_error("idg_plan_create: field of view too large (grid_size * cell_size must be < 1.4 rad)");
    return IDG_EINVAL;
  }
  for (int32_t c = 0; c < p.n_chan; ++c) {
    if (!(freqs_host[c] > 0.0) || (c > 0 && !(freqs_host[c] > freqs_host[c - 1]))) {
      set_error("idg_plan_create: channel frequencies must be positive and strictly ascending (PAPER.md:196)");
      return IDG_EINVAL;
    }
  }
  for (int64_t b = 0; b < p.n_baselines; ++b) {
    for (int k = 0; k < 2; ++k) {
      const int32_t st = baselines_host[b * 2 + k];
      if (st < 0 || st >= p.n_stations) {
        set_error("idg_plan_create: station index out of range in baselines");
        return IDG_EINVAL;
      }
    }
  }
  idg_plan* plan = new (std::nothrow) idg_plan();
  if (!plan) { set_error("host allocation failed"); return IDG_ENOMEM; }
  try {
    plan->par = p;
    plan->n_rows = static_cast<int64_t>(p.n_baselines) * p.n_times;
    plan->n_intervals = (p.n_times + p.aterm_period - 1) / p.aterm_period;
    plan->image_size = p.grid_size * p.cell_size;
    plan->uvw.assign(uvw_m_host, uvw_m_host + plan->n_rows * 3);
    plan->kappa.resize(p.n_chan);
    for (int32_t c = 0; c < p.n_chan; ++c) plan->kappa[c] = freqs_host[c] / kSpeedOfLight;
    plan->baselines.assign(baselines_host, baselines_host + static_cast<int64_t>(p.n_baselines) * 2);
    const int rc = plan_build(plan);
    if (rc != IDG_OK) { delete plan; return rc; }
  } catch (const std::bad_alloc&) {
    delete plan;
    set_error("host allocation failed");
    return IDG_ENOMEM;
  }
  *out = plan;
  return IDG_OK;
}

void idg_plan_destroy(idg_plan* plan) {
  if (!plan) return;
  free_device_state(plan->dev);
  delete plan;
}

int idg_plan_counts(const idg_plan* plan, int64_t* n_subgrids, int32_t* n_wlayers, int32_t* wl_min,
                    int64_t* n_vis_planned, int64_t* n_vis_dropped) {
  if (!plan) { set_error("idg_plan_counts: null plan"); return IDG_EINVAL; }
  if (n_subgrids) *n_subgrids = plan->n_subgrids;
  if (n_wlayers) *n_wlayers = plan->n_wlayers;
  if (wl_min) *wl_min = plan->wl_min;
  if (n_vis_planned) *n_vis_planned = plan->n_vis_planned;
  if (n_vis_dropped) *n_vis_dropped = plan->n_vis_dropped;
  return IDG_OK;
}

int idg_plan_export(const idg_plan* plan, int32_t* sub_host) {
  if (!plan || (!sub_host && plan->n_subgrids > 0)) { set_error("idg_plan_export: null argument"); return IDG_EINVAL; }
  if (plan->n_subgrids > 0) std::memcpy(sub_host, plan->sub.data(), plan->sub.size() * sizeof(int32_t));
  return IDG_OK;
}

size_t idg_workspace_bytes(const idg_plan* plan, int direction) {
  (void)direction;
  if (!plan) return 0;
  return stack_bytes(plan, plan->batch_capacity);
}

int idg_grid(const idg_plan* plan, const void* vis_dev, const void* aterms_dev, const float* taper_dev,
             void* grid_dev, void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
  if (!plan || !vis_dev || !aterms_dev || !taper_dev || !grid_dev) { set_error("idg_grid: null argument"); return IDG_EINVAL; }
  if (plan->n_subgrids == 0) return IDG_OK;
  if (!workspace_dev || workspace_bytes < idg_workspace_bytes(plan, IDG_GRID)) {
    set_error("idg_grid: workspace too small (see idg_workspace_bytes)");
    return IDG_ENOMEM;
  }
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  float2* stack = static_cast<float2*>(workspace_dev);
  const int L = plan->par.subgrid_size, Ng = plan->par.grid_size;
  for (size_t i = 0; i < plan->batches.size(); ++i) {
    const Batch& bt = plan->batches[i];
    const SubgridJob job = make_job(plan, d, bt.first, bt.count, aterms_dev, taper_dev);
    { ProfScope ps(IDG_K_GRIDDER, stream);
      IDG_CUDA(run_gridder(plan, job, static_cast<const float4*>(vis_dev), stack, stream)); }
    { ProfScope ps(IDG_K_FFT, stream);
      IDG_CUDA(launch_subgrid_fft(L, bt.count * 4, stack, +1, stream)); }
    { ProfScope ps(IDG_K_ADDER, stream);
      IDG_CUDA(launch_adder(d->meta, d->batch_csr[i], bt.first, L, Ng, plan->tiles_x, plan->tiles_y, stack,
                            static_cast<float2*>(grid_dev), stream)); }
  }
  return IDG_OK;
}

int idg_degrid(const idg_plan* plan, const void* grid_dev, const void* aterms_dev, const float* taper_dev,
               void* vis_dev, void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
  if (!plan || !vis_dev || !aterms_dev || !taper_dev || !grid_dev) { set_error("idg_degrid: null argument"); return IDG_EINVAL; }
  if (plan->n_subgrids == 0) return IDG_OK;
  if (!workspace_dev || workspace_bytes < idg_workspace_bytes(plan, IDG_DEGRID)) {
    set_error("idg_degrid: workspace too small (see idg_workspace_bytes)");
    return IDG_ENOMEM;
  }
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  float2* stack = static_cast<float2*>(workspace_dev);
  const int L = plan->par.subgrid_size, Ng = plan->par.grid_size;
  for (size_t i = 0; i < plan->batches.size(); ++i) {
    const Batch& bt = plan->batches[i];
    const SubgridJob job = make_job(plan, d, bt.first, bt.count, aterms_dev, taper_dev);
    { ProfScope ps(IDG_K_SPLITTER, stream);
      IDG_CUDA(launch_splitter(d->meta, bt.first, bt.count, L, Ng, static_cast<const float2*>(grid_dev), stack, stream)); }
    { ProfScope ps(IDG_K_IFFT, stream);
      IDG_CUDA(launch_subgrid_fft(L, bt.count * 4, stack, -1, stream)); }
    { ProfScope ps(IDG_K_DEGRIDDER, stream);
      IDG_CUDA(run_degridder(plan, job, stack, static_cast<float4*>(vis_dev), stream)); }
  }
  return IDG_OK;
}

// ---- host-buffer variants -------------------------------------------------------------------
namespace {
struct ArenaLayout { size_t vis, aterms, taper, grid, work, total; };
size_t align_up(size_t x) { return (x + 255) & ~size_t{255}; }
ArenaLayout arena_layout(const idg_plan* plan) {
  const idg_params& p = plan->par;
  const size_t L = p.subgrid_size, Ng = p.grid_size;
  ArenaLayout a{};
  size_t off = 0;
  a.vis = off;    off += align_up(static_cast<size_t>(plan->n_rows) * p.n_chan * 4 * sizeof(float2));
  a.aterms = off; off += align_up(static_cast<size_t>(p.n_stations) * plan->n_intervals * L * L * 4 * sizeof(float2));
  a.taper = off;  off += align_up(L * L * sizeof(float));
  a.grid = off;   off += align_up(static_cast<size_t>(plan->n_wlayers) * 4 * Ng * Ng * sizeof(float2));
  a.work = off;   off += align_up(stack_bytes(plan, plan->batch_capacity));
  a.total = off;
  return a;
}
}  // namespace

size_t idg_host_arena_bytes(const idg_plan* plan, int direction) {
  (void)direction;
  if (!plan) return 0;
  return arena_layout(plan).total;
}

int idg_grid_host(const idg_plan* plan, const void* vis_host, const void* aterms_host, const float* taper_host,
                  void* grid_host, void* arena_dev, size_t arena_bytes, void* cuda_stream) {
  if (!plan || !vis_host || !aterms_host || !taper_host || !grid_host || !arena_dev) {
    set_error("idg_grid_host: null argument");
    return IDG_EINVAL;
  }
  const ArenaLayout a = arena_layout(plan);
  if (arena_bytes < a.total) { set_error("idg_grid_host: arena too small (see idg_host_arena_bytes)"); return IDG_ENOMEM; }
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  char* base = static_cast<char*>(arena_dev);
  const idg_params& p = plan->par;
  const size_t L = p.subgrid_size, Ng = p.grid_size;
  const size_t vis_b = static_cast<size_t>(plan->n_rows) * p.n_chan * 4 * sizeof(float2);
  const size_t at_b = static_cast<size_t>(p.n_stations) * plan->n_intervals * L * L * 4 * sizeof(float2);
  const size_t grid_b = static_cast<size_t>(plan->n_wlayers) * 4 * Ng * Ng * sizeof(float2);
  IDG_CUDA(cudaMemcpyAsync(base + a.vis, vis_host, vis_b, cudaMemcpyHostToDevice, stream));
  IDG_CUDA(cudaMemcpyAsync(base + a.aterms, aterms_host, at_b, cudaMemcpyHostToDevice, stream));
  IDG_CUDA(cudaMemcpyAsync(base + a.taper, taper_host, L * L * sizeof(float), cudaMemcpyHostToDevice, stream));
  IDG_CUDA(cudaMemcpyAsync(base + a.grid, grid_host, grid_b, cudaMemcpyHostToDevice, stream));
  int rc = idg_grid(plan, base + a.vis, base + a.aterms, reinterpret_cast<const float*>(base + a.taper), base + a.grid,
                    base + a.work, a.total - a.work, cuda_stream);
  if (rc != IDG_OK) return rc;
  IDG_CUDA(cudaMemcpyAsync(grid_host, base + a.grid, grid_b, cudaMemcpyDeviceToHost, stream));
  IDG_CUDA(cudaStreamSynchronize(stream));
  return IDG_OK;
}

int idg_degrid_host(const idg_plan* plan, const void* grid_host, const void* aterms_host, const float* taper_host,
                    void* vis_host, void* arena_dev, size_t arena_bytes, void* cuda_stream) {
  if (!plan || !vis_host || !aterms_host || !taper_host || !grid_host || !arena_dev) {
    set_error("idg_degrid_host: null argument");
    return IDG_EINVAL;
  }
  const ArenaLayout a = arena_layout(plan);
  if (arena_bytes < a.total) { set_error("idg_degrid_host: arena too small (see idg_host_arena_bytes)"); return IDG_ENOMEM; }
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  char* base = static_cast<char*>(arena_dev);
  const idg_params& p = plan->par;
  const size_t L = p.subgrid_size, Ng = p.grid_size;
  const size_t vis_b = static_cast<size_t>(plan->n_rows) * p.n_chan * 4 * sizeof(float2);
  const size_t at_b = static_cast<size_t>(p.n_stations) * plan->n_intervals * L * L * 4 * sizeof(float2);
  const size_t grid_b = static_cast<size_t>(plan->n_wlayers) * 4 * Ng * Ng * sizeof(float2);
  // visibilities not covered by a subgrid must come back untouched: upload them first
  IDG_CUDA(cudaMemcpyAsync(base + a.vis, vis_host, vis_b, cudaMemcpyHostToDevice, stream));
  IDG_CUDA(cudaMemcpyAsync(base + a.aterms, aterms_host, at_b, cudaMemcpyHostToDevice, stream));
  IDG_CUDA(cudaMemcpyAsync(base + a.taper, taper_host, L * L * sizeof(float), cudaMemcpyHostToDevice, stream));
  IDG_CUDA(cudaMemcpyAsync(base + a.grid, grid_host, grid_b, cudaMemcpyHostToDevice, stream));
  int rc = idg_degrid(plan, base + a.grid, base + a.aterms, reinterpret_cast<const float*>(base + a.taper),
                      base + a.vis, base + a.work, a.total - a.work, cuda_stream);
  if (rc != IDG_OK) return rc;
  IDG_CUDA(cudaMemcpyAsync(vis_host, base + a.vis, vis_b, cudaMemcpyDeviceToHost, stream));
  IDG_CUDA(cudaStreamSynchronize(stream));
  return IDG_OK;
}

// ---- stage-level entry points ----------------------------------------------------------------
int idg_grid_subgrids(const idg_plan* plan, int64_t first, int64_t count, const void* vis_dev,
                      const void* aterms_dev, const float* taper_dev, void* subgrids_dev, int stage,
                      void* cuda_stream) {
  if (!plan || !vis_dev || !aterms_dev || !taper_dev || !subgrids_dev) { set_error("idg_grid_subgrids: null argument"); return IDG_EINVAL; }
  if (!range_ok(plan, first, count) || (stage != IDG_STAGE_GRIDDER && stage != IDG_STAGE_FFT)) {
    set_error("idg_grid_subgrids: bad range or stage");
    return IDG_EINVAL;
  }
  if (count == 0) return IDG_OK;
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  const SubgridJob job = make_job(plan, d, first, count, aterms_dev, taper_dev);
  IDG_CUDA(run_gridder(plan, job, static_cast<const float4*>(vis_dev), static_cast<float2*>(subgrids_dev), stream));
  if (stage == IDG_STAGE_FFT)
    IDG_CUDA(launch_subgrid_fft(plan->par.subgrid_size, count * 4, static_cast<float2*>(subgrids_dev), +1, stream));
  return IDG_OK;
}

int idg_degrid_subgrids(const idg_plan* plan, int64_t first, int64_t count, const void* subgrids_dev,
                        const void* aterms_dev, const float* taper_dev, void* vis_dev, void* cuda_stream) {
  if (!plan || !vis_dev || !aterms_dev || !taper_dev || !subgrids_dev) { set_error("idg_degrid_subgrids: null argument"); return IDG_EINVAL; }
  if (!range_ok(plan, first, count)) { set_error("idg_degrid_subgrids: bad range"); return IDG_EINVAL; }
  if (count == 0) return IDG_OK;
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  const SubgridJob job = make_job(plan, d, first, count, aterms_dev, taper_dev);
  IDG_CUDA(run_degridder(plan, job, static_cast<const float2*>(subgrids_dev), static_cast<float4*>(vis_dev),
                            static_cast<cudaStream_t>(cuda_stream)));
  return IDG_OK;
}

int idg_subgrid_fft(int32_t subgrid_size, int64_t n_planes, void* planes_dev, int direction, void* cuda_stream) {
  if (subgrid_size != 32 && subgrid_size != 64 && subgrid_size != 96 && subgrid_size != 128) {
    set_error("idg_subgrid_fft: subgrid_size must be 32, 64, 96 or 128");
    return IDG_EUNSUPPORTED;
  }
  if (n_planes < 0 || (n_planes > 0 && !planes_dev) || (direction != 1 && direction != -1)) {
    set_error("idg_subgrid_fft: bad argument");
    return IDG_EINVAL;
  }
  IDG_CUDA(launch_subgrid_fft(subgrid_size, n_planes, static_cast<float2*>(planes_dev), direction,
                              static_cast<cudaStream_t>(cuda_stream)));
  return IDG_OK;
}

int idg_adder(const idg_plan* plan, int64_t first, int64_t count, const void* subgrids_dev, void* grid_dev,
              void* cuda_stream) {
  if (!plan || !subgrids_dev || !grid_dev) { set_error("idg_adder: null argument"); return IDG_EINVAL; }
  if (!range_ok(plan, first, count)) { set_error("idg_adder: bad range"); return IDG_EINVAL; }
  if (count == 0) return IDG_OK;
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  // an arbitrary range needs its own tile lists: build, upload, run, free (test hook, synchronous)
  TileCsr csr;
  build_tile_csr(plan, first, count, &csr);
  DeviceCsr dc;
  cudaError_t e = upload_csr(csr, &dc);
  if (e == cudaSuccess) e = alloc_adder_scratch(dc.n_slots, dc.n_tiles, &dc.partials, &dc.counters);
  if (e != cudaSuccess) { cudaFree(dc.partials); cudaFree(dc.counters); free_csr(&dc); return cuda_fail(e, "idg_adder: tile list upload"); }
  e = launch_adder(d->meta, dc, first, plan->par.subgrid_size, plan->par.grid_size, plan->tiles_x, plan->tiles_y,
                   static_cast<const float2*>(subgrids_dev), static_cast<float2*>(grid_dev), stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
  cudaFree(dc.partials); cudaFree(dc.counters);
  free_csr(&dc);
  if (e != cudaSuccess) return cuda_fail(e, "idg_adder");
  return IDG_OK;
}

int idg_splitter(const idg_plan* plan, int64_t first, int64_t count, const void* grid_dev, void* subgrids_dev,
                 void* cuda_stream) {
  if (!plan || !subgrids_dev || !grid_dev) { set_error("idg_splitter: null argument"); return IDG_EINVAL; }
  if (!range_ok(plan, first, count)) { set_error("idg_splitter: bad range"); return IDG_EINVAL; }
  if (count == 0) return IDG_OK;
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  IDG_CUDA(launch_splitter(d->meta, first, count, plan->par.subgrid_size, plan->par.grid_size,
                           static_cast<const float2*>(grid_dev), static_cast<float2*>(subgrids_dev),
                           static_cast<cudaStream_t>(cuda_stream)));
  return IDG_OK;
}

int idg_profile_enable(int on) {
  std::lock_guard<std::mutex> lock(g_prof_mu);
  g_prof_on = on != 0;
  return IDG_OK;
}

int idg_profile_read(double* ms_out, int64_t* launches_out) {
  if (!ms_out || !launches_out) { set_error("idg_profile_read: null argument"); return IDG_EINVAL; }
  std::vector<ProfRecord> recs;
  {
    std::lock_guard<std::mutex> lock(g_prof_mu);
    recs.swap(g_prof_pending);
  }
  cudaError_t first_err = cudaSuccess;
  for (const ProfRecord& r : recs) {
    float ms = 0.f;
    cudaError_t e = cudaEventSynchronize(r.b);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, r.a, r.b);
    if (e == cudaSuccess) { ms_out[r.kind] += ms; launches_out[r.kind] += 1; }
    else if (first_err == cudaSuccess) first_err = e;
    cudaEventDestroy(r.a);
    cudaEventDestroy(r.b);
  }
  if (first_err != cudaSuccess) return cuda_fail(first_err, "idg_profile_read");
  return IDG_OK;
}

int idg_set_kernel_variant(int kind, int variant) {
  if ((kind != IDG_K_GRIDDER && kind != IDG_K_DEGRIDDER) ||
      (variant != IDG_VARIANT_SIMT && variant != IDG_VARIANT_TENSOR && variant != IDG_VARIANT_AUTO)) {
    set_error("idg_set_kernel_variant: bad kind or variant");
    return IDG_EINVAL;
  }
  g_variant[kind].store(variant);
  return IDG_OK;
}

int idg_get_kernel_variant(int kind) {
  if (kind < 0 || kind >= IDG_K_COUNT) return IDG_EINVAL;
  return g_variant[kind].load();
}

int idg_measure_alu_peaks(double* out_host) {
  if (!out_host) { set_error("idg_measure_alu_peaks: null argument"); return IDG_EINVAL; }
  IDG_CUDA(measure_alu_peaks(out_host));
  return IDG_OK;
}

int64_t idg_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

const char* idg_last_error(void) { return g_last_error.c_str(); }

const char* idg_version(void) { return "idg_b200 0.1 (sm_100a)"; }

}  // extern "C"
