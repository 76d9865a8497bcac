// C-ABI layer: argument validation, plan lifetime, lazy upload of the plan metadata, and the
// orchestration of the kernels per batch.  See include/idg_b200.h for the contract.
#include <atomic>
#include <functional>
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
static std::atomic<int> g_kmask[IDG_K_COUNT];        // which direct-sum kernels ran (idg_kernel_config_mask)

void set_error(const std::string& msg) { g_last_error = msg; }
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
void note_kernel(int kind, int bit) { g_kmask[kind].fetch_or(bit, std::memory_order_relaxed); }

namespace {

// ---- optional per-kernel timing with CUDA events on the caller's stream -----------------------
struct ProfRecord { int kind; cudaEvent_t a, b; };
std::mutex g_prof_mu;
bool g_prof_on = false;
std::vector<ProfRecord> g_prof_pending;
std::vector<cudaEvent_t> g_prof_pool;                // events of records already read, reused by later scopes

bool prof_event(cudaEvent_t* e) {                    // g_prof_mu held
  if (!g_prof_pool.empty()) { *e = g_prof_pool.back(); g_prof_pool.pop_back(); return true; }
  return cudaEventCreate(e) == cudaSuccess;
}

struct ProfScope {
  cudaStream_t stream;
  int kind;
  cudaEvent_t a = nullptr, b = nullptr;
  bool on = false;
  ProfScope(int kind_, cudaStream_t s) : stream(s), kind(kind_) {
    std::lock_guard<std::mutex> lock(g_prof_mu);
    on = g_prof_on;
    if (on) {
      if (!prof_event(&a) || !prof_event(&b)) { on = false; return; }
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

// fp64 partial sums [n_slots][4 pol][tile pixels][re, im] and one zeroed counter per tile
constexpr size_t kPartialBytes = static_cast<size_t>(4) * kTilePixels * 2 * sizeof(double);
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

cudaError_t upload_split(const KernelSplit& sp, DeviceSplit* out) {
  *out = DeviceSplit{};
  out->variant = sp.variant;
  out->n_tensor = static_cast<int32_t>(sp.tensor.size());
  out->n_simt = static_cast<int32_t>(sp.simt.size());
  if (sp.tensor.empty() || sp.simt.empty()) return cudaSuccess;      // one launch over the whole range: no lists
  cudaError_t e = upload(sp.tensor, &out->tensor);
  if (e != cudaSuccess) return e;
  return upload(sp.simt, &out->simt);
}

void free_split(DeviceSplit* s) {
  cudaFree(s->tensor); cudaFree(s->simt);
  *s = DeviceSplit{};
}

void free_device_state(DeviceState* d) {
  if (!d) return;
  cudaFree(d->uvw); cudaFree(d->kappa); cudaFree(d->meta); cudaFree(d->nprime);
  for (auto& c : d->batch_csr) free_csr(&c);
  for (auto& c : d->batch_grid_split) free_split(&c);
  for (auto& c : d->batch_degrid_split) free_split(&c);
  cudaFree(d->adder_partials); cudaFree(d->adder_counters);
  closure_plan_destroy(d->closure_fft);
  delete d;
}

// Uploads the plan metadata on first use (the only device memory the library owns).
int ensure_device(const idg_plan* plan, const DeviceState** out) {
  std::lock_guard<std::mutex> lock(plan->mu);
  int dev = 0;
  IDG_CUDA(cudaGetDevice(&dev));
  if (plan->dev) {
    if (plan->dev->device != dev) {
      set_error("the plan's metadata lives on device " + std::to_string(plan->dev->device) + " but the current device is " +
                std::to_string(dev) + " (one plan per device)");
      return IDG_EINVAL;
    }
    *out = plan->dev;
    return IDG_OK;
  }
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
  d->batch_grid_split.resize(plan->batches.size());
  d->batch_degrid_split.resize(plan->batches.size());
  for (size_t i = 0; i < plan->batches.size(); ++i) {
    if ((e = upload_csr(plan->batches[i].csr, &d->batch_csr[i])) != cudaSuccess ||
        (e = upload_split(plan->batches[i].grid_split, &d->batch_grid_split[i])) != cudaSuccess ||
        (e = upload_split(plan->batches[i].degrid_split, &d->batch_degrid_split[i])) != cudaSuccess) {
      free_device_state(d);
      return cuda_fail(e, "plan upload (tile and kernel lists)");
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
  j.weights = nullptr;
  j.index = nullptr;
  j.power_norm = plan->par.power_norm;
  j.dkappa = plan->dkappa;
  j.dkappa_f = static_cast<float>(plan->dkappa);
  j.first = first; j.count = count;
  j.subgrid_size = plan->par.subgrid_size; j.grid_size = plan->par.grid_size;
  j.n_times = plan->par.n_times; j.n_chan = plan->par.n_chan; j.n_intervals = plan->n_intervals;
  j.max_nt = plan->par.n_times < plan->par.aterm_period ? plan->par.n_times : plan->par.aterm_period;
  j.image_size = plan->image_size; j.w_step = plan->par.w_step;
  return j;
}

// The direct-sum step of one range of subgrids with the plan's kernel variant.  Under IDG_VARIANT_AUTO the
// choice is per SUBGRID (PAPER.md:247 fn 7): `sp` says how many subgrids take which kernel and, when both
// kinds occur, holds the two complementary index lists on the device.
cudaError_t run_gridder(SubgridJob job, const DeviceSplit& sp, const float4* vis, float2* out, cudaStream_t stream) {
  switch (sp.variant) {
    case IDG_VARIANT_SIMT:   return launch_gridder(job, vis, out, stream);
    case IDG_VARIANT_TENSOR: return launch_gridder_tc(job, vis, out, stream);
    case IDG_VARIANT_FP64:   return launch_gridder_f64(job, vis, out, nullptr, stream);
    default: break;
  }
  if (sp.n_simt == 0) return launch_gridder_tc(job, vis, out, stream);
  if (sp.n_tensor == 0) return launch_gridder(job, vis, out, stream);
  job.index = sp.tensor; job.count = sp.n_tensor;
  cudaError_t e = launch_gridder_tc(job, vis, out, stream);
  if (e != cudaSuccess) return e;
  job.index = sp.simt; job.count = sp.n_simt;
  return launch_gridder(job, vis, out, stream);
}

cudaError_t run_degridder(SubgridJob job, const DeviceSplit& sp, const float2* in, float4* vis, cudaStream_t stream) {
  switch (sp.variant) {
    case IDG_VARIANT_SIMT:   return launch_degridder(job, in, vis, stream);
    case IDG_VARIANT_TENSOR: return launch_degridder_tc(job, in, vis, stream);
    case IDG_VARIANT_FP64:   return launch_degridder_f64(job, in, nullptr, vis, nullptr, stream);
    default: break;
  }
  if (sp.n_simt == 0) return launch_degridder_tc(job, in, vis, stream);
  if (sp.n_tensor == 0) return launch_degridder(job, in, vis, stream);
  job.index = sp.tensor; job.count = sp.n_tensor;
  cudaError_t e = launch_degridder_tc(job, in, vis, stream);
  if (e != cudaSuccess) return e;
  job.index = sp.simt; job.count = sp.n_simt;
  return launch_degridder(job, in, vis, stream);
}

// The same for an arbitrary range (stage-level test hooks): the lists are built and uploaded for the call and
// freed after a stream synchronisation.
struct RangeSplit {
  DeviceSplit d;
  bool owned = false;
  ~RangeSplit() { if (owned) free_split(&d); }
  cudaError_t init(const idg_plan* plan, int64_t first, int64_t count, int direction) {
    KernelSplit sp;
    split_kernels(plan, first, count, direction, &sp);
    owned = true;
    return upload_split(sp, &d);
  }
  bool mixed() const { return d.tensor != nullptr; }
};

bool subgrid_size_ok(int L) { return L == 32 || L == 48 || L == 64 || L == 96 || L == 128 || L == 160; }

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
  if (!subgrid_size_ok(p.subgrid_size)) {
    set_error("idg_plan_create: subgrid_size must be 32, 48, 64, 96, 128 or 160");
    return IDG_EUNSUPPORTED;
  }
  for (int v : {p.gridder_variant, p.degridder_variant}) {
    if (v != IDG_VARIANT_AUTO && v != IDG_VARIANT_SIMT && v != IDG_VARIANT_TENSOR && v != IDG_VARIANT_FP64) {
      set_error("idg_plan_create: kernel variant must be IDG_VARIANT_AUTO, _SIMT, _TENSOR or _FP64");
      return IDG_EINVAL;
    }
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

namespace {

// One batch of the imaging direction: gridder, subgrid FFT, adder.  `before_adder` runs on the host
// between the FFT and the adder launches (the host-buffer call waits for the grid upload there).
int grid_batch(const idg_plan* plan, const DeviceState* d, size_t i, const void* vis_dev, const void* aterms_dev,
               const float* taper_dev, void* grid_dev, float2* stack, cudaStream_t stream,
               const std::function<int()>& before_adder, const float* weights_dev = nullptr) {
  const int L = plan->par.subgrid_size, Ng = plan->par.grid_size;
  const Batch& bt = plan->batches[i];
  SubgridJob job = make_job(plan, d, bt.first, bt.count, aterms_dev, taper_dev);
  job.weights = weights_dev;
  { ProfScope ps(IDG_K_GRIDDER, stream);
    IDG_CUDA(run_gridder(job, d->batch_grid_split[i], static_cast<const float4*>(vis_dev), stack, stream)); }
  { ProfScope ps(IDG_K_FFT, stream);
    IDG_CUDA(launch_subgrid_fft(L, bt.count * 4, stack, +1, stream)); }
  int rc = before_adder();
  if (rc != IDG_OK) return rc;
  { ProfScope ps(IDG_K_ADDER, stream);
    IDG_CUDA(launch_adder(d->meta, d->batch_csr[i], bt.first, bt.count, L, Ng, plan->tiles_x, plan->tiles_y, stack,
                          static_cast<float2*>(grid_dev), stream)); }
  return IDG_OK;
}

// One batch of the prediction direction: splitter, inverse subgrid FFT, degridder.
int degrid_batch(const idg_plan* plan, const DeviceState* d, size_t i, const void* grid_dev, const void* aterms_dev,
                 const float* taper_dev, void* vis_dev, float2* stack, cudaStream_t stream) {
  const int L = plan->par.subgrid_size, Ng = plan->par.grid_size;
  const Batch& bt = plan->batches[i];
  const SubgridJob job = make_job(plan, d, bt.first, bt.count, aterms_dev, taper_dev);
  // splitter (a6) and inverse subgrid FFT (a7) in one kernel: the transform gathers its input from the grid
  { ProfScope ps(IDG_K_IFFT, stream);
    IDG_CUDA(launch_split_ifft(d->meta, bt.first, bt.count, L, Ng, static_cast<const float2*>(grid_dev), stack, stream)); }
  { ProfScope ps(IDG_K_DEGRIDDER, stream);
    IDG_CUDA(run_degridder(job, d->batch_degrid_split[i], stack, static_cast<float4*>(vis_dev), stream)); }
  return IDG_OK;
}

}  // namespace

int idg_grid_weighted(const idg_plan* plan, const void* vis_dev, const float* weights_dev, const void* aterms_dev,
                      const float* taper_dev, void* grid_dev, void* workspace_dev, size_t workspace_bytes,
                      void* cuda_stream) {
  if (plan && plan->n_subgrids == 0) return IDG_OK;      // nothing planned (the arrays may be empty, i.e. null)
  if (!plan || !vis_dev || !aterms_dev || !taper_dev || !grid_dev) { set_error("idg_grid: null argument"); return IDG_EINVAL; }
  if (!workspace_dev || workspace_bytes < idg_workspace_bytes(plan, IDG_GRID)) {
    set_error("idg_grid: workspace too small (see idg_workspace_bytes)");
    return IDG_ENOMEM;
  }
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  for (size_t i = 0; i < plan->batches.size(); ++i) {
    rc = grid_batch(plan, d, i, vis_dev, aterms_dev, taper_dev, grid_dev, static_cast<float2*>(workspace_dev), stream,
                    [] { return IDG_OK; }, weights_dev);
    if (rc != IDG_OK) return rc;
  }
  return IDG_OK;
}

int idg_grid(const idg_plan* plan, const void* vis_dev, const void* aterms_dev, const float* taper_dev,
             void* grid_dev, void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
  return idg_grid_weighted(plan, vis_dev, nullptr, aterms_dev, taper_dev, grid_dev, workspace_dev, workspace_bytes,
                           cuda_stream);
}

int idg_degrid(const idg_plan* plan, const void* grid_dev, const void* aterms_dev, const float* taper_dev,
               void* vis_dev, void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
  if (plan && plan->n_subgrids == 0) return IDG_OK;      // nothing planned (the arrays may be empty, i.e. null)
  if (!plan || !vis_dev || !aterms_dev || !taper_dev || !grid_dev) { set_error("idg_degrid: null argument"); return IDG_EINVAL; }
  if (!workspace_dev || workspace_bytes < idg_workspace_bytes(plan, IDG_DEGRID)) {
    set_error("idg_degrid: workspace too small (see idg_workspace_bytes)");
    return IDG_ENOMEM;
  }
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  for (size_t i = 0; i < plan->batches.size(); ++i) {
    rc = degrid_batch(plan, d, i, grid_dev, aterms_dev, taper_dev, vis_dev, static_cast<float2*>(workspace_dev), stream);
    if (rc != IDG_OK) return rc;
  }
  return IDG_OK;
}

// ---- host-buffer variants -------------------------------------------------------------------
namespace {
struct ArenaLayout { size_t vis, aterms, taper, grid, grid_in, work, total; };
size_t align_up(size_t x) { return (x + 255) & ~size_t{255}; }
ArenaLayout arena_layout(const idg_plan* plan, int direction = IDG_GRID) {
  const idg_params& p = plan->par;
  const size_t L = p.subgrid_size, Ng = p.grid_size;
  ArenaLayout a{};
  size_t off = 0;
  a.vis = off;    off += align_up(static_cast<size_t>(plan->n_rows) * p.n_chan * 4 * sizeof(float2));
  a.aterms = off; off += align_up(static_cast<size_t>(p.n_stations) * plan->n_intervals * L * L * 4 * sizeof(float2));
  a.taper = off;  off += align_up(L * L * sizeof(float));
  a.grid = off;   off += align_up(static_cast<size_t>(plan->n_wlayers) * 4 * Ng * Ng * sizeof(float2));
  // imaging only: the caller's grid waits here until the subgrids have been added (see idg_grid_host)
  a.grid_in = off; if (direction == IDG_GRID) off += align_up(static_cast<size_t>(plan->n_wlayers) * 4 * Ng * Ng * sizeof(float2));
  a.work = off;   off += align_up(stack_bytes(plan, plan->batch_capacity));
  a.total = off;
  return a;
}
}  // namespace

size_t idg_host_arena_bytes(const idg_plan* plan, int direction) {
  if (!plan) return 0;
  return arena_layout(plan, direction).total;
}

namespace {

// Rows of the visibility table grouped by the first and by the last batch that touches them, as runs of
// consecutive rows: the host-buffer calls upload a row just before the first batch that reads it and
// download it right after the last batch that writes it, while the other batches compute.
void ensure_row_runs(const idg_plan* plan) {
  std::lock_guard<std::mutex> lock(plan->mu);
  if (!plan->rows_first.empty() || !plan->grid_rows.empty()) return;
  plan->grid_rows.assign(plan->n_wlayers, {0, 0});         // a plan without subgrids touches no row
  if (plan->batches.empty()) return;
  const size_t nb = plan->batches.size();
  std::vector<int32_t> first(plan->n_rows, -1), last(plan->n_rows, -1);
  for (size_t i = 0; i < nb; ++i) {
    const Batch& bt = plan->batches[i];
    for (int64_t s = bt.first; s < bt.first + bt.count; ++s) {
      const int32_t* m = &plan->sub[static_cast<size_t>(s) * 8];
      const int64_t r0 = static_cast<int64_t>(m[0]) * plan->par.n_times + m[1];
      for (int64_t r = r0; r < r0 + m[2]; ++r) {
        if (first[r] < 0) first[r] = static_cast<int32_t>(i);
        last[r] = static_cast<int32_t>(i);
      }
    }
  }
  auto runs = [&](const std::vector<int32_t>& tag, std::vector<std::vector<std::pair<int64_t, int64_t>>>* out) {
    out->assign(nb, {});
    for (int64_t r = 0; r < plan->n_rows;) {
      int64_t e = r + 1;
      while (e < plan->n_rows && tag[e] == tag[r]) ++e;
      if (tag[r] >= 0) (*out)[tag[r]].emplace_back(r, e);
      r = e;
    }
  };
  runs(first, &plan->rows_first);
  runs(last, &plan->rows_last);
  // master-grid rows under the subgrids of each w-layer: nothing outside them is read or written
  plan->grid_rows.assign(plan->n_wlayers, {plan->par.grid_size, 0});
  for (int64_t s = 0; s < plan->n_subgrids; ++s) {
    const int32_t* m = &plan->sub[static_cast<size_t>(s) * 8];
    auto& gr = plan->grid_rows[m[7] - plan->wl_min];
    gr.first = std::min(gr.first, m[6]);
    gr.second = std::max(gr.second, m[6] + plan->par.subgrid_size);
  }
  for (auto& gr : plan->grid_rows)
    if (gr.second <= gr.first) gr = {0, 0};
}

// Calls fn(byte offset, byte count) for the touched rows of every (layer, polarisation) plane of the master grid.
// row_align > 1 widens each range outwards to multiples of row_align (clamped to the grid).
cudaError_t for_grid_rows(const idg_plan* plan, const std::function<cudaError_t(size_t, size_t)>& fn, int row_align = 1) {
  const size_t Ng = plan->par.grid_size;
  for (int32_t k = 0; k < plan->n_wlayers; ++k) {
    auto gr = plan->grid_rows[k];
    if (gr.second <= gr.first) continue;
    if (row_align > 1) {
      gr.first = gr.first / row_align * row_align;
      gr.second = std::min<int32_t>(plan->par.grid_size, (gr.second + row_align - 1) / row_align * row_align);
    }
    const size_t n = static_cast<size_t>(gr.second - gr.first) * Ng * sizeof(float2);
    if (n == 0) continue;
    for (int p = 0; p < 4; ++p) {
      cudaError_t e = fn(((static_cast<size_t>(k) * 4 + p) * Ng + gr.first) * Ng * sizeof(float2), n);
      if (e != cudaSuccess) return e;
    }
  }
  return cudaSuccess;
}

// Copies the touched rows of every (layer, polarisation) plane of the master grid between host and device
// (kind says which way); returns the bytes moved through `bytes` when it is not null.
cudaError_t copy_grid_rows(const idg_plan* plan, void* dst, const void* src, cudaMemcpyKind kind, cudaStream_t stream,
                           int64_t* bytes) {
  const size_t Ng = plan->par.grid_size;
  int64_t total = 0;
  for (int32_t k = 0; k < plan->n_wlayers; ++k) {
    const auto gr = plan->grid_rows[k];
    const size_t n = static_cast<size_t>(gr.second - gr.first) * Ng * sizeof(float2);
    if (n == 0) continue;
    for (int p = 0; p < 4; ++p) {
      const size_t off = ((static_cast<size_t>(k) * 4 + p) * Ng + gr.first) * Ng * sizeof(float2);
      if (dst) {
        cudaError_t e = cudaMemcpyAsync(static_cast<char*>(dst) + off, static_cast<const char*>(src) + off, n, kind, stream);
        if (e != cudaSuccess) return e;
      }
      total += static_cast<int64_t>(n);
    }
  }
  if (bytes) *bytes = total;
  return cudaSuccess;
}

// a second stream and the events that order it against the caller's stream; all destroyed on return
struct CopyLane {
  cudaStream_t s = nullptr;
  std::vector<cudaEvent_t> ev;
  ~CopyLane() {
    for (cudaEvent_t e : ev) cudaEventDestroy(e);
    if (s) cudaStreamDestroy(s);
  }
  cudaError_t init() { return cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking); }
  cudaError_t event(cudaEvent_t* e) {
    cudaError_t rc = cudaEventCreateWithFlags(e, cudaEventDisableTiming);
    if (rc == cudaSuccess) ev.push_back(*e);
    return rc;
  }
  // `to` waits for everything enqueued on `from` so far
  cudaError_t order(cudaStream_t from, cudaStream_t to) {
    cudaEvent_t e;
    cudaError_t rc = event(&e);
    if (rc != cudaSuccess) return rc;
    if ((rc = cudaEventRecord(e, from)) != cudaSuccess) return rc;
    return cudaStreamWaitEvent(to, e, 0);
  }
};

}  // namespace

int idg_host_traffic_bytes(const idg_plan* plan, int direction, int64_t* h2d_bytes, int64_t* d2h_bytes) {
  if (!plan || (direction != IDG_GRID && direction != IDG_DEGRID)) { set_error("idg_host_traffic_bytes: bad argument"); return IDG_EINVAL; }
  if (plan->n_subgrids == 0) {                            // nothing is planned: the host calls move nothing
    if (h2d_bytes) *h2d_bytes = 0;
    if (d2h_bytes) *d2h_bytes = 0;
    return IDG_OK;
  }
  ensure_row_runs(plan);
  const idg_params& p = plan->par;
  const int64_t L = p.subgrid_size;
  const int64_t row_b = static_cast<int64_t>(p.n_chan) * 4 * sizeof(float2);
  const int64_t at_b = static_cast<int64_t>(p.n_stations) * plan->n_intervals * L * L * 4 * sizeof(float2);
  const int64_t tp_b = L * L * sizeof(float);
  int64_t grid_rows_b = 0, vis_rows = 0;
  copy_grid_rows(plan, nullptr, nullptr, cudaMemcpyHostToDevice, nullptr, &grid_rows_b);
  for (const auto& runs : plan->rows_first)
    for (const auto& run : runs) vis_rows += run.second - run.first;
  const bool partial_rows = plan->n_vis_planned != static_cast<int64_t>(plan->n_rows) * p.n_chan;
  int64_t up, down;
  if (direction == IDG_GRID) {
    up = vis_rows * row_b + at_b + tp_b + grid_rows_b;
    down = grid_rows_b;
  } else {
    up = grid_rows_b + at_b + tp_b + (partial_rows ? static_cast<int64_t>(plan->n_rows) * row_b : 0);
    down = vis_rows * row_b;
  }
  if (h2d_bytes) *h2d_bytes = up;
  if (d2h_bytes) *d2h_bytes = down;
  return IDG_OK;
}

int idg_grid_host(const idg_plan* plan, const void* vis_host, const void* aterms_host, const float* taper_host,
                  void* grid_host, void* arena_dev, size_t arena_bytes, void* cuda_stream) {
  if (plan && plan->n_subgrids == 0) return IDG_OK;       // nothing to add: grid_host stays as it is
  if (!plan || !vis_host || !aterms_host || !taper_host || !grid_host || !arena_dev) {
    set_error("idg_grid_host: null argument");
    return IDG_EINVAL;
  }
  const ArenaLayout a = arena_layout(plan);
  if (arena_bytes < a.total) { set_error("idg_grid_host: arena too small (see idg_host_arena_bytes)"); return IDG_ENOMEM; }
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  char* base = static_cast<char*>(arena_dev);
  const idg_params& p = plan->par;
  const size_t L = p.subgrid_size;
  const size_t row_b = static_cast<size_t>(p.n_chan) * 4 * sizeof(float2);
  const size_t at_b = static_cast<size_t>(p.n_stations) * plan->n_intervals * L * L * 4 * sizeof(float2);
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  ensure_row_runs(plan);
  // Copy lane: A-terms and taper, then per batch the visibility rows it is the first to read.  The compute
  // stream waits per batch, so uploads overlap the gridding of earlier batches.
  CopyLane lane;
  IDG_CUDA(lane.init());
  IDG_CUDA(lane.order(stream, lane.s));                 // the arena may still be in use by earlier work
  IDG_CUDA(cudaMemcpyAsync(base + a.aterms, aterms_host, at_b, cudaMemcpyHostToDevice, lane.s));
  IDG_CUDA(cudaMemcpyAsync(base + a.taper, taper_host, L * L * sizeof(float), cudaMemcpyHostToDevice, lane.s));
  // The caller's grid (accumulated into) is NOT on the critical path: the subgrids are added into a zeroed
  // device grid while the caller's grid goes up to a second buffer behind the visibilities, and the two are
  // summed once at the end.
  // (only the rows under a subgrid are added and moved.  The adder reads and writes whole tiles of tile_h rows,
  // so the zeroed range is widened to tile rows: nothing else of the device grid is ever read.)
  IDG_CUDA(for_grid_rows(plan, [&](size_t off, size_t n) { return cudaMemsetAsync(base + a.grid + off, 0, n, stream); },
                         plan->tile_h));
  for (size_t i = 0; i < plan->batches.size(); ++i) {
    for (const auto& run : plan->rows_first[i])
      IDG_CUDA(cudaMemcpyAsync(base + a.vis + run.first * row_b, static_cast<const char*>(vis_host) + run.first * row_b,
                               (run.second - run.first) * row_b, cudaMemcpyHostToDevice, lane.s));
    IDG_CUDA(lane.order(lane.s, stream));
    rc = grid_batch(plan, d, i, base + a.vis, base + a.aterms, reinterpret_cast<const float*>(base + a.taper),
                    base + a.grid, reinterpret_cast<float2*>(base + a.work), stream, [] { return IDG_OK; });
    if (rc != IDG_OK) return rc;
  }
  // only the master-grid rows under the subgrids move: the rest of grid_host is already what it will be
  IDG_CUDA(copy_grid_rows(plan, base + a.grid_in, grid_host, cudaMemcpyHostToDevice, lane.s, nullptr));
  IDG_CUDA(lane.order(lane.s, stream));
  IDG_CUDA(for_grid_rows(plan, [&](size_t off, size_t n) {
    return launch_grid_add(reinterpret_cast<const float2*>(base + a.grid_in + off), reinterpret_cast<float2*>(base + a.grid + off),
                           static_cast<int64_t>(n / sizeof(float2)), stream);
  }));
  IDG_CUDA(copy_grid_rows(plan, grid_host, base + a.grid, cudaMemcpyDeviceToHost, stream, nullptr));
  IDG_CUDA(cudaStreamSynchronize(stream));
  IDG_CUDA(cudaStreamSynchronize(lane.s));
  return IDG_OK;
}

int idg_degrid_host(const idg_plan* plan, const void* grid_host, const void* aterms_host, const float* taper_host,
                    void* vis_host, void* arena_dev, size_t arena_bytes, void* cuda_stream) {
  if (plan && plan->n_subgrids == 0) return IDG_OK;       // no planned visibility: vis_host stays as it is
  if (!plan || !vis_host || !aterms_host || !taper_host || !grid_host || !arena_dev) {
    set_error("idg_degrid_host: null argument");
    return IDG_EINVAL;
  }
  const ArenaLayout a = arena_layout(plan, IDG_DEGRID);
  if (arena_bytes < a.total) { set_error("idg_degrid_host: arena too small (see idg_host_arena_bytes)"); return IDG_ENOMEM; }
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  char* base = static_cast<char*>(arena_dev);
  const idg_params& p = plan->par;
  const size_t L = p.subgrid_size;
  const size_t row_b = static_cast<size_t>(p.n_chan) * 4 * sizeof(float2);
  const size_t vis_b = static_cast<size_t>(plan->n_rows) * row_b;
  const size_t at_b = static_cast<size_t>(p.n_stations) * plan->n_intervals * L * L * 4 * sizeof(float2);
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  ensure_row_runs(plan);
  CopyLane lane;
  IDG_CUDA(lane.init());
  IDG_CUDA(lane.order(stream, lane.s));
  // Visibilities no subgrid covers must come back untouched.  Rows no subgrid touches are simply never
  // downloaded; rows only partly covered exist only if the planner dropped visibilities, and then the
  // host's values go up first (on the copy lane, beside the grid upload).
  const bool partial_rows = plan->n_vis_planned != static_cast<int64_t>(plan->n_rows) * p.n_chan;
  if (partial_rows) {
    IDG_CUDA(cudaMemcpyAsync(base + a.vis, vis_host, vis_b, cudaMemcpyHostToDevice, lane.s));
    IDG_CUDA(lane.order(lane.s, stream));
  }
  // the splitter reads the grid only under the subgrids: those rows go up, nothing else
  IDG_CUDA(copy_grid_rows(plan, base + a.grid, grid_host, cudaMemcpyHostToDevice, stream, nullptr));
  IDG_CUDA(cudaMemcpyAsync(base + a.aterms, aterms_host, at_b, cudaMemcpyHostToDevice, stream));
  IDG_CUDA(cudaMemcpyAsync(base + a.taper, taper_host, L * L * sizeof(float), cudaMemcpyHostToDevice, stream));
  // per batch: predict, then download the rows it was the last to write while the next batch computes
  for (size_t i = 0; i < plan->batches.size(); ++i) {
    rc = degrid_batch(plan, d, i, base + a.grid, base + a.aterms, reinterpret_cast<const float*>(base + a.taper),
                      base + a.vis, reinterpret_cast<float2*>(base + a.work), stream);
    if (rc != IDG_OK) return rc;
    IDG_CUDA(lane.order(stream, lane.s));
    for (const auto& run : plan->rows_last[i])
      IDG_CUDA(cudaMemcpyAsync(static_cast<char*>(vis_host) + run.first * row_b, base + a.vis + run.first * row_b,
                               (run.second - run.first) * row_b, cudaMemcpyDeviceToHost, lane.s));
  }
  IDG_CUDA(cudaStreamSynchronize(stream));
  IDG_CUDA(cudaStreamSynchronize(lane.s));
  return IDG_OK;
}

// ---- w-stacking closure (outside the hot path) -------------------------------------------------
namespace {
int ensure_closure_fft(const idg_plan* plan, const DeviceState* d, void** out) {
  std::lock_guard<std::mutex> lock(plan->mu);
  DeviceState* dm = const_cast<DeviceState*>(d);
  if (!dm->closure_fft && closure_plan_create(plan->par.grid_size, &dm->closure_fft) != 0) {
    set_error("cuFFT plan creation failed for the master-grid transform");
    return IDG_ECUDA;
  }
  *out = dm->closure_fft;
  return IDG_OK;
}
}  // namespace

size_t idg_closure_workspace_bytes(const idg_plan* plan) {
  if (!plan) return 0;
  const size_t Ng = plan->par.grid_size;
  return 4 * Ng * Ng * sizeof(float2);
}

int idg_grid_to_image(const idg_plan* plan, const void* grid_dev, const float* corr_dev, void* image_dev,
                      void* workspace_dev, size_t workspace_bytes, void* cuda_stream) {
  if (!plan || !grid_dev || !image_dev) { set_error("idg_grid_to_image: null argument"); return IDG_EINVAL; }
  if (!workspace_dev || workspace_bytes < idg_closure_workspace_bytes(plan)) {
    set_error("idg_grid_to_image: workspace too small (see idg_closure_workspace_bytes)");
    return IDG_ENOMEM;
  }
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  void* fft = nullptr;
  if ((rc = ensure_closure_fft(plan, d, &fft)) != IDG_OK) return rc;
  IDG_CUDA(launch_grid_to_image(fft, static_cast<const float2*>(grid_dev), corr_dev, static_cast<float2*>(image_dev),
                                static_cast<float2*>(workspace_dev), plan->par.grid_size, plan->n_wlayers, plan->wl_min,
                                plan->par.w_step, plan->image_size, static_cast<cudaStream_t>(cuda_stream)));
  return IDG_OK;
}

int idg_image_to_grid(const idg_plan* plan, const void* image_dev, const float* corr_dev, void* grid_dev,
                      void* cuda_stream) {
  if (!plan || !grid_dev || !image_dev) { set_error("idg_image_to_grid: null argument"); return IDG_EINVAL; }
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  void* fft = nullptr;
  if ((rc = ensure_closure_fft(plan, d, &fft)) != IDG_OK) return rc;
  IDG_CUDA(launch_image_to_grid(fft, static_cast<const float2*>(image_dev), corr_dev, static_cast<float2*>(grid_dev),
                                plan->par.grid_size, plan->n_wlayers, plan->wl_min, plan->par.w_step, plan->image_size,
                                static_cast<cudaStream_t>(cuda_stream)));
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
  RangeSplit rs;
  IDG_CUDA(rs.init(plan, first, count, IDG_GRID));
  IDG_CUDA(run_gridder(job, rs.d, static_cast<const float4*>(vis_dev), static_cast<float2*>(subgrids_dev), stream));
  if (stage == IDG_STAGE_FFT)
    IDG_CUDA(launch_subgrid_fft(plan->par.subgrid_size, count * 4, static_cast<float2*>(subgrids_dev), +1, stream));
  if (rs.mixed()) IDG_CUDA(cudaStreamSynchronize(stream));      // the lists are freed on return
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
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  RangeSplit rs;
  IDG_CUDA(rs.init(plan, first, count, IDG_DEGRID));
  IDG_CUDA(run_degridder(job, rs.d, static_cast<const float2*>(subgrids_dev), static_cast<float4*>(vis_dev), stream));
  if (rs.mixed()) IDG_CUDA(cudaStreamSynchronize(stream));      // the lists are freed on return
  return IDG_OK;
}

int idg_grid_subgrids_f64(const idg_plan* plan, int64_t first, int64_t count, const void* vis_dev,
                          const void* aterms_dev, const float* taper_dev, void* subgrids_dev, void* cuda_stream) {
  if (!plan || !vis_dev || !aterms_dev || !taper_dev || !subgrids_dev) { set_error("idg_grid_subgrids_f64: null argument"); return IDG_EINVAL; }
  if (!range_ok(plan, first, count)) { set_error("idg_grid_subgrids_f64: bad range"); return IDG_EINVAL; }
  if (count == 0) return IDG_OK;
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  const SubgridJob job = make_job(plan, d, first, count, aterms_dev, taper_dev);
  IDG_CUDA(launch_gridder_f64(job, static_cast<const float4*>(vis_dev), nullptr, static_cast<double2*>(subgrids_dev),
                              static_cast<cudaStream_t>(cuda_stream)));
  return IDG_OK;
}

int idg_degrid_subgrids_f64(const idg_plan* plan, int64_t first, int64_t count, const void* subgrids_dev,
                            const void* aterms_dev, const float* taper_dev, void* vis_dev, void* cuda_stream) {
  if (!plan || !vis_dev || !aterms_dev || !taper_dev || !subgrids_dev) { set_error("idg_degrid_subgrids_f64: null argument"); return IDG_EINVAL; }
  if (!range_ok(plan, first, count)) { set_error("idg_degrid_subgrids_f64: bad range"); return IDG_EINVAL; }
  if (count == 0) return IDG_OK;
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  const SubgridJob job = make_job(plan, d, first, count, aterms_dev, taper_dev);
  IDG_CUDA(launch_degridder_f64(job, nullptr, static_cast<const double2*>(subgrids_dev), nullptr,
                                static_cast<double2*>(vis_dev), static_cast<cudaStream_t>(cuda_stream)));
  return IDG_OK;
}

int idg_power_norm_average(const idg_plan* plan, const void* aterms_dev, double* avg_dev, void* cuda_stream) {
  if (!plan || !aterms_dev || !avg_dev) { set_error("idg_power_norm_average: null argument"); return IDG_EINVAL; }
  if (plan->n_subgrids == 0) { set_error("idg_power_norm_average: the plan has no subgrids"); return IDG_EINVAL; }
  const DeviceState* d = nullptr;
  int rc = ensure_device(plan, &d);
  if (rc != IDG_OK) return rc;
  // the factor depends on (baseline, interval) only (|| M_q M_p^H ||_F = || M_p M_q^H ||_F, so conjugated
  // subgrids need no special case): weights = planned visibilities per (baseline, interval)
  const int32_t n_int = plan->n_intervals;
  std::vector<double> w(static_cast<size_t>(plan->par.n_baselines) * n_int, 0.0);
  for (int64_t s = 0; s < plan->n_subgrids; ++s) {
    const int32_t* e = &plan->sub[static_cast<size_t>(s) * 8];
    w[static_cast<size_t>(e[0]) * n_int + e[1] / plan->par.aterm_period] += static_cast<double>(e[2]) * e[4];
  }
  std::vector<int32_t> pairs;
  std::vector<double> weights;
  double wsum = 0.0;
  for (size_t i = 0; i < w.size(); ++i) {
    if (w[i] == 0.0) continue;
    const size_t b = i / n_int;
    pairs.push_back(plan->baselines[b * 2]); pairs.push_back(plan->baselines[b * 2 + 1]);
    pairs.push_back(static_cast<int32_t>(i % n_int));
    weights.push_back(w[i]);
    wsum += w[i];
  }
  const int L = plan->par.subgrid_size;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  int32_t* d_pairs = nullptr;
  double *d_w = nullptr, *d_scratch = nullptr;
  cudaError_t e = upload(pairs, &d_pairs);
  if (e == cudaSuccess) e = upload(weights, &d_w);
  if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void**>(&d_scratch), sizeof(double) * kPowerNormSlices * L * L);
  if (e == cudaSuccess)
    e = launch_power_norm_average(static_cast<const float4*>(aterms_dev), L, n_int, d_pairs, d_w,
                                  static_cast<int64_t>(weights.size()), wsum, d_scratch, avg_dev, stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
  cudaFree(d_pairs); cudaFree(d_w); cudaFree(d_scratch);
  if (e != cudaSuccess) return cuda_fail(e, "idg_power_norm_average");
  return IDG_OK;
}

int idg_subgrid_fft(int32_t subgrid_size, int64_t n_planes, void* planes_dev, int direction, void* cuda_stream) {
  if (!subgrid_size_ok(subgrid_size)) {
    set_error("idg_subgrid_fft: subgrid_size must be 32, 48, 64, 96, 128 or 160");
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
  e = launch_adder(d->meta, dc, first, count, plan->par.subgrid_size, plan->par.grid_size, plan->tiles_x, plan->tiles_y,
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
    std::lock_guard<std::mutex> lock(g_prof_mu);
    g_prof_pool.push_back(r.a);
    g_prof_pool.push_back(r.b);
  }
  if (first_err != cudaSuccess) return cuda_fail(first_err, "idg_profile_read");
  return IDG_OK;
}

int idg_plan_kernel_split(const idg_plan* plan, int direction, int64_t* n_tensor, int64_t* n_simt) {
  if (!plan || (direction != IDG_GRID && direction != IDG_DEGRID)) { set_error("idg_plan_kernel_split: bad argument"); return IDG_EINVAL; }
  int64_t nt = 0, ns = 0;
  for (const Batch& bt : plan->batches) {
    const KernelSplit& sp = direction == IDG_GRID ? bt.grid_split : bt.degrid_split;
    if (sp.variant == IDG_VARIANT_AUTO) { nt += static_cast<int64_t>(sp.tensor.size()); ns += static_cast<int64_t>(sp.simt.size()); }
    else if (sp.variant == IDG_VARIANT_TENSOR) nt += bt.count;
    else ns += bt.count;
  }
  if (n_tensor) *n_tensor = nt;
  if (n_simt) *n_simt = ns;
  return IDG_OK;
}

int idg_kernel_config_mask(int kind, int reset) {
  if (kind != IDG_K_GRIDDER && kind != IDG_K_DEGRIDDER) { set_error("idg_kernel_config_mask: bad kind"); return IDG_EINVAL; }
  return reset ? g_kmask[kind].exchange(0) : g_kmask[kind].load();
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
