// Host planner: visibility table -> subtables = subgrids.
//
// PAPER.md §2.2 :62-72 (every visibility in exactly one L x L subgrid, subgrids may overlap,
// centre snaps to a master-grid pixel), §2.4 :141-143 (subgrids snap to a w-layer), §3.1
// :186-200 (single pass per baseline: channel ranges that fit "comfortably", then grow in time;
// only the corners of a subtable are tested), §3.3 :255 (one A-term interval per subgrid).
// The deterministic reading (O1, R6-R9, R12) is restated here in C++; all arithmetic
// is IEEE fp64 in a fixed order (this file is compiled with -ffp-contract=off) so that the plan
// is bit-identical to the one the test oracle derives independently.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <tuple>

#include "idg_internal.h"

namespace idg {

namespace {

struct WorkItem { int32_t t0, lo, hi; };

struct Emitted { int32_t v[8]; };

inline bool emitted_less(const Emitted& a, const Emitted& b) {
  // order (wl, b, t0, c0)
  return std::make_tuple(a.v[7], a.v[0], a.v[1], a.v[3]) < std::make_tuple(b.v[7], b.v[0], b.v[1], b.v[3]);
}

}  // namespace

int plan_build(idg_plan* plan) {
  const idg_params& par = plan->par;
  const int32_t Ng = par.grid_size, L = par.subgrid_size, P = par.padding;
  const int32_t nT = par.n_times, nC = par.n_chan;
  const double S = plan->image_size;
  const double span_max = static_cast<double>(L - P - 1);
  const double comfort_span = par.comfort * span_max;
  const bool layered = par.w_step > 0.0;

  // uniformly spaced channels let the tensor-core gridder rotate its phasors along the channel axis
  plan->dkappa = 0.0;
  if (nC >= 2) {
    const double dk = (plan->kappa[nC - 1] - plan->kappa[0]) / (nC - 1);
    bool uniform = dk > 0.0;
    for (int32_t c = 0; c < nC && uniform; ++c)
      uniform = std::fabs(plan->kappa[c] - (plan->kappa[0] + c * dk)) <= 1e-9 * dk * nC;
    if (uniform) plan->dkappa = dk;
  }

  std::vector<Emitted> out;
  std::vector<double> X(static_cast<size_t>(nT) * nC), Y(X.size());
  std::vector<int64_t> WL(X.size());
  std::vector<char> FLIP(static_cast<size_t>(nT), 0);
  std::vector<WorkItem> work;
  int64_t dropped = 0;

  for (int32_t b = 0; b < par.n_baselines; ++b) {
    const double* rows = plan->uvw.data() + static_cast<size_t>(b) * nT * 3;
    for (int32_t t = 0; t < nT; ++t) {
      double um = rows[t * 3 + 0], vm = rows[t * 3 + 1], wm = rows[t * 3 + 2];
      // PAPER.md:178 (fn 4): a row with w < 0 is used as the row (-u,-v,-w) of the swapped baseline (R21)
      FLIP[t] = (par.positive_w != 0 && wm < 0.0) ? 1 : 0;
      if (FLIP[t]) { um = -um; vm = -vm; wm = -wm; }
      for (int32_t c = 0; c < nC; ++c) {
        const double k = plan->kappa[c];
        const size_t i = static_cast<size_t>(t) * nC + c;
        X[i] = (um * k) * S;            // master-grid pixels from the centre, this exact order
        Y[i] = (vm * k) * S;
        WL[i] = layered ? static_cast<int64_t>(std::floor((wm * k) / par.w_step)) : 0;
      }
    }
    auto at = [nC](int32_t t, int32_t c) { return static_cast<size_t>(t) * nC + c; };

    for (int32_t it = 0; it < plan->n_intervals; ++it) {
      const int32_t ta = it * par.aterm_period;
      const int32_t tb = std::min(ta + par.aterm_period, nT);
      work.clear();
      work.push_back({ta, 0, nC - 1});
      while (!work.empty()) {
        const WorkItem w = work.back();
        work.pop_back();
        const int32_t t0 = w.t0, lo = w.lo, hi = w.hi;
        const int64_t wl0 = WL[at(t0, lo)];
        // channel range at the first timestep that fits comfortably (R7)
        int32_t c1 = lo;
        while (c1 + 1 <= hi &&
               std::max(std::fabs(X[at(t0, c1 + 1)] - X[at(t0, lo)]),
                        std::fabs(Y[at(t0, c1 + 1)] - Y[at(t0, lo)])) <= comfort_span &&
               WL[at(t0, c1 + 1)] == wl0) {
          ++c1;
        }
        if (c1 < hi) work.push_back({t0, c1 + 1, hi});
        double xmin = std::min(X[at(t0, lo)], X[at(t0, c1)]), xmax = std::max(X[at(t0, lo)], X[at(t0, c1)]);
        double ymin = std::min(Y[at(t0, lo)], Y[at(t0, c1)]), ymax = std::max(Y[at(t0, lo)], Y[at(t0, c1)]);
        // grow in time while the corner bounding box still fits
        int32_t n = 1;
        while (t0 + n < tb) {
          const int32_t t = t0 + n;
          if (WL[at(t, lo)] != wl0 || WL[at(t, c1)] != wl0 || FLIP[t] != FLIP[t0]) break;
          const double nxmin = std::min(xmin, std::min(X[at(t, lo)], X[at(t, c1)]));
          const double nxmax = std::max(xmax, std::max(X[at(t, lo)], X[at(t, c1)]));
          const double nymin = std::min(ymin, std::min(Y[at(t, lo)], Y[at(t, c1)]));
          const double nymax = std::max(ymax, std::max(Y[at(t, lo)], Y[at(t, c1)]));
          if ((nxmax - nxmin) > span_max || (nymax - nymin) > span_max) break;
          xmin = nxmin; xmax = nxmax; ymin = nymin; ymax = nymax;
          ++n;
        }
        if (t0 + n < tb) work.push_back({t0 + n, lo, c1});
        // centre snaps to a master-grid pixel, round half up (R12)
        const int64_t cx = static_cast<int64_t>(std::floor((xmin + xmax) / 2.0 + 0.5)) + Ng / 2;
        const int64_t cy = static_cast<int64_t>(std::floor((ymin + ymax) / 2.0 + 0.5)) + Ng / 2;
        const int64_t x0 = cx - L / 2, y0 = cy - L / 2;
        const int32_t nc = c1 - lo + 1;
        if (x0 < 0 || y0 < 0 || x0 + L > Ng || y0 + L > Ng) {
          dropped += static_cast<int64_t>(n) * nc;
          continue;
        }
        Emitted e;
        e.v[0] = b; e.v[1] = t0; e.v[2] = n; e.v[3] = lo; e.v[4] = nc;
        e.v[5] = static_cast<int32_t>(x0); e.v[6] = static_cast<int32_t>(y0);
        e.v[7] = static_cast<int32_t>(wl0);
        out.push_back(e);
      }
    }
  }
  std::sort(out.begin(), out.end(), emitted_less);   // keys are unique: no stability issue

  plan->n_subgrids = static_cast<int64_t>(out.size());
  plan->sub.resize(out.size() * 8);
  int64_t planned = 0;
  int32_t wl_lo = 0, wl_hi = 0;
  for (size_t i = 0; i < out.size(); ++i) {
    std::memcpy(&plan->sub[i * 8], out[i].v, sizeof(out[i].v));
    planned += static_cast<int64_t>(out[i].v[2]) * out[i].v[4];
    if (i == 0) { wl_lo = wl_hi = out[i].v[7]; }
    wl_lo = std::min(wl_lo, out[i].v[7]);
    wl_hi = std::max(wl_hi, out[i].v[7]);
  }
  plan->n_vis_planned = planned;
  plan->n_vis_dropped = dropped;
  plan->wl_min = wl_lo;
  plan->n_wlayers = out.empty() ? 1 : (wl_hi - wl_lo + 1);

  plan->tile_w = tile_width(L);
  plan->tile_h = tile_height(L);
  plan->tiles_x = (Ng + plan->tile_w - 1) / plan->tile_w;
  plan->tiles_y = (Ng + plan->tile_h - 1) / plan->tile_h;

  // batches: contiguous ranges of the sorted subgrid list (§3.4 :259-267, R18)
  int64_t cap = par.max_batch_subgrids;
  if (cap <= 0) {
    const int64_t bytes_per = static_cast<int64_t>(L) * L * 4 * 8;
    cap = std::max<int64_t>(1, (int64_t{4} << 30) / bytes_per);
  }
  plan->batch_capacity = std::max<int64_t>(1, std::min<int64_t>(cap, std::max<int64_t>(plan->n_subgrids, 1)));
  plan->batches.clear();
  for (int64_t first = 0; first < plan->n_subgrids; first += plan->batch_capacity) {
    Batch bt;
    bt.first = first;
    bt.count = std::min(plan->batch_capacity, plan->n_subgrids - first);
    build_tile_csr(plan, bt.first, bt.count, &bt.csr);
    split_kernels(plan, bt.first, bt.count, IDG_GRID, &bt.grid_split);
    split_kernels(plan, bt.first, bt.count, IDG_DEGRID, &bt.degrid_split);
    plan->batches.push_back(std::move(bt));
  }
  return IDG_OK;
}

// For subgrids [first, first+count): which adder tiles (tile_w x tile_h master-grid pixels of one
// w-layer) does each overlap.  Lists are ascending in subgrid index, which fixes the summation
// order of the adder (R18: bitwise reproducible).
void build_tile_csr(const idg_plan* plan, int64_t first, int64_t count, TileCsr* out) {
  const int32_t L = plan->par.subgrid_size;
  const int32_t tx_n = plan->tiles_x, ty_n = plan->tiles_y;
  std::vector<std::pair<int32_t, int32_t>> pairs;   // (tile id, subgrid)
  pairs.reserve(static_cast<size_t>(count) * ((L + plan->tile_h - 1) / plan->tile_h + 1) * 2);
  for (int64_t s = first; s < first + count; ++s) {
    const int32_t* e = &plan->sub[static_cast<size_t>(s) * 8];
    const int32_t x0 = e[5], y0 = e[6], layer = e[7] - plan->wl_min;
    const int32_t tx0 = x0 / plan->tile_w, tx1 = (x0 + L - 1) / plan->tile_w;
    const int32_t ty0 = y0 / plan->tile_h, ty1 = (y0 + L - 1) / plan->tile_h;
    for (int32_t ty = ty0; ty <= ty1; ++ty)
      for (int32_t tx = tx0; tx <= tx1; ++tx)
        pairs.emplace_back((layer * ty_n + ty) * tx_n + tx, static_cast<int32_t>(s));
  }
  std::sort(pairs.begin(), pairs.end());
  // group by tile (subgrids ascending within a tile), then emit the tiles heaviest first so the
  // longest lists start early (the order of TILES does not affect any sum)
  struct Run { int32_t tile; size_t beg, end; };
  std::vector<Run> runs;
  for (size_t i = 0; i < pairs.size(); ++i) {
    if (i == 0 || pairs[i].first != pairs[i - 1].first) runs.push_back({pairs[i].first, i, i});
    runs.back().end = i + 1;
  }
  std::stable_sort(runs.begin(), runs.end(),
                   [](const Run& a, const Run& b) { return (a.end - a.beg) > (b.end - b.beg); });
  out->tile_ids.clear(); out->offsets.clear(); out->items.clear();
  out->items.reserve(pairs.size());
  for (const Run& r : runs) {
    out->tile_ids.push_back(r.tile);
    out->offsets.push_back(static_cast<int32_t>(out->items.size()));
    for (size_t i = r.beg; i < r.end; ++i) out->items.push_back(pairs[i].second);
  }
  out->offsets.push_back(static_cast<int32_t>(out->items.size()));
  // segments: a block walks at most kAdderSegment subgrids, so one dense tile does not serialise the launch
  struct Seg { int32_t tile, beg, end, k, n, slot; };
  std::vector<Seg> segs;
  out->n_slots = 0;
  for (size_t t = 0; t < out->tile_ids.size(); ++t) {
    const int32_t beg = out->offsets[t], end = out->offsets[t + 1];
    const int32_t n = (end - beg + kAdderSegment - 1) / kAdderSegment;
    for (int32_t k = 0; k < n; ++k) {
      const int32_t b = beg + k * kAdderSegment, e = std::min(end, b + kAdderSegment);
      segs.push_back({static_cast<int32_t>(t), b, e, k, n, n > 1 ? out->n_slots++ : -1});
    }
  }
  std::stable_sort(segs.begin(), segs.end(), [](const Seg& a, const Seg& b) { return (a.end - a.beg) > (b.end - b.beg); });
  out->segs.clear();
  out->segs.reserve(segs.size() * kSegStride);
  for (const Seg& g : segs) {
    const int32_t rec[kSegStride] = {g.tile, g.beg, g.end, g.k, g.n, g.slot};
    out->segs.insert(out->segs.end(), rec, rec + kSegStride);
  }
}

bool subgrid_conjugated(const idg_plan* plan, const int32_t* e) {
  if (!plan->par.positive_w) return false;
  return plan->uvw[(static_cast<size_t>(e[0]) * plan->par.n_times + e[1]) * 3 + 2] < 0.0;
}

// Kernel choice per subgrid (PAPER.md:247 fn 7, :239-241).  The tensor-core
// gridder pads every table row to whole 16-channel chunks: it runs at 0.96 of the ALU roofline on full chunks
// against the SIMT kernel's 0.55 (no padding), so it wins from a fill of about 0.6.
void split_kernels(const idg_plan* plan, int64_t first, int64_t count, int direction, KernelSplit* out) {
  out->tensor.clear(); out->simt.clear();
  out->variant = direction == IDG_GRID ? plan->par.gridder_variant : plan->par.degridder_variant;
  const int32_t max_nt = std::min(plan->par.n_times, plan->par.aterm_period);
  if (direction == IDG_GRID && out->variant != IDG_VARIANT_SIMT && out->variant != IDG_VARIANT_FP64 &&
      !gridder_tc_fits(plan->par.n_chan, max_nt))
    out->variant = IDG_VARIANT_SIMT;      // what launch_gridder_tc would run anyway: the reported split says so
  if (out->variant != IDG_VARIANT_AUTO) return;
  for (int64_t i = 0; i < count; ++i) {
    const int32_t* e = &plan->sub[static_cast<size_t>(first + i) * 8];
    const int32_t nt = e[2], nc = e[4];
    bool tensor;
    if (direction == IDG_GRID) tensor = 100 * nc >= 65 * ((nc + 15) / 16 * 16);     // chunk fill >= 65 %
    else                       tensor = static_cast<int64_t>(nt) * nc >= kDegridTensorMin;
    (tensor ? out->tensor : out->simt).push_back(static_cast<int32_t>(i));
  }
}

// Per-subgrid device metadata: the 8 plan fields plus stations (p, q), A-term interval,
// grid layer index and flags, so kernels need no second lookup.
void fill_meta(const idg_plan* plan, std::vector<int32_t>* meta) {
  meta->resize(static_cast<size_t>(plan->n_subgrids) * kMetaStride);
  for (int64_t s = 0; s < plan->n_subgrids; ++s) {
    const int32_t* e = &plan->sub[static_cast<size_t>(s) * 8];
    int32_t* m = &(*meta)[static_cast<size_t>(s) * kMetaStride];
    for (int i = 0; i < 8; ++i) m[i] = e[i];
    const bool conj = subgrid_conjugated(plan, e);     // conjugated rows belong to the swapped baseline (R21)
    m[8] = plan->baselines[static_cast<size_t>(e[0]) * 2 + (conj ? 1 : 0)];
    m[9] = plan->baselines[static_cast<size_t>(e[0]) * 2 + (conj ? 0 : 1)];
    m[10] = e[1] / plan->par.aterm_period;
    m[11] = e[7] - plan->wl_min;
    m[12] = conj ? kMetaConj : 0;
    m[13] = m[14] = m[15] = 0;
  }
}

}  // namespace idg
