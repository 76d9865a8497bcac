/* idg_b200.h -- C ABI of the B200-native image-domain-gridding (IDG) hot path.
 *
 * Method: arxiv 2502.17789 (Hodgson 2025, "That pesky A-term", the Pigi imager); citations
 * are "PAPER.md:<line>" of the paper text plus the section / equation they fall in.
 * "R<n>" are the readings of silent or ambiguous points listed in DESIGN.md.
 *
 * Path (§2.5 :152-174):
 *   imaging    : gridder (Eq. 10 :133-137) -> A-term sandwich + taper (:156, §3.3 :251-257)
 *                -> subgrid FFT (:157) -> adder (Eq. 6 :102, :158)
 *   prediction : splitter (:169) -> inverse subgrid FFT (:170) -> taper + A-term (Eq. 13 :173)
 *                -> degridder (Eq. 13 :171-174)
 *
 * Conventions:
 *   Ng grid size (even), cell [rad], S = Ng*cell; L subgrid size in {32,48,64,96,128,160}; P total
 *   kernel padding in pixels; kappa_c = nu_c / 299792458.0; row r = b*n_times + t
 *   (baseline-major); u = u_m(r)*kappa_c [wavelengths].
 *   subgrid s = (b, t0, nt, c0, nc, x0, y0, wl): rows b*n_times + t0 .. +nt, channels c0 .. +nc,
 *   lower-left master-grid pixel (x0, y0), w-layer wl (signed).  Centre cx = x0 + L/2,
 *   u0 = (cx - Ng/2)/S, v0 likewise, w0 = (wl + 1/2)*w_step if w_step > 0 else 0.
 *   subgrid pixel (y, x): l = (x - L/2)*S/L, m = (y - L/2)*S/L, n' = sqrt(1-l^2-m^2) - 1.
 *   phase [cycles] phi = (u-u0) l + (v-v0) m + (w-w0) n'.
 *   2x2 matrices are row-major: vis[r, c, 0..3] = (XX, XY, YX, YY); Jones M[st, it, y, x, 2, 2].
 *
 * All *_dev pointers are caller-owned device memory (16-byte aligned); all *_host pointers are
 * caller-owned host memory.  The library allocates on the device only what belongs to the plan:
 * the metadata it uploads on first use and the adder's scratch (fp64 partial sums of the tile
 * segments, one counter per tile), both freed by idg_plan_destroy.  Because that scratch is per
 * plan, calls on ONE plan must not overlap in time (one stream at a time); different plans are
 * independent.  All device work is enqueued on the
 * caller's stream (a cudaStream_t passed as void*; NULL = default stream) and the calls return
 * without synchronising unless stated.  Every function returns 0 on success or a negative
 * IDG_E* code; idg_last_error() gives a thread-local message.  There is no CPU fallback: a
 * device call on a machine without a usable sm_100 GPU returns IDG_ECUDA.
 */
#ifndef IDG_B200_H
#define IDG_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define IDG_API __attribute__((visibility("default")))
#else
#define IDG_API
#endif

#define IDG_OK            0
#define IDG_EINVAL       -1   /* bad argument (null pointer, non-ascending channels, bad sizes)  */
#define IDG_EUNSUPPORTED -2   /* subgrid size not in {32,48,64,96,128,160}                       */
#define IDG_ENOMEM       -3   /* workspace too small / host allocation failed                   */
#define IDG_ECUDA        -4   /* CUDA runtime error (message in idg_last_error)                 */

#define IDG_GRID   0          /* direction selectors for idg_workspace_bytes                    */
#define IDG_DEGRID 1

/* stage selectors for idg_grid_subgrids */
#define IDG_STAGE_GRIDDER 0   /* after gridder + A-term + taper (steps a1-a3), image domain     */
#define IDG_STAGE_FFT     1   /* after the subgrid FFT (step a4), uv domain                     */

typedef struct idg_plan idg_plan;          /* opaque; host-owned; immutable after create          */

typedef struct {
  int32_t grid_size;      /* Ng, even                                                            */
  int32_t subgrid_size;   /* L in {32, 48, 64, 96, 128, 160}                                     */
  int32_t padding;        /* P, total kernel padding in pixels, 0 <= P < L-1  (R8)               */
  int32_t n_stations;
  int32_t n_baselines;
  int32_t n_times;
  int32_t n_chan;
  int32_t aterm_period;   /* timesteps per A-term interval, >= 1 (R6)                            */
  double  cell_size;      /* rad                                                                 */
  double  w_step;         /* wavelengths; 0 => single layer with w0 = 0 (R9)                     */
  double  comfort;        /* fraction of the usable span a channel range may fill (R7); 0.75     */
  int64_t max_batch_subgrids; /* subgrids processed per batch (§3.4 :259-267, R18);
                                 0 => library default                                            */
  int32_t gridder_variant;   /* IDG_VARIANT_* of the gridder direct sum (0 = AUTO), see below    */
  int32_t degridder_variant; /* IDG_VARIANT_* of the degridder direct sum (0 = AUTO)             */
  int32_t positive_w;     /* != 0: rows with w < 0 are used as (-u,-v,-w) of the swapped baseline
                             with V^dagger, so that only layers wl >= 0 exist (PAPER.md:178
                             footnote 4, R21).  A subgrid never mixes the two kinds of row.      */
  int32_t power_norm;     /* != 0: the imaging sandwich is divided per pixel by the Frobenius
                             norm || M_p M_q^H ||_F (§3.3, R22); the caller corrects
                             the image by idg_power_norm_average.  Prediction is not normalised. */
} idg_params;

/* ---- planner: visibility table -> subgrids (§2.2 :62-72, §2.4 :141-143, §3.1
 * :186-200, §3.3 :255; the deterministic reading is DESIGN.md "O1").  Host only: works on a
 * machine without a GPU.
 *   uvw_m_host     [n_baselines*n_times, 3] float64 metres, row r = b*n_times + t
 *   freqs_host     [n_chan] float64 Hz, strictly ascending (R11) else IDG_EINVAL
 *   baselines_host [n_baselines, 2] int32 station pairs (p, q)
 * The plan keeps its own copies; the inputs may be freed after the call. */
IDG_API int  idg_plan_create(const idg_params* params, const double* uvw_m_host, const double* freqs_host,
                     const int32_t* baselines_host, idg_plan** out);
IDG_API void idg_plan_destroy(idg_plan* plan);

/* Counts: subgrids, number of w-layers W = wl_max - wl_min + 1 (1 if no subgrids), wl_min,
 * visibilities covered by a subgrid and visibilities dropped because their subgrid would
 * leave the master grid.  Any output pointer may be NULL. */
IDG_API int  idg_plan_counts(const idg_plan* plan, int64_t* n_subgrids, int32_t* n_wlayers, int32_t* wl_min,
                     int64_t* n_vis_planned, int64_t* n_vis_dropped);

/* sub_host [n_subgrids, 8] int32 rows (b, t0, nt, c0, nc, x0, y0, wl), sorted by (wl, b, t0, c0). */
IDG_API int  idg_plan_export(const idg_plan* plan, int32_t* sub_host);

/* Bytes of device workspace idg_grid / idg_degrid need (the subgrid stack of one batch,
 * PAPER.md:210 "a contiguous stack of L x L arrays"). */
IDG_API size_t idg_workspace_bytes(const idg_plan* plan, int direction);

/* ---- imaging direction, steps 2.i-2.iii of PAPER.md:155-158 over all subgrids of the plan.
 *   vis_dev    [n_rows, n_chan, 4] complex64 (interleaved re, im)
 *   aterms_dev [n_stations, n_intervals, L, L, 2, 2] complex64, n_intervals = ceil(n_times/aterm_period);
 *              applied as M_p X M_q^H (R5): pass A^-1 for paper-style imaging (Eq. 10)
 *   taper_dev  [L, L] float32 (R4, R15)
 *   grid_dev   [n_wlayers, 4, Ng, Ng] complex64, ACCUMULATED INTO (caller zeroes)
 * The adder is atomic-free and its summation order is fixed: results are bitwise reproducible. */
IDG_API int  idg_grid(const idg_plan* plan, const void* vis_dev, const void* aterms_dev, const float* taper_dev,
              void* grid_dev, void* workspace_dev, size_t workspace_bytes, void* cuda_stream);

/* The same with imaging weights applied as the visibilities are loaded ("weighting ...
 * performed by each thread"): vis[r, c, :] is multiplied by weights_dev[r, c]
 * (float32 [n_rows, n_chan]; NULL = idg_grid).  Flagged samples are weight 0: such a sample contributes an exact
 * zero whatever it holds (NaN and Inf included; it is selected out, not multiplied) and does not enter the
 * tensor-core gridder's per-segment scale.  A non-finite sample with a non-zero weight is the caller's error: the
 * result of every subgrid that covers it is undefined (NaN in its pixels). */
IDG_API int  idg_grid_weighted(const idg_plan* plan, const void* vis_dev, const float* weights_dev,
                       const void* aterms_dev, const float* taper_dev, void* grid_dev, void* workspace_dev,
                       size_t workspace_bytes, void* cuda_stream);

/* ---- prediction direction, steps 3.i-3.iii of PAPER.md:168-174.  Writes vis_dev[r, c, :]
 * for every visibility covered by a subgrid and leaves the others untouched.  The same taper
 * array multiplies (R4) and the same sandwich M_p X M_q^H is applied (R5: pass A). */
IDG_API int  idg_degrid(const idg_plan* plan, const void* grid_dev, const void* aterms_dev, const float* taper_dev,
                void* vis_dev, void* workspace_dev, size_t workspace_bytes, void* cuda_stream);

/* ---- the same two calls on HOST buffers (pinned memory recommended: pageable memory makes the
 * copies synchronous).  They copy the inputs to `arena_dev`, run the device path on `cuda_stream`,
 * copy the result back (grid_host is accumulated into: it is uploaded behind the visibilities and added
 * on the device after the subgrids) and synchronise before returning.  Only the master-grid rows under
 * a subgrid are moved, in either direction: the rest of grid_host is neither read nor written.  Copies run on a second stream and overlap compute batch by batch: a visibility row
 * goes up just before the first batch that reads it and comes down right after the last batch
 * that writes it, so a plan with smaller batches (idg_params.max_batch_subgrids) overlaps more.
 * idg_degrid_host uploads vis_host only when the planner left visibilities uncovered (they come
 * back untouched).  arena_dev must hold idg_host_arena_bytes(plan, direction) bytes. */
IDG_API size_t idg_host_arena_bytes(const idg_plan* plan, int direction);
/* Bytes one idg_grid_host / idg_degrid_host call moves over the bus in each direction: the visibility rows
 * and the master-grid rows that lie under a subgrid, the A-terms and the taper (nothing else is touched). */
IDG_API int  idg_host_traffic_bytes(const idg_plan* plan, int direction, int64_t* h2d_bytes, int64_t* d2h_bytes);
IDG_API int  idg_grid_host(const idg_plan* plan, const void* vis_host, const void* aterms_host,
                   const float* taper_host, void* grid_host, void* arena_dev, size_t arena_bytes,
                   void* cuda_stream);
IDG_API int  idg_degrid_host(const idg_plan* plan, const void* grid_host, const void* aterms_host,
                     const float* taper_host, void* vis_host, void* arena_dev, size_t arena_bytes,
                     void* cuda_stream);

/* ---- stage-level entry points (used by the parity tests; same kernels as above) ----------- */

/* Subgrids [first, first+count) through the gridder (+A-term+taper) and, if stage ==
 * IDG_STAGE_FFT, the subgrid FFT.  subgrids_dev [count, 4, L, L] complex64 (pol-major planes). */
IDG_API int  idg_grid_subgrids(const idg_plan* plan, int64_t first, int64_t count, const void* vis_dev,
                       const void* aterms_dev, const float* taper_dev, void* subgrids_dev,
                       int stage, void* cuda_stream);

/* Image-domain subgrids [first, first+count) (after the inverse FFT, before taper / A-term)
 * through taper + A-term + degridder into vis_dev. */
IDG_API int  idg_degrid_subgrids(const idg_plan* plan, int64_t first, int64_t count, const void* subgrids_dev,
                         const void* aterms_dev, const float* taper_dev, void* vis_dev,
                         void* cuda_stream);

/* Centred L x L DFT of `n_planes` planes in place, each scaled by 1/L^2 (R1, R2):
 * direction +1: out[gy,gx] = L^-2 sum in[y,x] exp(-2 pi i((gy-L/2)(y-L/2)+(gx-L/2)(x-L/2))/L)
 * direction -1: the same with exp(+...)  (Eq. 7-8 :107-117). */
IDG_API int  idg_subgrid_fft(int32_t subgrid_size, int64_t n_planes, void* planes_dev, int direction,
                     void* cuda_stream);

/* Adder / splitter for subgrids [first, first+count) (Eq. 6 :102, :158, :169):
 *   adder   : grid[wl - wl_min, pol, y0+gy, x0+gx] += subgrids[s - first, pol, gy, gx]
 *   splitter: subgrids[s - first, pol, gy, gx]      = grid[wl - wl_min, pol, y0+gy, x0+gx]   */
IDG_API int  idg_adder(const idg_plan* plan, int64_t first, int64_t count, const void* subgrids_dev,
               void* grid_dev, void* cuda_stream);
IDG_API int  idg_splitter(const idg_plan* plan, int64_t first, int64_t count, const void* grid_dev,
                  void* subgrids_dev, void* cuda_stream);

/* ---- per-kernel timing (CUDA events recorded on the caller's stream around every kernel
 * launch while enabled; off by default).  idg_profile_read waits for the recorded events,
 * adds their durations into ms_out[kind] / launches_out[kind] (kind = IDG_K_*, arrays of
 * IDG_K_COUNT) and clears the record. */
#define IDG_K_GRIDDER   0
#define IDG_K_FFT       1
#define IDG_K_ADDER     2
#define IDG_K_SPLITTER  3
#define IDG_K_IFFT      4
#define IDG_K_DEGRIDDER 5
#define IDG_K_COUNT     6
IDG_API int  idg_profile_enable(int on);
IDG_API int  idg_profile_read(double* ms_out, int64_t* launches_out);

/* ---- w-stacking closure either side of the path (Eq. 11 :145-148, Eq. 12 :164-166).
 * NOT part of the measured hot path; the master-grid FFT is cuFFT's (its plan and work area are
 * created on the first call and belong to the idg_plan).
 *   idg_grid_to_image: image[p, y, x] = corr[y, x] * sum_layers e^{+2 pi i w0 n'(l_x, m_y)} *
 *       sum_g grid[layer, p, g] e^{+2 pi i ((gy-Ng/2)(y-Ng/2) + (gx-Ng/2)(x-Ng/2)) / Ng}
 *   idg_image_to_grid: grid[layer, p, g] = sum_j corr[j] e^{-2 pi i w0 n'_j} image[p, j] e^{-2 pi i (...)/Ng}
 * w0 = (wl + 1/2) w_step (0 if w_step = 0), l_x = (x - Ng/2) S/Ng, no 1/Ng^2 factor in either direction.
 * corr_dev: optional real [Ng, Ng] factor (NULL = 1), e.g. 1 / (T_full * n_vis) for a dirty image or
 * 1 / T_full for a model (R4: the image-level taper correction is the caller's).
 * grid_dev [n_wlayers, 4, Ng, Ng] c64, image_dev [4, Ng, Ng] c64 (overwritten / read),
 * workspace_dev: idg_closure_workspace_bytes(plan) bytes for idg_grid_to_image (the grid is preserved);
 * idg_image_to_grid overwrites grid_dev and needs no workspace. */
IDG_API size_t idg_closure_workspace_bytes(const idg_plan* plan);
IDG_API int  idg_grid_to_image(const idg_plan* plan, const void* grid_dev, const float* corr_dev, void* image_dev,
                       void* workspace_dev, size_t workspace_bytes, void* cuda_stream);
IDG_API int  idg_image_to_grid(const idg_plan* plan, const void* image_dev, const float* corr_dev, void* grid_dev,
                       void* cuda_stream);

/* Kernel variant of the two direct-sum kernels: a PLAN parameter (idg_params.gridder_variant /
 * .degridder_variant), so two plans in one process may differ.
 * IDG_VARIANT_AUTO (0, the default): PER SUBGRID (PAPER.md:247 footnote 7, "swap the kernel design by a
 *   subgrid-occupancy heuristic"; :239-241), the tensor-core kernel where its operand slots are well filled
 *   (gridder: at least 65 % of the slots of a table row's 16-channel chunks carry visibilities; degridder:
 *   always, its idle warps cost nothing) and the shape fits its shared-memory tables, else the SIMT kernel.  A batch is then
 *   two launches over complementary index lists; the adder's order is untouched.
 * IDG_VARIANT_SIMT: all arithmetic on the FP32 / SFU pipes (packed FFMA2).
 * IDG_VARIANT_TENSOR: the phasor matrix is generated on the SIMT pipes and the 2x2 complex MACs run on the
 *   tensor cores (tcgen05, fp32 accumulation drained into registers).  Operands are split into a head and a
 *   remainder of 11 significant bits each: the gridder uses fp16 heads + fp16 remainders with ONE
 *   power-of-two scale per segment of a subgrid (at most 2560 visibilities), so its absolute error is about
 *   2^-22 of the segment's largest |component|: samples far below the segment maximum keep that ABSOLUTE
 *   accuracy, not their relative one (tests pin this with 1e6 of dynamic range inside one subgrid).  The
 *   degridder uses tf32 heads + tf32 remainders (relative 2^-22 per operand).
 * IDG_VARIANT_FP64: SIMT kernels with the phase, sin/cos and accumulation in fp64 (§5.3: the
 *   fp64 kernels are about 4.5x slower; §4.1 :289-293 accuracy experiment); inputs and the subgrid stack
 *   stay complex64 on the idg_grid / idg_degrid path, the *_f64 stage calls below keep fp64 end to end.
 * All but FP64 meet the 1e-5 bar with margin; FP64 is for accuracy studies. */
#define IDG_VARIANT_AUTO   0
#define IDG_VARIANT_SIMT   1
#define IDG_VARIANT_TENSOR 2
#define IDG_VARIANT_FP64   3

/* How IDG_VARIANT_AUTO splits the plan's subgrids between the tensor-core and the SIMT kernel of a direction
 * (IDG_GRID or IDG_DEGRID), summed over the batches.  A plan with a forced variant reports all subgrids under it
 * (FP64 counts as SIMT); a shape whose per-subgrid tables the tensor-core gridder cannot hold in shared memory (more
 * than 1264 channels, more than 128 rows per A-term interval) runs the SIMT gridder whatever was asked for and is
 * reported so.  Host only. */
IDG_API int  idg_plan_kernel_split(const idg_plan* plan, int direction, int64_t* n_tensor, int64_t* n_simt);

/* Which kernels the direct-sum step `kind` (IDG_K_GRIDDER or IDG_K_DEGRIDDER) has launched in this process
 * since the last reset, as a bit mask: bit 0 SIMT, bit 1 / 2 / 4 tensor-core with 1 / 2 / 4 compute groups
 * per CTA (the gridder picks by shared-memory fit; the degridder always runs 2), bit 8 fp64, bit 9 the tensor-core
 * gridder with phasor rotation along the channel axis (uniformly spaced channels; otherwise one sincos per pair).  reset != 0
 * clears the mask after reading.  For the tests, which must know what they exercised. */
#define IDG_KMASK_SIMT   (1 << 0)
#define IDG_KMASK_TC(ng) (1 << (ng))
#define IDG_KMASK_FP64   (1 << 8)
#define IDG_KMASK_ROT    (1 << 9)
IDG_API int  idg_kernel_config_mask(int kind, int reset);

/* fp64 stage calls: the two direct sums with their A-term /
 * taper step in double precision from the same complex64 / float32 inputs.
 *   idg_grid_subgrids_f64  : subgrids_dev [count, 4, L, L] complex128, stage IDG_STAGE_GRIDDER only
 *   idg_degrid_subgrids_f64: subgrids_dev [count, 4, L, L] complex128 in, vis_dev [n_rows, n_chan, 4]
 *                            complex128 out (planned visibilities of the range only) */
IDG_API int  idg_grid_subgrids_f64(const idg_plan* plan, int64_t first, int64_t count, const void* vis_dev,
                           const void* aterms_dev, const float* taper_dev, void* subgrids_dev,
                           void* cuda_stream);
IDG_API int  idg_degrid_subgrids_f64(const idg_plan* plan, int64_t first, int64_t count, const void* subgrids_dev,
                             const void* aterms_dev, const float* taper_dev, void* vis_dev,
                             void* cuda_stream);

/* Weighted average over the subgrids of the power-normalisation factor 1 / || M_p M_q^H ||_F, weights =
 * visibilities per subgrid ("the final image must then be corrected by the weighted average
 * of this normalisation factor across all subgrids", R22).  avg_dev [L, L] float64, overwritten.
 * Works for any plan (power_norm on or off); synchronises the stream. */
IDG_API int  idg_power_norm_average(const idg_plan* plan, const void* aterms_dev, double* avg_dev,
                            void* cuda_stream);

/* ---- the same average for callers that cannot allocate device memory ------------------------------------
 * idg_power_norm_average allocates (and frees) three device buffers per call.  Two kinds of caller cannot
 * live with that: one whose own pool took the whole device at start-up (master grids fill the card,
 * PAPER.md:399-405), where a raw cudaMalloc fails although the pool has room; and one that prepares the
 * correction while gridding batches run on other streams, because cudaMalloc / cudaFree synchronise the whole
 * device and stall them.  idg_power_norm_average_static calls no cudaMalloc, no cudaFree and no allocating
 * library routine, takes no plan (so it never triggers the plan's metadata upload) and does not synchronise:
 * the two kernels are enqueued on cuda_stream and avg_dev is valid when they have run.
 *
 * Its scratch (64 x L x L fp64 partial sums) is an array built into the library:
 * 64 x 96 x 96 x 8 B = 4.5 MiB of every GPU that loads the library, until the process exits.  Hence
 *   - subgrid_size > IDG_STATIC_MAX_SUBGRID_SIZE (96) is refused with IDG_EUNSUPPORTED and a message naming
 *     the limit (L = 128 and 160 need idg_power_norm_average);
 *   - all calls on one device share that array.  It needs no clearing (each call overwrites what it reads)
 *     and keeps the last call's partial sums, but two calls that overlap on the GPU -- different streams,
 *     different host threads, different plans -- race on it and both results are garbage.  Order them.
 *   - the first call on each device looks up the array's device address (one cudaGetSymbolAddress, with that
 *     device current).  Make that first call during set-up, before any stream capture begins.
 *
 * The caller passes everything else, already on the device (16-byte aligned):
 *   aterms_dev  [n_stations, n_intervals, L, L, 2, 2] complex64, as for idg_grid
 *   pairs_dev   [n_terms, 3] int32 (p, q, interval): the (baseline, interval) combinations that carry
 *               planned visibilities;  weights_dev [n_terms] float64: their visibility counts;
 *   weight_sum  the sum of the weights;  avg_dev [L, L] float64, overwritten.
 * idg_plan_power_norm_terms lists the terms of a plan on the HOST (no GPU needed), in the order
 * idg_power_norm_average uses, so that both calls return bit-identical averages: call it with capacity 0 to
 * get n_terms and weight_sum, then with pairs_host [n_terms, 3] / weights_host [n_terms] (capacity =
 * n_terms; IDG_ENOMEM if too small), and copy both into your own device memory once. */
#define IDG_STATIC_MAX_SUBGRID_SIZE 96
IDG_API int  idg_plan_power_norm_terms(const idg_plan* plan, int32_t* pairs_host, double* weights_host,
                               int64_t capacity, int64_t* n_terms, double* weight_sum);
IDG_API int  idg_power_norm_average_static(const void* aterms_dev, int32_t subgrid_size, int32_t n_intervals,
                                   const int32_t* pairs_dev, const double* weights_dev, int64_t n_terms,
                                   double weight_sum, double* avg_dev, void* cuda_stream);

/* Empirical ALU peaks of the current device, measured the way the paper measures its Table 1
 * (§5.1 :339-351): register-only loops timed with the SM cycle counter.  Synchronous.
 * out_host[7], per SM per clock: [0] FFMA lane-ops, [1] FFMA2 (packed fp32x2) FMA lane-ops,
 * [2] MUFU.EX2 lane-ops, [3] sin+cos pairs (__sincosf), [4] (visibility, pixel) pairs of the
 * gridder's instruction mix (phase FFMA + __sincosf + 8 FFMA2 per pair), [5] the same mix with
 * 16 scalar FFMA, [6] pairs of the operand-generation mix alone (phase FFMA + __sincosf + split of
 * cos and sin into a tf32 head and an exact remainder, the round-1 operand format: what is left on the SIMT pipes when the
 * MACs go to the tensor cores).  These are the
 * denominators of the ALU roofline. */
IDG_API int  idg_measure_alu_peaks(double* out_host);

/* Number of kernels the library has launched in this process (for bench.py's gpu_launches). */
IDG_API int64_t idg_launch_count(void);

IDG_API const char* idg_last_error(void);
IDG_API const char* idg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* IDG_B200_H */
