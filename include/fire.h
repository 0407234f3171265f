/*
 * fire.h -- C ABI of libfire: batched stochastic cellular-automata fire propagation on a raster
 * landscape plus the per-simulation fitness reduction against a reference burned map, the hot
 * path of arXiv 1701.03549 (Denham & Laneri), for NVIDIA B200 (sm_100a).
 *
 * The problem as the paper states it: given raster layers for vegetation, slope, aspect and wind
 * direction (Sec. 3.1), a parameter vector beta of Eq. 1, an
 * ignition point and a random seed, run the cellular automaton
 * until the fire stops by itself and score the final burnt map
 * against a reference map with Eq. 2.  The GA / Monte-Carlo search that calls
 * this millions of times (App. B, C) stays on the host.
 *
 * Conventions (DESIGN.md "Readings of the paper" R-4..R-9)
 *   - rasters are row-major [H][W]; row 0 is north, x grows east; angles are radians, compass
 *     bearings clockwise from north.  `aspect` = bearing the slope faces (downslope), `wind` =
 *     bearing the wind blows TOWARD, `slope` = inclination angle in [0, pi/2).
 *   - veg: 0 = impossible to burn, 1 = forest (I_f = 1), >= 2 = other burnable fuel (I_f = 0).
 *   - direction d = 0..7 = N, NE, E, SE, S, SW, W, NW is the direction of travel from the burning
 *     cell to the target cell; thresholds are indexed [cell of the TARGET][d].
 *   - bitmaps: cell (x, y) is bit (x & 31) (LSB = lowest x) of 32-bit word y*ceil(W/32) + (x >> 5);
 *     tail bits of a row are zero.
 *
 * Pointers: every array argument is a DEVICE pointer on the handle's device unless its name
 * ends in `_host`.  `stream` is a cudaStream_t passed as void* (NULL = default stream).
 * Ownership: the caller owns every array; the library borrows it until the enqueued work is
 * done.  The handle owns covariates, thresholds, scratch planes and queues.
 * Asynchrony: every call only enqueues work on `stream` unless stated otherwise; outputs are valid
 * once the caller has synchronised the stream.  A handle must not be used from two streams at once.
 * The one exception to "only enqueues": the handle's internal buffers are grow-only, and a call that has to
 * GROW one (a larger P in fire_params_upload, a larger S in fire_simulate_batch / fire_fitness /
 * fire_generation_host than any call before on this handle) first waits for `stream` (cudaStreamSynchronize),
 * because work already enqueued may still use the old buffer.  Repeating a call with sizes the handle has
 * already seen never synchronises.
 * Limits (violations return FIRE_EINVAL before anything is enqueued; the handle stays usable):
 *   1 <= W, H <= 8192;  P * W * H < 2^32 (threshold sectors are addressed by 32-bit indices: 137 GB of table);
 *   S * ceil(W/8) * ceil(H/8) < 2^31 per fire_simulate_batch call (state planes are addressed by 32-bit tile
 *   offsets; 2^30 when the two-plane kernel family is selected): 131,071 simulations on a 1024 x 1024 lattice,
 *   8,191 on 4096 x 4096 -- split larger batches over several calls, using sim_ids to keep the random streams.
 * Errors: 0 on success, a negative FIRE_E* code otherwise.  The library never throws, aborts or
 * prints.  Faults only the device can see (ignition outside the lattice or on a non-burnable
 * cell, sim_param outside [0, P)) are not errors: that simulation burns nothing, steps = 0 (R-12).
 * There is no CPU fallback: without a CUDA device every call returns FIRE_ECUDA.
 */
#ifndef FIRE_H
#define FIRE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FIRE_OK       0
#define FIRE_EINVAL  (-1)   /* null pointer, non-positive size, R < 2, a limit listed above exceeded */
#define FIRE_ENOMEM  (-2)   /* device allocation failed */
#define FIRE_ESTATE  (-3)   /* simulate before fire_params_upload, p out of range in download */
#define FIRE_ECUDA   (-4)   /* a CUDA call failed (sticky), or no CUDA device */
#define FIRE_ELIMIT  (-5)   /* fire_fitness_static: S beyond FIRE_FITNESS_STATIC_MAX_SIMS */

#define FIRE_METRIC_DELTA    0   /* Eq. 2: (#(A u A*) - #(A n A*)) / #A, 0 = perfect overlap */
#define FIRE_METRIC_JACCARD  1   /* #(A n A*) / #(A u A*) */

typedef struct fire_landscape fire_landscape;   /* opaque; one handle = one device */

/* Landscape ingest.  Derives and keeps, per cell, the
 * covariates of Eq. 1 in double precision (I_f, psi, omega_d, sigma_d) and the burnable bitmap.
 * veg u8[H][W]; slope, aspect, wind f32[H][W].  Precondition (R-20): finite values, 0 <= slope < pi/2.
 * The rasters may be freed once `stream` has passed this point.  1 <= W, H <= 8192. */
int fire_landscape_create(fire_landscape** out, const uint8_t* veg, const float* slope,
                          const float* aspect, const float* wind, int32_t W, int32_t H, void* stream);

/* Frees everything the handle owns.  Synchronises the device. */
int fire_landscape_destroy(fire_landscape* L);

/* Contagion-threshold precompute (a2; Eq. 1).  beta f32[P][5] = (beta_0 .. beta_4).
 * For every parameter vector p, burnable cell c and direction d:
 *   T[p][c][d] = min(rint(2^32 / (1 + exp(-(b0 + b1 I_f + b2 psi + b3 omega_d + b4 sigma_d)))), 2^32 - 1)
 * x in IEEE double in the written order, separate multiplies and adds (no FMA contraction); the logistic and the rounding in
 * double precision to within ONE count of the correctly rounded value (4e-8 of the entries differ by one count from a libm
 * evaluation, none by more: tests/test_gpu_parity.py); T = 0 on non-burnable cells.  A trial succeeds iff
 * rnd < T or T == 2^32 - 1 (R-11).  Replaces any previous table; allocates P*W*H*32 bytes. */
int fire_params_upload(fire_landscape* L, const float* beta, int32_t P, void* stream);

/* Batch of S independent simulations (a3-a6).
 * ignitions i32[S][2] = (x, y); sim_param i32[S] in [0, P); seeds u64[S];
 * sim_ids i32[S] or NULL: the `sim` field of the random-number key (NULL = 0..S-1), so that a
 * shard of a larger batch reproduces the same fires.  max_steps: 0 = until extinction.
 * The random word of trial (seed, sim, step t, target cell c = y*W + x, direction d) is word d & 3 of
 * Philox4x32-10(counter = (c, t, sim, d >> 2), key = (seed & 0xffffffff, seed >> 32)) (R-3).
 * out_burned u32[S][H][ceil(W/32)] final burnt map (every word is written);
 * out_steps u32[S] or NULL: number of CA steps until the fire stopped;
 * out_trials u64[S] or NULL: number of (target cell, direction) Bernoulli trials performed. */
int fire_simulate_batch(fire_landscape* L, const int32_t* ignitions, const int32_t* sim_param,
                        const uint64_t* seeds, const int32_t* sim_ids, int32_t S, uint32_t max_steps,
                        uint32_t* out_burned, uint32_t* out_steps, uint64_t* out_trials, void* stream);

/* Variant of the uphill test (PAPER.md:87 read literally): with an elevation raster f32[H][W] the slope term of
 * direction d applies iff slope > 0 and elevation[target] > elevation[source] (strictly), source = target - offset(d), instead
 * of the default local-plane test on the aspect (R-7).  Invalidates the threshold table: call fire_params_upload again. */
int fire_landscape_set_elevation(fire_landscape* L, const float* elevation, void* stream);

/* Per-class vegetation term: Eq. 1 has one vegetation term, beta_1 I_f with I_f = 1 for forest.
 * class_if_host f32[n_classes] (HOST memory, read before the call returns) gives every vegetation class v its own I_f
 * (classes >= n_classes get 0; class 0 cannot burn anyway); n_classes = 0 restores the paper's indicator (class 1 only).
 * Invalidates the threshold table: call fire_params_upload again. */
int fire_landscape_set_class_indicator(fire_landscape* L, const float* class_if_host, int32_t n_classes, void* stream);

/* Hazard map: out_count u32[H][W] = number of the S maps burned u32[S][H][ceil(W/32)] in which the
 * cell is burnt (divide by S for the burn probability of the cell over replicates). */
int fire_burn_count(fire_landscape* L, const uint32_t* burned, int32_t S, uint32_t* out_count, void* stream);

/* Time-of-burn output ("fire evolution in time"): out_time i32[S][H][W] (device; the caller's, sized
 * for the largest batch it will pass) receives, in every later fire_simulate_batch on this handle, the step at which each cell
 * ignited: 0 for the ignition cell, t + 1 for a cell ignited by the transition t -> t + 1, -1 for a cell that never burnt.
 * NULL switches the output off (default). */
int fire_set_time_output(fire_landscape* L, int32_t* out_time);

/* Fused fitness counts (Eq. 2): every later fire_simulate_batch on this handle also writes
 * out_counts u32[S][2] = (I, N*) against reference u32[H][ceil(W/32)], the values fire_fitness's out_counts would hold, while
 * it converts the state planes to burnt maps (one pass over the maps saved; out_burned is still written).  Both arrays are the
 * caller's (device), out_counts sized for the largest batch it will pass; both NULL switch the output off (default); one NULL and
 * one not is FIRE_EINVAL. */
int fire_set_fused_counts(fire_landscape* L, const uint32_t* reference, uint32_t* out_counts);

/* Fuel-dependent burn-out time ("a burnt cell gets inactive after a given time that depends on the
 * vegetation type", :145, :68, :273; reading R-21).  burn_time_host u8[n_classes] (HOST memory, read before the call
 * returns): steps a cell of vegetation class v stays ACTIVE once ignited, 1..8 (0 reads as 1; classes >= n_classes burn one
 * step).  An active cell is a source for each of its susceptible neighbours at EVERY step it is active: one trial
 * rnd(seed, sim, t, target, d) per step and pair, keyed as in fire_simulate_batch (the key holds the step, so a repeated pair
 * draws a fresh word); the run ends when no cell is active.  All ones (or n_classes = 0) is the paper's setting and the default.
 * Applies to every later fire_simulate_batch / fire_generation_host on this handle. */
int fire_set_burn_time(fire_landscape* L, const uint8_t* burn_time_host, int32_t n_classes, void* stream);

/* Fitness reduction (a7; Eq. 2).  reference u32[H][ceil(W/32)] = A, burned
 * u32[S][H][ceil(W/32)] = A*.  out_counts u32[S][2] or NULL = (I, N*) with I = #(A n A*), N* = #A*;
 * out_score f32[S]: metric 0 = (float)(N + N* - 2I) / (float)N, metric 1 = (float)I / (float)(N + N* - I),
 * N = #A; one IEEE divide (N = 0 gives inf/NaN, not an error).  out_ref_area u32[1] or NULL = N. */
int fire_fitness(fire_landscape* L, const uint32_t* reference, const uint32_t* burned, int32_t S,
                 int32_t metric, float* out_score, uint32_t* out_counts, uint32_t* out_ref_area, void* stream);

/* Fitness reduction that ALLOCATES NOTHING: for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it).  Same result as fire_fitness (Eq. 2; scores bit for bit) without a handle: reference
 * u32[H][ceil(W/32)], burned u32[S][H][ceil(W/32)], out_score f32[S], out_ref_area u32[1] or NULL, all DEVICE pointers on the
 * CURRENT device; the work is enqueued on `stream`.  The per-simulation counts (I, N*) and #A live in a static device array inside
 * the library, sized for S <= FIRE_FITNESS_STATIC_MAX_SIMS (128.25 KiB, held by every GPU that loads the library until the process
 * exits); a larger S returns FIRE_ELIMIT before anything is enqueued (split the batch: the score of a simulation does not depend
 * on the others).  The call makes no cudaMalloc / cudaFree and calls no allocating library routine.  EVERY call on a device
 * shares that one array (it is cleared at the start of each call): calls that overlap on the GPU -- two streams, or two host
 * threads -- race on it and give wrong scores; calls on one stream, or otherwise ordered, are safe. */
#define FIRE_FITNESS_STATIC_MAX_SIMS 16384
int fire_fitness_static(const uint32_t* reference, const uint32_t* burned, int32_t W, int32_t H, int32_t S,
                        int32_t metric, float* out_score, uint32_t* out_ref_area, void* stream);

/* Per-candidate statistics over R replicates (a8; BASELINE config 4).
 * counts u32[G*R][2] = (I, N*), candidate-major; x = ref_area + N* - 2I.
 * out_sums u64[G][2] = (sum x, sum x^2); out_mean_var f64[G][2] = mean and sample variance (R-16)
 * of delta = x / ref_area:  mean = sum x / (R N),  var = (R sum x^2 - (sum x)^2) / (R (R-1)) / N^2. */
int fire_fitness_group_stats(const uint32_t* counts, uint32_t ref_area, int32_t G, int32_t R,
                             uint64_t* out_sums, double* out_mean_var, void* stream);

/* Test hook: copies the threshold table of parameter vector p to out u32[H][W][8] (device). */
int fire_thresholds_download(fire_landscape* L, int32_t p, uint32_t* out, void* stream);

/* One GA generation with HOST buffers (end-to-end path): copies beta, ignitions, sim_param, seeds
 * (and sim_ids if not NULL) and the reference bitmap to the device, runs fire_params_upload,
 * fire_simulate_batch and fire_fitness on `stream`, copies scores (and counts / steps if not NULL)
 * back and SYNCHRONISES the stream.  Host arrays should be page-locked for full copy bandwidth.
 * The burnt maps stay on the device: *out_burned_dev (if not NULL) receives a device pointer to
 * u32[S][H][ceil(W/32)] owned by the handle, valid until the next call on this handle. */
int fire_generation_host(fire_landscape* L, const float* beta_host, int32_t P,
                         const int32_t* ignitions_host, const int32_t* sim_param_host,
                         const uint64_t* seeds_host, const int32_t* sim_ids_host, int32_t S,
                         uint32_t max_steps, const uint32_t* reference_host, int32_t metric,
                         float* out_score_host, uint32_t* out_counts_host, uint32_t* out_steps_host,
                         uint32_t** out_burned_dev, void* stream);

/* Number of kernel launches the library has enqueued on this handle so far (bench.py's gpu_launches). */
int64_t fire_launch_count(const fire_landscape* L);

/* Device timing of the propagation kernel alone (bench.py's roofline): while enabled, every
 * fire_simulate_batch brackets its propagation kernel with a pair of CUDA events on `stream` (at most 64
 * pairs are kept between reads).  fire_profile_read waits for the recorded events, writes their elapsed
 * milliseconds, oldest first, to ms_host (HOST memory, max_entries floats), sets *n_out and forgets them. */
int fire_set_profiling(fire_landscape* L, int32_t enabled);
int fire_profile_read(fire_landscape* L, float* ms_host, int32_t max_entries, int32_t* n_out);

/* Tuning knob (tests use it to show results do not depend on launch geometry, pin P-9):
 * threads per CTA of the propagation kernel (multiple of 32, 32..1024; 0 = default) and CTAs per SM
 * (0..32; 0 = default). */
int fire_set_launch_geometry(fire_landscape* L, int32_t threads_per_cta, int32_t ctas_per_sm);

/* Test hook (pin P-9): capacity, in cells, of the per-CTA frontier list of the propagation kernel:
 * the first `shared_entries` live in shared memory, the rest up to `total_entries` in a global spill
 * area; a simulation whose burning front ever exceeds `total_entries` is redone by the list-free
 * rescue kernel.  Results never depend on these values.  0 = default. */
int fire_set_list_capacity(fire_landscape* L, int32_t shared_entries, int32_t total_entries);

/* Tuning knob / test hook (pin P-9): order in which the simulations of a batch are handed to the resident
 * CTAs.  0 = default: largest expected fires first (by the mean contagion probability of their parameter
 * vector, a by-product of fire_params_upload); 1 = batch order.  Results never depend on it. */
int fire_set_schedule(fire_landscape* L, int32_t mode);

/* Test hook (pin P-9): which propagation kernel fire_simulate_batch launches.  0 = automatic (by batch size),
 * 1 = two-phase kernel (one CTA per simulation, one state plane, two block barriers per step), 2 = asynchronous-warp
 * kernel (one CTA per simulation, two state planes, one block barrier per step), 3 / 4 = the asynchronous-warp kernel as
 * thread-block clusters of 2 / 4 CTAs per simulation (one cluster barrier per step; frontier lists read through
 * distributed shared memory).  Results never depend on it. */
int fire_set_kernel(fire_landscape* L, int32_t family);

const char* fire_error_string(int code);

#ifdef __cplusplus
}
#endif
#endif /* FIRE_H */
