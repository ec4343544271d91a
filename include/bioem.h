/*
 * bioem.h -- C ABI of the B200-native BioEM hot path (arXiv:1609.06634).
 *
 * The library scores every experimental particle image against every calculated image
 * (model x orientation x CTF parameter set) over all in-plane centre displacements and
 * accumulates the marginal log-posterior per (image, model), with the maximising grid
 * parameters (paper sections 2-3; citations "P:<line>" are lines of PAPER.md, "R<k>" the
 * readings of DESIGN.md section 3).
 *
 * Conventions
 *   - every call returns an int: 0 = ok, negative = one of the BIOEM_E* codes; nothing throws or
 *     aborts across the ABI; bioem_last_error(ctx) returns a ctx-owned, NUL-terminated message.
 *   - INPUTS ARE COPIED: the caller keeps ownership of every pointer passed in and may free it
 *     after the call returns.  OUTPUTS ARE CALLER-ALLOCATED host arrays.
 *   - pointers are HOST pointers unless the argument list has an `is_device` flag set to 1, in
 *     which case they are CUDA device pointers on the context's device (e.g. torch data_ptr()).
 *   - all device work is enqueued on the cudaStream_t given at creation (NULL = default stream,
 *     e.g. torch.cuda.current_stream().cuda_stream); bioem_run returns after enqueueing and
 *     bioem_get_* synchronise that stream.
 *   - images are row-major [k][j] = [y][x], x fastest (R11); pixel (N/2, N/2) is the model
 *     origin.
 *   - there is NO CPU fallback: without a CUDA device bioem_create fails with BIOEM_ECUDA.
 */
#ifndef BIOEM_H
#define BIOEM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BIOEM_OK            0
#define BIOEM_EBADARG      (-1)   /* NULL / out-of-range argument                         */
#define BIOEM_EBADSTATE    (-2)   /* call order: something required has not been set yet   */
#define BIOEM_EOOM         (-3)   /* device allocation failed                              */
#define BIOEM_ECUDA        (-4)   /* CUDA runtime error (message in bioem_last_error)      */
#define BIOEM_EUNSUPPORTED (-5)   /* image size / grid size the kernels are not built for  */

#define BIOEM_TOPK 8              /* candidates per (image, model) re-scored in FP64 (a7)  */

typedef struct bioem_ctx bioem_ctx;

/* Create a context on CUDA device `device`; `cuda_stream` is a cudaStream_t (may be NULL). */
int bioem_create(bioem_ctx **out, int device, void *cuda_stream);
int bioem_destroy(bioem_ctx *ctx);
const char *bioem_last_error(const bioem_ctx *ctx);

/* Square images of n_pix x n_pix pixels of pixel_size_A Angstrom.  Supported n_pix:
 * 64, 96, 128, 160, 170, 192, 224, 256 (BIOEM_EUNSUPPORTED otherwise).  64 / 128 (max_shift <= 16) and 224 (max_shift <= 31) run
 * the tuned kernels; the other sizes -- 170 is the GroEL box of the paper's Table 1, 2 x 5 x 17 -- run the generic
 * two-step kernel, whose second step is a direct sum over n_pix / N1 residues (N1 = 32, or 2 for 170): same results, parity
 * tested, not tuned.  Clears images, models stay. */
int bioem_set_image_geometry(bioem_ctx *ctx, int n_pix, float pixel_size_A);

/* Models.  Atoms: uniform-density spheres, centre xyz_A [n][3], radius_A [n], total
 * weight [n] (R10); projected by Eq. 1 with 4x4 mid-point sub-sampling per pixel.
 * Density: cube of n_vox^3 voxels rho[z][y][x] of voxel_A Angstrom, origin at voxel n_vox/2,
 * projected as a trilinear central section of its 3-D DFT (R21); requires n_vox == n_pix and
 * voxel_A == pixel_size_A.  *model_id receives 0, 1, ... in order of addition. */
int bioem_clear_models(bioem_ctx *ctx);
int bioem_add_model_atoms(bioem_ctx *ctx, int n_atoms, const float *xyz_A, const float *radius_A,
                          const float *weight, int *model_id);
int bioem_add_model_density(bioem_ctx *ctx, int n_vox, float voxel_A, const float *rho, int *model_id);

/* Orientation grid: n unit quaternions (w,x,y,z), ACTIVE rotation r' = R(q) r,
 * projection along z' (R12).  log_prior [n] or NULL = uniform (-log n) (R7). */
int bioem_set_orientations_quat(bioem_ctx *ctx, int n, const float *q_wxyz, const float *log_prior);

/* CTF / envelope grid: CTF(s|a,A) Env(s|b), s = 2 pi x spatial frequency, a and b in A^2,
 * 0 <= A <= 1.  log_prior [n] or NULL = uniform. */
int bioem_set_ctf_grid(bioem_ctx *ctx, int n, const float *a_A2, const float *A, const float *b_A2,
                       const float *log_prior);

/* Helper (R8, R9): defocus [um], B-factor [A^2], voltage [kV] -> a = lambda_e dz / (2 pi), b = B / (8 pi^2). */
int bioem_ctf_from_defocus(float defocus_um, float bfactor_A2, float kV, float *a_A2, float *b_A2);

/* Centre displacements (Eq. 7): all integer (dx,dy) with |dx|,|dy| <= max_shift_px, circular
 * (R5, R6); 2*max_shift_px + 1 <= n_pix. */
int bioem_set_shift_range(bioem_ctx *ctx, int max_shift_px);

/* Replace the image stack: n_img images [n][N][N] float32 (host, or device if is_device). Runs the
 * observed-image preprocessing (a0: mean removal, spectra, C_o / C_oo sums).
 * BIOEM_EBADARG if an image is constant or not finite (C_oo - C_o^2/n is not > 0: the marginal over
 * N, mu, lambda of Eq. 8 does not exist for it); the stack is then left empty. */
int bioem_push_images(bioem_ctx *ctx, int n_img, const float *pixels, int is_device);

/* The hot path: all models x orientations x CTFs x shifts against all images (Eq. 9 on the grid,
 * P:126; Eqs. 11-12; closed-form marginal over N, mu, lambda).  Requires geometry,
 * >= 1 model, orientations, CTFs, a shift range and images (else BIOEM_EBADSTATE). */
int bioem_run(bioem_ctx *ctx);
/* Calculated-image cache.  The outputs of a1-a3 (projection spectra, CTF tables, T_c; "calculated once per
 * orientation and CTF set") depend on the models, grids and shift range only, so a bioem_run that follows another one with
 * nothing but the image stack replaced reuses them: this is how an image stack larger than device memory is scored in
 * subsets -- bioem_push_images(subset) + bioem_run + bioem_get_* per subset, results concatenated; images are
 * independent.  Every bioem_set_* / bioem_add_model_* / bioem_clear_models call drops the cache;
 * bioem_invalidate_precompute drops it explicitly (bench.py does, so that every timed step runs all of a0-a7). */
int bioem_invalidate_precompute(bioem_ctx *ctx);
/* Domain of validity.  bioem_run only enqueues; a calculated image that is empty or not finite (T_c = n C_cc - C_c^2 is
 * not > 0: the model projects to nothing inside the box) is detected on the device and reported as BIOEM_EBADARG by the first
 * bioem_get_* call.  The hot loop is FP32 on operands correctly rounded from FP64; the BIOEM_TOPK largest terms per
 * (image, model) are re-scored in FP64 and the argmax is taken among them.  The 1e-3 absolute accuracy of log_posterior
 * therefore holds when the terms outside the BIOEM_TOPK largest carry a small share of the sum, or carry a small FP32 error:
 * |delta log P| <~ (share of the sum outside the top BIOEM_TOPK) x n rho^2 / (1 - rho^2) x 1e-6, rho^2 = the squared
 * correlation of the best match.  rho^2 -> 1 (a noiseless planted image, R14) is clamped at
 * 1 - rho^2 >= 2^-24 in the FP32 loop and 1e-300 in the re-scoring: finite results, parity with the oracle not defined. */

/* Results of the last bioem_run, each [n_img][n_model] (image-major):
 *   log_posterior = log sum_theta w(theta) P_m,omega(theta), w uniform unless priors were given (R7);
 *   best = grid parameters of the largest term (R15: exact ties -> lowest flat index) and its value. */
int bioem_get_log_posterior(bioem_ctx *ctx, double *out);
int bioem_get_best(bioem_ctx *ctx, int32_t *orient_idx, int32_t *ctf_idx, int32_t *dx, int32_t *dy,
                   double *best_log_p);

/* Posterior as a function of the orientation (the paper's third output):
 *   out[img][model][o] = log sum_{ctf, d} w(o, ctf, d) P_m,omega(o, ctf, d)      (log-sum-exp over o gives log_posterior).
 * Off by default.  When enabled before bioem_run, the work items stay chunked (several orientations per thread block): each warp
 * closes its running sums at the end of every orientation into a shared-memory table, and the work item's epilogue combines
 * warps -> orientation -> work item in fixed order and writes 8 bytes per (image, model, orientation).  Measured 1.04x / 1.11x /
 * 1.06x the run time on Small / Paper-scale / Ensemble (the kernels are separate template instantiations: a run with the option
 * off executes the same code as before).  The table has 32 rows, so the chunk is capped at 32.  The terms that the FP64
 * re-scoring replaces (the 8 largest per image and model) are replaced here too; the others keep FP32 accuracy
 * (R24).  enable: 0 | 1.  get_: caller-allocated [n_img][n_model][n_orient] doubles; BIOEM_EBADSTATE if the
 * last run was made without the option.  On a context that holds an orientation slice (bioem_set_orientation_slice) the output
 * is that rank's part, [n_img][n_model][o_end - o_begin]: the values are those of the undivided run, bit for bit, and the ranks'
 * parts concatenated along the last axis are its output (shard.run_orientation_sharded gathers them). */
int bioem_set_orientation_posterior(bioem_ctx *ctx, int enable);
int bioem_get_orientation_log_posterior(bioem_ctx *ctx, double *out);

/* Ensemble posterior, Eq. 10: log P(M|Omega) = sum_omega log sum_m w_m P_m,omega (up to the constant
 * the paper drops), from the log-posteriors of the last bioem_run.  weights: host, [n_model], w_m >= 0 (the paper normalises
 * sum_m w_m = 1; not enforced), NULL = uniform 1/n_model.  out_total: one double.  out_per_image: [n_img] doubles (the
 * inner log-sums) or NULL.  FP64, fixed summation order. */
int bioem_get_ensemble_log_posterior(bioem_ctx *ctx, const double *weights, double *out_total, double *out_per_image);

/* Synthetic map (paper section 3.8: "print the synthetic map corresponding to a specific parameter set theta"): the calculated
 * image I_cal of Eq. 7 for theta = (orient, ctf, d = (dx, dy), N, mu) of `model`,
 *   out[k][j] = N * I1(k + dy, j + dx) - mu        (row-major [N][N] floats, caller-allocated; I1 of Eqs. 1-5 in FP64),
 * displaced the way the run scores it: wrapped around the box (displacement variant 0, R5) or cut off at the borders (variant 1,
 * R25); |dx|, |dy| < n_pix, not limited to the shift range.  fit_to_image = NULL: N = 1, mu = 0.  Otherwise a host image
 * [N][N] (e.g. the particle whose bioem_get_best parameters are passed): N and mu are the values that maximise the likelihood of
 * Eq. 8 for that image (least squares; a constant calculated image gives N = 0), returned in out_norm_offset[0..1] if not NULL.
 * Needs a completed bioem_run on this context (its spectra are reused; `orient` must lie in the context's orientation slice).
 * Synchronises the stream. */
int bioem_get_synthetic_map(bioem_ctx *ctx, int model, int orient, int ctf, int dx, int dy, const float *fit_to_image, float *out,
                            double *out_norm_offset);

/* Work decomposition of bioem_run: one work item (thread block) scores one image against `n_orient_per_item` consecutive
 * orientations x all CTFs x all shifts of one model (the image-stationary loop order of DESIGN.md section 8; P:199-203 has
 * the loops the other way round).  0 = automatic: >= 32 work items per SM, at most 32 orientations per item.  The value
 * fixes the order in which the FP32 partial sums are combined, so results are bit-identical between two runs only if it is
 * the same; ranks that shard one image stack set it explicitly.  Capped at 32 while the per-orientation
 * posterior is enabled (1 with the two-CTA cluster kernel of bioem_debug_set_kernel, which has no per-orientation table). */
int bioem_set_orientation_chunk(bioem_ctx *ctx, int n_orient_per_item);

/* Displacement variant (paper section 3.3).  0 (default): Fourier space -- one output-pruned inverse transform
 * per (image, calculated image), displacements wrap around the borders (R5); the hot path.  1: real space -- "the cross-correlation
 * is simply calculated for different displacements", the displaced calculated image is CROPPED at the borders instead of
 * wrapping: I_d(r) = I1(r + d) where r + d lies inside the box, 0 elsewhere, and Eq. 8 is applied to (I_obs, I_d) over
 * all n pixels, so C_co, C_c and C_cc depend on d (reading R25 in DESIGN.md).  The paper's route for very few displacements
 * (Fig. 2): (2D+1)^2 n multiply-adds per pair, FP64 throughout (no re-scoring step), deterministic.  Call BEFORE
 * bioem_push_images (the real-space variant keeps the mean-free images in real space); BIOEM_EBADSTATE at bioem_run otherwise.
 * The per-orientation posterior is available with it (running sums per (image, model, orientation), FP64); orientation slices are
 * not (BIOEM_EUNSUPPORTED). */
int bioem_set_displacement_variant(bioem_ctx *ctx, int variant);

/* ---- orientation sharding: the paper's MPI axis ("MPI over orientations"; no communication but one gather) ----
 * Every rank holds all models, grids and images and scores a contiguous SLICE [o_begin, o_end) of the orientation grid; indices,
 * priors and the uniform weight -log(n_orient) still refer to the full grid.  bioem_run is the four phases below on one
 * context; sharded, the ranks exchange two small buffers between them (paper_1609_06634_b200/shard.py does it with
 * torch.distributed):
 *   bioem_run_partial          a1-a6 on the slice: one partial {m, s, BIOEM_TOPK candidates} per (image, model, chunk of orientations)
 *   bioem_export_partials      -> all_gather over ranks (rank order = grid order)
 *   bioem_merge_partials       the fixed-order combine of ALL ranks' partials, on every rank (a6)
 *   bioem_rescore_local        FP64 values of the merged candidates whose orientation this rank holds, exactly 0.0 for the others (a7)
 *   bioem_export_rescore       -> all_reduce(SUM) over ranks -> bioem_import_rescore
 *   bioem_finish               corrected log-sum-exp, argmax, constants (a7): every rank then holds the full results.
 * The results are bit-identical to one GPU scoring the whole grid with the same bioem_set_orientation_chunk value: the chunk
 * partials are the same numbers and are combined in the same order.  Requirements (BIOEM_EBADSTATE / BIOEM_EBADARG otherwise):
 * an explicit orientation chunk, the same on all ranks; o_begin a multiple of it; the per-orientation posterior disabled.
 * set_orientation_slice(ctx, 0, -1) clears the slice.  Buffers: caller-allocated, host or device (is_device). */
int bioem_set_orientation_slice(bioem_ctx *ctx, int o_begin, int o_end);
int bioem_run_partial(bioem_ctx *ctx);
/* size of this context's partials: n_bytes of the blob bioem_export_partials writes, n_chunks = chunks per model in it */
int bioem_get_partials_size(bioem_ctx *ctx, int64_t *n_bytes, int32_t *n_chunks);
int bioem_export_partials(bioem_ctx *ctx, void *dst, int is_device);
/* blobs: n_blobs blobs, blob r at blobs + r * stride_bytes with chunks_of_blob[r] (host array) chunks per model, in grid order;
 * blobs = NULL merges this context's own partials (what bioem_run does). */
int bioem_merge_partials(bioem_ctx *ctx, int n_blobs, const void *blobs, int64_t stride_bytes, const int32_t *chunks_of_blob,
                         int is_device);
int bioem_rescore_local(bioem_ctx *ctx);
/* [n_img][n_model][BIOEM_TOPK] doubles */
int bioem_export_rescore(bioem_ctx *ctx, double *dst, int is_device);
int bioem_import_rescore(bioem_ctx *ctx, const double *src, int is_device);
int bioem_finish(bioem_ctx *ctx);

/* ---- test / debug entry points (not on the measured path) ---- */
/* Which fused kernel bioem_run may use: 0 automatic (packed register-resident kernel for n_pix 64 / 128 with max_shift <= 16,
 * tensor-memory kernel for n_pix 224 with max_shift <= 31, generic kernel otherwise), 1 generic kernel always, 3 the
 * two-CTA-cluster kernel of round 1 (n_pix 224, max_shift <= 31; kept as a cross-check of the tensor-memory kernel). */
int bioem_debug_set_kernel(bioem_ctx *ctx, int which);
/* The plan of the last bioem_run: kernel (1 generic, 2 packed, 3 cluster, 4 tensor memory, 6 real-space variant) and orientations
 * per work item. */
int bioem_get_run_plan(bioem_ctx *ctx, int *kernel, int *n_orient_per_item);
/* real-space calculated image I1 of (model, orient, ctf) [N][N] ("synthetic map"). */
int bioem_debug_calc_image(bioem_ctx *ctx, int model, int orient, int ctf, float *out_real);
/* per-shift terms log P + log w of one (image, calc image) pair, [dy+D][dx+D]:
 * _map: as the FP32 fused kernel computes them (a4+a5); _map_f64: as the FP64 re-scoring kernel (a7) does. */
int bioem_debug_shift_map(bioem_ctx *ctx, int img, int model, int orient, int ctf, double *out);
int bioem_debug_shift_map_f64(bioem_ctx *ctx, int img, int model, int orient, int ctf, double *out);
/* FP32-only result of the last run (before FP64 re-scoring), [n_img][n_model]. */
int bioem_debug_log_posterior_f32(bioem_ctx *ctx, double *out);
/* CUDA-event times of the last bioem_run [ms]: whole run, fused kernel only; number of kernel launches. */
int bioem_get_timing(bioem_ctx *ctx, double *ms_total, double *ms_fused_kernel);
int bioem_get_launch_count(bioem_ctx *ctx, int64_t *n_launches, int64_t *n_fused_launches);
/* FP32 FMA rate of this device measured with a register-resident FFMA loop [TFLOP/s] (context for bench.py's "alu" roofline,
 * whose denominator is the formula peak) and the device's MAXIMUM SM clock [MHz] (cudaDevAttrClockRate, not a clock sampled
 * while the loop ran: bench.py samples nvidia-smi for that). */
int bioem_measure_fp32_peak(bioem_ctx *ctx, double *tflops, double *sm_mhz);

/* Allocation-free entry point, for callers that may not call cudaMalloc (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it): Eq. 10 as bioem_get_ensemble_log_posterior computes it, but context-free, on
 * caller-supplied DEVICE arrays, enqueued on `cuda_stream` of CUDA device `device` without synchronising, and calling no
 * cudaMalloc / cudaFree or allocating library routine.  Its work array (the per-image inner log-sums) is a file-scope device
 * array of BIOEM_NOALLOC_MAX_IMG doubles (512 KiB) that every GPU loading the library holds until the process exits.
 *   log_p          device, [n_img][n_model] doubles: log P_m,omega, e.g. a device copy of bioem_get_log_posterior's output
 *   weights        device, [n_model] doubles, w_m >= 0 (a negative weight gives NaN outputs; nothing is read back to
 *                  check), or NULL = uniform 1 / n_model
 *   out_total      device, one double;  out_per_image  device, [n_img] doubles, or NULL
 * n_img > BIOEM_NOALLOC_MAX_IMG or n_model > BIOEM_NOALLOC_MAX_MODEL: BIOEM_EUNSUPPORTED, nothing enqueued (use the
 * allocating call).  Every call on a device shares the one work array: calls whose kernels may overlap on the GPU
 * (different streams, several host threads) RACE -- keep them on one stream or order them with events.  Nothing in the
 * array has to be cleared between calls (each call writes the entries it reads).  Same summation order as the allocating
 * call, so the two agree to rounding of log().  bioem_noalloc_prepare(device) takes the array's device address ahead of
 * time (otherwise the first call on a device does, which may load the module: do it before a capture begins).  These three
 * calls report errors through bioem_noalloc_last_error() (per host thread), not through a context. */
#define BIOEM_NOALLOC_MAX_IMG   65536
#define BIOEM_NOALLOC_MAX_MODEL 1024
int bioem_noalloc_prepare(int device);
int bioem_ensemble_log_posterior_noalloc(int device, void *cuda_stream, int n_img, int n_model, const double *log_p, const double *weights,
                                         double *out_total, double *out_per_image);
const char *bioem_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* BIOEM_H */
