/*
 * ulm_rca.h -- C-ABI boundary of the B200 (sm_100a) RCA projection beamformer.
 *
 * The library computes the Stage-1 "2D beamforming step" of the projection-based 3-D ULM pipeline of
 * arxiv 2511.21647 (Section II.A.1; acquisition geometry PAPER.md:113-117): row-column
 * array (RCA) delay-and-sum beamforming of multi-angle plane-wave channel data straight into per-frame
 * 2-D images -- the x-z image from the row-transmit events (received on the columns) and the y-z image
 * from the column-transmit events (received on the rows), "x-z plane for RC and y-z plane for CR"
 * (Fig. 1d) -- coherently compounded over the steering angles, with no 3-D volume written
 * to memory.  The paper prints no formula for this step; the exact definition implemented here is
 * DESIGN.md "Definition" (= SURVEY.md section 8(c)):
 *
 *   step 0 (RF input)  x[n] = rf[n] exp(-j 2 pi fc t_n), t_n = t_start + n/fs;
 *                      iq[n] = 2 sum_{m=-L..L} h[m] x[n-m]  (x = 0 outside the record),
 *                      h[m] ~ sinc(2 fc m/fs) (0.54 + 0.46 cos(pi m/L)), sum h = 1, L = (demod_taps-1)/2
 *   step 1 (x-z image) for pixel (x, z), row-tx angle th_k, column j at x_j:
 *                      tau = t0_k + (z cos th_k + y_ref sin th_k)/c + sqrt((x - x_j)^2 + z^2)/c
 *                      u = (tau - t_start) fs, n = floor(u), a = u - n   (term = 0 unless 0 <= n <= Ns-2)
 *                      P_xz(x, z) = sum_k sum_j w_j(x, z) ((1-a) iq_kj[n] + a iq_kj[n+1]) exp(+j 2 pi fc tau)
 *                      w_j = elem_window[j] * [f_number == 0 or |x - x_j| <= z / (2 f_number)]
 *   step 2 (y-z image) the same with x <-> y, columns <-> rows, x_ref for y_ref, grid_yz
 *   step 3             compound == 0: the k-sum is not taken (the paper's per-transmission slices S_k)
 *   step 4 (volume)    the same DAS at every voxel (x, y, z) for all events, V = V_RC + V_CR
 *                      (the "conventional 3D processing" the paper compares against)
 *
 * All pointers named d_* are DEVICE pointers owned by the caller; all other pointers are HOST pointers
 * that are only read during the call (the caller may free them at once).  No call throws, exits or
 * prints; failures are a status code plus ulm_rca_last_error().  There is no CPU fallback: without a
 * CUDA device every call that needs one fails with ULM_RCA_ECUDA.
 */
#ifndef ULM_RCA_H
#define ULM_RCA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ulm_rca_plan ulm_rca_plan; /* opaque, owned by the library */

typedef enum {
    ULM_RCA_OK = 0,
    ULM_RCA_EINVAL = 1,       /* NULL / non-finite / non-positive argument, inconsistent sizes        */
    ULM_RCA_ENOMEM = 2,       /* host or device allocation failed                                      */
    ULM_RCA_ECUDA = 3,        /* CUDA runtime error (text in ulm_rca_last_error)                       */
    ULM_RCA_EUNSUPPORTED = 4  /* valid request outside what the kernels cover                          */
} ulm_rca_status;

/* Array geometry (128 + 128 elements, pitch 0.214 mm).  Rows are long in x and indexed
 * along y, columns are long in y and indexed along x; element e of n sits at (e - (n-1)/2) * pitch. */
typedef struct {
    int32_t n_rows, n_cols;
    float pitch_m;
} ulm_rca_geometry;

/* One image grid: pixel (il, iz) is at lateral lat0_m + il*dlat_m (x for the x-z image, y for the y-z
 * image; dlat_m may be negative) and depth z0_m + iz*dz_m (z >= 0, dz_m > 0).  ref_m is the coordinate
 * of the reference slice along the transmit direction (y_ref for x-z, x_ref for y-z): the "central
 * slices along the transmit directions" of PAPER.md:31 (Fig. 1b) are ref_m = 0. */
typedef struct {
    int32_t n_lat;
    float lat0_m, dlat_m;
    int32_t n_ax;
    float z0_m, dz_m;
    float ref_m;
} ulm_rca_grid;

typedef struct {
    int32_t input_kind;         /* 0 = RF int16 real, 1 = IQ int16 interleaved (re, im)                */
    int32_t channels_per_event; /* n_rows + n_cols (rows first; only the aperture orthogonal to the
                                   transmitting one is read), or, when n_rows == n_cols, n_rows
                                   (orthogonal aperture only); 0 = n_rows + n_cols                     */
    int32_t n_samples;          /* samples per channel record (Ns >= 2)                                */
    float t_start_s;            /* time of sample 0                                                    */
    const float *t0_s;          /* HOST [n_row_tx + n_col_tx] per-event time offset, NULL = 0          */
    float f_number;             /* 0 = full aperture                                                   */
    const float *elem_window;   /* HOST [n_cols] weights of the column aperture (x-z image) followed by
                                   [n_rows] of the row aperture (y-z image); NULL = all ones           */
    int32_t demod_taps;         /* odd FIR length 2L+1; 0 = default 4*round(fs/fc)+1                   */
    int32_t compound;           /* 1 = sum over angles; 0 = one slice per event                        */
    int32_t max_frames;         /* largest n_frames a call will pass (sizes the plan's IQ scratch);
                                   0 = 32.  Larger calls are processed in batches of this size.        */
    int32_t build_volume;       /* 1 = also prepare ulm_rca_beamform_volume (needs equal axial grids)  */
    int32_t kernel;             /* 0 = auto (ring kernel where the shape fits); 1 = generic gather kernel;
                                   2 = shared-memory ring kernel or ULM_RCA_EUNSUPPORTED                 */
    int32_t precision;          /* format of the staged IQ scratch entries (mid = (a+b)/2, d = b-a of two
                                   neighbouring samples) and of the interpolation v = mid + a' d, a' in [-1/2, 1/2]:
                                   2 = full: fp32 throughout, 16 bytes per (sample, frame); nothing but fp32 rounding.
                                   3 = compact, 10 bytes: mid with 17 significant bits, d in fp16 (relative 2^-11,
                                       i.e. <= 2^-12 |d| per term), the weight a' carried as TWO fp16 terms
                                       (22 bits): holds max|err| <= 1e-4 max|image| on any int16 RF input, white
                                       noise included (the library's low-pass bounds |d| / |iq|).
                                   1 = compact-fast (opt-in): as 3 but a' rounded to ONE fp16 (another 2^-12 |d| per
                                       term, ~10 % faster DAS): within 1e-4 on band-limited echo data (|d| ~ 0.3 |iq|;
                                       1.1e-5 .. 1.4e-5 measured on the five BASELINE configs) but up to ~1.5e-4 on
                                       white noise -- select it only for echo-like input.
                                   0 = auto = 3 for RF input, 2 for IQ input (spectrum unknown).
                                   With the compact formats the low mantissa byte of a stored mid value is a byte of
                                   another frame of the same 4-frame chunk, so the result of frame f depends, by
                                   < 2^-16 relative per term (zero-mean), on which frames share its chunk.       */
    int32_t no_timing;          /* 1 = ulm_rca_beamform records no CUDA events around its kernels (and
                                   ulm_rca_plan_timing is unavailable); 0 = three cudaEventRecord per batch   */
    int32_t stage2_block;       /* P > 0: also prepare ulm_rca_stage2_project with sub-blocks of P x P voxel columns
                                   (P = 8; needs identical axial grids); 0 = not prepared           */
    int32_t clutter_frames;     /* n_t > 0: also prepare ulm_rca_clutter_filter for ensembles of up to n_t frames
                                   (32 .. 320; sizes the bf16 operand planes: ~8 bytes per slice value); 0 = not    */
    int32_t motion_frames;      /* > 0: also prepare ulm_rca_motion_estimate for calls of up to this many frames
                                   (scratch: ~20 MB per frame at the paper's slice sizes); 0 = not prepared        */
} ulm_rca_options;

/*
 * Build a plan: validates the arguments, derives the touched sample range, builds the per-angle
 * transmit-delay tables (fp64 on the host, split into integer + fraction), the demodulation filter and
 * mixer, tile windows and launch geometry, uploads them and allocates the IQ scratch.
 * Angles are in radians: row_tx_angles steer in the y-z plane, col_tx_angles in the x-z plane.
 * Event order in the channel data is row-tx angles (as given) then column-tx angles.
 * Either angle list may be empty (its image is then all zeros) but not both.
 * On success *out receives the plan; on failure *out is NULL.
 */
ulm_rca_status ulm_rca_plan_create(const ulm_rca_geometry *geometry,
                                   const float *row_tx_angles_rad, int32_t n_row_tx,
                                   const float *col_tx_angles_rad, int32_t n_col_tx,
                                   float c_mps, float fs_hz, float fc_hz,
                                   const ulm_rca_grid *grid_xz, const ulm_rca_grid *grid_yz,
                                   const ulm_rca_options *options, ulm_rca_plan **out);

/*
 * Beamform n_frames frames (steps 0-3).  With compound == 1, transmit events of an aperture whose transmit delay on
 * the reference slice is identical at every depth -- mirror angles +theta / -theta about a centred slice (ref_m = 0)
 * with equal t0 -- share the sample index, the interpolation weight and the phase of every (pixel, element) term, so
 * by linearity their channel data are added before demodulation and beamformed as one event ("folding"; detected at
 * plan creation by comparing the fp64 delay tables, exact up to the rounding order of the sums).
 * Enqueues on cuda_stream (a cudaStream_t passed as void*, NULL =
 * the legacy default stream) and returns without synchronising; results are valid once the caller has
 * synchronised that stream.  Never allocates.
 *   d_channel : int16 [frame][event][channel][sample] (x2 interleaved for IQ input), device memory
 *   d_out     : complex fp32 (re, im), device memory,
 *               compound == 1: [frame][ x-z: n_lat*n_ax | y-z: n_lat*n_ax ], axial index fastest
 *               compound == 0: [frame][event][lat][ax]
 * One call in flight per plan (the plan owns the IQ scratch).  n_frames == 0 is a no-op.
 * A plan belongs to the CUDA device that was current at plan_create; calls made while another device is current
 * fail with ULM_RCA_EINVAL.  Different plans (any filters, any devices) may be in flight at the same time.
 */
ulm_rca_status ulm_rca_beamform(const ulm_rca_plan *plan, const void *d_channel, int32_t n_frames,
                                void *d_out, void *cuda_stream);

/*
 * Conventional full 3-D DAS (step 4) on the grid x = grid_xz lateral, y = grid_yz lateral, z = the
 * (shared) axial grid: d_out_volume is complex fp32 [frame][x][y][z], z fastest.  Same stream and
 * ownership rules as ulm_rca_beamform.  Needs options.build_volume = 1.  Batches (max_frames) of one or two
 * frames are beamformed frame by frame from fp32 rows (das_volume_mirror_kernel on mirror-symmetric planes and
 * angles, else das_volume_kernel), larger ones by the generic kernel.
 */
ulm_rca_status ulm_rca_beamform_volume(const ulm_rca_plan *plan, const void *d_channel,
                                       int32_t n_frames, void *d_out_volume, void *cuda_stream);

/* Host convenience (this is the end-to-end call bench.py times as "e2e"): copies n_frames of HOST
 * channel data to an internal device buffer, beamforms, copies the images back to HOST memory and
 * synchronises.  The work is cut into chunks of 24 frames (12 for calls of fewer than 48 frames) and pipelined on two
 * internal streams through two device staging slots of one chunk each (upload of chunk i+1 overlaps the kernels and
 * the download of chunk i); only what the method reads is uploaded (the receive aperture of every event, the
 * touched sample range); pass pinned host memory for the overlap to take place.  Allocates the staging slots and
 * the streams on first use (freed by plan_destroy).  On any failure both streams are drained before the call
 * returns, so the caller's buffers are no longer in use.  One call in flight per plan. */
ulm_rca_status ulm_rca_beamform_host(ulm_rca_plan *plan, const void *h_channel, int32_t n_frames,
                                     void *h_out);

/* Byte sizes per frame of the three buffers above (any pointer may be NULL). */
ulm_rca_status ulm_rca_plan_sizes(const ulm_rca_plan *plan, size_t *channel_bytes_per_frame,
                                  size_t *out_bytes_per_frame, size_t *volume_bytes_per_frame);

/* Plan facts for benchmarks and tests: fills up to n values of
 *   [0] first touched sample  [1] touched samples per record  [2] IQ scratch bytes
 *   [3] kernel in use (1/2)   [4] frames per thread (F)       [5] pixels per tile
 *   [6] window entries per stage (W)  [7] ring stages  [8] tiles per projection (x-z)
 *   [9] dynamic shared memory bytes   [10] kernels launched by the last beamform call
 *   [11] tiles per projection (y-z)   [12] precision in use (1 compact-fast / 2 full / 3 compact)
 *   [13] scratch bytes per (sample, frame)   [14] bytes per frame ulm_rca_beamform_host uploads
 *   [15] transmit events beamformed per frame by ulm_rca_beamform after folding (see below; = n_row_tx + n_col_tx
 *        when nothing folds)
 *   [16] Stage 2: depth taps per (event, group) FIR executed by the kernel (0 = Stage 2 not prepared)
 *   [17] Stage 2: columns of the shared-memory slice tile (16 depths + halo)
 *   [18] .. [21] the ring kernel's work items of TWO frame groups (24 frames x 2 pixel rows per thread; used by calls
 *        of more than 12 frames when the scratch holds compact entries; 0 = not planned): window entries per group and
 *        stage, ring stages (each holds both groups' windows), tiles per projection x-z, y-z
 *   [22] 1 when single-frame volumes (ulm_rca_beamform_volume) run on mirror pairs: planes and angles of every
 *        aperture are mirror-symmetric (centred grid, symmetric angle set, equal start delays), 0 otherwise
 * [4] .. [9], [11] describe the work items of one frame group (12 frames x 4 pixel rows per thread). */
ulm_rca_status ulm_rca_plan_info(const ulm_rca_plan *plan, int64_t *values, int32_t n);

/* Mean device time per call of the kernels of the last n_calls (1..64) ulm_rca_beamform calls on this
 * plan, from CUDA events the library records on the caller's stream around its launches (first 4 batches
 * of each call): the demodulation/staging pre-pass and the DAS kernel(s).  Waits for those events; the
 * beamform calls themselves never synchronise. */
ulm_rca_status ulm_rca_plan_timing(const ulm_rca_plan *plan, int32_t n_calls, double *demod_ms, double *das_ms);

/* FP32 FMA throughput probe used for the roofline denominator: runs a register-only FFMA loop on every
 * SM on cuda_stream, synchronises, and returns the measured TFLOP/s (2 flop per FMA) in *tflops. */
ulm_rca_status ulm_rca_fp32_peak(double *tflops, void *cuda_stream);

/*
 * Stage 2 of the two-stage beamformer fused with the coherent compounding over all 2K transmissions and the sub-block
 * sum-projection ("the full volume V_k is reconstructed from [the slice] by extrapolating along the
 * transmit direction ... the compounded volume V is obtained by coherently summing all V_k-RC and V_k-CR";
 * the volume is divided into P x P x N sub-blocks that are "sum-projected along lateral (x) and
 * elevational (y) directions, resulting in projected planes V_p-m (m = 1 .. N/P x 2)"; P = 8).  The paper
 * prints no formula; the reading implemented is DESIGN.md section 11 (= oracle/stage2.py):
 *   voxel (lat, w, z_i) of event k, w = coordinate along the event's transmit direction, ref = the slice's position:
 *     tau0_k(z) = t0_k + (z cos th_k + ref sin th_k)/c + z/c,   B_k(lat, i) = S_k(lat, i) exp(-j 2 pi fc tau0_k(z_i)),
 *     q = i + (w - ref) tan(th_k/2) / dz,  n = floor(q),  b = q - n,  B_k = 0 outside the axial grid,
 *     V_k(lat, w, z_i) = [(1-b) B_k(lat, n) + b B_k(lat, n+1)] exp(+j 2 pi fc (tau0_k(z_i) + (w - ref) sin th_k / c)),
 *   V = sum of V_k over all row-tx (lat = x, w = y) and column-tx (lat = y, w = x) events on x = grid_xz lateral,
 *   y = grid_yz lateral, z = the common axial grid;  XZ_m(x, z) = sum over the m-th group of P consecutive y of V,
 *   YZ_m(y, z) = sum over the m-th group of P consecutive x of V (a last, shorter group is kept).
 * The volume is never formed (the group sums are complex FIRs along z with host-built taps).
 *   d_slices : complex fp32 [frame][event][lat][ax] -- exactly the compound == 0 output layout of ulm_rca_beamform
 *              (the paper filters these slices before Stage 2; any such array may be passed), device memory
 *   d_planes : complex fp32 [frame][ XZ: ceil(n_y/P) planes of n_x*n_ax | YZ: ceil(n_x/P) planes of n_y*n_ax ], axial
 *              index fastest, device memory
 * Needs options.stage2_block = P at plan_create (any `compound`); enqueues two kernels per batch of max_frames frames
 * on cuda_stream and returns without synchronising; never allocates; one call in flight per plan.
 */
ulm_rca_status ulm_rca_stage2_project(const ulm_rca_plan *plan, const void *d_slices, int32_t n_frames,
                                      void *d_planes, void *cuda_stream);

/* Byte sizes per frame of the two buffers of ulm_rca_stage2_project and the plane counts (any pointer may be NULL). */
ulm_rca_status ulm_rca_stage2_sizes(const ulm_rca_plan *plan, size_t *slices_bytes_per_frame,
                                    size_t *planes_bytes_per_frame, int32_t *n_planes_xz, int32_t *n_planes_yz);

/* Device time of the two kernels of the LAST batch of the last ulm_rca_stage2_project call (group sums, projection),
 * from CUDA events recorded on the caller's stream; waits for them.  Unavailable with options.no_timing. */
ulm_rca_status ulm_rca_stage2_timing(const ulm_rca_plan *plan, double *groupsum_ms, double *project_ms);

/*
 * Eigen-based clutter filter on the Stage-1 slice stacks ("parallelly computing the covariance matrix C
 * in C^{n_t x n_t} of I, performing a lightweight eigenvalue decomposition of C, and parallelly projecting to recover
 * blood flow signals", "applied ... immediately on 2D slices S_k-RC/CR obtained from Stage 1").  Reading (DESIGN.md
 * section 12 = oracle/clutter.py), per transmit event e with X[f][p] = slice value of pixel p in frame f:
 *   C[i][j] = sum_p conj(X[i][p]) X[j][p];   U_c = the clutter_rank eigenvectors of the largest eigenvalues of C;
 *   X_f[f][p] = X[f][p] - sum_m conj(U_c[f][m]) t_m[p],  t_m[p] = sum_f U_c[f][m] X[f][p]      (I_f = I (1 - U_c U_c^H)).
 * The paper gives no rule for the number of clutter components: clutter_rank (0 .. 24) is an argument.
 * C is formed on the tensor cores from bf16 (hi, lo) splits of the slices (three tcgen05.mma products per term, fp32
 * accumulation: relative error of C ~1e-5); the clutter subspace by blocked orthogonal iteration on 32 vectors (at most
 * 24 steps; it stops three steps after the leading clutter_rank eigenvalue estimates have settled to 1e-6) + a
 * Rayleigh-Ritz step, which is exact (to fp32) when lambda_{rank} is well separated from lambda_33 -- the tissue /
 * blood separation the filter is used for; for a flat spectrum the subspace, hence the result, is not determined.
 *   d_slices   : complex fp32 [frame][event][lat][ax] (compound == 0 layout), n_frames = n_t frames, device memory
 *   d_filtered : same layout and size; may be the same pointer as d_slices (in place)
 *   d_eigenvalues : NULL, or float [n_events][32]: the 32 largest eigenvalues of every C_e, descending
 *   d_covariance  : NULL, or complex fp32 [n_events][n_t][n_t]: the covariance matrices
 * Needs options.clutter_frames >= n_frames >= 32.  Enqueues five kernels on cuda_stream, never synchronises; one call in
 * flight per plan.
 */
ulm_rca_status ulm_rca_clutter_filter(const ulm_rca_plan *plan, const void *d_slices, int32_t n_frames,
                                      int32_t clutter_rank, void *d_filtered, void *d_eigenvalues, void *d_covariance,
                                      void *cuda_stream);

/* Device time of the five kernels of the last ulm_rca_clutter_filter call: ms5[0] bf16 split, [1] Gram (tcgen05),
 * [2] assembly of C, [3] eigen-subspace, [4] projection.  Waits for the events.  Unavailable with options.no_timing. */
ulm_rca_status ulm_rca_clutter_timing(const ulm_rca_plan *plan, double *ms5);

/*
 * Rigid motion estimation on the Stage-1 slices by Fourier-domain normalised cross-correlation ("each
 * frame is transformed into the Fourier domain, the correlation function between the two frames is computed, and the
 * displacement versus the reference frame is determined by locating the subpixel peak of the correlation function.  This
 * procedure requires two forward and one inverse Fourier transform"; "the K RC slices and K CR slices were used
 * separately to estimate motion within the x-z plane and the y-z plane.  K displacement vectors ... were first averaged,
 * and then the RC- and CR-averaged motions were vector-summed").  Reading: per slice, the B-mode
 * image |S| with its mean removed is zero-padded to the next powers of two; c(d) = IFFT2(FFT2(a_f) conj(FFT2(a_ref))) /
 * (|a_f| |a_ref|); the integer argmax (first in row-major order, signed) is refined by a 3-point parabola per axis; a
 * frame whose content moved by +s pixels relative to the reference gives +s.  Per frame the lateral / axial shifts are
 * averaged over the row-tx events (-> dx, dz) and the column-tx events (-> dy, dz) and scaled by the grid steps; the two
 * axial estimates are averaged (a literal vector sum would count the axial motion twice).
 *   d_slices    : complex fp32 [frame][event][lat][ax] (compound == 0 layout), device memory
 *   ref_frame   : index of the reference frame inside this call
 *   d_motion    : float4 [frame] = (dx, dy, dz in metres, mean NCC peak), device memory
 *   d_per_event : NULL, or float4 [frame][event] = (lateral shift in pixels, axial shift in pixels, NCC peak, 0)
 * Needs options.motion_frames >= n_frames and slices of at most 512 pixels along each axis.  Enqueues six kernels on
 * cuda_stream (hand-written warp FFTs in registers, two frames per complex transform; no library FFT), never
 * synchronises; one call in flight per plan.
 */
ulm_rca_status ulm_rca_motion_estimate(const ulm_rca_plan *plan, const void *d_slices, int32_t n_frames, int32_t ref_frame,
                                       void *d_motion, void *d_per_event, void *cuda_stream);

/* Device time (ms) of the six kernels of the last ulm_rca_motion_estimate call.  Unavailable with options.no_timing. */
ulm_rca_status ulm_rca_motion_timing(const ulm_rca_plan *plan, double *ms);

/* Parameters of ulm_rca_localize (none of them is given by the paper; PAPER.md:117 fixes only the 11-tap kernels). */
typedef struct {
    float sigma_lat_px, sigma_ax_px;   /* widths of the Gaussian-fitted PSF template along the lateral axis / depth, pixels  */
    float threshold_rel;               /* intensity threshold as a fraction of the frame's maximum |V|                         */
    float ncc_min;                     /* smallest NCC value of a localization                                                */
    int32_t capacity;                  /* localizations stored per plane at most                                               */
} ulm_rca_localize_params;

/*
 * Microbubble localization on the projected planes by separable sub-pixel 2-D normalised cross-correlation
 * ("the two projections are first normalized cross-correlated with the corresponding Gaussian-fitted 2D
 * PSFs ... sub-pixel regional peaks in the resulting correlating map are identified as localizations ... the 2D operation
 * was further decomposed into successive 1D correlations along each dimension"; 11-tap 1-D kernels;
 * "the maximum intensity of each volume was obtained ... for thresholding").  Reading:
 *   B = |V_p| of a plane (0 outside), g(a, b) = exp(-a^2 / 2 s_lat^2) exp(-b^2 / 2 s_ax^2), a, b = -5 .. 5;
 *   ncc(p) = sum_W (B - Bm)(g - gm) / sqrt(sum_W (B - Bm)^2 sum_W (g - gm)^2) over the 11 x 11 window W around p;
 *   a localization = an interior pixel with B >= threshold_rel * max over the frame's planes of B and ncc >= ncc_min
 *   whose ncc exceeds the 4 neighbours that follow it in row-major order and is not below the 4 that precede it, refined
 *   by a 3-point parabola of the NCC map along each axis.
 *   d_planes : complex fp32, the output layout of ulm_rca_stage2_project, n_frames frames, device memory
 *   d_loc    : float4 [frame][plane][capacity] = (lateral position, depth position in pixels, ncc, B), device memory;
 *              the order of the localizations of a plane is not fixed (atomic append), the set is
 *   d_count  : int32 [frame][plane] number of localizations found (if > capacity the surplus was dropped)
 * Needs options.stage2_block (the planes' geometry).  Enqueues two kernels per batch of max_frames frames; one call in
 * flight per plan.
 */
ulm_rca_status ulm_rca_localize(const ulm_rca_plan *plan, const void *d_planes, int32_t n_frames,
                                const ulm_rca_localize_params *params, void *d_loc, void *d_count, void *cuda_stream);

/*
 * ulm_rca_localize without a plan and WITHOUT ANY ALLOCATION -- for callers that cannot call cudaMalloc (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it).  Same operation, same kernels and same results as
 * ulm_rca_localize; the planes' geometry is passed as plain numbers:
 *   d_planes : complex fp32 [frame][n_planes_xz planes of n_lat_xz x n_z | n_planes_yz planes of n_lat_yz x n_z], depth
 *              index fastest (the output layout of ulm_rca_stage2_project), device memory; either plane set may be empty
 *   d_loc, d_count, params : as for ulm_rca_localize (outputs in device memory, owned by the caller)
 * The one scratch buffer of the operation -- the per-frame maximum of |V| that the intensity threshold needs -- lives in
 * a file-scope device array of ULM_RCA_LOCALIZE_STATIC_MAX_FRAMES unsigned ints (16 KB) that every GPU holding the
 * library keeps until the process exits; n_frames beyond that limit is refused with ULM_RCA_EINVAL (split the call).
 * The call clears the entries it uses (and d_count) on cuda_stream, enqueues the two kernels there and never
 * synchronises; it calls no cudaMalloc / cudaFree / allocating library routine (the first call on a device only looks up
 * the array's device address).  ALL calls on a device share that array: calls that can overlap on the GPU (different
 * streams without an ordering between them, or different host threads) race on it and may threshold against the wrong
 * maximum -- order them on one stream or with events.  The array keeps the last call's contents between calls.
 */
#define ULM_RCA_LOCALIZE_STATIC_MAX_FRAMES 4096
ulm_rca_status ulm_rca_localize_static(const void *d_planes, int32_t n_frames, int32_t n_z, int32_t n_planes_xz,
                                       int32_t n_lat_xz, int32_t n_planes_yz, int32_t n_lat_yz,
                                       const ulm_rca_localize_params *params, void *d_loc, void *d_count, void *cuda_stream);

/* Host-only view of the ring kernel's tile / window planning for ONE aperture (no CUDA device needed; used by the
 * CPU tests of the host logic): receive elements n_rx at `pitch_m`, transmit angles `angles_rad[n_tx]` with offsets
 * `t0_s` (NULL = 0), image grid `grid`.  Returns the number of tiles in *n_tiles, the stage length in entries in
 * *window, and, when the arrays are non-NULL (n_tiles * n_rx ints each), the per-(tile, element) window offsets
 * dj = floor(min receive excess over the tile) - 2 and stage lengths wj.  A tile is 384 consecutive positions of
 * (strip of 4 depth rows) x (lateral index), strips outer.  ULM_RCA_EUNSUPPORTED if the ring kernel does not
 * cover the shape. */
ulm_rca_status ulm_rca_ring_probe(int32_t n_rx, float pitch_m, const float *angles_rad, const float *t0_s, int32_t n_tx,
                                  float c_mps, float fs_hz, float t_start_s, const ulm_rca_grid *grid,
                                  int32_t *n_tiles, int32_t *window, int32_t *dj, int32_t *wj);

/* Host-only view of the event folding ulm_rca_plan_create applies to ONE aperture when compound == 1 (no CUDA device
 * needed; used by the CPU tests of the host logic): for the transmit angles `angles_rad[n_tx]` with offsets `t0_s`
 * (NULL = 0) and the reference slice / depth rows of `grid`, partner[k] receives the index of the later event whose
 * channel data are added to event k's (identical transmit delay on every depth row), -1 if event k is beamformed
 * alone, -2 if event k itself has been folded into an earlier event. */
ulm_rca_status ulm_rca_fold_probe(const float *angles_rad, const float *t0_s, int32_t n_tx, float c_mps, float fs_hz,
                                  const ulm_rca_grid *grid, int32_t *partner);

void ulm_rca_plan_destroy(ulm_rca_plan *plan); /* NULL-safe */

const char *ulm_rca_last_error(void); /* thread-local, valid until the next failing call */

#ifdef __cplusplus
}
#endif
#endif
