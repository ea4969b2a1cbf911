/*
 * tno_mf.h -- C ABI of the B200 matched-filter trajectory search.
 *
 * The operation (BASELINE.json:north_star; paper: Ganapathi, arXiv 2209.09848, section 3.2,
 * PAPER.md:L104-118, Eq. 5 "S = D * F" at L110, thresholding at L122): for a stack of
 * background-subtracted residual frames R_t and a bank of trajectory hypotheses k, score every
 * start pixel (x, y) with the matched filter "trajectory line convolved with the pixel response
 * function" (L106), evaluated sparsely (the paper's own suggestion of a "sparse convolution CUDA
 * kernel", L118):
 *
 *     c_t  = (x, y) + v (t - t0) + a (t - t0)^2              position at frame t
 *     N    = sum_t sum_{p in 5x5 window at round(c_t)} g(p - c_t) R_t(p) / sigma_t^2
 *     D    = sum_t sum_p g(p - c_t)^2 / sigma_t^2            taps outside the frame are
 *     SNR_k(x, y) = N / sqrt(D),  0 where D = 0              dropped from N and from D
 *
 * g(u) = exp(-|u|^2 / (2 prf_sigma^2)) (peak 1, sampled at pixel centres); round() is applied to
 * the displacement alone, round(c_t) = (x, y) + floor(d_t + 1/2), ties up (readings
 * c1-c8).  Outputs: the SNR maps and, per trajectory, the top-K pixels with SNR >= threshold
 * ordered by (SNR descending, y ascending, x ascending).
 *
 * Conventions
 *   - DEVICE pointers are CUDA device memory owned by the caller (e.g. a torch tensor's
 *     data_ptr()); HOST pointers are ordinary process memory.  Nothing passed in is retained
 *     after the call returns, and inputs are never written (except tno_mf_inject's frames).
 *   - tno_mf_search and tno_mf_inject validate on the host, enqueue their work on the context's
 *     stream and return without synchronising the device; results are valid once the caller
 *     synchronises that stream.  Host arrays are consumed before return.
 *   - Every function returns 0 on success or a negative TNO_MF_E* code; no exceptions, no
 *     exit().  After a failure tno_mf_last_error(ctx) describes it; outputs are unspecified.
 *   - A context is not thread-safe; distinct contexts are independent.  The only state outside a context is
 *     the thread-local text of the last tno_mf_create failure (tno_mf_last_error(NULL)).
 *   - There is no CPU fallback: without a CUDA device of compute capability 10.x,
 *     tno_mf_create fails with TNO_MF_EUNSUPPORTED / TNO_MF_ECUDA.
 *   - Behaviour for non-finite PIXELS is unspecified (pixels are not scanned).
 */
#ifndef TNO_MF_H
#define TNO_MF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TNO_MF_OK            0
#define TNO_MF_EINVAL       (-1)   /* bad argument (see each function) */
#define TNO_MF_ENOMEM       (-2)   /* host or device allocation failed */
#define TNO_MF_ECUDA        (-3)   /* CUDA runtime/driver error; text in tno_mf_last_error */
#define TNO_MF_EUNSUPPORTED (-4)   /* device is not sm_100-class, or no device */

typedef struct tno_mf_ctx tno_mf_ctx;                        /* opaque */

/* One trajectory hypothesis: velocity in px/frame, parallax term in px/frame^2
 * (north_star: "linear (vx,vy) or linear plus parallax term (ax,ay)"). */
typedef struct { float vx, vy, ax, ay; } tno_mf_traj;

/* One candidate.  Unused tail records are {-INFINITY, -1, -1, k}. */
typedef struct { float snr; int32_t x, y, k; } tno_mf_cand;  /* 16 bytes */

/* One source to inject: trajectory, start pixel at the reference epoch t0, amplitude in the
 * frames' flux units. */
typedef struct { tno_mf_traj traj; int32_t x, y; float amplitude; } tno_mf_source;  /* 28 bytes */

typedef struct {
    int32_t device;          /* CUDA device ordinal */
    void   *stream;          /* cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream);
                                NULL = the legacy default stream */
    int32_t topk;            /* K of the per-trajectory candidate list, >= 0; 0 = no list */
    float   snr_threshold;   /* candidate iff snr >= threshold; -INFINITY disables the cut */
    int32_t force_generic;   /* 0 = pick the fastest kernel that applies (normal use);
                                1 = always use the generic (non-TMA) kernel -- for tests */
    int32_t record_events;   /* != 0: bracket the main search kernel with CUDA events on the stream
                                so that tno_mf_last_kernel_ms can report its duration */
    int32_t workspace_limit_mb; /* 0 = default (<= 8 GB -- 40 GB in tno_mf_search_host, where the first chunk
                                hides the upload -- and <= 80 % of the free device memory);
                                > 0: cap, in MiB, of the partial-sum workspace of the separable
                                kernel -- a bank that needs more is searched in chunks of whole
                                batches (same results) */
    int32_t filter;          /* 0 = the Gaussian-PRF matched filter (the method); 1 = shift-stack, the comparison
                                method of PAPER.md:L118 (Rice & Laughlin 2020 "use a single non-zero value, set to 1,
                                for each time-slice"): the filter is 1 at round(c_t) and 0 elsewhere,
                                N = sum R_t(round(c_t))/sigma_t^2, D = sum [in frame]/sigma_t^2; prf_sigma is ignored
                                by the search (tno_mf_inject still renders with the PRF);
                                2 = pixel-integrated Gaussian PRF: the tap of pixel i is the flux fraction a source
                                at sub-pixel phase ph puts into it, Phi((i-ph+1/2)/prf_sigma) - Phi((i-ph-1/2)/prf_sigma)
                                per axis (PAPER.md:L41 describes the PRF by such fractions: ~50 % in the peak pixel);
                                3 = tabulated separable PRF, see tno_mf_set_prf_table; prf_sigma is ignored;
                                4 = tabulated non-separable PRF, see tno_mf_set_prf_table2d; prf_sigma is ignored.
                                In modes 2, 3 and 4 tno_mf_inject renders sources with the same taps. */
    int32_t sep_shape;       /* 0 = the separable kernel picks its shape by modelled cost (normal use): 4 positions per
                                thread x 5 slots per batch (tiles of 48 rows) or 5 x 4 (tiles of 60 rows);
                                1 / 2 = always the first / second shape -- for tests.  Same results up to rounding. */
} tno_mf_config;

/* Create a context on cfg->device.  Errors: EINVAL (NULL pointers, topk < 0, NaN threshold,
 * workspace_limit_mb < 0, filter not 0 .. 4, sep_shape not 0 .. 2), EUNSUPPORTED (no CUDA device / not compute capability 10.x), ECUDA, ENOMEM. */
int tno_mf_create(const tno_mf_config *cfg, tno_mf_ctx **out_ctx);

/* The search (formula above).
 *   frames        DEVICE  float32 [T][H][W], x fastest.  Read only.
 *   sigma_t       HOST    float32 [T], per-frame noise standard deviation, finite and > 0.
 *   trajectories  HOST    [n_traj]; finite values.
 *   prf_sigma     Gaussian PRF width in px, finite and > 0.   t0: reference epoch (frame units).
 *   out_snr       DEVICE  float32 [n_traj][H][W] (map k at out_snr + k*H*W), or NULL = no maps.
 *   out_topk      DEVICE  [n_traj][topk] records, or NULL (or topk == 0) = no lists.
 * Errors: EINVAL (NULL frames/sigma_t/trajectories, T/H/W/n_traj < 1, bad prf_sigma, sigma_t,
 * trajectory or t0 values, both outputs absent, shapes whose shifts do not fit 32-bit pixel
 * arithmetic, n_traj > 65535, H * W > 2^31, H > 262140 rows -- the same row limit holds for every call
 * that takes frames or maps), ENOMEM, ECUDA.
 * Any H, W >= 1 is computed correctly; the TMA kernel needs W % 4 == 0 and 16-byte aligned
 * frames (and y-shift ranges below 63 tile heights of 48 / 60 px), other inputs take the generic kernel.
 * The TMA kernel accumulates into a context-owned partial-sum workspace of (1 + ceil(y-shift range /
 * tile height)) * n_traj * H * W floats, capped (cfg.workspace_limit_mb); a larger bank is searched in chunks
 * of whole batches with identical results.  Results are bitwise reproducible, and for a given kernel
 * shape the map of a trajectory does not depend on the other trajectories of the call; with
 * cfg.sep_shape = 0 the shape (tile height 48 or 60) is picked per call from the bank and the frame
 * size, and the two shapes sum in different orders (differences of a few float32 ulps): pin
 * cfg.sep_shape to compare maps bit for bit across banks.  All element offsets are 64-bit. */
int tno_mf_search(tno_mf_ctx *ctx,
                  const float *frames, int32_t T, int32_t H, int32_t W,
                  const float *sigma_t,
                  const tno_mf_traj *trajectories, int32_t n_traj,
                  float prf_sigma, float t0,
                  float *out_snr,
                  tno_mf_cand *out_topk);

/* The search with frame times and pointing jitter in the track -- the filter is "the line of the trajectory
 * (including the pointing jitter)" and the frames of a sector are not equally spaced
 * ("the time-jump that occurs when TESS is transmitting frames to Earth", L116):
 *     c_t = (x, y) + v (tau_t - t0) + a (tau_t - t0)^2 + j_t
 *   frame_times  HOST float32 [T], tau_t in the time unit of the velocities, or NULL (tau_t = t).
 *   jitter_xy    HOST float32 [T][2], (jx_t, jy_t) in px, or NULL (no jitter).
 * Everything else as tno_mf_search, which is this call with both NULL.  Rounding, window, PRF and the
 * dropping of off-frame taps are unchanged (readings c1-c8, f1-f3); only the per-(trajectory,
 * frame) table differs, so the cost is the same.  Additional error: EINVAL for non-finite entries. */
int tno_mf_search_ex(tno_mf_ctx *ctx,
                     const float *frames, int32_t T, int32_t H, int32_t W,
                     const float *sigma_t, const float *frame_times, const float *jitter_xy,
                     const tno_mf_traj *trajectories, int32_t n_traj,
                     float prf_sigma, float t0,
                     float *out_snr,
                     tno_mf_cand *out_topk);

/* The search with per-pixel validity weights.  The paper sets bright pixels to 0 before filtering
 * ("the noise in those pixels will so high to make it impossible to detect a magnitude 20+ signal",
 * PAPER.md:L106) and keeps the normalisation of the full filter; here a masked pixel also leaves the
 * normalisation, which keeps the score in units of sigma next to masked stars:
 *     N = sum_t sum_p g(p - c_t) F_t(p) / sigma_t^2          F = frames AS GIVEN: the caller has zeroed
 *                                                            (or down-weighted) them, F = R * valid
 *     D = sum_t sum_p g(p - c_t)^2 valid_t(p) / sigma_t^2    SNR = N / sqrt(D), 0 where D = 0
 *   valid   DEVICE float32 [T][H][W], finite and >= 0: 1 = use, 0 = masked; other values act as relative
 *           inverse variances of the pixels.  Read only.  NULL = tno_mf_search_ex.
 * D is accumulated by a second pass of the same kernel over `valid` with squared taps: twice the time
 * and twice the workspace of tno_mf_search.  tno_mf_flux does not apply to a masked search (EINVAL).
 * Everything else as tno_mf_search_ex. */
int tno_mf_search_masked(tno_mf_ctx *ctx,
                         const float *frames, const float *valid, int32_t T, int32_t H, int32_t W,
                         const float *sigma_t, const float *frame_times, const float *jitter_xy,
                         const tno_mf_traj *trajectories, int32_t n_traj,
                         float prf_sigma, float t0,
                         float *out_snr,
                         tno_mf_cand *out_topk);

/* The search on a stack in HOST memory, results to HOST memory.  The stack is uploaded in bands of frame
 * rows on a second stream; the search of a band of tiles starts as soon as its rows (all T frames) are on the
 * device, so the transfer (the longer of the two on PCIe) hides the computation.  Same results, bit for bit,
 * as tno_mf_search_ex on the uploaded stack.
 *   frames_host    HOST float32 [T][H][W]; page-locked memory is needed for the overlap (pageable works, slower).
 *   out_snr_host   HOST float32 [n_traj][H][W] or NULL.     out_topk_host  HOST [n_traj][topk] or NULL.
 * Unlike the device-pointer calls this one RETURNS AFTER THE RESULTS ARE IN THE HOST BUFFERS (it synchronises
 * the context's stream).  The device copy of the stack and of the outputs lives in the context's workspace.
 * Errors: as tno_mf_search_ex. */
int tno_mf_search_host(tno_mf_ctx *ctx,
                       const float *frames_host, int32_t T, int32_t H, int32_t W,
                       const float *sigma_t, const float *frame_times, const float *jitter_xy,
                       const tno_mf_traj *trajectories, int32_t n_traj,
                       float prf_sigma, float t0,
                       float *out_snr_host,
                       tno_mf_cand *out_topk_host);

/* tno_mf_search_host for the paper's real chain: clipped bright pixels (PAPER.md:L106 -> `valid_host`, as in
 * tno_mf_search_masked) and the maximum over the filter bank (L112 -> `out_max_host`, `out_argk_host`, as in
 * tno_mf_search_max), with the same banded overlap of upload, search, finish and download.  The validity
 * weights travel with the frames, band by band (twice the upload); the two max maps are copied back at the end.
 *   valid_host     HOST float32 [T][H][W] or NULL (= unmasked).
 *   out_max_host   HOST float32 [H][W] or NULL.   out_argk_host  HOST int32 [H][W] or NULL (needs out_max_host).
 *   out_snr_host, out_topk_host as in tno_mf_search_host; at least one of the three outputs must be given.
 * Results are bit for bit those of tno_mf_search_max on the uploaded stacks.  tno_mf_search_host is this call
 * with valid_host, out_max_host and out_argk_host NULL.  Errors: as tno_mf_search_max. */
int tno_mf_search_host_max(tno_mf_ctx *ctx,
                           const float *frames_host, const float *valid_host, int32_t T, int32_t H, int32_t W,
                           const float *sigma_t, const float *frame_times, const float *jitter_xy,
                           const tno_mf_traj *trajectories, int32_t n_traj,
                           float prf_sigma, float t0,
                           float *out_max_host, int32_t *out_argk_host,
                           float *out_snr_host,
                           tno_mf_cand *out_topk_host);

/* Tabulated separable PRF for filter 3: `table` is HOST float32
 * [n_phase][5], row r = the fractions of the flux that fall into the pixels -2 .. +2 around the rounded
 * position for a source whose sub-pixel phase ph = c - round(c) lies in [-1/2 + r/n_phase, -1/2 + (r+1)/n_phase);
 * the search and tno_mf_inject use row floor((ph + 1/2) * n_phase) for x and for y (nearest tabulated phase, no
 * interpolation), the 2-D filter is the outer product.  Values must be finite and >= 0.  The table is copied;
 * n_phase = 0 removes it.  A context with filter 3 and no table fails its searches with EINVAL.
 * Errors: EINVAL, ENOMEM, ECUDA. */
int tno_mf_set_prf_table(tno_mf_ctx *ctx, const float *table, int32_t n_phase);

/* Tabulated NON-separable PRF for filter 4 (the TESS PRF, "approximately 50 % of
 * the flux in the peak pixel and 90 % in 2 x 2", is tabulated per 2-D sub-pixel phase and is not an outer product).
 * `table` is HOST float32 [n_phase_y][n_phase_x][5][5]: block (ry, rx) holds, at [j + 2][i + 2], the response of the
 * pixel at offset (i, j) from the rounded position for a source whose sub-pixel phases (phx, phy) fall into column
 * rx = floor((phx + 1/2) n_phase_x) and row ry = floor((phy + 1/2) n_phase_y) (clamped; no interpolation).
 * Values finite and >= 0; phases 1 .. 4096; both 0 removes the table.  The table is copied.
 * Searches of a context with filter 4 run the 25-tap formulation (one thread per trajectory and pixel, N and D
 * accumulated together: D is not separable either), at any H, W and alignment, with or without validity weights;
 * tno_mf_inject renders with the same blocks; tno_mf_flux does not apply (EINVAL).  A context with filter 4 and no
 * table fails its searches with EINVAL.  Errors: EINVAL, ENOMEM, ECUDA. */
int tno_mf_set_prf_table2d(tno_mf_ctx *ctx, const float *table, int32_t n_phase_y, int32_t n_phase_x);

/* Signal injection ("signal injection corresponds to adding a filter times a flux
 * to the raw data"): for each source m in order and every frame t,
 *     R_t(p) <- (float)((double)R_t(p) + amplitude_m * g(p - c_t))  on the 25 window taps,
 * taps outside the frame skipped.  Deterministic (sources are applied sequentially per frame).
 *   frames   DEVICE float32 [T][H][W], modified in place.     sources  HOST [n_sources].
 * Errors: EINVAL, ECUDA. */
int tno_mf_inject(tno_mf_ctx *ctx, float *frames, int32_t T, int32_t H, int32_t W,
                  const tno_mf_source *sources, int32_t n_sources,
                  float prf_sigma, float t0);

/* tno_mf_inject on the track that tno_mf_search_ex scores: frame times and pointing jitter enter the position of
 * the source exactly as they enter the filter, c_t = (x, y) + v (tau_t - t0) + a (tau_t - t0)^2 + j_t ("the line of
 * the trajectory (including the pointing jitter)"; injection = "adding a filter times a flux", L130),
 * so that injection and recovery are consistent for irregular cadence and jitter.
 *   frame_times HOST float32 [T] or NULL; jitter_xy HOST float32 [T][2] or NULL (both NULL = tno_mf_inject).
 * Errors: EINVAL (also: non-finite times / jitter, a displacement beyond 1e9 px), ENOMEM, ECUDA. */
int tno_mf_inject_ex(tno_mf_ctx *ctx, float *frames, int32_t T, int32_t H, int32_t W,
                     const float *frame_times, const float *jitter_xy,
                     const tno_mf_source *sources, int32_t n_sources,
                     float prf_sigma, float t0);

/* Interpreting scores (section 3.3): "We take the maximum score across the filter bank, which
 * then tells us the most likely trajectory, along with the score of that trajectory" (L112), and "we
 * compute the standard deviation sigma of the scores in the 255 x 255 square centered on a pixel. We
 * represent our scores in units of sigma" (L124):
 *     M(x, y) = max_k snr[k][y][x],  A(x, y) = the smallest k that attains it
 *     Z(x, y) = M(x, y) / sigma_box(x, y), sigma_box = population standard deviation of M over the
 *               pixels of the frame within (box-1)/2 of (x, y) in both axes; 0 where it vanishes
 *   snr       DEVICE float32 [n_traj][H][W] (e.g. out_snr of tno_mf_search).  Read only.
 *   box       odd, >= 1 (the paper uses 255).
 *   out_max   DEVICE float32 [H][W].                  out_argk  DEVICE int32 [H][W], or NULL.
 *   out_z     DEVICE float32 [H][W], or NULL.
 *   out_topk  DEVICE [topk] records of the pixels with the largest Z >= cfg.snr_threshold (now in
 *             units of sigma_box), ordered (Z descending, y, x ascending), record.snr = Z, record.k =
 *             A(x, y); unused tail {-INFINITY, -1, -1, -1}; or NULL (or topk == 0).
 * sigma_box is evaluated in float64 from summed-area tables; a variance below 1e-12 of the box's mean
 * square counts as zero.  Errors: EINVAL (NULL snr/out_max, sizes < 1, even box), ENOMEM, ECUDA. */
int tno_mf_best(tno_mf_ctx *ctx, const float *snr, int32_t n_traj, int32_t H, int32_t W, int32_t box,
                float *out_max, int32_t *out_argk, float *out_z, tno_mf_cand *out_topk);

/* Z of one score map without any device allocation (the Z(x, y) of tno_mf_best): for callers that
 * cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that forbid it.
 * tno_mf_best keeps its float64 summed-area tables in a context buffer that grows with cudaMalloc; this call keeps
 * them in a static device array of the library and enqueues its three kernels on the context's stream, nothing
 * else: no cudaMalloc, no cudaFree, no allocating library routine, no synchronisation.
 *   score     DEVICE float32 [H][W] (e.g. out_max of tno_mf_best / tno_mf_search_max).  Read only.
 *   box       odd, >= 1 (the paper uses 255).
 *   out_z     DEVICE float32 [H][W], must not alias score.  Bit for bit the out_z of
 *             tno_mf_best(score as a bank of one map).
 * Limit: H * W <= 1 048 576 pixels (e.g. 1024 x 1024); the static array is 16 MiB, and every GPU that loads the
 * library holds it until the process exits.  All calls on a device share the array, whatever their context or
 * stream: calls that overlap on the GPU race on it -- keep them on one stream or order them with events.  The
 * array keeps the last call's contents; every call overwrites the H * W entries it reads, so nothing has to be
 * cleared.  The first call on a device resolves the array's device address (cudaGetSymbolAddress, once per device):
 * make that call before a graph capture starts.
 * Errors: EINVAL (NULL or aliased pointers, sizes < 1, H * W beyond the limit -- the text names the limit and
 * tno_mf_best as the path for larger maps --, even box, device ordinal > 63), ECUDA. */
int tno_mf_local_z_static(tno_mf_ctx *ctx, const float *score, int32_t H, int32_t W, int32_t box, float *out_z);

/* Debug aid: fill the shared memory of every SM of the context's device with `pattern` (one kernel on the context's
 * stream that takes all the shared memory of an SM, a few waves of blocks).  Shared memory is not cleared between
 * kernels; a kernel that reads a word it never wrote computes with what an earlier kernel left there.  The GPU tests
 * call this with 0xffffffff (a NaN as a float) before every test, which turns such a read into a visible error --
 * what compute-sanitizer's initcheck would report.  No effect on results.  Errors: EINVAL (NULL ctx), ECUDA. */
int tno_mf_debug_poison_shared(tno_mf_ctx *ctx, uint32_t pattern);

/* The search with the max over the filter bank fused into its epilogue ("We take
 * the maximum score across the filter bank, which then tells us the most likely trajectory, along with the score
 * of that trajectory"): everything tno_mf_search_masked does, plus
 *   out_max    DEVICE float32 [H][W]   M(x, y) = max_k SNR_k(x, y)               (required)
 *   out_argk   DEVICE int32   [H][W]   the smallest k that attains it, or NULL
 * -- bit for bit what tno_mf_best computes from out_snr, without the maps having to exist: out_snr and out_topk
 * may both be NULL (a bank of 1024 trajectories on 2048^2 then needs no 17 GB of maps).  valid, frame_times and
 * jitter_xy may be NULL as in the other searches.  Z and the peaks follow with tno_mf_best(out_max as a bank of
 * one map) and tno_mf_peaks(Z, out_argk).  The running maximum lives in a 64-bit key per pixel (8 * H * W bytes of
 * workspace), updated with atomicMax: order independent, hence reproducible.  Errors as tno_mf_search_masked. */
int tno_mf_search_max(tno_mf_ctx *ctx, const float *frames, const float *valid, int32_t T, int32_t H, int32_t W,
                      const float *sigma_t, const float *frame_times, const float *jitter_xy,
                      const tno_mf_traj *trajectories, int32_t n_traj, float prf_sigma, float t0,
                      float *out_max, int32_t *out_argk, float *out_snr, tno_mf_cand *out_topk);

/* Non-maximum suppression of a score map, "so one object yields one candidate" (the paper
 * lists every score above 3 sigma as a candidate, L124, and one object lights up a neighbourhood):
 * pixel p is a peak iff score(p) >= cfg.snr_threshold and for every other pixel q of the frame with
 * |qx - px| <= radius and |qy - py| <= radius: score(p) > score(q), or score(p) == score(q) and p precedes q
 * in row-major order (of equal neighbours the first one survives).
 *   score      DEVICE float32 [H][W], e.g. out_z or out_max of tno_mf_best.  Read only.
 *   argk       DEVICE int32 [H][W] (out_argk of tno_mf_best) or NULL: fills record.k (else 0).
 *   radius     0 .. 1024 px (0: every pixel above the threshold is a peak).
 *   out_peaks  DEVICE float32 [H][W]: score at the peaks, -INFINITY elsewhere; or NULL.  Must not alias score.
 *   out_topk   DEVICE [topk] records of the highest peaks, ordered (score descending, y, x ascending), unused
 *              tail {-INFINITY, -1, -1, -1}; or NULL (or topk == 0).
 * Errors: EINVAL, ENOMEM, ECUDA. */
int tno_mf_peaks(tno_mf_ctx *ctx, const float *score, const int32_t *argk, int32_t H, int32_t W, int32_t radius,
                 float *out_peaks, tno_mf_cand *out_topk);

/* Flux estimate (the score "is a direct estimate of the total flux due to that moving
 * object, which allows to not only estimate the position and trajectory of a detection, but also the
 * magnitude"): the maximum-likelihood amplitude of a source on trajectory k starting at (x, y),
 *     A_k(x, y) = N / D = SNR_k(x, y) / sqrt(D_k(x, y)),        0 where D = 0,
 * in the flux units of the frames, from the SNR maps and the D tables of the LAST tno_mf_search(_ex) on
 * this context (same n_traj, H, W; the tables stay valid until the next search).
 *   snr       DEVICE float32 [n_traj][H][W] as written by that search.   out_flux  DEVICE, same shape.
 * Errors: EINVAL (NULL pointers, no matching preceding search), ECUDA. */
int tno_mf_flux(tno_mf_ctx *ctx, const float *snr, int32_t n_traj, int32_t H, int32_t W, float *out_flux);

/* High-resolution background model (section 3.1, Eq. 1-4): the step that produces the residual
 * stack the search runs on.  With the scattered light U(S_t) already removed, every pixel p is regressed on
 * the pointing jitter theta_t = (x_t, y_t),
 *     y_t(p) = B(p) + B_theta(p) . (x_t, y_t, x_t^2, y_t^2, x_t y_t) + eps,
 * with the Huber loss L_delta (Eq. 4) "through repeated least squares solves, alternated with clipping the
 * residuals (Huber 1977)" (L100):  beta_0 = least squares;  beta_{i+1} = beta_i + pinv(Phi) clip(y - Phi beta_i,
 * -delta, +delta), i = 0 .. n_iter-1;  all pixels share Phi (orthonormalised once on the host in float64).
 *   frames     DEVICE float32 [T][H][W]: data minus scattered light.     jitter_xy  HOST float32 [T][2], px.
 *   delta      Huber threshold in flux units, > 0 (INFINITY: plain least squares).    n_iter >= 0.
 *   out_coef   DEVICE float32 [6][H][W]: B, then the coefficients of x, y, x^2, y^2, xy; or NULL.  Columns of
 *              the basis that are linearly dependent on earlier ones (e.g. no jitter at all) get 0.
 *   out_resid  DEVICE float32 [T][H][W]: y - Phi beta, the input of tno_mf_search; may be `frames` itself
 *              (in place); or NULL.
 * Traffic: (n_iter + 3) * T*H*W*4 bytes (one read per pass, the last pass also writes), HBM-bound; the fast
 * kernel needs H*W % 4 == 0 and 16-byte aligned pointers, other stacks take a slower plain kernel with the
 * same results.  T >= 6 distinct jitter values are needed for all six coefficients to be identifiable.
 * Enqueues on the context's stream after a short synchronisation for the basis upload.
 * Errors: EINVAL, ENOMEM, ECUDA. */
int tno_mf_background(tno_mf_ctx *ctx, const float *frames, int32_t T, int32_t H, int32_t W,
                      const float *jitter_xy, float delta, int32_t n_iter, float *out_coef, float *out_resid);

/* Low-resolution scattered-light model (section 3.1, Eq. 1-4, second part):
 *     D_t = U(S_t) + B + B_theta . (x_t, y_t, x_t^2, y_t^2, x_t y_t) + eps_t,      L = sum_{t,i,j} L_delta(D_t - pred_t)
 * with D the data downsampled to N x N ("N = 512"), S_t an n x n image per frame ("n = 64"), U bilinear upsampling
 * (output pixel i has its centre at (i + 1/2) n / N - 1/2 input pixels, clamped to [0, n - 1], and takes the two
 * nearest input pixels per axis: "the 4 nearest low resolution points"), L_delta the Huber loss of Eq. 4.
 * "We minimize this convex loss over B, B_theta, S_t using the L-BFGS algorithm" (L94).
 *   D          DEVICE float32 [T][N][N].           jitter_xy  HOST float32 [T][2], px.        delta > 0.
 *   beta       DEVICE float32 [6][N][N]: B, then the coefficients of x, y, x^2, y^2, xy.
 *   S          DEVICE float32 [T][n][n].
 * tno_mf_scatter_lossgrad evaluates L (float64, written to HOST *out_loss) and its gradient (DEVICE g_beta
 * [6][N][N], g_S [T][n][n]) at (beta, S); it returns after the loss has arrived.
 * tno_mf_scatter_fit runs L-BFGS (10 pairs, Armijo backtracking) from the (beta, S) it is given -- zeros are the
 * paper's "regardless of the initial parameters" -- and overwrites them with the minimiser; it stops when
 * max_i |g_i| <= gtol, after max_iter iterations, when two consecutive iterations each decrease the loss by less
 * than 1e-9 of its value, or when no step decreases it at all (float32 resolution), and reports the
 * final loss, the iterations and the loss evaluations (HOST, each may be NULL).  Blocking.  The loss and the
 * prediction are determined by the data; the split of a time-constant smooth component between S and B is not.
 * Workspace: about 26 vectors of 6 N^2 + T n^2 floats and one [T][N][N] stack.  Errors: EINVAL, ENOMEM, ECUDA. */
int tno_mf_scatter_lossgrad(tno_mf_ctx *ctx, const float *D, int32_t T, int32_t N, int32_t n, const float *jitter_xy,
                            float delta, const float *beta, const float *S, double *out_loss, float *g_beta,
                            float *g_S);
int tno_mf_scatter_fit(tno_mf_ctx *ctx, const float *D, int32_t T, int32_t N, int32_t n, const float *jitter_xy,
                       float delta, int32_t max_iter, float gtol, float *beta, float *S, double *out_loss,
                       int32_t *out_iters, int32_t *out_evals);

/* The two ends of that solve.  tno_mf_downsample: out[t][y][x] = mean of the factor x factor block of frames
 * ("the data downsampled to 512 x 512 from 2048 x 2048", L69); frames DEVICE [T][H][W], out DEVICE
 * [T][H/factor][W/factor], factor divides H and W.  tno_mf_scatter_subtract: frames[t] -= U(S_t) with U from
 * n x n to H x W (same bilinear rule), in place -- the stack that tno_mf_background expects ("Once we solve for
 * scattered light S_t at low resolution, we hold it fixed, and re-estimate B, B_theta at high resolution", L98).
 * T <= 65535.  Asynchronous on the context's stream.  Errors: EINVAL, ECUDA. */
int tno_mf_downsample(tno_mf_ctx *ctx, const float *frames, int32_t T, int32_t H, int32_t W, int32_t factor,
                      float *out);
int tno_mf_scatter_subtract(tno_mf_ctx *ctx, float *frames, int32_t T, int32_t H, int32_t W, const float *S,
                            int32_t n);

/* Host-only planning query (no device work; ctx may be NULL): how the search would group
 * `trajectories` into batches that share one x-motion (vx, ax) -- the unit of work of the
 * separable kernel.  Writes, for each trajectory, its batch index and slot
 * within the batch to out_batch[n_traj] / out_slot[n_traj] (either may be NULL) and returns the
 * number of batches (>= 1), or a negative error.  max_entries: slots per batch (1..16);
 * max_spread: largest allowed difference of integer y-shifts inside a batch at any frame; a value
 * >= 2^30 means no limit and an even split of each x-motion into the fewest batches.  (The search
 * itself batches SLOTS, tno_mf_plan_slots; this query is the single-trajectory packing.) */
int tno_mf_plan(const tno_mf_traj *trajectories, int32_t n_traj, int32_t T, float t0,
                int32_t max_entries, int32_t max_spread,
                int32_t *out_batch, int32_t *out_slot);

/* Host-only planning query (no device work): how the separable kernel groups `trajectories` into batches of
 * SLOTS.  A batch shares one x-motion; a slot holds a y-motion (vy, ay) and, if it is in the bank, its mirror
 * image (-vy, -ay), which the kernel scores together at the cost of one (exact
 * algebra on the five y-taps).  Two trajectories share a slot only if the filter is symmetric under y -> -y
 * (`symmetric_filter` != 0: cfg.filter 0 and 1), no frame rounds an exact half-pixel tie, and there is no
 * pointing jitter in y; otherwise each sits alone.  Writes per trajectory its batch, its slot within the batch
 * and its member (0: the slot's own orientation, vy > 0 or (vy = 0, ay >= 0) for a pairable motion; 1: the
 * mirror image) to out_batch / out_slot / out_member [n_traj] (each may be NULL); returns the number of batches
 * or a negative error.  frame_times / jitter_xy as in tno_mf_search_ex (NULL = none).  max_slots in 1 .. 16
 * (the search uses 5). */
int tno_mf_plan_slots(const tno_mf_traj *trajectories, int32_t n_traj, int32_t T, float t0,
                      const float *frame_times, const float *jitter_xy, int32_t max_slots,
                      int32_t symmetric_filter, int32_t *out_batch, int32_t *out_slot, int32_t *out_member);

/* Counters of the last tno_mf_search on this context (host values, valid after the call
 * returns): number of kernel launches enqueued, and which search kernel was used
 * (0 = generic, 1 = separable TMA kernel).  NULL pointers are skipped. */
int tno_mf_last_stats(const tno_mf_ctx *ctx, int32_t *out_launches, int32_t *out_kernel);

/* Duration in milliseconds of the main search kernel of the last tno_mf_search, measured with
 * CUDA events recorded on the context's stream around that launch.  Needs
 * cfg.record_events != 0 (else EINVAL).  Blocks the host until the kernel has finished. */
int tno_mf_last_kernel_ms(tno_mf_ctx *ctx, float *out_ms);

/* Work of the last tno_mf_search in FP32 operations of the formulation it executed (DESIGN.md
 * "roofline"): multiply-adds of the shared x-pass (5 per staged pixel and batch, halo rows included),
 * multiply-adds of the y-pass (5 per SLOT x frame x pixel; a slot is one trajectory or a trajectory and
 * its mirror image (-vy, -ay)), and the additions of the y-pass (4 per batch x
 * frame x pixel: the sums and differences of the window rows that all slots of a batch share).  The
 * generic kernel reports x = 0, y = 25 per evaluation, no additions.  NULL pointers are skipped. */
int tno_mf_last_work(const tno_mf_ctx *ctx, double *out_fma_xpass, double *out_fma_ypass, double *out_add_ypass);

/* Release the context and its workspace.  The caller must have synchronised the stream.
 * NULL is accepted. */
int tno_mf_destroy(tno_mf_ctx *ctx);

/* Text of the last error on this context (or of the last failed tno_mf_create when ctx is
 * NULL).  Never NULL; valid until the next call on the same context. */
const char *tno_mf_last_error(const tno_mf_ctx *ctx);

/* Library version string, e.g. "tno_mf 0.1 (sm_100a)". */
const char *tno_mf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TNO_MF_H */
