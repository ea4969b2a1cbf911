// Launch wrappers of the kernels in libtno_mf.so (all enqueue on the given stream, no syncs).
#pragma once
#include <cuda.h>

#include "../../include/tno_mf.h"
#include "common.cuh"

namespace tno {

// ---- tables.cu ----
void launch_class_tables(cudaStream_t st, const float *cls_v, const float *cls_a,
                         const float *times /* DEVICE [T] or NULL */, const float *jitter /* DEVICE [T][2] or NULL */,
                         int32_t n_cls, int32_t n_x, int32_t T, double t0, double prf_sigma,
                         int32_t filter /* tno_mf_config::filter */, const float *prf_tab /* DEVICE [n_phase][5] */,
                         int32_t n_phase, int32_t *shift, float *g, double *gd);
void launch_border_tables(cudaStream_t st, const int32_t *shift, const double *gd, const double *qd,
                          const AxisBorder *border, const int64_t *off, int32_t n_cls, int32_t n_x,
                          int32_t max_n, int32_t T, int32_t W, int32_t H, double *out);
void launch_rsd_tables(cudaStream_t st, const TrajInfo *traj, int32_t n_traj, int64_t max_tiles,
                       const double *ab, const int64_t *off, int32_t n_x, int32_t T, float *rsd);

// ---- search_generic.cu ----
// One thread per (trajectory, pixel); any H, W; maps only.
// valid != NULL: D = sum g^2 valid / sigma^2 is accumulated next to N (masked search), rsd is not used
void launch_search_generic(cudaStream_t st, const float *frames, const float *valid, int32_t T, int32_t H, int32_t W,
                           const ClassTables &tab, const TrajInfo *traj, const float *rsd,
                           int32_t k_first, int32_t k_count, float *out_snr /* [k_count][H][W] */);

// filter 4: the 25 taps of (trajectory, frame) from the non-separable table tab2 [n_py][n_px][5][5]; tab.gd holds
// the phase rows / columns (tables.cu); N and D are accumulated together
void launch_search_generic25(cudaStream_t st, const float *frames, const float *valid, int32_t T, int32_t H, int32_t W,
                             const ClassTables &tab, const TrajInfo *traj, const float *tab2, int32_t n_px,
                             int32_t k_first, int32_t k_count, float *out_snr);

// ---- topk.cu ----
constexpr int32_t kCollectTile = 64;        // k_collect_from_map tiles are 64 x 64 pixels
constexpr int32_t kMaxTopk = 1024;
constexpr int32_t kMaxRows = 65535 * 4;     // frame rows: several kernels put rows / 4 into gridDim.y (DESIGN d2)
// candidates of maps [k_count][H][W] (trajectories k_first..) into tile slots
void launch_collect_from_map(cudaStream_t st, const float *maps, int32_t H, int32_t W,
                             int32_t k_first, int32_t k_count, const TopkSlots &slots);
// merge all tile slots of every trajectory into out_topk[K][ktop]
void launch_topk_merge(cudaStream_t st, const TopkSlots &slots, int32_t n_tiles, int32_t W,
                       tno_mf_cand *out_topk);

// ---- best.cu ---- (section 3.3: max over the filter bank, scores in local-sigma units)
void launch_max_map(cudaStream_t st, const float *snr, int32_t K, int32_t H, int32_t W, float *out_max,
                    int32_t *out_argk /* may be NULL */, int32_t n_sm);
// sat_ws: H*W*16 bytes of workspace (float64 summed-area tables of M and M^2)
void launch_local_z(cudaStream_t st, const float *m, int32_t H, int32_t W, int32_t box, void *sat_ws, float *z);
// out[k][y][x] = snr[k][y][x] * D_k(x, y)^(-1/2)  (flux estimate N / D)
void launch_flux(cudaStream_t st, const float *snr, const TrajInfo *traj, const float *rsd, int32_t K, int32_t H,
                 int32_t W, float *out);
// running maximum over the bank as 64-bit keys (score order << 32 | ~k): update from materialised maps, decode
void launch_max_keys_from_maps(cudaStream_t st, const float *maps, int32_t k0, int32_t kc, int64_t n_px, uint64_t *keys);
void launch_max_decode(cudaStream_t st, const uint64_t *keys, int64_t n_px, float *out_max, int32_t *out_argk);
void launch_nms(cudaStream_t st, const float *score, int32_t H, int32_t W, int32_t radius, float thr, float *out);
void launch_set_argk(cudaStream_t st, tno_mf_cand *cand, int32_t n, const int32_t *argk, int32_t W);

// ---- background.cu ---- (section 3.1: per-pixel Huber fit on the jitter basis)
struct BgRinv { float v[36]; };      // R^{-1} of the orthonormalised basis, row major
// Q: DEVICE [T][16] orthonormal basis, every coefficient twice + padding (see background.cu); out_resid may alias frames (in place)
void launch_background(cudaStream_t st, const float *frames, int32_t T, int64_t n_px, const float *Q,
                       const BgRinv &rinv, float delta, int32_t n_iter, float *out_coef, float *out_resid);

// ---- scatter.cu ---- (section 3.1: low-resolution scattered-light model, L-BFGS)
constexpr int kScatterHistory = 10;
struct ScatterProblem {
    const float *D;        // DEVICE [T][N][N] downsampled data
    int32_t T, N, n;
    const float *phi;      // DEVICE [T][8]: (1, x, y, x^2, y^2, xy, 0, 0) of the jitter
    const int32_t *bi0;    // DEVICE [N]: first input pixel of output pixel i (bilinear_table)
    const float *bw;       // DEVICE [N]: weight of the second input pixel
    const int32_t *blo, *bhi;   // DEVICE [n]: first and last output pixel whose stencil touches input pixel b
    float delta;
};
void bilinear_table(int32_t N, int32_t n, int32_t *i0, float *w);      // host
void launch_downsample(cudaStream_t st, const float *frames, int32_t T, int32_t H, int32_t W, int32_t f, float *out);
void launch_scatter_subtract(cudaStream_t st, float *frames, int32_t T, int32_t H, int32_t W, const float *S, int32_t n,
                             const int32_t *yi0, const float *yw, const int32_t *xi0, const float *xw);
// launches only; returns the number of kernels launched
int32_t scatter_lossgrad(cudaStream_t st, const ScatterProblem &pb, const float *beta, const float *S, float *psi,
                         double *partials, float *g_beta, float *g_S, double *loss_dev);
size_t scatter_ws_bytes(int32_t T, int32_t N, int32_t n);
// beta, S: DEVICE, start point in, minimiser out; synchronises the stream; returns 0 or a cudaError_t
int32_t scatter_fit(cudaStream_t st, const ScatterProblem &pb, float *beta, float *S, void *ws, int32_t max_iter,
                    float gtol, double *out_loss, int32_t *out_iters, int32_t *out_evals, int32_t *out_launches);

// ---- inject.cu ----
struct SourceDev { float vx, vy, ax, ay; int32_t x, y; float amp; };
void launch_inject(cudaStream_t st, float *frames, int32_t T, int32_t H, int32_t W,
                   const SourceDev *src, int32_t n_src, double prf_sigma, double t0, int32_t filter,
                   const float *prf_tab, int32_t n_phase, const float *times /* DEVICE [T] or NULL */,
                   const float *jitter /* DEVICE [T][2] or NULL */);

// ---- search_sep.cu ----
struct SepVariant {
    int32_t nb;           // slots per batch (a slot = a y-motion and its mirror image, plan.h)
    int32_t tile_h;       // positions (frame rows) per tile; the tile width is 64 columns
    int32_t rows;         // positions per consumer thread
};
int32_t sep_num_variants();
SepVariant sep_variant(int32_t v);
// per-(batch, frame) stage table size in 32-bit words
int32_t sep_table_words(int32_t v);
// tile rows of the position space [-2, H + 2)
int32_t sep_tile_rows(int32_t v, int32_t H);
void launch_sep_tables(cudaStream_t st, int32_t v, const ClassTables &tab, const int32_t *batch_xc,
                       const int32_t *slot_yc /* [n_batches][nb] y-class of the slot's tables, -1 = empty */,
                       const int32_t *slot_flip /* [n_batches][nb] 1: that class is the slot's mirror image */,
                       const int32_t *slot_q /* [n_batches][nb][2] planned index of the plus / minus member
                                                relative to the batch's first, -1 = absent */,
                       int32_t n_batches, int32_t squared /* 1: taps g^2 (D pass of the masked search) */,
                       float *stage_tab);
struct SepArgs {
    const float *frames;
    int32_t T, H, W;
    const float *stage_tab;       // [n_batches][T][table_words], first batch of the chunk
    const int32_t *batch_q;       // [n_batches] planned-order index q of the first member of each batch
    int32_t n_batches;            // batches of the chunk
    int32_t q0;                   // first planned-order index of the chunk
    float *pieces;                // [n_pieces][chunk entries][H][W] partial sums, zero on entry
    int64_t piece_stride;         // floats between pieces = chunk entries * H * W
    int32_t n_pieces;
    int32_t n_sm;
    int32_t ty0 = 0, ty1 = 0;     // tile rows [ty0, ty1) of the position space; ty1 = 0: up to the last one
};
// returns cudaError_t-like code (0 ok); *grid_out = number of CTAs used
int launch_search_sep(cudaStream_t st, int32_t v, const SepArgs &a, void *encode_fn, int32_t *grid_out,
                      const char **err);
// SNR = (sum of pieces) * D^(-1/2) for entries q0 .. q0 + q_count of the planned order (perm[q] =
// trajectory); maps to out_snr (may be NULL), candidates to the 64 x 64 tile slots (keys may be NULL)
// dpieces != NULL (masked search): SNR = (sum of pieces) / sqrt(sum of dpieces), 0 where that is 0
void launch_finish(cudaStream_t st, const float *pieces, const float *dpieces, int32_t n_pieces, int64_t piece_stride,
                   const int32_t *perm, int32_t q0, int32_t q_count, const TrajInfo *traj, const float *rsd,
                   int32_t H, int32_t W, int32_t fy0, int32_t fy1 /* rows of 64 x 64 tiles [fy0, fy1) */,
                   float *out_snr, uint64_t *maxkeys /* DEVICE [H][W] running (score, ~k) maximum, or NULL */,
                   const TopkSlots &slots);

// ---- api.cu: the opaque context as seen by an entry point in another file (local_z_static.cu) ----
struct CtxView { cudaStream_t stream; int32_t device; };
CtxView ctx_view(const tno_mf_ctx *ctx);
int ctx_fail(tno_mf_ctx *ctx, int code, const char *text);      // sets tno_mf_last_error(ctx), returns code
void ctx_set_launches(tno_mf_ctx *ctx, int32_t n);              // what tno_mf_last_stats reports

}  // namespace tno
