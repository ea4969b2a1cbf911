// Launch wrappers of the kernels in libtno_mf.so (all enqueue on the given stream, no syncs).
#pragma once
#include <cuda.h>

#include "../../include/tno_mf.h"
#include "common.cuh"

namespace tno {

// ---- tables.cu ----
void launch_class_tables(cudaStream_t st, const float *cls_v, const float *cls_a, int32_t n_cls,
                         int32_t T, double t0, double prf_sigma, int32_t *shift, float *g,
                         double *gd);
void launch_border_tables(cudaStream_t st, const int32_t *shift, const double *gd, const double *qd,
                          const AxisBorder *border, const int64_t *off, int32_t n_cls, int32_t n_x,
                          int32_t max_n, int32_t T, int32_t W, int32_t H, double *out);
void launch_rsd_tables(cudaStream_t st, const TrajInfo *traj, int32_t n_traj, int64_t max_cells,
                       const double *ab, const int64_t *off, int32_t n_x, int32_t T, float *rsd);

// ---- search_generic.cu ----
// One thread per (trajectory, pixel); any H, W; maps only.
void launch_search_generic(cudaStream_t st, const float *frames, int32_t T, int32_t H, int32_t W,
                           const ClassTables &tab, const TrajInfo *traj, const float *rsd,
                           int32_t k_first, int32_t k_count, float *out_snr /* [k_count][H][W] */);

// ---- topk.cu ----
constexpr int32_t kCollectTile = 64;        // k_collect_from_map tiles are 64 x 64 pixels
constexpr int32_t kMaxTopk = 1024;
// candidates of maps [k_count][H][W] (trajectories k_first..) into tile slots
void launch_collect_from_map(cudaStream_t st, const float *maps, int32_t H, int32_t W,
                             int32_t k_first, int32_t k_count, const TopkSlots &slots);
// merge all tile slots of every trajectory into out_topk[K][ktop]
void launch_topk_merge(cudaStream_t st, const TopkSlots &slots, int32_t n_tiles, int32_t W,
                       tno_mf_cand *out_topk);

// ---- inject.cu ----
struct SourceDev { float vx, vy, ax, ay; int32_t x, y; float amp; };
void launch_inject(cudaStream_t st, float *frames, int32_t T, int32_t H, int32_t W,
                   const SourceDev *src, int32_t n_src, double prf_sigma, double t0);

// ---- search_sep.cu ----
struct SepVariant {
    int32_t nb;           // entries per batch
    int32_t tile_h;       // output tile height (tile width is 64)
    int32_t max_spread;   // largest y-shift spread a batch may have
};
int32_t sep_num_variants();
SepVariant sep_variant(int32_t v);
// per-(batch, frame) stage table size in 32-bit words for variant v
int32_t sep_table_words(int32_t v);
void launch_sep_tables(cudaStream_t st, int32_t v, const ClassTables &tab, const int32_t *batch_xc,
                       const int32_t *batch_yc /* [n_batches][nb], -1 = empty */, int32_t n_batches,
                       float *stage_tab);
struct SepArgs {
    const float *frames;
    int32_t T, H, W;
    const float *stage_tab;       // [n_batches][T][table_words]
    const int32_t *batch_traj;    // [n_batches][nb] trajectory index or -1
    int32_t n_batches;
    const TrajInfo *traj;
    const float *rsd;
    float *out_snr;               // may be NULL
    TopkSlots slots;              // slots.keys may be NULL
    float *scratch;               // [grid][tile_h*64*nb] partial sums
    int32_t n_sm;
};
// returns cudaError_t-like code (0 ok); *grid_out = number of CTAs used
int launch_search_sep(cudaStream_t st, int32_t v, const SepArgs &a, void *encode_fn, int32_t *grid_out,
                      const char **err);
size_t sep_scratch_floats_per_cta(int32_t v);

}  // namespace tno
