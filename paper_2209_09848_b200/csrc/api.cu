// C ABI of libtno_mf.so (include/tno_mf.h): context, validation, planning, launches.
#include <cfloat>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "kernels.h"
#include "plan.h"

using namespace tno;

namespace {

thread_local std::string g_create_error = "";

struct DevBuf {
    void *p = nullptr;
    size_t cap = 0;
};

}  // namespace

struct tno_mf_ctx {
    tno_mf_config cfg;
    cudaStream_t stream = nullptr;
    int32_t n_sm = 0;
    void *encode_fn = nullptr;
    std::string err;
    int32_t last_launches = 0, last_kernel = 0;
    // host-fed search (tno_mf_search_host): rows [0, fed_rows) of every frame are on the device
    const float *feed_host = nullptr, *feed_host2 = nullptr;      // feed_host2: the validity weights of a masked search
    float *feed_dev = nullptr, *feed_dev2 = nullptr;
    int32_t fed_rows = 0, feed_T = 0, feed_H = 0, feed_W = 0;
    cudaStream_t copy_stream = nullptr, down_stream = nullptr;
    cudaEvent_t copy_ev = nullptr, start_ev = nullptr, fin_ev = nullptr;
    float *down_host = nullptr;       // host maps of tno_mf_search_host (NULL: no maps wanted)
    const float *down_dev = nullptr;
    int32_t down_rows = 0, down_K = 0;   // rows [0, down_rows) of every map are on their way to the host
    DevBuf stack, stack2, hmaps, htopk, hmax, bgq, prf_tab, prf_tab2, maxkeys, scat;
    int32_t prf_phases = 0;          // rows of prf_tab (tno_mf_set_prf_table), 0 = none
    int32_t prf2_py = 0, prf2_px = 0;   // phases of prf_tab2 (tno_mf_set_prf_table2d), 0 = none
    // geometry and tables of the last successful search (for tno_mf_flux)
    int32_t s_traj = 0, s_H = 0, s_W = 0;
    const TrajInfo *s_ti = nullptr;
    double last_fma_x = 0.0, last_fma_y = 0.0, last_add_y = 0.0;
    std::vector<cudaEvent_t> ev;      // pairs (before, after) around each main search kernel launch
    int32_t ev_used = 0;              // events recorded by the last search
    // grow-only device workspace
    DevBuf meta, shift, g, gd, ab, rsd, stage_tab, pieces, keys, counts, tmp_maps, src, sat, ztmp;
};

namespace {

int fail(tno_mf_ctx *ctx, int code, const char *fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx) ctx->err = buf; else g_create_error = buf;
    return code;
}

#define CU_TRY(ctx, expr)                                                                   \
    do {                                                                                    \
        cudaError_t e_ = (expr);                                                            \
        if (e_ != cudaSuccess)                                                              \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? TNO_MF_ENOMEM : TNO_MF_ECUDA, \
                        "%s: %s", #expr, cudaGetErrorString(e_));                           \
    } while (0)

// Debug aid (environment variable TNO_MF_POISON_WORKSPACE=1): every workspace buffer is filled with 0xff bytes -- NaN
// as floats, -1 as integers -- when it is allocated, so that a kernel that reads workspace it never wrote shows in the
// tests instead of computing with whatever the allocator handed out (profiles/r2_sanitizers.md).
bool poison_workspace() {
    static const bool on = [] { const char *v = getenv("TNO_MF_POISON_WORKSPACE"); return v && v[0] == '1'; }();
    return on;
}

// Grow-only buffer.  cudaFree synchronises the device, so replacing a buffer that earlier work on
// the stream may still read is safe.
int reserve(tno_mf_ctx *ctx, DevBuf &b, size_t bytes) {
    if (bytes <= b.cap) return TNO_MF_OK;
    if (b.p) { cudaFree(b.p); b.p = nullptr; b.cap = 0; }
    const size_t want = bytes + bytes / 8 + 256;
    cudaError_t e = cudaMalloc(&b.p, want);
    if (e != cudaSuccess) {
        cudaGetLastError();
        e = cudaMalloc(&b.p, bytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            b.p = nullptr;
            return fail(ctx, TNO_MF_ENOMEM, "device allocation of %zu bytes failed: %s", bytes,
                        cudaGetErrorString(e));
        }
        b.cap = bytes;
    } else {
        b.cap = want;
    }
    if (poison_workspace()) {
        cudaMemset(b.p, 0xff, b.cap);
        cudaDeviceSynchronize();
    }
    return TNO_MF_OK;
}

// host blob with 16-byte aligned sections, uploaded with one copy
struct Blob {
    std::vector<unsigned char> bytes;
    size_t add(const void *src, size_t n) {
        const size_t off = (bytes.size() + 15) & ~(size_t)15;
        bytes.resize(off + n);
        if (n) memcpy(bytes.data() + off, src, n);
        return off;
    }
};

AxisBorder make_border(const AxisClass &c, int32_t L) {
    AxisBorder b;
    b.lo = std::max(0, 2 - c.smin);
    b.hi = std::max(0, c.smax + 2);
    // lo/hi larger than the axis mean every pixel is clipped somewhere: fall back to identity
    if ((int64_t)b.lo + 1 + (int64_t)b.hi >= (int64_t)L) {
        b.identity = 1;
        b.n = L;
        b.lo = b.hi = 0;
    } else {
        b.identity = 0;
        b.n = b.lo + 1 + b.hi;
    }
    return b;
}

bool finite_f(float v) { return std::isfinite(v); }

// Record the next event of the (before, after) pairs that bracket the main search kernels.
int record_event(tno_mf_ctx *ctx) {
    if (!ctx->cfg.record_events) return TNO_MF_OK;
    if (ctx->ev_used == (int32_t)ctx->ev.size()) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) {
            cudaGetLastError();
            return fail(ctx, TNO_MF_ECUDA, "cudaEventCreate failed");
        }
        ctx->ev.push_back(e);
    }
    if (cudaEventRecord(ctx->ev[ctx->ev_used], ctx->stream) != cudaSuccess) {
        cudaGetLastError();
        return fail(ctx, TNO_MF_ECUDA, "cudaEventRecord failed");
    }
    ++ctx->ev_used;
    return TNO_MF_OK;
}

// Host-fed search: upload the rows [fed_rows, r_end) of every frame (one strided 2-D copy on the copy
// stream) and make the compute stream wait for them.  No-op for a device-resident stack.
int feed_rows(tno_mf_ctx *ctx, int32_t r_end) {
    if (!ctx->feed_host) return TNO_MF_OK;
    r_end = std::min(r_end, ctx->feed_H);
    if (r_end <= ctx->fed_rows) return TNO_MF_OK;
    const size_t pitch = (size_t)ctx->feed_H * ctx->feed_W * 4, off = (size_t)ctx->fed_rows * ctx->feed_W;
    CU_TRY(ctx, cudaMemcpy2DAsync(ctx->feed_dev + off, pitch, ctx->feed_host + off, pitch,
                                  (size_t)(r_end - ctx->fed_rows) * ctx->feed_W * 4, (size_t)ctx->feed_T,
                                  cudaMemcpyHostToDevice, ctx->copy_stream));
    if (ctx->feed_host2)
        CU_TRY(ctx, cudaMemcpy2DAsync(ctx->feed_dev2 + off, pitch, ctx->feed_host2 + off, pitch,
                                      (size_t)(r_end - ctx->fed_rows) * ctx->feed_W * 4, (size_t)ctx->feed_T,
                                      cudaMemcpyHostToDevice, ctx->copy_stream));
    CU_TRY(ctx, cudaEventRecord(ctx->copy_ev, ctx->copy_stream));
    CU_TRY(ctx, cudaStreamWaitEvent(ctx->stream, ctx->copy_ev, 0));
    ctx->fed_rows = r_end;
    return TNO_MF_OK;
}

// Host-fed search: once the rows [down_rows, r_end) of all maps are final on the compute stream, send them
// to the host on the download stream (PCIe is full duplex: this overlaps the upload of later bands).
int download_rows(tno_mf_ctx *ctx, int32_t r_end) {
    if (!ctx->down_host) return TNO_MF_OK;
    r_end = std::min(r_end, ctx->feed_H);
    if (r_end <= ctx->down_rows) return TNO_MF_OK;
    const size_t pitch = (size_t)ctx->feed_H * ctx->feed_W * 4, off = (size_t)ctx->down_rows * ctx->feed_W;
    CU_TRY(ctx, cudaEventRecord(ctx->fin_ev, ctx->stream));
    CU_TRY(ctx, cudaStreamWaitEvent(ctx->down_stream, ctx->fin_ev, 0));
    CU_TRY(ctx, cudaMemcpy2DAsync(ctx->down_host + off, pitch, ctx->down_dev + off, pitch,
                                  (size_t)(r_end - ctx->down_rows) * ctx->feed_W * 4, (size_t)ctx->down_K,
                                  cudaMemcpyDeviceToHost, ctx->down_stream));
    ctx->down_rows = r_end;
    return TNO_MF_OK;
}

}  // namespace

extern "C" {

const char *tno_mf_version(void) { return "tno_mf 0.1 (sm_100a)"; }

const char *tno_mf_last_error(const tno_mf_ctx *ctx) {
    return ctx ? ctx->err.c_str() : g_create_error.c_str();
}

int tno_mf_create(const tno_mf_config *cfg, tno_mf_ctx **out_ctx) {
    if (!cfg || !out_ctx) return fail(nullptr, TNO_MF_EINVAL, "tno_mf_create: NULL argument");
    *out_ctx = nullptr;
    if (cfg->topk < 0 || cfg->topk > kMaxTopk)
        return fail(nullptr, TNO_MF_EINVAL, "tno_mf_create: topk must be in [0, %d]", kMaxTopk);
    if (std::isnan(cfg->snr_threshold))
        return fail(nullptr, TNO_MF_EINVAL, "tno_mf_create: snr_threshold is NaN");
    if (cfg->filter < 0 || cfg->filter > 4 || cfg->workspace_limit_mb < 0 || cfg->sep_shape < 0 ||
        cfg->sep_shape > sep_num_variants())
        return fail(nullptr, TNO_MF_EINVAL, "tno_mf_create: filter must be 0 .. 4, workspace_limit_mb >= 0, sep_shape 0 .. %d",
                    sep_num_variants());
    int n_dev = 0;
    cudaError_t e = cudaGetDeviceCount(&n_dev);
    if (e != cudaSuccess || n_dev == 0) {
        cudaGetLastError();
        return fail(nullptr, TNO_MF_EUNSUPPORTED, "tno_mf_create: no CUDA device (%s); there is no CPU fallback",
                    e != cudaSuccess ? cudaGetErrorString(e) : "device count 0");
    }
    if (cfg->device < 0 || cfg->device >= n_dev)
        return fail(nullptr, TNO_MF_EINVAL, "tno_mf_create: device %d out of range [0, %d)", cfg->device, n_dev);
    cudaDeviceProp prop;
    CU_TRY(nullptr, cudaGetDeviceProperties(&prop, cfg->device));
    if (prop.major != 10)
        return fail(nullptr, TNO_MF_EUNSUPPORTED,
                    "tno_mf_create: device %d is sm_%d%d; this library is built for sm_100a only",
                    cfg->device, prop.major, prop.minor);
    CU_TRY(nullptr, cudaSetDevice(cfg->device));
    tno_mf_ctx *ctx = new (std::nothrow) tno_mf_ctx();
    if (!ctx) return fail(nullptr, TNO_MF_ENOMEM, "tno_mf_create: out of host memory");
    ctx->cfg = *cfg;
    ctx->stream = reinterpret_cast<cudaStream_t>(cfg->stream);
    ctx->n_sm = prop.multiProcessorCount;
    cudaDriverEntryPointQueryResult qres;
    e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ctx->encode_fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !ctx->encode_fn) {
        cudaGetLastError();
        delete ctx;
        return fail(nullptr, TNO_MF_ECUDA, "tno_mf_create: cuTensorMapEncodeTiled not available in the driver");
    }
    *out_ctx = ctx;
    return TNO_MF_OK;
}

int tno_mf_last_kernel_ms(tno_mf_ctx *ctx, float *out_ms) {
    if (!ctx || !out_ms) return TNO_MF_EINVAL;
    if (ctx->ev_used < 2)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_last_kernel_ms: no recorded search (cfg.record_events = 0?)");
    float total = 0.f;
    for (int32_t i = 0; i + 1 < ctx->ev_used; i += 2) {
        float ms = 0.f;
        CU_TRY(ctx, cudaEventSynchronize(ctx->ev[i + 1]));
        CU_TRY(ctx, cudaEventElapsedTime(&ms, ctx->ev[i], ctx->ev[i + 1]));
        total += ms;
    }
    *out_ms = total;
    return TNO_MF_OK;
}

int tno_mf_last_work(const tno_mf_ctx *ctx, double *out_fma_xpass, double *out_fma_ypass, double *out_add_ypass) {
    if (!ctx) return TNO_MF_EINVAL;
    if (out_fma_xpass) *out_fma_xpass = ctx->last_fma_x;
    if (out_fma_ypass) *out_fma_ypass = ctx->last_fma_y;
    if (out_add_ypass) *out_add_ypass = ctx->last_add_y;
    return TNO_MF_OK;
}

int tno_mf_destroy(tno_mf_ctx *ctx) {
    if (!ctx) return TNO_MF_OK;
    cudaSetDevice(ctx->cfg.device);
    DevBuf *bufs[] = {&ctx->meta, &ctx->shift, &ctx->g, &ctx->gd, &ctx->ab, &ctx->rsd, &ctx->stage_tab,
                      &ctx->pieces, &ctx->keys, &ctx->counts, &ctx->tmp_maps, &ctx->src, &ctx->sat, &ctx->ztmp,
                      &ctx->stack, &ctx->stack2, &ctx->hmaps, &ctx->htopk, &ctx->hmax, &ctx->bgq, &ctx->prf_tab,
                      &ctx->prf_tab2, &ctx->maxkeys, &ctx->scat};
    for (DevBuf *b : bufs)
        if (b->p) cudaFree(b->p);
    for (cudaEvent_t e : ctx->ev) cudaEventDestroy(e);
    if (ctx->copy_ev) cudaEventDestroy(ctx->copy_ev);
    if (ctx->start_ev) cudaEventDestroy(ctx->start_ev);
    if (ctx->fin_ev) cudaEventDestroy(ctx->fin_ev);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->down_stream) cudaStreamDestroy(ctx->down_stream);
    delete ctx;
    return TNO_MF_OK;
}

int tno_mf_last_stats(const tno_mf_ctx *ctx, int32_t *out_launches, int32_t *out_kernel) {
    if (!ctx) return TNO_MF_EINVAL;
    if (out_launches) *out_launches = ctx->last_launches;
    if (out_kernel) *out_kernel = ctx->last_kernel;
    return TNO_MF_OK;
}

int tno_mf_plan(const tno_mf_traj *trajectories, int32_t n_traj, int32_t T, float t0,
                int32_t max_entries, int32_t max_spread, int32_t *out_batch, int32_t *out_slot) {
    if (!trajectories || n_traj < 1 || T < 1 || max_entries < 1 || max_entries > 16 || max_spread < 0 ||
        !finite_f(t0))
        return TNO_MF_EINVAL;
    for (int32_t k = 0; k < n_traj; ++k)
        if (!finite_f(trajectories[k].vx) || !finite_f(trajectories[k].vy) ||
            !finite_f(trajectories[k].ax) || !finite_f(trajectories[k].ay))
            return TNO_MF_EINVAL;
    Plan plan;
    const int rc = build_classes(trajectories, n_traj, T, (double)t0, nullptr, nullptr, &plan);
    if (rc != TNO_MF_OK) return rc;
    build_batches(&plan, max_entries, max_spread);
    for (size_t b = 0; b < plan.batches.size(); ++b)
        for (size_t s = 0; s < plan.batches[b].traj.size(); ++s) {
            if (out_batch) out_batch[plan.batches[b].traj[s]] = (int32_t)b;
            if (out_slot) out_slot[plan.batches[b].traj[s]] = (int32_t)s;
        }
    return (int)plan.batches.size();
}

int tno_mf_plan_slots(const tno_mf_traj *trajectories, int32_t n_traj, int32_t T, float t0, const float *frame_times,
                      const float *jitter_xy, int32_t max_slots, int32_t symmetric_filter, int32_t *out_batch,
                      int32_t *out_slot, int32_t *out_member) {
    if (!trajectories || n_traj < 1 || T < 1 || max_slots < 1 || max_slots > 16 || !finite_f(t0))
        return TNO_MF_EINVAL;
    for (int32_t k = 0; k < n_traj; ++k)
        if (!finite_f(trajectories[k].vx) || !finite_f(trajectories[k].vy) ||
            !finite_f(trajectories[k].ax) || !finite_f(trajectories[k].ay))
            return TNO_MF_EINVAL;
    for (int32_t t = 0; t < T; ++t)
        if ((frame_times && !finite_f(frame_times[t])) ||
            (jitter_xy && (!finite_f(jitter_xy[2 * t]) || !finite_f(jitter_xy[2 * t + 1]))))
            return TNO_MF_EINVAL;
    Plan plan;
    const int rc = build_classes(trajectories, n_traj, T, (double)t0, frame_times, jitter_xy, &plan);
    if (rc != TNO_MF_OK) return rc;
    build_slot_batches(&plan, max_slots, symmetric_filter != 0);
    for (size_t b = 0; b < plan.slot_batches.size(); ++b)
        for (size_t s = 0; s < plan.slot_batches[b].slots.size(); ++s)
            for (int m = 0; m < 2; ++m) {
                const int32_t k = plan.slot_batches[b].slots[s].member[m];
                if (k < 0) continue;
                if (out_batch) out_batch[k] = (int32_t)b;
                if (out_slot) out_slot[k] = (int32_t)s;
                if (out_member) out_member[k] = m;
            }
    return (int)plan.slot_batches.size();
}

// ---- low-resolution scattered-light model (section 3.1) -------------------------------------------------
static int scatter_setup(tno_mf_ctx *ctx, const char *who, const float *D, int32_t T, int32_t N, int32_t n,
                         const float *jitter_xy, float delta, const float *beta, const float *S, size_t extra_bytes,
                         ScatterProblem *pb, unsigned char **ws) {
    if (!D || !jitter_xy || !beta || !S) return fail(ctx, TNO_MF_EINVAL, "%s: NULL pointer", who);
    if (T < 1 || N < 1 || n < 1 || n > N || (int64_t)T * N * N > ((int64_t)1 << 40))
        return fail(ctx, TNO_MF_EINVAL, "%s: need T >= 1 and 1 <= n <= N", who);
    if (!(delta > 0.f) || std::isnan(delta)) return fail(ctx, TNO_MF_EINVAL, "%s: delta must be > 0", who);
    std::vector<float> phi((size_t)T * 8, 0.f);
    for (int32_t t = 0; t < T; ++t) {
        const double x = jitter_xy[2 * t], y = jitter_xy[2 * t + 1];
        if (!finite_f(jitter_xy[2 * t]) || !finite_f(jitter_xy[2 * t + 1]))
            return fail(ctx, TNO_MF_EINVAL, "%s: jitter_xy[%d] is not finite", who, t);
        float *row = &phi[(size_t)t * 8];
        row[0] = 1.f; row[1] = (float)x; row[2] = (float)y; row[3] = (float)(x * x); row[4] = (float)(y * y);
        row[5] = (float)(x * y);
    }
    CU_TRY(ctx, cudaSetDevice(ctx->cfg.device));
    int rc;
    // one upload: phi [T][8] floats, then the bilinear table (first input pixel [N] int32, weight [N] float)
    const size_t phi_words = (size_t)T * 8;
    std::vector<int32_t> head(phi_words + 2 * (size_t)N + 2 * (size_t)n);
    std::memcpy(head.data(), phi.data(), phi_words * 4);
    int32_t *hi0 = head.data() + phi_words, *hlo = hi0 + 2 * (size_t)N, *hhi = hlo + n;
    bilinear_table(N, n, hi0, reinterpret_cast<float *>(hi0 + N));
    for (int32_t b = 0; b < n; ++b) { hlo[b] = N; hhi[b] = -1; }
    for (int32_t i = 0; i < N; ++i)
        for (int32_t b : {hi0[i], std::min(hi0[i] + 1, n - 1)}) {
            hlo[b] = std::min(hlo[b], i);
            hhi[b] = std::max(hhi[b], i);
        }
    const size_t phi_bytes = (head.size() * 4 + 255) & ~(size_t)255;
    if ((rc = reserve(ctx, ctx->scat, phi_bytes + extra_bytes))) return rc;
    unsigned char *base = static_cast<unsigned char *>(ctx->scat.p);
    CU_TRY(ctx, cudaMemcpyAsync(base, head.data(), head.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));      // head is a local buffer
    pb->D = D; pb->T = T; pb->N = N; pb->n = n; pb->phi = reinterpret_cast<const float *>(base); pb->delta = delta;
    pb->bi0 = reinterpret_cast<const int32_t *>(base) + phi_words;
    pb->bw = reinterpret_cast<const float *>(base) + phi_words + N;
    pb->blo = pb->bi0 + 2 * (size_t)N;
    pb->bhi = pb->blo + n;
    *ws = base + phi_bytes;
    return TNO_MF_OK;
}

int tno_mf_scatter_lossgrad(tno_mf_ctx *ctx, const float *D, int32_t T, int32_t N, int32_t n, const float *jitter_xy,
                            float delta, const float *beta, const float *S, double *out_loss, float *g_beta,
                            float *g_S) {
    if (!ctx) return TNO_MF_EINVAL;
    ctx->last_launches = 0;
    if (!out_loss || !g_beta || !g_S) return fail(ctx, TNO_MF_EINVAL, "tno_mf_scatter_lossgrad: NULL output");
    ScatterProblem pb;
    unsigned char *ws = nullptr;
    const size_t blocks = std::max<size_t>(8192, ((size_t)N * N + 255) / 256);       // kLossPartials of scatter.cu
    const size_t psi_bytes = ((size_t)T * N * N * 4 + 255) & ~(size_t)255;
    int rc = scatter_setup(ctx, "tno_mf_scatter_lossgrad", D, T, N, n, jitter_xy, delta, beta, S,
                           psi_bytes + (blocks + 8) * 8, &pb, &ws);
    if (rc) return rc;
    double *partials = reinterpret_cast<double *>(ws + psi_bytes);
    ctx->last_launches = scatter_lossgrad(ctx->stream, pb, beta, S, reinterpret_cast<float *>(ws), partials, g_beta, g_S,
                                          partials + blocks);
    CU_TRY(ctx, cudaMemcpyAsync(out_loss, partials + blocks, 8, cudaMemcpyDeviceToHost, ctx->stream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    CU_TRY(ctx, cudaGetLastError());
    return TNO_MF_OK;
}

int tno_mf_scatter_fit(tno_mf_ctx *ctx, const float *D, int32_t T, int32_t N, int32_t n, const float *jitter_xy,
                       float delta, int32_t max_iter, float gtol, float *beta, float *S, double *out_loss,
                       int32_t *out_iters, int32_t *out_evals) {
    if (!ctx) return TNO_MF_EINVAL;
    ctx->last_launches = 0;
    if (max_iter < 0 || !(gtol >= 0.f)) return fail(ctx, TNO_MF_EINVAL, "tno_mf_scatter_fit: max_iter, gtol must be >= 0");
    ScatterProblem pb;
    unsigned char *ws = nullptr;
    int rc = scatter_setup(ctx, "tno_mf_scatter_fit", D, T, N, n, jitter_xy, delta, beta, S,
                           scatter_ws_bytes(T, N, n), &pb, &ws);
    if (rc) return rc;
    double loss = 0.0;
    int32_t iters = 0, evals = 0, launches = 0;
    const int32_t e = scatter_fit(ctx->stream, pb, beta, S, ws, max_iter, gtol, &loss, &iters, &evals, &launches);
    ctx->last_launches = launches;
    if (e != 0) return fail(ctx, TNO_MF_ECUDA, "tno_mf_scatter_fit: %s", cudaGetErrorString((cudaError_t)e));
    if (out_loss) *out_loss = loss;
    if (out_iters) *out_iters = iters;
    if (out_evals) *out_evals = evals;
    return TNO_MF_OK;
}

int tno_mf_downsample(tno_mf_ctx *ctx, const float *frames, int32_t T, int32_t H, int32_t W, int32_t factor,
                      float *out) {
    if (!ctx) return TNO_MF_EINVAL;
    if (!frames || !out) return fail(ctx, TNO_MF_EINVAL, "tno_mf_downsample: NULL pointer");
    if (T < 1 || T > 65535 || H < 1 || W < 1 || factor < 1 || H % factor || W % factor || H / factor > kMaxRows)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_downsample: need 1 <= T <= 65535, factor dividing H and W, and "
                    "H / factor <= %d", kMaxRows);
    CU_TRY(ctx, cudaSetDevice(ctx->cfg.device));
    launch_downsample(ctx->stream, frames, T, H, W, factor, out);
    ctx->last_launches = 1;
    CU_TRY(ctx, cudaGetLastError());
    return TNO_MF_OK;
}

int tno_mf_scatter_subtract(tno_mf_ctx *ctx, float *frames, int32_t T, int32_t H, int32_t W, const float *S,
                            int32_t n) {
    if (!ctx) return TNO_MF_EINVAL;
    if (!frames || !S) return fail(ctx, TNO_MF_EINVAL, "tno_mf_scatter_subtract: NULL pointer");
    if (T < 1 || T > 65535 || H < 1 || H > kMaxRows || W < 1 || n < 1 || n > H || n > W)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_scatter_subtract: need 1 <= T <= 65535, H <= %d and 1 <= n <= min(H, W)",
                    kMaxRows);
    CU_TRY(ctx, cudaSetDevice(ctx->cfg.device));
    std::vector<int32_t> tabs(2 * ((size_t)H + W));          // y: first pixel [H], weight [H]; x: the same [W]
    bilinear_table(H, n, tabs.data(), reinterpret_cast<float *>(tabs.data() + H));
    bilinear_table(W, n, tabs.data() + 2 * H, reinterpret_cast<float *>(tabs.data() + 2 * H + W));
    int rc = reserve(ctx, ctx->scat, tabs.size() * 4);
    if (rc) return rc;
    CU_TRY(ctx, cudaMemcpyAsync(ctx->scat.p, tabs.data(), tabs.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));      // tabs is a local buffer
    const int32_t *d = static_cast<const int32_t *>(ctx->scat.p);
    launch_scatter_subtract(ctx->stream, frames, T, H, W, S, n, d, reinterpret_cast<const float *>(d + H), d + 2 * H,
                            reinterpret_cast<const float *>(d + 2 * H + W));
    ctx->last_launches = 1;
    CU_TRY(ctx, cudaGetLastError());
    return TNO_MF_OK;
}

int tno_mf_set_prf_table(tno_mf_ctx *ctx, const float *table, int32_t n_phase) {
    if (!ctx) return TNO_MF_EINVAL;
    if (n_phase < 0 || n_phase > (1 << 20) || (n_phase > 0 && !table))
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_set_prf_table: n_phase must be in [0, 2^20] and table non-NULL");
    for (int64_t i = 0; i < (int64_t)n_phase * 5; ++i)
        if (!finite_f(table[i]) || table[i] < 0.f)
            return fail(ctx, TNO_MF_EINVAL, "tno_mf_set_prf_table: table[%lld] is negative or not finite", (long long)i);
    CU_TRY(ctx, cudaSetDevice(ctx->cfg.device));
    ctx->prf_phases = 0;
    if (n_phase == 0) return TNO_MF_OK;
    int rc = reserve(ctx, ctx->prf_tab, (size_t)n_phase * 5 * sizeof(float));
    if (rc) return rc;
    // the caller's buffer may go away after the call
    CU_TRY(ctx, cudaMemcpyAsync(ctx->prf_tab.p, table, (size_t)n_phase * 5 * sizeof(float), cudaMemcpyHostToDevice,
                                ctx->stream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->prf_phases = n_phase;
    return TNO_MF_OK;
}

int tno_mf_set_prf_table2d(tno_mf_ctx *ctx, const float *table, int32_t n_phase_y, int32_t n_phase_x) {
    if (!ctx) return TNO_MF_EINVAL;
    if (n_phase_y < 0 || n_phase_x < 0 || n_phase_y > 4096 || n_phase_x > 4096 || (n_phase_y == 0) != (n_phase_x == 0) ||
        (n_phase_y > 0 && !table))
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_set_prf_table2d: phases must be in [0, 4096], both zero or both "
                    "positive, and table non-NULL");
    const int64_t n = (int64_t)n_phase_y * n_phase_x * 25;
    for (int64_t i = 0; i < n; ++i)
        if (!finite_f(table[i]) || table[i] < 0.f)
            return fail(ctx, TNO_MF_EINVAL, "tno_mf_set_prf_table2d: table[%lld] is negative or not finite", (long long)i);
    CU_TRY(ctx, cudaSetDevice(ctx->cfg.device));
    ctx->prf2_py = ctx->prf2_px = 0;
    if (n == 0) return TNO_MF_OK;
    int rc = reserve(ctx, ctx->prf_tab2, (size_t)n * sizeof(float));
    if (rc) return rc;
    // the caller's buffer may go away after the call
    CU_TRY(ctx, cudaMemcpyAsync(ctx->prf_tab2.p, table, (size_t)n * sizeof(float), cudaMemcpyHostToDevice, ctx->stream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->prf2_py = n_phase_y;
    ctx->prf2_px = n_phase_x;
    return TNO_MF_OK;
}

int tno_mf_inject(tno_mf_ctx *ctx, float *frames, int32_t T, int32_t H, int32_t W,
                  const tno_mf_source *sources, int32_t n_sources, float prf_sigma, float t0) {
    return tno_mf_inject_ex(ctx, frames, T, H, W, nullptr, nullptr, sources, n_sources, prf_sigma, t0);
}

int tno_mf_inject_ex(tno_mf_ctx *ctx, float *frames, int32_t T, int32_t H, int32_t W, const float *frame_times,
                     const float *jitter_xy, const tno_mf_source *sources, int32_t n_sources, float prf_sigma,
                     float t0) {
    if (!ctx) return TNO_MF_EINVAL;
    if (!frames || !sources || T < 1 || H < 1 || W < 1 || n_sources < 0)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_inject: NULL pointer or non-positive size");
    if (!(prf_sigma > 0.f) || !finite_f(prf_sigma) || !finite_f(t0))
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_inject: prf_sigma must be finite and > 0, t0 finite");
    if (ctx->cfg.filter == 3 && ctx->prf_phases == 0)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_inject: filter 3 needs a table (tno_mf_set_prf_table)");
    if (ctx->cfg.filter == 4 && ctx->prf2_py == 0)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_inject: filter 4 needs a table (tno_mf_set_prf_table2d)");
    for (int32_t t = 0; t < T; ++t) {
        if (frame_times && !finite_f(frame_times[t]))
            return fail(ctx, TNO_MF_EINVAL, "tno_mf_inject: frame_times[%d] is not finite", t);
        if (jitter_xy && (!finite_f(jitter_xy[2 * t]) || !finite_f(jitter_xy[2 * t + 1])))
            return fail(ctx, TNO_MF_EINVAL, "tno_mf_inject: jitter_xy[%d] is not finite", t);
    }
    if (n_sources == 0) return TNO_MF_OK;
    std::vector<SourceDev> host(n_sources);
    for (int32_t m = 0; m < n_sources; ++m) {
        const tno_mf_source &s = sources[m];
        if (!finite_f(s.traj.vx) || !finite_f(s.traj.vy) || !finite_f(s.traj.ax) || !finite_f(s.traj.ay) ||
            !finite_f(s.amplitude))
            return fail(ctx, TNO_MF_EINVAL, "tno_mf_inject: source %d has a non-finite value", m);
        host[m] = {s.traj.vx, s.traj.vy, s.traj.ax, s.traj.ay, s.x, s.y, s.amplitude};
        // the displacement must fit 32-bit pixel arithmetic, as in the search (reading d2)
        for (int32_t t = 0; t < T; ++t) {
            const double dt = (frame_times ? (double)frame_times[t] : (double)t) - (double)t0;
            int32_t sh;
            if (!axis_shift((double)s.traj.vx, (double)s.traj.ax, dt, jitter_xy ? (double)jitter_xy[2 * t] : 0.0, &sh) ||
                !axis_shift((double)s.traj.vy, (double)s.traj.ay, dt, jitter_xy ? (double)jitter_xy[2 * t + 1] : 0.0, &sh))
                return fail(ctx, TNO_MF_EINVAL, "tno_mf_inject: the displacement of source %d exceeds 1e9 px", m);
        }
    }
    CU_TRY(ctx, cudaSetDevice(ctx->cfg.device));
    // one upload: the sources, then frame_times [T] and jitter_xy [T][2] if given
    const size_t src_bytes = (host.size() * sizeof(SourceDev) + 15) & ~(size_t)15;
    std::vector<unsigned char> blob(src_bytes + (frame_times ? (size_t)T * 4 : 0) + (jitter_xy ? (size_t)T * 8 : 0) + 16);
    std::memcpy(blob.data(), host.data(), host.size() * sizeof(SourceDev));
    size_t o_tm = src_bytes, o_jt = (o_tm + (frame_times ? (size_t)T * 4 : 0) + 7) & ~(size_t)7;
    if (frame_times) std::memcpy(blob.data() + o_tm, frame_times, (size_t)T * 4);
    if (jitter_xy) std::memcpy(blob.data() + o_jt, jitter_xy, (size_t)T * 8);
    int rc = reserve(ctx, ctx->src, blob.size());
    if (rc) return rc;
    CU_TRY(ctx, cudaMemcpyAsync(ctx->src.p, blob.data(), blob.size(), cudaMemcpyHostToDevice, ctx->stream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));      // blob is a local buffer
    const unsigned char *base = static_cast<const unsigned char *>(ctx->src.p);
    launch_inject(ctx->stream, frames, T, H, W, reinterpret_cast<const SourceDev *>(base), n_sources,
                  (double)prf_sigma, (double)t0, ctx->cfg.filter,
                  static_cast<const float *>(ctx->cfg.filter == 4 ? ctx->prf_tab2.p : ctx->prf_tab.p),
                  ctx->cfg.filter == 4 ? (ctx->prf2_py << 16 | ctx->prf2_px) : ctx->prf_phases,
                  frame_times ? reinterpret_cast<const float *>(base + o_tm) : nullptr,
                  jitter_xy ? reinterpret_cast<const float *>(base + o_jt) : nullptr);
    CU_TRY(ctx, cudaGetLastError());
    return TNO_MF_OK;
}

int tno_mf_best(tno_mf_ctx *ctx, const float *snr, int32_t n_traj, int32_t H, int32_t W, int32_t box,
                float *out_max, int32_t *out_argk, float *out_z, tno_mf_cand *out_topk) {
    if (!ctx) return TNO_MF_EINVAL;
    ctx->last_launches = 0;
    if (!snr || !out_max) return fail(ctx, TNO_MF_EINVAL, "tno_mf_best: NULL snr or out_max");
    if (n_traj < 1 || H < 1 || W < 1 || (int64_t)H * W > (int64_t)1 << 31 || H > kMaxRows)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_best: n_traj, H, W must be >= 1, H*W <= 2^31 and H <= %d", kMaxRows);
    if (box < 1 || (box & 1) == 0) return fail(ctx, TNO_MF_EINVAL, "tno_mf_best: box must be odd and >= 1");
    CU_TRY(ctx, cudaSetDevice(ctx->cfg.device));
    cudaStream_t st = ctx->stream;
    const bool want_topk = out_topk != nullptr && ctx->cfg.topk > 0;
    int rc;
    int32_t *argk = out_argk;
    const size_t px = (size_t)H * W;
    if (want_topk && !argk) {          // the records carry the arg-max trajectory
        if ((rc = reserve(ctx, ctx->tmp_maps, px * 4))) return rc;
        argk = static_cast<int32_t *>(ctx->tmp_maps.p);
    }
    launch_max_map(st, snr, n_traj, H, W, out_max, argk, ctx->n_sm);
    ctx->last_launches += 1;
    if (out_z || want_topk) {
        float *z = out_z;
        if (!z) {
            if ((rc = reserve(ctx, ctx->ztmp, px * 4))) return rc;
            z = static_cast<float *>(ctx->ztmp.p);
        }
        if ((rc = reserve(ctx, ctx->sat, px * 16))) return rc;
        launch_local_z(st, out_max, H, W, box, ctx->sat.p, z);
        ctx->last_launches += 3;
        if (want_topk) {
            const int32_t ntx = (W + kCollectTile - 1) / kCollectTile, nty = (H + kCollectTile - 1) / kCollectTile;
            const int64_t n_tiles = (int64_t)ntx * nty;
            if ((rc = reserve(ctx, ctx->keys, (size_t)n_tiles * ctx->cfg.topk * 8))) return rc;
            if ((rc = reserve(ctx, ctx->counts, (size_t)n_tiles * 4))) return rc;
            TopkSlots slots;
            slots.keys = static_cast<uint64_t *>(ctx->keys.p);
            slots.counts = static_cast<int32_t *>(ctx->counts.p);
            slots.ktop = ctx->cfg.topk;
            slots.K = 1;
            slots.threshold = ctx->cfg.snr_threshold;
            launch_collect_from_map(st, z, H, W, 0, 1, slots);
            launch_topk_merge(st, slots, (int32_t)n_tiles, W, out_topk);
            launch_set_argk(st, out_topk, ctx->cfg.topk, argk, W);
            ctx->last_launches += 3;
        }
    }
    CU_TRY(ctx, cudaGetLastError());
    return TNO_MF_OK;
}

int tno_mf_peaks(tno_mf_ctx *ctx, const float *score, const int32_t *argk, int32_t H, int32_t W, int32_t radius,
                 float *out_peaks, tno_mf_cand *out_topk) {
    if (!ctx) return TNO_MF_EINVAL;
    ctx->last_launches = 0;
    if (!score) return fail(ctx, TNO_MF_EINVAL, "tno_mf_peaks: NULL score map");
    if (H < 1 || W < 1 || (int64_t)H * W > (int64_t)1 << 31 || H > kMaxRows)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_peaks: H, W must be >= 1, H*W <= 2^31 and H <= %d", kMaxRows);
    if (radius < 0 || radius > 1024) return fail(ctx, TNO_MF_EINVAL, "tno_mf_peaks: radius must be in [0, 1024]");
    const bool want_topk = out_topk != nullptr && ctx->cfg.topk > 0;
    if (!out_peaks && !want_topk) return fail(ctx, TNO_MF_EINVAL, "tno_mf_peaks: no output requested");
    if (out_peaks == score) return fail(ctx, TNO_MF_EINVAL, "tno_mf_peaks: out_peaks must not alias score");
    CU_TRY(ctx, cudaSetDevice(ctx->cfg.device));
    cudaStream_t st = ctx->stream;
    int rc;
    float *pk = out_peaks;
    if (!pk) {
        if ((rc = reserve(ctx, ctx->ztmp, (size_t)H * W * 4))) return rc;
        pk = static_cast<float *>(ctx->ztmp.p);
        if (pk == score) return fail(ctx, TNO_MF_EINVAL, "tno_mf_peaks: score is the context's scratch map");
    }
    launch_nms(st, score, H, W, radius, ctx->cfg.snr_threshold, pk);
    ctx->last_launches += 1;
    if (want_topk) {
        const int32_t ntx = (W + kCollectTile - 1) / kCollectTile, nty = (H + kCollectTile - 1) / kCollectTile;
        const int64_t n_tiles = (int64_t)ntx * nty;
        if ((rc = reserve(ctx, ctx->keys, (size_t)n_tiles * ctx->cfg.topk * 8))) return rc;
        if ((rc = reserve(ctx, ctx->counts, (size_t)n_tiles * 4))) return rc;
        TopkSlots slots;
        slots.keys = static_cast<uint64_t *>(ctx->keys.p);
        slots.counts = static_cast<int32_t *>(ctx->counts.p);
        slots.ktop = ctx->cfg.topk;
        slots.K = 1;
        slots.threshold = std::max(ctx->cfg.snr_threshold, -FLT_MAX);      // never the -inf of a suppressed pixel
        launch_collect_from_map(st, pk, H, W, 0, 1, slots);
        launch_topk_merge(st, slots, (int32_t)n_tiles, W, out_topk);
        ctx->last_launches += 2;
        if (argk) {
            launch_set_argk(st, out_topk, ctx->cfg.topk, argk, W);
            ctx->last_launches += 1;
        }
    }
    CU_TRY(ctx, cudaGetLastError());
    return TNO_MF_OK;
}

int tno_mf_search(tno_mf_ctx *ctx, const float *frames, int32_t T, int32_t H, int32_t W,
                  const float *sigma_t, const tno_mf_traj *trajectories, int32_t n_traj,
                  float prf_sigma, float t0, float *out_snr, tno_mf_cand *out_topk) {
    return tno_mf_search_ex(ctx, frames, T, H, W, sigma_t, nullptr, nullptr, trajectories, n_traj, prf_sigma, t0,
                            out_snr, out_topk);
}

int tno_mf_background(tno_mf_ctx *ctx, const float *frames, int32_t T, int32_t H, int32_t W,
                      const float *jitter_xy, float delta, int32_t n_iter, float *out_coef, float *out_resid) {
    if (!ctx) return TNO_MF_EINVAL;
    ctx->last_launches = 0;
    ctx->ev_used = 0;
    if (!frames || !jitter_xy) return fail(ctx, TNO_MF_EINVAL, "tno_mf_background: NULL frames or jitter_xy");
    if (T < 1 || H < 1 || W < 1) return fail(ctx, TNO_MF_EINVAL, "tno_mf_background: T, H, W must be >= 1");
    if (!(delta > 0.f) || std::isnan(delta)) return fail(ctx, TNO_MF_EINVAL, "tno_mf_background: delta must be > 0");
    if (n_iter < 0) return fail(ctx, TNO_MF_EINVAL, "tno_mf_background: n_iter must be >= 0");
    if (!out_coef && !out_resid) return fail(ctx, TNO_MF_EINVAL, "tno_mf_background: no output requested");
    for (int32_t t = 0; t < T; ++t)
        if (!finite_f(jitter_xy[2 * t]) || !finite_f(jitter_xy[2 * t + 1]))
            return fail(ctx, TNO_MF_EINVAL, "tno_mf_background: jitter_xy[%d] is not finite", t);
    // basis (1, x, y, x^2, y^2, x y), orthonormalised column by column in float64 (modified Gram-Schmidt,
    // two passes); a column that is (numerically) in the span of the earlier ones is dropped
    std::vector<double> q((size_t)T * 6), r(36, 0.0);
    for (int32_t t = 0; t < T; ++t) {
        const double x = jitter_xy[2 * t], y = jitter_xy[2 * t + 1];
        double *row = &q[(size_t)t * 6];
        row[0] = 1.0; row[1] = x; row[2] = y; row[3] = x * x; row[4] = y * y; row[5] = x * y;
    }
    bool kept[6];
    for (int k = 0; k < 6; ++k) {
        double norm0 = 0.0;
        for (int32_t t = 0; t < T; ++t) norm0 += q[(size_t)t * 6 + k] * q[(size_t)t * 6 + k];
        for (int pass = 0; pass < 2; ++pass)
            for (int m = 0; m < k; ++m) {
                if (!kept[m]) continue;
                double dot = 0.0;
                for (int32_t t = 0; t < T; ++t) dot += q[(size_t)t * 6 + m] * q[(size_t)t * 6 + k];
                r[m * 6 + k] += dot;
                for (int32_t t = 0; t < T; ++t) q[(size_t)t * 6 + k] -= dot * q[(size_t)t * 6 + m];
            }
        double norm = 0.0;
        for (int32_t t = 0; t < T; ++t) norm += q[(size_t)t * 6 + k] * q[(size_t)t * 6 + k];
        kept[k] = norm > 1e-20 * std::max(norm0, 1e-300) && norm > 0.0;
        const double inv = kept[k] ? 1.0 / std::sqrt(norm) : 0.0;
        r[k * 6 + k] = kept[k] ? std::sqrt(norm) : 0.0;
        for (int32_t t = 0; t < T; ++t) q[(size_t)t * 6 + k] *= inv;
        if (!kept[k]) for (int m = 0; m < k; ++m) r[m * 6 + k] = 0.0;
    }
    // R^{-1} by back substitution on the kept columns
    BgRinv rinv;
    double ri[36] = {0.0};
    for (int col = 0; col < 6; ++col) {
        if (!kept[col]) continue;
        for (int k = col; k >= 0; --k) {
            if (!kept[k]) continue;
            double v = (k == col) ? 1.0 : 0.0;
            for (int m = k + 1; m <= col; ++m) v -= r[k * 6 + m] * ri[m * 6 + col];
            ri[k * 6 + col] = v / r[k * 6 + k];
        }
    }
    for (int i = 0; i < 36; ++i) rinv.v[i] = (float)ri[i];
    std::vector<float> qf((size_t)T * 16, 0.f);         // row t: (q0,q0, q1,q1, ..., q5,q5, 0,0,0,0)
    for (int32_t t = 0; t < T; ++t)
        for (int k = 0; k < 6; ++k)
            qf[(size_t)t * 16 + 2 * k] = qf[(size_t)t * 16 + 2 * k + 1] = (float)q[(size_t)t * 6 + k];
    CU_TRY(ctx, cudaSetDevice(ctx->cfg.device));
    int rc;
    if ((rc = reserve(ctx, ctx->bgq, qf.size() * 4))) return rc;
    CU_TRY(ctx, cudaMemcpyAsync(ctx->bgq.p, qf.data(), qf.size() * 4, cudaMemcpyHostToDevice, ctx->stream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));      // qf is a local buffer
    if ((rc = record_event(ctx))) return rc;
    launch_background(ctx->stream, frames, T, (int64_t)H * W, static_cast<const float *>(ctx->bgq.p), rinv, delta,
                      n_iter, out_coef, out_resid);
    if ((rc = record_event(ctx))) return rc;
    ctx->last_launches = 1;
    CU_TRY(ctx, cudaGetLastError());
    return TNO_MF_OK;
}

int tno_mf_flux(tno_mf_ctx *ctx, const float *snr, int32_t n_traj, int32_t H, int32_t W, float *out_flux) {
    if (!ctx) return TNO_MF_EINVAL;
    if (!snr || !out_flux) return fail(ctx, TNO_MF_EINVAL, "tno_mf_flux: NULL snr or out_flux");
    if (!ctx->s_ti || n_traj != ctx->s_traj || H != ctx->s_H || W != ctx->s_W)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_flux: no preceding search with n_traj = %d, H = %d, W = %d on this "
                    "context", n_traj, H, W);
    CU_TRY(ctx, cudaSetDevice(ctx->cfg.device));
    launch_flux(ctx->stream, snr, ctx->s_ti, static_cast<const float *>(ctx->rsd.p), n_traj, H, W, out_flux);
    ctx->last_launches = 1;
    CU_TRY(ctx, cudaGetLastError());
    return TNO_MF_OK;
}

int tno_mf_search_ex(tno_mf_ctx *ctx, const float *frames, int32_t T, int32_t H, int32_t W,
                     const float *sigma_t, const float *frame_times, const float *jitter_xy,
                     const tno_mf_traj *trajectories, int32_t n_traj,
                     float prf_sigma, float t0, float *out_snr, tno_mf_cand *out_topk) {
    return tno_mf_search_masked(ctx, frames, nullptr, T, H, W, sigma_t, frame_times, jitter_xy, trajectories, n_traj,
                                prf_sigma, t0, out_snr, out_topk);
}

// The search proper; out_max / out_argk (tno_mf_search_max) may be NULL.
static int search_core(tno_mf_ctx *ctx, const float *frames, const float *valid, int32_t T, int32_t H, int32_t W,
                       const float *sigma_t, const float *frame_times, const float *jitter_xy,
                       const tno_mf_traj *trajectories, int32_t n_traj,
                       float prf_sigma, float t0, float *out_snr, tno_mf_cand *out_topk, float *out_max,
                       int32_t *out_argk) {
    if (!ctx) return TNO_MF_EINVAL;
    ctx->last_launches = 0;
    ctx->s_ti = nullptr;
    ctx->ev_used = 0;
    // ------------------------------------------------------------------ validation
    if (!frames || !sigma_t || !trajectories)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: NULL frames, sigma_t or trajectories");
    if (T < 1 || H < 1 || W < 1 || n_traj < 1)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: T, H, W and n_traj must be >= 1");
    if (n_traj > 65535) return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: at most 65535 trajectories per call");
    if ((int64_t)H * W > (int64_t)1 << 31 || H > kMaxRows)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: H*W must not exceed 2^31 pixels and H %d rows", kMaxRows);
    if (!(prf_sigma > 0.f) || !finite_f(prf_sigma))
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: prf_sigma must be finite and > 0");
    if (ctx->cfg.filter == 3 && ctx->prf_phases == 0)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: filter 3 needs a table (tno_mf_set_prf_table)");
    if (ctx->cfg.filter == 4 && ctx->prf2_py == 0)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: filter 4 needs a table (tno_mf_set_prf_table2d)");
    const bool nonsep = ctx->cfg.filter == 4;      // 25-tap formulation of the generic kernel only
    if (!finite_f(t0)) return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: t0 must be finite");
    const bool want_topk = out_topk != nullptr && ctx->cfg.topk > 0;
    if (!out_snr && !want_topk && !out_max)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: no output requested (out_snr NULL and no top-K)");
    if (out_argk && !out_max) return fail(ctx, TNO_MF_EINVAL, "tno_mf_search_max: out_argk needs out_max");
    for (int32_t t = 0; t < T; ++t)
        if (!(sigma_t[t] > 0.f) || !finite_f(sigma_t[t]))
            return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: sigma_t[%d] must be finite and > 0", t);
    for (int32_t k = 0; k < n_traj; ++k)
        if (!finite_f(trajectories[k].vx) || !finite_f(trajectories[k].vy) ||
            !finite_f(trajectories[k].ax) || !finite_f(trajectories[k].ay))
            return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: trajectory %d has a non-finite value", k);
    for (int32_t t = 0; t < T; ++t) {
        if (frame_times && !finite_f(frame_times[t]))
            return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: frame_times[%d] is not finite", t);
        if (jitter_xy && (!finite_f(jitter_xy[2 * t]) || !finite_f(jitter_xy[2 * t + 1])))
            return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: jitter_xy[%d] is not finite", t);
    }
    CU_TRY(ctx, cudaSetDevice(ctx->cfg.device));
    cudaStream_t st = ctx->stream;

    // ------------------------------------------------------------------ planning (host)
    Plan plan;
    if (build_classes(trajectories, n_traj, T, (double)t0, frame_times, jitter_xy, &plan) != TNO_MF_OK)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: a trajectory displacement exceeds 1e9 px");
    const int32_t n_x = (int32_t)plan.xcls.size(), n_y = (int32_t)plan.ycls.size();
    const int32_t n_cls = n_x + n_y;
    if (n_cls > 65535) return fail(ctx, TNO_MF_EINVAL, "tno_mf_search: too many distinct axis motions");

    // The separable kernel needs TMA-compatible frames (W % 4 == 0, 16-byte aligned) and a piece
    // count (1 + ceil(y-shift range / tile height)) that stays small.
    bool use_sep = !ctx->cfg.force_generic && !nonsep && (W % 4 == 0) &&
                   ((reinterpret_cast<uintptr_t>(frames) & 15u) == 0) &&
                   ((reinterpret_cast<uintptr_t>(valid) & 15u) == 0) && W >= 4;
    int32_t variant = -1, n_pieces = 1;
    const int32_t n_pass = valid ? 2 : 1;             // masked search: a second pass accumulates D
    SepVariant sv = {0, 0};
    if (use_sep) {
        // slots (mirror pairs where the filter is symmetric under y -> -y: the Gaussian and the single tap)
        // packed into batches; both kernel variants take the same batches
        // kernel shape: the one with the shorter modelled makespan.  A (tile, batch) work item costs, per frame and
        // position row, [ 30 (tile_h + 4) / tile_h for the x-pass + 2 (5 slots + 4) for the y-pass + 200 / rows for the
        // per-frame bookkeeping and latencies of a consumer warp + 15 slots / rows if the batch is not full (it then
        // takes the kernel's branchy path without the weight prefetch) ]; the persistent CTAs take ceil(items / SMs)
        // items each.  The three constants are fitted to the measured shape ratios of configs 2-5 (DESIGN.md section 6:
        // reproduced within 2 %).  Ties go to shape 0.
        const bool sym = ctx->cfg.filter == 0 || ctx->cfg.filter == 1;
        double best = 0.0;
        for (int32_t v = 0; v < sep_num_variants(); ++v) {
            const SepVariant cand = sep_variant(v);
            build_slot_batches(&plan, cand.nb, sym);
            double per_item = 0.0;
            for (const SlotBatch &bt : plan.slot_batches)
                per_item += 30.0 * (cand.tile_h + 4) / cand.tile_h + 2.0 * (5.0 * bt.slots.size() + 4.0) + 200.0 / cand.rows +
                            ((int32_t)bt.slots.size() < cand.nb ? 15.0 * bt.slots.size() / cand.rows : 0.0);
            per_item *= (double)cand.tile_h / (double)plan.slot_batches.size();
            const double items = (double)((W + 63) / 64) * sep_tile_rows(v, H) * (double)plan.slot_batches.size();
            const double cost = std::ceil(items / ctx->n_sm) * per_item;
            if (variant < 0 || cost < best * (1.0 - 1e-9)) { best = cost; variant = v; }
        }
        if (ctx->cfg.sep_shape > 0) variant = ctx->cfg.sep_shape - 1;
        sv = sep_variant(variant);
        build_slot_batches(&plan, sv.nb, sym);
        int64_t range = 0;
        for (const AxisClass &c : plan.ycls) range = std::max<int64_t>(range, (int64_t)c.smax - c.smin);
        const int64_t np = 1 + (range + sv.tile_h - 1) / sv.tile_h;
        if (np > 64) use_sep = false; else n_pieces = (int32_t)np;
    }
    ctx->last_kernel = use_sep ? 1 : 0;

    // ------------------------------------------------------------------ host metadata blob
    std::vector<float> cls_v(n_cls), cls_a(n_cls);
    std::vector<AxisBorder> border(n_cls);
    std::vector<int64_t> ab_off(n_cls);
    int64_t ab_total = 0;
    int32_t max_n = 0;
    for (int32_t c = 0; c < n_cls; ++c) {
        const AxisClass &ac = c < n_x ? plan.xcls[c] : plan.ycls[c - n_x];
        cls_v[c] = ac.v;
        cls_a[c] = ac.a;
        border[c] = make_border(ac, c < n_x ? W : H);
        ab_off[c] = ab_total;
        ab_total += (int64_t)border[c].n * T;
        max_n = std::max(max_n, border[c].n);
    }
    std::vector<float> qf(T);
    std::vector<double> qd(T);
    for (int32_t t = 0; t < T; ++t) {
        const double s = (double)sigma_t[t];
        qd[t] = 1.0 / (s * s);
        qf[t] = (float)qd[t];
    }
    std::vector<TrajInfo> tinfo(n_traj);
    int64_t rsd_total = 0, max_tiles = 0;               // (16 x 16 tiles of border cells: k_rsd_tables)
    for (int32_t k = 0; k < n_traj; ++k) {
        TrajInfo &ti = tinfo[k];
        ti.xc = plan.traj_xc[k];
        ti.yc = plan.traj_yc[k];
        ti.bx = border[ti.xc];
        ti.by = border[n_x + ti.yc];
        ti.rsd_off = rsd_total;
        const int64_t cells = (int64_t)ti.bx.n * ti.by.n;
        rsd_total += cells;
        max_tiles = std::max(max_tiles, (int64_t)((ti.bx.n + 15) / 16) * ((ti.by.n + 15) / 16));
    }
    // planned order q: batches in order, slots in order, plus member before minus member
    int32_t n_batches = 0;
    std::vector<int32_t> batch_xc, slot_yc, slot_flip, slot_q, perm, batch_q0;
    double slot_px = 0.0;                // slots summed over batches (work accounting)
    if (use_sep) {
        n_batches = (int32_t)plan.slot_batches.size();
        batch_xc.resize(n_batches);
        slot_yc.assign((size_t)n_batches * sv.nb, -1);
        slot_flip.assign((size_t)n_batches * sv.nb, 0);
        slot_q.assign((size_t)n_batches * sv.nb * 2, -1);
        batch_q0.resize(n_batches + 1);
        perm.reserve(n_traj);
        for (int32_t b = 0; b < n_batches; ++b) {
            const SlotBatch &bt = plan.slot_batches[b];
            batch_xc[b] = bt.xcls;
            batch_q0[b] = (int32_t)perm.size();
            for (size_t j = 0; j < bt.slots.size(); ++j) {
                const size_t slot = (size_t)b * sv.nb + j;
                slot_yc[slot] = bt.slots[j].ycls;
                slot_flip[slot] = bt.slots[j].flip;
                for (int m = 0; m < 2; ++m)
                    if (bt.slots[j].member[m] >= 0) {
                        slot_q[slot * 2 + m] = (int32_t)perm.size() - batch_q0[b];
                        perm.push_back(bt.slots[j].member[m]);
                    }
            }
            slot_px += (double)bt.slots.size();
        }
        batch_q0[n_batches] = (int32_t)perm.size();
    }
    Blob blob;
    const size_t o_v = blob.add(cls_v.data(), cls_v.size() * 4);
    const size_t o_a = blob.add(cls_a.data(), cls_a.size() * 4);
    const size_t o_qf = blob.add(qf.data(), qf.size() * 4);
    const size_t o_qd = blob.add(qd.data(), qd.size() * 8);
    const size_t o_bd = blob.add(border.data(), border.size() * sizeof(AxisBorder));
    const size_t o_off = blob.add(ab_off.data(), ab_off.size() * 8);
    const size_t o_ti = blob.add(tinfo.data(), tinfo.size() * sizeof(TrajInfo));
    const size_t o_bx = blob.add(batch_xc.data(), batch_xc.size() * 4);
    const size_t o_by = blob.add(slot_yc.data(), slot_yc.size() * 4);
    const size_t o_fl = blob.add(slot_flip.data(), slot_flip.size() * 4);
    const size_t o_sq = blob.add(slot_q.data(), slot_q.size() * 4);
    const size_t o_tm = blob.add(frame_times, frame_times ? (size_t)T * 4 : 0);
    const size_t o_jt = blob.add(jitter_xy, jitter_xy ? (size_t)T * 8 : 0);
    const size_t o_bq = blob.add(batch_q0.data(), batch_q0.size() * 4);
    const size_t o_perm = blob.add(perm.data(), perm.size() * 4);

    // ------------------------------------------------------------------ workspace
    int rc;
    const size_t ct = (size_t)n_cls * T;
    if ((rc = reserve(ctx, ctx->meta, blob.bytes.size()))) return rc;
    if ((rc = reserve(ctx, ctx->shift, ct * 4))) return rc;
    if ((rc = reserve(ctx, ctx->g, ct * 5 * 4))) return rc;
    if ((rc = reserve(ctx, ctx->gd, ct * 5 * 8))) return rc;
    if ((rc = reserve(ctx, ctx->ab, (size_t)ab_total * 8))) return rc;
    if ((rc = reserve(ctx, ctx->rsd, (size_t)rsd_total * 4))) return rc;
    const int32_t ntx = (W + kCollectTile - 1) / kCollectTile, nty = (H + kCollectTile - 1) / kCollectTile;
    const int64_t n_tiles = (int64_t)ntx * nty;           // candidate tiles (64 x 64 start pixels)
    if (want_topk) {
        if ((rc = reserve(ctx, ctx->keys, (size_t)n_tiles * n_traj * ctx->cfg.topk * 8))) return rc;
        if ((rc = reserve(ctx, ctx->counts, (size_t)n_tiles * n_traj * 4))) return rc;
    }
    // piece buffer: n_pieces partial-sum maps per entry; the bank is processed in chunks of whole
    // batches when it does not fit the budget (<= 8 GB, or 40 GB for a host-fed search whose first chunk hides the upload, and <= 80 % of what the device has free)
    const int64_t map_px = (int64_t)H * W;
    int64_t chunk_cap = n_traj;                            // entries per chunk
    if (use_sep) {
        if ((rc = reserve(ctx, ctx->stage_tab, (size_t)n_pass * n_batches * T * sep_table_words(variant) * 4)))
            return rc;
        const size_t per_entry = (size_t)n_pass * n_pieces * map_px * 4;
        const size_t want = per_entry * n_traj;
        const size_t limit = ctx->cfg.workspace_limit_mb > 0 ? (size_t)ctx->cfg.workspace_limit_mb << 20
                                                             : (size_t)(ctx->feed_host ? 40 : 8) << 30;
        size_t have = std::min(ctx->pieces.cap, limit);
        if (want > have) {
            size_t free_b = 0, total_b = 0;
            CU_TRY(ctx, cudaMemGetInfo(&free_b, &total_b));
            const size_t avail = (size_t)((double)(free_b + ctx->pieces.cap) * 0.8);
            const size_t budget = std::min<size_t>(want, std::min<size_t>(avail, limit));
            // a chunk holds at least one batch
            const size_t need = std::max<size_t>(budget, per_entry * (size_t)std::min<int64_t>(2 * sv.nb, n_traj));
            if (need > avail)
                return fail(ctx, TNO_MF_ENOMEM, "not enough device memory for the partial-sum buffer "
                            "(%zu bytes per trajectory, %zu available)", per_entry, avail);
            if ((rc = reserve(ctx, ctx->pieces, need))) return rc;
            have = need;
        }
        chunk_cap = std::min<int64_t>((int64_t)(have / per_entry), n_traj);
    }
    unsigned char *meta = static_cast<unsigned char *>(ctx->meta.p);
    CU_TRY(ctx, cudaMemcpyAsync(meta, blob.bytes.data(), blob.bytes.size(), cudaMemcpyHostToDevice, st));

    ClassTables tab;
    tab.shift = static_cast<const int32_t *>(ctx->shift.p);
    tab.g = static_cast<const float *>(ctx->g.p);
    tab.gd = static_cast<const double *>(ctx->gd.p);
    tab.qf = reinterpret_cast<const float *>(meta + o_qf);
    tab.qd = reinterpret_cast<const double *>(meta + o_qd);
    tab.cls_v = reinterpret_cast<const float *>(meta + o_v);
    tab.cls_a = reinterpret_cast<const float *>(meta + o_a);
    tab.n_x = n_x;
    tab.T = T;
    const TrajInfo *d_ti = reinterpret_cast<const TrajInfo *>(meta + o_ti);
    const int64_t *d_off = reinterpret_cast<const int64_t *>(meta + o_off);
    float *d_rsd = static_cast<float *>(ctx->rsd.p);

    // ------------------------------------------------------------------ table kernels
    launch_class_tables(st, reinterpret_cast<const float *>(meta + o_v), reinterpret_cast<const float *>(meta + o_a),
                        frame_times ? reinterpret_cast<const float *>(meta + o_tm) : nullptr,
                        jitter_xy ? reinterpret_cast<const float *>(meta + o_jt) : nullptr,
                        n_cls, n_x, T, (double)t0, (double)prf_sigma, ctx->cfg.filter,
                        static_cast<const float *>(ctx->prf_tab.p),
                        nonsep ? (ctx->prf2_py << 16 | ctx->prf2_px) : ctx->prf_phases, static_cast<int32_t *>(ctx->shift.p),
                        static_cast<float *>(ctx->g.p), static_cast<double *>(ctx->gd.p));
    launch_border_tables(st, tab.shift, tab.gd, tab.qd, reinterpret_cast<const AxisBorder *>(meta + o_bd), d_off,
                         n_cls, n_x, max_n, T, W, H, static_cast<double *>(ctx->ab.p));
    launch_rsd_tables(st, d_ti, n_traj, max_tiles, static_cast<const double *>(ctx->ab.p), d_off, n_x, T, d_rsd);
    ctx->last_launches += 3;
    CU_TRY(ctx, cudaGetLastError());

    TopkSlots slots;
    slots.keys = want_topk ? static_cast<uint64_t *>(ctx->keys.p) : nullptr;
    slots.counts = want_topk ? static_cast<int32_t *>(ctx->counts.p) : nullptr;
    slots.ktop = ctx->cfg.topk;
    slots.K = n_traj;
    slots.threshold = ctx->cfg.snr_threshold;

    uint64_t *mk = nullptr;                  // running (score, ~k) maximum per pixel, 0 = below every score
    if (out_max) {
        if ((rc = reserve(ctx, ctx->maxkeys, (size_t)map_px * 8))) return rc;
        mk = static_cast<uint64_t *>(ctx->maxkeys.p);
        CU_TRY(ctx, cudaMemsetAsync(mk, 0, (size_t)map_px * 8, st));
    }

    // ------------------------------------------------------------------ search
    if (use_sep) {
        const size_t tab_floats = (size_t)n_batches * T * sep_table_words(variant);
        for (int32_t pass = 0; pass < n_pass; ++pass) {
            launch_sep_tables(st, variant, tab, reinterpret_cast<const int32_t *>(meta + o_bx),
                              reinterpret_cast<const int32_t *>(meta + o_by),
                              reinterpret_cast<const int32_t *>(meta + o_fl),
                              reinterpret_cast<const int32_t *>(meta + o_sq), n_batches, pass,
                              static_cast<float *>(ctx->stage_tab.p) + pass * tab_floats);
            ctx->last_launches += 1;
        }
        CU_TRY(ctx, cudaGetLastError());
        const int32_t tabw = sep_table_words(variant);
        for (int32_t b0 = 0; b0 < n_batches;) {
            int32_t b1 = b0 + 1;
            while (b1 < n_batches && batch_q0[b1 + 1] - batch_q0[b0] <= chunk_cap) ++b1;
            const int32_t q0 = batch_q0[b0], qn = batch_q0[b1] - q0;
            SepArgs a;
            a.frames = frames; a.T = T; a.H = H; a.W = W;
            a.stage_tab = static_cast<const float *>(ctx->stage_tab.p) + (size_t)b0 * T * tabw;
            a.batch_q = reinterpret_cast<const int32_t *>(meta + o_bq) + b0;
            a.n_batches = b1 - b0;
            a.q0 = q0;
            a.pieces = static_cast<float *>(ctx->pieces.p);
            a.piece_stride = (int64_t)qn * map_px;
            a.n_pieces = n_pieces;
            a.n_sm = ctx->n_sm;
            const size_t pass_floats = (size_t)n_pieces * a.piece_stride;
            CU_TRY(ctx, cudaMemsetAsync(a.pieces, 0, n_pass * pass_floats * 4, st));
            const int32_t nfy = (H + kCollectTile - 1) / kCollectTile;   // rows of 64 x 64 output tiles
            int32_t fin_tiles = 0;                                        // ... already finished (banded)
            const bool banded_finish = ctx->feed_host && ctx->fed_rows < H && qn == n_traj;
            int64_t y_smax = INT32_MIN;                                   // largest y-shift of the bank
            for (const AxisClass &c : plan.ycls) y_smax = std::max<int64_t>(y_smax, c.smax);
            const float *np_ = static_cast<const float *>(ctx->pieces.p);
            // a host-fed stack arrives in bands of tile rows: the search of a band starts as soon as
            // its frame rows are on the device and overlaps the upload of the next bands
            const int32_t nty = sep_tile_rows(variant, H);
            const int32_t band = (ctx->feed_host && ctx->fed_rows < H) ? 4 : nty;
            for (int32_t ty0 = 0; ty0 < nty; ty0 += band) {
                a.ty0 = ty0;
                a.ty1 = std::min(nty, ty0 + band);
                if ((rc = feed_rows(ctx, a.ty1 == nty ? H : a.ty1 * sv.tile_h))) return rc;
                for (int32_t pass = 0; pass < n_pass; ++pass) {
                    // pass 1 of a masked search: the same kernel over the validity weights with squared taps
                    a.frames = pass ? valid : frames;
                    a.stage_tab = static_cast<const float *>(ctx->stage_tab.p) + pass * tab_floats + (size_t)b0 * T * tabw;
                    a.pieces = static_cast<float *>(ctx->pieces.p) + pass * pass_floats;
                    int32_t grid = 0;
                    const char *err = "";
                    if ((rc = record_event(ctx))) return rc;
                    if (launch_search_sep(st, variant, a, ctx->encode_fn, &grid, &err) != 0)
                        return fail(ctx, TNO_MF_ECUDA, "separable search kernel: %s", err);
                    if ((rc = record_event(ctx))) return rc;
                    ctx->last_launches += (ty0 > 0);
                }
                // host-fed, one chunk: the output rows that no later tile row can touch are finished and
                // sent to the host while the next bands are still being uploaded
                if (banded_finish && a.ty1 < nty) {
                    const int32_t fy1 = (int32_t)std::min<int64_t>(nfy, std::max<int64_t>(
                        fin_tiles, ((int64_t)a.ty1 * sv.tile_h - y_smax - 2) / kCollectTile));
                    if (fy1 > fin_tiles) {
                        launch_finish(st, np_, valid ? np_ + pass_floats : nullptr, n_pieces, a.piece_stride,
                                      reinterpret_cast<const int32_t *>(meta + o_perm), q0, qn, d_ti, d_rsd, H, W,
                                      fin_tiles, fy1, out_snr, mk, slots);
                        ctx->last_launches += 1;
                        fin_tiles = fy1;
                        if ((rc = download_rows(ctx, fy1 * kCollectTile))) return rc;
                    }
                }
            }
            // (all rows may be finished already: a bank whose y-shifts are all negative; launch_finish skips an empty range)
            launch_finish(st, np_, valid ? np_ + pass_floats : nullptr, n_pieces, a.piece_stride,
                          reinterpret_cast<const int32_t *>(meta + o_perm), q0, qn, d_ti, d_rsd, H, W, fin_tiles, nfy,
                          out_snr, mk, slots);
            CU_TRY(ctx, cudaGetLastError());
            ctx->last_launches += 2 + n_pass;              // memset, search(es), finish
            b0 = b1;
        }
        // work of the formulation: x-pass over the staged rows of every (tile, batch, frame),
        // y-pass per trajectory x frame x start pixel
        double rows = 0.0;
        for (int32_t ty = 0; ty < sep_tile_rows(variant, H); ++ty)
            rows += (double)(std::min(sv.tile_h, H + 2 - (ty * sv.tile_h - 2)) + 4);
        const double cols = 64.0 * (double)((W + 63) / 64);
        ctx->last_fma_x = n_pass * 5.0 * rows * cols * (double)n_batches * T;
        // y-pass: 5 multiply-adds per slot (one or two trajectories), position and frame; the sums and
        // differences of the window rows, 4 additions per position and frame, are shared by the batch
        ctx->last_fma_y = n_pass * 5.0 * slot_px * T * (double)H * W;
        ctx->last_add_y = n_pass * 4.0 * (rows - 4.0 * sep_tile_rows(variant, H)) * cols * (double)n_batches * T;
    } else {
        // generic path: maps are always materialised (caller's buffer, or a workspace chunk)
        if ((rc = feed_rows(ctx, H))) return rc;
        int32_t chunk = n_traj;
        float *maps = out_snr;
        if (!out_snr) {
            const int64_t budget = (int64_t)1 << 29;   // floats (2 GiB)
            chunk = (int32_t)std::max<int64_t>(1, std::min<int64_t>(n_traj, budget / map_px));
            if ((rc = reserve(ctx, ctx->tmp_maps, (size_t)chunk * map_px * 4))) return rc;
            maps = static_cast<float *>(ctx->tmp_maps.p);
        }
        ctx->last_fma_x = 0.0;
        ctx->last_add_y = 0.0;
        ctx->last_fma_y = n_pass * 25.0 * (double)n_traj * T * (double)H * W;
        if ((rc = record_event(ctx))) return rc;
        for (int32_t k0 = 0; k0 < n_traj; k0 += chunk) {
            const int32_t kc = std::min(chunk, n_traj - k0);
            float *dst = out_snr ? out_snr + (int64_t)k0 * map_px : maps;
            if (nonsep)
                launch_search_generic25(st, frames, valid, T, H, W, tab, d_ti, static_cast<const float *>(ctx->prf_tab2.p),
                                        ctx->prf2_px, k0, kc, dst);
            else
                launch_search_generic(st, frames, valid, T, H, W, tab, d_ti, d_rsd, k0, kc, dst);
            ctx->last_launches += 1;
            if (want_topk) {
                launch_collect_from_map(st, dst, H, W, k0, kc, slots);
                ctx->last_launches += 1;
            }
            if (mk) {
                launch_max_keys_from_maps(st, dst, k0, kc, map_px, mk);
                ctx->last_launches += 1;
            }
        }
        if ((rc = record_event(ctx))) return rc;
        CU_TRY(ctx, cudaGetLastError());
    }
    if (want_topk) {
        launch_topk_merge(st, slots, (int32_t)n_tiles, W, out_topk);
        ctx->last_launches += 1;
        CU_TRY(ctx, cudaGetLastError());
    }
    if (mk) {
        launch_max_decode(st, mk, map_px, out_max, out_argk);
        ctx->last_launches += 1;
        CU_TRY(ctx, cudaGetLastError());
    }
    ctx->s_traj = n_traj; ctx->s_H = H; ctx->s_W = W;
    ctx->s_ti = (valid || nonsep) ? nullptr : d_ti;    // tno_mf_flux needs the analytic (separable) D tables
    return TNO_MF_OK;
}

int tno_mf_search_masked(tno_mf_ctx *ctx, const float *frames, const float *valid, int32_t T, int32_t H, int32_t W,
                         const float *sigma_t, const float *frame_times, const float *jitter_xy,
                         const tno_mf_traj *trajectories, int32_t n_traj,
                         float prf_sigma, float t0, float *out_snr, tno_mf_cand *out_topk) {
    return search_core(ctx, frames, valid, T, H, W, sigma_t, frame_times, jitter_xy, trajectories, n_traj, prf_sigma, t0,
                       out_snr, out_topk, nullptr, nullptr);
}

int tno_mf_search_max(tno_mf_ctx *ctx, const float *frames, const float *valid, int32_t T, int32_t H, int32_t W,
                      const float *sigma_t, const float *frame_times, const float *jitter_xy,
                      const tno_mf_traj *trajectories, int32_t n_traj, float prf_sigma, float t0,
                      float *out_max, int32_t *out_argk, float *out_snr, tno_mf_cand *out_topk) {
    if (!ctx) return TNO_MF_EINVAL;
    if (!out_max) return fail(ctx, TNO_MF_EINVAL, "tno_mf_search_max: NULL out_max");
    return search_core(ctx, frames, valid, T, H, W, sigma_t, frame_times, jitter_xy, trajectories, n_traj, prf_sigma, t0,
                       out_snr, out_topk, out_max, out_argk);
}

int tno_mf_search_host(tno_mf_ctx *ctx, const float *frames_host, int32_t T, int32_t H, int32_t W,
                       const float *sigma_t, const float *frame_times, const float *jitter_xy,
                       const tno_mf_traj *trajectories, int32_t n_traj, float prf_sigma, float t0,
                       float *out_snr_host, tno_mf_cand *out_topk_host) {
    return tno_mf_search_host_max(ctx, frames_host, nullptr, T, H, W, sigma_t, frame_times, jitter_xy, trajectories,
                                  n_traj, prf_sigma, t0, nullptr, nullptr, out_snr_host, out_topk_host);
}

int tno_mf_search_host_max(tno_mf_ctx *ctx, const float *frames_host, const float *valid_host, int32_t T, int32_t H,
                           int32_t W, const float *sigma_t, const float *frame_times, const float *jitter_xy,
                           const tno_mf_traj *trajectories, int32_t n_traj, float prf_sigma, float t0,
                           float *out_max_host, int32_t *out_argk_host, float *out_snr_host,
                           tno_mf_cand *out_topk_host) {
    if (!ctx) return TNO_MF_EINVAL;
    if (!frames_host) return fail(ctx, TNO_MF_EINVAL, "tno_mf_search_host: NULL frames");
    if (T < 1 || H < 1 || W < 1 || n_traj < 1)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_search_host: T, H, W and n_traj must be >= 1");
    const bool want_topk = out_topk_host != nullptr && ctx->cfg.topk > 0;
    if (!out_snr_host && !want_topk && !out_max_host)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_search_host: no output requested");
    if (out_argk_host && !out_max_host)
        return fail(ctx, TNO_MF_EINVAL, "tno_mf_search_host_max: out_argk needs out_max");
    CU_TRY(ctx, cudaSetDevice(ctx->cfg.device));
    int rc;
    const size_t px = (size_t)H * W;
    if ((rc = reserve(ctx, ctx->stack, (size_t)T * px * 4))) return rc;
    if (valid_host && (rc = reserve(ctx, ctx->stack2, (size_t)T * px * 4))) return rc;
    if (out_snr_host && (rc = reserve(ctx, ctx->hmaps, (size_t)n_traj * px * 4))) return rc;
    if (want_topk && (rc = reserve(ctx, ctx->htopk, (size_t)n_traj * ctx->cfg.topk * sizeof(tno_mf_cand)))) return rc;
    if (out_max_host && (rc = reserve(ctx, ctx->hmax, px * 8))) return rc;
    if (!ctx->copy_stream) {
        CU_TRY(ctx, cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        CU_TRY(ctx, cudaEventCreateWithFlags(&ctx->copy_ev, cudaEventDisableTiming));
        CU_TRY(ctx, cudaEventCreateWithFlags(&ctx->start_ev, cudaEventDisableTiming));
        CU_TRY(ctx, cudaStreamCreateWithFlags(&ctx->down_stream, cudaStreamNonBlocking));
        CU_TRY(ctx, cudaEventCreateWithFlags(&ctx->fin_ev, cudaEventDisableTiming));
    }
    // the upload must not overtake earlier work of the context that still reads the device stack
    CU_TRY(ctx, cudaEventRecord(ctx->start_ev, ctx->stream));
    CU_TRY(ctx, cudaStreamWaitEvent(ctx->copy_stream, ctx->start_ev, 0));
    ctx->feed_host = frames_host;
    ctx->feed_dev = static_cast<float *>(ctx->stack.p);
    ctx->feed_host2 = valid_host;
    ctx->feed_dev2 = valid_host ? static_cast<float *>(ctx->stack2.p) : nullptr;
    ctx->fed_rows = 0;
    ctx->feed_T = T; ctx->feed_H = H; ctx->feed_W = W;
    float *d_maps = out_snr_host ? static_cast<float *>(ctx->hmaps.p) : nullptr;
    ctx->down_host = out_snr_host;
    ctx->down_dev = d_maps;
    ctx->down_rows = 0;
    ctx->down_K = n_traj;
    tno_mf_cand *d_topk = want_topk ? static_cast<tno_mf_cand *>(ctx->htopk.p) : nullptr;
    float *d_max = out_max_host ? static_cast<float *>(ctx->hmax.p) : nullptr;
    int32_t *d_argk = out_argk_host ? reinterpret_cast<int32_t *>(d_max + px) : nullptr;
    rc = search_core(ctx, ctx->feed_dev, ctx->feed_dev2, T, H, W, sigma_t, frame_times, jitter_xy, trajectories,
                     n_traj, prf_sigma, t0, d_maps, d_topk, d_max, d_argk);
    ctx->feed_host = ctx->feed_host2 = nullptr;
    if (rc == TNO_MF_OK) rc = download_rows(ctx, H);       // the rows no band could finish early
    ctx->down_host = nullptr;
    if (rc != TNO_MF_OK) {
        cudaStreamSynchronize(ctx->copy_stream);           // nothing of the caller's buffers is in flight on return
        cudaStreamSynchronize(ctx->down_stream);
        return rc;
    }
    if (d_topk)
        CU_TRY(ctx, cudaMemcpyAsync(out_topk_host, d_topk, (size_t)n_traj * ctx->cfg.topk * sizeof(tno_mf_cand),
                                    cudaMemcpyDeviceToHost, ctx->stream));
    if (d_max) CU_TRY(ctx, cudaMemcpyAsync(out_max_host, d_max, px * 4, cudaMemcpyDeviceToHost, ctx->stream));
    if (d_argk) CU_TRY(ctx, cudaMemcpyAsync(out_argk_host, d_argk, px * 4, cudaMemcpyDeviceToHost, ctx->stream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->down_stream));
    return TNO_MF_OK;
}

}  // extern "C"

// What an entry point that lives in another file (local_z_static.cu) needs of the opaque context.
namespace tno {
CtxView ctx_view(const tno_mf_ctx *ctx) { return CtxView{ctx->stream, ctx->cfg.device}; }
int ctx_fail(tno_mf_ctx *ctx, int code, const char *text) { return fail(ctx, code, "%s", text); }
void ctx_set_launches(tno_mf_ctx *ctx, int32_t n) { ctx->last_launches = n; }
}  // namespace tno
