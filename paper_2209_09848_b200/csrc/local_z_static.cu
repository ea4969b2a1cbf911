// tno_mf_local_z_static: the local z-score of a score map (section 3.3: "we compute the standard
// deviation of the scores in the 255 x 255 square centered on a pixel. We represent our scores in units of sigma")
// for callers that must not allocate device memory -- code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc.  tno_mf_best computes the same map with its float64 summed-area tables in a
// grow-only cudaMalloc'ed buffer of the context; here the tables live in a file-scope device array of fixed size,
// so the call enqueues three kernels and nothing else: no cudaMalloc, no cudaFree, no allocating library routine.
//
// The array: kStaticZMaxPx double2 = 16 MiB, held by every GPU that loads this library until the process exits.
// All calls on a device share it (whatever their context or stream): calls that overlap on the GPU race on it, so
// callers keep them on one stream or order them with events.  It keeps the last call's contents; nothing in it has
// to start at zero, because k_sat_rows_static overwrites each of the H * W entries that the later kernels read.
//
// The kernels are those of best.cu statement by statement (same float64 arithmetic in the same order), so the
// result is bit-identical to tno_mf_best's out_z for the same map (tests/test_zz_no_alloc.py).
#include <cstdio>
#include <mutex>

#include "kernels.h"

namespace tno {

constexpr int64_t kStaticZMaxPx = (int64_t)1 << 20;       // H * W of the largest map, e.g. 1024 x 1024
constexpr int32_t kStaticMaxDevices = 64;

// In host code this name is a host-side stand-in, not a device address: kernels get the address that
// cudaGetSymbolAddress returns for the current device (sat_static_address below).
static __device__ __align__(256) double2 g_sat_static[kStaticZMaxPx];

namespace {

std::mutex g_sat_mu;
double2 *g_sat_addr[kStaticMaxDevices];      // per device ordinal; NULL = not resolved yet

// Once per device, with that device current.
int sat_static_address(tno_mf_ctx *ctx, int32_t device, double2 **out) {
    std::lock_guard<std::mutex> lock(g_sat_mu);
    if (!g_sat_addr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_sat_static);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            char buf[200];
            snprintf(buf, sizeof buf, "tno_mf_local_z_static: cudaGetSymbolAddress failed on device %d: %s", device,
                     e != cudaSuccess ? cudaGetErrorString(e) : "NULL address");
            return ctx_fail(ctx, TNO_MF_ECUDA, buf);
        }
        g_sat_addr[device] = static_cast<double2 *>(p);
    }
    *out = g_sat_addr[device];
    return TNO_MF_OK;
}

// One block per row: inclusive prefix sums along x of (M, M^2) in float64 (best.cu: k_sat_rows).
__global__ void __launch_bounds__(256)
k_sat_rows_static(const float *__restrict__ m, int32_t W, double2 *__restrict__ sat) {
    __shared__ double2 wsum[8];
    const int32_t y = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int32_t per = (W + 255) / 256;
    const int32_t x0 = tid * per, x1 = min(W, x0 + per);
    const float *row = m + (int64_t)y * W;
    double2 loc = make_double2(0.0, 0.0);
    for (int32_t x = x0; x < x1; ++x) {
        const double v = (double)row[x];
        loc.x += v;
        loc.y += v * v;
    }
    double2 inc = loc;
    for (int o = 1; o < 32; o <<= 1) {
        const double a = __shfl_up_sync(0xffffffffu, inc.x, o), b = __shfl_up_sync(0xffffffffu, inc.y, o);
        if (lane >= o) { inc.x += a; inc.y += b; }
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    double2 run = make_double2(inc.x - loc.x, inc.y - loc.y);
    for (int32_t w = 0; w < warp; ++w) { run.x += wsum[w].x; run.y += wsum[w].y; }
    double2 *out = sat + (int64_t)y * W;
    for (int32_t x = x0; x < x1; ++x) {
        const double v = (double)row[x];
        run.x += v;
        run.y += v * v;
        out[x] = run;
    }
}

// One block per 32 columns, 32 warps: warp w walks the rows [w*chunk, (w+1)*chunk) of its columns, in place
// (best.cu: k_sat_cols).
__global__ void __launch_bounds__(1024)
k_sat_cols_static(double2 *__restrict__ sat, int32_t H, int32_t W) {
    __shared__ double2 tot[32][33];
    const int32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int32_t x = blockIdx.x * 32 + lane;
    const int32_t chunk = (H + 31) / 32;
    const int32_t y0 = warp * chunk, y1 = min(H, y0 + chunk);
    double2 s = make_double2(0.0, 0.0);
    if (x < W)
        for (int32_t y = y0; y < y1; ++y) {
            const double2 v = sat[(int64_t)y * W + x];
            s.x += v.x;
            s.y += v.y;
        }
    tot[warp][lane] = s;
    __syncthreads();
    double2 run = make_double2(0.0, 0.0);
    for (int32_t w = 0; w < warp; ++w) { run.x += tot[w][lane].x; run.y += tot[w][lane].y; }
    if (x < W)
        for (int32_t y = y0; y < y1; ++y) {
            double2 v = sat[(int64_t)y * W + x];
            run.x += v.x;
            run.y += v.y;
            sat[(int64_t)y * W + x] = run;
        }
}

// Z = M / sigma_box from the four corners of the clipped box (best.cu: k_local_z).
__global__ void __launch_bounds__(256)
k_local_z_static(const float *__restrict__ m, const double2 *__restrict__ sat, int32_t H, int32_t W, int32_t h,
                 float *__restrict__ z) {
    const int32_t x = blockIdx.x * 64 + (threadIdx.x & 63), y = blockIdx.y * 4 + (threadIdx.x >> 6);
    if (x >= W || y >= H) return;
    const int32_t x0 = max(0, x - h), x1 = min(W - 1, x + h), y0 = max(0, y - h), y1 = min(H - 1, y + h);
    auto at = [&](int32_t yy, int32_t xx) -> double2 {
        if (yy < 0 || xx < 0) return make_double2(0.0, 0.0);
        return sat[(int64_t)yy * W + xx];
    };
    const double2 a = at(y1, x1), b = at(y1, x0 - 1), c = at(y0 - 1, x1), d = at(y0 - 1, x0 - 1);
    const double n = (double)(y1 - y0 + 1) * (double)(x1 - x0 + 1);
    const double s = ((a.x - b.x) - c.x) + d.x, q = ((a.y - b.y) - c.y) + d.y;
    const double mean = s / n;
    const double var = q / n - mean * mean;
    const double floor_v = 1e-12 * (q / n);
    z[(int64_t)y * W + x] = var > floor_v ? (float)((double)m[(int64_t)y * W + x] / sqrt(var)) : 0.0f;
}

}  // namespace
}  // namespace tno

using namespace tno;

extern "C" int tno_mf_local_z_static(tno_mf_ctx *ctx, const float *score, int32_t H, int32_t W, int32_t box,
                                     float *out_z) {
    if (!ctx) return TNO_MF_EINVAL;
    ctx_set_launches(ctx, 0);
    if (!score || !out_z) return ctx_fail(ctx, TNO_MF_EINVAL, "tno_mf_local_z_static: NULL score or out_z");
    if (out_z == score) return ctx_fail(ctx, TNO_MF_EINVAL, "tno_mf_local_z_static: out_z must not alias score");
    if (H < 1 || W < 1 || H > kMaxRows)
        return ctx_fail(ctx, TNO_MF_EINVAL, "tno_mf_local_z_static: H and W must be >= 1 and H <= 262140 rows");
    if ((int64_t)H * W > kStaticZMaxPx) {
        char buf[200];
        snprintf(buf, sizeof buf,
                 "tno_mf_local_z_static: H * W = %lld exceeds the static scratch of %lld pixels (16 MiB); "
                 "use tno_mf_best for larger maps", (long long)H * W, (long long)kStaticZMaxPx);
        return ctx_fail(ctx, TNO_MF_EINVAL, buf);
    }
    if (box < 1 || (box & 1) == 0) return ctx_fail(ctx, TNO_MF_EINVAL, "tno_mf_local_z_static: box must be odd and >= 1");
    const CtxView v = ctx_view(ctx);
    if (v.device < 0 || v.device >= kStaticMaxDevices)
        return ctx_fail(ctx, TNO_MF_EINVAL, "tno_mf_local_z_static: device ordinal beyond 63");
    cudaError_t e = cudaSetDevice(v.device);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return ctx_fail(ctx, TNO_MF_ECUDA, cudaGetErrorString(e));
    }
    double2 *sat = nullptr;
    if (int rc = sat_static_address(ctx, v.device, &sat)) return rc;
    k_sat_rows_static<<<(unsigned)H, 256, 0, v.stream>>>(score, W, sat);
    k_sat_cols_static<<<(unsigned)((W + 31) / 32), 1024, 0, v.stream>>>(sat, H, W);
    const dim3 grid((unsigned)((W + 63) / 64), (unsigned)((H + 3) / 4));
    k_local_z_static<<<grid, 256, 0, v.stream>>>(score, sat, H, W, (box - 1) / 2, out_z);
    ctx_set_launches(ctx, 3);
    e = cudaGetLastError();
    if (e != cudaSuccess) return ctx_fail(ctx, TNO_MF_ECUDA, cudaGetErrorString(e));
    return TNO_MF_OK;
}
