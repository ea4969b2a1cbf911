// Table kernels: everything that depends on (trajectory class, frame) but not on the pixel.
//   k_class_tables   shift, phase, PRF taps per (class, t)        -- the sparse form of the filter
//                    of PAPER.md:L106 (trajectory line (x) PRF), 5 + 5 taps instead of R x C
//   k_border_tables  per-axis clipped sums of squared taps per (class, t, border class)
//   k_rsd_tables     D^(-1/2) per (trajectory, border class y, border class x)
// D = sum_t sum_p g(p - c_t)^2 / sigma_t^2 with off-frame taps dropped (BASELINE.json:north_star)
// is separable per frame, D = sum_t q_t Ax_t(x) Ay_t(y); it is evaluated in float64.
#include "kernels.h"

namespace tno {

__global__ void k_class_tables(const float *__restrict__ cls_v, const float *__restrict__ cls_a,
                               const float *__restrict__ times, const float *__restrict__ jitter,
                               int32_t n_cls, int32_t n_x, int32_t T, double t0, double prf_sigma, int32_t filter,
                               const float *__restrict__ prf_tab, int32_t n_phase,
                               int32_t *__restrict__ shift, float *__restrict__ g,
                               double *__restrict__ gd) {
    const int64_t id = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= (int64_t)n_cls * T) return;
    const int32_t c = (int32_t)(id / T), t = (int32_t)(id % T);
    const double v = (double)cls_v[c], a = (double)cls_a[c];
    // tau_t (default t) and the pointing jitter of the class's axis (default 0): PAPER.md L106, L116
    const double dt = __dsub_rn(times ? (double)times[t] : (double)t, t0);
    const double j = jitter ? (double)jitter[2 * t + (c < n_x ? 0 : 1)] : 0.0;
    // d = (v*dt + (a*dt)*dt) + j evaluated left to right, every operation separately rounded
    const double d = __dadd_rn(__dadd_rn(__dmul_rn(v, dt), __dmul_rn(__dmul_rn(a, dt), dt)), j);
    const double f = floor(__dadd_rn(d, 0.5));
    const double ph = __dsub_rn(d, f);
    shift[id] = (int32_t)f;
    const double inv = 1.0 / (2.0 * prf_sigma * prf_sigma);
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        const double u = (double)(i - 2) - ph;
        // filter 0: the expression the first version of this kernel had (bit-compatible tables);
        // 1 shift-stack, 2 pixel-integrated Gaussian, 3 tabulated: prf_tap (common.cuh)
        const double w = filter == 0 ? exp(-(u * u) * inv)
                       : filter == 4 ? 0.0 : prf_tap(filter, i, ph, prf_sigma, prf_tab, n_phase);
        g[id * 5 + i] = (float)w;
        gd[id * 5 + i] = w;
    }
    if (filter == 4) {
        // non-separable tabulated PRF: the class contributes the row (y) or column (x) of its phase in the 2-D
        // table; n_phase packs (n_phase_y << 16 | n_phase_x).  The 25 taps are looked up per trajectory and frame.
        const int32_t np = c < n_x ? (n_phase & 0xffff) : (n_phase >> 16);
        int32_t row = (int32_t)floor((ph + 0.5) * (double)np);
        row = row < 0 ? 0 : (row > np - 1 ? np - 1 : row);
        gd[id * 5] = (double)row;
    }
}

// out[off[c] + t * n + j] = (scale_q ? q_t : 1) * sum_{i : 0 <= rep(j) + s + i - 2 < L} gd[c][t][i]^2
__global__ void k_border_tables(const int32_t *__restrict__ shift, const double *__restrict__ gd,
                                const double *__restrict__ qd, const AxisBorder *__restrict__ border,
                                const int64_t *__restrict__ off, int32_t n_x, int32_t T, int32_t W,
                                int32_t H, double *__restrict__ out) {
    const int32_t c = blockIdx.y;
    const AxisBorder b = border[c];
    const int32_t L = (c < n_x) ? W : H;
    const int64_t id = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= (int64_t)b.n * T) return;
    const int32_t t = (int32_t)(id / b.n), j = (int32_t)(id % b.n);
    const int32_t p = border_rep(j, b, L) + shift[(int64_t)c * T + t] - 2;
    const double *w = gd + ((int64_t)c * T + t) * 5;
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 5; ++i)
        if (p + i >= 0 && p + i < L) s += w[i] * w[i];
    if (c < n_x) s *= qd[t];
    out[off[c] + id] = s;
}

// rsd[k][cy][cx] = 1 / sqrt(sum_t AX[xc][t][cx] * AY[yc][t][cy])   (0 where the sum is 0)
// A small contraction over t per trajectory.  One block per 16 x 16 tile of border cells: the 16 columns of AX and
// the 16 columns of AY the tile needs are staged in shared memory, kRsdFrames frames at a time, and every thread sums
// its cell in frame order.  (One thread per cell reading global memory re-read every AX and AY value once per cell:
// 0.27 ms at T = 1000, bound by L1/L2 traffic.)
constexpr int kRsdTile = 16, kRsdFrames = 32;
__global__ void __launch_bounds__(kRsdTile * kRsdTile)
k_rsd_tables(const TrajInfo *__restrict__ traj, const double *__restrict__ ab, const int64_t *__restrict__ off,
             int32_t n_x, int32_t T, float *__restrict__ rsd) {
    __shared__ double sx[kRsdFrames][kRsdTile], sy[kRsdFrames][kRsdTile];
    const TrajInfo ti = traj[blockIdx.y];
    const int32_t ncx = ti.bx.n, ncy = ti.by.n;
    const int32_t tiles_x = (ncx + kRsdTile - 1) / kRsdTile;
    const int32_t cx0 = (int32_t)(blockIdx.x % tiles_x) * kRsdTile, cy0 = (int32_t)(blockIdx.x / tiles_x) * kRsdTile;
    if (cy0 >= ncy) return;                                   // (block-uniform) the grid is sized for the largest table
    const int32_t tid = threadIdx.x, lx = tid % kRsdTile, ly = tid / kRsdTile;
    const double *ax = ab + off[ti.xc];
    const double *ay = ab + off[n_x + ti.yc];
    double D = 0.0;
    for (int32_t t0 = 0; t0 < T; t0 += kRsdFrames) {
        for (int32_t i = tid; i < kRsdFrames * kRsdTile; i += kRsdTile * kRsdTile) {
            const int32_t t = t0 + i / kRsdTile, c = i % kRsdTile;
            sx[i / kRsdTile][c] = (t < T && cx0 + c < ncx) ? __ldg(ax + (int64_t)t * ncx + cx0 + c) : 0.0;
            sy[i / kRsdTile][c] = (t < T && cy0 + c < ncy) ? __ldg(ay + (int64_t)t * ncy + cy0 + c) : 0.0;
        }
        __syncthreads();
#pragma unroll
        for (int32_t tt = 0; tt < kRsdFrames; ++tt) D += sx[tt][lx] * sy[tt][ly];     // (frames past T add 0 * 0)
        __syncthreads();
    }
    if (cx0 + lx < ncx && cy0 + ly < ncy)
        rsd[ti.rsd_off + (int64_t)(cy0 + ly) * ncx + cx0 + lx] = (D > 0.0) ? (float)(1.0 / sqrt(D)) : 0.0f;
}

void launch_class_tables(cudaStream_t st, const float *cls_v, const float *cls_a, const float *times,
                         const float *jitter, int32_t n_cls, int32_t n_x, int32_t T, double t0,
                         double prf_sigma, int32_t filter, const float *prf_tab, int32_t n_phase, int32_t *shift,
                         float *g, double *gd) {
    const int64_t n = (int64_t)n_cls * T;
    k_class_tables<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(cls_v, cls_a, times, jitter, n_cls, n_x, T,
                                                                 t0, prf_sigma, filter, prf_tab, n_phase, shift, g, gd);
}

void launch_border_tables(cudaStream_t st, const int32_t *shift, const double *gd, const double *qd,
                          const AxisBorder *border, const int64_t *off, int32_t n_cls, int32_t n_x,
                          int32_t max_n, int32_t T, int32_t W, int32_t H, double *out) {
    const int64_t n = (int64_t)max_n * T;
    dim3 grid((unsigned)((n + 255) / 256), (unsigned)n_cls);
    k_border_tables<<<grid, 256, 0, st>>>(shift, gd, qd, border, off, n_x, T, W, H, out);
}

void launch_rsd_tables(cudaStream_t st, const TrajInfo *traj, int32_t n_traj, int64_t max_tiles,
                       const double *ab, const int64_t *off, int32_t n_x, int32_t T, float *rsd) {
    dim3 grid((unsigned)max_tiles, (unsigned)n_traj);          // max_tiles: 16 x 16 tiles of the largest table
    k_rsd_tables<<<grid, kRsdTile * kRsdTile, 0, st>>>(traj, ab, off, n_x, T, rsd);
}

}  // namespace tno
