// Generic search kernel: one thread per (trajectory, start pixel), any H and W, no TMA.
// It is the path for shapes the separable TMA kernel does not take (W % 4 != 0, unaligned
// frames) and the in-library regression reference for it.  Same arithmetic definition:
//   N = sum_t q_t sum_{j,i} gy[j] gx[i] R_t(x + sx + i, y + sy + j),  off-frame taps dropped
// (BASELINE.json:north_star; Eq. 5, with the zeros of F skipped, L118).
// Each frame's 25 taps are summed in float32, the sum over frames is kept in float64.
#include "kernels.h"

namespace tno {

__global__ void __launch_bounds__(256)
k_search_generic(const float *__restrict__ frames, const float *__restrict__ valid, int32_t T, int32_t H, int32_t W,
                 ClassTables tab, const TrajInfo *__restrict__ traj, const float *__restrict__ rsd,
                 int32_t k_first, float *__restrict__ out_snr) {
    const int32_t x = blockIdx.x * 32 + threadIdx.x;
    const int32_t y = blockIdx.y * 8 + threadIdx.y;
    const int32_t kl = blockIdx.z, k = k_first + kl;
    if (x >= W || y >= H) return;
    const TrajInfo ti = traj[k];
    const int64_t cx0 = (int64_t)ti.xc * T, cy0 = (int64_t)(tab.n_x + ti.yc) * T;
    double acc = 0.0, accd = 0.0;
    for (int32_t t = 0; t < T; ++t) {
        const int32_t px = x + tab.shift[cx0 + t] - 2, py = y + tab.shift[cy0 + t] - 2;
        const float *gx = tab.g + (cx0 + t) * 5, *gy = tab.g + (cy0 + t) * 5;
        const float *f = frames + (int64_t)t * H * W;
        const float *vf = valid ? valid + (int64_t)t * H * W : nullptr;
        float p = 0.0f, pd = 0.0f;
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            const int32_t yy = py + j;
            if (yy < 0 || yy >= H) continue;
            const float *row = f + (int64_t)yy * W;
            float r = 0.0f, rd = 0.0f;
#pragma unroll
            for (int i = 0; i < 5; ++i) {
                const int32_t xx = px + i;
                if (xx >= 0 && xx < W) {
                    r = fmaf(gx[i], __ldg(row + xx), r);
                    if (vf) rd = fmaf(gx[i] * gx[i], __ldg(vf + (int64_t)yy * W + xx), rd);
                }
            }
            p = fmaf(gy[j], r, p);
            pd = fmaf(gy[j] * gy[j], rd, pd);
        }
        acc += (double)(p * tab.qf[t]);
        accd += (double)(pd * tab.qf[t]);
    }
    float s;
    if (valid) {
        s = accd > 0.0 ? (float)(acc / sqrt(accd)) : 0.0f;
    } else {
        const int32_t cx = border_class(x, ti.bx, W), cy = border_class(y, ti.by, H);
        s = (float)acc * rsd[ti.rsd_off + (int64_t)cy * ti.bx.n + cx];
    }
    out_snr[((int64_t)kl * H + y) * W + x] = s;
}

// Filter 4 (tno_mf_set_prf_table2d): a tabulated NON-separable PRF.  The 5 x 5 block of the frame
// is the one at (row of the y-phase, column of the x-phase) of the table [n_py][n_px][5][5]; D is not separable
// either, so it is accumulated next to N (with the validity weights, if any).
__global__ void __launch_bounds__(256)
k_search_generic25(const float *__restrict__ frames, const float *__restrict__ valid, int32_t T, int32_t H, int32_t W,
                   ClassTables tab, const TrajInfo *__restrict__ traj, const float *__restrict__ tab2, int32_t n_px,
                   int32_t k_first, float *__restrict__ out_snr) {
    const int32_t x = blockIdx.x * 32 + threadIdx.x;
    const int32_t y = blockIdx.y * 8 + threadIdx.y;
    const int32_t kl = blockIdx.z, k = k_first + kl;
    if (x >= W || y >= H) return;
    const TrajInfo ti = traj[k];
    const int64_t cx0 = (int64_t)ti.xc * T, cy0 = (int64_t)(tab.n_x + ti.yc) * T;
    double acc = 0.0, accd = 0.0;
    for (int32_t t = 0; t < T; ++t) {
        const int32_t px = x + tab.shift[cx0 + t] - 2, py = y + tab.shift[cy0 + t] - 2;
        const int32_t rx = (int32_t)tab.gd[(cx0 + t) * 5], ry = (int32_t)tab.gd[(cy0 + t) * 5];
        const float *g = tab2 + ((int64_t)ry * n_px + rx) * 25;
        const float *f = frames + (int64_t)t * H * W;
        const float *vf = valid ? valid + (int64_t)t * H * W : nullptr;
        float p = 0.0f, pd = 0.0f;
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            const int32_t yy = py + j;
            if (yy < 0 || yy >= H) continue;
            const float *row = f + (int64_t)yy * W;
#pragma unroll
            for (int i = 0; i < 5; ++i) {
                const int32_t xx = px + i;
                if (xx >= 0 && xx < W) {
                    const float w = __ldg(g + 5 * j + i);
                    p = fmaf(w, __ldg(row + xx), p);
                    pd = fmaf(w * w, vf ? __ldg(vf + (int64_t)yy * W + xx) : 1.0f, pd);
                }
            }
        }
        acc += (double)(p * tab.qf[t]);
        accd += (double)(pd * tab.qf[t]);
    }
    out_snr[((int64_t)kl * H + y) * W + x] = accd > 0.0 ? (float)(acc / sqrt(accd)) : 0.0f;
}

void launch_search_generic25(cudaStream_t st, const float *frames, const float *valid, int32_t T, int32_t H, int32_t W,
                             const ClassTables &tab, const TrajInfo *traj, const float *tab2, int32_t n_px,
                             int32_t k_first, int32_t k_count, float *out_snr) {
    dim3 block(32, 8);
    dim3 grid((unsigned)((W + 31) / 32), (unsigned)((H + 7) / 8), (unsigned)k_count);
    k_search_generic25<<<grid, block, 0, st>>>(frames, valid, T, H, W, tab, traj, tab2, n_px, k_first, out_snr);
}

void launch_search_generic(cudaStream_t st, const float *frames, const float *valid, int32_t T, int32_t H, int32_t W,
                           const ClassTables &tab, const TrajInfo *traj, const float *rsd,
                           int32_t k_first, int32_t k_count, float *out_snr) {
    dim3 block(32, 8);
    dim3 grid((unsigned)((W + 31) / 32), (unsigned)((H + 7) / 8), (unsigned)k_count);
    k_search_generic<<<grid, block, 0, st>>>(frames, valid, T, H, W, tab, traj, rsd, k_first, out_snr);
}

}  // namespace tno
