// Signal injection: R_t(p) <- (float)((double)R_t(p) + A g(p - c_t)) on the 25
// window taps of every frame.  One thread per frame applies the sources in order, so overlapping
// sources give a deterministic result.
#include "kernels.h"

namespace tno {

// d = (v*dt + (a*dt)*dt) + j, every operation separately rounded: the evaluation of k_class_tables (tables.cu)
__device__ __forceinline__ void axis_pos(double v, double a, double dt, double j, int32_t *s, double *ph) {
    const double d = __dadd_rn(__dadd_rn(__dmul_rn(v, dt), __dmul_rn(__dmul_rn(a, dt), dt)), j);
    const double f = floor(__dadd_rn(d, 0.5));
    *s = (int32_t)f;
    *ph = __dsub_rn(d, f);
}

__global__ void k_inject(float *__restrict__ frames, int32_t T, int32_t H, int32_t W,
                         const SourceDev *__restrict__ src, int32_t n_src, double prf_sigma,
                         double t0, int32_t filter, const float *__restrict__ prf_tab, int32_t n_phase,
                         const float *__restrict__ times, const float *__restrict__ jitter) {
    const int32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    const double dt = __dsub_rn(times ? (double)times[t] : (double)t, t0);
    const double jx = jitter ? (double)jitter[2 * t] : 0.0, jy = jitter ? (double)jitter[2 * t + 1] : 0.0;
    const double inv = 1.0 / (2.0 * prf_sigma * prf_sigma);
    float *f = frames + (int64_t)t * H * W;
    for (int32_t m = 0; m < n_src; ++m) {
        const SourceDev s = src[m];
        int32_t sx, sy;
        double phx, phy;
        axis_pos((double)s.vx, (double)s.ax, dt, jx, &sx, &phx);
        axis_pos((double)s.vy, (double)s.ay, dt, jy, &sy, &phy);
        for (int j = -2; j <= 2; ++j) {
            const int32_t py = s.y + sy + j;
            if (py < 0 || py >= H) continue;
            for (int i = -2; i <= 2; ++i) {
                const int32_t px = s.x + sx + i;
                if (px < 0 || px >= W) continue;
                const double ux = (double)i - phx, uy = (double)j - phy;
                // filters 2, 3 and 4 render the source with their own PRF; 0 and 1 with the point-sampled
                // Gaussian (shift-stack is a way to search, not a PRF)
                double g;
                if (filter == 4) {
                    // non-separable table [n_py][n_px][5][5], n_phase = n_py << 16 | n_px
                    const int32_t npx = n_phase & 0xffff, npy = n_phase >> 16;
                    int32_t rx = (int32_t)floor((phx + 0.5) * (double)npx), ry = (int32_t)floor((phy + 0.5) * (double)npy);
                    rx = rx < 0 ? 0 : (rx > npx - 1 ? npx - 1 : rx);
                    ry = ry < 0 ? 0 : (ry > npy - 1 ? npy - 1 : ry);
                    g = (double)prf_tab[((int64_t)ry * npx + rx) * 25 + 5 * (j + 2) + (i + 2)];
                } else {
                    g = filter >= 2 ? prf_tap(filter, i + 2, phx, prf_sigma, prf_tab, n_phase) *
                                          prf_tap(filter, j + 2, phy, prf_sigma, prf_tab, n_phase)
                                    : exp(-(ux * ux + uy * uy) * inv);
                }
                float *p = f + (int64_t)py * W + px;
                *p = (float)((double)*p + (double)s.amp * g);
            }
        }
    }
}

void launch_inject(cudaStream_t st, float *frames, int32_t T, int32_t H, int32_t W,
                   const SourceDev *src, int32_t n_src, double prf_sigma, double t0, int32_t filter,
                   const float *prf_tab, int32_t n_phase, const float *times, const float *jitter) {
    k_inject<<<(unsigned)((T + 63) / 64), 64, 0, st>>>(frames, T, H, W, src, n_src, prf_sigma, t0, filter, prf_tab,
                                                       n_phase, times, jitter);
}

}  // namespace tno
