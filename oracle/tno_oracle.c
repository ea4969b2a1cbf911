/*
 * tno_oracle.c -- TEST INFRASTRUCTURE, not product code.
 *
 * Plain, slow, float64 CPU oracle for the matched-filter trajectory search of
 * Ganapathi, "Maximum Likelihood Systematic Effect Modeling and Matched Filtering to Detect
 * Trans-Neptunian Objects with TESS" (arXiv 2209.09848).  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code with the
 * CUDA path under paper_2209_09848_b200/.
 *
 * What it computes (BASELINE.json:north_star; the paper's counterpart is Eq. 5, PAPER.md:L110,
 * "S = D * F", the dot product of the filter with the data at every pixel location, L108, with
 * the filter F = trajectory line convolved with the pixel response function, L106):
 *
 *   for trajectory k = (vx, vy, ax, ay), start pixel (x, y) at the reference epoch t0,
 *   frames t = 0..T-1:
 *       dt = t - t0
 *       dx = vx*dt + ax*dt*dt            dy likewise             displacement in px
 *       sx = floor(dx + 0.5), phx = dx - sx   (ties go up; phase in [-0.5, 0.5))  DESIGN.md c1
 *       for j in -2..2, i in -2..2:                              5x5 window at round(c_t)
 *           px = x + sx + i ; py = y + sy + j
 *           skip the tap if (px, py) is outside the frame        dropped from N and D
 *           g  = exp(-((i - phx)^2 + (j - phy)^2) / (2 prf_sigma^2))     peak-1 Gaussian PRF
 *           N += g * R_t[py][px] / sigma_t^2
 *           D += g * g / sigma_t^2
 *   SNR_k(x, y) = N / sqrt(D) if D > 0 else 0
 *
 * tno_oracle_point is this literally (one exp per tap).  tno_oracle_map evaluates the same sums
 * with (sx, sy, gx[i], gy[j]) computed once per (k, t) -- they do not depend on (x, y) -- and
 * is pinned against tno_oracle_point on small inputs by tests/test_oracle_pins.py.
 * tno_oracle_inject adds A * g(p - c_t) on the same 25 taps with the same rounding ("signal
 * injection corresponds to adding a filter times a flux to the raw data").
 *
 * Parity pins (tests/test_oracle_pins.py): closed form N/D = A and SNR = A sqrt(D) for an
 * injected noiseless source; zero in -> zero out; linearity; integer velocities reduce to
 * scipy.ndimage.correlate + integer shifts; brute force with exact rational displacements;
 * hand-listed tie cases; corner closed form; N(0,1) statistics on pure noise.
 *
 * Inputs are float32 where the C ABI of the product takes float32 (frames, sigma_t, trajectory
 * parameters, prf_sigma, t0); every value is promoted to double before any arithmetic.
 * Build: gcc -O2 -fopenmp -ffp-contract=off (no fast-math), see oracle/build.py.
 *
 * The frame buffer may be a WINDOW of the full frame: it holds rows [wy0, wy0+wh) and columns
 * [wx0, wx0+ww) of an H x W frame for each t.  A tap that is inside the frame but outside the
 * window is an error (return -1): the caller must pass a window with enough halo.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int T, H, W;            /* full frame geometry */
    int wx0, wy0, ww, wh;   /* window held by the buffer */
} geom_t;

static inline double disp(double v, double a, double dt) { return v * dt + a * dt * dt; }

/* Time of frame t and pointing jitter of frame t (readings f1-f3): the filter is "the line
 * of the trajectory (including the pointing jitter)" and the frames are not equally
 * spaced ("the time-jump that occurs when TESS is transmitting frames to Earth", L116).
 *     c_t = (x, y) + v (tau_t - t0) + a (tau_t - t0)^2 + j_t
 * times == NULL: tau_t = t;  jitter == NULL: j_t = 0;  jitter[2t], jitter[2t+1] = (jx_t, jy_t) in px. */
/* Per-pixel validity / inverse-variance weights (readings h1-h3; "We set the
 * value of bright pixels to 0 because the noise in those pixels will so high"): with valid != NULL
 *     N = sum g F_t(p) / sigma_t^2          (the frames F as they are: the caller has zeroed or
 *                                            down-weighted them, F = R * valid)
 *     D = sum g^2 valid_t(p) / sigma_t^2    (a masked pixel carries no information)
 * valid has the layout of the frames (same window); NULL = all ones. */
/* Filter of one axis at tap offset u = i - phase (readings g2, g3): the PRF as seen by the pixel grid.
 *   mode 0  the point-sampled Gaussian of BASELINE.json:north_star, exp(-u^2 / (2 s^2));
 *   mode 1  shift-stack (after Rice & Laughlin 2020: "a single non-zero value, set to 1, for
 *           each time-slice"): 1 at the rounded position (i = 0), else 0;
 *   mode 2  the pixel-integrated Gaussian: the flux of a unit source at sub-pixel phase `ph` that falls into
 *           pixel i, the integral of the normalised Gaussian density over [i - 1/2, i + 1/2]
 *           = Phi((u + 1/2) / s) - Phi((u - 1/2) / s)   (the PRF is the fraction of the flux
 *           per pixel, "50 % in the peak pixel, 90 % in 2 x 2");
 *   mode 3  a tabulated separable PRF: row floor((ph + 1/2) * n_phase) (clamped) of the table installed with
 *           tno_oracle_set_prf_table, [n_phase][5] fractions for taps i = -2 .. 2, phases uniform over
 *           [-1/2, 1/2).  The table is the ONE piece of global state of this file (test infrastructure). */
static double *g_prf_table = NULL;
static int g_prf_phases = 0;
int tno_oracle_set_prf_table(const double *table, int n_phase) {
    free(g_prf_table);
    g_prf_table = NULL;
    g_prf_phases = 0;
    if (!table || n_phase <= 0) return 0;
    g_prf_table = (double *)malloc(sizeof(double) * 5 * (size_t)n_phase);
    if (!g_prf_table) return -2;
    memcpy(g_prf_table, table, sizeof(double) * 5 * (size_t)n_phase);
    g_prf_phases = n_phase;
    return 0;
}
static inline double tap1(int mode, int i, double ph, double s) {
    if (mode == 1) return i == 0 ? 1.0 : 0.0;
    const double u = (double)i - ph;
    if (mode == 2) {
        const double r = 1.0 / (s * sqrt(2.0));
        return 0.5 * (erf((u + 0.5) * r) - erf((u - 0.5) * r));
    }
    if (mode == 3) {
        int row = (int)floor((ph + 0.5) * (double)g_prf_phases);
        if (row < 0) row = 0;
        if (row > g_prf_phases - 1) row = g_prf_phases - 1;
        return g_prf_table[5 * row + (i + 2)];
    }
    return exp(-(u * u) / (2.0 * s * s));
}
/*   mode 4  a tabulated NON-separable PRF (the real TESS PRF, "50 % of the flux in the peak pixel
 *           and 90 % in 2 x 2", is a 2-D table per 2-D sub-pixel phase, not an outer product): the table installed
 *           with tno_oracle_set_prf_table2d is [n_phase_y][n_phase_x][5][5]; a source at phases (phx, phy) takes
 *           the 5 x 5 block of row floor((phy + 1/2) n_phase_y), column floor((phx + 1/2) n_phase_x) (clamped),
 *           whose entry [j + 2][i + 2] is the response of the pixel at offset (i, j) from the rounded position.
 *           No interpolation.  Second piece of global state of this file. */
static double *g_prf_table2d = NULL;
static int g_prf_phases_y = 0, g_prf_phases_x = 0;
int tno_oracle_set_prf_table2d(const double *table, int n_phase_y, int n_phase_x) {
    free(g_prf_table2d);
    g_prf_table2d = NULL;
    g_prf_phases_y = g_prf_phases_x = 0;
    if (!table || n_phase_y <= 0 || n_phase_x <= 0) return 0;
    const size_t n = (size_t)25 * (size_t)n_phase_y * (size_t)n_phase_x;
    g_prf_table2d = (double *)malloc(sizeof(double) * n);
    if (!g_prf_table2d) return -2;
    memcpy(g_prf_table2d, table, sizeof(double) * n);
    g_prf_phases_y = n_phase_y;
    g_prf_phases_x = n_phase_x;
    return 0;
}
static inline int phase_row(double ph, int n) {
    int row = (int)floor((ph + 0.5) * (double)n);
    if (row < 0) row = 0;
    if (row > n - 1) row = n - 1;
    return row;
}
/* the filter value at tap (i, j) for any mode: per-axis products for the separable modes 1-3 */
static inline double tap2(int mode, int i, int j, double phx, double phy, double s) {
    if (mode == 4) {
        const int ry = phase_row(phy, g_prf_phases_y), rx = phase_row(phx, g_prf_phases_x);
        return g_prf_table2d[((size_t)(ry * g_prf_phases_x + rx) * 5 + (size_t)(j + 2)) * 5 + (size_t)(i + 2)];
    }
    return tap1(mode, i, phx, s) * tap1(mode, j, phy, s);
}
static inline double frame_dt(const float *times, int t, double t0) {
    return (times ? (double)times[t] : (double)t) - t0;
}
static inline double jit(const float *jitter, int t, int axis) {
    return jitter ? (double)jitter[2 * t + axis] : 0.0;
}

/* round-half-up of a displacement: integer shift s and phase d - s in [-0.5, 0.5) */
static inline void split(double d, int *s, double *ph) {
    double f = floor(d + 0.5);
    *s = (int)f;
    *ph = d - f;
}

int tno_oracle_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* literal definition, one exp per tap */
int tno_oracle_point_ex(const float *frames, int T, int H, int W,
                        int wx0, int wy0, int ww, int wh,
                        const float *sigma_t, const float *times, const float *jitter, const float *valid,
                        int mode, const float *traj4, float prf_sigma_f, float t0_f,
                        int x, int y, double *N_out, double *D_out, double *snr_out)
{
    const double vx = traj4[0], vy = traj4[1], ax = traj4[2], ay = traj4[3];
    const double s = prf_sigma_f, t0 = t0_f;
    double N = 0.0, D = 0.0;
    for (int t = 0; t < T; ++t) {
        const double dt = frame_dt(times, t, t0);
        int sx, sy; double phx, phy;
        split(disp(vx, ax, dt) + jit(jitter, t, 0), &sx, &phx);
        split(disp(vy, ay, dt) + jit(jitter, t, 1), &sy, &phy);
        const double sig = sigma_t[t];
        const double q = 1.0 / (sig * sig);
        for (int j = -2; j <= 2; ++j) {
            for (int i = -2; i <= 2; ++i) {
                const int px = x + sx + i, py = y + sy + j;
                if (px < 0 || px >= W || py < 0 || py >= H) continue;
                if (px < wx0 || px >= wx0 + ww || py < wy0 || py >= wy0 + wh) return -1;
                const double ux = (double)i - phx, uy = (double)j - phy;
                const double g = mode != 0 ? tap2(mode, i, j, phx, phy, s)
                                           : exp(-(ux * ux + uy * uy) / (2.0 * s * s));
                const size_t idx = ((size_t)t * wh + (size_t)(py - wy0)) * ww + (size_t)(px - wx0);
                const double R = frames[idx];
                N += g * R * q;
                D += valid ? g * g * q * (double)valid[idx] : g * g * q;
            }
        }
    }
    if (N_out) *N_out = N;
    if (D_out) *D_out = D;
    if (snr_out) *snr_out = (D > 0.0) ? N / sqrt(D) : 0.0;
    return 0;
}

int tno_oracle_point(const float *frames, int T, int H, int W,
                     int wx0, int wy0, int ww, int wh,
                     const float *sigma_t, const float *traj4, float prf_sigma_f, float t0_f,
                     int x, int y, double *N_out, double *D_out, double *snr_out)
{
    return tno_oracle_point_ex(frames, T, H, W, wx0, wy0, ww, wh, sigma_t, NULL, NULL, NULL, 0, traj4,
                               prf_sigma_f, t0_f, x, y, N_out, D_out, snr_out);
}

/* same sums, per-(k,t) quantities hoisted out of the pixel loop.
 * Region of start pixels: x in [x_lo, x_hi), y in [y_lo, y_hi).
 * out_snr / out_N / out_D: double [K][y_hi-y_lo][x_hi-x_lo]; out_N, out_D may be NULL. */
int tno_oracle_map_ex(const float *frames, int T, int H, int W,
                      int wx0, int wy0, int ww, int wh,
                      const float *sigma_t, const float *times, const float *jitter, const float *valid,
                      int mode, const float *traj, int K,
                      float prf_sigma_f, float t0_f,
                      int x_lo, int x_hi, int y_lo, int y_hi,
                      double *out_snr, double *out_N, double *out_D)
{
    const double s = prf_sigma_f, t0 = t0_f;
    const int rw = x_hi - x_lo, rh = y_hi - y_lo;
    if (rw <= 0 || rh <= 0 || K <= 0 || T <= 0) return -2;
    int *SX = (int *)malloc(sizeof(int) * (size_t)T * 2);
    double *G = (double *)malloc(sizeof(double) * (size_t)T * 11);
    double *G2 = mode == 4 ? (double *)malloc(sizeof(double) * (size_t)T * 25) : NULL;   /* mode 4: [t][j][i] */
    if (!SX || !G || (mode == 4 && !G2)) { free(SX); free(G); free(G2); return -3; }
    int err = 0;
    for (int k = 0; k < K; ++k) {
        const double vx = traj[4 * k + 0], vy = traj[4 * k + 1];
        const double ax = traj[4 * k + 2], ay = traj[4 * k + 3];
        for (int t = 0; t < T; ++t) {
            const double dt = frame_dt(times, t, t0);
            int sx, sy; double phx, phy;
            split(disp(vx, ax, dt) + jit(jitter, t, 0), &sx, &phx);
            split(disp(vy, ay, dt) + jit(jitter, t, 1), &sy, &phy);
            SX[2 * t] = sx; SX[2 * t + 1] = sy;
            for (int i = -2; i <= 2; ++i) {
                G[11 * t + (i + 2)] = mode == 4 ? 0.0 : tap1(mode, i, phx, s);
                G[11 * t + 5 + (i + 2)] = mode == 4 ? 0.0 : tap1(mode, i, phy, s);
            }
            if (mode == 4)
                for (int j = -2; j <= 2; ++j)
                    for (int i = -2; i <= 2; ++i) G2[25 * t + 5 * (j + 2) + (i + 2)] = tap2(4, i, j, phx, phy, s);
            const double sig = sigma_t[t];
            G[11 * t + 10] = 1.0 / (sig * sig);
        }
        double *Nk = (double *)calloc((size_t)rw * rh, sizeof(double));
        double *Dk = (double *)calloc((size_t)rw * rh, sizeof(double));
        if (!Nk || !Dk) { free(Nk); free(Dk); err = -3; break; }
#pragma omp parallel for schedule(static) reduction(min : err)
        for (int y = y_lo; y < y_hi; ++y) {
            double *Nr = Nk + (size_t)(y - y_lo) * rw;
            double *Dr = Dk + (size_t)(y - y_lo) * rw;
            for (int t = 0; t < T; ++t) {
                const int sx = SX[2 * t], sy = SX[2 * t + 1];
                const double *gx = G + 11 * t, *gy = G + 11 * t + 5;
                const double q = G[11 * t + 10];
                for (int j = -2; j <= 2; ++j) {
                    const int py = y + sy + j;
                    if (py < 0 || py >= H) continue;
                    if (py < wy0 || py >= wy0 + wh) { err = -1; continue; }
                    const float *row = frames + ((size_t)t * wh + (size_t)(py - wy0)) * ww;
                    const float *vrow = valid ? valid + ((size_t)t * wh + (size_t)(py - wy0)) * ww : NULL;
                    for (int i = -2; i <= 2; ++i) {
                        const double g = G2 ? G2[25 * t + 5 * (j + 2) + (i + 2)] : gx[i + 2] * gy[j + 2];
                        const double wN = g * q, wD = g * g * q;
                        int xa = x_lo, xb = x_hi;           /* start pixels with px inside the frame */
                        if (xa + sx + i < 0) xa = -(sx + i);
                        if (xb + sx + i > W) xb = W - (sx + i);
                        if (xa >= xb) continue;
                        if (xa + sx + i < wx0 || xb + sx + i > wx0 + ww) { err = -1; continue; }
                        const float *src = row + (sx + i - wx0);
                        const float *vsrc = vrow ? vrow + (sx + i - wx0) : NULL;
                        for (int x = xa; x < xb; ++x) {
                            Nr[x - x_lo] += wN * (double)src[x];
                            Dr[x - x_lo] += vsrc ? wD * (double)vsrc[x] : wD;
                        }
                    }
                }
            }
        }
        for (size_t p = 0; p < (size_t)rw * rh; ++p) {
            const double D = Dk[p];
            out_snr[(size_t)k * rw * rh + p] = (D > 0.0) ? Nk[p] / sqrt(D) : 0.0;
            if (out_N) out_N[(size_t)k * rw * rh + p] = Nk[p];
            if (out_D) out_D[(size_t)k * rw * rh + p] = D;
        }
        free(Nk); free(Dk);
        if (err) break;
    }
    free(SX); free(G); free(G2);
    return err;
}

int tno_oracle_map(const float *frames, int T, int H, int W,
                   int wx0, int wy0, int ww, int wh,
                   const float *sigma_t, const float *traj, int K,
                   float prf_sigma_f, float t0_f,
                   int x_lo, int x_hi, int y_lo, int y_hi,
                   double *out_snr, double *out_N, double *out_D)
{
    return tno_oracle_map_ex(frames, T, H, W, wx0, wy0, ww, wh, sigma_t, NULL, NULL, NULL, 0, traj, K,
                             prf_sigma_f, t0_f, x_lo, x_hi, y_lo, y_hi, out_snr, out_N, out_D);
}

/* Injection: for each source, in order, add amp * g(p - c_t) on the 25 taps of
 * every frame, computed in double and rounded once to float32:
 *     R <- (float)((double)R + amp * g).
 * Works on a full-frame buffer [T][H][W].  traj: [n][4] per source. */
int tno_oracle_inject_ex(float *frames, int T, int H, int W, const float *times, const float *jitter,
                         const float *traj, const int *xs, const int *ys, const float *amp, int n,
                         float prf_sigma_f, float t0_f)
{
    const double s = prf_sigma_f, t0 = t0_f;
    for (int m = 0; m < n; ++m) {
        const double vx = traj[4 * m + 0], vy = traj[4 * m + 1];
        const double ax = traj[4 * m + 2], ay = traj[4 * m + 3];
        const double A = amp[m];
        for (int t = 0; t < T; ++t) {
            const double dt = frame_dt(times, t, t0);
            int sx, sy; double phx, phy;
            split(disp(vx, ax, dt) + jit(jitter, t, 0), &sx, &phx);
            split(disp(vy, ay, dt) + jit(jitter, t, 1), &sy, &phy);
            for (int j = -2; j <= 2; ++j) {
                for (int i = -2; i <= 2; ++i) {
                    const int px = xs[m] + sx + i, py = ys[m] + sy + j;
                    if (px < 0 || px >= W || py < 0 || py >= H) continue;
                    const double ux = (double)i - phx, uy = (double)j - phy;
                    const double g = exp(-(ux * ux + uy * uy) / (2.0 * s * s));
                    float *p = frames + ((size_t)t * H + (size_t)py) * W + (size_t)px;
                    *p = (float)((double)*p + A * g);
                }
            }
        }
    }
    return 0;
}

/* The same with the filter of `mode` (tap2): the source as modes 1-4 see it. */
int tno_oracle_inject_mode(float *frames, int T, int H, int W, const float *times, const float *jitter, int mode,
                         const float *traj, const int *xs, const int *ys, const float *amp, int n,
                         float prf_sigma_f, float t0_f)
{
    const double s = prf_sigma_f, t0 = t0_f;
    for (int m = 0; m < n; ++m) {
        const double vx = traj[4 * m + 0], vy = traj[4 * m + 1];
        const double ax = traj[4 * m + 2], ay = traj[4 * m + 3];
        const double A = amp[m];
        for (int t = 0; t < T; ++t) {
            const double dt = frame_dt(times, t, t0);
            int sx, sy; double phx, phy;
            split(disp(vx, ax, dt) + jit(jitter, t, 0), &sx, &phx);
            split(disp(vy, ay, dt) + jit(jitter, t, 1), &sy, &phy);
            for (int j = -2; j <= 2; ++j) {
                for (int i = -2; i <= 2; ++i) {
                    const int px = xs[m] + sx + i, py = ys[m] + sy + j;
                    if (px < 0 || px >= W || py < 0 || py >= H) continue;
                    const double g = tap2(mode, i, j, phx, phy, s);
                    float *p = frames + ((size_t)t * H + (size_t)py) * W + (size_t)px;
                    *p = (float)((double)*p + A * g);
                }
            }
        }
    }
    return 0;
}

int tno_oracle_inject(float *frames, int T, int H, int W,
                      const float *traj, const int *xs, const int *ys, const float *amp, int n,
                      float prf_sigma_f, float t0_f)
{
    return tno_oracle_inject_ex(frames, T, H, W, NULL, NULL, traj, xs, ys, amp, n, prf_sigma_f, t0_f);
}

/* ------------------------------------------------------------------------------------------
 * Interpreting scores (section 3.3, L112 and L122-124; readings e1-e4).
 *
 * tno_oracle_best: "We take the maximum score across the filter bank, which then tells us the
 * most likely trajectory, along with the score of that trajectory" (L112):
 *     M(x, y) = max_k S_k(x, y),   A(x, y) = the smallest k that attains it.
 * Scores are float32 (they are the product's output format); comparisons are exact.
 *
 * tno_oracle_local_z: "we compute the standard deviation sigma of the scores in the 255 x 255
 * square centered on a pixel. We represent our scores in units of sigma" (L124):
 *     B(x, y)   = the pixels (x', y') of the frame with |x' - x| <= h and |y' - y| <= h, h = (box-1)/2
 *     mean      = sum_B M / |B|,   var = sum_B (M - mean)^2 / |B|      (population variance)
 *     Z(x, y)   = M(x, y) / sqrt(var)   if var > 0 else 0
 * The two-pass definition is evaluated literally for every pixel (O(H W box^2): small maps only).
 * tno_oracle_local_z_sep uses the separability of the box sums of M and M^2 (row sums, then
 * column sums of those, all float64, var = sum2/|B| - (sum/|B|)^2) and is pinned against the
 * literal form by tests/test_oracle_pins.py; it is what full-size maps are checked against.
 */
int tno_oracle_best(const float *snr, int K, int H, int W, float *out_max, int *out_argk) {
    if (!snr || K < 1 || H < 1 || W < 1 || !out_max || !out_argk) return -2;
    for (long p = 0; p < (long)H * W; ++p) {
        float m = snr[p];
        int a = 0;
        for (int k = 1; k < K; ++k) {
            const float v = snr[(long)k * H * W + p];
            if (v > m) { m = v; a = k; }
        }
        out_max[p] = m;
        out_argk[p] = a;
    }
    return 0;
}

int tno_oracle_local_z(const float *m, int H, int W, int box, double *out_z, double *out_sigma) {
    if (!m || H < 1 || W < 1 || box < 1 || (box & 1) == 0 || !out_z) return -2;
    const int h = (box - 1) / 2;
#pragma omp parallel for schedule(static)
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            const int y0 = y - h < 0 ? 0 : y - h, y1 = y + h >= H ? H - 1 : y + h;
            const int x0 = x - h < 0 ? 0 : x - h, x1 = x + h >= W ? W - 1 : x + h;
            const double n = (double)(y1 - y0 + 1) * (double)(x1 - x0 + 1);
            double s = 0.0;
            for (int yy = y0; yy <= y1; ++yy)
                for (int xx = x0; xx <= x1; ++xx) s += (double)m[(long)yy * W + xx];
            const double mean = s / n;
            double v = 0.0;
            for (int yy = y0; yy <= y1; ++yy)
                for (int xx = x0; xx <= x1; ++xx) {
                    const double d = (double)m[(long)yy * W + xx] - mean;
                    v += d * d;
                }
            v /= n;
            const double sd = v > 0.0 ? sqrt(v) : 0.0;
            if (out_sigma) out_sigma[(long)y * W + x] = sd;
            out_z[(long)y * W + x] = sd > 0.0 ? (double)m[(long)y * W + x] / sd : 0.0;
        }
    return 0;
}

int tno_oracle_local_z_sep(const float *m, int H, int W, int box, double *out_z, double *out_sigma) {
    if (!m || H < 1 || W < 1 || box < 1 || (box & 1) == 0 || !out_z) return -2;
    const int h = (box - 1) / 2;
    double *r1 = (double *)malloc(sizeof(double) * (size_t)H * W);
    double *r2 = (double *)malloc(sizeof(double) * (size_t)H * W);
    if (!r1 || !r2) { free(r1); free(r2); return -3; }
#pragma omp parallel for schedule(static)
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            const int x0 = x - h < 0 ? 0 : x - h, x1 = x + h >= W ? W - 1 : x + h;
            double s = 0.0, q = 0.0;
            for (int xx = x0; xx <= x1; ++xx) {
                const double v = (double)m[(long)y * W + xx];
                s += v;
                q += v * v;
            }
            r1[(long)y * W + x] = s;
            r2[(long)y * W + x] = q;
        }
#pragma omp parallel for schedule(static)
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            const int y0 = y - h < 0 ? 0 : y - h, y1 = y + h >= H ? H - 1 : y + h;
            const int x0 = x - h < 0 ? 0 : x - h, x1 = x + h >= W ? W - 1 : x + h;
            const double n = (double)(y1 - y0 + 1) * (double)(x1 - x0 + 1);
            double s = 0.0, q = 0.0;
            for (int yy = y0; yy <= y1; ++yy) {
                s += r1[(long)yy * W + x];
                q += r2[(long)yy * W + x];
            }
            const double mean = s / n;
            double v = q / n - mean * mean;
            if (v < 0.0) v = 0.0;
            const double sd = v > 0.0 ? sqrt(v) : 0.0;
            if (out_sigma) out_sigma[(long)y * W + x] = sd;
            out_z[(long)y * W + x] = sd > 0.0 ? (double)m[(long)y * W + x] / sd : 0.0;
        }
    free(r1);
    free(r2);
    return 0;
}
