// Interpreting scores (section 3.3):
//   k_max_map    M(x,y) = max_k S_k(x,y) and the smallest k that attains it -- "We take the maximum
//                score across the filter bank, which then tells us the most likely trajectory" (L112)
//   k_sat_rows / k_sat_cols   float64 summed-area tables of M and M^2
//   k_local_z    Z = M / sigma_box, sigma_box = population standard deviation of M in the box x box
//                square centred on the pixel, clipped to the frame -- "we compute the standard
//                deviation of the scores in the 255 x 255 square centered on a pixel. We represent
//                our scores in units of sigma" (L124)
//   k_set_argk   writes the arg-max trajectory into the candidate records of the Z map
// All of it is HBM-bound streaming work: K maps read once, then a few passes over one map.
#include "kernels.h"

namespace tno {

// grid-stride over groups of 4 pixels (n_px % 4 == 0 is not required: scalar tail)
__global__ void __launch_bounds__(256)
k_max_map(const float *__restrict__ snr, int32_t K, int64_t n_px, float *__restrict__ out_max,
          int32_t *__restrict__ out_argk) {
    const int64_t n4 = n_px / 4;
    // (out_argk == NULL has address 0: aligned)
    const bool vec = ((reinterpret_cast<uintptr_t>(snr) | reinterpret_cast<uintptr_t>(out_max) |
                       reinterpret_cast<uintptr_t>(out_argk)) & 15u) == 0 && (n_px % 4) == 0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x, id = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (vec) {
        for (int64_t i = id; i < n4; i += stride) {
            float4 m = __ldcs(reinterpret_cast<const float4 *>(snr) + i);
            int4 a = make_int4(0, 0, 0, 0);
            for (int32_t k = 1; k < K; ++k) {
                const float4 v = __ldcs(reinterpret_cast<const float4 *>(snr + (int64_t)k * n_px) + i);
                if (v.x > m.x) { m.x = v.x; a.x = k; }
                if (v.y > m.y) { m.y = v.y; a.y = k; }
                if (v.z > m.z) { m.z = v.z; a.z = k; }
                if (v.w > m.w) { m.w = v.w; a.w = k; }
            }
            reinterpret_cast<float4 *>(out_max)[i] = m;
            if (out_argk) reinterpret_cast<int4 *>(out_argk)[i] = a;
        }
    } else {
        for (int64_t i = id; i < n_px; i += stride) {
            float m = snr[i];
            int32_t a = 0;
            for (int32_t k = 1; k < K; ++k) {
                const float v = snr[(int64_t)k * n_px + i];
                if (v > m) { m = v; a = k; }
            }
            out_max[i] = m;
            if (out_argk) out_argk[i] = a;
        }
    }
}

// One block per row: inclusive prefix sums along x of (M, M^2) in float64.
__global__ void __launch_bounds__(256)
k_sat_rows(const float *__restrict__ m, int32_t W, double2 *__restrict__ sat) {
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

// One block per 32 columns, 32 warps: warp w walks the rows [w*chunk, (w+1)*chunk) of its columns
// (lanes across columns: 512-byte coalesced rows of double2), in place.
__global__ void __launch_bounds__(1024)
k_sat_cols(double2 *__restrict__ sat, int32_t H, int32_t W) {
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

__global__ void __launch_bounds__(256)
k_local_z(const float *__restrict__ m, const double2 *__restrict__ sat, int32_t H, int32_t W, int32_t h,
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
    // differences of large sums: a variance below this relative floor is rounding noise of a constant box
    const double floor_v = 1e-12 * (q / n);
    z[(int64_t)y * W + x] = var > floor_v ? (float)((double)m[(int64_t)y * W + x] / sqrt(var)) : 0.0f;
}

__global__ void k_set_argk(tno_mf_cand *__restrict__ cand, int32_t n, const int32_t *__restrict__ argk, int32_t W) {
    const int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    tno_mf_cand c = cand[i];
    c.k = (c.x >= 0) ? argk[(int64_t)c.y * W + c.x] : -1;
    cand[i] = c;
}

// Flux estimate A = N / D = SNR * D^(-1/2) per trajectory and start pixel (the score "is a
// direct estimate of the total flux due to that moving object ... but also the magnitude"), from the SNR
// maps and the D^(-1/2) tables of the search that produced them.
// VEC: four neighbouring pixels per thread (16-byte loads and stores; needs W % 4 == 0 and aligned pointers)
template <bool VEC>
__global__ void __launch_bounds__(256)
k_flux(const float *__restrict__ snr, const TrajInfo *__restrict__ traj, const float *__restrict__ rsd,
       int32_t H, int32_t W, float *__restrict__ out) {
    constexpr int PX = VEC ? 4 : 1;
    const int32_t x = (blockIdx.x * 64 + (threadIdx.x & 63)) * PX, y = blockIdx.y * 4 + (threadIdx.x >> 6);
    const int32_t k = blockIdx.z;
    if (x >= W || y >= H) return;
    const TrajInfo ti = traj[k];
    const float *rr = rsd + ti.rsd_off + (int64_t)border_class(y, ti.by, H) * ti.bx.n;
    const int64_t i = ((int64_t)k * H + y) * W + x;
    if (VEC) {
        float4 v = __ldcs(reinterpret_cast<const float4 *>(snr + i));
        v.x *= __ldg(rr + border_class(x, ti.bx, W));
        v.y *= __ldg(rr + border_class(x + 1, ti.bx, W));
        v.z *= __ldg(rr + border_class(x + 2, ti.bx, W));
        v.w *= __ldg(rr + border_class(x + 3, ti.bx, W));
        __stcs(reinterpret_cast<float4 *>(out + i), v);
    } else {
        out[i] = snr[i] * __ldg(rr + border_class(x, ti.bx, W));
    }
}

// Max over the bank fused into the search (tno_mf_search_max): the search keeps, per pixel, the maximum of the keys
// (score order << 32 | ~k) -- k_finish with atomicMax, the generic path with this kernel on its map chunks.
__global__ void __launch_bounds__(256)
k_max_keys_from_maps(const float *__restrict__ maps, int32_t k0, int32_t kc, int64_t n_px,
                     unsigned long long *__restrict__ keys) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_px) return;
    unsigned long long best = keys[i];
    for (int32_t k = 0; k < kc; ++k) {
        const unsigned long long key = make_key(maps[(int64_t)k * n_px + i], (uint32_t)(k0 + k));
        best = key > best ? key : best;
    }
    keys[i] = best;
}

__global__ void __launch_bounds__(256)
k_max_decode(const unsigned long long *__restrict__ keys, int64_t n_px, float *__restrict__ out_max,
             int32_t *__restrict__ out_argk) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_px) return;
    const unsigned long long key = keys[i];
    out_max[i] = ord_to_snr((uint32_t)(key >> 32));
    if (out_argk) out_argk[i] = (int32_t)(~(uint32_t)key);
}

void launch_max_keys_from_maps(cudaStream_t st, const float *maps, int32_t k0, int32_t kc, int64_t n_px, uint64_t *keys) {
    k_max_keys_from_maps<<<(unsigned)((n_px + 255) / 256), 256, 0, st>>>(maps, k0, kc, n_px,
                                                                        reinterpret_cast<unsigned long long *>(keys));
}

void launch_max_decode(cudaStream_t st, const uint64_t *keys, int64_t n_px, float *out_max, int32_t *out_argk) {
    k_max_decode<<<(unsigned)((n_px + 255) / 256), 256, 0, st>>>(reinterpret_cast<const unsigned long long *>(keys),
                                                                n_px, out_max, out_argk);
}

// Non-maximum suppression (reading e6): out = score where the pixel is >= thr and
// beats every other pixel of its (2r+1)^2 window (larger score, or equal score and earlier in row-major order),
// -inf elsewhere.  Only pixels above the threshold scan their window, and they stop at the first loss.
__global__ void __launch_bounds__(256)
k_nms(const float *__restrict__ score, int32_t H, int32_t W, int32_t r, float thr, float *__restrict__ out) {
    const int32_t x = blockIdx.x * 64 + (threadIdx.x & 63), y = blockIdx.y * 4 + (threadIdx.x >> 6);
    if (x >= W || y >= H) return;
    const float s = score[(int64_t)y * W + x];
    bool keep = s >= thr;
    if (keep) {
        const int32_t x0 = max(0, x - r), x1 = min(W - 1, x + r), y0 = max(0, y - r), y1 = min(H - 1, y + r);
        for (int32_t yy = y0; yy <= y1 && keep; ++yy) {
            const float *row = score + (int64_t)yy * W;
            for (int32_t xx = x0; xx <= x1; ++xx) {
                const float q = __ldg(row + xx);
                const bool earlier = yy < y || (yy == y && xx < x);
                if (q > s || (q == s && earlier)) { keep = false; break; }
            }
        }
    }
    out[(int64_t)y * W + x] = keep ? s : -INFINITY;
}

void launch_nms(cudaStream_t st, const float *score, int32_t H, int32_t W, int32_t radius, float thr, float *out) {
    dim3 grid((unsigned)((W + 63) / 64), (unsigned)((H + 3) / 4));
    k_nms<<<grid, 256, 0, st>>>(score, H, W, radius, thr, out);
}

void launch_flux(cudaStream_t st, const float *snr, const TrajInfo *traj, const float *rsd, int32_t K, int32_t H,
                 int32_t W, float *out) {
    const bool vec = W % 4 == 0 && ((reinterpret_cast<uintptr_t>(snr) | reinterpret_cast<uintptr_t>(out)) & 15u) == 0;
    if (vec) {
        dim3 grid((unsigned)((W / 4 + 63) / 64), (unsigned)((H + 3) / 4), (unsigned)K);
        k_flux<true><<<grid, 256, 0, st>>>(snr, traj, rsd, H, W, out);
    } else {
        dim3 grid((unsigned)((W + 63) / 64), (unsigned)((H + 3) / 4), (unsigned)K);
        k_flux<false><<<grid, 256, 0, st>>>(snr, traj, rsd, H, W, out);
    }
}

void launch_max_map(cudaStream_t st, const float *snr, int32_t K, int32_t H, int32_t W, float *out_max,
                    int32_t *out_argk, int32_t n_sm) {
    k_max_map<<<(unsigned)(n_sm * 8), 256, 0, st>>>(snr, K, (int64_t)H * W, out_max, out_argk);
}

void launch_local_z(cudaStream_t st, const float *m, int32_t H, int32_t W, int32_t box, void *sat_ws, float *z) {
    double2 *sat = static_cast<double2 *>(sat_ws);
    k_sat_rows<<<(unsigned)H, 256, 0, st>>>(m, W, sat);
    k_sat_cols<<<(unsigned)((W + 31) / 32), 1024, 0, st>>>(sat, H, W);
    dim3 grid((unsigned)((W + 63) / 64), (unsigned)((H + 3) / 4));
    k_local_z<<<grid, 256, 0, st>>>(m, sat, H, W, (box - 1) / 2, z);
}

void launch_set_argk(cudaStream_t st, tno_mf_cand *cand, int32_t n, const int32_t *argk, int32_t W) {
    k_set_argk<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(cand, n, argk, W);
}

}  // namespace tno
