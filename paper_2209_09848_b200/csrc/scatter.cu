// Low-resolution scattered-light model (section 3.1, Eq. 1-4, second part):
//     D_t = U(S_t) + B + B_theta . theta_t^k + eps,      L = sum_{t,i,j} L_delta(D_t - pred_t)_{ij}
// D: the data downsampled to N x N (512), S_t: n x n (64) per frame, U: bilinear upsampling, the background terms
// as in background.cu.  "We minimize this convex loss over B, B_theta, S_t using the L-BFGS algorithm" (L94).
//   k_downsample        block means, 2048^2 -> 512^2 (L69)
//   k_scatter_resid     one thread per low-resolution pixel walks the frames: residual, loss, dL/dbeta in registers,
//                       psi = clip(r) to a scratch stack
//   k_scatter_gs        dL/dS_t = -U^T psi_t as a gather: one thread per (t, a, b) sums its footprint (no atomics)
//   k_dot / k_sum_partials / k_axpy / k_absmax   the vector algebra of L-BFGS, two-stage reductions in a fixed
//                       order (float64), so a fit is reproducible run to run
//   scatter_fit         the L-BFGS driver (host loop, two-loop recursion, Armijo backtracking)
//   k_scatter_subtract  frames -= U(S_t) at full resolution, the hand-over to tno_mf_background
// Everything is HBM-bound streaming over a 1 GB stack (T = 1000, N = 512); the paper quotes ~40 s for this solve.
#include <algorithm>
#include <cmath>
#include <vector>

#include "kernels.h"

namespace tno {

// 1-D bilinear stencil of output pixel i (reading s2): centre at u = (i + 1/2) n / N - 1/2, clamped to [0, n - 1];
// inputs floor(u) and floor(u) + 1 (clamped) with weights 1 - frac(u), frac(u).  The host tabulates floor(u) and
// frac(u) per output pixel in float64 (bilinear_table) -- the kernels only look them up.
void bilinear_table(int32_t N, int32_t n, int32_t *i0, float *w) {
    for (int32_t i = 0; i < N; ++i) {
        double u = ((double)i + 0.5) * (double)n / (double)N - 0.5;
        u = std::min(std::max(u, 0.0), (double)(n - 1));
        const double f = std::floor(u);
        i0[i] = (int32_t)f;
        w[i] = (float)(u - f);
    }
}

__global__ void __launch_bounds__(256)
k_downsample(const float *__restrict__ frames, int32_t H, int32_t W, int32_t f, float *__restrict__ out) {
    const int32_t Wo = W / f, Ho = H / f;
    const int32_t x = blockIdx.x * 64 + (threadIdx.x & 63), y = blockIdx.y * 4 + (threadIdx.x >> 6), t = blockIdx.z;
    if (x >= Wo || y >= Ho) return;
    const float *src = frames + ((int64_t)t * H + (int64_t)y * f) * W + (int64_t)x * f;
    double s = 0.0;
    for (int32_t j = 0; j < f; ++j)
        for (int32_t i = 0; i < f; ++i) s += (double)__ldg(src + (int64_t)j * W + i);
    out[((int64_t)t * Ho + y) * Wo + x] = (float)(s / ((double)f * f));
}

constexpr int kRedBlocks = 1024;       // partial sums of every reduction
constexpr int kLossPartials = 8192;    // capacity of the loss partials (blocks of the evaluation kernels)

// block-wide sum in a fixed order -> partials[blockIdx.x]
__device__ __forceinline__ void block_sum_to(double v, double *__restrict__ partials) {
    __shared__ double sh[8];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += sh[w];
        partials[blockIdx.x] = s;
    }
}

__global__ void __launch_bounds__(256)
k_scatter_resid(const float *__restrict__ D, int32_t T, int32_t N, int32_t n, const float *__restrict__ phi /* [T][8] */,
                const int32_t *__restrict__ bi0, const float *__restrict__ bw, float delta, const float *__restrict__ beta, const float *__restrict__ S, float *__restrict__ psi,
                float *__restrict__ g_beta, double *__restrict__ partials) {
    const int64_t n_px = (int64_t)N * N;
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double loss = 0.0;
    if (p < n_px) {
        const int32_t i = (int32_t)(p / N), j = (int32_t)(p % N);
        const int32_t i0 = bi0[i], j0 = bi0[j], i1 = min(i0 + 1, n - 1), j1 = min(j0 + 1, n - 1);
        const float wy = bw[i], wx = bw[j];
        const float w00 = (1.f - wy) * (1.f - wx), w01 = (1.f - wy) * wx, w10 = wy * (1.f - wx), w11 = wy * wx;
        const int32_t o00 = i0 * n + j0, o01 = i0 * n + j1, o10 = i1 * n + j0, o11 = i1 * n + j1;
        float b[6], g[6];
#pragma unroll
        for (int k = 0; k < 6; ++k) { b[k] = beta[k * n_px + p]; g[k] = 0.f; }
#pragma unroll 4
        for (int32_t t = 0; t < T; ++t) {
            const float4 qa = __ldg(reinterpret_cast<const float4 *>(phi + 8 * (int64_t)t));
            const float2 qb = __ldg(reinterpret_cast<const float2 *>(phi + 8 * (int64_t)t + 4));
            const float q[6] = {qa.x, qa.y, qa.z, qa.w, qb.x, qb.y};
            const float *St = S + (int64_t)t * n * n;
            float pred = w00 * __ldg(St + o00) + w01 * __ldg(St + o01) + w10 * __ldg(St + o10) + w11 * __ldg(St + o11);
#pragma unroll
            for (int k = 0; k < 6; ++k) pred = fmaf(q[k], b[k], pred);
            const float r = D[(int64_t)t * n_px + p] - pred;
            const float a = fabsf(r);
            loss += (double)(a <= delta ? 0.5f * r * r : delta * (a - 0.5f * delta));       // Eq. 4
            const float c = fminf(fmaxf(r, -delta), delta);
            psi[(int64_t)t * n_px + p] = c;
#pragma unroll
            for (int k = 0; k < 6; ++k) g[k] = fmaf(q[k], c, g[k]);
        }
#pragma unroll
        for (int k = 0; k < 6; ++k) g_beta[k * n_px + p] = -g[k];
    }
    block_sum_to(loss, partials);
}

// ---- bulk-copy staged variant of k_scatter_resid (N % 4 == 0, aligned): the structure of k_background_bulk --------
// 128 consumer threads own four neighbouring pixels of a row each; a fifth warp requests every frame's 512 pixels
// as one cp.async.bulk (2 KB, one address translation) into a ring of 3 stages x 8 frames together with the 8 rows of
// phi.  The walk over the frames with ordinary loads (k_scatter_resid) is bound by TLB misses and by the few
// loads a thread can keep in flight (1.7 TB/s); see DESIGN.md 8f / 8g.
__device__ __forceinline__ uint32_t sc_smem(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void sc_wait(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n.reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n}\n"
            : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}

template <int NT, int NS, int FS, int SF /* floats of S staged per frame */>
__global__ void __launch_bounds__(NT + 32, 2048 / (NT + 32) > 4 ? 4 : 2048 / (NT + 32))
k_scatter_resid_bulk(const float *__restrict__ D, int32_t T, int32_t N, int32_t n, const float *__restrict__ phi,
                     const int32_t *__restrict__ bi0, const float *__restrict__ bw, float delta,
                     const float *__restrict__ beta, const float *__restrict__ S, float *__restrict__ psi,
                     float *__restrict__ g_beta, double *__restrict__ partials) {
    constexpr int PX = 2;                                        // neighbouring pixels per thread
    constexpr int PXF = NT * PX, STAGE = FS * (PXF + 8 + SF);
    extern __shared__ __align__(128) float ring[];               // [NS][STAGE]: FS x pixels, FS x phi, FS x rows of S_t
    __shared__ __align__(8) uint64_t bars[2 * NS];
    __shared__ double wsum[NT / 32];
    const uint32_t full = sc_smem(bars), empty = full + 8 * NS;
    const int32_t tid = threadIdx.x, lane = tid & 31;
    const int64_t n_px = (int64_t)N * N;
    const int64_t p0 = (int64_t)blockIdx.x * PXF, left = n_px - p0;
    const uint32_t bytes = (uint32_t)(left < PXF ? left : PXF) * 4u;
    if (tid == 0) {
        for (int s = 0; s < NS; ++s) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(full + 8 * s), "r"(1));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(empty + 8 * s), "r"(NT / 32));
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int32_t total = (T + FS - 1) / FS;
    // the rows of S_t that the pixels of this block touch: [ra, ra + nr), nr * n <= SF floats (checked by the host)
    const int64_t p_last = p0 + (left < PXF ? left : PXF) - 1;
    const int32_t ra = bi0[(int32_t)(p0 / N)], rb = min(bi0[(int32_t)(p_last / N)] + 1, n - 1);
    const uint32_t sbytes = (uint32_t)(rb - ra + 1) * n * 4u;
    if (tid >= NT) {
        if (lane == 0) {
            for (int32_t g = 0; g < total; ++g) {
                const uint32_t s = (uint32_t)g % NS, bar = full + 8 * s, dst = sc_smem(ring + s * STAGE);
                if (g >= NS) sc_wait(empty + 8 * s, ((uint32_t)(g / NS) - 1u) & 1u);
                const int32_t t0 = g * FS, nf = min(FS, T - t0);
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(nf * (bytes + 32u + sbytes))
                             : "memory");
                for (int32_t f = 0; f < nf; ++f)
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
                                     "r"(dst + f * (PXF * 4)), "l"(D + (int64_t)(t0 + f) * n_px + p0), "r"(bytes), "r"(bar)
                                 : "memory");
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
                                 "r"(dst + FS * (PXF * 4)), "l"(phi + 8 * (int64_t)t0), "r"(nf * 32u), "r"(bar)
                             : "memory");
                for (int32_t f = 0; f < nf; ++f)
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
                                     "r"(dst + (FS * (PXF + 8) + f * SF) * 4), "l"(S + ((int64_t)(t0 + f) * n + ra) * n),
                                     "r"(sbytes), "r"(bar)
                                 : "memory");
            }
        }
        return;
    }
    const bool live = (int64_t)tid * PX < left;
    const int64_t p = p0 + (int64_t)tid * PX;
    const int32_t i = live ? (int32_t)(p / N) : 0, j = live ? (int32_t)(p % N) : 0;     // PX pixels of one row: N % 4 == 0
    const int32_t i0 = bi0[i], i1 = min(i0 + 1, n - 1);
    const float wy = bw[i];
    int32_t o0[PX], dj[PX];
    float wx[PX];
#pragma unroll
    for (int k = 0; k < PX; ++k) {
        const int32_t j0 = bi0[j + k];
        o0[k] = (i0 - ra) * n + j0;
        dj[k] = min(j0 + 1, n - 1) - j0;
        wx[k] = bw[j + k];
    }
    const int32_t di = (i1 - i0) * n;
    float b[6][PX], g[6][PX];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const float2 v = live ? *reinterpret_cast<const float2 *>(beta + k * n_px + p) : make_float2(0.f, 0.f);
        b[k][0] = v.x; b[k][1] = v.y;
        g[k][0] = g[k][1] = 0.f;
    }
    double loss = 0.0;
    uint32_t st = 0, par = 0;
    for (int32_t t0 = 0; t0 < T; t0 += FS) {
        sc_wait(full + 8 * st, par);
        const float *sp = ring + st * STAGE;
        float lsum = 0.f;
#pragma unroll
        for (int f = 0; f < FS; ++f) {
            if (t0 + f < T) {
                const float2 dv = reinterpret_cast<const float2 *>(sp + f * PXF)[tid];
                const float4 qa = *reinterpret_cast<const float4 *>(sp + FS * PXF + f * 8);
                const float2 qb = *reinterpret_cast<const float2 *>(sp + FS * PXF + f * 8 + 4);
                const float q[6] = {qa.x, qa.y, qa.z, qa.w, qb.x, qb.y};
                const float d4[PX] = {dv.x, dv.y};
                const float *St = sp + FS * (PXF + 8) + f * SF;
                float c4[PX];
#pragma unroll
                for (int k = 0; k < PX; ++k) {
                    const float a00 = St[o0[k]], a01 = St[o0[k] + dj[k]];
                    const float a10 = St[o0[k] + di], a11 = St[o0[k] + di + dj[k]];
                    // the same expression as k_scatter_resid: four weights times four values
                    float pred = (1.f - wy) * (1.f - wx[k]) * a00 + (1.f - wy) * wx[k] * a01 + wy * (1.f - wx[k]) * a10 +
                                 wy * wx[k] * a11;
#pragma unroll
                    for (int m = 0; m < 6; ++m) pred = fmaf(q[m], b[m][k], pred);
                    const float r = d4[k] - pred;
                    const float a = fabsf(r);
                    lsum += a <= delta ? 0.5f * r * r : delta * (a - 0.5f * delta);       // Eq. 4
                    const float c = fminf(fmaxf(r, -delta), delta);
                    c4[k] = c;
#pragma unroll
                    for (int m = 0; m < 6; ++m) g[m][k] = fmaf(q[m], c, g[m][k]);
                }
                if (live)
                    *reinterpret_cast<float2 *>(psi + (int64_t)(t0 + f) * n_px + p) = make_float2(c4[0], c4[1]);
            }
        }
        if (live) loss += (double)lsum;
        __syncwarp();
        if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(empty + 8 * st) : "memory");
        if (++st == NS) { st = 0; par ^= 1u; }
    }
    if (live) {
#pragma unroll
        for (int k = 0; k < 6; ++k)
            *reinterpret_cast<float2 *>(g_beta + k * n_px + p) = make_float2(-g[k][0], -g[k][1]);
    }
    // loss of the block in a fixed order (consumer warps only: the producer warp has left)
    for (int o = 16; o > 0; o >>= 1) loss += __shfl_down_sync(0xffffffffu, loss, o);
    if (lane == 0) wsum[tid >> 5] = loss;
    asm volatile("bar.sync 1, %0;" ::"n"(NT) : "memory");
    if (tid == 0) {
        double s = 0.0;
        for (int w = 0; w < NT / 32; ++w) s += wsum[w];
        partials[blockIdx.x] = s;
    }
}

// ---- fused evaluation (N = 2 NT: one block per image row) -----------------------------------------------------------
// k_scatter_resid_bulk, but psi never goes to global memory: dL/dS_t = -A^T psi_t A is separable, and the column
// half of it, C[i][t][b] = sum_j wx(j, b) psi[t][i][j], only needs the row i the block owns.  The consumers put the
// clipped residuals of a stage (FS frames x N pixels) into a padded shared buffer, then thread (f, b) sums the <= max_sup
// columns under input column b -- pitch N + 1 makes the 8 frames x 4 columns of a warp hit 32 distinct banks -- and
// the block writes FS x n partial sums, coalesced, to cpart[i][t][b].  k_scatter_gs_rows finishes the row half.  One
// evaluation then reads the data once (T N^2 floats) and moves 2 T N n floats of partial sums: 1.3 GB instead of 3 GB at
// the paper's size.  Every sum has a fixed order: the gradient is reproducible bit for bit.
template <int NT, int NS, int FS, int SF>
__global__ void __launch_bounds__(NT + 32, 3)
k_scatter_fused(const float *__restrict__ D, int32_t T, int32_t N, int32_t n, const float *__restrict__ phi,
                const int32_t *__restrict__ bi0, const float *__restrict__ bw, const int32_t *__restrict__ blo,
                const int32_t *__restrict__ bhi, int32_t max_sup, float delta,
                const float *__restrict__ beta, const float *__restrict__ S, float *__restrict__ cpart,
                float *__restrict__ g_beta, double *__restrict__ partials, int32_t t_chunk) {
    // blockIdx.y: the chunk of frames [ta, tb) of this block; g_beta is then the block's partial sum, written to
    // g_beta + blockIdx.y * 6 N^2 (k_scatter_gbeta_sum adds the chunks in order).  Chunks exist to balance the blocks
    // over the SMs: N rows alone leave a second, nearly empty wave.
    constexpr int PX = 2;
    constexpr int PXF = NT * PX, STAGE = FS * (PXF + 8 + SF), PP = PXF + 1;
    const int32_t ta = blockIdx.y * t_chunk, tb = min(T, ta + t_chunk);
    extern __shared__ __align__(128) float ring[];               // [NS][STAGE], then psi rows [FS][PP], then weights
    __shared__ __align__(8) uint64_t bars[2 * NS];
    __shared__ double wsum[NT / 32];
    float *prow = ring + NS * STAGE;                             // clipped residuals of the current stage
    float *Wt = prow + FS * PP;                                  // [n][max_sup] column weights wx(blo[b] + c, b)
    const uint32_t full = sc_smem(bars), empty = full + 8 * NS;
    const int32_t tid = threadIdx.x, lane = tid & 31;
    const int64_t n_px = (int64_t)N * N;
    const int32_t i = blockIdx.x;                                // the image row of this block (N == PXF)
    const int64_t p0 = (int64_t)i * PXF;
    const uint32_t bytes = PXF * 4u;
    if (tid == 0) {
        for (int s = 0; s < NS; ++s) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(full + 8 * s), "r"(1));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(empty + 8 * s), "r"(NT / 32));
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int32_t total = (tb - ta + FS - 1) / FS;
    const int32_t ra = bi0[i], rb = min(ra + 1, n - 1);          // the rows of S_t under this image row
    const uint32_t sbytes = (uint32_t)(rb - ra + 1) * n * 4u;
    if (tid >= NT) {
        if (lane == 0) {
            for (int32_t g = 0; g < total; ++g) {
                const uint32_t s = (uint32_t)g % NS, bar = full + 8 * s, dst = sc_smem(ring + s * STAGE);
                if (g >= NS) sc_wait(empty + 8 * s, ((uint32_t)(g / NS) - 1u) & 1u);
                const int32_t t0 = ta + g * FS, nf = min(FS, tb - t0);
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(nf * (bytes + 32u + sbytes))
                             : "memory");
                for (int32_t f = 0; f < nf; ++f)
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
                                     "r"(dst + f * (PXF * 4)), "l"(D + (int64_t)(t0 + f) * n_px + p0), "r"(bytes), "r"(bar)
                                 : "memory");
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
                                 "r"(dst + FS * (PXF * 4)), "l"(phi + 8 * (int64_t)t0), "r"(nf * 32u), "r"(bar)
                             : "memory");
                for (int32_t f = 0; f < nf; ++f)
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
                                     "r"(dst + (FS * (PXF + 8) + f * SF) * 4), "l"(S + ((int64_t)(t0 + f) * n + ra) * n),
                                     "r"(sbytes), "r"(bar)
                                 : "memory");
            }
        }
        return;
    }
    // the weights of every input column over its support (at most max_sup image columns), once per block
    for (int32_t e = tid; e < n * max_sup; e += NT) {
        const int32_t b = e / max_sup, c = blo[b] + e % max_sup;
        float w = 0.f;
        if (c <= bhi[b]) {
            const int32_t c0 = bi0[c], c1 = min(c0 + 1, n - 1);
            const float v = bw[c];
            w = (c0 == b ? 1.f - v : 0.f) + (c1 == b ? v : 0.f);
        }
        Wt[e] = w;
    }
    const int64_t p = p0 + (int64_t)tid * PX;
    const int32_t j = tid * PX;
    const int32_t i1 = rb;
    const float wy = bw[i];
    // per pixel: the four bilinear weights (the products of k_scatter_resid, formed once) and the places of the four
    // values of S_t in the staged rows of stage 0, frame 0 (row ra of S_t is row 0 of the staged rows)
    float w00[PX], w01[PX], w10[PX], w11[PX];
    const float *s00[PX], *s01[PX], *s10[PX], *s11[PX];
    const int32_t di = (i1 - ra) * n;
#pragma unroll
    for (int k = 0; k < PX; ++k) {
        const int32_t j0 = bi0[j + k], dj = min(j0 + 1, n - 1) - j0;
        const float wx = bw[j + k];
        w00[k] = (1.f - wy) * (1.f - wx); w01[k] = (1.f - wy) * wx; w10[k] = wy * (1.f - wx); w11[k] = wy * wx;
        s00[k] = ring + FS * (PXF + 8) + j0;
        s01[k] = s00[k] + dj;
        s10[k] = s00[k] + di;
        s11[k] = s10[k] + dj;
    }
    float b[6][PX], g[6][PX];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const float2 v = *reinterpret_cast<const float2 *>(beta + k * n_px + p);
        b[k][0] = v.x; b[k][1] = v.y;
        g[k][0] = g[k][1] = 0.f;
    }
    double loss = 0.0;
    uint32_t st = 0, par = 0;
    // one frame of the stage at offset so (floats) for this thread's two pixels; returns the clipped residuals
    auto frame = [&](const float *sp, int32_t so, int f, float &lsum, float (&c4)[PX]) {
        const float2 dv = reinterpret_cast<const float2 *>(sp + f * PXF)[tid];
        const float4 qa = *reinterpret_cast<const float4 *>(sp + FS * PXF + f * 8);
        const float2 qb = *reinterpret_cast<const float2 *>(sp + FS * PXF + f * 8 + 4);
        const float q[6] = {qa.x, qa.y, qa.z, qa.w, qb.x, qb.y};
        const float d4[PX] = {dv.x, dv.y};
#pragma unroll
        for (int k = 0; k < PX; ++k) {
            const int32_t o = so + f * SF;
            // the same expression as k_scatter_resid: four weights times four values
            float pred = w00[k] * s00[k][o] + w01[k] * s01[k][o] + w10[k] * s10[k][o] + w11[k] * s11[k][o];
#pragma unroll
            for (int m = 0; m < 6; ++m) pred = fmaf(q[m], b[m][k], pred);
            const float r = d4[k] - pred;
            const float c = fminf(fmaxf(r, -delta), delta);
            lsum = fmaf(c, r - 0.5f * c, lsum);        // Eq. 4: c (r - c/2) = r^2/2 inside, delta (|r| - delta/2) outside
            c4[k] = c;
#pragma unroll
            for (int m = 0; m < 6; ++m) g[m][k] = fmaf(q[m], c, g[m][k]);
        }
    };
    for (int32_t t0 = ta; t0 < tb; t0 += FS) {
        sc_wait(full + 8 * st, par);
        const float *sp = ring + st * STAGE;
        const int32_t so = (int32_t)st * STAGE;
        float lsum = 0.f;
        if (t0 + FS <= tb) {                      // a full stage: no per-frame test
#pragma unroll
            for (int f = 0; f < FS; ++f) {
                float c4[PX];
                frame(sp, so, f, lsum, c4);
                prow[f * PP + j] = c4[0];
                prow[f * PP + j + 1] = c4[1];
            }
        } else {
#pragma unroll
            for (int f = 0; f < FS; ++f) {
                float c4[PX] = {0.f, 0.f};
                if (t0 + f < tb) frame(sp, so, f, lsum, c4);
                prow[f * PP + j] = c4[0];
                prow[f * PP + j + 1] = c4[1];
            }
        }
        loss += (double)lsum;
        // the stage's data is consumed: hand it back, then reduce the psi rows along the columns
        __syncwarp();
        if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(empty + 8 * st) : "memory");
        asm volatile("bar.sync 1, %0;" ::"n"(NT) : "memory");
        // thread -> (frame f = e % FS, input column b = e / FS): a warp covers FS frames x 32 / FS columns
        for (int32_t e = tid; e < FS * n; e += NT) {
            const int32_t f = e % FS, bb = e / FS;
            if (t0 + f < tb) {
                const int32_t lo = blo[bb];
                const float *pr = prow + f * PP + lo, *w = Wt + bb * max_sup;
                // only the support [blo, bhi] of the column: past it the weights are zero, but the row is not -- its
                // pad element is never written, and 0 x (whatever an earlier kernel left there, possibly NaN) is not 0
                const int32_t ns = min(max_sup, bhi[bb] - lo + 1);
                float sum = 0.f;
                for (int32_t c = 0; c < ns; ++c) sum = fmaf(w[c], pr[c], sum);
                cpart[((int64_t)i * T + (t0 + f)) * n + bb] = sum;
            }
        }
        asm volatile("bar.sync 1, %0;" ::"n"(NT) : "memory");      // prow is rewritten by the next stage
        if (++st == NS) { st = 0; par ^= 1u; }
    }
#pragma unroll
    for (int k = 0; k < 6; ++k)
        *reinterpret_cast<float2 *>(g_beta + (int64_t)blockIdx.y * 6 * n_px + k * n_px + p) = make_float2(-g[k][0], -g[k][1]);
    for (int o = 16; o > 0; o >>= 1) loss += __shfl_down_sync(0xffffffffu, loss, o);
    if (lane == 0) wsum[tid >> 5] = loss;
    asm volatile("bar.sync 1, %0;" ::"n"(NT) : "memory");
    if (tid == 0) {
        double s = 0.0;
        for (int w = 0; w < NT / 32; ++w) s += wsum[w];
        partials[blockIdx.y * gridDim.x + blockIdx.x] = s;
    }
}

// g_beta = sum over the chunks of the partial sums, in order
__global__ void __launch_bounds__(256)
k_scatter_gbeta_sum(const float *__restrict__ part, int32_t n_chunk, int64_t n, float *__restrict__ g_beta) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float s = part[i];
    for (int32_t c = 1; c < n_chunk; ++c) s += part[c * n + i];
    g_beta[i] = s;
}

// g_S[t][a][b] = - sum_i wy(i, a) cpart[i][t][b] over the image rows i under input row a (rlo[a] .. rhi[a]), in order
__global__ void __launch_bounds__(256)
k_scatter_gs_rows(const float *__restrict__ cpart, int32_t T, int32_t N, int32_t n, const int32_t *__restrict__ bi0,
                  const float *__restrict__ bw, const int32_t *__restrict__ blo, const int32_t *__restrict__ bhi,
                  float *__restrict__ g_S) {
    const int64_t id = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= (int64_t)T * n * n) return;
    const int32_t b = (int32_t)(id % n), a = (int32_t)((id / n) % n), t = (int32_t)(id / ((int64_t)n * n));
    float acc = 0.f;
    for (int32_t i = blo[a]; i <= bhi[a]; ++i) {
        const int32_t i0 = __ldg(bi0 + i), i1 = min(i0 + 1, n - 1);
        const float w = __ldg(bw + i);
        const float wy = (i0 == a ? 1.f - w : 0.f) + (i1 == a ? w : 0.f);
        acc = fmaf(wy, __ldg(cpart + ((int64_t)i * T + t) * n + b), acc);
    }
    g_S[id] = -acc;
}

// dL/dS[t][a][b] = - sum_{i,j} wy(i, a) wx(j, b) psi[t][i][j]: only pixels within one input pixel of (a, b) count
__global__ void __launch_bounds__(256)
k_scatter_gs(const float *__restrict__ psi, int32_t T, int32_t N, int32_t n, const int32_t *__restrict__ bi0,
             const float *__restrict__ bw, float *__restrict__ g_S) {
    const int64_t id = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= (int64_t)T * n * n) return;
    const int32_t b = (int32_t)(id % n), a = (int32_t)((id / n) % n), t = (int32_t)(id / ((int64_t)n * n));
    const int32_t f = (N + n - 1) / n;
    const int32_t ilo = max(0, (a - 1) * f - 1), ihi = min(N - 1, (a + 2) * f), jlo = max(0, (b - 1) * f - 1),
                  jhi = min(N - 1, (b + 2) * f);
    const float *P = psi + (int64_t)t * N * N;
    float acc = 0.f;
    for (int32_t i = ilo; i <= ihi; ++i) {
        const int32_t i0 = __ldg(bi0 + i), i1 = min(i0 + 1, n - 1);
        const float w = __ldg(bw + i);
        const float wy = (i0 == a ? 1.f - w : 0.f) + (i1 == a ? w : 0.f);
        if (wy == 0.f) continue;
        float row = 0.f;
        for (int32_t j = jlo; j <= jhi; ++j) {
            const int32_t j0 = __ldg(bi0 + j), j1 = min(j0 + 1, n - 1);
            const float v = __ldg(bw + j);
            const float wx = (j0 == b ? 1.f - v : 0.f) + (j1 == b ? v : 0.f);
            if (wx != 0.f) row = fmaf(wx, __ldg(P + (int64_t)i * N + j), row);
        }
        acc = fmaf(wy, row, acc);
    }
    g_S[id] = -acc;
}

// The same sum, separably and with every psi read exactly once, coalesced: one block per frame, one thread per
// column j walks down the rows; row i feeds the two input rows a = bi0[i] (weight 1 - w) and a + 1 (weight w), which
// are the same for the whole block, so two running sums per thread suffice; when a advances, the finished column
// sums C_a[j] go through shared memory and threads b < n reduce them along j over their support [blo[b], bhi[b]].
__global__ void __launch_bounds__(1024)
k_scatter_gs_cols(const float *__restrict__ psi, int32_t N, int32_t n, const int32_t *__restrict__ bi0,
                  const float *__restrict__ bw, const int32_t *__restrict__ blo, const int32_t *__restrict__ bhi,
                  int32_t strip_b, int32_t max_sup, float *__restrict__ g_S) {
    // blockIdx.y: a strip of strip_b input columns b and the image columns under them (strips overlap by the width of
    // a stencil; more, smaller blocks keep more loads in flight than one block per frame)
    extern __shared__ float C[];                 // [blockDim.x] column sums, then [strip_b][max_sup] weights
    float *Wt = C + blockDim.x;
    const int32_t t = blockIdx.x, tid = threadIdx.x;
    const int32_t b0 = blockIdx.y * strip_b, b1 = min(n, b0 + strip_b);
    const int32_t c_lo = blo[b0], c_hi = bhi[b1 - 1];
    const int32_t j = c_lo + tid;
    const bool active = j <= c_hi;
    const float *P = psi + (int64_t)t * N * N;
    float *out = g_S + (int64_t)t * n * n;
    const int32_t b = b0 + tid;
    const int32_t my_lo = b < b1 ? blo[b] : 0, my_hi = b < b1 ? min(bhi[b], blo[b] + max_sup - 1) : -1;
    // the weights of input column b over its support, once (the support is at most max_sup image columns wide)
    if (b < b1)
        for (int32_t c = my_lo; c <= my_hi; ++c) {
            const int32_t c0 = __ldg(bi0 + c), c1 = min(c0 + 1, n - 1);
            const float v = __ldg(bw + c);
            Wt[tid * max_sup + (c - my_lo)] = (c0 == b ? 1.f - v : 0.f) + (c1 == b ? v : 0.f);
        }
    const float *myW = Wt + tid * max_sup, *myC = C + (my_lo - c_lo);
    const int32_t my_n = my_hi - my_lo + 1;
    auto flush = [&](int32_t a, float acc) {
        if (active) C[tid] = acc;
        __syncthreads();
        if (b < b1) {
            float sum = 0.f;
            for (int32_t c = 0; c < my_n; ++c) sum = fmaf(myW[c], myC[c], sum);
            out[a * n + b] = -sum;
        }
        __syncthreads();
    };
    float acc0 = 0.f, acc1 = 0.f;
    int32_t cur = __ldg(bi0);
    constexpr int kAhead = 16;                    // rows loaded before they are used: 8 loads in flight per thread
    for (int32_t ib = 0; ib < N; ib += kAhead) {
        float vv[kAhead];
#pragma unroll
        for (int k = 0; k < kAhead; ++k)
            vv[k] = (active && ib + k < N) ? __ldcs(P + (int64_t)(ib + k) * N + j) : 0.f;
#pragma unroll
        for (int k = 0; k < kAhead; ++k) {
            const int32_t i = ib + k;
            if (i < N) {
                const int32_t a0 = __ldg(bi0 + i);
                const float w = __ldg(bw + i);
                if (a0 != cur) {                 // uniform over the block: the input row advances by one
                    flush(cur, acc0);
                    acc0 = acc1;
                    acc1 = 0.f;
                    cur = a0;
                }
                if (a0 + 1 <= n - 1) {
                    acc0 = fmaf(1.f - w, vv[k], acc0);
                    acc1 = fmaf(w, vv[k], acc1);
                } else {
                    acc0 += vv[k];               // clamped: both stencil points are the last input row
                }
            }
        }
    }
    flush(cur, acc0);
    for (int32_t a = cur + 1; a < n; ++a) {      // input rows below the last stencil (only if N < n, never here)
        flush(a, a == cur + 1 ? acc1 : 0.f);
    }
}

// ---- vector algebra of L-BFGS (float32 vectors, float64 reductions in a fixed order) -----------------------------
__global__ void __launch_bounds__(256)
k_dot(const float *__restrict__ x, const float *__restrict__ y, int64_t n, double *__restrict__ partials) {
    double s = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        s += (double)x[i] * (double)y[i];
    block_sum_to(s, partials);
}
__global__ void __launch_bounds__(256)
k_absmax(const float *__restrict__ x, int64_t n, double *__restrict__ partials) {
    __shared__ double sh[8];
    double m = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        m = fmax(m, fabs((double)x[i]));
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_down_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) m = fmax(m, sh[w]);
        partials[blockIdx.x] = fmax(m, sh[0]);
    }
}
// out[0] = sum (or max) of the n partials, one block, fixed tree
__global__ void __launch_bounds__(256)
k_sum_partials(const double *__restrict__ partials, int32_t n, int32_t take_max, double *__restrict__ out) {
    __shared__ double sh[256];
    double s = 0.0;
    for (int32_t i = threadIdx.x; i < n; i += 256) s = take_max ? fmax(s, partials[i]) : s + partials[i];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o)
            sh[threadIdx.x] = take_max ? fmax(sh[threadIdx.x], sh[threadIdx.x + o]) : sh[threadIdx.x] + sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = sh[0];
}
// The scalars of the two-loop recursion stay on the device (sc[]): the final stage of a reduction applies the
// recursion's formula and leaves the coefficient of the next vector update in sc[2], so the host enqueues the whole
// recursion without reading anything back.  sc[0], sc[1]: results for the host; sc[3]: |g|_inf;
// sc[8 + i]: rho_i; sc[8 + kScatterHistory + i]: alpha_i.
enum ScalarOp { kStore0 = 0, kAlpha = 1, kBeta = 3, kStore1 = 4 };
__global__ void __launch_bounds__(256)
k_reduce_op(const double *__restrict__ partials, int32_t n, int32_t op, int32_t i, double *__restrict__ sc) {
    __shared__ double sh[256];
    double s = 0.0;
    for (int32_t k = threadIdx.x; k < n; k += 256) s += partials[k];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        s = sh[0];
        double *rho = sc + 8, *alpha = sc + 8 + kScatterHistory;
        if (op == kStore0) sc[0] = s;
        else if (op == kStore1) sc[1] = s;
        else if (op == kAlpha) { alpha[i] = rho[i] * s; sc[2] = -alpha[i]; }          // q -= alpha_i y_i
        else if (op == kBeta) sc[2] = alpha[i] - rho[i] * s;                           // r += (alpha_i - beta) s_i
    }
}
// z = a x + b y   (z may alias x or y)
__global__ void __launch_bounds__(256)
k_axpby(float a, const float *x, float b, const float *y, int64_t n, int64_t n4, float *z) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n4 > 0) {
        if (i < n4) {
            const float4 u = reinterpret_cast<const float4 *>(x)[i];
            float4 v = make_float4(a * u.x, a * u.y, a * u.z, a * u.w);
            if (b != 0.f) {
                const float4 w = reinterpret_cast<const float4 *>(y)[i];
                v = make_float4(a * u.x + b * w.x, a * u.y + b * w.y, a * u.z + b * w.z, a * u.w + b * w.w);
            }
            reinterpret_cast<float4 *>(z)[i] = v;
        }
    } else if (i < n) {
        z[i] = a * x[i] + (b != 0.f ? b * y[i] : 0.f);
    }
}

// Reduction tail shared by the fused kernels below: every block leaves its partial sum(s) in partials[block] (and
// partials[grid + block]), the block that arrives last (a ticket counter, reset for the next launch) adds them up in
// index order -- the same tree whatever the arrival order, so the result is reproducible -- and applies the recursion's
// formula like k_reduce_op.
__device__ __forceinline__ void last_block_reduce(double v0, double v1, int32_t two, double *partials,
                                                  unsigned int *ticket, int32_t op, int32_t i, double *sc) {
    __shared__ double sh0[8], sh1[8];
    __shared__ double tr0[256], tr1[256];
    __shared__ bool last;
    for (int o = 16; o > 0; o >>= 1) {
        v0 += __shfl_down_sync(0xffffffffu, v0, o);
        v1 += __shfl_down_sync(0xffffffffu, v1, o);
    }
    if ((threadIdx.x & 31) == 0) { sh0[threadIdx.x >> 5] = v0; sh1[threadIdx.x >> 5] = v1; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { a += sh0[w]; b += sh1[w]; }
        partials[blockIdx.x] = a;
        if (two) partials[gridDim.x + blockIdx.x] = b;
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    double a = 0.0, b = 0.0;
    for (int32_t k = threadIdx.x; k < (int32_t)gridDim.x; k += 256) {
        a += __ldcg(partials + k);
        if (two) b += __ldcg(partials + gridDim.x + k);
    }
    tr0[threadIdx.x] = a; tr1[threadIdx.x] = b;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) { tr0[threadIdx.x] += tr0[threadIdx.x + o]; tr1[threadIdx.x] += tr1[threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        *ticket = 0;
        const double s = tr0[0];
        double *rho = sc + 8, *alpha = sc + 8 + kScatterHistory;
        if (op == kStore0) { sc[0] = s; if (two) sc[1] = tr1[0]; }
        else if (op == kAlpha) { alpha[i] = rho[i] * s; sc[2] = -alpha[i]; }          // q -= alpha_i y_i
        else if (op == kBeta) sc[2] = alpha[i] - rho[i] * s;                           // r += (alpha_i - beta) s_i
    }
}
// One step of the two-loop recursion in one pass: out = scale * (in + (float)sc[2] * v)  (v == NULL: out = scale * in),
// then the dot product of out with w, reduced and turned into the next coefficient by the last block.
__global__ void __launch_bounds__(256)
k_update_dot(const float *in, const float *v, float scale, const float *__restrict__ w, int64_t n, int64_t n4,
             float *out, double *partials, unsigned int *ticket, int32_t op, int32_t i, double *sc) {
    const float c = v ? (float)sc[2] : 0.f;
    double acc = 0.0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x, id = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (n4 > 0) {
        for (int64_t k = id; k < n4; k += stride) {
            float4 a = reinterpret_cast<const float4 *>(in)[k];
            if (v) {
                const float4 b = reinterpret_cast<const float4 *>(v)[k];
                a = make_float4(a.x + c * b.x, a.y + c * b.y, a.z + c * b.z, a.w + c * b.w);
            }
            a = make_float4(scale * a.x, scale * a.y, scale * a.z, scale * a.w);
            reinterpret_cast<float4 *>(out)[k] = a;
            const float4 q = reinterpret_cast<const float4 *>(w)[k];
            acc += (double)a.x * q.x + (double)a.y * q.y + (double)a.z * q.z + (double)a.w * q.w;
        }
    } else {
        for (int64_t k = id; k < n; k += stride) {
            float a = in[k];
            if (v) a = a + c * v[k];
            a = scale * a;
            out[k] = a;
            acc += (double)a * (double)w[k];
        }
    }
    last_block_reduce(acc, 0.0, 0, partials, ticket, op, i, sc);
}
// The new pair in one pass: s = xn - x, y = gn - g, and both s.y -> sc[0] and y.y -> sc[1]
__global__ void __launch_bounds__(256)
k_pair(const float *__restrict__ xn, const float *__restrict__ x, const float *__restrict__ gn, const float *__restrict__ g,
       int64_t n, float *__restrict__ s_out, float *__restrict__ y_out, double *partials, unsigned int *ticket,
       double *sc) {
    double sy = 0.0, yy = 0.0;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
        const float sv = xn[k] - x[k], yv = gn[k] - g[k];
        s_out[k] = sv;
        y_out[k] = yv;
        sy += (double)sv * (double)yv;
        yy += (double)yv * (double)yv;
    }
    last_block_reduce(sy, yy, 1, partials, ticket, kStore0, 0, sc);
}

// VEC: four neighbouring pixels of four rows (y, y + 4, y + 8, y + 12) per thread (W % 4 == 0, 16-byte aligned frames):
// the four 16-byte loads of the frame are requested before the stencil arithmetic, which keeps enough bytes in flight
// per SM for an in-place stream; the column stencil is looked up once for the four rows
template <bool VEC>
__global__ void __launch_bounds__(256, 4)
k_scatter_subtract(float *__restrict__ frames, int32_t H, int32_t W, const float *__restrict__ S, int32_t n,
                   const int32_t *__restrict__ yi0, const float *__restrict__ yw, const int32_t *__restrict__ xi0,
                   const float *__restrict__ xw) {
    constexpr int PX = VEC ? 4 : 1, RW = VEC ? 4 : 1;
    const int32_t x = (blockIdx.x * 64 + (threadIdx.x & 63)) * PX, y = blockIdx.y * (4 * RW) + (threadIdx.x >> 6),
                  t = blockIdx.z;
    if (x >= W || y >= H) return;
    float *p = frames + ((int64_t)t * H + y) * W + x;
    float4 v[RW];
    if (VEC) {
#pragma unroll
        for (int r = 0; r < RW; ++r)
            if (y + 4 * r < H) v[r] = __ldcs(reinterpret_cast<const float4 *>(p + (int64_t)4 * r * W));
    }
    int32_t j0[PX], j1[PX];
    float wx[PX];
#pragma unroll
    for (int k = 0; k < PX; ++k) {
        j0[k] = xi0[x + k];
        j1[k] = min(j0[k] + 1, n - 1);
        wx[k] = xw[x + k];
    }
#pragma unroll
    for (int r = 0; r < RW; ++r) {
        const int32_t yr = y + 4 * r;
        if (yr >= H) break;
        const int32_t i0 = yi0[yr], i1 = min(i0 + 1, n - 1);
        const float wy = yw[yr];
        const float *r0 = S + (int64_t)t * n * n + i0 * n, *r1 = S + (int64_t)t * n * n + i1 * n;
        float u[PX];
#pragma unroll
        for (int k = 0; k < PX; ++k)
            u[k] = (1.f - wy) * ((1.f - wx[k]) * __ldg(r0 + j0[k]) + wx[k] * __ldg(r0 + j1[k])) +
                   wy * ((1.f - wx[k]) * __ldg(r1 + j0[k]) + wx[k] * __ldg(r1 + j1[k]));
        if (VEC) {
            float4 w = v[r];
            w.x -= u[0]; w.y -= u[PX > 1 ? 1 : 0]; w.z -= u[PX > 2 ? 2 : 0]; w.w -= u[PX > 3 ? 3 : 0];
            __stcs(reinterpret_cast<float4 *>(p + (int64_t)4 * r * W), w);
        } else {
            p[0] -= u[0];
        }
    }
}

void launch_downsample(cudaStream_t st, const float *frames, int32_t T, int32_t H, int32_t W, int32_t f, float *out) {
    dim3 grid((unsigned)((W / f + 63) / 64), (unsigned)((H / f + 3) / 4), (unsigned)T);
    k_downsample<<<grid, 256, 0, st>>>(frames, H, W, f, out);
}

void launch_scatter_subtract(cudaStream_t st, float *frames, int32_t T, int32_t H, int32_t W, const float *S, int32_t n,
                             const int32_t *yi0, const float *yw, const int32_t *xi0, const float *xw) {
    if (W % 4 == 0 && (reinterpret_cast<uintptr_t>(frames) & 15u) == 0) {
        dim3 grid((unsigned)((W / 4 + 63) / 64), (unsigned)((H + 15) / 16), (unsigned)T);
        k_scatter_subtract<true><<<grid, 256, 0, st>>>(frames, H, W, S, n, yi0, yw, xi0, xw);
    } else {
        dim3 grid((unsigned)((W + 63) / 64), (unsigned)((H + 3) / 4), (unsigned)T);
        k_scatter_subtract<false><<<grid, 256, 0, st>>>(frames, H, W, S, n, yi0, yw, xi0, xw);
    }
}

// loss -> loss_dev[0] (DEVICE double), gradient -> g_beta, g_S.  psi: [T][N][N] scratch, partials: [>= blocks] doubles
int32_t scatter_lossgrad(cudaStream_t st, const ScatterProblem &pb, const float *beta, const float *S, float *psi,
                         double *partials, float *g_beta, float *g_S, double *loss_dev) {
    const int64_t n_px = (int64_t)pb.N * pb.N;
    int32_t blocks;
    const bool aligned = ((reinterpret_cast<uintptr_t>(pb.D) | reinterpret_cast<uintptr_t>(beta) |
                           reinterpret_cast<uintptr_t>(psi) | reinterpret_cast<uintptr_t>(g_beta)) & 15u) == 0;
    constexpr int NT = 256, NS = 2, FS = 8, SF = 192;     // 45.6 KB per CTA: four CTAs per SM, all 512 blocks of N = 512 resident
    // fused evaluation (one block per image row, psi stays on chip): N = 2 NT, two rows of S_t fit the staging area
    // image columns under one input column: two stencil widths, plus the half width of clamped columns at the edge
    // (input column 1 also "sees", with weight 0, the columns clamped to input column 0)
    const int32_t max_sup_f = 5 * ((pb.N + pb.n - 1) / pb.n) / 2 + 4;
    if (pb.N == 2 * NT && pb.n % 4 == 0 && 2 * pb.n <= SF && aligned && (reinterpret_cast<uintptr_t>(S) & 15u) == 0 &&
        (size_t)pb.n * max_sup_f * 4 <= 32 * 1024) {
        const size_t smem = ((size_t)NS * FS * (NT * 2 + 8 + SF) + (size_t)FS * (NT * 2 + 1) + (size_t)pb.n * max_sup_f) * 4;
        cudaFuncSetAttribute(k_scatter_fused<NT, NS, FS, SF>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        // chunks of frames: the number (<= 16, chunks of at least two stages, partial sums inside the scratch stack)
        // that wastes the least of the last wave of blocks, three blocks per SM
        int dev = 0, n_sm = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        const double slots = 3.0 * n_sm;
        int32_t n_chunk = 1;
        double best = std::ceil(pb.N / slots);
        for (int32_t c = 2; c <= 16; ++c) {
            const int32_t tc = ((pb.T + c - 1) / c + FS - 1) / FS * FS;
            if (tc < 2 * FS || (int64_t)(c - 1) * tc >= pb.T) continue;
            if ((int64_t)pb.N * pb.T * pb.n + (int64_t)c * 6 * n_px > (int64_t)pb.T * n_px || (int64_t)c * pb.N > kLossPartials)
                continue;
            const double cost = std::ceil(c * pb.N / slots) / c;
            if (cost < best - 1e-9) { best = cost; n_chunk = c; }
        }
        const int32_t t_chunk = n_chunk == 1 ? pb.T : ((pb.T + n_chunk - 1) / n_chunk + FS - 1) / FS * FS;
        float *gb_part = n_chunk == 1 ? g_beta : psi + (int64_t)pb.N * pb.T * pb.n;
        dim3 grid((unsigned)pb.N, (unsigned)n_chunk);
        k_scatter_fused<NT, NS, FS, SF><<<grid, NT + 32, smem, st>>>(
            pb.D, pb.T, pb.N, pb.n, pb.phi, pb.bi0, pb.bw, pb.blo, pb.bhi, max_sup_f, pb.delta, beta, S, psi, gb_part,
            partials, t_chunk);
        int32_t launched = 3;
        if (n_chunk > 1) {
            k_scatter_gbeta_sum<<<(unsigned)((6 * n_px + 255) / 256), 256, 0, st>>>(gb_part, n_chunk, 6 * n_px, g_beta);
            ++launched;
        }
        k_sum_partials<<<1, 256, 0, st>>>(partials, pb.N * n_chunk, 0, loss_dev);
        const int64_t ns = (int64_t)pb.T * pb.n * pb.n;
        k_scatter_gs_rows<<<(unsigned)((ns + 255) / 256), 256, 0, st>>>(psi, pb.T, pb.N, pb.n, pb.bi0, pb.bw, pb.blo, pb.bhi, g_S);
        return launched;
    }
    // rows of S a block of NT * 2 pixels can touch: those under its first and last image row, plus one
    const int64_t img_rows = std::min<int64_t>(pb.N, (NT * 2 + pb.N - 2) / pb.N + 1);
    const int64_t s_rows = std::min<int64_t>(pb.n, (img_rows * pb.n + pb.N - 1) / pb.N + 2);
    if (pb.N % 4 == 0 && pb.n % 4 == 0 && s_rows * pb.n <= SF && aligned &&
        (reinterpret_cast<uintptr_t>(S) & 15u) == 0) {
        constexpr int smem = NS * FS * (NT * 2 + 8 + SF) * 4;
        blocks = (int32_t)((n_px + NT * 2 - 1) / (NT * 2));
        cudaFuncSetAttribute(k_scatter_resid_bulk<NT, NS, FS, SF>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        k_scatter_resid_bulk<NT, NS, FS, SF><<<(unsigned)blocks, NT + 32, smem, st>>>(pb.D, pb.T, pb.N, pb.n, pb.phi, pb.bi0, pb.bw,
                                                                                pb.delta, beta, S, psi, g_beta, partials);
    } else {
        blocks = (int32_t)((n_px + 255) / 256);
        k_scatter_resid<<<(unsigned)blocks, 256, 0, st>>>(pb.D, pb.T, pb.N, pb.n, pb.phi, pb.bi0, pb.bw, pb.delta, beta, S,
                                                         psi, g_beta, partials);
    }
    k_sum_partials<<<1, 256, 0, st>>>(partials, blocks, 0, loss_dev);
    if (pb.N <= 1024) {
        // strips of input columns: 4 for the paper's n = 64; image columns of a strip <= N / strips + two stencils
        const int32_t n_strip = pb.n >= 16 ? 4 : 1, strip_b = (pb.n + n_strip - 1) / n_strip;
        const int32_t cols = std::min(pb.N, (pb.N + n_strip - 1) / n_strip + max_sup_f);
        const int32_t threads = ((std::max(cols, strip_b) + 31) / 32) * 32;
        const int32_t max_sup = max_sup_f;                                   // image columns under one input column
        dim3 grid((unsigned)pb.T, (unsigned)((pb.n + strip_b - 1) / strip_b));
        k_scatter_gs_cols<<<grid, threads, ((size_t)threads + (size_t)strip_b * max_sup) * 4, st>>>(
            psi, pb.N, pb.n, pb.bi0, pb.bw, pb.blo, pb.bhi, strip_b, max_sup, g_S);
    } else {
        const int64_t ns = (int64_t)pb.T * pb.n * pb.n;
        k_scatter_gs<<<(unsigned)((ns + 255) / 256), 256, 0, st>>>(psi, pb.T, pb.N, pb.n, pb.bi0, pb.bw, g_S);
    }
    return 3;
}

// ---- L-BFGS --------------------------------------------------------------------------------------
// x = [beta (6 N^2) | S (T n^2)].  Two-loop recursion over the last kScatterHistory (s, y) pairs, initial scaling
// s.y / y.y, Armijo backtracking from step 1 (first iteration: 1 / |g|); a pair enters the history only if
// s.y > 1e-10 |y|^2; a non-descent direction resets the history.  Stops at |g|_inf <= gtol, after max_iter
// iterations, when two consecutive iterations each decrease the loss by less than 1e-9 of its value, or when the
// line search cannot decrease it at all (float32 resolution reached).
size_t scatter_ws_bytes(int32_t T, int32_t N, int32_t n) {
    const size_t P = (size_t)6 * N * N + (size_t)T * n * n;
    const size_t blocks = std::max<size_t>(kLossPartials, ((size_t)N * N + 255) / 256);
    return (5 + 2 * (size_t)kScatterHistory) * P * 4 + (size_t)T * N * N * 4 + (blocks + 8 + 2 * kScatterHistory) * 8 + 256;
}

int32_t scatter_fit(cudaStream_t st, const ScatterProblem &pb, float *beta, float *S, void *ws, int32_t max_iter,
                    float gtol, double *out_loss, int32_t *out_iters, int32_t *out_evals, int32_t *out_launches) {
    const int64_t nb = (int64_t)6 * pb.N * pb.N, ns = (int64_t)pb.T * pb.n * pb.n, P = nb + ns;
    const size_t blocks = std::max<size_t>(kLossPartials, ((size_t)pb.N * pb.N + 255) / 256);
    float *x = static_cast<float *>(ws), *g = x + P, *xn = g + P, *gn = xn + P, *d = gn + P;
    float *hs = d + P, *hy = hs + (size_t)kScatterHistory * P, *psi = hy + (size_t)kScatterHistory * P;
    double *partials = reinterpret_cast<double *>((reinterpret_cast<uintptr_t>(psi + (size_t)pb.T * pb.N * pb.N) + 15) &
                                                  ~(uintptr_t)15);
    double *scal = partials + blocks;            // 8 + 2 * kScatterHistory doubles (k_reduce_op)
    unsigned int *ticket = reinterpret_cast<unsigned int *>(scal + 6);       // scal[6] is not used as a scalar
    cudaMemsetAsync(ticket, 0, 8, st);
    int32_t launches = 0, evals = 0;
    cudaError_t err = cudaSuccess;
    auto fetch = [&](double *dev) -> double {
        double h = 0.0;
        cudaError_t e = cudaMemcpyAsync(&h, dev, 8, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) err = e;
        return h;
    };
    auto dot_to = [&](const float *a, const float *b, int32_t op, int32_t i) {      // no read-back
        k_dot<<<kRedBlocks, 256, 0, st>>>(a, b, P, partials);
        k_reduce_op<<<1, 256, 0, st>>>(partials, kRedBlocks, op, i, scal);
        launches += 2;
    };
    auto dot = [&](const float *a, const float *b) -> double {
        dot_to(a, b, kStore0, 0);
        return fetch(scal);
    };
    // every vector of the workspace starts a multiple of P floats after the 256-byte aligned base
    const int64_t P4 = (P % 4 == 0 && (reinterpret_cast<uintptr_t>(ws) & 15u) == 0) ? P / 4 : 0;
    const unsigned vgrid = (unsigned)(((P4 > 0 ? P4 : P) + 255) / 256);
    auto axpby = [&](float a, const float *xx, float b, const float *yy, float *zz) {
        k_axpby<<<vgrid, 256, 0, st>>>(a, xx, b, yy, P, P4, zz);
        launches += 1;
    };
    auto eval = [&](const float *xx, float *gg) -> double {
        launches += scatter_lossgrad(st, pb, xx, xx + nb, psi, partials, gg, gg + nb, scal + 1);
        ++evals;
        return fetch(scal + 1);
    };
    cudaMemcpyAsync(x, beta, nb * 4, cudaMemcpyDeviceToDevice, st);
    cudaMemcpyAsync(x + nb, S, ns * 4, cudaMemcpyDeviceToDevice, st);
    double f = eval(x, g);
    std::vector<double> gamma(kScatterHistory);          // s.y / y.y of each pair (initial scaling of the recursion)
    int32_t hist = 0, head = 0, it = 0;          // pairs stored, slot of the next pair
    int32_t stalled = 0;                         // consecutive iterations without a relevant decrease
    for (; it < max_iter && err == cudaSuccess; ++it) {
        k_absmax<<<kRedBlocks, 256, 0, st>>>(g, P, partials);
        k_sum_partials<<<1, 256, 0, st>>>(partials, kRedBlocks, 1, scal + 3);
        launches += 2;
        // d = H g by the two-loop recursion, every scalar of it on the device.  Each step is ONE launch: the vector
        // update that the previous coefficient calls for, fused with the dot product that yields the next one.
        auto slot = [&](int32_t c) { return (head - 1 - c + 2 * kScatterHistory) % kScatterHistory; };
        auto step_dot = [&](const float *in, const float *v, float scale, const float *w, int32_t op, int32_t i) {
            k_update_dot<<<kRedBlocks, 256, 0, st>>>(in, v, scale, w, P, P4, d, partials, ticket, op, i, scal);
            launches += 1;
        };
        if (hist == 0) {
            step_dot(g, nullptr, 1.f, g, kStore0, 0);                                   // d = g, g.d
        } else {
            step_dot(g, nullptr, 1.f, hs + (size_t)slot(0) * P, kAlpha, slot(0));      // d = g, alpha of the newest pair
            for (int32_t c = 1; c < hist; ++c)                                          // d -= alpha y (previous pair)
                step_dot(d, hy + (size_t)slot(c - 1) * P, 1.f, hs + (size_t)slot(c) * P, kAlpha, slot(c));
            // d = gamma (d - alpha y) of the oldest pair, then the second loop from the oldest pair up
            step_dot(d, hy + (size_t)slot(hist - 1) * P, (float)gamma[(head - 1 + kScatterHistory) % kScatterHistory],
                     hy + (size_t)slot(hist - 1) * P, kBeta, slot(hist - 1));
            for (int32_t c = hist - 2; c >= 0; --c)                                     // d += (alpha - beta) s (previous pair)
                step_dot(d, hs + (size_t)slot(c + 1) * P, 1.f, hy + (size_t)slot(c) * P, kBeta, slot(c));
            step_dot(d, hs + (size_t)slot(0) * P, 1.f, g, kStore0, 0);                  // last update, g.d
        }
        double h4[4];                            // one read-back per direction: g.d and |g|_inf
        {
            cudaError_t e = cudaMemcpyAsync(h4, scal, 32, cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (e != cudaSuccess) { err = e; break; }
        }
        if (h4[3] <= (double)gtol) break;
        double dg = -h4[0];                      // directional derivative along -d
        if (!(dg < 0.0)) {                       // not a descent direction: steepest descent, empty history
            hist = 0;
            axpby(1.f, g, 0.f, g, d);
            dg = -dot(g, g);
            if (!(dg < 0.0)) break;
        }
        double step = (hist == 0) ? std::min(1.0, 1.0 / std::sqrt(-dg)) : 1.0;
        double fn = f;
        bool ok = false;
        for (int32_t ls = 0; ls < 40 && err == cudaSuccess; ++ls) {
            axpby(1.f, x, (float)-step, d, xn);
            fn = eval(xn, gn);
            if (fn <= f + 1e-4 * step * dg) { ok = true; break; }
            step *= 0.5;
        }
        if (!ok) break;
        // s = xn - x, y = gn - g into the history slot
        float *s_new = hs + (size_t)head * P, *y_new = hy + (size_t)head * P;
        k_pair<<<kRedBlocks, 256, 0, st>>>(xn, x, gn, g, P, s_new, y_new, partials, ticket, scal);
        launches += 1;
        double h2[2];
        {
            cudaError_t e = cudaMemcpyAsync(h2, scal, 16, cudaMemcpyDeviceToHost, st);
            if (e == cudaSuccess) e = cudaStreamSynchronize(st);
            if (e != cudaSuccess) { err = e; break; }
        }
        const double sy = h2[0], yy = h2[1];
        if (sy > 1e-10 * yy && yy > 0.0) {
            const double r = 1.0 / sy;           // rho of the new pair, to the device scalars
            cudaMemcpyAsync(scal + 8 + head, &r, 8, cudaMemcpyHostToDevice, st);
            cudaStreamSynchronize(st);           // r is a local
            gamma[head] = sy / yy;
            head = (head + 1) % kScatterHistory;
            hist = std::min(hist + 1, kScatterHistory);
        } else if (hist == kScatterHistory) {
            // the rejected pair was written over the oldest pair of a full history: that slot no longer holds a
            // valid pair, so it leaves the recursion (which reads slots head - 1 ... head - hist)
            hist = kScatterHistory - 1;
        }
        std::swap(x, xn);
        std::swap(g, gn);
        stalled = (f - fn <= 1e-9 * std::fabs(f)) ? stalled + 1 : 0;
        f = fn;
        if (stalled >= 2) { ++it; break; }
    }
    cudaMemcpyAsync(beta, x, nb * 4, cudaMemcpyDeviceToDevice, st);
    cudaMemcpyAsync(S, x + nb, ns * 4, cudaMemcpyDeviceToDevice, st);
    if (err == cudaSuccess) err = cudaStreamSynchronize(st);
    if (err == cudaSuccess) err = cudaGetLastError();
    *out_loss = f;
    *out_iters = it;
    *out_evals = evals;
    *out_launches = launches;
    return err == cudaSuccess ? 0 : (int32_t)err;
}

}  // namespace tno
