// High-resolution background model (section 3.1, Eq. 1-4): with the
// scattered light already removed, every pixel is regressed on the jitter basis
//     y_t(p) = B(p) + B_theta(p) . (x_t, y_t, x_t^2, y_t^2, x_t y_t) + eps
// with the Huber loss, "through repeated least squares solves, alternated with clipping the residuals
// (Huber 1977)"; all pixels share the design matrix, so "we can reuse the computation of the inverse of the
// Gram matrix" (L98).  The host orthonormalises the basis (Phi = Q R, float64), which makes that inverse the
// identity:  c_0 = Q^T y,  c_{i+1} = c_i + Q^T clip(y - Q c_i, -delta, +delta),  beta = R^{-1} c.
// One thread keeps c of its pixels in registers through all iterations; every iteration is one pass over
// the stack (4 bytes and 12 FMA per pixel and frame), the last pass writes the residuals.
//
// Q table on the device: [T][16] floats, row t = (q0,q0, q1,q1, ..., q5,q5, 0,0,0,0): every coefficient
// twice, so that a 16-byte shared-memory load yields two ready operands of the packed FFMA2.
#include "kernels.h"

namespace tno {

// ---- plain variant: one pixel per thread, ordinary loads; any n_px and alignment ---------------------------
__global__ void __launch_bounds__(256)
k_background_plain(const float *frames, int32_t T, int64_t n_px, const float *__restrict__ Q, BgRinv rinv,
                   float delta, int32_t n_iter, float *__restrict__ out_coef, float *out_resid) {
    // frames and out_resid may be the same buffer (in place): no __restrict__ on them
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_px) return;
    float c[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    for (int32_t it = 0; it <= n_iter; ++it) {
        float s[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        const float lim = it == 0 ? INFINITY : delta;          // pass 0: ordinary least squares (c = 0)
#pragma unroll 4
        for (int32_t t = 0; t < T; ++t) {
            float q[6];
#pragma unroll
            for (int k = 0; k < 6; ++k) q[k] = __ldg(Q + 16 * (int64_t)t + 2 * k);
            float r = frames[(int64_t)t * n_px + p];
#pragma unroll
            for (int k = 0; k < 6; ++k) r = fmaf(-q[k], c[k], r);
            r = fminf(fmaxf(r, -lim), lim);
#pragma unroll
            for (int k = 0; k < 6; ++k) s[k] = fmaf(q[k], r, s[k]);
        }
#pragma unroll
        for (int k = 0; k < 6; ++k) c[k] += s[k];
    }
    if (out_resid) {
#pragma unroll 4
        for (int32_t t = 0; t < T; ++t) {
            float r = frames[(int64_t)t * n_px + p];
#pragma unroll
            for (int k = 0; k < 6; ++k) r = fmaf(-__ldg(Q + 16 * (int64_t)t + 2 * k), c[k], r);
            out_resid[(int64_t)t * n_px + p] = r;
        }
    }
    if (out_coef) {
        // beta = R^{-1} c (upper triangular, rows of dropped columns are zero)
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            float b = 0.f;
#pragma unroll
            for (int m = 0; m < 6; ++m) b = fmaf(rinv.v[k * 6 + m], c[m], b);
            out_coef[(int64_t)k * n_px + p] = b;
        }
    }
}

// ---- bulk-copy staged variant -----------------------------------------------------------------------------
// The time series of a pixel has one sample per frame, one frame = H*W*4 bytes apart: a thread that walks it
// with ordinary loads touches a different 2 MB page at every step, and once T exceeds the reach of the TLB
// (measured: the plain kernel drops from 5.3 TB/s at T = 50 to 2.9 TB/s at T >= 100, whatever H and W are)
// every warp-load pays a miss.  Here one elected thread requests each frame's NT*4 pixels as ONE bulk copy
// (cp.async.bulk, one translation per 2 KB; a fifth warp does nothing else) into a ring of NS stages of FS frames,
// together with the FS rows of Q, completion on the stage's mbarrier; the ring runs on through the passes, so
// the first frames of the next pass are in flight while the last ones of this pass are consumed.  The
// arithmetic is packed (FFMA2 on pixel pairs): 24 FFMA2 + 8 FMNMX per 4 pixels and frame.
__device__ __forceinline__ uint32_t bg_smem(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void bg_wait(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n.reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n}\n"
            : "=r"(done) : "r"(bar), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void bg_bulk(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

template <int NT, int NS, int FS, int MB>
__global__ void __launch_bounds__(NT + 32, MB)
k_background_bulk(const float *frames, int32_t T, int64_t n_px, const float *__restrict__ Q /* [T][16] */,
                  BgRinv rinv, float delta, int32_t n_iter, float *__restrict__ out_coef, float *out_resid) {
    constexpr int PXF = NT * 4;                                  // floats of one frame's pixels in a stage
    constexpr int STAGE = FS * (PXF + 16);                       // + FS rows of Q
    extern __shared__ __align__(128) float ring[];               // [NS][STAGE]
    __shared__ __align__(8) uint64_t bars[2 * NS];               // full[NS], empty[NS]
    const uint32_t full = bg_smem(bars), empty = full + 8 * NS;
    const int32_t tid = threadIdx.x, lane = tid & 31;
    const int64_t p0 = (int64_t)blockIdx.x * PXF;
    const int64_t left = n_px - p0;
    const uint32_t bytes = (uint32_t)(left < PXF ? left : PXF) * 4u;     // multiple of 16: n_px % 4 == 0
    const bool live = (int64_t)tid * 4 < left;                   // idle threads still keep the barriers going
    const int64_t p = p0 + (int64_t)tid * 4;
    if (tid == 0) {
        for (int s = 0; s < NS; ++s) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(full + 8 * s), "r"(1));
            asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(empty + 8 * s), "r"(NT / 32));
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const int32_t n_pass = n_iter + 1 + (out_resid ? 1 : 0);
    const int32_t spp = (T + FS - 1) / FS;                       // stages per pass (a stage never straddles two)
    const int32_t total = n_pass * spp;
    int32_t iss = 0, iss_t0 = 0;                                 // next request: stage sequence number, first frame
    uint32_t iss_s = 0;
    auto issue = [&]() {
        const int32_t nf = min(FS, T - iss_t0);
        const uint32_t bar = full + 8 * iss_s, dst = bg_smem(ring + iss_s * STAGE);
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(nf * (bytes + 64u))
                     : "memory");
        for (int32_t f = 0; f < nf; ++f)
            bg_bulk(dst + f * (PXF * 4), frames + (int64_t)(iss_t0 + f) * n_px + p0, bytes, bar);
        bg_bulk(dst + FS * (PXF * 4), Q + 16 * (int64_t)iss_t0, nf * 64u, bar);
        ++iss;
        if (++iss_s == NS) iss_s = 0;
        iss_t0 += FS;
        if (iss_t0 >= T) iss_t0 = 0;
    };
    if (tid >= NT) {
        // producer warp: one lane keeps the ring full -- a stage is requested again as soon as the NT / 32 consumer
        // warps have released it; the consumers never issue a copy
        if (lane == 0)
            for (int32_t gq = 0; gq < total; ++gq) {
                if (gq >= NS) bg_wait(empty + 8 * iss_s, ((uint32_t)(gq / NS) - 1u) & 1u);
                issue();
            }
        return;
    }

    float2 cn[6][2];                                             // MINUS the coefficients, two pixel pairs
#pragma unroll
    for (int k = 0; k < 6; ++k) cn[k][0] = cn[k][1] = make_float2(0.f, 0.f);
    uint32_t st = 0, par = 0;                                    // stage and parity of the consumer
    int32_t g = 0;                                               // consumed stages, all passes
    // one stage: wait, FS frames through `body(frame in stage, t, pixels, q pairs)`, release, refill
    auto stage_loop = [&](auto body) {
        for (int32_t t0 = 0; t0 < T; t0 += FS, ++g) {
            bg_wait(full + 8 * st, par);
            const float *sp = ring + st * STAGE;
#pragma unroll
            for (int f = 0; f < FS; ++f) {
                if (t0 + f < T) {
                    const float4 v = reinterpret_cast<const float4 *>(sp + f * PXF)[tid];
                    const float4 *qr = reinterpret_cast<const float4 *>(sp + FS * PXF + f * 16);
                    const float4 qa = qr[0], qb = qr[1], qc = qr[2];
                    const float2 q2[6] = {make_float2(qa.x, qa.y), make_float2(qa.z, qa.w), make_float2(qb.x, qb.y),
                                          make_float2(qb.z, qb.w), make_float2(qc.x, qc.y), make_float2(qc.z, qc.w)};
                    body(t0 + f, v, q2);
                }
            }
            __syncwarp();
            if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(empty + 8 * st) : "memory");
            if (++st == NS) { st = 0; par ^= 1u; }
        }
    };
    for (int32_t it = 0; it <= n_iter; ++it) {
        float2 s[6][2];
#pragma unroll
        for (int k = 0; k < 6; ++k) s[k][0] = s[k][1] = make_float2(0.f, 0.f);
        const float lim = it == 0 ? INFINITY : delta;            // pass 0: ordinary least squares (c = 0)
        stage_loop([&](int32_t, const float4 &v, const float2 (&q2)[6]) {
            float2 r0 = make_float2(v.x, v.y), r1 = make_float2(v.z, v.w);
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                r0 = __ffma2_rn(q2[k], cn[k][0], r0);
                r1 = __ffma2_rn(q2[k], cn[k][1], r1);
            }
            r0.x = fminf(fmaxf(r0.x, -lim), lim);
            r0.y = fminf(fmaxf(r0.y, -lim), lim);
            r1.x = fminf(fmaxf(r1.x, -lim), lim);
            r1.y = fminf(fmaxf(r1.y, -lim), lim);
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                s[k][0] = __ffma2_rn(q2[k], r0, s[k][0]);
                s[k][1] = __ffma2_rn(q2[k], r1, s[k][1]);
            }
        });
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            cn[k][0].x -= s[k][0].x; cn[k][0].y -= s[k][0].y;
            cn[k][1].x -= s[k][1].x; cn[k][1].y -= s[k][1].y;
        }
    }
    if (out_resid) {
        stage_loop([&](int32_t t, const float4 &v, const float2 (&q2)[6]) {
            float2 r0 = make_float2(v.x, v.y), r1 = make_float2(v.z, v.w);
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                r0 = __ffma2_rn(q2[k], cn[k][0], r0);
                r1 = __ffma2_rn(q2[k], cn[k][1], r1);
            }
            if (live)
                *reinterpret_cast<float4 *>(out_resid + (int64_t)t * n_px + p) = make_float4(r0.x, r0.y, r1.x, r1.y);
        });
    }
    if (out_coef && live) {
        // beta = R^{-1} c (upper triangular, rows of dropped columns are zero)
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            float b[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int m = 0; m < 6; ++m) {
                b[0] = fmaf(rinv.v[k * 6 + m], -cn[m][0].x, b[0]);
                b[1] = fmaf(rinv.v[k * 6 + m], -cn[m][0].y, b[1]);
                b[2] = fmaf(rinv.v[k * 6 + m], -cn[m][1].x, b[2]);
                b[3] = fmaf(rinv.v[k * 6 + m], -cn[m][1].y, b[3]);
            }
            *reinterpret_cast<float4 *>(out_coef + (int64_t)k * n_px + p) = make_float4(b[0], b[1], b[2], b[3]);
        }
    }
}

void launch_background(cudaStream_t st, const float *frames, int32_t T, int64_t n_px, const float *Q,
                       const BgRinv &rinv, float delta, int32_t n_iter, float *out_coef, float *out_resid) {
    const bool vec = (n_px % 4 == 0) && ((reinterpret_cast<uintptr_t>(frames) | reinterpret_cast<uintptr_t>(out_coef) |
                                          reinterpret_cast<uintptr_t>(out_resid)) & 15u) == 0;
    if (vec) {
        // 128 consumer threads x 4 pixels + a producer warp, 3 stages of 8 frames (50.7 KB), 4 CTAs per SM: the best
        // of the swept
        // (NT, NS, FS, CTAs/SM) on config 3 -- see DESIGN.md 8f
        constexpr int NT = 128, NS = 3, FS = 8, MB = 4;
        constexpr int smem = NS * FS * (NT * 4 + 16) * 4;
        cudaFuncSetAttribute(k_background_bulk<NT, NS, FS, MB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        k_background_bulk<NT, NS, FS, MB><<<(unsigned)((n_px + NT * 4 - 1) / (NT * 4)), NT + 32, smem, st>>>(
            frames, T, n_px, Q, rinv, delta, n_iter, out_coef, out_resid);
    } else {
        k_background_plain<<<(unsigned)((n_px + 255) / 256), 256, 0, st>>>(frames, T, n_px, Q, rinv, delta, n_iter,
                                                                          out_coef, out_resid);
    }
}

}  // namespace tno
