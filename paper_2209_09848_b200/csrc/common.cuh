// Device-side structures shared by the kernels of libtno_mf.so.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

// Debug build (nvcc -DTNO_DEBUG_CHECKS, see profiles/r2_sanitizers.md): every shared-memory index, piece address
// and ring invariant the kernels rely on is checked on the device; a violation prints its place and traps, which
// the next CUDA call of the host reports as an error.  Compiled out otherwise.
#ifdef TNO_DEBUG_CHECKS
#include <cstdio>
#define TNO_CHECK(cond)                                                                                   \
    do {                                                                                                  \
        if (!(cond)) {                                                                                    \
            printf("TNO_CHECK failed: %s  at %s:%d (block %d thread %d)\n", #cond, __FILE__, __LINE__,    \
                   (int)blockIdx.x, (int)threadIdx.x);                                                    \
            __trap();                                                                                     \
        }                                                                                                 \
    } while (0)
#else
#define TNO_CHECK(cond) do { } while (0)
#endif

namespace tno {

// ---- axis classes -----------------------------------------------------------------------------
// Class c (x-classes first, then y-classes) has, for every frame t:
//   shift[c*T + t]        integer shift floor(d + 1/2)
//   g[(c*T + t)*5 + i]    float32 PRF taps exp(-(i-2 - phase)^2 / (2 sigma^2)), i = 0..4
//   gd[(c*T + t)*5 + i]   the same taps in float64 (for D and for the fused weights)
struct ClassTables {
    const int32_t *shift;
    const float *g;
    const double *gd;
    const float *qf;      // [T] 1 / sigma_t^2
    const double *qd;     // [T]
    const float *cls_v;   // [n classes] velocity of the class (px/frame)
    const float *cls_a;   // [n classes] parallax term (px/frame^2)
    int32_t n_x;          // number of x-classes (y-class j is class n_x + j)
    int32_t T;
};

// ---- border classes ---------------------------------------------------------------------------
// D depends on (x, y) only through which taps fall off the frame.  Along one axis of extent L a
// class with shifts in [smin, smax] clips only pixels closer than lo = max(0, 2 - smin) to the low
// edge or hi = max(0, smax + 2) to the high edge; all other pixels share one value.  Pixels are
// therefore mapped to lo + 1 + hi border classes (or to themselves when lo + 1 + hi >= L).
struct AxisBorder {
    int32_t lo, hi, n, identity;
};

__host__ __device__ inline int32_t border_class(int32_t p, const AxisBorder &b, int32_t L) {
    if (b.identity) return p;
    if (p < b.lo) return p;
    if (p >= L - b.hi) return b.lo + 1 + (p - (L - b.hi));
    return b.lo;
}
__host__ __device__ inline int32_t border_rep(int32_t c, const AxisBorder &b, int32_t L) {
    if (b.identity) return c;
    if (c <= b.lo) return c;
    return L - b.hi + (c - b.lo - 1);
}

// Per trajectory: its classes and where its D^(-1/2) table [ncy][ncx] lives.
struct TrajInfo {
    int32_t xc, yc;           // x-class index, y-class index (both into their own lists)
    AxisBorder bx, by;
    int64_t rsd_off;          // offset (floats) of this trajectory's table in the rsd array
};

// ---- candidates -------------------------------------------------------------------------------
// A candidate is one 64-bit key: order-preserving image of the float32 SNR in the high word, the
// complement of the pixel index y*W + x in the low word.  Larger key = earlier in the list
// (SNR descending, then y ascending, then x ascending).  0 = empty.
__device__ __forceinline__ uint32_t snr_to_ord(float s) {
    s += 0.0f;                                   // -0 -> +0
    uint32_t u = __float_as_uint(s);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ord_to_snr(uint32_t o) {
    uint32_t u = (o & 0x80000000u) ? (o & 0x7fffffffu) : ~o;
    return __uint_as_float(u);
}
__device__ __forceinline__ uint64_t make_key(float snr, uint32_t pixel_index) {
    return ((uint64_t)snr_to_ord(snr) << 32) | (uint32_t)(~pixel_index);
}

// Tile slots of the candidate pipeline: tile ti, trajectory k owns
//   keys[(ti * K + k) * ktop .. + ktop)   and   counts[ti * K + k]  (<= ktop).
struct TopkSlots {
    uint64_t *keys;
    int32_t *counts;
    int32_t ktop;
    int32_t K;
    float threshold;
};

// Filter of one axis at tap i (0 .. 4, offset i - 2 from the rounded position) for sub-pixel phase ph in
// [-1/2, 1/2): tno_mf_config::filter (include/tno_mf.h) -- 0 point-sampled Gaussian, 1 shift-stack single tap,
// 2 pixel-integrated Gaussian (the flux fraction per pixel), 3 tabulated (row of the phase).
__device__ __forceinline__ double prf_tap(int32_t filter, int i, double ph, double prf_sigma,
                                          const float *__restrict__ prf_tab, int32_t n_phase) {
    if (filter == 1) return i == 2 ? 1.0 : 0.0;
    const double u = (double)(i - 2) - ph;
    if (filter == 2) {
        const double r = 1.0 / (prf_sigma * sqrt(2.0));
        return 0.5 * (erf((u + 0.5) * r) - erf((u - 0.5) * r));
    }
    if (filter == 3) {
        int32_t row = (int32_t)floor((ph + 0.5) * (double)n_phase);
        row = row < 0 ? 0 : (row > n_phase - 1 ? n_phase - 1 : row);
        return (double)prf_tab[5 * row + i];
    }
    return exp(-(u * u) / (2.0 * prf_sigma * prf_sigma));
}

}  // namespace tno
