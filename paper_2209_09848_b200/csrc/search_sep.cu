// Separable, trajectory-batched matched-filter kernel for sm_100a, accumulating in coordinates
// that FOLLOW each trajectory.
//
// What it computes (BASELINE.json:north_star; Eq. 5, evaluated sparsely as
// suggested at L118): for a BATCH of trajectories that share one x-motion (vx, ax),
//     X_t(x, y')  = sum_i gx_t[i] R_t(x + sx_t + i - 2, y')                          (x-pass, shared)
//     N_e(x, y)  += sum_j (gy_{e,t}[j] / sigma_t^2) X_t(x, y + d_{e,t} + j - 2)        (y-pass, per entry)
// for all frames t, where d_{e,t} is the integer y-shift of entry e at frame t.
//
// The y-pass is indexed by the POSITION P = y + d_{e,t} of the track in frame t, not by the start
// pixel y: a CTA owns the frame-space rows P in [Y0, Y0 + HT) of a 64-column strip, so every entry
// reads the SAME rows P-2..P+2 of X_t.  A thread loads its R+4 window rows of X_t once per frame
// into registers and reuses them for all of its entries with static register indices (the
// start-pixel formulation needs one window per entry and is bound by shared-memory bandwidth).
// The price: the output row held by an accumulator, y = P - d_{e,t}, changes whenever d_{e,t}
// does.  Just before that happens (and every kSeg frames, and after the last frame) the entry's
// accumulators are added into the PIECE buffer piece[ty mod NP][entry][y][x] in global memory
// (L2 resident while hot) and cleared.  Tile rows ty and ty' contribute to the same output row
// only if |ty - ty'| < NP, so every piece address belongs to exactly one CTA and plain
// read-modify-write is race free and deterministic.  k_finish sums the NP pieces in a fixed order,
// multiplies by D^(-1/2), stores the map and collects the candidates.  The segment flushes also
// bound the FP32 rounding error of long sums (|dSNR| <= 1e-3 on bright tracks).
//
// Structure:
//   * persistent CTAs, one per SM, walk (tile, batch) work items batch-fastest, so the batches of
//     one tile run on neighbouring CTAs at the same time and share the frame tiles in L2;
//   * frame tiles of (HT + 4) rows x 76 columns are staged by TMA (cp.async.bulk.tensor.3d, zero
//     fill outside the frame = "dropped from N") into a STAGES-deep shared-memory ring together
//     with the per-(batch, frame) table (cp.async.bulk), completion on mbarriers;
//   * x-pass: 8 outputs per thread from four 16-byte shared loads; the row pitches (76 and 68
//     words) make a quarter-warp of 8 rows hit 32 distinct banks on both the loads and the stores;
//   * y-pass: R rows x 2 columns x NBW entries per thread in FP32 registers.
#include <cstdio>

#include "kernels.h"
#include "topk.cuh"

namespace tno {

// ------------------------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int32_t c0, int32_t c1,
                                            int32_t c2, uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, "
        "%3, %4}], [%5];" ::"r"(smem_u32(dst)),
        "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void bulk_load(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}

// ------------------------------------------------------------------------------------ configuration
constexpr int kTileW = 64;   // output tile width: 32 lanes x 2 columns
constexpr int kBoxW = 76;    // staged columns: 64 + 4 halo + up to 3 of alignment (the TMA start
                             // coordinate must be 16-byte aligned) = 71, padded to a pitch = 12 mod 32
constexpr int kXP = 68;      // pitch of the X rows (words), = 4 mod 32
constexpr int kSeg = 64;     // an entry's accumulators are flushed at least every kSeg frames
constexpr int kHdr = 16;     // header words of a stage table entry
// stage table entry (32-bit words), one per (batch, frame t):
//   [0] xo = 4*floor((sx - 2)/4), the 16-byte aligned x offset of the staged box relative to the tile
//   [1] o = sx - 2 - xo in 0..3, the column of the box at which the 5-tap window of output 0 starts
//   [2] number of entries of the batch (they occupy slots 0 .. n-1)
//   [3] flush mask: bit e set if entry e must be flushed after this frame
//   [4..8] gx[0..4]
//   [9] xo of frame t + STAGES - 1 (look-ahead for the producer)
//   [16 + 8e + 0..4] gy_e[0..4] / sigma_t^2   [16 + 8e + 5] d_{e,t}          (entry e; zeros if empty)

template <int R_, int NB_, int RG_, int STAGES_>
struct SepCfg {
    static constexpr int R = R_, NB = NB_, RG = RG_, STAGES = STAGES_;
    static constexpr int NW = RG;                  // warps: warp w owns positions w*R .. w*R + R - 1
    static constexpr int NT = 32 * NW;
    static constexpr int HT = R * RG;              // positions (rows) per tile
    static constexpr int XROWS = HT + 4;
    static constexpr int TABW = kHdr + 8 * NB;
    static constexpr int RBUF = (XROWS * kBoxW + 31) / 32 * 32;   // floats per stage (128-byte multiple)
    static constexpr int XBUF = XROWS * kXP;                      // floats per X buffer
    static constexpr uint32_t BOX_BYTES = XROWS * kBoxW * 4;
    static constexpr size_t SMEM = (size_t)(STAGES * RBUF + 2 * XBUF + STAGES * TABW) * 4 + STAGES * 8 + 64;
    static_assert((TABW * 4) % 16 == 0 && (XBUF * 4) % 16 == 0, "16-byte alignment of the sections");
    static_assert(NW % 8 == 0, "the order of the two passes alternates between halves of each SM sub-partition");
};

// Phase of an entry's periodic flush: a function of its y-motion alone, so that the summation order
// of a trajectory (and therefore its float32 result) does not depend on the rest of the bank.
__device__ __forceinline__ int32_t seg_phase(float v, float a) {
    uint32_t h = __float_as_uint(v) * 2654435761u ^ __float_as_uint(a) * 2246822519u;
    h ^= h >> 15;
    return (int32_t)(h % (uint32_t)kSeg);
}

// ------------------------------------------------------------------------------------ table kernel
template <class C>
__global__ void k_sep_tables(ClassTables tab, const int32_t *__restrict__ batch_xc,
                             const int32_t *__restrict__ batch_yc, int32_t n_batches,
                             float *__restrict__ stage_tab) {
    const int64_t id = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int32_t T = tab.T;
    if (id >= (int64_t)n_batches * T) return;
    const int32_t b = (int32_t)(id / T), t = (int32_t)(id % T);
    const int32_t xc = batch_xc[b];
    const int32_t *yc = batch_yc + (int64_t)b * C::NB;
    float *out = stage_tab + id * C::TABW;
    int32_t *outi = reinterpret_cast<int32_t *>(out);
    auto align4 = [](int32_t v) { return v & ~3; };          // floor to a multiple of 4 (two's complement)
    const int32_t sxm2 = tab.shift[(int64_t)xc * T + t] - 2;
    for (int i = 0; i < kHdr; ++i) outi[i] = 0;
    outi[0] = align4(sxm2);
    outi[1] = sxm2 - align4(sxm2);
    for (int i = 0; i < 5; ++i) out[4 + i] = tab.g[((int64_t)xc * T + t) * 5 + i];
    const int32_t f = t + C::STAGES - 1;
    if (f < T) outi[9] = align4(tab.shift[(int64_t)xc * T + f] - 2);
    int32_t n = 0, fmask = 0;
    for (int e = 0; e < C::NB; ++e) {
        float *oe = out + kHdr + 8 * e;
        int32_t *oi = reinterpret_cast<int32_t *>(oe);
        for (int j = 0; j < 8; ++j) oi[j] = 0;
        if (yc[e] < 0) continue;
        n = e + 1;
        const int32_t c = tab.n_x + yc[e];
        const int64_t ci = (int64_t)c * T + t;
        for (int j = 0; j < 5; ++j) oe[j] = (float)(tab.gd[ci * 5 + j] * tab.qd[t]);
        oi[5] = tab.shift[ci];
        // flush before the mapping position -> output row changes, once per kSeg frames, and after
        // the last frame
        const bool fl = (t == T - 1) || (tab.shift[ci + 1] != tab.shift[ci]) ||
                        ((t + 1 + seg_phase(tab.cls_v[c], tab.cls_a[c])) % kSeg == 0);
        if (fl) fmask |= 1 << e;
    }
    outi[2] = n;
    outi[3] = fmask;
}

// ------------------------------------------------------------------------------------ main kernel
template <class C>
__global__ void __launch_bounds__(C::NT, 1)
k_search_sep(const __grid_constant__ CUtensorMap map, const SepArgs a, const int32_t ntx,
             const int32_t nty) {
    constexpr int R = C::R, NB = C::NB, NW = C::NW, HT = C::HT;
    constexpr int S = C::STAGES, TABW = C::TABW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float *Rbuf = reinterpret_cast<float *>(smem_raw);
    float *Xbuf = Rbuf + S * C::RBUF;
    float *Tab = Xbuf + 2 * C::XBUF;
    uint64_t *bar = reinterpret_cast<uint64_t *>(Tab + S * TABW);

    const int32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int32_t r0 = warp * R;
    const int32_t T = a.T, H = a.H, W = a.W;
    // Half of the warps of every SM sub-partition (warp % 4) run the y-pass before the x-pass, the
    // other half after it, so that the latencies of one pass hide under the FFMAs of the other.
    const bool y_first = (warp & 4) != 0;

    if (tid == 0) {
        for (int s = 0; s < S; ++s) mbar_init(&bar[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    uint32_t phase = 0;   // bit s = parity to wait for on stage s
    // x-pass roles: group g = (block of 8 rows, half of the 64 columns); a quarter-warp takes the
    // 8 rows of the block at one 8-column chunk.  The last warps take the ragged tail.
    const int32_t xrow_in = lane & 7, xq_in = lane >> 3;

    const int32_t n_items = ntx * nty * a.n_batches;          // < 2^31 (checked by the host)
    for (int32_t item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int32_t b = item % a.n_batches;
        const int32_t tile = item / a.n_batches;
        const int32_t ty = tile / ntx;
        const int32_t x0 = (tile % ntx) * kTileW, Y0 = ty * HT - 2;
        // positions P >= H + 2 have no tap inside the frame: warps that hold only such positions
        // and the X rows only they would read are skipped (rows past the frame arrive as zeros)
        const int32_t xrows = min(HT, (H + 2 - Y0 + R - 1) / R * R) + 4;
        const int32_t x = x0 + 2 * lane;

        float2 acc[NB][R];
#pragma unroll
        for (int s = 0; s < NB; ++s)
#pragma unroll
            for (int i = 0; i < R; ++i) acc[s][i] = make_float2(0.f, 0.f);

        auto issue = [&](int32_t f, int32_t xo) {
            const int32_t st = f % S;
            mbar_expect_tx(&bar[st], C::BOX_BYTES + TABW * 4);
            tma_load_3d(Rbuf + st * C::RBUF, &map, x0 + xo, Y0 - 2, f, &bar[st]);
            bulk_load(Tab + st * TABW, a.stage_tab + ((int64_t)b * T + f) * TABW, TABW * 4, &bar[st]);
        };

        // ---------------- x-pass of frame fx: X[fx & 1] = row-wise 5-tap correlation of the staged box
        auto x_pass = [&](int32_t fx, int32_t &nxo) {
            const int32_t st = fx % S;
            mbar_wait(&bar[st], (phase >> st) & 1u);
            phase ^= 1u << st;
            const float *tb = Tab + st * TABW;
            const int32_t *tbi = reinterpret_cast<const int32_t *>(tb);
            nxo = tbi[9];
            const int32_t o = tbi[1];
            const float g0 = tb[4], g1 = tb[5], g2 = tb[6], g3 = tb[7], g4 = tb[8];
            const float *src = Rbuf + st * C::RBUF;
            float *dst = Xbuf + (fx & 1) * C::XBUF;
            const int32_t ngroups = 2 * ((xrows + 7) >> 3);
            for (int32_t g = NW - 1 - warp; g < ngroups; g += NW) {
                const int32_t row = 8 * (g >> 1) + xrow_in, q = 4 * (g & 1) + xq_in;
                if (row < xrows) {
                    const float4 *p4 = reinterpret_cast<const float4 *>(src + row * kBoxW + 8 * q);
                    const float4 u0 = p4[0], u1 = p4[1], u2 = p4[2], u3 = p4[3];
                    const float r[16] = {u0.x, u0.y, u0.z, u0.w, u1.x, u1.y, u1.z, u1.w,
                                         u2.x, u2.y, u2.z, u2.w, u3.x, u3.y, u3.z, u3.w};
                    float v[8];
#define TNO_TAPS(O)                                                                                   \
    _Pragma("unroll") for (int c = 0; c < 8; ++c)                                                     \
        v[c] = fmaf(g4, r[O + c + 4],                                                                 \
                    fmaf(g3, r[O + c + 3], fmaf(g2, r[O + c + 2], fmaf(g1, r[O + c + 1], g0 * r[O + c]))));
                    switch (o) {                       // uniform across the CTA
                        case 0: TNO_TAPS(0) break;
                        case 1: TNO_TAPS(1) break;
                        case 2: TNO_TAPS(2) break;
                        default: TNO_TAPS(3) break;
                    }
#undef TNO_TAPS
                    float4 *d4 = reinterpret_cast<float4 *>(dst + row * kXP + 8 * q);
                    d4[0] = make_float4(v[0], v[1], v[2], v[3]);
                    d4[1] = make_float4(v[4], v[5], v[6], v[7]);
                }
            }
        };

        // ---------------- y-pass of frame i: one register window of X for all entries of the batch
        auto y_pass = [&](int32_t i) {
            const float *th = Tab + (i % S) * TABW;
            const float *tb = th + kHdr;
            const float2 *xp = reinterpret_cast<const float2 *>(Xbuf + (i & 1) * C::XBUF + r0 * kXP) + lane;
            float2 win[R + 4];
#pragma unroll
            for (int r = 0; r < R + 4; ++r) win[r] = xp[r * (kXP / 2)];
            const int32_t n = reinterpret_cast<const int32_t *>(th)[2];
            const int32_t fmask = reinterpret_cast<const int32_t *>(th)[3];
#define TNO_ENTRY(s)                                                                                  \
    {                                                                                                 \
        const float4 wa = *reinterpret_cast<const float4 *>(tb + 8 * (s));                            \
        const float w4 = tb[8 * (s) + 4];                                                             \
        _Pragma("unroll") for (int r = 0; r < R; ++r) {                                               \
            float2 c = acc[s][r];                                                                     \
            c.x = fmaf(wa.x, win[r].x, c.x);     c.y = fmaf(wa.x, win[r].y, c.y);                     \
            c.x = fmaf(wa.y, win[r + 1].x, c.x); c.y = fmaf(wa.y, win[r + 1].y, c.y);                 \
            c.x = fmaf(wa.z, win[r + 2].x, c.x); c.y = fmaf(wa.z, win[r + 2].y, c.y);                 \
            c.x = fmaf(wa.w, win[r + 3].x, c.x); c.y = fmaf(wa.w, win[r + 3].y, c.y);                 \
            c.x = fmaf(w4, win[r + 4].x, c.x);   c.y = fmaf(w4, win[r + 4].y, c.y);                   \
            acc[s][r] = c;                                                                            \
        }                                                                                             \
    }
            if (n == NB) {          // full batch: straight-line code
#pragma unroll
                for (int s = 0; s < NB; ++s) TNO_ENTRY(s)
            } else {
#pragma unroll
                for (int s = 0; s < NB; ++s)
                    if (s < n) TNO_ENTRY(s)
            }
#undef TNO_ENTRY
            if (fmask != 0) {
                // ---------------- flush: piece[ty mod NP][entry][P - d][x] += acc, acc = 0
                float *pbase = a.pieces + (int64_t)(ty % a.n_pieces) * a.piece_stride;
                const int32_t *bq = a.batch_q + (int64_t)b * NB;
#pragma unroll
                for (int s = 0; s < NB; ++s) {
                    if (fmask & (1 << s)) {
                        const int32_t d = reinterpret_cast<const int32_t *>(tb)[8 * s + 5];
                        const int32_t yb = Y0 + r0 - d;
                        const int64_t q = __ldg(bq + s) - a.q0;
                        float *p0 = pbase + (q * H + yb) * (int64_t)W + x;
                        float2 old[R];
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const bool in = (uint32_t)(yb + r) < (uint32_t)H && x < W;
                            old[r] = in ? __ldcg(reinterpret_cast<const float2 *>(p0 + (int64_t)r * W))
                                        : make_float2(0.f, 0.f);
                        }
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const bool in = (uint32_t)(yb + r) < (uint32_t)H && x < W;
                            if (in)
                                __stcg(reinterpret_cast<float2 *>(p0 + (int64_t)r * W),
                                       make_float2(old[r].x + acc[s][r].x, old[r].y + acc[s][r].y));
                            acc[s][r] = make_float2(0.f, 0.f);
                        }
                    }
                }
            }
        };

        __syncthreads();    // every warp is done with the previous item's buffers
        if (tid == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            const int32_t *gi = reinterpret_cast<const int32_t *>(a.stage_tab + (int64_t)b * T * TABW);
            for (int32_t f = 0; f < S && f < T; ++f) issue(f, __ldg(gi + (int64_t)f * TABW));
        }

        const bool y_active = r0 < xrows - 4;
        for (int32_t i = -1; i < T; ++i) {
            int32_t nxo = 0;
            if (y_first) {
                if (i >= 0 && y_active) y_pass(i);
                if (i + 1 < T) x_pass(i + 1, nxo);
            } else {
                if (i + 1 < T) x_pass(i + 1, nxo);
                if (i >= 0 && y_active) y_pass(i);
            }
            __syncthreads();
            if (tid == 0 && i >= 0 && i + S < T) issue(i + S, nxo);
        }
    }
}

// ------------------------------------------------------------------------------------ finishing kernel
// One block per (64 x 64 tile, entry q of the chunk): SNR = (sum of the pieces) * D^(-1/2), map
// store, candidates >= threshold into the tile's slot (BASELINE.json:north_star a4, a5).
__global__ void __launch_bounds__(256)
k_finish(const float *__restrict__ pieces, int32_t n_pieces, int64_t piece_stride,
         const int32_t *__restrict__ perm, int32_t q0, const TrajInfo *__restrict__ traj,
         const float *__restrict__ rsd, int32_t H, int32_t W, float *__restrict__ out_snr,
         TopkSlots slots) {
    __shared__ uint64_t list[kCollectTile * kCollectTile];
    __shared__ int32_t count;
    const int32_t tid = threadIdx.x, lane = tid & 31;
    const int32_t ql = blockIdx.z, k = perm[q0 + ql];
    const int32_t x0 = blockIdx.x * kCollectTile, y0 = blockIdx.y * kCollectTile;
    const bool want_topk = slots.keys != nullptr;
    if (tid == 0) count = 0;
    __syncthreads();
    const TrajInfo ti = traj[k];
    const float *rs = rsd + ti.rsd_off;
    const bool interior = !ti.bx.identity && !ti.by.identity && x0 >= ti.bx.lo &&
                          x0 + kCollectTile <= W - ti.bx.hi && y0 >= ti.by.lo &&
                          y0 + kCollectTile <= H - ti.by.hi;
    const float rs_in = interior ? __ldg(rs + (int64_t)ti.by.lo * ti.bx.n + ti.bx.lo) : 0.f;
    const float *pin = pieces + (int64_t)ql * H * W;
    float *om = out_snr ? out_snr + (int64_t)k * H * W : nullptr;
#pragma unroll
    for (int it = 0; it < kCollectTile * kCollectTile / 4 / 256; ++it) {
        const int32_t idx = it * 256 + tid;
        const int32_t y = y0 + (idx >> 4), x = x0 + 4 * (idx & 15);
        const bool in = (y < H) && (x < W);          // W % 4 == 0: the four columns are in or out together
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (in) {
            const int64_t off = (int64_t)y * W + x;
            for (int32_t c = 0; c < n_pieces; ++c) {
                const float4 p = __ldcs(reinterpret_cast<const float4 *>(pin + c * piece_stride + off));
                v.x += p.x; v.y += p.y; v.z += p.z; v.w += p.w;
            }
            if (interior) {
                v.x *= rs_in; v.y *= rs_in; v.z *= rs_in; v.w *= rs_in;
            } else {
                const float *rr = rs + (int64_t)border_class(y, ti.by, H) * ti.bx.n;
                v.x *= __ldg(rr + border_class(x, ti.bx, W));
                v.y *= __ldg(rr + border_class(x + 1, ti.bx, W));
                v.z *= __ldg(rr + border_class(x + 2, ti.bx, W));
                v.w *= __ldg(rr + border_class(x + 3, ti.bx, W));
            }
            if (om) *reinterpret_cast<float4 *>(om + off) = v;
        }
        if (want_topk) {
            const uint32_t pix = (uint32_t)(y * W + x);
            const float thr = slots.threshold;
            warp_push(in && v.x >= thr, make_key(v.x, pix), list, &count, lane);
            warp_push(in && v.y >= thr, make_key(v.y, pix + 1u), list, &count, lane);
            warp_push(in && v.z >= thr, make_key(v.z, pix + 2u), list, &count, lane);
            warp_push(in && v.w >= thr, make_key(v.w, pix + 3u), list, &count, lane);
        }
    }
    if (want_topk) {
        __syncthreads();
        const int64_t tile = (int64_t)blockIdx.y * gridDim.x + blockIdx.x;
        tile_flush<256>(list, count, slots, tile, k, tid);
    }
}

// ------------------------------------------------------------------------------------ host side
// (rows per thread, entries per batch, warps, stages): tile 64 positions x 64 columns, 512 threads
using V0 = SepCfg<4, 8, 16, 5>;
using V1 = SepCfg<4, 10, 16, 5>;

int32_t sep_num_variants() { return 2; }
SepVariant sep_variant(int32_t v) { return v == 0 ? SepVariant{V0::NB, V0::HT} : SepVariant{V1::NB, V1::HT}; }
int32_t sep_table_words(int32_t v) { return v == 0 ? V0::TABW : V1::TABW; }
int32_t sep_tile_rows(int32_t v, int32_t H) {
    const int32_t ht = sep_variant(v).tile_h;
    return (H + 4 + ht - 1) / ht;
}

void launch_sep_tables(cudaStream_t st, int32_t v, const ClassTables &tab, const int32_t *batch_xc,
                       const int32_t *batch_yc, int32_t n_batches, float *stage_tab) {
    const int64_t n = (int64_t)n_batches * tab.T;
    const unsigned grid = (unsigned)((n + 127) / 128);
    if (v == 0) k_sep_tables<V0><<<grid, 128, 0, st>>>(tab, batch_xc, batch_yc, n_batches, stage_tab);
    else k_sep_tables<V1><<<grid, 128, 0, st>>>(tab, batch_xc, batch_yc, n_batches, stage_tab);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *,
                                  const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

template <class C>
static int launch_t(cudaStream_t st, const SepArgs &a, void *encode_fn, int32_t *grid_out, const char **err) {
    CUtensorMap map;
    EncodeTiledFn enc = reinterpret_cast<EncodeTiledFn>(encode_fn);
    const cuuint64_t dims[3] = {(cuuint64_t)a.W, (cuuint64_t)a.H, (cuuint64_t)a.T};
    const cuuint64_t strides[2] = {(cuuint64_t)a.W * 4, (cuuint64_t)a.W * a.H * 4};
    const cuuint32_t estr[3] = {1, 1, 1};
    const cuuint32_t box[3] = {(cuuint32_t)kBoxW, (cuuint32_t)C::XROWS, 1};
    const CUresult r = enc(&map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float *>(a.frames), dims,
                           strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        *err = "cuTensorMapEncodeTiled failed";
        return (int)r;
    }
    const cudaError_t e0 = cudaFuncSetAttribute(k_search_sep<C>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                (int)C::SMEM);
    if (e0 != cudaSuccess) {
        *err = cudaGetErrorString(e0);
        return (int)e0;
    }
    const int32_t ntx = (a.W + kTileW - 1) / kTileW, nty = (a.H + 4 + C::HT - 1) / C::HT;
    const int64_t n_items = (int64_t)ntx * nty * a.n_batches;
    if (n_items >= ((int64_t)1 << 31)) {
        *err = "too many (tile, batch) work items";
        return -1;
    }
    const int32_t grid = (int32_t)(n_items < a.n_sm ? n_items : a.n_sm);
    *grid_out = grid;
    k_search_sep<C><<<grid, C::NT, C::SMEM, st>>>(map, a, ntx, nty);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        *err = cudaGetErrorString(e);
        return (int)e;
    }
    return 0;
}

int launch_search_sep(cudaStream_t st, int32_t v, const SepArgs &a, void *encode_fn, int32_t *grid_out,
                      const char **err) {
    return v == 0 ? launch_t<V0>(st, a, encode_fn, grid_out, err) : launch_t<V1>(st, a, encode_fn, grid_out, err);
}

void launch_finish(cudaStream_t st, const float *pieces, int32_t n_pieces, int64_t piece_stride,
                   const int32_t *perm, int32_t q0, int32_t q_count, const TrajInfo *traj, const float *rsd,
                   int32_t H, int32_t W, float *out_snr, const TopkSlots &slots) {
    dim3 grid((unsigned)((W + kCollectTile - 1) / kCollectTile),
              (unsigned)((H + kCollectTile - 1) / kCollectTile), (unsigned)q_count);
    k_finish<<<grid, 256, 0, st>>>(pieces, n_pieces, piece_stride, perm, q0, traj, rsd, H, W, out_snr, slots);
}

}  // namespace tno
