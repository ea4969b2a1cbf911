// Separable, trajectory-batched matched-filter kernel for sm_100a, accumulating in coordinates
// that FOLLOW each trajectory.
//
// What it computes (BASELINE.json:north_star; Eq. 5, evaluated sparsely as
// suggested at L118): for a BATCH of trajectories that share one x-motion (vx, ax),
//     X_t(x, y')  = sum_i gx_t[i] R_t(x + sx_t + i - 2, y')                          (x-pass, shared)
//     N_e(x, y)  += sum_j (gy_{e,t}[j] / sigma_t^2) X_t(x, y + d_{e,t} + j - 2)        (y-pass, per entry)
// for all frames t, where d_{e,t} is the integer y-shift of entry e at frame t.
//
// MIRROR PAIRS.  The entries of a batch are grouped into SLOTS (plan.h): a slot holds a y-motion (v, a) and its
// mirror image (-v, -a).  The mirror's shift is -d and its five taps are the reversed taps, so with the even and
// odd parts of the taps, s_j = (w[2+j] + w[2-j]) / 2 and d_j = (w[2+j] - w[2-j]) / 2,
//     E += w[2] X(P) + s_1 (X(P+1) + X(P-1)) + s_2 (X(P+2) + X(P-2))
//     O +=             d_1 (X(P+1) - X(P-1)) + d_2 (X(P+2) - X(P-2))
//     N_plus(x, P - d) = E + O,     N_minus(x, P + d) = E - O
// both members cost 5 multiply-adds per position and frame instead of 10 (the sums and differences of the
// window rows are shared by all slots of the batch).  Exact algebra: results differ from the tap-by-tap sum
// only by rounding.  A slot without a mirror in the bank is evaluated the same way (E + O only), so the map of
// a trajectory does not depend on the rest of the bank.
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
// only if |ty - ty'| < NP, so every piece address belongs to exactly one CTA; the adds are
// red.global.add.v2.f32 (no read latency), issued in a fixed order per address, hence
// deterministic.  k_finish sums the NP pieces in a fixed order, multiplies by D^(-1/2), stores the
// map and collects the candidates.  The segment flushes also bound the FP32 rounding error of long
// sums (|dSNR| <= 1e-3 on bright tracks).
//
// Structure:
//   * persistent CTAs, one per SM, walk (tile, batch) work items batch-fastest, so the batches of
//     one tile run on neighbouring CTAs at the same time and share the frame tiles in L2;
//   * warp-specialised: one producer warpgroup (80 or 56 registers per thread after setmaxnreg), each of
//     whose four warps owns every fourth frame -- it requests the frame's TMA box, runs its whole x-pass and
//     hands one of its two X buffers to the consumers -- and 12 consumer warps (144 or 152 registers) that run
//     the y-pass; the roles are linked by mbarrier rings only, there is no barrier among the producers and no
//     CTA-wide barrier in the frame loop;
//   * frame tiles of (HT + 4) rows x 76 columns are staged by TMA (cp.async.bulk.tensor.3d, zero
//     fill outside the frame = "dropped from N") together with the per-(batch, frame) table row
//     (cp.async.bulk), completion on mbarriers;
//   * x-pass: 8 outputs per thread from four 16-byte shared loads, the next step's loads issued ahead; the row
//     pitches (76 and 68 words) make a quarter-warp of 8 rows hit 32 distinct banks on both loads and stores;
//   * y-pass: R positions x 2 columns x NB slots x (E, O) per thread in FP32 registers, packed FFMA2
//     (fma.rn.f32x2: two columns per instruction, two issue cycles); the warp index goes through a shuffle so
//     that ranges, bases, ring positions and barrier addresses are uniform-datapath values, the only per-lane
//     register is the byte offset of the thread's two columns, and all shared loads of a frame (header, first
//     weights, window) are requested together ahead of their first use;
//   * two shapes are compiled (R x NB = 4 x 5 and 5 x 4, tiles of 48 and 60 positions); the host picks one per
//     search by modelled cost (api.cu).
#include <algorithm>
#include <cstdio>

#include "kernels.h"
#include "topk.cuh"

namespace tno {

// ------------------------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
// The mbarrier helpers take 32-bit shared-window addresses (smem base computed once per thread).
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!done);
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, int32_t c0, int32_t c1,
                                            int32_t c2, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, "
        "%3, %4}], [%5];" ::"r"(smem_u32(dst)),
        "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void bulk_load(void *dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}

// ------------------------------------------------------------------------------------ configuration
constexpr int kTileW = 64;   // output tile width: 32 lanes x 2 columns
constexpr int kBoxW = 76;    // staged columns: 64 + 4 halo + up to 3 of alignment (the TMA start
                             // coordinate must be 16-byte aligned) = 71, padded to a pitch = 12 mod 32
constexpr int kXP = 68;      // pitch of the X rows (words), = 4 mod 32
constexpr int kSeg = 128;    // an entry's accumulators are flushed at least every kSeg frames
constexpr int kHdr = 16;     // header words of a stage table entry
constexpr int kPW = 4;       // producer warps (one warpgroup: setmaxnreg is per warpgroup)
// stage table entry (32-bit words), one per (batch, frame t):
//   [0] xo = 4*floor((sx - 2)/4), the 16-byte aligned x offset of the staged box relative to the tile
//   [1] o = sx - 2 - xo in 0..3, the column of the box at which the 5-tap window of output 0 starts
//   [2..6] gx[0..4]
//   [8] number of slots of the batch (they occupy slots 0 .. n-1)
//   [9] flush mask: bit s set if slot s must be flushed after this frame
//   [10] wait mask: bit s set if the previous flush of slot s is at most XR frames back
//   [11], [12..15] d_2 / sigma_t^2 of slot 4 and of slots 0..3: the consumers read [8..15] with two 16-byte loads
//   [16 + 8s + 0..4] (w[2], s_1, s_2, d_1, d_2) / sigma_t^2 of slot s (zeros if empty)
//   [16 + 8s + 5] d_{s,t}    [16 + 8s + 6], [.. + 7] planned-order index of the plus / minus member relative
//                            to the first one of the batch, -1 = absent

template <int R_, int NB_, int CW_, int SB_, int XR_, int PREGS_ = 80>
struct SepCfg {
    static constexpr int R = R_, NB = NB_, CW = CW_, SB = SB_, XR = XR_;      // NB = slots per batch
    static constexpr int NT = 32 * (CW + kPW);     // consumer warps 0 .. CW-1, then the producer warpgroup
    static constexpr int HT = R * CW;              // positions (rows) per tile: consumer warp w owns w*R ..
    static constexpr int XROWS = HT + 4;
    static constexpr int TS = 16;                  // table stages, >= SB + XR + 2 (ring invariants in the kernel)
    static constexpr int TABW = kHdr + 8 * NB;
    static constexpr int RBUF = (XROWS * kBoxW + 31) / 32 * 32;   // floats per box stage (128-byte multiple)
    static constexpr int XBUF = XROWS * kXP;                      // floats per X buffer
    static constexpr uint32_t BOX_BYTES = XROWS * kBoxW * 4;
    static constexpr int NBAR = SB + 2 * XR + NB;
    static constexpr size_t SMEM = (size_t)(SB * RBUF + XR * XBUF + TS * TABW) * 4 + NBAR * 8 + 64;
    // register split: setmaxnreg moves registers between the warpgroups of the CTA, the total stays
    // what the launch allocated (NT x the per-thread count ptxas derives from __launch_bounds__)
    static constexpr int LREGS = 65536 / NT / 8 * 8;
    static constexpr int PREGS = PREGS_;
    static constexpr int CREGS_RAW = (NT * LREGS - kPW * 32 * PREGS) / (CW * 32) / 8 * 8;
    static constexpr int CREGS = CREGS_RAW > 232 ? 232 : CREGS_RAW;
    static_assert(CW % 4 == 0 && (CW * 32 * CREGS + kPW * 32 * PREGS) <= NT * LREGS, "register budget");
    static_assert((SB & (SB - 1)) == 0 && (XR & (XR - 1)) == 0 && (TS & (TS - 1)) == 0 && TS >= SB + XR + 2,
                  "ring sizes are powers of two");
    static_assert((TABW * 4) % 16 == 0 && (XBUF * 4) % 16 == 0, "16-byte alignment of the sections");
    static_assert(NB <= 5, "the header holds d_2 of five slots");
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
                             const int32_t *__restrict__ slot_yc, const int32_t *__restrict__ slot_flip,
                             const int32_t *__restrict__ slot_q, int32_t n_batches, int32_t squared,
                             float *__restrict__ stage_tab) {
    const int64_t id = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int32_t T = tab.T;
    if (id >= (int64_t)n_batches * T) return;
    const int32_t b = (int32_t)(id / T), t = (int32_t)(id % T);
    const int32_t xc = batch_xc[b];
    const int32_t *yc = slot_yc + (int64_t)b * C::NB;
    float *out = stage_tab + id * C::TABW;
    int32_t *outi = reinterpret_cast<int32_t *>(out);
    auto align4 = [](int32_t v) { return v & ~3; };          // floor to a multiple of 4 (two's complement)
    const int32_t sxm2 = tab.shift[(int64_t)xc * T + t] - 2;
    for (int i = 0; i < kHdr; ++i) outi[i] = 0;
    outi[0] = align4(sxm2);
    outi[1] = sxm2 - align4(sxm2);
    // squared = 1: the taps of the D pass over the validity weights, sum g^2 V / sigma^2
    for (int i = 0; i < 5; ++i) {
        const double gv = tab.gd[((int64_t)xc * T + t) * 5 + i];
        out[2 + i] = squared ? (float)(gv * gv) : tab.g[((int64_t)xc * T + t) * 5 + i];
    }
    int32_t n = 0, fmask = 0, fwait = 0;
    for (int e = 0; e < C::NB; ++e) {
        float *oe = out + kHdr + 8 * e;
        int32_t *oi = reinterpret_cast<int32_t *>(oe);
        for (int j = 0; j < 8; ++j) oi[j] = 0;
        oi[6] = oi[7] = -1;
        if (yc[e] < 0) continue;
        n = e + 1;
        const int32_t flip = slot_flip[(int64_t)b * C::NB + e];
        const int32_t c = tab.n_x + yc[e];
        const int64_t ci = (int64_t)c * T + t;
        // taps of the slot's orientation: those of the class, reversed if the class is the mirror image
        double w[5];
        for (int j = 0; j < 5; ++j) {
            const double gv = tab.gd[ci * 5 + (flip ? 4 - j : j)];
            w[j] = (squared ? gv * gv : gv) * tab.qd[t];
        }
        oe[0] = (float)w[2];
        oe[1] = (float)(0.5 * (w[3] + w[1]));
        oe[2] = (float)(0.5 * (w[4] + w[0]));
        oe[3] = (float)(0.5 * (w[3] - w[1]));
        oe[4] = (float)(0.5 * (w[4] - w[0]));
        out[e < 4 ? 12 + e : 11] = oe[4];
        oi[5] = flip ? -tab.shift[ci] : tab.shift[ci];
        oi[6] = slot_q[((int64_t)b * C::NB + e) * 2];
        oi[7] = slot_q[((int64_t)b * C::NB + e) * 2 + 1];
        // flush before the mapping position -> output row changes, once per kSeg frames, and after
        // the last frame.  The phase of the periodic flush is that of the slot's orientation.
        const float ov = (flip ? -tab.cls_v[c] : tab.cls_v[c]) + 0.0f, oa = (flip ? -tab.cls_a[c] : tab.cls_a[c]) + 0.0f;
        const int32_t ph = seg_phase(ov, oa);
        const bool fl = (t == T - 1) || (tab.shift[ci + 1] != tab.shift[ci]) || ((t + 1 + ph) % kSeg == 0);
        if (fl) {
            fmask |= 1 << e;
            // was the slot also flushed after one of the frames t - XR .. t - 1 ?  (t < XR: the
            // last frame of the CTA's previous work item, where every slot is flushed, is that close)
            if (t < C::XR) fwait |= 1 << e;
            for (int32_t u = max(t - C::XR, 0); u < t; ++u)
                if (tab.shift[ci - t + u + 1] != tab.shift[ci - t + u] || (u + 1 + ph) % kSeg == 0) fwait |= 1 << e;
        }
    }
    outi[8] = n;
    outi[9] = fmask;
    outi[10] = fwait;
}

// ------------------------------------------------------------------------------------ main kernel
// Predicated red.global.add.v2.f32 (fire and forget: no read latency, no branch).
__device__ __forceinline__ void red_add_v2_if(bool pred, float *addr, float2 v) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.u32 p, %0, 0;\n"
        "@p red.global.add.v2.f32 [%1], {%2, %3};\n"
        "}\n" ::"r"((uint32_t)pred),
        "l"(addr), "f"(v.x), "f"(v.y)
        : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// One arrival for the whole (converged) warp: elect.sync picks the lane, no thread index needed.
__device__ __forceinline__ void mbar_arrive_one(uint32_t bar) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "elect.sync _|p, 0xffffffff;\n"
        "@p mbarrier.arrive.shared::cta.b64 _, [%0];\n"
        "}\n" ::"r"(bar)
        : "memory");
}

// x-pass of one thread and step: 8 outputs X(c .. c+7) = sum_i g[i] R(c + O + i) from the 16 staged values
// R(c .. c+15) of its row (four 16-byte loads), O = 0..3 the offset of the window in the 16-byte aligned box.
struct XIn { float4 a, b, c, d; };
__device__ __forceinline__ XIn xpass_load(const float *p) {
    const float4 *p4 = reinterpret_cast<const float4 *>(p);
    return XIn{p4[0], p4[1], p4[2], p4[3]};
}
template <int O>
__device__ __forceinline__ void xpass_step(const XIn &u, float *dst, const float (&g)[5]) {
    const float r[16] = {u.a.x, u.a.y, u.a.z, u.a.w, u.b.x, u.b.y, u.b.z, u.b.w,
                         u.c.x, u.c.y, u.c.z, u.c.w, u.d.x, u.d.y, u.d.z, u.d.w};
    float v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = g[0] * r[O + j];
#pragma unroll
    for (int i = 1; i < 5; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = fmaf(g[i], r[O + j + i], v[j]);
    reinterpret_cast<float4 *>(dst)[0] = make_float4(v[0], v[1], v[2], v[3]);
    reinterpret_cast<float4 *>(dst)[1] = make_float4(v[4], v[5], v[6], v[7]);
}
// One frame of one producer warp.  Row groups of 8: a quarter-warp takes 8 rows at one offset of 8 columns (lane & 7 =
// row, lane >> 3 = octet of columns: 32 distinct banks for the 16-byte loads at pitch 76 and the 16-byte stores at
// pitch 68), the warp covers 8 rows x 32 columns per step and walks the two halves of each group; the loads of the
// next step are issued before the arithmetic of the current one (in program order ahead of its stores, which the
// compiler must assume may alias them).  A last group of m <= 4 rows (the 52 rows of the first kernel shape: m = 4)
// is done in ONE step with lane & 3 = row and lane >> 2 = octet, all 64 columns: half the instructions of a
// half-empty group of 8.
template <int O>
__device__ __forceinline__ void xpass_frame4(const float *srcb, float *dstb, int32_t lane, int32_t xrows,
                                            const float (&g)[5]) {
    const int32_t row_in = lane & 7, oct_in = lane >> 3;
    const float *src = srcb + row_in * kBoxW + 8 * oct_in;
    float *dst = dstb + row_in * kXP + 8 * oct_in;
    const int32_t nfull = xrows >> 3, m = xrows & 7;          // row groups with all 8 rows, rows of the last group
    const bool tail8 = m > 4 && row_in < m;                   // this lane's row of a last group of 5 .. 7 rows
    XIn u = xpass_load(src);                    // left half of the current row group
    for (int32_t i = 0; i < nfull; ++i) {
        const XIn w = xpass_load(src + 32);     // right half
        xpass_step<O>(u, dst, g);
        src += 8 * kBoxW;
        if (i + 1 < nfull || tail8) u = xpass_load(src);
        xpass_step<O>(w, dst + 32, g);
        dst += 8 * kXP;
    }
    if (m > 4) {
        if (tail8) {
            const XIn w = xpass_load(src + 32);
            xpass_step<O>(u, dst, g);
            xpass_step<O>(w, dst + 32, g);
        }
    } else if (m > 0) {
        const int32_t r4 = lane & 3, o8 = lane >> 2;
        if (r4 < m) {
            const XIn t = xpass_load(srcb + (8 * nfull + r4) * kBoxW + 8 * o8);
            xpass_step<O>(t, dstb + (8 * nfull + r4) * kXP + 8 * o8, g);
        }
    }
}

// One frame of one producer warp: this lane's rows row_in, row_in + 8, ... of the box, columns 8 oct_in .. + 7
// and 32 + 8 oct_in .. + 7.  The loads of the next step are issued before the arithmetic of the current one
// (in program order ahead of its stores, which the compiler must assume may alias them).
template <int O>
__device__ __forceinline__ void xpass_frame(const float *src, float *dst, int32_t nfull, bool tail,
                                            const float (&g)[5]) {
    XIn u = xpass_load(src);                    // left half of the current row group
    for (int32_t i = 0; i < nfull; ++i) {
        const XIn w = xpass_load(src + 32);     // right half
        xpass_step<O>(u, dst, g);
        src += 8 * kBoxW;
        if (i + 1 < nfull || tail) u = xpass_load(src);
        xpass_step<O>(w, dst + 32, g);
        dst += 8 * kXP;
    }
    if (tail) {
        const XIn w = xpass_load(src + 32);
        xpass_step<O>(u, dst, g);
        xpass_step<O>(w, dst + 32, g);
    }
}

// Warp-specialised, persistent.  Per CTA-local frame counter n (frames of all its work items in
// sequence) three rings connect the roles:
//   box[n % SB]  TMA -> producer       full_box  (tx bytes; also covers tab[n % TS])
//   X[n % XR]    producer -> consumers x_full   (1 arrival),  x_empty (CW arrivals)
//   tab[n % TS]  TMA -> producer (gx) and consumers (weights, d, masks)
// Frame n belongs to producer warp n % kPW (XR = kPW, SB = 2 kPW: the warp's own X buffer and its two
// box stages).  The warp requests frame n + SB when it has finished frame n, which it started only
// after all consumers had released frame n - XR, i.e. had finished frame n - XR - 1 completely: the
// table stage (n + SB) % TS was last used by frame n + SB - TS <= n - XR - 1 for TS >= SB + XR + 1,
// even though a consumer releases X before it runs the flush of that frame (which still reads d from
// the table).
template <class C>
__global__ void __launch_bounds__(C::NT, 1)
k_search_sep(const __grid_constant__ CUtensorMap map, const SepArgs a, const int32_t ntx,
             const int32_t nty) {      // nty tile rows starting at a.ty0
    constexpr int R = C::R, NB = C::NB, CW = C::CW, HT = C::HT;
    constexpr int SB = C::SB, XR = C::XR, TS = C::TS, TABW = C::TABW;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float *Rbuf = reinterpret_cast<float *>(smem_raw);
    float *Xbuf = Rbuf + SB * C::RBUF;
    float *Tab = Xbuf + XR * C::XBUF;
    const uint32_t full_box = smem_u32(Tab + TS * TABW);   // mbarriers, 8 bytes each:
    const uint32_t x_full = full_box + 8 * SB;             //   [SB] box + table landed, [XR] X produced,
    const uint32_t x_empty = x_full + 8 * XR;              //   [XR] X consumed by all consumer warps,
    const uint32_t f_done = x_empty + 8 * XR;              //   [NB] k-th flush of entry e finished by all of them

    const int32_t tid = threadIdx.x, lane = tid & 31;
    // (through a shuffle the warp index is warp-uniform for the compiler: role tests, row ranges and barrier
    // addresses derived from it live in uniform registers instead of being recomputed from the thread index)
    const int32_t warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int32_t T = a.T, H = a.H, W = a.W;
    const int32_t n_items = ntx * nty * a.n_batches;          // < 2^31 (checked by the host)

    if (tid == 0) {
        for (int s = 0; s < SB; ++s) mbar_init(full_box + 8 * (s), 1);
        for (int s = 0; s < XR; ++s) { mbar_init(x_full + 8 * (s), 1); mbar_init(x_empty + 8 * (s), CW); }
        for (int s = 0; s < NB; ++s) mbar_init(f_done + 8 * (s), CW);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= CW) {
        // =============================================================== producers: TMA + x-pass
        // Producer warp pw owns the CTA-local frames n = pw, pw + kPW, ...: it requests their boxes (two
        // stages of its own, so the next box is in flight while it works), runs the whole x-pass of the
        // frame and hands X[n % XR] = X[pw] to the consumers.  The four warps work on four consecutive
        // frames at the same time and never synchronise with each other; the per-frame costs (two
        // mbarrier waits, the table row, the hand-over) are paid once per warp and frame.
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(C::PREGS));
        static_assert(XR % kPW == 0 && SB % kPW == 0, "whole X buffers and box stages per producer warp");
        constexpr int BST = SB / kPW, XST = XR / kPW;       // box stages and X buffers of one producer warp
        const int32_t pw = warp - CW;
        // position of this warp's next frame to REQUEST (iss_*) and to PROCESS (item, t) in the CTA's
        // sequence of (work item, frame)
        int32_t iss_item = blockIdx.x, iss_t = pw;
        uint32_t iss_k = 0;      // (ring counters are unsigned: their divisions and remainders are shifts and masks)
        auto advance = [&](int32_t &it, int32_t &tt) {
            tt += kPW;
            while (tt >= T) { tt -= T; it += gridDim.x; }
        };
        while (iss_t >= T) { iss_t -= T; iss_item += gridDim.x; }
        int32_t item = iss_item, t = iss_t;
        // (the divisions that split a work item into batch and tile are redone only when the item changes)
        int32_t iss_cached = -1, iss_b = 0, iss_x0 = 0, iss_y0 = 0;
        auto iss_one = [&]() {          // lane 0: request frame (iss_item, iss_t) into this warp's next box stage
            if (iss_item != iss_cached) {
                iss_cached = iss_item;
                iss_b = iss_item % a.n_batches;
                const int32_t tl = a.ty0 * ntx + iss_item / a.n_batches;
                iss_x0 = (tl % ntx) * kTileW;
                iss_y0 = (tl / ntx) * HT - 4;
            }
            const int32_t b = iss_b;
            const int32_t *row = reinterpret_cast<const int32_t *>(a.stage_tab + ((int64_t)b * T + iss_t) * TABW);
            const uint32_t sb = pw + kPW * (iss_k % BST), n = pw + kPW * iss_k;
            TNO_CHECK(iss_item >= 0 && iss_item < n_items && iss_t >= 0 && iss_t < T && b < a.n_batches);
            TNO_CHECK(sb >= 0 && sb < SB && ((__ldg(row) & 3) == 0) && (uint32_t)__ldg(row + 1) < 4u);
            TNO_CHECK(iss_y0 + 4 < (a.ty0 + nty) * HT && iss_x0 < ntx * kTileW);
            mbar_expect_tx(full_box + 8 * (sb), C::BOX_BYTES + TABW * 4);
            tma_load_3d(Rbuf + sb * C::RBUF, &map, iss_x0 + __ldg(row), iss_y0, iss_t, full_box + 8 * (sb));
            bulk_load(Tab + (n & (TS - 1)) * TABW, row, TABW * 4, full_box + 8 * (sb));
        };
        if (lane == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            for (int f = 0; f < BST && iss_item < n_items; ++f) {
                iss_one();
                ++iss_k;
                advance(iss_item, iss_t);
            }
        }
        iss_k = BST;        // (all lanes keep the same counters; only lane 0 issues)
        {
            int32_t ii = blockIdx.x, tt = pw;
            while (tt >= T) { tt -= T; ii += gridDim.x; }
            for (int f = 0; f < BST; ++f) advance(ii, tt);
            iss_item = ii; iss_t = tt;
        }
        int32_t cached = -1, xrows = 0;
        for (uint32_t k = 0; item < n_items; ++k) {
            if (item != cached) {
                cached = item;
                const int32_t Y0 = (a.ty0 + item / a.n_batches / ntx) * HT - 2;
                // positions P >= H + 2 have no tap inside the frame: the X rows only they would read are skipped
                xrows = min(HT, (H + 2 - Y0 + R - 1) / R * R) + 4;
            }
            const uint32_t sb = pw + kPW * (k % BST), xb = pw + kPW * (k % XST), n = pw + kPW * k;
            mbar_wait(full_box + 8 * (sb), (k / BST) & 1);
            if (k >= XST) mbar_wait(x_empty + 8 * (xb), (k / XST + 1) & 1);
            const float *tb = Tab + (n & (TS - 1)) * TABW;
            const int32_t o = reinterpret_cast<const int32_t *>(tb)[1];
            float g[5];
#pragma unroll
            for (int i = 0; i < 5; ++i) g[i] = tb[2 + i];
            TNO_CHECK(xrows >= 4 + R && xrows <= C::XROWS && (uint32_t)o < 4u && sb < SB);
            TNO_CHECK((xrows + 7) / 8 * 8 * kBoxW <= C::RBUF + 8 * kBoxW);      // loads stay inside the staging ring
            if constexpr (C::XROWS % 8 != 0 && C::XROWS % 8 <= 4) {
                // (the shape whose full tiles end in a group of <= 4 rows: that group in one step)
                const float *src = Rbuf + sb * C::RBUF;
                float *dst = Xbuf + xb * C::XBUF;
                switch (o) {                                        // uniform across the CTA
                    case 0: xpass_frame4<0>(src, dst, lane, xrows, g); break;
                    case 1: xpass_frame4<1>(src, dst, lane, xrows, g); break;
                    case 2: xpass_frame4<2>(src, dst, lane, xrows, g); break;
                    default: xpass_frame4<3>(src, dst, lane, xrows, g); break;
                }
            } else {
                const int32_t row_in = lane & 7, oct_in = lane >> 3;
                const float *src = Rbuf + sb * C::RBUF + row_in * kBoxW + 8 * oct_in;
                float *dst = Xbuf + xb * C::XBUF + row_in * kXP + 8 * oct_in;
                const int32_t nfull = xrows >> 3;                   // row groups with all 8 rows
                const bool tail = row_in < (xrows & 7);             // this lane's row of the last, partial group
                switch (o) {
                    case 0: xpass_frame<0>(src, dst, nfull, tail, g); break;
                    case 1: xpass_frame<1>(src, dst, nfull, tail, g); break;
                    case 2: xpass_frame<2>(src, dst, nfull, tail, g); break;
                    default: xpass_frame<3>(src, dst, nfull, tail, g); break;
                }
            }
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(x_full + 8 * (xb));
                // this warp is done with box stage sb: request the frame that uses it next
                if (iss_item < n_items) { iss_k = k + BST; iss_one(); }
            }
            advance(iss_item, iss_t);
            advance(item, t);
        }
    } else {
        // =============================================================== consumers: y-pass + flush
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(C::CREGS));
        const int32_t r0 = warp * R;
        uint32_t n = 0;           // CTA-local frame counter (unsigned: ring positions are shifts and masks)
        uint32_t fpar = 0;        // bit s = parity of the number of flushes of slot s so far
        // The only per-lane quantity a consumer keeps: the byte offset of its two columns, both in a row of X
        // and in a row of a piece map.  Everything else below (window base, piece base, rows) is the same for
        // the whole warp and stays in uniform registers; the loads are explicit ld.shared with immediate row
        // offsets.
        uint32_t lane8 = 8u * (uint32_t)lane;
        asm volatile("" : "+r"(lane8));
        const uint32_t xwu = smem_u32(Xbuf + r0 * kXP);
        for (int32_t item = blockIdx.x; item < n_items; item += gridDim.x) {
            // flush coordinates of the item: the members of the batch have planned indices q_first + (the
            // offsets in the table), a member's piece map starts at ebase + offset*H*W (column x0 of the tile;
            // this lane's two columns are lane8 bytes further), and the accumulator row r of this warp holds
            // output row yr0 + r - d (plus member) or yr0 + r + d (minus member)
            const int32_t b = item % a.n_batches, tile = a.ty0 * ntx + item / a.n_batches;
            const int32_t ty = tile / ntx;
            const int32_t x0 = (tile % ntx) * kTileW;
            float *ebase = a.pieces + (int64_t)(ty % a.n_pieces) * a.piece_stride +
                           (int64_t)(__ldg(a.batch_q + b) - a.q0) * H * W + x0;
            // bytes of a row of the tile that lie inside the frame (columns past it are never flushed)
            const uint32_t wlim = 4u * (uint32_t)min(kTileW, W - x0);
            const int32_t yr0 = ty * HT - 2 + r0;
            // else: positions without any tap in the frame
            const bool y_active = r0 < min(HT, H + 4 - ty * HT);

            float2 accE[NB][R], accO[NB][R];
#pragma unroll
            for (int s = 0; s < NB; ++s)
#pragma unroll
                for (int i = 0; i < R; ++i) accE[s][i] = accO[s][i] = make_float2(0.f, 0.f);

            for (int32_t t = 0; t < T; ++t) {
                const uint32_t xr = n & (XR - 1);
                mbar_wait(x_full + 8 * (xr), (n / XR) & 1);
                const float *th = Tab + (n & (TS - 1)) * TABW;
                const float *tb = th + kHdr;
                // number of slots and flush mask of the frame (and d_2 of slot 4), read together ahead of the FFMAs,
                // but requested after the window: the header's move into uniform registers waits for its load, and
                // the warp issues in order
                int4 hq;
                if (y_active) {
                    // ---------------- y-pass: one register window of X for all slots of the batch, and the
                    // sums and differences of its rows about each of this thread's R positions
                    const uint32_t xw = xwu + (uint32_t)xr * (C::XBUF * 4) + lane8;
                    TNO_CHECK(xw + (R + 3) * (kXP * 4) + 8 <= smem_u32(Xbuf + (xr + 1) * C::XBUF));   // inside X[xr]
                    // (the weights of slot 0 are requested before the window, not after the sums that need it)
                    const float4 wa0 = *reinterpret_cast<const float4 *>(tb);
                    float2 win[R + 4];
#pragma unroll
                    for (int r = 0; r < R + 4; ++r)
                        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];"
                                     : "=f"(win[r].x), "=f"(win[r].y) : "r"(xw + (uint32_t)(r * kXP * 4)));
                    asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                                 : "=r"(hq.x), "=r"(hq.y), "=r"(hq.z), "=r"(hq.w) : "r"(smem_u32(th + 8)));
                    TNO_CHECK(hq.x >= 1 && hq.x <= NB && (hq.y >> NB) == 0);
                    float2 A1[R], B1[R], A2[R], B2[R];
                    const float2 neg1 = make_float2(-1.f, -1.f);
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        A1[r] = __fadd2_rn(win[r + 3], win[r + 1]);
                        B1[r] = __ffma2_rn(neg1, win[r + 1], win[r + 3]);       // exact difference
                        A2[r] = __fadd2_rn(win[r + 4], win[r]);
                        B2[r] = __ffma2_rn(neg1, win[r], win[r + 4]);
                    }
                    const int32_t nfill = hq.x;
#define TNO_FMAS(s)                                                                                      \
    {                                                                                                    \
        const float2 w0 = make_float2(wa.x, wa.x), w1 = make_float2(wa.y, wa.y),                         \
                     w2 = make_float2(wa.z, wa.z), w3 = make_float2(wa.w, wa.w), w5 = make_float2(w4, w4); \
        _Pragma("unroll") for (int r = 0; r < R; ++r) accE[s][r] = __ffma2_rn(w0, win[r + 2], accE[s][r]); \
        _Pragma("unroll") for (int r = 0; r < R; ++r) accO[s][r] = __ffma2_rn(w3, B1[r], accO[s][r]);      \
        _Pragma("unroll") for (int r = 0; r < R; ++r) accE[s][r] = __ffma2_rn(w1, A1[r], accE[s][r]);      \
        _Pragma("unroll") for (int r = 0; r < R; ++r) accO[s][r] = __ffma2_rn(w5, B2[r], accO[s][r]);      \
        _Pragma("unroll") for (int r = 0; r < R; ++r) accE[s][r] = __ffma2_rn(w2, A2[r], accE[s][r]);      \
    }
                    // d_2 of all slots: one 16-byte load and one word
                    const float4 d2q = *reinterpret_cast<const float4 *>(th + 12);
                    const float d2v[5] = {d2q.x, d2q.y, d2q.z, d2q.w, __int_as_float(hq.w)};
                    if (nfill == NB) {
                        // full batch: straight-line code, the weights of slot s + 1 are loaded
                        // before the FFMAs of slot s (the empty asm keeps ptxas from hoisting more
                        // loads than the register budget holds)
                        float4 wa = wa0;
#pragma unroll
                        for (int s = 0; s < NB; ++s) {
                            float4 wan = wa;
                            if (s + 1 < NB) wan = *reinterpret_cast<const float4 *>(tb + 8 * (s + 1));
                            const float w4 = d2v[s];
                            TNO_FMAS(s)
                            asm volatile("" ::: "memory");
                            wa = wan;
                        }
                    } else {
#pragma unroll
                        for (int s = 0; s < NB; ++s)
                            if (s < nfill) {
                                const float4 wa = s == 0 ? wa0 : *reinterpret_cast<const float4 *>(tb + 8 * s);
                                const float w4 = d2v[s];
                                TNO_FMAS(s)
                            }
                    }
#undef TNO_FMAS
                } else {
                    hq = *reinterpret_cast<const int4 *>(th + 8);
                }
                const int32_t fmask = hq.y;
                __syncwarp();
                {
                    // (the ring position again from the frame counter: nothing is kept across the FFMAs for it)
                    uint32_t n2 = n;
                    asm volatile("" : "+r"(n2));
                    mbar_arrive_one(x_empty + 8 * (n2 & (XR - 1)));  // this warp no longer reads X[xr]
                }
                if (fmask != 0) {
                    const int32_t fwait = reinterpret_cast<const int32_t *>(th)[10];
                    // ---------------- flush: piece[ty mod NP][member][P -+ d][x] += E +- O, E = O = 0
#pragma unroll
                    for (int s = 0; s < NB; ++s) {
                        if (fmask & (1 << s)) {
                            // The output rows a warp holds change with d, so successive flushes of a
                            // slot touch the same addresses from different warps: flush k starts only
                            // after every consumer warp has finished flush k - 1 of that slot, which
                            // fixes the order of the float adds per address.  If flush k - 1 is more
                            // than XR frames back that is already implied by X[n] being there (the
                            // producers waited for every consumer to release frame n - XR, which each
                            // did after its flushes of the frames before); otherwise wait on f_done --
                            // also needed so that no warp arrives twice in one phase of f_done.
                            if (fwait & (1 << s)) mbar_wait(f_done + 8 * (s), ((fpar >> s) & 1u) ^ 1u);
                            fpar ^= 1u << s;
                            if (y_active) {
                                const int4 dq = *reinterpret_cast<const int4 *>(tb + 8 * s + 4);   // (d_2, d, q+, q-)
                                const int32_t yp = yr0 - dq.y, ym = yr0 + dq.y;
                                // (through the empty asm the lane offset is a value of this frame: the addresses
                                // are formed here from uniform registers, not carried through the frame loop)
                                uint32_t l8 = lane8;
                                asm volatile("" : "+r"(l8));
                                float *pp = reinterpret_cast<float *>(
                                    reinterpret_cast<char *>(ebase + ((int64_t)dq.z * H + yp) * W) + l8);
                                float *pm = reinterpret_cast<float *>(
                                    reinterpret_cast<char *>(ebase + ((int64_t)dq.w * H + ym) * W) + l8);
                                asm volatile("" : "+l"(pp), "+l"(pm));      // one address each, then += W per row
                                const bool hp = dq.z >= 0 && l8 < wlim, hm = dq.w >= 0 && l8 < wlim;
                                TNO_CHECK(dq.z < 2 * NB && dq.w < 2 * NB && (dq.z >= 0 || dq.w >= 0));
                                TNO_CHECK(__ldg(a.batch_q + b) - a.q0 + max(dq.z, dq.w) < a.piece_stride / ((int64_t)H * W));
#ifdef TNO_DEBUG_CHECKS
                                for (int r = 0; r < R; ++r) {
                                    // every address a predicated-on reduction touches lies in this tile row's piece
                                    const float *lo = a.pieces + (int64_t)(ty % a.n_pieces) * a.piece_stride;
                                    if (hp && (uint32_t)(yp + r) < (uint32_t)H)
                                        TNO_CHECK(pp + (int64_t)r * W >= lo && pp + (int64_t)r * W + 1 < lo + a.piece_stride);
                                    if (hm && (uint32_t)(ym + r) < (uint32_t)H)
                                        TNO_CHECK(pm + (int64_t)r * W >= lo && pm + (int64_t)r * W + 1 < lo + a.piece_stride);
                                }
#endif
#pragma unroll
                                for (int r = 0; r < R; ++r, pp += W, pm += W) {
                                    // the piece addresses are owned by this CTA, and f_done orders the adds
                                    // of successive flushes; rows outside the frame are predicated off
                                    const float2 e = accE[s][r], o = accO[s][r];
                                    red_add_v2_if(hp && (uint32_t)(yp + r) < (uint32_t)H, pp,
                                                  make_float2(e.x + o.x, e.y + o.y));
                                    red_add_v2_if(hm && (uint32_t)(ym + r) < (uint32_t)H, pm,
                                                  make_float2(e.x - o.x, e.y - o.y));
                                    accE[s][r] = accO[s][r] = make_float2(0.f, 0.f);
                                }
                            }
                            __syncwarp();
                            mbar_arrive_one(f_done + 8 * (s));
                        }
                    }
                }
                ++n;
            }
        }
    }
}

// ------------------------------------------------------------------------------------ finishing kernel
// One block per (64 x 64 tile, entry q of the chunk): SNR = (sum of the pieces) * D^(-1/2), map
// store, candidates >= threshold into the tile's slot (BASELINE.json:north_star a4, a5).
__global__ void __launch_bounds__(256)
k_finish(const float *__restrict__ pieces, const float *__restrict__ dpieces, int32_t n_pieces, int64_t piece_stride,
         const int32_t *__restrict__ perm, int32_t q0, const TrajInfo *__restrict__ traj,
         const float *__restrict__ rsd, int32_t H, int32_t W, int32_t fy0, float *__restrict__ out_snr,
         unsigned long long *__restrict__ maxkeys, TopkSlots slots) {
    __shared__ uint64_t list[kCollectTile * kCollectTile];
    __shared__ int32_t count;
    const int32_t tid = threadIdx.x, lane = tid & 31;
    const int32_t ql = blockIdx.z, k = perm[q0 + ql];
    const int32_t x0 = blockIdx.x * kCollectTile, y0 = (fy0 + blockIdx.y) * kCollectTile;
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
            if (n_pieces <= 4) {
                // the usual case: all loads in flight together, summed in piece order (a missing piece adds +0)
                float4 p[4];
#pragma unroll
                for (int32_t c = 0; c < 4; ++c)
                    p[c] = c < n_pieces ? __ldcs(reinterpret_cast<const float4 *>(pin + c * piece_stride + off))
                                        : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                for (int32_t c = 0; c < 4; ++c) { v.x += p[c].x; v.y += p[c].y; v.z += p[c].z; v.w += p[c].w; }
            } else {
                for (int32_t c = 0; c < n_pieces; ++c) {
                    const float4 p = __ldcs(reinterpret_cast<const float4 *>(pin + c * piece_stride + off));
                    v.x += p.x; v.y += p.y; v.z += p.z; v.w += p.w;
                }
            }
            if (dpieces) {
                // masked search: D was accumulated like N, from the validity weights
                float4 dsum = make_float4(0.f, 0.f, 0.f, 0.f);
                const float *din = dpieces + (int64_t)ql * H * W;
                for (int32_t c = 0; c < n_pieces; ++c) {
                    const float4 p = __ldcs(reinterpret_cast<const float4 *>(din + c * piece_stride + off));
                    dsum.x += p.x; dsum.y += p.y; dsum.z += p.z; dsum.w += p.w;
                }
                v.x = dsum.x > 0.f ? v.x / sqrtf(dsum.x) : 0.f;
                v.y = dsum.y > 0.f ? v.y / sqrtf(dsum.y) : 0.f;
                v.z = dsum.z > 0.f ? v.z / sqrtf(dsum.z) : 0.f;
                v.w = dsum.w > 0.f ? v.w / sqrtf(dsum.w) : 0.f;
            } else if (interior) {
                v.x *= rs_in; v.y *= rs_in; v.z *= rs_in; v.w *= rs_in;
            } else {
                const float *rr = rs + (int64_t)border_class(y, ti.by, H) * ti.bx.n;
                v.x *= __ldg(rr + border_class(x, ti.bx, W));
                v.y *= __ldg(rr + border_class(x + 1, ti.bx, W));
                v.z *= __ldg(rr + border_class(x + 2, ti.bx, W));
                v.w *= __ldg(rr + border_class(x + 3, ti.bx, W));
            }
            if (om) *reinterpret_cast<float4 *>(om + off) = v;
            if (maxkeys) {
                // fused max over the bank: key = (score, ~k), so the maximum of the keys is
                // the largest score and, of equal scores, the smallest k -- order independent, hence exact
                atomicMax(maxkeys + off, make_key(v.x, (uint32_t)k));
                atomicMax(maxkeys + off + 1, make_key(v.y, (uint32_t)k));
                atomicMax(maxkeys + off + 2, make_key(v.z, (uint32_t)k));
                atomicMax(maxkeys + off + 3, make_key(v.w, (uint32_t)k));
            }
        }
        // (one vote per warp and row group: most groups hold no candidate, and the four ballots below are skipped)
        if (want_topk &&
            __any_sync(0xffffffffu, in && fmaxf(fmaxf(v.x, v.y), fmaxf(v.z, v.w)) >= slots.threshold)) {
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
        const int64_t tile = (int64_t)(fy0 + blockIdx.y) * gridDim.x + blockIdx.x;
        tile_flush<256>(list, count, slots, tile, k, tid);
    }
}

// ------------------------------------------------------------------------------------ host side
// (rows per thread, slots per batch, consumer warps, box stages, X buffers): tiles of CW x R positions x 64
// columns.  A slot costs 4 R accumulator registers (E and O, two columns), the window and its sums and
// differences 2 (R + 4) + 8 R.
using V0 = SepCfg<4, 5, 12, 4, 8>;            // tiles of 48 positions, 5 slots: banks with 5 slots per x-motion (config 3)
using V1 = SepCfg<5, 4, 12, 4, 8, 56>;        // tiles of 60 positions, 4 slots: the per-frame bookkeeping of a warp is
                                              // spread over 5 positions instead of 4 (config 4: 8 x 8 grid = 4 slots)
// (measured alternatives: 8 consumer warps x 6 rows is 4-10 % slower on every config)

int32_t sep_num_variants() { return 2; }
SepVariant sep_variant(int32_t v) {
    return v == 0 ? SepVariant{V0::NB, V0::HT, V0::R} : SepVariant{V1::NB, V1::HT, V1::R};
}
int32_t sep_table_words(int32_t v) { return v == 0 ? V0::TABW : V1::TABW; }
int32_t sep_tile_rows(int32_t v, int32_t H) {
    const int32_t ht = sep_variant(v).tile_h;
    return (H + 4 + ht - 1) / ht;
}

void launch_sep_tables(cudaStream_t st, int32_t v, const ClassTables &tab, const int32_t *batch_xc,
                       const int32_t *slot_yc, const int32_t *slot_flip, const int32_t *slot_q, int32_t n_batches,
                       int32_t squared, float *stage_tab) {
    const int64_t n = (int64_t)n_batches * tab.T;
    const unsigned grid = (unsigned)((n + 127) / 128);
    if (v == 0)
        k_sep_tables<V0><<<grid, 128, 0, st>>>(tab, batch_xc, slot_yc, slot_flip, slot_q, n_batches, squared, stage_tab);
    else
        k_sep_tables<V1><<<grid, 128, 0, st>>>(tab, batch_xc, slot_yc, slot_flip, slot_q, n_batches, squared, stage_tab);
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
    const int32_t ntx = (a.W + kTileW - 1) / kTileW, nty_all = (a.H + 4 + C::HT - 1) / C::HT;
    const int32_t nty = (a.ty1 > 0 ? std::min(a.ty1, nty_all) : nty_all) - a.ty0;     // tile rows of this launch
    if (a.ty0 < 0 || nty < 1) {
        *err = "empty tile-row range";
        return -1;
    }
    const int64_t n_items = (int64_t)ntx * nty * a.n_batches;
    if (n_items >= ((int64_t)1 << 31) || (n_items / a.n_sm + 1) * a.T >= ((int64_t)1 << 31)) {
        *err = "too many (tile, batch, frame) steps";
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

void launch_finish(cudaStream_t st, const float *pieces, const float *dpieces, int32_t n_pieces, int64_t piece_stride,
                   const int32_t *perm, int32_t q0, int32_t q_count, const TrajInfo *traj, const float *rsd,
                   int32_t H, int32_t W, int32_t fy0, int32_t fy1, float *out_snr, uint64_t *maxkeys,
                   const TopkSlots &slots) {
    if (fy1 <= fy0 || q_count <= 0) return;      // nothing left to finish (the banded host search may be done early)
    dim3 grid((unsigned)((W + kCollectTile - 1) / kCollectTile), (unsigned)(fy1 - fy0), (unsigned)q_count);
    k_finish<<<grid, 256, 0, st>>>(pieces, dpieces, n_pieces, piece_stride, perm, q0, traj, rsd, H, W, fy0, out_snr,
                                   reinterpret_cast<unsigned long long *>(maxkeys), slots);
}

}  // namespace tno
