// Candidate pipeline kernels: tile collection from a stored map, and the per-trajectory merge.
#include "kernels.h"
#include "topk.cuh"

namespace tno {

// One block per (64 x 64 tile, trajectory): threshold the map tile, append with warp_push, keep
// the tile's ktop best.
__global__ void __launch_bounds__(256)
k_collect_from_map(const float *__restrict__ maps, int32_t H, int32_t W, int32_t k_first,
                   TopkSlots slots) {
    __shared__ uint64_t list[kCollectTile * kCollectTile];
    __shared__ int32_t count;
    const int32_t tid = threadIdx.x, lane = tid & 31;
    const int32_t kl = blockIdx.z, k = k_first + kl;
    const int32_t x0 = blockIdx.x * kCollectTile, y0 = blockIdx.y * kCollectTile;
    if (tid == 0) count = 0;
    __syncthreads();
    const float *m = maps + (int64_t)kl * H * W;
    for (int32_t i = tid; i < kCollectTile * kCollectTile; i += 256) {
        const int32_t x = x0 + (i & (kCollectTile - 1)), y = y0 + i / kCollectTile;
        bool pred = false;
        float s = 0.0f;
        if (x < W && y < H) {
            s = m[(int64_t)y * W + x];
            pred = s >= slots.threshold;
        }
        warp_push(pred, make_key(s, (uint32_t)(y * W + x)), list, &count, lane);
    }
    __syncthreads();
    const int64_t tile = (int64_t)blockIdx.y * gridDim.x + blockIdx.x;
    tile_flush<256>(list, count, slots, tile, k, tid);
}

// One block per trajectory: exact selection of the ktop largest keys among the candidates of all
// tile slots (keys are unique: the pixel index is part of the key), then one small sort.
//   1. N = sum of the tile counts; if N <= ktop every candidate is selected;
//   2. else a most-significant-digit radix select (13-bit digits, shared-memory histogram) finds
//      the ktop-th largest key; each pass reads the candidates (L2 resident) once;
//   3. the selected keys are gathered into shared memory, sorted (bitonic, shuffles for strides
//      < 32) and written as records.
constexpr int kMergeThreads = 512;
constexpr int kDigitBits = 13, kBins = 1 << kDigitBits;

__global__ void __launch_bounds__(kMergeThreads)
k_topk_merge(TopkSlots slots, int32_t n_tiles, int32_t W, int32_t P, tno_mf_cand *__restrict__ out) {
    extern __shared__ uint64_t buf[];          // [0, P) selected keys
    __shared__ uint32_t hist[kBins];
    __shared__ uint32_t wsum[kMergeThreads / 32];
    __shared__ uint32_t sel_bin, sel_before, total, fill;
    const int32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, k = blockIdx.x, ktop = slots.ktop;
    constexpr int NWARP = kMergeThreads / 32;

    // visit every candidate key of trajectory k: warp per tile, lanes over the slot entries
    auto for_each_key = [&](auto &&fn) {
        for (int32_t tile = warp; tile < n_tiles; tile += NWARP) {
            const int32_t c = slots.counts[(int64_t)tile * slots.K + k];
            const uint64_t *src = slots.keys + ((int64_t)tile * slots.K + k) * (int64_t)ktop;
            for (int32_t r = lane; r < c; r += 32) fn(src[r]);
        }
    };

    if (tid == 0) { total = 0; fill = 0; }
    for (int32_t i = tid; i < P; i += kMergeThreads) buf[i] = 0ull;
    __syncthreads();
    {
        uint32_t n = 0;
        for (int32_t tile = tid; tile < n_tiles; tile += kMergeThreads) n += (uint32_t)slots.counts[(int64_t)tile * slots.K + k];
        for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xffffffffu, n, o);
        if (lane == 0 && n) atomicAdd(&total, n);
    }
    __syncthreads();
    const uint32_t N = total;
    uint64_t kth = 0ull;                       // select keys >= kth
    if (N > (uint32_t)ktop) {
        uint64_t prefix = 0ull;                // value of the digits fixed so far (high bits of kth)
        uint32_t remaining = (uint32_t)ktop;   // rank of the wanted key among the keys matching prefix
        int32_t shift = 64;
        while (shift > 0) {
            const int32_t bits = shift >= kDigitBits ? kDigitBits : shift;
            const int32_t lo = shift - bits;   // digit = (key >> lo) & (2^bits - 1)
            const int32_t nb = 1 << bits;
            for (int32_t i = tid; i < nb; i += kMergeThreads) hist[i] = 0u;
            __syncthreads();
            for_each_key([&](uint64_t key) {
                const bool match = (shift == 64) || ((key >> shift) == (prefix >> shift));
                if (match) atomicAdd(&hist[(uint32_t)(key >> lo) & (uint32_t)(nb - 1)], 1u);
            });
            __syncthreads();
            // find, from the top bin down, the bin in which the cumulative count reaches `remaining`
            const int32_t per = nb / kMergeThreads;                 // bins per thread (>= 1: nb >= 512)
            uint32_t local = 0;
            for (int32_t j = 0; j < per; ++j) local += hist[nb - 1 - (tid * per + j)];
            uint32_t incl = local;
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += v;
            }
            if (lane == 31) wsum[warp] = incl;
            __syncthreads();
            uint32_t before = incl - local;
            for (int32_t w = 0; w < warp; ++w) before += wsum[w];
            if (before < remaining && remaining <= before + local) {
                uint32_t acc = before;
                for (int32_t j = 0; j < per; ++j) {
                    const int32_t bin = nb - 1 - (tid * per + j);
                    if (remaining <= acc + hist[bin]) { sel_bin = (uint32_t)bin; sel_before = acc; break; }
                    acc += hist[bin];
                }
            }
            __syncthreads();
            prefix |= (uint64_t)sel_bin << lo;
            remaining -= sel_before;
            const uint32_t in_bin = hist[sel_bin];
            shift = lo;
            __syncthreads();
            if (in_bin == remaining) break;    // every key with this prefix is selected
        }
        kth = prefix;                          // digits below `shift` are zero: keys >= kth are exactly the ktop best
    }
    for_each_key([&](uint64_t key) {
        if (key >= kth) buf[atomicAdd(&fill, 1u)] = key;
    });
    __syncthreads();
    block_sort_desc<kMergeThreads>(buf, P, tid);
    for (int32_t i = tid; i < ktop; i += kMergeThreads) {
        const uint64_t key = buf[i];
        tno_mf_cand c;
        if (key != 0ull) {
            const uint32_t idx = ~(uint32_t)key;
            c.snr = ord_to_snr((uint32_t)(key >> 32));
            c.x = (int32_t)(idx % (uint32_t)W);
            c.y = (int32_t)(idx / (uint32_t)W);
        } else {
            c.snr = -INFINITY; c.x = -1; c.y = -1;
        }
        c.k = k;
        out[(int64_t)k * ktop + i] = c;
    }
}

void launch_collect_from_map(cudaStream_t st, const float *maps, int32_t H, int32_t W,
                             int32_t k_first, int32_t k_count, const TopkSlots &slots) {
    dim3 grid((unsigned)((W + kCollectTile - 1) / kCollectTile),
              (unsigned)((H + kCollectTile - 1) / kCollectTile), (unsigned)k_count);
    k_collect_from_map<<<grid, 256, 0, st>>>(maps, H, W, k_first, slots);
}

void launch_topk_merge(cudaStream_t st, const TopkSlots &slots, int32_t n_tiles, int32_t W,
                       tno_mf_cand *out_topk) {
    int32_t P = 32;
    while (P < slots.ktop) P <<= 1;
    const size_t smem = (size_t)P * sizeof(uint64_t);
    k_topk_merge<<<(unsigned)slots.K, kMergeThreads, smem, st>>>(slots, n_tiles, W, P, out_topk);
}

}  // namespace tno
