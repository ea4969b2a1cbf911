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

// One block per trajectory: stream all tile slots through a sorted buffer of the P best.
__global__ void __launch_bounds__(256)
k_topk_merge(TopkSlots slots, int32_t n_tiles, int32_t W, int32_t P, tno_mf_cand *__restrict__ out) {
    extern __shared__ uint64_t buf[];          // [0, P) best so far (sorted), [P, 2P) incoming
    const int32_t tid = threadIdx.x, k = blockIdx.x, ktop = slots.ktop;
    for (int32_t i = tid; i < P; i += 256) buf[i] = 0ull;
    const int32_t G = P / ktop;                // tiles per round
    for (int32_t tile0 = 0; tile0 < n_tiles; tile0 += G) {
        int32_t any = 0;
        for (int32_t i = tid; i < P; i += 256) {
            const int32_t g = i / ktop, r = i - g * ktop;
            const int64_t tile = (int64_t)tile0 + g;
            uint64_t v = 0ull;
            if (g < G && tile < n_tiles && r < slots.counts[tile * slots.K + k])
                v = slots.keys[(tile * slots.K + k) * (int64_t)ktop + r];
            buf[P + i] = v;
            any |= (v != 0ull);
        }
        if (__syncthreads_or(any)) block_sort_desc<256>(buf, 2 * P, tid);
    }
    __syncthreads();
    for (int32_t i = tid; i < ktop; i += 256) {
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
    int32_t P = 512;
    while (P < slots.ktop) P <<= 1;
    const size_t smem = (size_t)2 * P * sizeof(uint64_t);
    k_topk_merge<<<(unsigned)slots.K, 256, smem, st>>>(slots, n_tiles, W, P, out_topk);
}

}  // namespace tno
