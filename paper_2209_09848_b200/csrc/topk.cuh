// Candidate selection primitives (BASELINE.json:north_star "(d) warp-shuffle top-K";
// PAPER.md:L122 "we take all scores above a threshold as potential candidates").
// Candidates are 64-bit keys (common.cuh); "better" = larger key.
#pragma once
#include "common.cuh"

namespace tno {

// Warp-aggregated append: one shared-memory atomic per warp, positions handed out by ballot +
// shuffle.  Must be called by all 32 lanes of a warp.
__device__ __forceinline__ void warp_push(bool pred, uint64_t key, uint64_t *list, int32_t *count,
                                          int32_t lane) {
    const unsigned m = __ballot_sync(0xffffffffu, pred);
    if (m == 0u) return;
    const int32_t leader = __ffs(m) - 1;
    int32_t base = 0;
    if (lane == leader) base = atomicAdd(count, __popc(m));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (pred) list[base + __popc(m & ((1u << lane) - 1u))] = key;
}

// Block-wide bitonic sort, descending, of n keys in shared memory (n a power of two >= 32,
// NT a multiple of 32).  Strides below 32 are done in registers with warp shuffles; larger
// strides through shared memory.  Ends with a __syncthreads().
template <int NT>
__device__ void block_sort_desc(uint64_t *keys, int32_t n, int32_t tid) {
    for (int32_t k = 2; k <= n; k <<= 1) {
        int32_t j = k >> 1;
        for (; j >= 32; j >>= 1) {
            for (int32_t i = tid; i < n; i += NT) {
                const int32_t p = i ^ j;
                if (p > i) {
                    const uint64_t a = keys[i], b = keys[p];
                    const bool desc = (i & k) == 0;
                    if ((a < b) == desc) { keys[i] = b; keys[p] = a; }
                }
            }
            __syncthreads();
        }
        for (int32_t base = 0; base < n; base += NT) {
            const int32_t i = base + tid;
            if (i < n) {                       // uniform per warp: n and NT are multiples of 32
                uint64_t v = keys[i];
                const bool desc = (i & k) == 0;
                for (int32_t jj = j; jj > 0; jj >>= 1) {
                    const uint64_t o = __shfl_xor_sync(0xffffffffu, v, jj);
                    const bool lower = (i & jj) == 0;
                    const bool want_max = (lower == desc);
                    v = want_max ? (v > o ? v : o) : (v < o ? v : o);
                }
                keys[i] = v;
            }
        }
        __syncthreads();
    }
}

// Write one tile's candidates (list[0..n), unordered) to its slot, keeping the ktop best when
// there are more.  `list` must have room for the next power of two >= max(n, 32).  Block-uniform
// arguments; all NT threads call.  Ends with a __syncthreads().
template <int NT>
__device__ void tile_flush(uint64_t *list, int32_t n, const TopkSlots &slots, int64_t tile,
                           int32_t k, int32_t tid) {
    const int32_t ktop = slots.ktop;
    if (n > ktop) {
        int32_t np2 = 32;
        while (np2 < n) np2 <<= 1;
        for (int32_t i = n + tid; i < np2; i += NT) list[i] = 0ull;
        __syncthreads();
        block_sort_desc<NT>(list, np2, tid);
        n = ktop;
    }
    uint64_t *dst = slots.keys + (tile * slots.K + k) * (int64_t)ktop;
    for (int32_t i = tid; i < n; i += NT) dst[i] = list[i];
    if (tid == 0) slots.counts[tile * slots.K + k] = n;
    __syncthreads();
}

}  // namespace tno
