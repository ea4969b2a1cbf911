// tno_mf_debug_poison_shared: fills the shared memory of every SM with a bit pattern (tests: 0xffffffff, a NaN when
// read as a float).  Shared memory is not cleared between kernels, so a kernel that reads a word of it that it never
// wrote -- even to multiply it by a zero weight -- computes with whatever an earlier kernel left there.
// compute-sanitizer's initcheck would find that; it is closed on this pool (profiles/r2_sanitizers.md), so the GPU
// tests call this before every test instead (tests/conftest.py): such a read then meets a NaN instead of, usually,
// a harmless finite number.
#include "kernels.h"

namespace tno {
namespace {

__global__ void __launch_bounds__(256)
k_poison_shared(uint32_t pattern, uint32_t words, uint32_t *sink) {
    extern __shared__ uint32_t sm[];
    for (uint32_t i = threadIdx.x; i < words; i += blockDim.x) sm[i] = pattern;
    __syncthreads();
    // (a read that depends on run-time data keeps the stores from being optimised away)
    if (sink && sm[(threadIdx.x * 2654435761u) % words] != pattern) sink[0] = 1u;
}

}  // namespace
}  // namespace tno

using namespace tno;

extern "C" int tno_mf_debug_poison_shared(tno_mf_ctx *ctx, uint32_t pattern) {
    if (!ctx) return TNO_MF_EINVAL;
    const CtxView v = ctx_view(ctx);
    cudaError_t e = cudaSetDevice(v.device);
    int n_sm = 0, max_smem = 0;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, v.device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, v.device);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_poison_shared, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return ctx_fail(ctx, TNO_MF_ECUDA, cudaGetErrorString(e));
    }
    // one block per SM at a time (it takes all the shared memory), a few waves to reach every SM; then the same with
    // blocks of a quarter, an eighth and a sixteenth of it, several per SM: the shared-memory carve-out of an SM
    // follows the kernel that runs on it, and what a later kernel finds is what was written under a similar split
    int32_t launches = 0;
    for (int div = 1; div <= 16; div = div == 1 ? 4 : div * 2) {
        const uint32_t bytes = ((uint32_t)max_smem / (uint32_t)div) & ~15u;
        k_poison_shared<<<(unsigned)(4 * div * n_sm), 256, bytes, v.stream>>>(pattern, bytes / 4u, nullptr);
        ++launches;
    }
    ctx_set_launches(ctx, launches);
    e = cudaGetLastError();
    if (e != cudaSuccess) return ctx_fail(ctx, TNO_MF_ECUDA, cudaGetErrorString(e));
    return TNO_MF_OK;
}
