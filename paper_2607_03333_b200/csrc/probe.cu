// libspork: a read-only HBM stream (bench support).  The attention kernels are almost pure READ streams;
// MEASURED_PEAKS.json's figure is a copy (read + write).  bench.py times this kernel beside them so that
// the roofline line can also say how far a kernel is from what a plain read of the same bytes reaches.
// It streams the way the attention kernel does: persistent CTAs (2 per SM), one thread per CTA keeping a
// ring of 16 KiB bulk copies (cp.async.bulk global -> shared, mbarrier completion) in flight; nothing is
// done with the data.
#include "spork_internal.h"
#include "umma.cuh"

using namespace spork::ptx;

namespace {

constexpr int PROBE_SLOT = 16384, PROBE_NSLOT = 6;

__global__ void __launch_bounds__(32, 2) read_probe_kernel(const uint8_t *__restrict__ p, size_t n_chunks) {
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t base = smem_u32(smem), bars = base + PROBE_NSLOT * PROBE_SLOT;
    if (threadIdx.x == 0) {
        for (int s = 0; s < PROBE_NSLOT; ++s) mbar_init(bars + 8 * s, 1);
        mbar_fence_init();
    }
    __syncwarp();
    if (threadIdx.x != 0) return;
    // chunk c of this CTA = global chunk blockIdx.x + c * gridDim.x
    const size_t mine = n_chunks > blockIdx.x ? (n_chunks - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    size_t issued = 0, done = 0;
    for (; issued < mine && issued < (size_t)PROBE_NSLOT; ++issued) {
        mbar_expect_tx(bars + 8 * (uint32_t)issued, PROBE_SLOT);
        bulk_g2s(base + (uint32_t)issued * PROBE_SLOT, p + (blockIdx.x + issued * gridDim.x) * (size_t)PROBE_SLOT, PROBE_SLOT,
                 bars + 8 * (uint32_t)issued);
    }
    for (; done < mine; ++done) {
        const uint32_t s = (uint32_t)(done % PROBE_NSLOT);
        mbar_wait(bars + 8 * s, (uint32_t)(done / PROBE_NSLOT) & 1);
        if (issued < mine) {
            mbar_expect_tx(bars + 8 * s, PROBE_SLOT);
            bulk_g2s(base + s * PROBE_SLOT, p + (blockIdx.x + issued * gridDim.x) * (size_t)PROBE_SLOT, PROBE_SLOT, bars + 8 * s);
            ++issued;
        }
    }
}

}  // namespace

extern "C" int spork_hbm_read_probe(spork_ctx *c, const void *buf, size_t bytes, void *stream) {
    if (!c || !buf || ((uintptr_t)buf & 15) || bytes < (size_t)PROBE_SLOT) return SPORK_ERR_INVALID;
    constexpr int SMEM = PROBE_NSLOT * PROBE_SLOT + 64;
    if (!(c->smem_attr_done & 16u)) {
        SPORK_CUDA(cudaFuncSetAttribute(read_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM));
        c->smem_attr_done |= 16u;
    }
    read_probe_kernel<<<c->num_sms * 2, 32, SMEM, (cudaStream_t)stream>>>((const uint8_t *)buf, bytes / PROBE_SLOT);
    SPORK_CUDA(cudaGetLastError());
    return SPORK_OK;
}
