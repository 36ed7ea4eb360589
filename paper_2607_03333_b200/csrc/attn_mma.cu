// libspork: the bandwidth path -- bf16 KV, D = 128, page = 16 tokens.
//
// One persistent CTA = 4 consumer warps + 1 producer warp, 2 CTAs per SM.
// The producer walks the block table and stages each (page, kv head) block of
// K and of V (4 KiB each, already in its 128-byte-swizzled shared-memory
// image) with ONE cp.async.bulk per block into a 3-stage ring of 64-token
// tiles, signalled through mbarriers.  Consumers hold the Q rows of the item
// as mma A fragments and run S = Q K^T, an online softmax in the exp2 domain
// and O += P V on the tensor cores (mma.sync m16n8k16 bf16, fp32 accumulate):
// the GQA heads of every member of a fork group are packed as rows against
// one stream of shared-prefix K/V, so a prefix page is read from HBM once per
// group.  Warps split an item as (row tiles of 16) x (token parts of a tile);
// token parts are combined through shared memory, and every item writes one
// normalised partial (o, lse) per row for the merge kernel.
#include <math.h>

#include "spork_internal.h"
#include "umma.cuh"      // mbarrier / bulk-copy / ex2 / pack wrappers shared with the tcgen05 kernel

using namespace spork;
using namespace spork::ptx;

namespace {

constexpr int D = 128;
constexpr int NSTAGE = 3;
constexpr int TILE_PAGES = 4;
constexpr int TILE_TOKENS = TILE_PAGES * PS;       // 64
constexpr int HEAD_BLOCK = PS * D * 2;             // 4096 B
constexpr int STAGE_BYTES = 2 * TILE_PAGES * HEAD_BLOCK;  // K then V: 32 KiB
constexpr int N_CONSUMER_WARPS = 4;
constexpr int N_THREADS = (N_CONSUMER_WARPS + 1) * 32;
constexpr int COMB_REC_BYTES = 64 * 32 * 4 + 8 * 4 * 4;   // O[64][32 lanes] + (m0,m1,l0,l1) per quad
constexpr int SMEM_BYTES = NSTAGE * STAGE_BYTES + 2 * COMB_REC_BYTES + 2 * NSTAGE * 8 + 128;
constexpr int CTAS_PER_SM = 2;
constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;

__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
        "{%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void consumer_bar() {   // the 4 consumer warps only
    asm volatile("bar.sync 1, %0;" ::"n"(N_CONSUMER_WARPS * 32) : "memory");
}

struct Params {
    const WorkItem *items;
    const int32_t *cta_ptr;       // this CTA runs items [cta_ptr[b], cta_ptr[b + 1])
    const int32_t *seq_len;       // device lengths: open-ended items end there
    const int32_t *rowmap;
    const uint16_t *q;
    const uint8_t *k_pool, *v_pool;
    const int32_t *table;
    int table_stride, Hq, Hkv, G;
    float scale_log2;     // scale * log2(e)
    float *ws_o, *ws_lse;
};

// Per-warp state for one item: 16 rows x 128 dims of O (fp32 C fragments),
// running max (raw scores * scale_log2) and the per-thread part of the row sums.
struct RowState {
    float o[16][4];
    float m[2], l[2];
};

// NT n-tiles of 8 tokens (NT = 2: one page, NT = 4: two pages), starting at
// page slot `pg0` of the stage.  `t_base` = global token index of the first token.
template <int NT>
__device__ __forceinline__ void process_block(RowState &st, const uint32_t (&qa)[8][4], uint32_t k_base,
                                              uint32_t v_base, int pg0, int lane, float scale_log2,
                                              bool need_mask, int t_base, int tok_end, int lim_r0,
                                              int lim_r1, int valid_pages /* pages with data, from pg0 */) {
    constexpr int NP = NT / 2;
    float s[NT][4];
#pragma unroll
    for (int j = 0; j < NT; ++j) s[j][0] = s[j][1] = s[j][2] = s[j][3] = 0.f;
    const int mi = lane >> 3, r8 = lane & 7;
    // ---- S = Q K^T ------------------------------------------------------------
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        // token row inside the page = 8 * (mi >> 1) + r8: row group (mi >> 1), row r8 of the atom
        const uint32_t pbase = k_base + (pg0 + p) * HEAD_BLOCK + ((mi >> 1) << 11) + r8 * 128;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
            const int c = 2 * ks + (mi & 1);                    // 16-byte chunk 0..15
            const uint32_t addr = pbase + ((c >> 3) << 10) + (((c & 7) ^ r8) << 4);
            uint32_t b0, b1, b2, b3;
            ldsm_x4(addr, b0, b1, b2, b3);
            mma_bf16(s[2 * p], qa[ks], b0, b1);
            mma_bf16(s[2 * p + 1], qa[ks], b2, b3);
        }
    }
    // ---- mask + row max -------------------------------------------------------
    const int tq = (lane & 3) * 2;
    float mx0 = -INFINITY, mx1 = -INFINITY;
#pragma unroll
    for (int j = 0; j < NT; ++j) {
        if (need_mask) {
            const int t = t_base + 8 * j + tq;
            if (t >= tok_end || t > lim_r0) s[j][0] = -INFINITY;
            if (t + 1 >= tok_end || t + 1 > lim_r0) s[j][1] = -INFINITY;
            if (t >= tok_end || t > lim_r1) s[j][2] = -INFINITY;
            if (t + 1 >= tok_end || t + 1 > lim_r1) s[j][3] = -INFINITY;
        }
        mx0 = fmaxf(mx0, fmaxf(s[j][0], s[j][1]));
        mx1 = fmaxf(mx1, fmaxf(s[j][2], s[j][3]));
    }
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 1));
    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, 2));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 1));
    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, 2));
    const float mn0 = fmaxf(st.m[0], mx0 * scale_log2), mn1 = fmaxf(st.m[1], mx1 * scale_log2);
    const float mu0 = mn0 == -INFINITY ? 0.f : mn0, mu1 = mn1 == -INFINITY ? 0.f : mn1;
    const float a0 = ex2(st.m[0] - mu0), a1 = ex2(st.m[1] - mu1);
    st.m[0] = mn0;
    st.m[1] = mn1;
    // ---- P = exp2(S * c - m), row sums, bf16 A fragments --------------------------
    uint32_t pa[NP][4];
    float sum0 = 0.f, sum1 = 0.f;
#pragma unroll
    for (int j = 0; j < NT; ++j) {
        const float p0 = ex2(fmaf(s[j][0], scale_log2, -mu0));
        const float p1 = ex2(fmaf(s[j][1], scale_log2, -mu0));
        const float p2 = ex2(fmaf(s[j][2], scale_log2, -mu1));
        const float p3 = ex2(fmaf(s[j][3], scale_log2, -mu1));
        sum0 += p0 + p1;
        sum1 += p2 + p3;
        pa[j >> 1][(j & 1) * 2 + 0] = pack_bf16(p0, p1);
        pa[j >> 1][(j & 1) * 2 + 1] = pack_bf16(p2, p3);
    }
    st.l[0] = st.l[0] * a0 + sum0;
    st.l[1] = st.l[1] * a1 + sum1;
#pragma unroll
    for (int n = 0; n < 16; ++n) {
        st.o[n][0] *= a0; st.o[n][1] *= a0;
        st.o[n][2] *= a1; st.o[n][3] *= a1;
    }
    // ---- O += P V (skip pages that were not staged: stale smem may hold anything) -----
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        if (p < valid_pages) {
            const uint32_t pbase = v_base + (pg0 + p) * HEAD_BLOCK + ((mi & 1) << 11) + r8 * 128;
#pragma unroll
            for (int cp = 0; cp < 8; ++cp) {
                const int c = 2 * cp + (mi >> 1);
                const uint32_t addr = pbase + ((c >> 3) << 10) + (((c & 7) ^ r8) << 4);
                uint32_t b0, b1, b2, b3;
                ldsm_x4_t(addr, b0, b1, b2, b3);
                mma_bf16(st.o[2 * cp], pa[p], b0, b1);
                mma_bf16(st.o[2 * cp + 1], pa[p], b2, b3);
            }
        }
    }
}

// merge the record at `rec` (written by another warp, same lane layout) into st
__device__ __forceinline__ void comb_merge(RowState &st, const float *rec, int lane) {
    const float *ml = rec + 64 * 32 + (lane >> 2) * 4;
    const float mb0 = ml[0], mb1 = ml[1], lb0 = ml[2], lb1 = ml[3];
    const float M0 = fmaxf(st.m[0], mb0), M1 = fmaxf(st.m[1], mb1);
    const float u0 = M0 == -INFINITY ? 0.f : M0, u1 = M1 == -INFINITY ? 0.f : M1;
    const float fa0 = ex2(st.m[0] - u0), fb0 = ex2(mb0 - u0);
    const float fa1 = ex2(st.m[1] - u1), fb1 = ex2(mb1 - u1);
#pragma unroll
    for (int n = 0; n < 16; ++n) {
        st.o[n][0] = st.o[n][0] * fa0 + rec[(n * 4 + 0) * 32 + lane] * fb0;
        st.o[n][1] = st.o[n][1] * fa0 + rec[(n * 4 + 1) * 32 + lane] * fb0;
        st.o[n][2] = st.o[n][2] * fa1 + rec[(n * 4 + 2) * 32 + lane] * fb1;
        st.o[n][3] = st.o[n][3] * fa1 + rec[(n * 4 + 3) * 32 + lane] * fb1;
    }
    st.l[0] = st.l[0] * fa0 + lb0 * fb0;
    st.l[1] = st.l[1] * fa1 + lb1 * fb1;
    st.m[0] = M0;
    st.m[1] = M1;
}
__device__ __forceinline__ void comb_store(const RowState &st, float *rec, int lane) {
#pragma unroll
    for (int n = 0; n < 16; ++n)
#pragma unroll
        for (int e = 0; e < 4; ++e) rec[(n * 4 + e) * 32 + lane] = st.o[n][e];
    if ((lane & 3) == 0) {
        float *ml = rec + 64 * 32 + (lane >> 2) * 4;
        ml[0] = st.m[0]; ml[1] = st.m[1]; ml[2] = st.l[0]; ml[3] = st.l[1];
    }
}

__global__ void __launch_bounds__(N_THREADS, CTAS_PER_SM) attn_mma_kernel(const Params P) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 127) & ~(uintptr_t)127);
    const uint32_t stage_base = smem_u32(smem);
    float *comb = (float *)(smem + NSTAGE * STAGE_BYTES);
    const uint32_t bar_base = stage_base + NSTAGE * STAGE_BYTES + 2 * COMB_REC_BYTES;
    // full[s] at bar_base + 8 s, empty[s] at bar_base + 8 (NSTAGE + s)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(bar_base + 8 * s, 1);
            mbar_init(bar_base + 8 * (NSTAGE + s), N_CONSUMER_WARPS);
        }
        mbar_fence_init();
    }
    __syncthreads();

    // let the merge kernel's blocks become resident now; they wait for this grid to finish
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    uint32_t stage = 0, phase = 0;   // ring position, carried across items by both roles
    const int item_begin = P.cta_ptr[blockIdx.x], item_end = P.cta_ptr[blockIdx.x + 1];

    if (warp == N_CONSUMER_WARPS) {
        // ============================ producer ============================
        for (int idx = item_begin; idx < item_end; ++idx) {
            const WorkItem it = load_item(P.items, idx, P.seq_len);
            const int page0 = it.tok0 / PS;
            const int n_pages = (it.tok1 + PS - 1) / PS - page0;
            const int n_tiles = (n_pages + TILE_PAGES - 1) / TILE_PAGES;
            const int32_t *row = P.table + (size_t)it.table_seq * P.table_stride + page0;
            const size_t head_off = (size_t)it.kvh * HEAD_BLOCK;
            const size_t page_stride = (size_t)P.Hkv * HEAD_BLOCK;
            int e0 = 0, e1 = 0, e2 = 0, e3 = 0;
            for (int tile = 0; tile < n_tiles; ++tile) {
                if ((tile & 31) == 0) {      // each lane fetches the 4 table entries of one tile
                    const int pb = (tile + lane) * TILE_PAGES;
                    e0 = pb + 0 < n_pages ? row[pb + 0] : 0;
                    e1 = pb + 1 < n_pages ? row[pb + 1] : 0;
                    e2 = pb + 2 < n_pages ? row[pb + 2] : 0;
                    e3 = pb + 3 < n_pages ? row[pb + 3] : 0;
                }
                const int src = tile & 31;
                const int p0 = __shfl_sync(0xffffffffu, e0, src), p1 = __shfl_sync(0xffffffffu, e1, src);
                const int p2 = __shfl_sync(0xffffffffu, e2, src), p3 = __shfl_sync(0xffffffffu, e3, src);
                if (lane == 0) {
                    const int np = min(TILE_PAGES, n_pages - tile * TILE_PAGES);
                    const uint32_t full = bar_base + 8 * stage, empty = bar_base + 8 * (NSTAGE + stage);
                    mbar_wait(empty, phase ^ 1);
                    mbar_expect_tx(full, (uint32_t)np * 2 * HEAD_BLOCK);
                    const uint32_t kdst = stage_base + stage * STAGE_BYTES;
                    const uint32_t vdst = kdst + TILE_PAGES * HEAD_BLOCK;
                    const int pg[4] = {p0, p1, p2, p3};
#pragma unroll
                    for (int p = 0; p < TILE_PAGES; ++p)
                        if (p < np) {
                            const size_t off = (size_t)pg[p] * page_stride + head_off;
                            bulk_g2s(kdst + p * HEAD_BLOCK, P.k_pool + off, HEAD_BLOCK, full);
                            bulk_g2s(vdst + p * HEAD_BLOCK, P.v_pool + off, HEAD_BLOCK, full);
                        }
                }
                if (++stage == NSTAGE) { stage = 0; phase ^= 1; }
            }
        }
        return;
    }

    // ================================ consumers ================================
    const int g = lane >> 2, tq = (lane & 3) * 2;
    for (int idx = item_begin; idx < item_end; ++idx) {
        const WorkItem it = load_item(P.items, idx, P.seq_len);
        const int RT = it.nrows <= 16 ? 1 : (it.nrows <= 32 ? 2 : 4);   // row tiles of 16
        const int TP = N_CONSUMER_WARPS / RT;                             // token parts of a tile
        const int rt = warp % RT, tp = warp / RT;
        const int TW = TILE_TOKENS / TP;                                  // tokens per warp per tile

        // ---- Q rows of this warp's row tile as A fragments --------------------------
        uint32_t qa[8][4];
        const int rr0 = rt * 16 + g, rr1 = rr0 + 8;
        int lim_r0 = 0, lim_r1 = 0;
        {
            const uint16_t *q0 = nullptr, *q1 = nullptr;
            if (rr0 < it.nrows) {
                const int lr = it.rb0 + rr0;
                q0 = P.q + ((size_t)item_qrow(it, P.rowmap, lr, P.G) * P.Hq + it.kvh * P.G + lr % P.G) * D;
                lim_r0 = it.lim0 + lr / P.G;
            }
            if (rr1 < it.nrows) {
                const int lr = it.rb0 + rr1;
                q1 = P.q + ((size_t)item_qrow(it, P.rowmap, lr, P.G) * P.Hq + it.kvh * P.G + lr % P.G) * D;
                lim_r1 = it.lim0 + lr / P.G;
            }
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
                const int d0 = 16 * ks + tq;
                qa[ks][0] = q0 ? *reinterpret_cast<const uint32_t *>(q0 + d0) : 0u;
                qa[ks][1] = q1 ? *reinterpret_cast<const uint32_t *>(q1 + d0) : 0u;
                qa[ks][2] = q0 ? *reinterpret_cast<const uint32_t *>(q0 + d0 + 8) : 0u;
                qa[ks][3] = q1 ? *reinterpret_cast<const uint32_t *>(q1 + d0 + 8) : 0u;
            }
        }
        const int min_lim = it.lim0 + it.rb0 / P.G;   // smallest visibility limit of the item

        RowState st;
#pragma unroll
        for (int n = 0; n < 16; ++n) st.o[n][0] = st.o[n][1] = st.o[n][2] = st.o[n][3] = 0.f;
        st.m[0] = st.m[1] = -INFINITY;
        st.l[0] = st.l[1] = 0.f;

        const int n_tiles = (it.tok1 - it.tok0 + TILE_TOKENS - 1) / TILE_TOKENS;
        for (int tile = 0; tile < n_tiles; ++tile) {
            const uint32_t full = bar_base + 8 * stage, empty = bar_base + 8 * (NSTAGE + stage);
            mbar_wait(full, phase);
            const uint32_t k_base = stage_base + stage * STAGE_BYTES;
            const uint32_t v_base = k_base + TILE_PAGES * HEAD_BLOCK;
            const int tile_t0 = it.tok0 + tile * TILE_TOKENS;
            const int nv = min(TILE_TOKENS, it.tok1 - tile_t0);            // valid tokens in the tile
            const int nvp = (nv + PS - 1) / PS;                            // staged pages
            const bool need_mask = nv < TILE_TOKENS || tile_t0 + TILE_TOKENS - 1 > min_lim;
            bool wrote_smem = false;
            if ((nv & (PS - 1)) && (nvp - 1) * PS >= tp * TW && (nvp - 1) * PS < (tp + 1) * TW) {
                // the last staged page is partially filled: its tail rows hold whatever the pool
                // held (possibly NaN patterns).  P is 0 there; make V 0 as well.
                uint8_t *vpage = smem + stage * STAGE_BYTES + (TILE_PAGES + nvp - 1) * HEAD_BLOCK;
                const int r_first = nv & (PS - 1);
                for (int i = lane; i < (PS - r_first) * 16; i += 32) {
                    const int r = r_first + (i >> 4), c = i & 15;
                    *reinterpret_cast<uint4 *>(vpage + swz_chunk_off(2, r, c)) = make_uint4(0, 0, 0, 0);
                }
                __syncwarp();
                wrote_smem = true;
            }
            if (TW == 64) {
#pragma unroll 1
                for (int sb = 0; sb < 2; ++sb) {
                    const int pg0 = sb * 2;
                    if (pg0 < nvp)
                        process_block<4>(st, qa, k_base, v_base, pg0, lane, P.scale_log2, need_mask,
                                         tile_t0 + pg0 * PS, it.tok1, lim_r0, lim_r1, nvp - pg0);
                }
            } else if (TW == 32) {
                const int pg0 = tp * 2;
                if (pg0 < nvp)
                    process_block<4>(st, qa, k_base, v_base, pg0, lane, P.scale_log2, need_mask,
                                     tile_t0 + pg0 * PS, it.tok1, lim_r0, lim_r1, nvp - pg0);
            } else {
                const int pg0 = tp;
                if (pg0 < nvp)
                    process_block<2>(st, qa, k_base, v_base, pg0, lane, P.scale_log2, need_mask,
                                     tile_t0 + pg0 * PS, it.tok1, lim_r0, lim_r1, nvp - pg0);
            }
            if (wrote_smem) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(empty);
            if (++stage == NSTAGE) { stage = 0; phase ^= 1; }
        }

        // ---- finish the row sums (quad reduce), combine token parts, write the partial --------
        st.l[0] += __shfl_xor_sync(0xffffffffu, st.l[0], 1);
        st.l[0] += __shfl_xor_sync(0xffffffffu, st.l[0], 2);
        st.l[1] += __shfl_xor_sync(0xffffffffu, st.l[1], 1);
        st.l[1] += __shfl_xor_sync(0xffffffffu, st.l[1], 2);
        float *rec0 = comb, *rec1 = comb + COMB_REC_BYTES / 4;
        if (TP == 4) {
            if (warp == 2) comb_store(st, rec0, lane);
            if (warp == 3) comb_store(st, rec1, lane);
            consumer_bar();
            if (warp == 0) comb_merge(st, rec0, lane);
            if (warp == 1) comb_merge(st, rec1, lane);
            consumer_bar();
            if (warp == 1) comb_store(st, rec0, lane);
            consumer_bar();
            if (warp == 0) comb_merge(st, rec0, lane);
            consumer_bar();
        } else if (TP == 2) {
            if (warp == 2) comb_store(st, rec0, lane);
            if (warp == 3) comb_store(st, rec1, lane);
            consumer_bar();
            if (warp == 0) comb_merge(st, rec0, lane);
            if (warp == 1) comb_merge(st, rec1, lane);
            consumer_bar();
        }
        if (tp == 0) {
            const float inv0 = st.l[0] > 0.f ? 1.f / st.l[0] : 0.f;
            const float inv1 = st.l[1] > 0.f ? 1.f / st.l[1] : 0.f;
            if (rr0 < it.nrows) {
                float *o = P.ws_o + (size_t)(it.part_base + rr0) * D + tq;
#pragma unroll
                for (int n = 0; n < 16; ++n)
                    *reinterpret_cast<float2 *>(o + 8 * n) = make_float2(st.o[n][0] * inv0, st.o[n][1] * inv0);
                if ((lane & 3) == 0)
                    P.ws_lse[it.part_base + rr0] =
                        st.l[0] > 0.f ? (st.m[0] + log2f(st.l[0])) * LN2 : -INFINITY;
            }
            if (rr1 < it.nrows) {
                float *o = P.ws_o + (size_t)(it.part_base + rr1) * D + tq;
#pragma unroll
                for (int n = 0; n < 16; ++n)
                    *reinterpret_cast<float2 *>(o + 8 * n) = make_float2(st.o[n][2] * inv1, st.o[n][3] * inv1);
                if ((lane & 3) == 0)
                    P.ws_lse[it.part_base + rr1] =
                        st.l[1] > 0.f ? (st.m[1] + log2f(st.l[1])) * LN2 : -INFINITY;
            }
        }
    }
    // When launched programmatically behind the tcgen05 kernel this grid may start before that one
    // has finished; do not complete before it has, so that merge_kernel (which waits for THIS grid)
    // sees both kernels' partials.  A no-op for a normal launch.
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

}  // namespace

namespace spork {

int attn_mma_grid(spork_ctx *c) { return c->num_sms * CTAS_PER_SM; }

int launch_attn_mma(spork_ctx *c, const LayerIO &io, bool programmatic, cudaStream_t st) {
    const Plan &P = c->plan;
    if (P.n_items == 0) return SPORK_OK;
    if (!(c->smem_attr_done & 8u)) {       // per handle (= per device), not per process
        SPORK_CUDA(cudaFuncSetAttribute(attn_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        SMEM_BYTES));
        c->smem_attr_done |= 8u;
    }
    Params p;
    p.items = P.d_items;
    p.cta_ptr = P.d_cta_ptr;
    p.seq_len = c->d_len;
    p.rowmap = P.d_rowmap;
    p.q = (const uint16_t *)io.q;
    p.k_pool = (const uint8_t *)io.k_pool;
    p.v_pool = (const uint8_t *)io.v_pool;
    p.table = c->d_table;
    p.table_stride = c->table_stride;
    p.Hq = c->cfg.num_q_heads;
    p.Hkv = c->cfg.num_kv_heads;
    p.G = c->G;
    p.scale_log2 = c->cfg.scale * LOG2E;
    p.ws_o = (float *)c->ws_o.p;
    p.ws_lse = (float *)c->ws_lse.p;
    const int grid = P.grid;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(N_THREADS);
    cfg.dynamicSmemBytes = SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = programmatic ? 1 : 0;   // overlap the tail of the tcgen05 kernel
    SPORK_CUDA(cudaLaunchKernelEx(&cfg, attn_mma_kernel, p));
    c->last_launches++;
    c->plan.info.grid = grid;
    SPORK_CUDA(cudaGetLastError());
    return SPORK_OK;
}

}  // namespace spork
