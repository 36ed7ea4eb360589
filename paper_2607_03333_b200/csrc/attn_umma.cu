// libspork: the tensor path -- bf16 KV, D = 128, page = 16 tokens, up to 128 query rows
// per work item on the 5th-generation tensor cores (tcgen05.mma, accumulators in TMEM).
//
// One persistent CTA = producer warp + one MMA-issuing thread + 4 softmax warps; 2 CTAs per SM
// (256 TMEM columns and < 113 KiB of shared memory each), so one CTA's softmax overlaps the
// other's MMAs.  Per 64-token tile of an item:
//   producer : one cp.async.bulk per (page, kv head) block of K, then of V, into a ring of
//              16 KiB slots (K and V are separate slots, released separately)
//   MMA      : S[128 x 64] = Q K^T   (A = Q in smem, B = K pages, both K-major SW128)
//              O[128 x 128] += P V   (A = P in TMEM as packed bf16, B = V pages, MN-major SW128)
//              S(i+1) is issued before P V(i): it runs while the softmax of tile i is busy
//   softmax  : thread r owns query row r (TMEM lane r): tcgen05.ld of S, mask, row max,
//              exp2, row sum, bf16 P back into TMEM over the S columns.  The running max is
//              only raised when it grows by more than 2^8 (P stays <= 256, exact in bf16's
//              exponent range), so O is rescaled in TMEM rarely.
// The fork group's GQA rows of all members are the 128 M-rows of one tile, so a shared prefix
// page is read from HBM once per group.  Every item writes one normalised partial (o, lse)
// per row for merge_kernel.
#include <math.h>

#include "spork_internal.h"
#include "umma.cuh"

using namespace spork;
using namespace spork::ptx;

namespace {

constexpr int D = 128;
constexpr int TILE_PAGES = 4;
constexpr int TILE_TOKENS = TILE_PAGES * PS;          // 64
constexpr int HEAD_BLOCK = PS * D * 2;                // 4096 B: one (page, kv head) block
constexpr int SLOT_BYTES = TILE_PAGES * HEAD_BLOCK;   // 16 KiB: a K tile or a V tile
constexpr int NSLOT = 5;
constexpr int Q_BYTES = 128 * D * 2;                  // 32 KiB
constexpr int Q_HALF = Q_BYTES / 2;                   // dims [64, 128) start here
constexpr int N_THREADS = 192;
constexpr int CTAS_PER_SM = 2;
constexpr int TMEM_COLS = 256;                        // O: [0,128)  S/P buffer b: [128 + 64 b, +64)
constexpr int BAR_OFF = Q_BYTES + NSLOT * SLOT_BYTES;
constexpr int SMEM_BYTES = BAR_OFF + 256;
constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;
constexpr float RESCALE_THRESHOLD = 8.f;              // log2 units

struct UParams {
    const WorkItem *items;
    const int32_t *cta_ptr;
    const uint16_t *q;
    const uint8_t *k_pool, *v_pool;
    const int32_t *table;
    int table_stride, Hq, Hkv, G;
    float scale_log2;
    float *ws_o, *ws_lse;
};

// barrier slots (8 bytes each) from BAR_OFF
enum : int {
    B_FULL = 0,                 // [NSLOT] bulk copies landed
    B_EMPTY = NSLOT,            // [NSLOT] MMAs reading the slot completed
    B_SFULL = 2 * NSLOT,        // [2] S(b) complete
    B_PFULL = 2 * NSLOT + 2,    // [2] P(b) written (4 softmax warps)
    B_PVDONE = 2 * NSLOT + 4,   // [2] P V of a tile with parity b complete
    B_QFULL = 2 * NSLOT + 6,    // Q staged
    B_OFREE = 2 * NSLOT + 7,    // epilogue finished reading O
    B_COUNT = 2 * NSLOT + 8
};

__global__ void __launch_bounds__(N_THREADS, CTAS_PER_SM) attn_umma_kernel(const UParams P) {
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bars = sbase + BAR_OFF;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + BAR_OFF + 8 * B_COUNT);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    auto bar = [&](int i) { return bars + 8u * (uint32_t)i; };

    if (threadIdx.x == 0) {
        if (sbase & 1023u) __trap();   // the 128-byte swizzle is a function of the smem address
        for (int s = 0; s < NSLOT; ++s) {
            mbar_init(bar(B_FULL + s), 1);
            mbar_init(bar(B_EMPTY + s), 1);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(bar(B_SFULL + b), 1);
            mbar_init(bar(B_PFULL + b), 4);
            mbar_init(bar(B_PVDONE + b), 1);
        }
        mbar_init(bar(B_QFULL), 1);
        mbar_init(bar(B_OFREE), 4);
        mbar_fence_init();
    }
    if (warp == 1) {
        tmem_alloc(smem_u32(tmem_slot), TMEM_COLS);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tbase = *tmem_slot;
    const uint32_t tO = tbase;
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    const int item_begin = P.cta_ptr[blockIdx.x], item_end = P.cta_ptr[blockIdx.x + 1];

    if (warp == 0) {
        // ================================ producer ================================
        uint32_t ld = 0;   // loads issued so far: slot = ld % NSLOT, phase = (ld / NSLOT) & 1
        for (int idx = item_begin; idx < item_end; ++idx) {
            const WorkItem it = P.items[idx];
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
                    const int pg[4] = {p0, p1, p2, p3};
#pragma unroll
                    for (int kv = 0; kv < 2; ++kv) {
                        const uint32_t slot = (ld + kv) % NSLOT, ph = ((ld + kv) / NSLOT) & 1;
                        mbar_wait(bar(B_EMPTY + slot), ph ^ 1);
                        mbar_expect_tx(bar(B_FULL + slot), (uint32_t)np * HEAD_BLOCK);
                        const uint32_t dst = sbase + Q_BYTES + slot * SLOT_BYTES;
                        const uint8_t *pool = kv ? P.v_pool : P.k_pool;
#pragma unroll
                        for (int p = 0; p < TILE_PAGES; ++p)
                            if (p < np)
                                bulk_g2s(dst + p * HEAD_BLOCK, pool + (size_t)pg[p] * page_stride + head_off,
                                         HEAD_BLOCK, bar(B_FULL + slot));
                    }
                }
                ld += 2;
            }
        }
    } else if (warp == 1) {
        // ================================ MMA issuer (one thread) ================================
        if (lane == 0) {
            uint32_t g0 = 0;   // tiles issued before this item (global tile counter)
            int j = 0;
            for (int idx = item_begin; idx < item_end; ++idx, ++j) {
                const WorkItem it = P.items[idx];
                const int n_tok = it.tok1 - it.tok0;
                const int n_tiles = (n_tok + TILE_TOKENS - 1) / TILE_TOKENS;
                auto pages_of_tile = [&](int i) {
                    return (min(TILE_TOKENS, n_tok - i * TILE_TOKENS) + PS - 1) / PS;
                };
                auto issue_s = [&](int i) {
                    const uint32_t g = g0 + i, b = g & 1, ldk = 2 * g;
                    const uint32_t slot = ldk % NSLOT, ph = (ldk / NSLOT) & 1;
                    mbar_wait(bar(B_FULL + slot), ph);
                    tc_fence_after();
                    const uint32_t id = idesc_bf16(128, PS * pages_of_tile(i), 0, 0);
                    const uint32_t ka = sbase + Q_BYTES + slot * SLOT_BYTES;
                    const uint32_t tS = tbase + 128 + 64 * b;
#pragma unroll
                    for (int ks = 0; ks < 8; ++ks) {
                        const uint64_t ad = smem_desc_sw128(sbase + (ks >> 2) * Q_HALF + (ks & 3) * 32, 16, 1024);
                        const uint64_t bd = smem_desc_sw128(ka + (ks >> 2) * 1024 + (ks & 3) * 32, 16, 2048);
                        mma_ss(tS, ad, bd, id, ks > 0);
                    }
                    mma_commit(bar(B_EMPTY + slot));
                    mma_commit(bar(B_SFULL + b));
                };
                mbar_wait(bar(B_QFULL), j & 1);
                tc_fence_after();
                issue_s(0);
                for (int i = 0; i < n_tiles; ++i) {
                    if (i + 1 < n_tiles) issue_s(i + 1);
                    const uint32_t g = g0 + i, b = g & 1, ldv = 2 * g + 1;
                    const uint32_t slot = ldv % NSLOT, ph = (ldv / NSLOT) & 1;
                    mbar_wait(bar(B_PFULL + b), (g >> 1) & 1);
                    mbar_wait(bar(B_FULL + slot), ph);
                    if (i == 0 && j > 0) mbar_wait(bar(B_OFREE), (j - 1) & 1);
                    tc_fence_after();
                    const uint32_t id = idesc_bf16(128, D, 0, 1);
                    const uint32_t va = sbase + Q_BYTES + slot * SLOT_BYTES;
                    const uint32_t tP = tbase + 128 + 64 * b;
                    const int nvp = pages_of_tile(i);
#pragma unroll
                    for (int pg = 0; pg < TILE_PAGES; ++pg)
                        if (pg < nvp) {
                            const uint64_t bd = smem_desc_sw128(va + pg * HEAD_BLOCK, 1024, 2048);
                            mma_ts(tO, tP + pg * 8, bd, id, (i > 0) || (pg > 0));
                        }
                    mma_commit(bar(B_EMPTY + slot));
                    mma_commit(bar(B_PVDONE + b));
                }
                g0 += n_tiles;
            }
        }
        __syncwarp();
    } else {
        // ================================ softmax warps ================================
        const int lg = warp & 3;                       // TMEM lane group this warp may access
        const int r = lg * 32 + lane;                  // query row of the item owned by this thread
        const uint32_t lane_addr = (uint32_t)(lg * 32) << 16;
        const int st = threadIdx.x - 64;               // 0..127 among the softmax threads
        uint32_t g0 = 0;
        for (int idx = item_begin; idx < item_end; ++idx) {
            const WorkItem it = P.items[idx];
            const int n_tok = it.tok1 - it.tok0;
            const int n_tiles = (n_tok + TILE_TOKENS - 1) / TILE_TOKENS;
            // ---- Q rows -> smem (K-major, 128-byte swizzle); rows beyond nrows are zero ----
            {
                const int c = st & 15;                 // 16-byte chunk of the row
#pragma unroll 4
                for (int k = 0; k < 16; ++k) {
                    const int row = (st >> 4) + 8 * k;
                    uint4 v = make_uint4(0, 0, 0, 0);
                    if (row < it.nrows) {
                        const int lr = it.rb0 + row;
                        const uint16_t *src =
                            P.q + ((size_t)(it.qrow0 + lr / P.G) * P.Hq + it.kvh * P.G + lr % P.G) * D + c * 8;
                        v = *reinterpret_cast<const uint4 *>(src);
                    }
                    const int off = (c >> 3) * Q_HALF + (row >> 3) * 1024 + (row & 7) * 128 +
                                    (((c & 7) ^ (row & 7)) << 4);
                    *reinterpret_cast<uint4 *>(smem + off) = v;
                }
                fence_async_smem();
                asm volatile("bar.sync 1, 128;" ::: "memory");
                if (st == 0) mbar_arrive(bar(B_QFULL));
            }
            const int lim_r = it.lim0 + (it.rb0 + r) / P.G;
            const int min_lim = it.lim0 + it.rb0 / P.G;
            float m_used = -INFINITY, l = 0.f, lr = 0.f;   // l: exact row sum (lse); lr: sum of the bf16 weights

            if (lg * 32 >= it.nrows) {
                // none of this warp's 32 rows exists (few-row item): only keep the barriers moving;
                // whatever S/P/O hold in these lanes never leaves TMEM
                for (int i = 0; i < n_tiles; ++i) {
                    const uint32_t g = g0 + i, b = g & 1;
                    mbar_wait(bar(B_SFULL + b), (g >> 1) & 1);
                    if (lane == 0) mbar_arrive(bar(B_PFULL + b));
                    __syncwarp();
                }
                const uint32_t gl = g0 + n_tiles - 1;
                mbar_wait(bar(B_PVDONE + (gl & 1)), (gl >> 1) & 1);
                if (lane == 0) mbar_arrive(bar(B_OFREE));
                __syncwarp();
                g0 += n_tiles;
                continue;
            }

            for (int i = 0; i < n_tiles; ++i) {
                const uint32_t g = g0 + i, b = g & 1;
                const uint32_t tS = tbase + 128 + 64 * b + lane_addr;
                mbar_wait(bar(B_SFULL + b), (g >> 1) & 1);
                tc_fence_after();
                uint32_t s0[32], s1[32];
                tmem_ld32(tS, s0);
                tmem_ld32(tS + 32, s1);
                tmem_wait_ld();
                const int tile_t0 = it.tok0 + i * TILE_TOKENS;
                const int nv = min(TILE_TOKENS, it.tok1 - tile_t0);
                if (nv < TILE_TOKENS || tile_t0 + TILE_TOKENS - 1 > min_lim) {
                    const int vis = min(nv, lim_r - tile_t0 + 1);   // visible tokens of the tile for this row
#pragma unroll
                    for (int t = 0; t < 32; ++t) {
                        if (t >= vis) s0[t] = 0xff800000u;           // -inf
                        if (t + 32 >= vis) s1[t] = 0xff800000u;
                    }
                }
                float mx = -INFINITY;
#pragma unroll
                for (int t = 0; t < 32; ++t)
                    mx = fmaxf(mx, fmaxf(__uint_as_float(s0[t]), __uint_as_float(s1[t])));
                const float mxs = mx * P.scale_log2;
                const bool grow = mxs > m_used + RESCALE_THRESHOLD;
                if (__any_sync(0xffffffffu, grow)) {
                    const float m_new = grow ? mxs : m_used;
                    const float alpha = grow ? (m_used == -INFINITY ? 0.f : ex2(m_used - m_new)) : 1.f;
                    l *= alpha;
                    lr *= alpha;
                    if (i > 0) {
                        // O holds tiles [0, i): wait for P V(i - 1), rescale this thread's row
                        mbar_wait(bar(B_PVDONE + ((g - 1) & 1)), ((g - 1) >> 1) & 1);
                        tc_fence_after();
#pragma unroll 1
                        for (int cb = 0; cb < 4; ++cb) {
                            uint32_t o[32];
                            tmem_ld32(tO + lane_addr + cb * 32, o);
                            tmem_wait_ld();
#pragma unroll
                            for (int t = 0; t < 32; ++t) o[t] = __float_as_uint(__uint_as_float(o[t]) * alpha);
                            tmem_st32(tO + lane_addr + cb * 32, o);
                        }
                        tmem_wait_st();
                    }
                    m_used = m_new;
                }
                const float mu = m_used == -INFINITY ? 0.f : m_used;
                uint32_t p[32];
                float sum0 = 0.f, sum1 = 0.f, rs0 = 0.f, rs1 = 0.f;
#pragma unroll
                for (int t = 0; t < 16; ++t) {
                    const float a0 = ex2(fmaf(__uint_as_float(s0[2 * t]), P.scale_log2, -mu));
                    const float a1 = ex2(fmaf(__uint_as_float(s0[2 * t + 1]), P.scale_log2, -mu));
                    const float c0 = ex2(fmaf(__uint_as_float(s1[2 * t]), P.scale_log2, -mu));
                    const float c1 = ex2(fmaf(__uint_as_float(s1[2 * t + 1]), P.scale_log2, -mu));
                    p[t] = pack_bf16(a0, a1);
                    p[16 + t] = pack_bf16(c0, c1);
                    // o is normalised by the sum of the ROUNDED weights the tensor core uses, so that
                    // o = sum(p v) / sum(p) stays a true weighted mean (a one-hot row returns V exactly
                    // even when the running max is stale and p is not a power of two); lse keeps the
                    // exact sum
                    sum0 += a0 + a1;
                    sum1 += c0 + c1;
                    rs0 += __uint_as_float(p[t] << 16) + __uint_as_float(p[t] & 0xffff0000u);
                    rs1 += __uint_as_float(p[16 + t] << 16) + __uint_as_float(p[16 + t] & 0xffff0000u);
                }
                l += sum0 + sum1;
                lr += rs0 + rs1;
                tmem_st32(tS, p);
                tmem_wait_st();
                if ((nv & (PS - 1)) && lg == 0) {
                    // the last staged page is partially filled: its tail rows hold whatever the pool
                    // held (possibly NaN patterns).  P is 0 there; make V 0 as well (the warp of rows
                    // 0..31 does it: it is active in every item).
                    const uint32_t ldv = 2 * g + 1, slot = ldv % NSLOT, ph = (ldv / NSLOT) & 1;
                    mbar_wait(bar(B_FULL + slot), ph);
                    const int nvp = (nv + PS - 1) / PS;
                    uint8_t *vpage = smem + Q_BYTES + slot * SLOT_BYTES + (nvp - 1) * HEAD_BLOCK;
                    const int r_first = nv & (PS - 1);
                    for (int e = lane; e < (PS - r_first) * 16; e += 32) {
                        const int rr = r_first + (e >> 4), cc = e & 15;
                        *reinterpret_cast<uint4 *>(vpage + swz_chunk_off(2, rr, cc)) = make_uint4(0, 0, 0, 0);
                    }
                    fence_async_smem();
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_PFULL + b));
            }

            // ---- epilogue: O / l -> partial rows ------------------------------------------------
            {
                const uint32_t gl = g0 + n_tiles - 1;
                mbar_wait(bar(B_PVDONE + (gl & 1)), (gl >> 1) & 1);
                tc_fence_after();
                const float inv = lr > 0.f ? 1.f / lr : 0.f;
                float *dst = P.ws_o + (size_t)(it.part_base + r) * D;
#pragma unroll 1
                for (int cb = 0; cb < 4; ++cb) {
                    uint32_t o[32];
                    tmem_ld32(tO + lane_addr + cb * 32, o);
                    tmem_wait_ld();
                    if (r < it.nrows) {
#pragma unroll
                        for (int t = 0; t < 8; ++t)
                            *reinterpret_cast<float4 *>(dst + cb * 32 + 4 * t) =
                                make_float4(__uint_as_float(o[4 * t]) * inv, __uint_as_float(o[4 * t + 1]) * inv,
                                            __uint_as_float(o[4 * t + 2]) * inv, __uint_as_float(o[4 * t + 3]) * inv);
                    }
                }
                if (r < it.nrows)
                    P.ws_lse[it.part_base + r] = l > 0.f ? (m_used + log2f(l)) * LN2 : -INFINITY;
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(B_OFREE));
            }
            g0 += n_tiles;
        }
    }

    // ---- teardown: every MMA has completed (the softmax warps waited for the last P V) ----
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tbase, TMEM_COLS);
    }
}

}  // namespace

namespace spork {

int attn_umma_grid(spork_ctx *c) { return c->num_sms * CTAS_PER_SM; }

int launch_attn_umma(spork_ctx *c, const void *q, cudaStream_t st) {
    const Plan &P = c->plan;
    if (P.n_items_umma == 0) return SPORK_OK;
    static bool attr_set = false;
    if (!attr_set) {
        SPORK_CUDA(cudaFuncSetAttribute(attn_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        SMEM_BYTES));
        attr_set = true;
    }
    UParams p;
    p.items = (const WorkItem *)P.items.p + P.n_items;        // the tensor-path items follow the others
    p.cta_ptr = (const int32_t *)P.cta_ptr.p + (P.grid + 1);
    p.q = (const uint16_t *)q;
    p.k_pool = (const uint8_t *)c->k_pool;
    p.v_pool = (const uint8_t *)c->v_pool;
    p.table = c->d_table;
    p.table_stride = c->table_stride;
    p.Hq = c->cfg.num_q_heads;
    p.Hkv = c->cfg.num_kv_heads;
    p.G = c->G;
    p.scale_log2 = c->cfg.scale * LOG2E;
    p.ws_o = (float *)c->ws_o.p;
    p.ws_lse = (float *)c->ws_lse.p;
    attn_umma_kernel<<<P.grid_umma, N_THREADS, SMEM_BYTES, st>>>(p);
    c->last_launches++;
    SPORK_CUDA(cudaGetLastError());
    return SPORK_OK;
}

}  // namespace spork
