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
constexpr int Q_BYTES = 128 * D * 2;                  // 32 KiB: the 128 rows of one pipe
constexpr int Q_HALF = Q_BYTES / 2;                   // dims [64, 128) start here
constexpr int PIPE_COLS = 256;                        // TMEM columns of one pipe: O [0,128), S/P buffer b [128 + 64 b, +64)
constexpr float LOG2E = 1.4426950408889634f;
constexpr float LN2 = 0.6931471805599453f;
constexpr float RESCALE_THRESHOLD = 8.f;              // log2 units
// share of a tile's exp2 pairs computed on the FMA pipe instead of the MUFU unit (ex2_poly2): pair j of a
// thread's 32 is emulated when (j * EMU_NUM) % EMU_DEN < EMU_NUM.  Default 0: measured on config 4 the
// emulation only costs (k = 16: 544 / 568 / 600 / 634 us at 0, 1/4, 1/3, 1/2) -- a softmax warp is bound by
// its own dependent instruction stream (~2,200 clocks per 64-token tile), not by the
// MUFU unit, so extra FMA-pipe work lengthens it.  Kept as a build-time knob (-DSPORK_EMU_NUM / _DEN).
#ifndef SPORK_EMU_NUM
#define SPORK_EMU_NUM 0
#endif
#ifndef SPORK_EMU_DEN
#define SPORK_EMU_DEN 1
#endif
constexpr int EMU_NUM = SPORK_EMU_NUM, EMU_DEN = SPORK_EMU_DEN;
__host__ __device__ constexpr bool emulated_pair(int j) { return (j * EMU_NUM) % EMU_DEN < EMU_NUM; }

// NP = number of softmax pipes of a CTA = row blocks of 128 it runs against ONE stream of K/V:
//   NP = 1: items of <= 128 rows, 2 CTAs per SM, 5-slot ring each
//   NP = 2: items of <= 256 rows (verify with many drafts), 1 CTA per SM, 10-slot ring; every
//           K/V tile is fetched once for both row blocks
//   SP = 2 (NP = 1 only): every row's 64 scores of a tile are split over TWO threads (8 softmax warps,
//           4 per SM sub-partition instead of 2) for items whose time is the softmax's, not HBM's:
//           4-slot ring, the row max and the row sums are exchanged through shared memory
//   F8 (NP = SP = 1): the FP8-KV variant (e4m3 K/V bytes, bf16 Q).  The bulk copies land 8 KiB e4m3 tiles
//           in a 6-slot ring.  K is consumed where it lands: S = Q K^T runs in kind::f8f6f4, with Q split
//           into TWO e4m3 terms when it is staged (q = hi + lo exactly for a bf16 q: 4 + 4 significant bits),
//           so the scores are as exact as the bf16 path's.  V is widened (exactly) to fp16 by two converter
//           warps, half a tile each, into one of TWO operand slots in the swizzled image the bf16 path
//           stages directly; P is packed as fp16 and P V runs in kind::f16.  Softmax, epilogue, merge and
//           planner are the bf16 kernel's.
template <int NP, int SP, bool F8 = false>
struct Cfg {
    static_assert(SP == 1 || NP == 1, "split rows only with one pipe");
    static_assert(!F8 || (NP == 1 && SP == 1), "FP8-KV: the default kernel shape only");
    static constexpr int NSLOT = F8 ? 6 : (NP == 2 ? 10 : (SP == 2 ? 4 : 5));
    static constexpr int RING_SLOT = F8 ? SLOT_BYTES / 2 : SLOT_BYTES;   // bytes of one landed K or V tile
    static constexpr int N_SOFTMAX = NP * 128 * SP;
    static constexpr int N_CONV = F8 ? 64 : 0;                            // converter threads (2 warps)
    static constexpr int N_THREADS = 64 + N_SOFTMAX + N_CONV;
    static constexpr int CTAS_PER_SM = NP == 1 ? 2 : 1;
    static constexpr int TMEM_COLS = NP * PIPE_COLS;
    static constexpr int OPER_OFF = NP * Q_BYTES;                         // F8: two fp16 V operand slots
    static constexpr int RING_OFF = OPER_OFF + (F8 ? 2 * SLOT_BYTES : 0);
    static constexpr int BAR_OFF = RING_OFF + NSLOT * RING_SLOT;
    // barrier slots (8 bytes each) from BAR_OFF
    static constexpr int B_FULL = 0;                  // [NSLOT] bulk copies landed
    static constexpr int B_EMPTY = NSLOT;             // [NSLOT] MMAs (F8: converters) reading the slot completed
    static constexpr int B_PIPE = 2 * NSLOT;          // per pipe: 7 barriers, see P_*
    static constexpr int B_QFULL = B_PIPE + 7 * NP;   // Q staged
    static constexpr int B_OPER = B_QFULL + 1;        // F8: V operand slot b empty [2] ("full" arrives on P_PFULL + b)
    static constexpr int B_COUNT = B_OPER + (F8 ? 2 : 0);
    static constexpr int XCH_OFF = BAR_OFF + 8 * B_COUNT + 16;     // float [2][2][128] (SP = 2)
    static constexpr int QEXP_OFF = XCH_OFF + (SP == 2 ? 2048 : 0);   // F8: uint8 [2][128], per-row power-of-two Q scaling
    static constexpr int SMEM_BYTES = QEXP_OFF + (F8 ? 256 : 0);
};
enum : int { O_VEMPTY = 0 };
enum : int {
    P_SFULL = 0,    // [2] S(b) complete
    P_PFULL = 2,    // [2] P(b) written (4 softmax warps)
    P_PVDONE = 4,   // [2] P V of a tile with parity b complete
    P_OFREE = 6     // epilogue finished reading O
};

struct UParams {
    const WorkItem *items;
    const int32_t *cta_ptr;
    const int32_t *seq_len;       // device lengths: open-ended items end there
    const int32_t *rowmap;
    const uint16_t *q;
    const uint8_t *k_pool, *v_pool;
    const int32_t *table;
    int table_stride, Hq, Hkv, G;
    float scale_log2;
    float *ws_o, *ws_lse;
    int wait_prev;                // launched programmatically behind a kernel that still READS ws_o / ws_lse
                                  // (the merge of the previous layer): wait for it before the first partial
};

template <int NP, int SP, bool F8>
__global__ void __launch_bounds__(Cfg<NP, SP, F8>::N_THREADS, Cfg<NP, SP, F8>::CTAS_PER_SM)
attn_umma_kernel(const UParams P) {
    using C = Cfg<NP, SP, F8>;
    constexpr int NSLOT = C::NSLOT;
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = smem_u32(smem);
    const uint32_t ring = sbase + C::RING_OFF;
    const uint32_t bars = sbase + C::BAR_OFF;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(smem + C::BAR_OFF + 8 * C::B_COUNT);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    auto bar = [&](int i) { return bars + 8u * (uint32_t)i; };
    auto pbar = [&](int w, int i) { return bars + 8u * (uint32_t)(C::B_PIPE + 7 * w + i); };

    if (threadIdx.x == 0) {
        if (sbase & 1023u) __trap();   // the 128-byte swizzle is a function of the smem address
        for (int s = 0; s < NSLOT; ++s) {
            mbar_init(bar(C::B_FULL + s), 1);
            // F8: even slots hold K tiles (freed by the S MMAs' commit), odd slots V tiles (freed by both converter warps)
            mbar_init(bar(C::B_EMPTY + s), (F8 && (s & 1)) ? 2 : 1);
        }
        for (int w = 0; w < NP; ++w) {
            for (int b = 0; b < 2; ++b) {
                mbar_init(pbar(w, P_SFULL + b), 1);
                mbar_init(pbar(w, P_PFULL + b), 4 * SP + (F8 ? 2 : 0));   // F8: + the two V converter warps (see below)
                mbar_init(pbar(w, P_PVDONE + b), 1);
            }
            mbar_init(pbar(w, P_OFREE), 4 * SP);
        }
        mbar_init(bar(C::B_QFULL), 1);
        if constexpr (F8) {
            // V operand slot b is "full" on P_PFULL + b together with P(b): tile T uses S/P buffer T & 1 AND V slot
            // T & 1, and the MMA warp needs both before P V -- one wait instead of two (a wait costs ~190 clocks)
            for (int b = 0; b < 2; ++b) mbar_init(bar(C::B_OPER + O_VEMPTY + b), 1);    // tcgen05.commit
        }
        mbar_fence_init();
    }
    if (warp == 1) {
        tmem_alloc(smem_u32(tmem_slot), C::TMEM_COLS);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tbase = *tmem_slot;
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    const int item_begin = P.cta_ptr[blockIdx.x], item_end = P.cta_ptr[blockIdx.x + 1];

    if (warp == 0) {
        // ================================ producer ================================
        uint32_t ld = 0;   // loads issued so far: slot = ld % NSLOT, phase = (ld / NSLOT) & 1
        for (int idx = item_begin; idx < item_end; ++idx) {
            const WorkItem it = load_item(P.items, idx, P.seq_len);
            const int page0 = it.tok0 / PS;
            const int n_pages = (it.tok1 + PS - 1) / PS - page0;
            const int n_tiles = (n_pages + TILE_PAGES - 1) / TILE_PAGES;
            const int32_t *row = P.table + (size_t)it.table_seq * P.table_stride + page0;
            constexpr int HB = F8 ? HEAD_BLOCK / 2 : HEAD_BLOCK;     // bytes of a (page, kv head) block in the pool
            const size_t head_off = (size_t)it.kvh * HB;
            const size_t page_stride = (size_t)P.Hkv * HB;
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
                        mbar_wait(bar(C::B_EMPTY + slot), ph ^ 1);
                        mbar_expect_tx(bar(C::B_FULL + slot), (uint32_t)np * HB);
                        const uint32_t dst = ring + slot * C::RING_SLOT;
                        const uint8_t *pool = kv ? P.v_pool : P.k_pool;
#pragma unroll
                        for (int p = 0; p < TILE_PAGES; ++p)
                            if (p < np)
                                bulk_g2s(dst + p * HB, pool + (size_t)pg[p] * page_stride + head_off,
                                         HB, bar(C::B_FULL + slot));
                    }
                }
                ld += 2;
            }
        }
    } else if (warp == 1) {
        // ================================ MMA issuer ================================
        // The whole warp runs this loop in lockstep (waits, counters, descriptors stay warp-uniform);
        // one elected lane issues the tcgen05 instructions of a step.
        const uint64_t q_desc = smem_desc_sw128(sbase, 16, 1024);     // K-major, 8-row groups 1 KiB apart
        // operand tiles: the ring itself, or (F8) the two fp16 slots the converter warps fill
        const uint32_t v_base = F8 ? sbase + C::OPER_OFF : ring;
        // K-major, 8-token groups 2 KiB apart (e4m3: 128-byte rows hold all 128 dims, groups 1 KiB apart)
        const uint64_t k_desc = smem_desc_sw128(ring, 16, F8 ? 1024 : 2048);
        const uint64_t v_desc = smem_desc_sw128(v_base, 1024, 2048);    // MN-major: dim halves 1 KiB, 8-token groups 2 KiB
        constexpr uint32_t ID_PV = F8 ? idesc_f16(128, D, 0, 1) : idesc_bf16(128, D, 0, 1);
        uint32_t gt = 0;            // tiles of all items so far: K of tile gt is load 2 gt, V is 2 gt + 1
        uint32_t g0[NP];            // tiles pipe w has run (its S/P buffer and barrier phases)
        int jw[NP];                 // items pipe w has run
#pragma unroll
        for (int w = 0; w < NP; ++w) { g0[w] = 0; jw[w] = 0; }
        int j = 0;
        for (int idx = item_begin; idx < item_end; ++idx, ++j) {
            const WorkItem it = load_item(P.items, idx, P.seq_len);
            const int n_tok = it.tok1 - it.tok0;
            const int n_tiles = (n_tok + TILE_TOKENS - 1) / TILE_TOKENS;
            const int npipe = (NP > 1 && it.nrows > 128) ? 2 : 1;   // pipe 1 sits idle on a <= 128-row item
            auto pages_of_tile = [&](int i) {
                return (min(TILE_TOKENS, n_tok - i * TILE_TOKENS) + PS - 1) / PS;
            };
            auto issue_s = [&](int i) {
                const uint32_t ldk = 2 * (gt + i);
                const uint32_t slot = ldk % NSLOT, ph = (ldk / NSLOT) & 1;
                mbar_wait(bar(C::B_FULL + slot), ph);
                tc_fence_after();
                const uint32_t id = F8 ? idesc_f16(128, PS * pages_of_tile(i), 0, 0) : idesc_bf16(128, PS * pages_of_tile(i), 0, 0);
                const uint64_t kd = smem_desc_advance(k_desc, slot * C::RING_SLOT);
                if (elect_one()) {
#pragma unroll
                    for (int w = 0; w < NP; ++w) {
                        if (w < npipe) {
                            const uint32_t b = (g0[w] + i) & 1;
                            const uint32_t tS = tbase + w * PIPE_COLS + 128 + 64 * b;
                            if constexpr (F8) {
                                // 4 K-steps of 32 e4m3 dims, for the hi and the lo term of Q (16 KiB apart)
#pragma unroll
                                for (int ks = 0; ks < 8; ++ks)
                                    mma_ss_f8(tS, smem_desc_advance(q_desc, (ks >> 2) * Q_HALF + (ks & 3) * 32),
                                              smem_desc_advance(kd, (ks & 3) * 32), id, ks > 0);
                            } else {
#pragma unroll
                                for (int ks = 0; ks < 8; ++ks)
                                    mma_ss(tS, smem_desc_advance(q_desc, w * Q_BYTES + (ks >> 2) * Q_HALF + (ks & 3) * 32),
                                           smem_desc_advance(kd, (ks >> 2) * 1024 + (ks & 3) * 32), id, ks > 0);
                            }
                            mma_commit(pbar(w, P_SFULL + b));
                        }
                    }
                    mma_commit(bar(C::B_EMPTY + slot));
                }
                __syncwarp();
            };
            mbar_wait(bar(C::B_QFULL), j & 1);
            tc_fence_after();
            issue_s(0);
            for (int i = 0; i < n_tiles; ++i) {
                if (i + 1 < n_tiles) issue_s(i + 1);
                const uint32_t ldv = 2 * (gt + i) + 1;
                // F8: tile T's V sits in operand slot T & 1, filled by the converter warps
                const uint32_t slot = F8 ? (gt + i) & 1 : ldv % NSLOT, ph = F8 ? ((gt + i) >> 1) & 1 : (ldv / NSLOT) & 1;
                const uint32_t v_full = bar(C::B_FULL + slot);      // (F8: V's readiness arrives on P_PFULL)
                const uint32_t v_empty = F8 ? bar(C::B_OPER + O_VEMPTY + slot) : bar(C::B_EMPTY + slot);
                const uint64_t vd = smem_desc_advance(v_desc, slot * SLOT_BYTES);
                const int nvp = pages_of_tile(i);
#pragma unroll
                for (int w = 0; w < NP; ++w) {
                    if (w < npipe) {
                        const uint32_t g = g0[w] + i, b = g & 1;
                        mbar_wait(pbar(w, P_PFULL + b), (g >> 1) & 1);
                        if (!F8 && w == 0) mbar_wait(v_full, ph);
                        if (i == 0 && jw[w] > 0) mbar_wait(pbar(w, P_OFREE), (jw[w] - 1) & 1);
                        tc_fence_after();
                        const uint32_t tO = tbase + w * PIPE_COLS;
                        const uint32_t tP = tO + 128 + 64 * b;
                        if (elect_one()) {
                            mma_ts(tO, tP, vd, ID_PV, i > 0);
#pragma unroll
                            for (int pg = 1; pg < TILE_PAGES; ++pg)
                                if (pg < nvp) mma_ts(tO, tP + pg * 8, smem_desc_advance(vd, pg * HEAD_BLOCK), ID_PV, 1);
                            mma_commit(pbar(w, P_PVDONE + b));
                            if (w == npipe - 1) mma_commit(v_empty);
                        }
                        __syncwarp();
                    }
                }
            }
            gt += n_tiles;
#pragma unroll
            for (int w = 0; w < NP; ++w)
                if (w < npipe) { g0[w] += n_tiles; jw[w]++; }
        }
    } else if (F8 && warp >= 2 + C::N_SOFTMAX / 32) {
        // ================================ converter warps (FP8-KV) ================================
        // Warp cw widens pages cw and cw + 2 of every landed V tile, e4m3 -> fp16 (exact), into V operand
        // slot (tile & 1): the block image the bf16 path stages directly (swz_chunk_off(2, ...)).  The e4m3
        // block is 16 rows of 128 bytes, 16-byte chunks XOR-swizzled by (row & 7); a quarter warp takes one
        // chunk column of 8 rows, which is conflict-free for the loads and for the stores.  Rows of a
        // partially filled last page are written as zeros (pool memory may hold NaN codes).  A tile's
        // loads are issued before the warp waits for its operand slot and the landing slot is released as
        // soon as they have arrived.  (K is not widened: the S MMAs read the landed e4m3 tile.)
        const int cw = warp - (2 + C::N_SOFTMAX / 32);
        uint32_t ct = 0;                                  // tiles of all items so far
        for (int idx = item_begin; idx < item_end; ++idx) {
            const WorkItem it = load_item(P.items, idx, P.seq_len);
            const int n_tok = it.tok1 - it.tok0;
            const int n_tiles = (n_tok + TILE_TOKENS - 1) / TILE_TOKENS;
            for (int i = 0; i < n_tiles; ++i, ++ct) {
                const int nv = min(TILE_TOKENS, n_tok - i * TILE_TOKENS);
                const int np = (nv + PS - 1) / PS;
                const uint32_t ld = 2 * ct + 1, slot = ld % NSLOT, ph = (ld / NSLOT) & 1, vb = ct & 1;
                mbar_wait(bar(C::B_FULL + slot), ph);
                const uint8_t *src = smem + C::RING_OFF + slot * C::RING_SLOT;
                uint8_t *dst = smem + C::OPER_OFF + vb * SLOT_BYTES;
                uint4 v[2][4];
#pragma unroll
                for (int u = 0; u < 2; ++u)
#pragma unroll
                    for (int q4 = 0; q4 < 4; ++q4) {
                        const int pg = cw + 2 * u, row = (lane & 7) + 8 * (q4 & 1), c8 = (lane >> 3) + 4 * (q4 >> 1);
                        v[u][q4] = pg < np ? *reinterpret_cast<const uint4 *>(src + pg * (HEAD_BLOCK / 2) + row * 128 +
                                                                              ((c8 ^ (row & 7)) << 4))
                                           : make_uint4(0, 0, 0, 0);
                    }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar(C::B_EMPTY + slot));      // the landing slot is free again
                mbar_wait(bar(C::B_OPER + O_VEMPTY + vb), ((ct >> 1) & 1) ^ 1);
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const int pg = cw + 2 * u;
                    if (pg >= np) continue;
                    const int valid = (pg == np - 1 && (nv & (PS - 1))) ? (nv & (PS - 1)) : PS;
#pragma unroll
                    for (int q4 = 0; q4 < 4; ++q4) {
                        const int row = (lane & 7) + 8 * (q4 & 1), c8 = (lane >> 3) + 4 * (q4 >> 1);
                        uint4 a, b;
                        e4m3x4_to_f16x4(v[u][q4].x, a.x, a.y);
                        e4m3x4_to_f16x4(v[u][q4].y, a.z, a.w);
                        e4m3x4_to_f16x4(v[u][q4].z, b.x, b.y);
                        e4m3x4_to_f16x4(v[u][q4].w, b.z, b.w);
                        if (row >= valid) a = b = make_uint4(0, 0, 0, 0);
                        *reinterpret_cast<uint4 *>(dst + pg * HEAD_BLOCK + swz_chunk_off(2, row, 2 * c8)) = a;
                        *reinterpret_cast<uint4 *>(dst + pg * HEAD_BLOCK + swz_chunk_off(2, row, 2 * c8 + 1)) = b;
                    }
                }
                fence_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive(pbar(0, P_PFULL + vb));
            }
        }
    } else {
        // ================================ softmax warps ================================
        const int w = NP > 1 ? (warp - 2) >> 2 : 0;    // pipe: rows [128 w, 128 w + 128) of the item
        const int h = SP > 1 ? (warp - 2) >> 2 : 0;    // SP = 2: which 32 of a tile's 64 scores this thread owns
        const int lg = warp & 3;                       // TMEM lane group this warp may access
        const int r = w * 128 + lg * 32 + lane;        // query row of the item owned by this thread
        const uint32_t lane_addr = (uint32_t)(lg * 32) << 16;
        const uint32_t tO = tbase + w * PIPE_COLS;
        const int st = threadIdx.x - 64;               // 0 .. N_SOFTMAX-1 among the softmax threads
        uint32_t g0 = 0, gt = 0;                       // tiles this pipe has run / tiles of all items so far
        // Q rows of an item -> smem (K-major, 128-byte swizzle); rows beyond nrows are zero.  Each pipe
        // stages its own 128 rows.  All 16 loads of a thread are in flight together.  Called for the
        // NEXT item as soon as this thread has seen the last S of the current item complete (its Q
        // image is then dead), i.e. before the epilogue: the global-load latency and the next item's
        // first S MMA hide under the last P V and the write-back of the partials.
        auto stage_q = [&](const WorkItem &qi, int parity) {
            const int c = st & 15;                     // 16-byte chunk of the row
            constexpr int QT = 128 * SP, NK = 16 / SP;  // threads staging one pipe's image, rows per thread
            uint4 v[NK];
#pragma unroll
            for (int k = 0; k < NK; ++k) {
                const int row = w * 128 + ((st & (QT - 1)) >> 4) + (QT / 16) * k;
                v[k] = make_uint4(0, 0, 0, 0);
                if (F8 && c == 0 && row >= qi.nrows) smem[C::QEXP_OFF + parity * 128 + (row & 127)] = 134;   // scale 1
                if (row < qi.nrows) {
                    const int lr = qi.rb0 + row;
                    const uint16_t *src =
                        P.q + ((size_t)item_qrow(qi, P.rowmap, lr, P.G) * P.Hq + qi.kvh * P.G + lr % P.G) * D + c * 8;
                    v[k] = *reinterpret_cast<const uint4 *>(src);
                    if constexpr (F8) {
                        // bf16 -> two e4m3 terms, q * 2^s = hi + lo: the row is first scaled by the power of two
                        // that brings its largest magnitude into [128, 256) (e4m3 tops out at 448; the softmax
                        // thread of the row undoes it in its score scale), hi = the scaled q rounded to e4m3
                        // (4 significant bits), lo = the residual, again e4m3: exact for a bf16 q (8 significant
                        // bits) down to elements 2^-17 of the row's largest.  The 8 hi bytes go to v[k].x/.y,
                        // the 8 lo bytes to v[k].z/.w.
                        const uint32_t *u = reinterpret_cast<const uint32_t *>(&v[k]);
                        float mx = 0.f;
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            mx = fmaxf(mx, fmaxf(fabsf(__uint_as_float(u[e] << 16)), fabsf(__uint_as_float(u[e] & 0xffff0000u))));
#pragma unroll
                        for (int o = 1; o < 16; o <<= 1)       // the row's 16 chunks = one half warp (the other half may sit this row out)
                            mx = fmaxf(mx, __shfl_xor_sync(lane < 16 ? 0x0000ffffu : 0xffff0000u, mx, o));
                        uint32_t eb = (__float_as_uint(mx) >> 23) & 0xffu;       // biased exponent of the row maximum
                        eb = min(max(eb, 32u), 220u);                            // (zero / tiny / huge rows: a harmless scale)
                        const float qs = __uint_as_float((261u - eb) << 23);    // 2^(7 - e)
                        if (c == 0) smem[C::QEXP_OFF + parity * 128 + row] = (uint8_t)eb;
                        uint32_t hi8[2], lo8[2];
#pragma unroll
                        for (int e2 = 0; e2 < 2; ++e2) {
                            float f[4], g[4];
                            f[0] = __uint_as_float(u[2 * e2] << 16) * qs;
                            f[1] = __uint_as_float(u[2 * e2] & 0xffff0000u) * qs;
                            f[2] = __uint_as_float(u[2 * e2 + 1] << 16) * qs;
                            f[3] = __uint_as_float(u[2 * e2 + 1] & 0xffff0000u) * qs;
                            const uint32_t h = pack_e4m3(f[0], f[1]) | (pack_e4m3(f[2], f[3]) << 16);
                            uint32_t h01, h23;
                            e4m3x4_to_f16x4(h, h01, h23);
                            unpack_f16(h01, g[0], g[1]);
                            unpack_f16(h23, g[2], g[3]);
                            hi8[e2] = h;
                            lo8[e2] = pack_e4m3(f[0] - g[0], f[1] - g[1]) | (pack_e4m3(f[2] - g[2], f[3] - g[3]) << 16);
                        }
                        v[k] = make_uint4(hi8[0], hi8[1], lo8[0], lo8[1]);
                    }
                }
            }
#pragma unroll
            for (int k = 0; k < NK; ++k) {
                const int rp = ((st & (QT - 1)) >> 4) + (QT / 16) * k;   // row inside the pipe's 32 KiB image
                if constexpr (F8) {
                    // e4m3 images: rows of 128 bytes (all 128 dims), 16-byte chunks XOR-swizzled by the row;
                    // chunk c of the bf16 row (8 dims) is half of e4m3 chunk c / 2; hi image, lo image 16 KiB on
                    const int off = (rp >> 3) * 1024 + (rp & 7) * 128 + ((((c >> 1) & 7) ^ (rp & 7)) << 4) + (c & 1) * 8;
                    *reinterpret_cast<uint2 *>(smem + off) = make_uint2(v[k].x, v[k].y);
                    *reinterpret_cast<uint2 *>(smem + Q_HALF + off) = make_uint2(v[k].z, v[k].w);
                    continue;
                }
                const int off = w * Q_BYTES + (c >> 3) * Q_HALF + (rp >> 3) * 1024 + (rp & 7) * 128 +
                                (((c & 7) ^ (rp & 7)) << 4);
                *reinterpret_cast<uint4 *>(smem + off) = v[k];
            }
            fence_async_smem();
            asm volatile("bar.sync 1, %0;" ::"n"(C::N_SOFTMAX) : "memory");
            if (st == 0) mbar_arrive(bar(C::B_QFULL));
        };
        if (item_begin < item_end) stage_q(P.items[item_begin], 0);
        for (int idx = item_begin; idx < item_end; ++idx) {
            const WorkItem it = load_item(P.items, idx, P.seq_len);
            const bool has_next = idx + 1 < item_end;
            const int n_tok = it.tok1 - it.tok0;
            const int n_tiles = (n_tok + TILE_TOKENS - 1) / TILE_TOKENS;
            // 0: this pipe sits the item out (NP = 2, <= 128 rows: the MMA warp knows); 1: none of this warp's
            // 32 rows exists (few-row item): only keep the barriers moving, whatever S/P/O hold in these
            // lanes never leaves TMEM; 2: softmax
            const int mode = (NP > 1 && w * 128 >= it.nrows) ? 0 : (w * 128 + lg * 32 >= it.nrows ? 1 : 2);
            const int lim_r = it.lim0 + (it.rb0 + r) / P.G;
            const int min_lim = it.lim0 + (it.rb0 + w * 128) / P.G;
            float m_used = -INFINITY, l = 0.f, lr = 0.f;   // l: exact row sum (lse); lr: sum of the bf16 weights
            // score scale of this thread's row (log2 domain); F8: times the inverse of the row's Q scaling
            float scale_log2 = P.scale_log2;
            if constexpr (F8) {
                const uint32_t eb = smem[C::QEXP_OFF + ((idx - item_begin) & 1) * 128 + (r & 127)];
                scale_log2 *= __uint_as_float((eb - 7u) << 23);                  // 2^(e - 7)
            }

            if (mode == 1) {
                for (int i = 0; i < n_tiles; ++i) {
                    const uint32_t g = g0 + i, b = g & 1;
                    mbar_wait(pbar(w, P_SFULL + b), (g >> 1) & 1);
                    if (lane == 0) mbar_arrive(pbar(w, P_PFULL + b));
                    __syncwarp();
                }
            }

            if constexpr (SP == 2) {
                // ---- split rows: this thread owns scores [32 h, 32 h + 32) of its row in every tile ----
                float *xch = reinterpret_cast<float *>(smem + C::XCH_OFF);      // [2][2][128]
                auto pair_sync = [&]() {                 // the two warps that share TMEM lane group lg
                    asm volatile("bar.sync %0, 64;" ::"r"(2 + lg) : "memory");
                };
                const int rr = lg * 32 + lane;
                for (int i = 0; mode == 2 && i < n_tiles; ++i) {
                    const uint32_t g = g0 + i, b = g & 1;
                    const uint32_t tS = tO + 128 + 64 * b + lane_addr;
                    mbar_wait(pbar(w, P_SFULL + b), (g >> 1) & 1);
                    tc_fence_after();
                    uint32_t sc[32];
                    tmem_ld32(tS + 32 * h, sc);
                    tmem_wait_ld();
                    const int tile_t0 = it.tok0 + i * TILE_TOKENS;
                    const int nv = min(TILE_TOKENS, it.tok1 - tile_t0);
                    if (nv < TILE_TOKENS || tile_t0 + TILE_TOKENS - 1 > min_lim) {
                        const int vis = min(nv, lim_r - tile_t0 + 1) - 32 * h;
#pragma unroll
                        for (int t = 0; t < 32; ++t)
                            if (t >= vis) sc[t] = 0xff800000u;           // -inf
                    }
                    float mxa[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
#pragma unroll
                    for (int t = 0; t < 32; ++t) mxa[t & 3] = fmaxf(mxa[t & 3], __uint_as_float(sc[t]));
                    float mx = fmaxf(fmaxf(mxa[0], mxa[1]), fmaxf(mxa[2], mxa[3]));
                    // row max over both halves (double buffered by tile parity: a thread is at most one
                    // pair barrier ahead of its partner)
                    xch[((g & 1) * 2 + h) * 128 + rr] = mx;
                    pair_sync();
                    mx = fmaxf(mx, xch[((g & 1) * 2 + (h ^ 1)) * 128 + rr]);
                    const float mxs = mx * P.scale_log2;
                    const bool grow = mxs > m_used + RESCALE_THRESHOLD;
                    if (__any_sync(0xffffffffu, grow)) {          // same rows, same values: both halves agree
                        const float m_new = grow ? mxs : m_used;
                        const float alpha = grow ? (m_used == -INFINITY ? 0.f : ex2(m_used - m_new)) : 1.f;
                        l *= alpha;
                        lr *= alpha;
                        if (i > 0) {
                            mbar_wait(pbar(w, P_PVDONE + ((g - 1) & 1)), ((g - 1) >> 1) & 1);
                            tc_fence_after();
#pragma unroll 1
                            for (int cb = 2 * h; cb < 2 * h + 2; ++cb) {     // this half's 64 columns of O
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
                    uint32_t p[16];
                    float sum0 = 0.f, sum1 = 0.f, rs0 = 0.f, rs1 = 0.f;
#pragma unroll
                    for (int t = 0; t < 8; ++t) {
                        const float a0 = ex2(fmaf(__uint_as_float(sc[4 * t]), P.scale_log2, -mu));
                        const float a1 = ex2(fmaf(__uint_as_float(sc[4 * t + 1]), P.scale_log2, -mu));
                        const float c0 = ex2(fmaf(__uint_as_float(sc[4 * t + 2]), P.scale_log2, -mu));
                        const float c1 = ex2(fmaf(__uint_as_float(sc[4 * t + 3]), P.scale_log2, -mu));
                        p[2 * t] = pack_bf16(a0, a1);
                        p[2 * t + 1] = pack_bf16(c0, c1);
                        sum0 += a0 + a1;
                        sum1 += c0 + c1;
                        rs0 += __uint_as_float(p[2 * t] << 16) + __uint_as_float(p[2 * t] & 0xffff0000u);
                        rs1 += __uint_as_float(p[2 * t + 1] << 16) + __uint_as_float(p[2 * t + 1] & 0xffff0000u);
                    }
                    l += sum0 + sum1;
                    lr += rs0 + rs1;
                    // P columns [16 h, 16 h + 16) lie over S columns both halves have already read
                    tmem_st16(tS + 16 * h, p);
                    tmem_wait_st();
                    if ((nv & (PS - 1)) && lg == 0 && h == 0) {
                        const uint32_t ldv = 2 * (gt + i) + 1, slot = ldv % NSLOT, ph = (ldv / NSLOT) & 1;
                        mbar_wait(bar(C::B_FULL + slot), ph);
                        const int nvp = (nv + PS - 1) / PS;
                        uint8_t *vpage = smem + C::RING_OFF + slot * SLOT_BYTES + (nvp - 1) * HEAD_BLOCK;
                        const int r_first = nv & (PS - 1);
                        for (int e = lane; e < (PS - r_first) * 16; e += 32) {
                            const int r2 = r_first + (e >> 4), cc = e & 15;
                            *reinterpret_cast<uint4 *>(vpage + swz_chunk_off(2, r2, cc)) = make_uint4(0, 0, 0, 0);
                        }
                        fence_async_smem();
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(pbar(w, P_PFULL + b));
                }
                if (has_next) stage_q(P.items[idx + 1], (idx + 1 - item_begin) & 1);
                if (mode == 1) {
                    const uint32_t gl = g0 + n_tiles - 1;
                    mbar_wait(pbar(w, P_PVDONE + (gl & 1)), (gl >> 1) & 1);
                    if (lane == 0) mbar_arrive(pbar(w, P_OFREE));
                    __syncwarp();
                }
                if (mode == 2) {
                    const uint32_t gl = g0 + n_tiles - 1;
                    mbar_wait(pbar(w, P_PVDONE + (gl & 1)), (gl >> 1) & 1);
                    tc_fence_after();
                    pair_sync();                                   // the partner has read the last row max
                    xch[(0 * 2 + h) * 128 + rr] = l;
                    xch[(1 * 2 + h) * 128 + rr] = lr;
                    pair_sync();
                    l += xch[(0 * 2 + (h ^ 1)) * 128 + rr];
                    lr += xch[(1 * 2 + (h ^ 1)) * 128 + rr];
                    pair_sync();                                   // ... before the next item's first tile
                    const float inv = lr > 0.f ? 1.f / lr : 0.f;
                    float *dst = P.ws_o + (size_t)(it.part_base + r) * D;
                    if (P.wait_prev && idx == item_begin) asm volatile("griddepcontrol.wait;" ::: "memory");
#pragma unroll 1
                    for (int cb = 2 * h; cb < 2 * h + 2; ++cb) {
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
                    if (r < it.nrows && h == 0)
                        P.ws_lse[it.part_base + r] = l > 0.f ? (m_used + log2f(l)) * LN2 : -INFINITY;
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(pbar(w, P_OFREE));
                }
                if (mode != 0) g0 += n_tiles;
                gt += n_tiles;
            } else {

            for (int i = 0; mode == 2 && i < n_tiles; ++i) {
                const uint32_t g = g0 + i, b = g & 1;
                const uint32_t tS = tO + 128 + 64 * b + lane_addr;
                mbar_wait(pbar(w, P_SFULL + b), (g >> 1) & 1);
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
                float mxa[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};   // 4 independent chains
#pragma unroll
                for (int t = 0; t < 32; ++t)
                    mxa[t & 3] = fmaxf(mxa[t & 3], fmaxf(__uint_as_float(s0[t]), __uint_as_float(s1[t])));
                const float mx = fmaxf(fmaxf(mxa[0], mxa[1]), fmaxf(mxa[2], mxa[3]));
                const float mxs = mx * scale_log2;
                const bool grow = mxs > m_used + RESCALE_THRESHOLD;
                if (__any_sync(0xffffffffu, grow)) {
                    const float m_new = grow ? mxs : m_used;
                    const float alpha = grow ? (m_used == -INFINITY ? 0.f : ex2(m_used - m_new)) : 1.f;
                    l *= alpha;
                    lr *= alpha;
                    if (i > 0) {
                        // O holds tiles [0, i): wait for P V(i - 1), rescale this thread's row
                        mbar_wait(pbar(w, P_PVDONE + ((g - 1) & 1)), ((g - 1) >> 1) & 1);
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
                // packed fp32 pairs for the scale, the exact sum and the sum of the rounded weights
                float se0 = 0.f, se1 = 0.f, se2 = 0.f, se3 = 0.f, sr0 = 0.f, sr1 = 0.f, sr2 = 0.f, sr3 = 0.f;
                const float nmu = -mu;
#pragma unroll
                for (int t = 0; t < 16; ++t) {
                    float x0, x1, y0, y1;
                    ffma2(x0, x1, __uint_as_float(s0[2 * t]), __uint_as_float(s0[2 * t + 1]), scale_log2, nmu);
                    ffma2(y0, y1, __uint_as_float(s1[2 * t]), __uint_as_float(s1[2 * t + 1]), scale_log2, nmu);
                    float a0, a1, c0, c1;
                    if (emulated_pair(2 * t)) ex2_poly2(x0, x1, a0, a1); else { a0 = ex2(x0); a1 = ex2(x1); }
                    if (emulated_pair(2 * t + 1)) ex2_poly2(y0, y1, c0, c1); else { c0 = ex2(y0); c1 = ex2(y1); }
                    p[t] = F8 ? pack_f16(a0, a1) : pack_bf16(a0, a1);
                    p[16 + t] = F8 ? pack_f16(c0, c1) : pack_bf16(c0, c1);
                    // o is normalised by the sum of the ROUNDED weights the tensor core uses, so that
                    // o = sum(p v) / sum(p) stays a true weighted mean (a one-hot row returns V exactly
                    // even when the running max is stale and p is not a power of two); lse keeps the
                    // exact sum
                    fadd2(se0, se1, a0, a1);
                    fadd2(se2, se3, c0, c1);
                    if constexpr (F8) {
                        float r0, r1, r2, r3;
                        unpack_f16(p[t], r0, r1);
                        unpack_f16(p[16 + t], r2, r3);
                        fadd2(sr0, sr1, r0, r1);
                        fadd2(sr2, sr3, r2, r3);
                    } else {
                    fadd2(sr0, sr1, __uint_as_float(p[t] << 16), __uint_as_float(p[t] & 0xffff0000u));
                    fadd2(sr2, sr3, __uint_as_float(p[16 + t] << 16), __uint_as_float(p[16 + t] & 0xffff0000u));
                    }
                }
                l += (se0 + se1) + (se2 + se3);
                lr += (sr0 + sr1) + (sr2 + sr3);
                tmem_st32(tS, p);
                tmem_wait_st();
                if (!F8 && (nv & (PS - 1)) && w == 0 && lg == 0) {
                    // the last staged page is partially filled: its tail rows hold whatever the pool
                    // held (possibly NaN patterns).  P is 0 there; make V 0 as well.  The warp of rows
                    // 0..31 does it (active in every item); the MMA thread issues pipe 0's P V, which
                    // waits for this warp, before any other pipe's.
                    const uint32_t ldv = 2 * (gt + i) + 1, slot = ldv % NSLOT, ph = (ldv / NSLOT) & 1;
                    mbar_wait(bar(C::B_FULL + slot), ph);
                    const int nvp = (nv + PS - 1) / PS;
                    uint8_t *vpage = smem + C::RING_OFF + slot * SLOT_BYTES + (nvp - 1) * HEAD_BLOCK;
                    const int r_first = nv & (PS - 1);
                    for (int e = lane; e < (PS - r_first) * 16; e += 32) {
                        const int rr = r_first + (e >> 4), cc = e & 15;
                        *reinterpret_cast<uint4 *>(vpage + swz_chunk_off(2, rr, cc)) = make_uint4(0, 0, 0, 0);
                    }
                    fence_async_smem();
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(pbar(w, P_PFULL + b));
            }

            if (has_next) stage_q(P.items[idx + 1], (idx + 1 - item_begin) & 1);

            if (mode == 1) {
                const uint32_t gl = g0 + n_tiles - 1;
                mbar_wait(pbar(w, P_PVDONE + (gl & 1)), (gl >> 1) & 1);
                if (lane == 0) mbar_arrive(pbar(w, P_OFREE));
                __syncwarp();
            }
            // ---- epilogue: O / l -> partial rows ------------------------------------------------
            if (mode == 2) {
                const uint32_t gl = g0 + n_tiles - 1;
                mbar_wait(pbar(w, P_PVDONE + (gl & 1)), (gl >> 1) & 1);
                tc_fence_after();
                const float inv = lr > 0.f ? 1.f / lr : 0.f;
                float *dst = P.ws_o + (size_t)(it.part_base + r) * D;
                if (P.wait_prev && idx == item_begin) asm volatile("griddepcontrol.wait;" ::: "memory");
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
                if (lane == 0) mbar_arrive(pbar(w, P_OFREE));
            }
            if (mode != 0) g0 += n_tiles;
            gt += n_tiles;
            }   // SP == 1
        }
    }

    // ---- teardown: every MMA has completed (the softmax warps waited for the last P V) ----
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tbase, C::TMEM_COLS);
    }
    // When launched programmatically behind another attention kernel this grid may start before
    // that one has finished; do not complete before it has, so that merge_kernel (which waits for
    // the LAST attention grid) sees every kernel's partials.  A no-op for a normal launch.
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

}  // namespace

namespace spork {

// variant 0: one pipe (the default kernel), 1: two pipes, 2: one pipe with split rows
int attn_umma_grid(spork_ctx *c, int variant) {
    return c->num_sms * (variant == 1 ? Cfg<2, 1>::CTAS_PER_SM : Cfg<1, 1>::CTAS_PER_SM);
}

template <int NP, int SP, bool F8 = false>
static int launch_np(spork_ctx *c, const UParams &p, int grid, bool programmatic, cudaStream_t st) {
    constexpr uint32_t bit = 1u << (F8 ? 3 : (NP == 2 ? 1 : (SP == 2 ? 2 : 0)));
    if (!(c->smem_attr_done & bit)) {      // per handle (= per device), not per process
        SPORK_CUDA(cudaFuncSetAttribute(attn_umma_kernel<NP, SP, F8>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        Cfg<NP, SP, F8>::SMEM_BYTES));
        c->smem_attr_done |= bit;
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(Cfg<NP, SP, F8>::N_THREADS);
    cfg.dynamicSmemBytes = Cfg<NP, SP, F8>::SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = programmatic ? 1 : 0;   // may start while the previous kernel drains
    SPORK_CUDA(cudaLaunchKernelEx(&cfg, attn_umma_kernel<NP, SP, F8>, p));
    c->last_launches++;
    SPORK_CUDA(cudaGetLastError());
    return SPORK_OK;
}

// np = 2: the many-row items' list (launched first; two-pipe or split-row kernel), np = 1: the others
int launch_attn_umma(spork_ctx *c, const LayerIO &io, int np, bool programmatic, bool wait_prev, cudaStream_t st) {
    const Plan &P = c->plan;
    const int n = np == 2 ? P.n_items_umma2 : P.n_items_umma;
    if (n == 0) return SPORK_OK;
    UParams p;
    // item lists: [mma.sync][tcgen05 NP=1][tcgen05 NP=2]; cta_ptr arrays in the same order
    p.items = P.d_items + P.n_items + (np == 2 ? P.n_items_umma : 0);
    p.cta_ptr = P.d_cta_ptr + (P.grid + 1) + (np == 2 ? P.grid_umma + 1 : 0);
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
    p.wait_prev = wait_prev ? 1 : 0;
    if (c->cfg.dtype == SPORK_E4M3) return np == 1 ? launch_np<1, 1, true>(c, p, P.grid_umma, programmatic, st) : SPORK_ERR_INVALID;
    if (np == 1) return launch_np<1, 1>(c, p, P.grid_umma, programmatic, st);
    return P.variant2 == 2 ? launch_np<1, 2>(c, p, P.grid_umma2, programmatic, st)
                           : launch_np<2, 1>(c, p, P.grid_umma2, programmatic, st);
}

}  // namespace spork
