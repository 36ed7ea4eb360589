// libspork: LSE-weighted combination of one (q row, q head)'s partials by one warp.
//   M = max lse_s, w_s = exp(lse_s - M), out = sum w_s o_s / sum w_s, lse = M + ln sum w_s
// An empty partial has lse = -inf and weight 0; no partial at all: out = 0, lse = -inf.
// A row's partials come from up to MAX_ROW_REFS segments (one per cascade level it shares with other
// members of its fork group, plus its private tail), each cut into `nsplit` pieces.
// The partials were written by the attention kernel(s) just before and sit in L2: every
// partial is read once, with ld.global.cg.
#pragma once

#include <math.h>

#include "spork_internal.h"

namespace spork {

__device__ __forceinline__ float merge_warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// The splits of one row, flattened over its refs.  Lane i < nref holds ref i: the partial row of its
// split 0 (for GQA head j of the row's kv head), its number of splits and their stride.
struct RowSplits {
    int base, nsplit, stride, cum_end;   // per lane (ref `lane`)
    int nref, total;                     // warp-uniform
};
__device__ __forceinline__ RowSplits load_row_splits(const QRowDesc &d, const RowRef *__restrict__ refs,
                                                     const StreamDesc *__restrict__ streams, int kvh, int lane) {
    RowSplits r;
    r.nref = d.nref;
    r.base = 0;
    r.nsplit = 0;
    r.stride = 0;
    if (lane < d.nref) {
        const RowRef ref = refs[d.ref0 + lane];
        const StreamDesc sd = streams[ref.stream + kvh];
        r.base = sd.part_base + ref.off;       // GQA head 0 of the row
        r.nsplit = sd.nsplit;
        r.stride = sd.stride;
    }
    int x = r.nsplit;                    // inclusive scan over the (<= 8) refs
#pragma unroll
    for (int o = 1; o < MAX_ROW_REFS; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    r.cum_end = x;
    r.total = __shfl_sync(0xffffffffu, x, MAX_ROW_REFS - 1);
    return r;
}
// partial row of split s of GQA head j (every lane may ask for a different s; all lanes must call);
// -1 beyond the end
__device__ __forceinline__ int split_row(const RowSplits &r, int s, int j) {
    int row = -1;
    for (int i = 0; i < r.nref; ++i) {
        const int ce = __shfl_sync(0xffffffffu, r.cum_end, i), ns = __shfl_sync(0xffffffffu, r.nsplit, i);
        const int b = __shfl_sync(0xffffffffu, r.base, i), st = __shfl_sync(0xffffffffu, r.stride, i);
        if (s >= ce - ns && s < ce) row = b + (s - (ce - ns)) * st + j;
    }
    return row;
}

// Lane s owns the weight of split s; the partial rows are fetched 8 splits at a time with
// every load of a batch in flight before the first use (pure L2 latency otherwise).
template <int NI>   // float4 per lane per row: 1 for D <= 128, 2 for D <= 256
__device__ __forceinline__ void merge_row(const RowSplits &rs, int j, int D, const float *ws_o, const float *ws_lse,
                                          float *out_row, float *lse_out, int lane) {
    const int n = rs.total;
    const int row_first = split_row(rs, lane, j);                 // split `lane`
    const float lse_first = row_first >= 0 ? __ldcg(ws_lse + row_first) : -INFINITY;
    float M = lse_first;
    for (int s0 = 32; s0 < n; s0 += 32) {
        const int row = split_row(rs, s0 + lane, j);
        if (row >= 0) M = fmaxf(M, __ldcg(ws_lse + row));
    }
    M = merge_warp_max(M);
    const int nv = D >> 2;                        // float4 per row (<= 64)
    float4 *o = reinterpret_cast<float4 *>(out_row);
    if (M == -INFINITY) {
        for (int c = lane; c < nv; c += 32) o[c] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (lane == 0) *lse_out = -INFINITY;
        return;
    }
    float4 acc[NI];
#pragma unroll
    for (int i = 0; i < NI; ++i) acc[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    float W = 0.f;
    for (int s0 = 0; s0 < n; s0 += 32) {
        const int nb = min(32, n - s0);
        const int row_l = s0 == 0 ? row_first : split_row(rs, s0 + lane, j);
        const float wl = row_l >= 0 ? expf((s0 == 0 ? lse_first : __ldcg(ws_lse + row_l)) - M) : 0.f;
        for (int b0 = 0; b0 < nb; b0 += 8) {
            float4 v[NI][8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int row = __shfl_sync(0xffffffffu, row_l, (b0 + u) & 31);   // -1 beyond the last split
                const float4 *po = reinterpret_cast<const float4 *>(ws_o + (size_t)max(row, 0) * D);
#pragma unroll
                for (int i = 0; i < NI; ++i) {
                    const int c = lane + 32 * i;
                    v[i][u] = (row >= 0 && b0 + u < nb && c < nv) ? __ldcg(po + c) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const float ws = b0 + u < nb ? __shfl_sync(0xffffffffu, wl, (b0 + u) & 31) : 0.f;
                W += ws;
#pragma unroll
                for (int i = 0; i < NI; ++i) {
                    acc[i].x = fmaf(ws, v[i][u].x, acc[i].x);
                    acc[i].y = fmaf(ws, v[i][u].y, acc[i].y);
                    acc[i].z = fmaf(ws, v[i][u].z, acc[i].z);
                    acc[i].w = fmaf(ws, v[i][u].w, acc[i].w);
                }
            }
        }
    }
    const float inv = 1.f / W;
#pragma unroll
    for (int i = 0; i < NI; ++i) {
        const int c = lane + 32 * i;
        if (c < nv) o[c] = make_float4(acc[i].x * inv, acc[i].y * inv, acc[i].z * inv, acc[i].w * inv);
    }
    if (lane == 0) *lse_out = M + logf(W);
}

// The same combine for JB consecutive GQA heads of one (q row, kv head) at once -- their partial rows
// are contiguous (JB x D floats per split), so one warp streams JB * 512 B per split with every load
// of a split in flight: one descriptor fetch and JB times the memory-level parallelism per warp.
// JB is a power of two <= 8; lane `e` of a batch owns the weight of (split e / JB, head e % JB).
// The JB heads start at GQA head j0.
template <int NI, int JB>
__device__ __forceinline__ void merge_heads(const RowSplits &rs, int j0, int D, const float *ws_o, const float *ws_lse,
                                            float *out_rows, float *lse_out, int lane) {
    const int n = rs.total;
    constexpr int SB = 32 / JB;                 // splits per batch of 32 lanes
    const int jj = lane % JB, sl = lane / JB;
    // ---- row maxima ----
    float M = -INFINITY;
    for (int s0 = 0; s0 < n; s0 += SB) {
        const int row = split_row(rs, s0 + sl, j0);
        if (row >= 0) M = fmaxf(M, __ldcg(ws_lse + row + jj));
    }
#pragma unroll
    for (int o = JB; o < 32; o <<= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));   // lanes of head jj
    const int nv = D >> 2;
    float4 acc[JB][NI];
    float W[JB];
#pragma unroll
    for (int k = 0; k < JB; ++k) {
        W[k] = 0.f;
#pragma unroll
        for (int i = 0; i < NI; ++i) acc[k][i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    for (int s0 = 0; s0 < n; s0 += SB) {
        const int row_l = split_row(rs, s0 + sl, j0);        // head j0's partial row of split s0 + sl
        const float wl = (row_l >= 0 && M != -INFINITY) ? expf(__ldcg(ws_lse + row_l + jj) - M) : 0.f;
        const int nb = min(SB, n - s0);
        for (int sb = 0; sb < nb; ++sb) {
            const int row = __shfl_sync(0xffffffffu, row_l, sb * JB);
            const float4 *po = reinterpret_cast<const float4 *>(ws_o + (size_t)row * D);
            float4 v[JB][NI];
#pragma unroll
            for (int k = 0; k < JB; ++k)
#pragma unroll
                for (int i = 0; i < NI; ++i) {
                    const int c = lane + 32 * i;
                    v[k][i] = c < nv ? __ldcg(po + (size_t)k * nv + c) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
#pragma unroll
            for (int k = 0; k < JB; ++k) {
                const float w = __shfl_sync(0xffffffffu, wl, sb * JB + k);
                W[k] += w;
#pragma unroll
                for (int i = 0; i < NI; ++i) {
                    acc[k][i].x = fmaf(w, v[k][i].x, acc[k][i].x);
                    acc[k][i].y = fmaf(w, v[k][i].y, acc[k][i].y);
                    acc[k][i].z = fmaf(w, v[k][i].z, acc[k][i].z);
                    acc[k][i].w = fmaf(w, v[k][i].w, acc[k][i].w);
                }
            }
        }
    }
#pragma unroll
    for (int k = 0; k < JB; ++k) {
        const float inv = W[k] > 0.f ? 1.f / W[k] : 0.f;     // no partial / all empty: out = 0
        float4 *o = reinterpret_cast<float4 *>(out_rows + (size_t)k * D);
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            const int c = lane + 32 * i;
            if (c < nv) o[c] = make_float4(acc[k][i].x * inv, acc[k][i].y * inv, acc[k][i].z * inv, acc[k][i].w * inv);
        }
        const float Mk = __shfl_sync(0xffffffffu, M, k);     // lane k holds head k's maximum
        if (lane == 0) lse_out[k] = W[k] > 0.f ? Mk + logf(W[k]) : -INFINITY;
    }
}

// Four consecutive GQA heads of one (q row, kv head), FOUR splits in flight: every partial row of a batch
// (4 splits x 4 heads x 512 B) and its lse are requested before anything is used, so a warp pays one memory
// round trip per four splits instead of one per split plus one for the maxima (the merge is pure latency:
// ncu showed 37 % long-scoreboard stalls at 20 warps per SM).  Batches are combined with a running maximum.
// Lane e < 16 owns the weight of (split e / 4, head e % 4).
template <int NI>
__device__ __forceinline__ void merge_heads4(const RowSplits &rs, int j0, int D, const float *ws_o, const float *ws_lse,
                                             float *out_rows, float *lse_out, int lane) {
    const int n = rs.total, nv = D >> 2;
    const int jj = lane & 3, sl = lane >> 2;
    float4 acc[4][NI];
    float W[4], M = -INFINITY;               // M: running maximum of head jj (the same on every lane with that jj)
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        W[k] = 0.f;
#pragma unroll
        for (int i = 0; i < NI; ++i) acc[k][i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    for (int s0 = 0; s0 < n; s0 += 4) {
        const int row_l = split_row(rs, s0 + sl, j0);                 // head j0's partial row of split s0 + sl
        const bool mine = sl < 4 && row_l >= 0;
        const float lse_l = mine ? __ldcg(ws_lse + row_l + jj) : -INFINITY;
        float4 v[4][4][NI];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int row = __shfl_sync(0xffffffffu, row_l, u * 4);
            const float4 *po = reinterpret_cast<const float4 *>(ws_o + (size_t)max(row, 0) * D);
#pragma unroll
            for (int k = 0; k < 4; ++k)
#pragma unroll
                for (int i = 0; i < NI; ++i) {
                    const int c = lane + 32 * i;
                    v[u][k][i] = (row >= 0 && c < nv) ? __ldcg(po + (size_t)k * nv + c) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
        }
        float m = lse_l;
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
        const float M_new = fmaxf(M, m);
        const float alpha_l = (M == -INFINITY) ? 0.f : expf(M - M_new);     // M_new = -inf: nothing yet, acc = 0 anyway
        const float w_l = (mine && M_new != -INFINITY) ? expf(lse_l - M_new) : 0.f;
        M = M_new;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float alpha = __shfl_sync(0xffffffffu, alpha_l, k);
            W[k] *= alpha;
#pragma unroll
            for (int i = 0; i < NI; ++i) {
                acc[k][i].x *= alpha; acc[k][i].y *= alpha; acc[k][i].z *= alpha; acc[k][i].w *= alpha;
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float w = __shfl_sync(0xffffffffu, w_l, u * 4 + k);
                W[k] += w;
#pragma unroll
                for (int i = 0; i < NI; ++i) {
                    acc[k][i].x = fmaf(w, v[u][k][i].x, acc[k][i].x);
                    acc[k][i].y = fmaf(w, v[u][k][i].y, acc[k][i].y);
                    acc[k][i].z = fmaf(w, v[u][k][i].z, acc[k][i].z);
                    acc[k][i].w = fmaf(w, v[u][k][i].w, acc[k][i].w);
                }
            }
        }
    }
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float inv = W[k] > 0.f ? 1.f / W[k] : 0.f;     // no partial / all empty: out = 0
        float4 *o = reinterpret_cast<float4 *>(out_rows + (size_t)k * D);
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            const int c = lane + 32 * i;
            if (c < nv) o[c] = make_float4(acc[k][i].x * inv, acc[k][i].y * inv, acc[k][i].z * inv, acc[k][i].w * inv);
        }
        const float Mk = __shfl_sync(0xffffffffu, M, k);     // lane k holds head k's maximum
        if (lane == 0) lse_out[k] = W[k] > 0.f ? Mk + logf(W[k]) : -INFINITY;
    }
}

}  // namespace spork
