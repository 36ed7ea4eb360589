// libspork: LSE-weighted combination of one (q row, q head)'s partials by one warp.
//   M = max lse_s, w_s = exp(lse_s - M), out = sum w_s o_s / sum w_s, lse = M + ln sum w_s
// An empty partial has lse = -inf and weight 0; no partial at all: out = 0, lse = -inf.
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

// Lane s owns the weight of split s; the partial rows are fetched 8 splits at a time with
// every load of a batch in flight before the first use (pure L2 latency otherwise).
// The two streams a row draws its partials from (none: nsplit = 0).
struct RowStreams {
    StreamDesc pre, suf;
};
__device__ __forceinline__ RowStreams load_row_streams(const StreamDesc *__restrict__ streams, const QRowDesc &d,
                                                       int kvh) {
    RowStreams r{{0, 0, 0, 0}, {0, 0, 0, 0}};
    if (d.pre_stream >= 0) r.pre = streams[d.pre_stream + kvh];
    if (d.suf_stream >= 0) r.suf = streams[d.suf_stream + kvh];
    return r;
}

template <int NI>   // float4 per lane per row: 1 for D <= 128, 2 for D <= 256
__device__ __forceinline__ void merge_row(const RowStreams &rs, const QRowDesc &d, int j, int D,
                                          const float *ws_o, const float *ws_lse, float *out_row,
                                          float *lse_out, int lane) {
    const StreamDesc &pre = rs.pre, &suf = rs.suf;
    const int pre0 = pre.part_base + d.pre_off + j;
    const int suf0 = suf.part_base + d.suf_off + j;
    const int n = pre.nsplit + suf.nsplit;
    auto part = [&](int s) -> size_t {
        return s < pre.nsplit ? (size_t)pre0 + (size_t)s * pre.stride
                              : (size_t)suf0 + (size_t)(s - pre.nsplit) * suf.stride;
    };
    const float lse_mine = lane < n ? __ldcg(ws_lse + part(lane)) : -INFINITY;   // split `lane`
    float M = lse_mine;
    for (int s = lane + 32; s < n; s += 32) M = fmaxf(M, __ldcg(ws_lse + part(s)));
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
        const float wl = lane < nb ? expf((s0 == 0 ? lse_mine : __ldcg(ws_lse + part(s0 + lane))) - M)
                                   : 0.f;                                   // weight of split s0+lane
        for (int b0 = 0; b0 < nb; b0 += 8) {
            float4 v[NI][8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const bool have = b0 + u < nb;          // no load beyond the last split
                const float4 *po = reinterpret_cast<const float4 *>(ws_o + part(have ? s0 + b0 + u : 0) * D);
#pragma unroll
                for (int i = 0; i < NI; ++i) {
                    const int c = lane + 32 * i;
                    v[i][u] = have && c < nv ? __ldcg(po + c) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const float ws = __shfl_sync(0xffffffffu, wl, (b0 + u) & 31);   // 0 beyond nb
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
template <int NI, int JB>
__device__ __forceinline__ void merge_heads(const RowStreams &rs, const QRowDesc &d, int j0, int D,
                                            const float *ws_o, const float *ws_lse, float *out_rows,
                                            float *lse_out, int lane) {
    const StreamDesc &pre = rs.pre, &suf = rs.suf;
    const int pre0 = pre.part_base + d.pre_off + j0;
    const int suf0 = suf.part_base + d.suf_off + j0;
    const int n = pre.nsplit + suf.nsplit;
    auto part = [&](int s) -> size_t {          // partial row of (split s, head j0)
        return s < pre.nsplit ? (size_t)pre0 + (size_t)s * pre.stride
                              : (size_t)suf0 + (size_t)(s - pre.nsplit) * suf.stride;
    };
    constexpr int SB = 32 / JB;                 // splits per batch of 32 lanes
    const int jj = lane % JB, sl = lane / JB;
    // ---- row maxima ----
    float M = -INFINITY;
    for (int s = sl; s < n; s += SB) M = fmaxf(M, __ldcg(ws_lse + part(s) + jj));
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
        const int s_mine = s0 + sl;
        const float wl = (s_mine < n && M != -INFINITY) ? expf(__ldcg(ws_lse + part(s_mine) + jj) - M) : 0.f;
        const int nb = min(SB, n - s0);
        for (int sb = 0; sb < nb; ++sb) {
            const float4 *po = reinterpret_cast<const float4 *>(ws_o + part(s0 + sb) * D);
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

}  // namespace spork
