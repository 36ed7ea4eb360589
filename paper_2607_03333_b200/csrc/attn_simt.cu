// libspork: generic CUDA-core attention kernel (fp32 KV, or bf16 / e4m3 KV with D != 128)
// and the LSE merge kernel shared by both attention paths.
//
// simt kernel: one CTA per work item, one warp per query row at a time.  A
// lane owns one token for the score pass (full dot product, 16-byte loads) and
// D/32 output dims for the value pass.  fp32 accumulation, accurate expf/logf:
// this is the path that has to meet 1e-5 on fp32 KV (config 1), not a
// bandwidth target.
#include <cuda_fp16.h>
#include <math.h>

#include "spork_internal.h"
#include "merge.cuh"

using namespace spork;

namespace {

constexpr int SIMT_WARPS = 4;

__device__ __forceinline__ float bf16_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }

// byte offset of 16-byte chunk c of row r inside a (page, kv head) block
__device__ __forceinline__ int chunk_off(int swizzled, int chunks_per_row, int r, int c) {
    if (swizzled) return swz_chunk_off(chunks_per_row >> 3, r, c);
    return (r * chunks_per_row + c) * 16;
}

template <typename T> struct Elt;
template <> struct Elt<float> {
    static constexpr int PER_CHUNK = 4;
    static __device__ __forceinline__ void unpack(const uint4 &v, float *f) {
        f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y);
        f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
    }
    static __device__ __forceinline__ float load(const uint8_t *p) { return *reinterpret_cast<const float *>(p); }
};
template <> struct Elt<uint16_t> {
    static constexpr int PER_CHUNK = 8;
    static __device__ __forceinline__ void unpack(const uint4 &v, float *f) {
        f[0] = bf16_lo(v.x); f[1] = bf16_hi(v.x); f[2] = bf16_lo(v.y); f[3] = bf16_hi(v.y);
        f[4] = bf16_lo(v.z); f[5] = bf16_hi(v.z); f[6] = bf16_lo(v.w); f[7] = bf16_hi(v.w);
    }
    static __device__ __forceinline__ float load(const uint8_t *p) {
        return __uint_as_float((uint32_t)(*reinterpret_cast<const uint16_t *>(p)) << 16);
    }
};

// e4m3 ("fn") byte -> fp32, exact: the byte's magnitude bits shifted into an fp16 pattern read 2^-8 too
// small (subnormals included); s.1111.111 is NaN
__device__ __forceinline__ float e4m3_to_f32(uint32_t b) {
    const float v = __half2float(__ushort_as_half((unsigned short)(((b & 0x80u) << 8) | ((b & 0x7fu) << 7)))) * 256.f;
    return (b & 0x7fu) == 0x7fu ? __int_as_float(0x7fffffff) : v;
}
template <> struct Elt<uint8_t> {
    static constexpr int PER_CHUNK = 16;
    static __device__ __forceinline__ void unpack(const uint4 &v, float *f) {
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 16; ++i) f[i] = e4m3_to_f32((w[i >> 2] >> (8 * (i & 3))) & 0xffu);
    }
    static __device__ __forceinline__ float load(const uint8_t *p) { return e4m3_to_f32(*p); }
};

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// T: stored K / V element, TQ: stored Q element (the same type, except e4m3 KV with bf16 queries)
template <typename T, typename TQ, int DMAX>
__global__ void __launch_bounds__(SIMT_WARPS * 32) attn_simt_kernel(
    const WorkItem *__restrict__ items, const int32_t *__restrict__ seq_len,
    const int32_t *__restrict__ rowmap, const TQ *__restrict__ q, const uint8_t *__restrict__ k_pool,
    const uint8_t *__restrict__ v_pool, const int32_t *__restrict__ table, int table_stride, int Hq,
    int Hkv, int G, int D, int swizzled, float scale, float *__restrict__ ws_o,
    float *__restrict__ ws_lse) {
    __shared__ float qs[SIMT_WARPS][DMAX];
    const WorkItem it = load_item(items, blockIdx.x, seq_len);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int E = Elt<T>::PER_CHUNK;
    const int cpr = D / E;                       // 16-byte chunks per row
    const size_t head_block = (size_t)PS * D * sizeof(T);
    const int32_t *row_tab = table + (size_t)it.table_seq * table_stride;
    constexpr int NACC = DMAX / 32;

    for (int r = warp; r < it.nrows; r += SIMT_WARPS) {
        const int lr = it.rb0 + r;
        const int qrow = item_qrow(it, rowmap, lr, G), h = it.kvh * G + lr % G;
        const int lim = it.lim0 + lr / G;
        __syncwarp();
        for (int d = lane; d < D; d += 32)
            qs[warp][d] = Elt<TQ>::load(reinterpret_cast<const uint8_t *>(q + ((size_t)qrow * Hq + h) * D + d));
        __syncwarp();
        float m = -INFINITY, l = 0.f, acc[NACC];
#pragma unroll
        for (int i = 0; i < NACC; ++i) acc[i] = 0.f;

        for (int tb = it.tok0; tb < it.tok1; tb += 32) {
            const int t = tb + lane;
            const bool valid = t < it.tok1 && t <= lim;
            float s = -INFINITY;
            size_t blk = 0;
            if (valid) {
                blk = ((size_t)row_tab[t / PS] * Hkv + it.kvh) * head_block;
                const uint8_t *kp = k_pool + blk;
                float dot = 0.f;
                for (int c = 0; c < cpr; ++c) {
                    uint4 v = *reinterpret_cast<const uint4 *>(kp + chunk_off(swizzled, cpr, t % PS, c));
                    float f[E];
                    Elt<T>::unpack(v, f);
#pragma unroll
                    for (int e = 0; e < E; ++e) dot = fmaf(qs[warp][c * E + e], f[e], dot);
                }
                s = dot * scale;
            }
            const float m_new = fmaxf(m, warp_max(s));
            if (m_new == -INFINITY) continue;   // nothing visible yet (warp-uniform)
            const float alpha = expf(m - m_new);   // m = -inf -> 0
            const float p = valid ? expf(s - m_new) : 0.f;
            l = l * alpha + warp_sum(p);
#pragma unroll
            for (int i = 0; i < NACC; ++i) acc[i] *= alpha;
            m = m_new;
            const int nt = min(32, it.tok1 - tb);
            // value pass: 8 tokens' V elements are requested before the first is used (each is a dependent
            // global load: one at a time, the 32 tokens of a chunk cost 32 memory latencies)
            for (int t0 = 0; t0 < nt; t0 += 8) {
                float pt[8], vv[8][NACC];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int tt = t0 + u;                                   // (tt < 32 always: nt <= 32, t0 % 8 == 0)
                    pt[u] = __shfl_sync(0xffffffffu, p, tt & 31);
                    const unsigned long long b = __shfl_sync(0xffffffffu, (unsigned long long)blk, tt & 31);
                    if (tt >= nt) pt[u] = 0.f;
                    const uint8_t *vp = v_pool + b;
                    const int rr = (tb + tt) % PS;
#pragma unroll
                    for (int i = 0; i < NACC; ++i) {
                        const int d = lane + 32 * i;
                        vv[u][i] = 0.f;
                        if (pt[u] != 0.f && d < D) {        // p = 0: masked or beyond the range -- keeps 0 * garbage out
                            const int off = chunk_off(swizzled, cpr, rr, d / E) + (d % E) * (int)sizeof(T);
                            vv[u][i] = Elt<T>::load(vp + off);
                        }
                    }
                }
#pragma unroll
                for (int u = 0; u < 8; ++u)
#pragma unroll
                    for (int i = 0; i < NACC; ++i) acc[i] = fmaf(pt[u], vv[u][i], acc[i]);
            }
        }
        const size_t prow = (size_t)it.part_base + r;
        const float inv = l > 0.f ? 1.f / l : 0.f;
#pragma unroll
        for (int i = 0; i < NACC; ++i) {
            int d = lane + 32 * i;
            if (d < D) ws_o[prow * D + d] = acc[i] * inv;
        }
        if (lane == 0) ws_lse[prow] = l > 0.f ? m + logf(l) : -INFINITY;
    }
}

// one warp per (q row, q head): LSE-weighted combination of that row's partials
//   M = max lse_s, w_s = exp(lse_s - M), out = sum w_s o_s / sum w_s, lse = M + ln sum w_s
// an empty partial has lse = -inf and weight 0; no partial at all: out = 0, lse = -inf.
// Launched with programmatic stream serialisation: blocks may become resident while the
// attention kernel still runs and wait in griddepcontrol.wait until its partials are visible.
// Lane s owns the weight of split s; the partial rows are fetched 8 splits at a time with
// every load of a batch in flight before the first use (the kernel is pure L2 latency).
template <int NI>   // float4 per lane per row: 1 for D <= 128, 2 for D <= 256
__global__ void __launch_bounds__(128) merge_kernel(const QRowDesc *__restrict__ qd,
                                                    const RowRef *__restrict__ refs,
                                                    const StreamDesc *__restrict__ streams, int n_qrows, int Hq,
                                                    int G, int D, const float *ws_o, const float *ws_lse,
                                                    float *__restrict__ out, float *__restrict__ lse) {
    // one warp per (q row, q head): the most warps, for calls with few rows (decode)
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= n_qrows * Hq) return;
    const int qrow = w / Hq, h = w % Hq;
    const QRowDesc d = qd[qrow];                 // written before the attention kernel was launched
    const RowSplits rs = load_row_splits(d, refs, streams, h / G, lane);
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // a next layer's attention kernel may queue up
    asm volatile("griddepcontrol.wait;" ::: "memory");
    merge_row<NI>(rs, h % G, D, ws_o, ws_lse, out + (size_t)w * D, lse + w, lane);
}

template <int NI>
__global__ void __launch_bounds__(128) merge_heads_kernel(const QRowDesc *__restrict__ qd,
                                                          const RowRef *__restrict__ refs,
                                                          const StreamDesc *__restrict__ streams, int n_qrows,
                                                          int Hq, int G, int D, const float *ws_o,
                                                          const float *ws_lse, float *__restrict__ out,
                                                          float *__restrict__ lse) {
    // one warp per (q row, kv head): its G heads' partial rows are contiguous; for calls with many rows
    // (verify, large decode batches), where bytes in flight per warp matter more than the warp count
    const int Hkv = Hq / G;
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= n_qrows * Hkv) return;
    const int qrow = w / Hkv, kvh = w % Hkv;
    const QRowDesc d = qd[qrow];                 // written before the attention kernel was launched
    const RowSplits rs = load_row_splits(d, refs, streams, kvh, lane);
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const size_t row0 = (size_t)qrow * Hq + (size_t)kvh * G;
    constexpr int JB = NI == 1 ? 8 : 4;
    int j = 0;
    for (; j + JB <= G; j += JB)
        merge_heads<NI, JB>(rs, j, D, ws_o, ws_lse, out + (row0 + j) * D, lse + row0 + j, lane);
    if (G - j >= 4 && JB > 4) {
        merge_heads<NI, 4>(rs, j, D, ws_o, ws_lse, out + (row0 + j) * D, lse + row0 + j, lane);
        j += 4;
    }
    if (G - j >= 2) {
        merge_heads<NI, 2>(rs, j, D, ws_o, ws_lse, out + (row0 + j) * D, lse + row0 + j, lane);
        j += 2;
    }
    for (; j < G; ++j)
        merge_row<NI>(rs, j, D, ws_o, ws_lse, out + (row0 + j) * D, lse + row0 + j, lane);
}

// one warp per (q row, kv head, group of 4 GQA heads): merge_heads4 (G % 4 == 0)
template <int NI>
__global__ void __launch_bounds__(128) merge_heads4_kernel(const QRowDesc *__restrict__ qd,
                                                           const RowRef *__restrict__ refs,
                                                           const StreamDesc *__restrict__ streams, int n_qrows,
                                                           int Hq, int G, int D, const float *ws_o,
                                                           const float *ws_lse, float *__restrict__ out,
                                                           float *__restrict__ lse) {
    const int Hkv = Hq / G, Q4 = G >> 2;
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= n_qrows * Hkv * Q4) return;
    const int qrow = w / (Hkv * Q4), kvh = (w / Q4) % Hkv, j0 = (w % Q4) * 4;
    const QRowDesc d = qd[qrow];                 // written before the attention kernel was launched
    const RowSplits rs = load_row_splits(d, refs, streams, kvh, lane);
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const size_t row0 = (size_t)qrow * Hq + (size_t)kvh * G + j0;
    merge_heads4<NI>(rs, j0, D, ws_o, ws_lse, out + row0 * D, lse + row0, lane);
}

}  // namespace

namespace spork {

int launch_attn_simt(spork_ctx *c, const LayerIO &io, cudaStream_t st) {
    const Plan &P = c->plan;
    if (P.n_items == 0) return SPORK_OK;
    const WorkItem *items = P.d_items;
    float *wo = (float *)c->ws_o.p, *wl = (float *)c->ws_lse.p;
    const uint8_t *kp = (const uint8_t *)io.k_pool, *vp = (const uint8_t *)io.v_pool;
    const spork_config &f = c->cfg;
    dim3 grid(P.n_items), block(SIMT_WARPS * 32);
#define SPORK_SIMT(T, TQ, DMAX)                                                                    \
    attn_simt_kernel<T, TQ, DMAX><<<grid, block, 0, st>>>(items, c->d_len, P.d_rowmap, (const TQ *)io.q, kp, vp, \
                                                          c->d_table, c->table_stride, f.num_q_heads, \
                                                          f.num_kv_heads, c->G, f.head_dim,        \
                                                          c->swizzled, f.scale, wo, wl)
    if (f.dtype == SPORK_F32) {
        if (f.head_dim <= 64) SPORK_SIMT(float, float, 64);
        else if (f.head_dim <= 128) SPORK_SIMT(float, float, 128);
        else SPORK_SIMT(float, float, 256);
    } else if (f.dtype == SPORK_E4M3) {
        if (f.head_dim <= 64) SPORK_SIMT(uint8_t, uint16_t, 64);
        else if (f.head_dim <= 128) SPORK_SIMT(uint8_t, uint16_t, 128);
        else SPORK_SIMT(uint8_t, uint16_t, 256);
    } else {
        if (f.head_dim <= 64) SPORK_SIMT(uint16_t, uint16_t, 64);
        else if (f.head_dim <= 128) SPORK_SIMT(uint16_t, uint16_t, 128);
        else SPORK_SIMT(uint16_t, uint16_t, 256);
    }
#undef SPORK_SIMT
    c->last_launches++;
    SPORK_CUDA(cudaGetLastError());
    return SPORK_OK;
}

int launch_merge(spork_ctx *c, const LayerIO &io, cudaStream_t st) {
    const Plan &P = c->plan;
    if (P.n_qrows == 0) return SPORK_OK;
    // enough (q row, kv head) pairs to fill the SMs: the grouped kernel (measured: verify k = 16 merge
    // 60 -> 37 us, config 3 14 -> 12 us; config 2 / 5 with 256 / 512 pairs are faster per head)
    const bool grouped = P.n_qrows * c->cfg.num_kv_heads >= 1024;
    const bool by4 = grouped && c->G % 4 == 0 && c->cfg.head_dim <= 128;    // four heads per warp, four splits in flight
    const int warps = P.n_qrows * (by4 ? c->cfg.num_kv_heads * (c->G / 4)
                                       : (grouped ? c->cfg.num_kv_heads : c->cfg.num_q_heads));
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(ceil_div(warps, 4));
    cfg.blockDim = dim3(128);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    auto kern = by4 ? merge_heads4_kernel<1>
                    : (grouped ? (c->cfg.head_dim <= 128 ? merge_heads_kernel<1> : merge_heads_kernel<2>)
                               : (c->cfg.head_dim <= 128 ? merge_kernel<1> : merge_kernel<2>));
    SPORK_CUDA(cudaLaunchKernelEx(&cfg, kern, P.d_qdesc, P.d_refs, P.d_streams, P.n_qrows,
                                  (int)c->cfg.num_q_heads, c->G, (int)c->cfg.head_dim,
                                  (const float *)c->ws_o.p, (const float *)c->ws_lse.p,
                                  io.out, io.lse));
    c->last_launches++;
    SPORK_CUDA(cudaGetLastError());
    return SPORK_OK;
}

}  // namespace spork
