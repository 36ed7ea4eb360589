// libspork: D2 confidence score (Eq. 2)
//   c = min_{i=2..L} exp(l_i),  l_i = log-probability of the top-1 token at position i of the span
//     = min_i 1 / sum_v exp(x_iv - max_v x_iv)
// A pure HBM stream over the logits (4 bytes per element, one ex2 per element):
//   conf_partial_kernel : grid (splits, rows): one CTA reduces a slice of one row's vocabulary to
//                         (max, sum of exp relative to that max), 16-byte loads, 8 values per
//                         rescale of the running sum
//   conf_span_kernel    : one warp per span combines the slices of each row and takes the minimum
#include <limits.h>
#include <math.h>
#include <string.h>

#include <algorithm>
#include <mutex>

#include "spork_internal.h"

using namespace spork;

namespace {

constexpr int THREADS = 256;
constexpr float LOG2E = 1.4426950408889634f;

__device__ __forceinline__ float ex2f(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// running (m, s): s = sum exp2((x - m) * log2 e) over the values seen, m their maximum
__device__ __forceinline__ void absorb8(float &m, float &s, const float (&x)[8]) {
    float mx = fmaxf(fmaxf(fmaxf(x[0], x[1]), fmaxf(x[2], x[3])), fmaxf(fmaxf(x[4], x[5]), fmaxf(x[6], x[7])));
    if (mx > m) {                        // rare after the first batches
        s *= ex2f((m - mx) * LOG2E);     // m = -inf: s is 0 and stays 0
        m = mx;
    }
    // (x - m) first: exact for x == m, so the top-1 term is exactly 1
    float a = 0.f, b = 0.f;
#pragma unroll
    for (int i = 0; i < 8; i += 2) {
        a += ex2f((x[i] - m) * LOG2E);
        b += ex2f((x[i + 1] - m) * LOG2E);
    }
    s += a + b;
}

__device__ __forceinline__ void combine(float &m, float &s, float m2, float s2) {
    const float M = fmaxf(m, m2);
    if (M == -INFINITY) return;
    s = s * ex2f((m - M) * LOG2E) + s2 * ex2f((m2 - M) * LOG2E);
    m = M;
}

__global__ void __launch_bounds__(THREADS) conf_partial_kernel(const float *__restrict__ logits, int vocab,
                                                               int chunk, int splits, int vec,
                                                               const int32_t *__restrict__ rows,
                                                               float2 *__restrict__ part) {
    // grid.x = rows x splits (a 1-D grid: no 65,535 limit on the row count)
    const int row = rows[blockIdx.x / splits], sx = blockIdx.x % splits;   // only rows i >= 2 of their span are read
    const float *x = logits + (size_t)row * vocab;
    const int v0 = sx * chunk, v1 = min(vocab, v0 + chunk);
    float m = -INFINITY, s = 0.f;
    // vec: every row is 16-byte aligned (vocab % 4 == 0 and an aligned base; chunk is a multiple of 8)
    if (vec) {
        // 4 batches of 8 values (8 x 16-byte loads) in flight per thread before the first exp
        constexpr int NB = 4;
        for (int v = v0 + threadIdx.x * 8; v < v1; v += THREADS * 8 * NB) {
            float t[NB][8];
#pragma unroll
            for (int k = 0; k < NB; ++k) {
                const int vk = v + k * THREADS * 8;
                if (vk + 8 <= v1) {
                    const float4 a = __ldcs(reinterpret_cast<const float4 *>(x + vk));
                    const float4 b = __ldcs(reinterpret_cast<const float4 *>(x + vk + 4));
                    t[k][0] = a.x; t[k][1] = a.y; t[k][2] = a.z; t[k][3] = a.w;
                    t[k][4] = b.x; t[k][5] = b.y; t[k][6] = b.z; t[k][7] = b.w;
                } else {
#pragma unroll
                    for (int i = 0; i < 8; ++i) t[k][i] = vk + i < v1 ? x[vk + i] : -INFINITY;
                }
            }
#pragma unroll
            for (int k = 0; k < NB; ++k) absorb8(m, s, t[k]);
        }
    } else {
        for (int v = v0 + threadIdx.x * 8; v < v1; v += THREADS * 8) {
            float t[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) t[i] = v + i < v1 ? x[v + i] : -INFINITY;
            absorb8(m, s, t);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
        combine(m, s, __shfl_xor_sync(0xffffffffu, m, o), __shfl_xor_sync(0xffffffffu, s, o));
    __shared__ float2 red[THREADS / 32];
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = make_float2(m, s);
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < THREADS / 32; ++w) combine(m, s, red[w].x, red[w].y);
        part[(size_t)row * splits + sx] = make_float2(m, s);
    }
}

__global__ void __launch_bounds__(128) conf_span_kernel(const int32_t *__restrict__ span_indptr, int n_spans,
                                                        const float2 *__restrict__ part, int splits,
                                                        float *__restrict__ conf) {
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= n_spans) return;
    float c = 1.f;                                           // empty minimum (A-23)
    for (int row = span_indptr[w] + 1; row < span_indptr[w + 1]; ++row) {     // i = 2 .. L
        float m = -INFINITY, s = 0.f;
        for (int k = lane; k < splits; k += 32) {
            const float2 p = part[(size_t)row * splits + k];
            combine(m, s, p.x, p.y);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1)
            combine(m, s, __shfl_xor_sync(0xffffffffu, m, o), __shfl_xor_sync(0xffffffffu, s, o));
        c = fminf(c, 1.f / s);                               // exp(x_max - lse) = 1 / sum exp(x - x_max)
    }
    if (lane == 0) conf[w] = c;
}

}  // namespace

extern "C" int spork_confidence(spork_ctx *c, int n_spans, const int32_t *span_indptr, const float *logits,
                                int vocab, float *confidence_out, void *stream) {
    if (!c || n_spans < 0 || vocab < 1) return SPORK_ERR_INVALID;
    c->last_launches = 0;
    if (n_spans == 0) return SPORK_OK;
    if (!span_indptr || !confidence_out || span_indptr[0] != 0) return SPORK_ERR_INVALID;
    for (int s = 0; s < n_spans; ++s)
        if (span_indptr[s + 1] < span_indptr[s]) return SPORK_ERR_INVALID;
    const int n_pos = span_indptr[n_spans];
    if (n_pos > 0 && !logits) return SPORK_ERR_INVALID;
    cudaStream_t st = (cudaStream_t)stream;
    // enough CTAs to keep every SM's loads in flight: >= 8 per SM
    int splits = n_pos > 0 ? ceil_div(8 * c->num_sms, std::max(1, n_pos - n_spans)) : 1;
    splits = std::max(1, std::min(splits, ceil_div(vocab, THREADS * 8)));
    const int chunk = ceil_div(ceil_div(vocab, splits), THREADS * 8) * THREADS * 8;
    splits = ceil_div(vocab, chunk);
    int rc = devbuf_reserve(&c->ws_conf, (size_t)std::max(1, n_pos) * splits * sizeof(float2), st);
    if (rc != SPORK_OK) return rc;
    // device descriptors: span_indptr, then the list of rows that enter a minimum (all but the first of
    // each span); cached across calls with the same spans (the probes of a batch keep their shape
    // from step to step)
    const size_t ib = 4 * (size_t)(n_spans + 1);
    int n_rows = 0;
    const bool same = c->conf_key.size() == (size_t)n_spans + 1 &&
                      memcmp(c->conf_key.data(), span_indptr, ib) == 0 && c->conf_desc.p;
    if (same) {
        n_rows = n_pos - n_spans;
        for (int s = 0; s < n_spans; ++s) n_rows += span_indptr[s + 1] == span_indptr[s];   // empty spans skip nothing
    } else {
        rc = devbuf_reserve(&c->conf_desc, ib + 4 * (size_t)n_pos + 64, st);
        if (rc != SPORK_OK) return rc;
        StageSlot *slot;
        rc = stage_acquire(c, ib + 4 * (size_t)n_pos, &slot);
        if (rc != SPORK_OK) return rc;
        memcpy(slot->h, span_indptr, ib);
        int32_t *rows = (int32_t *)((char *)slot->h + ib);
        for (int s = 0; s < n_spans; ++s)
            for (int i = span_indptr[s] + 1; i < span_indptr[s + 1]; ++i) rows[n_rows++] = i;
        rc = stage_commit(c, slot, ib + 4 * (size_t)n_rows, st);
        if (rc != SPORK_OK) return rc;
        SPORK_CUDA(cudaMemcpyAsync(c->conf_desc.p, slot->d, ib + 4 * (size_t)n_rows, cudaMemcpyDeviceToDevice, st));
        rc = stage_done(c, slot, st);
        if (rc != SPORK_OK) return rc;
        c->conf_key.assign(span_indptr, span_indptr + n_spans + 1);
    }
    const int32_t *d_span = (const int32_t *)c->conf_desc.p;
    const int32_t *d_rows = (const int32_t *)((const char *)c->conf_desc.p + ib);
    if (n_rows > 0) {
        if ((int64_t)splits * n_rows > INT_MAX) return SPORK_ERR_INVALID;
        const int vec = (vocab & 3) == 0 && ((uintptr_t)logits & 15) == 0;   // else scalar loads (e.g. a sliced tensor)
        conf_partial_kernel<<<(unsigned)(splits * n_rows), THREADS, 0, st>>>(logits, vocab, chunk, splits, vec, d_rows,
                                                                             (float2 *)c->ws_conf.p);
        c->last_launches++;
    }
    conf_span_kernel<<<ceil_div(n_spans, 4), 128, 0, st>>>(d_span, n_spans, (const float2 *)c->ws_conf.p, splits,
                                                           confidence_out);
    c->last_launches++;
    SPORK_CUDA(cudaGetLastError());
    return SPORK_OK;
}

// ---------------------------------------------------------------------------------------------------
// spork_confidence_static: the same score for callers that cannot allocate (CUDA-graph capture, tight
// serving loops).  The per-(row, slice) partials live in a file-scope device array instead of the
// context's grown buffer, and the spans are read from DEVICE memory, so the call is two launches and
// nothing else: no cudaMalloc / cudaFree, no staging copy, no host read of device memory.
//   conf_partial_static_kernel : conf_partial_kernel without the row list -- CTA (row, slice) finds out
//                                from the device span_indptr whether its row opens a span (Eq. 2 skips
//                                i = 1) and leaves if so
//   conf_span_static_kernel    : conf_span_kernel over the static array, span bounds clamped to the rows
// Every GPU that loads libspork holds the array (256 KiB) until the process exits.  All calls share it:
// a slot the span kernel reads is written by the partial kernel of the same call (nothing has to start
// at zero, stale contents of earlier calls are never read), but two calls that overlap on the GPU
// (different streams, or graph branches) race on it.
namespace {

constexpr int STATIC_MAX_ROWS = SPORK_CONFIDENCE_STATIC_MAX_ROWS;
constexpr int STATIC_MAX_PARTS = 2 * STATIC_MAX_ROWS;          // float2 each: 256 KiB
constexpr int STATIC_MAX_DEVICES = 64;

static __device__ __align__(256) float2 conf_static_scratch[STATIC_MAX_PARTS];

// The array's name is a host-side stand-in in host code: the device address is resolved once per
// device (with that device current) and kept here.
struct StaticDev {
    float2 *part = nullptr;
    int num_sms = 0;
};
StaticDev g_static_dev[STATIC_MAX_DEVICES];
std::mutex g_static_mu;

__global__ void __launch_bounds__(THREADS) conf_partial_static_kernel(const float *__restrict__ logits, int vocab,
                                                                      int chunk, int splits, int vec,
                                                                      const int32_t *__restrict__ span_indptr,
                                                                      int n_spans, float2 *__restrict__ part) {
    const int row = blockIdx.x / splits, sx = blockIdx.x % splits;
    // the last j with span_indptr[j] <= row is the span holding the row (empty spans repeat a value)
    int lo = 0, hi = n_spans;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (span_indptr[mid] <= row) lo = mid; else hi = mid - 1;
    }
    if (span_indptr[lo] == row) return;                       // i = 1 of its span: not part of the minimum
    const float *x = logits + (size_t)row * vocab;
    const int v0 = sx * chunk, v1 = min(vocab, v0 + chunk);
    float m = -INFINITY, s = 0.f;
    if (vec) {
        constexpr int NB = 4;
        for (int v = v0 + threadIdx.x * 8; v < v1; v += THREADS * 8 * NB) {
            float t[NB][8];
#pragma unroll
            for (int k = 0; k < NB; ++k) {
                const int vk = v + k * THREADS * 8;
                if (vk + 8 <= v1) {
                    const float4 a = __ldcs(reinterpret_cast<const float4 *>(x + vk));
                    const float4 b = __ldcs(reinterpret_cast<const float4 *>(x + vk + 4));
                    t[k][0] = a.x; t[k][1] = a.y; t[k][2] = a.z; t[k][3] = a.w;
                    t[k][4] = b.x; t[k][5] = b.y; t[k][6] = b.z; t[k][7] = b.w;
                } else {
#pragma unroll
                    for (int i = 0; i < 8; ++i) t[k][i] = vk + i < v1 ? x[vk + i] : -INFINITY;
                }
            }
#pragma unroll
            for (int k = 0; k < NB; ++k) absorb8(m, s, t[k]);
        }
    } else {
        for (int v = v0 + threadIdx.x * 8; v < v1; v += THREADS * 8) {
            float t[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) t[i] = v + i < v1 ? x[v + i] : -INFINITY;
            absorb8(m, s, t);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
        combine(m, s, __shfl_xor_sync(0xffffffffu, m, o), __shfl_xor_sync(0xffffffffu, s, o));
    __shared__ float2 red[THREADS / 32];
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = make_float2(m, s);
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < THREADS / 32; ++w) combine(m, s, red[w].x, red[w].y);
        part[(size_t)row * splits + sx] = make_float2(m, s);
    }
}

// conf_span_kernel with the span bounds clamped to [0, n_pos]: the spans come from device memory here and
// cannot be validated on the host, so a bad span_indptr gives wrong scores, never a read outside the array
__global__ void __launch_bounds__(128) conf_span_static_kernel(const int32_t *__restrict__ span_indptr, int n_spans,
                                                               int n_pos, const float2 *__restrict__ part, int splits,
                                                               float *__restrict__ conf) {
    const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (w >= n_spans) return;
    const int r0 = max(0, span_indptr[w]), r1 = min(n_pos, span_indptr[w + 1]);
    float c = 1.f;                                           // empty minimum (A-23)
    for (int row = r0 + 1; row < r1; ++row) {                // i = 2 .. L
        float m = -INFINITY, s = 0.f;
        for (int k = lane; k < splits; k += 32) {
            const float2 p = part[(size_t)row * splits + k];
            combine(m, s, p.x, p.y);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1)
            combine(m, s, __shfl_xor_sync(0xffffffffu, m, o), __shfl_xor_sync(0xffffffffu, s, o));
        c = fminf(c, 1.f / s);
    }
    if (lane == 0) conf[w] = c;
}

}  // namespace

extern "C" int spork_confidence_static(int n_spans, const int32_t *span_indptr, int n_pos, const float *logits,
                                       int vocab, float *confidence_out, void *stream) {
    if (n_spans < 0 || n_pos < 0 || vocab < 1) return SPORK_ERR_INVALID;
    if (n_pos > STATIC_MAX_ROWS) return SPORK_ERR_LIMIT;
    int dev = -1;
    SPORK_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return SPORK_ERR_LIMIT;
    StaticDev sd;
    {
        std::lock_guard<std::mutex> lock(g_static_mu);
        if (!g_static_dev[dev].part) {          // set-up, once per device, that device current
            float2 *p = nullptr;
            int sms = 0;
            SPORK_CUDA(cudaGetSymbolAddress((void **)&p, conf_static_scratch));
            SPORK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
            if (!p || sms < 1) return SPORK_ERR_CUDA;
            g_static_dev[dev].num_sms = sms;
            g_static_dev[dev].part = p;
        }
        sd = g_static_dev[dev];
    }
    if (n_spans == 0) return SPORK_OK;          // (a set-up call: the address is resolved, nothing runs)
    if (!span_indptr || !confidence_out || (n_pos > 0 && !logits)) return SPORK_ERR_INVALID;
    cudaStream_t st = (cudaStream_t)stream;
    int splits = 1, chunk = THREADS * 8;
    if (n_pos > 0) {
        // as spork_confidence (>= 8 CTAs per SM; the CTAs of span-opening rows leave at once), then what
        // the array holds: at least 2 slices per row
        splits = ceil_div(8 * sd.num_sms, n_pos);
        splits = std::max(1, std::min(splits, ceil_div(vocab, THREADS * 8)));
        splits = std::min(splits, STATIC_MAX_PARTS / n_pos);
        chunk = ceil_div(ceil_div(vocab, splits), THREADS * 8) * THREADS * 8;
        splits = ceil_div(vocab, chunk);
        const int vec = (vocab & 3) == 0 && ((uintptr_t)logits & 15) == 0;
        conf_partial_static_kernel<<<(unsigned)(splits * n_pos), THREADS, 0, st>>>(logits, vocab, chunk, splits, vec,
                                                                                   span_indptr, n_spans, sd.part);
    }
    conf_span_static_kernel<<<ceil_div(n_spans, 4), 128, 0, st>>>(span_indptr, n_spans, n_pos, sd.part, splits,
                                                                 confidence_out);
    SPORK_CUDA(cudaGetLastError());
    return SPORK_OK;
}
