/*
 * spork_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU fp64 implementation of what the Spork
 * fork / decode / verify / release path computes.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may call it.  It shares no code with paper_2607_03333_b200/csrc (the CUDA
 * path): no headers, no helpers, no tables.
 *
 * What it follows
 * ---------------
 * The paper fixes WHEN things happen and what they must preserve:
 *   - fork shares the main stream's prefix KV with the probe ("Fork a
 *     completions request ... {D1 cache hit}", Algorithm 1 step 6,
 *     PAPER.md:262; section 4.1);
 *   - main and probe decode concurrently over that prefix;
 *   - D3 verifies k draft tokens in one decode step and accepts the longest
 *     greedy-matching prefix (section 4.3 steps 1-3);
 *   - a probe that ends / is rejected / times out / is superseded drops its
 *     KV.
 * The paper gives no arithmetic for any of it, so everything numerical is the
 * plain textbook definition written out, under the readings A-1..A-25 of
 * SURVEY.md section 8(c) (restated in DESIGN.md "Readings"):
 *   A-1  allocation = lowest free id first, requests in array order
 *   A-2  refcount[p] = number of live block-table entries pointing at p
 *   A-3  fork copies the WHOLE partially filled tail page
 *   A-8  softmax scale passed in (1/sqrt(D))      A-9  lse is a natural log
 *   A-10 q head h -> kv head h / (Hq/Hkv)         A-12 decode sees all len tokens
 *   A-13 verify row j of k sees tokens t <= len-k+j (drafts already appended)
 *   A-15 an empty part has lse = -inf and weight 0 (never 0*NaN)
 * Attention (the "exact up to rounding order" case): for query row q, keys
 * k_t, values v_t, t = 0..n-1:
 *     s_t = scale * <q, k_t>,  m = max_t s_t,  Z = sum_t exp(s_t - m),
 *     out = sum_t exp(s_t - m) / Z * v_t,      lse = m + ln Z.
 * No blocking, no online softmax, no cascade in the main routine; the cascade
 * (prefix / suffix partials merged by log-sum-exp) exists only as a second
 * routine used to pin the first.
 *
 * Pins: tests/test_oracle_attention.py, tests/test_oracle_alloc.py (closed
 * forms, invariants, brute force, torch float64 SDPA, exhaustive allocator
 * scripts against an independently written model).  No function here is
 * "parity unpinned".
 *
 * Storage: K/V/Q are kept in their storage dtype (fp32, or bf16 as uint16 bit
 * patterns rounded once by the input generator) and widened exactly to fp64
 * on every read.
 *
 * FP8-KV variant (ORACLE_E4M3KV, reading B-4):
 * K and V are stored as e4m3 bytes (1 sign, 4 exponent bits with bias 7, 3
 * mantissa bits; no infinities; exponent 15 with mantissa 7 is NaN; exponent 0
 * is subnormal: m/8 * 2^-6), Q stays bf16.  Only the widening differs: the
 * definition above is applied to the exactly widened values.  Pinned against
 * torch.float8_e4m3fn -> float64 on all 256 codes (tests/test_oracle_fp8.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK 0
#define ORACLE_ERR_INVALID (-1)
#define ORACLE_ERR_OOM (-2)
#define ORACLE_ERR_NO_SLOT (-3)
#define ORACLE_ERR_TOO_LONG (-4)
#define ORACLE_ERR_INVALID_SEQ (-5)
#define ORACLE_ERR_SHARED (-6)

#define ORACLE_F32 0
#define ORACLE_BF16 1
#define ORACLE_E4M3KV 2   /* K, V: e4m3 bytes; Q: bf16 */

typedef struct oracle_ctx {
    int dtype, Hq, Hkv, D, ps;
    int num_pages, max_seqs, max_pages_per_seq;
    double scale;
    int store_kv;
    size_t elt;            /* bytes per stored element */
    int32_t *refcount;     /* [num_pages]  0 <=> free (A-2) */
    int32_t *table;        /* [max_seqs][max_pages_per_seq] */
    int32_t *len;          /* [max_seqs] */
    uint8_t *live;         /* [max_seqs] */
    uint8_t *kpool, *vpool;/* [num_pages][Hkv][ps][D] storage dtype (plain row-major) */
} oracle_ctx;

/* ---- exact widening ------------------------------------------------------ */
static double widen_f32(const uint8_t *base, size_t idx) {
    float f;
    memcpy(&f, base + idx * 4, 4);
    return (double)f;
}
static double widen_bf16(const uint8_t *base, size_t idx) {
    uint16_t h;
    uint32_t u;
    float f;
    memcpy(&h, base + idx * 2, 2);
    u = ((uint32_t)h) << 16;
    memcpy(&f, &u, 4);
    return (double)f;
}
/* e4m3 ("fn": finite + NaN): value = (-1)^s * 2^(e-7) * (1 + m/8), e = 1..15;
 * e = 0: (-1)^s * 2^-6 * m/8; s.1111.111 is NaN */
static double widen_e4m3(const uint8_t *base, size_t idx) {
    uint8_t b = base[idx];
    int sgn = b >> 7, e = (b >> 3) & 15, m = b & 7;
    double v;
    if (e == 15 && m == 7) return NAN;
    v = e == 0 ? ldexp((double)m / 8.0, -6) : ldexp(1.0 + (double)m / 8.0, e - 7);
    return sgn ? -v : v;
}
/* one stored K / V element */
static double load_elt(const oracle_ctx *c, const uint8_t *base, size_t idx) {
    if (c->dtype == ORACLE_F32) return widen_f32(base, idx);
    if (c->dtype == ORACLE_BF16) return widen_bf16(base, idx);
    return widen_e4m3(base, idx);
}
/* one stored Q element (the KV dtype, except for e4m3 KV, whose queries are bf16) */
static double load_q(const oracle_ctx *c, const uint8_t *base, size_t idx) {
    return c->dtype == ORACLE_F32 ? widen_f32(base, idx) : widen_bf16(base, idx);
}
static size_t q_elt(const oracle_ctx *c) { return c->dtype == ORACLE_F32 ? 4 : 2; }

static size_t page_elems(const oracle_ctx *c) { return (size_t)c->Hkv * c->ps * c->D; }

static size_t kv_index(const oracle_ctx *c, int page, int head, int slot) {
    return (((size_t)page * c->Hkv + head) * c->ps + slot) * c->D;
}

/* ---- lifetime ------------------------------------------------------------ */
oracle_ctx *oracle_create(int dtype, int Hq, int Hkv, int D, int ps, int num_pages, int max_seqs,
                          int max_pages_per_seq, double scale, int store_kv) {
    oracle_ctx *c;
    if (Hq <= 0 || Hkv <= 0 || D <= 0 || ps <= 0 || Hq % Hkv || num_pages <= 0 || max_seqs <= 0 ||
        max_pages_per_seq <= 0 || (dtype != ORACLE_F32 && dtype != ORACLE_BF16 && dtype != ORACLE_E4M3KV))
        return NULL;
    c = (oracle_ctx *)calloc(1, sizeof(*c));
    if (!c) return NULL;
    c->dtype = dtype; c->Hq = Hq; c->Hkv = Hkv; c->D = D; c->ps = ps;
    c->num_pages = num_pages; c->max_seqs = max_seqs; c->max_pages_per_seq = max_pages_per_seq;
    c->scale = scale; c->store_kv = store_kv;
    c->elt = dtype == ORACLE_F32 ? 4 : (dtype == ORACLE_BF16 ? 2 : 1);
    c->refcount = (int32_t *)calloc((size_t)num_pages, sizeof(int32_t));
    c->table = (int32_t *)malloc((size_t)max_seqs * max_pages_per_seq * sizeof(int32_t));
    c->len = (int32_t *)calloc((size_t)max_seqs, sizeof(int32_t));
    c->live = (uint8_t *)calloc((size_t)max_seqs, 1);
    if (c->table) memset(c->table, 0xff, (size_t)max_seqs * max_pages_per_seq * sizeof(int32_t));
    if (store_kv) {
        c->kpool = (uint8_t *)calloc((size_t)num_pages * page_elems(c), c->elt);
        c->vpool = (uint8_t *)calloc((size_t)num_pages * page_elems(c), c->elt);
    }
    if (!c->refcount || !c->table || !c->len || !c->live || (store_kv && (!c->kpool || !c->vpool))) {
        free(c->refcount); free(c->table); free(c->len); free(c->live); free(c->kpool); free(c->vpool);
        free(c);
        return NULL;
    }
    return c;
}

void oracle_destroy(oracle_ctx *c) {
    if (!c) return;
    free(c->refcount); free(c->table); free(c->len); free(c->live); free(c->kpool); free(c->vpool);
    free(c);
}

/* ---- allocator (A-1: lowest free id first) --------------------------------- */
static int count_free_pages(const oracle_ctx *c) {
    int n = 0, p;
    for (p = 0; p < c->num_pages; ++p) n += (c->refcount[p] == 0);
    return n;
}

static int alloc_page(oracle_ctx *c) {
    int p;
    for (p = 0; p < c->num_pages; ++p)
        if (c->refcount[p] == 0) { c->refcount[p] = 1; return p; }
    return -1;
}

static int pages_of(const oracle_ctx *c, int len) { return (len + c->ps - 1) / c->ps; }

static int seq_ok(const oracle_ctx *c, int s) { return s >= 0 && s < c->max_seqs && c->live[s]; }

int oracle_seq_create(oracle_ctx *c, int n, int32_t *ids_out) {
    int i, s, nfree = 0;
    for (s = 0; s < c->max_seqs; ++s) nfree += !c->live[s];
    if (n < 0) return ORACLE_ERR_INVALID;
    if (nfree < n) return ORACLE_ERR_NO_SLOT;       /* all-or-nothing */
    for (i = 0, s = 0; i < n; ++s)
        if (!c->live[s]) { c->live[s] = 1; c->len[s] = 0; ids_out[i++] = s; }
    return ORACLE_OK;
}

/* append: the "prefill / decode wrote KV" event (Algorithm 1 steps 1-5).
 * k_src, v_src: [sum n_tokens][Hkv][D] storage dtype.  Requests in array order,
 * positions ascending; a page is allocated at each page boundary. */
int oracle_append(oracle_ctx *c, int n, const int32_t *seq_ids, const int32_t *n_tokens,
                  const void *k_src, const void *v_src) {
    int i, j, h, need = 0;
    size_t tok = 0;
    /* validate the whole batch first: a failing batch changes nothing.  The same
     * sequence may appear twice, so track lengths as they would evolve. */
    int32_t *tmp_len = (int32_t *)malloc((size_t)c->max_seqs * sizeof(int32_t));
    if (!tmp_len) return ORACLE_ERR_INVALID;
    memcpy(tmp_len, c->len, (size_t)c->max_seqs * sizeof(int32_t));
    for (i = 0; i < n; ++i) {
        int s = seq_ids[i], nl;
        if (!seq_ok(c, s) || n_tokens[i] < 0) { free(tmp_len); return ORACLE_ERR_INVALID_SEQ; }
        nl = tmp_len[s] + n_tokens[i];
        if (pages_of(c, nl) > c->max_pages_per_seq) { free(tmp_len); return ORACLE_ERR_TOO_LONG; }
        need += pages_of(c, nl) - pages_of(c, tmp_len[s]);
        tmp_len[s] = nl;
    }
    free(tmp_len);
    if (need > count_free_pages(c)) return ORACLE_ERR_OOM;
    for (i = 0; i < n; ++i) {
        int s = seq_ids[i];
        for (j = 0; j < n_tokens[i]; ++j, ++tok) {
            int L = c->len[s], slot = L % c->ps, page;
            if (slot == 0) c->table[(size_t)s * c->max_pages_per_seq + L / c->ps] = alloc_page(c);
            page = c->table[(size_t)s * c->max_pages_per_seq + L / c->ps];
            if (c->store_kv) {
                for (h = 0; h < c->Hkv; ++h) {
                    size_t dst = kv_index(c, page, h, slot) * c->elt;
                    size_t src = ((tok * c->Hkv + h) * c->D) * c->elt;
                    memcpy(c->kpool + dst, (const uint8_t *)k_src + src, c->D * c->elt);
                    memcpy(c->vpool + dst, (const uint8_t *)v_src + src, c->D * c->elt);
                }
            }
            c->len[s] = L + 1;
        }
    }
    return ORACLE_OK;
}

/* fork: Algorithm 1 step 6 -- child shares the parent's full
 * pages (refcount++), gets a private copy of the partially filled tail page
 * (A-3), and the parent's length.  Children take the lowest free slots in
 * request order; the same parent may repeat; all-or-nothing. */
int oracle_fork(oracle_ctx *c, int n, const int32_t *parents, int32_t *children_out) {
    int i, j, s, nfree = 0, need = 0;
    if (n < 0) return ORACLE_ERR_INVALID;
    for (i = 0; i < n; ++i) {
        if (!seq_ok(c, parents[i])) return ORACLE_ERR_INVALID_SEQ;
        need += (c->len[parents[i]] % c->ps) != 0;
    }
    for (s = 0; s < c->max_seqs; ++s) nfree += !c->live[s];
    if (nfree < n) return ORACLE_ERR_NO_SLOT;
    if (need > count_free_pages(c)) return ORACLE_ERR_OOM;
    for (i = 0; i < n; ++i) {
        int p = parents[i], child = -1, L = c->len[p], nf = L / c->ps;
        const int32_t *pt = c->table + (size_t)p * c->max_pages_per_seq;
        int32_t *ct;
        for (s = 0; s < c->max_seqs; ++s) if (!c->live[s]) { child = s; break; }
        ct = c->table + (size_t)child * c->max_pages_per_seq;
        c->live[child] = 1;
        for (j = 0; j < nf; ++j) { ct[j] = pt[j]; c->refcount[pt[j]] += 1; }
        if (L % c->ps) {
            int np = alloc_page(c);
            if (c->store_kv) {
                size_t bytes = page_elems(c) * c->elt;
                memcpy(c->kpool + (size_t)np * bytes, c->kpool + (size_t)pt[nf] * bytes, bytes);
                memcpy(c->vpool + (size_t)np * bytes, c->vpool + (size_t)pt[nf] * bytes, bytes);
            }
            ct[nf] = np;
        }
        c->len[child] = L;
        children_out[i] = child;
    }
    return ORACLE_OK;
}

/* release: probe finished / rejected / timed out / superseded (PAPER.md:211,
 * :503, :585) or main finished.  Double release or a repeated id in one batch is
 * rejected without any state change. */
int oracle_release(oracle_ctx *c, int n, const int32_t *seq_ids) {
    int i, j;
    for (i = 0; i < n; ++i) {
        if (!seq_ok(c, seq_ids[i])) return ORACLE_ERR_INVALID_SEQ;
        for (j = 0; j < i; ++j) if (seq_ids[j] == seq_ids[i]) return ORACLE_ERR_INVALID_SEQ;
    }
    for (i = 0; i < n; ++i) {
        int s = seq_ids[i], np = pages_of(c, c->len[s]);
        int32_t *t = c->table + (size_t)s * c->max_pages_per_seq;
        for (j = 0; j < np; ++j) { c->refcount[t[j]] -= 1; t[j] = -1; }
        c->len[s] = 0;
        c->live[s] = 0;
    }
    return ORACLE_OK;
}

/* truncate: rollback of rejected drafts (section 4.3 step 3).
 * Frees whole pages beyond ceil(new_len/ps).  ORACLE_ERR_SHARED if the kept
 * tail page is partially filled and shared (a later append would write into a
 * page other sequences read). */
int oracle_truncate(oracle_ctx *c, int n, const int32_t *seq_ids, const int32_t *new_len) {
    int i, j;
    for (i = 0; i < n; ++i) {
        int s = seq_ids[i];
        if (!seq_ok(c, s)) return ORACLE_ERR_INVALID_SEQ;
        for (j = 0; j < i; ++j) if (seq_ids[j] == s) return ORACLE_ERR_INVALID_SEQ;
        if (new_len[i] < 0 || new_len[i] > c->len[s]) return ORACLE_ERR_INVALID;
        if (new_len[i] % c->ps) {
            int pg = c->table[(size_t)s * c->max_pages_per_seq + new_len[i] / c->ps];
            if (c->refcount[pg] > 1) return ORACLE_ERR_SHARED;
        }
    }
    for (i = 0; i < n; ++i) {
        int s = seq_ids[i], keep = pages_of(c, new_len[i]), np = pages_of(c, c->len[s]);
        int32_t *t = c->table + (size_t)s * c->max_pages_per_seq;
        for (j = keep; j < np; ++j) { c->refcount[t[j]] -= 1; t[j] = -1; }
        c->len[s] = new_len[i];
    }
    return ORACLE_OK;
}

/* ---- export (bit-exact parity of the integer state) ---------------------- */
int oracle_export_seq(const oracle_ctx *c, int seq, int32_t *len_out, int32_t *table_out) {
    int j, np;
    if (seq < 0 || seq >= c->max_seqs) return ORACLE_ERR_INVALID_SEQ;
    if (!c->live[seq]) { *len_out = -1; return ORACLE_OK; }
    *len_out = c->len[seq];
    np = pages_of(c, c->len[seq]);
    for (j = 0; j < np; ++j) table_out[j] = c->table[(size_t)seq * c->max_pages_per_seq + j];
    return ORACLE_OK;
}

int oracle_export_refcounts(const oracle_ctx *c, int32_t *out) {
    memcpy(out, c->refcount, (size_t)c->num_pages * sizeof(int32_t));
    return ORACLE_OK;
}

/* logical K/V of tokens [t0, t0+n) of one sequence, storage dtype, [n][Hkv][D] */
int oracle_read_kv(const oracle_ctx *c, int seq, int t0, int n, void *k_out, void *v_out) {
    int t, h;
    if (!seq_ok(c, seq) || !c->store_kv || t0 < 0 || n < 0 || t0 + n > c->len[seq])
        return ORACLE_ERR_INVALID;
    for (t = 0; t < n; ++t) {
        int page = c->table[(size_t)seq * c->max_pages_per_seq + (t0 + t) / c->ps];
        int slot = (t0 + t) % c->ps;
        for (h = 0; h < c->Hkv; ++h) {
            size_t src = kv_index(c, page, h, slot) * c->elt;
            size_t dst = (((size_t)t * c->Hkv + h) * c->D) * c->elt;
            memcpy((uint8_t *)k_out + dst, c->kpool + src, c->D * c->elt);
            memcpy((uint8_t *)v_out + dst, c->vpool + src, c->D * c->elt);
        }
    }
    return ORACLE_OK;
}

/* ---- attention: the plain definition ---------------------------------------
 * One query row (sequence seq, q head h, query vector q[D] in storage dtype)
 * over tokens [t0, t1) of the sequence, walking the block table token by
 * token.  out[D], *lse in fp64.  If p_out != NULL it receives the t1-t0
 * softmax probabilities.  Empty range: out = 0, lse = -inf (A-15). */
static int attend_range(const oracle_ctx *c, int seq, int h, const uint8_t *q, int t0, int t1,
                        double *out, double *lse, double *p_out) {
    int D = c->D, kvh = h / (c->Hq / c->Hkv), n = t1 - t0, t, d;
    const int32_t *tab = c->table + (size_t)seq * c->max_pages_per_seq;
    double *s, m, Z;
    for (d = 0; d < D; ++d) out[d] = 0.0;
    if (n <= 0) { *lse = -INFINITY; return ORACLE_OK; }
    s = (double *)malloc((size_t)n * sizeof(double));
    if (!s) return ORACLE_ERR_INVALID;
    m = -INFINITY;
    for (t = 0; t < n; ++t) {                        /* s_t = scale * <q, k_t> */
        size_t ki = kv_index(c, tab[(t0 + t) / c->ps], kvh, (t0 + t) % c->ps);
        double acc = 0.0;
        for (d = 0; d < D; ++d) acc += load_q(c, q, (size_t)d) * load_elt(c, c->kpool, ki + d);
        s[t] = c->scale * acc;
        if (s[t] > m) m = s[t];
    }
    Z = 0.0;
    for (t = 0; t < n; ++t) Z += exp(s[t] - m);      /* Z = sum exp(s_t - m) */
    for (t = 0; t < n; ++t) {                        /* out = sum p_t v_t */
        size_t vi = kv_index(c, tab[(t0 + t) / c->ps], kvh, (t0 + t) % c->ps);
        double p = exp(s[t] - m) / Z;
        if (p_out) p_out[t] = p;
        for (d = 0; d < D; ++d) out[d] += p * load_elt(c, c->vpool, vi + d);
    }
    *lse = m + log(Z);
    free(s);
    return ORACLE_OK;
}

/* decode (q_len = 1, A-12): q [n][Hq][D] storage dtype; out [n][Hq][D], lse [n][Hq] fp64.
 * Fork groups are ignored entirely: each sequence attends all of its own tokens. */
int oracle_decode(const oracle_ctx *c, int n, const int32_t *seq_ids, const void *q, double *out,
                  double *lse) {
    int i, rc = ORACLE_OK;
    if (!c->store_kv) return ORACLE_ERR_INVALID;
    for (i = 0; i < n; ++i) if (!seq_ok(c, seq_ids[i])) return ORACLE_ERR_INVALID_SEQ;
#pragma omp parallel for schedule(dynamic, 1)
    for (i = 0; i < n * c->Hq; ++i) {
        int si = i / c->Hq, h = i % c->Hq, s = seq_ids[si];
        const uint8_t *qr = (const uint8_t *)q + ((size_t)si * c->Hq + h) * c->D * q_elt(c);
        int r = attend_range(c, s, h, qr, 0, c->len[s], out + ((size_t)si * c->Hq + h) * c->D,
                             lse + (size_t)si * c->Hq + h, NULL);
        if (r != ORACLE_OK) rc = r;
    }
    return rc;
}

/* verify (A-13): q [sum k][Hq][D], ragged by q_indptr[n+1]; the k_i draft
 * tokens' KV are the last k_i tokens of sequence i; row j attends tokens
 * t <= len_i - k_i + j.  out [sum k][Hq][D], lse [sum k][Hq]. */
int oracle_verify(const oracle_ctx *c, int n, const int32_t *seq_ids, const int32_t *q_indptr,
                  const void *q, double *out, double *lse) {
    int i, rc = ORACLE_OK, rows;
    if (!c->store_kv) return ORACLE_ERR_INVALID;
    for (i = 0; i < n; ++i) {
        int k = q_indptr[i + 1] - q_indptr[i];
        if (!seq_ok(c, seq_ids[i])) return ORACLE_ERR_INVALID_SEQ;
        if (k < 1 || k > c->len[seq_ids[i]]) return ORACLE_ERR_INVALID;
    }
    rows = q_indptr[n] * c->Hq;
#pragma omp parallel for schedule(dynamic, 1)
    for (i = 0; i < rows; ++i) {
        int row = i / c->Hq, h = i % c->Hq, si = 0, s, k, j, r;
        const uint8_t *qr = (const uint8_t *)q + (size_t)i * c->D * q_elt(c);
        while (q_indptr[si + 1] <= row) ++si;
        s = seq_ids[si]; k = q_indptr[si + 1] - q_indptr[si]; j = row - q_indptr[si];
        r = attend_range(c, s, h, qr, 0, c->len[s] - k + j + 1, out + (size_t)i * c->D, lse + i, NULL);
        if (r != ORACLE_OK) rc = r;
    }
    return rc;
}

/* single row over an arbitrary token range, optionally returning probabilities
 * (used by the pins: softmax rows sum to 1; partials for the cascade routine) */
int oracle_attend_range(const oracle_ctx *c, int seq, int h, const void *q_row, int t0, int t1,
                        double *out, double *lse, double *p_out) {
    if (!seq_ok(c, seq) || !c->store_kv || h < 0 || h >= c->Hq || t0 < 0 || t1 > c->len[seq])
        return ORACLE_ERR_INVALID;
    return attend_range(c, seq, h, (const uint8_t *)q_row, t0, t1, out, lse, p_out);
}

/* log-sum-exp merge of two partials (the cascade formula):
 *   M = max(lse_a, lse_b), w_x = exp(lse_x - M),
 *   o = (w_a o_a + w_b o_b)/(w_a + w_b), lse = M + ln(w_a + w_b);
 * an empty part (lse = -inf) has weight 0 and is skipped. */
void oracle_merge2(int D, const double *oa, double lsea, const double *ob, double lseb, double *out,
                   double *lse) {
    int d;
    double M, wa, wb;
    if (lsea == -INFINITY && lseb == -INFINITY) {
        for (d = 0; d < D; ++d) out[d] = 0.0;
        *lse = -INFINITY;
        return;
    }
    if (lsea == -INFINITY) { for (d = 0; d < D; ++d) out[d] = ob[d]; *lse = lseb; return; }
    if (lseb == -INFINITY) { for (d = 0; d < D; ++d) out[d] = oa[d]; *lse = lsea; return; }
    M = lsea > lseb ? lsea : lseb;
    wa = exp(lsea - M); wb = exp(lseb - M);
    for (d = 0; d < D; ++d) out[d] = (wa * oa[d] + wb * ob[d]) / (wa + wb);
    *lse = M + log(wa + wb);
}

/* cascade reference: split the sequence at token `split` (page aligned, 0 <= split <= len),
 * attend [0,split) and [split,len) separately, merge.  Used ONLY to pin oracle_decode. */
int oracle_cascade_row(const oracle_ctx *c, int seq, int h, const void *q_row, int split, double *out,
                       double *lse) {
    int r, D = c->D;
    double *oa, *ob, la, lb;
    if (!seq_ok(c, seq) || split < 0 || split > c->len[seq] || split % c->ps) return ORACLE_ERR_INVALID;
    oa = (double *)malloc(2 * (size_t)D * sizeof(double));
    if (!oa) return ORACLE_ERR_INVALID;
    ob = oa + D;
    r = attend_range(c, seq, h, (const uint8_t *)q_row, 0, split, oa, &la, NULL);
    if (r == ORACLE_OK) r = attend_range(c, seq, h, (const uint8_t *)q_row, split, c->len[seq], ob, &lb, NULL);
    if (r == ORACLE_OK) oracle_merge2(D, oa, la, ob, lb, out, lse);
    free(oa);
    return r;
}

/* ---- dense (unpaged) form of the same definition ---------------------------
 * K, V: [n][D] storage dtype for ONE kv head; used for sampled outputs of the
 * full-size configs where no paged oracle state is built, and pinned against
 * the paged routine. */
int oracle_attend_dense(int dtype, int D, double scale, const void *q_row, const void *K,
                        const void *V, int n, double *out, double *lse) {
    oracle_ctx tmp;
    int t, d;
    double *s, m = -INFINITY, Z = 0.0;
    memset(&tmp, 0, sizeof(tmp));
    tmp.dtype = dtype;
    for (d = 0; d < D; ++d) out[d] = 0.0;
    if (n <= 0) { *lse = -INFINITY; return ORACLE_OK; }
    s = (double *)malloc((size_t)n * sizeof(double));
    if (!s) return ORACLE_ERR_INVALID;
    for (t = 0; t < n; ++t) {
        double acc = 0.0;
        for (d = 0; d < D; ++d)
            acc += load_q(&tmp, (const uint8_t *)q_row, (size_t)d) *
                   load_elt(&tmp, (const uint8_t *)K, (size_t)t * D + d);
        s[t] = scale * acc;
        if (s[t] > m) m = s[t];
    }
    for (t = 0; t < n; ++t) Z += exp(s[t] - m);
    for (t = 0; t < n; ++t) {
        double p = exp(s[t] - m) / Z;
        for (d = 0; d < D; ++d) out[d] += p * load_elt(&tmp, (const uint8_t *)V, (size_t)t * D + d);
    }
    *lse = m + log(Z);
    free(s);
    return ORACLE_OK;
}

/* exact widening of n stored K/V elements (for the pins of the storage formats) */
void oracle_widen(int dtype, const void *src, long n, double *out) {
    oracle_ctx tmp;
    long i;
    memset(&tmp, 0, sizeof(tmp));
    tmp.dtype = dtype;
    for (i = 0; i < n; ++i) out[i] = load_elt(&tmp, (const uint8_t *)src, (size_t)i);
}

/* threads the OpenMP loops above may use (timing only: bench.py's single-thread baseline) */
void oracle_set_num_threads(int n) {
#ifdef _OPENMP
    extern void omp_set_num_threads(int);
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
