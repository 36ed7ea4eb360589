"""Seeded synthetic inputs for the Spork fork / cascade-decode / verify path.

This package is the ONLY code shared by the CUDA path's tests/bench and the CPU
oracle.  It holds no attention, softmax, merge or allocator arithmetic: it draws
random numbers, rounds them to the storage dtype, and replays a fixed script of
C-ABI-shaped calls (seq_create / append / fork / release) against whatever
"engine" object it is handed.

Recipe (BASELINE.json configs):
the paper's serving traffic (GAIA / HotpotQA / tau2-bench / BrowseComp on Qwen3
models) is not available, so only its *shape* statistics are
used: context ~15K, CoT ~2,000 tokens, probe <= 50
tokens, drafts ~18-30 tokens, 1-3 probes
per turn (Algorithm 1).  Values are iid N(0,1) (config 3: 1 %
of keys scaled x8), seed 0, one independent numpy sub-stream per
(config, tensor, group-or-sequence) so that any subset can be regenerated
without generating the rest.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import List, Optional, Sequence

import numpy as np

PAGE_SIZE = 16

# tensor ids of the independent sub-streams
T_SUFFIX_LEN = 0
T_PREFIX_K = 1
T_PREFIX_V = 2
T_SUFFIX_K = 3
T_SUFFIX_V = 4
T_Q = 5
T_OUTLIER_PREFIX = 6
T_OUTLIER_SUFFIX = 7
T_CHURN = 8
T_MISC = 9
T_COT_K = 10
T_COT_V = 11


def rng(cfg_no: int, tensor_no: int, index: int = 0) -> np.random.Generator:
    """Independent sub-stream; seed 0 everywhere."""
    return np.random.default_rng([0, int(cfg_no), int(tensor_no), int(index)])


# ----------------------------------------------------------------------------
# storage dtype helpers (bit manipulation only)
# ----------------------------------------------------------------------------
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit pattern (uint16), round-to-nearest-even."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    b = x.view(np.uint32)
    lsb = (b >> np.uint32(16)) & np.uint32(1)
    r = (b + np.uint32(0x7FFF) + lsb) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(u: np.ndarray) -> np.ndarray:
    """bf16 bit pattern (uint16) -> float32 (exact)."""
    u = np.ascontiguousarray(u, dtype=np.uint16)
    return (u.astype(np.uint32) << np.uint32(16)).view(np.float32)


def f32_to_e4m3_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> e4m3 ("fn") bit pattern (uint8): round-to-nearest-even, saturating at +-448.
    Format: 1 sign, 4 exponent bits (bias 7), 3 mantissa bits; exponent 0 is subnormal (m/8 * 2^-6)."""
    x = np.ascontiguousarray(x, dtype=np.float32).astype(np.float64)
    a = np.minimum(np.abs(x), 448.0)
    _, e = np.frexp(a)                           # a = f * 2^e, f in [0.5, 1)
    quantum = np.ldexp(1.0, np.maximum(e - 1, -6) - 3)   # spacing of the format at a (2^-9 below 2^-6)
    q = np.minimum(np.rint(a / quantum) * quantum, 448.0)   # np.rint: ties to even
    _, e2 = np.frexp(q)
    eb = np.where(q >= 2.0 ** -6, e2 - 1 + 7, 0)
    m = np.where(eb > 0, (q / np.ldexp(1.0, eb - 7) - 1.0) * 8.0, q / 2.0 ** -9)
    bits = (eb.astype(np.int64) << 3) | m.astype(np.int64) | (np.signbit(x).astype(np.int64) << 7)
    return bits.astype(np.uint8)


def e4m3_bits_to_f32(u: np.ndarray) -> np.ndarray:
    """e4m3 bit pattern (uint8) -> float32 (exact; 0x7f / 0xff are NaN)."""
    u = np.ascontiguousarray(u, dtype=np.uint8).astype(np.int64)
    e, m = (u >> 3) & 15, u & 7
    v = np.where(e == 0, np.ldexp(m / 8.0, -6), np.ldexp(1.0 + m / 8.0, e - 7))
    v = np.where((e == 15) & (m == 7), np.nan, v)
    return np.where(u >> 7, -v, v).astype(np.float32)


def to_storage(x: np.ndarray, dtype: str) -> np.ndarray:
    """Round float32 values once to the storage dtype ('f32', 'bf16' or 'e4m3')."""
    if dtype == "f32":
        return np.ascontiguousarray(x, dtype=np.float32)
    if dtype == "bf16":
        return f32_to_bf16_bits(x)
    if dtype == "e4m3":
        return f32_to_e4m3_bits(x)
    raise ValueError(dtype)


def storage_to_f64(x: np.ndarray, dtype: str) -> np.ndarray:
    """Exact widening of stored values (for test-side independent checks)."""
    if dtype == "f32":
        return np.asarray(x, dtype=np.float32).astype(np.float64)
    if dtype == "bf16":
        return bf16_bits_to_f32(x).astype(np.float64)
    if dtype == "e4m3":
        return e4m3_bits_to_f32(x).astype(np.float64)
    raise ValueError(dtype)


def storage_np_dtype(dtype: str):
    return {"f32": np.float32, "bf16": np.uint16, "e4m3": np.uint8}[dtype]


def q_dtype_of(dtype: str) -> str:
    """Storage dtype of the queries: the KV dtype, except that an e4m3 KV cache is queried in bf16."""
    return "bf16" if dtype == "e4m3" else dtype


# ----------------------------------------------------------------------------
# configs (BASELINE.json `configs`)
# ----------------------------------------------------------------------------
@dataclass(frozen=True)
class SporkConfig:
    name: str
    cfg_no: int
    dtype: str            # 'f32' | 'bf16' (KV and Q storage dtype) | 'e4m3' (KV; Q is bf16)
    Hq: int
    Hkv: int
    D: int
    n_groups: int
    group_size: int       # main + probes
    prefix_len: int       # P, shared by the whole fork group
    suffix_lo: int        # private suffix ~ U{lo..hi}, both inclusive (A-19)
    suffix_hi: int
    k_draft: int = 0      # 0: decode (q_len=1); >0: verify with k drafts/seq
    outlier_frac: float = 0.0   # config 3: Bernoulli per (token, kv head) on K
    outlier_scale: float = 8.0
    page_size: int = PAGE_SIZE

    @property
    def n_seqs(self) -> int:
        return self.n_groups * self.group_size

    @property
    def G(self) -> int:
        return self.Hq // self.Hkv

    @property
    def scale(self) -> float:
        return 1.0 / float(np.sqrt(self.D))

    @property
    def elt_bytes(self) -> int:
        return {"f32": 4, "bf16": 2, "e4m3": 1}[self.dtype]

    @property
    def q_dtype(self) -> str:
        return q_dtype_of(self.dtype)

    @property
    def token_bytes(self) -> int:
        """B_tok = K and V bytes of one token, one layer."""
        return 2 * self.Hkv * self.D * self.elt_bytes

    def scaled(self, **kw) -> "SporkConfig":
        return replace(self, **kw)


CFG1 = SporkConfig("cfg1_tiny_fp32", 1, "f32", 4, 1, 64, 1, 3, 256, 0, 32)
CFG2 = SporkConfig("cfg2_qwen3_4b_decode", 2, "bf16", 32, 8, 128, 16, 2, 4096, 1, 2048)
CFG3 = SporkConfig("cfg3_qwen3_32b_decode", 3, "bf16", 64, 8, 128, 32, 4, 8192, 1, 2000,
                   outlier_frac=0.01)
CFG4 = SporkConfig("cfg4_qwen3_32b_verify", 4, "bf16", 64, 8, 128, 16, 4, 16384, 0, 512,
                   k_draft=8)
CFG5 = SporkConfig("cfg5_qwen3_30b_a3b_decode", 5, "bf16", 32, 4, 128, 16, 8, 32768, 1, 4096)

CONFIGS = {1: CFG1, 2: CFG2, 3: CFG3, 4: CFG4, 5: CFG5}


# ----------------------------------------------------------------------------
# workload = lengths + lazily generated values
# ----------------------------------------------------------------------------
class Workload:
    """Lengths are drawn eagerly; K/V/Q values are generated per group / per
    sequence on demand from their own sub-streams (cheap to regenerate, so a
    full-size run never needs all of them on the host at once)."""

    def __init__(self, cfg: SporkConfig, k_per_seq: Optional[Sequence[int]] = None):
        self.cfg = cfg
        r = rng(cfg.cfg_no, T_SUFFIX_LEN)
        self.suffix_len = r.integers(cfg.suffix_lo, cfg.suffix_hi + 1,
                                     size=cfg.n_seqs).astype(np.int64)
        if k_per_seq is None:
            self.k = np.full(cfg.n_seqs, cfg.k_draft, dtype=np.int64)
        else:
            self.k = np.asarray(k_per_seq, dtype=np.int64)
            assert self.k.shape == (cfg.n_seqs,)
        # private tokens appended after the fork: suffix + drafts (A-14: L = P + s + k)
        self.private_len = self.suffix_len + self.k
        self.total_len = cfg.prefix_len + self.private_len

    # ---- group / sequence bookkeeping -------------------------------------
    def group_of(self, seq: int) -> int:
        return seq // self.cfg.group_size

    def members(self, g: int) -> List[int]:
        gs = self.cfg.group_size
        return list(range(g * gs, (g + 1) * gs))

    def unique_tokens(self) -> int:
        """sum_groups (P + sum_members (s + k))."""
        return int(self.cfg.n_groups * self.cfg.prefix_len + self.private_len.sum())

    def unique_kv_bytes(self) -> int:
        return self.unique_tokens() * self.cfg.token_bytes

    def naive_tokens(self) -> int:
        return int(self.total_len.sum())

    def q_rows(self) -> np.ndarray:
        """query rows per sequence (1 for decode, k for verify)."""
        return np.where(self.k > 0, self.k, 1).astype(np.int64)

    def flops(self) -> float:
        """4*D flops per (query row, q head, attended token); verify rows are
        causal within the drafts (row j sees L-k+j+1 tokens)."""
        c = self.cfg
        tot = 0.0
        for i in range(c.n_seqs):
            L, k = int(self.total_len[i]), int(self.k[i])
            if k == 0:
                att = L
            else:
                att = sum(L - k + j + 1 for j in range(k))
            tot += 4.0 * c.D * c.Hq * att
        return tot

    # ---- values -------------------------------------------------------------
    def _normal(self, tensor_no: int, index: int, n_tok: int, heads: int) -> np.ndarray:
        c = self.cfg
        r = rng(c.cfg_no, tensor_no, index)
        return r.standard_normal((n_tok, heads, c.D), dtype=np.float32)

    def _outliers(self, x: np.ndarray, tensor_no: int, index: int) -> np.ndarray:
        c = self.cfg
        if c.outlier_frac <= 0.0:
            return x
        r = rng(c.cfg_no, tensor_no, index)
        mask = r.random((x.shape[0], x.shape[1])) < c.outlier_frac   # per (token, kv head), A-17
        x = x.copy()
        x[mask] *= np.float32(c.outlier_scale)
        return x

    def prefix_kv(self, g: int):
        """K, V of group g's shared prefix, storage dtype, [P][Hkv][D]."""
        c = self.cfg
        k = self._outliers(self._normal(T_PREFIX_K, g, c.prefix_len, c.Hkv), T_OUTLIER_PREFIX, g)
        v = self._normal(T_PREFIX_V, g, c.prefix_len, c.Hkv)
        return to_storage(k, c.dtype), to_storage(v, c.dtype)

    def suffix_kv(self, seq: int):
        """K, V of sequence seq's private tokens (suffix then drafts), [s+k][Hkv][D]."""
        c = self.cfg
        n = int(self.private_len[seq])
        k = self._outliers(self._normal(T_SUFFIX_K, seq, n, c.Hkv), T_OUTLIER_SUFFIX, seq)
        v = self._normal(T_SUFFIX_V, seq, n, c.Hkv)
        return to_storage(k, c.dtype), to_storage(v, c.dtype)

    def q(self, seq: int) -> np.ndarray:
        """query rows of one sequence, storage dtype, [q_rows][Hq][D]."""
        c = self.cfg
        n = int(self.q_rows()[seq])
        return to_storage(self._normal(T_Q, seq, n, c.Hq), c.q_dtype)

    def q_all(self) -> np.ndarray:
        return np.concatenate([self.q(i) for i in range(self.cfg.n_seqs)], axis=0)

    def q_indptr(self) -> np.ndarray:
        return np.concatenate([[0], np.cumsum(self.q_rows())]).astype(np.int32)

    def group_indptr(self) -> np.ndarray:
        c = self.cfg
        return (np.arange(c.n_groups + 1) * c.group_size).astype(np.int32)

    def dense_kv(self, seq: int):
        """Logical K, V of one whole sequence, storage dtype, [L][Hkv][D]
        (prefix of its group followed by its private tokens)."""
        pk, pv = self.prefix_kv(self.group_of(seq))
        sk, sv = self.suffix_kv(seq)
        return np.concatenate([pk, sk], axis=0), np.concatenate([pv, sv], axis=0)


# ----------------------------------------------------------------------------
# the call script (same calls, same order, for every engine)
# ----------------------------------------------------------------------------
def build_state(engine, wl: Workload, interleave: bool = True, values: bool = True) -> np.ndarray:
    """Replays SURVEY.md 8(d) "Placement" through an engine exposing
    seq_create(n)->ids, append(seq_ids, n_tokens, k, v), fork(parents)->children.

    Mains are prefilled first (one append of P tokens each), probes are forked
    from their main at L = P (Algorithm 1 step 6), then private
    tokens are appended round-robin one page at a time across all sequences so
    that private pages interleave as under continuous batching.
    Returns seq_ids[n_seqs] in workload order (main first within each group).
    values=False replays the same calls with all-zero K/V (for engines whose allocator is all that
    matters, e.g. the fork-churn baseline): block tables and refcounts are the same.
    """
    c = wl.cfg
    mains = np.asarray(engine.seq_create(c.n_groups), dtype=np.int32)
    zeros = None if values else np.zeros((max(c.prefix_len, 1), c.Hkv, c.D), storage_np_dtype(c.dtype))
    for g in range(c.n_groups):
        pk, pv = wl.prefix_kv(g) if values else (zeros[:c.prefix_len], zeros[:c.prefix_len])
        engine.append(mains[g:g + 1], np.array([c.prefix_len], np.int32), pk, pv)
    seq_ids = np.zeros(c.n_seqs, dtype=np.int32)
    n_probe = c.group_size - 1
    if n_probe > 0:
        parents = np.repeat(mains, n_probe).astype(np.int32)
        children = np.asarray(engine.fork(parents), dtype=np.int32)
    for g in range(c.n_groups):
        seq_ids[g * c.group_size] = mains[g]
        for j in range(n_probe):
            seq_ids[g * c.group_size + 1 + j] = children[g * n_probe + j]

    priv = [wl.suffix_kv(i) for i in range(c.n_seqs)] if values else None
    done = np.zeros(c.n_seqs, dtype=np.int64)
    step = c.page_size if interleave else int(max(1, wl.private_len.max()))
    while True:
        todo = np.nonzero(done < wl.private_len)[0]
        if todo.size == 0:
            break
        n_tok = np.minimum(step, wl.private_len[todo] - done[todo]).astype(np.int32)
        if values:
            ks = np.concatenate([priv[i][0][done[i]:done[i] + n] for i, n in zip(todo, n_tok)], axis=0)
            vs = np.concatenate([priv[i][1][done[i]:done[i] + n] for i, n in zip(todo, n_tok)], axis=0)
        else:
            ks = vs = np.zeros((int(n_tok.sum()), c.Hkv, c.D), storage_np_dtype(c.dtype))
        engine.append(seq_ids[todo], n_tok, ks, vs)
        done[todo] += n_tok
    return seq_ids


# ----------------------------------------------------------------------------
# successive probes (Algorithm 1 steps 4-6; Fig. 4)
# ----------------------------------------------------------------------------
class SuccessiveWorkload(Workload):
    """Probe r (r = 1 .. group_size-1) of a group is forked after the main stream has decoded
    r * stride further CoT tokens, so it shares P + r * stride tokens with the main stream (and with
    every later probe), not just P.  Token content per group: prefix(g), then the group's CoT stream
    cot(g) of (group_size-1) * stride tokens (the main stream's tokens between the fork points), then
    each sequence's private tokens (suffix, then drafts) from its own sub-stream."""

    def __init__(self, cfg: SporkConfig, stride: int, k_per_seq: Optional[Sequence[int]] = None):
        super().__init__(cfg, k_per_seq)
        self.stride = int(stride)
        gs = cfg.group_size
        r = np.arange(cfg.n_seqs) % gs                       # 0: main, r: probe r
        self.fork_extra = np.where(r == 0, (gs - 1) * self.stride, r * self.stride).astype(np.int64)
        self.total_len = cfg.prefix_len + self.fork_extra + self.private_len

    def cot_kv(self, g: int):
        c = self.cfg
        n = (c.group_size - 1) * self.stride
        k = self._outliers(self._normal(T_COT_K, g, n, c.Hkv), T_OUTLIER_PREFIX, 1_000_000 + g)
        v = self._normal(T_COT_V, g, n, c.Hkv)
        return to_storage(k, c.dtype), to_storage(v, c.dtype)

    def unique_tokens(self) -> int:
        """Nested sharing: every token is counted once per group.  A fork point that is not page
        aligned duplicates its partially filled page into the probe (those tokens are private copies)."""
        c = self.cfg
        dup = sum((c.prefix_len + r * self.stride) % c.page_size for r in range(1, c.group_size))
        return int(c.n_groups * (c.prefix_len + (c.group_size - 1) * self.stride + dup) + self.private_len.sum())

    def single_level_tokens(self) -> int:
        """What a cascade with ONE shared level reads: the group-wide common prefix (up to the first
        fork point) once, everything beyond it once per member."""
        c = self.cfg
        if c.group_size < 2:
            return self.naive_tokens()
        shared = ((c.prefix_len + self.stride) // c.page_size) * c.page_size
        return int(c.n_groups * shared + (self.total_len - shared).sum())

    def dense_kv(self, seq: int):
        g = self.group_of(seq)
        pk, pv = self.prefix_kv(g)
        ck, cv = self.cot_kv(g)
        sk, sv = self.suffix_kv(seq)
        e = int(self.fork_extra[seq])
        return np.concatenate([pk, ck[:e], sk], axis=0), np.concatenate([pv, cv[:e], sv], axis=0)


def build_state_successive(engine, wl: SuccessiveWorkload) -> np.ndarray:
    """The call script of one paper turn per group (Algorithm 1): main prefilled,
    then for r = 1 .. R: main decodes `stride` more CoT tokens (step 5), probe r is forked from it
    (step 6); afterwards every stream appends its private tokens round-robin one page at a time."""
    c = wl.cfg
    mains = np.asarray(engine.seq_create(c.n_groups), dtype=np.int32)
    for g in range(c.n_groups):
        pk, pv = wl.prefix_kv(g)
        engine.append(mains[g:g + 1], np.array([c.prefix_len], np.int32), pk, pv)
    seq_ids = np.zeros(c.n_seqs, dtype=np.int32)
    seq_ids[0::c.group_size] = mains
    cot = [wl.cot_kv(g) for g in range(c.n_groups)]
    st = wl.stride
    for r in range(1, c.group_size):
        ks = np.concatenate([cot[g][0][(r - 1) * st:r * st] for g in range(c.n_groups)], axis=0)
        vs = np.concatenate([cot[g][1][(r - 1) * st:r * st] for g in range(c.n_groups)], axis=0)
        engine.append(mains, np.full(c.n_groups, st, np.int32), ks, vs)
        seq_ids[r::c.group_size] = np.asarray(engine.fork(mains), dtype=np.int32)
    priv = [wl.suffix_kv(i) for i in range(c.n_seqs)]
    done = np.zeros(c.n_seqs, dtype=np.int64)
    while True:
        todo = np.nonzero(done < wl.private_len)[0]
        if todo.size == 0:
            break
        n_tok = np.minimum(c.page_size, wl.private_len[todo] - done[todo]).astype(np.int32)
        ks = np.concatenate([priv[i][0][done[i]:done[i] + n] for i, n in zip(todo, n_tok)], axis=0)
        vs = np.concatenate([priv[i][1][done[i]:done[i] + n] for i, n in zip(todo, n_tok)], axis=0)
        engine.append(seq_ids[todo], n_tok, ks, vs)
        done[todo] += n_tok
    return seq_ids


def churn_parents(cfg_no: int, n_forks: int, live_ids: np.ndarray, index: int = 0) -> np.ndarray:
    """Config 5 fork churn: parents drawn uniformly from the live sequences."""
    r = rng(cfg_no, T_CHURN, index)
    return np.asarray(live_ids, dtype=np.int32)[r.integers(0, len(live_ids), size=n_forks)]


# ---------------------------------------------------------------------------
# D2 confidence: synthetic next-token logits of probe tool-name spans
# ---------------------------------------------------------------------------
T_LOGITS = 40


def probe_logits(n_spans: int, vocab: int, seed: int = 0, max_len: int = 5):
    """fp32 logits [n_pos][vocab] and span_indptr[n_spans + 1] for `n_spans` tool-name spans of
    1..max_len generated tokens each ("typically 1-4 tokens" after the opening
    quote, which is the span's first row).  Rows are N(0, 2^2) noise; one token per row is
    lifted by U(0, 14) so that top-1 probabilities spread over (0, 1) as in Fig. 8
    (PAPER.md:215-223).  Stand-in for real probe logits (no model weights here)."""
    r = rng(0, T_LOGITS, seed)
    lens = r.integers(1, max_len + 1, size=n_spans)
    indptr = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    n_pos = int(indptr[-1])
    x = (2.0 * r.standard_normal((n_pos, vocab), dtype=np.float32)).astype(np.float32)
    top = r.integers(0, vocab, size=n_pos)
    x[np.arange(n_pos), top] += r.uniform(0.0, 14.0, size=n_pos).astype(np.float32)
    return x, indptr
