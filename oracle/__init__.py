"""CPU fp64 oracle for the Spork fork / decode / verify / release path.

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import this package.  It
shares no code with paper_2607_03333_b200 (the CUDA path) and never imports it.

The arithmetic lives in spork_oracle.c (plain C, fp64); this file only builds
that file with gcc and marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "spork_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

F32, BF16, E4M3KV = 0, 1, 2
DTYPES = {"f32": F32, "bf16": BF16, "e4m3": E4M3KV}      # "e4m3": K, V e4m3 bytes, Q bf16
KV_NP = {"f32": np.float32, "bf16": np.uint16, "e4m3": np.uint8}   # storage arrays are bit patterns
Q_NP = {"f32": np.float32, "bf16": np.uint16, "e4m3": np.uint16}

OK = 0
ERR_INVALID, ERR_OOM, ERR_NO_SLOT, ERR_TOO_LONG, ERR_INVALID_SEQ, ERR_SHARED = -1, -2, -3, -4, -5, -6


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp spork_oracle.c -> liboracle.so (in-tree)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-Wall", "-Wextra",
           "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        P, I, D = C.c_void_p, C.c_int, C.c_double
        sig = {
            "oracle_create": ([I] * 8 + [D, I], P),
            "oracle_destroy": ([P], None),
            "oracle_seq_create": ([P, I, P], I),
            "oracle_append": ([P, I, P, P, P, P], I),
            "oracle_fork": ([P, I, P, P], I),
            "oracle_release": ([P, I, P], I),
            "oracle_truncate": ([P, I, P, P], I),
            "oracle_export_seq": ([P, I, P, P], I),
            "oracle_export_refcounts": ([P, P], I),
            "oracle_read_kv": ([P, I, I, I, P, P], I),
            "oracle_decode": ([P, I, P, P, P, P], I),
            "oracle_verify": ([P, I, P, P, P, P, P], I),
            "oracle_attend_range": ([P, I, I, P, I, I, P, P, P], I),
            "oracle_merge2": ([I, P, D, P, D, P, P], None),
            "oracle_cascade_row": ([P, I, I, P, I, P, P], I),
            "oracle_attend_dense": ([I, I, D, P, P, P, I, P, P], I),
            "oracle_widen": ([I, P, C.c_long, P], None),
            "oracle_num_threads": ([], I),
            "oracle_set_num_threads": ([I], None),
        }
        for name, (args, res) in sig.items():
            f = getattr(_lib, name)
            f.argtypes = args
            f.restype = res
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32).reshape(-1))


def num_threads() -> int:
    return int(lib().oracle_num_threads())


class OracleError(RuntimeError):
    def __init__(self, code: int):
        super().__init__(f"oracle error {code}")
        self.code = code


class Oracle:
    """numpy-facing handle; also the 'engine' interface of synth.build_state."""

    def __init__(self, dtype: str, Hq: int, Hkv: int, D: int, num_pages: int, max_seqs: int,
                 max_pages_per_seq: int, scale: float, page_size: int = 16, store_kv: bool = True):
        self.dtype, self.Hq, self.Hkv, self.D, self.ps = dtype, Hq, Hkv, D, page_size
        self.num_pages, self.max_seqs, self.max_pages_per_seq = num_pages, max_seqs, max_pages_per_seq
        self.scale = scale
        self.np_dtype = KV_NP[dtype]
        self.q_dtype = Q_NP[dtype]
        self._h = lib().oracle_create(DTYPES[dtype], Hq, Hkv, D, page_size, num_pages, max_seqs,
                                      max_pages_per_seq, float(scale), int(store_kv))
        if not self._h:
            raise MemoryError("oracle_create failed")

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @staticmethod
    def _chk(rc: int, raise_on_error: bool = True) -> int:
        if rc != OK and raise_on_error:
            raise OracleError(rc)
        return rc

    # ---- state calls --------------------------------------------------------
    def seq_create(self, n: int) -> np.ndarray:
        ids = np.zeros(n, np.int32)
        self._chk(lib().oracle_seq_create(self._h, n, _p(ids)))
        return ids

    def append(self, seq_ids, n_tokens, k: np.ndarray, v: np.ndarray, check: bool = True) -> int:
        s, nt = _i32(seq_ids), _i32(n_tokens)
        k = np.ascontiguousarray(k, dtype=self.np_dtype)
        v = np.ascontiguousarray(v, dtype=self.np_dtype)
        assert k.size == int(nt.sum()) * self.Hkv * self.D and v.size == k.size
        return self._chk(lib().oracle_append(self._h, len(s), _p(s), _p(nt), _p(k), _p(v)), check)

    def fork(self, parents, check: bool = True):
        p = _i32(parents)
        ch = np.full(len(p), -1, np.int32)
        rc = self._chk(lib().oracle_fork(self._h, len(p), _p(p), _p(ch)), check)
        return ch if check else (rc, ch)

    def release(self, seq_ids, check: bool = True) -> int:
        s = _i32(seq_ids)
        return self._chk(lib().oracle_release(self._h, len(s), _p(s)), check)

    def truncate(self, seq_ids, new_len, check: bool = True) -> int:
        s, nl = _i32(seq_ids), _i32(new_len)
        return self._chk(lib().oracle_truncate(self._h, len(s), _p(s), _p(nl)), check)

    # ---- partial-token accept ---------------------------------
    def accept(self, seq_ids, q_indptr, draft_tokens, target_tokens, check: bool = True):
        """PAPER.md:236-237 (section 4.3): the engine "verifies the draft ... the first k matching tokens
        are accepted".  Sequence i holds k_i = q_indptr[i+1] - q_indptr[i] drafts as its last k_i tokens;
        target_tokens[j] is the target model's greedy token at draft position j.  accept_len_i = the
        number of leading positions with draft == target; the rejected drafts' KV is dropped:
        truncate(seq_i, len_i - (k_i - accept_len_i)).  Returns (rc, accept_len[n])."""
        acc = accept_len(q_indptr, draft_tokens, target_tokens)
        qi = np.asarray(q_indptr, dtype=np.int64)
        k = qi[1:] - qi[:-1]
        new_len = np.array([self.export_seq(int(s))[0] for s in seq_ids], dtype=np.int64) - (k - acc)
        rc = self.truncate(seq_ids, new_len.astype(np.int32), check)
        return rc, acc

    # ---- export -------------------------------------------------------------
    def export_seq(self, seq: int):
        """(len, table[ceil(len/ps)]); len = -1 if the slot is not live."""
        ln = np.zeros(1, np.int32)
        tab = np.full(self.max_pages_per_seq, -1, np.int32)
        self._chk(lib().oracle_export_seq(self._h, int(seq), _p(ln), _p(tab)))
        L = int(ln[0])
        return L, tab[:max(0, (L + self.ps - 1) // self.ps)].copy()

    def export_refcounts(self) -> np.ndarray:
        out = np.zeros(self.num_pages, np.int32)
        self._chk(lib().oracle_export_refcounts(self._h, _p(out)))
        return out

    def read_kv(self, seq: int, t0: int, n: int):
        k = np.zeros((n, self.Hkv, self.D), self.np_dtype)
        v = np.zeros_like(k)
        self._chk(lib().oracle_read_kv(self._h, int(seq), int(t0), int(n), _p(k), _p(v)))
        return k, v

    # ---- attention ----------------------------------------------------------
    def decode(self, seq_ids, q: np.ndarray):
        s = _i32(seq_ids)
        q = np.ascontiguousarray(q, dtype=self.q_dtype)
        assert q.shape == (len(s), self.Hq, self.D)
        out = np.zeros((len(s), self.Hq, self.D), np.float64)
        lse = np.zeros((len(s), self.Hq), np.float64)
        self._chk(lib().oracle_decode(self._h, len(s), _p(s), _p(q), _p(out), _p(lse)))
        return out, lse

    def verify(self, seq_ids, q_indptr, q: np.ndarray, check: bool = True):
        s, qi = _i32(seq_ids), _i32(q_indptr)
        q = np.ascontiguousarray(q, dtype=self.q_dtype)
        rows = int(qi[-1])
        assert q.shape == (rows, self.Hq, self.D)
        out = np.zeros((rows, self.Hq, self.D), np.float64)
        lse = np.zeros((rows, self.Hq), np.float64)
        rc = self._chk(lib().oracle_verify(self._h, len(s), _p(s), _p(qi), _p(q), _p(out), _p(lse)),
                       check)
        return (out, lse) if check else (rc, out, lse)

    def attend_range(self, seq: int, h: int, q_row: np.ndarray, t0: int, t1: int, probs: bool = False):
        q_row = np.ascontiguousarray(q_row, dtype=self.q_dtype)
        out = np.zeros(self.D, np.float64)
        lse = np.zeros(1, np.float64)
        p = np.zeros(max(0, t1 - t0), np.float64) if probs else None
        self._chk(lib().oracle_attend_range(self._h, int(seq), int(h), _p(q_row), int(t0), int(t1),
                                            _p(out), _p(lse), _p(p)))
        return (out, float(lse[0]), p) if probs else (out, float(lse[0]))

    def cascade_row(self, seq: int, h: int, q_row: np.ndarray, split: int):
        q_row = np.ascontiguousarray(q_row, dtype=self.q_dtype)
        out = np.zeros(self.D, np.float64)
        lse = np.zeros(1, np.float64)
        self._chk(lib().oracle_cascade_row(self._h, int(seq), int(h), _p(q_row), int(split), _p(out),
                                           _p(lse)))
        return out, float(lse[0])


def merge2(oa: np.ndarray, lsea: float, ob: np.ndarray, lseb: float):
    oa = np.ascontiguousarray(oa, np.float64)
    ob = np.ascontiguousarray(ob, np.float64)
    out = np.zeros_like(oa)
    lse = np.zeros(1, np.float64)
    lib().oracle_merge2(len(oa), _p(oa), float(lsea), _p(ob), float(lseb), _p(out), _p(lse))
    return out, float(lse[0])


def attend_dense(dtype: str, scale: float, q_row: np.ndarray, K: np.ndarray, V: np.ndarray):
    """Plain definition on an unpaged [n][D] K/V of one kv head (storage dtype)."""
    q_row = np.ascontiguousarray(q_row, dtype=Q_NP[dtype])
    K = np.ascontiguousarray(K, dtype=KV_NP[dtype])
    V = np.ascontiguousarray(V, dtype=KV_NP[dtype])
    n, D = K.shape
    out = np.zeros(D, np.float64)
    lse = np.zeros(1, np.float64)
    rc = lib().oracle_attend_dense(DTYPES[dtype], D, float(scale), _p(q_row), _p(K), _p(V), n, _p(out),
                                   _p(lse))
    if rc != OK:
        raise OracleError(rc)
    return out, float(lse[0])


def set_num_threads(n: int) -> None:
    """Threads of the oracle's OpenMP loops (bench.py's single-thread baseline; results do not depend on it)."""
    lib().oracle_set_num_threads(int(n))


def widen(dtype: str, a: np.ndarray) -> np.ndarray:
    """The oracle's exact widening of stored K/V elements (bit patterns) to float64."""
    a = np.ascontiguousarray(a, dtype=KV_NP[dtype])
    out = np.zeros(a.shape, np.float64)
    lib().oracle_widen(DTYPES[dtype], _p(a), a.size, _p(out))
    return out


def accept_len(q_indptr, draft_tokens, target_tokens) -> np.ndarray:
    """Longest greedy-matching prefix per sequence, written out position by
    position: walk the drafts of sequence i from the first; stop at the first mismatch."""
    qi = np.asarray(q_indptr, dtype=np.int64)
    d = np.asarray(draft_tokens)
    t = np.asarray(target_tokens)
    out = np.zeros(len(qi) - 1, dtype=np.int32)
    for i in range(len(qi) - 1):
        a = 0
        for j in range(int(qi[i]), int(qi[i + 1])):
            if int(d[j]) != int(t[j]):
                break
            a += 1
        out[i] = a
    return out


def confidence(logits, span_indptr) -> np.ndarray:
    """D2 confidence score, Eq. 2: c = min_{i=2..L} exp(l_i), l_i the
    log-probability of the TOP-1 token at position i of the tool-name span.  logits: [n_pos][V], the
    spans are consecutive row ranges [span_indptr[s], span_indptr[s+1]); the first row of a span is
    skipped (i starts at 2: "the opening quote is always high-probability boilerplate"); a span of
    L <= 1 rows has an empty minimum, read as 1 (reading A-23).  fp64, the plain definition:
    l_i = x_max - ln sum_v exp(x_v)."""
    x = np.asarray(logits, dtype=np.float64)
    sp = np.asarray(span_indptr, dtype=np.int64)
    out = np.ones(len(sp) - 1, dtype=np.float64)
    for s in range(len(sp) - 1):
        c = 1.0
        for i in range(int(sp[s]) + 1, int(sp[s + 1])):
            row = x[i]
            m = float(row.max())
            lse = m + np.log(np.sum(np.exp(row - m)))
            c = min(c, float(np.exp(m - lse)))
        out[s] = c
    return out
