"""paper_2607_03333_b200 -- Python binding of libspork (the C ABI in include/spork.h).

Argument marshalling only: every step of the path (allocator, fork, append,
release, cascade decode attention, verify attention, merge) runs in the CUDA
kernels of libspork.so.  PyTorch is used for device memory and streams.  There
is no CPU fallback: constructing a `Spork` without the built library or without
a CUDA device raises.

Method names mirror the ABI: seq_create, append, fork, release, truncate,
decode_attn, verify_attn, export, export_refcounts, read_kv, status.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

from . import build as _build

F32, BF16, E4M3 = 0, 1, 2
PAGE_SIZE = 16

OK = 0
ERR_STALE = -9
ERR_LIMIT = -10
CONFIDENCE_STATIC_MAX_ROWS = 16384
ERR_INVALID, ERR_OOM, ERR_NO_SLOT, ERR_TOO_LONG, ERR_INVALID_SEQ, ERR_SHARED, ERR_CUDA, ERR_DEVICE = (
    -1, -2, -3, -4, -5, -6, -7, -8)

# every symbol include/spork.h declares (tests check that the library exports them all)
ABI_SYMBOLS = [
    "spork_page_bytes", "spork_create", "spork_destroy", "spork_seq_create", "spork_append",
    "spork_fork", "spork_release", "spork_truncate", "spork_decode_attn", "spork_verify_attn",
    "spork_decode_attn_host", "spork_verify_attn_host", "spork_export", "spork_export_refcounts",
    "spork_read_kv", "spork_free_pages", "spork_status", "spork_last_plan", "spork_last_launches",
    "spork_accept", "spork_confidence", "spork_set_timing", "spork_last_kernel_ms", "spork_set_tensor_path_min_rows", "spork_set_many_row_variant", "spork_set_stream_k", "spork_strerror",
    "spork_set_cascade_levels", "spork_layers", "spork_write_kv_layer", "spork_decode_attn_layers",
    "spork_verify_attn_layers", "spork_hbm_read_probe",
    "spork_turn_prepare", "spork_turn_append", "spork_turn_verify", "spork_turn_accept", "spork_turn_decode",
    "spork_turn_sync", "spork_turn_destroy", "spork_confidence_static",
]


class SporkConfig(C.Structure):
    _fields_ = [("dtype", C.c_int32), ("num_q_heads", C.c_int32), ("num_kv_heads", C.c_int32),
                ("head_dim", C.c_int32), ("page_size", C.c_int32), ("num_pages", C.c_int32),
                ("max_seqs", C.c_int32), ("max_pages_per_seq", C.c_int32), ("scale", C.c_float)]


class PlanInfo(C.Structure):
    _fields_ = [("n_items", C.c_int32), ("n_prefix_items", C.c_int32), ("chunk_tokens", C.c_int32),
                ("grid", C.c_int32), ("kernel", C.c_int32), ("plan_cached", C.c_int32),
                ("unique_tokens", C.c_int64), ("naive_tokens", C.c_int64),
                ("partial_rows", C.c_int64), ("launches", C.c_int32), ("n_umma_items", C.c_int32),
                ("n_two_pipe_items", C.c_int32), ("stream_k", C.c_int32), ("plan_host_us", C.c_float),
                ("plan_builds", C.c_int32), ("n_levels", C.c_int32), ("reserved", C.c_int32)]

    def as_dict(self):
        return {k: (float if t is C.c_float else int)(getattr(self, k)) for k, t in self._fields_ if k != "reserved"}


_lib = None


def lib_path() -> str:
    return _build.LIB


def load(build_if_missing: bool = True):
    """dlopen libspork.so (building it first if needed) and declare the ABI signatures."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build() if build_if_missing else _build.LIB
    if not os.path.exists(path):
        raise RuntimeError(f"libspork.so not found at {path}; run python -m paper_2607_03333_b200.build")
    lib = C.CDLL(path)
    P, I, I32 = C.c_void_p, C.c_int, C.c_int32
    sig = {
        "spork_page_bytes": ([P], C.c_size_t),
        "spork_create": ([P, P, P, P], I),
        "spork_destroy": ([P], I),
        "spork_seq_create": ([P, I, P], I),
        "spork_append": ([P, I, P, P, P, P, P], I),
        "spork_fork": ([P, I, P, P, P], I),
        "spork_release": ([P, I, P, P], I),
        "spork_truncate": ([P, I, P, P, P], I),
        "spork_decode_attn": ([P, I, P, P, P, P, P, P], I),
        "spork_verify_attn": ([P, I, P, P, P, P, P, P, P], I),
        "spork_decode_attn_host": ([P, I, P, P, P, P, P, P], I),
        "spork_verify_attn_host": ([P, I, P, P, P, P, P, P, P], I),
        "spork_export": ([P, I32, P, P], I),
        "spork_export_refcounts": ([P, P], I),
        "spork_read_kv": ([P, I32, I32, I32, P, P], I),
        "spork_free_pages": ([P, P], I),
        "spork_status": ([P], I),
        "spork_last_plan": ([P, P], I),
        "spork_last_launches": ([P], I),
        "spork_accept": ([P, I, P, P, P, P, P, P], I),
        "spork_confidence": ([P, I, P, P, I, P, P], I),
        "spork_confidence_static": ([I, P, I, P, I, P, P], I),
        "spork_set_timing": ([P, I], I),
        "spork_set_tensor_path_min_rows": ([P, I], I),
        "spork_set_many_row_variant": ([P, I], I),
        "spork_set_stream_k": ([P, I], I),
        "spork_set_cascade_levels": ([P, I], I),
        "spork_layers": ([P, I, P, P, P], I),
        "spork_write_kv_layer": ([P, I, I, P, P, P, P, P], I),
        "spork_decode_attn_layers": ([P, I, I, P, P, P, P, P, P], I),
        "spork_verify_attn_layers": ([P, I, I, P, P, P, P, P, P, P], I),
        "spork_last_kernel_ms": ([P, P, P], I),
        "spork_hbm_read_probe": ([P, P, C.c_size_t, P], I),
        "spork_turn_prepare": ([P, I, P, P, P, P, P], I),
        "spork_turn_append": ([P, I, P, P, P], I),
        "spork_turn_verify": ([P, P, P, P, P], I),
        "spork_turn_accept": ([P, P, P, P, P], I),
        "spork_turn_decode": ([P, P, P, P, P], I),
        "spork_turn_sync": ([P, P], I),
        "spork_turn_destroy": ([P], I),
        "spork_strerror": ([I], C.c_char_p),
    }
    for name, (args, res) in sig.items():
        f = getattr(lib, name)
        f.argtypes = args
        f.restype = res
    _lib = lib
    return lib


class SporkError(RuntimeError):
    def __init__(self, code: int):
        msg = load().spork_strerror(code).decode()
        super().__init__(f"spork error {code}: {msg}")
        self.code = code


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32).reshape(-1))


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Spork:
    """One libspork handle plus the torch-allocated KV pools it works on."""

    def __init__(self, dtype: str, Hq: int, Hkv: int, D: int, num_pages: int, max_seqs: int,
                 max_pages_per_seq: int, scale: float, device: str = "cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libspork needs a CUDA device (there is no CPU fallback)")
        self.torch = torch
        self.lib = load()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.dtype, self.Hq, self.Hkv, self.D = dtype, Hq, Hkv, D
        self.num_pages, self.max_seqs, self.max_pages_per_seq = num_pages, max_seqs, max_pages_per_seq
        self.scale = float(scale)
        self.ps = PAGE_SIZE
        # host arrays are bit patterns: K / V in np_dtype, queries in q_np_dtype ("e4m3": fp8 cache, bf16 queries)
        self.np_dtype = {"f32": np.float32, "bf16": np.uint16, "e4m3": np.uint8}[dtype]
        self.q_np_dtype = np.float32 if dtype == "f32" else np.uint16
        self.torch_dtype = torch.float32 if dtype == "f32" else torch.bfloat16
        self.cfg = SporkConfig({"f32": F32, "bf16": BF16, "e4m3": E4M3}[dtype], Hq, Hkv, D, PAGE_SIZE, num_pages,
                               max_seqs, max_pages_per_seq, self.scale)
        self.page_bytes = int(self.lib.spork_page_bytes(C.byref(self.cfg)))
        # caller-owned pools: raw bytes (torch.empty: contents arbitrary on purpose)
        self.k_pool = torch.empty(num_pages * self.page_bytes, dtype=torch.uint8, device=self.device)
        self.v_pool = torch.empty(num_pages * self.page_bytes, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
        h = C.c_void_p()
        rc = self.lib.spork_create(C.byref(self.cfg), self.k_pool.data_ptr(), self.v_pool.data_ptr(),
                                   C.byref(h))
        if rc != OK:
            raise SporkError(rc)
        self._h = h

    # ---- lifetime -------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            self.lib.spork_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def _st(self):
        return C.c_void_p(self.stream.cuda_stream)

    def _enter(self):
        """our stream waits for work queued on torch's current stream (caller-made inputs)"""
        cur = self.torch.cuda.current_stream(self.device)
        if cur != self.stream:
            self.stream.wait_stream(cur)

    def _leave(self):
        """torch's current stream waits for ours, so results are safe to use there"""
        cur = self.torch.cuda.current_stream(self.device)
        if cur != self.stream:
            cur.wait_stream(self.stream)

    def _hold(self, *tensors):
        """caller tensors are read on OUR stream: tell the caching allocator, so that memory freed on the
        caller's stream is not reused before our kernels have read it"""
        for t in tensors:
            if t is not None and t.is_cuda:
                t.record_stream(self.stream)
        self._keep = tensors

    @staticmethod
    def _chk(rc: int, check: bool = True) -> int:
        if rc != OK and check:
            raise SporkError(rc)
        return rc

    def _dev(self, a: np.ndarray):
        """numpy storage array (float32 / bf16 bit patterns) -> device tensor on our stream."""
        t = self.torch.from_numpy(np.ascontiguousarray(a))
        with self.torch.cuda.stream(self.stream):
            return t.to(self.device, non_blocking=False)

    # ---- state calls ----------------------------------------------------------
    def seq_create(self, n: int) -> np.ndarray:
        ids = np.zeros(n, np.int32)
        self._chk(self.lib.spork_seq_create(self._h, n, _p(ids)))
        return ids

    def append(self, seq_ids, n_tokens, k, v, check: bool = True) -> int:
        """k, v: numpy storage arrays or device tensors, [sum n_tokens][Hkv][D]."""
        s, nt = _i32(seq_ids), _i32(n_tokens)
        kd = k if hasattr(k, "data_ptr") else self._dev(np.asarray(k, dtype=self.np_dtype))
        vd = v if hasattr(v, "data_ptr") else self._dev(np.asarray(v, dtype=self.np_dtype))
        total = int(nt[nt > 0].sum()) if len(nt) else 0
        assert kd.numel() * kd.element_size() == total * self.Hkv * self.D * np.dtype(self.np_dtype).itemsize
        self._enter()
        rc = self.lib.spork_append(self._h, len(s), _p(s), _p(nt), kd.data_ptr(), vd.data_ptr(), self._st)
        self._hold(kd, vd)
        return self._chk(rc, check)

    def fork(self, parents, check: bool = True):
        p = _i32(parents)
        ch = np.full(len(p), -1, np.int32)
        rc = self._chk(self.lib.spork_fork(self._h, len(p), _p(p), _p(ch), self._st), check)
        return ch if check else (rc, ch)

    def release(self, seq_ids, check: bool = True) -> int:
        s = _i32(seq_ids)
        return self._chk(self.lib.spork_release(self._h, len(s), _p(s), self._st), check)

    def truncate(self, seq_ids, new_len, check: bool = True) -> int:
        s, nl = _i32(seq_ids), _i32(new_len)
        return self._chk(self.lib.spork_truncate(self._h, len(s), _p(s), _p(nl), self._st), check)

    def accept(self, seq_ids, q_indptr, draft_tokens, target_tokens, check: bool = True):
        """Longest greedy-matching prefix per sequence + rollback of the rejected drafts.
        draft_tokens / target_tokens: device int32 tensors (or numpy arrays).  Returns (rc, accept_len)."""
        torch = self.torch
        s, qi = _i32(seq_ids), _i32(q_indptr)
        d = draft_tokens if hasattr(draft_tokens, "data_ptr") else self._dev(np.asarray(draft_tokens, dtype=np.int32))
        t = target_tokens if hasattr(target_tokens, "data_ptr") else self._dev(np.asarray(target_tokens, dtype=np.int32))
        assert d.dtype == torch.int32 and t.dtype == torch.int32
        acc = np.zeros(len(s), np.int32)
        self._enter()            # drafts / targets may have been produced on torch's current stream
        rc = self.lib.spork_accept(self._h, len(s), _p(s), _p(qi), C.c_void_p(d.data_ptr()),
                                   C.c_void_p(t.data_ptr()), _p(acc), self._st)
        self._hold(d, t)
        return self._chk(rc, check), acc

    def confidence(self, span_indptr, logits, out=None, check: bool = True):
        """Eq. 2 confidence per span.  logits: device fp32 tensor [n_pos][vocab] (or numpy).  Returns a
        device fp32 tensor [n_spans]."""
        torch = self.torch
        sp = _i32(span_indptr)
        x = logits if hasattr(logits, "data_ptr") else self._dev(np.asarray(logits, dtype=np.float32))
        assert x.dtype == torch.float32 and x.is_contiguous()
        n = len(sp) - 1
        if out is None:
            out = torch.empty((n,), dtype=torch.float32, device=self.device)
        self._enter()            # the logits may still be in flight on torch's current stream
        rc = self.lib.spork_confidence(self._h, n, _p(sp), C.c_void_p(x.data_ptr()), int(x.shape[1]),
                                       C.c_void_p(out.data_ptr()), self._st)
        self._leave()            # ... and the scores are read there
        self._hold(x, out)
        self._chk(rc, check)
        return out if check else (rc, out)

    def confidence_static(self, span_indptr, logits, out, check: bool = True):
        """spork_confidence_static: Eq. 2 confidence with no allocation anywhere (see spork.h).  All three
        arguments are device tensors the caller owns: span_indptr int32 [n_spans + 1], logits fp32
        [n_pos][vocab] (at most CONFIDENCE_STATIC_MAX_ROWS rows), out fp32 [n_spans].  Runs on this
        context's stream; returns the error code."""
        torch = self.torch
        assert span_indptr.dtype == torch.int32 and span_indptr.is_cuda and span_indptr.is_contiguous()
        assert logits.dtype == torch.float32 and logits.is_cuda and logits.is_contiguous() and logits.dim() == 2
        n = int(span_indptr.numel()) - 1
        assert out.dtype == torch.float32 and out.is_cuda and out.is_contiguous() and out.numel() == n
        self._enter()
        with torch.cuda.device(self.device):       # the call resolves its scratch on the CURRENT device
            rc = self.lib.spork_confidence_static(n, C.c_void_p(span_indptr.data_ptr()), int(logits.shape[0]),
                                                  C.c_void_p(logits.data_ptr()), int(logits.shape[1]),
                                                  C.c_void_p(out.data_ptr()), self._st)
        self._leave()
        self._hold(span_indptr, logits, out)
        return self._chk(rc, check)

    def turn(self, group_indptr, seq_ids, q_indptr) -> "Turn":
        """Prepares a capturable partial-token-accept turn over this batch (see spork.h, spork_turn_*)."""
        return Turn(self, group_indptr, seq_ids, q_indptr)

    # ---- attention ------------------------------------------------------------
    def decode_attn(self, group_indptr, seq_ids, q, out=None, lse=None, check: bool = True):
        """q: device tensor [n_seq][Hq][D] in the storage dtype (or numpy storage array).
        Returns device fp32 tensors (out [n_seq][Hq][D], lse [n_seq][Hq])."""
        torch = self.torch
        gi, s = _i32(group_indptr), _i32(seq_ids)
        qd = q if hasattr(q, "data_ptr") else self._dev(np.asarray(q, dtype=self.q_np_dtype))
        n = len(s)
        if out is None:
            out = torch.empty((n, self.Hq, self.D), dtype=torch.float32, device=self.device)
        if lse is None:
            lse = torch.empty((n, self.Hq), dtype=torch.float32, device=self.device)
        self._enter()
        rc = self.lib.spork_decode_attn(self._h, len(gi) - 1, _p(gi), _p(s), qd.data_ptr(),
                                        out.data_ptr(), lse.data_ptr(), self._st)
        self._leave()
        self._hold(qd, out, lse)
        self._chk(rc, check)
        return (out, lse) if check else (rc, out, lse)

    def verify_attn(self, group_indptr, seq_ids, q_indptr, q, out=None, lse=None, check: bool = True):
        torch = self.torch
        gi, s, qi = _i32(group_indptr), _i32(seq_ids), _i32(q_indptr)
        qd = q if hasattr(q, "data_ptr") else self._dev(np.asarray(q, dtype=self.q_np_dtype))
        rows = int(qi[-1]) if len(qi) else 0
        if out is None:
            out = torch.empty((rows, self.Hq, self.D), dtype=torch.float32, device=self.device)
        if lse is None:
            lse = torch.empty((rows, self.Hq), dtype=torch.float32, device=self.device)
        self._enter()
        rc = self.lib.spork_verify_attn(self._h, len(gi) - 1, _p(gi), _p(s), _p(qi), qd.data_ptr(),
                                        out.data_ptr(), lse.data_ptr(), self._st)
        self._leave()
        self._hold(qd, out, lse)
        self._chk(rc, check)
        return (out, lse) if check else (rc, out, lse)

    # ---- multi-layer step -------------------------------------
    def layers(self, n_layers: int):
        """Allocates and registers the K/V pools of layers 1 .. n_layers-1 (layer 0 = the pools made at
        construction); block tables, refcounts and lengths are shared by all layers."""
        torch = self.torch
        self.k_pools = [self.k_pool] + [torch.empty_like(self.k_pool) for _ in range(n_layers - 1)]
        self.v_pools = [self.v_pool] + [torch.empty_like(self.v_pool) for _ in range(n_layers - 1)]
        kp = (C.c_void_p * n_layers)(*[t.data_ptr() for t in self.k_pools])
        vp = (C.c_void_p * n_layers)(*[t.data_ptr() for t in self.v_pools])
        self._chk(self.lib.spork_layers(self._h, n_layers, kp, vp, self._st))
        self.n_layers = n_layers

    def write_kv_layer(self, layer: int, seq_ids, n_tokens, k, v, check: bool = True) -> int:
        """K/V of the last n_tokens[i] tokens of each sequence into layer `layer`'s pools."""
        s, nt = _i32(seq_ids), _i32(n_tokens)
        kd = k if hasattr(k, "data_ptr") else self._dev(np.asarray(k, dtype=self.np_dtype))
        vd = v if hasattr(v, "data_ptr") else self._dev(np.asarray(v, dtype=self.np_dtype))
        self._enter()
        rc = self.lib.spork_write_kv_layer(self._h, int(layer), len(s), _p(s), _p(nt), kd.data_ptr(),
                                           vd.data_ptr(), self._st)
        self._hold(kd, vd)
        return self._chk(rc, check)

    def attn_layers(self, group_indptr, seq_ids, q_layers, out_layers, lse_layers, q_indptr=None):
        """One plan, len(q_layers) x (attention, merge) launches back to back.  q_layers / out_layers /
        lse_layers: lists of device tensors, one per layer."""
        gi, s = _i32(group_indptr), _i32(seq_ids)
        L = len(q_layers)
        qp = (C.c_void_p * L)(*[t.data_ptr() for t in q_layers])
        op = (C.c_void_p * L)(*[t.data_ptr() for t in out_layers])
        lp = (C.c_void_p * L)(*[t.data_ptr() for t in lse_layers])
        self._enter()
        if q_indptr is None:
            rc = self.lib.spork_decode_attn_layers(self._h, L, len(gi) - 1, _p(gi), _p(s), qp, op, lp, self._st)
        else:
            qi = _i32(q_indptr)
            rc = self.lib.spork_verify_attn_layers(self._h, L, len(gi) - 1, _p(gi), _p(s), _p(qi), qp, op, lp,
                                                   self._st)
        self._leave()
        self._hold(*q_layers, *out_layers, *lse_layers)
        self._chk(rc)

    def decode_attn_host(self, group_indptr, seq_ids, q_host, out_host, lse_host):
        """HOST (pinned) tensors in, HOST tensors out; copies run inside the call."""
        gi, s = _i32(group_indptr), _i32(seq_ids)
        self._chk(self.lib.spork_decode_attn_host(self._h, len(gi) - 1, _p(gi), _p(s), q_host.data_ptr(),
                                                  out_host.data_ptr(), lse_host.data_ptr(), self._st))

    def verify_attn_host(self, group_indptr, seq_ids, q_indptr, q_host, out_host, lse_host):
        gi, s, qi = _i32(group_indptr), _i32(seq_ids), _i32(q_indptr)
        self._chk(self.lib.spork_verify_attn_host(self._h, len(gi) - 1, _p(gi), _p(s), _p(qi),
                                                  q_host.data_ptr(), out_host.data_ptr(),
                                                  lse_host.data_ptr(), self._st))

    # ---- export ---------------------------------------------------------------
    def export(self, seq: int):
        """(len, table[ceil(len/16)]) read from the device; len = -1 if the slot is not live."""
        ln = np.zeros(1, np.int32)
        tab = np.full(self.max_pages_per_seq, -1, np.int32)
        self._chk(self.lib.spork_export(self._h, int(seq), _p(ln), _p(tab)))
        L = int(ln[0])
        return L, tab[:max(0, (L + self.ps - 1) // self.ps)].copy()

    export_seq = export   # same name as the oracle's engine interface

    def export_refcounts(self) -> np.ndarray:
        out = np.zeros(self.num_pages, np.int32)
        self._chk(self.lib.spork_export_refcounts(self._h, _p(out)))
        return out

    def read_kv(self, seq: int, t0: int, n: int):
        k = np.zeros((n, self.Hkv, self.D), self.np_dtype)
        v = np.zeros_like(k)
        self._chk(self.lib.spork_read_kv(self._h, int(seq), int(t0), int(n), _p(k), _p(v)))
        return k, v

    def free_pages(self) -> int:
        out = np.zeros(1, np.int32)
        self._chk(self.lib.spork_free_pages(self._h, _p(out)))
        return int(out[0])

    def status(self) -> int:
        return int(self.lib.spork_status(self._h))

    def last_plan(self) -> dict:
        info = PlanInfo()
        self._chk(self.lib.spork_last_plan(self._h, C.byref(info)))
        return info.as_dict()

    def last_launches(self) -> int:
        return int(self.lib.spork_last_launches(self._h))

    def set_timing(self, enable: bool):
        self._chk(self.lib.spork_set_timing(self._h, int(bool(enable))))

    def set_tensor_path_min_rows(self, min_rows: int):
        """Planner knob: segments with >= min_rows rows per KV head run on the tcgen05 kernel."""
        self._chk(self.lib.spork_set_tensor_path_min_rows(self._h, int(min_rows)))

    def set_many_row_variant(self, mode: int):
        """Planner knob: which tcgen05 kernel runs segments of more than 128 rows.  0 (default): the
        one-pipe kernel in row blocks of 128; 1: the two-pipe kernel (row blocks of 256 over one K/V
        stream); 2: the split-row kernel."""
        self._chk(self.lib.spork_set_many_row_variant(self._h, int(mode)))

    def set_cascade_levels(self, max_levels: int):
        """Planner knob: deepest cascade built for a fork group (1: the group-wide prefix only)."""
        self._chk(self.lib.spork_set_cascade_levels(self._h, int(max_levels)))

    def set_stream_k(self, enable: bool):
        """Planner knob: equal-work contiguous schedule for single-row-block calls (default on)."""
        self._chk(self.lib.spork_set_stream_k(self._h, int(bool(enable))))

    def hbm_read_probe(self, buf):
        """Bench support: one read-only pass over the device tensor `buf` on our stream."""
        self._chk(self.lib.spork_hbm_read_probe(self._h, C.c_void_p(buf.data_ptr()),
                                                C.c_size_t(buf.numel() * buf.element_size()), self._st))

    def last_kernel_ms(self):
        """(attention kernel ms, merge kernel ms) of the last attention call (synchronises)."""
        a, m = C.c_float(), C.c_float()
        self._chk(self.lib.spork_last_kernel_ms(self._h, C.byref(a), C.byref(m)))
        return float(a.value), float(m.value)

    def synchronize(self):
        self.stream.synchronize()


class Turn:
    """A prepared turn: append drafts -> verify -> accept + rollback -> append one token -> decode, each
    call nothing but kernel launches on the handle's stream over the DEVICE tensors it is given, so the
    caller can capture them (torch.cuda.graph(..., stream=spk.stream)) and replay.  Argument marshalling
    only; tensors must stay alive (and in place) for as long as a captured graph is replayed."""

    def __init__(self, spk: Spork, group_indptr, seq_ids, q_indptr):
        self.spk = spk
        gi, s, qi = _i32(group_indptr), _i32(seq_ids), _i32(q_indptr)
        self.n, self.rows = len(s), int(qi[-1])
        h = C.c_void_p()
        spk._chk(spk.lib.spork_turn_prepare(spk._h, len(gi) - 1, _p(gi), _p(s), _p(qi), spk._st, C.byref(h)))
        self._t = h

    def append(self, which: int, k, v):
        """which = 0: the k_i drafts of every sequence ([sum k][Hkv][D]); 1: one token each ([n][Hkv][D])."""
        self.spk._enter()        # (no-ops under torch.cuda.graph(stream=spk.stream): that IS the current stream)
        rc = self.spk.lib.spork_turn_append(self._t, int(which), C.c_void_p(k.data_ptr()), C.c_void_p(v.data_ptr()),
                                            self.spk._st)
        self.spk._leave()
        self.spk._chk(rc)

    def verify(self, q, out, lse):
        self.spk._enter()
        rc = self.spk.lib.spork_turn_verify(self._t, C.c_void_p(q.data_ptr()), C.c_void_p(out.data_ptr()),
                                            C.c_void_p(lse.data_ptr()), self.spk._st)
        self.spk._leave()
        self.spk._chk(rc)

    def accept(self, draft_tokens, target_tokens, accept_len=None):
        a = C.c_void_p(accept_len.data_ptr()) if accept_len is not None else None
        self.spk._enter()
        rc = self.spk.lib.spork_turn_accept(self._t, C.c_void_p(draft_tokens.data_ptr()),
                                            C.c_void_p(target_tokens.data_ptr()), a, self.spk._st)
        self.spk._leave()
        self.spk._chk(rc)

    def decode(self, q, out, lse):
        self.spk._enter()
        rc = self.spk.lib.spork_turn_decode(self._t, C.c_void_p(q.data_ptr()), C.c_void_p(out.data_ptr()),
                                            C.c_void_p(lse.data_ptr()), self.spk._st)
        self.spk._leave()
        self.spk._chk(rc)

    def sync(self, check: bool = True) -> int:
        """Host mirror of the lengths <- device (synchronises); the other Spork calls work again."""
        return self.spk._chk(self.spk.lib.spork_turn_sync(self._t, self.spk._st), check)

    def close(self):
        if getattr(self, "_t", None):
            self.spk.lib.spork_turn_destroy(self._t)
            self._t = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
