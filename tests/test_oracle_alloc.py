"""Pins for the oracle's allocator / fork / release / truncate (CPU only).

The integer state is pinned by (1) invariants checked after every call,
(2) an independently written ~40-line Python model of readings A-1..A-5
 compared on EVERY script of bounded length over a tiny pool
(exhaustive, not sampled) and on long random scripts, and (3) the north_star
invariants: refcounts return to zero after release, fork with a partial tail
allocates exactly one page, an aligned fork allocates none.
"""
import itertools

import numpy as np
import pytest

import oracle

PS = 4          # small page so that short scripts cross page boundaries


class Model:
    """Independent restatement of the allocator readings (not a port of the C code)."""

    def __init__(self, num_pages, max_seqs, mpps, ps):
        self.rc = [0] * num_pages
        self.seqs = {}                   # id -> list of page ids ; lens separately
        self.lens = {}
        self.num_pages, self.max_seqs, self.mpps, self.ps = num_pages, max_seqs, mpps, ps

    def _free_pages(self):
        return [p for p, c in enumerate(self.rc) if c == 0]

    def _free_slots(self):
        return [s for s in range(self.max_seqs) if s not in self.seqs]

    def _take(self):
        p = self._free_pages()[0]
        self.rc[p] = 1
        return p

    def create(self):
        fs = self._free_slots()
        if not fs:
            return oracle.ERR_NO_SLOT, None
        self.seqs[fs[0]], self.lens[fs[0]] = [], 0
        return 0, fs[0]

    def append(self, s, n):
        if s not in self.seqs:
            return oracle.ERR_INVALID_SEQ
        new_pages = -(-(self.lens[s] + n) // self.ps) - len(self.seqs[s])
        if len(self.seqs[s]) + new_pages > self.mpps:
            return oracle.ERR_TOO_LONG
        if new_pages > len(self._free_pages()):
            return oracle.ERR_OOM
        for _ in range(new_pages):
            self.seqs[s].append(self._take())
        self.lens[s] += n
        return 0

    def fork(self, parents):
        if any(p not in self.seqs for p in parents):
            return oracle.ERR_INVALID_SEQ, None
        if len(self._free_slots()) < len(parents):
            return oracle.ERR_NO_SLOT, None
        if sum(1 for p in parents if self.lens[p] % self.ps) > len(self._free_pages()):
            return oracle.ERR_OOM, None
        kids = []
        for p in parents:
            c = self._free_slots()[0]
            full = self.lens[p] // self.ps
            shared = list(self.seqs[p][:full])
            for pg in shared:
                self.rc[pg] += 1
            if self.lens[p] % self.ps:
                shared.append(self._take())
            self.seqs[c], self.lens[c] = shared, self.lens[p]
            kids.append(c)
        return 0, kids

    def release(self, ids):
        if any(s not in self.seqs for s in ids) or len(set(ids)) != len(ids):
            return oracle.ERR_INVALID_SEQ
        for s in ids:
            for pg in self.seqs.pop(s):
                self.rc[pg] -= 1
            self.lens.pop(s)
        return 0

    def truncate(self, s, n):
        if s not in self.seqs:
            return oracle.ERR_INVALID_SEQ
        if n < 0 or n > self.lens[s]:
            return oracle.ERR_INVALID
        if n % self.ps and self.rc[self.seqs[s][n // self.ps]] > 1:
            return oracle.ERR_SHARED
        keep = -(-n // self.ps)
        for pg in self.seqs[s][keep:]:
            self.rc[pg] -= 1
        self.seqs[s] = self.seqs[s][:keep]
        self.lens[s] = n
        return 0


def mk(num_pages=8, max_seqs=3, mpps=4):
    return oracle.Oracle("f32", 1, 1, 2, num_pages, max_seqs, mpps, 1.0, page_size=PS, store_kv=True)


def check_same(o, m):
    np.testing.assert_array_equal(o.export_refcounts(), np.array(m.rc, np.int32))
    for s in range(m.max_seqs):
        L, tab = o.export_seq(s)
        if s in m.seqs:
            assert L == m.lens[s] and list(tab) == m.seqs[s], (s, L, tab, m.lens[s], m.seqs[s])
        else:
            assert L == -1
    # invariants (SURVEY.md 8(c) pins): sum refcount == sum ceil(len/ps); free + used == NP
    rc = o.export_refcounts()
    assert rc.sum() == sum(-(-l // PS) for l in m.lens.values())
    assert (rc == 0).sum() + (rc > 0).sum() == o.num_pages and (rc >= 0).all()


def apply(o, m, op, check=True):
    kind = op[0]
    z = np.zeros
    if kind == "c":
        rc_m, sid = m.create()
        try:
            ids = o.seq_create(1)
            rc_o = 0
            assert ids[0] == sid
        except oracle.OracleError as e:
            rc_o = e.code
    elif kind == "a":
        _, s, n = op
        rc_m = m.append(s, n)
        rc_o = o.append([s], [n], z((n, 1, 2), np.float32), z((n, 1, 2), np.float32), check=False)
    elif kind == "f":
        parents = list(op[1:])
        rc_m, kids = m.fork(parents)
        rc_o, ch = o.fork(parents, check=False)
        if rc_m == 0:
            assert list(ch) == kids
    elif kind == "r":
        ids = list(op[1:])
        rc_m = m.release(ids)
        rc_o = o.release(ids, check=False)
    elif kind == "t":
        _, s, n = op
        rc_m = m.truncate(s, n)
        rc_o = o.truncate([s], [n], check=False)
    assert rc_o == rc_m, (op, rc_o, rc_m)
    if check:
        check_same(o, m)


OPS = ([("c",)] + [("a", s, n) for s in range(2) for n in (1, 4, 6)] + [("a", 2, 3)]
       + [("f", p) for p in range(3)] + [("f", 0, 0)] + [("f", 0, 1)]
       + [("r", s) for s in range(3)] + [("r", 0, 1)]
       + [("t", s, n) for s in range(2) for n in (0, 2)])


def test_exhaustive_short_scripts_against_independent_model():
    """every script of length 3 over 3 slots / 8 pages, from the empty state and after each
    of a set of seeding prefixes (all |OPS|^3 continuations of each; exhaustive, not sampled)"""
    prefixes = [
        [],
        [("c",), ("a", 0, 6)],                      # one sequence with a partial tail
        [("c",), ("a", 0, 8), ("f", 0)],            # aligned fork
        [("c",), ("a", 0, 5), ("f", 0, 0)],         # partial-tail fork x2 (slots full)
        [("c",), ("c",), ("a", 1, 3), ("a", 0, 9), ("r", 1)],   # hole at page 0
    ]
    n = 0
    for pre in prefixes:
        depth = 3
        for script in itertools.product(OPS, repeat=depth):
            o, m = mk(), Model(8, 3, 4, PS)
            for op in pre:
                apply(o, m, op)
            for i, op in enumerate(script):       # return codes every step, full state at the end
                apply(o, m, op, check=(i == depth - 1))
            o.close()
            n += 1
    assert n == len(prefixes) * len(OPS) ** 3


def test_long_random_scripts_against_model():
    r = np.random.default_rng(0)
    for trial in range(30):
        o, m = oracle.Oracle("f32", 1, 1, 2, 40, 8, 6, 1.0, page_size=PS), Model(40, 8, 6, PS)
        for _ in range(300):
            kind = r.choice(["c", "a", "a", "f", "f", "r", "t"])
            s = int(r.integers(0, 8))
            if kind == "c":
                op = ("c",)
            elif kind == "a":
                op = ("a", s, int(r.integers(0, 9)))
            elif kind == "f":
                op = ("f",) + tuple(int(x) for x in r.integers(0, 8, size=int(r.integers(1, 4))))
            elif kind == "r":
                op = ("r",) + tuple(set(int(x) for x in r.integers(0, 8, size=int(r.integers(1, 3)))))
            else:
                op = ("t", s, int(r.integers(0, 20)))
            apply(o, m, op)
        live = [s for s in m.seqs]
        if live:
            apply(o, m, ("r",) + tuple(live))
        assert (o.export_refcounts() == 0).all()          # refcounts return to zero
        o.close()


def test_fork_page_accounting_and_tail_copy():
    r = np.random.default_rng(1)
    o = oracle.Oracle("bf16", 2, 2, 4, 32, 8, 8, 0.5, page_size=16)
    (main,) = o.seq_create(1)
    k = r.integers(0, 2 ** 15, size=(37, 2, 4)).astype(np.uint16)
    v = r.integers(0, 2 ** 15, size=(37, 2, 4)).astype(np.uint16)
    o.append([main], [32], k[:32], v[:32])
    used = (o.export_refcounts() > 0).sum()
    (c0,) = o.fork([main])                         # aligned: zero pages allocated (A-4)
    assert (o.export_refcounts() > 0).sum() == used
    assert list(o.export_seq(c0)[1]) == list(o.export_seq(main)[1])
    np.testing.assert_array_equal(o.export_refcounts()[:2], [2, 2])
    o.append([main], [5], k[32:], v[32:])          # main now has a partial tail (5 of 16)
    used = (o.export_refcounts() > 0).sum()
    c1, c2 = o.fork([main, main])                  # unaligned: exactly one page each
    assert (o.export_refcounts() > 0).sum() == used + 2
    Lm, tm = o.export_seq(main)
    for c in (c1, c2):
        L, t = o.export_seq(c)
        assert L == Lm == 37 and list(t[:2]) == list(tm[:2]) and t[2] != tm[2]
        ck, cv = o.read_kv(c, 0, 37)               # tail valid slots bit-equal (A-3)
        np.testing.assert_array_equal(ck, k)
        np.testing.assert_array_equal(cv, v)
        assert o.export_refcounts()[t[2]] == 1
    assert c1 != c2 and o.export_seq(c1)[1][2] != o.export_seq(c2)[1][2]
    # child's first append after an aligned fork allocates its own page
    o.append([c0], [1], k[:1], v[:1])
    assert o.export_seq(c0)[1][2] not in (tm[2], o.export_seq(c1)[1][2], o.export_seq(c2)[1][2])
    # fork of a fork, parent released before children (A-5)
    (gc,) = o.fork([c1])
    o.release([main, c1])
    gk, gv = o.read_kv(gc, 0, 37)
    np.testing.assert_array_equal(gk, k)
    o.release([c0, c2, gc])
    assert (o.export_refcounts() == 0).all()
    # double release rejected without state change
    assert o.release([gc], check=False) == oracle.ERR_INVALID_SEQ


def test_all_or_nothing_on_oom_and_no_slot():
    o = oracle.Oracle("f32", 1, 1, 2, 3, 4, 4, 1.0, page_size=4)
    z = lambda n: np.zeros((n, 1, 2), np.float32)
    (a,) = o.seq_create(1)
    o.append([a], [6], z(6), z(6))                 # 2 of 3 pages used, partial tail
    before = o.export_refcounts().copy()
    rc, _ = o.fork([a, a], check=False)            # needs 2 tail pages, 1 free
    assert rc == oracle.ERR_OOM
    np.testing.assert_array_equal(o.export_refcounts(), before)
    assert o.export_seq(1)[0] == -1                # no child slot was taken
    assert o.append([a], [9], z(9), z(9), check=False) == oracle.ERR_OOM
    assert o.export_seq(a)[0] == 6
    o.seq_create(3)
    rc, _ = o.fork([a], check=False)
    assert rc == oracle.ERR_NO_SLOT
    assert o.append([a], [20], z(20), z(20), check=False) == oracle.ERR_TOO_LONG


def test_lowest_free_id_first_after_holes():
    o = oracle.Oracle("f32", 1, 1, 2, 8, 4, 8, 1.0, page_size=4)
    z = lambda n: np.zeros((n, 1, 2), np.float32)
    a, b, c = o.seq_create(3)
    o.append([a, b, c], [4, 4, 4], z(12), z(12))   # pages 0,1,2 in request order
    assert [o.export_seq(s)[1][0] for s in (a, b, c)] == [0, 1, 2]
    o.release([b])
    o.append([c], [8], z(8), z(8))                 # takes the hole (1) first, then 3
    assert list(o.export_seq(c)[1]) == [2, 1, 3]
    (d,) = o.seq_create(1)
    assert d == b                                  # lowest free slot first
