"""GPU parity of the integer state (block tables, lengths, refcounts, error codes):
random scripts of seq_create / append / fork / truncate / release replayed on the
oracle and on libspork.  Bit-exact under the lowest-free-id policy (reading A-1)."""
import numpy as np
import pytest

import oracle
import synth
from _harness import assert_state_equal

pytestmark = pytest.mark.gpu


def _mk(dtype, Hq, Hkv, D, npg, ms, mp):
    import paper_2607_03333_b200 as sp
    o = oracle.Oracle(dtype, Hq, Hkv, D, npg, ms, mp, 0.125)
    s = sp.Spork(dtype, Hq, Hkv, D, npg, ms, mp, 0.125)
    return o, s


def _kv(r, n, Hkv, D, dtype):
    k = synth.to_storage(r.standard_normal((n, Hkv, D), dtype=np.float32), dtype)
    v = synth.to_storage(r.standard_normal((n, Hkv, D), dtype=np.float32), dtype)
    return k, v


@pytest.mark.parametrize("seed,dtype,npg", [(0, "f32", 40), (1, "bf16", 24), (2, "bf16", 200), (3, "f32", 12)])
def test_random_scripts(seed, dtype, npg):
    Hq, Hkv, D = 4, 2, 64
    ms, mp = 12, 9
    o, s = _mk(dtype, Hq, Hkv, D, npg, ms, mp)
    r = np.random.default_rng([7, seed])
    live = []
    codes = {}
    for step in range(160):
        op = r.choice(["create", "append", "fork", "truncate", "release", "bad"],
                      p=[0.1, 0.38, 0.2, 0.12, 0.15, 0.05])
        if op == "create":
            n = int(r.integers(1, 3))
            try:
                a = o.seq_create(n)
                ok = True
            except oracle.OracleError as e:
                ok, code = False, e.code
            if ok:
                b = s.seq_create(n)
                assert np.array_equal(a, b)
                live += list(a)
            else:
                import paper_2607_03333_b200 as sp
                with pytest.raises(sp.SporkError) as ei:
                    s.seq_create(n)
                assert ei.value.code == code
        elif op == "append" and live:
            n = int(r.integers(1, 4))
            ids = r.choice(live, size=n)          # repeats allowed
            nt = r.integers(0, 40, size=n)
            k, v = _kv(r, int(nt.sum()), Hkv, D, dtype)
            rc_o = o.append(ids, nt, k, v, check=False)
            rc_s = s.append(ids, nt, k, v, check=False)
            assert rc_o == rc_s, (step, "append", rc_o, rc_s)
            codes[rc_o] = codes.get(rc_o, 0) + 1
        elif op == "fork" and live:
            n = int(r.integers(1, 4))
            par = r.choice(live, size=n)
            rc_o, ch_o = o.fork(par, check=False)
            rc_s, ch_s = s.fork(par, check=False)
            assert rc_o == rc_s, (step, "fork", rc_o, rc_s)
            codes[rc_o] = codes.get(rc_o, 0) + 1
            if rc_o == 0:
                assert np.array_equal(ch_o, ch_s)
                live += list(ch_o)
        elif op == "truncate" and live:
            sid = int(r.choice(live))
            L, _ = o.export_seq(sid)
            nl = int(r.integers(0, L + 1))
            rc_o = o.truncate([sid], [nl], check=False)
            rc_s = s.truncate([sid], [nl], check=False)
            assert rc_o == rc_s, (step, "truncate", rc_o, rc_s)
            codes[rc_o] = codes.get(rc_o, 0) + 1
        elif op == "release" and live:
            n = min(len(live), int(r.integers(1, 3)))
            ids = list(r.choice(live, size=n, replace=False))
            assert o.release(ids, check=False) == s.release(ids, check=False) == 0
            for i in ids:
                live.remove(i)
        elif op == "bad":
            # invalid ids, double release within a batch, truncate beyond len
            assert o.release([ms + 3], check=False) == s.release([ms + 3], check=False) != 0
            if live:
                x = int(live[0])
                assert o.release([x, x], check=False) == s.release([x, x], check=False) != 0
                assert o.truncate([x], [10 ** 6], check=False) == s.truncate([x], [10 ** 6], check=False) != 0
                dead = [i for i in range(ms) if i not in live]
                if dead:
                    assert o.fork([dead[0]], check=False)[0] == s.fork([dead[0]], check=False)[0] != 0
        if step % 8 == 7 or step == 159:
            assert_state_equal(o, s, live)
            # invariants: sum refcount == sum ceil(len/ps); free + used == NP
            rc = s.export_refcounts()
            tot = sum((s.export(int(i))[0] + 15) // 16 for i in live)
            assert int(rc.sum()) == tot
            assert s.free_pages() == int((rc == 0).sum())
    # stored K/V agree for every live sequence
    for i in live:
        L, _ = o.export_seq(int(i))
        if L:
            ko, vo = o.read_kv(int(i), 0, L)
            ks, vs = s.read_kv(int(i), 0, L)
            assert np.array_equal(ko, ks) and np.array_equal(vo, vs)
    o.release(live)
    s.release(live)
    assert not s.export_refcounts().any() and s.free_pages() == npg and s.status() == 0
    assert len(codes) >= 2, f"script never hit an error path: {codes}"


def test_truncate_shared_tail_is_rejected():
    import paper_2607_03333_b200 as sp
    o, s = _mk("bf16", 4, 2, 64, 32, 6, 8)
    r = np.random.default_rng(5)
    a_o, a_s = o.seq_create(1), s.seq_create(1)
    k, v = _kv(r, 70, 2, 64, "bf16")
    o.append(a_o, [70], k, v)
    s.append(a_s, [70], k, v)
    c_o, c_s = o.fork(a_o), s.fork(a_s)
    # 70 tokens = 4 full pages shared + a private tail copy each
    for nl, want in [(40, oracle.ERR_SHARED), (64, 0)]:
        rc_o = o.truncate(c_o, [nl], check=False)
        rc_s = s.truncate(c_s, [nl], check=False)
        assert rc_o == rc_s == want
    assert sp.ERR_SHARED == oracle.ERR_SHARED
    assert_state_equal(o, s, [int(a_o[0]), int(c_o[0])])
    # after the parent is released the pages are exclusively the child's: truncate is legal
    o.release(a_o)
    s.release(a_s)
    assert o.truncate(c_o, [40], check=False) == s.truncate(c_s, [40], check=False) == 0
    assert_state_equal(o, s, [int(c_o[0])])


def test_oom_and_no_slot_change_nothing():
    o, s = _mk("f32", 4, 2, 64, 6, 3, 8)
    r = np.random.default_rng(9)
    a = o.seq_create(1)
    s.seq_create(1)
    k, v = _kv(r, 70, 2, 64, "f32")          # 5 pages of 6
    o.append(a, [70], k, v)
    s.append(a, [70], k, v)
    k2, v2 = _kv(r, 40, 2, 64, "f32")        # needs 2 more pages... only 1 free
    assert o.append(a, [40], k2, v2, check=False) == s.append(a, [40], k2, v2, check=False) == oracle.ERR_OOM
    rc_o, _ = o.fork([a[0], a[0]], check=False)     # two tail copies, one page free
    rc_s, _ = s.fork([a[0], a[0]], check=False)
    assert rc_o == rc_s == oracle.ERR_OOM
    assert_state_equal(o, s, a)
    ch_o, ch_s = o.fork(a), s.fork(a)
    assert np.array_equal(ch_o, ch_s)
    ch_o, ch_s = o.fork(a[:0]), s.fork(a[:0])       # empty batch
    rc_o, _ = o.fork([a[0], a[0]], check=False)     # only one slot left
    rc_s, _ = s.fork([a[0], a[0]], check=False)
    assert rc_o == rc_s == oracle.ERR_NO_SLOT
    assert_state_equal(o, s, [0, 1])
    assert s.free_pages() == 0
