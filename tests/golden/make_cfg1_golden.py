"""Writes tests/golden/cfg1_oracle.txt: the oracle's out/lse for config 1.

Calls only oracle/ and synth/ (never the CUDA path).  Run from the repo root:
    python tests/golden/make_cfg1_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import synth   # noqa: E402


def compute():
    c = synth.CFG1
    wl = synth.Workload(c)
    o = oracle.Oracle(c.dtype, c.Hq, c.Hkv, c.D, 64, 8, 32, c.scale)
    ids = synth.build_state(o, wl)
    out, lse = o.decode(ids, wl.q_all())
    tabs = [o.export_seq(int(s)) for s in ids]
    return wl, ids, out, lse, tabs, o.export_refcounts()


def main():
    wl, ids, out, lse, tabs, rc = compute()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg1_oracle.txt")
    with open(path, "w") as f:
        f.write("# config 1 (BASELINE.json configs[0]); oracle fp64; written by make_cfg1_golden.py\n")
        f.write("suffix_len " + " ".join(str(int(x)) for x in wl.suffix_len) + "\n")
        for s, (L, t) in zip(ids, tabs):
            f.write(f"seq {int(s)} len {L} table " + " ".join(str(int(x)) for x in t) + "\n")
        f.write("refcount_nonzero " + " ".join(f"{i}:{int(v)}" for i, v in enumerate(rc) if v) + "\n")
        for i in range(out.shape[0]):
            for h in range(out.shape[1]):
                f.write(f"lse {i} {h} {lse[i, h]:.17g}\n")
                f.write(f"out {i} {h} " + " ".join(f"{x:.17g}" for x in out[i, h, :8]) + "\n")
    print("wrote", path)


if __name__ == "__main__":
    main()
