"""Writes tests/golden/oracle_full_<config>.txt: the oracle's WHOLE profile I(q_k), every k, for the full-size
BASELINE.json configs 3, 4 and 5 (Eq. 2), where the oracle is far too slow to run inside the
test suite (cfg5: 2.56e12 sinc terms in fp64).

Calls ONLY oracle/ and the seeded input generators; nothing here touches the CUDA path.  The paper prints no
I(q) values (its profiles are figures), so these are oracle outputs, not paper numbers; the oracle itself is
pinned by tests/test_oracle_pins.py.  Cost on 16 host cores: cfg3 ~2.5 min, cfg4 (65 conformers) ~10 s,
cfg5 ~25 min.

    python tests/golden/make_golden_full.py [--out DIR] cfg3 cfg4 cfg5
"""
import argparse
import hashlib
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle as orc                                   # noqa: E402
from paper_1306_2258_b200 import workloads as wl                   # noqa: E402

# cfg4: every 16th conformer and the last one (65 of 1024), all 64 q each
CFG4_CONFORMERS = list(range(0, 1024, 16)) + [1023]
HEAD = ["# oracle (fp64, Eq. 2 of arxiv 1306.2258, PAPER.md:41-42), EVERY q index; written by tests/golden/make_golden_full.py",
        "# columns: config  conformer  k  q_k(float32 repr)  I(q_k)  sum|terms|   ; the '# input' line = sha256[:16] of the input bytes"]


def digest(w):
    h = hashlib.sha256()
    for a in (w.xyz, w.type, w.fftab, w.q):
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()[:16]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.dirname(os.path.abspath(__file__)))
    ap.add_argument("configs", nargs="+", choices=["cfg3", "cfg4", "cfg5"])
    a = ap.parse_args()
    os.makedirs(a.out, exist_ok=True)
    for name in a.configs:
        w = wl.CONFIGS[name]()
        t0 = time.time()
        lines = list(HEAD)
        if name == "cfg4":
            lines.append(f"# input cfg4 {digest(w)} N={w.N} T={w.T} M={w.M} B={w.B}")
            for b in CFG4_CONFORMERS:
                I, A = orc.debye_sym(w.xyz[b], w.type, w.fftab, w.q, return_abs=True)
                lines += [f"cfg4 {b} {k} {float(w.q[k])!r} {float(I[k])!r} {float(A[k])!r}" for k in range(w.M)]
        else:
            lines.append(f"# input {name} {digest(w)} N={w.N} T={w.T} M={w.M}")
            I, A, nthr = orc.debye_sym(w.xyz, w.type, w.fftab, w.q, return_abs=True, return_threads=True)
            lines += [f"{name} 0 {k} {float(w.q[k])!r} {float(I[k])!r} {float(A[k])!r}" for k in range(w.M)]
            print(name, "threads", nthr, flush=True)
        path = os.path.join(a.out, f"oracle_full_{name}.txt")
        with open(path, "w") as f:
            f.write("\n".join(lines) + "\n")
        print(name, "done in", round(time.time() - t0, 1), "s ->", path, flush=True)


if __name__ == "__main__":
    main()
