"""Writes tests/golden/oracle_profiles.txt: oracle values of I(q_k) (Eq. 2) at sampled q indices
of the full-size BASELINE.json configs, where the oracle is too slow to run inside the test suite.

Calls ONLY oracle/ and the seeded input generators; nothing here touches the CUDA path.  The paper prints no
I(q) values (its profiles are figures), so these are oracle outputs, not paper numbers; the oracle itself is
pinned by tests/test_oracle_pins.py.

    python tests/golden/make_golden.py            # ~10 min on 8 cores
"""
import hashlib
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle as orc                                   # noqa: E402
from paper_1306_2258_b200 import workloads as wl                   # noqa: E402

SAMPLES = {
    "cfg2": list(range(0, 101, 10)),
    "cfg3": [0, 1, 37, 100, 150, 163, 180, 190, 199],
    "cfg3_8k": list(range(0, 200, 13)) + [199],
    "cfg5": [0, 2, 8, 40, 64, 72, 100, 112, 120, 124, 127],     # dense at high q: condition number ~400 there
}
CONFORMERS = [0, 1, 511, 1023]


def digest(w):
    h = hashlib.sha256()
    for a in (w.xyz, w.type, w.fftab, w.q):
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()[:16]


def main():
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_profiles.txt")
    lines = ["# oracle (fp64, Eq. 2 of arxiv 1306.2258, PAPER.md:41-42) at sampled q indices; written by tests/golden/make_golden.py",
             "# columns: config  conformer  k  q_k(float32 repr)  I(q_k)  sum|terms|   ; one '# input' line per config = sha256[:16] of the input bytes"]
    for name, ks in SAMPLES.items():
        w = wl.cfg3(n_bp=200, tag="cfg3_8k") if name == "cfg3_8k" else wl.CONFIGS[name]()
        t0 = time.time()
        I, A = orc.debye_sym(w.xyz, w.type, w.fftab[:, ks].copy(), w.q[ks].copy(), return_abs=True)
        lines.append(f"# input {name} {digest(w)} N={w.N} T={w.T} M={w.M}")
        for k, i, a in zip(ks, I, A):
            lines.append(f"{name} 0 {k} {float(w.q[k])!r} {float(i)!r} {float(a)!r}")
        print(name, "done in", round(time.time() - t0, 1), "s", flush=True)
    w = wl.cfg4()
    lines.append(f"# input cfg4 {digest(w)} N={w.N} T={w.T} M={w.M} B={w.B}")
    for b in CONFORMERS:
        I, A = orc.debye_sym(w.xyz[b], w.type, w.fftab, w.q, return_abs=True)
        for k in range(0, w.M, 9):
            lines.append(f"cfg4 {b} {k} {float(w.q[k])!r} {float(I[k])!r} {float(A[k])!r}")
    with open(out, "w") as f:
        f.write("\n".join(lines) + "\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
