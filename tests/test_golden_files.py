"""The stored oracle profiles (tests/golden/) belong to the inputs the generators produce today: every file's '# input'
line carries sha256[:16] of the input bytes, and the whole-profile files hold every q index (SURVEY.md section 7 step 2:
"cached in the repo with an input hash").  CPU only."""
import hashlib
import os

import numpy as np
import pytest

from paper_1306_2258_b200 import workloads as wl

GDIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def digest(w):
    h = hashlib.sha256()
    for a in (w.xyz, w.type, w.fftab, w.q):
        h.update(np.ascontiguousarray(a).tobytes())
    return h.hexdigest()[:16]


def parse(fn):
    inputs, rows = {}, {}
    for line in open(os.path.join(GDIR, fn)):
        if line.startswith("# input"):
            _, _, name, dg, *_ = line.split()
            inputs[name] = dg
        elif not line.startswith("#") and line.strip():
            name, b, k, q, I, A = line.split()
            rows.setdefault(name, []).append((int(b), int(k), float(q), float(I), float(A)))
    return inputs, rows


@pytest.mark.parametrize("fn,name,n_conf", [("oracle_full_cfg3.txt", "cfg3", 1), ("oracle_full_cfg5.txt", "cfg5", 1),
                                             ("oracle_full_cfg4.txt", "cfg4", 65)])
def test_whole_profiles_match_todays_inputs(fn, name, n_conf):
    inputs, rows = parse(fn)
    w = wl.CONFIGS[name]()
    assert inputs[name] == digest(w)
    r = rows[name]
    assert len(r) == n_conf * w.M
    assert sorted({k for _, k, *_ in r}) == list(range(w.M))
    for b, k, q, I, A in r:
        assert q == float(w.q[k]) and I > 0 and A >= I * (1 - 1e-12)
    # q = 0: I(0) = (sum f(0))^2 exactly (reading R3)
    tot = w.fftab.astype(np.float64)[w.type, 0].sum() ** 2
    for b, k, q, I, A in r:
        if k == 0:
            assert abs(I - tot) <= 1e-12 * tot


def test_sampled_profiles_match_todays_inputs():
    inputs, rows = parse("oracle_profiles.txt")
    for name, dg in inputs.items():
        w = wl.cfg3(n_bp=200, tag="cfg3_8k") if name == "cfg3_8k" else wl.CONFIGS[name]()
        assert dg == digest(w), name
