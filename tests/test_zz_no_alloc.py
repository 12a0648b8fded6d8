"""debye_profile_static (include/debye.h): the entry point that allocates nothing -- its scratch is a fixed __device__ array of
the library -- against the existing allocating path (debye_profile, which takes the same one-launch kernel with its records in
the cudaMalloc'ed workspace) and against the oracle, on calls in a row that share the array.

Named test_zz_* so that pytest collects it LAST (`pytest --collect-only -q`): the suite runs with `pytest -x`.  It depends on
nothing the other tests leave behind: it passes alone in a fresh process and after the rest of the suite."""
import ctypes as C

import numpy as np
import pytest

from oracle import oracle as orc
from paper_1306_2258_b200 import workloads as wl

TOL32 = 1e-4          # the FP32-accumulation tolerance of tests/test_parity_gpu.py (BASELINE.json north_star)


def rel(a, b):
    a, b = np.asarray(a), np.asarray(b)
    return float(np.max(np.abs(a - b) / np.abs(b)))


@pytest.fixture(scope="module")
def db():
    from paper_1306_2258_b200 import binding
    binding.lib()
    return binding


def to_dev(w):
    import torch
    return tuple(torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (w.xyz, w.type, w.fftab, w.q))


@pytest.mark.gpu
def test_static_scratch_entry_matches_the_allocating_path_on_calls_in_a_row(db):
    import torch
    # different sizes, type counts and grids back to back: the second and third call find the first one's records in the
    # array (more CTAs, more type pairs, more slots than they use themselves); the last case is the largest the array holds
    cases = [wl.small_random(41, 1500, 6, 101),                      # q_0 = 0, 100 chain indices
             wl.small_random(42, 300, 2, 24, q_min=0.025),           # q_0 = dq: q_k = (k + 1) dq; few CTAs, 3 type pairs
             wl.small_random(43, 1000, 5, 51),
             wl.small_random(44, 2048, 8, 129, q_max=0.8)]           # N, T and non-zero q count at the limits
    dev = [to_dev(w) for w in cases]
    hints = [db.q_hint(w.q) for w in cases]
    outs = [torch.full((w.M,), float("nan"), dtype=torch.float64, device="cuda") for w in cases]
    # the existing path first (it allocates its workspace), then one warm-up call of the new one (module load, symbol look-up)
    want = [db.debye_profile(*d, hint=h).cpu().numpy() for d, h in zip(dev, hints)]
    db.debye_profile_static(*dev[0], outs[0], hints[0])
    torch.cuda.synchronize()
    outs[0].fill_(float("nan"))
    free0 = torch.cuda.mem_get_info()[0]
    for rounds in range(2):                                         # two passes over the cases: eight calls in a row, no sync between
        for d, h, o in zip(dev, hints, outs):
            assert db.debye_profile_static(*d, o, h) is o
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                    # the device's free memory did not move: nothing was allocated
    for w, o, ref_gpu in zip(cases, outs, want):
        got = o.cpu().numpy()
        assert np.isfinite(got).all(), w.name
        assert rel(got, ref_gpu) <= TOL32, (w.name, rel(got, ref_gpu))
        # same kernel, same grid, same unit ranges: not merely close
        assert got.tobytes() == ref_gpu.tobytes(), (w.name, rel(got, ref_gpu))
        assert rel(got, orc.debye_sym(w.xyz, w.type, w.fftab, w.q)) <= TOL32, w.name
    # a wrong hint is caught on the device (NaN, never a wrong number), as in the allocating path
    x, t, f, q = dev[2]
    q_bad = q.clone()
    q_bad[7] *= 1.01
    o = torch.zeros(cases[2].M, dtype=torch.float64, device="cuda")
    db.debye_profile_static(x, t, f, q_bad, o, hints[2])
    assert torch.isnan(o).all()
    # ... and the array is still good for the next call
    o2 = torch.empty_like(o)
    db.debye_profile_static(x, t, f, q, o2, hints[2])
    assert o2.cpu().numpy().tobytes() == want[2].tobytes()


@pytest.mark.gpu
def test_static_scratch_entry_on_a_side_stream_and_refusals_leave_the_output_alone(db):
    import torch
    w = wl.small_random(45, 800, 4, 64)
    x, t, f, q = to_dev(w)
    h = db.q_hint(w.q)
    want = db.debye_profile(x, t, f, q, hint=h).cpu().numpy()
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    o = torch.empty(w.M, dtype=torch.float64, device="cuda")
    with torch.cuda.stream(s):
        db.debye_profile_static(x, t, f, q, o, h, stream=s)
        db.debye_profile_static(x, t, f, q, o, h, stream=s)
    s.synchronize()
    assert o.cpu().numpy().tobytes() == want.tobytes()
    # beyond the limits: refused before anything is launched, the output keeps its contents
    big = wl.small_random(46, 2049, 3, 32)
    xb, tb, fb, qb = to_dev(big)
    ob = torch.full((32,), -1.0, dtype=torch.float64, device="cuda")
    with pytest.raises(db.LibdebyeError, match="2048") as ei:
        db.debye_profile_static(xb, tb, fb, qb, ob, db.q_hint(big.q))
    assert ei.value.code == db.DEBYE_EUNSUPPORTED
    torch.cuda.synchronize()
    assert (ob == -1.0).all()


def test_static_scratch_entry_states_and_enforces_its_limits():
    """Host-side only (no GPU): the limits are what include/debye.h says, and every size beyond them -- or a call without the
    uniform-grid hint -- is refused with DEBYE_EUNSUPPORTED and a message that names the limit, before any CUDA call."""
    from paper_1306_2258_b200 import binding
    L = binding.lib()
    n_max, t_max, q_max, nbytes = binding.static_limits()
    assert (n_max, t_max, q_max) == (2048, 8, 128)
    assert nbytes == (256 + 36) * 128 * 8 and nbytes <= 1 << 20          # modest: under 1 MiB per GPU
    buf = (C.c_char * 4096)()
    p = C.cast(buf, C.c_void_p)
    H0 = (1 << 8) | (1 << 9) | (1 << 10)      # DEBYE_QHINT | _UNIFORM | _START0
    H1 = (1 << 8) | (1 << 9) | (1 << 11)      # ... | _STARTDQ
    EINVAL, EUNSUP = 1, 2

    def call(N, T, M, flags, ptr=p):
        st = L.debye_profile_static(ptr, ptr, N, ptr, T, ptr, M, ptr, flags, None)
        return st, L.debye_profile_static_error().decode()

    assert call(10, 2, 5, H0, None)[0] == EINVAL
    assert call(0, 2, 5, H0)[0] == EINVAL
    st, msg = call(n_max + 1, 2, 5, H0)
    assert st == EUNSUP and "2049" in msg and "2048" in msg
    st, msg = call(100, t_max + 1, 5, H0)
    assert st == EUNSUP and "9 types" in msg and "8" in msg
    st, msg = call(100, 2, q_max + 2, H0)          # 129 non-zero q values on a grid from 0
    assert st == EUNSUP and "129" in msg and "128" in msg
    st, msg = call(100, 2, q_max + 1, H1)          # 129 non-zero q values on a grid from dq
    assert st == EUNSUP and "129" in msg
    for flags in (0, 1 << 8, (1 << 8) | (1 << 9)):   # no hint, "not uniform", uniform with a general start
        st, msg = call(100, 2, 5, flags)
        assert st == EUNSUP and "DEBYE_QHINT" in msg
    for flags in (H0 | 1, H0 | (1 << 2), H0 | (1 << 4)):   # FP64, MUFU, accurate: they need the allocated workspace
        st, msg = call(100, 2, 5, flags)
        assert st == EUNSUP and "recurrence" in msg
