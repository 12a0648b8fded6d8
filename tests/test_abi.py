"""CPU-only checks of the boundary: libdebye.so loads, exports every symbol include/debye.h declares, and rejects
bad arguments with the documented status codes before touching CUDA (no compute calls here)."""
import ctypes as C
import os
import re

import pytest

from paper_1306_2258_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "debye.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(debye_[a-z_0-9]+)\s*\(", src)))


def test_library_loads_and_exports_every_declared_symbol():
    L = binding.lib()
    names = declared_symbols()
    assert set(binding.EXPORTS) == set(names), (names, binding.EXPORTS)
    for n in names:
        assert getattr(L, n) is not None
    assert L.debye_version() >= 100


def test_strerror_and_status_codes():
    L = binding.lib()
    assert L.debye_strerror(0) == b"ok"
    for st in (1, 2, 3, 4, 99):
        assert len(L.debye_strerror(st)) > 0


def test_argument_validation_happens_before_cuda():
    L = binding.lib()
    buf = (C.c_char * 4096)()
    p = C.cast(buf, C.c_void_p)
    EINVAL, EUNSUP = 1, 2
    ok_args = dict(N=10, T=2, M=5)
    assert L.debye_profile(None, p, 10, p, 2, p, 5, p, 0, None) == EINVAL
    assert L.debye_profile(p, None, 10, p, 2, p, 5, p, 0, None) == EINVAL
    assert L.debye_profile(p, p, 10, None, 2, p, 5, p, 0, None) == EINVAL
    assert L.debye_profile(p, p, 10, p, 2, None, 5, p, 0, None) == EINVAL
    assert L.debye_profile(p, p, 10, p, 2, p, 5, None, 0, None) == EINVAL
    assert L.debye_profile(p, p, 0, p, 2, p, 5, p, 0, None) == EINVAL
    assert L.debye_profile(p, p, 10, p, 0, p, 5, p, 0, None) == EINVAL
    assert L.debye_profile(p, p, 10, p, 33, p, 5, p, 0, None) == EINVAL
    assert L.debye_profile(p, p, 10, p, 2, p, 0, p, 0, None) == EINVAL
    assert L.debye_profile(p, p, 10, p, 2, p, 4097, p, 0, None) == EINVAL
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, (1 << 2) | (1 << 3), None) == EINVAL      # two sinc variants
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, (1 << 0) | (1 << 2), None) == EINVAL      # fp64 + fp32 variant
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, 1 << 20, None) == EINVAL                  # unknown flag
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, 1 << 9, None) == EINVAL                   # hint sub-bit without DEBYE_QHINT
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, (1 << 8) | (1 << 10), None) == EINVAL     # start bit without uniform
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, (1 << 8) | (1 << 9) | (1 << 10) | (1 << 11), None) == EINVAL
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, 1 << 12, None) == EINVAL                  # pieces hint without DEBYE_QHINT
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, (1 << 8) | (1 << 12) | (1 << 9), None) == EINVAL   # pieces and uniform
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, (1 << 8) | (3 << 16), None) == EINVAL     # piece count without the pieces bit
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, (1 << 8) | (1 << 12) | (16 << 21), None) == EINVAL  # more than 128 accumulators
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, (1 << 5) | (1 << 3), None) == EINVAL      # centred and recurrence
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, 1 << 5, None) == EUNSUP                   # centred form without the pieces hint
    assert L.debye_profile(p, p, 10, p, 2, p, 5, p, (1 << 5) | (1 << 8) | (1 << 9), None) == EUNSUP
    assert L.debye_profile(p, p, (1 << 24) + 1, p, 2, p, 5, p, 0, None) == EUNSUP
    assert L.debye_profile_batch(p, p, 10, 0, p, 2, p, 5, p, 0, None) == EINVAL
    assert L.debye_profile_host(None, p, 10, p, 2, p, 5, p, 0, None) == EINVAL
    assert L.debye_partials_shard(p, p, 10, 1, p, 2, 5, p, p, 0, 2, 2, None) == EINVAL          # rank outside [0, world)
    assert L.debye_partials_shard(p, p, 10, 1, p, 2, 5, p, p, 0, 0, 0, None) == EINVAL
    assert L.debye_partials_shard(None, p, 10, 1, p, 2, 5, p, p, 0, 0, 2, None) == EINVAL
    assert L.debye_profile_from_partials(None, 2, p, p, 1, 2, 5, p, None) == EINVAL
    assert L.debye_profile_peratom(None, p, 10, p, 5, p, 0, None) == EINVAL
    assert L.debye_profile_peratom(p, p, 0, p, 5, p, 0, None) == EINVAL
    assert L.debye_profile_peratom(p, p, 10, p, 4097, p, 0, None) == EINVAL
    assert L.debye_profile_peratom(p, p, 10, p, 5, p, 1 << 3, None) == EUNSUP                   # recurrence demanded without a grid hint
    assert L.debye_profile_peratom(p, p, 10, p, 5, p, (1 << 3) | (1 << 2), None) == EINVAL      # recurrence and MUFU
    assert L.debye_profile_peratom(p, p, 10, p, 5, p, (1 << 3) | 1, None) == EINVAL             # recurrence and FP64
    assert L.debye_profile_peratom(p, p, 10, p, 5, p, 1 << 10, None) == EINVAL                  # hint sub-bit without DEBYE_QHINT
    assert L.debye_profile_peratom(p, p, (1 << 24) + 1, p, 5, p, 0, None) == EUNSUP
    assert L.debye_profile_from_partials(p, 0, p, p, 1, 2, 5, p, None) == EINVAL
    assert L.debye_profile_from_partials(p, 2, p, p, 1, 33, 5, p, None) == EINVAL
    assert L.debye_partials(p, p, 10, 1, None, 2, 5, p, None, 0, None) == EINVAL
    del ok_args


def test_workspace_and_launch_info_are_host_side():
    L = binding.lib()
    assert L.debye_workspace_bytes(0, 1, 2, 5, 0) == 0
    small = L.debye_workspace_bytes(1000, 1, 5, 51, 0)
    big = L.debye_workspace_bytes(200000, 1, 20, 128, 0)
    assert 0 < small < big < (1 << 30)
    # O(N + CTAs*T^2*M), never O(N^2): doubling N adds ~20 bytes per atom
    a, b = L.debye_workspace_bytes(100000, 1, 5, 64, 0), L.debye_workspace_bytes(200000, 1, 5, 64, 0)
    assert 15 * 100000 < b - a < 25 * 100000
    info = binding.launch_info(10000, 1, 5, 101, "auto")
    # no hint: setup(+pack: N*B <= 16384), recurrence sized for 100 and for 101 chain indices, centred form (general start), MUFU,
    # reduce, epilogue -- the device runs one of the four pairs launches, the others return at once
    assert info == {"n_launches": 7, "q_chunk": 104, "n_chunks": 1}
    assert binding.launch_info(50000, 1, 4, 200, "recur") == {"n_launches": 5, "q_chunk": 104, "n_chunks": 2}
    assert binding.launch_info(1000, 1, 5, 51, "fp64")["n_chunks"] == 2
    assert binding.launch_info(1000, 1, 5, 300, "mufu") == {"n_launches": 4, "q_chunk": 104, "n_chunks": 3}


def test_binding_refuses_non_cuda_inputs():
    import numpy as np
    import torch
    x = torch.zeros(4, 3)
    with pytest.raises(binding.LibdebyeError):
        binding.debye_profile(x, torch.zeros(4, dtype=torch.int32), torch.zeros(1, 2), torch.zeros(2))
    with pytest.raises(binding.LibdebyeError):
        binding.debye_profile_host(np.zeros((4, 3)), np.zeros(4, np.int32), np.zeros((1, 2), np.float32),
                                   np.zeros(2, np.float32))       # float64 xyz


def test_q_hint_classifies_grids_on_the_host():
    """debye_q_hint applies the device's classification to a host copy of q (include/debye.h, DEBYE_QHINT_*)."""
    import numpy as np
    from paper_1306_2258_b200 import workloads as wl
    H, U, Z, D = 1 << 8, 1 << 9, 1 << 10, 1 << 11
    assert binding.q_hint(wl.q_grid(0.5, 101)) == H | U | Z                    # starts at 0
    assert binding.q_hint(wl.q_grid(1.0, 50, 0.02)) == H | U | D               # the paper's grid k/50, k = 1..50
    P = 1 << 12

    def pieces(n, K):
        return H | P | ((n - 1) << 16) | ((K // 8 - 1) << 21)
    # uniform with a general start, descending, or a few uniform pieces: the piecewise-uniform hint (centred product form) with
    # the number of pieces and the accumulators per thread the launch is sized for
    assert binding.q_hint(wl.q_grid(0.9, 64, 0.3)) == pieces(1, 64)
    assert binding.q_hint(wl.q_grid(0.3, 31)[::-1].copy()) == pieces(1, 32)
    assert binding.q_hint(wl.q_grid(0.9, 200, 0.3)) == pieces(2, 104)          # more than 128 points: equal pieces
    # pieces only where they pay (pieces x (start-up + accumulators) against 8 cycles per q of the MUFU kernel): not for lone points
    assert binding.q_hint(np.array([0.0, 0.1, 0.25], np.float32)) == H and binding.q_hint_pieces(np.array([0.0, 0.1, 0.25], np.float32)) == pieces(2, 8)
    saxs_waxs = np.concatenate([np.arange(51) * 0.005, 0.25 + 0.01 * np.arange(1, 51)]).astype(np.float32)
    assert binding.q_hint(saxs_waxs) == pieces(2, 56) and binding.pieces_of(binding.q_hint(saxs_waxs)) == (2, 56)
    assert binding.q_hint(np.delete(wl.q_grid(0.5, 101), 37)) == pieces(2, 64)  # a dropped point: 37 + 63
    # a grid from 0 or dq with more than 256 chain indices would need more than two recurrence chunks (chain form): pieces instead
    assert binding.q_hint(wl.q_grid(1.7, 1000)) == pieces(8, 128) and binding.q_hint(wl.q_grid(1.7, 257)) == H | U | Z
    assert binding.q_hint(wl.q_grid(2.57, 257, 0.01)) == pieces(3, 88) and binding.q_hint(wl.q_grid(2.56, 256, 0.01)) == H | U | D
    assert binding.q_hint_pieces(wl.q_grid(0.5, 101)) == pieces(1, 104)        # any uniform grid can be forced into the centred form ...
    assert binding.q_hint(wl.q_grid(0.5, 101)) == H | U | Z                    # ... but from 0 or dq the telescoped form is preferred
    rng = np.random.default_rng(5)
    assert binding.q_hint(np.sort(rng.uniform(0, 0.7, 40)).astype(np.float32)) == H      # no structure: the MUFU kernel
    assert binding.q_hint_pieces(np.sort(rng.uniform(0, 0.7, 40)).astype(np.float32)) in (0, pieces(20, 8))     # pairs of points are "uniform"
    assert binding.q_hint_pieces(np.sort(rng.uniform(0, 0.7, 200)).astype(np.float32)) == 0
    assert binding.pieces_of(H | U) == (0, 0)
    assert binding.q_hint(np.array([0.0], np.float32)) == H | U | Z
    assert binding.q_hint(np.array([0.3], np.float32)) in (H | U | D, pieces(1, 8))
    # a grid is uniform if every q[k] is within 1.5 float ulps of ITSELF of the line through the end points: grids rounded once
    # from the exact line pass at every size and range, a jitter of 2 ulps of q_max at low k does not
    for qmax, M, qmin in ((0.5, 101, 0.0), (1.0, 50, 0.02), (0.3, 128, 0.0), (1.7, 4096, 0.0), (0.9, 64, 0.3), (25.0, 999, 0.0)):
        assert binding.q_hint(wl.q_grid(qmax, M, qmin)) & (U | P), (qmax, M, qmin)
        assert binding.q_hint(np.linspace(qmin, qmax, M, dtype=np.float32)) & (U | P)
        assert binding.q_hint((np.arange(M) * np.float32((qmax - qmin) / (M - 1)) + np.float32(qmin)).astype(np.float32)) & (U | P) or M > 500
    g = wl.q_grid(0.5, 101)
    j = g.copy(); j[3] = np.nextafter(np.nextafter(j[3], np.float32(1)), np.float32(1)); j[7] += 2 * np.spacing(np.float32(0.5))
    assert not binding.q_hint(j) & U                                          # not uniform as a whole ...
    assert binding.q_hint(j) == pieces(3, 96)                                 # ... but three uniform pieces (7 + the lone jittered point + 93)
    L = binding.lib()
    assert L.debye_q_hint(None, 5) == 0
    # with a hint exactly one pairs instantiation is launched
    assert binding.launch_info(10000, 1, 5, 101, "auto", hint=H | U | Z) == {"n_launches": 4, "q_chunk": 100, "n_chunks": 1}
    assert binding.launch_info(10000, 1, 5, 101, "auto", hint=H | U | D) == {"n_launches": 4, "q_chunk": 104, "n_chunks": 1}
    assert binding.launch_info(10000, 1, 5, 101, "auto", hint=H)["n_launches"] == 4
    assert binding.launch_info(10000, 1, 5, 101, "auto", hint=pieces(2, 56)) == {"n_launches": 4, "q_chunk": 56, "n_chunks": 2}
