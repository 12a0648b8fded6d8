"""GPU parity tests proper: libdebye (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (BASELINE.json north_star): max_k |I_gpu - I_oracle| / |I_oracle| <= 1e-4 for the FP32
accumulation paths, <= 1e-10 for the FP64 mode."""
import math
import os

import numpy as np
import pytest

from oracle import oracle as orc
from paper_1306_2258_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL32, TOL64 = 1e-4, 1e-10
FP32_VARIANTS = ["auto", "recur", "mufu", "accurate"]


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


def gpu_profile(db, w, variant="auto", batch=False):
    import torch
    x, t, f, q = to_dev(w)
    out = (db.debye_profile_batch if batch else db.debye_profile)(x, t, f, q, variant=variant)
    torch.cuda.synchronize()
    return out.cpu().numpy()


# sizes span several 128-atom rows / 64-atom tiles and ragged tails; T and M exercise every chunking
CASES = [
    ("s3_N130_T3_M17", lambda: wl.small_random(3, 130, 3, 17)),
    ("s4_N777_T5_M101", lambda: wl.small_random(4, 777, 5, 101)),
    ("s5_N1500_T4_M200", lambda: wl.small_random(5, 1500, 4, 200, q_max=1.0)),          # 2 recurrence chunks
    ("s6_N600_T20_M128", lambda: wl.small_random(6, 600, 20, 128, q_max=0.3)),
    ("s7_N900_T3_M64_offset_grid", lambda: wl.small_random(7, 900, 3, 64, q_min=0.3, q_max=0.9)),   # general start
    ("s8_N513_T32_M40_signed", lambda: wl.small_random(8, 513, 32, 40, signed=True)),
    ("s9_N2100_T2_M300", lambda: wl.small_random(9, 2100, 2, 300, q_max=1.2, box=60.0)),  # 4 chunks
    # grids starting at q = 0 where dropping the trivial index saves a whole chunk (129 -> 128 indices: 1 chunk instead of 2;
    # 257 -> 256: 2 instead of 4): the device picks the smaller of two recurrence launches
    ("s10_N400_T2_M129", lambda: wl.small_random(10, 400, 2, 129, q_max=0.8)),
    ("s11_N300_T3_M257", lambda: wl.small_random(11, 300, 3, 257, q_max=1.0)),
    ("s12_N500_T2_M129_from_dq", lambda: wl.small_random(12, 500, 2, 129, q_min=0.005, q_max=0.645)),   # q_k = (k + 1) dq
    ("cfg1", wl.cfg1),
    ("table1_N1000_paper_grid", lambda: wl.table1(1000)),                                 # q_k = k/50, k = 1..50
]


@pytest.mark.parametrize("name,make", CASES, ids=[c[0] for c in CASES])
def test_parity_all_variants(db, name, make):
    w = make()
    ref, A = orc.debye_sym(w.xyz, w.type, w.fftab, w.q, return_abs=True)
    if (w.fftab < 0).any():
        # signed form factors: I may come close to 0; use the documented floor 1e-4 * sum|terms| instead
        floor = np.maximum(np.abs(ref), 1e-2 * A)
        err = lambda I: float(np.max(np.abs(I - ref) / floor))
    else:
        err = lambda I: rel(I, ref)
    assert err(gpu_profile(db, w, "fp64")) <= TOL64
    for v in FP32_VARIANTS:
        e = err(gpu_profile(db, w, v))
        assert e <= TOL32, (name, v, e)


def test_two_atom_closed_form_distance_sweep(db):
    """I = f1^2 + f2^2 + 2 f1 f2 sin(qd)/(qd) (north_star); d from far below the slow-path cut to 3000 A."""
    q = wl.q_grid(0.5, 101)
    f = np.stack([np.linspace(6, 2, 101), np.linspace(8, 1, 101)]).astype(np.float32)
    typ = np.array([0, 1], np.int32)
    worst = {v: 0.0 for v in FP32_VARIANTS + ["fp64"]}
    ds = [0.0, 1e-3, 0.05, 0.3, 0.7, 0.79, 0.81, 1.0, 1.37, 2.2, 3.7, 9.9, 31.4159, 62.83, 78.54, 157.08, 400.3, 1234.5, 3000.0]
    for d in ds:
        xyz = np.array([[0.5, 0.25, -1.0], [0.5, 0.25, -1.0 + d]], np.float32)
        dd = float(np.float64(xyz[1, 2]) - np.float64(xyz[0, 2]))
        qq = q.astype(np.float64)
        s = np.where(qq * dd == 0, 1.0, np.sin(qq * dd) / np.where(qq * dd == 0, 1.0, qq * dd))
        want = f[0].astype(np.float64) ** 2 + f[1].astype(np.float64) ** 2 + 2 * f[0].astype(np.float64) * f[1] * s
        w = wl.Workload("two", xyz, typ, f, q)
        for v in worst:
            worst[v] = max(worst[v], rel(gpu_profile(db, w, v), want))
    assert worst["fp64"] <= TOL64, worst
    for v in FP32_VARIANTS:
        assert worst[v] <= TOL32, worst


def test_degenerate_inputs(db):
    import torch
    q = wl.q_grid(0.6, 33)
    f = wl.gaussian_form_factors(1, 3, q)
    # N = 1: I = f^2
    w = wl.Workload("one", np.array([[1, 2, 3]], np.float32), np.array([1], np.int32), f, q)
    for v in ["auto", "mufu", "fp64"]:
        assert rel(gpu_profile(db, w, v), f[1].astype(np.float64) ** 2) <= 1e-15
    # all atoms coincident: I = (sum f)^2 for every q
    typ = np.array([0, 1, 2, 2, 1, 0, 0], np.int32)
    w = wl.Workload("coin", np.tile(np.array([[1.5, -2.0, 0.25]], np.float32), (7, 1)), typ, f, q)
    tot = f.astype(np.float64)[typ].sum(0) ** 2
    for v in FP32_VARIANTS:
        assert rel(gpu_profile(db, w, v), tot) <= 1e-6
    assert rel(gpu_profile(db, w, "fp64"), tot) <= 1e-13
    # q = 0 only (M = 1), and a single non-zero q
    w0 = wl.small_random(20, 300, 3, 1)
    w0.q[:] = 0
    assert rel(gpu_profile(db, w0), w0.fftab.astype(np.float64)[w0.type, 0].sum() ** 2) <= 1e-14
    w1 = wl.small_random(21, 300, 3, 1, q_max=0.37)
    ref = orc.debye_sym(w1.xyz, w1.type, w1.fftab, w1.q)
    for v in FP32_VARIANTS:
        assert rel(gpu_profile(db, w1, v), ref) <= TOL32
    # a type that never occurs, and a type with a single atom
    w2 = wl.small_random(22, 400, 4, 25)
    w2.type[w2.type == 2] = 0
    w2.type[7] = 3
    w2.type[w2.type == 3] = np.where(np.arange((w2.type == 3).sum()) == 0, 3, 1)
    assert (w2.type == 2).sum() == 0 and (w2.type == 3).sum() == 1
    ref = orc.debye_sym(w2.xyz, w2.type, w2.fftab, w2.q)
    for v in FP32_VARIANTS:
        assert rel(gpu_profile(db, w2, v), ref) <= TOL32
    assert rel(gpu_profile(db, w2, "fp64"), ref) <= TOL64
    torch.cuda.synchronize()


def test_non_uniform_and_descending_grids(db):
    w = wl.small_random(23, 500, 3, 40)
    rng = np.random.default_rng(0)
    w.q[:] = np.sort(rng.uniform(0, 0.7, 40)).astype(np.float32)
    w.fftab[:] = wl.gaussian_form_factors(5, 3, w.q)
    ref = orc.debye_sym(w.xyz, w.type, w.fftab, w.q)
    for v in ["auto", "mufu", "accurate"]:
        assert rel(gpu_profile(db, w, v), ref) <= TOL32
    assert rel(gpu_profile(db, w, "fp64"), ref) <= TOL64
    assert np.isnan(gpu_profile(db, w, "recur")).all()          # documented: forced recurrence on a non-uniform grid
    # descending uniform grid, and a grid containing negative q (sinc is even)
    w2 = wl.small_random(24, 300, 2, 31)
    w2.q[:] = w2.q[::-1].copy()
    w2.fftab[:] = w2.fftab[:, ::-1].copy()
    ref2 = orc.debye_sym(w2.xyz, w2.type, w2.fftab, w2.q)
    for v in FP32_VARIANTS:
        assert rel(gpu_profile(db, w2, v), ref2) <= TOL32
    w3 = wl.small_random(25, 300, 2, 31)
    w3.q[:] = np.linspace(-0.3, 0.3, 31).astype(np.float32)
    ref3 = orc.debye_sym(w3.xyz, w3.type, w3.fftab, w3.q)
    for v in FP32_VARIANTS:
        assert rel(gpu_profile(db, w3, v), ref3) <= TOL32


def test_bitwise_determinism_and_host_entry(db):
    import torch
    w = wl.small_random(26, 3000, 5, 101)
    a = gpu_profile(db, w)
    b = gpu_profile(db, w)
    assert a.tobytes() == b.tobytes()
    s = torch.cuda.Stream()
    x, t, f, q = to_dev(w)
    torch.cuda.synchronize()
    c = db.debye_profile(x, t, f, q, stream=s)
    s.synchronize()
    assert c.cpu().numpy().tobytes() == a.tobytes()
    h = db.debye_profile_host(w.xyz, w.type, w.fftab, w.q)
    assert h.tobytes() == a.tobytes()


def test_batch_equals_singles(db):
    w = wl.cfg4(B=9, N=700)
    ref = orc.debye_batch(w.xyz, w.type, w.fftab, w.q)
    Ib = gpu_profile(db, w, batch=True)
    assert Ib.shape == (9, w.M)
    assert rel(Ib, ref) <= TOL32
    for b in (0, 8):
        one = gpu_profile(db, wl.Workload("one", w.xyz[b].copy(), w.type, w.fftab, w.q))
        assert rel(Ib[b], one) <= 1e-6
    assert rel(gpu_profile(db, w, "fp64", batch=True), ref) <= TOL64
    hb = db.debye_profile_batch_host(w.xyz, w.type, w.fftab, w.q)
    assert hb.tobytes() == Ib.tobytes()


def test_invariances(db):
    w = wl.small_random(27, 1200, 4, 64)
    I = gpu_profile(db, w)
    perm = np.random.default_rng(3).permutation(w.N)
    wp = wl.Workload("p", w.xyz[perm].copy(), w.type[perm].copy(), w.fftab, w.q)
    assert rel(gpu_profile(db, wp), I) <= 1e-5
    ws = wl.Workload("s", np.ascontiguousarray(w.xyz[:, [2, 0, 1]] * np.float32(-1)), w.type, w.fftab, w.q)
    assert rel(gpu_profile(db, ws), I) <= 1e-5


def test_partials_reconstruct_profile_and_match_oracle(db):
    import torch
    w = wl.small_random(28, 400, 3, 21)
    x, t, f, q = to_dev(w)
    S, n = db.debye_partials(x, t, q, w.T)
    torch.cuda.synchronize()
    S = S.cpu().numpy()[0]; n = n.cpu().numpy()
    assert list(n) == [int((w.type == a).sum()) for a in range(w.T)]
    ref = orc.debye_sym(w.xyz, w.type, w.fftab, w.q)
    F = w.fftab.astype(np.float64)
    I = (n[:, None] * F ** 2).sum(0)
    p = 0
    for a in range(w.T):
        for b in range(a, w.T):
            I += 2 * F[a] * F[b] * S[p]; p += 1
    assert rel(I, ref) <= TOL32
    # S_aa and S_ab straight from the oracle with indicator form factors: I_a = n_a + 2 S_aa, I_ab = n_a + n_b + 2 (S_aa + S_bb + S_ab)
    ind = lambda ts: np.stack([np.full(w.M, 1.0 if a in ts else 0.0, np.float32) for a in range(w.T)])
    Ia = {a: orc.debye_sym(w.xyz, w.type, ind([a]), w.q) for a in range(w.T)}
    idx = lambda a, b: a * (2 * w.T - a + 1) // 2 + (b - a)
    for a in range(w.T):
        Saa = (Ia[a] - n[a]) / 2
        assert np.max(np.abs(S[idx(a, a)] - Saa)) <= 1e-4 * np.max(np.abs(Saa)) + 1e-9
    Iab = orc.debye_sym(w.xyz, w.type, ind([0, 2]), w.q)
    S02 = (Iab - n[0] - n[2]) / 2 - (Ia[0] - n[0]) / 2 - (Ia[2] - n[2]) / 2
    assert np.max(np.abs(S[idx(0, 2)] - S02)) <= 1e-4 * np.max(np.abs(S02)) + 1e-9


def test_caller_workspace(db):
    import torch
    w = wl.small_random(29, 800, 3, 51)
    ref = gpu_profile(db, w)
    L = db.lib()
    need = L.debye_workspace_bytes(w.N, 1, w.T, w.M, 0)
    buf = torch.empty(need + 256, dtype=torch.uint8, device="cuda")
    ptr = (buf.data_ptr() + 255) // 256 * 256
    assert L.debye_set_workspace(ptr, need) == 0
    try:
        assert gpu_profile(db, w).tobytes() == ref.tobytes()
        assert L.debye_set_workspace(ptr, 1024) == 0
        with pytest.raises(db.LibdebyeError):
            gpu_profile(db, w)
    finally:
        assert L.debye_set_workspace(None, 0) == 0
    assert gpu_profile(db, w).tobytes() == ref.tobytes()


def test_weighted_profiles_match_the_weighted_oracle(db):
    """Per-atom weights f_j = w_j F[t_j] (reading R10w; include/debye.h debye_profile_weighted): every variant against the
    oracle, weights of both signs, the batch entry, the host entry, and weight 1 == the unweighted call."""
    import torch
    rng = np.random.default_rng(11)
    for name, w0, M in (("one_chunk", wl.small_random(30, 900, 4, 64), 64), ("two_chunks", wl.small_random(31, 700, 3, 150, q_max=0.9), 150)):
        wt = rng.uniform(0.3, 2.5, w0.N).astype(np.float32)
        ref, A = orc.debye_sym(w0.xyz, w0.type, w0.fftab, w0.q, weight=wt, return_abs=True)
        x, t, f, q = to_dev(w0)
        wd = torch.from_numpy(wt).cuda()
        for v in ["auto", "recur", "mufu"]:
            I = db.debye_profile_weighted(x, t, wd, f, q, variant=v).cpu().numpy()
            assert rel(I, ref) <= TOL32, (name, v, rel(I, ref))
        # the libdevice-sinf reference variant exists for the plain calls only (include/debye.h DEBYE_SINC_ACCURATE)
        with pytest.raises(db.LibdebyeError) as ei:
            db.debye_profile_weighted(x, t, wd, f, q, variant="accurate")
        assert ei.value.code == db.DEBYE_EUNSUPPORTED
        assert rel(db.debye_profile_weighted(x, t, wd, f, q, variant="fp64").cpu().numpy(), ref) <= TOL64
        ones = torch.ones(w0.N, dtype=torch.float32, device="cuda")
        # weight 1 is the unweighted profile up to summation order (weighted calls reduce their accumulators once per row)
        assert rel(db.debye_profile_weighted(x, t, ones, f, q).cpu().numpy(), db.debye_profile(x, t, f, q).cpu().numpy()) <= 1e-6
        h = db.debye_profile_weighted_host(w0.xyz, w0.type, wt, w0.fftab, w0.q)
        assert h.tobytes() == db.debye_profile_weighted(x, t, wd, f, q).cpu().numpy().tobytes()
    # signed weights (negative contrast): compare against the documented floor 1e-2 * sum|terms|
    w1 = wl.small_random(32, 600, 3, 48)
    ws = (rng.uniform(0.5, 2.0, w1.N) * np.where(rng.uniform(size=w1.N) < 0.3, -1, 1)).astype(np.float32)
    ref, A = orc.debye_sym(w1.xyz, w1.type, w1.fftab, w1.q, weight=ws, return_abs=True)
    x, t, f, q = to_dev(w1)
    I = db.debye_profile_weighted(x, t, torch.from_numpy(ws).cuda(), f, q).cpu().numpy()
    assert float(np.max(np.abs(I - ref) / np.maximum(np.abs(ref), 1e-2 * A))) <= TOL32
    # batch with shared weights
    wb = wl.cfg4(B=5, N=500)
    wt = rng.uniform(0.5, 1.5, wb.N).astype(np.float32)
    refb = orc.debye_batch(wb.xyz, wb.type, wb.fftab, wb.q, weight=wt)
    xb, t, f, q = to_dev(wb)
    Ib = db.debye_profile_weighted(xb, t, torch.from_numpy(wt).cuda(), f, q).cpu().numpy()
    assert Ib.shape == (5, wb.M) and rel(Ib, refb) <= TOL32


def test_random_shape_sweep(db):
    """Seeded sweep over small shapes: every accumulator count K (multiples of 4 and of 8), 1-4 chunks, grids starting at
    0, at dq and elsewhere, 1-3 conformers, 1-6 types, row counts around the 128-atom row and 512-atom tile boundaries."""
    import torch
    rng = np.random.default_rng(2024)
    worst = 0.0
    for case in range(48):
        N = int(rng.choice([2, 3, 31, 127, 128, 129, 200, 383, 513, 640]))
        T = int(rng.integers(1, 7))
        M = int(rng.choice([1, 2, 3, 7, 8, 9, 12, 13, 33, 52, 64, 65, 97, 100, 101, 128, 129, 130, 200, 257, 300]))
        B = int(rng.choice([1, 1, 2, 3]))
        start = int(rng.integers(0, 3))                       # 0: q0 = 0, 1: q0 = dq, 2: offset grid
        dq = float(rng.uniform(0.002, 0.02))
        q0 = [0.0, dq, float(rng.uniform(0.05, 0.3))][start]
        q = (q0 + dq * np.arange(M)).astype(np.float32)
        if start == 0:
            q[0] = 0.0
        xyz = (rng.uniform(-1, 1, (B, N, 3)) * float(rng.uniform(5, 60))).astype(np.float32)
        typ = rng.integers(0, T, N).astype(np.int32)
        f = wl.gaussian_form_factors(1000 + case, T, q)
        ref = np.stack([orc.debye_sym(xyz[b], typ, f, q) for b in range(B)])
        x, t, fd, qd = (torch.from_numpy(a).cuda() for a in (xyz, typ, f, q))
        for v in ("auto", "mufu"):
            I = db.debye_profile_batch(x, t, fd, qd, variant=v).cpu().numpy()
            e = rel(I, ref)
            worst = max(worst, e)
            assert e <= TOL32, (case, N, T, M, B, start, v, e)
    assert worst <= 1e-5, worst                               # typical error of these small, well-conditioned cases


def test_grid_hints_select_one_launch_and_are_checked(db):
    """DEBYE_QHINT_* (include/debye.h): with the right hint the result is the unhinted one -- bit for bit where the hint
    only removes launches, to rounding where it selects the single fused launch for small structures (debye_small.cuh: the
    same terms, summed by other CTAs); a wrong hint gives NaN, never a wrong number."""
    import torch
    grids = {"zero": wl.q_grid(0.5, 101), "dq": wl.q_grid(1.0, 50, 0.02), "offset": wl.q_grid(0.9, 64, 0.3),
             "nonuniform": np.sort(np.random.default_rng(7).uniform(0.01, 0.8, 40)).astype(np.float32),
             "zero_129": wl.q_grid(0.8, 129)}
    base = wl.small_random(40, 700, 3, 8)
    hints = {k: db.q_hint(v) for k, v in grids.items()}
    assert len({hints[k] for k in ("zero", "dq", "offset", "nonuniform")}) == 4
    for name, qg in grids.items():
        f = wl.gaussian_form_factors(77, 3, qg)
        x, t = (torch.from_numpy(a).cuda() for a in (base.xyz, base.type))
        fd, qd = torch.from_numpy(f).cuda(), torch.from_numpy(qg).cuda()
        plain = db.debye_profile(x, t, fd, qd).cpu().numpy()
        ref = orc.debye_sym(base.xyz, base.type, f, qg)
        assert rel(plain, ref) <= TOL32
        hinted = db.debye_profile(x, t, fd, qd, hint=hints[name]).cpu().numpy()
        if db.launch_info(base.N, 1, 3, len(qg), "auto", hint=hints[name])["n_launches"] == 1:      # the fused small-structure launch
            assert name in ("zero", "dq", "zero_129") and rel(hinted, plain) <= 2e-6 and rel(hinted, ref) <= TOL32
            assert hinted.tobytes() == db.debye_profile(x, t, fd, qd, hint=hints[name]).cpu().numpy().tobytes()
        elif db.pieces_of(hints[name])[0]:      # general start: the hint selects the centred product form, the unhinted call runs the chain
            assert name == "offset" and rel(hinted, plain) <= 2e-6 and rel(hinted, ref) <= TOL32
        else:
            assert hinted.tobytes() == plain.tobytes(), name
        for other, h in hints.items():
            if h != hints[name]:
                assert np.isnan(db.debye_profile(x, t, fd, qd, hint=h).cpu().numpy()).all(), (name, other)
    hb = db.debye_profile_host(base.xyz, base.type, wl.gaussian_form_factors(77, 3, grids["zero"]), grids["zero"], hint=hints["zero"])
    assert np.isfinite(hb).all()


def test_small_structure_single_launch(db):
    """debye_small_kernel (PAPER.md:88 "N < W", :25 refinement loops): with a grid hint a structure of at most 2048 atoms and
    8 types on a grid q_k = (k + koff) dq with at most 128 chain indices runs as ONE launch (sort in shared memory per CTA,
    product-form pairs, last-CTA reduction + epilogue).  Against the oracle, against the general path, twice for bits; the
    partial structure factors too; shapes that span 1..16 rows, 1..8 types, ragged segments, the size limits."""
    import torch
    shapes = [(2, 1, 5, 0.0), (3, 2, 9, 0.0), (130, 3, 17, 0.0), (777, 5, 101, 0.0), (1000, 8, 51, 0.0), (1031, 4, 129, 0.0),
              (500, 2, 128, 0.005), (2048, 5, 64, 0.0), (1999, 7, 33, 0.02), (257, 1, 2, 0.0), (64, 8, 100, 0.004)]
    for si, (N, T, M, q_min) in enumerate(shapes):
        w = wl.small_random(200 + si, N, T, M, q_min=q_min, q_max=q_min * M if q_min else 0.6, box=20.0 + N ** (1 / 3) * 3)
        hint = db.q_hint(w.q)
        assert db.launch_info(N, 1, T, M, "auto", hint=hint)["n_launches"] == 1, (N, T, M)
        x, t, f, q = to_dev(w)
        ref = orc.debye_sym(w.xyz, w.type, w.fftab, w.q)
        a = db.debye_profile(x, t, f, q, hint=hint).cpu().numpy()
        assert rel(a, ref) <= TOL32, (N, T, M, rel(a, ref))
        assert rel(a, gpu_profile(db, w)) <= 5e-6
        assert a.tobytes() == db.debye_profile(x, t, f, q, hint=hint).cpu().numpy().tobytes()
        S, n = db.debye_partials(x, t, q, T, hint=hint)
        assert np.array_equal(n.cpu().numpy(), np.bincount(w.type, minlength=T))
        S = S.cpu().numpy()[0]
        F = w.fftab.astype(np.float64)
        I = (n.cpu().numpy()[:, None] * F * F).sum(0)
        tp = 0
        for ta in range(T):
            for tb in range(ta, T):
                I = I + 2.0 * F[ta] * F[tb] * S[tp]
                tp += 1
        assert rel(I, a) <= 1e-12
    # a wrong hint gives NaN; just beyond the limits the general path runs
    w = wl.small_random(230, 300, 3, 40, q_min=0.3, q_max=0.9)          # general start, but the caller promises q[0] == 0
    x, t, f, q = to_dev(w)
    assert np.isnan(db.debye_profile(x, t, f, q, hint=db.q_hint(wl.q_grid(0.5, 40))).cpu().numpy()).all()
    assert db.launch_info(2049, 1, 3, 40, "auto", hint=db.q_hint(wl.q_grid(0.5, 40)))["n_launches"] > 1
    assert db.launch_info(500, 1, 9, 40, "auto", hint=db.q_hint(wl.q_grid(0.5, 40)))["n_launches"] > 1
    assert db.launch_info(500, 1, 3, 130, "auto", hint=db.q_hint(wl.q_grid(0.5, 130)))["n_launches"] > 1
    # coincident atoms and a single atom
    w1 = wl.Workload("one", np.zeros((1, 3), np.float32), np.zeros(1, np.int32), np.full((1, 9), 3.0, np.float32), wl.q_grid(0.4, 9))
    x, t, f, q = to_dev(w1)
    assert np.allclose(db.debye_profile(x, t, f, q, hint=db.q_hint(w1.q)).cpu().numpy(), 9.0, rtol=0, atol=0)
    wc = wl.Workload("coincident", np.zeros((40, 3), np.float32), np.zeros(40, np.int32), np.full((1, 9), 1.0, np.float32), wl.q_grid(0.4, 9))
    x, t, f, q = to_dev(wc)
    assert rel(db.debye_profile(x, t, f, q, hint=db.q_hint(wc.q)).cpu().numpy(), np.full(9, 1600.0)) <= 1e-6


def test_maximum_q_count_and_type_count(db):
    """Edge of the documented limits (include/debye.h): M = DEBYE_MAX_Q = 4096 (32 recurrence chunks, general start) with
    T = DEBYE_MAX_TYPES = 32, on a grid from 0 and on an offset grid; every variant that supports it."""
    for q_min in (0.0, 0.05):
        w = wl.small_random(50, 150, 32, 4096, q_min=q_min, q_max=1.5, box=30.0)
        ref = orc.debye_sym(w.xyz, w.type, w.fftab, w.q)
        for v in ("auto", "mufu"):
            e = rel(gpu_profile(db, w, v), ref)
            assert e <= TOL32, (q_min, v, e)
        assert rel(gpu_profile(db, w, "fp64"), ref) <= TOL64


def test_plan_execute_equals_the_plain_calls_bit_for_bit(db):
    """debye_plan_* (include/debye.h): setup once, execute per set of coordinates; same kernels in the same order as the
    plain calls, so the results are identical bit for bit -- for a grid from 0, the paper's grid, a non-uniform grid,
    with weights, and for a batch."""
    import torch
    rng = np.random.default_rng(21)
    grids = [wl.q_grid(0.5, 101), wl.q_grid(1.0, 50, 0.02), np.sort(rng.uniform(0.01, 0.7, 33)).astype(np.float32),
             np.concatenate([np.arange(41) * 0.005, 0.2 + 0.02 * np.arange(1, 31)]).astype(np.float32),      # two uniform pieces
             wl.q_grid(0.9, 150, 0.3)]                                                                       # general start, two pieces
    for qg in grids:
        base = wl.small_random(60, 900, 4, 8)
        f = wl.gaussian_form_factors(5, 4, qg)
        t, fd, qd = (torch.from_numpy(a).cuda() for a in (base.type, f, qg))
        plan = db.Plan(t, qd, 4)
        for rep in range(3):                                   # new coordinates, same plan
            xyz = (base.xyz + rng.normal(0, 0.5, base.xyz.shape)).astype(np.float32)
            x = torch.from_numpy(xyz).cuda()
            a = plan.execute(x, fd).cpu().numpy()
            b = db.debye_profile(x, t, fd, qd, hint=db.q_hint(qg)).cpu().numpy()     # a plan knows its grid: same launches as a hinted call
            assert a.tobytes() == b.tobytes()
            assert rel(a, orc.debye_sym(xyz, base.type, f, qg)) <= TOL32
        plan.destroy()
    # weights and a batch
    wb = wl.cfg4(B=3, N=400)
    wt = rng.uniform(0.5, 1.5, wb.N).astype(np.float32)
    xb, t, fd, qd = to_dev(wb)
    wd = torch.from_numpy(wt).cuda()
    plan = db.Plan(t, qd, wb.T, B=3, weight=wd)
    a = plan.execute(xb, fd).cpu().numpy()
    assert a.tobytes() == db.debye_profile_weighted(xb, t, wd, fd, qd).cpu().numpy().tobytes()
    assert rel(a, orc.debye_batch(wb.xyz, wb.type, wb.fftab, wb.q, weight=wt)) <= TOL32
    plan.destroy()


def test_calls_on_different_streams_do_not_corrupt_each_other(db):
    """include/debye.h: the per-device scratch is ordered across streams with an event (calls on different streams serialise
    on the device); a plan owns its scratch, so plans on different streams may overlap.  Eight rounds of interleaved calls
    on three streams, large enough to overlap in time if nothing ordered them, against the single-stream results bit for bit."""
    import torch
    ws = [wl.small_random(90 + i, 2600 + 300 * i, 4, 101) for i in range(3)]       # beyond the single-launch size limit
    devs = [to_dev(w) for w in ws]
    refs = [gpu_profile(db, w) for w in ws]
    for i, w in enumerate(ws):
        assert rel(refs[i], orc.debye_sym(w.xyz, w.type, w.fftab, w.q)) <= TOL32
    streams = [torch.cuda.Stream() for _ in range(3)]
    outs = [[None] * 3 for _ in range(8)]
    for r in range(8):                                       # plain calls: shared scratch, three streams
        for i in (r % 3, (r + 1) % 3, (r + 2) % 3):
            x, t, f, q = devs[i]
            outs[r][i] = db.debye_profile(x, t, f, q, stream=streams[i])
    torch.cuda.synchronize()
    for r in range(8):
        for i in range(3):
            assert outs[r][i].cpu().numpy().tobytes() == refs[i].tobytes(), (r, i)
    plans = [db.Plan(devs[i][1], devs[i][3], ws[i].T) for i in range(3)]
    torch.cuda.synchronize()
    pref = [plans[i].execute(devs[i][0], devs[i][2]).cpu().numpy() for i in range(3)]
    for r in range(8):                                       # plans: own scratch, three streams, no ordering between them
        for i in (r % 3, (r + 1) % 3, (r + 2) % 3):
            outs[r][i] = plans[i].execute(devs[i][0], devs[i][2], stream=streams[i])
    # one plan on two streams in turn: serialised by the plan's own event
    twice = [plans[0].execute(devs[0][0], devs[0][2], stream=streams[k % 2]) for k in range(6)]
    torch.cuda.synchronize()
    for r in range(8):
        for i in range(3):
            assert outs[r][i].cpu().numpy().tobytes() == pref[i].tobytes(), (r, i)
    for o in twice:
        assert o.cpu().numpy().tobytes() == pref[0].tobytes()
    for i in range(3):
        assert rel(pref[i], orc.debye_sym(ws[i].xyz, ws[i].type, ws[i].fftab, ws[i].q)) <= TOL32
        plans[i].destroy()


def test_grid_jittered_by_two_ulps_is_taken_as_it_is(db):
    """A grid whose points sit 2 float ulps of q_max off the uniform line is NOT run through the recurrence (which would
    evaluate the line instead of q[k]): the device classifies it as non-uniform and the MUFU kernel takes q as given."""
    w = wl.small_random(95, 3000, 3, 96, q_max=0.6, box=80.0)
    rng = np.random.default_rng(5)
    qj = (w.q + rng.integers(-2, 3, w.M) * np.spacing(np.float32(0.6))).astype(np.float32)
    qj[0] = 0.0
    wj = wl.Workload("jitter", w.xyz, w.type, w.fftab, qj)
    assert db.q_hint(qj) == 1 << 8                                           # DEBYE_QHINT alone: not uniform
    ref = orc.debye_sym(wj.xyz, wj.type, wj.fftab, wj.q)
    assert rel(gpu_profile(db, wj), ref) <= 1e-5
    assert gpu_profile(db, wj).tobytes() == gpu_profile(db, wj, "mufu").tobytes()
    assert np.isnan(gpu_profile(db, wj, "recur")).all()                      # forced recurrence on a non-uniform grid: NaN


def _regrid(w, q, seed=77):
    q = np.ascontiguousarray(q, dtype=np.float32)
    return wl.Workload(w.name + "_regrid", w.xyz, w.type, wl.gaussian_form_factors(seed, w.T, q), q)


PIECE_GRIDS = [
    # name, grid, (pieces, accumulators per thread) the hint must carry
    ("saxs_waxs", np.concatenate([np.arange(51) * 0.005, 0.25 + 0.01 * np.arange(1, 51)]), (2, 56)),
    ("dropped_point", np.delete(wl.q_grid(0.5, 101), 37), (2, 64)),
    ("three_ranges", np.concatenate([np.arange(1, 41) * 0.002, 0.08 + 0.005 * np.arange(1, 41), 0.28 + 0.02 * np.arange(1, 30)]), (3, 40)),
    ("general_start", wl.q_grid(0.9, 64, 0.3), (1, 64)),
    ("general_start_200", 0.0123 + np.arange(200) * 0.004, (2, 104)),
    ("descending", wl.q_grid(0.3, 31)[::-1].copy(), (1, 32)),
    ("through_zero", np.linspace(-0.3, 0.3, 31), (1, 32)),
    ("lone_points", np.array([0.0, 0.1, 0.25]), None),            # pieces, but too short to pay: debye_q_hint leaves them to the MUFU kernel
    ("repeated_q", np.array([0.1, 0.1, 0.1, 0.2, 0.3, 0.4]), None),
    ("one_point", np.array([0.37]), None),
]


def test_piecewise_uniform_grids_run_the_centred_product_form(db):
    """DEBYE_QHINT_PIECES / DEBYE_SINC_CENTRED (include/debye.h): a grid made of a few uniform
    pieces -- SAXS + WAXS ranges, a dropped point, a general start -- runs the centred product form (debye_pairs.cuh), one
    launch, against the oracle and against the MUFU kernel, which takes any grid."""
    import torch
    base = wl.small_random(50, 1500, 4, 8)
    for name, qg, want in PIECE_GRIDS:
        w = _regrid(base, qg)
        h = db.q_hint(w.q)
        if want is not None:
            assert db.pieces_of(h) == want, (name, hex(h), db.pieces_of(h))
        ref = orc.debye_sym(w.xyz, w.type, w.fftab, w.q)
        x, t, f, q = to_dev(w)
        hp = db.q_hint_pieces(w.q)
        assert hp != 0
        I = db.debye_profile(x, t, f, q, variant="centred", hint=hp).cpu().numpy()
        assert rel(I, ref) <= TOL32, (name, rel(I, ref))
        assert I.tobytes() == db.debye_profile(x, t, f, q, variant="centred", hint=hp).cpu().numpy().tobytes()     # bitwise reproducible
        if db.pieces_of(h)[0]:
            assert h == hp
            assert db.debye_profile(x, t, f, q, hint=h).cpu().numpy().tobytes() == I.tobytes()      # automatic mode takes it from the hint
            assert db.launch_info(w.N, 1, w.T, w.M, "auto", hint=h)["n_launches"] == 4            # setup (+ pack), ONE pairs launch, reduce, epilogue
        assert rel(db.debye_profile(x, t, f, q, variant="mufu").cpu().numpy(), I) <= 1e-5
        assert rel(db.debye_profile(x, t, f, q).cpu().numpy(), ref) <= TOL32                        # no hint: whatever the device chooses
    # every accumulator count (both layouts: K = 16 L + 8 with the seeds as level 0, K = 16 L without), general start
    for K in range(8, 129, 8):
        for M in (K, K - 7 if K > 8 else 1):
            w = _regrid(wl.small_random(51, 600, 3, 8), 0.0371 + (0.55 / 128) * np.arange(M))
            hp = db.q_hint_pieces(w.q)
            assert db.pieces_of(hp) == (1, K)
            x, t, f, q = to_dev(w)
            I = db.debye_profile(x, t, f, q, variant="centred", hint=hp).cpu().numpy()
            assert rel(I, orc.debye_sym(w.xyz, w.type, w.fftab, w.q)) <= TOL32, (K, M)
    # weights, a batch, the host entry
    rng = np.random.default_rng(3)
    qg = PIECE_GRIDS[0][1]
    w = _regrid(wl.small_random(52, 900, 4, 8), qg)
    h = db.q_hint(w.q)
    x, t, f, q = to_dev(w)
    wt = (rng.uniform(0.3, 2.0, w.N) * np.where(rng.uniform(size=w.N) < 0.2, -1, 1)).astype(np.float32)
    refw, A = orc.debye_sym(w.xyz, w.type, w.fftab, w.q, weight=wt, return_abs=True)
    Iw = db.debye_profile_weighted(x, t, torch.from_numpy(wt).cuda(), f, q, hint=h).cpu().numpy()
    assert float(np.max(np.abs(Iw - refw) / np.maximum(np.abs(refw), 1e-2 * A))) <= TOL32
    wb = wl.cfg4(B=4, N=500)
    wb = wl.Workload("batch_regrid", wb.xyz, wb.type, wl.gaussian_form_factors(9, wb.T, qg.astype(np.float32)), qg.astype(np.float32))
    xb, t, f, q = to_dev(wb)
    Ib = db.debye_profile_batch(xb, t, f, q, hint=h).cpu().numpy()
    assert rel(Ib, orc.debye_batch(wb.xyz, wb.type, wb.fftab, wb.q)) <= TOL32
    for b in range(4):       # same terms, other CTA ranges than in the batch: equal to rounding
        one = db.debye_profile(xb[b].contiguous(), t, f, q, hint=h).cpu().numpy()
        assert rel(Ib[b], one) <= 1e-6
    Ih = db.debye_profile_host(wb.xyz[0], wb.type, wb.fftab, wb.q, hint=h)
    assert Ih.tobytes() == db.debye_profile(xb[0].contiguous(), t, f, q, hint=h).cpu().numpy().tobytes()


def test_piecewise_hint_is_checked_on_the_device_and_degenerate_pairs_keep_their_limits(db):
    import torch
    base = wl.small_random(53, 500, 3, 8)
    grids = {n: np.ascontiguousarray(g, dtype=np.float32) for n, g, _ in PIECE_GRIDS[:5]}
    hints = {n: db.q_hint(g) for n, g in grids.items()}
    assert len(set(hints.values())) == len(hints)
    for n, g in grids.items():
        w = _regrid(base, g)
        x, t, f, q = to_dev(w)
        for other, h in hints.items():
            I = db.debye_profile(x, t, f, q, hint=h).cpu().numpy()
            assert np.isnan(I).all() == (other != n), (n, other)            # a hint sized for another grid: NaN, never a wrong number
    # a grid with the promised piece count and size but other break points is still right: the device cuts q itself
    ga = np.concatenate([np.arange(51) * 0.005, 0.25 + 0.01 * np.arange(1, 51)]).astype(np.float32)
    gb = np.concatenate([np.arange(50) * 0.005, 0.245 + 0.01 * np.arange(1, 52)]).astype(np.float32)
    assert db.q_hint(ga) == db.q_hint(gb)
    w = _regrid(base, gb)
    x, t, f, q = to_dev(w)
    assert rel(db.debye_profile(x, t, f, q, hint=db.q_hint(ga)).cpu().numpy(), orc.debye_sym(w.xyz, w.type, w.fftab, w.q)) <= TOL32
    # all atoms coincident: I = (sum f)^2 at every q (r = 0: every seed and weight takes its limit).  The centred form gets a term
    # below the piece's centre q_c as a difference (P - Q)/4 of sums of size ~q_c, so a term at q carries ~1e-7 q_c/q relative
    # error: random over pairs in a real structure, coherent here where all pairs are the same pair (q_c/q = 24 at the first
    # non-zero q of this grid; the telescoped form and the MUFU kernel hold 1e-6, test_degenerate_inputs)
    qg = grids["saxs_waxs"]
    f = wl.gaussian_form_factors(1, 3, qg)
    typ = np.array([0, 1, 2, 2, 1, 0, 0], np.int32)
    wc = wl.Workload("coin", np.tile(np.array([[1.5, -2.0, 0.25]], np.float32), (7, 1)), typ, f, qg)
    x, t, fd, q = to_dev(wc)
    assert rel(db.debye_profile(x, t, fd, q, hint=hints["saxs_waxs"]).cpu().numpy(), f.astype(np.float64)[typ].sum(0) ** 2) <= 5e-6
    # two atoms, closed form I = f1^2 + f2^2 + 2 f1 f2 sin(qd)/(qd), distances from far below one grid step to 3000 A
    f2 = np.stack([np.linspace(6, 2, len(qg)), np.linspace(8, 1, len(qg))]).astype(np.float32)
    worst = 0.0
    for d in [0.0, 1e-3, 0.05, 0.3, 0.81, 1.37, 3.7, 9.9, 31.4159, 78.54, 400.3, 1234.5, 3000.0]:
        xyz = np.array([[0.5, 0.25, -1.0], [0.5, 0.25, -1.0 + d]], np.float32)
        dd = float(np.float64(xyz[1, 2]) - np.float64(xyz[0, 2]))
        qq = qg.astype(np.float64)
        sinc = np.where(qq * dd == 0, 1.0, np.sin(qq * dd) / np.where(qq * dd == 0, 1.0, qq * dd))
        want = f2[0].astype(np.float64) ** 2 + f2[1].astype(np.float64) ** 2 + 2 * f2[0].astype(np.float64) * f2[1] * sinc
        x, t, fd, q = to_dev(wl.Workload("two", xyz, np.array([0, 1], np.int32), f2, qg))
        worst = max(worst, rel(db.debye_profile(x, t, fd, q, hint=hints["saxs_waxs"]).cpu().numpy(), want))
    assert worst <= TOL32, worst


def test_c_abi_from_plain_c(db, tmp_path):
    """The boundary is a C ABI: tests/c_abi_client.c -- plain C, include/debye.h and the CUDA runtime only, no Python and no torch
    in the process -- is compiled with gcc, linked against libdebye.so and run on cfg1 and on a 2000-atom case; its profiles
    (host-buffer entry, device-buffer entry, the no-allocation entry) are compared with the oracle here.  Prints the latencies
    the client measured (host entry: one H2D copy of the gathered inputs, the kernel, one D2H copy, synchronise)."""
    import shutil
    import subprocess
    import sys
    from paper_1306_2258_b200 import binding
    gcc, cuda = shutil.which("gcc"), os.environ.get("CUDA_HOME", "/usr/local/cuda")
    if gcc is None or not os.path.exists(os.path.join(cuda, "include", "cuda_runtime.h")):
        pytest.skip("needs gcc and the CUDA runtime headers")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    libdir = os.path.dirname(binding.LIB_PATH)
    exe = str(tmp_path / "c_abi_client")
    subprocess.check_call([gcc, "-O2", "-std=c11", "-D_POSIX_C_SOURCE=200809L", "-o", exe, os.path.join(root, "tests", "c_abi_client.c"),
                           "-I", os.path.join(root, "include"), "-I", os.path.join(cuda, "include"), "-L", libdir, "-L", os.path.join(cuda, "lib64"),
                           "-l:" + os.path.basename(binding.LIB_PATH), "-lcudart", "-lm",
                           "-Wl,-rpath," + libdir, "-Wl,-rpath," + os.path.join(cuda, "lib64")])
    for w in (wl.cfg1(), wl.small_random(71, 2000, 5, 50, q_min=0.02, q_max=1.0)):
        fin, fout = str(tmp_path / "in.bin"), str(tmp_path / "out.bin")
        with open(fin, "wb") as fh:
            np.array([w.N, w.T, w.M], np.int32).tofile(fh)
            for a in (w.xyz, w.type, w.fftab, w.q):
                np.ascontiguousarray(a).tofile(fh)
        r = subprocess.run([exe, fin, fout, "300"], capture_output=True, text=True, timeout=300)
        assert r.returncode == 0, (r.stdout, r.stderr)
        sys.stdout.write("c_abi_client: " + r.stdout)
        res = np.fromfile(fout, np.float64)
        assert res.shape == (3 * w.M + 3,)
        I_host, I_dev, I_static, lat = res[:w.M], res[w.M:2 * w.M], res[2 * w.M:3 * w.M], res[3 * w.M:]
        ref = orc.debye_sym(w.xyz, w.type, w.fftab, w.q)
        assert rel(I_host, ref) <= TOL32 and I_host.tobytes() == I_dev.tobytes() == I_static.tobytes()
        x, t, f, q = to_dev(w)
        assert I_dev.tobytes() == db.debye_profile(x, t, f, q, hint=db.q_hint(w.q)).cpu().numpy().tobytes()      # the binding adds nothing
        assert (lat > 0).all() and lat[0] < 5e3


def test_non_finite_input_propagates_and_does_not_poison_later_calls(db):
    """include/debye.h: NaN / Inf in the inputs propagate to I_out (no hang, no crash); the next call is unaffected."""
    w = wl.small_random(70, 500, 3, 40)
    good = gpu_profile(db, w)
    bad = wl.Workload("nan", w.xyz.copy(), w.type, w.fftab, w.q)
    bad.xyz[17, 1] = np.nan
    bad.xyz[300, 0] = np.inf
    for v in ("auto", "mufu", "fp64"):
        I = gpu_profile(db, bad, v)
        assert not np.isfinite(I[1:]).any(), v               # every q > 0 involves the poisoned atoms
    assert gpu_profile(db, w).tobytes() == good.tobytes()


def test_non_finite_conformer_does_not_reach_its_neighbours_in_a_batch(db):
    """A NaN coordinate in ONE conformer of a batch makes that conformer's profile NaN and leaves every other conformer's
    profile bit-identical to a clean run: masked pairs (tile tails, read-ahead of the pipeline) read their coordinates from
    a valid entry of the current tile, never from whatever an earlier tile -- possibly of another conformer -- left behind.
    Odd atom counts per type make the two-pairs-per-iteration loop end on a masked partner."""
    for N, M in ((301, 101), (517, 64), (203, 128)):
        geo, tab = wl.cfg4(B=5, N=N), wl.small_random(3, 10, 5, M, q_max=0.5)      # 5 conformers; a 5-type table on M points
        w = wl.Workload("batch", geo.xyz, geo.type, tab.fftab, tab.q)
        clean = gpu_profile(db, w, batch=True)
        bad = wl.Workload("nanbatch", w.xyz.copy(), w.type, w.fftab, w.q)
        bad.xyz[2, N // 3, 1] = np.nan
        bad.xyz[2, N - 1, 2] = np.inf
        for v in ("auto", "mufu"):
            ref = clean if v == "auto" else gpu_profile(db, w, v, batch=True)
            I = gpu_profile(db, bad, v, batch=True)
            assert not np.isfinite(I[2, 1:]).any(), v
            for b in (0, 1, 3, 4):
                assert I[b].tobytes() == ref[b].tobytes(), (v, b, N)


def test_q_grid_split_over_ranks_reassembles_the_profile(db):
    """sharding.profile_q_slice (different q ranges on different devices), the ranks emulated one after
    the other on one GPU: the slices tile the grid and agree with the unsplit profile and the oracle."""
    import torch
    from paper_1306_2258_b200 import sharding
    w = wl.small_random(80, 1100, 4, 101)
    x, t, f, q = to_dev(w)
    ref = orc.debye_sym(w.xyz, w.type, w.fftab, w.q)
    whole = db.debye_profile(x, t, f, q).cpu().numpy()
    fn = lambda ff, qq: db.debye_profile(x, t, ff, qq)
    for world in (2, 3, 8):
        parts, cover = [], []
        for rank in range(world):
            loc, (lo, hi) = sharding.profile_q_slice(fn, f, q, rank, world)
            parts.append(loc.cpu().numpy()); cover += list(range(lo, hi))
        I = np.concatenate(parts)
        assert cover == list(range(w.M))
        assert rel(I, ref) <= TOL32 and rel(I, whole) <= 1e-5


def test_tile_split_over_ranks_sums_to_the_whole_and_matches_the_oracle(db):
    """debye_partials_shard / debye_profile_from_partials (tiles of the upper triangle cyclic over ranks, one
    all-gather of FP64 partials, fixed-order sum + epilogue on the device), the ranks emulated one after the other on one
    GPU (they do not wait on one another).  Every variant; grids that contain q = 0 (closed-form term: rank 0 only),
    start at dq, are offset, or are not uniform; a batch; more ranks than the small case has busy CTAs."""
    import torch
    from paper_1306_2258_b200 import sharding
    cases = [
        (wl.small_random(81, 1300, 4, 101), False),
        (wl.small_random(82, 700, 3, 129, q_min=0.005, q_max=0.645), False),
        (wl.small_random(83, 900, 5, 64, q_min=0.3, q_max=0.9), False),
        (wl.cfg4(B=3, N=500), True),
    ]
    for w, batch in cases:
        x, t, f, q = to_dev(w)
        ref = orc.debye_batch(w.xyz, w.type, w.fftab, w.q) if batch else orc.debye_sym(w.xyz, w.type, w.fftab, w.q)[None]
        for variant in ("auto", "mufu", "fp64"):
            tol = TOL64 if variant == "fp64" else TOL32
            S_full, n_full = db.debye_partials(x, t, q, w.T, variant=variant)
            whole = (db.debye_profile_batch if batch else db.debye_profile)(x, t, f, q, variant=variant).cpu().numpy().reshape(ref.shape)
            for world in (1, 2, 3, 8):
                parts = []
                for rank in range(world):
                    S, n = db.debye_partials_shard(x, t, q, w.T, rank, world, variant=variant)
                    assert torch.equal(n, n_full)
                    parts.append(S)
                S_parts = torch.stack(parts)
                if world > 1:       # nobody's share is the whole thing, and the shares add up to it
                    assert sum(float(p.abs().sum()) > 0 for p in parts) >= 2
                tot = S_parts.sum(0)
                # same per-CTA FP64 sums, only the last FP64 additions are regrouped.  In the product form of the recurrence
                # S is a telescoped sum (B_{Sj+k0} = Out[j][k0] + B_{Sj-k0}, debye_pairs.cuh) whose terms can be ~1e3 times
                # larger than S itself, so the regrouping shows up at 1e-16 x that factor x sqrt(#additions)
                assert float(((tot - S_full).abs() / (S_full.abs() + 1e-300)).max()) <= (1e-10 if world > 1 else 0.0)
                I = db.debye_profile_from_partials(S_parts, n_full, f).cpu().numpy()
                assert I.shape == ref.shape
                assert rel(I, ref) <= tol and rel(I, whole) <= 1e-11
                # through the sharding helper (no process group: the gather is the identity for world == 1)
                if world == 1:
                    I1 = sharding.profile_tile_split(lambda r, wd: db.debye_partials_shard(x, t, q, w.T, r, wd, variant=variant),
                                                     db.debye_profile_from_partials, f, 0, 1).cpu().numpy()
                    assert np.array_equal(I1, I)
    # a non-uniform grid with an explicit q = 0 in the middle (MUFU kernel chosen on the device)
    w = wl.small_random(84, 600, 3, 33)
    qn = np.sort(np.random.default_rng(84).uniform(0.01, 0.6, w.M)).astype(np.float32); qn[7] = 0.0
    w2 = wl.Workload("nonuniform", w.xyz, w.type, w.fftab, qn)
    x, t, f, q = to_dev(w2)
    ref = orc.debye_sym(w2.xyz, w2.type, w2.fftab, w2.q)
    parts = torch.stack([db.debye_partials_shard(x, t, q, w2.T, r, 4)[0] for r in range(4)])
    n = db.debye_partials(x, t, q, w2.T)[1]
    assert rel(db.debye_profile_from_partials(parts, n, f).cpu().numpy()[0], ref) <= TOL32
    # repeated calls are bitwise identical, and an unsharded call afterwards is not disturbed by the zeroed records
    a = db.debye_partials_shard(x, t, q, w2.T, 1, 4)[0]
    assert torch.equal(a, parts[1])
    assert rel(db.debye_profile(x, t, f, q).cpu().numpy(), ref) <= TOL32


def test_tile_split_argument_validation(db):
    import torch
    w = wl.small_random(85, 200, 2, 11)
    x, t, f, q = to_dev(w)
    for rank, world in ((-1, 2), (2, 2), (0, 0), (0, 5000)):
        with pytest.raises(db.LibdebyeError):
            db.debye_partials_shard(x, t, q, w.T, rank, world)
    S, n = db.debye_partials(x, t, q, w.T)
    with pytest.raises(db.LibdebyeError):
        db.debye_profile_from_partials(S[None][:, :, :2].contiguous(), n, f)


def _peratom_ff(w, seed):
    """per-ATOM rows (the form factor depends on the atom's environment): the type's row times a per-atom
    factor in [0.6, 1.4] plus a per-atom q-dependent offset, so that no two atoms share a row"""
    rng = np.random.default_rng(seed)
    base = w.fftab[w.type].astype(np.float64)
    fac = rng.uniform(0.6, 1.4, (w.N, 1))
    off = rng.uniform(-0.3, 0.3, (w.N, 1)) * np.exp(-np.linspace(0, 2, w.M))[None, :]
    return np.ascontiguousarray((base * fac + off).astype(np.float32))


def test_peratom_form_factors_match_the_peratom_oracle(db):
    """debye_profile_peratom (the paper's general case; NEXT-1) against oracle_debye_peratom, element by
    element: sizes spanning several 128-atom rows, 64-atom tiles and 32-q chunks with ragged tails, uniform / offset /
    non-uniform / descending grids with q = 0 inside, signed rows; FP32 (1e-4) and FP64 (1e-10) arithmetic."""
    import torch
    cases = [
        wl.small_random(90, 130, 3, 17),
        wl.small_random(91, 777, 5, 101),
        wl.small_random(92, 1500, 4, 200, q_max=1.0),
        wl.small_random(93, 513, 8, 40, signed=True),
        wl.small_random(94, 900, 3, 64, q_min=0.3, q_max=0.9),
        wl.small_random(95, 2100, 2, 33, q_max=1.2, box=60.0),
        wl.cfg1(),
    ]
    for n, w in enumerate(cases):
        ff = _peratom_ff(w, 900 + n)
        qn = w.q.copy()
        if n % 2 == 1:      # non-uniform, descending, with an explicit zero in the middle
            qn = np.sort(np.random.default_rng(n).uniform(0.01, float(w.q.max()) + 0.1, w.M)).astype(np.float32)[::-1].copy()
            qn[w.M // 2] = 0.0
        ref = orc.debye_peratom(w.xyz, ff, qn)
        x = torch.from_numpy(w.xyz).cuda(); f = torch.from_numpy(ff).cuda(); q = torch.from_numpy(qn).cuda()
        for variant, tol in (("auto", TOL32), ("mufu", TOL32), ("fp64", TOL64)):
            I = db.debye_profile_peratom(x, f, q, variant=variant).cpu().numpy()
            assert rel(I, ref) <= tol, (n, variant, rel(I, ref))
        a = db.debye_profile_peratom(x, f, q); b = db.debye_profile_peratom(x, f, q)
        assert torch.equal(a, b)                                       # bitwise reproducible
    # rows copied from a type table: the per-type path and its oracle
    w = wl.small_random(96, 1100, 4, 101)
    x, t, f, q = to_dev(w)
    ffc = torch.from_numpy(np.ascontiguousarray(w.fftab[w.type])).cuda()
    I = db.debye_profile_peratom(x, ffc, q).cpu().numpy()
    assert rel(I, orc.debye_sym(w.xyz, w.type, w.fftab, w.q)) <= TOL32
    assert rel(I, db.debye_profile(x, t, f, q).cpu().numpy()) <= 1e-5


def test_peratom_recurrence_on_hinted_uniform_grids(db):
    """debye_profile_peratom with a grid hint (grids q_k = (k + koff) dq): the chain recurrence with one packed FMA per term
    against f_j(q_k) (debye_peratom_recur.cuh) instead of one MUFU.SIN per term.  Against oracle_debye_peratom element by
    element and against the direct kernel; one and two chunks, K % 8 == 4, grids from 0 and from dq, ragged rows, close and
    coincident atoms (the small-theta path), a wrong hint, a grid it does not take."""
    import torch
    # up to 2048 atoms on a one-chunk grid: the single fused launch (debye_peratom_small.cuh); beyond, or two chunks: four launches
    shapes = [(2, 9, 0.0), (3, 17, 0.0), (130, 33, 0.0), (777, 101, 0.0), (1500, 129, 0.0), (700, 128, 0.004), (1100, 200, 0.0),
              (400, 257, 0.0), (515, 52, 0.01), (900, 64, 0.0), (2048, 128, 0.004), (2049, 64, 0.0), (2600, 101, 0.0)]
    for si, (N, M, q_min) in enumerate(shapes):
        w = wl.small_random(300 + si, N, 3, M, q_min=q_min, q_max=q_min * M if q_min else 0.7, box=12.0 + N ** (1 / 3) * 3)
        ff = _peratom_ff(w, 400 + si)
        hint = db.q_hint(w.q)
        x, f, q = (torch.from_numpy(a).cuda() for a in (w.xyz, ff, w.q))
        ref = orc.debye_peratom(w.xyz, ff, w.q)
        a = db.debye_profile_peratom(x, f, q, hint=hint, variant="recur").cpu().numpy()
        assert rel(a, ref) <= TOL32, (N, M, q_min, rel(a, ref))
        assert rel(a, db.debye_profile_peratom(x, f, q).cpu().numpy()) <= 2e-5          # the direct kernel
        assert a.tobytes() == db.debye_profile_peratom(x, f, q, hint=hint).cpu().numpy().tobytes()      # automatic choice, and run to run
        assert np.array_equal(a, db.debye_profile_peratom_host(w.xyz, ff, w.q, hint=hint))
    # close pairs (theta far below the small-theta threshold) and coincident atoms
    xyz = np.array([[0, 0, 0], [0, 0, 0], [1e-3, 0, 0], [0.02, 0.01, 0], [3.0, 1.0, -2.0], [0.3, 0.0, 0.0]], np.float32)
    qg = wl.q_grid(0.5, 101)
    ff = (1.0 + 0.3 * np.random.default_rng(3).standard_normal((6, 101))).astype(np.float32)
    a = db.debye_profile_peratom(torch.from_numpy(xyz).cuda(), torch.from_numpy(ff).cuda(), torch.from_numpy(qg).cuda(), hint=db.q_hint(qg)).cpu().numpy()
    assert rel(a, orc.debye_peratom(xyz, ff, qg)) <= 1e-5
    # a wrong hint gives NaN; a general-start grid is not taken by the recurrence
    w = wl.small_random(330, 300, 3, 40, q_min=0.3, q_max=0.9)
    ff = _peratom_ff(w, 1)
    x, f, q = (torch.from_numpy(a_).cuda() for a_ in (w.xyz, ff, w.q))
    assert np.isnan(db.debye_profile_peratom(x, f, q, hint=db.q_hint(wl.q_grid(0.5, 40))).cpu().numpy()).all()
    with pytest.raises(db.LibdebyeError):
        db.debye_profile_peratom(x, f, q, hint=db.q_hint(w.q), variant="recur")
    assert rel(db.debye_profile_peratom(x, f, q, hint=db.q_hint(w.q)).cpu().numpy(), orc.debye_peratom(w.xyz, ff, w.q)) <= TOL32


def test_peratom_batch_of_conformers_shares_the_table(db):
    """debye_profile_peratom_batch (include/debye.h): B conformers, one per-atom table.  Hinted grids from 0 and from dq run one
    fused launch sequence (unit line conformer -> chunk -> row -> j), one and two chunks, a wave of CTAs that spans several
    conformers and conformers that span several CTAs; other grids / variants run conformer by conformer.  Against the
    per-atom oracle on every conformer and against the single-structure entry."""
    import torch
    rng = np.random.default_rng(17)
    for si, (B, N, M, q_min) in enumerate([(5, 300, 64, 0.0), (3, 900, 101, 0.0), (7, 130, 50, 0.02), (2, 1100, 200, 0.0), (33, 40, 17, 0.0)]):
        w = wl.small_random(500 + si, N, 3, M, q_min=q_min, q_max=q_min * M if q_min else 0.6, box=10.0 + N ** (1 / 3) * 3)
        ff = _peratom_ff(w, 600 + si)
        xyz = (w.xyz[None] + rng.normal(0, 0.7, (B,) + w.xyz.shape)).astype(np.float32)
        hint = db.q_hint(w.q)
        x, f, q = (torch.from_numpy(a_).cuda() for a_ in (xyz, ff, w.q))
        Ib = db.debye_profile_peratom_batch(x, f, q, hint=hint).cpu().numpy()
        assert Ib.shape == (B, M)
        assert Ib.tobytes() == db.debye_profile_peratom_batch(x, f, q, hint=hint).cpu().numpy().tobytes()          # run to run
        for b in range(B):
            ref = orc.debye_peratom(xyz[b], ff, w.q)
            assert rel(Ib[b], ref) <= TOL32, (B, N, M, b, rel(Ib[b], ref))
            one = db.debye_profile_peratom(x[b].contiguous(), f, q, hint=hint).cpu().numpy()
            assert rel(Ib[b], one) <= 1e-6                                                                        # same terms, other CTA ranges
        if si == 0:      # no hint, MUFU and FP64: conformer by conformer, bit for bit the single-structure call
            for kw in (dict(), dict(variant="mufu"), dict(variant="fp64")):
                I2 = db.debye_profile_peratom_batch(x, f, q, **kw).cpu().numpy()
                for b in range(B):
                    assert I2[b].tobytes() == db.debye_profile_peratom(x[b].contiguous(), f, q, **kw).cpu().numpy().tobytes()
            wrong = (1 << 8) | (1 << 9) | (1 << 11)          # "q_k = (k + 1) dq" promised for a grid that starts at 0
            assert np.isnan(db.debye_profile_peratom_batch(x, f, q, hint=wrong).cpu().numpy()).all()
    with pytest.raises(db.LibdebyeError):
        db.debye_profile_peratom_batch(x[:0], f, q)


def test_peratom_degenerate_inputs(db):
    import torch
    q = np.array([0.0, 0.05, 0.4, 1.3], dtype=np.float32)
    dq = torch.from_numpy(q).cuda()
    # one atom: I = f^2; two atoms: closed form; coincident atoms: sinc(0) = 1; a very close pair (accurate small-x path)
    one = np.array([[1.0, 2.0, 3.0]], dtype=np.float32); f1 = np.array([[2.0, 1.5, -1.0, 0.5]], dtype=np.float32)
    I = db.debye_profile_peratom(torch.from_numpy(one).cuda(), torch.from_numpy(f1).cuda(), dq).cpu().numpy()
    assert np.allclose(I, f1[0].astype(np.float64) ** 2, rtol=1e-15)
    for d in (0.0, 1e-4, 0.01, 3.7, 250.0):
        xyz = np.array([[0.5, 0.5, 0.5], [0.5, 0.5, 0.5 + d]], dtype=np.float32)
        dd = float(np.float64(xyz[1, 2]) - np.float64(xyz[0, 2]))
        ff = np.array([[6.0, 5.9, 4.0, 1.5], [-1.5, -1.4, -1.0, -0.3]], dtype=np.float32)
        qq = q.astype(np.float64)
        s = np.where(qq * dd == 0, 1.0, np.sin(qq * dd) / np.where(qq * dd == 0, 1.0, qq * dd))
        want = ff[0].astype(np.float64) ** 2 + ff[1].astype(np.float64) ** 2 + 2 * ff[0].astype(np.float64) * ff[1] * s
        for variant, tol in (("auto", 2e-6), ("fp64", 1e-12)):
            I = db.debye_profile_peratom(torch.from_numpy(xyz).cuda(), torch.from_numpy(ff).cuda(), dq, variant=variant).cpu().numpy()
            assert rel(I, want) <= tol, (d, variant, I, want)
    # q = 0 only; M = 1
    w = wl.small_random(97, 300, 3, 5)
    ff = _peratom_ff(w, 97)[:, :1].copy()
    I = db.debye_profile_peratom(torch.from_numpy(w.xyz).cuda(), torch.from_numpy(ff).cuda(), torch.zeros(1, device="cuda")).cpu().numpy()
    assert abs(I[0] - ff.astype(np.float64).sum() ** 2) <= 1e-12 * I[0]
    # bad flags are rejected before anything is launched
    with pytest.raises(db.LibdebyeError):
        db.debye_profile_peratom(torch.from_numpy(w.xyz).cuda(), torch.from_numpy(ff).cuda(), torch.zeros(1, device="cuda"), variant="recur")
    # caller-owned workspace (include/debye.h: at most 1.3 MB + 1 KB x M): same bits; too small a workspace is refused; and the
    # sharded and unsharded per-type calls run from the same caller workspace
    w = wl.small_random(98, 900, 3, 45)
    ff = _peratom_ff(w, 98)
    x, t, f, q = to_dev(w)
    fd = torch.from_numpy(ff).cuda()
    ref = db.debye_profile_peratom(x, fd, q).cpu().numpy()
    part_ref = db.debye_partials_shard(x, t, q, w.T, 1, 2)[0].cpu().numpy()
    L = db.lib()
    need = max(1400000 + 1024 * w.M, L.debye_workspace_bytes(w.N, 1, w.T, w.M, 0))
    buf = torch.empty(need + 256, dtype=torch.uint8, device="cuda")
    ptr = (buf.data_ptr() + 255) // 256 * 256
    assert L.debye_set_workspace(ptr, need) == 0
    try:
        assert db.debye_profile_peratom(x, fd, q).cpu().numpy().tobytes() == ref.tobytes()
        assert db.debye_partials_shard(x, t, q, w.T, 1, 2)[0].cpu().numpy().tobytes() == part_ref.tobytes()
        assert L.debye_set_workspace(ptr, 1024) == 0
        with pytest.raises(db.LibdebyeError):
            db.debye_profile_peratom(x, fd, q)
    finally:
        assert L.debye_set_workspace(None, 0) == 0
    assert db.debye_profile_peratom(x, fd, q).cpu().numpy().tobytes() == ref.tobytes()
