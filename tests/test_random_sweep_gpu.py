"""Seeded random sweep: shapes, q grids and entry points drawn at random, every result compared element by element with the
CPU oracle (Eq. (2)).  The fixed cases of test_parity_gpu.py are chosen by hand around the tile, chunk and piece
boundaries; this sweep covers the combinations nobody thought of.  Tolerances as there (north_star): 1e-4 FP32, 1e-10 FP64,
relative to max(|I|, 1e-2 sum|terms|) (signed form factors: I may come close to 0)."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_1306_2258_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL32, TOL64 = 1e-4, 1e-10
GRID_KINDS = ["zero", "dq", "general", "pieces", "random", "descending", "repeat"]


@pytest.fixture(scope="module")
def db():
    from paper_1306_2258_b200 import binding
    binding.lib()
    return binding


def make_grid(kind, M, rng):
    """An input recipe only (none of the method's arithmetic): the kinds of q grid the library distinguishes."""
    k = np.arange(M, dtype=np.float64)
    if kind == "zero":                       # q_k = k dq
        return k * rng.uniform(0.002, 0.02)
    if kind == "dq":                         # q_k = (k + 1) dq: the paper's own grid
        return (k + 1) * rng.uniform(0.002, 0.02)
    if kind == "general":                    # uniform, arbitrary start
        return rng.uniform(0.05, 0.5) + k * rng.uniform(0.001, 0.01)
    if kind == "pieces":                     # 2..4 uniform pieces with their own steps
        cuts = np.sort(rng.choice(np.arange(1, M), size=min(int(rng.integers(1, 4)), M - 1), replace=False)) if M > 1 else []
        q, start, prev = [], rng.uniform(0.0, 0.1), 0
        for c in list(cuts) + [M]:
            q += list(start + np.arange(c - prev) * rng.uniform(0.001, 0.01))
            start, prev = q[-1] + rng.uniform(0.02, 0.1), c
        return np.array(q)
    if kind == "random":
        return np.sort(rng.uniform(0.0, 1.0, M))
    if kind == "descending":
        return (k[::-1] + rng.integers(0, 2)) * rng.uniform(0.002, 0.02)
    q = np.sort(rng.uniform(0.0, 0.8, M))    # "repeat": repeated q values
    q[M // 2:] = q[: M - M // 2]
    return q


def err(I, ref, A):
    return float(np.max(np.abs(np.asarray(I) - ref) / np.maximum(np.abs(ref), 1e-2 * A)))


def draw_case(seed):
    rng = np.random.default_rng(0xD0E5 + seed)
    N = int(rng.choice([1, 2, 3, 31, 33, 127, 128, 129, 255, 257, 400, 777, 1025])) if rng.random() < 0.5 else int(rng.integers(1, 1300))
    T = int(rng.choice([1, 2, 3, 5, 8, 9, 20, 32]))
    M = int(rng.choice([1, 2, 7, 8, 9, 16, 24, 51, 64, 100, 101, 127, 128, 129, 130, 200, 256, 257, 258, 300, 513]))
    kind = GRID_KINDS[int(rng.integers(0, len(GRID_KINDS)))]
    box = float(rng.choice([0.5, 5.0, 25.0, 80.0, 400.0, 4000.0]))
    w = wl.small_random(int(rng.integers(1, 1 << 30)), N, T, M, box=box, signed=bool(rng.random() < 0.3))
    xyz = w.xyz.copy()
    if rng.random() < 0.3 and N > 10:        # coincident and nearly coincident atoms (sinc -> 1, PAPER.md:41 reading R2)
        k = int(rng.integers(1, N // 2))
        xyz[:k] = xyz[N - k:]
        xyz[k:2 * k] = xyz[N - 2 * k:N - k] + np.float32(1e-4)
    w = wl.with_grid(w, make_grid(kind, M, rng).astype(np.float32), f"sweep{seed}")
    return rng, w, xyz, f"seed {seed}: N={N} T={T} M={M} grid={kind} box={box}"


@pytest.mark.parametrize("seed", range(24))
def test_random_case_against_the_oracle_through_every_entry(db, seed):
    import torch
    rng, w, xyz, desc = draw_case(seed)
    N, T, M = w.N, w.T, w.M
    ref, A = orc.debye_sym(xyz, w.type, w.fftab, w.q, return_abs=True)
    x, t, f, q = (torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (xyz, w.type, w.fftab, w.q))
    res = {"auto": db.debye_profile(x, t, f, q), "mufu": db.debye_profile(x, t, f, q, variant="mufu")}
    h = db.q_hint(w.q)
    if h:
        res["hint"] = db.debye_profile(x, t, f, q, hint=h)
    hp = db.q_hint_pieces(w.q)
    if hp:
        res["pieces hint"] = db.debye_profile(x, t, f, q, hint=hp)
    res["host entry"] = db.debye_profile_host(xyz, w.type, w.fftab, w.q)
    plan = db.Plan(t, q, T)
    res["plan"] = plan.execute(x, f)
    # tile split over 3 ranks, run one after the other on this GPU (no kernel waits on another): parts summed in rank order
    parts = []
    for r in range(3):
        S, n = db.debye_partials_shard(x, t, q, T, r, 3, hint=h or 0)
        parts.append(S)
    res["tile split"] = db.debye_profile_from_partials(torch.stack(parts), n, f)[0]
    lim = db.static_limits()
    if h and not (h & db.QHINT_PIECES) and N <= lim[0] and T <= lim[1] and M <= lim[2] + 1:
        try:
            res["static"] = db.debye_profile_static(x, t, f, q, torch.empty(M, dtype=torch.float64, device="cuda"), h)
        except db.LibdebyeError as e:       # beyond its limits (e.g. M non-zero q values): refused, never wrong
            assert e.code in (db.DEBYE_EUNSUPPORTED, db.DEBYE_EINVAL), desc
    torch.cuda.synchronize()
    plan.destroy()
    for name, I in res.items():
        I = I.cpu().numpy() if hasattr(I, "cpu") else I
        e = err(I, ref, A)
        assert e <= TOL32, (desc, name, e)
    if seed % 4 == 0:
        e = err(db.debye_profile(x, t, f, q, variant="fp64").cpu().numpy(), ref, A)
        assert e <= TOL64, (desc, "fp64", e)
    if seed % 3 == 0:                        # per-atom weights (reading R10w)
        wt = rng.uniform(0.5, 1.5, N).astype(np.float32)
        refw, Aw = orc.debye_sym(xyz, w.type, w.fftab, w.q, weight=wt, return_abs=True)
        e = err(db.debye_profile_weighted(x, t, torch.from_numpy(wt).cuda(), f, q).cpu().numpy(), refw, Aw)
        assert e <= TOL32, (desc, "weighted", e)
    if M <= 258 and N <= 700:                # per-atom table, two conformers sharing it
        ff = wl.peratom_table(w, seed=seed)
        xb = np.stack([xyz, xyz * np.float32(0.9)])
        Ib = db.debye_profile_peratom_batch(torch.from_numpy(xb).cuda(), torch.from_numpy(ff).cuda(), q, hint=h or 0).cpu().numpy()
        I1 = db.debye_profile_peratom(x, torch.from_numpy(ff).cuda(), q).cpu().numpy()
        for b in range(2):
            rp, Ap = orc.debye_peratom(xb[b], ff, w.q, return_abs=True)
            assert err(Ib[b], rp, Ap) <= TOL32, (desc, "per-atom batch", b)
            if b == 0:
                assert err(I1, rp, Ap) <= TOL32, (desc, "per-atom")
