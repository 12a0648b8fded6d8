"""Pins for the CPU oracle (oracle/debye_oracle.c): everything here is fixed by the paper's equations or by
mathematics, not by the oracle itself.  CPU only.

PAPER.md:37-39 (Eq. 1), PAPER.md:41-42 (Eq. 2), PAPER.md:88 ("only j <= k").  The paper prints no I(q)
value (Figs 6-7 are images), so there is no numeric fixture to quote; the pins are closed forms, the
definition Eq. (1) by brute-force quadrature, invariances and identities -- chosen so that a dropped self
term, a missing factor 2, a wrong sign, a transposed fftab or a wrong q index fails at least one."""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from paper_1306_2258_b200 import workloads as wl

RT = 1e-12


def rel(a, b):
    return np.max(np.abs(np.asarray(a) - np.asarray(b)) / np.abs(np.asarray(b)))


def test_two_atom_closed_form():
    # I(q) = f1^2 + f2^2 + 2 f1 f2 sin(qd)/(qd)   (north_star; from Eq. 2)
    d = 3.7
    xyz = np.array([[0.25, -1.0, 2.0], [0.25, -1.0, 2.0 + d]], dtype=np.float32)
    dd = float(np.float64(xyz[1, 2]) - np.float64(xyz[0, 2]))
    q = np.array([0.0, 0.013, 0.2, 0.5, 1.0, 3.0], dtype=np.float32)
    f = np.array([[6.0, 5.9, 5.0, 3.5, 2.0, 1.1], [-1.5, -1.5, -1.4, -1.0, -0.7, -0.2]], dtype=np.float32)
    typ = np.array([0, 1], dtype=np.int32)
    qq = q.astype(np.float64)
    s = np.where(qq == 0, 1.0, np.sin(qq * dd) / np.where(qq == 0, 1.0, qq * dd))
    f1, f2 = f[0].astype(np.float64), f[1].astype(np.float64)
    want = f1 ** 2 + f2 ** 2 + 2 * f1 * f2 * s
    assert rel(orc.debye_full(xyz, typ, f, q), want) < RT
    assert rel(orc.debye_sym(xyz, typ, f, q), want) < RT
    # a transposed fftab or swapped types must change the answer (guards the indexing)
    assert rel(orc.debye_full(xyz, typ[::-1].copy(), f, q), want) < RT   # symmetric under swapping both atoms


def test_I0_is_square_of_sum():
    w = wl.small_random(1, 300, 4, 5, signed=True)
    I = orc.debye_full(w.xyz, w.type, w.fftab, w.q)
    tot = w.fftab.astype(np.float64)[w.type, 0].sum()
    assert w.q[0] == 0.0
    assert abs(I[0] - tot ** 2) / tot ** 2 < RT


@pytest.mark.parametrize("seed", [0, 1])
def test_eq1_orientational_average_equals_eq2(seed):
    # Eq. (2) is the exact orientational average of Eq. (1).
    rng = np.random.default_rng(100 + seed)
    N = 20
    x = rng.uniform(-12, 12, (N, 3)).astype(np.float32)
    typ = rng.integers(0, 3, N).astype(np.int32)
    q = np.array([0.05, 0.31, 0.77, 1.0], dtype=np.float32)
    f = rng.uniform(-2, 7, (3, 4)).astype(np.float32)
    I2 = orc.debye_full(x, typ, f, q)
    for m, qq in enumerate(q):
        I1 = orc.eq1_quadrature(x.astype(np.float64), f.astype(np.float64)[typ, m], float(qq))
        assert abs(I1 - I2[m]) / abs(I2[m]) < 1e-11, (m, I1, I2[m])


def test_full_equals_sym_and_row_slabs_add_up():
    w = wl.small_random(2, 257, 5, 9, signed=True)
    If, Af = orc.debye_full(w.xyz, w.type, w.fftab, w.q, return_abs=True)
    Is, As = orc.debye_sym(w.xyz, w.type, w.fftab, w.q, return_abs=True)
    assert rel(Is, If) < 1e-13 and rel(As, Af) < 1e-13
    a = orc.debye_sym(w.xyz, w.type, w.fftab, w.q, rows=(0, 100))
    b = orc.debye_sym(w.xyz, w.type, w.fftab, w.q, rows=(100, 257), threads=3)
    assert rel(a + b, If) < 1e-13
    assert (Af >= np.abs(If)).all()


def test_polyhedra_and_coincident():
    q = np.array([0.0, 0.1, 0.9, 2.5], dtype=np.float32)
    qq = q.astype(np.float64)
    f = np.array([[2.0, 1.9, 1.5, 0.6]], dtype=np.float32)
    ff = f[0].astype(np.float64)
    d = 2.0
    sinc = lambda u: np.where(u == 0, 1.0, np.sin(u) / np.where(u == 0, 1.0, u))
    tri = np.array([[0, 0, 0], [d, 0, 0], [d / 2, d * math.sqrt(3) / 2, 0]], dtype=np.float64)
    # regular tetrahedron with edge 2*sqrt(2)*s from alternating cube corners (exact in fp32 for s=1)
    tet = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=np.float64)
    dt = 2 * math.sqrt(2)
    I = orc.debye_full(tet.astype(np.float32), np.zeros(4, np.int32), f, q)
    assert rel(I, 4 * ff ** 2 + 12 * ff ** 2 * sinc(qq * dt)) < RT
    x3 = tri.astype(np.float32)
    d01 = np.linalg.norm(x3[0].astype(np.float64) - x3[1]); d02 = np.linalg.norm(x3[0].astype(np.float64) - x3[2])
    d12 = np.linalg.norm(x3[1].astype(np.float64) - x3[2])
    I = orc.debye_full(x3, np.zeros(3, np.int32), f, q)
    assert rel(I, 3 * ff ** 2 + 2 * ff ** 2 * (sinc(qq * d01) + sinc(qq * d02) + sinc(qq * d12))) < RT
    # all atoms coincident: I = (sum f)^2 for every q (reading R2: sinc(0) = 1)
    xc = np.tile(np.array([[1.5, -2.0, 0.25]], dtype=np.float32), (7, 1))
    f2 = np.array([[2.0, 1.9, 1.5, 0.6], [-1.0, -0.5, 0.25, 3.0]], dtype=np.float32)
    typ = np.array([0, 1, 0, 0, 1, 1, 0], dtype=np.int32)
    tot = f2.astype(np.float64)[typ].sum(axis=0)
    assert rel(orc.debye_sym(xc, typ, f2, q), tot ** 2) < RT


def test_chain_closed_form():
    n, d = 400, 1.5
    xyz = np.zeros((n, 3), dtype=np.float32); xyz[:, 1] = np.arange(n) * d       # exact in fp32
    q = wl.q_grid(0.8, 17)
    I = orc.debye_sym(xyz, np.zeros(n, np.int32), np.ones((1, 17), np.float32), q)
    assert rel(I, orc.chain_closed_form(n, d, q.astype(np.float64))) < 1e-11


def test_lattice_closed_forms():
    w = wl.cubic_lattice(6, 5, 7, 2.5, 9, 0.7)
    I = orc.debye_sym(w.xyz, w.type, w.fftab, w.q)
    assert rel(I, orc.lattice_closed_form(6, 5, 7, 2.5, w.q.astype(np.float64))) < 1e-11
    w2 = wl.cubic_lattice(5, 6, 4, 2.0, 7, 0.9, T=2)
    I2 = orc.debye_full(w2.xyz, w2.type, w2.fftab, w2.q)
    assert rel(I2, orc.lattice_closed_form(5, 6, 4, 2.0, w2.q.astype(np.float64), fa=1.0, fb=2.0)) < 1e-11


def test_low_q_expansion():
    # I(q) = I(0) - q^2/6 S2 + O(q^4), S2 = sum_ij f_i f_j r_ij^2 = 2 [F sum f_i |x_i|^2 - |sum f_i x_i|^2]
    w = wl.small_random(3, 500, 3, 2, q_max=1e-3)
    x = w.xyz.astype(np.float64); f = w.fftab.astype(np.float64)[w.type, 1]
    F = f.sum()
    S2 = 2 * (F * (f * (x ** 2).sum(1)).sum() - ((f[:, None] * x).sum(0) ** 2).sum())
    I = orc.debye_sym(w.xyz, w.type, w.fftab, w.q)
    qq = float(w.q[1])
    lead = F ** 2 - qq ** 2 / 6 * S2
    assert abs(I[1] - lead) / (qq ** 2 / 6 * S2) < 1e-3        # remainder is O(q^4)
    assert I[1] < F ** 2


def test_invariances():
    w = wl.small_random(4, 200, 4, 6, signed=True)
    I = orc.debye_sym(w.xyz, w.type, w.fftab, w.q)
    rng = np.random.default_rng(5)
    perm = rng.permutation(w.N)
    assert rel(orc.debye_sym(w.xyz[perm], w.type[perm], w.fftab, w.q), I) < 1e-12
    # transforms exact in fp32: axis swap, sign flip, power-of-two translation on a coarse grid
    assert rel(orc.debye_sym(w.xyz[:, [2, 0, 1]] * np.float32(-1), w.type, w.fftab, w.q), I) < 1e-12
    xg = np.round(w.xyz * 64) / 64
    Ig = orc.debye_sym(xg.astype(np.float32), w.type, w.fftab, w.q)
    assert rel(orc.debye_sym((xg + 32.0).astype(np.float32), w.type, w.fftab, w.q), Ig) < 1e-12
    # general rotation + translation, applied in double and rounded once: agreement to fp32 input rounding
    A = rng.normal(size=(3, 3)); Q, _ = np.linalg.qr(A)
    xr = (w.xyz.astype(np.float64) @ Q.T + np.array([3.0, -7.0, 11.0])).astype(np.float32)
    assert rel(orc.debye_sym(xr, w.type, w.fftab, w.q), I) < 2e-5


def test_scaling_identities_and_bound():
    w = wl.small_random(6, 150, 3, 5)
    I = orc.debye_sym(w.xyz, w.type, w.fftab, w.q)
    assert (I >= 0).all()
    assert rel(orc.debye_sym(w.xyz, w.type, w.fftab * np.float32(2.0), w.q), 4 * I) < 1e-13    # I(alpha f) = alpha^2 I
    # I(q; s x) = I(s q; x) with s = 2 (exact in fp32)
    assert rel(orc.debye_sym(w.xyz * np.float32(2), w.type, w.fftab, w.q),
               orc.debye_sym(w.xyz, w.type, w.fftab, w.q * np.float32(2))) < 1e-13
    # |I - sum f^2| <= 2 sum_{i<j} |f_i f_j| / (q r_ij)
    x = w.xyz.astype(np.float64); r = np.sqrt(((x[:, None] - x[None]) ** 2).sum(-1))
    iu = np.triu_indices(w.N, 1)
    for m in range(1, w.M):
        f = w.fftab.astype(np.float64)[w.type, m]
        bound = 2 * (np.abs(f[iu[0]] * f[iu[1]]) / (float(w.q[m]) * r[iu])).sum()
        assert abs(I[m] - (f ** 2).sum()) <= bound


def test_workloads_are_reproducible_and_shaped():
    a, b = wl.cfg1(), wl.cfg1()
    assert a.xyz.tobytes() == b.xyz.tobytes() and a.type.tobytes() == b.type.tobytes()
    x = a.xyz.astype(np.float64)
    r = np.sqrt(((x[:, None] - x[None]) ** 2).sum(-1)) + 1e9 * np.eye(a.N)
    assert r.min() >= 1.2 - 1e-5 and np.linalg.norm(x, axis=1).max() <= 15.0 + 1e-4
    assert a.q[0] == 0 and abs(a.q[-1] - 0.5) < 1e-7 and a.M == 51 and a.T == 5
    w3 = wl.cfg3(n_bp=200)
    assert w3.N == 8000 and w3.T == 4 and w3.M == 200
    assert [int((w3.type == t).sum()) for t in range(4)] == [400, 2400, 3600, 1600]


def test_weighted_oracle_pins():
    """Per-atom weights (reading R10w: f_j(q) = w_j F[t_j](q)).  Pins that do not go through the
    weighted code path: closed forms, and identities against the UNWEIGHTED oracle on transformed inputs."""
    rng = np.random.default_rng(5)
    q = wl.q_grid(0.9, 13)
    f = wl.gaussian_form_factors(3, 3, q)
    # (1) two atoms: I = w1^2 f1^2 + w2^2 f2^2 + 2 w1 w2 f1 f2 sin(qd)/(qd)
    d = 3.25
    xyz = np.array([[0, 0, 0], [0, d, 0]], np.float32)
    typ = np.array([0, 2], np.int32)
    w = np.array([1.5, -0.75], np.float32)                     # contrast may be negative
    qq, F = q.astype(np.float64), f.astype(np.float64)
    s = np.where(qq == 0, 1.0, np.sin(qq * d) / np.where(qq == 0, 1.0, qq * d))
    want = (1.5 * F[0]) ** 2 + (0.75 * F[2]) ** 2 + 2 * 1.5 * (-0.75) * F[0] * F[2] * s
    assert np.max(np.abs(orc.debye_sym(xyz, typ, f, q, weight=w) - want)) <= 1e-12 * np.max(np.abs(want))
    assert np.max(np.abs(orc.debye_full(xyz, typ, f, q, weight=w) - want)) <= 1e-12 * np.max(np.abs(want))
    # (2) weight 1 is the unweighted oracle, bit for bit; full == sym with weights
    N = 40
    xyz = (rng.uniform(-8, 8, (N, 3))).astype(np.float32)
    typ = rng.integers(0, 3, N).astype(np.int32)
    assert np.array_equal(orc.debye_sym(xyz, typ, f, q, weight=np.ones(N, np.float32)), orc.debye_sym(xyz, typ, f, q))
    w = rng.uniform(0.25, 3.0, N).astype(np.float32)
    assert rel(orc.debye_sym(xyz, typ, f, q, weight=w), orc.debye_full(xyz, typ, f, q, weight=w)) <= 1e-13
    # (3) an atom of integer weight n is n coincident atoms of weight 1 (sinc(0) = 1 between the copies)
    wi = rng.integers(1, 4, N)
    dup = np.repeat(np.arange(N), wi)
    assert rel(orc.debye_sym(xyz, typ, f, q, weight=wi.astype(np.float32)), orc.debye_sym(xyz[dup], typ[dup], f, q)) <= 1e-12
    # (4) one weight per type is a rescaled form-factor table
    c = np.array([0.5, 2.0, 1.25], np.float32)                  # exactly representable, products exact in fp32
    assert rel(orc.debye_sym(xyz, typ, f, q, weight=c[typ]), orc.debye_sym(xyz, typ, (f * c[:, None]).astype(np.float32), q)) <= 1e-6
    # (5) I(0) = (sum_j w_j f_j(0))^2
    I = orc.debye_sym(xyz, typ, f, q, weight=w)
    assert abs(I[0] - (w.astype(np.float64) * F[typ, 0]).sum() ** 2) <= 1e-12 * I[0]


def test_peratom_oracle_pins():
    """oracle_debye_peratom (reading R10p: one form-factor row per ATOM) against what the paper and the
    mathematics fix: the two-atom closed form with two different atoms, I(0) = (sum_j f_j(0))^2, Eq. (1) by spherical
    quadrature with a different form factor on every atom, the reduction to the per-type oracle when the rows are copies
    of a type table, separability (f_j(q) = w_j g(q) gives g^2 times the profile of point scatterers w_j), the triangle
    closed form, invariance under a permutation that moves the rows with the atoms, full == sym."""
    rng = np.random.default_rng(77)
    # two atoms, different per-atom rows, one negative
    d = 4.3
    xyz = np.array([[1.0, 2.0, -0.5], [1.0, 2.0 + d, -0.5]], dtype=np.float32)
    dd = float(np.float64(xyz[1, 1]) - np.float64(xyz[0, 1]))
    q = np.array([0.0, 0.02, 0.3, 0.9, 2.5], dtype=np.float32)
    ff = np.array([[7.0, 6.9, 5.5, 3.0, 1.0], [-2.0, -1.9, -1.5, -0.8, -0.1]], dtype=np.float32)
    qq = q.astype(np.float64)
    s = np.where(qq == 0, 1.0, np.sin(qq * dd) / np.where(qq == 0, 1.0, qq * dd))
    f1, f2 = ff[0].astype(np.float64), ff[1].astype(np.float64)
    want = f1 ** 2 + f2 ** 2 + 2 * f1 * f2 * s
    for sym in (False, True):
        assert rel(orc.debye_peratom(xyz, ff, q, sym=sym), want) < RT
    # a transposed table read (ff[m][j] instead of ff[j][m]) or a shifted q index would fail the next three
    N, M = 18, 4
    x = rng.uniform(-10, 10, (N, 3)).astype(np.float32)
    q = np.array([0.0, 0.21, 0.6, 1.1], dtype=np.float32)
    ff = rng.uniform(-1, 6, (N, M)).astype(np.float32)
    I = orc.debye_peratom(x, ff, q)
    assert rel(I, orc.debye_peratom(x, ff, q, sym=False)) < RT
    assert abs(I[0] - ff[:, 0].astype(np.float64).sum() ** 2) < RT * I[0]                 # I(0) = (sum f)^2
    for m in range(1, M):                                                                   # Eq. (1)
        I1 = orc.eq1_quadrature(x.astype(np.float64), ff[:, m].astype(np.float64), float(q[m]))
        assert abs(I1 - I[m]) <= 1e-9 * abs(I[m])
    perm = rng.permutation(N)
    assert rel(orc.debye_peratom(x[perm], ff[perm], q), I) < 1e-11
    # rows copied from a type table: the per-type oracle (R10)
    w = wl.small_random(78, 150, 4, 9, signed=True)
    assert rel(orc.debye_peratom(w.xyz, w.fftab[w.type], w.q), orc.debye_sym(w.xyz, w.type, w.fftab, w.q)) < RT
    # ... times a per-atom weight: the weighted oracle (R10w)
    wt = rng.uniform(0.3, 1.7, w.N).astype(np.float32)
    ffw = (w.fftab[w.type].astype(np.float64) * wt[:, None].astype(np.float64))
    ffw32 = ffw.astype(np.float32)
    if np.array_equal(ffw32.astype(np.float64), ffw):      # only exact products are comparable bit for bit; else loosen
        tolw = RT
    else:
        tolw = 1e-6
    assert rel(orc.debye_peratom(w.xyz, ffw32, w.q), orc.debye_sym(w.xyz, w.type, w.fftab, w.q, weight=wt)) < tolw
    # separable rows f_j(q) = c_j g(q), c_j small integers and g powers of two (products exact in float32)
    c = rng.integers(-3, 5, N).astype(np.float32)
    g = np.array([2.0, 1.0, 0.5, 0.25], dtype=np.float32)
    ones = np.ones((1, M), dtype=np.float32)
    pts = orc.debye_sym(x, np.zeros(N, np.int32), ones, q, weight=c)
    assert rel(orc.debye_peratom(x, c[:, None] * g[None, :], q), g.astype(np.float64) ** 2 * pts) < 1e-11
    # equilateral triangle, three different atoms: I = sum f^2 + 2 (f1 f2 + f1 f3 + f2 f3) sinc(q a)
    a = 2.0
    tri = np.array([[0, 0, 0], [a, 0, 0], [a / 2, a * math.sqrt(3) / 2, 0]], dtype=np.float32)
    ft = np.array([[3.0], [5.0], [-2.0]], dtype=np.float32)
    qa = np.array([0.7], dtype=np.float32)
    dists = [np.linalg.norm(tri[i].astype(np.float64) - tri[j].astype(np.float64)) for i, j in ((0, 1), (0, 2), (1, 2))]
    sincs = [math.sin(float(qa[0]) * dd_) / (float(qa[0]) * dd_) for dd_ in dists]
    want = 9 + 25 + 4 + 2 * (15 * sincs[0] - 6 * sincs[1] - 10 * sincs[2])
    assert abs(orc.debye_peratom(tri, ft, qa)[0] - want) < 1e-12 * abs(want)
