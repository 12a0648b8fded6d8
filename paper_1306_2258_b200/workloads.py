"""Seeded synthetic workloads shaped like the paper's (§III: "randomly generated
proteins", 50 q on (0,1]; Figs 6-7: lysozyme / DNA-like elongated structures) and BASELINE.json's five
configs.  Shared by the oracle-side tests and the CUDA-side tests / bench.

This module holds NONE of the method's arithmetic (no distances, no sinc, no sums): it only draws
coordinates, type labels, form-factor tables and q grids.  The form-factor *table* is an input of the
method (SURVEY.md §8(c) reading 9), so filling it with seeded 4-Gaussian values is input generation.

PRNG: SplitMix64 used as a counter-based generator (output n depends only on (seed, n)), so every stream
is reproducible and vectorisable.  All geometry is drawn in float64 and rounded ONCE to float32; both the
oracle and libdebye receive the same float32/int32 bytes.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
BASE_SEED = 1306225800


class Stream:
    """SplitMix64 stream: u64 #n = mix(seed + (n+1)*gamma).  `uniform(n)` consumes n outputs."""

    def __init__(self, seed: int):
        self.seed = np.uint64(seed & 0xFFFFFFFFFFFFFFFF)
        self.pos = 0

    def bits(self, n: int) -> np.ndarray:
        idx = np.arange(self.pos + 1, self.pos + n + 1, dtype=np.uint64)
        self.pos += n
        with np.errstate(over="ignore"):
            z = self.seed + idx * _GAMMA
            z = (z ^ (z >> np.uint64(30))) * _M1
            z = (z ^ (z >> np.uint64(27))) * _M2
            z = z ^ (z >> np.uint64(31))
        return z

    def uniform(self, n: int) -> np.ndarray:
        return (self.bits(n) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)

    def normal(self, n: int) -> np.ndarray:
        """Box-Muller, cosine branch, two uniforms per normal."""
        u = self.uniform(2 * n).reshape(n, 2)
        return np.sqrt(-2.0 * np.log(1.0 - u[:, 0])) * np.cos(2.0 * math.pi * u[:, 1])

    def unit_vectors(self, n: int) -> np.ndarray:
        u = self.uniform(2 * n).reshape(n, 2)
        z = 2.0 * u[:, 0] - 1.0
        phi = 2.0 * math.pi * u[:, 1]
        s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
        return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


@dataclass
class Workload:
    name: str
    xyz: np.ndarray            # float32 [N,3] or [B,N,3]
    type: np.ndarray           # int32 [N]
    fftab: np.ndarray          # float32 [T,M]
    q: np.ndarray              # float32 [M]
    meta: dict = field(default_factory=dict)

    @property
    def N(self): return int(self.type.shape[0])
    @property
    def T(self): return int(self.fftab.shape[0])
    @property
    def M(self): return int(self.q.shape[0])
    @property
    def B(self): return int(self.xyz.shape[0]) if self.xyz.ndim == 3 else 1
    @property
    def pairs(self): return self.N * (self.N - 1) // 2
    @property
    def pair_q(self): return self.pairs * self.M * self.B


# ----------------------------------------------------------------------------------------------------
# pieces
# ----------------------------------------------------------------------------------------------------
def q_grid(q_max: float, M: int, q_min: float = 0.0) -> np.ndarray:
    """M points uniform on [q_min, q_max], both ends included; float32(q_min + (q_max-q_min) k/(M-1))."""
    if M == 1:
        return np.array([q_max], dtype=np.float32)
    k = np.arange(M, dtype=np.float64)
    return (q_min + (q_max - q_min) * k / (M - 1)).astype(np.float32)


def gaussian_form_factors(seed: int, T: int, q: np.ndarray, n_gauss: int = 4,
                          a=(0.5, 6.0), b=(0.5, 40.0), c=(0.0, 1.0)) -> np.ndarray:
    """f_t(q) = sum_g a_tg exp(-b_tg (q/4pi)^2) + c_t with seeded coefficients (BASELINE.json configs[0]);
    no published table is reproduced."""
    s = Stream(seed)
    A = a[0] + (a[1] - a[0]) * s.uniform(T * n_gauss).reshape(T, n_gauss)
    Bc = b[0] + (b[1] - b[0]) * s.uniform(T * n_gauss).reshape(T, n_gauss)
    C = c[0] + (c[1] - c[0]) * s.uniform(T)
    x = (q.astype(np.float64) / (4.0 * math.pi)) ** 2
    f = (A[:, :, None] * np.exp(-Bc[:, :, None] * x[None, None, :])).sum(axis=1) + C[:, None]
    return f.astype(np.float32)


def types_from_cdf(seed: int, N: int, cdf) -> np.ndarray:
    u = Stream(seed).uniform(N)
    return np.searchsorted(np.asarray(cdf, dtype=np.float64), u, side="right").astype(np.int32).clip(0, len(cdf) - 1)


_PROTEIN_CDF = (0.50, 0.65, 0.85, 0.86, 1.00)   # C, N, O, S, H  (BASELINE.json configs[0])


def sphere_min_spacing(seed: int, N: int, radius: float, dmin: float) -> np.ndarray:
    """Uniform points in a ball with sequential rejection at minimum spacing dmin."""
    s = Stream(seed)
    out = np.empty((N, 3))
    n = 0
    while n < N:
        cand = (2.0 * s.uniform(3 * 256).reshape(256, 3) - 1.0) * radius
        for p in cand:
            if p @ p > radius * radius:
                continue
            if n and (((out[:n] - p) ** 2).sum(axis=1) < dmin * dmin).any():
                continue
            out[n] = p
            n += 1
            if n == N:
                break
    return out


def confined_walk(seed: int, steps: int, step_len: float, inside, start) -> np.ndarray:
    """Random walk with fixed step length; a step leaving the region (`inside(p)` False) is redrawn."""
    s = Stream(seed)
    pts = np.empty((steps, 3))
    p = np.asarray(start, dtype=np.float64)
    pts[0] = p
    buf = s.unit_vectors(4096)
    bi = 0
    for m in range(1, steps):
        while True:
            if bi == len(buf):
                buf = s.unit_vectors(4096)
                bi = 0
            cand = p + step_len * buf[bi]
            bi += 1
            if inside(cand):
                break
        p = cand
        pts[m] = p
    return pts


def blob(seed: int, n_backbone: int, radius: float, atoms_per_step: int = 8, jitter: float = 1.5) -> np.ndarray:
    """Globular protein-like blob: 3.8 A random walk confined to a ball, `atoms_per_step` atoms per
    backbone point with Gaussian side-chain jitter (BASELINE.json configs[1])."""
    r2 = radius * radius
    bb = confined_walk(seed, n_backbone, 3.8, lambda p: p @ p <= r2, (0.0, 0.0, 0.0))
    nz = Stream(seed + 1000).normal(n_backbone * atoms_per_step * 3).reshape(n_backbone, atoms_per_step, 3)
    return (bb[:, None, :] + jitter * nz).reshape(-1, 3)


# ----------------------------------------------------------------------------------------------------
# the five BASELINE.json configs (+ extras)
# ----------------------------------------------------------------------------------------------------
def cfg1() -> Workload:
    s = BASE_SEED + 1
    q = q_grid(0.5, 51)
    return Workload("cfg1_sphere_1k", sphere_min_spacing(s, 1000, 15.0, 1.2).astype(np.float32),
                    types_from_cdf(s + 10, 1000, _PROTEIN_CDF), gaussian_form_factors(s + 20, 5, q), q)


def cfg2(N: int = 10000, M: int = 101, q_max: float = 0.5, q_min: float = 0.0, tag: str = "cfg2_globular_10k",
         seed_off: int = 2) -> Workload:
    s = BASE_SEED + seed_off
    q = q_grid(q_max, M, q_min)
    nb = (N + 7) // 8
    radius = 30.0 * (N / 10000.0) ** (1.0 / 3.0)      # constant density when N changes (sweep T)
    xyz = blob(s, nb, radius)[:N]
    return Workload(tag, xyz.astype(np.float32), types_from_cdf(s + 10, N, _PROTEIN_CDF),
                    gaussian_form_factors(s + 20, 5, q), q)


def cfg3(n_bp: int = 1250, tag: str = "cfg3_helix_50k") -> Workload:
    """Straight B-form-like duplex: 10.5 bp/turn, 3.4 A rise, radius 10 A, 20 atoms per nucleotide
    (1 P, 6 O, 9 C, 4 N), Gaussian offsets sigma 0.7 A.  n_bp=1250 -> N=50,000 (length 4247 A);
    n_bp=200 -> N=8,000 (680 A), the literal-length reading of BASELINE.json configs[2]."""
    s = BASE_SEED + 3
    b = np.arange(n_bp, dtype=np.float64)[:, None, None]
    st = np.arange(2, dtype=np.float64)[None, :, None]
    m = np.arange(20, dtype=np.float64)[None, None, :]
    rho = 10.0 - 0.45 * m
    phi = 2.0 * math.pi * b / 10.5 + math.pi * st + 0.1 * m
    pos = np.stack([rho * np.cos(phi), rho * np.sin(phi), 3.4 * b + 0.0 * st + 0.0 * m], axis=-1).reshape(-1, 3)
    pos = pos + 0.7 * Stream(s).normal(pos.shape[0] * 3).reshape(-1, 3)
    tm = np.empty(20, dtype=np.int32)
    tm[0] = 0; tm[1:7] = 1; tm[7:16] = 2; tm[16:20] = 3          # P, O, C, N
    typ = np.tile(tm, n_bp * 2)
    q = q_grid(1.0, 200)
    return Workload(tag, pos.astype(np.float32), typ, gaussian_form_factors(s + 20, 4, q), q)


def cfg4(B: int = 1024, N: int = 2000, tag: str = "cfg4_batch_1024x2k") -> Workload:
    s = BASE_SEED + 4
    base = blob(s, (N + 7) // 8, 17.5)[:N]
    noise = Stream(s + 2000).normal(B * N * 3).reshape(B, N, 3)
    q = q_grid(0.4, 64)
    return Workload(tag, (base[None] + 2.0 * noise).astype(np.float32), types_from_cdf(s + 10, N, _PROTEIN_CDF),
                    gaussian_form_factors(s + 20, 5, q), q)


def cfg5(N: int = 200000, tag: str = "cfg5_coarse_200k") -> Workload:
    s = BASE_SEED + 5
    hi = np.array([150.0, 150.0, 400.0])
    xyz = confined_walk(s, N, 3.8, lambda p: (p >= 0.0).all() and (p <= hi).all(), (75.0, 75.0, 200.0))
    typ = np.minimum((Stream(s + 10).uniform(N) * 20).astype(np.int32), 19)
    q = q_grid(0.3, 128)
    fs = Stream(s + 20)
    a = 20.0 + 90.0 * fs.uniform(20)
    bb = 150.0 + 350.0 * fs.uniform(20)
    x = (q.astype(np.float64) / (4.0 * math.pi)) ** 2
    f = a[:, None] * np.exp(-bb[:, None] * x[None, :])
    return Workload(tag, xyz.astype(np.float32), typ, f.astype(np.float32), q)


def table1(N: int) -> Workload:
    """Workload shaped like the paper's Table I rows: 'random protein' of N atoms,
    50 q uniformly spaced on 0 < q <= 1.0 (q_k = k/50, k=1..50)."""
    w = cfg2(N=N, M=50, q_max=1.0, q_min=0.02, tag=f"table1_N{N}", seed_off=100 + int(round(math.log2(N) * 8)))
    return w


def small_random(seed: int, N: int, T: int, M: int, q_max: float = 0.6, box: float = 25.0, q_min: float = 0.0,
                 signed: bool = False) -> Workload:
    """Uniform points in a cube, i.i.d. uniform types; for parity tests that span tiles and ragged tails."""
    s = Stream(BASE_SEED + 7000 + seed)
    xyz = (s.uniform(N * 3).reshape(N, 3) - 0.5) * box
    typ = np.minimum((s.uniform(N) * T).astype(np.int32), T - 1)
    q = q_grid(q_max, M, q_min)
    f = gaussian_form_factors(BASE_SEED + 8000 + seed, T, q)
    if signed:   # neutron-like scattering lengths may be negative
        sign = np.where(s.uniform(T) < 0.4, -1.0, 1.0).astype(np.float32)
        f = f * sign[:, None]
    return Workload(f"rand_s{seed}_N{N}_T{T}_M{M}", xyz.astype(np.float32), typ, f, q)


def cubic_lattice(nx: int, ny: int, nz: int, a: float, M: int, q_max: float, T: int = 1) -> Workload:
    """Simple cubic lattice, unit form factors (T=1) or types by coordinate parity (T=2)."""
    g = np.stack(np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij"), axis=-1).reshape(-1, 3)
    typ = ((g.sum(axis=1) % 2) if T == 2 else np.zeros(len(g))).astype(np.int32)
    q = q_grid(q_max, M)
    f = np.ones((T, M), dtype=np.float32)
    if T == 2:
        f[1] *= 2.0
    return Workload(f"lattice_{nx}x{ny}x{nz}", (g * a).astype(np.float32), typ, f, q, {"n": (nx, ny, nz), "a": a})


def with_grid(w: Workload, q, tag: str, seed: int = 4242) -> Workload:
    """The same structure on another q grid (form factors of the same 4-Gaussian family, re-drawn for that grid)."""
    q = np.ascontiguousarray(q, dtype=np.float32)
    return Workload(f"{w.name}_{tag}", w.xyz, w.type, gaussian_form_factors(BASE_SEED + seed, w.T, q), q, dict(w.meta))


def grid_general_start(w: Workload) -> np.ndarray:
    """Uniform, M points, same range, but starting 2.46 steps above 0 (neither 0 nor dq): a detector edge."""
    dq = float(w.q[-1] - w.q[0]) / max(1, w.M - 1)
    return ((2.46 + np.arange(w.M, dtype=np.float64)) * dq).astype(np.float32)


def grid_two_pieces(w: Workload) -> np.ndarray:
    """M points in two uniform pieces: the lower half of the config's range at its own step, then a coarser range (twice the
    step) up to 1.5 x q_max -- a SAXS range followed by a WAXS range."""
    dq = float(w.q[-1] - w.q[0]) / max(1, w.M - 1)
    n1 = (w.M + 1) // 2
    lo = np.arange(n1, dtype=np.float64) * dq
    hi = lo[-1] + 2.0 * dq * np.arange(1, w.M - n1 + 1, dtype=np.float64)
    return np.concatenate([lo, hi]).astype(np.float32)


GRIDS = {"general_start": grid_general_start, "two_pieces": grid_two_pieces}
CONFIGS = {"cfg1": cfg1, "cfg2": cfg2, "cfg3": cfg3, "cfg4": cfg4, "cfg5": cfg5}


def peratom_table(w: Workload, seed: int = 0) -> np.ndarray:
    """ff[N][M] float32 for the per-ATOM path (the form factors "cannot be factored out of the equation, because the non-uniform density of the water layer
    atoms around the molecule creates an intractable number of possible f_k f_j combinations" --
    excluded volume and hydration layer): the type's row times a seeded per-atom factor in [0.6, 1.4] (a stand-in for the
    solvent-accessible fraction), plus a seeded per-atom offset in [-0.3, 0.3] that decays with q (a hydration-shell-like
    term), so that no two atoms share a row.  An input recipe only: none of the method's arithmetic."""
    rng = np.random.default_rng(0x5EED0000 + seed)
    base = w.fftab[w.type].astype(np.float64)
    fac = rng.uniform(0.6, 1.4, (w.N, 1))
    off = rng.uniform(-0.3, 0.3, (w.N, 1)) * np.exp(-np.linspace(0.0, 2.0, w.M))[None, :]
    return np.ascontiguousarray((base * fac + off).astype(np.float32))
