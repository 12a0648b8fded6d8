"""Multi-GPU plumbing for libdebye: the path shards over independent structures /
conformers with NO data-path collective -- each rank owns a contiguous slice of the batch and writes its own
rows of I_out.  torch.distributed is used only to agree on timing (max over ranks) and, optionally, to gather the
per-rank profiles to rank 0."""
from __future__ import annotations


def shard_range(n_items: int, rank: int, world: int):
    """Contiguous, balanced slice [lo, hi) of n_items owned by `rank` (sizes differ by at most one)."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    base, extra = divmod(n_items, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def max_over_ranks(value: float, device=None) -> float:
    """Max of a scalar over all ranks (identity without an initialised process group)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def gather_profiles(local, n_total: int, rank: int, world: int):
    """All-gather the per-rank rows I[lo:hi, M] into the full [n_total, M] array (every rank gets it)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or world == 1:
        return local
    M = local.shape[1]
    sizes = [shard_range(n_total, r, world) for r in range(world)]
    mx = max(hi - lo for lo, hi in sizes)
    pad = torch.zeros((mx, M), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    bufs = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(bufs, pad)
    return torch.cat([bufs[r][: hi - lo] for r, (lo, hi) in enumerate(sizes)], dim=0)


# ---- one structure over several GPUs: split of the q grid ------------------------------------------------------------------
# The paper's own multi-device idea (different q ranges on different devices).  Every rank holds all atoms
# and computes a contiguous slice of the q grid with the ordinary single-GPU call (distances are recomputed per rank, as in
# the paper's proposal); the only exchange is an all-gather of the M/world profile values.  A contiguous slice of a uniform
# grid is uniform, so every rank keeps the recurrence kernel.
def q_slice(M: int, rank: int, world: int):
    """[lo, hi) of the q grid owned by `rank`."""
    return shard_range(M, rank, world)


def profile_q_slice(profile_fn, fftab, q, rank: int, world: int):
    """This rank's part of one profile: profile_fn(fftab[:, lo:hi], q[lo:hi]) -> values [hi - lo] (empty slices allowed).
    `profile_fn` is the single-GPU call with xyz / type bound (e.g. lambda f, q: binding.debye_profile(xyz, type, f, q))."""
    lo, hi = q_slice(q.shape[0], rank, world)
    if hi == lo:
        return fftab.new_zeros(0, dtype=__import__("torch").float64), (lo, hi)
    return profile_fn(fftab[:, lo:hi].contiguous(), q[lo:hi].contiguous()), (lo, hi)


def gather_q_slices(local, M: int, rank: int, world: int):
    """All-gather the per-rank slices of one profile into the full [M] profile (every rank gets it)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or world == 1:
        return local
    sizes = [q_slice(M, r, world) for r in range(world)]
    mx = max(hi - lo for lo, hi in sizes)
    pad = torch.zeros(mx, dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    bufs = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(bufs, pad)
    return torch.cat([bufs[r][: hi - lo] for r, (lo, hi) in enumerate(sizes)], dim=0)


# ---- one structure over several GPUs: split by tiles of the upper triangle ---------------------------------------------------
# tiles are independent units, every GPU holds all coordinates (<= 3.2 MB), pairs CTA c of the static
# schedule belongs to rank c mod world (cyclic keeps the triangular load balanced), and the one exchange step is an
# all-gather of the FP64 partial structure factors S_ab[T(T+1)/2][M] (<= 215 KB per conformer) followed by a fixed-order sum
# (bitwise reproducible for a given world size) and the form-factor epilogue, both inside debye_profile_from_partials.
# Unlike the q-range split above, no distance is computed twice.
def gather_partials(S_part, world: int):
    """All-gather [B, n_tp, M] parts into [world, B, n_tp, M] in rank order (identity reshape without a process group)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or world == 1:
        return S_part[None].contiguous()
    out = torch.empty((world,) + tuple(S_part.shape), dtype=S_part.dtype, device=S_part.device)
    dist.all_gather(list(out.unbind(0)), S_part.contiguous())   # views of one buffer: rank order, no extra copy
    return out


def assert_same_schedule(pairs_grid: int, world: int, device=None):
    """The tile split assigns pairs CTA c of ONE static schedule to rank c mod world, so every rank must have built the
    same schedule: the same pairs grid (it depends on the device's SM count and the kernel's occupancy, binding.launch_info).
    Raises on every rank if the ranks disagree (mixed GPU models, differently built libraries)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or world == 1:
        return
    t = torch.tensor([int(pairs_grid), -int(pairs_grid)], dtype=torch.int64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    if int(t[0]) != -int(t[1]):
        raise RuntimeError(f"tile split: ranks disagree on the pairs grid (max {int(t[0])}, min {-int(t[1])}); "
                           "every rank must run the same GPU model and library build")


def profile_tile_split(partials_shard_fn, from_partials_fn, fftab, rank: int, world: int):
    """One profile of one structure (or batch) on `world` GPUs: partials_shard_fn(rank, world) -> (S_part, n) is this rank's
    tile share (binding.debye_partials_shard with xyz / type / q bound), the parts are all-gathered, and
    from_partials_fn(S_parts, n, fftab) -> I[B, M] (binding.debye_profile_from_partials) sums them in rank order and applies
    the epilogue.  Every rank returns the full profile."""
    S_part, n = partials_shard_fn(rank, world)
    return from_partials_fn(gather_partials(S_part, world), n, fftab)
