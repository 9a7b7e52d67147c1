"""Band sharding of the SHO project / add path across ranks.

Bands are independent in both steps -- eq. (25) carries the band index k as a free index
 and step (3) adds into each band separately -- so N ranks shard the
band axis with NO data-path collective: the plan (atoms, boxes) is replicated, rank r owns the bands
``band_range(nbands, r, N)`` of psi and the matching slab ``coeff[:, lo:hi, :]``.  The only
communication is the timing protocol of bench.py (barrier + max over ranks).

No method arithmetic here, no CUDA: plain index bookkeeping plus two tiny ``torch.distributed`` helpers
that work on any backend (nccl on the GPUs, gloo in the CPU tests).
"""
from __future__ import annotations


def band_range(nbands: int, rank: int, world: int) -> tuple[int, int]:
    """Half-open range [lo, hi) of the bands rank ``rank`` of ``world`` owns: contiguous, ascending,
    sizes differing by at most one (the first ``nbands % world`` ranks get the extra band)."""
    nbands, rank, world = int(nbands), int(rank), int(world)
    if world < 1 or not (0 <= rank < world) or nbands < 0:
        raise ValueError("band_range: need 0 <= rank < world and nbands >= 0")
    base, extra = divmod(nbands, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def band_owner(band: int, nbands: int, world: int) -> int:
    """The rank that owns ``band`` under ``band_range``."""
    band, nbands, world = int(band), int(nbands), int(world)
    if not (0 <= band < nbands):
        raise ValueError("band_owner: band out of range")
    base, extra = divmod(nbands, world)
    cut = extra * (base + 1)
    return band // (base + 1) if band < cut else extra + (band - cut) // max(base, 1)


def max_over_ranks(values, device=None):
    """Element-wise MAX of a list of floats over all ranks (bench.py: device times are reported as the
    max over ranks).  Identity when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def gather_band_slabs(local, nbands: int, band_axis: int = 1):
    """Test / driver helper: all-gather the per-rank band slabs of a tensor (coefficients
    ``[natoms][nb_local][N_SHO]`` with band_axis=1, psi ``[nb_local][Nz][Ny][Nx]`` with band_axis=0) into
    the full-band tensor on every rank.  NOT on the hot path: project and add never need it."""
    import torch
    import torch.distributed as dist

    world, rank = dist.get_world_size(), dist.get_rank()
    lo, hi = band_range(nbands, rank, world)
    if local.shape[band_axis] != hi - lo:
        raise ValueError("gather_band_slabs: local slab has %d bands, rank %d owns %d" % (local.shape[band_axis], rank, hi - lo))
    widest = -(-nbands // world)
    moved = local.movedim(band_axis, 0).contiguous()
    pad = torch.zeros((widest,) + tuple(moved.shape[1:]), dtype=moved.dtype, device=moved.device)
    pad[: hi - lo] = moved
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    out = []
    for r in range(world):
        rlo, rhi = band_range(nbands, r, world)
        out.append(parts[r][: rhi - rlo])
    return torch.cat(out, dim=0).movedim(0, band_axis).contiguous()
