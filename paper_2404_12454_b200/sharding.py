"""Host-side sharding of the field sum over detector rows.

Pixels are independent, so N ranks need no data-path collective: each rank evaluates a band of rows
with the same beamlet records.  The band helpers only build detector descriptors and run on the CPU;
`gather_rows` is the one optional collective after the path ("outputs stay sharded or one all-gather of
16 B per pixel"), through torch.distributed -- NCCL over NVLink for device tensors, gloo for host tensors.
"""
from __future__ import annotations


def row_range(n_v: int, rank: int, world: int):
    """Contiguous, balanced split of n_v rows: the first n_v % world ranks get one extra row."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, extra = divmod(n_v, world)
    v0 = rank * base + min(rank, extra)
    return v0, v0 + base + (1 if rank < extra else 0)


def row_band(detector: dict, rank: int, world: int) -> dict:
    """Sub-detector covering this rank's rows of `detector` (strong scaling).  Pixel (iu, iv_local) of
    the band sits exactly where pixel (iu, v0 + iv_local) of the full detector sits."""
    n_v = int(detector["n_v"])
    v0, v1 = row_range(n_v, rank, world)
    shift = (0.5 * (v0 + v1 - 1) - 0.5 * (n_v - 1)) * float(detector["dv"])
    out = dict(detector)
    out["n_v"] = v1 - v0
    out["origin"] = [float(o) + shift * float(e) for o, e in zip(detector["origin"], detector["e_v"])]
    out["row_offset"] = v0
    return out


def weak_band(detector: dict, rank: int, world: int) -> dict:
    """Rank r's own full-size band of a `world`-times taller detector (weak scaling, bench.py)."""
    band = int(detector["n_v"]) * float(detector["dv"])
    shift = (rank - 0.5 * (world - 1)) * band
    out = dict(detector)
    out["origin"] = [float(o) + shift * float(e) for o, e in zip(detector["origin"], detector["e_v"])]
    return out


def gather_rows(band_field, n_v: int, group=None):
    """All-gather the finished row bands of `row_band` into the full (n_v, n_u) field on every rank.
    `band_field` is this rank's (rows, n_u) complex tensor (device tensor -> NCCL, host tensor -> gloo); bands may
    differ by one row, so they are padded to the tallest one for the collective (complex viewed as real pairs)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    v0, v1 = row_range(n_v, rank, world)
    if band_field.shape[0] != v1 - v0:
        raise ValueError("band_field does not have this rank's rows")
    tallest = -(-n_v // world)
    real = torch.view_as_real(band_field.contiguous())
    pad = real.new_zeros((tallest,) + tuple(real.shape[1:]))
    pad[: v1 - v0] = real
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    out = real.new_empty((n_v,) + tuple(real.shape[1:]))
    for r in range(world):
        a, b = row_range(n_v, r, world)
        out[a:b] = parts[r][: b - a]
    return torch.view_as_complex(out)
