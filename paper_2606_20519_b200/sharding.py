"""Multi-GPU use of the path.

A single block does not shard (replicas only).  A block LIST shards by independent
units: blocks are assigned to ranks by n^3 cost, largest first; each rank projects
its blocks with hpsd_project, then ONE all-gather of the output svec pieces makes the
whole vector available everywhere.  Host-side logic only; the projection itself is the
C-ABI call.  Covered on CPU by world_size-2 gloo tests with a stand-in projector.
"""
from __future__ import annotations

from typing import Callable, List, Optional, Sequence

import torch


def assign_blocks(sizes: Sequence[int], world_size: int) -> List[List[int]]:
    """Longest-processing-time assignment of block indices to ranks by n^3 cost."""
    order = sorted(range(len(sizes)), key=lambda b: (-int(sizes[b]) ** 3, b))
    load = [0] * world_size
    owned: List[List[int]] = [[] for _ in range(world_size)]
    for b in order:
        r = min(range(world_size), key=lambda k: (load[k], k))
        owned[r].append(b)
        load[r] += int(sizes[b]) ** 3
    for lst in owned:
        lst.sort()
    return owned


def project_sharded(sizes: Sequence[int], in_svec: torch.Tensor, group=None,
                    projector: Optional[Callable[[Sequence[int], torch.Tensor], torch.Tensor]] = None) -> torch.Tensor:
    """Project a block list with the blocks spread over the ranks of `group`.

    Every rank passes the full in_svec and gets the full out_svec.  `projector(sizes, svec)`
    defaults to the CUDA hpsd_project binding; tests pass a stand-in on CPU."""
    import torch.distributed as dist

    if projector is None:
        from .binding import project as projector  # noqa: PLC0415
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    offs = [0]
    for n in sizes:
        offs.append(offs[-1] + int(n) * int(n))
    owned = assign_blocks(sizes, world)
    mine = owned[rank]
    my_sizes = [int(sizes[b]) for b in mine]
    if mine:
        my_in = torch.cat([in_svec[offs[b]:offs[b + 1]] for b in mine])
    else:
        my_in = in_svec.new_zeros(0)
    my_out = projector(my_sizes, my_in) if mine else my_in
    # one all-gather of the (padded) per-rank pieces
    lens = [sum(int(sizes[b]) ** 2 for b in owned[r]) for r in range(world)]
    pad = max(lens) if lens else 0
    buf = in_svec.new_zeros(pad)
    buf[: my_out.numel()] = my_out
    gathered = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(gathered, buf, group=group)
    out = torch.empty_like(in_svec)
    for r in range(world):
        pos = 0
        for b in owned[r]:
            ln = offs[b + 1] - offs[b]
            out[offs[b]:offs[b + 1]] = gathered[r][pos:pos + ln]
            pos += ln
    return out
