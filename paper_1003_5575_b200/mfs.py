"""Row f4: the sum of the per-GPU grids of a channel-sharded job (PAPER.md :108-120).

Every rank grids its own block of channels onto its own grid (no collective on the timed path,
DESIGN.md section 9).  A multi-frequency-synthesis image needs the sum of those grids: `reduce_grids`
is a deterministic all-reduce made of two exchanges and one kernel of ours,

    all-to-all (rank r receives slice r of every rank's grid, in rank order)
    gridder_sum_parts (FP64 sum of the `world` slices in rank order, one rounding to FP32)
    all-gather (every rank receives every summed slice)

so the result is independent of the collective library's reduction algorithm and order: bit-identical
from run to run and on every rank.  torch.distributed supplies the exchanges (NCCL over NVLink on
GPUs; gloo on CPU for the host-logic tests, which pass their own `sum_parts`).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def slice_len(numel: int, world: int) -> int:
    """Elements per rank slice: the smallest multiple of 4 (float4 kernels) that covers numel / world."""
    per = -(-numel // world)
    return -(-per // 4) * 4


def sum_parts_cuda(parts: torch.Tensor) -> torch.Tensor:
    """parts: CUDA float32 [n_parts][len] -> float32 [len], FP64 accumulation in part order (our kernel)."""
    from . import gridder
    lib = gridder.load_library()
    if not parts.is_cuda or parts.dtype != torch.float32 or not parts.is_contiguous():
        raise ValueError("sum_parts_cuda wants a contiguous CUDA float32 tensor [n_parts][len]")
    n_parts, length = parts.shape
    out = torch.empty(length, dtype=torch.float32, device=parts.device)
    rc = lib.gridder_sum_parts(parts.data_ptr(), n_parts, length, length, out.data_ptr(),
                               torch.cuda.current_stream(parts.device).cuda_stream)
    if rc != gridder.OK:
        raise gridder.GridderError(rc, "gridder_sum_parts")
    return out


def reduce_grids(grid: torch.Tensor, group=None, sum_parts=None) -> torch.Tensor:
    """In place: grid <- sum over ranks of grid, the same bits on every rank.  `sum_parts` maps a
    [world][slice] tensor to its FP64 fixed-order sum over dim 0 (default: the CUDA kernel)."""
    world = dist.get_world_size(group)
    if world == 1:
        return grid
    if not grid.is_contiguous() or grid.dtype != torch.float32:
        raise ValueError("reduce_grids wants a contiguous float32 grid")
    sum_parts = sum_parts or sum_parts_cuda
    flat = grid.view(-1)
    numel = flat.numel()
    L = slice_len(numel, world)
    send = flat
    if world * L != numel:                                   # pad so that every rank's slice has L elements
        send = torch.zeros(world * L, dtype=flat.dtype, device=flat.device)
        send[:numel] = flat
    recv = torch.empty(world * L, dtype=flat.dtype, device=flat.device)
    dist.all_to_all_single(recv, send, group=group)          # recv[p L : (p+1) L] = rank p's slice `rank`
    mine = sum_parts(recv.view(world, L))
    out = torch.empty(world * L, dtype=flat.dtype, device=flat.device)
    dist.all_gather_into_tensor(out, mine.contiguous(), group=group)
    flat.copy_(out[:numel])
    return grid
