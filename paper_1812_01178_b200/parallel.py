"""Multi-GPU slab sweeps (Algorithm 1 L222-258, L156/L174): one process per GPU, every rank
is one partition of the PDD / PPT method along the slab direction.  This module is plumbing only: the arithmetic (local
elimination, spikes, interface solve, correction) runs in the CUDA kernels behind `binding.Slab`; here the interface rows
travel between ranks with `torch.distributed` (NCCL on GPUs; the same functions run on CPU tensors over gloo, which is
how the exchange pattern is tested without GPUs).

  PDD  (Alg.1 steps 4 and 6): rank r sends its xt_first plane to r-1 and its xt_last plane to r+1 and receives
       xt_last of r-1 and xt_first of r+1 -- two neighbour messages of one plane each, no host synchronisation.
  PPT  (L156, L174): one all-gather of every rank's two planes; each rank then applies its two rows of Z^-1.
"""
import torch
import torch.distributed as dist

from . import binding as tdx


def slab_bounds(n_global, world):
    """Rows [start, stop) of each rank: the partition map of tdx_partition_bounds (reading A5)."""
    s = tdx.partition_bounds(n_global, world)
    return [(int(s[r]), int(s[r + 1])) for r in range(world)]


def exchange_pdd(iface, rank, world, group=None):
    """iface: [2][plane] = (xt_first, xt_last) of this rank.  Returns nbr [2][plane] = (xt_last of rank-1, xt_first of
    rank+1); the plane of a missing neighbour is left as zeros (never read)."""
    nbr = torch.zeros_like(iface)
    ops = []
    if rank >= 1:
        ops.append(dist.P2POp(dist.isend, iface[0], rank - 1, group))
        ops.append(dist.P2POp(dist.irecv, nbr[0], rank - 1, group))
    if rank <= world - 2:
        ops.append(dist.P2POp(dist.isend, iface[1], rank + 1, group))
        ops.append(dist.P2POp(dist.irecv, nbr[1], rank + 1, group))
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    return nbr


def exchange_ppt(iface, rank, world, group=None):
    """iface: [2][plane] of this rank.  Returns the gathered [world][2][plane] (rank-major)."""
    out = torch.empty((world,) + tuple(iface.shape), dtype=iface.dtype, device=iface.device)
    if world == 1:
        out[0].copy_(iface)
        return out
    if iface.is_cuda:
        dist.all_gather_into_tensor(out, iface.contiguous(), group=group)
    else:                                                       # gloo: list form
        parts = [out[r] for r in range(world)]
        dist.all_gather(parts, iface.contiguous(), group=group)
    return out


class SlabSweep:
    """x = (I - alpha delta2_dir)^-1 d on a field whose `direction` is split over `world` ranks; in place on the rank's
    slab tensor [nz_loc][ny_loc][nx] (float64, CUDA).  `across` = tdx.MODE_PDD or tdx.MODE_PPT between ranks,
    `local_mode` / `P_local` inside the rank."""

    def __init__(self, slab_grid, direction, rank, world, faces_global, bc_global, alpha, across, local_mode, P_local, group=None,
                 slab=None):
        """slab: an object with eliminate(field, iface, stream) / correct(field, iface_own, iface_nbr, stream) / close();
        default: the CUDA kernels behind tdx.Slab.  (The CPU tests of this class's control flow and exchange pattern pass
        a stand-in, since the kernels need a device.)"""
        self.slab = slab if slab is not None else tdx.Slab(slab_grid, direction, rank, world, faces_global, bc_global, alpha, across, local_mode, P_local)
        self.rank, self.world, self.across, self.group = rank, world, across, group
        g = slab_grid
        self.plane = (g.nx * g.nz) if direction == 1 else (g.nx * g.ny)
        self.iface = None

    def sweep(self, field):
        if self.iface is None or self.iface.device != field.device:
            self.iface = torch.empty((2, self.plane), dtype=torch.float64, device=field.device)
        stream = torch.cuda.current_stream().cuda_stream if field.is_cuda else 0
        self.slab.eliminate(field, self.iface, stream)
        if self.world == 1:
            return field
        if self.across == tdx.MODE_PDD:
            nbr = exchange_pdd(self.iface, self.rank, self.world, self.group)
        else:
            nbr = exchange_ppt(self.iface, self.rank, self.world, self.group)
        self.slab.correct(field, self.iface, nbr, stream)
        return field

    def close(self):
        self.slab.close()
