"""z-slab decomposition of ONE registration over several GPUs (volumes of
512x512x256 and up; BASELINE.json keeps the 256x256x100 class on one GPU, where an iteration is ~100 us and
the exchange would eat the gain).

Partition.  Rank r owns a contiguous range of z planes and holds, of the displacement field(s), those planes
plus a halo of H = ceil(3 sigma) + 1 planes on every interior side.  The images S and M are replicated on
every rank (268 MB each at 512x512x256): the trilinear gather of PAPER.md L179 reaches anywhere along z and
never leaves the device.  One iteration on a rank is

    demons_warp_force_slab   u -> u'   on the whole slab (image accesses in global planes)
    demons_smooth            u' -> u   on the whole slab (clamps at the slab ends)
    halo refresh             the H outermost planes of every interior side are overwritten with the neighbour's
                             own planes (torch.distributed send/recv: NCCL over NVLink on GPUs)

The gradient of the warped image (variants 2-5) is wrong on the outermost plane of an interior side, the force
there is wrong, and the Gaussian carries that R planes inwards: R + 1 halo planes keep the own planes exact.
They are BIT-IDENTICAL to the single-GPU result (same kernels, same arithmetic per voxel); the three metrics
are summed over own planes on each rank and added over the ranks once, at the end (every BASELINE.json
configuration fixes the iteration count; the stopping rule would need that sum every iteration).

Pyramid levels below the finest are an eighth of the work or less: every rank runs them whole, redundantly
(`demons_register` on the restricted pair), prolongs, and keeps its slab -- no exchange, same bits.

All arithmetic is in libdemons.so; this module is plumbing: slab bookkeeping, torch allocations, and the
exchange.  `LocalExchange` moves the halos between the slabs of several ranks held by ONE process (one GPU):
tests/test_gpu_parity.py uses it to check the decomposition against the undivided registration.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

from . import binding as B


@dataclass(frozen=True)
class Slab:
    rank: int
    world: int
    own0: int   # first own plane (global)
    own1: int   # one past the last own plane (global)
    lo: int     # first plane held (global): own0 - halo, clipped to the volume
    hi: int     # one past the last plane held (global)
    halo: int

    @property
    def count(self):       # planes held
        return self.hi - self.lo

    @property
    def own_begin(self):   # first own plane, local index
        return self.own0 - self.lo

    @property
    def own_count(self):
        return self.own1 - self.own0


def halo_planes(sigma: float) -> int:
    """R + 1: R = ceil(3 sigma) for the Gaussian, one more for the central difference of the warped image."""
    return int(math.ceil(3.0 * float(sigma))) + 1


def plan(nz: int, world: int, halo: int):
    """Balanced contiguous split of nz planes over `world` ranks.  Every rank must own at least `halo` planes,
    so that a halo is filled by the adjacent rank alone."""
    if world < 1 or nz < world:
        raise ValueError("more ranks than planes")
    slabs = []
    for r in range(world):
        own0, own1 = (r * nz) // world, ((r + 1) * nz) // world
        if world > 1 and own1 - own0 < halo:
            raise ValueError(f"rank {r} would own {own1 - own0} planes, fewer than the halo of {halo}")
        slabs.append(Slab(r, world, own0, own1, max(0, own0 - halo), min(nz, own1 + halo), halo))
    return slabs


class LocalExchange:
    """Halo refresh between the slabs of all ranks held by one process (the single-GPU stand-in)."""

    def __init__(self, slabs):
        self.slabs = slabs

    def refresh(self, fields):
        """fields[r]: (3, count_r, ny, nx) tensor of rank r.  Interior halos <- the neighbour's own planes."""
        for s in self.slabs:
            f = fields[s.rank]
            if s.rank > 0:                       # lower halo: planes [lo, own0) from rank - 1
                n = self.slabs[s.rank - 1]
                f[:, 0:s.own0 - s.lo].copy_(fields[n.rank][:, s.lo - n.lo:s.own0 - n.lo])
            if s.rank < s.world - 1:             # upper halo: planes [own1, hi) from rank + 1
                n = self.slabs[s.rank + 1]
                f[:, s.own1 - s.lo:s.hi - s.lo].copy_(fields[n.rank][:, s.own1 - n.lo:s.hi - n.lo])


class DistExchange:
    """Halo refresh of THIS rank's slab over torch.distributed (NCCL on GPUs, gloo on CPU): per neighbour one
    send of own boundary planes and one receive into the halo, per component (contiguous slices)."""

    def __init__(self, slab: Slab):
        self.slab = slab

    def refresh(self, field):
        import torch.distributed as dist
        s = self.slab
        ops, keep = [], []
        for nb_rank, send_planes, recv_planes in (
                (s.rank - 1, (s.own0 - s.lo, s.own0 - s.lo + s.halo), (0, s.own0 - s.lo)),
                (s.rank + 1, (s.own1 - s.lo - s.halo, s.own1 - s.lo), (s.own1 - s.lo, s.hi - s.lo))):
            if nb_rank < 0 or nb_rank >= s.world:
                continue
            # every rank owns at least `halo` planes (plan()), so a halo is exactly `halo` planes deep
            for c in range(field.shape[0]):
                out = field[c, send_planes[0]:send_planes[1]]
                inp = field[c, recv_planes[0]:recv_planes[1]]
                keep.append(out)
                ops.append(dist.P2POp(dist.isend, out, nb_rank))
                ops.append(dist.P2POp(dist.irecv, inp, nb_rank))
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()


def iterate_slabs(engines, slabs, dS, dM, fields, scratch, iters, sigma, exchange, metrics=None, fields_b=None,
                  scratch_b=None, eps=0.0):
    """`iters` iterations on the slabs in `fields` (a list with one entry per rank this process holds; one entry
    under torch.distributed).  engines[i]: binding.Demons created with the WHOLE volume's dims; metrics (optional):
    float64 device tensors (iters, 3) per held rank, filled with the sums over own planes.  Everything is enqueued
    on torch's current stream, so that kernels, halo copies and NCCL transfers are ordered.

    Limits, checked here: exactly `iters` iterations run -- the stopping rule of PAPER.md L145 needs the three sums
    added over all ranks after every iteration, which this loop does not do, so eps > 0 is refused rather than
    ignored; and every slab must carry a halo of at least halo_planes(sigma) planes (plan() has already refused
    splits in which a rank owns fewer planes than its halo, i.e. world > nz / halo)."""
    if eps is not None and float(eps) > 0.0:
        raise ValueError("iterate_slabs runs fixed iteration counts: the stopping rule (eps > 0) needs the metrics "
                         "summed over the ranks every iteration, which the slab loop does not do")
    need = halo_planes(sigma)
    for s in slabs:
        if s.world > 1 and s.halo < need:
            raise ValueError(f"slab of rank {s.rank} has a halo of {s.halo} planes; sigma = {sigma} needs {need}")
    import torch
    dims = engines[0].dims
    local = isinstance(exchange, LocalExchange)
    st = torch.cuda.current_stream()
    for it in range(iters):
        for i, s in enumerate(slabs):
            m = metrics[i][it] if metrics is not None else None
            B.demons_warp_force_slab(engines[i].ctx, dims, s.lo, s.count, s.own_begin, s.own_count, dS, dM, fields[i],
                                     scratch[i], fields_b[i] if fields_b else None, scratch_b[i] if scratch_b else None,
                                     m, st)
            ldims = (dims[0], dims[1], s.count)
            B.demons_smooth(engines[i].ctx, ldims, scratch[i], fields[i], 3, sigma, st)
            if fields_b:
                B.demons_smooth(engines[i].ctx, ldims, scratch_b[i], fields_b[i], 3, sigma, st)
        exchange.refresh(fields if local else fields[0])
        if fields_b:
            exchange.refresh(fields_b if local else fields_b[0])


def coarse_levels_replicated(dims, spacing, variant, alpha, sigma, dS, dM, iters_coarse, device):
    """The pyramid levels below the finest, run whole (every rank does the same work, no exchange): restrict the
    pair, register it with the remaining levels, prolong.  Returns the initial field(s) of the finest level for the
    whole volume, (u, u_b or None)."""
    import torch
    st = torch.cuda.current_stream()
    fine = B.Demons(dims, spacing, variant, alpha, sigma, levels=1, device=device)
    cd = B.demons_level_dims(fine.ctx, 1)
    cshape = (cd[2], cd[1], cd[0])
    S1 = torch.empty((2,) + cshape, dtype=torch.float32, device=device)   # S then M: one L2 window covers both
    B.demons_restrict(fine.ctx, dims, dS, S1[0], st)
    B.demons_restrict(fine.ctx, dims, dM, S1[1], st)
    coarse = B.Demons(cd, spacing, variant, alpha, sigma, levels=len(iters_coarse), device=device)
    if len(iters_coarse) == 1:
        B.demons_set_option(coarse.ctx, "zero_start", 1)
    ic = variant == B.INVERSE_CONSISTENT
    uc = torch.empty((3,) + cshape, dtype=torch.float32, device=device)
    ubc = torch.empty_like(uc) if ic else None
    B.demons_register(coarse.ctx, S1[0], S1[1], uc, ubc, iters_coarse, 0.0, None, None, st)
    shape = (dims[2], dims[1], dims[0])
    u = torch.empty((3,) + shape, dtype=torch.float32, device=device)
    B.demons_prolong(fine.ctx, cd, uc, dims, u, st)
    ub = None
    if ic:
        ub = torch.empty_like(u)
        B.demons_prolong(fine.ctx, cd, ubc, dims, ub, st)
    torch.cuda.synchronize()
    coarse.close()
    fine.close()
    return u, ub
