"""Multi-GPU domain decomposition: one process per GPU, the halo exchange of PAPER.md:76-78 over torch.distributed.

Every rank holds its part of the mesh as an ordinary context whose cut flux-point pairs name ghosts (include/frb200.h
`fr_halo_desc`; fr_inputs.partition.split_case builds such cases).  A right-hand side is the library's three phases
(`fr_rhs_phase`) with two point-to-point exchanges in between: U_f after S1 and, for Navier-Stokes, G_f after S5 -- one
contiguous message per peer and exchange, `ncclSend` / `ncclRecv` over NVLink 5 / NVSwitch when the process group is NCCL.
The library packs and unpacks with its own kernels; this module only moves the buffers (no arithmetic).  With the gloo
backend the same code runs on host copies of the buffers (CPU tests of the plumbing).

The transfers run on torch's current stream, which must be the stream the context was set up with.
"""
import numpy as np


class _DevBuf:
    """A device buffer of the library seen by torch (zero-copy) through __cuda_array_interface__."""

    def __init__(self, ptr, n, dtype):
        self.__cuda_array_interface__ = dict(shape=(int(n),), typestr="<f8" if dtype == np.float64 else "<f4",
                                             data=(int(ptr), False), version=2)


class HaloExchange:
    """Moves the send buffers of a context into the peers' receive buffers."""

    def __init__(self, ctx, dist=None):
        import torch
        self.ctx, self.dist, self.torch = ctx, dist, torch
        self.peers = ctx.halo["peers"]
        self.buf = {}
        for which in (0, 1):
            s, r, n = ctx.halo_buffers(which)
            if n:
                self.buf[which] = (torch.as_tensor(_DevBuf(s, n, ctx.dtype), device="cuda"),
                                   torch.as_tensor(_DevBuf(r, n, ctx.dtype), device="cuda"), 5 if which == 0 else 15)

    def segments(self, which):
        """[(peer rank, send view, receive view)]: V * count contiguous values per peer."""
        snd, rcv, V = self.buf[which]
        return [(p["rank"], snd[V * p["start"]:V * (p["start"] + p["count"])], rcv[V * p["start"]:V * (p["start"] + p["count"])])
                for p in self.peers]

    def exchange(self, which):
        if which not in self.buf:
            return
        dist = self.dist
        ops = []
        for peer, s, r in self.segments(which):
            ops += [dist.P2POp(dist.isend, s, peer), dist.P2POp(dist.irecv, r, peer)]
        for w in dist.batch_isend_irecv(ops):
            w.wait()


def partitioned_rhs(ctx, xch, u_ptrs, dudt_ptrs):
    """One right-hand side of this rank's part: three library phases, two exchanges."""
    ctx.rhs_phase(0, u_ptrs)
    xch.exchange(0)
    ctx.rhs_phase(1, u_ptrs)
    xch.exchange(1)
    ctx.rhs_phase(2, u_ptrs, dudt_ptrs)


def partitioned_rk_step(ctx, xch, dt, nstages=5):
    """One Runge-Kutta step on the internal state: every stage is the three phases with the stage update fused into the last."""
    for i in range(nstages):
        ctx.rk_stage_phase(dt, i, 0)
        xch.exchange(0)
        ctx.rk_stage_phase(dt, i, 1)
        xch.exchange(1)
        ctx.rk_stage_phase(dt, i, 2)


def local_exchange(xchs, which):
    """All ranks in one process on one device (tests on a single GPU): copy every rank's segments into its peers' receive
    buffers with device copies, the ranks' phases having been launched one after the other (no kernel waits on another)."""
    for r, x in enumerate(xchs):
        if which not in x.buf:
            continue
        for peer, s, _ in x.segments(which):
            back = [seg for seg in xchs[peer].segments(which) if seg[0] == r]
            back[0][2].copy_(s)
