"""z-slab decomposition of the exchange step over ranks: the plumbing around the C calls.

One process per GPU; rank r owns the planes [r nz, (r + 1) nz) of a domain cut along z (periodic in the rank index).
The method's arithmetic is all in the CUDA kernels (csrc/pm_slab.cuh, the fold kernel, the return kernel); this module
only says WHICH buffer goes to WHOM, through torch.distributed point-to-point calls (NCCL on GPUs, gloo in the CPU tests):

    Step 2 (Eq. 3)  a rank's low  z ghost planes -> the LOWER neighbour's `recv_hi`
                                     a rank's high z ghost planes -> the UPPER neighbour's `recv_lo`
    Step 4 fill-back (L79, R16)      a rank's bottom owned planes of the return mesh -> the lower neighbour's high ghost planes,
                                     its top owned planes -> the upper neighbour's low ghost planes
    state halo (before pm_deposit)   the same pattern as the fill-back, for the six state fields

Step 2 has a second form, `peer_put=True`: no message at all.  The ranks exchange CUDA IPC handles of their slab memory once;
from then on the pack kernel of every rank stores its ghost planes straight into the neighbours' receive slabs through
peer-mapped memory (pm_slab_put: compute step and transfer in one kernel, NVLink between the GPUs of a node), and the only
host-side action per step is "drain the stream, then a barrier" so that every rank folds after every put has landed
(include/pm.h says why one barrier per step is enough).

With world size 2 both neighbours are the same peer; messages between one pair of ranks match in the order they are posted,
so every rank posts "to lower, to upper" and "from upper, from lower" -- the peer's first message is its "to lower" one, which
is what this rank's "from upper" slot expects.  With world size 1 a rank is its own neighbour (plain copies): the result is
then the periodic single-domain step, bit for bit.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def slab_neighbours(rank: int, size: int):
    """(lower, upper) neighbour of a rank in the periodic chain of z slabs."""
    return (rank - 1) % size, (rank + 1) % size


def exchange_slabs(send_lo, send_hi, recv_lo, recv_hi, rank: int = 0, size: int = 1, group=None):
    """send_lo -> lower neighbour's recv_hi, send_hi -> upper neighbour's recv_lo; fills this rank's recv_lo / recv_hi.
    All four are 1-d tensors of equal length (device tensors with NCCL, CPU tensors with gloo).  Blocks until done."""
    if size == 1:
        recv_hi.copy_(send_lo)
        recv_lo.copy_(send_hi)
        return
    lo, hi = slab_neighbours(rank, size)
    if send_lo.is_cuda and dist.get_backend(group) == "gloo":
        # device tensors over a CPU-only backend (two ranks sharing one GPU in the tests): stage through host memory
        host = [t.cpu() for t in (send_lo, send_hi)]
        got = [torch.empty_like(host[0]), torch.empty_like(host[1])]
        exchange_slabs(host[0], host[1], got[0], got[1], rank, size, group)
        recv_lo.copy_(got[0])
        recv_hi.copy_(got[1])
        return
    ops = [dist.P2POp(dist.isend, send_lo, lo, group), dist.P2POp(dist.isend, send_hi, hi, group),
           dist.P2POp(dist.irecv, recv_hi, hi, group), dist.P2POp(dist.irecv, recv_lo, lo, group)]
    for req in dist.batch_isend_irecv(ops):
        req.wait()


def exchange_state_halo(fields, g: int, plane: int, nz: int, rank: int = 0, size: int = 1, group=None):
    """Fill the g ghost planes below and above the nz owned planes of every field (flat tensors of (nz + 2g) * plane values)
    with the neighbours' boundary planes: the halo exchange a hydro code does anyway."""
    gp = g * plane
    for f in fields:
        v = f.view(-1)
        exchange_slabs(v[gp:2 * gp], v[nz * plane:nz * plane + gp], v[0:gp], v[(nz + g) * plane:(nz + 2 * g) * plane],
                       rank, size, group)


class SlabStep:
    """One rank's exchange step on its z slab: the C calls in order, with the three exchanges between them."""

    def __init__(self, ctx, rank: int = 0, size: int = 1, group=None, peer_put: bool = False):
        assert ctx.params.get("z_slab", 0) == 1, "the ctx must be created with z_slab = 1"
        self.ctx, self.rank, self.size, self.group = ctx, rank, size, group
        self.d = ctx.pm_slab_describe()
        self.peer_put = peer_put
        if peer_put:
            if size == 1:
                ctx.pm_slab_connect_ipc(None, None)            # its own neighbour on both sides
            else:
                handles = [None] * size
                dist.all_gather_object(handles, ctx.pm_slab_ipc_export(), group=group)
                lo, hi = slab_neighbours(rank, size)
                ctx.pm_slab_connect_ipc(handles[lo], handles[hi])
        p = ctx.params
        self.g, self.plane, self.nz = self.d["state_ghost_planes"], p["nx"] * p["ny"], p["nz"]

    # The slab memory is written and read by kernels on the ctx's stream.  torch.distributed (NCCL) and Tensor.copy_ work on
    # torch's current stream, which is the stream pm.Context hands to pm_create by default: stream order is all that is needed.

    def _xchg(self, grp):
        d = self.d
        if d[grp + "_send_lo"] is None:
            return
        exchange_slabs(d[grp + "_send_lo"], d[grp + "_send_hi"], d[grp + "_recv_lo"], d[grp + "_recv_hi"], self.rank, self.size, self.group)

    def _landed(self):
        """Every rank's put of this step is complete: drain this rank's stream, then meet the others."""
        self.ctx.stream.synchronize()
        if self.size > 1:
            dist.barrier(group=self.group)

    def halo(self, state):
        exchange_state_halo(state.fields(), self.g, self.plane, self.nz, self.rank, self.size, self.group)

    def step(self, state, sinks, sne, dt, halo: bool = True):
        """state: pm.DeviceState whose fields hold (nz + 2g) planes.  halo=False when the caller has filled the ghost planes."""
        c = self.ctx
        if halo:
            self.halo(state)
        c.pm_deposit(state, sinks, sne, dt)
        if self.peer_put:
            c.pm_slab_put()                     # Step 2: ghost planes -> the neighbours' receive slabs, stored by the pack kernel
            self._landed()
        else:
            c.pm_slab_pack()
            self._xchg("buf")                   # Step 2: ghost planes -> neighbours, as messages
        c.pm_fold_ghosts()
        c.pm_apply_limited(state)
        self._xchg("ret")                       # owner -> ghost copy of (eta, v_old) for Step 4 (R16)
        self._xchg("rtr")
        c.pm_return_to_particles(sinks)
