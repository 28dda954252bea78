"""Host-side logic of the z-slab decomposition on CPU, world size 2 over gloo: WHICH planes go to WHOM.

Each rank takes the particles whose host cell lies in its slab, lets the ORACLE deposit them (on the periodic global grid, so
the x / y directions are already folded), cuts out its slab with g ghost planes per side, packs the ghost planes as the
library does ([channel][plane][row]), sends them with paper_2509_18261_b200.sharded.exchange_slabs -- the function the GPU
path uses -- and adds what it receives onto its boundary planes in the fixed order.  The result must be the single-domain
oracle's buffer restricted to the slab.  The state halo exchange is checked the same way (bit-exact copies).  With two ranks
the lower and the upper neighbour are the same peer: the test fails if the two messages of a pair are swapped.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import pm_oracle as po  # noqa: E402
from paper_2509_18261_b200 import inputs, sharded  # noqa: E402

N, G = 24, 4


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _slab_planes(a, z0, nz, g):
    """planes [z0 - g, z0 + nz + g) of a periodic global mesh (n, n, n)"""
    return np.ascontiguousarray(a[np.arange(z0 - g, z0 + nz + g) % a.shape[0]])


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = inputs.scaled_mixed(N, 240, seed_index=5)
        nz = N // world
        z0 = rank * nz
        # several particles right at the cuts, so that ghost planes carry something in both directions
        w.sinks.z[:4] = np.array([0.4, nz - 0.3, nz + 0.6, N - 0.2])
        w.sne.z[:8] = np.array([0.1, 1.7, nz - 2.2, nz - 0.1, nz + 0.2, nz + 2.9, N - 1.1, N - 0.05])
        full = po.Oracle(w.params, w.state.copy(), w.sinks.copy(), w.sne.copy())
        full.deposit(w.dt)
        mine_k = (w.sinks.z >= z0) & (w.sinks.z < z0 + nz)
        mine_n = (w.sne.z >= z0) & (w.sne.z < z0 + nz)
        sk = inputs.Sinks(*(getattr(w.sinks, f)[mine_k].copy() for f in ("x", "y", "z", "vx", "vy", "vz", "m")))
        sn = inputs.SNe(*(getattr(w.sne, f)[mine_n].copy() for f in ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej")))
        loc = po.Oracle(w.params, w.state.copy(), sk, sn)
        loc.deposit(w.dt)
        chans = [loc.A[0]] + [loc.S[f] for f in range(5)]                  # the six GPU channels (R29)
        ref = [full.A[0]] + [full.S[f] for f in range(5)]
        scale = [full.Aabs[0]] + [full.Sabs[f] for f in range(5)]
        slabs = [_slab_planes(c.reshape(N, N, N), z0, nz, G) for c in chans]
        # nothing of this rank's particles lands outside its slab + g ghost planes
        for c, s in zip(chans, slabs):
            assert np.isclose(np.abs(c).sum(), np.abs(s).sum(), rtol=1e-12)
        plane = N * N
        pack = lambda sl: torch.from_numpy(np.concatenate([s[sl].reshape(-1) for s in slabs]))
        send_lo, send_hi = pack(slice(0, G)), pack(slice(nz + G, nz + 2 * G))
        recv_lo, recv_hi = torch.empty_like(send_lo), torch.empty_like(send_hi)
        sharded.exchange_slabs(send_lo, send_hi, recv_lo, recv_hi, rank, world)
        worst = 0.0
        for ch in range(6):
            owned = slabs[ch][G:G + nz].copy()
            owned[:G] += recv_lo[ch * G * plane:(ch + 1) * G * plane].numpy().reshape(G, N, N)           # from the lower neighbour
            owned[nz - G:] += recv_hi[ch * G * plane:(ch + 1) * G * plane].numpy().reshape(G, N, N)      # from the upper neighbour
            want = ref[ch].reshape(N, N, N)[z0:z0 + nz]
            tol = 1e-12 * np.abs(want) + 64 * np.finfo(float).eps * scale[ch].reshape(N, N, N)[z0:z0 + nz] + 1e-300
            err = np.abs(owned - want)
            assert np.all(err <= tol), f"rank {rank} channel {ch}: {err.max()}"
            assert np.array_equal(owned != 0, want != 0)
            worst = max(worst, float(np.abs(recv_lo).sum() + np.abs(recv_hi).sum()))
        assert worst > 0.0                                                   # the cuts were really crossed
        # state halo: ghost planes poisoned, then filled by the exchange; must equal the global field's planes bit for bit
        fields = []
        for f in w.state.fields():
            a = _slab_planes(f, z0, nz, G)
            a[:G] = np.nan
            a[-G:] = np.nan
            fields.append(torch.from_numpy(a))
        sharded.exchange_state_halo(fields, G, plane, nz, rank, world)
        for t, f in zip(fields, w.state.fields()):
            assert np.array_equal(t.numpy(), _slab_planes(f, z0, nz, G))
        out[rank] = (int(mine_k.sum()), int(mine_n.sum()))
    finally:
        dist.destroy_process_group()


def test_slab_exchange_gloo_world2():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert sorted(res) == [0, 1]
    assert res[0][0] + res[1][0] == 24 and res[0][1] + res[1][1] == 216      # every particle belongs to exactly one slab


def test_neighbours_and_self_exchange():
    assert sharded.slab_neighbours(0, 1) == (0, 0)
    assert sharded.slab_neighbours(0, 2) == (1, 1) and sharded.slab_neighbours(1, 2) == (0, 0)
    assert sharded.slab_neighbours(0, 8) == (7, 1) and sharded.slab_neighbours(7, 8) == (6, 0)
    a, b = torch.arange(6.0), torch.arange(6.0) + 10
    rl, rh = torch.zeros(6), torch.zeros(6)
    sharded.exchange_slabs(a, b, rl, rh)                 # one rank: its low ghosts fold onto its own top planes and vice versa
    assert torch.equal(rh, a) and torch.equal(rl, b)


class _FakeSlabCtx:
    """Stands in for pm.Context in SlabStep's set-up and call sequence (no GPU): records what it is asked to do."""

    def __init__(self, rank):
        self.rank = rank
        self.params = {"z_slab": 1, "nx": 8, "ny": 8, "nz": 8}
        self.calls = []
        self.connected = None

        class _S:
            def synchronize(self_inner):
                self.calls.append("sync")
        self.stream = _S()

    def pm_slab_describe(self):
        keys = [g + "_" + s for g in ("buf", "ret", "rtr") for s in ("send_lo", "send_hi", "recv_lo", "recv_hi")]
        return dict({k: None for k in keys}, state_ghost_planes=4)

    def pm_slab_ipc_export(self):
        return ("handle-of-rank-%d" % self.rank).encode().ljust(64, b".")

    def pm_slab_connect_ipc(self, lower, upper):
        self.connected = (lower, upper)

    def __getattr__(self, name):                     # pm_deposit, pm_slab_put, pm_fold_ghosts, ... : just note the order
        if name.startswith("pm_"):
            return lambda *a, **k: self.calls.append(name)
        raise AttributeError(name)


def _peer_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ctx = _FakeSlabCtx(rank)
        step = sharded.SlabStep(ctx, rank, world, peer_put=True)

        class _NoFields:
            def fields(self):
                return []
        step.step(_NoFields(), None, None, 0.1)
        out[rank] = (ctx.connected, list(ctx.calls))
    finally:
        dist.destroy_process_group()


def test_peer_put_setup_hands_every_rank_its_two_neighbours_handles_world3():
    """SlabStep(peer_put=True): all ranks publish the IPC handle of their slab memory, every rank connects to the handle of
    rank - 1 (its low ghost planes go there) and of rank + 1, periodic in the rank index; a step then puts, drains its stream
    and meets the others BEFORE it folds.  Three ranks, so that lower and upper neighbour differ."""
    world, port = 3, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_peer_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    h = lambda r: ("handle-of-rank-%d" % r).encode().ljust(64, b".")
    for r in range(3):
        connected, calls = res[r]
        assert connected == (h((r - 1) % 3), h((r + 1) % 3))
        assert calls == ["pm_deposit", "pm_slab_put", "sync", "pm_fold_ghosts", "pm_apply_limited", "pm_return_to_particles"]
    # one rank: its own neighbour on both sides, no handle travels
    ctx = _FakeSlabCtx(0)
    sharded.SlabStep(ctx, 0, 1, peer_put=True)
    assert ctx.connected == (None, None)
