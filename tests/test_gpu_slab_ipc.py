"""z-slab decomposition with TWO PROCESSES, peer-memory form of Step 2: each rank's pack kernel stores its
ghost planes straight into the other rank's receive slabs (pm_slab_put), the slab memory being mapped into the neighbour
process through a CUDA IPC handle -- the mechanism that carries the transfer over NVLink when the ranks sit on different GPUs
of a node.  This box has one GPU, so all ranks use cuda:0 (two ranks: both neighbours are the same peer; three: they differ); no kernel of one rank ever waits for a kernel of the other (the only
synchronisation is "drain the stream, then a host barrier", sharded.SlabStep._landed).  The control plane is gloo; the state
halo and the return-mesh fill-back travel through sharded.exchange_slabs (staged through host memory on this backend).

Each rank runs three steps on its half of the domain; the parent glues the halves and compares with the single-domain oracle:
step 1 to the strict tolerances of tests/parity.py, the free-running trajectory to 1e-9."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2509_18261_b200 import inputs  # noqa: E402

pytestmark = pytest.mark.gpu
N, NPART, SEED, STEPS = 48, 1400, 12, 3


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def workload(world):
    """The same on every rank and in the parent: seeded, a fifth of the particles within 3 cells of a cut."""
    w = inputs.scaled_mixed(N, NPART, seed_index=SEED)
    h = N // world
    rng = np.random.default_rng(SEED)
    for prt in (w.sinks, w.sne):
        k = max(prt.n // 5, 2)
        prt.z[:k] = np.mod(rng.choice([float(h * r) for r in range(world)], size=k) + rng.uniform(-3.0, 3.0, size=k), float(N))
    return w


def _worker(rank, world, port, outdir):
    import torch.distributed as dist

    from paper_2509_18261_b200 import pm, sharded
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        dev = torch.device("cuda:0")
        torch.cuda.set_device(dev)
        w = workload(world)
        h = N // world
        z0 = rank * h
        p = dict(w.params, nz=h, z_slab=1)
        p["x0"] = (p["x0"][0], p["x0"][1], p["x0"][2] + z0 * p["dx"])
        ctx = pm.Context(p, device="cuda:0")
        g = ctx.ghost_width()
        idx = np.arange(z0 - g, z0 + h + g) % N
        fields = []
        for f in w.state.fields():
            a = np.ascontiguousarray(f[idx])
            a[:g] = np.nan                               # the halo exchange has to fill the ghost planes
            a[-g:] = np.nan
            fields.append(torch.from_numpy(a).to(dev))
        state = pm.DeviceState(*fields)
        sel_k = np.nonzero((w.sinks.z >= z0) & (w.sinks.z < z0 + h))[0]
        sel_n = np.nonzero((w.sne.z >= z0) & (w.sne.z < z0 + h))[0]
        sk = inputs.Sinks(*(np.ascontiguousarray(getattr(w.sinks, f)[sel_k]) for f in ("x", "y", "z", "vx", "vy", "vz", "m")))
        sn = inputs.SNe(*(np.ascontiguousarray(getattr(w.sne, f)[sel_n]) for f in ("x", "y", "z", "vx", "vy", "vz", "e_sn", "m_ej")))
        sinks = pm.DeviceSinks.from_host(sk, dev) if sk.n else None
        sne = pm.DeviceSNe.from_host(sn, dev) if sn.n else None
        step = sharded.SlabStep(ctx, rank, world, peer_put=True)
        out = {"sel_k": sel_k}
        for s in range(STEPS):
            step.step(state, sinks, sne, w.dt)
            ctx.pm_check()
            for name, t in zip(("rho", "mx", "my", "mz", "etot", "eint"), state.fields()):
                out[f"{name}{s}"] = t.view(h + 2 * g, N, N)[g:-g].cpu().numpy()
            out[f"m{s}"] = sinks.m.cpu().numpy() if sinks is not None else np.zeros(0)
            out[f"dm{s}"] = sinks.dm.cpu().numpy() if sinks is not None else np.zeros(0)
        torch.cuda.synchronize()
        dist.barrier()                                   # nobody frees slab memory a neighbour may still be mapped to mid-step
        ctx.close()
        np.savez(os.path.join(outdir, f"rank{rank}.npz"), **out)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_processes_put_their_ghost_planes_into_each_other(tmp_path, world):
    mode = subprocess.run(["nvidia-smi", "--query-gpu=compute_mode", "--format=csv,noheader", "--id=0"],
                          capture_output=True, text=True).stdout.strip()
    if mode and mode != "Default":
        pytest.skip(f"GPU 0 is in compute mode {mode!r}: two processes cannot share it")
    import torch.multiprocessing as mp

    from tests import parity
    port = _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r = [np.load(os.path.join(str(tmp_path), f"rank{k}.npz")) for k in range(world)]
    w = workload(world)
    o = parity.make_oracle(w)
    parity.CONTEXT["test"] = f"{world}_processes_peer_put"
    for s in range(STEPS):
        o.step(w.dt)
        got = {f: np.concatenate([r[k][f"{f}{s}"] for k in range(world)], axis=0) for f in ("rho", "mx", "my", "mz", "etot", "eint")}
        m = np.zeros(w.sinks.n)
        dm = np.zeros(w.sinks.n)
        for k in range(world):
            m[r[k]["sel_k"]] = r[k][f"m{s}"]
            dm[r[k]["sel_k"]] = r[k][f"dm{s}"]
        if s == 0:
            parity.close_strict(got["rho"], o.state.rho, "rho")
            parity.close_strict(m, o.sinks.m, "sink m")
            parity.close_strict(dm, o.sink_diag["dm"], "sink dm")
        for f, ref in (("rho", o.state.rho), ("etot", o.state.etot)):
            assert np.all(np.abs(got[f] - ref) <= 1e-9 * np.abs(ref)), f"{f}, step {s}"
        for f, ref in (("mx", o.state.mx), ("my", o.state.my), ("mz", o.state.mz)):
            assert np.all(np.abs(got[f] - ref) <= 1e-9 * (np.abs(ref) + np.abs(o.state.rho))), f"{f}, step {s}"
        assert np.all(np.abs(m - o.sinks.m) <= 1e-9 * np.abs(o.sinks.m)), f"sink m, step {s}"
    # sinks at the cuts really used the other rank's cells
    h = N // world
    near = np.min(np.abs(w.sinks.z[:, None] - np.array([float(h * r) for r in range(world + 1)])[None, :]), axis=1) < 3.0
    assert near.sum() >= 2 and np.all(o.sink_diag["dm"][near] > 0)
    V = float(w.params["dx"]) ** 3
    mass = V * got["rho"].sum() + m.sum()
    mass0 = V * w.state.rho.sum() + w.sinks.m.sum()
    assert abs((mass - mass0) - STEPS * w.sne.m_ej.sum()) <= 1e-12 * mass
    parity.dump_margins()
