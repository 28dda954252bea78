"""Host-side logic of bench.py on CPU: the whole-job aggregate and the max-over-ranks rule with world_size 2 (gloo).
The path itself does not shard ("replicas only"), so the only multi-rank logic is this aggregation."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = 10.0 + 5.0 * rank                      # rank 1 is the slow replica
        total = bench.reduce_max(ms, world, torch.device("cpu"))
        out[rank] = (total, bench.whole_job_value(1000, 4, world, total))
    finally:
        dist.destroy_process_group()


def test_replicas_max_over_ranks_gloo_world2():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 15.0                       # the max, on every rank
    assert res[0][1] == pytest.approx(2 * 1000 * 4 / 15e-3 / 1e6)   # units of BOTH replicas over the slowest rank's time


def test_single_rank_is_identity():
    assert bench.reduce_max(3.25, 1, None) == 3.25
    assert bench.whole_job_value(512 ** 3, 10, 1, 116.0) == pytest.approx(512 ** 3 * 10 / 0.116 / 1e6)


def test_algorithmic_bytes_dense_limits():
    """With every cell touched and every tile live the per-kernel figures are SURVEY.md 8(d)'s: apply 176 B/cell, reset +
    write-back 48 B per buffer cell, fold 3 x 48 B per ghost cell, gathers 40 / 32 B per cell; the deposit kernels carry no
    write-back (8(d) books it once, with the reset)."""
    N, Nb = 512 ** 3, 520 ** 3
    b = bench.algorithmic_bytes(N, Nb, 10 ** 5, 9 * 10 ** 5, 1.0, 1.0, 1.0)
    assert b["apply"] == 176.0 * N
    assert b["zero"] == 48.0 * Nb
    assert b["fold"] == 3 * 48.0 * (Nb - N)
    assert b["sinks"] == 40.0 * N + 80.0 * 10 ** 5 and b["sne"] == 32.0 * N + 64.0 * 9 * 10 ** 5
    b0 = bench.algorithmic_bytes(N, Nb, 0, 0, 0.0, 0.0, 0.0, 0.0, 0.0)
    assert b0["apply"] == 0.0 and b0["sne"] == 0.0 and b0["sinks"] == 0.0 and b0["zero"] == 0.0
    # SN deposit at config 5's probed cell fraction (T_SN ~ 0.48): ~2.1 GB, not the 6.4 GB of round 1's line
    assert 2.0e9 < bench.algorithmic_bytes(N, Nb, 10 ** 5, 9 * 10 ** 5, 0.55, 0.12, 0.48)["sne"] < 2.2e9


_OMP_SCRIPT = """
import sys
import numpy as np
sys.path.insert(0, {root!r})
from oracle import pm_oracle as po
from paper_2509_18261_b200 import inputs
w = inputs.scaled_mixed(40, 800, seed_index=5)
o = po.Oracle(w.params, w.state, w.sinks, w.sne, keep_abs=False, omp=True)
for _ in range(2):
    o.step(w.dt)
np.savez({out!r}, threads=po.lib_omp().orc_threads(), m=w.sinks.m, **{{f: getattr(w.state, f) for f in w.state.FIELDS}})
"""


def test_openmp_build_of_the_oracle_is_the_same_program(tmp_path):
    """bench.py's all-cores leg times oracle/pm_oracle.c compiled with -fopenmp.  The pragmas must
    not change what is computed: on a small mixed workload the two builds agree to the reorder tolerance (the OpenMP build's
    sums depend on the order of its atomic additions), conserve the same totals, and the plain build -- the parity reference --
    stays deterministic.  The OpenMP build runs in a process of its own, so that this one stays single-threaded for the
    tests that fork."""
    import hashlib
    import subprocess

    import numpy as np

    from oracle import pm_oracle as po
    from paper_2509_18261_b200 import inputs

    def run():
        w = inputs.scaled_mixed(40, 800, seed_index=5)
        o = po.Oracle(w.params, w.state, w.sinks, w.sne, keep_abs=False)
        for _ in range(2):
            o.step(w.dt)
        return w

    a, b = run(), run()
    digest = lambda w: hashlib.sha256(b"".join(getattr(w.state, f).tobytes() for f in w.state.FIELDS)).hexdigest()
    assert digest(a) == digest(b), "the plain build must not depend on anything but its inputs"
    assert po.lib().orc_threads() == 1
    out = str(tmp_path / "omp.npz")
    subprocess.check_call([sys.executable, "-c", _OMP_SCRIPT.format(root=ROOT, out=out)])
    c = np.load(out)
    assert int(c["threads"]) >= 1
    for f in a.state.FIELDS:
        x, y = getattr(a.state, f), c[f]
        assert np.all(np.abs(x - y) <= 1e-9 * np.abs(x) + 1e-12 * np.abs(x).max()), f
    assert abs(a.state.rho.sum() - c["rho"].sum()) <= 1e-12 * a.state.rho.sum()
    assert np.allclose(a.sinks.m, c["m"], rtol=1e-11, atol=0)
