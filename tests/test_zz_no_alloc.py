"""pm_gravity_deposit_noalloc (include/pm.h): the entry point that allocates nothing -- its ghost-zoned accumulation mesh is a
file-scope __device__ array of the library -- against the existing path, pm_gravity_deposit on a ctx, on the same seeded
inputs.  Both run the same kernels; only the order of the fp64 atomic additions differs, so the tolerance is the one of
tests/test_gpu_gravity.py: 1e-12 relative per cell, cell membership exact, total mass to 1e-13.

The file is named to be collected last: the array is shared by every call of the process and keeps the last call's contents,
so the test must pass alone in a fresh process and after all the other tests."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2509_18261_b200 import inputs, pm

DEV = "cuda:0"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def existing_path(w, with_gas):
    ctx = pm.Context(w.params, device=DEV)
    out = torch.empty(w.rho_gas.shape, dtype=torch.float64, device=DEV)
    ctx.pm_gravity_deposit(dev(w.rho_gas) if with_gas else None, dev(w.x), dev(w.y), dev(w.z), dev(w.m), out)
    ctx.pm_check()
    ctx.close()
    return out.cpu().numpy()


def compare(got, ref, w, with_gas):
    assert np.all(np.abs(got - ref) <= 1e-12 * np.abs(ref) + 1e-300), "rho_tot against pm_gravity_deposit"
    if not with_gas:
        assert np.array_equal(got != 0, ref != 0), "cell membership"
    V = float(w.params["dx"]) ** 3
    want = (float(w.rho_gas.sum()) * V if with_gas else 0.0) + float(w.m.sum())
    assert abs(float(got.sum()) * V - want) <= 1e-13 * want, "total mass"


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_ctx_path():
    # call 1: the largest mesh the array holds (64^3), gas + 200 000 particles; call 2: a smaller, odd, non-cubic mesh with an
    # offset origin and dx != 1, particles only -- it runs on top of what call 1 left in the array
    wa = inputs.gravity_workload(64, 200_000)
    wb = inputs.gravity_workload(36, 30_000, seed_index=7, shape=(41, 36, 50), dx=0.25, x0=(-3.0, 1.5, 10.0))
    ref_a, ref_b = existing_path(wa, True), existing_path(wb, False)

    ins_a = [dev(a) for a in (wa.rho_gas, wa.x, wa.y, wa.z, wa.m)]
    ins_b = [dev(a) for a in (wb.x, wb.y, wb.z, wb.m)]
    out_a = torch.full(wa.rho_gas.shape, np.nan, dtype=torch.float64, device=DEV)
    out_b = torch.full(wb.rho_gas.shape, np.nan, dtype=torch.float64, device=DEV)
    flag = torch.full((1,), -1, dtype=torch.int32, device=DEV)

    pm.pm_gravity_deposit_noalloc(wa.params, *ins_a, out_a, outside=flag)
    pm.pm_gravity_deposit_noalloc(wb.params, None, *ins_b, out_b)                      # straight after, same stream
    torch.cuda.synchronize()
    assert int(flag.item()) == 0
    compare(out_a.cpu().numpy(), ref_a, wa, True)
    compare(out_b.cpu().numpy(), ref_b, wb, False)

    # a third call, same shapes as the first (every kernel it launches is loaded by now): the device's free memory must not
    # move across it, and the result is again the first call's
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info(DEV)
    out_a.fill_(np.nan)
    pm.pm_gravity_deposit_noalloc(wa.params, *ins_a, out_a, outside=flag)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info(DEV)
    assert free1 == free0, "device memory was allocated or freed during the call"
    compare(out_a.cpu().numpy(), ref_a, wa, True)


@pytest.mark.gpu
def test_outside_flag_and_in_place_update():
    w = inputs.gravity_workload(24, 1000)
    gas = dev(w.rho_gas)
    flag = torch.zeros(1, dtype=torch.int32, device=DEV)
    x = w.x.copy()
    x[17] = 24.0                                                   # on the upper face: outside [x0, x0 + n dx)
    pm.pm_gravity_deposit_noalloc(w.params, gas, dev(x), dev(w.y), dev(w.z), dev(w.m), gas, outside=flag)   # in place
    assert int(flag.item()) == 1
    V = float(w.params["dx"]) ** 3
    want = float(w.rho_gas.sum()) * V + float(w.m.sum()) - float(w.m[17])          # the outsider is skipped
    assert abs(float(gas.sum().item()) * V - want) <= 1e-13 * want
    # the flag word lives in the shared array too: the next call starts from 0 again
    out = torch.empty_like(gas)
    pm.pm_gravity_deposit_noalloc(w.params, None, dev(w.x), dev(w.y), dev(w.z), dev(w.m), out, outside=flag)
    assert int(flag.item()) == 0
    # no particles: rho_tot = rho_gas
    e = torch.empty(0, dtype=torch.float64, device=DEV)
    g2 = dev(w.rho_gas)
    pm.pm_gravity_deposit_noalloc(w.params, g2, e, e, e, e, out)
    assert torch.equal(out, g2)


def test_sizes_beyond_the_array_are_refused_with_a_clear_error():
    """Argument checks come before any CUDA call: this part runs without a GPU."""
    L = pm.lib()
    x0 = (C.c_double * 3)(0.0, 0.0, 0.0)
    fake = C.c_void_p(256)                                         # never dereferenced: the call is refused first
    assert (66 + 4) * 68 * 68 <= pm.PM_NOALLOC_MAX_GHOSTED_CELLS < (67 + 4) * 69 * 69      # cubes up to 66^3 fit
    rc = L.pm_gravity_deposit_noalloc(0, None, 128, 64, 64, x0, 1.0, None, 0, None, None, None, None, fake, None)
    assert rc == pm.PM_EINVAL
    msg = L.pm_noalloc_last_error().decode()
    assert "PM_NOALLOC_MAX_GHOSTED_CELLS" in msg and str(pm.PM_NOALLOC_MAX_GHOSTED_CELLS) in msg and "128 x 64 x 64" in msg
    assert L.pm_gravity_deposit_noalloc(0, None, 2, 8, 8, x0, 1.0, None, 0, None, None, None, None, fake, None) == pm.PM_EINVAL
    assert L.pm_gravity_deposit_noalloc(0, None, 8, 8, 8, x0, 0.0, None, 0, None, None, None, None, fake, None) == pm.PM_EINVAL
    assert L.pm_gravity_deposit_noalloc(0, None, 8, 8, 8, x0, 1.0, None, -1, None, None, None, None, fake, None) == pm.PM_EINVAL
    assert L.pm_gravity_deposit_noalloc(0, None, 8, 8, 8, x0, 1.0, None, 5, None, None, None, None, fake, None) == pm.PM_EINVAL
    assert L.pm_gravity_deposit_noalloc(0, None, 8, 8, 8, None, 1.0, None, 0, None, None, None, None, fake, None) == pm.PM_EINVAL
    assert L.pm_gravity_deposit_noalloc(99, None, 8, 8, 8, x0, 1.0, None, 0, None, None, None, None, fake, None) == pm.PM_EINVAL
    # the same refusal through the Python binding (needs device tensors, so only where there is a GPU)
    if torch.cuda.is_available():
        big = {"nx": 67, "ny": 67, "nz": 67, "x0": (0.0, 0.0, 0.0), "dx": 1.0}
        out = torch.empty(67 ** 3, dtype=torch.float64, device=DEV)
        e = torch.empty(0, dtype=torch.float64, device=DEV)
        with pytest.raises(pm.PmError, match="PM_NOALLOC_MAX_GHOSTED_CELLS"):
            pm.pm_gravity_deposit_noalloc(big, None, e, e, e, e, out)
