"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol include/pm.h declares,
argument validation that needs no GPU works, and the product path fails loudly (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest
import torch

from paper_2509_18261_b200 import inputs, pm

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built():
    return pm.build()


def declared_functions():
    src = open(os.path.join(ROOT, "include", "pm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pm_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_six_entry_points():
    names = declared_functions()
    for f in ("pm_create", "pm_deposit", "pm_fold_ghosts", "pm_apply_limited", "pm_return_to_particles", "pm_destroy"):
        assert f in names


def test_library_exports_every_declared_symbol(built):
    L = C.CDLL(built)
    for name in declared_functions():
        assert hasattr(L, name), f"{name} declared in include/pm.h but not exported"
    assert sorted(pm.EXPORTS) == declared_functions()


def test_params_struct_matches_header():
    src = open(os.path.join(ROOT, "include", "pm.h")).read()
    start = src.index("typedef struct {", src.index("Plain data")) + len("typedef struct {")
    body = src[start:src.index("} pm_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        m = re.match(r"\s*(int32_t|double)\s+(.*)", decl.strip(), flags=re.S)
        if m:
            fields += [re.sub(r"\[.*\]", "", n).strip() for n in m.group(2).split(",")]
    assert fields == [f for f, _ in pm.PmParams._fields_]


def test_argument_validation_without_gpu(built):
    L = pm.lib()
    h = C.c_void_p()
    assert L.pm_create(None, 0, None, C.byref(h)) == pm.PM_EINVAL
    p = pm.make_params(inputs.default_params(8))          # 8 < 2g+1 = 9
    assert L.pm_create(C.byref(p), 0, None, C.byref(h)) == pm.PM_EINVAL
    p = pm.make_params(inputs.default_params(16))
    p.sn_nsub = 9
    assert L.pm_create(C.byref(p), 0, None, C.byref(h)) == pm.PM_EINVAL
    assert L.pm_fold_ghosts(None) == pm.PM_EINVAL
    assert L.pm_destroy(None) == pm.PM_EINVAL
    assert L.pm_gravity_deposit(None, None, 0, None, None, None, None, None) == pm.PM_EINVAL
    assert L.pm_gravity_kick(None, None, None, None, 0, None, None, None, None, None, None, 0.0, None, None, None) == pm.PM_EINVAL
    assert L.pm_drift(None, 0, None, None, None, None, None, None, 0.0) == pm.PM_EINVAL


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback(built):
    """Without a GPU the product path must fail, not compute on the CPU."""
    L = pm.lib()
    h = C.c_void_p()
    p = pm.make_params(inputs.default_params(16))
    rc = L.pm_create(C.byref(p), 0, None, C.byref(h))
    assert rc in (pm.PM_ECUDA, pm.PM_ENOMEM) and not h.value


def test_product_does_not_import_oracle():
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2509_18261_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(root, f)).read()
                assert "pm_oracle" not in txt and "import oracle" not in txt and "from oracle" not in txt, f
