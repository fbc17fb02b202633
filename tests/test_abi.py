"""The C-ABI library builds, loads and exports every symbol include/pasta.h declares (no GPU needed),
validates arguments before touching the device, and fails loudly without one."""
import ctypes as C
import os
import re

import pytest

import paper_1412_8502_b200 as pasta
from paper_1412_8502_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "pasta.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pasta_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    lib = pasta.load()
    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), "libpasta_b200.so does not export %s" % n
    assert sorted(binding.SIGNATURES) == names


def test_params_struct_layout_and_defaults():
    p = pasta.default_params()
    assert p.struct_size == C.sizeof(pasta.Params)
    assert (p.a, p.b, p.c, p.Lambda) == (110.0, -26.0, 24.0, 1.25)  # Table I
    assert p.alpha_hbarc == 1.44 and p.lambda_ == 10.0 and p.mass == 939.0 and p.r_c == 20.0
    assert p.scale_per_step == 1.0 and p.thermostat_interval == 0 and p.energy_every_step == 1
    assert pasta.load().pasta_version().startswith(b"pasta-b200")


def test_argument_validation_happens_before_any_device_work():
    lib = pasta.load()
    h = C.c_void_p()
    p = pasta.default_params()
    bad = [
        dict(N=0), dict(Y_P=1.5), dict(Y_P=-0.1), dict(density=0.0), dict(T=-1.0),
        dict(N=2048, density=0.05),  # L/2 = 17.2 < r_c = 20  (nearest image ambiguous)
    ]
    base = dict(N=51200, Y_P=0.4, density=0.08, T=1.0)
    for b in bad:
        a = dict(base, **b)
        rc = lib.pasta_create(C.byref(h), a["N"], a["Y_P"], a["density"], a["T"], C.byref(p), 1, None)
        assert rc == -1 and h.value is None, (b, lib.pasta_last_error())
    assert b"r_c" in lib.pasta_last_error()
    for field, val in (("r_c", 0.0), ("Lambda", 0.0), ("mass", -1.0), ("scale_per_step", 0.0),
                       ("thermostat_interval", -1), ("cell_subdiv", 0), ("struct_size", 8)):
        q = pasta.default_params()
        setattr(q, field, val)
        assert lib.pasta_create(C.byref(h), 51200, 0.4, 0.08, 1.0, C.byref(q), 1, None) == -1
    q = pasta.default_params(r_nuc=11.5, coulomb_all_pairs=1)  # the paper's Coulomb sum needs a 120 fm box (D26); L = 86 fm here
    assert lib.pasta_create(C.byref(h), 51200, 0.4, 0.08, 1.0, C.byref(q), 1, None) == -1
    assert b"120" in lib.pasta_last_error()
    assert lib.pasta_create(None, 51200, 0.4, 0.08, 1.0, C.byref(p), 1, None) == -1
    assert lib.pasta_step(None, 1, 2.0) == -1 and lib.pasta_destroy(None) == 0
    assert lib.pasta_launch_count(None) == 0


def test_no_cpu_fallback_without_a_device():
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    lib = pasta.load()
    h = C.c_void_p()
    p = pasta.default_params()
    rc = lib.pasta_create(C.byref(h), 51200, 0.4, 0.08, 1.0, C.byref(p), 1, None)
    assert rc == -2 and h.value is None  # PASTA_ECUDA
    assert b"no CPU fallback" in lib.pasta_last_error()
    with pytest.raises(RuntimeError):
        pasta.Sim(2048, 0.3, 0.05, 1.0)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1412_8502_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle|#include.*oracle|oracle[./]", text, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            assert "paper_1412_8502_b200 import" not in open(os.path.join(ROOT, "oracle", f)).read()
