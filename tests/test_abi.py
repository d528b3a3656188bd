"""The C-ABI library builds without a GPU, loads, and exports every symbol include/msm.h declares
(no compute calls here). Also: the binding lists the same names, and calls that need a device fail
with a status code instead of crashing or falling back to the CPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "msm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(msm_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2510_05961_b200 import build, msm
    build.build()
    return msm.lib()


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert len(names) >= 11
    for n in names:
        assert hasattr(lib, n), n


def test_binding_lists_the_header_names(lib):
    from paper_2510_05961_b200 import msm
    assert sorted(msm.EXPORTS) == _declared()


def test_struct_sizes_match_header():
    """ctypes mirrors of msm_params_t / msm_plan_info_t have the C layout (sizes from gcc)."""
    import subprocess
    import tempfile
    from paper_2510_05961_b200 import msm
    prog = '#include <stdio.h>\n#include "msm.h"\nint main(void){printf("%zu %zu\\n", sizeof(msm_params_t), sizeof(msm_plan_info_t));return 0;}\n'
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "s.c")
        open(c, "w").write(prog)
        exe = os.path.join(d, "s")
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe])
        a, b = (int(v) for v in subprocess.check_output([exe]).split())
    assert ctypes.sizeof(msm.Params) == a
    assert ctypes.sizeof(msm.PlanInfo) == b


def test_status_strings(lib):
    for s in range(8):
        assert lib.msm_status_string(s)


def test_argument_errors_need_no_device(lib):
    from paper_2510_05961_b200 import msm
    assert lib.msm_plan_create(None, None) == 1
    h = ctypes.c_void_p()
    assert lib.msm_plan_create(None, ctypes.byref(h)) == 1 and not h
    prm = msm.Params()
    prm.box[:] = [20.0, 20.0, 20.0]; prm.periodic[:] = [1, 1, 1]
    prm.h, prm.a, prm.p, prm.levels, prm.precision, prm.mu, prm.max_particles, prm.device = 2.0, 6.0, 5, 2, 0, -1, 8, 0
    assert lib.msm_plan_create(ctypes.byref(prm), ctypes.byref(h)) == 1       # odd order
    prm.p, prm.a = 4, 11.0
    assert lib.msm_plan_create(ctypes.byref(prm), ctypes.byref(h)) == 3       # a > L/2
    prm.a = 6.0; prm.periodic[:] = [1, 0, 0]
    assert lib.msm_plan_create(ctypes.byref(prm), ctypes.byref(h)) == 2       # one periodic axis (T4)
    assert lib.msm_evaluate(None, 0, None, None, None, None, None, None, None) == 1


def test_no_cpu_fallback_without_device(lib):
    """Without a CUDA device plan creation fails with MSM_ERR_CUDA (the product never routes
    through the oracle or any CPU path)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    from paper_2510_05961_b200 import msm
    with pytest.raises(msm.MsmError) as e:
        msm.Plan((20.0,) * 3, (1, 1, 1), 2.0, 6.0, 4, 2)
    assert e.value.status == 7


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2510_05961_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".hpp", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "msm_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "libmsm_b200" not in txt and "csrc" not in txt.replace("paper_2510_05961_b200/csrc)", ""), f
