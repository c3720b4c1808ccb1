"""CPU-side checks of the boundary: the in-tree CUDA library builds/loads and exports every function that
include/dualip.h declares; the ctypes mirrors match the C structs; no compute call is made (no GPU here)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "dualip.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dualip_[a-z_]+)\s*\(", src)))


def test_header_declares_the_boundary_calls():
    names = _declared_functions()
    for need in ("dualip_create", "dualip_grad", "dualip_solve", "dualip_set_c", "dualip_get_info",
                 "dualip_destroy", "dualip_strerror", "dualip_opts_default"):
        assert need in names


def test_library_exports_every_declared_symbol():
    import __graft_entry__ as ge
    ge.build()
    import paper_2606_07777_b200 as pkg
    lib = pkg.load_library()
    for name in _declared_functions():
        assert hasattr(lib, name), name
    assert set(_declared_functions()) == set(pkg.EXPORTED_SYMBOLS)


def test_struct_mirrors_match_the_header():
    import paper_2606_07777_b200 as pkg
    assert ctypes.sizeof(pkg.Scalars) == 6 * 8
    o = pkg.binding.make_opts()
    assert (o.projection, o.p0, o.reduction, o.borrow, o.validate, o.momentum) == (0, 1.0, 0, 0, 1, 1)
    # sizes and field offsets as gcc lays out include/dualip.h, against the ctypes mirrors
    import subprocess, tempfile
    fields = {"dualip_opts": ["projection", "p0", "reduction", "use_graph", "tuning", "precondition", "step_rule", "eta_min", "eta_max"],
              "dualip_info": ["I", "L", "group_lanes", "smem_bytes", "fix_scale_s", "streaming", "ntiles", "grad_kernel_count",
                              "precondition", "L_step", "duals", "lambda_lo_smem", "checked_build", "checks_failed", "long_rows", "long_row_threshold"],
              "dualip_scalars": ["g", "r_2", "gap"], "dualip_trace": ["capacity", "lambda", "eta"],
              "dualip_tuning": ["direct_kernel", "stages", "tile_units", "lambda_plan", "step_deal"]}
    src = '#include <stdio.h>\n#include <stddef.h>\n#include "dualip.h"\nint main(void){\n'
    for st, fl in fields.items():
        src += f'printf("{st} %zu\\n", sizeof({st}));\n'
        for f in fl:
            src += f'printf("{st}.{f} %zu\\n", offsetof({st}, {f}));\n'
    src += "return 0;}\n"
    with tempfile.TemporaryDirectory() as td:
        cpath, exe = os.path.join(td, "abi.c"), os.path.join(td, "abi")
        open(cpath, "w").write(src)
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", exe, cpath])
        got = dict(line.split() for line in subprocess.check_output([exe]).decode().splitlines())
    mirrors = {"dualip_opts": pkg.Opts, "dualip_info": pkg.Info, "dualip_scalars": pkg.Scalars, "dualip_trace": pkg.binding._Trace,
               "dualip_tuning": pkg.binding.Tuning}
    rename = {"lambda": "lam"}
    for st, fl in fields.items():
        assert int(got[st]) == ctypes.sizeof(mirrors[st]), st
        for f in fl:
            assert int(got[f"{st}.{f}"]) == getattr(mirrors[st], rename.get(f, f)).offset, f"{st}.{f}"
    lib = pkg.load_library()
    assert lib.dualip_strerror(0) == b"ok" and lib.dualip_strerror(-3).startswith(b"duplicate")


def test_argument_errors_need_no_gpu():
    """EINVAL is decided before any CUDA call; everything else fails loudly with ECUDA on a GPU-less host
    (no CPU fallback)."""
    import torch
    import paper_2606_07777_b200 as pkg
    rp = np.array([0, 2], dtype=np.int64); idx = np.array([0, 1], dtype=np.int32)
    c = np.array([-1, -.5], dtype=np.float32); a = np.ones(2, dtype=np.float32); b = np.ones(2, dtype=np.float32)
    with pytest.raises(pkg.DualipError) as e:
        pkg.Problem.create(1, 0, 1, rp, idx, c, a, b)
    assert e.value.code == -1
    with pytest.raises(pkg.DualipError) as e:
        pkg.Problem.create(1, 2, 9, rp, idx, c, a, b)
    assert e.value.code == -1
    with pytest.raises(pkg.DualipError) as e:
        pkg.Problem.create(1, 2, 1, rp, idx, c, a, b, pkg.binding.make_opts(projection=7))
    assert e.value.code == -1
    if not torch.cuda.is_available():
        with pytest.raises(pkg.DualipError) as e:
            pkg.Problem.create(1, 2, 1, rp, idx, c, a, b)
        assert e.value.code == -5


def test_product_never_imports_the_oracle():
    """The CUDA path and the oracle share no code and neither imports the other."""
    for base, _, files in os.walk(os.path.join(ROOT, "paper_2606_07777_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(base, f)).read()
                assert "oracle" not in txt.lower() or f == "__init__.py" and "import oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2606_07777_b200" not in txt and "from paper_2606_07777_b200" not in txt
            assert "#include \"dualip" not in txt.replace("dualip_oracle", "")
