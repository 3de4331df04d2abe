"""CPU-side checks of the boundary: the C-ABI library builds, loads, exports every symbol that
include/nsm.h declares, and the ctypes structs match the C layout.  No compute calls."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2210_13641_b200 import build
    build.build()
    import paper_2210_13641_b200 as nsm
    return nsm.load_library()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "nsm.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nsm_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    import paper_2210_13641_b200 as nsm
    syms = declared_symbols()
    assert len(syms) >= 18
    for s in syms:
        assert hasattr(lib, s), s
    assert sorted(nsm.EXPORTS) == syms


def test_struct_layouts_match_c(lib, tmp_path):
    """sizeof/offsetof from a C program compiled against include/nsm.h vs the ctypes mirror."""
    import paper_2210_13641_b200.binding as B
    prog = tmp_path / "layout.c"
    fields_cfg = [n for n, _ in B.NsmFieldConfig._fields_]
    fields_b = [n for n, _ in B.NsmRayBatch._fields_]
    fields_s = [n for n, _ in B.NsmStepStats._fields_]
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "nsm.h"', 'int main(void){']
    fields_mc = [n for n, _ in B.NsmMarchConfig._fields_]
    fields_mr = [n for n, _ in B.NsmMarchResult._fields_]
    for typ, fs in (("nsm_field_config", fields_cfg), ("nsm_ray_batch", fields_b), ("nsm_step_stats", fields_s),
                    ("nsm_march_config", fields_mc), ("nsm_march_result", fields_mr)):
        lines.append(f'printf("%zu\\n", sizeof({typ}));')
        for f in fs:
            lines.append(f'printf("%zu\\n", offsetof({typ}, {f}));')
    lines.append("return 0;}")
    prog.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(prog), "-o", str(exe)], check=True)
    vals = [int(x) for x in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    want = []
    for cls in (B.NsmFieldConfig, B.NsmRayBatch, B.NsmStepStats, B.NsmMarchConfig, B.NsmMarchResult):
        want.append(C.sizeof(cls))
        want += [getattr(cls, n).offset for n, _ in cls._fields_]
    assert vals == want


def test_no_gpu_means_loud_failure(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_2210_13641_b200 as nsm
    from workloads import configs
    with pytest.raises(RuntimeError):
        nsm.Field(configs.config1().field)
    # the C entry point itself refuses too (no CPU fallback)
    cfg = nsm.make_config(configs.config1().field)
    h = C.c_void_p()
    assert lib.nsm_create_field(C.byref(cfg), None, C.byref(h)) == 3   # NSM_ERR_CUDA
    assert b"no CPU fallback" in lib.nsm_last_error() or b"CUDA" in lib.nsm_last_error()


def test_version_and_error_strings(lib):
    assert lib.nsm_version().startswith(b"nsm")
    cfg = __import__("paper_2210_13641_b200").make_config(__import__("workloads.configs", fromlist=["x"]).config1().field)
    cfg.n_features = 3
    h = C.c_void_p()
    assert lib.nsm_create_field(C.byref(cfg), None, C.byref(h)) == 1   # NSM_ERR_INVALID_ARG, validated before CUDA
    assert b"n_features" in lib.nsm_last_error()


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2210_13641_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "nsm_oracle" not in txt, fn
