"""The boundary without a GPU: libarc_b200.so loads, exports every function include/arc.h declares, the ctypes
mirrors of its structs have the C compiler's sizes and offsets, the calls that need no device answer, and the
ones that do fail loudly (there is no CPU fallback).  No compute call is made here."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest

from paper_1807_07094_b200 import arc, build as arc_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "arc.h")


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(arc_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    arc_build.build()
    return arc.lib()


def test_every_declared_entry_point_is_exported_and_bound(lib):
    names = _declared_functions()
    assert len(names) >= 19
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in include/arc.h but not exported by libarc_b200.so"
        assert n in arc.EXPORTS, f"{n} is declared in include/arc.h but missing from the binding's EXPORTS"
        assert hasattr(arc, n), f"the Python binding has no function named {n}"
    assert sorted(arc.EXPORTS) == names


def test_library_links_only_the_cuda_runtime(lib):
    out = subprocess.run(["ldd", arc.LIB_PATH], capture_output=True, text=True).stdout
    out = re.sub(r"\(0x[0-9a-f]+\)", "", out)             # load addresses are random hex: "c10" may turn up in one
    for forbidden in ("torch", "python", "oracle", "c10", "cublas", "nccl"):
        assert forbidden not in out.lower(), out


def test_struct_layouts_match_the_c_compiler(tmp_path):
    """sizeof / offsetof of every public struct, from gcc on include/arc.h, against the ctypes mirrors"""
    structs = {"arc_params": arc.arc_params, "arc_rates": arc.arc_rates, "arc_stats": arc.arc_stats,
               "arc_raylog": arc.arc_raylog}
    lines = ['#include <stdio.h>', '#include <stddef.h>', f'#include "{HEADER}"', "int main(void){"]
    for sname, ct in structs.items():
        lines.append(f'printf("{sname} %zu\\n", sizeof({sname}));')
        for fname, _ in ct._fields_:
            cname = "async" if fname == "async_" else fname
            lines.append(f'printf("{sname}.{fname} %zu\\n", offsetof({sname}, {cname}));')
    lines.append("return 0;}")
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-std=c99", "-o", str(exe), str(src)])
    got = dict(l.split() for l in subprocess.check_output([str(exe)], text=True).splitlines())
    for sname, ct in structs.items():
        assert int(got[sname]) == C.sizeof(ct), sname
        for fname, _ in ct._fields_:
            assert int(got[f"{sname}.{fname}"]) == getattr(ct, fname).offset, f"{sname}.{fname}"


def test_enums_match_the_header():
    src = open(HEADER).read()
    for name in ("ARC_F32", "ARC_F64", "ARC_HOST", "ARC_DEVICE", "ARC_OK", "ARC_EINVAL", "ARC_ENOMEM", "ARC_ECUDA",
                 "ARC_ESTATE", "ARC_EOVERFLOW", "ARC_END_SPLIT", "ARC_END_DEPLETED", "ARC_END_ESCAPED",
                 "ARC_DEPOSIT_AUTO", "ARC_DEPOSIT_RED", "ARC_DEPOSIT_AGG", "ARC_DEPOSIT_QUAD",
                 "ARC_GEOM_NONE", "ARC_GEOM_FC", "ARC_GEOM_FC_SECONDARY", "ARC_GEOM_FC2", "ARC_DT_NEUTRAL", "ARC_DT_INTENSITY"):
        m = re.search(rf"\b{name}\s*=\s*(-?\d+)", src)
        assert m, name
        assert int(m.group(1)) == getattr(arc, name), name
    for name in ("ARC_MAX_BINS", "ARC_MAX_LEVEL"):
        m = re.search(rf"#define\s+{name}\s+(\d+)", src)
        assert int(m.group(1)) == getattr(arc, name)


def test_calls_that_need_no_device(lib):
    assert "sm_100a" in arc.arc_version()
    p = arc.arc_default_params()
    assert (p.l0, p.Lmax, p.Phi, p.tau_term, p.eps_sub) == (1, 13, 3.0, 30.0, 0.1)      # PAPER.md:45, :154; G6-G7
    assert lib.arc_destroy(None) in (arc.ARC_OK, arc.ARC_EINVAL)
    assert lib.arc_trace(None, 0, None) == arc.ARC_EINVAL
    assert lib.arc_update_chemistry(None, C.c_double(1.0)) == arc.ARC_EINVAL
    assert lib.arc_pix2vec(None, None, -1, None) == arc.ARC_EINVAL
    assert lib.arc_pix2vec(None, None, 0, None) == arc.ARC_OK


def test_bad_arguments_are_rejected_before_any_device_work():
    for N, box, dt in ((0, 1.0, arc.ARC_F32), (2048, 1.0, arc.ARC_F32), (8, -1.0, arc.ARC_F64), (8, 1.0, 7)):
        with pytest.raises(arc.ArcError) as e:
            arc.arc_create_grid(N, box, dt)
        assert e.value.code == arc.ARC_EINVAL


def test_no_cpu_fallback_without_a_device():
    """on a box without a GPU the product path must fail loudly, never compute on the host"""
    import torch
    if torch.cuda.is_available():
        pytest.skip("this box has a GPU")
    with pytest.raises(arc.ArcError) as e:
        arc.arc_create_grid(8, 1.0, arc.ARC_F64)
    assert e.value.code == arc.ARC_ECUDA


def test_missing_library_raises_instead_of_falling_back(tmp_path):
    code = ("import sys; sys.path.insert(0, %r)\n"
            "from paper_1807_07094_b200 import arc\n"
            "arc.LIB_PATH = %r\n"
            "try:\n    arc.lib()\nexcept ImportError as e:\n    print('RAISED', e)\n" % (ROOT, str(tmp_path / "nope.so")))
    out = subprocess.check_output([sys.executable, "-c", code], text=True)
    assert "RAISED" in out and "no CPU fallback" in out


def test_product_package_never_touches_the_oracle():
    pkg = os.path.join(ROOT, "paper_1807_07094_b200")
    for dirpath, _, files in os.walk(pkg):
        if "build" in os.path.relpath(dirpath, pkg).split(os.sep):
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "arc_oracle" not in text, f
    otext = open(os.path.join(ROOT, "oracle", "oracle.py")).read() + open(os.path.join(ROOT, "oracle", "arc_oracle.c")).read()
    assert "libarc_b200" not in otext and "paper_1807_07094_b200.arc" not in otext
    assert not re.search(r'#include\s+"[^"]*arc\.h"', otext)
