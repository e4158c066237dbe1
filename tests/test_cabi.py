"""The C-ABI library loads without a GPU and exports every symbol include/md_b200.h declares.
No compute call is made here (there is no CPU fallback to call)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2003_14061_b200.build import build
    build()
    import paper_2003_14061_b200 as md
    return md, md.load_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "md_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"MD_API\s+[^;(]*?\b(md_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported_and_bound(lib):
    md, L = lib
    syms = declared_symbols()
    assert len(syms) >= 20 and "md_step" in syms and "md_create" in syms
    for s in syms:
        assert getattr(L, s) is not None, s
    assert sorted(md.EXPORTS) == syms          # the binding declares exactly the header's calls


def test_no_other_symbols_leak(lib):
    import subprocess
    md, _ = lib
    out = subprocess.run(["nm", "-D", "--defined-only", md.LIB_PATH], capture_output=True, text=True).stdout
    names = [l.split()[-1] for l in out.splitlines() if " T " in l]
    assert sorted(names) == declared_symbols()


def test_calls_that_need_no_device(lib):
    md, L = lib
    assert b"sm_100a" in L.md_version()
    from paper_2003_14061_b200.binding import _Params
    p = _Params()
    L.md_params_default(ctypes.byref(p))
    assert p.temperature == 1.0 and p.device == -1 and p.lattice == 0


def test_struct_sizes_match_header(lib):
    """ctypes mirrors of md_params / md_energy / md_info have the C layout (checked against a compiled probe)."""
    import subprocess
    import tempfile
    from paper_2003_14061_b200.binding import _Energy, _Info, _Params, _Peaks, _PushoffOpts, _PushoffReport
    src = ('#include <stdio.h>\n#include "md_b200.h"\nint main(){printf("%zu %zu %zu %zu %zu %zu\\n",'
           'sizeof(md_params),sizeof(md_energy),sizeof(md_info),sizeof(md_pushoff_opts),sizeof(md_pushoff_report),'
           'sizeof(md_peaks));return 0;}\n')
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "p.c")
        open(c, "w").write(src)
        exe = os.path.join(d, "p")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe], check=True)
        sizes = [int(x) for x in subprocess.run([exe], capture_output=True, text=True).stdout.split()]
    assert sizes == [ctypes.sizeof(x) for x in (_Params, _Energy, _Info, _PushoffOpts, _PushoffReport, _Peaks)]


def test_product_fails_loudly_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    md, _ = lib
    with pytest.raises(md.MDError):
        md.MDSystem(4096, 1.12, 0.4, 0.005, density=0.8)


def test_product_does_not_import_oracle():
    """Nothing under the product package imports, includes, links or loads anything from oracle/."""
    pkg = os.path.join(ROOT, "paper_2003_14061_b200")
    bad = re.compile(r"(^\s*(from|import)\s+oracle\b|#include\s*[<\"][^>\"]*oracle|md_oracle|libmd_oracle|orc_[a-z_]+\()", re.M)
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h")):
                assert not bad.search(open(os.path.join(dp, f)).read()), f
