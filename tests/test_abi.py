"""CPU-side checks of the boundary: libmarut.so builds for sm_100a, loads without a GPU, exports every symbol
include/marut.h declares, and refuses to compute without a device (no fallback).  No compute calls here."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "marut.h")


@pytest.fixture(scope="module")
def libpath():
    from paper_2605_26388_b200 import build

    return build.build()


def declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(marut_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_exported(libpath):
    names = declared_symbols()
    assert {"marut_mesh_create", "marut_rhs", "marut_ssprk_stage", "marut_max_dt", "marut_chem_source"} <= set(names)
    L = ctypes.CDLL(libpath)
    for n in names:
        assert hasattr(L, n), n
    from paper_2605_26388_b200 import binding

    assert sorted(binding.SYMBOLS) == names


def test_library_is_sm100a_only(libpath):
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_header_compiles_as_plain_c(tmp_path):
    c = tmp_path / "t.c"
    c.write_text('#include "marut.h"\nint main(void){ marut_mesh_desc d; (void)d; return MARUT_OK; }\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(c), "-o",
                    str(tmp_path / "t.o")], check=True)


def test_no_device_means_error_not_fallback(libpath):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2605_26388_b200 as mb
    import workloads as wl

    c = wl.make_case("c1", cells=2)
    with pytest.raises(mb.MarutError) as e:
        mb.MarutMesh(c.mesh)
    assert e.value.status == 3 and "no CPU fallback" in str(e.value)


def test_product_never_touches_oracle():
    """the package and bench.py's CUDA arm import nothing from oracle/ (and oracle/ nothing from the package)"""
    pkg = os.path.join(ROOT, "paper_2605_26388_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "marut_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2605_26388_b200" not in txt and "from paper_2605_26388_b200" not in txt, f
            assert "csrc/" not in txt and '#include "marut' not in txt.replace('#include "marut_oracle', ""), f


def test_desc_struct_layout_matches_binding():
    """offsets of marut_mesh_desc as gcc lays them out == the ctypes mirror"""
    from paper_2605_26388_b200 import binding

    fields = [n for n, _ in binding._Desc._fields_]
    prog = '#include <stdio.h>\n#include <stddef.h>\n#include "marut.h"\nint main(void){' + "".join(
        f'printf("%zu\\n", offsetof(marut_mesh_desc, {n}));' for n in fields) + 'printf("%zu\\n", sizeof(marut_mesh_desc));return 0;}'
    import tempfile

    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "o.c"), "w").write(prog)
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), os.path.join(d, "o.c"), "-o", os.path.join(d, "o")], check=True)
        out = subprocess.run([os.path.join(d, "o")], capture_output=True, text=True).stdout.split()
    offs = [int(x) for x in out]
    assert offs[:-1] == [getattr(binding._Desc, n).offset for n in fields]
    assert offs[-1] == ctypes.sizeof(binding._Desc)
    assert np.dtype(np.int32).itemsize == ctypes.sizeof(ctypes.c_int)
