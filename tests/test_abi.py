"""The C-ABI boundary without a GPU: the library builds for sm_100a, loads, and exports every
symbol include/genga.h declares; host-side argument checking; no compute call is made."""
import ctypes
import os
import re
import subprocess

import pytest

from conftest import ROOT
from paper_2309_08217_b200 import binding, build


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "genga.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(genga_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_all_exported(lib):
    syms = declared_symbols()
    assert len(syms) >= 20
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in genga.h but not exported"
    assert sorted(binding.SYMBOLS) == syms


def test_params_struct_matches_header(lib):
    # field order and count of genga_params in the header == the ctypes mirror
    text = open(os.path.join(ROOT, "include", "genga.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} genga_params;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        for part in decl.split(","):
            names.append(re.findall(r"[A-Za-z_0-9]+", part)[-1])
    assert names == [f[0] for f in binding.GengaParams._fields_]


def test_defaults_and_workspace_size(lib):
    p = binding.default_params()
    assert abs(p.G - 0.01720209895 ** 2) < 1e-20 and p.M_star == 1.0
    assert (p.n1, p.n2, p.pair_rule, p.v_is_heliocentric) == (3.0, 0.0, binding.PAIR_MUTUAL_HILL, 1)
    sizes = [lib.genga_workspace_bytes(n, ctypes.byref(p)) for n in (0, 1, 512, 513, 40000)]
    assert all(s > 0 and s % 256 == 0 for s in sizes)
    assert sizes == sorted(sizes) and sizes[3] > sizes[2]
    assert lib.genga_workspace_bytes(-1, ctypes.byref(p)) == 0


def test_argument_errors_without_device(lib):
    p = binding.default_params()
    h = ctypes.c_void_p(0)
    assert lib.genga_create(ctypes.byref(h), -1, None, None, None, ctypes.byref(p)) == binding.EINVAL
    assert lib.genga_create(None, 4, None, None, None, ctypes.byref(p)) == binding.EINVAL
    # no workspace given
    assert lib.genga_create(ctypes.byref(h), 4, None, None, None, ctypes.byref(p)) == binding.ENOMEM
    assert lib.genga_kick(None, 1.0, 0) == binding.EINVAL
    assert lib.genga_drift(None, 1.0) == binding.EINVAL
    assert lib.genga_step(None, 1.0, 0) == binding.EINVAL
    assert lib.genga_destroy(None) == binding.EINVAL
    assert lib.genga_strerror(binding.ECAPACITY).decode().startswith("encounter")
    assert b"sm_100a" in lib.genga_version()


def test_binding_refuses_to_run_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(binding.GengaError):
        binding.Genga(torch.zeros(2, dtype=torch.float64), torch.zeros(2, 3, dtype=torch.float64),
                      torch.zeros(2, 3, dtype=torch.float64))


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2309_08217_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "genga_oracle" not in src, f


def test_params_struct_layout_matches_the_c_compiler(tmp_path):
    # sizeof and every offsetof of genga_params as gcc lays the header out == the ctypes mirror (types and padding,
    # not just names); the header must also compile as plain C
    fields = [f[0] for f in binding.GengaParams._fields_]
    src = tmp_path / "layout.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "genga.h"\nint main(void) {\n'
                   '  printf("%zu\\n", sizeof(genga_params));\n'
                   + "".join(f'  printf("%zu\\n", offsetof(genga_params, {f}));\n' for f in fields)
                   + "  return 0;\n}\n")
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)],
                   check=True)
    out = [int(v) for v in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()]
    assert out[0] == ctypes.sizeof(binding.GengaParams)
    assert out[1:] == [getattr(binding.GengaParams, f).offset for f in fields]
