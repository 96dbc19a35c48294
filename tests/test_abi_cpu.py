"""-m "not gpu": the C-ABI library builds, loads and exports every symbol include/nsgpu.h declares;
create fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes
import os

import numpy as np
import pytest

from paper_2509_13307_b200 import build, nsgpu, workloads as W
from tests.util import header_exports


@pytest.fixture(scope="module")
def libpath():
    return build.build()


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    names = header_exports()
    assert set(names) == set(nsgpu.EXPORTS)
    for n in names:
        assert hasattr(L, n), n


def test_binding_struct_sizes_match_c_layout(tmp_path):
    """compile a C program against include/nsgpu.h (the header is plain C) and compare sizeof with ctypes."""
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    src = tmp_path / "sz.c"
    src.write_text('#include <stdio.h>\n#include "nsgpu.h"\nint main(void){printf("%zu %zu %zu %zu %zu\\n",'
                   'sizeof(nsgpu_prior1d),sizeof(nsgpu_emulator),sizeof(nsgpu_theory),sizeof(nsgpu_run_opts),'
                   'sizeof(nsgpu_result));return 0;}\n')
    exe = tmp_path / "sz"
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(root, "include"), str(src), "-o", str(exe)])
    got = [int(x) for x in subprocess.check_output([str(exe)]).split()]
    want = [ctypes.sizeof(t) for t in (nsgpu._Prior1d, nsgpu._Emulator, nsgpu._Theory, nsgpu._RunOpts, nsgpu._Result)]
    assert got == want


def test_create_without_gpu_fails_loudly(libpath):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    wl = W.toy_identity(D=3)
    with pytest.raises(nsgpu.NsgpuError) as e:
        nsgpu.Context(wl, max_batch=8)
    assert e.value.status == nsgpu.ECUDA and "no CPU fallback" in str(e.value)


def test_product_does_not_import_the_oracle():
    import subprocess, sys
    code = ("import sys; import paper_2509_13307_b200.nsgpu, paper_2509_13307_b200.workloads, "
            "paper_2509_13307_b200.build; assert not any(m == 'oracle' or m.startswith('oracle.') for m in sys.modules)")
    subprocess.check_call([sys.executable, "-c", code], cwd=os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def test_binding_flag_constants_match_the_header():
    """the flag bits the binding ORs into nsgpu_create are the header's #defines"""
    import re
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    hdr = open(os.path.join(root, "include", "nsgpu.h")).read()
    defs = {m.group(1): int(m.group(2)) for m in re.finditer(r"#define\s+NSGPU_(\w+)\s+(\d+)u\b", hdr)}
    for name in ("MLP_AUTO", "MLP_SIMT", "MLP_TC", "CHI2_STREAMED", "CHI2_TILED", "MLP_CLUSTER", "MLP_NO_CLUSTER",
                 "SHEAR_STREAM", "NO_PDL"):
        assert getattr(nsgpu, name) == defs[name], name
    bits = [defs[n] for n in defs if defs[n]]
    assert len(set(bits)) == len(bits) and all(b & (b - 1) == 0 for b in bits)      # distinct single bits


def test_examples_import_without_the_oracle_and_parse_their_arguments():
    import subprocess, sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for mod in ("model_comparison", "cmb_evidence"):
        out = subprocess.run([sys.executable, "-m", f"paper_2509_13307_b200.examples.{mod}", "--help"], cwd=root,
                             capture_output=True, text=True)
        assert out.returncode == 0 and "--seeds" in out.stdout, out.stderr
    code = ("import sys; import paper_2509_13307_b200.examples.model_comparison, paper_2509_13307_b200.examples.cmb_evidence; "
            "assert not any(m == 'oracle' or m.startswith('oracle.') for m in sys.modules)")
    subprocess.check_call([sys.executable, "-c", code], cwd=root)
