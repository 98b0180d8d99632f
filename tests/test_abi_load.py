"""CPU-side checks of the C-ABI boundary (no compute calls): libpsd.so builds for sm_100a,
loads, and exports every symbol include/psd.h declares; the binding mirrors the header."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols(header="psd.h", macro="PSD_API"):
    src = open(os.path.join(ROOT, "include", header)).read()
    return sorted(set(re.findall(macro + r"\s+[\w\s\*]+?\b(psd_\w+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    syms = header_symbols()
    for name in ("psd_build_tets", "psd_deposit_uniform", "psd_deposit_patches"):
        assert name in syms
    assert len(syms) >= 10


def test_library_builds_loads_and_exports_every_symbol():
    from paper_1612_09491_b200 import _build, binding
    path = _build.build()
    lib = ctypes.CDLL(path)
    syms = header_symbols()
    for name in syms:
        assert hasattr(lib, name), f"{name} declared in psd.h but not exported"
    assert sorted(binding.EXPORTS) == syms
    assert binding.version().startswith("libpsd sm_100a")


def test_peaks_library_builds_loads_and_exports_every_symbol():
    from paper_1612_09491_b200 import _build, peaks
    lib = ctypes.CDLL(_build.build(target=_build.PEAKS_LIB))
    syms = header_symbols("psd_peaks.h", "PSD_PEAKS_API")
    assert len(syms) == 4
    for name in syms:
        assert hasattr(lib, name), f"{name} declared in psd_peaks.h but not exported"
    assert sorted(peaks.EXPORTS) == syms


def test_stats_struct_matches_header_layout():
    """psd_stats: the ctypes mirror must have the same size as the C struct (checked by
    compiling a one-line C program against the header)."""
    import subprocess
    import tempfile
    from paper_1612_09491_b200 import binding
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "sz.c")
        open(c, "w").write('#include <stdio.h>\n#include "psd.h"\nint main(void){printf("%zu %zu",'
                           'sizeof(psd_stats),sizeof(psd_patch));return 0;}\n')
        exe = os.path.join(d, "sz")
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), c, "-o", exe], check=True)
        out = subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()
    assert int(out[0]) == ctypes.sizeof(binding.PsdStats)
    assert int(out[1]) == ctypes.sizeof(binding.PsdPatch)


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_1612_09491_b200 as psd
    with pytest.raises(RuntimeError):
        psd.Context(0)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1612_09491_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "psd_oracle" not in txt and "from oracle" not in txt and "import oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1612_09491_b200" not in txt and "psd_geom" not in txt, f
