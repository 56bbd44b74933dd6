"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol
include/mcdc.h declares; the binding's struct layouts match the header."""
import ctypes as C
import os
import re
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    import __graft_entry__ as ge
    ge.build()
    from paper_2305_07636_b200 import binding
    L = binding.load_library()
    header = open(os.path.join(ROOT, "include", "mcdc.h")).read()
    declared = set(re.findall(r"\b(mcdc_[a-z_]+)\s*\(", header))
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    for name in declared:
        assert hasattr(L, name), name


def test_struct_layouts_match_header(tmp_path):
    from paper_2305_07636_b200 import binding as b
    src = tmp_path / "sz.c"
    src.write_text('#include <stdio.h>\n#include "mcdc.h"\nint main(void){printf("%zu %zu %zu %zu %zu %zu %zu\\n",'
                   "sizeof(mcdc_materials),sizeof(mcdc_geometry),sizeof(mcdc_source),sizeof(mcdc_tally_mesh),"
                   "sizeof(mcdc_census),sizeof(mcdc_run_params),sizeof(mcdc_counters));return 0;}\n")
    exe = tmp_path / "sz"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(src)], check=True)
    sizes = [int(x) for x in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    mine = [C.sizeof(t) for t in (b.Materials, b.Geometry, b.Source, b.TallyMesh, b.Census, b.RunParams, b.Counters)]
    assert sizes == mine


def test_no_gpu_means_loud_failure():
    import torch
    if torch.cuda.is_available():
        return
    import pytest
    import mcdc_inputs as mi
    from paper_2305_07636_b200 import Problem, McdcError
    with pytest.raises((McdcError, RuntimeError)):
        Problem(mi.config1()).run()
