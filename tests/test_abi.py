"""The C-ABI library builds, loads and exports every symbol include/md.h declares (no compute calls: no GPU here)."""
import ctypes
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "md.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(md_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    import paper_1212_6332_b200 as md
    L = md.lib()
    names = declared_symbols()
    assert {"md_create", "md_build_neighbors", "md_compute_forces", "md_step", "md_workspace_bytes"} <= set(names)
    for n in names:
        assert hasattr(L, n), n
    assert b"sm_100a" in L.md_version()
    assert L.md_strerror(-2).decode().startswith("box")
    assert [L.md_kernel_name(k).decode() for k in range(len(md.KERNEL_CLASSES))] == list(md.KERNEL_CLASSES)


def test_workspace_query_and_argument_errors_need_no_gpu():
    import paper_1212_6332_b200 as md
    import workloads
    L = md.lib()
    w = workloads.config(0)
    d = md.MdDesc()
    d.n_atoms, d.n_boxes, d.n_types = w.n_atoms, 1, 1
    d.box = (ctypes.c_double * 3)(*w.box)
    d.cutoff, d.skin, d.pot_kind, d.taper_on = 4.9, 0.3, 0, 4.4
    n = ctypes.c_size_t()
    assert L.md_workspace_bytes(ctypes.byref(d), ctypes.byref(n)) == 0
    # positions(3 double4) + velocities + list (capacity x 4 B) ...: a few hundred bytes per atom plus 1 MiB staging
    assert 864 * 300 < n.value - (1 << 20) < 864 * 2000
    d.box = (ctypes.c_double * 3)(10.0, 30.0, 30.0)
    assert L.md_workspace_bytes(ctypes.byref(d), ctypes.byref(n)) == md.MD_EBOX
    d.box = (ctypes.c_double * 3)(*w.box)
    d.n_boxes = 5
    assert L.md_workspace_bytes(ctypes.byref(d), ctypes.byref(n)) == md.MD_EINVAL
    d.n_boxes, d.n_types = 1, 9
    assert L.md_workspace_bytes(ctypes.byref(d), ctypes.byref(n)) == md.MD_EINVAL
    assert L.md_step(None, 1, 1.0) == md.MD_EINVAL and L.md_destroy(None) == 0


def test_python_struct_matches_c_layout():
    """sizeof(md_desc) as the C compiler sees it == ctypes' view (a mismatch would scramble every call)."""
    import subprocess, tempfile
    import paper_1212_6332_b200 as md
    src = '#include <stdio.h>\n#include "md.h"\nint main(){printf("%zu %zu\\n", sizeof(md_desc), sizeof(md_stats));return 0;}\n'
    with tempfile.TemporaryDirectory() as t:
        open(os.path.join(t, "s.c"), "w").write(src)
        subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), "-o", os.path.join(t, "s"), os.path.join(t, "s.c")], check=True)
        a, b = map(int, subprocess.run([os.path.join(t, "s")], capture_output=True, text=True, check=True).stdout.split())
    assert a == ctypes.sizeof(md.MdDesc) and b == ctypes.sizeof(md.MdStats)


def test_no_gpu_means_loud_failure():
    import torch
    import pytest
    import paper_1212_6332_b200 as md
    import workloads
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        md.MDSystem(workloads.config(0))
