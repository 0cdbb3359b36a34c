"""md_kinetic_energy_noalloc (include/md.h): the entry point that allocates nothing, its scratch a fixed device array of the
library.  Collected last on purpose (the suite runs with pytest -x).  The GPU test checks it against the existing path
(md_get_energies: block partials in the system's workspace) on two calls in a row that share the scratch array."""
import ctypes as C

import numpy as np
import pytest

import workloads

E_REL = 1e-12        # the energy tolerance of tests/test_gpu_parity.py (BASELINE.json north_star)


def test_rejects_bad_sizes_before_touching_the_device():
    """Argument errors are decided on the host: no GPU needed, and the message names the limit."""
    import paper_1212_6332_b200 as md
    L = md.lib()
    mass = (C.c_double * 1)(63.546)
    err = C.create_string_buffer(256)
    dummy = C.c_void_p(256)                                   # never dereferenced: the size check comes first
    rc = L.md_kinetic_energy_noalloc(None, dummy, None, mass, 1, md.MD_NOALLOC_MAX_ATOMS + 1, dummy, err, len(err))
    assert rc == md.MD_EINVAL
    assert b"exceeds MD_NOALLOC_MAX_ATOMS = 4194304" in err.value
    assert L.md_kinetic_energy_noalloc(None, dummy, None, mass, 1, -1, dummy, err, len(err)) == md.MD_EINVAL
    assert b"negative" in err.value
    assert L.md_kinetic_energy_noalloc(None, dummy, None, mass, 1, 10, None, err, len(err)) == md.MD_EINVAL
    assert L.md_kinetic_energy_noalloc(None, dummy, None, mass, 5, 10, dummy, err, len(err)) == md.MD_EINVAL
    assert L.md_kinetic_energy_noalloc(None, dummy, None, mass, 2, 10, dummy, err, len(err)) == md.MD_EINVAL   # types NULL
    bad = (C.c_double * 1)(0.0)
    assert L.md_kinetic_energy_noalloc(None, dummy, None, bad, 1, 10, dummy, None, 0) == md.MD_EINVAL          # err may be NULL
    text = open(md.__file__.replace("__init__.py", "csrc/md_noalloc.cu")).read()
    text = "\n".join(line.split("//")[0] for line in text.splitlines())
    assert "cudaMalloc" not in text and "cudaFree" not in text and "cudaGetSymbolAddress" in text


@pytest.mark.gpu
def test_no_alloc_kinetic_energy_matches_md_get_energies_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "this test needs the B200"
    import paper_1212_6332_b200 as md
    # 32,000 atoms of one species (32 block partials), then 2,000 atoms of two species in 4 boxes (2 partials), then 864 atoms
    # (1 partial), then 16,384 atoms of two species (16 partials): a call that read partials left by the call before it, or
    # an arrival counter left non-zero, would be wrong
    cases = (workloads.config("3a", scale=20), workloads.alloy(workloads.config(2, scale=4), 77, 0.4), workloads.config(0),
             workloads.alloy(workloads.config("3a", scale=16), 78))
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    for it, w in enumerate(cases):                               # calls back to back on one stream, one shared scratch
        sysm = md.MDSystem(w)
        try:
            want = float(np.sum(sysm.energies()[1]))             # existing path: k_ekin_partial + k_ekin_boxes over the workspace
            v = sysm.velocities(device_out=True)
            types = torch.as_tensor(np.ascontiguousarray(w.types, dtype=np.int32)).cuda() if len(w.mass) > 1 else None
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
            md.kinetic_energy_noalloc(v, types, w.mass, out[:1])
            md.kinetic_energy_noalloc(v, types, w.mass, out[1:])        # and again at once: same bits (fixed summation order)
            torch.cuda.synchronize()
            if it > 0:                                           # (the very first launch may load the kernel's code)
                assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the device's free memory"
            got = out.cpu().numpy()
            assert got[0] == got[1]
            assert abs(got[0] - want) <= E_REL * abs(want), (w.name, got[0], want)
            # independent check of both: the definition in numpy from the velocities the caller holds
            m = np.asarray(w.mass, dtype=np.float64)[np.asarray(w.types) if len(w.mass) > 1 else np.zeros(w.n_atoms, dtype=int)]
            ref = 0.5 * 103.642696526805 * float(np.sum(m * np.sum(np.asarray(w.velocities) ** 2, axis=1)))
            assert abs(got[0] - ref) <= 1e-11 * abs(ref)
        finally:
            sysm.close()
    # n_atoms = 0 is legal and gives 0; a size beyond the fixed scratch is refused with a message that names the limit
    md.kinetic_energy_noalloc(torch.empty((0, 3), dtype=torch.float64, device="cuda"), None, [63.546], out[:1])
    assert float(out[0]) == 0.0
    err = C.create_string_buffer(256)
    rc = md.lib().md_kinetic_energy_noalloc(C.c_void_p(torch.cuda.current_stream().cuda_stream), C.c_void_p(out.data_ptr()), None,
                                            (C.c_double * 1)(63.546), 1, md.MD_NOALLOC_MAX_ATOMS + 1, C.c_void_p(out.data_ptr()),
                                            err, len(err))
    assert rc == md.MD_EINVAL and b"exceeds MD_NOALLOC_MAX_ATOMS" in err.value
