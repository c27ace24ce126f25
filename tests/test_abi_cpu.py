"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol include/wpcd.h declares
(no compute calls without a GPU), and the host-side input recipe is what DESIGN.md states."""
import ctypes
import os
import re

import numpy as np

from paper_2106_00454_b200 import inputs as inp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "wpcd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(wpcd_[A-Za-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_2106_00454_b200 import build
    lib = ctypes.CDLL(build.build())
    names = _declared()
    assert {"wpcd_build_channels", "wpcd_diag_batched", "wpcd_onshell_T", "wpcd_phase_shifts"} <= set(names)
    for nm in names:
        assert hasattr(lib, nm), nm
    # the binding's export list is the header's, and every definition has C linkage inside ONE extern "C" block
    src = open(os.path.join(ROOT, "paper_2106_00454_b200", "wpcd.py")).read()
    exports = re.search(r"EXPORTS = \[(.*?)\]", src, flags=re.S).group(1)
    assert sorted(re.findall(r'"(wpcd_[A-Za-z_0-9]+)"', exports)) == names
    api = open(os.path.join(ROOT, "paper_2106_00454_b200", "csrc", "api.cu")).read()
    assert api.count('extern "C" {') == 1 and api.rstrip().endswith('}  // extern "C"')
    # no undeclared debug exports in the product build
    import subprocess
    dyn = subprocess.run(["nm", "-D", "--defined-only", build.LIB], capture_output=True, text=True).stdout
    assert sorted(set(re.findall(r"\bT (wpcd_[A-Za-z_0-9]+)", dyn))) == names
    lib.wpcd_strerror.restype = ctypes.c_char_p
    assert lib.wpcd_strerror(0) == b"ok" and lib.wpcd_strerror(-2) == b"unsupported size"
    # without a device the handle cannot be created and says so (no CPU fallback)
    import torch
    if not torch.cuda.is_available():
        h = ctypes.c_void_p()
        assert lib.wpcd_create(ctypes.byref(h), 0) == -4 and not h.value


def test_static_workspace_constant_matches_the_header():
    """wpcd_diag_batched_static: the binding's limit is the header's WPCD_STATIC_WORK_BYTES, the array is a file-scope
    __device__ array in the .cu file that resolves its address with cudaGetSymbolAddress, and the entry point's translation
    units call no allocator."""
    from paper_2106_00454_b200 import wpcd
    hdr = open(os.path.join(ROOT, "include", "wpcd.h")).read()
    m = re.search(r"#define WPCD_STATIC_WORK_BYTES \((\d+)u << (\d+)\)", hdr)
    assert m and (int(m.group(1)) << int(m.group(2))) == wpcd.Handle.STATIC_WORK_BYTES == 16 << 20
    jac = open(os.path.join(ROOT, "paper_2106_00454_b200", "csrc", "jacobi.cu")).read()
    assert "static __device__ __align__(256) unsigned char wpcd_static_work[WPCD_STATIC_WORK_BYTES];" in jac
    assert "cudaGetSymbolAddress(&ptr, wpcd_static_work)" in jac
    for f in ("jacobi.cu", "jacobi_small.cu", "api.cu"):
        src = open(os.path.join(ROOT, "paper_2106_00454_b200", "csrc", f)).read()
        src = re.sub(r"//.*", "", src)
        assert not re.search(r"\bcuda(Malloc\w*|Free\w*|HostAlloc)\s*\(", src), f


def test_input_recipe():
    p = inp.grid_edges(100)
    assert len(p) == 101 and p[0] == 0 and abs(p[100] - 127.96) < 0.01 and np.all(np.diff(p) > 0)
    s = inp.sample_scales(1024)
    assert s.shape == (1024, 3) and np.allclose(s[0], [1.012573, 0.986790, 1.064042], atol=1e-6)
    assert 0.6 < s.min() < 0.62 and 1.30 < s.max() < 1.32        # range 0.61...1.31
    assert len(inp.CHANNELS_J4) == 14 and sum(c for _, c, _ in inp.CHANNELS_J4) == 4
    tl, ecm = inp.energies(350)
    assert tl[0] == 1.0 and tl[-1] == 350.0 and np.allclose(ecm, tl / 2)


def test_binding_does_not_import_oracle():
    for fn in ("wpcd.py", "inputs.py", "build.py", "__init__.py"):
        src = open(os.path.join(ROOT, "paper_2106_00454_b200", fn)).read()
        assert not re.search(r"^\s*(from|import)\s+\.*oracle", src, flags=re.M), fn
        assert "liboracle" not in src, fn


def test_jacobi_block_tournament_invariants():
    """Host logic of wpcd_diag_batched's schedule through the C-ABI test hooks: in a sweep every pair of real blocks
    meets exactly once, every block sits in at most one slot per step, and the pipelining rule holds -- every real
    pivot of the next step is fed by exactly one tile of the running step and no tile feeds two pivots."""
    from paper_2106_00454_b200 import build
    lib = ctypes.CDLL(build.build())
    I, J = ctypes.c_int(), ctypes.c_int()
    for nb in (2, 3, 5, 6, 7, 13, 25, 26, 50, 100):
        m = max(6, nb + (nb & 1))
        met = set()
        for t in range(m - 1):
            slots, seen = [], set()
            for s in range(m // 2):
                assert lib.wpcd_jacobi_schedule(m, nb, t, s, ctypes.byref(I), ctypes.byref(J)) == 0
                slots.append((I.value, J.value))
                for b in (I.value, J.value):
                    if b >= 0:
                        assert 0 <= b < nb and b not in seen
                        seen.add(b)
                if J.value >= 0:
                    assert I.value < J.value and (I.value, J.value) not in met
                    met.add((I.value, J.value))
            assert seen == set(range(nb))                       # every real block sits somewhere
            tn = (t + 1) % (m - 1)
            nxt = []
            for s in range(m // 2):
                lib.wpcd_jacobi_schedule(m, nb, tn, s, ctypes.byref(I), ctypes.byref(J))
                nxt.append((I.value, J.value))
            fed = {}
            for s1 in range(m // 2):
                for s2 in range(s1 + 1, m // 2):
                    cs = lib.wpcd_jacobi_critical_slot(m, nb, t, tn, s1, s2)
                    blocks1 = {b for b in slots[s1] if b >= 0}
                    blocks2 = {b for b in slots[s2] if b >= 0}
                    # brute force: real pivots of step tn with one block in each of the two slots
                    want = [k for k, (a, b) in enumerate(nxt)
                            if b >= 0 and ((a in blocks1 and b in blocks2) or (a in blocks2 and b in blocks1))]
                    assert len(want) <= 1
                    assert cs == (want[0] if want else -1), (nb, t, s1, s2, cs, want)
                    if cs >= 0:
                        assert cs not in fed
                        fed[cs] = (s1, s2)
            assert set(fed) == {k for k, (a, b) in enumerate(nxt) if b >= 0}
        assert met == {(a, b) for a in range(nb) for b in range(a + 1, nb)}
    assert lib.wpcd_jacobi_schedule(4, 4, 0, 0, ctypes.byref(I), ctypes.byref(J)) == -1   # m < 6 rejected
