"""CPU-side checks of the C-ABI boundary: the library loads and exports every symbol that
include/*.h declares (no compute calls), and argument validation that needs no GPU."""
import ctypes
import glob
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    names = set()
    for h in glob.glob(os.path.join(ROOT, "include", "*.h")):
        src = open(h).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(trimeg_[a-z0-9_]+)\s*\(", src))
    return sorted(names)


@pytest.fixture(scope="module")
def lib():
    from paper_2601_14301_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def test_header_declares_the_path():
    names = _declared_symbols()
    for must in ("trimeg_mesh_create", "trimeg_field_upload", "trimeg_push", "trimeg_locate",
                 "trimeg_gather", "trimeg_rhs", "trimeg_sort", "trimeg_compact", "trimeg_push_host"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    for name in _declared_symbols():
        assert hasattr(lib, name), name


def test_binding_names_match_header():
    from paper_2601_14301_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_symbols()
    L = binding.load()
    assert b"sm_100a" in L.trimeg_version()
    assert binding.strerror(0) == "ok"
    for code in (-1, -2, -3, -4, -5):
        assert binding.strerror(code) not in ("ok", "unknown error")


def test_sass_is_sm100a_and_locator_has_no_fma_in_contains():
    """The cubin embedded in the library targets sm_100a, and the SASS of locate_kernel has no DFMA where the
    contains() test lives (rule L2: every operation individually rounded): the kernel body (hinted walk) and the
    complete 3x3 rule (the subroutine with the most DMULs) multiply and add separately; fused multiply-adds appear
    only in the (r, theta) guess (sqrt, atan2), which never decides anything (rule L1)."""
    import subprocess
    from paper_2601_14301_b200 import binding
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    assert "sm_100a" in out.stdout
    sass = subprocess.run(["cuobjdump", "-sass", binding.LIB_PATH], capture_output=True, text=True).stdout
    fn = [f for f in re.split(r"\n\s*Function : ", sass) if f.startswith("_ZN6trimeg13locate_kernel")]
    assert len(fn) == 1
    ins = [(int(a, 16), op) for a, op in re.findall(r"/\*([0-9a-f]{4,})\*/\s+(?:@!?U?P\d+\s+)?([A-Z][A-Z0-9_.]*)", fn[0])]
    targets = sorted({int(t, 16) for t in re.findall(r"CALL\.REL\.NOINC\s+(0x[0-9a-f]+)", fn[0])})
    assert targets, "locate_full / ring_sector_guess are expected as subroutines"
    bounds = [0] + targets + [max(a for a, _ in ins) + 16]
    regions = [[op for a, op in ins if lo <= a < hi] for lo, hi in zip(bounds[:-1], bounds[1:])]
    body = regions[0]
    full = max(regions[1:], key=lambda r: sum(op.startswith("DMUL") for op in r))
    for r in (body, full):
        assert sum(op.startswith("DMUL") for op in r) >= 4 and sum(op.startswith("DADD") for op in r) >= 4
        assert not any(op.startswith("DFMA") for op in r)
    assert any(op.startswith("DFMA") for r in regions for op in r)      # the guess does use them: the parse sees DFMAs


def test_invalid_arguments_are_rejected_without_a_gpu(lib):
    from paper_2601_14301_b200 import binding
    L = binding.load()
    h = ctypes.c_void_p(0)
    p = binding.trimeg_params(R0=10, a=1, B0=1, q0=1.4, q2=2.0, rho0=1 / 60, qs_over_ms=1, T=2, kappa_n=1,
                              kappa_T=6.9, eom_variant=0, weight_mode=0)
    dp = ctypes.POINTER(ctypes.c_double)
    r_bad = (ctypes.c_double * 3)(0.0, 0.5, 0.4)
    r_ok = (ctypes.c_double * 3)(0.0, 0.5, 1.0)
    assert L.trimeg_mesh_create(ctypes.byref(h), 2, 32, ctypes.cast(r_bad, dp), None, None, ctypes.byref(p)) == binding.ERR_MESH
    assert L.trimeg_mesh_create(ctypes.byref(h), 1, 32, ctypes.cast(r_ok, dp), None, None, ctypes.byref(p)) == binding.ERR_INVALID_ARG
    assert L.trimeg_mesh_create(None, 2, 32, ctypes.cast(r_ok, dp), None, None, ctypes.byref(p)) == binding.ERR_INVALID_ARG
    # sagitta rule L4: 3 sectors, thin second ring
    r_thin = (ctypes.c_double * 3)(0.0, 0.9, 1.0)
    assert L.trimeg_mesh_create(ctypes.byref(h), 2, 3, ctypes.cast(r_thin, dp), None, None, ctypes.byref(p)) == binding.ERR_MESH
    p.T = -1.0
    assert L.trimeg_mesh_create(ctypes.byref(h), 2, 32, ctypes.cast(r_ok, dp), None, None, ctypes.byref(p)) == binding.ERR_INVALID_ARG
    assert L.trimeg_mesh_destroy(None) == binding.ERR_INVALID_ARG
    assert L.trimeg_push(None, None, 0, 0.1, 1, None) == binding.ERR_INVALID_ARG


def test_no_cpu_fallback_when_no_device():
    """Without a CUDA device mesh_create must fail with ERR_CUDA (loudly), not compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2601_14301_b200 import binding, inputs
    with pytest.raises(binding.TrimegError) as e:
        binding.context_for(inputs.WORKLOADS["cfg1"])
    assert e.value.code in (binding.ERR_CUDA, binding.ERR_ALLOC)
