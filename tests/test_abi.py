"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads without a GPU,
exports every symbol include/tlb.h declares, validates parameters, and refuses to run without a
device (no CPU fallback).  No compute call is made here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2109_12565_b200 import binding
    binding.build()
    binding.load_library()
    return binding


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "tlb.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tlb_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(binding):
    lib = binding.load_library()
    names = _declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.SYMBOLS) == names


def test_library_is_sm100a_and_product_never_imports_oracle(binding):
    import subprocess
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True)
    assert "sm_100a" in out.stdout
    pkg = os.path.join(ROOT, "paper_2109_12565_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), f
                assert "tlb_oracle" not in text, f


def test_params_struct_and_defaults(binding):
    assert ctypes.sizeof(binding.TLBParams) == 22 * 8 + 8 * 4
    p = binding.default_params()
    assert (p.tau, p.tau_g, p.rho0, p.G12, p.G11a, p.G11r) == (1.0, 1.0, 1.0, 0.405, -9.0, 8.1)
    assert (p.T_bottom, p.T_top, p.T_ref, p.alpha_g, p.thermal, p.periodic_y) == (1.0, 0.0, 0.5, 1e-4, 1, 0)
    with pytest.raises(KeyError):
        binding.default_params(no_such_field=1)


def test_workspace_bytes_and_validation(binding):
    lib = binding.load_library()
    n = ctypes.c_size_t()
    p = binding.default_params()
    assert lib.tlb_workspace_bytes(4096, 2048, ctypes.byref(p), ctypes.byref(n)) == 0
    pops = 2 * 27 * 4096 * 2050 * 8
    assert pops < n.value < pops * 1.12  # two population buffers dominate
    for bad in (dict(tau=0.5), dict(tau_g=0.3), dict(rho0=0.0), dict(post_w=4, post_h=4, post_period=16, periodic_y=1),
                dict(post_w=4, post_h=1024, post_period=16), dict(pop_precision=16), dict(n_droplets=-1)):
        q = binding.default_params(**bad)
        assert lib.tlb_workspace_bytes(4096, 2048, ctypes.byref(q), ctypes.byref(n)) == binding.TLB_EINVAL, bad
    q = binding.default_params(pop_precision=32)  # fp32 population storage: half-size buffers + a host staging area
    m = ctypes.c_size_t()
    assert lib.tlb_workspace_bytes(4096, 2048, ctypes.byref(q), ctypes.byref(m)) == 0 and m.value < n.value
    assert lib.tlb_workspace_bytes(0, 8, ctypes.byref(p), ctypes.byref(n)) == binding.TLB_EINVAL
    assert lib.tlb_workspace_bytes(8, 8, None, ctypes.byref(n)) == binding.TLB_EINVAL
    assert b"fallback" in lib.tlb_error_string(binding.TLB_ECUDA)
    assert lib.tlb_step(None, 1) == binding.TLB_EINVAL


def test_no_cpu_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(binding.TLBError) as e:
        binding.TLB(16, 16)
    assert e.value.code == binding.TLB_ECUDA
    # the C call itself also refuses (fake, aligned, non-NULL workspace pointer; never dereferenced)
    lib = binding.load_library()
    p = binding.default_params()
    h = ctypes.c_void_p()
    rc = lib.tlb_create(16, 16, ctypes.byref(p), 1 << 20, 1 << 30, None, ctypes.byref(h))
    assert rc == binding.TLB_ECUDA and not h.value


def test_header_is_plain_c(tmp_path):
    """include/tlb.h is a C ABI: it compiles as C99 (no C++ or CUDA types in the signatures)."""
    import subprocess
    src = tmp_path / "t.c"
    src.write_text('#include "tlb.h"\nint main(void) { tlb_params p; tlb_rough_walls r; (void)p; (void)r; return TLB_OK; }\n')
    inc = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include")
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", inc, "-c", str(src), "-o", str(tmp_path / "t.o")])
