"""CPU-side checks of the C-ABI boundary: libns.so builds, loads, and exports every symbol that
include/ns.h declares; argument validation works without a GPU; there is no CPU fallback."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libns():
    from paper_2401_09843_b200 import build, binding
    build.build()
    return binding.lib()


def declared_symbols(header="ns.h", prefix="ns_"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(" + prefix + r"[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_exported(libns):
    from paper_2401_09843_b200 import binding
    syms = declared_symbols()
    assert len(syms) >= 15
    for s in syms:
        assert hasattr(libns, s), f"libns.so does not export {s}"
    assert sorted(binding.EXPORTS) == syms
    syms3 = declared_symbols("ns_mg.h", "ns_mg_")
    assert len(syms3) >= 12
    for s in syms3:
        assert hasattr(libns, s), f"libns.so does not export {s}"
    assert sorted(binding.EXPORTS_MG) == syms3
    syms2 = declared_symbols("ns2d.h", "ns2d_")
    assert len(syms2) >= 15
    for s in syms2:
        assert hasattr(libns, s), f"libns.so does not export {s}"
    assert sorted(binding.EXPORTS_2D) == syms2


def test_no_torch_types_in_header():
    text = open(os.path.join(ROOT, "include", "ns.h")).read()
    assert "torch" not in text.lower()
    assert "at::" not in text and "Tensor" not in text


def test_create_rejects_bad_arguments(libns):
    from paper_2401_09843_b200 import binding
    h = ctypes.c_void_p()
    for N, batch, dtype in [(7, 1, 0), (1024, 1, 0), (8, 1, 0), (32, 0, 0), (32, 1, 5), (41, 1, 0), (14, 1, 0), (642, 1, 0),
                            (768, 1, 0)]:
        rc = libns.ns_create(ctypes.byref(h), N, batch, None, dtype, None)
        assert rc == binding.NS_ERR_INVALID_ARG, (N, batch, dtype, rc)
        assert not h.value
        assert len(libns.ns_last_error(None)) > 0
    p = binding.ns_params(0.0, 0.0, 0.5, -1.0, -1.0, 0)  # s < 1
    assert libns.ns_create(ctypes.byref(h), 32, 1, ctypes.byref(p), 0, None) == binding.NS_ERR_INVALID_ARG
    assert libns.ns_create(None, 32, 1, None, 0, None) == binding.NS_ERR_INVALID_ARG
    assert libns.ns_destroy(None) == binding.NS_ERR_INVALID_ARG
    assert libns.ns_step(None, 0.1) == binding.NS_ERR_INVALID_ARG
    for N, batch, dtype in [(14, 1, 0), (97, 1, 0), (1024, 1, 0), (256, 0, 0), (256, 1, 7)]:
        assert libns.ns2d_create(ctypes.byref(h), N, batch, None, dtype, None) == binding.NS_ERR_INVALID_ARG and not h.value
    assert libns.ns2d_destroy(None) == binding.NS_ERR_INVALID_ARG and libns.ns2d_step(None, 0.1) == binding.NS_ERR_INVALID_ARG
    # ns_mg.h: decomposition checks come before any device is touched
    dev = (ctypes.c_int * 4)(0, 0, 0, 0)
    for N, P, dtype in [(64, 0, 0), (64, 17, 0), (64, 3, 0), (50, 2, 0), (16, 2, 0), (64, 2, 9), (80, 2, 1)]:
        assert libns.ns_mg_create(ctypes.byref(h), N, P, dev, None, dtype) == binding.NS_ERR_INVALID_ARG, (N, P, dtype)
        assert not h.value and len(libns.ns_mg_last_error(None)) > 0
    assert libns.ns_mg_create(ctypes.byref(h), 64, 2, None, None, 0) == binding.NS_ERR_INVALID_ARG
    assert libns.ns_mg_destroy(None) == binding.NS_ERR_INVALID_ARG and libns.ns_mg_step(None, 0.1) == binding.NS_ERR_INVALID_ARG


def test_no_cpu_fallback(libns):
    """Without a CUDA device ns_create must fail loudly (NS_ERR_CUDA), never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2401_09843_b200 import binding
    h = ctypes.c_void_p()
    rc = libns.ns_create(ctypes.byref(h), 32, 1, None, 0, None)
    assert rc == binding.NS_ERR_CUDA
    assert b"no usable CUDA device" in libns.ns_last_error(None)
    with pytest.raises(binding.NSError):
        binding.Solver(32, stream=0)
    assert libns.ns2d_create(ctypes.byref(h), 256, 4, None, 0, None) == binding.NS_ERR_CUDA
    dev = (ctypes.c_int * 2)(0, 0)
    assert libns.ns_mg_create(ctypes.byref(h), 64, 2, dev, None, 0) == binding.NS_ERR_CUDA
    with pytest.raises(binding.NSError):
        binding.SolverMG(64, [0, 0])
    with pytest.raises(binding.NSError):
        binding.Solver2D(256, stream=0)


def test_product_does_not_import_oracle():
    """The product package must not reference oracle/ (the oracle is test infrastructure)."""
    pkg = os.path.join(ROOT, "paper_2401_09843_b200")
    for dirpath, _d, files in os.walk(pkg):
        if "build" in os.path.relpath(dirpath, pkg).split(os.sep)[:1] and dirpath != pkg:
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "ns_oracle" not in text and "from oracle" not in text and "import oracle" not in text, f
    otext = open(os.path.join(ROOT, "oracle", "ns_oracle.py")).read() + open(os.path.join(ROOT, "oracle", "ns_oracle.cpp")).read()
    assert "paper_2401_09843_b200" not in otext.replace("paper_2401_09843_b200/csrc/", "")


def test_sass_is_blackwell_native():
    """The built library carries the sm_100a paths the design names (B200_PROFILING.md 'What proves a Blackwell-native
    kernel'): TMA bulk copies (UBLKCP) in every fused z kernel, tensor-map TMA loads (UTMALDG) in the persistent column kernel, tensor-memory parking (STTM / LDTM after a
    tcgen05.alloc) in the long-line kernels, and no cuFFT / cuBLAS dependency.  Static check with cuobjdump / ldd."""
    import shutil
    import subprocess
    from paper_2401_09843_b200 import binding
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([cuobjdump, "-sass", binding.LIB_PATH], capture_output=True, text=True, check=True).stdout
    assert "sm_100a" in sass
    per_fn, name = {}, None
    for line in sass.splitlines():
        if "Function :" in line:
            name = line.split("Function :")[1].strip()
            per_fn[name] = set()
        elif name is not None:
            for m in ("UBLKCP", "UTMALDG", "LDTM", "STTM", "UTCATOMSWS", "DFMA"):
                if m in line:
                    per_fn[name].add(m)
    z = {k: v for k, v in per_fn.items() if "z_fused" in k or "z_pair" in k or "y2d_kernel" in k}
    assert len(z) >= 12 and all("UBLKCP" in v for v in z.values())
    tm = {k: v for k, v in per_fn.items() if "z_pair" in k or "y2d_kernel" in k or "_tmem_kernel" in k}
    assert len(tm) >= 12 and all({"LDTM", "STTM", "UTCATOMSWS"} <= v for v in tm.values())
    # the persistent forward column kernel: tensor-map TMA loads (cp.async.bulk.tensor) and twiddles in tensor memory
    ring = {k: v for k, v in per_fn.items() if "col_fwd_ring_kernel" in k}
    assert len(ring) >= 1 and all({"UTMALDG", "LDTM", "STTM"} <= v for v in ring.values())
    ldd = subprocess.run(["ldd", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "cufft" not in ldd.lower() and "cublas" not in ldd.lower()
