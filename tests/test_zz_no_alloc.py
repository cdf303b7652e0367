"""The allocation-free entry point (include/ns_noalloc.h): ns_noalloc_energy_spectrum accumulates the shell spectrum of a
caller-held device array in a static __device__ scratch array of the library.  Collected LAST on purpose (the file name): the
suite runs with pytest -x, and this is an addition outside the hot path.

GPU test: its output against the existing path (ns_energy_spectrum of a solver handle holding the same state) within the tolerance
the other spectrum tests use (1e-13 absolute at total energy 0.5), on two calls in a row with different shapes -- the second must
not see the first one's bins."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_noalloc_symbol_is_declared_exported_and_validates_on_the_cpu():
    from paper_2401_09843_b200 import binding, build
    build.build()
    L = binding.lib()
    text = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "ns_noalloc.h")).read(), flags=re.S)
    syms = sorted(set(re.findall(r"\b(ns_noalloc_[a-z_0-9]+)\s*\(", text)))
    assert syms == sorted(binding.EXPORTS_NOALLOC) == ["ns_noalloc_energy_spectrum"]
    assert hasattr(L, syms[0])
    assert int(re.search(r"#define NS_NOALLOC_MAX_VALUES (\d+)", text).group(1)) == binding.NS_NOALLOC_MAX_VALUES
    # argument validation needs no GPU: sizes beyond the static scratch are rejected with a clear message, nothing is truncated
    err = ctypes.create_string_buffer(256)
    dummy = ctypes.c_void_p(256)          # never dereferenced by the checks
    for N, batch, dtype, nbins in [(64, 1, 0, 0), (64, 1, 0, 5000), (63, 1, 0, 16), (64, 0, 0, 16), (64, 1, 7, 16), (64, 17, 0, 1024)]:
        rc = L.ns_noalloc_energy_spectrum(dummy, N, batch, dtype, nbins, dummy, 1, None, err, 256)
        assert rc == binding.NS_ERR_INVALID_ARG and len(err.value) > 0, (N, batch, dtype, nbins)
    assert b"exceeds the static scratch" in err.value
    assert L.ns_noalloc_energy_spectrum(None, 64, 1, 0, 16, dummy, 1, None, err, 256) == binding.NS_ERR_INVALID_ARG
    # the file of the entry point calls no allocator
    src = open(os.path.join(ROOT, "paper_2401_09843_b200", "csrc", "ns_noalloc.cu")).read()
    code = re.sub(r"//.*", "", src)
    assert "cudaMalloc" not in code and "cudaFree" not in code and "cudaGetSymbolAddress" in code


@pytest.mark.gpu
def test_noalloc_energy_spectrum_matches_the_handle_path_twice():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2401_09843_b200 import binding, inputs
    binding.lib()

    def state(N, batch, seed):
        us = np.stack([inputs.gaussian_field(N, seed + i, lambda k: 1.0 / (1.0 + k) ** 2, e_tot=0.5) * (1.0 + 0.25 * i) for i in range(batch)])
        s = binding.Solver(N, batch=batch)
        s.set_initial(us)
        return s, s.get_spectral()

    # call 1: batch 3 at 64^3, full range of bins, device output
    s1, uh1 = state(64, 3, 11)
    want1 = s1.energy_spectrum(64)
    d1 = torch.from_numpy(uh1).cuda()
    out1 = torch.full((3, 64), -1.0, dtype=torch.float64, device="cuda")
    binding.energy_spectrum_noalloc(d1, 64, 64, out=out1)
    torch.cuda.synchronize()
    got1 = out1.cpu().numpy()
    assert np.abs(got1 - want1).max() < 1e-13
    assert abs(got1[0].sum() - 0.5) < 1e-12                           # Parseval: total energy of the recipe
    # call 2, right after: another state, fewer samples and FEWER bins (a stale scratch would show), host output, fp64 from 48^3
    s2, uh2 = state(48, 2, 23)
    want2 = s2.energy_spectrum(20)
    got2 = binding.energy_spectrum_noalloc(torch.from_numpy(uh2).cuda(), 48, 20)
    assert got2.shape == (2, 20) and np.abs(got2 - want2).max() < 1e-13
    # and the first request again: identical to its first answer up to the order of the atomic sums
    free0 = torch.cuda.mem_get_info()[0]
    again = binding.energy_spectrum_noalloc(d1, 64, 64)
    assert torch.cuda.mem_get_info()[0] == free0                      # a call (past the one-time symbol set-up) takes no device memory
    assert np.abs(again - got1).max() < 1e-14
    # fp32 state against the fp32 handle path
    s3 = binding.Solver(64, batch=1, dtype="f32")
    s3.set_spectral(uh1[:1].astype(np.complex64))
    got3 = binding.energy_spectrum_noalloc(torch.from_numpy(uh1[:1].astype(np.complex64)).cuda(), 64, 64)
    assert np.abs(got3 - s3.energy_spectrum(64)).max() < 1e-12
    # beyond the static scratch: rejected, not truncated
    with pytest.raises(binding.NSError, match="exceeds the static scratch"):
        binding.energy_spectrum_noalloc(torch.zeros((5, 3, 16, 16, 9), dtype=torch.complex128, device="cuda"), 16, 4096)
