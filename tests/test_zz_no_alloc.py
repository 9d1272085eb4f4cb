"""pa_overlap_hist_static -- the one entry point of the library that allocates nothing (include/pa_b200.h,
csrc/pa_static.cu).

It exists for users who cannot allocate at the moment they want the order-parameter histogram: code running while
another component owns all of the GPU's memory, loops that must not stall the device on cudaMalloc / cudaFree, code
that is handed a device pointer and a stream and nothing else.  Its accumulation bins are a fixed 131 328-byte array
inside the library (L <= 128) that every call on a GPU shares and that keeps the previous call's counts, so the
things to check are: (1) the result equals the context path's pa_overlap_hist bit for bit (integer work: no
tolerance), (2) it still does on the second and later calls, when the array is dirty -- same input twice (stale counts
would double), a large lattice followed by a small one and back, (3) sizes beyond the limit are refused, not truncated.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It holds no state of its own, so it passes alone in a fresh process (first call on the device = the set-up
call) as well as after the other GPU tests (library already loaded, scratch untouched until now).
"""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _population(L, R0, seed, betas, theta=2):
    """a population with structure in its overlap histogram: a few annealing steps through the context path"""
    from paper_2006_00561_b200 import binding
    pa = binding.PopulationAnnealer(L, R0, P=4, seed=seed)
    for b in betas:
        pa.step(b, theta)
    return pa


@pytest.mark.gpu
def test_static_overlap_hist_equals_the_context_path_on_consecutive_calls():
    import torch
    from paper_2006_00561_b200 import binding
    from oracle import pa_oracle as orc
    cases = []
    # A: shared-memory histogram path, even R;  B: L = 128 accumulates straight into the scratch bins (global atomics);
    # C: odd R (the last replica has no partner), small lattice after a large one.  (pa_step wants |dbeta| 2N < 700.)
    for L, R0, seed, betas in [(32, 3000, 11, (0.2, 0.4, 0.5)), (128, 301, 12, (0.02, 0.04, 0.06)), (16, 1001, 13, (0.25, 0.5, 0.8))]:
        pa = _population(L, R0, seed, betas)
        spins_host = pa.spins()
        want = pa.overlap_hist()                                       # existing path: bins in the context's workspace
        assert want.sum() == pa.R // 2
        assert np.array_equal(want, orc.overlap_hist(L, spins_host))   # and that path agrees with the oracle here
        cases.append((L, pa.R, torch.from_numpy(spins_host.view(np.int32)).cuda(), want))
        pa.close()
    torch.cuda.synchronize()
    A, B, Cc = cases
    # two calls in a row on the same input: the second one finds the first one's counts in the array
    for L, R, spins, want in (A, A, B, B, Cc, A, B):
        got = binding.overlap_hist_static(spins, L, R)
        assert got.dtype == np.uint64 and got.shape == (L * L + 1,)
        assert np.array_equal(got, want), (L, R)
    # device destination: enqueued on the current stream, nothing synchronised by the call
    for L, R, spins, want in (Cc, Cc, A):
        out = torch.full((L * L + 1,), -1, dtype=torch.int64, device="cuda")
        binding.overlap_hist_static(spins, L, R, out=out)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy().astype(np.uint64), want), (L, R)
    # fewer replicas than the tensor holds, and the empty cases
    L, R, spins, _ = A
    half = binding.overlap_hist_static(spins, L, 1000)
    assert np.array_equal(half, orc.overlap_hist(L, spins[:1000].cpu().numpy().view(np.uint32)))
    for r in (0, 1):
        assert binding.overlap_hist_static(spins, L, r).sum() == 0
    assert np.array_equal(binding.overlap_hist_static(spins, L, R), A[3])


@pytest.mark.gpu
def test_static_overlap_hist_refuses_what_it_cannot_hold():
    import torch
    from paper_2006_00561_b200 import binding
    spins = torch.zeros(4 * 256 * 256 // 32, dtype=torch.int32, device="cuda")
    with pytest.raises(binding.PaError) as e:
        binding.overlap_hist_static(spins, 256, 4)       # 65 537 bins > the 16 385 the built-in array holds
    assert e.value.code == binding.PA_EINVAL and "too large for the static scratch" in str(e.value)
    with pytest.raises(binding.PaError) as e:
        binding.overlap_hist_static(spins, 24, 4)
    assert e.value.code == binding.PA_EINVAL
    lib = binding.load_library()
    host = np.zeros(64, np.uint32)
    hist = np.zeros(65, np.uint64)
    rc = lib.pa_overlap_hist_static(C.c_void_p(host.ctypes.data), 8, 4, C.c_void_p(hist.ctypes.data), 0, None)
    assert rc == binding.PA_EINVAL and b"not a device pointer" in lib.pa_static_last_error()
    # and a good call still works afterwards
    ok = binding.overlap_hist_static(torch.zeros(64 * 2, dtype=torch.int32, device="cuda"), 8, 64)
    assert ok[64] == 32 and ok.sum() == 32   # identical lattices: q = N


def test_static_entry_point_rejects_oversize_before_touching_cuda():
    """-m "not gpu": the size limit is checked first, so the refusal needs no device"""
    from paper_2006_00561_b200 import binding
    lib = binding.load_library()
    hist = np.zeros(10, np.uint64)
    rc = lib.pa_overlap_hist_static(None, 256, 4, C.c_void_p(hist.ctypes.data), 0, None)
    assert rc == binding.PA_EINVAL
    assert b"L <= 128" in lib.pa_static_last_error()


def test_static_entry_point_source_allocates_nothing():
    """the translation unit of the no-allocation call names no allocating CUDA routine outside its comments"""
    src = open(os.path.join(ROOT, "paper_2006_00561_b200", "csrc", "pa_static.cu")).read()
    code = re.sub(r"//[^\n]*", "", re.sub(r"/\*.*?\*/", "", src, flags=re.S))
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMallocHost", "cudaMallocAsync", "cudaMemPool",
                   "new ", "malloc(", "std::vector", "std::string"):
        assert banned not in code, banned
    assert "cudaGetSymbolAddress" in code and "static __device__ __align__(256)" in code
