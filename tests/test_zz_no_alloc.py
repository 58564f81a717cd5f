"""admm_phit_apply_static (include/admm_b200.h): the Eq. (6) contraction W = G . Phi through the entry point that
allocates nothing (its split-K scratch is a static __device__ array), against the existing handle-based path
(admm_contract_probe, which = 0) on the same seeded inputs, within the bar the contraction tests use (tests/test_gpu_parity.py:
|difference| < 1e-6 of the sum of |terms| of an output), on two calls in a row that share the scratch.

Collected last on purpose (the file name): the suite runs with `pytest -x`."""
import gc
import os
import re

import numpy as np
import pytest

from conftest import have_cuda

gpu = [pytest.mark.gpu, pytest.mark.skipif(not have_cuda(), reason="needs a CUDA device")]


def _marked(f):
    for m in gpu:
        f = m(f)
    return f


TOL = 1e-6          # tests/test_gpu_parity.py::test_contractions_match_fp64_matmul


@pytest.fixture(scope="module")
def b():
    from paper_2509_08602_b200 import binding
    return binding


def _existing_path(b, w, small):
    h = b.admm_setup(w.phi, w.point_class, w.classes)
    out = b.admm_contract_probe(h, 0, small)
    h.close()
    return out


@_marked
def test_two_calls_in_a_row_match_the_existing_path(b):
    import torch
    from workloads import make_workload
    w = make_workload(0, n_target=900, n_lowdose=1711, n_iso=12)          # N = 2611, n = 288: ragged tiles, several splits
    rng = np.random.default_rng(23)
    P = np.abs(w.phi.astype(np.float64))
    phi = torch.from_numpy(w.phi).cuda()
    # the second call is smaller than the first (fewer plans, so fewer tiles and another split count): whatever the first call left
    # in the shared scratch must not show in it
    for Bp in (81, 9):
        small = rng.standard_normal((Bp, w.N)).astype(np.float32)
        want = _existing_path(b, w, small)
        g = torch.from_numpy(small).cuda()
        out = torch.full((Bp, w.n), float("nan"), dtype=torch.float64, device="cuda")
        b.admm_phit_apply_static(phi, g, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        scale = np.abs(small.astype(np.float64)) @ P
        assert np.isfinite(got).all()
        assert np.max(np.abs(got - want) / scale) < TOL, Bp
        exact = small.astype(np.float64) @ w.phi.astype(np.float64)
        assert np.max(np.abs(got - exact) / scale) < TOL, Bp
        # same call again: same bits (the partial sums are added in split order whichever block arrives last)
        out2 = torch.empty_like(out)
        # device-wide free memory must not drop across a call.  (Device-wide, because torch's own counters cannot see a cudaMalloc made
        # by the library; one-sided and after a gc pass, because handles and tensors that EARLIER tests left to the garbage collector
        # may be released at any moment, which only raises it.)
        gc.collect()
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        b.admm_phit_apply_static(phi, g, out2)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] >= free_before
        assert torch.equal(out, out2)


@_marked
def test_strided_inputs_and_a_side_stream(b):
    import torch
    from workloads import make_workload
    w = make_workload(0, n_target=40, n_lowdose=57, n_iso=1)              # N = 97, n = 24: less than one tile, one split
    rng = np.random.default_rng(29)
    small = rng.standard_normal((5, w.N)).astype(np.float32)
    want = _existing_path(b, w, small)
    phi = torch.zeros((w.N, w.n + 7), dtype=torch.float32, device="cuda"); phi[:, : w.n] = torch.from_numpy(w.phi).cuda()
    g = torch.zeros((5, w.N + 3), dtype=torch.float32, device="cuda"); g[:, : w.N] = torch.from_numpy(small).cuda()
    out = torch.empty((5, w.n), dtype=torch.float64, device="cuda")
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        b.admm_phit_apply_static(phi[:, : w.n], g[:, : w.N], out)
    s.synchronize()
    scale = np.abs(small.astype(np.float64)) @ np.abs(w.phi.astype(np.float64))
    assert np.max(np.abs(out.cpu().numpy() - want) / scale) < TOL


@_marked
def test_sizes_beyond_the_scratch_are_refused(b):
    import torch
    n, Bp = 32768, 64                                                      # 2097152 outputs > 2093056
    phi = torch.zeros((16, n), dtype=torch.float32, device="cuda")
    g = torch.zeros((Bp, 16), dtype=torch.float32, device="cuda")
    out = torch.full((Bp, n), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(b.AdmmError) as e:
        b.admm_phit_apply_static(phi, g, out)
    assert e.value.status == b.ADMM_EINVAL and "exceeds the static scratch" in str(e.value)
    assert bool((out == 7.0).all())                                        # untouched
    # one plan fewer fits
    b.admm_phit_apply_static(phi, g[:63], out[:63])
    torch.cuda.synchronize()
    assert bool((out[:63] == 0.0).all()) and bool((out[63] == 7.0).all())
    # host pointers are refused, not dereferenced
    import ctypes as C
    hp = np.zeros((4, 4), np.float32); ho = np.zeros((4, 4), np.float64)
    err = C.create_string_buffer(256)
    st = b._lib.admm_phit_apply_static(hp.ctypes.data, 4, 4, 4, hp.ctypes.data, 4, 4, ho.ctypes.data, 0, None, err, 256)
    assert st == b.ADMM_EINVAL and b"memory of the given device" in err.value


def test_source_calls_no_allocating_routine():
    """By construction: the translation unit of the entry point names no allocation routine and no library that allocates
    (a check a run cannot make: an allocation freed again inside the call leaves free memory as it was)."""
    src = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_2509_08602_b200", "csrc", "no_alloc.cu")).read()
    code = re.sub(r"//[^\n]*", "", src)                                   # comments may name them
    for word in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMemPool", "cublas", "cusolver", "new ", "malloc(", "std::vector", "admm_internal.h"):
        assert word not in code, word
    assert "static __device__ __align__(256)" in code and "cudaGetSymbolAddress" in code
