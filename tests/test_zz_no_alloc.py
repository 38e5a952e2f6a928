"""frs_dot_noalloc, the one entry point of libfrs.so that allocates nothing (include/frs.h, csrc/k_dot_noalloc.cu).

It is there for callers that cannot let this library call cudaMalloc: a process whose framework allocator has already claimed
the GPU's memory (an allocation behind its back fails, or takes what the framework counted on), and a latency-bound loop in
which cudaMalloc / cudaFree would stall every stream of the device.  Its scratch is a fixed array in the library's device
code that every call shares and that keeps the last call's contents -- so the GPU test makes two calls in a row, the second
on fewer CTAs than the first with the first call's partial sums still lying in the slots beyond them, and holds each against
frs_dot, the existing path through a context.

This file is named to be collected LAST (`pytest --collect-only -q tests`): the suite runs with pytest -x, and a failure here
must not hide the other tests.  It passes on its own in a fresh process (the first call does the per-device set-up) and
after the rest of the suite.
"""
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

# frs_dot is compared with fp64 numpy dots at 1e-12 relative elsewhere (tests/test_gpu_patches.py); the two GPU paths
# run the same arithmetic in the same order, so they are held to that bound against each other and to it against numpy.
RTOL = 1e-12


@pytest.fixture(scope="module")
def frs():
    import paper_2406_09144_b200 as m
    from paper_2406_09144_b200 import build as b
    b.build(verbose=False)
    m.load_library()
    return m


def test_object_file_calls_no_allocating_routine(frs):
    """The translation unit of the entry point refers to no cudaMalloc* / cudaFree* / cudaHostAlloc / stream-ordered
    allocation symbol (what `nm -u` of its object shows), and it does look the scratch address up with
    cudaGetSymbolAddress."""
    obj = os.path.join(ROOT, "paper_2406_09144_b200", "build", "k_dot_noalloc.o")
    assert os.path.exists(obj)
    und = subprocess.run(["nm", "-u", obj], capture_output=True, text=True, check=True).stdout
    names = set(re.findall(r"U (\w+)", und))
    assert "cudaGetSymbolAddress" in names
    banned = [n for n in names if re.search(r"alloc|cudaFree|MemPool|malloc|_Znw|_Zna", n, re.I)]
    assert banned == [], banned


def test_sizes_beyond_the_maximum_are_refused_without_touching_the_gpu(frs):
    """n > FRS_DOT_NOALLOC_MAX_N, a ragged n, NULL and misaligned pointers come back as FRS_EINVAL with a text that says
    why -- checked before any CUDA call, so this runs without a GPU (the pointers are never dereferenced)."""
    lib = frs.lib()
    header = open(os.path.join(ROOT, "include", "frs.h")).read()
    assert re.search(r"#define FRS_DOT_NOALLOC_MAX_N \(1LL << 28\)", header) and frs.FRS_DOT_NOALLOC_MAX_N == 1 << 28
    fake = 1 << 20                                   # aligned, never dereferenced
    assert lib.frs_dot_noalloc(0, None, fake, fake, frs.FRS_DOT_NOALLOC_MAX_N + 4, fake) == frs.FRS_EINVAL
    msg = lib.frs_dot_noalloc_last_error().decode()
    assert "beyond the maximum" in msg and str(1 << 28) in msg
    assert lib.frs_dot_noalloc(0, None, fake, fake, 6, fake) == frs.FRS_EINVAL
    assert "multiple of 4" in lib.frs_dot_noalloc_last_error().decode()
    assert lib.frs_dot_noalloc(0, None, None, fake, 8, fake) == frs.FRS_EINVAL
    assert lib.frs_dot_noalloc(0, None, fake + 4, fake, 8, fake) == frs.FRS_EINVAL
    assert "aligned" in lib.frs_dot_noalloc_last_error().decode()
    assert lib.frs_dot_noalloc(64, None, fake, fake, 8, fake) == frs.FRS_EINVAL


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_existing_path(frs):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    rng = np.random.default_rng(20240609)
    ctx = frs.Context(64, 64, 1)                     # the existing path: frs_dot through a context (which allocates)
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    # first call: 1184 CTAs (the whole scratch array), a ragged tail; second call straight after it: 3 CTAs, other data,
    # with the first call's partials still in slots 3 .. 1183; third: back to a size in between
    for n in (4 * 1_250_003, 4 * 700, 4 * 40_001):
        a = rng.normal(size=n).astype(np.float32)
        b = (rng.normal(size=n) + 0.25 * a).astype(np.float32)
        da, db = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
        out.fill_(float("nan"))
        frs.dot_noalloc(da, db, out)
        got = float(out.item())                      # .item() synchronises the stream the call was enqueued on
        want = ctx.dot(da, db)
        ref = float(np.dot(a.astype(np.float64), b.astype(np.float64)))
        scale = float(np.dot(np.abs(a).astype(np.float64), np.abs(b).astype(np.float64)))
        assert np.isfinite(got)
        assert abs(got - want) <= RTOL * scale, (n, got, want)
        assert abs(got - ref) <= RTOL * scale, (n, got, ref)
        assert got == want, "same arithmetic in the same order: the two paths should agree to the last bit"
    # on a stream of the caller's own, twice over the same input: the same bits both times
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    vals = []
    for _ in range(2):
        out.fill_(float("nan"))
        st.wait_stream(torch.cuda.current_stream())
        frs.dot_noalloc(da, db, out, stream=st)
        st.synchronize()
        vals.append(float(out.item()))
    assert vals[0] == vals[1] == want
    # a refused call enqueues nothing and leaves the output alone
    out.fill_(-1.0)
    with pytest.raises(frs.FrsError, match="multiple of 4"):
        frs.dot_noalloc(da[:6], db[:6], out)
    assert float(out.item()) == -1.0
