"""CPU-only checks of the product side: the library builds for sm_100a, exports every symbol
include/frs.h declares, its host-replayable FFT logic is right, and it refuses to run without a GPU."""
import os
import re

import numpy as np
import pytest

import paper_2406_09144_b200 as frs
from paper_2406_09144_b200 import build as frs_build
from oracle import frs_oracle as o

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def library():
    frs_build.build(verbose=False)
    return frs.load_library()


def test_library_exports_every_declared_symbol(library):
    header = open(os.path.join(ROOT, "include", "frs.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(frs_[a-z_0-9]+)\s*\(", header))
    assert declared == set(frs.EXPORTS), declared ^ set(frs.EXPORTS)
    for name in declared:
        assert hasattr(library, name)
    assert b"sm_100a" in library.frs_version()


@pytest.mark.parametrize("n", [16, 32, 64, 128, 256, 512, 1024, 2048, 4096])
def test_stage_logic_replayed_on_cpu_matches_dft(library, n):
    rng = np.random.default_rng(n)
    x = (rng.normal(size=n) + 1j * rng.normal(size=n)).astype(np.complex64)
    ref = np.fft.fft(x.astype(np.complex128))
    if n <= 64:
        ref = o.dft_naive(x.astype(np.complex128))
    got = frs.selftest_fft_host(x)
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) < 5e-7
    inv = frs.selftest_fft_host(got, inverse=True)
    assert np.linalg.norm(inv / n - x) / np.linalg.norm(x) < 1e-6
    # a delta at position q -> pure phase ramp: catches any index permutation exactly
    for q in (1, n // 2 + 1, n - 1):
        d = np.zeros(n, np.complex64)
        d[q] = 1
        assert np.allclose(frs.selftest_fft_host(d), np.exp(-2j * np.pi * q * np.arange(n) / n), atol=2e-6)


@pytest.mark.parametrize("n", [256, 512, 1024, 2048, 4096])
def test_dif_core_replayed_on_cpu_matches_dft(library, n):
    """The DIF/DIT core of the column convolution (csrc/fft_dif.cuh), replayed thread by thread: the permuted spectrum,
    sorted through its own register <-> frequency map, is the DFT; the inverse brings a sorted spectrum back."""
    rng = np.random.default_rng(100 + n)
    x = (rng.normal(size=n) + 1j * rng.normal(size=n)).astype(np.complex64)
    ref = np.fft.fft(x.astype(np.complex128))
    got = frs.selftest_dif_host(x)
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) < 8e-7
    inv = frs.selftest_dif_host(got, inverse=True)
    assert np.linalg.norm(inv / n - x) / np.linalg.norm(x) < 1.5e-6
    for q in (1, n // 2 + 1, n - 1):
        d = np.zeros(n, np.complex64)
        d[q] = 1
        assert np.allclose(frs.selftest_dif_host(d), np.exp(-2j * np.pi * q * np.arange(n) / n), atol=3e-6)
        assert np.allclose(frs.selftest_dif_host(d, inverse=True), np.exp(2j * np.pi * q * np.arange(n) / n), atol=3e-6)
    with pytest.raises(frs.FrsError):
        frs.selftest_dif_host(np.zeros(128, np.complex64))


@pytest.mark.parametrize("n", [256, 512, 1024, 2048, 4096])
def test_dif_exchange_is_race_free_and_conflict_free(library, n):
    """What compute-sanitizer's racecheck would look at (the tool is closed on the GPU pool, profiles/r2_sanitizer.md):
    every shared-memory access of two consecutive columns, lane by lane -- no two threads touch a slot (one of them
    writing) without a barrier that orders them (a block barrier, or a warp sync between lanes of one warp), no slot
    out of range, no bank conflict in any 128-bit access, and the register <-> frequency map is a bijection."""
    conflict, hazards, oob, used, alloc, dup = frs.selftest_dif_exchange(n)
    assert conflict == 1 and hazards == 0 and oob == 0 and dup == 0
    assert used == n and used <= alloc


@pytest.mark.parametrize("nf", [16, 32, 64, 128, 256, 512, 1024, 2048, 4096])
def test_tma_copy_geometry_covers_and_fits(library, nf):
    """The tensor copies that feed the passes (csrc/tmap.h): the row gather must cover all nf + 1 bins of a
    row pair, land inside the exchange buffer, and use 128-byte aligned boxes whenever TMA is used; the
    column copies must tile a column of `rows` samples exactly."""
    for rows in (32, 256, 4096):
        box_bins, bin_copies, box_pairs, col_copies, xbuf, use_tma = frs.selftest_tma_geometry(nf, rows)
        assert box_bins * bin_copies >= nf + 1                      # every bin kx = 0..nf is fetched
        assert box_bins * (bin_copies - 1) < nf + 1                 # ... by no more copies than needed
        assert box_bins * bin_copies <= xbuf                        # 16-byte slots: lands inside the buffer
        assert xbuf % 8 == 0 and xbuf >= nf + nf // 16              # 128-byte multiple, padded positions fit
        if use_tma:
            assert (box_bins * 16) % 128 == 0                       # consecutive boxes stay 128-byte aligned
        assert box_pairs * col_copies == rows // 2 and box_pairs <= 256
        assert (box_pairs * 16) % 128 == 0
    with pytest.raises(frs.FrsError):
        frs.selftest_tma_geometry(24, 64)


def test_selftest_rejects_bad_sizes(library):
    with pytest.raises(frs.FrsError):
        frs.selftest_fft_host(np.zeros(24, np.complex64))


def test_no_cpu_fallback(library):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        frs.Context(64, 64)
    import ctypes as C
    h = C.c_void_p()
    assert library.frs_create(64, 64, 1, 0, None, C.byref(h)) == frs.FRS_ECUDA
    assert library.frs_create(48, 64, 1, 0, None, C.byref(h)) == frs.FRS_EINVAL      # not a power of two
    assert library.frs_create(64, 8192, 1, 0, None, C.byref(h)) == frs.FRS_EINVAL


def test_tf32_dft_stage_needs_the_three_term_split():
    """Arithmetic of the tensor-core alternative: a radix-16 DFT stage as a TF32 GEMM.  One pass of
    TF32 (10-bit mantissa, fp32 accumulate) misses the 1e-5 parity bar by two orders of magnitude; the 3-term split
    x_hi W_hi + x_lo W_hi + x_hi W_lo meets it -- at three times the tensor-core work.  Emulated in numpy."""
    def tf32(a):
        b = np.asarray(a, np.float32).view(np.uint32)
        b = (b + np.uint32(0x1000)) & np.uint32(0xFFFFE000)          # round to 10 explicit mantissa bits
        return b.view(np.float32)
    rng = np.random.default_rng(16)
    x = rng.normal(size=(4096, 16)) + 1j * rng.normal(size=(4096, 16))
    w = np.exp(-2j * np.pi * np.outer(np.arange(16), np.arange(16)) / 16)
    ref = x @ w
    xr = np.concatenate([x.real, x.imag], 1).astype(np.float32)      # [p][32] real form
    wr = np.block([[w.real, w.imag], [-w.imag, w.real]]).astype(np.float32)   # [32][32]
    def gemm(a, b):                                                  # exact products of tf32 operands, fp32 accumulate
        return (a.astype(np.float64) @ b.astype(np.float64)).astype(np.float32)
    def err(y):
        return np.linalg.norm((y[:, :16] + 1j * y[:, 16:]) - ref) / np.linalg.norm(ref)
    one = gemm(tf32(xr), tf32(wr))
    xh, wh = tf32(xr), tf32(wr)
    xl, wl = tf32(xr - xh), tf32(wr - wh)
    three = gemm(xh, wh) + gemm(xl, wh) + gemm(xh, wl)
    assert err(one) > 1e-4                                           # ~3e-4: fails the bar on its own
    assert err(three) < 2e-6                                         # the split restores fp32-class accuracy


def test_amp_model_size_matches_oracle_bins():
    """frs_amp_model_size is host arithmetic (no GPU): bins and theta length of the radial grid equal the oracle's."""
    import ctypes as C
    from oracle import prior_oracle as po
    import paper_2406_09144_b200 as frs
    lib = frs.load_library()
    for ny, nx in ((32, 32), (64, 256), (512, 128), (1024, 1024)):
        nb, nt = C.c_int(0), C.c_int(0)
        assert lib.frs_amp_model_size(ny, nx, C.byref(nb), C.byref(nt)) == 0
        t = po.bins(ny, nx)[2]
        assert nb.value == len(t) and nt.value == po.ntheta(len(t))
    assert lib.frs_amp_model_size(48, 32, C.byref(nb), C.byref(nt)) != 0
