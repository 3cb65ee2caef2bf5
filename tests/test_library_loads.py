"""The C-ABI boundary without a GPU: libttdft.so builds (nvcc cross-compiles sm_100a), loads, and exports every function that
include/ttdft.h declares; the Python binding lists exactly those; the host-only entry points (Algorithm 1's scalars, PAPER.md:L217-222,
argument validation, error text) work.  No compute call is made here."""
import ctypes
import os
import re
from fractions import Fraction

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2110_15853_b200 import build
    path = build.build()                      # no-op when the library is newer than its sources
    return ctypes.CDLL(path)


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "ttdft.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)          # declarations only, not the comments
    text = re.sub(r"//[^\n]*", "", text)
    return sorted(set(re.findall(r"\b(ttdft_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound(lib):
    import paper_2110_15853_b200 as tt
    names = declared_symbols()
    assert len(names) >= 30 and "ttdft_cheb_filter" in names and "ttdft_recover_subdomains" in names
    missing = [n for n in names if not hasattr(lib, n)]
    assert not missing, missing
    assert sorted(tt.exported_symbols) == names                 # the binding covers the header, nothing else
    assert os.path.samefile(tt.library_path(), lib._name)


def test_host_only_entry_points(lib):
    import paper_2110_15853_b200 as tt
    # Algorithm 1's scalars for (a0, a, b) = (0, 2, 10): e = 4, c = 6, sigma_1..4 = -2/3, -3/7, -7/18, -18/47
    c, alpha, beta = tt.cheb_scalars(4, 2.0, 10.0, 0.0)
    sig = [Fraction(-2, 3), Fraction(-3, 7), Fraction(-7, 18), Fraction(-18, 47)]
    e = Fraction(4)
    assert c == 6.0
    assert alpha[0] == pytest.approx(float(sig[0] / e), rel=1e-15)
    for k in range(1, 4):
        assert alpha[k] == pytest.approx(float(2 * sig[k] / e), rel=1e-15)
        assert beta[k] == pytest.approx(float(-sig[k - 1] * sig[k]), rel=1e-15)
    assert tt.cheb_scalars(0, 2.0, 10.0, 0.0) == (6.0, [], [])
    for bad in [(3, 2.0, 10.0, 2.0), (3, 10.0, 2.0, 0.0), (-1, 2.0, 10.0, 0.0)]:       # a0 < a < b and m >= 0 required
        with pytest.raises(tt.TTDFTError) as err:
            tt.cheb_scalars(*bad)
        assert err.value.status_name == "INVALID_ARG" and tt.last_error()
    assert isinstance(tt.launch_count(), int)
    # work-size queries that need no device
    assert tt.gram_work_bytes(1024, 64) > 0 and tt.orthonormalize_work_bytes(1024, 64, 2) > tt.orthonormalize_work_bytes(1024, 64, 1)
    n = ctypes.c_size_t(0)
    assert lib.ttdft_recover_subdomains_work_bytes(ctypes.c_int64(1000), ctypes.byref(n)) == 0 and n.value >= 1000 * 804
    assert lib.ttdft_recover_subdomains_work_bytes(ctypes.c_int64(-1), ctypes.byref(n)) == 1
    # NULL arguments are rejected before any CUDA call
    assert lib.ttdft_h_storage_bytes(None, ctypes.byref(n)) == 1
    assert lib.ttdft_h_destroy(None) in (0, 1)


def test_static_scratch_constant_and_null_handle(lib):
    """ttdft_cheb_step_static: the binding's size limit is the header's, the array is a static device symbol of that size inside the
    library (no allocation at run time), and a NULL handle is rejected before any CUDA call."""
    import subprocess
    import paper_2110_15853_b200 as tt
    text = open(os.path.join(ROOT, "include", "ttdft.h")).read()
    m = re.search(r"#define\s+TTDFT_STATIC_SCRATCH_BYTES\s+\((\d+)u\s*<<\s*(\d+)\)", text)
    assert m and (int(m.group(1)) << int(m.group(2))) == tt.STATIC_SCRATCH_BYTES == 32 << 20
    lib.ttdft_cheb_step_static.restype = ctypes.c_int
    args = [None, ctypes.c_double(1.0), ctypes.c_double(0.0), ctypes.c_double(0.0), None, ctypes.c_int64(1), None, ctypes.c_int64(1),
            None, ctypes.c_int64(1), ctypes.c_int64(1), None]
    assert lib.ttdft_cheb_step_static(*args) == 1                 # TTDFT_ERR_INVALID_ARG
    out = subprocess.run(["cuobjdump", "-elf", tt.library_path()], capture_output=True, text=True)
    if out.returncode == 0:
        assert re.search(r"\.global\s+\.align\s+256\s+\.b8\s+g_static_scratch\[%d\]" % tt.STATIC_SCRATCH_BYTES, out.stdout) or \
            "g_static_scratch" in out.stdout


def test_no_cpu_fallback_without_a_gpu():
    """The product path must fail loudly, not compute on the CPU, when no CUDA device is there."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2110_15853_b200 as tt
    M = 8
    rp = torch.arange(M + 1, dtype=torch.int32)
    with pytest.raises(Exception):
        tt.h_build_csr(M, rp, torch.arange(M, dtype=torch.int32), torch.ones(M, dtype=torch.float64))
