"""The C-ABI boundary without a GPU: libqe_hpsi.so builds, loads, and exports every function include/qe_hpsi.h
declares; the ctypes binding names exactly those functions; the entry points that need no device behave as the
header says (status strings, NULL handles, argument errors). No compute call is made here.
PAPER.md:L112/L152/L156 (flat library API), L168 (external H builder)."""
import ctypes
import os
import re

import pytest

from paper_2104_10502_b200 import build as libbuild
from paper_2104_10502_b200 import qe_hpsi

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "qe_hpsi.h")
TEST_HEADER = os.path.join(ROOT, "include", "qe_hpsi_test.h")


def declared_functions(headers=(HEADER, TEST_HEADER)):
    """Names of every function prototype in include/*.h (comments stripped)."""
    src = "\n".join(open(h).read() for h in headers)
    src = re.sub(r"/\*.*?\*/", " ", src, flags=re.S)
    src = re.sub(r"//[^\n]*", " ", src)
    src = re.sub(r"^\s*#.*$", " ", src, flags=re.M)
    names = re.findall(r"\b(qe_hpsi_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


@pytest.fixture(scope="module")
def lib():
    libbuild.build()  # no-op when the .so is newer than its sources; nvcc cross-compiles without a GPU
    return qe_hpsi.load_library()


def test_header_declares_the_three_north_star_calls():
    names = declared_functions()
    for n in ("qe_hpsi_create", "qe_hpsi_apply", "qe_hpsi_destroy", "qe_hpsi_gsphere"):
        assert n in names


def test_library_exports_every_declared_symbol(lib):
    raw = ctypes.CDLL(qe_hpsi.LIB_PATH)
    for n in declared_functions():
        assert hasattr(raw, n), f"{n} declared in include/qe_hpsi.h but not exported by libqe_hpsi.so"


def test_binding_covers_exactly_the_header():
    assert sorted(qe_hpsi.SIGNATURES) == declared_functions()


def test_status_strings(lib):
    seen = set()
    for code in (0, -1, -2, -3, -4, -5):
        s = lib.qe_hpsi_strerror(code).decode()
        assert s and s != "unknown status"
        seen.add(s)
    assert len(seen) == 6
    assert lib.qe_hpsi_strerror(-99).decode() == "unknown status"


def test_null_handle_behaviour(lib):
    null = ctypes.c_void_p(None)
    assert lib.qe_hpsi_destroy(null) == qe_hpsi.QE_HPSI_OK  # header: NULL is a no-op
    assert lib.qe_hpsi_npw(null) == qe_hpsi.QE_HPSI_ESTATE
    assert lib.qe_hpsi_nsticks(null) == qe_hpsi.QE_HPSI_ESTATE
    assert lib.qe_hpsi_nplanes(null) == qe_hpsi.QE_HPSI_ESTATE
    assert lib.qe_hpsi_apply(null, null, 0, null, 0, 1, null) == qe_hpsi.QE_HPSI_ESTATE
    assert lib.qe_hpsi_apply_host(null, null, 0, null, 0, 1) == qe_hpsi.QE_HPSI_ESTATE
    assert lib.qe_hpsi_launch_count(null, 1) == qe_hpsi.QE_HPSI_ESTATE


def test_argument_errors_are_reported_before_any_device_work(lib):
    """EINVAL / EGRID come from host-side validation, so they are testable without a CUDA device."""
    import numpy as np

    at = np.diag([7.0, 7.0, 7.0]).reshape(-1)
    xk = np.zeros(3)
    pd, pi = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int32)
    npw = ctypes.c_int64(0)

    def gs(nr, ecut=8.0, npw_ref=ctypes.byref(npw)):
        n = np.asarray(nr, dtype=np.int32)
        return lib.qe_hpsi_gsphere(at.ctypes.data_as(pd), xk.ctypes.data_as(pd), ecut, n.ctypes.data_as(pi), npw_ref, None)

    assert gs((14, 15, 15)) == qe_hpsi.QE_HPSI_EGRID  # 14 = 2 * 7
    assert gs((5, 15, 15)) == qe_hpsi.QE_HPSI_EGRID  # sphere (|n| <= 3) wider than the box
    assert gs((15, 15, 750)) == qe_hpsi.QE_HPSI_EGRID  # above QE_HPSI_MAX_N
    assert gs((15, 15, 15), ecut=-1.0) == qe_hpsi.QE_HPSI_EINVAL
    assert gs((15, 15, 15), npw_ref=None) == qe_hpsi.QE_HPSI_EINVAL
    out = ctypes.c_void_p(None)
    n = np.asarray((15, 15, 15), dtype=np.int32)
    rc = lib.qe_hpsi_create(ctypes.byref(out), at.ctypes.data_as(pd), 8.0, xk.ctypes.data_as(pd), n.ctypes.data_as(pi),
                            None, 0, None, 0, 0, None, None, 1, 0, None)
    assert rc == qe_hpsi.QE_HPSI_EINVAL and out.value is None  # vr_dev NULL


def test_precision_is_an_explicit_flag_and_bad_flag_words_are_rejected(lib):
    """The accuracy class of the projector contractions is chosen by the caller, never by size or environment; malformed
    flag words are EINVAL before any device work (include/qe_hpsi.h, qe_hpsi_create)."""
    import numpy as np

    at = np.diag([7.0, 7.0, 7.0]).reshape(-1)
    xk = np.zeros(3)
    n = np.asarray((15, 15, 15), dtype=np.int32)
    pd, pi = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int32)
    fake = ctypes.c_void_p(0x1000)  # never dereferenced: the flag check comes first

    def create(flags):
        out = ctypes.c_void_p(None)
        rc = lib.qe_hpsi_create(ctypes.byref(out), at.ctypes.data_as(pd), 8.0, xk.ctypes.data_as(pd), n.ctypes.data_as(pi),
                                fake, 0, None, 0, 0, None, None, 1, flags, None)
        assert out.value is None
        return rc

    q = qe_hpsi
    assert create(1 << 20) == q.QE_HPSI_EINVAL  # unknown bit
    assert create(q.QE_HPSI_FP64_DMMA | q.QE_HPSI_PROJ_INT8) == q.QE_HPSI_EINVAL  # two accuracy classes
    assert create(q.QE_HPSI_PROJ_CERTIFY) == q.QE_HPSI_EINVAL  # certify without the int8 path
    assert create(q.QE_HPSI_PROJ_DIGITS(6)) == q.QE_HPSI_EINVAL  # digits without the int8 path
    assert create(q.QE_HPSI_PROJ_3M_ALL) == q.QE_HPSI_EINVAL
    assert create(q.QE_HPSI_PROJ_INT8 | q.QE_HPSI_PROJ_DIGITS(3)) == q.QE_HPSI_EINVAL  # 4..7 only
    assert create(q.QE_HPSI_PROJ_INT8 | q.QE_HPSI_PROJ_DIGITS(8)) == q.QE_HPSI_EINVAL
    assert q.QE_HPSI_PROJ_DIGITS(6) == 6 << 8 and q.QE_HPSI_PROJ_3M_A6 == 2 << 12
    # the source reads no environment variable that changes the arithmetic
    src = open(os.path.join(ROOT, "paper_2104_10502_b200", "csrc", "qe_hpsi.cu")).read()
    for name in ("QE_HPSI_OZAKI", "QE_HPSI_OZ_3M", "QE_HPSI_OZ_KMAX"):
        assert name not in src


def test_product_header_holds_no_measurement_helpers():
    prod = declared_functions((HEADER,))
    for n in ("qe_hpsi_probe_fp64", "qe_hpsi_profile", "qe_hpsi_profile_read", "qe_hpsi_launch_count", "qe_hpsi_fft_local",
              "qe_hpsi_nonlocal", "qe_hpsi_get_becp", "qe_hpsi_test_set_int8_kmax"):
        assert n not in prod and n in declared_functions((TEST_HEADER,))
    assert "qe_hpsi_last_error" in prod  # SURVEY.md 8(b) name


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    """No fallback: a missing .so is a RuntimeError, never a silent CPU path."""
    monkeypatch.setattr(qe_hpsi, "_lib", None)
    monkeypatch.setattr(qe_hpsi, "LIB_PATH", str(tmp_path / "libqe_hpsi.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        qe_hpsi.load_library()
