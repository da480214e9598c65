import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(autouse=True)
def _guard_bands_checked_at_destroy(monkeypatch, request):
    """Every handle a GPU test destroys first has its guard bands verified (qe_hpsi_test_check_guards): a kernel that wrote
    past the end of any workspace of the handle fails the test that used it. Stands in for compute-sanitizer memcheck, which
    the GPU pool does not run (profiles/r2_sanitizer.md)."""
    from paper_2104_10502_b200 import qe_hpsi

    orig = qe_hpsi.Hpsi.destroy

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value is not None:
            bad = self.check_guards()
            orig(self)
            assert bad == 0, f"{bad} device buffer(s) of the handle were written past their end"
        else:
            orig(self)

    monkeypatch.setattr(qe_hpsi.Hpsi, "destroy", destroy)
    # the Gamma-symmetric projector mode is a scheduling choice from 2^20 entries of beta on; the tests run it on the tiny cases too
    import os
    have = "gpu" in request.node.keywords and os.path.exists(qe_hpsi.LIB_PATH)
    if have:
        qe_hpsi.qe_hpsi_test_set_sym_min(0)
    yield
    if have:
        qe_hpsi.qe_hpsi_test_set_sym_min(-1)
