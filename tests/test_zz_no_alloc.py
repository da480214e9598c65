"""qe_hpsi_overlap_static (include/qe_hpsi.h): the reduced matrix <a_i|b_j> of the iterative diagonaliser (PAPER.md:L162,
L168) from the entry point that allocates nothing -- split-K partials in the library's file-scope device array instead of
a handle's workspace -- against the existing path (Hpsi.overlap on a handle) on the same inputs, two calls in a row.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

from paper_2104_10502_b200 import qe_hpsi
from tests import _gpu

pytestmark = pytest.mark.gpu


def _scale(a, b, npw):
    an = torch.linalg.vector_norm(a[:, :npw], dim=1)
    bn = torch.linalg.vector_norm(b[:, :npw], dim=1)
    return (an[:, None] * bn[None, :]).cpu().numpy()


@pytest.mark.parametrize("cfg,na,nb", [("T1_general_k", 5, 7), (1, 128, 128), (1, 37, 61)])
def test_overlap_static_matches_the_handle_path_on_two_calls_in_a_row(cfg, na, nb):
    h, inp = _gpu.make(cfg)
    npw = h.npw
    a1 = _gpu.gen_psi_dev(inp, 0, na)
    b1 = _gpu.gen_psi_dev(inp, 100, nb)
    a2 = _gpu.gen_psi_dev(inp, 300, na)  # second call: other inputs, so stale partials of the first would show
    b2 = _gpu.gen_psi_dev(inp, 17, nb)
    qe_hpsi.qe_hpsi_overlap_static_init()
    for a, b in ((a1, b1), (a2, b2)):
        ref = h.overlap(a, b)
        out = torch.full((na, nb + 3), 9.0, dtype=torch.complex128, device="cuda")
        qe_hpsi.qe_hpsi_overlap_static(a, b, npw, out[:, :nb])
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        err = np.abs(got[:, :nb] - ref.cpu().numpy()) / _scale(a, b, npw)
        assert err.max() <= 1e-13  # the tolerance of test_overlap_against_oracle: |error| <= 1e-13 |a||b|
        assert np.all(got[:, nb:] == 9.0)
        # same K slices, kernel and reduction order: in fact the same bits
        assert torch.equal(out[:, :nb].contiguous().view(torch.float64), ref.contiguous().view(torch.float64))
    h.destroy()


def test_overlap_static_rejects_sizes_beyond_the_static_scratch_and_allocates_nothing():
    n = qe_hpsi.QE_HPSI_OVERLAP_STATIC_MAX
    a = torch.zeros((n + 1, 64), dtype=torch.complex128, device="cuda")
    b = torch.zeros((4, 64), dtype=torch.complex128, device="cuda")
    out = torch.full((n + 1, n + 1), 5.0, dtype=torch.complex128, device="cuda")
    with pytest.raises(qe_hpsi.QeHpsiError) as ei:
        qe_hpsi.qe_hpsi_overlap_static(a, b, 64, out[:, :4])
    assert ei.value.status == -1  # QE_HPSI_EINVAL
    with pytest.raises(qe_hpsi.QeHpsiError):
        qe_hpsi.qe_hpsi_overlap_static(b, a, 64, out[:4, :])
    with pytest.raises(qe_hpsi.QeHpsiError):
        qe_hpsi.qe_hpsi_overlap_static(b, b, 65, out[:4, :4])  # ld < npw
    torch.cuda.synchronize()
    assert torch.all(out == 5.0)
    # no device memory is taken by a call (the driver's free-memory figure before and after)
    qe_hpsi.qe_hpsi_overlap_static(b, b, 64, out[:4, :4])
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        qe_hpsi.qe_hpsi_overlap_static(b, b, 64, out[:4, :4])
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    assert torch.all(out[:4, :4] == 0.0)  # zero inputs: every partial of the call was written, none left over
    # npw = 0: zeros, rest untouched
    out.fill_(5.0)
    qe_hpsi.qe_hpsi_overlap_static(b, b, 0, out[:4, :4])
    torch.cuda.synchronize()
    assert torch.all(out[:4, :4] == 0.0) and torch.all(out[4:, :] == 5.0)
