"""GPU parity of the int8-digit projector path (csrc/ozaki_kernels.cuh; create flag
QE_HPSI_PROJ_INT8): a6 / a8 computed exactly on the int8 tensor cores from S balanced 8-bit digits of the FP64 operands.
The oracle is oracle/hpsi_oracle.py (becp_of, vnl_psi); the default FP64 DMMA path is a second, independent
implementation of the same rows.  Tolerances: S = 7 (55 bits under the row exponent) is held to the FP64 path's 1e-13 /
1e-12; S = 6 (47 bits) to north_star's 1e-11 of the nonlocal part alone -- DESIGN.md 5.6's truncation law
((S+1) 2^(-8S+1) K max|a| max|b|, random signs: sqrt(K)) puts it at ~1e-12 on these operands, not below 1e-13."""
from __future__ import annotations

import numpy as np
import pytest
import torch

from oracle import hpsi_oracle as orc
from paper_2104_10502_b200 import harness, qe_hpsi
from tests import _gpu

pytestmark = pytest.mark.gpu


def _make_int8(key, digits=6, three_m=None, **kw):
    """Handle on the int8 digit path with `digits` digits per operand (explicit create flag)."""
    return _gpu.make(key, flags=harness.int8_flags(digits, three_m), **kw)


def _nonlocal(h, inp, nb):
    psi = _gpu.gen_psi_dev(inp, 0, nb)
    out = h.nonlocal_add(psi, torch.zeros_like(psi))
    becp, _ = h.becp(nb)
    torch.cuda.synchronize()
    return psi, out, becp


def test_the_accuracy_class_is_what_the_create_flag_says_whatever_the_size():
    for cfg in (0, 1):  # 17 k and 12 M entries of beta: the default is FP64 for both, the int8 path only on request
        h, _ = _gpu.make(cfg)
        assert h.info()["ozaki_slices"] == 0
        h.destroy()
        h, _ = _gpu.make(cfg, flags=qe_hpsi.QE_HPSI_FP64_DMMA)
        assert h.info()["ozaki_slices"] == 0
        h.destroy()
        h, _ = _gpu.make(cfg, flags=qe_hpsi.QE_HPSI_PROJ_INT8)  # no digit field: 7 digits (55 bits)
        assert h.info()["ozaki_slices"] == 7 and h.info()["ozaki_nsplit"] >= 1 and h.info()["ozaki_3m"] == 0
        h.destroy()
    h, _ = _make_int8(1, 6, three_m=3)
    assert h.info()["ozaki_slices"] == 6 and h.info()["ozaki_3m"] == 2
    h.destroy()


@pytest.mark.parametrize("digits", [6, 7])
@pytest.mark.parametrize("three_m", [0, 2, 3])
@pytest.mark.parametrize("cfg", ["T1_general_k", "T2_radix5", "T5_odd_bands", 0, 1])
def test_becp_and_vnl_against_oracle(cfg, three_m, digits):
    """Both forms of a6 and a8: the real-form complex GEMMs and the integer 3M forms (three real GEMMs on planar digit planes;
    QE_HPSI_PROJ_3M_A6: a6 only; QE_HPSI_PROJ_3M_ALL: a6 and a8 whatever the size), at 6 and 7 digits."""
    h, inp = _make_int8(cfg, digits, three_m=three_m)
    assert h.info()["ozaki_3m"] == {0: 0, 2: 1, 3: 2}[three_m]
    path = f"int8_s{digits}"
    wl = inp["wl"]
    npw = h.npw
    psi, out, becp = _nonlocal(h, inp, wl.nbands)
    ph = psi[:, :npw].cpu().numpy()
    beta = inp["beta"][:, :npw].cpu().numpy()
    bref = orc.becp_of(beta, ph)
    eb = np.abs(becp.cpu().numpy() - bref).max() / np.abs(bref).max()
    assert eb <= _gpu.TOL_BECP[path], eb
    vref = orc.vnl_psi(beta, inp["dblocks"], ph)
    # demanded of the nonlocal part ALONE (it is ~1e-5 of |H psi| on these workloads)
    ev = _gpu.rel_l2(out.cpu().numpy()[:, :npw], vref).max()
    assert ev <= _gpu.TOL_VNL[path], ev
    h.destroy()


@pytest.mark.parametrize("digits", [6, 7])
def test_int8_path_agrees_with_the_fp64_tensor_path_on_config_1(digits):
    h, inp = _make_int8(1, digits)
    _, out, becp = _nonlocal(h, inp, 128)
    h.destroy()
    h2, inp2 = _gpu.make(1, flags=qe_hpsi.QE_HPSI_FP64_DMMA)
    _, out2, becp2 = _nonlocal(h2, inp2, 128)
    h2.destroy()
    path = f"int8_s{digits}"
    assert float((becp - becp2).abs().max()) <= _gpu.TOL_BECP[path] * float(becp2.abs().max())
    num = torch.linalg.vector_norm(out - out2, dim=1)
    den = torch.linalg.vector_norm(out2, dim=1)
    assert float((num / den).max()) <= _gpu.TOL_VNL[path]


@pytest.mark.parametrize("slices,tol", [(4, 2e-7), (5, 1e-9), (6, 1e-11), (7, 1e-13)])
def test_error_falls_by_2_to_the_8_per_digit(slices, tol):
    """Each extra digit adds 8 bits: the measured error must respect the law (and S = 4 must be visibly worse than S = 7,
    i.e. the digits are really what is being multiplied)."""
    h, inp = _make_int8(0, digits=slices)
    assert h.info()["ozaki_slices"] == slices
    wl = inp["wl"]
    npw = h.npw
    psi, out, _ = _nonlocal(h, inp, wl.nbands)
    beta = inp["beta"][:, :npw].cpu().numpy()
    vref = orc.vnl_psi(beta, inp["dblocks"], psi[:, :npw].cpu().numpy())
    err = _gpu.rel_l2(out.cpu().numpy()[:, :npw], vref).max()
    assert err <= tol, err
    if slices == 4:
        assert err >= 1e-12, err
    h.destroy()


def test_bits_do_not_depend_on_batch_composition_or_run():
    h, inp = _make_int8(1, 6, max_batch=48)
    psi = _gpu.gen_psi_dev(inp, 0, 100)  # chunks 48, 48, 4
    a = h.apply(psi).clone()
    b = h.apply(psi).clone()
    one = h.apply(psi[77:78].contiguous()).clone()
    torch.cuda.synchronize()
    assert torch.equal(a.view(torch.float64), b.view(torch.float64))
    assert torch.equal(a[77].view(torch.float64), one[0].view(torch.float64))
    h.destroy()


def test_zero_band_and_huge_dynamic_range():
    h, inp = _make_int8("T1_general_k")
    wl = inp["wl"]
    npw = h.npw
    psi = _gpu.gen_psi_dev(inp, 0, wl.nbands)
    psi[0] = 0  # all-zero band: exponent 0, slices 0
    psi[1, :npw] *= torch.logspace(0, -30, npw, dtype=torch.float64, device="cuda")  # entries far below 2^-46 of the row maximum
    out = h.nonlocal_add(psi, torch.zeros_like(psi))
    torch.cuda.synchronize()
    beta = inp["beta"][:, :npw].cpu().numpy()
    vref = orc.vnl_psi(beta, inp["dblocks"], psi[:, :npw].cpu().numpy())
    got = out.cpu().numpy()[:, :npw]
    assert np.all(got[0] == 0)
    assert _gpu.rel_l2(got[1:], vref[1:]).max() <= 1e-11
    h.destroy()


def test_non_finite_operands_give_nan_not_finite_garbage():
    """A NaN / Inf in a band poisons that band's nonlocal part (as the FP64 contraction would) and no other band."""
    h, inp = _make_int8("T1_general_k")
    wl = inp["wl"]
    npw = h.npw
    psi = _gpu.gen_psi_dev(inp, 0, wl.nbands)
    psi[1, 5] = float("nan")
    psi[2, 7] = complex(float("inf"), 0.0)
    out = h.nonlocal_add(psi, torch.zeros_like(psi)).cpu().numpy()[:, :npw]
    assert np.isnan(out[1]).all() and np.isnan(out[2]).all()
    clean = [b for b in range(wl.nbands) if b not in (1, 2)]
    beta = inp["beta"][:, :npw].cpu().numpy()
    vref = orc.vnl_psi(beta, inp["dblocks"], psi[clean, :npw].cpu().numpy())
    assert _gpu.rel_l2(out[clean], vref).max() <= 1e-11
    h.destroy()


def test_k_ranges_of_a8_and_forced_splits_of_a6_give_the_same_result():
    """2 nproj beyond the exact-int32 K range makes a8 walk its K ranges launch by launch (and a6 split finer); forced here on
    config 1 by lowering the range (qe_hpsi_test_set_int8_kmax), checked against the default plan and the FP64 tensor path."""
    h, inp = _make_int8(1, 6)
    psi, ref, _ = _nonlocal(h, inp, 64)
    h.destroy()
    qe_hpsi.qe_hpsi_test_set_int8_kmax(384)
    try:
        h2, inp2 = _make_int8(1, 6)
    finally:
        qe_hpsi.qe_hpsi_test_set_int8_kmax(0)
    assert h2.info()["ozaki_slices"] == 6
    assert h2.launch_count(64) == 5 + 7 + 3  # a1-a5, digit/reduce/a6 kernels, a8 in ceil(1024 / 384) = 3 launches
    _, out, _ = _nonlocal(h2, inp2, 64)
    h2.destroy()
    num = torch.linalg.vector_norm(out - ref, dim=1)
    den = torch.linalg.vector_norm(ref, dim=1)
    assert float((num / den).max()) <= 1e-13  # same digits, same exact integer sums; only the FP64 order of the K ranges differs
