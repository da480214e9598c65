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


def _make_int8(key, digits=6, three_m=None, nosym=False, **kw):
    """Handle on the int8 digit path with `digits` digits per operand (explicit create flag). nosym: keep the general complex
    contraction at k = 0 (QE_HPSI_NO_GAMMA_SYM), where the default is the Gamma-symmetric real form over the half sphere."""
    return _gpu.make(key, flags=harness.int8_flags(digits, three_m) | (qe_hpsi.QE_HPSI_NO_GAMMA_SYM if nosym else 0), **kw)


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
        assert h.info()["gamma_sym"] == 1  # k = 0, generator projectors: real forms over the half sphere
        h.destroy()
    h, _ = _make_int8(1, 6, three_m=3, nosym=True)
    assert h.info()["ozaki_slices"] == 6 and h.info()["ozaki_3m"] == 2 and h.info()["gamma_sym"] == 0
    h.destroy()


@pytest.mark.parametrize("digits", [6, 7])
@pytest.mark.parametrize("three_m", [0, 2, 3, "sym"])
@pytest.mark.parametrize("cfg", ["T1_general_k", "T2_radix5", "T5_odd_bands", 0, 1])
def test_becp_and_vnl_against_oracle(cfg, three_m, digits):
    """All forms of a6 and a8: the real-form complex GEMMs, the integer 3M forms (three real GEMMs on planar digit planes;
    QE_HPSI_PROJ_3M_A6: a6 only; QE_HPSI_PROJ_3M_ALL: a6 and a8 whatever the size) -- all with QE_HPSI_NO_GAMMA_SYM so that the
    k = 0 cases take them too -- and ("sym") the default: at k = 0 the Gamma-symmetric real forms over the half sphere."""
    if three_m == "sym":
        h, inp = _make_int8(cfg, digits)
        assert h.info()["gamma_sym"] == (0 if cfg in ("T1_general_k", "T5_odd_bands") else 1) and h.info()["ozaki_3m"] == 0
    else:
        h, inp = _make_int8(cfg, digits, three_m=three_m, nosym=True)
        assert h.info()["ozaki_3m"] == {0: 0, 2: 1, 3: 2}[three_m] and h.info()["gamma_sym"] == 0
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
    h, inp = _make_int8(1, 6, nosym=True)
    psi, ref, _ = _nonlocal(h, inp, 64)
    h.destroy()
    qe_hpsi.qe_hpsi_test_set_int8_kmax(384)
    try:
        h2, inp2 = _make_int8(1, 6, nosym=True)
        h3, inp3 = _make_int8(1, 6)  # the symmetric real forms: K of a8 is nproj = 512 -> 2 ranges
    finally:
        qe_hpsi.qe_hpsi_test_set_int8_kmax(0)
    assert h2.info()["ozaki_slices"] == 6
    assert h2.launch_count(64) == 5 + 7 + 3  # a1-a5, digit/reduce/a6 kernels, a8 in ceil(1024 / 384) = 3 launches
    assert h3.info()["gamma_sym"] == 1 and h3.launch_count(64) == 5 + 9 + 2
    _, out, _ = _nonlocal(h2, inp2, 64)
    _, out3, _ = _nonlocal(h3, inp3, 64)
    h2.destroy()
    h3.destroy()
    n3 = torch.linalg.vector_norm(out3 - ref, dim=1) / torch.linalg.vector_norm(ref, dim=1)
    assert float(n3.max()) <= 1e-11  # other digits (half-sphere rows): agreement at the accuracy class, not bitwise
    num = torch.linalg.vector_norm(out - ref, dim=1)
    den = torch.linalg.vector_norm(ref, dim=1)
    assert float((num / den).max()) <= 1e-13  # same digits, same exact integer sums; only the FP64 order of the K ranges differs


# ---- QE_HPSI_PROJ_CERTIFY: a-posteriori check + FP64 re-computation -----------------------------------
def _outer_shell_psi(inp, sp, nb, frac=0.9):
    """Adversarial bands for a per-row-exponent fixed-point scheme: psi lives only on the outer shell |k+G|^2 > frac ecut,
    where the Gaussian projectors are 1e-5 .. 1e-10 of their row maxima, so <beta|psi> is carried by digits the 47-bit split
    has mostly truncated (config 1: e^(-q^2 rc^2 / 2) = 7e-5 at rc 0.8 and 4e-10 at rc 1.2 for q^2 = 30)."""
    psi = _gpu.gen_psi_dev(inp, 300, nb)
    wl = inp["wl"]
    shell = torch.as_tensor(sp["g2kin"] > frac * wl.ecutwfc, device="cuda")
    psi[:, :shell.numel()] *= shell.to(torch.complex128)[None]
    psi /= torch.linalg.vector_norm(psi, dim=1)[:, None]
    return psi


def test_certified_path_recomputes_the_bands_the_47_bit_split_gets_wrong():
    """S = 6 WITHOUT the certificate exceeds north_star's 1e-11 on the nonlocal part of outer-shell bands; the certified handle
    flags exactly those bands, re-computes them on the FP64 tensor path and meets the tolerance; ordinary bands in the same
    call keep their int8 result."""
    h6, inp = _make_int8(1, 6)
    wl = inp["wl"]
    sp = _gpu.oracle_sphere(wl)
    npw = h6.npw
    n_adv, n_ok = 5, 7
    psi = torch.cat([_gpu.gen_psi_dev(inp, 0, n_ok), _outer_shell_psi(inp, sp, n_adv)])
    order = torch.as_tensor([0, 7, 1, 8, 2, 9, 3, 10, 4, 11, 5, 6], device="cuda")  # interleave: adversarial bands at 1, 3, 5, 7, 9
    psi = psi[order].contiguous()
    adv = np.array([1, 3, 5, 7, 9])
    ok = np.array([b for b in range(n_adv + n_ok) if b not in adv])
    beta = inp["beta"][:, :npw].cpu().numpy()
    vref = orc.vnl_psi(beta, inp["dblocks"], psi[:, :npw].cpu().numpy())
    plain = h6.nonlocal_add(psi, torch.zeros_like(psi)).cpu().numpy()[:, :npw]
    e_plain = _gpu.rel_l2(plain, vref)
    assert e_plain[adv].min() > 1e-11, e_plain  # the uncertified 47-bit path really fails here ...
    assert e_plain[ok].max() <= 1e-11, e_plain  # ... and only here
    h6.destroy()
    hc, _ = _gpu.make(1, flags=harness.int8_flags(6, certify=True), beta=inp["beta"])
    assert hc.info()["certify"] == 1
    sent = torch.zeros_like(psi)
    sent[:, npw:] = 3.0  # pad columns must stay untouched
    out = hc.nonlocal_add(psi, sent)
    rel, redo = hc.proj_check(psi.shape[0])
    torch.cuda.synchronize()
    got = out.cpu().numpy()[:, :npw]
    e_cert = _gpu.rel_l2(got, vref)
    redo = redo.cpu().numpy()
    rel = rel.cpu().numpy()
    assert np.array_equal(np.nonzero(redo)[0], adv), (redo, rel)
    assert e_cert.max() <= 1e-11, e_cert
    assert np.all(out.cpu().numpy()[:, npw:] == 3.0)
    # qe_hpsi_nonlocal accumulates on top of the caller's array in this mode too
    base = torch.as_tensor(vref, device="cuda") * (0.5 - 0.25j)
    acc = torch.zeros_like(psi)
    acc[:, :npw] = base
    hc.nonlocal_add(psi, acc)
    torch.cuda.synchronize()
    assert _gpu.rel_l2(acc.cpu().numpy()[:, :npw], vref * (1.5 - 0.25j)).max() <= 1e-11
    # the estimate tracks the true error of the int8 result (within the factor the 8 probes give), flagged or not
    ratio = rel / np.maximum(e_plain, 1e-300)
    assert np.all(ratio > 0.3) and np.all(ratio < 3.0), (rel, e_plain)
    # the whole H psi through qe_hpsi_apply takes the same decision and is the FP64 handle's result for the flagged bands
    hps = hc.apply(psi)
    _, redo2 = hc.proj_check(psi.shape[0])
    assert np.array_equal(redo2.cpu().numpy(), redo)
    hf, _ = _gpu.make(1, beta=inp["beta"], flags=qe_hpsi.QE_HPSI_NO_GAMMA_SYM)  # the re-computation is the general complex contraction
    ref = hf.apply(psi)
    torch.cuda.synchronize()
    d = torch.linalg.vector_norm(hps[:, :npw] - ref[:, :npw], dim=1) / torch.linalg.vector_norm(ref[:, :npw], dim=1)
    assert float(d.max()) <= 1e-13
    # a looser caller tolerance keeps every int8 result; tolerance 0 re-computes everything
    hc.set_proj_tolerance(1e-3)
    hc.nonlocal_add(psi, torch.zeros_like(psi))
    assert int(hc.proj_check(psi.shape[0])[1].sum()) == 0
    hc.set_proj_tolerance(0.0)
    allf = hc.nonlocal_add(psi, torch.zeros_like(psi))
    assert int(hc.proj_check(psi.shape[0])[1].sum()) == psi.shape[0]
    fp = hf.nonlocal_add(psi, torch.zeros_like(psi))
    torch.cuda.synchronize()
    assert torch.equal(allf[:, :npw].view(torch.float64), fp[:, :npw].view(torch.float64))  # the re-computation IS the FP64 path
    hc.destroy()
    hf.destroy()


@pytest.mark.parametrize("cfg", ["T1_general_k", "T5_odd_bands", 0])
def test_certified_path_small_cases_chunking_nan_and_graph(cfg):
    """max_batch smaller than the probe count and than the band count (several chunks), a NaN band (re-computed: FP64
    semantics), bit-reproducibility, and CUDA-graph capture (the decision never leaves the device)."""
    hc, inp = _gpu.make(cfg, flags=harness.int8_flags(6, three_m=3, certify=True), max_batch=3)
    wl = inp["wl"]
    npw = hc.npw
    psi = _gpu.gen_psi_dev(inp, 0, wl.nbands)
    beta = inp["beta"][:, :npw].cpu().numpy()
    vref = orc.vnl_psi(beta, inp["dblocks"], psi[:, :npw].cpu().numpy())
    a = hc.nonlocal_add(psi, torch.zeros_like(psi))
    b = hc.nonlocal_add(psi, torch.zeros_like(psi))
    torch.cuda.synchronize()
    assert torch.equal(a.view(torch.float64), b.view(torch.float64))
    assert _gpu.rel_l2(a.cpu().numpy()[:, :npw], vref).max() <= 1e-11
    bad = psi.clone()
    bad[1, 3] = float("nan")
    o = hc.nonlocal_add(bad, torch.zeros_like(bad)).cpu().numpy()[:, :npw]
    assert np.isnan(o[1]).any() and not np.isnan(np.delete(o, 1, 0)).any()
    # graph capture of the full apply
    ref = hc.apply(psi).clone()
    buf, out = psi.clone(), torch.zeros_like(psi)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        hc.apply(buf, out, side)
    torch.cuda.current_stream().wait_stream(side)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        hc.apply(buf, out, torch.cuda.current_stream())
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out[:, :npw].view(torch.float64), ref[:, :npw].view(torch.float64))
    del g
    hc.destroy()
