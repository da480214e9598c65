"""Pins for the oracle functions of the rows SURVEY.md 8(f) marks "next": overlap operator S (NEXT-2), reduced
matrices of the Davidson step (NEXT-3), charge density (NEXT-4).  PAPER.md:L226 names them ("application of the
overlap operator", "charge density generation"), L162/L168 the iterative diagonaliser that needs the reduced
matrices; it prints no formula, so the pins are closed forms, brute force and invariants (DESIGN.md section 2,
items 18-20)."""
import cmath
import math

import numpy as np
import pytest

from oracle import hpsi_oracle as orc
from tests._problem import problem, random_psi

TINY = ["T1_general_k", "T2_radix5", "T5_odd_bands"]


# ---- S ------------------------------------------------------------------------------------------------------
def test_spsi_identity_when_q_vanishes():
    pr = problem("T1_general_k")
    q = np.zeros_like(pr["dblocks"])
    np.testing.assert_array_equal(orc.spsi_of(pr["beta"], q, pr["psi"]), pr["psi"])


def test_spsi_rank_one_closed_form():
    """One projector, q = [[q0]]: S psi = psi + q0 beta <beta|psi>; with psi = beta: (1 + q0 |beta|^2) beta."""
    rng = np.random.default_rng(5)
    npw = 37
    beta = (rng.standard_normal((1, npw)) + 1j * rng.standard_normal((1, npw)))
    psi = (rng.standard_normal((2, npw)) + 1j * rng.standard_normal((2, npw)))
    q0 = 0.37
    q = np.array([[[q0]]])
    got = orc.spsi_of(beta, q, psi)
    for b in range(2):
        ov = sum(beta[0, g].conjugate() * psi[b, g] for g in range(npw))  # python loop, not the oracle's matmul
        np.testing.assert_allclose(got[b], psi[b] + q0 * ov * beta[0], atol=1e-13)
    nb2 = float((abs(beta[0]) ** 2).sum())
    np.testing.assert_allclose(orc.spsi_of(beta, q, beta)[0], (1 + q0 * nb2) * beta[0], atol=1e-12)


@pytest.mark.parametrize("cfg", TINY)
def test_spsi_is_hermitian_and_brute_force(cfg):
    pr = problem(cfg)
    beta, db = pr["beta"], pr["dblocks"]
    rng = np.random.default_rng(11)
    q = rng.uniform(-1, 1, db.shape)
    q = 0.5 * (q + q.transpose(0, 2, 1))
    npw = beta.shape[1]
    phi, psi = random_psi(npw, 2, 7), random_psi(npw, 2, 8)
    sp, sf = orc.spsi_of(beta, q, psi), orc.spsi_of(beta, q, phi)
    for i in range(2):
        for j in range(2):
            assert abs(np.vdot(phi[i], sp[j]) - np.vdot(sf[i], psi[j])) < 1e-12
    # brute force on a few rows: triple loop over atoms, i, j
    nat, nh, _ = q.shape
    for g in (0, npw // 2, npw - 1):
        acc = psi[0, g]
        for a in range(nat):
            for i in range(nh):
                for j in range(nh):
                    acc += beta[a * nh + i, g] * q[a, i, j] * np.vdot(beta[a * nh + j], psi[0])
        assert abs(acc - sp[0, g]) < 1e-12 * max(1.0, abs(acc))


# ---- reduced matrices ------------------------------------------------------------------------------------------
def test_overlap_against_python_loops_and_symmetries():
    rng = np.random.default_rng(2)
    a = rng.standard_normal((3, 29)) + 1j * rng.standard_normal((3, 29))
    b = rng.standard_normal((4, 29)) + 1j * rng.standard_normal((4, 29))
    m = orc.overlap_of(a, b)
    assert m.shape == (3, 4)
    for i in range(3):
        for j in range(4):
            ref = sum(a[i, g].conjugate() * b[j, g] for g in range(29))
            assert abs(m[i, j] - ref) < 1e-13
    np.testing.assert_allclose(orc.overlap_of(b, a), m.conj().T, atol=1e-13)  # <b|a> = conj(<a|b>)
    qmat, _ = np.linalg.qr((rng.standard_normal((29, 5)) + 1j * rng.standard_normal((29, 5))))
    np.testing.assert_allclose(orc.overlap_of(qmat.T, qmat.T), np.eye(5), atol=1e-13)  # orthonormal set -> identity


@pytest.mark.parametrize("cfg", TINY)
def test_projected_hamiltonian_is_hermitian(cfg):
    pr = problem(cfg)
    psi = pr["psi"]
    hp = orc.hpsi_dual(pr["fft_index"], pr["g2kin"], pr["nr"], pr["vr"], psi, pr["beta"], pr["dblocks"])
    hm = orc.overlap_of(psi, hp)
    np.testing.assert_allclose(hm, hm.conj().T, atol=1e-11 * np.abs(hm).max())


# ---- density ---------------------------------------------------------------------------------------------------
def _tiny_sphere():
    at = np.diag([7.0, 8.0, 9.0])
    nr = (8, 9, 10)
    sp = orc.gsphere(at, np.zeros(3), 6.0, nr)
    return at, nr, sp


def test_density_single_plane_wave_is_constant():
    at, nr, sp = _tiny_sphere()
    npw = sp["miller"].shape[0]
    psi = np.zeros((1, npw), complex)
    psi[0, npw // 3] = 0.6 - 0.8j
    rho = orc.density_of(sp["fft_index"], nr, psi, np.array([2.0]), 0.25)
    np.testing.assert_allclose(rho, 2.0 * 0.25 * 1.0, atol=1e-13)


def test_density_two_plane_waves_closed_form():
    """c1 e^{iG1 r} + c2 e^{iG2 r}: |psi|^2 = |c1|^2 + |c2|^2 + 2 Re(c1 conj(c2) e^{i(G1-G2) r}), r = sum (i_j/N_j) a_j."""
    at, nr, sp = _tiny_sphere()
    npw = sp["miller"].shape[0]
    g1, g2 = 1, npw - 2
    c1, c2 = 0.3 + 0.4j, -0.5 + 0.2j
    psi = np.zeros((1, npw), complex)
    psi[0, g1], psi[0, g2] = c1, c2
    rho = orc.density_of(sp["fft_index"], nr, psi, np.array([1.5]), 1.0)
    dm = sp["miller"][g1].astype(int) - sp["miller"][g2].astype(int)
    for i in (0, 3, 7):
        for j in (0, 4, 8):
            for k in (0, 5, 9):
                ph = 2 * math.pi * (dm[0] * i / nr[0] + dm[1] * j / nr[1] + dm[2] * k / nr[2])
                ref = 1.5 * (abs(c1) ** 2 + abs(c2) ** 2 + 2 * (c1 * c2.conjugate() * cmath.exp(1j * ph)).real)
                assert abs(rho[i, j, k] - ref) < 1e-13


@pytest.mark.parametrize("cfg", TINY)
def test_density_integrates_to_the_occupations(cfg):
    """Parseval: (1/N) sum_r rho(r) = scale * sum_b occ_b ||c_b||^2; rho >= 0; linear in occ."""
    pr = problem(cfg)
    psi = pr["psi"]
    nb = psi.shape[0]
    occ = np.linspace(2.0, 0.5, nb)
    rho = orc.density_of(pr["fft_index"], pr["nr"], psi, occ, 0.5)
    assert rho.min() >= 0.0
    norms = (np.abs(psi) ** 2).sum(1)
    assert abs(rho.mean() - 0.5 * (occ * norms).sum()) < 1e-12 * rho.mean()
    r1 = orc.density_of(pr["fft_index"], pr["nr"], psi[:1], occ[:1], 0.5)
    r2 = orc.density_of(pr["fft_index"], pr["nr"], psi[1:], occ[1:], 0.5)
    np.testing.assert_allclose(r1 + r2, rho, atol=1e-13 * rho.max())


def test_psi_r_matches_explicit_dft():
    """psi_r uses numpy.fft as the DFT step; pin it to the oracle's explicit DFT matrices (no FFT library)."""
    at, nr, sp = _tiny_sphere()
    npw = sp["miller"].shape[0]
    psi = random_psi(npw, 1, 3)[0]
    box = np.zeros(nr, complex)
    box.reshape(-1)[sp["fft_index"]] = psi
    np.testing.assert_allclose(orc.psi_r(sp["fft_index"], nr, psi), orc.dft3_explicit(box, +1), atol=1e-12)
