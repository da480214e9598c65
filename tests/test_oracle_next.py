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


# ---- Gamma-only path (NEXT-1) ---------------------------------------------------------------------------------------
def _gamma_problem(cfg, nb=3):
    """k = 0 tiny case: half-sphere psi / beta with real G = 0 components (inputs of a real-wavefunction calculation)."""
    pr = problem(cfg)
    assert np.all(np.asarray(pr["wl"].xk) == 0.0)
    ip, im = orc.gamma_half(pr["miller"])
    psi_h = pr["psi"][:nb, ip].copy()
    psi_h[:, 0] = psi_h[:, 0].real
    beta_h = pr["beta"][:, ip].copy()
    beta_h[:, 0] = beta_h[:, 0].real
    return pr, ip, im, psi_h, beta_h


def test_gamma_half_is_a_partition_of_the_sphere():
    pr = problem("T2_radix5")
    m = pr["miller"].astype(int)
    ip, im = orc.gamma_half(m)
    npw = m.shape[0]
    assert ip[0] == 0 and tuple(m[0]) == (0, 0, 0) and im[0] == 0  # G = 0 first, its own negative
    assert np.all(np.diff(ip) > 0)  # canonical order preserved
    np.testing.assert_array_equal(m[im], -m[ip])
    both = np.concatenate([ip, im[1:]])
    assert both.size == npw and np.array_equal(np.sort(both), np.arange(npw))  # each G exactly once
    assert 2 * ip.size - 1 == npw
    # brute force of the half rule on every sphere point
    for i, (a, b, c) in enumerate(m.tolist()):
        assert (i in set(ip.tolist())) == ((a, b, c) > (0, 0, -1) and (a > 0 or (a == 0 and (b > 0 or (b == 0 and c >= 0)))))


@pytest.mark.parametrize("cfg", ["T2_radix5", "T2b_radix5_20", "T3_aliased", 0])
def test_gamma_expansion_gives_real_psi_and_closed_result(cfg):
    pr, ip, im, psi_h, beta_h = _gamma_problem(cfg)
    npw = pr["miller"].shape[0]
    full = orc.gamma_expand(psi_h, ip, im, npw)
    for b in range(full.shape[0]):
        assert np.abs(orc.psi_r(pr["fft_index"], pr["nr"], full[b]).imag).max() < 1e-12  # psi(r) is real
    beta_f = orc.gamma_expand(beta_h, ip, im, npw)
    hf = orc.hpsi_dual(pr["fft_index"], pr["g2kin"], pr["nr"], pr["vr"], full, beta_f, pr["dblocks"])
    # H of a real field with real V and Hermitian-completed projectors is a real field: h(-G) = conj(h(G))
    np.testing.assert_allclose(hf[:, im], np.conj(hf[:, ip]), atol=1e-12 * np.abs(hf).max())
    # becp is real
    assert np.abs(orc.becp_of(beta_f, full).imag).max() < 1e-13
    got = orc.hpsi_gamma(pr["miller"], pr["fft_index"], pr["g2kin"], pr["nr"], pr["vr"], psi_h, beta_h, pr["dblocks"])
    np.testing.assert_array_equal(got, hf[:, ip])
    # and it is the dense-H (Level A, explicit DFT matrices) result restricted to the half sphere
    hd = orc.dense_h(pr["miller"], pr["g2kin"], pr["nr"], pr["vr"], beta_f, pr["dblocks"])
    np.testing.assert_allclose(got, orc.hpsi_dense(hd, full)[:, ip], atol=1e-11 * np.abs(got).max())


def test_gamma_single_plane_wave_pair_in_constant_potential():
    """psi = c e^{iGr} + conj(c) e^{-iGr} (a real cosine) in V0 without projectors: H psi = (|G|^2 + V0) psi."""
    pr, ip, im, psi_h, _ = _gamma_problem("T2_radix5", nb=1)
    psi_h[:] = 0.0
    g = ip.size // 2
    psi_h[0, g] = 0.3 - 0.7j
    v0 = 0.83
    vr = np.full(pr["nr"], v0)
    got = orc.hpsi_gamma(pr["miller"], pr["fft_index"], pr["g2kin"], pr["nr"], vr, psi_h)
    ref = np.zeros_like(psi_h)
    ref[0, g] = (pr["g2kin"][ip[g]] + v0) * psi_h[0, g]
    np.testing.assert_allclose(got, ref, atol=1e-13)


# ---- Davidson pieces (NEXT-3) -----------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg", ["T1_general_k", "T2_radix5"])
def test_hdiag_and_sdiag_are_the_diagonals_of_the_dense_operators(cfg):
    pr = problem(cfg)
    npw = pr["miller"].shape[0]
    ddiag = np.stack([np.diag(np.diag(d)) for d in pr["dblocks"]])  # D with its off-diagonal entries dropped
    hd = orc.dense_h(pr["miller"], pr["g2kin"], pr["nr"], pr["vr"], pr["beta"], ddiag)
    got = orc.hdiag_of(pr["g2kin"], pr["vr"].mean(), pr["beta"], pr["dblocks"])
    np.testing.assert_allclose(got, np.diag(hd).real, atol=1e-12 * np.abs(got).max())
    rng = np.random.default_rng(4)
    q = rng.uniform(-0.2, 0.2, pr["dblocks"].shape)
    q = 0.5 * (q + q.transpose(0, 2, 1))
    sd = orc.dense_s(pr["beta"], q, npw)
    qdiag = np.stack([np.diag(np.diag(x)) for x in q])
    np.testing.assert_allclose(orc.sdiag_of(npw, pr["beta"], q), np.diag(orc.dense_s(pr["beta"], qdiag, npw)).real, atol=1e-13)
    # dense S applied to psi is spsi_of
    np.testing.assert_allclose((sd @ pr["psi"].T).T, orc.spsi_of(pr["beta"], q, pr["psi"]), atol=1e-12)


def test_precond_and_rotate_against_python_loops():
    rng = np.random.default_rng(9)
    r = rng.standard_normal((2, 11)) + 1j * rng.standard_normal((2, 11))
    hd, sd, e = rng.uniform(0, 30, 11), rng.uniform(0.8, 1.3, 11), np.array([-0.4, 2.5])
    got = orc.precond_of(r, e, hd, sd)
    for b in range(2):
        for g in range(11):
            x = hd[g] - e[b] * sd[g]
            assert abs(got[b, g] - r[b, g] / (0.5 * (1 + x + math.sqrt(1 + (x - 1) ** 2)))) < 1e-14
    # limits: x = 1 -> 3/2; x >> 1 -> x
    assert abs(orc.precond_of(np.ones((1, 1)), [0.0], np.array([1.0]), np.array([1.0]))[0, 0] - 1 / 1.5) < 1e-15
    assert abs(orc.precond_of(np.ones((1, 1)), [0.0], np.array([1e8]), np.array([1.0]))[0, 0] * 1e8 - 1) < 1e-7
    x = rng.standard_normal((3, 7)) + 1j * rng.standard_normal((3, 7))
    c = rng.standard_normal((2, 3)) + 1j * rng.standard_normal((2, 3))
    y = orc.rotate_of(x, c)
    for k in range(2):
        for g in range(7):
            assert abs(y[k, g] - sum(c[k, j] * x[j, g] for j in range(3))) < 1e-14
