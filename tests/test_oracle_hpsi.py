"""Pins for the oracle's H|psi> (oracle/hpsi_oracle.py) against what the mathematics fixes.

PAPER.md prints no formula or worked example for H|psi> (it names the operation, and its three
terms); BASELINE.json's north_star gives H_GG' and the invariants used here: single plane wave
in constant V0, FFT round trip, Hermiticity, brute-force matrix-vector products. SURVEY.md 8(c) adds the closed
forms (cosine shift, rank-1 projector), translation covariance and time reversal. Each test is chosen so that
a plausible mistake (dropped term, wrong sign / index / transposed operand / missing 1/N) fails it.
"""
import cmath
import math

import numpy as np
import pytest

from oracle import hpsi_oracle as orc
from paper_2104_10502_b200 import inputs
from tests._problem import problem, random_psi, sphere

TINY = ["T1_general_k", "T2_radix5", "T2b_radix5_20", "T3_aliased", "T4_noproj", "T5_odd_bands"]


# ---------------------------------------------------------------------------------------------------------
# DFT building blocks
# ---------------------------------------------------------------------------------------------------------


@pytest.mark.parametrize("n", [1, 2, 3, 5, 8, 9, 10, 12, 15])
def test_dft_matrix_against_python_loops(n):
    for sign in (+1, -1):
        w = orc.dft_matrix(n, sign)
        for m in range(n):
            for i in range(n):
                ref = cmath.exp(sign * 2j * math.pi * ((m * i) % n) / n)
                assert abs(w[m, i] - ref) < 1e-15


@pytest.mark.parametrize("shape", [(4, 6, 5), (8, 9, 10), (15, 12, 18)])
def test_dft3_explicit_special_cases(shape):
    rng = np.random.default_rng(3)
    x = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    n = x.size
    fwd = orc.dft3_explicit(x, -1)
    inv = orc.dft3_explicit(x, +1)
    # library special case (third opinion): numpy.fft.fftn is exp(-), ifftn is exp(+)/N
    np.testing.assert_allclose(fwd, np.fft.fftn(x), rtol=0, atol=1e-12 * np.abs(x).sum())
    np.testing.assert_allclose(inv, np.fft.ifftn(x) * n, rtol=0, atol=1e-12 * np.abs(x).sum())
    # round trip and Parseval
    np.testing.assert_allclose(orc.dft3_explicit(inv, -1) / n, x, atol=1e-12)
    assert abs((np.abs(fwd) ** 2).sum() / n - (np.abs(x) ** 2).sum()) < 1e-10 * (np.abs(x) ** 2).sum()
    # delta at a known point -> plane wave with the right sign and axis assignment
    d = np.zeros(shape, complex)
    p = (1, 2, 3)
    d[p] = 1.0
    i1, i2, i3 = np.meshgrid(*[np.arange(s) for s in shape], indexing="ij")
    ph = 2 * np.pi * (p[0] * i1 / shape[0] + p[1] * i2 / shape[1] + p[2] * i3 / shape[2])
    np.testing.assert_allclose(orc.dft3_explicit(d, +1), np.exp(1j * ph), atol=1e-12)


def test_vloc_coeffs_of_cosine():
    nr = (6, 8, 10)
    i1, i2, i3 = np.meshgrid(*[np.arange(s) for s in nr], indexing="ij")
    m0 = (1, -2, 3)
    ph = 2 * np.pi * (m0[0] * i1 / nr[0] + m0[1] * i2 / nr[1] + m0[2] * i3 / nr[2])
    vr = 0.7 + 2 * 0.3 * np.cos(ph) - 2 * 0.2 * np.sin(ph)  # = 0.7 + (0.3+0.2i) e^{i ph} + c.c.
    vt = orc.vloc_coeffs(vr)
    ref = np.zeros(nr, complex)
    ref[0, 0, 0] = 0.7
    ref[m0[0] % 6, m0[1] % 8, m0[2] % 10] = 0.3 + 0.2j
    ref[-m0[0] % 6, -m0[1] % 8, -m0[2] % 10] = 0.3 - 0.2j
    np.testing.assert_allclose(vt, ref, atol=1e-14)


# ---------------------------------------------------------------------------------------------------------
# closed forms
# ---------------------------------------------------------------------------------------------------------


def _all_levels(p, psi, vr, beta, db):
    """H psi by Level A (dense), A' (all rows) and B (dual space)."""
    nr = p["nr"]
    h = orc.dense_h(p["miller"], p["g2kin"], nr, vr, beta, db)
    a = orc.hpsi_dense(h, psi)
    rows = np.arange(p["miller"].shape[0])
    ap = orc.hpsi_rows(rows, p["miller"], p["g2kin"], nr, orc.vloc_coeffs(vr), psi, beta, db)
    b = orc.hpsi_dual(p["fft_index"], p["g2kin"], nr, vr, psi, beta, db)
    return a, ap, b


@pytest.mark.parametrize("cfg", ["T1_general_k", "T5_odd_bands"])
def test_single_plane_wave_in_constant_potential(cfg):
    """north_star invariant: psi = delta_{G,G0}, V = V0, no projectors -> hpsi = (|k+G0|^2 + V0) delta."""
    p = problem(cfg)
    npw = p["miller"].shape[0]
    v0 = -0.37
    vr = np.full(p["nr"], v0)
    for g0 in (0, npw // 3, npw - 1):
        psi = np.zeros((1, npw), complex)
        psi[0, g0] = 1.0 - 2.0j
        for out in _all_levels(p, psi, vr, None, None):
            ref = np.zeros_like(psi)
            ref[0, g0] = (p["g2kin"][g0] + v0) * psi[0, g0]
            np.testing.assert_allclose(out, ref, atol=1e-13)
    # and for a general psi: (|k+G|^2 + V0) c(G)
    psi = random_psi(npw, 3, 11)
    for out in _all_levels(p, psi, vr, None, None):
        np.testing.assert_allclose(out, (p["g2kin"] + v0)[None] * psi, atol=1e-13)


@pytest.mark.parametrize("cfg", ["T1_general_k", "T2_radix5"])
def test_cosine_potential_is_a_shift(cfg):
    """V(r) = V1 e^{iG0.r} + conj  =>  (V psi)(G) = V1 psi(G-G0) + conj(V1) psi(G+G0), out-of-sphere terms dropped
    (grids here are unaliased: N_j >= 2(nmax-nmin)+1 + |G0| margin is checked)."""
    p = problem(cfg)
    nr = p["nr"]
    mil = p["miller"]
    npw = mil.shape[0]
    m0 = np.array([1, 0, -1])
    span = mil.max(0) - mil.min(0)
    assert all(span[j] + abs(m0[j]) < nr[j] for j in range(3))
    v1 = 0.3 - 0.45j
    i1, i2, i3 = np.meshgrid(*[np.arange(s) for s in nr], indexing="ij")
    ph = 2 * np.pi * (m0[0] * i1 / nr[0] + m0[1] * i2 / nr[1] + m0[2] * i3 / nr[2])
    vr = 2 * (v1 * np.exp(1j * ph)).real
    psi = random_psi(npw, 2, 5)
    lut = {tuple(m): i for i, m in enumerate(mil.tolist())}
    ref = p["g2kin"][None] * psi
    for ig, m in enumerate(mil.tolist()):
        lo = lut.get((m[0] - m0[0], m[1] - m0[1], m[2] - m0[2]))
        hi = lut.get((m[0] + m0[0], m[1] + m0[1], m[2] + m0[2]))
        if lo is not None:
            ref[:, ig] += v1 * psi[:, lo]
        if hi is not None:
            ref[:, ig] += np.conj(v1) * psi[:, hi]
    for out in _all_levels(p, psi, vr, None, None):
        np.testing.assert_allclose(out, ref, atol=1e-13)


def test_rank_one_projector_closed_form():
    """One projector b(G), D = d: hpsi_nl = d * b * (b^H psi), with pure-Python sums as the brute force."""
    p = problem("T2_radix5")
    npw = p["miller"].shape[0]
    b = random_psi(npw, 1, 21)  # [1,npw] arbitrary complex "projector"
    d = np.array([[[0.8]]])
    psi = random_psi(npw, 2, 22)
    vr = np.zeros(p["nr"])
    ref = p["g2kin"][None] * psi
    for ib in range(2):
        s = 0j
        for g in range(npw):
            s += b[0, g].conjugate() * psi[ib, g]
        for g in range(npw):
            ref[ib, g] += 0.8 * b[0, g] * s
    for out in _all_levels(p, psi, vr, b, d):
        np.testing.assert_allclose(out, ref, atol=1e-13)


def test_nonlocal_brute_force_loops():
    """a6-a8 against explicit Python loops over (atom, i, j, G') with non-symmetric-looking index roles."""
    p = problem("T5_odd_bands")
    beta, db = p["beta"], p["dblocks"]
    psi = p["psi"][:2]
    nat, nh, _ = db.shape
    npw = psi.shape[1]
    becp = np.zeros((nat * nh, 2), complex)
    for q in range(nat * nh):
        for ib in range(2):
            becp[q, ib] = sum(beta[q, g].conjugate() * psi[ib, g] for g in range(npw))
    np.testing.assert_allclose(orc.becp_of(beta, psi), becp, atol=1e-14)
    ref = np.zeros_like(psi)
    for a in range(nat):
        for i in range(nh):
            for j in range(nh):
                for ib in range(2):
                    ref[ib] += beta[a * nh + i] * db[a, i, j] * becp[a * nh + j, ib]
    np.testing.assert_allclose(orc.vnl_psi(beta, db, psi), ref, atol=1e-14)


# ---------------------------------------------------------------------------------------------------------
# whole-H invariants
# ---------------------------------------------------------------------------------------------------------


@pytest.mark.parametrize("cfg", TINY)
def test_levels_agree_and_dense_h_is_hermitian(cfg):
    p = problem(cfg)
    a, ap, b = _all_levels(p, p["psi"], p["vr"], p["beta"], p["dblocks"])
    assert orc.rel_l2(ap, a).max() < 1e-13
    assert orc.rel_l2(b, a).max() < 1e-13
    h = orc.dense_h(p["miller"], p["g2kin"], p["nr"], p["vr"], p["beta"], p["dblocks"])
    assert np.abs(h - h.conj().T).max() < 1e-14 * np.abs(h).max()


def test_config0_dense_matches_dual_space():
    p = problem(0)
    h = orc.dense_h(p["miller"], p["g2kin"], p["nr"], p["vr"], p["beta"], p["dblocks"])
    assert np.abs(h - h.conj().T).max() < 1e-14 * np.abs(h).max()
    a = orc.hpsi_dense(h, p["psi"])
    b = orc.hpsi_dual(p["fft_index"], p["g2kin"], p["nr"], p["vr"], p["psi"], p["beta"], p["dblocks"])
    assert orc.rel_l2(b, a).max() < 1e-13


@pytest.mark.parametrize("cfg", ["T1_general_k", "T3_aliased", 0])
def test_hermiticity_of_dual_space_application(cfg):
    p = problem(cfg)
    npw = p["miller"].shape[0]
    phi, psi = random_psi(npw, 2, 31), random_psi(npw, 2, 32)
    f = lambda x: orc.hpsi_dual(p["fft_index"], p["g2kin"], p["nr"], p["vr"], x, p["beta"], p["dblocks"])
    hpsi, hphi = f(psi), f(phi)
    lhs = (phi.conj() * hpsi).sum(1)
    rhs = np.conj((psi.conj() * hphi).sum(1))
    assert np.abs(lhs - rhs).max() < 1e-13 * np.abs(lhs).max()


@pytest.mark.parametrize("cfg", ["T1_general_k", "T5_odd_bands"])
def test_translation_covariance(cfg):
    """Shift atoms and V(r) by a grid vector t, psi(G) -> psi(G) e^{-iG.t}  =>  hpsi(G) -> hpsi(G) e^{-iG.t}.
    Catches structure-factor sign, index wrap and axis-order mistakes."""
    p = problem(cfg)
    wl = p["wl"]
    nr = p["nr"]
    s = np.array([1, 3, 2])
    mil = p["miller"].astype(np.float64)
    phase = np.exp(-2j * np.pi * (mil @ (s / np.array(nr))))
    vr2 = np.roll(p["vr"], shift=tuple(s), axis=(0, 1, 2))  # V'(r) = V(r - t)
    atoms2 = p["atoms"] + (s / np.array(nr))[None, :]
    beta2 = inputs.gen_beta(wl, p["miller"], atoms2).numpy()
    h1 = orc.hpsi_dual(p["fft_index"], p["g2kin"], nr, p["vr"], p["psi"], p["beta"], p["dblocks"])
    h2 = orc.hpsi_dual(p["fft_index"], p["g2kin"], nr, vr2, p["psi"] * phase[None], beta2, p["dblocks"])
    assert orc.rel_l2(h2, h1 * phase[None]).max() < 1e-12


def test_time_reversal_at_gamma():
    """k = 0, real V, real D, real Y_lm: psi(-G) = conj psi(G)  =>  hpsi(-G) = conj hpsi(G)."""
    p = problem("T2b_radix5_20")
    mil = p["miller"]
    lut = {tuple(m): i for i, m in enumerate(mil.tolist())}
    minus = np.array([lut[(-m[0], -m[1], -m[2])] for m in mil.tolist()])
    x = random_psi(mil.shape[0], 2, 41)
    psi = x + np.conj(x[:, minus])
    h = orc.hpsi_dual(p["fft_index"], p["g2kin"], p["nr"], p["vr"], psi, p["beta"], p["dblocks"])
    assert np.abs(h[:, minus] - np.conj(h)).max() < 1e-13 * np.abs(h).max()


def test_linearity():
    p = problem("T1_general_k")
    npw = p["miller"].shape[0]
    x, y = random_psi(npw, 1, 51), random_psi(npw, 1, 52)
    f = lambda v: orc.hpsi_dual(p["fft_index"], p["g2kin"], p["nr"], p["vr"], v, p["beta"], p["dblocks"])
    al = 0.3 - 1.1j
    np.testing.assert_allclose(f(x + al * y), f(x) + al * f(y), atol=1e-13)


def test_config1_sampled_rows_match_dual_space():
    """Level A' (the definition, no FFT of psi) vs Level B at a config too large for dense H."""
    p = problem(1, nbands=3)
    wl = p["wl"]
    npw = p["miller"].shape[0]
    rows = inputs.aux_choice(wl.seed, 1, npw, 24)
    vt = orc.vloc_coeffs(p["vr"])
    ap = orc.hpsi_rows(rows, p["miller"], p["g2kin"], p["nr"], vt, p["psi"], p["beta"], p["dblocks"])
    b = orc.hpsi_dual(p["fft_index"], p["g2kin"], p["nr"], p["vr"], p["psi"], p["beta"], p["dblocks"])
    assert np.abs(ap - b[:, rows]).max() < 1e-13 * np.abs(b).max()


def test_sampled_rows_with_becp_accumulated_over_atom_chunks():
    """The `becp=` branch of hpsi_rows (what the full-size GPU tests use: beta streamed in atom chunks, only its columns at
    the sampled rows kept) against the dense definition on a tiny case and against the in-memory branch on config 1."""
    p = problem("T1_general_k")
    wl, npw = p["wl"], p["miller"].shape[0]
    rows = np.array([0, 3, npw // 2, npw - 1])
    vt = orc.vloc_coeffs(p["vr"])
    nh = wl.nh
    becp = np.zeros((wl.nproj, p["psi"].shape[0]), complex)
    for a in range(wl.natoms):  # one atom per chunk
        becp[a * nh:(a + 1) * nh] = orc.becp_of(p["beta"][a * nh:(a + 1) * nh], p["psi"])
    got = orc.hpsi_rows(rows, p["miller"], p["g2kin"], p["nr"], vt, p["psi"], p["beta"][:, rows], p["dblocks"], becp=becp)
    hd = orc.dense_h(p["miller"], p["g2kin"], p["nr"], p["vr"], p["beta"], p["dblocks"])
    ref = orc.hpsi_dense(hd, p["psi"])[:, rows]
    assert np.abs(got - ref).max() < 1e-13 * np.abs(ref).max()
    # full beta passed together with becp: the columns are picked inside
    got2 = orc.hpsi_rows(rows, p["miller"], p["g2kin"], p["nr"], vt, p["psi"], p["beta"], p["dblocks"], becp=becp)
    assert np.array_equal(got, got2)
    # a wrong becp must show (the branch really uses what it is given)
    bad = orc.hpsi_rows(rows, p["miller"], p["g2kin"], p["nr"], vt, p["psi"], p["beta"][:, rows], p["dblocks"], becp=2 * becp)
    assert np.abs(bad - ref).max() > 1e-6 * np.abs(ref).max()


# ---------------------------------------------------------------------------------------------------------
# the error metric every parity assertion goes through
# ---------------------------------------------------------------------------------------------------------


def test_rel_l2_is_per_band_relative_to_the_reference():
    """rel_l2(x, ref)[b] = ||x_b - ref_b||_2 / ||ref_b||_2 over the entries of band b, hand-built so that a wrong axis,
    a wrong normaliser, a dropped square root or an average over bands each gives a different number."""
    ref = np.array([[3.0, 4.0j, 0.0], [3.0, 4.0j, 0.0], [0.0, 0.0, 10.0], [6.0, 8.0j, 0.0]])  # norms 5, 5, 10, 10
    x = ref.copy()
    x[1, 1] += 5e-3            # off by a known vector of norm 5e-3 -> 1e-3 exactly
    x[2] += np.array([3e-6j, 0.0, 4e-6])  # norm 5e-6 against 10 -> 5e-7
    x[3, 2] += 1e-2j           # purely imaginary error in an entry where ref is 0 -> 1e-3 of norm 10
    err = orc.rel_l2(x, ref)
    assert err.shape == (4,) and err.dtype == np.float64
    assert err[0] == 0.0
    np.testing.assert_allclose(err[1:], [1e-3, 5e-7, 1e-3], rtol=1e-9)  # x = ref + e is rounded: (10 + 4e-6) - 10 is exact to 1e-10
    # one bad band among many good ones is not averaged away, and the good ones stay exact
    big = np.tile(ref[:1], (1000, 1))
    y = big.copy()
    y[417, 0] += 0.05
    e = orc.rel_l2(y, big)
    assert e[417] == pytest.approx(1e-2, rel=1e-12) and np.count_nonzero(e) == 1
    # relative to ||ref||, not to ||x||: scaling x's error direction changes the numerator only
    r1 = np.array([[1.0, 0.0]])
    assert orc.rel_l2(np.array([[3.0, 0.0]]), r1)[0] == pytest.approx(2.0, rel=1e-15)   # ||x-ref|| / ||ref|| = 2, / ||x|| would be 2/3
    # invariant under a common scale, linear in the error
    np.testing.assert_allclose(orc.rel_l2(8.0 * x, 8.0 * ref), err, rtol=1e-13)  # power of two: exact scaling
    np.testing.assert_allclose(orc.rel_l2(ref + 3.0 * (x - ref), ref), 3.0 * err, rtol=1e-9)
    # long-double accumulation: tiny errors on a large reference do not vanish in the subtraction of squares
    ref2 = np.full((1, 4096), 1.0 + 0j)
    x2 = ref2 * (1.0 + 2.0 ** -50)
    assert orc.rel_l2(x2, ref2)[0] == pytest.approx(2.0 ** -50, rel=1e-6)


# ---------------------------------------------------------------------------------------------------------
# generators(inputs.py holds no method arithmetic; these check the recipe of SURVEY 8(c) items 6-10)
# ---------------------------------------------------------------------------------------------------------


def test_generators_follow_the_recipe():
    p = problem(0)
    wl = p["wl"]
    assert np.allclose((np.abs(p["psi"]) ** 2).sum(1), 1.0, atol=1e-13)
    # V(r) real with Hermitian V(G) supported on |G|^2 <= 100
    vt = np.fft.fftn(p["vr"]) / p["vr"].size
    assert np.abs(vt - np.conj(np.roll(vt[::-1, ::-1, ::-1], 1, (0, 1, 2)))).max() < 1e-14
    bvec = 2 * np.pi / 10.0
    n = orc.signed_index(np.arange(36), 36) * bvec
    g2 = n[:, None, None] ** 2 + n[None, :, None] ** 2 + n[None, None, :] ** 2
    assert np.abs(vt[g2 > 100.0 + 1e-9]).max() < 1e-14
    assert np.abs(vt[g2 <= 100.0]).max() > 1e-3
    # atoms: minimum-image separation >= 3 bohr
    a = np.array(wl.at).reshape(3, 3)
    d = p["atoms"][0] - p["atoms"][1]
    d -= np.round(d)
    assert np.linalg.norm(d @ a) >= 3.0
    # D symmetric, diagonal per l at config 0; 2x2-per-l coupling at config 1
    db = p["dblocks"]
    assert db.shape == (2, 4, 4) and np.allclose(db, np.transpose(db, (0, 2, 1)))
    assert np.count_nonzero(db[0] - np.diag(np.diag(db[0]))) == 0
    assert db[0, 1, 1] == db[0, 2, 2] == db[0, 3, 3] != db[0, 0, 0]
    d1 = inputs.gen_dblocks(inputs.CONFIGS[1])
    assert d1.shape == (64, 8, 8) and np.allclose(d1, np.transpose(d1, (0, 2, 1)))
    assert d1[0, 0, 1] != 0 and d1[0, 2, 5] != 0 and d1[0, 2, 3] == 0 and d1[0, 0, 2] == 0
    assert np.abs(d1).max() <= 1.0


def test_beta_formula_spot_check():
    """beta_{a,(n,l,m)}(G) = q^l e^{-q^2 rc^2/2} Y_lm e^{-i q.tau}/sqrt(Omega) recomputed with math.* scalars."""
    p = problem("T1_general_k")
    wl = p["wl"]
    a = np.array(wl.at).reshape(3, 3)
    b = 2 * np.pi * np.linalg.inv(a).T
    om = abs(np.linalg.det(a))
    for ig in (0, 17, p["miller"].shape[0] - 1):
        q = p["miller"][ig].astype(float) @ b + np.array(wl.xk)
        q2 = float(q @ q)
        for ia in (0, 1):
            tau = p["atoms"][ia] @ a
            sf = cmath.exp(-1j * float(q @ tau))
            exp8 = math.exp(-q2 * 0.8**2 / 2) / math.sqrt(om)
            exp12 = math.exp(-q2 * 1.2**2 / 2) / math.sqrt(om)
            y0, y1 = 1 / math.sqrt(4 * math.pi), math.sqrt(3 / (4 * math.pi))
            ref = [exp8 * y0, exp12 * y0] + [exp8 * y1 * q[c] for c in range(3)] + [exp12 * y1 * q[c] for c in range(3)]
            got = p["beta"][ia * 8:(ia + 1) * 8, ig]
            np.testing.assert_allclose(got, np.array(ref) * sf, rtol=1e-12, atol=1e-15)
