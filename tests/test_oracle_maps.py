"""Pins for the oracle's G-sphere maps (a0). PAPER.md:L176 (vi) names the operation; SURVEY.md 8(c) items 2-3
fix the readings (inclusive cutoff, ascending-FFT-index canonical order)."""
import math
import os

import numpy as np
import pytest

from oracle import hpsi_oracle as orc
from paper_2104_10502_b200 import inputs
from tests._problem import sphere

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "npw_counts.txt")) as f:
    for line in f:
        if line.strip() and not line.startswith("#"):
            c, npw, s, p = (int(x) for x in line.split())
            GOLD[c] = (npw, s, p)


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_npw_sticks_planes_match_survey_counts(cfg):
    wl = inputs.CONFIGS[cfg]
    sp = sphere(cfg)
    npw, s_gold, p_gold = GOLD[cfg]
    assert sp["miller"].shape[0] == npw
    n1, n2, n3 = wl.nr
    idx = sp["fft_index"].astype(np.int64)
    sticks = np.unique(idx // n3)
    planes = np.unique(idx // (n2 * n3))
    assert sticks.size == s_gold
    assert planes.size == p_gold


@pytest.mark.parametrize("cfg", [0, 1, 3, "T1_general_k", "T5_odd_bands", "T3_aliased"])
def test_map_structure(cfg):
    wl = inputs.get_workload(cfg)
    sp = sphere(cfg)
    idx = sp["fft_index"].astype(np.int64)
    assert np.all(np.diff(idx) > 0), "fft_index must be strictly increasing (canonical order)"
    assert np.array_equal(orc.fft_index_of(sp["miller"], wl.nr), idx), "miller <-> fft_index round trip"
    # g2kin = |k+G|^2 recomputed through an independent route (numpy matmul with inv-based reciprocal lattice)
    a = np.array(wl.at).reshape(3, 3)
    b = 2 * np.pi * np.linalg.inv(a).T
    q = sp["miller"].astype(np.float64) @ b + np.array(wl.xk)[None, :]
    np.testing.assert_allclose(sp["g2kin"], (q * q).sum(1), rtol=1e-12, atol=1e-12)
    assert sp["g2kin"].max() <= wl.ecutwfc
    if not any(wl.xk):
        # closed under G -> -G at k = 0
        s = {tuple(m) for m in sp["miller"].tolist()}
        assert all((-m[0], -m[1], -m[2]) in s for m in s)


@pytest.mark.parametrize("cfg", ["T1_general_k", "T5_odd_bands", "T2_radix5"])
def test_sphere_brute_force_python_loops(cfg):
    """Independent enumeration: pure-Python loops over a Miller cube (not the FFT box), math.* arithmetic."""
    wl = inputs.get_workload(cfg)
    a = np.array(wl.at).reshape(3, 3)
    b = (2 * np.pi * np.linalg.inv(a).T).tolist()
    k = list(wl.xk)
    found = {}
    r = 12
    for n1 in range(-r, r + 1):
        for n2 in range(-r, r + 1):
            for n3 in range(-r, r + 1):
                q = [k[c] + n1 * b[0][c] + n2 * b[1][c] + n3 * b[2][c] for c in range(3)]
                q2 = math.fsum(x * x for x in q)
                if q2 <= wl.ecutwfc:
                    found[(n1, n2, n3)] = q2
    sp = sphere(cfg)
    got = {tuple(m): g for m, g in zip(sp["miller"].tolist(), sp["g2kin"].tolist())}
    assert set(found) == set(got)
    for m, q2 in found.items():
        assert abs(got[m] - q2) <= 1e-12 * max(1.0, q2)
    # canonical order = ascending wrapped linear index
    n1, n2, n3 = wl.nr
    order = sorted(found, key=lambda m: ((m[0] % n1) * n2 + (m[1] % n2)) * n3 + (m[2] % n3))
    assert [tuple(m) for m in sp["miller"].tolist()] == order


def test_cutoff_is_inclusive_and_margin():
    # |G|^2 = 25 exactly reachable? For L=10 cubic: G^2 = (2pi/10)^2 * n^2 -- irrational multiples, so test the
    # inclusive rule on a cell built to hit the cutoff exactly: L = 2 pi, ecut = 9 -> (3,0,0) has q2 == 9.
    L = orc.TWO_PI
    sp = orc.gsphere((L, 0, 0, 0, L, 0, 0, 0, L), (0, 0, 0), 9.0, (8, 8, 8))
    s = {tuple(m) for m in sp["miller"].tolist()}
    assert (3, 0, 0) in s and (0, -3, 0) in s and (2, 2, 1) in s and (2, 2, 2) not in s
    # the five configs keep every lattice point well away from the cutoff (SURVEY table: >= 5.7e-5 relative)
    for cfg in (0, 1, 3):
        wl = inputs.CONFIGS[cfg]
        g2 = sphere(cfg)["g2kin"]
        assert (wl.ecutwfc - g2.max()) / wl.ecutwfc > 1e-5


def test_signed_index_convention():
    assert orc.signed_index(np.arange(8), 8).tolist() == [0, 1, 2, 3, -4, -3, -2, -1]
    assert orc.signed_index(np.arange(5), 5).tolist() == [0, 1, 2, -2, -1]
