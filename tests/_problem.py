"""Test helper: assemble one H|psi> problem (numpy, host) from a workload using the ORACLE's sphere.

Lives in tests/ because it imports oracle/ (allowed only for tests, smoke and the bench's cpu_baseline leg).
"""
from __future__ import annotations

import functools

import numpy as np

from oracle import hpsi_oracle as orc
from paper_2104_10502_b200 import inputs


@functools.lru_cache(maxsize=8)
def sphere(key):
    wl = inputs.get_workload(key)
    return orc.gsphere(wl.at, wl.xk, wl.ecutwfc, wl.nr)


@functools.lru_cache(maxsize=4)
def problem(key, nbands=None, with_beta=True):
    """dict(wl, miller, fft_index, g2kin, vr, atoms, beta, dblocks, psi) as numpy arrays (ld = npw)."""
    wl = inputs.get_workload(key)
    sp = sphere(key)
    nb = wl.nbands if nbands is None else nbands
    vr = inputs.gen_vloc(wl).numpy()
    atoms = inputs.gen_atoms(wl)
    beta = inputs.gen_beta(wl, sp["miller"], atoms).numpy() if with_beta else None
    db = inputs.gen_dblocks(wl)
    psi = inputs.gen_psi(wl, sp["miller"], 0, nb).numpy()
    return dict(wl=wl, miller=sp["miller"], fft_index=sp["fft_index"], g2kin=sp["g2kin"], vr=vr, atoms=atoms,
                beta=beta, dblocks=db, psi=psi, nr=tuple(wl.nr))


def random_psi(npw, nb, seed):
    v = np.stack([inputs.aux_normal_complex(seed, b, npw).numpy() for b in range(nb)])
    return v / np.linalg.norm(v, axis=1, keepdims=True)
