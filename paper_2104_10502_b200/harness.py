"""Harness shared by tests/, bench.py and __graft_entry__.smoke(): build every input of a BASELINE.json workload on the
GPU with the seeded generators (inputs.py) and the library's own sphere, and create a handle. Not part of the binding
(qe_hpsi.py mirrors the C ABI and nothing else) and holds no method arithmetic."""
from __future__ import annotations

import numpy as np
import torch

from . import inputs, qe_hpsi


def from_workload(wl, max_batch=None, flags=0, device="cuda", beta=None):
    """Returns (Hpsi, dict of inputs). `beta` lets several handles share one generated projector array."""
    wl = inputs.get_workload(wl)
    mil = qe_hpsi.qe_hpsi_gsphere(wl.at, wl.xk, wl.ecutwfc, wl.nr)
    npw = mil.shape[0]
    ld = inputs.pad8(npw)
    vr = inputs.gen_vloc(wl, device="cpu").to(device)  # input generation only (CPU FFT); not the product path
    atoms = inputs.gen_atoms(wl)
    mil_d = torch.as_tensor(mil, device=device)
    if wl.nproj:
        if beta is None:
            beta = torch.zeros((wl.nproj, ld), dtype=torch.complex128, device=device)
            step = 16
            for a0 in range(0, wl.natoms, step):
                na = min(step, wl.natoms - a0)
                inputs.gen_beta(wl, mil_d, atoms, a0, na, ld=ld, device=device, out=beta[a0 * wl.nh:(a0 + na) * wl.nh])
        blk = np.arange(wl.natoms + 1, dtype=np.int32) * wl.nh
        db = inputs.gen_dblocks(wl)
    else:
        beta, blk, db = None, None, None
    mb = wl.batch if max_batch is None else max_batch
    h = qe_hpsi.Hpsi(wl.at, wl.ecutwfc, wl.xk, wl.nr, vr, beta, blk, db, max_batch=mb, flags=flags)
    return h, dict(wl=wl, miller=mil, miller_dev=mil_d, ld=ld, vr=vr, atoms=atoms, beta=beta, dblocks=db, blk=blk)


def int8_flags(digits=6, three_m=None, certify=False):
    """Create flags of the int8 digit path: digits 4..7, three_m in {None (by size), 0 (off), 2 (a6 only), 3 (a6 and a8)}."""
    f = qe_hpsi.QE_HPSI_PROJ_INT8 | qe_hpsi.QE_HPSI_PROJ_DIGITS(digits)
    if three_m is not None:
        f |= {0: qe_hpsi.QE_HPSI_PROJ_3M_OFF, 2: qe_hpsi.QE_HPSI_PROJ_3M_A6, 3: qe_hpsi.QE_HPSI_PROJ_3M_ALL}[three_m]
    if certify:
        f |= qe_hpsi.QE_HPSI_PROJ_CERTIFY
    return f
