"""GPU-test helpers: build a handle for a workload on cuda:0 and produce the ORACLE reference for selected bands
from exactly the inputs the GPU used (device arrays copied to the host; beta streamed in atom chunks so that
config 4's 25 GB never has to sit in host memory)."""
from __future__ import annotations

import os

import numpy as np
import torch

from oracle import hpsi_oracle as orc
from paper_2104_10502_b200 import inputs, qe_hpsi


INT8 = 1 << 16  # test-only pseudo flag: force the int8 digit path (QE_HPSI_OZAKI=6) where the library's size rule would not


class force_int8:
    """with force_int8(flags) as f: create handles with flags f; tiny workloads otherwise default to the FP64 tensor path."""

    def __init__(self, flags, digits=6):
        self.on, self.flags, self.digits = bool(flags & INT8), flags & ~INT8, digits

    def __enter__(self):
        if self.on:
            os.environ["QE_HPSI_OZAKI"] = str(self.digits)
        return self.flags

    def __exit__(self, *exc):
        if self.on:
            del os.environ["QE_HPSI_OZAKI"]


def make(key, max_batch=None, flags=0):
    with force_int8(flags) as f:
        h, inp = qe_hpsi.from_workload(key, max_batch=max_batch, flags=f)
    if flags & INT8:
        assert inputs.get_workload(key).nproj == 0 or h.info()["ozaki_slices"] == 6
    return h, inp


def gen_psi_dev(inp, band0, nb):
    wl = inp["wl"]
    return inputs.gen_psi(wl, inp["miller_dev"], band0, nb, ld=inp["ld"], device="cuda")


def oracle_sphere(wl):
    return orc.gsphere(wl.at, wl.xk, wl.ecutwfc, wl.nr)


def oracle_hpsi(inp, sp, psi_host, atom_chunk=32, parts=False):
    """Level B oracle (dual space) for psi_host [nb, npw] using the GPU's own V(r), beta (streamed D2H) and D."""
    wl = inp["wl"]
    npw = sp["miller"].shape[0]
    vr = inp["vr"].cpu().numpy()
    loc = orc.hpsi_dual(sp["fft_index"], sp["g2kin"], tuple(wl.nr), vr, psi_host, None, None)
    vnl = np.zeros_like(psi_host)
    if wl.nproj:
        nh = wl.nh
        for a0 in range(0, wl.natoms, atom_chunk):
            a1 = min(wl.natoms, a0 + atom_chunk)
            bc = inp["beta"][a0 * nh:a1 * nh, :npw].cpu().numpy()
            vnl += orc.vnl_psi(bc, inp["dblocks"][a0:a1], psi_host)
    if parts:
        return loc, vnl
    return loc + vnl


def rel_l2(x, ref):
    return orc.rel_l2(x, ref)
