"""Seeded synthetic input generators for the H|psi> workloads (BASELINE.json `configs`).

This module serves BOTH the CPU oracle (tests) and the CUDA path (tests, bench). It holds none of the
method's arithmetic: no sphere enumeration, no FFT of psi, no Hamiltonian term. It only turns
(config, seed, integer keys) into the arrays the method consumes: psi(G), V(r), atom positions, beta(G), D.
The G-sphere (Miller indices) is an INPUT here: callers pass the `miller` array they got from the oracle
(tests) or from `qe_hpsi_gsphere` (bench), so the generator never decides sphere membership.

Recipe = SURVEY.md section 8(c) items 6-11 (the paper, PAPER.md, has no formulas; BASELINE.json `configs`
fix the distributions). Random numbers are counter-based: value = f(seed, stream, integer key), so the
generation order never matters and every array can be produced in pieces on any device.

All generators are torch functions with a `device` argument (CPU here, CUDA for the 25 GB beta of config 4).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
import torch

TWO_PI = 6.283185307179586

# ----------------------------------------------------------------------------------------------------------
# workload table
# ----------------------------------------------------------------------------------------------------------


@dataclass(frozen=True)
class Workload:
    """One H|psi> workload. Lengths in bohr, energies in Ry. `at` rows are the lattice vectors."""

    name: str
    at: tuple  # 3x3 row-major
    ecutwfc: float
    xk: tuple  # Cartesian k in bohr^-1
    nr: tuple  # FFT grid N1,N2,N3
    nbands: int
    batch: int  # bands per qe_hpsi_apply call
    natoms: int
    channels: tuple  # per-atom projector channels: (l, rc) in order; each expands to 2l+1 m's
    dmode: str  # "diag" (config 0) | "pair" (configs 1+: symmetric 2x2 per l coupling the two rc channels)
    seed: int
    min_sep: float = 3.0
    cfg_id: int = -1

    @property
    def nh(self) -> int:
        return sum(2 * l + 1 for l, _ in self.channels)

    @property
    def nproj(self) -> int:
        return self.natoms * self.nh

    @property
    def omega(self) -> float:
        a = np.array(self.at, dtype=np.float64).reshape(3, 3)
        return float(abs(np.linalg.det(a)))


def _cubic(L):
    return (L, 0.0, 0.0, 0.0, L, 0.0, 0.0, 0.0, L)


_SP1 = ((0, 1.0), (1, 1.0))  # config 0: s, p with rc = 1 -> 4 projectors
_SP2 = ((0, 0.8), (0, 1.2), (1, 0.8), (1, 1.2))  # configs 1+: 1+1+3+3 = 8 projectors

_BASE_SEED = 2104 * 10**4 + 10502


def _mk(i, name, at, ecut, xk, nr, nb, batch, nat, ch, dmode):
    return Workload(name, at, ecut, xk, nr, nb, batch, nat, ch, dmode, _BASE_SEED + i, cfg_id=i)


_K3 = 0.25 * TWO_PI / 25.0

CONFIGS = {
    0: _mk(0, "cfg0_tiny_gamma_36", _cubic(10.0), 25.0, (0.0, 0.0, 0.0), (36, 36, 36), 16, 16, 2, _SP1, "diag"),
    1: _mk(1, "cfg1_64atom_gamma_80", _cubic(20.5), 30.0, (0.0, 0.0, 0.0), (80, 80, 80), 128, 128, 64, _SP2, "pair"),
    2: _mk(2, "cfg2_216atom_gamma_125", _cubic(30.0), 40.0, (0.0, 0.0, 0.0), (125, 125, 125), 512, 512, 216, _SP2, "pair"),
    3: _mk(3, "cfg3_128atom_k_96x96x144", (25.0, 0, 0, 0, 25.0, 0, 0, 0, 37.5), 35.0, (_K3, _K3, _K3),
           (96, 96, 144), 256, 256, 128, _SP2, "pair"),
    4: _mk(4, "cfg4_512atom_gamma_192", _cubic(40.0), 50.0, (0.0, 0.0, 0.0), (192, 192, 192), 1024, 128, 512, _SP2, "pair"),
}

_KT1 = 0.25 * TWO_PI / 6.0
# Tiny auxiliary cases for the dense-H oracle on features config 0 lacks.
TINY = {
    "T1_general_k": _mk(101, "T1_general_k", (6.0, 0, 0, 0, 6.0, 0, 0, 0, 9.0), 9.0, (_KT1, _KT1, _KT1),
                        (12, 12, 18), 5, 5, 2, _SP2, "pair"),
    "T2_radix5": _mk(102, "T2_radix5", _cubic(7.0), 8.0, (0.0, 0.0, 0.0), (15, 15, 15), 4, 4, 1, _SP2, "pair"),
    "T2b_radix5_20": _mk(106, "T2b_radix5_20", _cubic(7.0), 8.0, (0.0, 0.0, 0.0), (20, 20, 20), 3, 3, 1, _SP1, "diag"),
    # aliased: N just >= 2*nmax+1 (nmax = 3 at L=7, ecut=8) so V*psi wraps; cyclic identity must still hold
    "T3_aliased": _mk(103, "T3_aliased", _cubic(7.0), 8.0, (0.0, 0.0, 0.0), (8, 8, 8), 4, 4, 1, _SP2, "pair"),
    "T4_noproj": _mk(104, "T4_noproj", _cubic(7.0), 8.0, (0.0, 0.0, 0.0), (10, 12, 9), 4, 4, 0, _SP2, "pair"),
    "T5_odd_bands": _mk(105, "T5_odd_bands", (6.0, 0.5, 0, 0, 6.5, 0.3, 0.2, 0, 7.0), 9.0, (0.11, -0.07, 0.05),
                        (12, 15, 16), 7, 7, 2, _SP1, "diag"),
}


def get_workload(key) -> Workload:
    if isinstance(key, Workload):
        return key
    if key in CONFIGS:
        return CONFIGS[key]
    if isinstance(key, str) and key.isdigit():
        return CONFIGS[int(key)]
    return TINY[key]


# ----------------------------------------------------------------------------------------------------------
# counter-based RNG (64-bit mix hash -> 53-bit uniforms -> Box-Muller), torch int64 with wraparound
# ----------------------------------------------------------------------------------------------------------

STREAM_PSI, STREAM_V, STREAM_ATOMS, STREAM_D, STREAM_AUX = 1, 2, 3, 4, 5


def _s64(x: int) -> int:
    """Python int -> the signed 64-bit value with the same bits."""
    x &= (1 << 64) - 1
    return x - (1 << 64) if x >= (1 << 63) else x


_C1 = _s64(0xBF58476D1CE4E5B9)
_C2 = _s64(0x94D049BB133111EB)
_GOLD = _s64(0x9E3779B97F4A7C15)


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    return (z >> s) & ((1 << (64 - s)) - 1)


def _mix64(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lsr(z, 30)) * _C1
    z = (z ^ _lsr(z, 27)) * _C2
    return z ^ _lsr(z, 31)


def _hash_key(seed: int, stream: int, words) -> torch.Tensor:
    """words: list of int64 tensors (broadcastable) or Python ints. Returns int64 hash tensor."""
    dev = None
    for w in words:
        if isinstance(w, torch.Tensor):
            dev = w.device
            break
    h = torch.tensor(_s64(seed * 0x9E3779B97F4A7C15 + stream * 0xD1B54A32D192ED03 + 0x2545F4914F6CDD1D),
                     dtype=torch.int64, device=dev)
    h = _mix64(h)
    for i, w in enumerate(words):
        if not isinstance(w, torch.Tensor):
            w = torch.tensor(int(w), dtype=torch.int64, device=dev)
        w = w.to(torch.int64)
        h = _mix64(h ^ _mix64(w + _s64(_GOLD * (i + 1))))
    return h


def _uniform(h: torch.Tensor, lane: int) -> torch.Tensor:
    """53-bit uniform in (0,1) from hash h and a lane number."""
    z = _mix64(h + _s64(_GOLD * (lane + 1)))
    return (_lsr(z, 11).to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)


def _normal_pair(h: torch.Tensor):
    u1 = _uniform(h, 0)
    u2 = _uniform(h, 1)
    r = torch.sqrt(-2.0 * torch.log(u1))
    return r * torch.cos(TWO_PI * u2), r * torch.sin(TWO_PI * u2)


# ----------------------------------------------------------------------------------------------------------
# geometry helpers (input generation only; the method's own reciprocal-lattice arithmetic lives elsewhere)
# ----------------------------------------------------------------------------------------------------------


def _recip_np(at) -> np.ndarray:
    a = np.array(at, dtype=np.float64).reshape(3, 3)
    return TWO_PI * np.linalg.inv(a).T  # rows b_i with a_i . b_j = 2 pi delta_ij


def _gcart(wl: Workload, miller: torch.Tensor) -> torch.Tensor:
    """Cartesian G (no k) for int Miller triples [n,3] -> float64 [n,3]."""
    b = torch.tensor(_recip_np(wl.at), dtype=torch.float64, device=miller.device)
    return miller.to(torch.float64) @ b


# ----------------------------------------------------------------------------------------------------------
# psi
# ----------------------------------------------------------------------------------------------------------


def gen_psi(wl: Workload, miller, band0: int = 0, nbands: int | None = None, ld: int | None = None,
            device="cpu") -> torch.Tensor:
    """psi[b][ig] complex128, shape [nbands, ld] (ld >= npw, pad columns zero).

    SURVEY 8(c) item 6: re, im ~ N(0,1) keyed by (band, Miller triple), times 1/(1+|G|^2) (literal |G|^2, not
    |k+G|^2), each band normalised to sum |c|^2 = 1.
    """
    wl = get_workload(wl)
    miller = torch.as_tensor(miller, device=device).to(torch.int64)
    npw = miller.shape[0]
    nbands = wl.nbands - band0 if nbands is None else nbands
    ld = npw if ld is None else ld
    g = _gcart(wl, miller)
    w = 1.0 / (1.0 + (g * g).sum(1))
    out = torch.zeros((nbands, ld), dtype=torch.complex128, device=device)
    step = max(1, (1 << 24) // max(npw, 1))
    for b0 in range(0, nbands, step):
        b1 = min(nbands, b0 + step)
        bands = torch.arange(band0 + b0, band0 + b1, dtype=torch.int64, device=device)[:, None]
        h = _hash_key(wl.seed, STREAM_PSI, [bands, miller[None, :, 0], miller[None, :, 1], miller[None, :, 2]])
        re, im = _normal_pair(h)
        c = torch.complex(re * w, im * w)
        c = c / torch.sqrt((c.real**2 + c.imag**2).sum(1, keepdim=True))
        out[b0:b1, :npw] = c
    return out


# ----------------------------------------------------------------------------------------------------------
# local potential V(r)
# ----------------------------------------------------------------------------------------------------------


def gen_vloc_g(wl: Workload, device="cpu"):
    """V(G) on the support |G|^2 <= 100. Returns (miller_v [nv,3] int64, vg [nv] c128)
    with V(-G) = conj V(G) and V(0) real. Complex normal times exp(-|G|^2/4)."""
    wl = get_workload(wl)
    a = np.array(wl.at, dtype=np.float64).reshape(3, 3)
    gmax = 10.0
    nmax = [int(math.floor(gmax * np.linalg.norm(a[j]) / TWO_PI)) + 1 for j in range(3)]
    for j in range(3):
        # the support must fit the grid without wrapping onto itself
        nmax[j] = min(nmax[j], (wl.nr[j] - 1) // 2)
    r = [torch.arange(-n, n + 1, dtype=torch.int64, device=device) for n in nmax]
    m = torch.stack(torch.meshgrid(*r, indexing="ij"), dim=-1).reshape(-1, 3)
    g = _gcart(wl, m)
    g2 = (g * g).sum(1)
    keep = g2 <= gmax * gmax
    m, g2 = m[keep], g2[keep]
    # lexicographic sign of the triple: first non-zero component
    sgn = torch.sign(m[:, 0]) * 4 + torch.sign(m[:, 1]) * 2 + torch.sign(m[:, 2])
    pos = sgn > 0
    zero = sgn == 0
    rep = torch.where(pos[:, None] | zero[:, None], m, -m)  # canonical representative of the +-G pair
    h = _hash_key(wl.seed, STREAM_V, [rep[:, 0], rep[:, 1], rep[:, 2]])
    re, im = _normal_pair(h)
    im = torch.where(pos, im, -im)
    im = torch.where(zero, torch.zeros_like(im), im)
    damp = torch.exp(-g2 / 4.0)
    return m, torch.complex(re * damp, im * damp)


def gen_vloc(wl: Workload, device="cpu") -> torch.Tensor:
    """Real V(r) [N1,N2,N3] float64 = sum_G V(G) exp(+i G.r) on the grid r = sum_j (i_j/N_j) a_j."""
    wl = get_workload(wl)
    m, vg = gen_vloc_g(wl, device=device)
    n1, n2, n3 = wl.nr
    box = torch.zeros((n1, n2, n3), dtype=torch.complex128, device=device)
    box[m[:, 0] % n1, m[:, 1] % n2, m[:, 2] % n3] = vg
    vr = torch.fft.ifftn(box) * float(n1 * n2 * n3)
    assert float(vr.imag.abs().max()) <= 1e-10 * max(1.0, float(vr.real.abs().max())), "V(r) not real"
    return vr.real.contiguous()


# ----------------------------------------------------------------------------------------------------------
# atoms, projectors, D
# ----------------------------------------------------------------------------------------------------------


def gen_atoms(wl: Workload) -> np.ndarray:
    """Fractional coordinates [natoms,3], sequential rejection sampling with minimum-image separation
    >= wl.min_sep bohr. CPU/numpy: at most 512 atoms."""
    wl = get_workload(wl)
    a = np.array(wl.at, dtype=np.float64).reshape(3, 3)
    shifts = np.array([[i, j, k] for i in (-1, 0, 1) for j in (-1, 0, 1) for k in (-1, 0, 1)], dtype=np.float64)
    pos = np.zeros((wl.natoms, 3))
    n = 0
    attempt = 0
    while n < wl.natoms:
        h = _hash_key(wl.seed, STREAM_ATOMS, [n, attempt])
        f = np.array([float(_uniform(h, i)) for i in range(3)])
        attempt += 1
        ok = True
        if n:
            d = f[None, :] - pos[:n]  # fractional differences
            d = d - np.round(d)
            dc = (d[:, None, :] + shifts[None, :, :]) @ a
            ok = bool(np.sqrt((dc * dc).sum(-1)).min() >= wl.min_sep)
        if ok:
            pos[n] = f
            n += 1
            attempt = 0
        assert attempt < 100000, "atom placement did not terminate"
    return pos


_Y00 = 0.28209479177387814  # 1/sqrt(4 pi)
_Y1 = 0.4886025119029199  # sqrt(3/(4 pi))


def gen_beta(wl: Workload, miller, atoms_frac, atom0: int = 0, natoms: int | None = None, ld: int | None = None,
             device="cpu", out: torch.Tensor | None = None) -> torch.Tensor:
    """beta[p][ig] complex128 for atoms atom0..atom0+natoms-1 -> [natoms*nh, ld].

    beta_{a,(n,l,m)}(G) = q^l exp(-q^2 rc_n^2/2) Y_lm(q^) exp(-i q.tau_a)/sqrt(Omega), q = k+G, real Y_lm with
    q^l Y_1c evaluated as the polynomial sqrt(3/4pi) q_c (c = x,y,z). Atoms outermost; channel order as
    `wl.channels`, m innermost."""
    wl = get_workload(wl)
    miller = torch.as_tensor(miller, device=device).to(torch.int64)
    npw = miller.shape[0]
    natoms = wl.natoms - atom0 if natoms is None else natoms
    ld = npw if ld is None else ld
    nh = wl.nh
    if out is None:
        out = torch.zeros((natoms * nh, ld), dtype=torch.complex128, device=device)
    if natoms == 0 or npw == 0:
        return out
    q = _gcart(wl, miller) + torch.tensor(wl.xk, dtype=torch.float64, device=device)[None, :]
    q2 = (q * q).sum(1)
    a = np.array(wl.at, dtype=np.float64).reshape(3, 3)
    tau = torch.tensor(np.asarray(atoms_frac)[atom0:atom0 + natoms] @ a, dtype=torch.float64, device=device)
    inv_sqrt_omega = 1.0 / math.sqrt(wl.omega)
    radial = []  # per projector within an atom: real [npw]
    for l, rc in wl.channels:
        e = torch.exp(-q2 * (rc * rc / 2.0)) * inv_sqrt_omega
        if l == 0:
            radial.append(e * _Y00)
        elif l == 1:
            for c in range(3):
                radial.append(e * (_Y1 * q[:, c]))
        else:
            raise NotImplementedError("l > 1")
    radial = torch.stack(radial, 0)  # [nh, npw]
    for ia in range(natoms):
        ph = q @ tau[ia]
        sf = torch.complex(torch.cos(ph), -torch.sin(ph))
        out[ia * nh:(ia + 1) * nh, :npw] = radial * sf[None, :]
    return out


def gen_dblocks(wl: Workload) -> np.ndarray:
    """D blocks [natoms, nh, nh] float64, real symmetric, entries U(-1,1) Ry."""
    wl = get_workload(wl)
    nh = wl.nh
    d = np.zeros((wl.natoms, nh, nh))

    def u(a, l, e):
        h = _hash_key(wl.seed, STREAM_D, [a, l, e])
        return 2.0 * float(_uniform(h, 0)) - 1.0

    for a in range(wl.natoms):
        if wl.dmode == "diag":
            off = 0
            for l, _ in wl.channels:
                v = u(a, l, 0)
                for m in range(2 * l + 1):
                    d[a, off + m, off + m] = v
                off += 2 * l + 1
        else:  # "pair": channels come as (l, rc1), (l, rc2) for each l
            off = 0
            chans = list(wl.channels)
            i = 0
            while i < len(chans):
                l = chans[i][0]
                assert chans[i + 1][0] == l
                m2 = 2 * l + 1
                d11, d12, d22 = u(a, l, 0), u(a, l, 1), u(a, l, 2)
                for m in range(m2):
                    p, q = off + m, off + m2 + m
                    d[a, p, p] = d11
                    d[a, q, q] = d22
                    d[a, p, q] = d[a, q, p] = d12
                off += 2 * m2
                i += 2
    return d


def aux_normal_complex(seed: int, key: int, n: int, device="cpu") -> torch.Tensor:
    """Complex normal vector of length n keyed by (seed, key): probe vectors for the Hermiticity tests."""
    idx = torch.arange(n, dtype=torch.int64, device=device)
    re, im = _normal_pair(_hash_key(seed, STREAM_AUX, [key, idx]))
    return torch.complex(re, im)


def aux_choice(seed: int, key: int, n: int, k: int) -> np.ndarray:
    """k distinct integers in [0, n), seeded, sorted."""
    idx = torch.arange(n, dtype=torch.int64)
    h = _hash_key(seed, STREAM_AUX, [key + 7919, idx])
    order = torch.argsort(_lsr(h, 1))
    return np.sort(order[:k].numpy())


def pad8(n: int) -> int:
    """Leading dimension used by the harness: npw rounded up to a multiple of 8 elements (128 B rows)."""
    return (n + 7) // 8 * 8
