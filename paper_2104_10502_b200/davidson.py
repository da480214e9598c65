"""Block Davidson driver around the library's H|psi> / S|psi> (the paper's KS_Solvers call the
Hamiltonian builder through exactly this kind of loop).

Host orchestration only. Every arithmetic operation on O(npw) data runs in libqe_hpsi.so: qe_hpsi_apply(_hs) (H psi,
S psi), qe_hpsi_overlap (reduced matrices), qe_hpsi_rotate (basis rotation), qe_hpsi_residual (h - e s and its squared
norms), qe_hpsi_hdiag / qe_hpsi_precond (preconditioner), qe_hpsi_scale (normalisation). What torch does here: row
copies between band arrays, O(nev) scalar work on the norms, and the small dense generalized eigenproblem of the
reduced matrices (at most 4 nev x 4 nev) via torch.linalg on the device -- the role LAXlib / cuSOLVER play in the
paper.
"""
from __future__ import annotations

import torch


def _herm(m):
    return 0.5 * (m + m.conj().transpose(-1, -2))


def _reduced_eig(hr, sr, nev):
    """lowest nev eigenpairs of hr v = e sr v (both Hermitian, sr positive definite) via Cholesky reduction."""
    l = torch.linalg.cholesky(_herm(sr))
    a = torch.linalg.solve_triangular(l, _herm(hr), upper=False)
    a = torch.linalg.solve_triangular(l, a.conj().transpose(-1, -2), upper=False).conj().transpose(-1, -2)
    e, w = torch.linalg.eigh(_herm(a))
    v = torch.linalg.solve_triangular(l.conj().transpose(-1, -2), w[:, :nev], upper=True)
    return e[:nev], v  # v: [m, nev], columns S-orthonormal in the basis


def davidson(h, psi0, vbar, use_s=False, tol=1e-9, max_iter=60, max_basis=4):
    """Lowest nev = psi0.shape[0] eigenpairs of H c = e S c (S = 1 unless use_s; then h.set_s must have been called).

    h: qe_hpsi.Hpsi; psi0 [nev, ld] complex128 CUDA start vectors (linearly independent); vbar = mean of V(r).
    Returns (e [nev] float64 CUDA, psi [nev, ld], info dict). Convergence: ||H c - e S c|| <= tol * max(1, |e|) per band.
    """
    nev, ld = int(psi0.shape[0]), int(psi0.shape[1])
    npw = h.npw
    dev = psi0.device
    mmax = max_basis * nev
    x = torch.zeros((mmax, ld), dtype=torch.complex128, device=dev)
    hx = torch.zeros_like(x)
    sx = torch.zeros_like(x) if use_s else x
    hd, sd = h.hdiag(vbar, want_s=use_s)

    def apply(block, hout, sout):
        if use_s:
            h.apply_hs(block, hout, sout)
        else:
            h.apply(block, hout)

    x[:nev] = psi0
    x[:nev, npw:] = 0
    apply(x[:nev], hx[:nev], sx[:nev] if use_s else None)
    m = nev
    napply = nev
    e = None
    resn = None
    for it in range(max_iter):
        hr = h.overlap(x[:m], hx[:m])
        sr = h.overlap(x[:m], sx[:m])
        e, v = _reduced_eig(hr, sr, nev)
        coef = v.transpose(0, 1).contiguous()  # [nev, m]
        psi = h.rotate(x[:m], coef)
        hpsi = h.rotate(hx[:m], coef)
        spsi = h.rotate(sx[:m], coef) if use_s else psi
        r, rn2 = h.residual(hpsi, spsi, e)  # r = H c - e S c over the sphere entries, |r|^2 per band
        resn = rn2.sqrt()
        unconv = (resn > tol * torch.clamp(e.abs(), min=1.0)).nonzero().flatten()
        k = int(unconv.numel())
        if k == 0:
            return e, psi, dict(iterations=it, applies=napply, residual=float(resn.max()), converged=True)
        if m + k > mmax:  # restart from the current Ritz vectors
            x[:nev], hx[:nev] = psi, hpsi
            if use_s:
                sx[:nev] = spsi
            m = nev
        t = r[unconv].contiguous()
        h.precond(t, e[unconv].contiguous(), hd, sd)
        _, tn2 = h.residual(t, t, torch.zeros(k, dtype=torch.float64, device=dev), r=t)  # e = 0: t unchanged, |t|^2
        h.scale(t, tn2.rsqrt())
        x[m:m + k] = t
        apply(x[m:m + k], hx[m:m + k], sx[m:m + k] if use_s else None)
        napply += k
        m += k
    return e, psi, dict(iterations=max_iter, applies=napply, residual=float(resn.max()), converged=False)
