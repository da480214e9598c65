"""CPU ORACLE for H|psi> -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain, slow, obviously-correct numpy (fp64 / complex128) implementation of what the CUDA library
`libqe_hpsi.so` computes. Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline /
`--impl reference` legs may import this file. It shares no code with `paper_2104_10502_b200/csrc` and does not
import the binding; the product path never imports it.

What is computed (PAPER.md is a review paper with no formulas; it names the operation and its three terms:
"Hamiltonian builds (i.e. the application of the one-particle Hamiltonian to ... Bloch states)"
section III; "local-potential, pseudopotential, kinetic-energy contributions to the Hamiltonian", PAPER.md:L224-226
section III.C; "generation of plane waves and of their mapping to FFT grids", PAPER.md:L176 (vi)). The formula
is BASELINE.json north_star's

    H_GG' = |k+G|^2 delta_GG' + V(G-G') + sum_a sum_ij beta_ai(G) D^a_ij conj(beta_aj(G'))

in Rydberg atomic units, with the readings of SURVEY.md 8(c) / DESIGN.md section 3:
  * V(G-G') := Vt[(n-n') mod N], Vt[m] = (1/N) sum_i V(r_i) exp(-2 pi i sum_j m_j i_j / N_j)  (3-D DFT of
    the INPUT real-space array, cyclically wrapped). With this reading the dual-space procedure equals the
    definition identically (cyclic convolution theorem).
  * sphere: |k+G|^2 <= ecutwfc inclusive, FP64, un-fused operations in the order written in `gsphere`.
  * canonical order of the sphere: ascending FFT linear index idx = (i1*N2 + i2)*N3 + i3 of the wrapped triple.
  * psi(r) = sum_G c(G) exp(+i(k+G).r): grid array = un-normalised DFT with exp(+2 pi i ...); back-transform
    exp(-2 pi i ...) with 1/N.

Three levels:
  Level A  `dense_h` + matvec      -- the definition written out (tiny cases only); uses explicit DFT matrices,
                                     never numpy.fft.
  Level A' `hpsi_rows`             -- the definition evaluated for sampled rows G (any size); explicit DFT
                                     matrices for Vt, never an FFT of psi.
  Level B  `hpsi_dual`             -- scatter -> inverse DFT -> V(r) multiply -> forward DFT -> gather, with
                                     numpy.fft as the library DFT step; also the timed CPU baseline.

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): closed forms (single plane wave in constant V0; cosine
potential shift; rank-1 projector), FFT round trip / Parseval / naive O(n^2) DFT, Hermiticity, translation
covariance, time reversal at k=0, linearity, A == A' == B on tiny cases, independently enumerated npw counts
(tests/golden/npw_counts.txt from SURVEY.md 8 table). The functions of the "next" rows at the end of the file
(`spsi_of`, `overlap_of`, `psi_r`, `density_of`) are pinned in tests/test_oracle_next.py (rank-1 closed form, brute-force
loops, Hermiticity, single / two plane-wave closed forms, Parseval, explicit DFT matrices). The error metric `rel_l2`
(the gate of every parity assertion) is pinned by hand-built vectors with known per-band errors
(test_rel_l2_is_per_band_relative_to_the_reference); the `becp=` branch of `hpsi_rows` by
test_sampled_rows_with_becp_accumulated_over_atom_chunks. Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

TWO_PI = 6.283185307179586


# ----------------------------------------------------------------------------------------------------------
# a0: reciprocal lattice, G-sphere and its maps  (PAPER.md:L176 (vi))
# ----------------------------------------------------------------------------------------------------------


def recip(at):
    """Reciprocal rows b_j (a_i . b_j = 2 pi delta_ij) and signed cell volume. Operation order:
    c1 = a2 x a3, c2 = a3 x a1, c3 = a1 x a2, each component (u*v) - (w*z) with every product rounded;
    vol = (a1x*c1x + a1y*c1y) + a1z*c1z;  b_jc = (2pi * c_jc) / vol."""
    a = np.asarray(at, dtype=np.float64).reshape(3, 3)

    def cross(u, v):
        return np.array([u[1] * v[2] - u[2] * v[1], u[2] * v[0] - u[0] * v[2], u[0] * v[1] - u[1] * v[0]])

    c = [cross(a[1], a[2]), cross(a[2], a[0]), cross(a[0], a[1])]
    vol = (a[0, 0] * c[0][0] + a[0, 1] * c[0][1]) + a[0, 2] * c[0][2]
    b = np.array([[(TWO_PI * c[j][k]) / vol for k in range(3)] for j in range(3)])
    return b, vol


def kfrac(at, xk):
    """Fractional k: kappa_j = ((a_jx*kx + a_jy*ky) + a_jz*kz) / 2pi."""
    a = np.asarray(at, dtype=np.float64).reshape(3, 3)
    k = np.asarray(xk, dtype=np.float64)
    return np.array([((a[j, 0] * k[0] + a[j, 1] * k[1]) + a[j, 2] * k[2]) / TWO_PI for j in range(3)])


def signed_index(i, n):
    """Wrapped FFT index i in [0,n) -> Miller index: i if i < (n+1)//2 else i - n."""
    i = np.asarray(i)
    return np.where(i >= (n + 1) // 2, i - n, i)


def gsphere(at, xk, ecutwfc, nr):
    """Enumerate the whole FFT box in ascending linear index and keep |k+G|^2 <= ecutwfc.

    Returns dict(miller int32 [npw,3], fft_index int32 [npw] (strictly increasing), g2kin float64 [npw]).
    Arithmetic per point, un-fused, in this order: m_j = n_j + kappa_j;  q_c = (m1*b1c + m2*b2c) + m3*b3c;
    q2 = (qx*qx + qy*qy) + qz*qz; keep iff q2 <= ecutwfc; g2kin = q2."""
    n1, n2, n3 = (int(x) for x in nr)
    b, _ = recip(at)
    kap = kfrac(at, xk)
    m1 = signed_index(np.arange(n1), n1).astype(np.float64) + kap[0]
    m2 = signed_index(np.arange(n2), n2).astype(np.float64) + kap[1]
    m3 = signed_index(np.arange(n3), n3).astype(np.float64) + kap[2]
    mil, idx, g2 = [], [], []
    for i1 in range(n1):  # plane by plane to bound memory at 192^3
        q = []
        for c in range(3):
            t = (m1[i1] * b[0, c] + m2[:, None] * b[1, c]) + m3[None, :] * b[2, c]
            q.append(t)
        q2 = (q[0] * q[0] + q[1] * q[1]) + q[2] * q[2]
        i2s, i3s = np.nonzero(q2 <= ecutwfc)  # row-major: ascending i2 then i3
        if i2s.size:
            idx.append((i1 * n2 + i2s) * n3 + i3s)
            g2.append(q2[i2s, i3s])
            mil.append(np.stack([np.full(i2s.shape, signed_index(i1, n1)), signed_index(i2s, n2),
                                 signed_index(i3s, n3)], 1))
    if not idx:
        return dict(miller=np.zeros((0, 3), np.int32), fft_index=np.zeros(0, np.int32), g2kin=np.zeros(0))
    return dict(miller=np.concatenate(mil).astype(np.int32), fft_index=np.concatenate(idx).astype(np.int32),
                g2kin=np.concatenate(g2))


def fft_index_of(miller, nr):
    """miller -> linear FFT index of the wrapped triple (the inverse of the map above)."""
    m = np.asarray(miller, dtype=np.int64)
    n1, n2, n3 = nr
    return ((m[:, 0] % n1) * n2 + (m[:, 1] % n2)) * n3 + (m[:, 2] % n3)


# ----------------------------------------------------------------------------------------------------------
# explicit DFT (the definition; no FFT library)
# ----------------------------------------------------------------------------------------------------------


def dft_matrix(n, sign):
    """W[m, i] = exp(sign * 2 pi i * m*i / n), angle reduced with integer (m*i mod n) so it stays accurate."""
    mi = np.outer(np.arange(n), np.arange(n)) % n
    ang = (TWO_PI / n) * mi
    # exact values at multiples of a quarter turn
    w = np.cos(ang) + 1j * sign * np.sin(ang)
    q = (4 * mi) % n == 0
    quarter = (4 * mi) // n
    exact = np.array([1, 1j * sign, -1, -1j * sign], dtype=np.complex128)
    w[q] = exact[quarter[q] % 4]
    return w


def dft3_explicit(x, sign):
    """Un-normalised 3-D DFT of x[N1,N2,N3] with exp(sign*2 pi i ...) along every axis, by explicit
    DFT-matrix products (O(N (N1+N2+N3)))."""
    x = np.asarray(x, dtype=np.complex128)
    n1, n2, n3 = x.shape
    y = np.tensordot(dft_matrix(n1, sign), x, axes=([1], [0]))  # [m1, i2, i3]
    y = np.tensordot(dft_matrix(n2, sign), y, axes=([1], [1])).transpose(1, 0, 2)  # [m1, m2, i3]
    y = np.tensordot(y, dft_matrix(n3, sign), axes=([2], [1]))  # [m1, m2, m3]
    return y


def vloc_coeffs(vr):
    """Vt[m] = (1/N) sum_i V(r_i) exp(-2 pi i sum_j m_j i_j/N_j): DFT coefficients of the input V(r) array."""
    vr = np.asarray(vr, dtype=np.float64)
    return dft3_explicit(vr, -1) / vr.size


# ----------------------------------------------------------------------------------------------------------
# nonlocal pieces (a6, a7, a8)
# ----------------------------------------------------------------------------------------------------------


def becp_of(beta, psi):
    """a6: becp[p][b] = sum_G conj(beta[p][G]) psi[b][G].  beta [nproj,npw], psi [nb,npw] -> [nproj,nb]."""
    return np.conj(beta) @ psi.T


def dbecp_of(dblocks, becp):
    """a7: dbecp[a,i][b] = sum_j D^a_ij becp[a,j][b].  dblocks [nat,nh,nh] real; becp [nat*nh, nb]."""
    nat, nh, _ = dblocks.shape
    if nat == 0:
        return becp.copy()
    return np.einsum("aij,ajb->aib", dblocks, becp.reshape(nat, nh, -1)).reshape(nat * nh, -1)


def vnl_psi(beta, dblocks, psi):
    """a6-a8: sum_a sum_ij beta_ai(G) D^a_ij <beta_aj|psi_b>  -> [nb, npw]."""
    if beta is None or beta.shape[0] == 0:
        return np.zeros_like(psi)
    return (beta.T @ dbecp_of(dblocks, becp_of(beta, psi))).T


# ----------------------------------------------------------------------------------------------------------
# Level A: dense H from the definition
# ----------------------------------------------------------------------------------------------------------


def dense_h(miller, g2kin, nr, vr, beta=None, dblocks=None):
    """H[G,G'] = g2kin[G] delta + Vt[(n-n') mod N] + sum_a beta_a(G) D^a beta_a(G')^H.  npw x npw complex128."""
    m = np.asarray(miller, dtype=np.int64)
    npw = m.shape[0]
    vt = vloc_coeffs(vr)
    d = m[:, None, :] - m[None, :, :]
    h = vt[d[..., 0] % nr[0], d[..., 1] % nr[1], d[..., 2] % nr[2]].astype(np.complex128)
    h[np.arange(npw), np.arange(npw)] += g2kin
    if beta is not None and beta.shape[0] > 0:
        nat, nh, _ = dblocks.shape
        for a in range(nat):
            ba = beta[a * nh:(a + 1) * nh]  # [nh, npw]
            h += ba.T @ (dblocks[a] @ np.conj(ba))
    return h


def hpsi_dense(h, psi):
    """psi [nb,npw] -> (H psi) [nb,npw]."""
    return (h @ psi.T).T


# ----------------------------------------------------------------------------------------------------------
# Level A': the definition for sampled rows
# ----------------------------------------------------------------------------------------------------------


def hpsi_rows(rows, miller, g2kin, nr, vt, psi, beta=None, dblocks=None, becp=None):
    """(H psi_b)(G) for G in `rows` (indices into the sphere) and every band of psi [nb,npw] -> [nb,len(rows)].

    vt = vloc_coeffs(vr) (pass it in: it is shared by all rows). If `becp` [nproj, nb] is given it is used
    as <beta|psi> (lets the caller accumulate it over chunks of a beta too large for host memory); then `beta`
    only needs its columns at `rows`: pass beta[:, rows] as `beta` with beta_is_rows semantics (shape
    [nproj, len(rows)])."""
    m = np.asarray(miller, dtype=np.int64)
    rows = np.asarray(rows, dtype=np.int64)
    out = np.zeros((psi.shape[0], rows.size), dtype=np.complex128)
    for j, g in enumerate(rows):
        d = m[g][None, :] - m  # n - n'
        vrow = vt[d[:, 0] % nr[0], d[:, 1] % nr[1], d[:, 2] % nr[2]]
        out[:, j] = psi @ vrow + g2kin[g] * psi[:, g]
    if beta is not None and beta.shape[0] > 0:
        if becp is None:
            becp = becp_of(beta, psi)
            bcols = beta[:, rows]
        else:
            bcols = beta if beta.shape[1] == rows.size else beta[:, rows]
        out += (bcols.T @ dbecp_of(dblocks, becp)).T
    return out


# ----------------------------------------------------------------------------------------------------------
# Level B: dual-space application (library FFT as the DFT step) -- also the timed CPU baseline
# ----------------------------------------------------------------------------------------------------------


def vloc_psi_dual(fft_index, nr, vr, psi):
    """a1-a5 without the kinetic term: gather( DFT-[ V(r) * DFT+[ scatter(psi) ] ] / N ) per band."""
    n = int(nr[0]) * int(nr[1]) * int(nr[2])
    out = np.empty_like(psi)
    for b in range(psi.shape[0]):
        box = np.zeros(n, dtype=np.complex128)
        box[fft_index] = psi[b]
        pr = np.fft.ifftn(box.reshape(nr)) * n  # un-normalised exp(+)
        vp = np.fft.fftn(vr * pr) / n  # exp(-) with 1/N
        out[b] = vp.reshape(-1)[fft_index]
    return out


def hpsi_dual(fft_index, g2kin, nr, vr, psi, beta=None, dblocks=None):
    """Level B: H psi = g2kin*psi + dual-space local term + nonlocal term. psi [nb,npw] -> [nb,npw]."""
    out = vloc_psi_dual(fft_index, nr, vr, psi)
    out += g2kin[None, :] * psi
    if beta is not None and beta.shape[0] > 0:
        out += vnl_psi(beta, dblocks, psi)
    return out


def rel_l2(x, ref):
    """Per-band relative L2 error ||x-ref||/||ref|| (long-double norms). x, ref [nb, npw]."""
    d = (x - ref).astype(np.clongdouble)
    r = ref.astype(np.clongdouble)
    num = np.sqrt((d.real**2 + d.imag**2).sum(-1))
    den = np.sqrt((r.real**2 + r.imag**2).sum(-1))
    return np.asarray(num / den, dtype=np.float64)


# ----------------------------------------------------------------------------------------------------------
# Rows marked "next" in SURVEY.md 8(f): overlap operator S, reduced matrices of the Davidson step, charge density
# ("application of the overlap operator", "charge density generation"; iterative diagonaliser
# calling H|psi> and S|psi>).  The paper prints no formula; these are the textbook
# definitions in the conventions fixed above (DESIGN.md section 2 items 18-20).
# ----------------------------------------------------------------------------------------------------------


def spsi_of(beta, qblocks, psi):
    """NEXT-2: S psi = psi + sum_a sum_ij beta_ai(G) q^a_ij <beta_aj|psi>  (ultrasoft/PAW overlap operator with
    per-atom real symmetric q blocks [nat,nh,nh]).  psi [nb,npw] -> [nb,npw]."""
    return psi + vnl_psi(beta, qblocks, psi)


def overlap_of(a, b):
    """NEXT-3: reduced matrix M[i][j] = <a_i|b_j> = sum_G conj(a[i][G]) b[j][G].  a [na,npw], b [nb,npw] -> [na,nb].
    With a = psi, b = H psi (S psi) this is the projected Hamiltonian (overlap) of the Davidson step."""
    return np.conj(a) @ b.T


def psi_r(fft_index, nr, psi_b):
    """psi(r_i) = sum_G c(G) exp(+2 pi i n.i/N) on the full grid for one band (un-normalised inverse DFT,
    reading 4 of DESIGN.md section 2; the Bloch phase has modulus 1 and drops out of |psi(r)|^2)."""
    n = int(nr[0]) * int(nr[1]) * int(nr[2])
    box = np.zeros(n, dtype=np.complex128)
    box[fft_index] = psi_b
    return np.fft.ifftn(box.reshape(nr)) * n


def density_of(fft_index, nr, psi, occ, scale):
    """NEXT-4: rho(r_i) = scale * sum_b occ[b] |psi_b(r_i)|^2 on the [N1,N2,N3] grid (scale = 1/Omega gives
    electrons per bohr^3 for normalised bands)."""
    rho = np.zeros(tuple(int(x) for x in nr), dtype=np.float64)
    for b in range(psi.shape[0]):
        pr = psi_r(fft_index, nr, psi[b])
        rho += occ[b] * (pr.real**2 + pr.imag**2)
    return scale * rho


# ----------------------------------------------------------------------------------------------------------
# NEXT-1: Gamma-only path (k = 0, real wavefunctions; the paper ports "Gamma-point specific algorithms" for every
# kernel).  Only the half sphere is stored: c(-G) = conj(c(G)).  The oracle is the definition: expand
# to the full sphere, apply the full-sphere H, restrict (DESIGN.md section 2 item 21).
# ----------------------------------------------------------------------------------------------------------


def gamma_half(miller):
    """Half sphere of a k = 0 sphere in canonical order: keep G = (n1,n2,n3) with n1 > 0, or n1 == 0 and n2 > 0, or
    n1 == n2 == 0 and n3 >= 0 (G = 0 included), in the order they have in the full sphere.
    Returns (idx_plus [ngw] positions of G in the full sphere, idx_minus [ngw] positions of -G)."""
    m = np.asarray(miller, dtype=np.int64)
    keep = (m[:, 0] > 0) | ((m[:, 0] == 0) & (m[:, 1] > 0)) | ((m[:, 0] == 0) & (m[:, 1] == 0) & (m[:, 2] >= 0))
    idx_plus = np.nonzero(keep)[0]
    pos = {tuple(v): i for i, v in enumerate(m.tolist())}
    idx_minus = np.array([pos[(-a, -b, -c)] for a, b, c in m[idx_plus].tolist()], dtype=np.int64)
    return idx_plus, idx_minus


def gamma_expand(x_half, idx_plus, idx_minus, npw):
    """[nb, ngw] half-sphere coefficients -> [nb, npw] full sphere with x(-G) = conj(x(G)) (G = 0 kept as given)."""
    full = np.zeros((x_half.shape[0], npw), dtype=np.complex128)
    full[:, idx_minus] = np.conj(x_half)
    full[:, idx_plus] = x_half
    return full


def hpsi_gamma(miller, fft_index, g2kin, nr, vr, psi_half, beta_half=None, dblocks=None):
    """(H psi) on the half sphere for real wavefunctions: expand psi and beta to the full sphere (Hermitian
    completion), apply Level B, restrict to the half sphere.  psi_half [nb, ngw] with Im psi(G=0) = 0."""
    ip, im = gamma_half(miller)
    npw = np.asarray(miller).shape[0]
    psi = gamma_expand(psi_half, ip, im, npw)
    beta = gamma_expand(beta_half, ip, im, npw) if beta_half is not None and beta_half.shape[0] else None
    return hpsi_dual(fft_index, g2kin, nr, vr, psi, beta, dblocks)[:, ip]


# ----------------------------------------------------------------------------------------------------------
# NEXT-3, the rest of the Davidson step around H|psi> ("iterative diagonalization", L168 "RCI"):
# diagonal of H and S for the preconditioner, the preconditioner itself, and the basis rotation.
# ----------------------------------------------------------------------------------------------------------


def hdiag_of(g2kin, vbar, beta=None, dblocks=None):
    """Preconditioner diagonal h_diag(G) = |k+G|^2 + vbar + sum_a sum_i D^a_ii |beta_ai(G)|^2 with vbar = mean of V(r)
    (= Vt[0], the diagonal of the local term).  Only the i = j terms of D enter (the usual plane-wave-code choice):
    it is the exact diagonal of H when every D^a is diagonal, and of H with D replaced by diag(D) otherwise."""
    out = np.asarray(g2kin, dtype=np.float64) + float(vbar)
    if beta is not None and beta.shape[0]:
        nat, nh, _ = dblocks.shape
        dii = np.stack([np.diag(dblocks[a]) for a in range(nat)]).reshape(-1)  # [nproj]
        out = out + dii @ (beta.real**2 + beta.imag**2)
    return out


def sdiag_of(npw, beta=None, qblocks=None):
    """s_diag(G) = 1 + sum_a sum_i q^a_ii |beta_ai(G)|^2 (same convention as hdiag_of)."""
    return hdiag_of(np.ones(npw), 0.0, beta, qblocks)


def precond_of(r, e, hdiag, sdiag):
    """Davidson preconditioner (the smooth form used by plane-wave codes): x = hdiag(G) - e_b sdiag(G),
    r_b(G) / ( (1 + x + sqrt(1 + (x-1)^2)) / 2 ).  r [nb,npw], e [nb]."""
    x = hdiag[None, :] - np.asarray(e)[:, None] * sdiag[None, :]
    return r / (0.5 * (1.0 + x + np.sqrt(1.0 + (x - 1.0) ** 2)))


def rotate_of(x, coef):
    """Basis rotation y[k][G] = sum_j coef[k][j] x[j][G].  x [nx,npw], coef [ny,nx] -> [ny,npw]."""
    return coef @ x


def dense_s(beta, qblocks, npw):
    """S[G,G'] = delta + sum_a beta_a(G) q^a beta_a(G')^H (tiny cases)."""
    s = np.eye(npw, dtype=np.complex128)
    if beta is not None and beta.shape[0]:
        nat, nh, _ = qblocks.shape
        for a in range(nat):
            ba = beta[a * nh:(a + 1) * nh]
            s += ba.T @ (qblocks[a] @ np.conj(ba))
    return s
