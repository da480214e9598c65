"""GPU parity: libqe_hpsi.so (through the C ABI / ctypes binding) against the CPU oracle, element by element, on
the same seeded inputs. Tolerance: relative L2 error <= 1e-11 per band (BASELINE.json north_star); index maps
bit-exact. PAPER.md:L105, L224-226, L176 (vi); readings in DESIGN.md section 3."""
import numpy as np
import pytest
import torch

from oracle import hpsi_oracle as orc
from paper_2104_10502_b200 import harness, inputs, qe_hpsi
from tests import _gpu

pytestmark = pytest.mark.gpu
TOL = 1e-11
TINY = ["T1_general_k", "T2_radix5", "T2b_radix5_20", "T3_aliased", "T4_noproj", "T5_odd_bands"]


@pytest.mark.parametrize("cfg", TINY + [0, 1, 2, 3, 4])
def test_maps_bit_exact(cfg):
    wl = inputs.get_workload(cfg)
    sp = _gpu.oracle_sphere(wl)
    mil = qe_hpsi.qe_hpsi_gsphere(wl.at, wl.xk, wl.ecutwfc, wl.nr)
    assert mil.dtype == np.int32 and np.array_equal(mil, sp["miller"])
    vr = torch.zeros(tuple(wl.nr), dtype=torch.float64, device="cuda")
    h = qe_hpsi.Hpsi(wl.at, wl.ecutwfc, wl.xk, wl.nr, vr, max_batch=1)
    m2, idx, g2 = h.maps()
    assert np.array_equal(m2.cpu().numpy(), sp["miller"])
    assert np.array_equal(idx.cpu().numpy(), sp["fft_index"])
    assert np.array_equal(g2.cpu().numpy().view(np.int64), sp["g2kin"].view(np.int64)), "g2kin must match bit for bit"
    info = h.info()
    n3 = wl.nr[2]
    assert info["S"] == np.unique(sp["fft_index"].astype(np.int64) // n3).size
    assert info["P"] == np.unique(sp["fft_index"].astype(np.int64) // (n3 * wl.nr[1])).size
    h.destroy()


@pytest.mark.parametrize("flags", [0, qe_hpsi.QE_HPSI_GENERIC_FFT, qe_hpsi.QE_HPSI_FP64_DMMA, _gpu.INT8, _gpu.INT8_S7])
@pytest.mark.parametrize("cfg", TINY + [0])
def test_small_cases_against_dense_h(cfg, flags):
    """Level A (dense H from the definition) on every tiny case and config 0; both radix plans."""
    h, inp = _gpu.make(cfg, flags=flags)
    wl = inp["wl"]
    sp = _gpu.oracle_sphere(wl)
    npw = h.npw
    psi = _gpu.gen_psi_dev(inp, 0, wl.nbands)
    hpsi = torch.full_like(psi, 7.0)  # sentinel: pad columns must stay untouched, the rest overwritten
    h.apply(psi, hpsi)
    torch.cuda.synchronize()
    beta = inp["beta"][:, :npw].cpu().numpy() if wl.nproj else None
    hd = orc.dense_h(sp["miller"], sp["g2kin"], tuple(wl.nr), inp["vr"].cpu().numpy(), beta, inp["dblocks"])
    ref = orc.hpsi_dense(hd, psi[:, :npw].cpu().numpy())
    got = hpsi.cpu().numpy()
    err = _gpu.rel_l2(got[:, :npw], ref)
    assert err.max() <= TOL, err
    assert np.all(got[:, npw:] == 7.0)
    h.destroy()


@pytest.mark.parametrize("cfg", ["T1_general_k", "T5_odd_bands", 0])
def test_stages_local_and_becp(cfg):
    h, inp = _gpu.make(cfg)
    wl = inp["wl"]
    sp = _gpu.oracle_sphere(wl)
    npw = h.npw
    psi = _gpu.gen_psi_dev(inp, 0, wl.nbands)
    ph = psi[:, :npw].cpu().numpy()
    loc_ref, vnl_ref = _gpu.oracle_hpsi(inp, sp, ph, parts=True)
    loc = h.fft_local(psi)
    torch.cuda.synchronize()
    assert _gpu.rel_l2(loc.cpu().numpy()[:, :npw], loc_ref).max() <= TOL
    out = h.nonlocal_add(psi, loc.clone())
    becp, dbecp = h.becp(wl.nbands)
    torch.cuda.synchronize()
    beta = inp["beta"][:, :npw].cpu().numpy()
    bref = orc.becp_of(beta, ph)
    assert np.abs(becp.cpu().numpy() - bref).max() <= 1e-13 * max(1.0, np.abs(bref).max())
    dref = orc.dbecp_of(inp["dblocks"], bref)
    assert np.abs(dbecp.cpu().numpy() - dref).max() <= 1e-13 * max(1.0, np.abs(dref).max())
    assert _gpu.rel_l2(out.cpu().numpy()[:, :npw], loc_ref + vnl_ref).max() <= TOL
    h.destroy()


def test_closed_form_plane_wave_in_constant_potential():
    """north_star invariant straight on the GPU path: psi = delta_G0, V = V0 -> (|k+G0|^2 + V0) delta."""
    wl = inputs.get_workload(0)
    v0 = 0.625
    vr = torch.full(tuple(wl.nr), v0, dtype=torch.float64, device="cuda")
    h = qe_hpsi.Hpsi(wl.at, wl.ecutwfc, wl.xk, wl.nr, vr, max_batch=4)
    _, _, g2 = h.maps()
    npw = h.npw
    picks = [0, 1, npw // 2, npw - 1]
    psi = torch.zeros((4, npw), dtype=torch.complex128, device="cuda")
    for b, g in enumerate(picks):
        psi[b, g] = 1.0 - 0.5j
    out = h.apply(psi)
    ref = torch.zeros_like(psi)
    for b, g in enumerate(picks):
        ref[b, g] = (g2[g] + v0) * psi[b, g]
    assert float((out - ref).abs().max()) <= 1e-13
    h.destroy()


def test_batch_composition_and_chunking_do_not_change_bits():
    """A band's result must not depend on which other bands share the call (reading 13)."""
    h, inp = _gpu.make(0, max_batch=5)  # 16 bands -> chunks 5,5,5,1
    psi = _gpu.gen_psi_dev(inp, 0, 16)
    full = h.apply(psi).clone()
    one = torch.stack([h.apply(psi[b:b + 1].contiguous())[0] for b in (0, 7, 15)])
    torch.cuda.synchronize()
    assert torch.equal(full[[0, 7, 15]].view(torch.float64), one.view(torch.float64))
    h.destroy()


@pytest.mark.parametrize("path", ["fp64", "fp64_general", "int8_s7", "int8_s6", "int8_s6_cert"])
def test_config1_all_bands(path):
    h, inp = _gpu.make(1, flags=_gpu.PATHS[path])
    wl = inp["wl"]
    sp = _gpu.oracle_sphere(wl)
    psi = _gpu.gen_psi_dev(inp, 0, wl.nbands)
    out = h.apply(psi)
    vnl = h.nonlocal_add(psi, torch.zeros_like(psi))
    torch.cuda.synchronize()
    loc_ref, vnl_ref = _gpu.oracle_hpsi(inp, sp, psi[:, :h.npw].cpu().numpy(), parts=True)
    ref = loc_ref + vnl_ref
    err = _gpu.rel_l2(out.cpu().numpy()[:, :h.npw], ref)
    assert err.max() <= TOL, err.max()
    evnl = _gpu.rel_l2(vnl.cpu().numpy()[:, :h.npw], vnl_ref)
    assert evnl.max() <= _gpu.TOL_VNL[path], f"config 1 {path}: nonlocal part alone {evnl.max():.2e}"
    # Level A' (definition, sampled rows) at full scale, no FFT of psi involved
    rows = inputs.aux_choice(wl.seed, 3, h.npw, 16)
    bands = [0, 63, 127]
    vt = orc.vloc_coeffs(inp["vr"].cpu().numpy())
    beta = inp["beta"][:, :h.npw].cpu().numpy()
    ap = orc.hpsi_rows(rows, sp["miller"], sp["g2kin"], tuple(wl.nr), vt, psi[bands, :h.npw].cpu().numpy(), beta,
                       inp["dblocks"])
    got = out.cpu().numpy()[bands][:, rows]
    assert np.abs(got - ap).max() <= 1e-12 * np.abs(ref).max()
    h.destroy()


def _sample_bands(wl):
    """First and last band of every `batch`-band call plus 8 seeded random bands (SURVEY.md 8(c) pin table)."""
    s = set()
    for b0 in range(0, wl.nbands, wl.batch):
        s.add(b0)
        s.add(min(wl.nbands, b0 + wl.batch) - 1)
    s.update(int(x) for x in inputs.aux_choice(wl.seed, 7, wl.nbands, 8))
    return sorted(s)


@pytest.mark.parametrize("cfg", [2, 3, 4])
def test_full_size_against_oracle_every_projector_path(cfg):
    """BASELINE.json's full sizes in the launch configuration bench.py times (calls of `batch` bands, beta borrowed), ALL
    bands applied, for each projector path (FP64 default, FP64 with the general contraction, int8 S = 7, int8 S = 6):
      * sampled bands (first + last of every call, 8 random): H psi against oracle Level B, and the NONLOCAL PART ALONE
        (qe_hpsi_nonlocal on zeros) against the oracle's nonlocal part -- it is ~1e-5 of |H psi| here, so only this isolates
        a6 / a8 at their full-size shapes (23-37 K splits, 64 K blocks x 3 planes); becp of the sampled bands against orc.becp_of;
      * every band: Hermitian probes <phi|H psi_b> = <H phi|psi_b> and <phi|V_NL psi_b> = <V_NL phi|psi_b>;
      * Level A' (the definition, sampled rows, no FFT of psi) with becp accumulated over atom chunks.
    The oracle runs once per config (beta streamed device -> host in atom chunks)."""
    wl = inputs.get_workload(cfg)
    sample = _sample_bands(wl)
    shared = {}
    report = {}
    for path, pflags in _gpu.PATHS.items():
        if path == "fp64_general" and any(x != 0.0 for x in wl.xk):
            continue  # at k != 0 the default FP64 path is the general contraction already
        h, inp = _gpu.make(cfg, flags=qe_hpsi.QE_HPSI_BORROW_BETA | pflags, beta=shared.get("beta"))
        assert h.info()["gamma_sym"] == (0 if path == "fp64_general" or any(x != 0.0 for x in wl.xk) else 1)
        npw = h.npw
        if not shared:
            shared["beta"] = inp["beta"]
            sp = _gpu.oracle_sphere(wl)
            psi_s = torch.cat([_gpu.gen_psi_dev(inp, b, 1) for b in sample])[:, :npw].cpu().numpy()
            phi = inputs.aux_normal_complex(wl.seed, 99, npw).numpy()
            phi /= np.linalg.norm(phi)
            loc_ref, vnl_ref, becp_ref = _gpu.oracle_hpsi(inp, sp, np.concatenate([psi_s, phi[None]]), want_becp=True)
            shared.update(sp=sp, psi_s=psi_s, phi=phi, loc=loc_ref, vnl=vnl_ref, becp=becp_ref)
        sp, phi = shared["sp"], shared["phi"]
        loc_ref, vnl_ref, becp_ref = shared["loc"], shared["vnl"], shared["becp"]
        phi_d = torch.as_tensor(phi, device="cuda")
        hphi_d = torch.as_tensor(loc_ref[-1] + vnl_ref[-1], device="cuda")
        vphi_d = torch.as_tensor(vnl_ref[-1], device="cuda")
        got_h, got_v, got_b = {}, {}, {}
        herm = herm_v = 0.0
        scale_h = scale_v = 0.0
        for b0 in range(0, wl.nbands, wl.batch):  # exactly bench.py's calls
            n = min(wl.batch, wl.nbands - b0)
            psi = _gpu.gen_psi_dev(inp, b0, n)
            out = h.apply(psi)
            vnl = h.nonlocal_add(psi, torch.zeros_like(psi))
            becp, _ = h.becp(n)
            torch.cuda.synchronize()
            for b in sample:
                if b0 <= b < b0 + n:
                    got_h[b] = out[b - b0, :npw].cpu().numpy()
                    got_v[b] = vnl[b - b0, :npw].cpu().numpy()
                    got_b[b] = becp[:, b - b0].cpu().numpy()
            herm = max(herm, float(((phi_d.conj()[None] * out[:, :npw]).sum(1) - (hphi_d.conj()[None] * psi[:, :npw]).sum(1)).abs().max()))
            herm_v = max(herm_v, float(((phi_d.conj()[None] * vnl[:, :npw]).sum(1) - (vphi_d.conj()[None] * psi[:, :npw]).sum(1)).abs().max()))
            scale_h = max(scale_h, float(torch.linalg.vector_norm(out[:, :npw], dim=1).max()))
            scale_v = max(scale_v, float(torch.linalg.vector_norm(vnl[:, :npw], dim=1).max()))
            del psi, out, vnl, becp
        eh = _gpu.rel_l2(np.stack([got_h[b] for b in sample]), loc_ref[:-1] + vnl_ref[:-1])
        ev = _gpu.rel_l2(np.stack([got_v[b] for b in sample]), vnl_ref[:-1])
        gb = np.stack([got_b[b] for b in sample], 1)
        eb = np.abs(gb - becp_ref[:, :-1]).max() / np.abs(becp_ref[:, :-1]).max()
        report[path] = dict(hpsi=eh.max(), vnl=ev.max(), becp=eb, herm=herm / scale_h, herm_vnl=herm_v / scale_v)
        msg = f"config {cfg} {path}: " + ", ".join(f"{k} {v:.2e}" for k, v in report[path].items())
        print(msg)
        assert eh.max() <= TOL, msg
        assert ev.max() <= _gpu.TOL_VNL[path], msg
        assert eb <= _gpu.TOL_BECP[path], msg
        assert herm <= 1e-11 * scale_h, msg
        assert herm_v <= _gpu.TOL_VNL[path] * 10 * scale_v, msg  # a dot product with a unit vector: same scale as the L2 error
        if path == "fp64":  # Level A' on the FP64 result (the other paths are within TOL of it by the assertions above)
            rows = inputs.aux_choice(wl.seed, 3, npw, 16)
            vt = orc.vloc_coeffs(inp["vr"].cpu().numpy())
            bcols = inp["beta"][:, torch.as_tensor(rows, device="cuda")].cpu().numpy()
            ap = orc.hpsi_rows(rows, sp["miller"], sp["g2kin"], tuple(wl.nr), vt, shared["psi_s"][:3], bcols, inp["dblocks"],
                               becp=becp_ref[:, :3])
            got = np.stack([got_h[b] for b in sample[:3]])[:, rows]
            ea = np.abs(got - ap).max() / np.abs(loc_ref[:3]).max()
            assert ea <= 1e-12, f"config {cfg}: Level A' rows {ea:.2e}"
        h.destroy()
        del h
        torch.cuda.empty_cache()


@pytest.mark.parametrize("flags", [0, _gpu.INT8, _gpu.INT8_S7, harness.int8_flags(6, three_m=3, certify=True)])
@pytest.mark.parametrize("cfg", ["T1_general_k", "T5_odd_bands", 0])
def test_apply_writes_nothing_outside_its_output_rows(cfg, flags):
    """Caller-side guard bands: hpsi is a window in the middle of a sentinel-filled allocation (guard rows before and after,
    pad columns inside); after apply / nonlocal / apply_host-style chunking every byte outside [b][0..npw) is untouched.
    (The handle's own workspaces carry guard bands too, verified at destroy: tests/conftest.py.)"""
    h, inp = _gpu.make(cfg, flags=flags, max_batch=5)
    wl = inp["wl"]
    npw, nb = h.npw, wl.nbands
    ld = inp["ld"] + 8  # a row stride larger than the generator's
    psi = torch.zeros((nb, ld), dtype=torch.complex128, device="cuda")
    psi[:, :inp["ld"]] = _gpu.gen_psi_dev(inp, 0, nb)
    guard = 3
    buf = torch.full((nb + 2 * guard, ld), complex(7.0, -7.0), dtype=torch.complex128, device="cuda")
    win = buf[guard:guard + nb]
    h.apply(psi, win)
    h.nonlocal_add(psi, win)
    torch.cuda.synchronize()
    host = buf.cpu().numpy()
    assert np.all(host[:guard] == complex(7.0, -7.0)) and np.all(host[guard + nb:] == complex(7.0, -7.0))
    assert np.all(host[guard:guard + nb, npw:] == complex(7.0, -7.0))
    assert np.isfinite(host[guard:guard + nb, :npw]).all() and not np.any(host[guard:guard + nb, :npw] == complex(7.0, -7.0))
    assert h.check_guards() == 0
    h.destroy()


def test_gamma_symmetric_projector_mode_is_detected_and_matches_the_general_contraction():
    """At k = 0 the FP64 path contracts psi = u + i v over the half sphere when EVERY projector passes the bit-exact check
    beta(-G) = +-conj beta(G) and D couples equal signs only; otherwise it must fall back. Both against the oracle
    (the other tests) and against the general complex contraction (here, nonlocal part alone)."""
    for cfg, want in (("T1_general_k", 0), ("T5_odd_bands", 0), ("T2_radix5", 1), ("T2b_radix5_20", 1), ("T3_aliased", 1), (0, 1), (1, 1)):
        h, inp = _gpu.make(cfg)
        assert h.info()["gamma_sym"] == want, cfg
        wl = inp["wl"]
        if not want:
            h.destroy()
            continue
        hg, _ = _gpu.make(cfg, flags=qe_hpsi.QE_HPSI_NO_GAMMA_SYM, beta=inp["beta"])
        assert hg.info()["gamma_sym"] == 0
        npw = h.npw
        psi = _gpu.gen_psi_dev(inp, 0, min(wl.nbands, 37))
        a = h.nonlocal_add(psi, torch.zeros_like(psi))
        b = hg.nonlocal_add(psi, torch.zeros_like(psi))
        ba, _ = h.becp(psi.shape[0]) if psi.shape[0] <= h.max_batch else (None, None)
        torch.cuda.synchronize()
        d = torch.linalg.vector_norm(a[:, :npw] - b[:, :npw], dim=1) / torch.linalg.vector_norm(b[:, :npw], dim=1)
        assert float(d.max()) <= 1e-13, (cfg, float(d.max()))
        assert torch.equal(a[:, npw:], torch.zeros_like(a[:, npw:]))
        assert h.launch_count(1) == 5 + 6 and hg.launch_count(1) == 5 + 4
        h.destroy()
        hg.destroy()
    # a projector set WITHOUT the symmetry (one entry nudged by one ulp) and a D that couples s with p: the general path, still right
    h0, inp = _gpu.make(0)
    wl = inp["wl"]
    sp = _gpu.oracle_sphere(wl)
    npw = h0.npw
    h0.destroy()
    beta = inp["beta"].clone()
    beta[3, 11] = torch.nextafter(beta[3, 11].real, torch.tensor(2.0, dtype=torch.float64, device="cuda")) + 1j * beta[3, 11].imag
    psi = _gpu.gen_psi_dev(inp, 0, wl.nbands)
    h1 = qe_hpsi.Hpsi(wl.at, wl.ecutwfc, wl.xk, wl.nr, inp["vr"], beta, inp["blk"], inp["dblocks"], max_batch=wl.batch)
    assert h1.info()["gamma_sym"] == 0
    ref = orc.vnl_psi(beta[:, :npw].cpu().numpy(), inp["dblocks"], psi[:, :npw].cpu().numpy())
    assert _gpu.rel_l2(h1.nonlocal_add(psi, torch.zeros_like(psi)).cpu().numpy()[:, :npw], ref).max() <= 1e-12
    h1.destroy()
    dmix = np.array(inp["dblocks"], dtype=np.float64).copy()
    dmix[:, 0, 1] = dmix[:, 1, 0] = 0.37  # config 0 orders [s; px, py, pz]: couples l = 0 with l = 1 (classes 0 and 1)
    h2 = qe_hpsi.Hpsi(wl.at, wl.ecutwfc, wl.xk, wl.nr, inp["vr"], inp["beta"], inp["blk"], dmix, max_batch=wl.batch)
    assert h2.info()["gamma_sym"] == 0
    ref = orc.vnl_psi(inp["beta"][:, :npw].cpu().numpy(), dmix, psi[:, :npw].cpu().numpy())
    assert _gpu.rel_l2(h2.nonlocal_add(psi, torch.zeros_like(psi)).cpu().numpy()[:, :npw], ref).max() <= 1e-12
    h2.destroy()
    # both classes really occur in the generator's projectors (s: +, p: -), so the i*beta rows are exercised
    h3, _ = _gpu.make(0)
    assert h3.info()["gamma_sym"] == 1
    h3.destroy()
    # outside the tests the mode starts at 2^20 entries of beta (config 0 has 17 k: launch-latency bound, general form)
    qe_hpsi.qe_hpsi_test_set_sym_min(-1)
    try:
        h4, _ = _gpu.make(0)
        h5, _ = _gpu.make(1)
        assert h4.info()["gamma_sym"] == 0 and h5.info()["gamma_sym"] == 1
        h4.destroy()
        h5.destroy()
    finally:
        qe_hpsi.qe_hpsi_test_set_sym_min(0)


@pytest.mark.parametrize("cfg,nb", [("T2_radix5", 3), ("T3_aliased", 5), (0, 16), (1, 37), (1, 64)])
def test_tma_fed_symmetric_kernels_give_the_bits_of_the_cp_async_ones(cfg, nb, monkeypatch):
    """zgemm_tma_kernels.cuh moves the operand tiles of the Gamma-symmetric FP64 a6 / a8 by TMA; tiles, DMMA order and epilogues
    are those of k_becp / k_vnl_add, so becp and the nonlocal part must be bit-identical (ragged K tail, row tail, column
    tail, and a second call with fewer bands over stale workspace columns)."""
    h, inp = _gpu.make(cfg)
    assert h.info()["gamma_sym"] == 1
    monkeypatch.setenv("QE_HPSI_SYM_TMA", "0")
    h0, _ = _gpu.make(cfg, beta=inp["beta"])
    monkeypatch.delenv("QE_HPSI_SYM_TMA")
    nb = min(nb, h.max_batch)
    for band0, n in ((0, nb), (50, max(1, nb // 2))):
        psi = _gpu.gen_psi_dev(inp, band0, n)
        base = _gpu.gen_psi_dev(inp, 200, n)
        a = h.nonlocal_add(psi, base.clone())
        ba, da = h.becp(n)
        b = h0.nonlocal_add(psi, base.clone())
        bb, db = h0.becp(n)
        torch.cuda.synchronize()
        assert torch.equal(ba.view(torch.float64), bb.view(torch.float64))
        assert torch.equal(da.view(torch.float64), db.view(torch.float64))
        assert torch.equal(a.view(torch.float64), b.view(torch.float64))
        assert not torch.equal(a, base)
    h.destroy()
    h0.destroy()


@pytest.mark.parametrize("cfg,nb", [("T1_general_k", 5), ("T5_odd_bands", 3), ("T3_aliased", 5), (0, 16), (1, 37), (3, 24)])
def test_tma_fed_general_kernels_give_the_bits_of_the_cp_async_ones(cfg, nb, monkeypatch):
    """The general complex a6 / a8 (3M form; k != 0 or QE_HPSI_NO_GAMMA_SYM) with TMA operand tiles against the cp.async
    kernels: becp, dbecp and the nonlocal part bit for bit, on two calls with different band counts."""
    flags = qe_hpsi.QE_HPSI_NO_GAMMA_SYM
    h, inp = _gpu.make(cfg, flags=flags)
    monkeypatch.setenv("QE_HPSI_ZG_TMA", "0")
    h0, _ = _gpu.make(cfg, flags=flags, beta=inp["beta"])
    monkeypatch.delenv("QE_HPSI_ZG_TMA")
    nb = min(nb, h.max_batch)
    for band0, n in ((0, nb), (50, max(1, nb // 2))):
        psi = _gpu.gen_psi_dev(inp, band0, n)
        base = _gpu.gen_psi_dev(inp, 200, n)
        a = h.nonlocal_add(psi, base.clone())
        ba, da = h.becp(n)
        b = h0.nonlocal_add(psi, base.clone())
        bb, db = h0.becp(n)
        torch.cuda.synchronize()
        assert torch.equal(ba.view(torch.float64), bb.view(torch.float64))
        assert torch.equal(da.view(torch.float64), db.view(torch.float64))
        assert torch.equal(a.view(torch.float64), b.view(torch.float64))
        assert not torch.equal(a, base)
    h.destroy()
    h0.destroy()


@pytest.mark.parametrize("cfg", ["T2_radix5", "T1_general_k", 0])
@pytest.mark.parametrize("dmode", ["diag", "full"])
def test_ragged_projector_blocks_and_tails(cfg, dmode):
    """13 projectors in blocks of 5 and 8 (K tail of the 16-projector tiles, ldp padding, a ragged class mask), 5 bands: the
    nonlocal part alone against becp_of / the block-diagonal D written out.  diag D keeps the Gamma-symmetric form at k = 0,
    a full random block couples s with p and must take the general contraction."""
    import scipy.linalg
    h0, inp = _gpu.make(cfg)
    wl = inp["wl"]
    npw = h0.npw
    h0.destroy()
    if wl.nproj < 13:  # 8 rows: 5 more as combinations of rows of equal parity (s with s, p with p), so the symmetry classes stay exact
        ia, ib = ([0, 1, 2, 3, 4], [1, 0, 3, 4, 2]) if wl.nh == 8 else ([0, 4, 1, 2, 3], [4, 0, 2, 3, 1])
        beta = torch.cat([inp["beta"], inp["beta"][ia] * 0.7 + inp["beta"][ib] * 0.4]).contiguous()
        assert beta.shape[0] == 13
    else:
        beta = inp["beta"][:13].contiguous()
    rng = np.random.default_rng(11)
    blocks = []
    for n in (5, 8):
        d = rng.standard_normal((n, n))
        blocks.append(np.diag(np.diag(d)) if dmode == "diag" else (d + d.T) / 2)
    h = qe_hpsi.Hpsi(wl.at, wl.ecutwfc, wl.xk, wl.nr, inp["vr"], beta, [0, 5, 13], blocks, max_batch=5)
    k0 = all(x == 0.0 for x in wl.xk)
    assert h.info()["gamma_sym"] == (1 if (k0 and dmode == "diag") else 0)
    psi = _gpu.gen_psi_dev(inp, 0, 5)
    got = h.nonlocal_add(psi, torch.zeros_like(psi))
    ba, da = h.becp(5)
    torch.cuda.synchronize()
    bh, ph = beta[:, :npw].cpu().numpy(), psi[:, :npw].cpu().numpy()
    becp = orc.becp_of(bh, ph)
    dbecp = scipy.linalg.block_diag(*blocks) @ becp
    ref = (bh.T @ dbecp).T
    assert np.abs(ba.cpu().numpy() - becp).max() <= 1e-13 * np.abs(becp).max()
    assert np.abs(da.cpu().numpy() - dbecp).max() <= 1e-13 * np.abs(dbecp).max()
    assert _gpu.rel_l2(got.cpu().numpy()[:, :npw], ref).max() <= 1e-12
    assert torch.equal(got[:, npw:], torch.zeros_like(got[:, npw:]))
    h.destroy()


def test_apply_host_matches_device_path():
    h, inp = _gpu.make(0, max_batch=6)
    psi = _gpu.gen_psi_dev(inp, 0, 16)
    dev = h.apply(psi).cpu()
    ph = psi.cpu().pin_memory()
    hh = torch.zeros_like(ph).pin_memory()
    h.apply_host(ph, hh)
    assert torch.equal(hh[:, :h.npw].view(torch.float64), dev[:, :h.npw].view(torch.float64))
    h.destroy()


def test_argument_errors():
    wl = inputs.get_workload("T2_radix5")
    vr = torch.zeros(tuple(wl.nr), dtype=torch.float64, device="cuda")
    with pytest.raises(qe_hpsi.QeHpsiError) as e:
        qe_hpsi.Hpsi(wl.at, wl.ecutwfc, wl.xk, (14, 15, 15), torch.zeros((14, 15, 15), dtype=torch.float64, device="cuda"))
    assert e.value.status == qe_hpsi.QE_HPSI_EGRID  # 14 = 2*7
    with pytest.raises(qe_hpsi.QeHpsiError) as e:
        qe_hpsi.Hpsi(wl.at, wl.ecutwfc, wl.xk, (5, 15, 15), torch.zeros((5, 15, 15), dtype=torch.float64, device="cuda"))
    assert e.value.status == qe_hpsi.QE_HPSI_EGRID  # sphere wider than the box
    h = qe_hpsi.Hpsi(wl.at, wl.ecutwfc, wl.xk, wl.nr, vr, max_batch=2)
    psi = torch.zeros((2, h.npw), dtype=torch.complex128, device="cuda")
    with pytest.raises(qe_hpsi.QeHpsiError) as e:
        h.apply(psi, psi)  # aliasing
    assert e.value.status == qe_hpsi.QE_HPSI_EINVAL
    with pytest.raises(qe_hpsi.QeHpsiError) as e:
        h.apply(psi[:, :h.npw - 1].contiguous())  # ld < npw
    assert e.value.status == qe_hpsi.QE_HPSI_EINVAL
    out = h.apply(torch.zeros((0, h.npw), dtype=torch.complex128, device="cuda"))  # empty input is fine
    assert out.shape[0] == 0
    # a complex128 array that is only 8-byte aligned (a view into a float64 buffer at an odd offset)
    import ctypes
    big = torch.zeros((3, h.npw + 8), dtype=torch.complex128, device="cuda")
    out2 = torch.zeros_like(big)
    lib = qe_hpsi.load_library()
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    rc = lib.qe_hpsi_apply(h._h, ctypes.c_void_p(big.data_ptr() + 8), h.npw + 8, ctypes.c_void_p(out2.data_ptr()), h.npw + 8, 2, st)
    assert rc == qe_hpsi.QE_HPSI_EINVAL
    rc = lib.qe_hpsi_apply(h._h, ctypes.c_void_p(big.data_ptr()), h.npw + 8, ctypes.c_void_p(out2.data_ptr() + 8), h.npw + 8, 2, st)
    assert rc == qe_hpsi.QE_HPSI_EINVAL
    h.destroy()


# every FFT length with a fast-path plan (two-pass: fft2p_kernels.cuh, three-pass: fft3p_kernels.cuh) plus a few
# lengths that only the generic multi-pass plan serves, each placed on each of the three axes in turn
FFT2P_LENGTHS = [8, 9, 10, 12, 15, 16, 18, 20, 36, 48, 64, 72, 80, 96, 100, 108, 120, 128, 144, 160, 180, 192, 240, 256]
FFT3P_LENGTHS = [125, 150, 200, 216, 250, 288, 300, 320, 360, 384]
GENERIC_LENGTHS = [24, 45, 135, 243]


@pytest.mark.parametrize("n", FFT2P_LENGTHS + FFT3P_LENGTHS + GENERIC_LENGTHS)
def test_local_term_for_every_fft_length(n):
    """Local + kinetic term (nproj = 0) on anisotropic cells whose grid is (n, 9, 10), (9, n, 10), (9, 10, n) with the
    sphere using the full index range of every axis, against oracle Level B on the same arrays."""
    ecut = 4.0
    gen = torch.Generator().manual_seed(1000 + n)
    for axis in range(3):
        nr = [9, 10, 12][axis:] + [9, 10, 12][:axis]
        nr = [nr[0], nr[1], nr[2]]
        nr[axis] = n
        at = np.zeros((3, 3))
        for j in range(3):
            nmax = (nr[j] - 1) // 2
            at[j, j] = 2.0 * np.pi * (nmax + 0.4) / np.sqrt(ecut)
        xk = np.array([0.0, 0.0, 0.0]) if axis == 0 else 0.02 * 2 * np.pi / at.diagonal() * np.array([1.0, -2.0, 1.5])
        sp = orc.gsphere(at, xk, ecut, nr)
        npw = sp["miller"].shape[0]
        assert npw > 0
        vr = torch.randn(tuple(nr), dtype=torch.float64, generator=gen)
        nb = 3
        ld = inputs.pad8(npw)
        psi = torch.zeros((nb, ld), dtype=torch.complex128)
        psi[:, :npw] = torch.randn((nb, npw), dtype=torch.complex128, generator=gen)
        h = qe_hpsi.Hpsi(at, ecut, xk, nr, vr.cuda(), max_batch=2)  # 3 bands through chunks of 2 and 1
        assert h.npw == npw
        out = h.apply(psi.cuda())
        torch.cuda.synchronize()
        ref = orc.hpsi_dual(sp["fft_index"], sp["g2kin"], tuple(nr), vr.numpy(), psi[:, :npw].numpy(), None, None)
        err = _gpu.rel_l2(out.cpu().numpy()[:, :npw], ref)
        assert err.max() <= TOL, (n, axis, nr, err)
        h.destroy()


@pytest.mark.parametrize("n", [48, 64, 96, 108, 120, 128, 144, 160, 192, 240, 256])
def test_x_stage_quarter_pruning(n, monkeypatch):
    """Grids that hold the sphere twice over along x (x_hi < N1 / 4, the density-grid rule): the x stage skips the known-zero
    half of its radix-RA inputs and the unused half of its outputs (k2t_x_vmul<RA, RB, HALF>).  Local + kinetic term against
    oracle Level B, and against the unpruned kernel (same sums up to the sign of an exact zero)."""
    ecut = 4.0
    gen = torch.Generator().manual_seed(2000 + n)
    nr = [n, 9, 10]
    at = np.zeros((3, 3))
    for j in range(3):
        nmax = (nr[j] // 4 - 1) if j == 0 else (nr[j] - 1) // 2
        at[j, j] = 2.0 * np.pi * (nmax + 0.4) / np.sqrt(ecut)
    xk = np.zeros(3)
    sp = orc.gsphere(at, xk, ecut, nr)
    npw = sp["miller"].shape[0]
    assert np.abs(sp["miller"][:, 0]).max() == n // 4 - 1
    vr = torch.randn(tuple(nr), dtype=torch.float64, generator=gen)
    nb = 3
    psi = torch.zeros((nb, inputs.pad8(npw)), dtype=torch.complex128)
    psi[:, :npw] = torch.randn((nb, npw), dtype=torch.complex128, generator=gen)
    h = qe_hpsi.Hpsi(at, ecut, xk, nr, vr.cuda(), max_batch=2)
    assert h.info()["x_half"] == 1
    out = h.apply(psi.cuda())
    monkeypatch.setenv("QE_HPSI_X_HALF", "0")
    h0 = qe_hpsi.Hpsi(at, ecut, xk, nr, vr.cuda(), max_batch=2)
    monkeypatch.delenv("QE_HPSI_X_HALF")
    assert h0.info()["x_half"] == 0
    out0 = h0.apply(psi.cuda())
    torch.cuda.synchronize()
    ref = orc.hpsi_dual(sp["fft_index"], sp["g2kin"], tuple(nr), vr.numpy(), psi[:, :npw].numpy(), None, None)
    assert _gpu.rel_l2(out.cpu().numpy()[:, :npw], ref).max() <= TOL
    assert _gpu.rel_l2(out.cpu().numpy()[:, :npw], out0.cpu().numpy()[:, :npw]).max() <= 1e-15
    # the density kernel shares the pruned inverse pass (k2t_x_rho<RA, RB, HALF>)
    occ = torch.tensor([2.0, 1.0, 0.5], dtype=torch.float64, device="cuda")
    rho = torch.full(tuple(nr), 0.25, dtype=torch.float64, device="cuda")
    h.density(psi.cuda(), occ, 0.5, rho)
    torch.cuda.synchronize()
    rref = 0.25 + orc.density_of(sp["fft_index"], tuple(nr), psi[:, :npw].numpy(), occ.cpu().numpy(), 0.5)
    assert np.abs(rho.cpu().numpy() - rref).max() <= 1e-12 * np.abs(rref).max()
    h.destroy()
    h0.destroy()


def test_handles_created_and_applied_from_two_host_threads():
    """Two host threads, each with its own stream and handle (per-device kernel attributes under a mutex, the tensor-map
    encoder looked up once, maps of psi encoded per call): same bits as the single-threaded result."""
    import threading
    h0, inp = _gpu.make(1)
    psi = _gpu.gen_psi_dev(inp, 0, 24)
    ref = h0.apply(psi).clone()
    torch.cuda.synchronize()
    h0.destroy()
    results, errors = {}, []

    def work(tag, flags):
        try:
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                for _ in range(3):
                    h, _ = _gpu.make(1, flags=flags, beta=inp["beta"])
                    out = h.apply(psi)
                    st.synchronize()
                    h.destroy()
                results[tag] = out
        except Exception as e:  # noqa: BLE001
            errors.append((tag, repr(e)))

    ts = [threading.Thread(target=work, args=("sym", 0)), threading.Thread(target=work, args=("gen", qe_hpsi.QE_HPSI_NO_GAMMA_SYM))]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not errors, errors
    assert torch.equal(results["sym"].view(torch.float64), ref.view(torch.float64))
    npw = inp["miller"].shape[0]
    assert _gpu.rel_l2(results["gen"].cpu().numpy()[:, :npw], ref.cpu().numpy()[:, :npw]).max() <= 1e-13


def test_apply_can_be_captured_in_a_cuda_graph():
    """qe_hpsi_apply enqueues kernels only (no allocation, no host sync): it can be stream-captured and replayed, which
    is how a launch-latency-bound caller (config 0: 9 launches for 16 bands) should drive it. Replays must reproduce the
    eager result bit for bit, also after psi is overwritten in place."""
    h, inp = _gpu.make(0)
    wl = inp["wl"]
    npw = h.npw
    psi = _gpu.gen_psi_dev(inp, 0, wl.nbands)
    ref1 = h.apply(psi).clone()
    psi2 = _gpu.gen_psi_dev(inp, 50, wl.nbands)
    ref2 = h.apply(psi2).clone()
    torch.cuda.synchronize()
    buf = psi.clone()
    out = torch.zeros_like(buf)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        h.apply(buf, out, side)  # warm-up on the capture stream
    torch.cuda.current_stream().wait_stream(side)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        h.apply(buf, out, torch.cuda.current_stream())
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out[:, :npw].view(torch.float64), ref1[:, :npw].view(torch.float64))
    buf.copy_(psi2)
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out[:, :npw].view(torch.float64), ref2[:, :npw].view(torch.float64))
    del g
    h.destroy()
