#!/usr/bin/env python
"""bench.py -- H|psi> band-applications/s on B200 (BASELINE.json metric), with roofline and CPU-oracle baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path (a1-a8) over all `nbands` bands of the workload, applied in calls of
`batch` bands (config 4: 1024 bands as 8 calls of 128). `value` = bands/s with psi/hpsi resident in HBM; `e2e` =
the same through qe_hpsi_apply_host with pinned HOST buffers (H2D of psi and D2H of hpsi inside the timed region).
Default workload: config 4 (the configuration north_star's target is quoted on; fits one GPU). Inputs are seeded
synthetic data. N > 1 (torchrun): every rank runs the same workload on its own bands
(k-point-pool style sharding, no data-path collective): weak scaling, max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "hpsi_band_applications_per_s"
UNIT = "bands/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--detail", action="store_true", help="extra pass with per-FFT-kernel events (stderr table)")
    ap.add_argument("--graph", type=int, default=-1, help="replay the step from a CUDA graph: 1 on, 0 off, -1 (default) only "
                    "for launch-latency-bound workloads (a step under 0.5 ms); stage timers are taken in a separate eager pass")
    ap.add_argument("--dmma", action="store_true", help="projector contractions on the FP64 tensor pipe (create flag "
                    "QE_HPSI_FP64_DMMA) instead of the default int8 digit path")
    ap.add_argument("--next", action="store_true", help="also time the SURVEY 8(f) rows (apply_hs, overlap, density): "
                    "adds a next_rows object to the JSON line")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------------
# clocks sampling during the timed region
# ---------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------------
# roofline model (DESIGN.md section 6 / SURVEY.md 8(d)): algorithmic bytes and flops per band
# ---------------------------------------------------------------------------------------------------------
def model(wl, info):
    npw, S, P = info["npw"], info["S"], info["P"]
    n1, n2, n3 = wl.nr
    b_fft = 16.0 * (3 * npw + 4 * S * n3 + 4 * P * n2 * n3) + 8.0 * n1 * n2 * n3 / wl.batch
    b_beta = 2 * 16.0 * wl.nproj * npw / wl.batch
    f_proj = 2 * 8.0 * wl.nproj * npw
    return dict(b_fft=b_fft, b_beta=b_beta, f_proj=f_proj)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json", d
    return 6650.0, "fallback (B200_PROFILING.md)", {}


def committed_traffic(cfg, kernel):
    """dram bytes per launch of `kernel` from the committed ncu --set full capture (profiles/traffic.json)."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        d = json.load(f)
    return d.get(f"cfg{cfg}", {}).get(kernel)


# ---------------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands on the host cores, on a bounded sample
# ---------------------------------------------------------------------------------------------------------
def oracle_sample_time(wl, nbands_sample=2, atoms_sample=16):
    """Times oracle Level B (hpsi_dual) on `nbands_sample` bands of the workload. The local+kinetic part runs on
    the full grid; the nonlocal part runs on the first `atoms_sample` atoms and its time is scaled by
    natoms/atoms_sample (config 4's beta is 25 GB; the oracle's cost is linear in the number of atoms).
    Returns (seconds per band extrapolated to the full workload, description, threads)."""
    from oracle import hpsi_oracle as orc
    from paper_2104_10502_b200 import inputs

    sp = orc.gsphere(wl.at, wl.xk, wl.ecutwfc, wl.nr)
    vr = inputs.gen_vloc(wl).numpy()
    atoms = inputs.gen_atoms(wl)
    na = min(atoms_sample, wl.natoms)
    beta = inputs.gen_beta(wl, sp["miller"], atoms, 0, na).numpy() if na else None
    db = inputs.gen_dblocks(wl)[:na] if na else None
    psi = inputs.gen_psi(wl, sp["miller"], 0, nbands_sample).numpy()
    t0 = time.perf_counter()
    orc.hpsi_dual(sp["fft_index"], sp["g2kin"], tuple(wl.nr), vr, psi, None, None)
    t_loc = time.perf_counter() - t0
    t_nl = 0.0
    if na:
        t0 = time.perf_counter()
        orc.vnl_psi(beta, db, psi)
        t_nl = (time.perf_counter() - t0) * (wl.natoms / na)
    per_band = (t_loc + t_nl) / nbands_sample
    desc = (f"oracle Level B on {nbands_sample} bands of {wl.name}: local+kinetic on the full {wl.nr} grid, "
            f"nonlocal on {na}/{wl.natoms} atoms scaled linearly")
    return per_band, desc, torch.get_num_threads()


def time_next_rows(h, wl, inp, psi, hpsi, batch, npw, dmma, hbm_peak):
    """CUDA-event timings of the rows SURVEY.md 8(f) marks next, on one chunk of `batch` bands of the workload:
    qe_hpsi_apply_hs (H psi and S psi), qe_hpsi_overlap (<psi|H psi>, batch x batch), qe_hpsi_density."""
    from paper_2104_10502_b200 import inputs, qe_hpsi
    nb = min(batch, psi.shape[0])
    p, hp = psi[:nb], hpsi[:nb]
    sp = torch.empty_like(p)
    out = {}

    def ev_time(fn, reps=3):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    if wl.nproj:
        rng = np.random.default_rng(7)
        q = rng.uniform(-1, 1, (wl.natoms, wl.nh, wl.nh))
        h.set_s(0.5 * (q + q.transpose(0, 2, 1)))
    if wl.nproj and h.info().get("ozaki_slices", 0):
        # the int8 digit path against the FP64 tensor path of the same library, on the nonlocal part alone (a6-a8 only)
        h2 = qe_hpsi.Hpsi(wl.at, wl.ecutwfc, wl.xk, wl.nr, inp["vr"], inp["beta"], np.arange(wl.natoms + 1, dtype=np.int32) * wl.nh,
                          inp["dblocks"], max_batch=batch, flags=qe_hpsi.QE_HPSI_BORROW_BETA | qe_hpsi.QE_HPSI_FP64_DMMA)
        a = h.nonlocal_add(p, torch.zeros_like(p))
        b = h2.nonlocal_add(p, torch.zeros_like(p))
        torch.cuda.synchronize()
        err = torch.linalg.vector_norm(a[:, :npw] - b[:, :npw], dim=1) / torch.linalg.vector_norm(b[:, :npw], dim=1)
        full = torch.linalg.vector_norm(h.apply(p)[:, :npw] - h2.apply(p)[:, :npw], dim=1) / torch.linalg.vector_norm(h2.apply(p)[:, :npw], dim=1)
        out["int8_vs_fp64_tensor_path"] = {"digits": h.info()["ozaki_slices"], "bands": nb, "max_rel_l2_nonlocal_part": float(err.max()),
                                           "max_rel_l2_hpsi": float(full.max())}
        h2.destroy()
        del a, b, err, full
    ms = ev_time(lambda: h.apply_hs(p, hp, sp))
    fl = 3 * 8.0 * wl.nproj * npw * nb  # a6 once + a8 twice
    out["apply_hs"] = {"ms": ms, "bands_per_s": nb / ms * 1e3, "proj_tflops": fl / ms * 1e-9 if wl.nproj else None,
                       "bound": "tensor", "frac_of_dmma_peak": fl / ms * 1e-9 / dmma if wl.nproj else None}
    m = torch.empty((nb, nb), dtype=torch.complex128, device="cuda")
    ms = ev_time(lambda: h.overlap(p, hp, m))
    fl = 8.0 * nb * nb * npw
    by = 2 * 16.0 * nb * npw
    out["overlap"] = {"ms": ms, "shape": [nb, nb, npw], "tflops": fl / ms * 1e-9, "gbs": by / ms * 1e-6,
                      "bound": "hbm" if by / (hbm_peak * 1e9) > fl / (dmma * 1e12) else "tensor",
                      "frac": max(by / (hbm_peak * 1e9), fl / (dmma * 1e12)) / (ms * 1e-3)}
    occ = torch.full((nb,), 2.0, dtype=torch.float64, device="cuda")
    rho = torch.zeros(tuple(wl.nr), dtype=torch.float64, device="cuda")
    ms = ev_time(lambda: h.density(p, occ, 1.0 / wl.omega, rho))
    n1, n2, n3 = wl.nr
    info = h.info()
    by = nb * 16.0 * (npw + 2 * info["S"] * n3 + 2 * info["P"] * n2 * n3) + 16.0 * n1 * n2 * n3 * -(-nb // info["fft_nb"])
    out["density"] = {"ms": ms, "bands_per_s": nb / ms * 1e3, "algorithmic_gbs": by / ms * 1e-6, "bound": "hbm",
                      "frac": by / ms * 1e-6 / hbm_peak}
    # NEXT-3, rest of the Davidson step: preconditioner diagonals (beta streamed once), preconditioner, rotation
    if wl.nproj:
        ms = ev_time(lambda: h.hdiag(0.0, want_s=True))
        by = 2 * 16.0 * wl.nproj * npw  # beta read once for hdiag and once for sdiag
        out["hdiag_sdiag"] = {"ms": ms, "gbs": by / ms * 1e-6, "bound": "hbm", "frac": by / ms * 1e-6 / hbm_peak}
    hd, _ = h.hdiag(0.0)
    ev = torch.zeros(nb, dtype=torch.float64, device="cuda")
    ms = ev_time(lambda: h.precond(sp, ev, hd))
    by = 2 * 16.0 * nb * npw
    out["precond"] = {"ms": ms, "gbs": by / ms * 1e-6, "bound": "hbm", "frac": by / ms * 1e-6 / hbm_peak}
    coef = torch.eye(nb, dtype=torch.complex128, device="cuda")
    ms = ev_time(lambda: h.rotate(p, coef, sp))
    fl = 8.0 * nb * nb * npw
    out["rotate"] = {"ms": ms, "shape": [npw, nb, nb], "tflops": fl / ms * 1e-9, "bound": "tensor", "frac": fl / ms * 1e-9 / dmma}
    # NEXT-1: the same chunk as a real-wavefunction problem on the half sphere (k = 0 configs only)
    if all(x == 0.0 for x in wl.xk):
        mil_h = qe_hpsi.qe_hpsi_gamma_gsphere(wl.at, wl.ecutwfc, wl.nr)
        ngw = mil_h.shape[0]
        ldg = inputs.pad8(ngw)
        mh = torch.as_tensor(mil_h, device="cuda")
        bh = None
        blk = db = None
        if wl.nproj:
            bh = torch.zeros((wl.nproj, ldg), dtype=torch.complex128, device="cuda")
            for a0 in range(0, wl.natoms, 16):
                na = min(16, wl.natoms - a0)
                inputs.gen_beta(wl, mh, inp["atoms"], a0, na, ld=ldg, device="cuda", out=bh[a0 * wl.nh:(a0 + na) * wl.nh])
            bh[:, 0] = bh[:, 0].real.to(torch.complex128)
            blk = np.arange(wl.natoms + 1, dtype=np.int32) * wl.nh
            db = inp["dblocks"]
        g = qe_hpsi.HpsiGamma(wl.at, wl.ecutwfc, wl.nr, inp["vr"], bh, blk, db, max_batch=nb, flags=qe_hpsi.QE_HPSI_BORROW_BETA)
        pg = inputs.gen_psi(wl, mh, 0, nb, ld=ldg, device="cuda")
        pg[:, 0] = pg[:, 0].real.to(torch.complex128)
        hg = torch.empty_like(pg)
        ms = ev_time(lambda: g.apply(pg, hg))
        flg = 2 * 2 * 2.0 * wl.nproj * (2 * ngw) * nb / 2  # two real GEMMs over 2*ngw real components: 2*M*N*K each
        out["gamma_apply"] = {"ms": ms, "bands_per_s": nb / ms * 1e3, "ngw": ngw, "real_proj_tflops": flg / ms * 1e-9,
                              "speedup_vs_complex_path": None}
        g.destroy()
        del bh, pg, hg
    return out


def run_reference(args, wl, rank):
    if rank != 0:
        return
    times = []
    desc, cores = "", 0
    for i in range(args.warmup + args.steps):
        per_band, desc, cores = oracle_sample_time(wl)
        if i >= args.warmup:
            times.append(per_band)
    per_band = float(np.mean(times))
    val = 1.0 / per_band
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": per_band * wl.nbands * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "nbands": wl.nbands, "batch": wl.batch, "grid": list(wl.nr), "nproj": wl.nproj},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------
def main():
    args = parse()
    from paper_2104_10502_b200 import inputs

    wl = inputs.get_workload(args.config)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, wl, rank)
        return

    from paper_2104_10502_b200 import qe_hpsi, sharding

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the H|psi> path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    # ---- inputs, resident in HBM ---------------------------------------------------------------------
    t_setup = time.perf_counter()
    h, inp = qe_hpsi.from_workload(wl, flags=qe_hpsi.QE_HPSI_BORROW_BETA | (qe_hpsi.QE_HPSI_FP64_DMMA if args.dmma else 0))
    info = h.info()
    npw, ld = h.npw, inp["ld"]
    nb, batch = wl.nbands, wl.batch
    psi = torch.empty((nb, ld), dtype=torch.complex128, device="cuda")
    band0, _ = sharding.weak_band_range(rank, nb)  # rank r applies H to its own bands (keys rank*nb ...)
    calls = sharding.batches(nb, batch)
    for b0, n in calls:
        psi[b0:b0 + n] = inputs.gen_psi(wl, inp["miller_dev"], band0 + b0, n, ld=ld, device="cuda")
    hpsi = torch.zeros_like(psi)
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t_setup
    stream = torch.cuda.current_stream()

    def step():
        for b0, n in calls:
            h.apply(psi[b0:b0 + n], hpsi[b0:b0 + n], stream)

    # inputs per step (psi 6.3 GB + beta 25 GB at config 4) exceed the 126 MB L2; for small configs flush L2
    flush = None
    if (psi.numel() * 16 + (inp["beta"].numel() * 16 if inp["beta"] is not None else 0)) < (512 << 20):
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    # launch-latency-bound workloads: capture the step (apply enqueues kernels only) and replay it
    use_graph = args.graph == 1
    if args.graph == -1:
        t0 = time.perf_counter()
        step()
        torch.cuda.synchronize()
        use_graph = (time.perf_counter() - t0) < 0.5e-3
    prof_eager = None
    if use_graph:
        h.profile(1)
        step()
        torch.cuda.synchronize()
        prof_eager = h.profile_read()  # stage timers cannot record inside a capture: one eager pass
        h.profile(0)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            cap = torch.cuda.current_stream()
            for b0, n in calls:
                h.apply(psi[b0:b0 + n], hpsi[b0:b0 + n], cap)
        eager_step = step

        def step():  # noqa: F811
            graph.replay()

        for _ in range(3):
            step()
        barrier()
    else:
        h.profile(1)
    sampler = ClockSampler(torch.cuda.current_device())
    sampler.start()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    torch.cuda.profiler.start()  # cudaProfilerStart: `ncu --profile-from-start off` sees only the timed steps
    for k in range(args.steps):
        if flush is not None:
            flush.fill_(k)
        evs[k][0].record(stream)
        step()
        evs[k][1].record(stream)
    barrier()
    torch.cuda.profiler.stop()
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = float(sum(step_ms))
    prof = prof_eager if use_graph else h.profile_read()
    h.profile(0)
    total_ms = sharding.max_over_ranks(total_ms, dist, "cuda")
    ms_per_step = total_ms / args.steps
    value = sharding.aggregate_bands_per_s(world, nb, ms_per_step)

    # ---- e2e through the host-buffer entry point ------------------------------------------------------
    e2e = None
    if not args.no_e2e:
        ph = torch.empty((nb, ld), dtype=torch.complex128).pin_memory()
        hh = torch.empty((nb, ld), dtype=torch.complex128).pin_memory()
        ph.copy_(psi)
        for _ in range(2):
            h.apply_host(ph, hh)
        barrier()
        t0 = time.perf_counter()
        ne = max(2, min(args.steps, 3))
        for _ in range(ne):
            h.apply_host(ph, hh)  # synchronous: returns after the last D2H copy
        t_e2e = (time.perf_counter() - t0) / ne
        t_e2e = sharding.max_over_ranks(t_e2e, dist, "cuda")
        # the e2e result must be the device path's result
        assert torch.equal(hh[:, :npw].view(torch.float64), hpsi[:, :npw].cpu().view(torch.float64)), "e2e != device path"
        e2e = {"value": world * nb / t_e2e, "unit": UNIT, "h2d_bytes_per_step": nb * npw * 16,
               "d2h_bytes_per_step": nb * npw * 16, "ms_per_step": t_e2e * 1e3}
        del ph, hh

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline --------------------------------------------------------------------------------------
    m = model(wl, info)
    hbm_peak, peak_src, mp = peaks()
    dmma, dfma = qe_hpsi.qe_hpsi_probe_fp64(300.0)
    chunks_per_step = (nb + batch - 1) // batch
    stage = {k: (v[0] / max(v[1], 1), v[1]) for k, v in prof.items()}  # avg ms per span
    t_becp, t_vnl, t_fft = stage["a6_becp"][0], stage["a8_vnl_add"][0], stage["a1_a5_fft_chain"][0]
    flops_launch = 8.0 * wl.nproj * npw * min(batch, nb)  # per ZGEMM launch (one chunk)
    roof_t = max((m["b_fft"] + m["b_beta"]) / (hbm_peak * 1e9), m["f_proj"] / (dmma * 1e12))  # s per band
    oz_s = info.get("ozaki_slices", 0)
    int8 = None
    if wl.nproj and oz_s and t_vnl + t_becp > t_fft:
        # projector contractions on the int8 tensor cores: S (S+1) / 2 digit-pair products per real product, each exact
        pairs = oz_s * (oz_s + 1) // 2
        m3 = info.get("ozaki_3m", 0)  # 1: a6 in the integer 3M form (3 real products per complex one), 2: a8 too
        a8_is_top = t_vnl >= t_becp
        kname, t_k = (("k_oz_vnl3<S> (a8, 3M form)" if m3 == 2 else "k_oz_gemm<S,1> (a8)"), t_vnl) if a8_is_top else \
            (("k_oz_gemm<S,2> x 3 (a6, 3M form)" if m3 else "k_oz_gemm<S,0> (a6)"), t_becp)
        ops_launch = pairs * flops_launch  # 4 real MACs per complex MAC x 2 ops x pairs
        if (a8_is_top and m3 == 2) or (not a8_is_top and m3 >= 1):
            ops_launch *= 0.75
        ach = ops_launch / (t_k * 1e-3) * 1e-12
        bf16_sus = float(mp.get("bf16_tflops_sustained", 0.0)) or 1414.0
        peak = 2.0 * bf16_sus
        t_slice = stage["a6_a8_int8_digits"][0]
        roofline = {"bound": "tensor", "kernel": kname, "achieved": ach, "peak": peak, "unit": "TOP/s", "frac": ach / peak,
                    "traffic": committed_traffic(args.config, ("k_oz_vnl3" if m3 == 2 else "k_oz_gemm_a8") if a8_is_top else
                                                  ("k_oz_gemm_a6_3m" if m3 else "k_oz_gemm_a6")),
                    "peak_source": "int8 dense = 2 x MEASURED_PEAKS.json bf16_tflops_sustained (guide's nominal int8 : bf16 ratio; "
                    "the kernel runs inside a long step); a register-free UTCIMMA loop on the same chip measured 4540 TOP/s "
                    "(profiles/r1g_int8.md)", "ms_per_launch": t_k, "ops_per_launch": ops_launch, "digits": oz_s,
                    "digit_pairs": pairs, "fp64_equivalent_tflops": flops_launch / (t_k * 1e-3) * 1e-12,
                    "vs_fp64_dmma_peak": flops_launch / (t_k * 1e-3) * 1e-12 / dmma,
                    "digit_kernels_ms_per_launch": t_slice,
                    "note": "achieved = executed int8 ops of the S-digit split (every one of them is needed for the FP64 result); "
                            "fp64_equivalent_tflops = 8 flops per complex MAC / time, comparable with the FP64 DMMA peak"}
        a6_units = (0.75 if m3 >= 1 else 1.0) + (0.75 if m3 == 2 else 1.0)  # integer 3M forms: 6 of the 8 tile-GEMM units each
        t_int8 = pairs * m["f_proj"] * 0.5 * a6_units / (peak * 1e12)
        b_beta8 = 2.0 * oz_s * 2 * wl.nproj * npw / wl.batch  # int8 digit planes of beta, streamed once by a6 and once by a8
        roof8 = max((m["b_fft"] + b_beta8) / (hbm_peak * 1e9), t_int8)
        int8 = {"bands_per_s": 1.0 / roof8, "frac": value / world * roof8, "int8_tops": peak, "bytes_per_band": m["b_fft"] + b_beta8,
                "int8_ops_per_band": pairs * m["f_proj"] * 0.5 * a6_units, "note": "max(bytes/HBM, digit-pair int8 ops/int8 tensor peak) per band"}
    elif wl.nproj and t_vnl + t_becp > t_fft:
        kname, t_k = ("k_vnl_add", t_vnl) if t_vnl >= t_becp else ("k_becp", t_becp)
        ach = flops_launch / (t_k * 1e-3) * 1e-12
        roofline = {"bound": "tensor", "kernel": kname, "achieved": ach, "peak": dmma, "unit": "TFLOP/s", "frac": ach / dmma,
                    "traffic": committed_traffic(args.config, kname), "peak_source": "FP64 DMMA (mma.sync m8n8k4) register-resident "
                    "loop measured live by qe_hpsi_probe_fp64; MEASURED_PEAKS.json has no FP64 entry",
                    "ms_per_launch": t_k, "flops_per_launch": flops_launch,
                    "executed_dmma_frac": ach / dmma * 0.75,
                    "note": "achieved counts the algorithmic 8 flops per complex MAC; the 3M product executes 6, so frac can "
                            "exceed 1 (DESIGN.md section 6); executed_dmma_frac = frac x 0.75 is the pipe utilisation"}
    else:
        bytes_launch = m["b_fft"] * min(batch, nb)
        ach = bytes_launch / (t_fft * 1e-3) * 1e-9
        roofline = {"bound": "hbm", "kernel": "a1-a5 FFT chain (5 kernels per sub-chunk)", "achieved": ach, "peak": hbm_peak,
                    "unit": "GB/s", "frac": ach / hbm_peak, "traffic": committed_traffic(args.config, "fft_chain"),
                    "peak_source": peak_src, "ms_per_launch": t_fft, "bytes_per_launch": bytes_launch}
    stages = {"a6_becp_ms": t_becp, "a7_ms": stage["a7_reduce_dmul"][0], "a1_a5_fft_ms": t_fft, "a8_vnl_add_ms": t_vnl,
              "per": f"chunk of {min(batch, nb)} bands", "chunks_per_step": chunks_per_step,
              "becp_tflops": flops_launch / (t_becp * 1e-3) * 1e-12 if t_becp else None,
              "vnl_tflops": flops_launch / (t_vnl * 1e-3) * 1e-12 if t_vnl else None,
              "fft_algorithmic_gbs": m["b_fft"] * min(batch, nb) / (t_fft * 1e-3) * 1e-9 if t_fft else None,
              "int8_digit_kernels_ms": stage["a6_a8_int8_digits"][0] * 2 if oz_s else None}

    cpu = None
    if not args.no_cpu_baseline:
        per_band, desc, cores = oracle_sample_time(wl)
        cpu = {"value": 1.0 / per_band, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": wl.name, "nbands": nb, "batch": batch, "grid": list(wl.nr), "npw": npw, "nproj": wl.nproj,
                       "sticks": info["S"], "planes": info["P"], "fft_band_chunk": info["fft_nb"], "split_k": info["ozaki_nsplit"] if info.get("ozaki_slices") else info["nsplit"], "projector_path": (f"int8 digits x{info['ozaki_slices']} (tcgen05)" + ({0: "", 1: ", a6 in the integer 3M form", 2: ", a6 and a8 in the integer 3M form"}[info.get("ozaki_3m", 0)])) if info.get("ozaki_slices") else "fp64 dmma (3M)", "cuda_graph": bool(use_graph),
                       "l2": "inputs per step exceed L2" if flush is None else "L2 flushed (256 MB write) between steps",
                       "sharding": "bands / k-point pools per rank, no collective"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": h.launch_count(batch) * chunks_per_step * args.steps if nb % batch == 0
            else sum(h.launch_count(min(batch, nb - b0)) for b0 in range(0, nb, batch)) * args.steps,
            "roofline": roofline,
            "combined_roofline": {"bands_per_s": 1.0 / roof_t, "frac": value / world * roof_t, "hbm_gbs": hbm_peak,
                                  "fp64_tensor_tflops": dmma, "fp64_dfma_tflops": dfma, "bytes_per_band": m["b_fft"] + m["b_beta"],
                                  "proj_flops_per_band": m["f_proj"], "note": "max(bytes/HBM, projector flops/FP64 tensor) per band"},
            "stages": stages, "cpu_baseline": cpu, "setup_s": t_setup}
    if int8 is not None:
        line["combined_roofline_int8"] = int8
        line["dtype"] = f"f64 (projector contractions: exact int8 digit products, {oz_s} digits per operand)"
    if args.next:
        torch.cuda.profiler.start()  # the next-rows pass is visible to `ncu --profile-from-start off` too
        line["next_rows"] = time_next_rows(h, wl, inp, psi, hpsi, batch, npw, dmma, hbm_peak)
        torch.cuda.profiler.stop()
        if "gamma_apply" in line["next_rows"]:
            line["next_rows"]["gamma_apply"]["speedup_vs_complex_path"] = line["next_rows"]["gamma_apply"]["bands_per_s"] / (value / world)
    print(json.dumps(line), flush=True)

    if args.detail:
        h.profile(2)
        (eager_step if use_graph else step)()
        torch.cuda.synchronize()
        d = h.profile_read()
        h.profile(0)
        for k, (ms, cnt) in d.items():
            if cnt:
                sys.stderr.write(f"{k:18s} total {ms:10.3f} ms over {cnt} spans\n")
    h.destroy()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
