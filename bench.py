#!/usr/bin/env python
"""bench.py -- H|psi> band-applications/s on B200 (BASELINE.json metric), with roofline and CPU-oracle baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path (a1-a8) over all `nbands` bands of the workload, applied in calls of
`batch` bands (config 4: 1024 bands as 8 calls of 128). `value` = bands/s with psi/hpsi resident in HBM; `e2e` =
the same through qe_hpsi_apply_host with pinned HOST buffers (H2D of psi and D2H of hpsi inside the timed region).
Default workload: config 4 (the configuration north_star's target is quoted on; fits one GPU). Inputs are seeded
synthetic data. N > 1 (torchrun): every rank runs the same workload on its own bands
(k-point-pool style sharding, no data-path collective): weak scaling, max-over-ranks time.

The headline (`value`, `e2e`, `roofline`, `combined_roofline`, `dtype` "f64") is the library's DEFAULT arithmetic: FP64
throughout, projector contractions on the FP64 tensor pipe. The opt-in int8 digit paths (create flag QE_HPSI_PROJ_INT8: 55-bit
and 47-bit block fixed point, and the certified 47-bit path) are timed on the same inputs as named sub-objects under
`int8_paths`, each with its measured error against the FP64 path beside it; they are not the headline.
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
    ap.add_argument("--path", default="fp64", choices=["fp64", "fp64_general", "int8_s7", "int8_s6", "int8_s6_certified"],
                    help="arithmetic of the HEADLINE leg (default fp64 = the library default; the others for profiling runs)")
    ap.add_argument("--no-int8", action="store_true", help="skip the int8_paths legs")
    ap.add_argument("--no-next", action="store_true", help="skip the next_rows object (SURVEY 8(f) rows: apply_hs, overlap, "
                    "density, Davidson pieces, Gamma-only apply)")
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
def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def oracle_sample_time(wl, bands_per_core=2, atoms_sample=32, max_bands=128):
    """Times oracle Level B (hpsi_dual), as it stands, on all host cores this process may use: 2 bands per core (at most
    `max_bands`), bands spread over the cores by a thread pool (numpy's FFT and BLAS release the GIL). The local + kinetic
    part runs on the full grid; the nonlocal part on the first `atoms_sample` atoms for all sampled bands at once (config 4's
    beta is 25 GB; the oracle's cost is linear in the number of atoms) with its time scaled by natoms / atoms_sample.
    Returns (seconds per band of the full workload at this core count, description, cores)."""
    from concurrent.futures import ThreadPoolExecutor

    from oracle import hpsi_oracle as orc
    from paper_2104_10502_b200 import inputs

    cores = host_cores()
    nbs = max(2, min(max_bands, bands_per_core * cores, wl.nbands))
    sp = orc.gsphere(wl.at, wl.xk, wl.ecutwfc, wl.nr)
    vr = inputs.gen_vloc(wl).numpy()
    atoms = inputs.gen_atoms(wl)
    na = min(atoms_sample, wl.natoms)
    beta = inputs.gen_beta(wl, sp["miller"], atoms, 0, na).numpy() if na else None
    db = inputs.gen_dblocks(wl)[:na] if na else None
    psi = inputs.gen_psi(wl, sp["miller"], 0, nbs).numpy()
    nr = tuple(wl.nr)

    def one(b):
        return orc.hpsi_dual(sp["fft_index"], sp["g2kin"], nr, vr, psi[b:b + 1], None, None)

    t0 = time.perf_counter()
    with ThreadPoolExecutor(cores) as ex:
        list(ex.map(one, range(nbs)))
    t_loc = time.perf_counter() - t0
    t_nl = 0.0
    if na:
        t0 = time.perf_counter()
        orc.vnl_psi(beta, db, psi)  # BLAS threads over the cores
        t_nl = (time.perf_counter() - t0) * (wl.natoms / na)
    per_band = (t_loc + t_nl) / nbs
    desc = (f"oracle Level B on {nbs} bands of {wl.name} ({bands_per_core} per core) spread over {cores} host cores: local+kinetic "
            f"on the full {wl.nr} grid ({t_loc:.1f} s), nonlocal on {na}/{wl.natoms} atoms scaled linearly ({t_nl:.1f} s)")
    return per_band, desc, cores


def ev_time(fn, reps=3):
    """mean ms of `reps` calls of fn after one warm-up, CUDA events on the current stream"""
    fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def time_next_rows(h, wl, inp, psi, hpsi, batch, npw, dmma, hbm_peak, hpsi_bands_per_s):
    """CUDA-event timings of the rows SURVEY.md 8(f) marks next, on one chunk of `batch` bands of the workload, FP64 handle:
    qe_hpsi_apply_hs (H psi and S psi), qe_hpsi_overlap, qe_hpsi_density, the Davidson pieces, qe_hpsi_gamma_apply."""
    from paper_2104_10502_b200 import inputs, qe_hpsi
    nb = min(batch, psi.shape[0])
    p, hp = psi[:nb], hpsi[:nb]
    sp = torch.empty_like(p)
    out = {"per": f"one chunk of {nb} bands, FP64 handle"}
    if wl.nproj:
        rng = np.random.default_rng(7)
        q = rng.uniform(-1, 1, (wl.natoms, wl.nh, wl.nh))
        h.set_s(0.5 * (q + q.transpose(0, 2, 1)))
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
    # NEXT-3, rest of the Davidson step: preconditioner diagonals (beta streamed once), preconditioner, rotation, residual
    if wl.nproj:
        ms = ev_time(lambda: h.hdiag(0.0, want_s=True))
        by = 2 * 16.0 * wl.nproj * npw  # beta read once for hdiag and once for sdiag
        out["hdiag_sdiag"] = {"ms": ms, "gbs": by / ms * 1e-6, "bound": "hbm", "frac": by / ms * 1e-6 / hbm_peak}
    hd, _ = h.hdiag(0.0)
    ev = torch.zeros(nb, dtype=torch.float64, device="cuda")
    ms = ev_time(lambda: h.precond(sp, ev, hd))
    by = 2 * 16.0 * nb * npw
    out["precond"] = {"ms": ms, "gbs": by / ms * 1e-6, "bound": "hbm", "frac": by / ms * 1e-6 / hbm_peak}
    ms = ev_time(lambda: h.residual(hp, p, ev, r=sp))
    by = 3 * 16.0 * nb * npw
    out["residual"] = {"ms": ms, "gbs": by / ms * 1e-6, "bound": "hbm", "frac": by / ms * 1e-6 / hbm_peak}
    coef = torch.eye(nb, dtype=torch.complex128, device="cuda")
    ms = ev_time(lambda: h.rotate(p, coef, sp))
    fl = 8.0 * nb * nb * npw
    out["rotate"] = {"ms": ms, "shape": [npw, nb, nb], "tflops": fl / ms * 1e-9, "bound": "tensor", "frac": fl / ms * 1e-9 / dmma}
    del sp, rho
    # NEXT-1: the same chunk as a real-wavefunction problem on the half sphere (k = 0 configs only), FP64
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
                              "frac_of_dmma_peak": flg / ms * 1e-9 / dmma,
                              "speedup_vs_complex_path": nb / ms * 1e3 / hpsi_bands_per_s}
        g.destroy()
        del bh, pg, hg
    return out


def run_reference(args, wl, rank):
    if rank != 0:
        return
    times = []
    desc, cores = "", 0
    for i in range(args.warmup + args.steps):
        per_band, desc, cores = oracle_sample_time(wl, bands_per_core=1, atoms_sample=16, max_bands=16)
        if i >= args.warmup:
            times.append(per_band)
    per_band = float(np.mean(times))
    val = 1.0 / per_band
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": per_band * wl.nbands * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "nbands": wl.nbands, "batch": wl.batch, "grid": list(wl.nr), "nproj": wl.nproj},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc + "; each step is this "
                             "bounded sample, ms_per_step is its per-band time x nbands (an extrapolation, stated)"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


PATH_FLAGS = {"fp64": lambda hz: 0, "fp64_general": lambda hz: 32,  # 32 = QE_HPSI_NO_GAMMA_SYM
              "int8_s7": lambda hz: hz.int8_flags(7), "int8_s6": lambda hz: hz.int8_flags(6),
              "int8_s6_certified": lambda hz: hz.int8_flags(6, certify=True)}
PATH_DTYPE = {"fp64": "f64", "fp64_general": "f64",
              "int8_s7": "f64 operands as 7 int8 digits (55-bit block fixed point) in the projector contractions, FP64 elsewhere",
              "int8_s6": "f64 operands as 6 int8 digits (47-bit block fixed point) in the projector contractions, FP64 elsewhere",
              "int8_s6_certified": "as int8_s6, each chunk checked a posteriori and failing bands re-computed in FP64"}


class Leg:
    """One timed arm: a handle with a given projector arithmetic on the shared inputs."""

    def __init__(self, name, wl, inp, psi, hpsi, calls, dist):
        from paper_2104_10502_b200 import harness, qe_hpsi
        self.name, self.wl, self.psi, self.hpsi, self.calls, self.dist = name, wl, psi, hpsi, calls, dist
        t0 = time.perf_counter()
        blk = inp["blk"]
        self.h = qe_hpsi.Hpsi(wl.at, wl.ecutwfc, wl.xk, wl.nr, inp["vr"], inp["beta"], blk, inp["dblocks"], max_batch=wl.batch,
                              flags=qe_hpsi.QE_HPSI_BORROW_BETA | PATH_FLAGS[name](harness))
        torch.cuda.synchronize()
        self.create_s = time.perf_counter() - t0
        self.stream = torch.cuda.current_stream()
        self.graph = None

    def eager_step(self):
        for b0, n in self.calls:
            self.h.apply(self.psi[b0:b0 + n], self.hpsi[b0:b0 + n], self.stream)

    def step(self):
        if self.graph is not None:
            self.graph.replay()
        else:
            self.eager_step()

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()
        torch.cuda.synchronize()

    def maybe_graph(self, mode):
        """launch-latency-bound workloads: capture the step (apply enqueues kernels only) and replay it"""
        use = mode == 1
        if mode == -1:
            t0 = time.perf_counter()
            self.eager_step()
            torch.cuda.synchronize()
            use = (time.perf_counter() - t0) < 0.5e-3
        if use:
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                cap = torch.cuda.current_stream()
                for b0, n in self.calls:
                    self.h.apply(self.psi[b0:b0 + n], self.hpsi[b0:b0 + n], cap)
            self.graph = g
            for _ in range(3):
                self.step()
        return use

    def timed(self, steps, warmup, flush, profiler=False):
        """W warm-ups, then K steps between barriers, CUDA events on the launching stream, stage timers OFF.
        Returns (ms per step max over ranks, per-step list, clocks)."""
        from paper_2104_10502_b200 import sharding
        for _ in range(max(warmup, 3)):
            self.step()
        self.barrier()
        sampler = ClockSampler(torch.cuda.current_device())
        sampler.start()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        self.barrier()
        if profiler:
            torch.cuda.profiler.start()  # cudaProfilerStart: `ncu --profile-from-start off` sees only the timed steps
        for k in range(steps):
            if flush is not None:
                flush.fill_(k)
            evs[k][0].record(self.stream)
            self.step()
            evs[k][1].record(self.stream)
        self.barrier()
        if profiler:
            torch.cuda.profiler.stop()
        clocks = sampler.stop()
        step_ms = [a.elapsed_time(b) for a, b in evs]
        total = sharding.max_over_ranks(float(sum(step_ms)), self.dist, "cuda")
        return total / steps, step_ms, clocks

    def stage_pass(self, steps):
        """the same steps again, eagerly, with the library's CUDA-event stage timers on: average ms per span"""
        self.h.profile(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(self.stream)
        for _ in range(steps):
            self.eager_step()
        e1.record(self.stream)
        torch.cuda.synchronize()
        prof = self.h.profile_read()
        self.h.profile(0)
        return {k: (v[0] / max(v[1], 1), v[1]) for k, v in prof.items()}, e0.elapsed_time(e1) / steps

    def e2e(self, steps):
        from paper_2104_10502_b200 import sharding
        nb, ld, npw = self.psi.shape[0], self.psi.shape[1], self.h.npw
        ph = torch.empty((nb, ld), dtype=torch.complex128).pin_memory()
        hh = torch.empty((nb, ld), dtype=torch.complex128).pin_memory()
        ph.copy_(self.psi)
        for _ in range(2):
            self.h.apply_host(ph, hh)
        self.barrier()
        t0 = time.perf_counter()
        ne = max(2, min(steps, 3))
        for _ in range(ne):
            self.h.apply_host(ph, hh)  # synchronous: returns after the last D2H copy
        t = sharding.max_over_ranks((time.perf_counter() - t0) / ne, self.dist, "cuda")
        # the e2e result must be the device path's result
        assert torch.equal(hh[:, :npw].view(torch.float64), self.hpsi[:, :npw].cpu().view(torch.float64)), "e2e != device path"
        world = 1 if self.dist is None else self.dist.get_world_size()
        return {"value": world * nb / t, "unit": UNIT, "h2d_bytes_per_step": nb * npw * 16, "d2h_bytes_per_step": nb * npw * 16,
                "ms_per_step": t * 1e3}

    def launches(self, steps):
        return sum(self.h.launch_count(n) for _, n in self.calls) * steps

    def close(self):
        self.graph = None
        self.h.destroy()
        torch.cuda.empty_cache()


def int8_roofline(leg, stage, m, mp, hbm_peak, dmma, args, value, world):
    """roofline objects of an int8 leg: the dominant digit GEMM against the int8 tensor peak, and the combined int8 roofline"""
    wl, info = leg.wl, leg.h.info()
    npw, nbc = leg.h.npw, min(wl.batch, wl.nbands)
    oz_s = info["ozaki_slices"]
    pairs = oz_s * (oz_s + 1) // 2
    m3 = info.get("ozaki_3m", 0)  # 1: a6 in the integer 3M form (3 real products per complex one), 2: a8 too
    gsym = bool(info.get("gamma_sym"))  # Gamma-symmetric real forms over the half sphere: half of the real-form complex MACs
    t_becp, t_vnl = stage["a6_becp"][0], stage["a8_vnl_add"][0]
    a8_is_top = t_vnl >= t_becp
    if gsym:
        kname, t_k = ("k_oz_gemm<S,4> (a8, Gamma-symmetric real form)", t_vnl) if a8_is_top else ("k_oz_gemm<S,2> (a6, Gamma-symmetric real form)", t_becp)
    else:
        kname, t_k = (("k_oz_vnl3<S> (a8, 3M form)" if m3 == 2 else "k_oz_gemm<S,1> (a8)"), t_vnl) if a8_is_top else \
            (("k_oz_gemm<S,2> x 3 (a6, 3M form)" if m3 else "k_oz_gemm<S,0> (a6)"), t_becp)
    flops_launch = 8.0 * wl.nproj * npw * nbc
    ops_launch = pairs * flops_launch  # 4 real MACs per complex MAC x 2 ops x pairs
    if gsym:
        ops_launch *= 0.5
    elif (a8_is_top and m3 == 2) or (not a8_is_top and m3 >= 1):
        ops_launch *= 0.75
    ach = ops_launch / (t_k * 1e-3) * 1e-12
    bf16_sus = float(mp.get("bf16_tflops_sustained", 0.0)) or 1414.0
    peak = 2.0 * bf16_sus
    tkey = (("k_oz_gemm_a8_sym" if a8_is_top else "k_oz_gemm_a6_sym") if gsym else
            (("k_oz_vnl3" if m3 == 2 else "k_oz_gemm_a8") if a8_is_top else ("k_oz_gemm_a6_3m" if m3 else "k_oz_gemm_a6")))
    roofline = {"bound": "tensor", "kernel": kname, "achieved": ach, "peak": peak, "unit": "TOP/s", "frac": ach / peak,
                "traffic": committed_traffic(args.config, tkey) if oz_s == 6 else (committed_traffic(args.config, tkey + "_s7") if oz_s == 7 and gsym else None),
                "peak_source": "int8 dense = 2 x MEASURED_PEAKS.json bf16_tflops_sustained (guide's nominal int8 : bf16 ratio; the "
                "kernel runs inside a long, power-capped step). Against the chip's measured int8 burst (register-free UTCIMMA loop, "
                "4540 TOP/s, profiles/r1g_int8.md) the same kernel is at " + f"{ach / 4540.0:.2f}" + "; ncu (profiles/r2l_capture.md): tensor pipe 67-82 % of active cycles", "ms_per_launch": t_k, "ops_per_launch": ops_launch, "digits": oz_s,
                "digit_pairs": pairs, "fp64_equivalent_tflops": flops_launch / (t_k * 1e-3) * 1e-12,
                "digit_kernels_ms_per_launch": stage["a6_a8_int8_digits"][0]}
    units = (0.75 if m3 >= 1 else 1.0) + (0.75 if m3 == 2 else 1.0)  # integer 3M forms: 6 of the 8 tile-GEMM units each
    if gsym:
        units = 1.0  # two real forms over the half sphere: half of the real-form complex MACs each
    t_int8 = pairs * m["f_proj"] * 0.5 * units / (peak * 1e12)
    b_beta8 = (3 if m3 >= 1 else 2) * oz_s * wl.nproj * npw / wl.batch + (3 if m3 == 2 else 2) * oz_s * wl.nproj * npw / wl.batch
    if gsym:
        b_beta8 = 2.0 * oz_s * wl.nproj * npw / wl.batch  # half-sphere real-form planes, streamed once by a6 and once by a8
    roof8 = max((m["b_fft"] + b_beta8) / (hbm_peak * 1e9), t_int8)
    combined = {"bands_per_s": 1.0 / roof8, "frac": value / world * roof8, "int8_tops": peak, "bytes_per_band": m["b_fft"] + b_beta8,
                "int8_ops_per_band": pairs * m["f_proj"] * 0.5 * units,
                "note": "max(bytes/HBM, digit-pair int8 ops / int8 tensor peak) per band; NOT the north_star roofline (that one is "
                        "defined on the FP64 tensor pipe and is printed for the FP64 leg only)"}
    return roofline, combined


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

    from paper_2104_10502_b200 import harness, qe_hpsi, sharding

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the H|psi> path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    # ---- cpu_baseline first (rank 0, N = 1 only): the oracle on the host cores, before the GPU legs, outside any timed region
    cpu = None
    if not args.no_cpu_baseline and rank == 0 and world == 1:
        per_band, desc, cores = oracle_sample_time(wl)
        cpu = {"value": 1.0 / per_band, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}

    # ---- inputs, resident in HBM ---------------------------------------------------------------------
    t_setup = time.perf_counter()
    h0, inp = harness.from_workload(wl, flags=qe_hpsi.QE_HPSI_BORROW_BETA, max_batch=1)  # generators + the library's sphere
    h0.destroy()
    ld = inp["ld"]
    nb, batch = wl.nbands, wl.batch
    psi = torch.empty((nb, ld), dtype=torch.complex128, device="cuda")
    band0, _ = sharding.weak_band_range(rank, nb)  # rank r applies H to its own bands (keys rank*nb ...)
    calls = sharding.batches(nb, batch)
    for b0, n in calls:
        psi[b0:b0 + n] = inputs.gen_psi(wl, inp["miller_dev"], band0 + b0, n, ld=ld, device="cuda")
    hpsi = torch.zeros_like(psi)
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t_setup

    # inputs per step (psi 6.3 GB + beta 25 GB at config 4) exceed the 126 MB L2; for small configs flush L2
    flush = None
    if (psi.numel() * 16 + (inp["beta"].numel() * 16 if inp["beta"] is not None else 0)) < (512 << 20):
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    # ---- headline leg ------------------------------------------------------------------------------------
    leg = Leg(args.path, wl, inp, psi, hpsi, calls, dist)
    h = leg.h
    info = h.info()
    npw = h.npw
    for _ in range(max(args.warmup, 3)):
        leg.eager_step()
    leg.barrier()
    use_graph = leg.maybe_graph(args.graph)
    ms_per_step, step_ms, clocks = leg.timed(args.steps, args.warmup, flush, profiler=True)
    value = sharding.aggregate_bands_per_s(world, nb, ms_per_step)
    launches = leg.launches(args.steps)
    stage, stage_pass_ms = leg.stage_pass(max(1, min(args.steps, 5)))  # separate eager pass: stage timers never run in the timed steps
    e2e = None if args.no_e2e else leg.e2e(args.steps)
    ref_vnl = None
    if wl.nproj and args.path == "fp64" and not args.no_int8:
        pb = psi[:min(batch, nb)]
        ref_vnl = h.nonlocal_add(pb, torch.zeros_like(pb))  # FP64 nonlocal part of the first chunk: the legs' error reference
        torch.cuda.synchronize()

    if rank != 0:
        leg.close()
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline --------------------------------------------------------------------------------------
    m = model(wl, info)
    hbm_peak, peak_src, mp = peaks()
    dmma, dfma = qe_hpsi.qe_hpsi_probe_fp64(300.0)
    chunks_per_step = (nb + batch - 1) // batch
    t_becp, t_vnl, t_fft = stage["a6_becp"][0], stage["a8_vnl_add"][0], stage["a1_a5_fft_chain"][0]
    flops_launch = 8.0 * wl.nproj * npw * min(batch, nb)  # per ZGEMM launch (one chunk)
    roof_t = max((m["b_fft"] + m["b_beta"]) / (hbm_peak * 1e9), m["f_proj"] / (dmma * 1e12))  # s per band
    oz_s = info.get("ozaki_slices", 0)
    combined8 = None
    if wl.nproj and oz_s and t_vnl + t_becp > t_fft:
        roofline, combined8 = int8_roofline(leg, stage, m, mp, hbm_peak, dmma, args, value, world)
    elif wl.nproj and t_vnl + t_becp > t_fft:
        kname, t_k = ("k_vnl_add", t_vnl) if t_vnl >= t_becp else ("k_becp", t_becp)
        gsym = bool(info.get("gamma_sym"))
        ex = 0.5 if gsym else 0.75  # executed / algorithmic flops
        ach = flops_launch / (t_k * 1e-3) * 1e-12
        kern = ("k_vnl_tma" if kname == "k_vnl_add" else "k_becp_tma") + ("<ZgS, ZF_SYM> (Gamma-symmetric real form, TMA-fed)" if gsym
                                                                           else "<ZgV0, ZF_3M> (3M complex form, TMA-fed)")
        roofline = {"bound": "tensor", "kernel": kern,
                    "achieved": ach, "peak": dmma, "unit": "TFLOP/s", "frac": ach / dmma,
                    "traffic": committed_traffic(args.config, kname + ("_sym" if gsym else "")),
                    "peak_source": "FP64 DMMA (mma.sync m8n8k4) register-resident "
                    "loop measured live by qe_hpsi_probe_fp64; MEASURED_PEAKS.json has no FP64 entry",
                    "ms_per_launch": t_k, "flops_per_launch": flops_launch, "executed_flops_per_launch": flops_launch * ex,
                    "executed_dmma_frac": ach / dmma * ex,
                    "note": "achieved counts the ALGORITHMIC 8 flops per complex MAC of north_star's F_proj; the kernel executes fewer in "
                            "the same FP64 arithmetic, so frac can exceed 1: " + ("at k = 0 with projectors that pass the bit-exact "
                            "beta(-G) = +-conj beta(G) check psi = u + i v is contracted as two real problems over the half sphere, 4 "
                            "executed flops per complex MAC (DESIGN.md section 5.8)" if gsym else "the 3M complex product executes 6 "
                            "(DESIGN.md section 6)") + "; executed_dmma_frac is the DMMA pipe utilisation"}
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
              "fft_frac_of_hbm": m["b_fft"] * min(batch, nb) / (t_fft * 1e-3) * 1e-9 / hbm_peak if t_fft else None,
              "int8_digit_kernels_ms": stage["a6_a8_int8_digits"][0] * 2 if oz_s else None,
              "certify_ms": stage["certify_check_redo"][0] if info.get("certify") else None,
              "measured_in": "a separate eager pass right after the timed steps (stage timers are off inside them)",
              "stage_pass_ms_per_step": stage_pass_ms}

    proj_path = ("fp64 dmma (Gamma-symmetric real form over the half sphere)" if info.get("gamma_sym") else "fp64 dmma (3M)") if not oz_s else (f"int8 digits x{oz_s} (tcgen05)" + {0: "", 1: ", a6 in the integer 3M form",
                2: ", a6 and a8 in the integer 3M form"}[info.get("ozaki_3m", 0)] + (", certified" if info.get("certify") else ""))
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": PATH_DTYPE[args.path],
            "data": "synthetic",
            "config": {"workload": wl.name, "nbands": nb, "batch": batch, "grid": list(wl.nr), "npw": npw, "nproj": wl.nproj,
                       "sticks": info["S"], "planes": info["P"], "fft_band_chunk": info["fft_nb"],
                       "split_k": info["ozaki_nsplit"] if oz_s else info["nsplit"], "projector_path": proj_path,
                       "cuda_graph": bool(use_graph),
                       "l2": "inputs per step exceed L2" if flush is None else "L2 flushed (256 MB write) between steps",
                       "sharding": "bands / k-point pools per rank, no collective"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline}
    if not oz_s:
        line["combined_roofline"] = {"bands_per_s": 1.0 / roof_t, "frac": value / world * roof_t, "hbm_gbs": hbm_peak,
                                     "fp64_tensor_tflops": dmma, "fp64_dfma_tflops": dfma, "bytes_per_band": m["b_fft"] + m["b_beta"],
                                     "proj_flops_per_band": m["f_proj"],
                                     "note": "north_star's roofline: max(bytes/HBM, projector flops/FP64 tensor peak) per band"}
    else:
        line["combined_roofline_int8"] = combined8
    line["stages"] = stages
    line["cpu_baseline"] = cpu
    line["setup_s"] = t_setup
    line["create_s"] = leg.create_s

    if not args.no_next and args.path == "fp64":
        torch.cuda.profiler.start()  # the next-rows pass is visible to `ncu --profile-from-start off` too
        line["next_rows"] = time_next_rows(h, wl, inp, psi, hpsi, batch, npw, dmma, hbm_peak, value / world)
        torch.cuda.profiler.stop()

    if args.detail:
        h.profile(2)
        leg.eager_step()
        torch.cuda.synchronize()
        d = h.profile_read()
        h.profile(0)
        for k, (ms, cnt) in d.items():
            if cnt:
                sys.stderr.write(f"{k:18s} total {ms:10.3f} ms over {cnt} spans\n")
    leg.close()

    # ---- the same FP64 step with the general complex contraction (QE_HPSI_NO_GAMMA_SYM): what k != 0 or unsymmetric projectors get
    if wl.nproj and args.path == "fp64" and info.get("gamma_sym") and not args.no_int8 and world == 1:
        lg = Leg("fp64_general", wl, inp, psi, hpsi, calls, None)
        for _ in range(3):
            lg.eager_step()
        torch.cuda.synchronize()
        k = max(2, min(args.steps, 3))
        msg, _, clkg = lg.timed(k, 3, flush)
        stg, _ = lg.stage_pass(1)
        vg = nb / msg * 1e3
        pb = psi[:min(batch, nb)]
        got = lg.h.nonlocal_add(pb, torch.zeros_like(pb))
        dg = torch.linalg.vector_norm(got[:, :npw] - ref_vnl[:, :npw], dim=1) / torch.linalg.vector_norm(ref_vnl[:, :npw], dim=1)
        line["fp64_general_contraction"] = {
            "value": vg, "unit": UNIT, "ms_per_step": msg, "steps": k, "dtype": "f64", "projector_path": "fp64 dmma (3M complex form)",
            "combined_roofline_frac": vg * roof_t, "a6_becp_ms": stg["a6_becp"][0], "a8_vnl_add_ms": stg["a8_vnl_add"][0],
            "executed_dmma_frac_a8": flops_launch / (stg["a8_vnl_add"][0] * 1e-3) * 1e-12 / dmma * 0.75, "clocks": clkg,
            "max_rel_l2_nonlocal_part_vs_headline_leg": float(dg.max()),
            "note": "the same step with create flag QE_HPSI_NO_GAMMA_SYM: 6 executed flops per complex MAC instead of 4; this is the "
                    "form config 3 (general k) and unsymmetric projector sets run"}
        del got, dg
        lg.close()

    # ---- the opt-in int8 digit paths on the same inputs: named sub-objects, each with its measured error ---------------
    if wl.nproj and args.path == "fp64" and not args.no_int8 and world == 1:
        legs = {}
        for name in ("int8_s7", "int8_s6", "int8_s6_certified"):
            try:
                lg = Leg(name, wl, inp, psi, hpsi, calls, None)
            except qe_hpsi.QeHpsiError as e:  # e.g. QE_HPSI_ENOMEM for the digit planes: reported, never a silent path change
                legs[name] = {"unavailable": str(e)}
                torch.cuda.empty_cache()
                continue
            for _ in range(3):
                lg.eager_step()
            torch.cuda.synchronize()
            lg.maybe_graph(args.graph)
            k = max(2, min(args.steps, 5))
            ms8, _, clk8 = lg.timed(k, 3, flush)
            st8, _ = lg.stage_pass(2)
            v8 = nb / ms8 * 1e3
            r8, c8 = int8_roofline(lg, st8, m, mp, hbm_peak, dmma, args, v8, 1)
            pb = psi[:min(batch, nb)]
            got = lg.h.nonlocal_add(pb, torch.zeros_like(pb))
            err = torch.linalg.vector_norm(got[:, :npw] - ref_vnl[:, :npw], dim=1) / torch.linalg.vector_norm(ref_vnl[:, :npw], dim=1)
            i8 = lg.h.info()
            obj = {"value": v8, "unit": UNIT, "ms_per_step": ms8, "steps": k, "dtype": PATH_DTYPE[name], "digits": i8["ozaki_slices"],
                   "forms_3m": i8["ozaki_3m"], "certified": bool(i8["certify"]),
                   "max_rel_l2_error_nonlocal_part_vs_fp64_path": float(err.max()), "error_measured_on": f"{pb.shape[0]} bands (first chunk)",
                   "clocks": clk8, "roofline": r8, "combined_roofline_int8": c8, "gpu_launches": lg.launches(k),
                   "stages": {"a6_becp_ms": st8["a6_becp"][0], "a1_a5_fft_ms": st8["a1_a5_fft_chain"][0], "a8_vnl_add_ms": st8["a8_vnl_add"][0],
                              "digit_kernels_ms": st8["a6_a8_int8_digits"][0] * 2,
                              "certify_ms": st8["certify_check_redo"][0] if i8["certify"] else None},
                   "create_s": lg.create_s, "digit_plane_bytes": i8["workspace_bytes"],
                   "speedup_vs_fp64_headline": v8 / value}
            if i8["certify"]:
                rel, redo = lg.h.proj_check(pb.shape[0])
                obj["a_posteriori_estimate_max"] = float(rel.max())
                obj["bands_recomputed_in_fp64"] = int(redo.sum())
            del got, err
            legs[name] = obj
            lg.close()
        line["int8_paths"] = legs
        line["int8_paths_note"] = ("opt-in accuracy classes (create flag QE_HPSI_PROJ_INT8), NOT the headline: block fixed point under a "
                                   "per-row exponent; oracle parity of their nonlocal part at full size is in tests/test_gpu_parity.py")
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
