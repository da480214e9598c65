"""The N>1 path on CPU: two `gloo` ranks shard the bands of a tiny workload with no data-path collective, each
applies H (the ORACLE stands in for the GPU library here: this test is about the host-side sharding logic), and
the gathered result equals the single-process application band for band. Also the max-over-ranks timing
reduction bench.py uses. PAPER.md:L236-238 (one rank per GPU, k-point pools); DESIGN.md section 8."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import hpsi_oracle as orc
from paper_2104_10502_b200 import inputs, sharding


def test_split_bands_covers_everything_once():
    for total in (0, 1, 7, 16, 1024, 1025):
        for world in (1, 2, 3, 8):
            parts = sharding.split_bands(total, world)
            assert len(parts) == world
            assert parts[0][0] == 0 and sum(n for _, n in parts) == total
            for (a0, an), (b0, _) in zip(parts, parts[1:]):
                assert a0 + an == b0
            sizes = [n for _, n in parts]
            assert max(sizes) - min(sizes) <= 1


def test_weak_ranges_are_disjoint_and_batches_cover():
    r = [sharding.weak_band_range(k, 1024) for k in range(4)]
    assert r == [(0, 1024), (1024, 1024), (2048, 1024), (3072, 1024)]
    assert sharding.batches(1024, 128) == [(128 * i, 128) for i in range(8)]
    assert sharding.batches(7, 3) == [(0, 3), (3, 3), (6, 1)]
    assert sharding.batches(0, 4) == []
    assert sharding.aggregate_bands_per_s(8, 1024, 1000.0) == 8192.0


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, key, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = inputs.get_workload(key)
        sp = orc.gsphere(wl.at, wl.xk, wl.ecutwfc, wl.nr)
        vr = inputs.gen_vloc(wl).numpy()
        atoms = inputs.gen_atoms(wl)
        beta = inputs.gen_beta(wl, sp["miller"], atoms).numpy()
        db = inputs.gen_dblocks(wl)
        # strong split of the workload's bands: replicated V / beta / D, disjoint psi, no exchange
        b0, nb = sharding.split_bands(wl.nbands, world)[rank]
        psi = inputs.gen_psi(wl, sp["miller"], b0, nb).numpy()
        out = np.zeros((0, sp["miller"].shape[0]), np.complex128)
        for o, n in sharding.batches(nb, 2):
            part = orc.hpsi_dual(sp["fft_index"], sp["g2kin"], tuple(wl.nr), vr, psi[o:o + n], beta, db)
            out = np.concatenate([out, part])
        # the benchmark's only communication: barrier + MAX of the timed milliseconds
        dist.barrier()
        ms = sharding.max_over_ranks(10.0 + 5.0 * rank, dist)
        gathered = [None] * world
        dist.all_gather_object(gathered, (b0, nb, out))  # test-side check only; not part of the path
        if rank == 0:
            q.put((ms, gathered))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("key", ["T5_odd_bands"])
def test_two_rank_band_sharding_matches_single_process(key):
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, key, q)) for r in range(world)]
    for p in procs:
        p.start()
    ms, gathered = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ms == 15.0  # the slowest rank's time
    wl = inputs.get_workload(key)
    sp = orc.gsphere(wl.at, wl.xk, wl.ecutwfc, wl.nr)
    psi = inputs.gen_psi(wl, sp["miller"], 0, wl.nbands).numpy()
    ref = orc.hpsi_dual(sp["fft_index"], sp["g2kin"], tuple(wl.nr), inputs.gen_vloc(wl).numpy(), psi,
                        inputs.gen_beta(wl, sp["miller"], inputs.gen_atoms(wl)).numpy(), inputs.gen_dblocks(wl))
    got = np.zeros_like(ref)
    seen = np.zeros(wl.nbands, bool)
    for b0, nb, out in gathered:
        assert not seen[b0:b0 + nb].any()
        got[b0:b0 + nb] = out
        seen[b0:b0 + nb] = True
    assert seen.all()
    assert orc.rel_l2(got, ref).max() <= 1e-14  # same arithmetic per band, whatever the shard it ran in
