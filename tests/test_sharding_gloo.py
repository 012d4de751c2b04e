"""The N > 1 path on CPU: two gloo processes, each grids its row range (the oracle stands in for the GPU kernels, which
need a device), sharding.reduce_grid combines them; the sum must equal the single-process result (pin P8, partition
invariance) and degridding each rank's rows from the broadcast model must reproduce the full prediction."""
import os
import socket

import numpy as np
import pytest

from paper_2508_17187_b200 import sharding
from paper_2508_17187_b200 import workloads as W

torch = pytest.importorskip("torch")


def test_row_range_partitions_exactly():
    for nrow in (0, 1, 7, 351 * 3, 1000):
        for world in (1, 2, 3, 8):
            r = [sharding.row_range(nrow, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == nrow
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            sizes = [hi - lo for lo, hi in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.row_range(10, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    from oracle import lra_ref
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = W.make_workload(W.small_config(5))
        rp = lra_ref.plan_for(wl)
        lo, hi = sharding.row_range(wl.cfg.nrow, rank, world)
        g, sw = rp.grid(wl.uvw[lo:hi], wl.freq, wl.cf_index[lo:hi], wl.vis[lo:hi], wl.wt[lo:hi], wl.tau, nthreads=2)
        tg, tsw = torch.from_numpy(g), torch.from_numpy(sw)
        sharding.reduce_grid(tg, tsw)
        model = torch.from_numpy(np.repeat(wl.model_grid.astype(np.complex128), wl.cfg.nterms, axis=0)) if rank == 0 \
            else torch.zeros((wl.cfg.nterms, wl.cfg.ncorr, wl.cfg.ny, wl.cfg.nx), dtype=torch.complex128)
        sharding.broadcast_model(model, src=0)
        v = rp.degrid(wl.uvw[lo:hi], wl.freq, wl.cf_index[lo:hi], model.numpy(), wl.tau, nthreads=2)
        np.savez(os.path.join(out, f"r{rank}.npz"), grid=tg.numpy(), sumwt=tsw.numpy(), vis=v, lo=lo, hi=hi)
    finally:
        dist.destroy_process_group()


def test_two_rank_grid_reduce_and_degrid(tmp_path, ref):
    import torch.multiprocessing as mp
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    wl = W.make_workload(W.small_config(5))
    rp = ref.plan_for(wl)
    want, want_sw = rp.grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, wl.tau)
    model = np.repeat(wl.model_grid.astype(np.complex128), wl.cfg.nterms, axis=0)
    want_v = rp.degrid(wl.uvw, wl.freq, wl.cf_index, model, wl.tau)
    parts = [np.load(tmp_path / f"r{k}.npz") for k in range(world)]
    for p in parts:
        assert np.abs(p["grid"] - want).max() <= 1e-12 * np.abs(want).max()       # P8: grid(A u B) = grid(A) + grid(B)
        assert np.abs(p["sumwt"] - want_sw).max() <= 1e-12 * np.abs(want_sw).max()
        assert np.array_equal(p["vis"], want_v[int(p["lo"]):int(p["hi"])])         # no collective after the broadcast
    assert parts[0]["hi"] == parts[1]["lo"]
