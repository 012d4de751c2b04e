"""The N > 1 path with liblra itself (not the oracle) doing the work:
rows split with sharding.row_range, every shard binned and gridded by its own plan into a private grid, the grids and
sums of weights added, and the total compared with the ORACLE's single-pass grid at north_star's tolerances.
  * two plans on one device (always runs on a GPU box): the per-shard product path and the accumulation;
  * two NCCL ranks, one per GPU, through sharding.reduce_grid / broadcast_model (skipped below two devices)."""
import os
import socket

import numpy as np
import pytest

from paper_2508_17187_b200 import sharding
from paper_2508_17187_b200 import workloads as W

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def _close(got, want, what):
    got, want = np.asarray(got, np.complex128), np.asarray(want, np.complex128)
    assert np.linalg.norm((got - want).ravel()) <= 1e-5 * np.linalg.norm(want.ravel()), what
    assert np.abs(got - want).max() <= 1e-4 * np.abs(want).max(), what


def _shard_grid(B, wl, lo, hi, device=0):
    """bin + grid of rows [lo, hi) with a plan of its own; returns device tensors (grid, sumwt) and the plan."""
    c = wl.cfg
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(f"cuda:{device}")
    plan = B.lra_plan_create(c.nx, c.ny, c.ncorr, c.nterms, c.oversampling, wl.scale_u, wl.scale_v, wl.cf.support,
                             wl.cf.offset, wl.cf.data, tile=c.tile, tile_x=c.tile_x, sort_mode=B.LRA_SORT_TILE_CF, device=device)
    B.lra_bin(plan, d(wl.uvw[lo:hi]), wl.freq, d(wl.cf_index[lo:hi]))
    g = torch.zeros((c.nterms, c.ncorr, c.ny, c.nx), dtype=torch.complex64, device=f"cuda:{device}")
    sw = torch.zeros((c.nterms, c.ncorr), dtype=torch.float64, device=f"cuda:{device}")
    B.lra_grid(plan, d(wl.vis[lo:hi]), d(wl.wt[lo:hi]), None if wl.tau is None else d(wl.tau), g, sw)
    return g, sw, plan


def test_two_plans_one_device_sum_to_the_oracle_grid(ref):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2508_17187_b200 import binding as B
    wl = W.make_workload(W.small_config(5))
    c = wl.cfg
    want, want_sw = ref.plan_for(wl, sort_mode=1).grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, wl.tau)
    parts = [_shard_grid(B, wl, *sharding.row_range(c.nrow, k, 3)) for k in range(3)]
    try:
        torch.cuda.synchronize()
        g = sum(p[0] for p in parts)
        sw = sum(p[1] for p in parts)
        _close(g.cpu().numpy(), want, "sum of three shard grids")
        assert np.abs(sw.cpu().numpy() - want_sw).max() <= 1e-6 * np.abs(want_sw).max()
        # degrid: every shard predicts its own rows from the same model grid, no exchange afterwards
        model = want.astype(np.complex64)
        want_v = ref.plan_for(wl, sort_mode=1).degrid(wl.uvw, wl.freq, wl.cf_index, model.astype(np.complex128), wl.tau)
        dm = torch.from_numpy(model).cuda()
        dt = None if wl.tau is None else torch.from_numpy(wl.tau).cuda()
        for k, (_, _, plan) in enumerate(parts):
            lo, hi = sharding.row_range(c.nrow, k, 3)
            out = torch.empty((hi - lo, c.nchan, c.ncorr), dtype=torch.complex64, device="cuda")
            B.lra_degrid(plan, dm, dt, None, out)
            torch.cuda.synchronize()
            _close(out.cpu().numpy(), want_v[lo:hi], f"degrid of shard {k}")
    finally:
        for p in parts:
            B.lra_plan_destroy(p[2])


def _nccl_worker(rank, world, port, out):
    import torch.distributed as dist
    from paper_2508_17187_b200 import binding as B
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    try:
        wl = W.make_workload(W.small_config(5))
        lo, hi = sharding.row_range(wl.cfg.nrow, rank, world)
        g, sw, plan = _shard_grid(B, wl, lo, hi, device=rank)
        sharding.reduce_grid(g, sw)                       # the one data-path collective
        # the model grid is the oracle's (written by the parent before the spawn), held by rank 0 only
        model = torch.from_numpy(np.load(os.path.join(out, "model.npy"))).cuda() if rank == 0 else torch.zeros_like(g)
        sharding.broadcast_model(model, src=0)
        res = torch.empty((hi - lo, wl.cfg.nchan, wl.cfg.ncorr), dtype=torch.complex64, device=f"cuda:{rank}")
        B.lra_degrid(plan, model, None if wl.tau is None else torch.from_numpy(wl.tau).cuda(), None, res)
        torch.cuda.synchronize()
        np.savez(os.path.join(out, f"r{rank}.npz"), grid=g.cpu().numpy(), sumwt=sw.cpu().numpy(), vis=res.cpu().numpy(), lo=lo, hi=hi)
        B.lra_plan_destroy(plan)
    finally:
        dist.destroy_process_group()


def test_two_nccl_ranks_reduce_to_the_oracle_grid(tmp_path, ref):
    if not torch.cuda.is_available() or torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    wl = W.make_workload(W.small_config(5))
    rp = ref.plan_for(wl, sort_mode=1)
    want, want_sw = rp.grid(wl.uvw, wl.freq, wl.cf_index, wl.vis, wl.wt, wl.tau)
    model = want.astype(np.complex64)
    np.save(tmp_path / "model.npy", model)
    mp.spawn(_nccl_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    parts = [np.load(tmp_path / f"r{k}.npz") for k in range(2)]
    for p in parts:
        _close(p["grid"], want, "all-reduced grid")
        assert np.abs(p["sumwt"] - want_sw).max() <= 1e-6 * np.abs(want_sw).max()
    want_v = rp.degrid(wl.uvw, wl.freq, wl.cf_index, model.astype(np.complex128), wl.tau)
    for p in parts:
        _close(p["vis"], want_v[int(p["lo"]):int(p["hi"])], "degrid after broadcast")
