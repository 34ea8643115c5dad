"""N > 1 path on CPU: world_size-2 `gloo` run of the energy-sharded sweep.

Each rank takes the energy slice `paper_2205_15000_b200.sharding` gives it, computes the un-finalised
accumulators of its slice (the oracle stands in for the kernels here — there is no GPU), the five fields are
summed with one all-reduce, and every rank finalises with the whole table's denominator.  The result must equal
the unsharded sweep: this is the statement that the path shards by energy with a single exchange step.
"""
import os
import socket

import numpy as np
import pytest

import oracle
import workloads as wlmod
from paper_2205_15000_b200 import sharding

torch = pytest.importorskip("torch")


def test_energy_slices_partition_the_table():
    for ne, world in ((512, 8), (512, 3), (40, 3), (16, 2), (7, 7), (33, 2)):
        got = []
        for r in range(world):
            sl = sharding.energy_slice(ne, world, r)
            got += list(range(ne))[sl]
        assert got == list(range(ne)), (ne, world)
        sizes = [len(range(ne)[sharding.energy_slice(ne, world, r)]) for r in range(world)]
        unit = 32 if ne % 32 == 0 and ne // 32 >= world else 1
        assert max(sizes) - min(sizes) <= unit
    z, w, dsum = sharding.matsubara_shard(0.1, 128, 4, 2)
    assert np.allclose(z.imag, 0.1 * (np.arange(64, 96) + 0.5)) and np.all(z.real == 0) and np.all(w == 1)
    assert abs(dsum - np.sum(1.0 / (np.arange(128) + 0.5))) < 1e-12
    with pytest.raises(ValueError):
        sharding.energy_slice(8, 2, 2)


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = wlmod.make_workload(1, pts_per_xi=4, n_angles=8, n_energies=12)
    o = oracle.Oracle.from_workload(wl)
    z, w, dsum = sharding.matsubara_shard(wl.t, wl.n_energies, world, rank)
    stores = o.reset_stores(wl.delta0, wl.Aext_x, wl.Aext_y, z)
    res = None
    for _ in range(2):                                       # two Jacobi sweeps: the stores stay rank-local
        r = o.raw_sweep(wl.delta0, wl.Aext_x, wl.Aext_y, z, w, stores)
        stores = r["stores"]
        acc = torch.from_numpy(np.stack([r["num"].real, r["num"].imag, r["Jx"], r["Jy"], r["I"]]))
        dist.all_reduce(acc)                                 # the one exchange step of the path
        a = acc.numpy()
        D = np.log(wl.t) + dsum
        res = dict(delta_new=-2j * wl.t * (a[0] + 1j * a[1]) / D * wl.mask, jx=2.0 * wl.charge_sign * wl.t * a[2] * wl.mask,
                   jy=2.0 * wl.charge_sign * wl.t * a[3] * wl.mask, fe_I=wl.t * a[4] * wl.mask)
    np.savez(out + f".{rank}.npz", **res)
    dist.destroy_process_group()


def test_world2_gloo_sharded_sweep_matches_full(tmp_path):
    import torch.multiprocessing as mp
    world, port, out = 2, _free_port(), str(tmp_path / "shard")
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    wl = wlmod.make_workload(1, pts_per_xi=4, n_angles=8, n_energies=12)
    o = oracle.Oracle.from_workload(wl)
    st = None
    for _ in range(2):
        ref = o.sweep(wl.delta0, wl.Aext_x, wl.Aext_y, wl.n_energies, st)
        st = ref["stores"]
    for rank in range(world):
        got = np.load(out + f".{rank}.npz")
        for key in ("delta_new", "jx", "jy", "fe_I"):
            err = np.max(np.abs(got[key] - ref[key])) / max(np.max(np.abs(ref[key])), 1e-6)
            assert err < 1e-12, (rank, key, err)


class _FakeContext:
    """Stands in for ScContext on a box without a GPU: the same four members `sharding.attach` touches.  Its sweep
    computes this rank's accumulators with the oracle (in place of the kernels), runs the hook, and finalises —
    the order of operations of sc_riccati_sweep with a hook set (include/sc_riccati.h, sc_set_allreduce_hook)."""

    def __init__(self, wl):
        self.wl, self.o = wl, oracle.Oracle.from_workload(wl)
        self.n_components, self.ny, self.nx, self.device = 1, wl.ny, wl.nx, torch.device("cpu")
        self.stores = None

    def sc_set_energies(self, z, w, denominator_sum):
        self.z, self.w, self.dsum = np.asarray(z), np.asarray(w), denominator_sum

    def sc_set_allreduce_hook(self, acc, fn):
        self.acc, self.fn = acc, fn

    def sweep(self):
        wl = self.wl
        if self.stores is None:
            self.stores = self.o.reset_stores(wl.delta0, wl.Aext_x, wl.Aext_y, self.z)
        r = self.o.raw_sweep(wl.delta0, wl.Aext_x, wl.Aext_y, self.z, self.w, self.stores)
        self.stores = r["stores"]
        self.acc.copy_(torch.from_numpy(np.stack([r["num"].real, r["num"].imag, r["Jx"], r["Jy"], r["I"]])))
        self.fn()
        a = self.acc.numpy()
        D = np.log(wl.t) + self.dsum
        return dict(delta_new=-2j * wl.t * (a[0] + 1j * a[1]) / D * wl.mask, jx=2.0 * wl.charge_sign * wl.t * a[2] * wl.mask,
                    jy=2.0 * wl.charge_sign * wl.t * a[3] * wl.mask, fe_I=wl.t * a[4] * wl.mask)


def _attach_worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = wlmod.make_workload(1, pts_per_xi=4, n_angles=8, n_energies=64)     # whole warps of energies: 32 per rank
    ctx = _FakeContext(wl)
    acc = sharding.attach(ctx, wl.t, wl.n_energies)          # the function bench.py --gpus N calls
    assert acc.shape == (5, wl.ny, wl.nx) and len(ctx.z) == 32 and ctx.z.imag[0] == wl.t * (32 * rank + 0.5)
    for _ in range(2):
        res = ctx.sweep()
    np.savez(out + f".{rank}.npz", **res)
    dist.destroy_process_group()


def test_world2_gloo_attach_runs_the_hook_path(tmp_path):
    import torch.multiprocessing as mp
    world, port, out = 2, _free_port(), str(tmp_path / "attach")
    mp.spawn(_attach_worker, args=(world, port, out), nprocs=world, join=True)
    wl = wlmod.make_workload(1, pts_per_xi=4, n_angles=8, n_energies=64)
    o = oracle.Oracle.from_workload(wl)
    st = None
    for _ in range(2):
        ref = o.sweep(wl.delta0, wl.Aext_x, wl.Aext_y, wl.n_energies, st)
        st = ref["stores"]
    for rank in range(world):
        got = np.load(out + f".{rank}.npz")
        for key in ("delta_new", "jx", "jy", "fe_I"):
            err = np.max(np.abs(got[key] - ref[key])) / max(np.max(np.abs(ref[key])), 1e-6)
            assert err < 1e-12, (rank, key, err)
