"""World-size-2 gloo tests (CPU) of the N>1 plumbing: atom sharding, output gather, MAX timing."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import synth_liz as sl
from paper_2308_16317_b200 import shard


def test_shard_atoms_partitions():
    for total in (1, 4, 7, 16):
        for world in (1, 2, 3, 8):
            got = [a for r in range(world) for a in shard.shard_atoms(total, world, r)]
            assert got == list(range(total))
            sizes = [len(shard.shard_atoms(total, world, r)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.shard_atoms(4, 2, 2)


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = sl.custom_config(13, 1, False, n_atoms=3, n_energies=2)
        mine = shard.shard_atoms(cfg.n_atoms, world, rank)
        local = sl.make_batch(cfg, n_atoms=len(mine), atom_offset=mine.start)
        # stand-in for the per-item result: something that identifies (atom occupancy, energy) uniquely
        k = cfg.k
        tau = torch.zeros((local.batch, k, k), dtype=torch.complex128)
        for b in range(local.batch):
            tau[b] = complex(float(local.species[b].sum()), float(local.z[b].imag)) * torch.eye(k, dtype=torch.complex128)
        counts = [len(shard.shard_atoms(cfg.n_atoms, world, r)) * cfg.n_energies for r in range(world)]
        full = shard.gather_tau00(tau, counts)
        tmax = shard.max_over_ranks(10.0 + rank)
        if rank == 0:
            np.save(out, full.numpy())
            assert tmax == 10.0 + world - 1
    finally:
        dist.destroy_process_group()


def test_two_rank_sharding_gathers_in_global_batch_order(tmp_path):
    out = str(tmp_path / "full.npy")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    full = np.load(out)
    cfg = sl.custom_config(13, 1, False, n_atoms=3, n_energies=2)
    glob = sl.make_batch(cfg)
    assert full.shape == (6, 4, 4)
    for b in range(6):
        assert full[b, 0, 0] == complex(float(glob.species[b].sum()), float(glob.z[b].imag))
