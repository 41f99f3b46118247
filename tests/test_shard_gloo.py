"""-m "not gpu": the index arithmetic of the slab decomposition (fsp_shard_planes / fsp_shard_block, the very numbers
the P2P copy kernel is launched with) pushed through a real world-size-2 exchange on CPU (gloo): a labelled array
B1x_r[kx][yl][z] = label(kx, y, z) goes through the forward transpose, must arrive as B1y_s[kxl][y][z] with the right
labels, and come back unchanged through the backward transpose."""
import os

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2405_02603_b200 import binding


def label(kx, y, z):
    return kx * 1_000_000 + y * 1_000 + z


def _apply_block(dst, src, blk):
    nrun, run_len, so, ss, do, ds = blk
    for i in range(nrun):
        dst[do + i * ds: do + i * ds + run_len] = src[so + i * ss: so + i * ss + run_len]


def _exchange(rank, world, send_src, recv_dst, N, direction):
    """Every rank sends to every rank the runs of fsp_shard_block, packed; the receiver places them with the same block."""
    Nx, Ny, Nz = N
    for dst_rank in range(world):
        for src_rank in range(world):
            blk = binding.shard_block(Nx, Ny, Nz, world, src_rank, dst_rank, direction)
            nrun, run_len, so, ss, do, ds = blk
            if src_rank == rank:
                packed = torch.stack([send_src[so + i * ss: so + i * ss + run_len] for i in range(nrun)]) if nrun else torch.empty(0)
                if dst_rank == rank:
                    got = packed
                else:
                    dist.send(packed.contiguous(), dst=dst_rank)
            if dst_rank == rank:
                if src_rank != rank:
                    got = torch.empty((nrun, run_len), dtype=torch.float64)
                    dist.recv(got, src=src_rank)
                for i in range(nrun):
                    recv_dst[do + i * ds: do + i * ds + run_len] = got[i]


def _worker(rank, world, port, N, ret):
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        Nx, Ny, Nz = N
        yl = Ny // world
        k0, npl = binding.shard_planes(Nx, world, rank)
        kx, y, z = np.meshgrid(np.arange(Nx + 1), rank * yl + np.arange(yl), np.arange(Nz), indexing="ij")
        b1x = torch.from_numpy(label(kx, y, z).astype(np.float64).ravel())
        b1y = torch.full((npl * Ny * Nz,), -1.0, dtype=torch.float64)
        _exchange(rank, world, b1x, b1y, N, 0)
        kx, y, z = np.meshgrid(k0 + np.arange(npl), np.arange(Ny), np.arange(Nz), indexing="ij")
        ok_fwd = bool(np.array_equal(b1y.numpy(), label(kx, y, z).astype(np.float64).ravel()))
        back = torch.full_like(b1x, -2.0)
        _exchange(rank, world, b1y, back, N, 1)
        ok_bwd = bool(torch.equal(back, b1x))
        ret[rank] = (ok_fwd, ok_bwd, k0, npl)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("N", [(8, 8, 8), (16, 4, 6)])
def test_shard_blocks_through_a_world_size_2_exchange(N):
    world = 2
    with mp.Manager() as m:
        ret = m.dict()
        mp.spawn(_worker, args=(world, 29500 + (os.getpid() + sum(N)) % 2000, N, ret), nprocs=world, join=True)
        res = dict(ret)
    assert all(res[r][0] and res[r][1] for r in range(world)), res
    # the slabs of planes are contiguous, disjoint and cover 0 .. Nx
    planes = sorted((res[r][2], res[r][3]) for r in range(world))
    assert planes[0][0] == 0 and planes[0][0] + planes[0][1] == planes[1][0] and planes[1][0] + planes[1][1] == N[0] + 1


def test_shard_layout_properties_for_any_rank_count():
    """Host-only: for P = 1 .. 16 the blocks of all (src, dst) pairs tile both workspaces exactly once."""
    Nx, Ny, Nz = 32, 48, 5
    for P in (1, 2, 3, 4, 6, 8, 12, 16):
        yl = Ny // P
        tot = 0
        for r in range(P):
            k0, npl = binding.shard_planes(Nx, P, r)
            tot += npl
            cover = np.zeros(npl * Ny * Nz, dtype=np.int32)          # B1y of rank r as a forward destination
            for s in range(P):
                nrun, run_len, so, ss, do, ds = binding.shard_block(Nx, Ny, Nz, P, s, r, 0)
                assert nrun == npl and run_len == yl * Nz and ss == yl * Nz and so == k0 * yl * Nz
                for i in range(nrun):
                    cover[do + i * ds: do + i * ds + run_len] += 1
            assert (cover == 1).all()
            cover = np.zeros((Nx + 1) * yl * Nz, dtype=np.int32)      # B1x of rank r as a backward destination
            for s in range(P):
                nrun, run_len, so, ss, do, ds = binding.shard_block(Nx, Ny, Nz, P, s, r, 1)
                for i in range(nrun):
                    cover[do + i * ds: do + i * ds + run_len] += 1
            assert (cover == 1).all()
        assert tot == Nx + 1
    with pytest.raises(binding.FspError):
        binding.shard_block(Nx, Ny, Nz, 5, 0, 0, 0)    # Ny % P != 0
