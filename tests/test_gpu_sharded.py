"""-m gpu: the slab-decomposed solve (include/fsp.h "slab decomposition") against the single-GPU solve
and the oracle.  One device stands in for P ranks WITHOUT any kernel waiting on another: the P sharded plans live in
one process, their transpose targets are plain device pointers, and the three phases are run for all ranks in turn
with a device synchronisation between phases (what the barriers do on a real node)."""
import numpy as np
import pytest

import oracle
from paper_2405_02603_b200 import binding, workloads as W
from tests.analytic import rel_l2, rel_max

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def sharded_solve(N, h, alg, P, rho_np):
    plans = [binding.ShardedPlan(N, h, alg, r, P) for r in range(P)]
    try:
        bufs = [p.buffers() for p in plans]
        for p in plans:
            p.precompute_green()
            p.set_peers([b[0] for b in bufs], [b[1] for b in bufs])
        yl = N[1] // P
        rho = torch.from_numpy(rho_np).cuda()
        slabs = [rho[:, r * yl:(r + 1) * yl, :].contiguous() for r in range(P)]
        outs = [torch.empty_like(s) for s in slabs]
        for ph in range(3):
            for r, p in enumerate(plans):
                p.phase(ph, slabs[r], outs[r])
            torch.cuda.synchronize()     # = the barrier between phases on a real node
        return torch.cat(outs, dim=1).cpu().numpy(), sum(p.bytes for p in plans)
    finally:
        for p in plans:
            p.destroy()


@pytest.mark.parametrize("N,P,alg", [((64, 64, 64), 2, "HE"), ((64, 64, 64), 4, "VG2"), ((32, 16, 64), 8, "HE"),
                                     ((256, 256, 64), 2, "HE"), ((128, 256, 256), 4, "VG2"), ((16, 64, 512), 3, None)])
def test_sharded_solve_equals_single_gpu_solve_and_oracle(N, P, alg):
    if alg is None:   # Ny % P != 0 is refused
        with pytest.raises(binding.FspError):
            binding.ShardedPlan(N, (0.1,) * 3, binding.HOCKNEY, 0, P)
        return
    w = W.random_density(N, seed=sum(N) + P)
    balg, oalg = (binding.HOCKNEY, oracle.HOCKNEY) if alg == "HE" else (binding.VICO_2, oracle.VICO_2)
    got, shard_bytes = sharded_solve(w.N, w.h, balg, P, w.rho)
    with binding.Plan(w.N, w.h, balg) as p:
        single = p.precompute_green().solve(torch.from_numpy(w.rho).cuda()).cpu().numpy()
        single_bytes = p.bytes
    ref = oracle.OraclePlan(w.N, w.h, oalg).precompute_green().solve(w.rho)
    assert np.isfinite(got).all()
    assert rel_l2(got, ref) <= 1e-12 and rel_max(got, ref) <= 1e-10
    assert rel_max(got, single) <= 1e-14      # same kernels on the same numbers, plane by plane
    assert shard_bytes > 0 and single_bytes > 0


def test_sharded_phases_need_peers_and_spectrum():
    N, h = (32, 32, 32), (0.1,) * 3
    with binding.ShardedPlan(N, h, binding.HOCKNEY, 0, 2) as p:
        rho = torch.zeros(p.slab, dtype=torch.float64, device="cuda")
        with pytest.raises(binding.FspError):
            p.phase(0, rho, rho)              # peers not set
        a = p.buffers()
        with pytest.raises(binding.FspError):
            p.set_peers([a[0], 0], [a[1], 0])  # null peer
        p.set_peers([a[0], a[0]], [a[1], a[1]])
        with pytest.raises(binding.FspError) as e:
            p.phase(0, rho, rho)
        assert e.value.code == -2             # not precomputed


def test_two_processes_share_one_device_through_ipc_handles():
    """The launch a multi-GPU node would use (torchrun, one process per rank, workspace addresses exchanged as CUDA IPC
    handles, barriers between the phases), with both ranks on this box's one device and gloo barriers: no kernel waits
    on another process's kernel.  Checks the IPC path and the assembled field against the single-GPU solve."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    port = 29600 + os.getpid() % 300
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(root, "bench.py"), "--sharded", "--gpus", "2", "--workload", "64", "--steps", "2",
           "--warmup", "1"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=root)
    assert res.returncode == 0, res.stderr[-2000:]
    line = json.loads([l for l in res.stdout.splitlines() if l.startswith("{")][-1])
    assert line["mode"] == "sharded" and line["n_gpus"] == 2
    assert line["max_rel_diff_vs_single_gpu_solve"] <= 1e-14
