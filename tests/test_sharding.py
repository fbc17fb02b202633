"""Target-sharded evaluation on several GPUs.  One GPU is all any run here has,
so: the partition (host arithmetic) is checked on the CPU, alone and across a world_size-2 gloo group; on the GPU the
ranks are played ONE AFTER ANOTHER on the single device (no kernel ever waits for another rank) and their partial
forces must add up bit-exactly to the one-GPU evaluation; and two processes sharing the one GPU run sharded MD steps
through the real torch.distributed callback (gloo carries the CUDA tensors) and must reproduce the unsharded
trajectory bit for bit."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

import paper_1412_8502_b200 as pasta
from paper_1412_8502_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    import socket

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("N,Np,cp,cn,world", [(409600, 122880, 3.1, 1.0, 8), (51200, 20480, 2.0, 1.0, 3), (2048, 0, 1.0, 1.0, 4),
                                               (2048, 2048, 5.0, 1.0, 5), (7, 3, 1.0, 1.0, 16), (1000, 1, 100.0, 1.0, 2)])
def test_shard_bounds_cover_and_balance(N, Np, cp, cn, world):
    b = pasta.shard_bounds(N, Np, cp, cn, world)
    assert len(b) == world + 1 and b[0] == 0 and b[-1] == N
    assert all(b[r] <= b[r + 1] for r in range(world))                     # contiguous, disjoint, complete
    cost = lambda lo, hi: cp * (min(hi, Np) - min(lo, Np)) + cn * (max(hi, Np) - max(lo, Np))
    total = cost(0, N)
    for r in range(world):                                                 # every rank within one target of its share
        assert abs(cost(b[r], b[r + 1]) - total / world) <= max(cp, cn) + 1e-9
    assert pasta.shard_bounds(N, Np, cp, cn, 1) == [0, N]
    for bad in ((0, 0, 1.0, 1.0, 2), (10, 11, 1.0, 1.0, 2), (10, 5, 0.0, 1.0, 2), (10, 5, 1.0, 1.0, 0)):
        with pytest.raises(pasta.PastaError):
            pasta.shard_bounds(*bad)


GLOO_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import paper_1412_8502_b200 as pasta
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
b = pasta.shard_bounds(409600, 122880, 3.1, 1.0, world)
mine = torch.tensor([b[rank], b[rank + 1]], dtype=torch.int64)
every = [torch.zeros(2, dtype=torch.int64) for _ in range(world)]
dist.all_gather(every, mine)
# what the force all-reduce does with partial results: every particle is non-zero on exactly one rank
F = torch.zeros(409600, dtype=torch.float64)
F[b[rank]:b[rank + 1]] = torch.arange(b[rank], b[rank + 1], dtype=torch.float64) + 0.25
dist.all_reduce(F)
if rank == 0:
    print(json.dumps({"ranges": [e.tolist() for e in every], "ok": bool(torch.equal(F, torch.arange(409600, dtype=torch.float64) + 0.25))}))
dist.destroy_process_group()
"""


def test_partition_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(GLOO_WORKER % ROOT)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), str(script)]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=240, env=dict(os.environ, OMP_NUM_THREADS="1"))
    assert out.returncode == 0, out.stderr[-2000:]
    d = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    (a0, a1), (b0, b1) = d["ranges"]
    assert a0 == 0 and a1 == b0 and b1 == 409600 and d["ok"]


@pytest.mark.gpu
@pytest.mark.parametrize("cfg_like,world,paper_mode", [((20000, 0.3, 0.05, 17.0), 3, False), ((30000, 0.05, 0.002, 20.0), 4, False),
                                                       ((20000, 0.4, 0.01, 20.0), 3, True)])
def test_ranks_played_in_turn_add_up_bit_exactly(orc, cfg_like, world, paper_mode):
    """Dense chunk path, (second case: cold, dilute, wide box) the neighbour-list path, and (third) the paper's range
    split with the all-pairs Coulomb kernel, whose proton targets are sharded by the same window."""
    import torch

    N, Y_P, density, r_c = cfg_like
    p = pasta.default_params(r_c=r_c, r_nuc=11.5, coulomb_all_pairs=1) if paper_mode else pasta.default_params(r_c=r_c)
    with pasta.Sim(N, Y_P, density, 0.5, params=p, seed=5) as sim:
        F1, pe1 = sim.forces()
        e1 = sim.particle_energies().clone()
        calls = []
        parts, eparts = [], []
        for r in range(world):
            sim.set_shard(r, world, allreduce=lambda t: calls.append(t.numel()))   # a "collective" that adds nothing
            F, _ = sim.forces()
            parts.append(F.clone())
            eparts.append(sim.particle_energies().clone())
        assert calls == [4 * N] * world   # forces and energies are summed as one contiguous run: one collective per evaluation
        owners = sum((q != 0).any(dim=1).to(torch.int32) for q in parts)
        # every particle on exactly one rank (in the paper's mode too: the all-pairs Coulomb kernel takes a proton's owner
        # from its chunk, so that nuclear and Coulomb parts are added on one rank in the one-GPU order)
        assert int(owners.max()) == 1 and int((owners == 0).sum()) <= 2
        assert torch.equal(sum(parts), F1) and torch.equal(sum(eparts), e1)
        # ... and the sharded evaluation against the ORACLE, at the gates of the unsharded parity tests (D17, D22)
        from test_gpu_parity import PE_TOL, _alts, _check_forces, _np, _oparams

        xs, _, is_p, L, _ = sim.get_state()
        xs, is_p = _np(xs), _np(is_p)
        op = orc.Params(r_c=r_c, r_nuc=11.5, coul_nocut=1.0) if paper_mode else _oparams(orc, sim.params)
        Fo, eo, peo, d = orc.forces(xs, is_p, L, op)
        _check_forces(_np(sum(parts)), Fo, alternates=None if paper_mode else _alts(orc, xs, is_p, L, op),
                      boundary_pairs=d["boundary_pairs"])
        assert abs(float(sum(eparts).sum()) - peo) <= PE_TOL * abs(peo)
        Np = int(sim.get_state()[2].sum())
        b = pasta.shard_bounds(N, Np, *sim.shard_costs(), world)
        sizes = [int((q != 0).any(dim=1).sum()) for q in parts]
        # ownership goes by a chunk's FIRST target; a chunk of the cell-block builder gathers slots of several rows
        assert N - 2 <= sum(sizes) <= N and all(abs(sizes[r] - (b[r + 1] - b[r])) <= 0.05 * N for r in range(world))
        sim.set_shard(0, 1)
        F, pe = sim.forces()
        assert torch.equal(F, F1) and pe == pe1


SHARD_WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import paper_1412_8502_b200 as pasta
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
torch.cuda.set_device(0)                      # both ranks share the one GPU; only the HOST waits in the collective
cases = {
    "dense": (6000, 0.3, 0.05, dict(r_c=17.0, thermostat_interval=5), 12),
    "dilute_lists_scaling_box": (8000, 0.2, 0.001, dict(r_c=20.0, thermostat_interval=5, scale_per_step=1.0004), 40),
    "paper_mode": (5000, 0.4, 0.0028, dict(r_c=20.0, r_nuc=11.5, coulomb_all_pairs=1, thermostat_interval=4), 10),
}
out = {}
for name, (N, Y_P, density, prm, steps) in cases.items():
    sim = pasta.Sim(N, Y_P, density, 0.5, params=pasta.default_params(**prm), seed=3)
    if world > 1:
        sim.set_shard(rank, world)
    sim.step(steps, 2.0)
    x, v, _, L, step = sim.get_state()
    F, pe = sim.forces()
    ke, pe2 = sim.energy()
    out[name] = {"x": x.cpu(), "v": v.cpu(), "F": F.cpu(), "pe": pe, "ke": ke, "L": L, "stats": sim.list_stats()}
    dist.barrier()
    sim.close()
if rank == 0:
    torch.save(out, sys.argv[1])
dist.barrier()
dist.destroy_process_group()
"""


@pytest.mark.gpu
def test_two_sharded_processes_reproduce_the_unsharded_trajectory(tmp_path):
    import torch

    script = tmp_path / "worker.py"
    script.write_text(SHARD_WORKER % ROOT)
    res = {}
    for world in (1, 2):
        out_file = tmp_path / ("w%d.pt" % world)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=%d" % world, "--master-addr",
               "127.0.0.1", "--master-port", str(_free_port()), str(script), str(out_file)]
        out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=dict(os.environ, OMP_NUM_THREADS="1"))
        assert out.returncode == 0, out.stderr[-3000:]
        res[world] = torch.load(out_file)
    for case in res[1]:
        one, two = res[1][case], res[2][case]
        for k in ("x", "v", "F"):
            assert torch.equal(one[k], two[k]), (case, k)
        assert one["pe"] == two["pe"] and one["ke"] == two["ke"] and one["L"] == two["L"] and one["stats"] == two["stats"], case
    assert res[1]["dilute_lists_scaling_box"]["stats"]["list_builds"] < 20   # that case really ran on reused lists
