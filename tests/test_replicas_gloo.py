"""N > 1 path on CPU: world_size-2 `gloo` processes exercise the replica plumbing bench.py uses
(rank -> configuration, barrier, max-over-ranks time, whole-job aggregate).  The path shards by
independent configurations with no data-path collective ("Multi-GPU")."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys, time
sys.path.insert(0, %(root)r)
import numpy as np
import gf_inputs as gi
from paper_1305_3440_b200.replicas import Replicas

rep = Replicas(backend="gloo")
assert rep.world == 2
seed = rep.config_seed(1)
U = gi.smooth_random_gauge((4, 4, 4, 4), 0.3, seed)          # this rank's own configuration
rep.barrier()
t_mine = 0.010 * (rep.rank + 1)                               # rank 1 is the slow one
t_max = rep.max_over_ranks(t_mine)
units = 1000 * (rep.rank + 1)
out = {"rank": rep.rank, "seed": seed, "items": rep.my_items(5), "t_max": t_max,
       "thr": rep.job_throughput(units, t_mine), "sum": rep.sum_over_ranks(units),
       "checksum": float(np.abs(U).sum()), "root": rep.is_root}
rep.barrier()
print("RESULT " + json.dumps(out), flush=True)
rep.close()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def test_two_rank_replica_plumbing(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % {"root": ROOT})
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    res = {}
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        line = [l for l in out.splitlines() if l.startswith("RESULT ")][0]
        r = json.loads(line[len("RESULT "):])
        res[r["rank"]] = r
    assert res[0]["seed"] == 1 and res[1]["seed"] == 2                   # one configuration per rank
    assert res[0]["checksum"] != res[1]["checksum"]
    assert res[0]["items"] == [0, 2, 4] and res[1]["items"] == [1, 3]    # ensemble split, no overlap
    for r in res.values():
        assert r["t_max"] == pytest.approx(0.020)                          # slowest rank
        assert r["sum"] == 3000.0
        assert r["thr"] == pytest.approx(3000.0 / 0.020)                   # all ranks' units / max time
    assert res[0]["root"] and not res[1]["root"]


def test_single_process_is_a_no_op():
    sys.path.insert(0, ROOT)
    from paper_1305_3440_b200.replicas import Replicas
    env = {k: os.environ.pop(k) for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK") if k in os.environ}
    try:
        rep = Replicas()
        assert rep.world == 1 and rep.rank == 0 and rep.is_root
        assert rep.config_seed(7) == 7 and rep.my_items(3) == [0, 1, 2]
        assert rep.max_over_ranks(1.5) == 1.5 and rep.job_throughput(10, 2.0) == 5.0
        rep.barrier()
        rep.close()
    finally:
        os.environ.update(env)


def test_bench_reference_arm_runs_on_rank0_only():
    """Under torchrun the reference arm prints on rank 0 and the other ranks exit 0 without work."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


# ---------------------------------------------------------------- slab decomposition, host logic

SLAB_WORKER = r"""
import json, os, sys
sys.path.insert(0, %(root)r)
import torch.distributed as dist
import paper_1305_3440_b200 as gf
from paper_1305_3440_b200.slabs import SlabRank, local_dims, neighbours

dist.init_process_group("gloo")
rank = dist.get_rank()


class FakeSlab:
    # this slab's share of theta falls by 10x per iteration; rank 1's share is 3x rank 0's
    def __init__(self, gauge):
        self.gauge, self.it, self.ops = gauge, 0, []
    def iterate(self, n, *a):
        self.it += n
        self.ops.append(("iterate", n))
    def measure(self, precision):
        self.ops.append(("measure",))
        th = (1 + 2 * rank) * 10.0 ** (-self.it)
        if self.gauge == gf.GF_COULOMB:
            return [0.5, 0.5], [th, th / 2]
        return [0.25 * (rank + 1)], [th]

out = {"rank": rank}
lan = SlabRank((8, 4, 4, 4), gauge=gf.GF_LANDAU, _field=FakeSlab(gf.GF_LANDAU))
out["dims"] = list(lan.dims)
out["nb"] = list(neighbours(lan.rank, lan.nslabs))
F, th = lan.measure(gf.GF_F64)
out["F"], out["th0"] = F[0], th[0]
out["fix"] = list(lan.fix_until(gf.GF_OVERRELAX, 1.7, 0.0, gf.GF_F64, 1e-6, 100, 2))
out["ops"] = lan.field.ops
cou = SlabRank((8, 4, 4, 4), gauge=gf.GF_COULOMB, _field=FakeSlab(gf.GF_COULOMB))
out["fixc"] = list(cou.fix_until(gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64, 2e-4, 3, 1))
out["fixc_nc"] = list(SlabRank((8, 4, 4, 4), gauge=gf.GF_COULOMB, _field=FakeSlab(gf.GF_COULOMB)).fix_until(
    gf.GF_STOCHASTIC, 1.0, 0.8, gf.GF_F64, 1e-30, 3, 2))
print("RESULT " + json.dumps(out), flush=True)
dist.destroy_process_group()
"""


def test_two_rank_slab_host_logic(tmp_path):
    """SlabRank's control flow under gloo with a stand-in slab: slab geometry, the scalar all-reduce of
    F and theta, and a stopping decision that is the same on every rank (so that all slabs keep
    issuing the same sequence of operations, which gf_set_slab's ordering requires)."""
    script = tmp_path / "slab_worker.py"
    script.write_text(SLAB_WORKER % {"root": ROOT})
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    res = {}
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        r = json.loads([l for l in out.splitlines() if l.startswith("RESULT ")][0][len("RESULT "):])
        res[r["rank"]] = r
    assert res[0]["dims"] == [4, 4, 4, 4] and res[0]["nb"] == [1, 1] and res[1]["nb"] == [0, 0]
    for r in res.values():
        assert r["F"] == pytest.approx(0.75) and r["th0"] == pytest.approx(4.0)      # shares added up
        # theta = 4 * 10^-it, checked every 2 iterations: 4e-8 < 1e-6 first at it = 8 on BOTH ranks
        assert r["fix"][0] == 0 and r["fix"][1] == 8 and r["fix"][2] == pytest.approx(4e-8)
        # Coulomb: max over all slices of all slabs = rank 1's 3 * 10^-it: below 2e-4 at it = 5 > max_iter 3
        assert r["fixc"][0] == 1 and r["fixc"][1] == 3 and r["fixc"][2] == pytest.approx(3e-3)
        assert r["fixc_nc"][1] == 3                                                   # last block is shortened
    assert res[0]["ops"] == res[1]["ops"]                                             # same operation sequence
    assert res[0]["ops"][:3] == [["measure"], ["iterate", 2], ["measure"]]
