"""CPU checks of the N > 1 host path of bench.py ("replicas only"): two processes, gloo backend,
rendezvous on 127.0.0.1.  The data path has no collective; the only exchange is the MAX over ranks of the timings."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms_step, region_ms, e2e_ms = [(100.0, 130.0, 140.0), (125.0, 128.0, 135.0)][rank]      # rank 1 is slower per step
    a, b = bench.reduce_max_over_ranks([ms_step, region_ms], world)
    c = bench.reduce_max_over_ranks([e2e_ms], world)[0]
    out[rank] = (a, b, c, bench.job_value(1000, world, a))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_job_value_world2():
    import torch.multiprocessing as mp
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for r in (0, 1):
        a, b, c, v = res[r]
        assert a == 125.0 and b == 130.0 and c == 140.0          # element-wise max, identical on both ranks
        assert v == pytest.approx(2 * 1000 / 0.125)              # two replicas in the time of the slower one


def _shard_worker(rank, world, port, out):
    """One rank of the sharded build's host path on CPU: shard_of() -> (rank, world); a partial J, K (here from the
    oracle's loop over this rank's share of the bra pairs; on a GPU from adft_jk_build_ex with shard_rank/shard_count);
    allreduce_jk() sums them in place over the group."""
    import numpy as np
    import torch
    import torch.distributed as dist
    import oracle
    from paper_2406_11185_b200 import api, workloads as W
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    assert api.shard_of() == (rank, world)
    w = W.make("0b")
    bs = oracle.basis_from_workload(w)
    Q = oracle.schwarz(bs)
    npair = bs.nshells * (bs.nshells + 1) // 2
    lo, hi = rank * npair // world, (rank + 1) * npair // world
    Jp, Kp, cnt = oracle.jk_range(bs, w.D, w.tau, Q, lo, hi)
    J = torch.from_numpy(np.asarray(Jp, np.float64)); K = torch.from_numpy(np.asarray(Kp, np.float64))
    api.allreduce_jk(J, K)
    api.allreduce_jk(J.clone(), None)                   # a J-only build reduces one matrix
    out[rank] = (J.numpy().copy(), K.numpy().copy(), cnt["kept"])
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_build_allreduce_world2():
    import numpy as np
    import torch.multiprocessing as mp
    import oracle
    from paper_2406_11185_b200 import workloads as W
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_shard_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    w = W.make("0b")
    bs = oracle.basis_from_workload(w)
    Jo, Ko, cnt = oracle.jk(bs, w.D, w.tau)
    assert res[0][2] + res[1][2] == cnt["kept"] and res[0][2] > 0 and res[1][2] > 0
    for r in (0, 1):                                     # every rank ends with the full matrices
        assert np.abs(res[r][0] - Jo).max() <= 1e-12 and np.abs(res[r][1] - Ko).max() <= 1e-12
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1])


def test_shard_of_without_process_group():
    from paper_2406_11185_b200 import api
    assert api.shard_of() == (0, 1)
    api.allreduce_jk(None, None)                         # no group: nothing to do


def test_world1_is_identity():
    import bench
    assert bench.reduce_max_over_ranks([3.5, 7.25], 1) == [3.5, 7.25]
    assert bench.job_value(10, 1, 500.0) == pytest.approx(20.0)


def test_reference_arm_other_ranks_exit_without_work():
    """--impl reference under torchrun: rank 0 alone runs and prints; the other ranks exit 0 and print nothing."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_reference_arm_rank0_line():
    env = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "quartets/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
