"""N>1 path on CPU: two gloo ranks, each running its shard (keyed by global game index);
the gathered result must equal the unsharded run.  Exercises the shard description that
bench.py uses under torchrun (workloads.shard_for_rank) with the oracle as the engine."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2511_07312_b200 import workloads as W

CFG = dict(name="shard_test", variant=0, num_games=48, seed=5, max_plies=60, auto_reset=1)
STEPS = 130


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _play(env, steps):
    rewards = []
    for _ in range(steps):
        r, d = env.step(env.sample_uniform(env.legal_mask()))
        rewards.append(r.copy())
    return env.get_boards(), np.stack(rewards)


def _worker(rank, world, port, out_path):
    from oracle import orc
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    kw = W.shard_for_rank(CFG, rank, world)
    env = orc.Env(CFG["num_games"], **kw)
    boards, rewards = _play(env, STEPS)
    t = torch.from_numpy(boards)
    gathered = [torch.empty_like(t) for _ in range(world)]
    dist.all_gather(gathered, t)           # test plumbing only: the data path has no collective
    elapsed = torch.tensor([float(rank + 1)])
    dist.all_reduce(elapsed, op=dist.ReduceOp.MAX)  # bench.py's only reduction: max time
    if rank == 0:
        np.save(out_path, torch.cat(gathered).numpy())
        assert elapsed.item() == float(world)
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shards_equal_unsharded_run(tmp_path):
    from oracle import orc
    world = 2
    out = str(tmp_path / "gathered.npy")
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    sharded = np.load(out)
    full = orc.Env(world * CFG["num_games"], variant=CFG["variant"], seed=CFG["seed"],
                   max_plies=CFG["max_plies"], auto_reset=1)
    boards, _ = _play(full, STEPS)
    assert np.array_equal(sharded, boards)
    assert (boards[:, 124] >= 2).all()  # every game went through at least two auto-resets


def test_shard_description():
    a = W.shard_for_rank(W.CONFIGS[2], 0, 8)
    b = W.shard_for_rank(W.CONFIGS[2], 7, 8)
    assert a["game_base"] == 0 and b["game_base"] == 7 * 65536
    assert {k: v for k, v in a.items() if k != "game_base"} == {k: v for k, v in b.items() if k != "game_base"}


def test_sharded_oracle_plumbing_equals_one_oracle():
    """tests/oracle_shards.py (the all-games parity plumbing of the -m gpu tests): three worker
    processes over a ragged split reproduce the single-process oracle output by output."""
    from oracle import orc
    from oracle_shards import ShardedOracle
    n, kw = 150, dict(variant=0, seed=9, max_plies=30, auto_reset=1)
    one = orc.Env(n, **kw)
    with ShardedOracle(n, procs=3, with_obs_before=True, **kw) as sh:
        assert len(sh._workers) == 3
        for t in range(45):
            ob = one.encode_obs().reshape(n, -1)
            m = one.legal_mask(); a = one.sample_uniform(m); r, d = one.step(a)
            sh.step(want_mask=True, want_obs_before=True, want_obs_after=True, want_boards=True)
            assert np.array_equal(sh.act, a) and np.array_equal(sh.rew, r) and np.array_equal(sh.done, d), t
            assert np.array_equal(sh.mask, m) and np.array_equal(sh.obs_before, ob), t
            assert np.array_equal(sh.obs, one.encode_obs().reshape(n, -1)), t
            assert np.array_equal(sh.boards, one.get_boards()), t
        assert np.array_equal(sh.get_boards(), one.get_boards())


def test_bench_gpus_n_starts_n_ranks_by_itself():
    """`python bench.py --gpus 2` with no launcher around it re-executes itself under torch.distributed.run
    with two ranks on 127.0.0.1.  Checked without a GPU on the reference arm: both
    ranks report in over gloo, rank 0 alone times the oracle and prints the one JSON line."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=600, env=env, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(x) for x in out.stdout.splitlines() if x.startswith("{")]
    assert len(lines) == 1
    assert lines[0]["impl"] == "reference" and lines[0]["n_gpus"] == 2
    assert lines[0]["config"]["ranks_started"] == 2
    assert lines[0]["value"] > 0
    # a workload that does not shard says so instead of starting ranks
    bad = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--workload", "cfg4"],
                         capture_output=True, text=True, timeout=120, env=env, cwd=root)
    assert bad.returncode != 0 and "cfg2" in bad.stderr
