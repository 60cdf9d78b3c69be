"""N > 1 host logic on CPU: world_size-2 gloo run of the sharding helpers."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys, importlib.util
    import numpy as np, torch, torch.distributed as dist
    sys.path.insert(0, %r)
    spec = importlib.util.spec_from_file_location("sharding", os.path.join(%r, "paper_2605_08916_b200", "sharding.py"))
    sharding = importlib.util.module_from_spec(spec); spec.loader.exec_module(sharding)
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    # contiguous global id ranges cover every chain exactly once
    n_total = 1001
    b, e = sharding.shard_range(n_total, rank, world)
    ids = torch.zeros(n_total, dtype=torch.int64); ids[b:e] = 1
    dist.all_reduce(ids)
    assert (ids == 1).all()
    assert sharding.shard_offset(589824, rank) == 589824 * rank
    # the per-resolve exchange: sum of the private accumulation buffers and of the counters
    rng = np.random.default_rng(rank)
    acc = torch.from_numpy(rng.random((64, 4)).astype(np.float32))
    tot, tours, muts = sharding.allreduce_totals(acc, 10 + rank, 100 * (rank + 1))
    want = sum(torch.from_numpy(np.random.default_rng(r).random((64, 4)).astype(np.float32)) for r in range(world))
    assert torch.allclose(tot, want) and tours == sum(10 + r for r in range(world)) and muts == sum(100 * (r + 1) for r in range(world))
    assert torch.equal(acc, torch.from_numpy(np.random.default_rng(rank).random((64, 4)).astype(np.float32)))  # input untouched
    # counters as 16-bit limbs in an fp32 buffer: the sum over ranks is exact (what k_pack_frame / k_resolve rely on)
    mine = [2**40 + 65535 * (rank + 1), 2**33 - 1 - rank]
    t = torch.tensor(sharding.limbs(mine[0]) + sharding.limbs(mine[1]), dtype=torch.float32)
    dist.all_reduce(t)
    assert sharding.from_limbs(t[:4]) == sum(2**40 + 65535 * (r + 1) for r in range(world))
    assert sharding.from_limbs(t[4:]) == sum(2**33 - 1 - r for r in range(world))
    dist.destroy_process_group()
    print("ok", rank)
""") % (ROOT, ROOT)


def test_two_rank_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), LOCAL_RANK=str(r))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    for p in procs:
        out, _ = p.communicate(timeout=240)
        assert p.returncode == 0, out
        assert "ok" in out
