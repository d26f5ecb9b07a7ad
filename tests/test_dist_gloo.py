"""N > 1 path on CPU: world_size-2 gloo processes check the head sharding (no data-path collective) and
the max-over-ranks / whole-job aggregation bench.py relies on."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip('torch')
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402


def _free_port():
    with socket.socket() as s:
        s.bind(('127.0.0.1', 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR='127.0.0.1', MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group('gloo', rank=rank, world_size=world)
    from paper_2607_02584_b200 import dist as rd
    heads = rd.shard_heads(25, world, rank)                       # 25 units over 2 ranks: 13 + 12
    gathered = [None] * world
    dist.all_gather_object(gathered, heads.tolist())
    ms = rd.max_over_ranks(3.0 + rank)                            # rank 1 is the slow one
    thr = rd.aggregate_throughput(len(heads), 3.0 + rank)
    if rank == 0:
        out.put((gathered, ms, thr))
    dist.destroy_process_group()


def test_world_size_2_head_sharding_and_timing():
    ctx = mp.get_context('spawn')
    out = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    gathered, ms, thr = out.get()
    assert gathered[0] == list(range(0, 13)) and gathered[1] == list(range(13, 25))   # disjoint, contiguous, complete
    assert ms == 4.0                                              # max over ranks
    assert abs(thr - 25 / 4.0e-3) < 1e-6                          # all units / slowest rank's time


def test_shard_heads_properties():
    from paper_2607_02584_b200 import dist as rd
    for n in (0, 1, 7, 12, 40, 41):
        for w in (1, 2, 3, 8):
            parts = [rd.shard_heads(n, w, r) for r in range(w)]
            cat = np.concatenate(parts)
            assert cat.tolist() == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    with pytest.raises(ValueError):
        rd.shard_heads(4, 2, 2)


def test_gpus_flag_starts_the_ranks_itself():
    """`--gpus 2` without a launcher (no WORLD_SIZE): the program starts two ranks and ONE line comes out, saying 2."""
    import json
    import subprocess
    import sys
    from paper_2607_02584_b200 import dist as rd
    assert rd.needs_relaunch(2, env={}) and not rd.needs_relaunch(1, env={}) and not rd.needs_relaunch(2, env={'WORLD_SIZE': '2'})
    argv = rd.torchrun_argv(4, 'bench.py', ['--gpus', '4'], port=1234)
    assert argv[1:] == ['-m', 'torch.distributed.run', '--nnodes=1', '--nproc-per-node', '4', '--master-addr', '127.0.0.1',
                        '--master-port', '1234', 'bench.py', '--gpus', '4']
    env = {k: v for k, v in os.environ.items() if k not in ('WORLD_SIZE', 'RANK', 'LOCAL_RANK', 'MASTER_ADDR', 'MASTER_PORT')}
    probe = os.path.join(os.path.dirname(os.path.abspath(__file__)), 'spawn_probe.py')
    r = subprocess.run([sys.executable, probe, '--gpus', '2'], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(x) for x in r.stdout.splitlines() if x.startswith('{')]
    assert lines == [{'n_ranks': 2, 'units': 12, 'slowest_ms': 2.0}], r.stdout
