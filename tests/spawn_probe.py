"""Helper of tests/test_dist_gloo.py (not a test): a stand-in for bench.py's `--gpus N` start-up on CPU.  Started WITHOUT a
launcher it must start N ranks itself (paper_2607_02584_b200.dist.relaunch_under_torchrun); each rank joins a gloo group
and rank 0 prints ONE JSON line with the number of ranks that took part."""
import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument('--gpus', type=int, default=1)
    args = ap.parse_args()
    from paper_2607_02584_b200 import dist as rd
    if rd.needs_relaunch(args.gpus):
        sys.exit(rd.relaunch_under_torchrun(args.gpus, os.path.abspath(__file__), sys.argv[1:]))
    import torch
    import torch.distributed as dist
    world, rank = int(os.environ.get('WORLD_SIZE', '1')), int(os.environ.get('RANK', '0'))
    if world > 1:
        dist.init_process_group('gloo')
    mine = rd.shard_heads(12, world, rank)
    total = rd.aggregate_throughput(len(mine), 1.0 + rank) * 1e-3 * (1.0 + (world - 1))     # units of all ranks
    if rank == 0:
        print(json.dumps({'n_ranks': world, 'units': round(total), 'slowest_ms': rd.max_over_ranks(1.0 + rank)}))
    else:
        rd.max_over_ranks(1.0 + rank)
    if world > 1:
        dist.destroy_process_group()


if __name__ == '__main__':
    main()
