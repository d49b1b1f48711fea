"""Worker for tests/test_multi_rank.py: run under torch.distributed.run with the gloo backend (CPU).
Exercises the multi-rank plumbing bench.py uses for its weak-scaling replicas: rendezvous, barrier,
max-over-ranks timing and the whole-job aggregation.  No GPU, no oracle, no kernels."""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

import bench  # noqa: E402
import synth_inputs as si  # noqa: E402


def main():
    rank, world, local = bench.dist_setup(world_hint := int(os.environ.get("WORLD_SIZE", "1")))
    assert world == world_hint and 0 <= rank < world and local == rank
    dev = torch.device("cpu")
    bench.barrier(world)
    # every rank "measures" a different step time; the job time is the slowest rank's
    my_ms = 10.0 + 5.0 * rank
    job_ms = bench.max_over_ranks(my_ms, world, dev)
    assert job_ms == 10.0 + 5.0 * (world - 1), job_ms
    # replicas only: each rank runs the full config-3 batch, no data-path collective
    fl = bench.flops_of(si.CFG3)
    value = world * fl / (job_ms * 1e-3) / 1e12
    bench.barrier(world)
    if rank == 0:
        print(json.dumps({"world": world, "job_ms": job_ms, "value": value, "per_rank_flops": fl}), flush=True)
    import torch.distributed as dist
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
