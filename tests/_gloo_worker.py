"""Worker of tests/test_multirank_cpu.py: the host logic of `bench.py --gpus N` ("replicas
only": one block per rank, no data-path collective) on a world of 2 CPU ranks over gloo."""
import os
import sys

import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    assert world == 2
    # each rank measured its own replica: the job's time is the slowest rank's
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, torch.device("cpu"))
    assert ms == 15.0, ms
    # whole-job value = units of all ranks / that time (weak scaling: work per rank fixed)
    v = bench.whole_job_value(ncells=1000, stages=3, steps=2, world=world, ms=ms)
    assert abs(v - 2 * 1000 * 3 * 2 / 15e-3) < 1e-6 * v
    # the workload generator is seeded: every rank builds the same block, no exchange needed
    from paper_2406_11669_b200 import workloads as wl
    w = wl.make(1, 8)
    t = torch.from_numpy(w.prims[0]).clone()
    ref = t.clone()
    dist.broadcast(ref, src=0)
    assert torch.equal(t, ref)
    dist.barrier()
    if rank == 0:
        print("GLOO_OK")
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
