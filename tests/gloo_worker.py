"""world_size-2 CPU check of the N > 1 plumbing of bench.py (launched by test_library_host.py under torchrun):
rendezvous on 127.0.0.1, barrier, and the max-over-ranks reduction of the per-rank step time (gloo here, nccl
on the GPU box).  The path itself is "replicas only": no data-path collective exists."""
import torch
import torch.distributed as dist

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
dist.barrier()
t = torch.tensor([10.0 + rank], dtype=torch.float64)      # per-rank ms_per_step
dist.all_reduce(t, op=dist.ReduceOp.MAX)
assert t.item() == 10.0 + world - 1
points = 1000
value = world * points / (t.item() * 1e-3)                   # whole-job throughput over all replicas
dist.barrier()
if rank == 0:
    print("gloo ok %d %.1f" % (world, value))
dist.destroy_process_group()
