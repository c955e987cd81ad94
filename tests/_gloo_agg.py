"""Helper of tests/test_bench_cpu.py: the reductions bench.py applies to its replicas, over a gloo group."""
import torch
import torch.distributed as dist

dist.init_process_group("gloo")
r = dist.get_rank()
t = torch.tensor([10.0 + r, 20.0 - r, 3.0 * (r + 1)], dtype=torch.float64)
dist.all_reduce(t, op=dist.ReduceOp.MAX)
u = torch.tensor([100.0 * (r + 1), 7.0], dtype=torch.float64)
dist.all_reduce(u, op=dist.ReduceOp.SUM)
if r == 0:
    print("AGG", t.tolist(), u.tolist())
dist.destroy_process_group()
