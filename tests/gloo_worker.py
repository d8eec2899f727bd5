"""world_size-2 gloo worker for tests/test_host_logic.py (launched with torch.distributed.run)."""
import sys

from paper_2606_15991_b200 import dist as tdist

rank, local_rank, world = tdist.init("gloo")
assert world == 2
tdist.barrier()
assert tdist.max_over_ranks(1.0 + rank) == 2.0
assert tdist.sum_over_ranks(10.0 * (rank + 1)) == 30.0
shares = [tdist.units_for_rank(257, r, world) for r in range(world)]
assert shares[0][0] == 0 and shares[-1][1] == 257 and shares[0][1] == shares[1][0]
assert abs((shares[0][1] - shares[0][0]) - (shares[1][1] - shares[1][0])) <= 1
tdist.barrier()
print(f"GLOO_OK rank{rank}", flush=True)
tdist.shutdown()
sys.exit(0)
