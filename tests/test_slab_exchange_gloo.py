"""The exchange step of the slab decomposition (paper_1812_01178_b200/parallel.py; Alg.1 steps 4 and 6, L156) on CPU:
three ranks over gloo.  No arithmetic happens here -- only which plane reaches which rank."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
from paper_1812_01178_b200 import parallel
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
plane = 6
iface = torch.empty((2, plane), dtype=torch.float64)
iface[0] = 100.0 * rank + torch.arange(plane, dtype=torch.float64)          # xt_first of this rank
iface[1] = 100.0 * rank + 50.0 + torch.arange(plane, dtype=torch.float64)   # xt_last of this rank
nbr = parallel.exchange_pdd(iface, rank, world)
ar = torch.arange(plane, dtype=torch.float64)
if rank >= 1:
    assert torch.equal(nbr[0], 100.0 * (rank - 1) + 50.0 + ar), nbr            # xt_last of rank-1
else:
    assert torch.equal(nbr[0], torch.zeros(plane, dtype=torch.float64))
if rank <= world - 2:
    assert torch.equal(nbr[1], 100.0 * (rank + 1) + ar), nbr                   # xt_first of rank+1
else:
    assert torch.equal(nbr[1], torch.zeros(plane, dtype=torch.float64))
g = parallel.exchange_ppt(iface, rank, world)
assert g.shape == (world, 2, plane)
for r in range(world):
    assert torch.equal(g[r, 0], 100.0 * r + ar) and torch.equal(g[r, 1], 100.0 * r + 50.0 + ar)
dist.barrier()
if rank == 0:
    print("exchange ok", world)
dist.destroy_process_group()
'''


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_neighbour_exchange_and_all_gather_three_ranks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "3", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), str(script)]
    out = subprocess.run(cmd, cwd=ROOT, env=dict(os.environ, OMP_NUM_THREADS="1"), capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-3000:]
    assert "exchange ok 3" in out.stdout


def test_slab_bounds_follow_the_partition_map():
    sys.path.insert(0, ROOT)
    from paper_1812_01178_b200 import parallel
    assert parallel.slab_bounds(70, 4) == [(0, 18), (18, 36), (36, 53), (53, 70)]
    assert parallel.slab_bounds(288, 8) == [(36 * r, 36 * (r + 1)) for r in range(8)]
