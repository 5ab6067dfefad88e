"""Host logic of the sharded (multi-GPU) path on CPU: the row split of the C ABI (wpg_shard_rows) and the grid
reduce / counter all-reduce of paper_1905_03213_b200/sharded.py in a world_size-2 gloo group.  The ranks' private
grids are made by the oracle on each rank's shard (there is no GPU here); the reduced grid on rank 0 must equal the
oracle's grid of all rows (P12: gridding is additive), and the counters must add up."""
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_1905_03213_b200 import sharded

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("nrow,row_block,world", [(0, 0, 3), (10, 0, 3), (7, 0, 8), (2016 * 5 + 17, 2016, 2),
                                                   (2016 * 5 + 17, 2016, 4), (130816 * 360, 130816, 8), (5, 100, 2)])
def test_shard_rows_partition(nrow, row_block, world):
    prev = 0
    sizes = []
    for rank in range(world):
        r0, r1 = sharded.shard_rows(nrow, world, rank, row_block)
        assert r0 == prev and r1 >= r0                       # contiguous, disjoint, in rank order
        if row_block and r1 < nrow:
            assert r1 % row_block == 0                       # whole time steps
        sizes.append(r1 - r0)
        prev = r1
    assert prev == nrow                                      # covers every row exactly once
    unit = row_block or 1
    assert max(sizes) - min(sizes) < 2 * unit                # balanced to within one unit (the last unit may be partial)


def test_shard_rows_argument_errors():
    from paper_1905_03213_b200 import wpgrid
    for args in ((10, 0, 0, 0), (10, 0, 2, 2), (10, 0, 2, -1), (-1, 0, 2, 0), (10, -5, 2, 0)):
        with pytest.raises(wpgrid.WpgError):
            sharded.shard_rows(args[0], args[2], args[3], args[1])


WORKER = r'''
import os, sys
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
from paper_1905_03213_b200 import sharded, synth
from oracle import gridder as ogrid, wkernel as owk
rank = int(os.environ["RANK"])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%%s" %% os.environ["MASTER_PORT"], rank=rank, world_size=2)
wl = synth.config2(nvis=2016 * 7 + 5, noise=False)
st = owk.build_stack(wl.Nw, wl.w_max, wl.support, wl.oversample, wl.grid_N, wl.cell)
rb = wl.notes["row_block"]
r0, r1 = sharded.shard_rows(wl.uvw.shape[0], 2, rank, rb)
part, pstats = ogrid.grid(wl.uvw[r0:r1], wl.vis[r0:r1], wl.weight[r0:r1], wl.freq, st)     # this rank's private grid
g = torch.from_numpy(part)
sharded.reduce_grid(g, dist, dst=0)
tot = sharded.reduce_stats(pstats, dist, torch.device("cpu"))
ok = True
if rank == 0:
    ref, rstats = ogrid.grid(wl.uvw, wl.vis, wl.weight, wl.freq, st)
    err = float(np.max(np.abs(g.numpy() - ref)) / np.max(np.abs(ref)))
    ok = err <= 1e-13 and tot == rstats
    print("RESULT", rank, r0, r1, err, tot == rstats, flush=True)
else:
    print("RESULT", rank, r0, r1, 0.0, True, flush=True)
dist.destroy_process_group()
sys.exit(0 if ok else 1)
'''


def test_reduce_of_private_grids_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    port = str(31500 + os.getpid() % 2000)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=port)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    lines = [[l for l in o[0].splitlines() if l.startswith("RESULT")][0].split() for o in outs]
    assert int(lines[0][2]) == 0 and int(lines[0][3]) == int(lines[1][2])        # shards meet
    assert int(lines[0][3]) % 2016 == 0 and int(lines[1][3]) == 2016 * 7 + 5
