"""The N>1 path on CPU: world_size-2 gloo processes exercise the host-side sharding logic.

The data path has no collective (slices are independent); what more than one rank adds is the shard
arithmetic, the max-over-ranks timing / sum-over-ranks unit count of bench.py, and the rule that only rank 0 runs and
prints the reference arm.
"""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2006_09808_b200 import shard

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("batch,world", [(1024, 8), (7, 2), (5, 4), (3, 4), (0, 2), (1, 1)])
def test_shard_bounds_partition_the_batch(batch, world):
    spans = [shard.shard_bounds(batch, r, world) for r in range(world)]
    assert spans[0][0] == 0 and spans[-1][1] == batch
    assert all(spans[i][1] == spans[i + 1][0] for i in range(world - 1))       # contiguous, in rank order
    sizes = [hi - lo for lo, hi in spans]
    assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard.shard_bounds(batch, world, world)


_WORKER = r"""
import os, sys, json
import numpy as np
import torch.distributed as dist
sys.path.insert(0, {root!r})
from paper_2006_09808_b200 import shard, synth
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
# strong split of one stack: every rank generates only its own slices; together they are the unsplit stack
lo, hi = shard.shard_bounds(5, rank, world)
mine = synth.generate(1, nslices=hi - lo, first_slice=lo)["field"]
full = synth.generate(1, nslices=5)["field"]
same = bool(np.array_equal(mine, full[lo:hi]))
# weak scaling as in bench.py: distinct stacks per rank
first = shard.weak_first_slice(16, rank)
# whole-job throughput: sum of units over max of time
value, units, ms = shard.job_throughput(1000.0 * (rank + 1), 10.0 * (rank + 1))
out = dict(rank=rank, lo=lo, hi=hi, same=same, first=first, value=value, units=units, ms=ms,
           mx=shard.max_over_ranks(rank + 1.5), sm=shard.sum_over_ranks(rank + 1.5))
with open(os.path.join({outdir!r}, "rank%d.json" % rank), "w") as f:
    json.dump(out, f)
dist.destroy_process_group()
"""


def _torchrun(args, port, timeout=240):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port)] + args
    env = dict(os.environ, OMP_NUM_THREADS="1")
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, cwd=ROOT, env=env)


def test_two_ranks_gloo_shard_and_reduce(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, outdir=str(tmp_path)))
    r = _torchrun([str(script)], 29731)
    assert r.returncode == 0, r.stderr[-2000:]
    res = [json.loads((tmp_path / ("rank%d.json" % k)).read_text()) for k in range(2)]
    assert [d["rank"] for d in res] == [0, 1]
    assert (res[0]["lo"], res[0]["hi"], res[1]["lo"], res[1]["hi"]) == (0, 3, 3, 5)
    assert all(d["same"] for d in res)                        # shards reassemble to the unsplit stack
    assert [d["first"] for d in res] == [0, 16]
    for d in res:                                             # every rank sees the same global numbers
        assert d["units"] == 3000.0 and d["ms"] == 20.0 and np.isclose(d["value"], 3000.0 / 0.020)
        assert d["mx"] == 2.5 and d["sm"] == 4.0


def test_reference_arm_prints_on_rank0_only():
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "3",
                   "--workload", "C0"], 29732)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
