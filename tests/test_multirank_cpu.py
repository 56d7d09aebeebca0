"""The N > 1 path of bench.py is "replicas only": one seeded CCD stack per rank, no data-path
collective, a barrier and a max-over-ranks reduction of the device time.  This covers that host logic with
world_size-2 gloo process groups on CPU (no GPU, no CUDA library calls)."""
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
# per-rank stacks: seed shifted by 100 * rank, as run_ours does
st, vx, vy, pd, desc = bench.make_workload("c1", seed_shift=100 * rank)
local_ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
ms = bench.max_over_ranks(local_ms, dist, torch.device("cpu"), world)
T, H, W = st.img.shape
value = bench.whole_job_value(float(H) * W * len(vx) * T, world, ms)
# one file per rank: two processes writing to one pipe can interleave their lines
open(os.path.join({out!r}, "rank%d.json" % rank), "w").write(
    json.dumps(dict(rank=rank, ms=ms, value=value, checksum=float(np.abs(st.img).sum()))))
dist.barrier()
dist.destroy_process_group()
"""


def test_two_rank_gloo_replicas(tmp_path):
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT, out=str(tmp_path)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), str(script)]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    import json
    recs = [json.loads((tmp_path / f"rank{r}.json").read_text()) for r in (0, 1)]
    assert [r["rank"] for r in recs] == [0, 1]
    assert recs[0]["ms"] == recs[1]["ms"] == 15.0                       # max over ranks, on every rank
    evals = 64 * 64 * 256 * 5
    assert np.isclose(recs[0]["value"], 2 * evals / 15e-3)              # whole-job aggregate over both replicas
    assert recs[0]["checksum"] != recs[1]["checksum"]                   # one independent stack per rank


def test_row_bands_partition_the_image():
    """--shard rows: the bands of the ranks tile [0, H) exactly, for any world size."""
    sys.path.insert(0, ROOT)
    import bench
    for H in (1, 7, 64, 4096, 4097):
        for world in (1, 2, 3, 4, 8):
            bands = [bench.row_band(r, world, H) for r in range(world)]
            assert bands[0][0] == 0 and bands[-1][1] == H
            assert all(a[1] == b[0] for a, b in zip(bands[:-1], bands[1:]))
            assert max(b[1] - b[0] for b in bands) - min(b[1] - b[0] for b in bands) <= 1
    vx = bench.whole_job_value(100.0, 4, 1000.0)
    assert vx == 400.0   # per-rank evaluations x ranks / seconds


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "c1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""
