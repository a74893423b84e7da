"""Host-side checks of bench.py's multi-rank logic (no GPU): `gloo`, world size 2, rendezvous on 127.0.0.1.

The path does not shard (replicas only), so the only cross-rank steps are the barrier and the MAX over
ranks of the device time; and `--impl reference` must print one line from rank 0 only."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
t = bench.max_over_ranks(10.0 + 5.0 * rank, 2, torch.device("cpu"))   # rank 1 is the slow one
v = bench.job_mlups(1000, 7, 2, t * 1e-3)
dist.barrier()
print("RESULT", rank, t, v, flush=True)
dist.destroy_process_group()
"""


def test_time_is_the_max_over_ranks_and_value_is_the_job_aggregate(tmp_path):
    port = _free_port()
    src = tmp_path / "w.py"
    src.write_text(WORKER.format(root=ROOT, port=port))
    procs = [subprocess.Popen([sys.executable, str(src), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(2)]
    outs = [p.communicate(timeout=240) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    for o, _ in outs:
        line = [l for l in o.splitlines() if l.startswith("RESULT")][0].split()
        assert float(line[2]) == 15.0                                  # both ranks see the slowest rank's time
        assert float(line[3]) == pytest.approx(1000 * 7 * 2 / 15e-3 / 1e6)  # units of ALL ranks / that time


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1, None) == 3.5
    assert bench.job_mlups(16_000_000, 400, 1, 0.16) == pytest.approx(40000.0)


def test_reference_arm_prints_one_line_from_rank_0_only():
    env = dict(os.environ, OMP_NUM_THREADS="4")
    outs = []
    for rank in (0, 1):
        e = dict(env, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank))
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                            "--warmup", "0", "--reference-budget", "6"], capture_output=True, text=True, env=e, timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        outs.append(r.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["gpu_launches"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"] > 0
    assert line["e2e"] == {"value": line["value"], "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}


def test_traffic_figure_comes_from_the_committed_profile():
    sys.path.insert(0, ROOT)
    import bench
    t, src = bench.load_traffic()
    assert t is None or 0.9 * 153 * 16e6 < t < 1.3 * 153 * 16e6
    assert (t is None) == (src is None) and (src is None or os.path.exists(os.path.join(ROOT, src)))
    th, _ = bench.load_traffic("thermal")  # fused flow + thermal kernel: (19 + 7) x 4 B x 2 + 1 flag byte = 209 B/cell
    assert th is None or 0.9 * 209 * 16e6 < th < 1.3 * 209 * 16e6
    s16, _ = bench.load_traffic("s16")      # 16-bit population storage: 19 x 2 B x 2 + 1 flag byte = 77 B/cell
    assert s16 is None or 0.9 * 77 * 16e6 < s16 < 1.3 * 77 * 16e6
