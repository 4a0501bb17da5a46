"""Host-side logic of bench.py on CPU: roofline arithmetic, JSON fields of the reference arm, and the
N > 1 path's max-over-ranks reduction with gloo, world_size 2 (no GPU, no collective on the data path)."""
from __future__ import annotations

import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_roofline_times_match_survey_table():
    sys.path.insert(0, ROOT)
    import bench
    import corrgen
    peaks = {"hbm_gbs": 6540.5, "bf16_tflops": 1676.3, "source": "test", "int8_tops": 3352.6, "int8_source": "test"}
    # c2 t_a = 150.3 us, c4 t_b = 160.3 us at these denominators
    t_a, t_b = bench.roofline_times(corrgen.CONFIGS["c2"], peaks)
    assert abs(t_a * 1e6 - 150.3) < 0.2 and t_b < t_a
    t_a, t_b = bench.roofline_times(corrgen.CONFIGS["c4"], peaks)
    assert abs(t_b * 1e6 - 160.3) < 0.3 and t_a < t_b
    w = corrgen.CONFIGS["c2"]
    assert w.cmacs == 10000 * 768 * 2080 and w.in_bytes == 983040000 and w.vis_bytes == 12779520


def test_channel_sharding_covers_every_channel_once():
    sys.path.insert(0, ROOT)
    import bench
    for n_chan, world in [(768, 8), (768, 5), (128, 3), (7, 8), (1536, 2)]:
        ranges = [bench.shard_channels(n_chan, world, r) for r in range(world)]
        assert ranges[0][0] == 0 and ranges[-1][1] == n_chan
        assert all(a[1] == b[0] for a, b in zip(ranges, ranges[1:]))
        sizes = [b - a for a, b in ranges]
        assert max(sizes) - min(sizes) <= 1


def test_shard_plan_gives_window_arguments():
    """Strong scaling: every rank's corr_create / corr_set_chan_window arguments tile the ONE cube."""
    sys.path.insert(0, ROOT)
    import bench
    import corrgen
    w = corrgen.CONFIGS["c2"]
    covered = []
    for rank in range(5):
        c0, c1, create_args, window_args = bench.shard_plan(w, 5, rank)
        assert create_args == (w.n_inputs, c1 - c0, w.n_time, w.dtype) and window_args == (w.n_chan, c0)
        covered += list(range(c0, c1))
    assert covered == list(range(w.n_chan))


def test_reference_arm_prints_contract_line():
    env = dict(os.environ, OMP_NUM_THREADS="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "c1",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "CMAC/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["vs_baseline"] is None


WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
rank, world, d = bench.dist_setup(2)
assert world == 2 and d is not None
t = bench.reduce_max(d, 1.0 + rank, torch.device("cpu"))
assert t == 2.0, t
import corrgen
w = corrgen.scaled(corrgen.CONFIGS["c2"], n_chan=11)
c0, c1, create_args, window_args = bench.shard_plan(w, world, rank)
# the two ranks' windows tile the cube: exchange the edges and check (the only "collective" is this test's own)
edges = torch.tensor([float(c0), float(c1)])
gathered = [torch.zeros(2) for _ in range(world)]
dist.all_gather(gathered, edges)
assert gathered[0][0] == 0 and gathered[0][1] == gathered[1][0] and gathered[1][1] == w.n_chan, gathered
assert create_args[1] == c1 - c0 and window_args == (w.n_chan, c0)
d.barrier()
d.destroy_process_group()
print("ok", rank)
"""


def test_max_over_ranks_with_gloo_world_size_2(tmp_path):
    pytest.importorskip("torch")
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT="29617", CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    for p in procs:
        out, err = p.communicate(timeout=300)
        assert p.returncode == 0 and "ok" in out, err[-2000:]
