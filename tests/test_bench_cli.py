"""bench.py command-line contract, on the CPU box: the reference arm prints one well-formed JSON line; `--gpus N`
without a torchrun environment launches N ranks itself, and without a CUDA device every rank fails loudly (there is
no CPU fallback for the product arm)."""
import json
import os
import subprocess
import sys

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BENCH = os.path.join(ROOT, "bench.py")


def _clean_env():
    env = dict(os.environ)
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT"):
        env.pop(k, None)
    return env


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, BENCH, "--impl", "reference", "--steps", "1", "--warmup", "0"],
                         cwd=ROOT, env=_clean_env(), capture_output=True, text=True, timeout=900)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.strip().startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "evals/s" and d["higher_is_better"] is True
    assert d["value"] > 1e6 and d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["value"] == d["value"] and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["gpu_launches"] == 0 and d["vs_baseline"] is None and "C3" in d["config"]["workload"]


@pytest.mark.skipif(torch.cuda.is_available(), reason="needs a box WITHOUT a CUDA device")
def test_gpus_n_spawns_n_ranks_and_fails_loudly_without_cuda():
    out = subprocess.run([sys.executable, BENCH, "--gpus", "2", "--steps", "1", "--warmup", "1"],
                         cwd=ROOT, env=_clean_env(), capture_output=True, text=True, timeout=600)
    assert out.returncode != 0
    err = out.stderr
    assert "spawning 2 ranks" in err
    assert "rank 0 of 2: no CUDA device" in err and "rank 1 of 2: no CUDA device" in err
    assert not [l for l in out.stdout.splitlines() if l.strip().startswith("{")]      # no number without a GPU


def test_world_size_mismatch_is_refused():
    env = dict(_clean_env(), WORLD_SIZE="2", RANK="0", LOCAL_RANK="0")
    out = subprocess.run([sys.executable, BENCH, "--gpus", "4"], cwd=ROOT, env=env, capture_output=True, text=True,
                         timeout=300)
    assert out.returncode != 0 and "WORLD_SIZE=2" in (out.stderr + out.stdout)


def test_roofline_numbers_come_from_the_committed_captures():
    """bench.py quotes ncu numbers (executed FP64 instructions per term, DRAM bytes per launch) beside its live
    measurements; they are parsed from the summaries under profiles/ at start-up, never typed into bench.py."""
    sys.path.insert(0, ROOT)
    import bench
    src = open(BENCH).read()
    for algo, kt in bench.KERNEL_TABLE.items():
        assert "executed" not in kt and "traffic" not in kt            # nothing remembered in the table itself
        got = bench.load_capture(dict(kt))
        rows = bench.parse_capture(os.path.join(ROOT, kt["capture"]), kt["section"])
        assert rows["launch__grid_size"][1] == 148
        rd, wr = rows["dram__bytes_read.sum"], rows["dram__bytes_write.sum"]
        scale = {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6}
        assert got["traffic"] == round(rd[1] * scale[rd[0]] + wr[1] * scale[wr[0]])
        assert str(got["traffic"]) not in src
        assert abs(got["executed"] - kt["algorithmic"]) < 0.15 and got["other"] > 1.0
    direct = bench.load_capture(dict(bench.KERNEL_TABLE["direct"]))
    assert direct["traffic"] == 3126784 and abs(direct["executed"] - 16.04) < 0.005 and abs(direct["other"] - 9.5) < 0.05
    missing = bench.load_capture(dict(bench.KERNEL_TABLE["direct"], capture="profiles/does_not_exist.md"))
    assert missing["executed"] is None and missing["traffic"] is None
