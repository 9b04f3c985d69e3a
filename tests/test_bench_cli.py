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


def _strong_worker(rank, world, port, out_path):
    import numpy as np
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import gen
    import oracle
    oracle.set_num_threads(2)
    w = gen.Workload(**{**gen.workload(4).__dict__, "n_across": 15, "det_n": 37})      # tilted, 37 rows: bands of 19 + 18
    xy = oracle.lattice(w.n_across, w.pupil_diameter)
    inp = gen.make_inputs(w, xy)
    rec = oracle.propagate(inp["xy"], oracle.waist(w.overlap_factor, w.pitch), w.wavelength,
                           inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"])
    det = inp["detector"]
    calls = []

    def evaluate(band):
        calls.append((band["row_offset"], band["n_v"]))
        return torch.as_tensor(oracle.field(oracle.to_detector(rec, band), band, w.wavelength))

    summary, full = bench.strong_scaling(evaluate, det, rank, world, dist, steps=2)
    assert len(calls) == 3 and len(set(calls)) == 1                 # one warm-up + two timed steps, always this rank's band
    ref = oracle.field(oracle.to_detector(rec, det), det, w.wavelength)
    err = float(np.linalg.norm(full.numpy() - ref) / np.linalg.norm(ref))
    if rank == 0:
        with open(out_path, "w") as f:
            json.dump({"summary": summary, "err": err, "band": list(calls[0])}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_strong_scaling_bookkeeping_world2_gloo(tmp_path):
    """bench.py's N > 1 measurement of SURVEY 8(e) -- one detector, rows partitioned, bands all-gathered -- driven on
    the CPU by two gloo ranks with the oracle as the per-rank evaluator: every rank ends with the full field."""
    import socket
    import torch.multiprocessing as mp
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    out = str(tmp_path / "strong.json")
    mp.spawn(_strong_worker, args=(2, port, out), nprocs=2, join=True)
    d = json.load(open(out))
    s = d["summary"]
    assert d["err"] < 1e-11 and d["band"] == [0, 19]
    assert s["scaling"] == "strong" and s["world"] == 2 and s["rows_per_rank"] == [19, 18] and s["steps"] == 2
    assert s["eval_ms_per_step"] > 0 and s["gather_ms_per_step"] > 0 and s["gather_bytes_per_rank"] == 37 * 37 * 16
