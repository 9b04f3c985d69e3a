"""N > 1 path on CPU: world_size-2 gloo run of the row sharding (no data-path collective; the only
communication is the gather of the finished bands).  The per-rank evaluator here is the oracle."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, tilt, out_path):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import gen
    import oracle
    from paper_2404_12454_b200 import sharding
    oracle.set_num_threads(2)
    w = gen.workload(4 if tilt else 0)
    if tilt:
        w = gen.Workload(**{**w.__dict__, "n_across": 15, "det_n": 37})
    xy = oracle.lattice(w.n_across, w.pupil_diameter)
    inp = gen.make_inputs(w, xy)
    rec = oracle.propagate(inp["xy"], oracle.waist(w.overlap_factor, w.pitch), w.wavelength,
                           inp["abcd_mode"], inp["abcd"], inp["l0"], inp["base"], inp["weight"])
    det = inp["detector"]
    band = sharding.row_band(det, rank, world)
    fld = oracle.field(oracle.to_detector(rec, band), band, w.wavelength)
    parts = [None] * world
    dist.all_gather_object(parts, (band["row_offset"], fld))
    # the library's own gather (one all-gather of the padded bands) must give every rank the same full field
    full_g = sharding.gather_rows(torch.as_tensor(fld), det["n_v"]).numpy()
    mine = np.concatenate([f for _, f in sorted(parts, key=lambda t: t[0])])
    assert full_g.shape == mine.shape and np.array_equal(full_g, mine)
    if rank == 0:
        full = oracle.field(oracle.to_detector(rec, det), det, w.wavelength)
        got = np.zeros_like(full)
        seen = np.zeros(full.shape[0], dtype=int)
        for v0, f in parts:
            got[v0:v0 + f.shape[0]] = f
            seen[v0:v0 + f.shape[0]] += 1
        err = np.linalg.norm(got - full) / np.linalg.norm(full)
        np.save(out_path, np.array([err, float(seen.min()), float(seen.max())]))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("tilt", [False, True])
def test_row_sharding_world2_gloo(tmp_path, tilt):
    out = str(tmp_path / "res.npy")
    mp.spawn(_worker, args=(2, _free_port(), tilt, out), nprocs=2, join=True)
    err, smin, smax = np.load(out)
    assert smin == 1 and smax == 1          # every row computed exactly once
    assert err < 1e-11


def test_row_range_partitions():
    from paper_2404_12454_b200.sharding import row_range, weak_band
    for n_v in (1, 7, 64, 1000, 1024):
        for world in (1, 2, 3, 8):
            r = [row_range(n_v, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n_v
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    d = dict(n_u=4, n_v=10, du=1.0, dv=2.0, origin=[0.0, 0.0, 0.0], e_u=[1, 0, 0], e_v=[0, 1, 0])
    assert weak_band(d, 0, 2)["origin"][1] == -10.0 and weak_band(d, 1, 2)["origin"][1] == 10.0
