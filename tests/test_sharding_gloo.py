"""N > 1 path on CPU (gloo, world_size 2): the sharding plan of paper_2110_00256_b200/sharding.py.  Each rank runs
the ORACLE on its shard (the CUDA path needs a GPU); the concatenation of the shards must equal the single-process
result exactly, because particles are independent and the Philox stream is keyed on the global particle id."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
N, SEED, STEP = 6001, 5, 3   # odd size: unbalanced shards


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _population():
    from paper_2110_00256_b200 import workloads as w
    p, e, b = w.config1(seed=1, n=N, species=0)
    rng = np.random.default_rng(0)
    tau = np.where(rng.uniform(size=N) < 0.1, -0.3, 0.7)
    return p, e, b, tau


def _tables(orc):
    tp = orc.TableParams(qs_n_chi=12, qs_n_xi=16, bw_n_chi=12, bw_n_xi=16)
    lnG = np.linspace(-6, 5, 12)
    qs = np.tile(np.linspace(-8.0, 0.0, 16), (12, 1))
    return orc.Tables(tp, lnG, qs, np.full(12, -3.0), np.tile(np.linspace(0, 0.5, 16), (12, 1)))


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_2110_00256_b200 import sharding
    p, e, b, tau = _population()
    lo, hi = sharding.shard_range(rank, world, N)
    sl = slice(lo, hi)
    o = oracle.generate_photons(_tables(oracle), 1, 1, [a[sl] for a in p], [a[sl] for a in e], [a[sl] for a in b],
                                tau[sl], SEED, STEP, ids=np.arange(lo, hi, dtype=np.uint64))
    offset, total = sharding.secondary_offsets(o["n_fired"])
    slowest = sharding.max_over_ranks(1.0 + rank)
    np.savez(os.path.join(out_dir, "rank%d.npz" % rank), lo=lo, hi=hi, offset=offset, total=total, slowest=slowest,
             tau=o["tau"], px=o["p"][0], ph=o["ph_p"][0], ph_tau=o["ph_tau"], parent=o["parent"] + lo)
    dist.destroy_process_group()


def test_two_ranks_equal_one(orc, tmp_path):
    world, port = 2, _free_port()
    mp.start_processes(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True, start_method="spawn")
    p, e, b, tau = _population()
    ref = orc.generate_photons(_tables(orc), 1, 1, p, e, b, tau, SEED, STEP)
    parts = [np.load(os.path.join(tmp_path, "rank%d.npz" % r)) for r in range(world)]
    assert parts[0]["lo"] == 0 and parts[0]["hi"] == parts[1]["lo"] and parts[1]["hi"] == N
    assert abs((parts[0]["hi"] - parts[0]["lo"]) - (parts[1]["hi"] - parts[1]["lo"])) <= 1
    assert all(float(q["slowest"]) == 2.0 for q in parts)                         # max over ranks
    assert int(parts[0]["total"]) == int(parts[1]["total"]) == ref["n_fired"]
    assert int(parts[0]["offset"]) == 0 and int(parts[1]["offset"]) == len(parts[0]["parent"])
    for key, whole in (("tau", ref["tau"]), ("px", ref["p"][0]), ("ph", ref["ph_p"][0]), ("ph_tau", ref["ph_tau"]),
                       ("parent", ref["parent"])):
        assert np.array_equal(np.concatenate([q[key] for q in parts]), whole), key


def test_shard_range_covers_everything():
    from paper_2110_00256_b200 import sharding
    for n, world in ((10, 3), (7, 8), (1 << 24, 8), (0, 2)):
        r = [sharding.shard_range(k, world, n) for k in range(world)]
        assert r[0][0] == 0 and r[-1][1] == n and all(r[k][1] == r[k + 1][0] for k in range(world - 1))
