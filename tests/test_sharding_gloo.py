"""The N > 1 path on CPU: world_size 2 over gloo.

Fixed-temperature tracking shards package-id ranges; the integer tallies summed with one all-reduce must equal the
single-process tallies exactly.  The compute of each rank is played by the oracle here (tests may use it; there is
no GPU in this container): with unit weights every absorption adds exactly one package energy, so the per-shell
tallies are integers."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2408_13807_b200 import sharding, synth  # noqa: E402

N_PKG = 6001          # odd on purpose: ragged split
SEED = 5


def _counts(orc, p, first, count):
    o = orc.Oracle(p)
    o.set_fixed_temperature(np.linspace(10.0, 20.0, p.n_shells))
    o.run(N_PKG, seed=SEED, mode=1, first_id=first, n_run=count)
    e_pkg = o.sums["injected"] / max(count, 1)
    a = np.rint(o.absorbed / e_pkg).astype(np.int64)
    assert np.allclose(a * e_pkg, o.absorbed, rtol=1e-9, atol=0)
    esc = np.rint(o.escaped / e_pkg).astype(np.int64)
    c = o.counters
    return a, esc, np.array([c["packages"], c["crossings"], c["scatterings"], c["absorptions"]], dtype=np.int64)


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import dies_oracle as orc
        p = synth.config1()
        first, count = sharding.package_range(N_PKG, rank, world)
        a, esc, cnt = _counts(orc, p, first, count)
        ta, te, tc = sharding.allreduce_tallies(torch.from_numpy(a), torch.from_numpy(esc), torch.from_numpy(cnt))
        slow = sharding.max_over_ranks(10.0 + rank, "cpu")
        if rank == 0:
            np.savez(out, a=ta.numpy(), esc=te.numpy(), cnt=tc.numpy(), slow=slow)
    finally:
        dist.destroy_process_group()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_package_ranges_tile_exactly():
    for n in (0, 1, 7, 6001, 10**7):
        for world in (1, 2, 3, 8):
            r = [sharding.package_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and sum(c for _, c in r) == n
            assert all(r[k][0] + r[k][1] == r[k + 1][0] for k in range(world - 1))
            assert max(c for _, c in r) - min(c for _, c in r) <= 1
    with pytest.raises(ValueError):
        sharding.package_range(10, 2, 2)
    assert len({sharding.replica_seed(1, s, r) for s in range(50) for r in range(8)}) == 400


def test_allreduce_refuses_floating_point_tallies():
    with pytest.raises(TypeError):
        sharding.allreduce_tallies(torch.zeros(4, dtype=torch.float64))


def test_fixed_T_shards_sum_to_the_single_run(tmp_path):
    from oracle import dies_oracle as orc
    out = str(tmp_path / "sum.npz")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    got = np.load(out)
    a, esc, cnt = _counts(orc, synth.config1(), 0, N_PKG)
    assert np.array_equal(got["a"], a)
    assert np.array_equal(got["esc"], esc)
    assert np.array_equal(got["cnt"], cnt)
    assert got["cnt"][0] == N_PKG and a.sum() > 0
    assert float(got["slow"]) == 11.0


# ------------------------------------------------------------------ config 5: the spheres of a batch dealt to ranks
N_MODELS, N_BATCH_PKG = 5, 1500


def _batch():
    return synth.config5(n_models=N_MODELS, n_packages=N_BATCH_PKG, n_shells=8, n_freq=16, n_T=50)


def _batch_T(orc, b, first):
    """Temperatures of the models of (sub-)batch b, whose first model has index `first` in the whole batch."""
    T = []
    for i in range(b.n_models):
        o = orc.Oracle(b.model(i))
        o.run(b.n_packages, seed=SEED, model_index=first + i)
        T.append(o.temperature())
    return np.array(T)


def _batch_worker(rank, world, port, outdir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import dies_oracle as orc
        sub, first = sharding.batch_shard(_batch(), rank, world)
        T = _batch_T(orc, sub, first)
        n_all = sharding.sum_over_ranks(sub.n_models * sub.n_packages, "cpu")
        np.savez(os.path.join(outdir, f"shard{rank}.npz"), T=T, first=first, n_all=n_all)
    finally:
        dist.destroy_process_group()


def test_batch_shards_tile_the_models():
    b = _batch()
    for world in (1, 2, 3, 5, 8):
        firsts, total = [], 0
        for rank in range(world):
            sub, first = sharding.batch_shard(b, rank, world)
            assert np.array_equal(sub.rho, b.rho[first:first + sub.n_models])
            assert np.array_equal(sub.ext_bin_intensity, b.ext_bin_intensity[first:first + sub.n_models])
            assert len(sub.meta["tau_V"]) == sub.n_models
            firsts.append(first); total += sub.n_models
        assert total == b.n_models and firsts == sorted(firsts)


def test_batch_shards_reproduce_the_whole_batch(tmp_path):
    """World size 2 over gloo, no data-path collective: each rank follows its spheres with their indices of the whole
    batch in the Philox counter; the concatenated temperatures equal those of the one-process batch exactly."""
    from oracle import dies_oracle as orc
    mp.spawn(_batch_worker, args=(2, _free_port(), str(tmp_path)), nprocs=2, join=True)
    parts = [np.load(tmp_path / f"shard{r}.npz") for r in range(2)]
    assert int(parts[0]["first"]) == 0 and int(parts[1]["first"]) == 3
    assert float(parts[0]["n_all"]) == N_MODELS * N_BATCH_PKG
    T = np.concatenate([q["T"] for q in parts])
    assert np.array_equal(T, _batch_T(orc, _batch(), 0))


def test_bench_gpus_n_starts_its_own_ranks(monkeypatch):
    """`python bench.py --gpus N` (the form the driver uses for N = 1, and a user for any N) must launch N ranks when
    it is not already one of them; under torchrun (WORLD_SIZE set) it must not spawn again."""
    import bench

    calls = []
    monkeypatch.setattr(bench.subprocess, "call", lambda cmd: calls.append(cmd) or 0)
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    with pytest.raises(SystemExit) as e:
        bench.main(["--gpus", "4", "--steps", "5", "--workload", "config5"])
    assert e.value.code == 0 and len(calls) == 1
    cmd = calls[0]
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert cmd[-6:] == ["--gpus", "4", "--steps", "5", "--workload", "config5"] and cmd[-7].endswith("bench.py")
    # the reference arm never spawns (rank 0 alone times the oracle): it goes straight to run_reference
    seen = []
    monkeypatch.setattr(bench, "run_reference", lambda a, rank, world: seen.append((rank, world)))
    bench.main(["--gpus", "4", "--impl", "reference"])
    assert seen == [(0, 1)] and len(calls) == 1
    # a rank of a running job does not spawn
    monkeypatch.setenv("WORLD_SIZE", "4")
    monkeypatch.setenv("RANK", "3")
    ours = []
    monkeypatch.setattr(bench, "run_ours", lambda a, rank, world, lr: ours.append((rank, world)))
    bench.main(["--gpus", "4"])
    assert ours == [(3, 4)] and len(calls) == 1
