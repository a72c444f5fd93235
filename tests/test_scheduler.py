"""Host-side scheduler: the C-ABI scheduling primitives against the paper's worked
example (Figure 2), brute force on tiny inputs and textbook bounds; multi-rank sharding
with a world-size-2 gloo group on CPU.  No GPU needed."""
import itertools
import os
import subprocess
import sys

import numpy as np
import pytest

import paper_2508_06628_b200 as ts
from paper_2508_06628_b200 import scheduler as sch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_fig2_conservative_max_scaler_golden():
    probes, expect = [], None
    for line in open(os.path.join(ROOT, "tests", "golden", "paper_fig2_memory_scaler.txt")):
        f = line.split()
        if not f or f[0].startswith("#"):
            continue
        if f[0] == "probe":
            assert int(f[1]) * float(f[2]) == float(f[3])          # the paper's own products 800, 720
            probes.append((int(f[1]), float(f[2])))
        elif f[0] == "max_memory_scaler":
            expect = float(f[1])
    got = sch.conservative_max_scaler([p[0] for p in probes], [p[1] for p in probes])
    assert got == expect == 720.0


def test_admission_never_exceeds_budget_and_is_maximal():
    rng = np.random.default_rng(0)
    for _ in range(50):
        cost = rng.uniform(1, 100, size=rng.integers(1, 30))
        budget = rng.uniform(0, cost.sum() * 1.2)
        n, used = ts.ts_sched_fill(cost, budget)
        assert used == pytest.approx(cost[:n].sum()) and used <= budget
        assert n == len(cost) or used + cost[n] > budget


def _brute_force_bins(cost, cap):
    n = len(cost)
    for nb in range(1, n + 1):
        for assign in itertools.product(range(nb), repeat=n):
            load = np.zeros(nb)
            for c, a in zip(cost, assign):
                load[a] += c
            if (load <= cap + 1e-12).all():
                return nb
    return n


def test_binpack_is_valid_and_near_optimal_on_tiny_inputs():
    rng = np.random.default_rng(1)
    for _ in range(20):
        cost = rng.integers(1, 10, size=rng.integers(1, 8)).astype(float)
        cap = 10.0
        bins, nb = ts.ts_sched_binpack(cost, cap)
        for b in range(nb):
            assert 0 < cost[bins == b].sum() <= cap
        opt = _brute_force_bins(cost, cap)
        assert opt <= nb <= np.floor(11 * opt / 9 + 6 / 9)          # FFD bound (Dosa 2007)
    with pytest.raises(ts.TsError):
        ts.ts_sched_binpack([11.0], 10.0)


def test_partition_lpt_bound_and_cover():
    rng = np.random.default_rng(2)
    for _ in range(20):
        cost = rng.uniform(1, 50, size=rng.integers(1, 9))
        R = int(rng.integers(1, 4))
        rank, load = ts.ts_sched_partition(cost, R)
        assert sorted(np.concatenate([np.flatnonzero(rank == r) for r in range(R)]).tolist()) == list(range(len(cost)))
        for r in range(R):
            assert load[r] == pytest.approx(cost[rank == r].sum())
        opt = min(max(sum(c for c, a in zip(cost, assign) if a == r) for r in range(R))
                  for assign in itertools.product(range(R), repeat=len(cost)))
        assert load.max() <= (4 / 3 - 1 / (3 * R)) * opt + 1e-9     # Graham's LPT bound


def test_byte_estimate_tracks_atoms_times_density():
    import workloads as wl
    b = wl.cfg3(n_systems=6, dtype="f32", n_range=(32, 400), clean=False)
    by = sch.batch_system_bytes(b)
    n = np.diff(b.sys_offset)
    assert np.all(np.argsort(by, kind="stable") == np.argsort(n, kind="stable"))   # same density: ordered by atoms
    assert sch.admit(by, by[:3].sum()) == 3


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
import paper_2508_06628_b200 as ts
import bench
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
rank, world = dist.get_rank(), dist.get_world_size()
cost = np.array([864., 256., 2048., 32., 500., 1000., 108., 700.])
rk, load = ts.ts_sched_partition(cost, world)
mine = np.flatnonzero(rk == rank)
owned = torch.zeros(len(cost), dtype=torch.int64); owned[mine] = 1
dist.all_reduce(owned)                                   # every system owned exactly once across ranks
assert owned.tolist() == [1] * len(cost), owned
t = bench.max_over_ranks([0.5 + rank, 2.0 - rank], world, device="cpu")
assert t == [0.5 + world - 1, 2.0], t
ids = bench.rank_system_ids(rank, 4)
assert ids == list(range(rank * 4, rank * 4 + 4))
dist.barrier(); dist.destroy_process_group()
print("ok", rank)
"""


def test_world_size_2_gloo_sharding(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(_WORKER.format(root=ROOT))
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29571")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    for r, p in enumerate(procs):
        out, _ = p.communicate(timeout=240)
        assert p.returncode == 0 and f"ok {r}" in out, out


def test_take_and_concat_are_pure_container_work():
    import workloads as wl
    b = wl.cfg3(n_systems=5, dtype="f64", n_range=(32, 120), clean=False)
    t = sch.take_systems(b, [3, 1])
    ref = wl.take(b, [3, 1])
    for name in ("pos", "vel", "mass", "type", "system_idx", "sys_offset", "cell", "sys_uid"):
        assert np.array_equal(np.asarray(getattr(t, name)), np.asarray(getattr(ref, name))), name
    c = sch.concat_systems([sch.take_systems(b, [0]), t])
    assert c.n_systems == 3 and c.n_atoms == int(np.diff(b.sys_offset)[[0, 3, 1]].sum())
    assert np.array_equal(c.pos[c.sys_offset[1]:c.sys_offset[2]], b.pos[b.sys_offset[3]:b.sys_offset[4]])


_SHARD_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
import workloads as wl
from paper_2508_06628_b200 import scheduler as sch
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
store = dist.TCPStore("127.0.0.1", int(os.environ["STORE_PORT"]), world, rank == 0)
dist.init_process_group("gloo", store=store, rank=rank, world_size=world)
b = wl.cfg3(n_systems=9, dtype="f64", n_range=(32, 200), clean=False)
runner = sch.ShardedRunner(store=store)
# fixed-length mode: every rank "steps" its shard with a stand-in (the real step_fn is a SimState run: no CPU path
# exists, by design); the gather must return every system exactly once, with the data of the right system
def step_fn(sub, systems):
    assert sub.n_systems == len(systems)
    return {{s: (rank, float(sub.pos[sub.sys_offset[k]:sub.sys_offset[k + 1]].sum())) for k, s in enumerate(systems)}}
res = runner.run_fixed(b, step_fn)
mine, load = runner.shard(sch.batch_system_bytes(b))
assert load.max() <= 1.34 * load.sum() / world + sch.batch_system_bytes(b).max()
if rank == 0:
    assert sorted(res) == list(range(9))
    for s, (r, v) in res.items():
        assert abs(v - float(b.pos[b.sys_offset[s]:b.sys_offset[s + 1]].sum())) < 1e-9
    assert {{r for r, _ in res.values()}} == {{0, 1}}
else:
    assert res is None
# in-flight mode: one shared counter hands out stream ids; ranks claim different amounts, nothing is lost or doubled
claimed = []
while True:
    ids = runner.next_ids(1 + rank * 2, 23)
    if not ids and len(claimed) and claimed[-1] >= 0:
        pass
    if not ids:
        break
    claimed += ids
every = [None] * world
dist.all_gather_object(every, claimed)
flat = sorted(i for part in every for i in part)
assert flat == list(range(23)), flat
dist.barrier(); dist.destroy_process_group()
print("ok", rank)
"""


def test_sharded_runner_world_size_2_gloo(tmp_path):
    script = tmp_path / "s.py"
    script.write_text(_SHARD_WORKER.format(root=ROOT))
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29573", STORE_PORT="29575")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True))
    for r, p in enumerate(procs):
        out, _ = p.communicate(timeout=240)
        assert p.returncode == 0 and f"ok {r}" in out, out
