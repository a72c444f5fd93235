"""Host-side batch scheduler (8(e)).

Decisions only: which systems share a batch, which slot a fresh system takes, which rank owns a
system.  The arithmetic of the decisions lives in libts (ts_estimate_system_bytes, ts_sched_*);
every simulation step runs in the CUDA kernels behind SimState.

  * estimate / admission: the paper sizes batches from a memory scaler found by probing for OOM
    (PAPER.md:66, :76-88); here the bytes are known analytically, and `admit` is the
    InFlightAutobatcher's "samples systems from the stream until memory is full".
  * InFlightRelaxer: "After every few steps of optimization, the convergence function is executed
    on the entire batch.  Any converged batches are removed ... and new systems are sampled from
    the stream".  Stream ids 0, 1, 2, ... fill slots in increasing id (R24); results
    do not depend on the check cadence or on batch composition (R22).
  * partition_systems: systems are independent, so multi-GPU = sharding by system
    with no exchange step.
"""
import numpy as np

import paper_2508_06628_b200 as ts


def system_bytes(n_atoms, volume, r_list, slack=1.25, dtype="f32"):
    """Bytes one system adds to a batch (boundary arrays + workspace): the n_atoms_x_density scaler
    of PAPER.md:88 with a known coefficient."""
    dt = ts.TS_F32 if dtype in ("f32", ts.TS_F32) else ts.TS_F64
    return ts.ts_estimate_system_bytes(n_atoms, volume, r_list, slack, dt)


def batch_system_bytes(batch, slack=1.25):
    """Per-system byte estimate for a workloads.Batch-like object."""
    off = np.asarray(batch.sys_offset)
    vol = np.abs(np.linalg.det(np.asarray(batch.cell, dtype=np.float64)))
    r_list = float(np.max(batch.potential.rc)) + float(batch.skin)
    return np.array([system_bytes(int(off[s + 1] - off[s]), float(vol[s]), r_list, slack, batch.dtype)
                     for s in range(len(vol))], dtype=np.float64)


def admit(costs, budget):
    """Longest prefix of the stream that fits `budget` (same unit as costs)."""
    return ts.ts_sched_fill(costs, budget)[0]


def conservative_max_scaler(n_systems, scalers):
    """Figure 2 step 4."""
    return ts.ts_sched_max_scaler(n_systems, scalers)


def binning_autobatch(costs, capacity):
    """BinningAutobatcher: list of index arrays, one per bin, first-fit decreasing."""
    bins, nb = ts.ts_sched_binpack(costs, capacity)
    return [np.flatnonzero(bins == b) for b in range(nb)]


def partition_systems(costs, n_ranks):
    """rank of each system (longest-processing-time first) and the per-rank load."""
    return ts.ts_sched_partition(costs, n_ranks)


def take_systems(b, systems):
    """The systems `systems` of a batch-like object as a new batch-like object (container work only)."""
    from types import SimpleNamespace
    off = np.asarray(b.sys_offset)
    idx = np.concatenate([np.arange(off[s], off[s + 1]) for s in systems]) if len(systems) else np.zeros(0, np.int64)
    sizes = [int(off[s + 1] - off[s]) for s in systems]
    new_off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    vel = getattr(b, "vel", None)
    return SimpleNamespace(
        name=getattr(b, "name", "batch"), pos=np.asarray(b.pos)[idx], vel=None if vel is None else np.asarray(vel)[idx],
        mass=np.asarray(b.mass)[idx], type=np.asarray(b.type)[idx],
        system_idx=np.repeat(np.arange(len(systems), dtype=np.int32), sizes), sys_offset=new_off,
        cell=np.asarray(b.cell)[list(systems)], potential=b.potential, mass_conv=b.mass_conv, kB=b.kB, skin=b.skin,
        dtype=getattr(b, "dtype", "f64"), sys_uid=np.asarray(b.sys_uid)[list(systems)],
        md=dict(getattr(b, "md", {}) or {}), fire=dict(getattr(b, "fire", {}) or {}),
        n_atoms=int(new_off[-1]), n_systems=len(systems))


def concat_systems(batches):
    """One batch-like object out of several (container work only; potential and units of the first)."""
    from types import SimpleNamespace
    b0 = batches[0]
    sizes = np.concatenate([np.diff(np.asarray(b.sys_offset)) for b in batches]).astype(np.int64)
    new_off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    cat = lambda name: np.concatenate([np.asarray(getattr(b, name)) for b in batches])
    zero_vel = lambda b: np.zeros_like(np.asarray(b.pos)) if getattr(b, "vel", None) is None else np.asarray(b.vel)
    return SimpleNamespace(
        name=getattr(b0, "name", "batch"), pos=cat("pos"), vel=np.concatenate([zero_vel(b) for b in batches]),
        mass=cat("mass"), type=cat("type"), system_idx=np.repeat(np.arange(sizes.size, dtype=np.int32), sizes),
        sys_offset=new_off, cell=cat("cell"), potential=b0.potential, mass_conv=b0.mass_conv, kB=b0.kB, skin=b0.skin,
        dtype=getattr(b0, "dtype", "f64"), sys_uid=cat("sys_uid"), md=dict(getattr(b0, "md", {}) or {}),
        fire=dict(getattr(b0, "fire", {}) or {}), n_atoms=int(new_off[-1]), n_systems=int(sizes.size))


class InFlightRelaxer:
    """FIRE relaxation of a stream of equal-size systems with converged systems swapped out.

    make_batch(ids) -> workloads.Batch-like object holding the systems `ids` (all the same atom
    count); n_slots systems are resident at a time (pass None to size it from `budget_bytes`).
    """

    def __init__(self, make_batch, n_total, fire, n_slots=None, budget_bytes=None, k_check=10, device="cuda:0",
                 engine=None, slack=1.25, pipelined=True):
        self.make_batch, self.n_total, self.fire, self.k_check = make_batch, int(n_total), dict(fire), int(k_check)
        self.pipelined = bool(pipelined)
        probe = make_batch([0])
        self.bytes_per_system = float(batch_system_bytes(probe, slack)[0])
        if n_slots is None:
            if budget_bytes is None:
                raise ValueError("give n_slots or budget_bytes")
            n_slots = admit(np.full(self.n_total, self.bytes_per_system), float(budget_bytes))
            if n_slots < 1:
                raise MemoryError("not even one system fits the byte budget")
        self.n_slots = min(int(n_slots), self.n_total)
        self.device, self.engine, self.slack = device, engine, slack
        self.results = {}           # id -> dict(pos, energy, fire_steps, status)
        self.failed = []
        self.peak_resident = 0

    def run(self, target=None, max_rounds=100000):
        if self.pipelined:
            return self._run_pipelined(target, max_rounds)
        return self._run_blocking(target, max_rounds)

    def _run_pipelined(self, target, max_rounds):
        """The same schedule with the device kept busy: ts_fire_step number r is enqueued BEFORE the status of call
        r - 1 is read (ts_fire_status_async into page-locked buffers, one event per call), and everything the host does
        with that status -- picking the finished systems, cutting the fresh ones from the stream, staging their upload --
        runs while call r computes.  A system that had converged in call r - 1 is frozen in call r (R22), and a slot
        refilled during round r is ignored in the stale snapshot of call r, so every id ends exactly as in the blocking
        loop; only the round in which a slot is refilled moves by one."""
        from .state import SimState
        target = self.n_total if target is None else int(target)
        ids = list(range(self.n_slots))
        next_id = self.n_slots
        b = self.make_batch(ids)
        st = SimState(b, device=self.device, engine=self.engine, slack=self.slack)
        torch = st.torch
        off = np.asarray(b.sys_offset).astype(np.int64)
        n_s = int(off[1] - off[0])
        S = self.n_slots
        slot_id = np.array(ids, dtype=np.int64)          # stream id resident in each slot, -1 = idle
        valid_from = np.zeros(S, dtype=np.int64)         # first call whose status describes the system now in the slot
        fp = ts.fire_params(**self.fire)
        pin = lambda shape, dt: torch.empty(shape, dtype=dt).pin_memory()
        snaps = [(pin((S,), torch.int32), pin((S,), torch.int32), torch.cuda.Event()) for _ in range(2)]
        stage = st.pinned_stage(S * n_s, S)
        pos_host, energy_host, sel_host = pin((S * n_s, 3), st.tdtype), pin((S,), torch.float64), pin((S * n_s,), torch.int64)
        lane = np.arange(n_s, dtype=np.int64)
        n_done = 0
        stream = torch.cuda.current_stream()

        def harvest(q):
            """Act on the status of call q (call q + 1 is already enqueued).  True when the run is over."""
            nonlocal n_done, next_id
            status_t, steps_t, ev = snaps[q % 2]
            ev.synchronize()
            status, steps = status_t.numpy(), steps_t.numpy()
            fin = (status == ts.TS_FIRE_CONVERGED) | (status == ts.TS_FIRE_FAILED)
            done = np.nonzero((slot_id >= 0) & (valid_from <= q) & fin)[0]
            self.peak_resident = max(self.peak_resident, int((slot_id >= 0).sum()))
            if done.size == 0:
                return False
            m = done.size * n_s
            # host work first (the device is stepping): row numbers of the finished systems, the fresh batch, its staging
            sel_host[:m].copy_(torch.from_numpy((off[done][:, None] + lane[None, :]).reshape(-1)))
            n_conv = int((status[done] == ts.TS_FIRE_CONVERGED).sum())
            take = 0 if n_done + n_conv >= target else min(done.size, self.n_total - next_id)
            new_ids = list(range(next_id, next_id + take))
            fresh = self.make_batch(new_ids) if take > 0 else None
            # enqueued behind the running call: the finished systems (frozen, so unchanged by that call) come back ...
            sel = sel_host[:m].to(st.device, non_blocking=True)
            pos_host[:m].copy_(st.pos.index_select(0, sel), non_blocking=True)
            energy_host.copy_(st.energy[:S], non_blocking=True)
            # ... and the fresh ones go into their slots; the swap synchronises, which also completes the copies above
            if take > 0:
                st.swap_systems(done[:take].astype(np.int32), fresh, stage)
            else:
                stream.synchronize()
            pos_done, energy = pos_host[:m].numpy(), energy_host.numpy()
            for k, s_ in enumerate(done):
                sid = int(slot_id[s_])
                self.results[sid] = {"pos": pos_done[k * n_s:(k + 1) * n_s].copy(), "energy": float(energy[s_]),
                                     "fire_steps": int(steps[s_]), "status": int(status[s_]), "slot": int(s_)}
                if status[s_] == ts.TS_FIRE_CONVERGED:
                    n_done += 1
                else:
                    self.failed.append(sid)
                slot_id[s_] = -1
            if n_done >= target:
                return True
            if take > 0:
                next_id += take
                slot_id[done[:take]] = new_ids
                valid_from[done[:take]] = q + 2              # call q + 1 was enqueued before the swap: its status is stale
            return not (slot_id >= 0).any()

        try:
            for r in range(max_rounds):
                st.fire_step(fp, self.k_check)
                status_t, steps_t, ev = snaps[r % 2]
                st.fire_status_async(status_t, steps_t)
                ev.record(stream)
                if r > 0 and harvest(r - 1):
                    break
            rep = st.poll()
            if rep.flags:
                raise ts.TsError(8, "InFlightRelaxer", f"device flags {rep.flags}")
        finally:
            self.unfinished = [int(i) for i in slot_id if i >= 0]
            st.close()
        return self.results

    def _run_blocking(self, target=None, max_rounds=100000):
        from .state import SimState
        target = self.n_total if target is None else int(target)
        ids = list(range(self.n_slots))
        next_id = self.n_slots
        b = self.make_batch(ids)
        st = SimState(b, device=self.device, engine=self.engine, slack=self.slack)
        off = np.asarray(b.sys_offset)
        slot_id = np.array(ids, dtype=np.int64)          # stream id resident in each slot, -1 = idle
        fp = ts.fire_params(**self.fire)
        n_done = 0
        try:
            for _ in range(max_rounds):
                st.fire_step(fp, self.k_check)
                mask, status, steps = st.converged_mask()
                done = [s for s in range(self.n_slots) if slot_id[s] >= 0 and status[s] in (ts.TS_FIRE_CONVERGED, ts.TS_FIRE_FAILED)]
                self.peak_resident = max(self.peak_resident, int((slot_id >= 0).sum()))
                if not done:
                    continue
                # only the finished systems come back to the host (device-side row selection, then one copy)
                rows = np.concatenate([np.arange(off[s], off[s + 1]) for s in done])
                sel = st.torch.from_numpy(rows).to(st.device)
                pos_done = st.pos.index_select(0, sel).cpu().numpy()
                energy = st.numpy("energy")
                at = 0
                for s in done:
                    n_s = int(off[s + 1] - off[s])
                    rec = {"pos": pos_done[at:at + n_s].copy(), "energy": float(energy[s]), "fire_steps": int(steps[s]),
                           "status": int(status[s]), "slot": s}
                    at += n_s
                    sid = int(slot_id[s])
                    self.results[sid] = rec
                    if status[s] == ts.TS_FIRE_CONVERGED:
                        n_done += 1
                    else:
                        self.failed.append(sid)
                    slot_id[s] = -1
                if n_done >= target:
                    break
                free = [s for s in done]
                take = min(len(free), self.n_total - next_id)
                if take > 0:
                    new_ids = list(range(next_id, next_id + take))
                    next_id += take
                    st.swap_systems(free[:take], self.make_batch(new_ids))
                    for s, sid in zip(free[:take], new_ids):
                        slot_id[s] = sid
                if not (slot_id >= 0).any():
                    break
            rep = st.poll()
            if rep.flags:
                raise ts.TsError(8, "InFlightRelaxer", f"device flags {rep.flags}")
        finally:
            self.unfinished = [int(i) for i in slot_id if i >= 0]
            st.close()
        return self.results


class RaggedInFlightRelaxer:
    """InFlightAutobatcher for systems of DIFFERENT sizes (Fig. 3).

    make_system(id) -> a one-system workloads.Batch-like object.  The first fill admits stream ids 0, 1, 2, ... until
    `budget_bytes` (ts_estimate_system_bytes per system, admission by ts_sched_fill) is full; that batch fixes the
    capacity of the state (atoms, systems, pair slots).  Every k_check FIRE steps the finished systems are read out
    and ts_repack_systems re-lays the batch: the running systems, then as many fresh ids as fit the three capacities.
    Results do not depend on the cadence or on who shared a batch with whom (R22): every id equals its solo run.
    """

    def __init__(self, make_system, n_total, fire, budget_bytes, k_check=10, device="cuda:0", engine=None, slack=1.25):
        self.make_system, self.n_total, self.fire, self.k_check = make_system, int(n_total), dict(fire), int(k_check)
        self.budget, self.device, self.engine, self.slack = float(budget_bytes), device, engine, float(slack)
        self.results, self.failed, self.unfinished = {}, [], []
        self.n_repacks, self.peak_atoms, self.peak_systems = 0, 0, 0
        self._cache = {}

    def _sys(self, sid):
        if sid not in self._cache:
            self._cache[sid] = self.make_system(sid)
        return self._cache[sid]

    def _pairs(self, b):
        vol = float(abs(np.linalg.det(np.asarray(b.cell, dtype=np.float64)[0])))
        r_list = float(np.max(b.potential.rc)) + float(b.skin)
        return ts.ts_estimate_system_pairs(int(np.asarray(b.pos).shape[0]), vol, r_list, self.slack)

    def _admit(self, next_id, atoms_free, systems_free, pairs_free, bytes_free=None, look_ahead=256):
        """How many of the ids next_id, next_id + 1, ... fit: the shortest of the prefixes the budgets allow."""
        ids = list(range(next_id, min(self.n_total, next_id + look_ahead)))
        if not ids or systems_free < 1:
            return []
        subs = [self._sys(i) for i in ids]
        n_at = np.array([np.asarray(b.pos).shape[0] for b in subs], dtype=np.float64)
        n_pr = np.array([self._pairs(b) for b in subs], dtype=np.float64)
        take = min(ts.ts_sched_fill(n_at, float(atoms_free))[0], ts.ts_sched_fill(n_pr, float(pairs_free))[0], int(systems_free))
        if bytes_free is not None:
            cost = np.array([batch_system_bytes(b, self.slack)[0] for b in subs])
            take = min(take, ts.ts_sched_fill(cost, float(bytes_free))[0])
        return ids[:take]

    def run(self, target=None, max_rounds=100000):
        from .state import SimState
        target = self.n_total if target is None else int(target)
        first = self._admit(0, 1e18, 1 << 30, 1e18, bytes_free=self.budget, look_ahead=self.n_total)
        if not first:
            raise MemoryError("not even one system fits the byte budget")
        st = SimState(concat_systems([self._sys(i) for i in first]), device=self.device, engine=self.engine, slack=self.slack)
        cap_atoms, cap_sys, cap_pairs = st.capacity()
        slot_id = list(first)
        next_id = first[-1] + 1
        for i in first:
            self._cache.pop(i, None)
        pairs_of = {}
        fp = ts.fire_params(**self.fire)
        n_done = 0
        try:
            for _ in range(max_rounds):
                self.peak_atoms, self.peak_systems = max(self.peak_atoms, st.N), max(self.peak_systems, st.S)
                st.fire_step(fp, self.k_check)
                mask, status, steps = st.converged_mask()
                done = [s for s in range(st.S) if status[s] in (ts.TS_FIRE_CONVERGED, ts.TS_FIRE_FAILED)]
                if not done:
                    continue
                pos, energy, off = st.numpy("pos"), st.numpy("energy"), st.sys_offset
                for s in done:
                    sid = slot_id[s]
                    self.results[sid] = {"pos": pos[off[s]:off[s + 1]].copy(), "energy": float(energy[s]),
                                         "fire_steps": int(steps[s]), "status": int(status[s])}
                    if status[s] == ts.TS_FIRE_CONVERGED:
                        n_done += 1
                    else:
                        self.failed.append(sid)
                keep = [s for s in range(st.S) if s not in set(done)]
                if n_done >= target:
                    slot_id = [slot_id[s] for s in keep]
                    break
                kept_atoms = int(sum(off[s + 1] - off[s] for s in keep))
                kept_pairs = 0
                cells = st.numpy("cell")
                r_list = float(st._pot.arrs[3].max()) + st.skin
                for s in keep:
                    vol = float(abs(np.linalg.det(cells[s].astype(np.float64))))
                    kept_pairs += ts.ts_estimate_system_pairs(int(off[s + 1] - off[s]), vol, r_list, self.slack)
                new_ids = self._admit(next_id, cap_atoms - kept_atoms, cap_sys - len(keep), cap_pairs - kept_pairs)
                if not keep and not new_ids:
                    slot_id = []
                    break
                fresh = concat_systems([self._sys(i) for i in new_ids]) if new_ids else None
                st.repack(keep, fresh)
                self.n_repacks += 1
                slot_id = [slot_id[s] for s in keep] + list(new_ids)
                for i in new_ids:
                    self._cache.pop(i, None)
                next_id += len(new_ids)
            rep = st.poll()
            if rep.flags:
                raise ts.TsError(ts.TS_ERR_STICKY, "RaggedInFlightRelaxer", f"device flags {rep.flags}")
        finally:
            self.unfinished = [int(i) for i in slot_id]
            st.close()
        return self.results


class BinRunner:
    """BinningAutobatcher as a runner: the systems of `batch` are packed into bins
    of at most `budget_bytes` (first-fit decreasing on ts_estimate_system_bytes, ts_sched_binpack) and the bins are
    stepped back to back on two CUDA streams, each bin as its own SimState; results come back in the order of `batch`."""

    def __init__(self, batch, budget_bytes, device="cuda:0", engine=None, slack=1.25):
        self.batch, self.device, self.engine, self.slack = batch, device, engine, slack
        self.costs = batch_system_bytes(batch, slack)
        self.bins = binning_autobatch(self.costs, float(budget_bytes))
        self._take = take_systems

    def run_md(self, n_steps, want=ts.TS_WANT_ENERGY):
        """n_steps of the batch's MD parameters on every bin; returns dict(pos, vel, force, energy, kinetic, virial)."""
        import torch
        from .state import SimState
        b = self.batch
        N, S = b.n_atoms, b.n_systems
        out = {"pos": np.zeros((N, 3)), "vel": np.zeros((N, 3)), "force": np.zeros((N, 3)), "energy": np.zeros(S),
               "kinetic": np.zeros(S), "virial": np.zeros((S, 3, 3))}
        streams = [torch.cuda.Stream(device=self.device) for _ in range(2)]
        live = []                                            # (state, systems of the bin, stream) of the bins in flight

        def collect(entry):
            st, systems, stream = entry
            stream.synchronize()
            rep = st.poll()
            if rep.flags:
                raise ts.TsError(ts.TS_ERR_STICKY, "BinRunner", f"device flags {rep.flags}")
            sub_off = st.sys_offset
            for k, s in enumerate(systems):
                a0, a1 = int(b.sys_offset[s]), int(b.sys_offset[s + 1])
                for name in ("pos", "vel", "force"):
                    out[name][a0:a1] = st.numpy(name)[sub_off[k]:sub_off[k + 1]]
                for name in ("energy", "kinetic", "virial"):
                    out[name][s] = st.numpy(name)[k]
            st.close()

        for n, systems in enumerate(self.bins):
            stream = streams[n % 2]
            if len(live) == 2:                               # at most two bins resident: the one stepping and the next
                collect(live.pop(0))
            with torch.cuda.stream(stream):
                st = SimState(self._take(b, [int(s) for s in systems]), device=self.device, engine=self.engine, slack=self.slack)
                st.md_step(dict(b.md), n_steps, want)
            live.append((st, [int(s) for s in systems], stream))
        while live:
            collect(live.pop(0))
        return out


class ShardedRunner:
    """Multi-GPU sharding by system (SURVEY 8(e), 8(f) NEXT-3; PAPER.md:64 systems are independent, :116 multi-GPU is the
    paper's future work): one process per GPU, no collective on the step path.

    Fixed-length runs: `partition_systems` (longest-processing-time first on the byte scaler) gives every rank its
    systems; each rank steps its own SimState; the per-system results are gathered on rank 0 (host objects).
    In-flight runs: the ranks draw stream ids from ONE shared counter in the process group's store (`next_ids`), so a
    rank that relaxes its systems faster simply takes more of the stream.
    `step_fn(sub_batch, system_indices) -> {system index: result}` does the device work (a SimState run); the runner
    itself holds no arithmetic, so its partition / queue / gather logic is testable on CPU ranks with a stand-in."""

    def __init__(self, rank=None, world=None, store=None):
        import torch.distributed as dist
        self.dist = dist
        self.on = dist.is_available() and dist.is_initialized()
        self.rank = (dist.get_rank() if self.on else 0) if rank is None else rank
        self.world = (dist.get_world_size() if self.on else 1) if world is None else world
        self.store = store

    def shard(self, costs):
        """Systems of this rank (sorted) and the load of every rank."""
        rank_of, load = partition_systems(np.asarray(costs, dtype=np.float64), self.world)
        return np.flatnonzero(rank_of == self.rank), load

    def run_fixed(self, batch, step_fn, costs=None, take=None):
        """Every rank steps its shard of `batch`; rank 0 returns {system index: result} for all systems, others None."""
        take = take_systems if take is None else take
        costs = batch_system_bytes(batch) if costs is None else costs
        mine, _ = self.shard(costs)
        local = step_fn(take(batch, [int(s) for s in mine]), [int(s) for s in mine]) if mine.size else {}
        return self.gather(local)

    def next_ids(self, n, n_total, key="ts_next_id"):
        """Claim up to n stream ids from the shared counter (atomic add in the store); [] when the stream is dry."""
        if n <= 0:
            return []
        if self.store is None:                                # single process
            start = getattr(self, "_local_next", 0)
            self._local_next = start + n
        else:
            start = self.store.add(key, n) - n
        return list(range(start, min(start + n, n_total)))

    def gather(self, local):
        """Per-system results of all ranks on rank 0 (the end-of-run gather of SURVEY 8(e))."""
        if not self.on or self.world == 1:
            return dict(local)
        parts = [None] * self.world if self.rank == 0 else None
        self.dist.gather_object(dict(local), parts, dst=0)
        if self.rank != 0:
            return None
        out = {}
        for p in parts:
            out.update(p)
        return out
