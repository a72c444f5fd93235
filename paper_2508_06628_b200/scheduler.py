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


class InFlightRelaxer:
    """FIRE relaxation of a stream of equal-size systems with converged systems swapped out.

    make_batch(ids) -> workloads.Batch-like object holding the systems `ids` (all the same atom
    count); n_slots systems are resident at a time (pass None to size it from `budget_bytes`).
    """

    def __init__(self, make_batch, n_total, fire, n_slots=None, budget_bytes=None, k_check=10, device="cuda:0",
                 engine=None, slack=1.25):
        self.make_batch, self.n_total, self.fire, self.k_check = make_batch, int(n_total), dict(fire), int(k_check)
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
                pos = st.numpy("pos")
                energy = st.numpy("energy")
                for s in done:
                    rec = {"pos": pos[off[s]:off[s + 1]].copy(), "energy": float(energy[s]), "fire_steps": int(steps[s]),
                           "status": int(status[s]), "slot": s}
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
