"""SimState: the caller-owned device arrays of one ragged batch plus its libts handle.

PyTorch provides device memory and the stream; all computation happens behind the C ABI.
"""
import ctypes as C

import numpy as np

import paper_2508_06628_b200 as ts


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2508_06628_b200 needs a CUDA device (there is no CPU fallback)")
    return torch


class _Pot:
    """Host tables of a potential, kept alive for ts_state_create."""

    def __init__(self, pot):
        self.kind = pot.kind if isinstance(pot.kind, int) else ts.KINDS[pot.kind]
        self.n_types = int(pot.n_types)
        nt2 = self.n_types ** 2
        self.arrs = [np.ascontiguousarray(np.asarray(getattr(pot, k), dtype=np.float64).reshape(nt2))
                     for k in ("p0", "p1", "p2", "rc")]
        p = [a.ctypes.data_as(C.c_void_p) for a in self.arrs]
        self.c = ts.ts_potential(self.kind, self.n_types, p[0], p[1], p[2], p[3], int(bool(pot.shift_energy)))


class PinnedStage:
    """Page-locked upload buffers for swap_systems, allocated once (cudaHostAlloc is slow) and reused by every swap.
    A swap synchronises before it returns, so the buffers are free again when the next swap fills them."""

    def __init__(self, torch, tdtype, max_atoms, max_systems):
        pin = lambda shape, dt: torch.empty(shape, dtype=dt).pin_memory()
        self.buf = {"pos": pin((max_atoms, 3), tdtype), "vel": pin((max_atoms, 3), tdtype), "mass": pin((max_atoms,), tdtype),
                    "type": pin((max_atoms,), torch.int32), "cell": pin((max_systems, 3, 3), tdtype),
                    "uid": pin((max_systems,), torch.int32)}

    def view(self, key, shape):
        b = self.buf[key]
        if shape[0] > b.shape[0]:
            raise ValueError(f"pinned stage too small for {key}: {shape[0]} > {b.shape[0]}")
        return b[:shape[0]]


class SimState:
    """One batch on the device.  `batch` is duck-typed (workloads.Batch): pos, vel, mass, type,
    system_idx, cell, potential, mass_conv, kB, skin, sys_uid."""

    def __init__(self, batch, dtype=None, skin=None, slack=1.25, device="cuda:0", engine=None, pinned_src=None):
        torch = _torch()
        self.torch = torch
        self.device = torch.device(device)
        dtype = dtype or getattr(batch, "dtype", "f64")
        self.dtype = ts.TS_F32 if dtype in ("f32", ts.TS_F32) else ts.TS_F64
        self.tdtype = torch.float32 if self.dtype == ts.TS_F32 else torch.float64
        self.npdtype = np.float32 if self.dtype == ts.TS_F32 else np.float64
        self.N = int(np.asarray(batch.pos).shape[0])
        self.S = int(np.asarray(batch.cell).shape[0])
        self.N_cap, self.S_cap = self.N, self.S                 # what ts_repack_systems may fill (sizes at create)
        self.sys_offset = np.asarray(batch.sys_offset, dtype=np.int64).copy() if hasattr(batch, "sys_offset") else None
        self.skin = float(batch.skin if skin is None else skin)
        self.slack = float(slack)
        self.units = ts.ts_units(float(batch.mass_conv), float(batch.kB))
        self._pot = _Pot(batch.potential)
        dev = self.device

        def up(a, dt, shape):
            t = torch.from_numpy(np.ascontiguousarray(np.asarray(a).reshape(shape))).to(dt)
            return t.to(dev, non_blocking=False).contiguous()

        self.pos = up(batch.pos, self.tdtype, (self.N, 3))
        vel = batch.vel if getattr(batch, "vel", None) is not None else np.zeros((self.N, 3))
        self.vel = up(vel, self.tdtype, (self.N, 3))
        self.mass = up(batch.mass, self.tdtype, (self.N,))
        self.type = up(batch.type, torch.int32, (self.N,))
        self.system_idx = up(batch.system_idx, torch.int32, (self.N,))
        self.cell = up(batch.cell, self.tdtype, (self.S, 3, 3))
        self.force = torch.zeros((self.N, 3), dtype=self.tdtype, device=dev)
        self.energy = torch.zeros(self.S, dtype=torch.float64, device=dev)
        self.virial = torch.zeros((self.S, 3, 3), dtype=torch.float64, device=dev)
        self.kinetic = torch.zeros(self.S, dtype=torch.float64, device=dev)
        uid = getattr(batch, "sys_uid", None)
        self.sys_uid = None if uid is None else torch.from_numpy(np.asarray(uid).astype(np.int64)).to(torch.int32).to(dev)
        self.desc = self._make_desc()
        self.nbr = ts.ts_nbr_params(self.skin, self.slack)
        with torch.cuda.device(self.device):
            self.workspace_bytes = ts.ts_workspace_bytes(self.desc, self._pot.c, self.nbr)
            self.workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=dev)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) & ~255
            self.handle = ts.ts_state_create(self.desc, self._pot.c, self.nbr, self._ws_ptr, self.workspace_bytes)
        if engine is not None:
            ts.ts_set_engine(self.handle, int(engine))

    def _make_desc(self):
        p = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        return ts.ts_state_desc(self.N, self.S, self.dtype, self.units, p(self.pos), p(self.vel), p(self.force),
                                p(self.mass), p(self.type), p(self.system_idx), p(self.cell), p(self.energy),
                                p(self.virial), p(self.kinetic), p(self.sys_uid))

    def close(self):
        if getattr(self, "handle", None) is not None:
            self.torch.cuda.synchronize(self.device)
            ts.ts_state_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------ C-ABI calls
    def build_neighbors(self):
        ts.ts_build_neighbors(self.handle)

    def compute_forces(self, want=ts.TS_WANT_ENERGY | ts.TS_WANT_VIRIAL):
        ts.ts_compute_forces(self.handle, want)

    def md_step(self, params, n_steps, want=ts.TS_WANT_ENERGY):
        if isinstance(params, dict):
            params = ts.md_params(**params)
        ts.ts_md_step(self.handle, params, n_steps, want)

    def fire_step(self, params, n_steps):
        if isinstance(params, dict):
            params = ts.fire_params(**params)
        ts.ts_fire_step(self.handle, params, n_steps)

    def poll(self):
        return ts.ts_poll(self.handle)

    def converged_mask(self):
        return ts.ts_converged_mask(self.handle, self.S)

    def fire_status_async(self, status, steps):
        """FIRE status / step counts into pinned int32 host tensors [S], enqueued on the current stream (no sync)."""
        ts.ts_fire_status_async(self.handle, status.data_ptr() if status is not None else 0,
                                steps.data_ptr() if steps is not None else 0)

    def get_neighbors(self):
        return ts.ts_get_neighbors(self.handle, self.N)

    def get_resident_neighbors(self, system):
        """(off, j, shift) of the list the system-resident engine would use for `system` at the current positions."""
        n = int(self.sys_offset[system + 1] - self.sys_offset[system])
        return ts.ts_get_resident_neighbors(self.handle, int(system), n)

    def set_system_steps(self, steps):
        ts.ts_set_system_steps(self.handle, steps)

    def get_system_steps(self):
        return ts.ts_get_system_steps(self.handle, self.S)

    def set_engine(self, engine):
        ts.ts_set_engine(self.handle, engine)

    def invalidate(self):
        ts.ts_invalidate(self.handle)

    def launch_count(self):
        return ts.ts_launch_count(self.handle)

    def swap_systems(self, slots, fresh, stage=None):
        """Replace the systems in `slots` by those of `fresh` (duck-typed batch, same sizes).  stage: a PinnedStage
        (page-locked upload buffers): the uploads are then enqueued without blocking on the work already in the stream."""
        d, alive = self._upload_fresh(fresh, stage)
        ts.ts_swap_systems(self.handle, slots, d)   # synchronises: the uploads may be released afterwards
        del alive

    def pinned_stage(self, max_atoms, max_systems):
        return PinnedStage(self.torch, self.tdtype, max_atoms, max_systems)

    def _upload_fresh(self, fresh, stage=None):
        """Device copies of a duck-typed batch for a swap / repack and their descriptor (kept alive by the caller)."""
        torch = self.torch
        n = int(np.asarray(fresh.cell).shape[0])
        nat = int(np.asarray(fresh.pos).shape[0])
        dev = self.device

        def up(a, dt, shape, key=None):
            src = torch.from_numpy(np.ascontiguousarray(np.asarray(a).reshape(shape)))
            if stage is None:
                return src.to(dt).to(dev).contiguous()
            buf = stage.view(key, shape)                   # page-locked, in the device dtype
            buf.copy_(src)
            return buf.to(dev, non_blocking=True)

        vel = fresh.vel if getattr(fresh, "vel", None) is not None else np.zeros((nat, 3))
        keep = [up(fresh.pos, self.tdtype, (nat, 3), "pos"), up(vel, self.tdtype, (nat, 3), "vel"),
                up(fresh.mass, self.tdtype, (nat,), "mass"), up(fresh.type, torch.int32, (nat,), "type"),
                up(fresh.cell, self.tdtype, (n, 3, 3), "cell"),
                up(np.asarray(fresh.sys_uid).astype(np.int64), torch.int32, (n,), "uid")]
        p = lambda t: C.c_void_p(t.data_ptr())
        d = ts.ts_state_desc(nat, n, self.dtype, self.units, p(keep[0]), p(keep[1]), None, p(keep[2]), p(keep[3]),
                             None, p(keep[4]), None, None, None, p(keep[5]))
        return d, keep

    def repack(self, keep_slots, fresh=None):
        """Ragged in-flight replacement (ts_repack_systems): the batch becomes the kept slots, in order, followed by
        the systems of `fresh` (duck-typed batch, any sizes).  Raises TsError(WORKSPACE_TOO_SMALL) when the new batch
        does not fit the capacity of the state; nothing has changed then."""
        keep_slots = [int(k) for k in keep_slots]
        old = self.sys_offset
        sizes = [int(old[k + 1] - old[k]) for k in keep_slots]
        if fresh is not None:
            d, alive = self._upload_fresh(fresh)
            fn = np.diff(np.asarray(fresh.sys_offset)).astype(np.int32)
            ts.ts_repack_systems(self.handle, keep_slots, d, fn)
            sizes += [int(x) for x in fn]
            del alive
        else:
            ts.ts_repack_systems(self.handle, keep_slots, None, np.zeros(0, np.int32))
        self.sys_offset = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
        self.N, self.S = int(self.sys_offset[-1]), len(sizes)

    def capacity(self):
        """(atoms, systems, pair slots) the state was created with."""
        return ts.ts_get_capacity(self.handle)

    # ------------------------------------------------------------------ graph export / external model (NEXT-2)
    def export_edges(self, cap=None):
        """The current Verlet list as device tensors: edge_index [2, n_edges] (int64) and the integer image shifts
        [n_edges, 3] in the state dtype: r_ij = pos[j] - pos[i] + shift @ cell[system].  Reads one scalar back
        (the edge count) to slice the tensors."""
        torch = self.torch
        if cap is None:
            cap = self.capacity()[2]
        if getattr(self, "_edges", None) is None or self._edges[0].shape[1] < cap:
            self._edges = (torch.empty((2, cap), dtype=torch.int64, device=self.device),
                           torch.empty((cap, 3), dtype=self.tdtype, device=self.device),
                           torch.zeros(1, dtype=torch.int64, device=self.device))
        ei, es, ne = self._edges
        ts.ts_export_edges(self.handle, ei[0].data_ptr(), ei[1].data_ptr(), es.data_ptr(), ei.shape[1], ne.data_ptr())
        n = int(ne.item())
        if n > ei.shape[1]:
            raise ts.TsError(ts.TS_ERR_WORKSPACE_TOO_SMALL, "export_edges", f"{n} edges > capacity {ei.shape[1]}")
        return ei[:, :n], es[:n]

    def export_edges_static(self, edge_index, edge_shift, n_edges):
        """ts_export_edges_static into the CALLER's device tensors (edge_index [2, cap] int64, edge_shift [cap, 3] in
        the state dtype, n_edges [1] int64): no allocation, no read-back; scratch in the library's static array."""
        ts.ts_export_edges_static(self.handle, edge_index[0].data_ptr(), edge_index[1].data_ptr(), edge_shift.data_ptr(),
                                  edge_index.shape[1], n_edges.data_ptr())

    def md_step_external(self, params, phase):
        if isinstance(params, dict):
            params = ts.md_params(**params)
        ts.ts_md_step_external(self.handle, params, phase)

    def fire_step_external(self, params, phase):
        if isinstance(params, dict):
            params = ts.fire_params(**params)
        ts.ts_fire_step_external(self.handle, params, phase)

    # ------------------------------------------------------------------ host views
    def numpy(self, name):
        """Host copy of a boundary array, cut to the live batch (a repack may have shrunk it below the capacity)."""
        t = getattr(self, name)
        n = self.S if name in ("cell", "energy", "virial", "kinetic", "sys_uid") else self.N
        return t[:n].detach().cpu().numpy()
