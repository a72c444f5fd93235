"""GPU test of ts_export_edges_static: the edge export whose scratch lives in a file-scope device array of the
library (include/ts.h), for callers that must not allocate.  Its output must equal ts_export_edges' on two calls in a
row -- the second on a different state, so that what the first call left in the shared array would show if it
mattered -- and a state beyond the stated limit must be refused.  Edge lists are integers: the comparison is exact.

Collected last on purpose (the name): the suite runs with pytest -x."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ts():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2508_06628_b200 as m
    m.lib()
    return m


def _both_exports(ts, torch, st):
    """(existing path, static path) for the current positions of `st`; the caller's buffers are filled with a
    sentinel first, so an entry the kernel did not write cannot pass."""
    ei, es = st.export_edges()
    ei, es = ei.clone(), es.clone()
    cap = st.capacity()[2]
    oi = torch.full((2, cap), -7, dtype=torch.int64, device=st.device)
    os_ = torch.full((cap, 3), -7.0, dtype=st.tdtype, device=st.device)
    on = torch.full((1,), -7, dtype=torch.int64, device=st.device)
    before = torch.cuda.memory_allocated()
    st.export_edges_static(oi, os_, on)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before            # torch's view: nothing was allocated around the call
    n = int(on.item())
    return (ei, es), (oi[:, :n], os_[:n]), n


def test_static_scratch_export_equals_workspace_export_twice(ts):
    import torch
    assert ts.ts_static_scratch_setup() == 16384
    # call 1: 3 x 108 fcc argon atoms, box < 2 r_list (image shifts matter), fp64
    a = wl.cfg1(n_systems=3, reps=3)
    sa = ts.SimState(a, engine=0)
    sa.md_step_external(ts.md_params(**a.md), ts.TS_PHASE_INIT)
    (ei, es), (oi, os_), n = _both_exports(ts, torch, sa)
    assert n == ei.shape[1] and n > 0
    assert torch.equal(oi, ei) and torch.equal(os_, es)
    # call 2, directly after, another state: more systems of other sizes, fp32 -- every entry of the shared array
    # that call 1 wrote is now stale
    b = wl.cfg3(n_systems=7, dtype="f32", n_range=(32, 200))
    sb = ts.SimState(b, engine=0)
    sb.md_step_external(ts.md_params(**b.md), ts.TS_PHASE_INIT)
    (ei2, es2), (oi2, os2), n2 = _both_exports(ts, torch, sb)
    assert n2 == ei2.shape[1] and n2 > 0 and n2 != n
    assert torch.equal(oi2, ei2) and torch.equal(os2, es2)
    # and the first state again after a few steps (positions moved; the list is skin-checked / rebuilt inside)
    sa.md_step(ts.md_params(**a.md), 30)
    (ei3, es3), (oi3, os3), n3 = _both_exports(ts, torch, sa)
    assert n3 == ei3.shape[1] and torch.equal(oi3, ei3) and torch.equal(os3, es3)
    sa.close(); sb.close()


def test_static_scratch_export_refuses_more_systems_than_the_array_holds(ts):
    import torch
    few = wl.cfg4(range(32), n_atoms=16, clean=False)
    big = wl.concat([few] * 513)                               # 16,416 systems > 16,384
    assert big.n_systems > ts.ts_static_scratch_setup()
    st = ts.SimState(big, engine=0)
    cap = 1024
    oi = torch.full((2, cap), -7, dtype=torch.int64, device=st.device)
    os_ = torch.full((cap, 3), -7.0, dtype=st.tdtype, device=st.device)
    on = torch.full((1,), -7, dtype=torch.int64, device=st.device)
    with pytest.raises(ts.TsError) as err:
        st.export_edges_static(oi, os_, on)
    assert err.value.code == ts.TS_ERR_WORKSPACE_TOO_SMALL and "16384" in str(err.value)
    torch.cuda.synchronize()
    assert int(on.item()) == -7 and int(oi.min().item()) == -7 and int(oi.max().item()) == -7     # nothing was written
    st.close()
