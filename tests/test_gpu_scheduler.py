"""In-flight scheduler on the GPU: every stream id is relaxed exactly once, the
slots never exceed the byte budget, and each final state passes the oracle's own convergence check."""
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


def test_inflight_relaxer_small_stream(ts, orc):
    from paper_2508_06628_b200 import scheduler as sch
    n_total, n_atoms = 14, 64
    make = lambda ids: wl.cfg4(ids, n_atoms=n_atoms)
    fire = dict(make([0]).fire, f_max=1e-4, max_steps=20000)
    per = sch.batch_system_bytes(make([0]))[0]
    r = sch.InFlightRelaxer(make, n_total, fire, budget_bytes=5.5 * per, k_check=10)
    assert r.n_slots == 5                                     # admission from the byte budget (a9)
    res = r.run()
    assert sorted(res) == list(range(n_total)) and r.unfinished == []
    assert r.peak_resident <= r.n_slots
    for sid, rec in res.items():
        assert rec["status"] == ts.TS_FIRE_CONVERGED
        b = wl.with_(make([sid]), pos=rec["pos"])
        o = orc.energy_forces(b)
        assert np.sqrt((o["F"] ** 2).sum(1)).max() < fire["f_max"]             # R30(ii)
        assert abs(rec["energy"] - o["E"][0]) <= 1e-12 * max(abs(o["E"][0]), o["Eabs"][0])
    # batch-composition independence (R22): a different slot count gives the same step counts and minima
    r2 = sch.InFlightRelaxer(make, n_total, fire, n_slots=3, k_check=7)
    res2 = r2.run()
    for sid in res:
        assert res2[sid]["fire_steps"] == res[sid]["fire_steps"]
        assert np.abs(res2[sid]["pos"] - res[sid]["pos"]).max() <= 1e-6


def test_estimate_covers_actual_list_size(ts):
    """Predicted bytes >= bytes actually used (nnz within capacity) on cfg2- and cfg3-shaped batches."""
    for b in (wl.cfg2(n_systems=3, dtype="f32"), wl.cfg3(n_systems=10, dtype="f32", n_range=(32, 600))):
        st = ts.SimState(b, engine=0)
        st.build_neighbors()
        rep = st.poll()
        assert rep.flags == 0 and rep.nnz <= rep.nnz_capacity
        from paper_2508_06628_b200 import scheduler as sch
        assert sch.batch_system_bytes(b).sum() >= 4 * rep.nnz
        st.close()
