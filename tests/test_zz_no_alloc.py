"""qa_ground_state_open_static (the entry point that allocates nothing: its workspace is a static __device__ array inside the
library) against qa_ground_state_open with a caller-allocated workspace.  Same kernels, same arithmetic: N must be equal
and E must agree to the 1e-9 relative of the parity tests (it is in fact bit-identical).  Collected last on purpose (file
name): the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

from paper_2404_04994_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    from paper_2404_04994_b200 import api as _api
    assert torch.cuda.is_available()
    return _api


def _pair(api, m, Vg, **kw):
    ref = m.ground_state(Vg, **kw)                      # workspace: a torch allocation of the binding
    got = m.ground_state_static(Vg, **kw)               # workspace: the library's static array
    torch.cuda.synchronize()
    N0, E0 = ref["N"].cpu().numpy(), ref["E"].cpu().numpy()
    N1, E1 = got["N"].cpu().numpy(), got["E"].cpu().numpy()
    assert np.array_equal(N0, N1)
    assert np.allclose(E0, E1, rtol=1e-9, atol=1e-9 * m.inverse()[1])
    return N1, E1


def test_static_workspace_two_calls_in_a_row(api):
    """Two calls in a row on the shared array, different sweeps and sizes (the second finds the first one's contents), on the
    three-launch path that really goes through the workspace (16 dots: prologue -> walk -> finish), then the pruned walk
    (its work counter must start at zero in every call) and a 13-dot array."""
    assert api.lib().qa_static_workspace_bytes() == 16 << 20
    assert api.lib().qa_static_workspace_init() == 0
    w = wl.random_open(16, 16, 3001, seed=77, lo=-0.7, hi=3.3)
    m = api.Model(w.C_dd, w.C_gd)
    Vg = torch.from_numpy(w.Vg).cuda()
    Na, _ = _pair(api, m, Vg)
    assert api.last_launch_plan()[0] == ["qa_prologue_lanes_kernel", "qa_minplus_walk_kernel", "qa_minplus_finish_kernel"]
    w2 = wl.random_open(16, 16, 1777, seed=78, lo=-0.5, hi=2.9)
    Vg2 = torch.from_numpy(w2.Vg).cuda()
    Nb, _ = _pair(api, m, Vg2)
    # the first sweep once more: the array now holds the second call's data
    Nc, _ = _pair(api, m, Vg)
    assert np.array_equal(Na, Nc)
    assert Nb.shape == (1777, 16)
    for variant in (2, 0):
        m.set_walk_variant(variant)
        _pair(api, m, Vg2)
        _pair(api, m, Vg2)
    m.set_walk_variant(1)
    _pair(api, m, Vg, algorithm="thresholded", t=0.3)
    w3 = wl.random_open(13, 13, 999, seed=79)
    m3 = api.Model(w3.C_dd, w3.C_gd)
    _pair(api, m3, torch.from_numpy(w3.Vg).cuda())
    _pair(api, m3, torch.from_numpy(w3.Vg).cuda())


def test_static_workspace_caller_buffers_and_limit(api):
    """Outputs in buffers the caller made beforehand (nothing is allocated between the two calls), and the size limit: a sweep
    whose workspace exceeds the 16 MiB is refused with QA_ERR_STATIC_WORKSPACE before anything is enqueued."""
    w = wl.config4(40, 35)
    m = api.Model(w.C_dd, w.C_gd)
    Vg = torch.from_numpy(w.Vg).cuda()
    ref = m.ground_state(Vg)
    out = {"N": torch.full((w.P, 16), -7, dtype=torch.int32, device="cuda"),
           "E": torch.full((w.P,), np.nan, dtype=torch.float64, device="cuda")}
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    for _ in range(2):
        m.ground_state_static(Vg, out=out)
        torch.cuda.synchronize()
        assert torch.equal(out["N"], ref["N"]) and torch.equal(out["E"], ref["E"])
        out["N"].fill_(-7)
    assert torch.cuda.memory_allocated() == before
    # limit: 16 MiB / 664 B per pixel at 16 dots
    lib = api.lib()
    P_big = 30000
    assert lib.qa_workspace_bytes(m._h, P_big) > (16 << 20)
    big = torch.zeros((P_big, w.C_gd.shape[1]), dtype=torch.float64, device="cuda")
    with pytest.raises(api.QaError) as ei:
        m.ground_state_static(big)
    assert ei.value.status == 9 and "static workspace holds" in str(ei.value)
    P_ok = 25000
    assert lib.qa_workspace_bytes(m._h, P_ok) <= (16 << 20)
    r = m.ground_state_static(big[:P_ok])
    torch.cuda.synchronize()
    assert int(r["N"].min()) >= 0
    # empty sweep: nothing to do, no error
    assert m.ground_state_static(big[:0])["N"].shape == (0, 16)
