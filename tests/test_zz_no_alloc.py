"""clt_diagnostics_static: the one entry point that uses no memory but the library's own (its scratch is a file-scope
static __device__ array, include/clt.h).  Checked against the existing path (clt_diagnostics + clt_suggest_dt, whose
block partials live in the caller's workspace) on calls in a row.  Collected last on purpose (file name)."""
import numpy as np
import pytest

from paper_1812_00525_b200 import inputs
from parity_util import make_gpu

pytestmark = pytest.mark.gpu

SUMS = ("kinetic", "magnetic", "magnetic_pert", "magnetic_n1")


def _compare(g, out, cfl, what):
    """The static-scratch result in `out` (already enqueued) against the existing path on the same state: the tolerances of
    test_diagnostics_and_suggest_dt_match_oracle (sums 1e-12, max |div B| 1e-10, dt 1e-13 relative)."""
    import torch
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    ref = g.diagnostics()
    for q, k in enumerate(SUMS):
        assert abs(got[q] - ref[k]) <= 1e-12 * abs(ref[k]), (what, k, got[q], ref[k])
    assert abs(got[4] - ref["max_divB"]) <= 1e-10 * abs(ref["max_divB"]) + 1e-15, (what, got[4], ref["max_divB"])
    dt = g.suggest_dt(cfl)
    assert abs(got[5] - dt) <= 1e-13 * dt, (what, got[5], dt)
    assert np.all(np.isfinite(got[:6])) and got[0] >= 0 and got[1] > 0


@pytest.mark.parametrize("phi_scheme", [0, 1])
def test_static_scratch_diagnostics_match_the_workspace_path_on_calls_in_a_row(phi_scheme):
    import torch
    # several tiles and a ragged tail in both directions; a second, smaller grid afterwards reads nothing the first left behind
    big = inputs.make_custom_problem(77, 16, 53, index=31, amplitude_scale=30.0)
    small = inputs.make_custom_problem(40, 8, 21, index=32, amplitude_scale=30.0)
    g = make_gpu(big, phi_scheme=phi_scheme)
    out = torch.full((6,), float("nan"), dtype=torch.float64, device="cuda")
    launches = g.launch_count
    g.diagnostics_static(out, 0.5)                       # first call: initial state
    assert g.launch_count == launches + 2                # the reduction kernel and the final kernel, nothing else
    _compare(g, out, 0.5, "first call")
    g.step(3)
    out.fill_(float("nan"))
    g.diagnostics_static(out, 0.4)                       # second call in a row: the state has moved, other cfl
    _compare(g, out, 0.4, "second call")
    # two calls back to back on one stream without anything in between: the second overwrites the scratch of the first
    out2 = torch.full((6,), float("nan"), dtype=torch.float64, device="cuda")
    g.diagnostics_static(out, 0.4)
    g.diagnostics_static(out2, 0.4)
    torch.cuda.synchronize()
    assert torch.equal(out, out2)
    h = make_gpu(small, phi_scheme=phi_scheme)
    out.fill_(float("nan"))
    h.diagnostics_static(out, 0.0)                       # cfl <= 0: params.cfl
    _compare(h, out, small.cfg.cfl, "smaller grid after a larger one")


def test_static_scratch_rejects_grids_beyond_its_limit_and_host_pointers():
    import torch
    from paper_1812_00525_b200 import clt
    prob = inputs.make_problem(1)
    g = make_gpu(prob)
    with pytest.raises((clt.CltError, TypeError)):
        g.diagnostics_static(np.empty(6), 0.5)           # a host pointer is refused
    with pytest.raises(clt.CltError) as e:
        g.diagnostics_static(torch.empty(6, dtype=torch.float64), 0.5)       # host tensor: not device memory
    assert e.value.code == clt.CLT_EINVAL
    # ceil((nR-4)/32) * (nZ-4) = 1 * 16386 > 16384 reduction CTAs: refused, with a text that says why
    c = prob.cfg
    big = clt.Clt(9, 5, 16390, c.Rmin, c.Rmax, c.Zmin, c.Zmax, c.phi_extent, c.gamma, c.eta, c.nu, c.D, c.kappa, prob.dt, c.cfl)
    out = torch.zeros(6, dtype=torch.float64, device="cuda")
    with pytest.raises(clt.CltError) as e:
        big.diagnostics_static(out, 0.5)
    assert e.value.code == clt.CLT_ENOMEM
    assert b"16384" in big.L.clt_last_cuda_error(big.h)
    big.close()
