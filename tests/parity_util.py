"""Helpers shared by the GPU parity tests: build both sides from one seeded problem, error metric H4."""
import numpy as np

import oracle as orc
from paper_1812_00525_b200 import inputs

RHS_TOL = 1e-12      # BASELINE.json north_star: relative L-infinity per RHS call
STEP_TOL = 1e-9      # ... and after 100 RK4 steps


def make_oracle(prob, **over):
    c = prob.cfg
    par = dict(gamma=c.gamma, eta=c.eta, nu=c.nu, D=c.D, kappa=c.kappa, dt=prob.dt)
    par.update(over)
    o = orc.Oracle(c.nR, c.nphi, c.nZ, c.Rmin, c.Rmax, c.Zmin, c.Zmax, c.phi_extent, **par)
    o.set_equilibrium(prob.U0)
    o.set_state(prob.U)
    return o


def make_gpu(prob, set_eq=True, **over):
    from paper_1812_00525_b200 import clt
    c = prob.cfg
    par = dict(gamma=c.gamma, eta=c.eta, nu=c.nu, D=c.D, kappa=c.kappa, dt=prob.dt, cfl=c.cfl)
    par.update(over)
    phi_scheme = par.pop("phi_scheme", 0)
    g = clt.Clt(c.nR, c.nphi, c.nZ, c.Rmin, c.Rmax, c.Zmin, c.Zmax, c.phi_extent, **par)
    if phi_scheme:
        g.set_phi_scheme(phi_scheme)
    if set_eq:
        g.set_equilibrium(np.ascontiguousarray(prob.U0))
    g.set_state(np.ascontiguousarray(prob.U))
    return g


def rel_linf(got, exp):
    """Per leading-index field: max|g - c| / max(max|c|, tiny) over all nodes (boundary layers must agree too)."""
    out = []
    for f in range(exp.shape[0]):
        s = max(np.abs(exp[f]).max(), 1e-300)
        out.append(float(np.abs(got[f] - exp[f]).max() / s))
    return out


def assert_close(got, exp, tol, what):
    errs = rel_linf(got, exp)
    assert max(errs) <= tol, f"{what}: rel Linf per field {errs} > {tol}"
    return errs


def rel_linf_physical(got, exp):
    """Reading R10: the state is rho, p, the vector v and the vector B; a vector's error is measured in
    the max-norm of the whole vector, i.e. each component's max|g - c| is divided by the largest component's max|c|.
    Needed where one component is orders of magnitude smaller than the others (config 5's v_phi ~ 1e-7 next to
    p ~ 1e-2): there a 1-ulp difference in the stored total p already moves grad(p - p0), hence v_phi, by 1e-9 of
    itself (tests/test_oracle_pins.py::test_rounding_noise_floor_of_the_oracle_itself)."""
    groups = [[0], [1], [2, 3, 4], [5, 6, 7]]
    out = []
    for grp in groups:
        s = max(max(np.abs(exp[f]).max() for f in grp), 1e-300)
        out.append(max(float(np.abs(got[f] - exp[f]).max() / s) for f in grp))
    return out


def assert_close_physical(got, exp, tol, what):
    errs = rel_linf_physical(got, exp)
    assert max(errs) <= tol, f"{what}: rel Linf per physical field (rho, p, v, B) {errs} > {tol}"
    return errs
