"""Helpers shared by the GPU parity tests: build both sides from one seeded problem, error metric H4."""
import ctypes
import functools
import json
import os
import subprocess

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


@functools.lru_cache(maxsize=None)
def oracle_run(index, steps):
    """BASELINE.json config `index` through the oracle, once per test session: the RHS of the initial state, the state
    after `steps` RK4 steps and its diagnostics.  (Configs 3-5 cost the oracle minutes; several tests compare with them.)"""
    prob = inputs.make_problem(index)
    o = make_oracle(prob)
    K = o.rhs()
    o.step(steps)
    return {"prob": prob, "K": K, "U": o.get_state(), "diag": o.diagnostics()}


def fma_oracle(prob, tmpdir, **over):
    """The oracle's own source built with FMA contraction (gcc -ffp-contract=fast -march=native): same arithmetic, other
    rounding.  Two oracle builds differ by nothing but round-off, so their distance is the rounding-noise floor of a
    run -- the yardstick reading R10 is measured against.  Returns None where the host has no FMA."""
    src = os.path.join(os.path.dirname(orc.__file__), "clt_oracle.c")
    so = os.path.join(str(tmpdir), "liboracle_fma.so")
    r = subprocess.run(["gcc", "-O2", "-ffp-contract=fast", "-march=native", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-o", so,
                        src, "-lm"], capture_output=True)
    if r.returncode != 0 or "fma" not in open("/proc/cpuinfo").read():
        return None
    c = prob.cfg
    par = dict(gamma=c.gamma, eta=c.eta, nu=c.nu, D=c.D, kappa=c.kappa, dt=prob.dt)
    par.update(over)
    o = orc.Oracle(c.nR, c.nphi, c.nZ, c.Rmin, c.Rmax, c.Zmin, c.Zmax, c.phi_extent, **par)
    L2 = ctypes.CDLL(so)
    for name in ("oracle_create", "oracle_destroy", "oracle_set_equilibrium", "oracle_set_state", "oracle_get_state",
                 "oracle_step", "oracle_rhs"):
        getattr(L2, name).argtypes = getattr(o.L, name).argtypes
        getattr(L2, name).restype = getattr(o.L, name).restype
    o.close()
    o.L = L2                      # same prototypes, other rounding: rebind this instance to the FMA build
    o.h = L2.oracle_create(c.nR, c.nphi, c.nZ, c.Rmin, c.Rmax, c.Zmin, c.Zmax, c.phi_extent, par["gamma"], par["eta"],
                           par["nu"], par["D"], par["kappa"], par["dt"])
    o.set_equilibrium(prob.U0)
    o.set_state(prob.U)
    return o


def record_margin(key, value):
    """Observed parity margins go to gpurun_out/parity_margins.json when CLT_RECORD_MARGINS is set (BASELINE.md section 4
    quotes them); a plain run records nothing."""
    if not os.environ.get("CLT_RECORD_MARGINS"):
        return
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    path = os.path.join(root, "gpurun_out", "parity_margins.json")
    os.makedirs(os.path.dirname(path), exist_ok=True)
    data = json.load(open(path)) if os.path.exists(path) else {}
    data[key] = value
    json.dump(data, open(path, "w"), indent=1, sort_keys=True)


def make_gpu(prob, set_eq=True, **over):
    from paper_1812_00525_b200 import clt
    c = prob.cfg
    par = dict(gamma=c.gamma, eta=c.eta, nu=c.nu, D=c.D, kappa=c.kappa, dt=prob.dt, cfl=c.cfl)
    par.update(over)
    phi_scheme = par.pop("phi_scheme", 0)
    if par.pop("textbook_rk4", False):       # the -DCLT_TEXTBOOK_RK4 build of the same sources (A/B only)
        par["lib_path"] = clt.LIB_TEXTBOOK_PATH
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
