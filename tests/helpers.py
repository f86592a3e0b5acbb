"""Small helpers shared by the tests (no method arithmetic beyond numpy reference formulas
that the individual tests state and cite)."""
import numpy as np

import workloads as W


def random_periodic_case(nx, ny, nz, seed=0, amp=0.2, **kw):
    """Smooth-ish random positive state on a periodic box; returns a Case."""
    rng = np.random.default_rng(seed)
    lx, ly, lz = kw.pop("lx", 2.0), kw.pop("ly", 3.0), kw.pop("lz", 2.5)

    def f():
        return rng.uniform(-1.0, 1.0, (nz, ny, nx))
    rho = 1.0 + amp * f()
    u, v, w = 0.7 * f(), 0.7 * f(), 0.7 * f()
    p = 1.0 + amp * f()
    gamma = kw.get("gamma", 1.4)
    base = dict(name="rand", nx=nx, ny=ny, nz=nz, lx=lx, ly=ly, lz=lz, gamma=gamma,
                w0=W.conserved_from_primitive(rho, u, v, w, p, gamma))
    base.update(kw)
    return W.Case(**base), (rho, u, v, w, p)


def field_err(a, b, floor=0.0):
    """Field-wise normalised max error (SURVEY 8(c) comparison rule): max|a-b| / max(max|b|, floor)."""
    a = np.asarray(a)
    b = np.asarray(b)
    scale = max(float(np.max(np.abs(b))), floor)
    return float(np.max(np.abs(a - b)) / (scale if scale > 0 else 1.0))


def natural_scales(case):
    """Per-equation magnitudes used as a FLOOR of the normalisation: state scale W_v = (rho, rho c, rho c,
    rho c, rho c^2) and advective rate (|u|+c)_max * largest metric.  A field whose reference is itself at
    round-off level (e.g. the mass RHS of the divergence-free Taylor-Green field, ~1e-15) has no meaningful
    relative error; it is measured against 1e-3 of these scales instead."""
    w = case.w0
    g = case.gamma
    rho = w[0]
    vel2 = (w[1] ** 2 + w[2] ** 2 + w[3] ** 2) / rho ** 2
    p = (g - 1) * (w[4] - 0.5 * rho * vel2)
    c = np.sqrt(g * p / rho)
    rc = float(np.max(rho * c))
    Wv = np.array([float(rho.max()), rc, rc, rc, float(np.max(rho * c * c))])
    if case.y_nodes is not None:
        dy = float(np.min(np.diff(case.y_nodes)))
    elif case.bc_y_lo == W.BC_PERIODIC:
        dy = case.ly / case.ny
    else:
        dy = (case.y_wall_hi - case.y_wall_lo) / case.ny
    met = max(case.nx / case.lx, 1.0 / dy, case.nz / case.lz)
    rate = float(np.max(np.sqrt(vel2) + c)) * met
    return 1e-3 * Wv, 1e-3 * Wv * rate
