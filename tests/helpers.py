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


def field_err(a, b):
    """Field-wise normalised max error (SURVEY 8(c) comparison rule)."""
    a = np.asarray(a)
    b = np.asarray(b)
    scale = np.max(np.abs(b))
    return float(np.max(np.abs(a - b)) / (scale if scale > 0 else 1.0))
