"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 0-4).

This module holds case descriptions (grid / gas / scheme parameters as plain numbers)
and initial conserved fields.  It contains none of the method's arithmetic (no flux,
sensor, derivative, RK or dt code) and imports neither the oracle nor the CUDA path;
both bindings marshal a `Case` into their own C structs.  All randomness comes from
numpy's PCG64 seeded explicitly, so every field is reproducible.

The paper's own workloads are the authors' production DNS set-ups (not in
the container); these stand in for them with the same structure: periodic box,
two-wall channel with tanh-stretched y, wall + free stream (recipe: DESIGN.md,
SURVEY.md section 8(d)).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

BC_PERIODIC, BC_WALL_ISOTHERMAL, BC_FREESTREAM = 0, 1, 2
BC_HALO = 3                                  # bc_z of a z slab of a sharded run: ghost planes come from the neighbours
VISC_NONE, VISC_POWER, VISC_SUTHERLAND = 0, 1, 2
FLUX_CENTRAL, FLUX_WENO, FLUX_HYBRID = 0, 1, 2


@dataclasses.dataclass
class Case:
    """One problem: parameters in the layout of the C ABI structs plus the initial field."""
    name: str
    # grid
    nx: int
    ny: int
    nz: int
    lx: float
    ly: float
    lz: float
    y_nodes: Optional[np.ndarray] = None     # ny node coordinates, None = uniform
    y_wall_lo: float = 0.0
    y_wall_hi: float = 0.0
    bc_x: int = BC_PERIODIC
    bc_y_lo: int = BC_PERIODIC
    bc_y_hi: int = BC_PERIODIC
    bc_z: int = BC_PERIODIC
    t_wall_lo: float = 1.0
    t_wall_hi: float = 1.0
    nz_global: int = 0                       # z nodes of the whole domain when this case is a slab (bc_z = BC_HALO)
    # gas
    gamma: float = 1.4
    rgas: float = 1.0
    prandtl: float = 0.72
    visc_law: int = VISC_NONE
    mu_ref: float = 0.0
    t_ref: float = 1.0
    suth_s_over_tref: float = 110.4 / 288.15
    pow_exp: float = 0.76
    u_ref: float = 1.0
    l_ref: float = 1.0
    freestream: tuple = (1.0, 0.0, 0.0, 0.0, 2.5)
    accel: tuple = (0.0, 0.0, 0.0)           # uniform body acceleration (channel driving force)
    # scheme
    central_order: int = 6
    weno_order: int = 5
    visc_order: int = 6
    flux_mode: int = FLUX_CENTRAL
    sensor_threshold: float = 0.2
    weno_eps: float = 1e-6
    weno_variant: int = 0                    # 0: Jiang-Shu weights, 1: WENO-Z
    cfl: float = 0.5
    dt_fixed: float = 0.0
    dt_every: int = 1
    # run
    nsteps: int = 1
    w0: Optional[np.ndarray] = None          # [5, nz, ny, nx] conserved, float64

    @property
    def npoints(self) -> int:
        return self.nx * self.ny * self.nz

    def replace(self, **kw) -> "Case":
        return dataclasses.replace(self, **kw)


def conserved_from_primitive(rho, u, v, w, p, gamma):
    """Pack (rho, u, v, w, p) into the conserved array [5, nz, ny, nx] (input marshalling only)."""
    out = np.empty((5,) + rho.shape, dtype=np.float64)
    out[0] = rho
    out[1] = rho * u
    out[2] = rho * v
    out[3] = rho * w
    out[4] = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w)
    return out


def _grid_xyz(nx, ny, nz, lx, ly, lz, y_nodes=None):
    x = np.arange(nx) * (lx / nx)
    y = np.arange(ny) * (ly / ny) if y_nodes is None else np.asarray(y_nodes)
    z = np.arange(nz) * (lz / nz)
    return np.meshgrid(z, y, x, indexing="ij")  # Z, Y, X with shape [nz, ny, nx]


# ----------------------------------------------------------------------------------------
# config 0: inviscid Taylor-Green vortex (closed form, no seed)
# ----------------------------------------------------------------------------------------
def taylor_green(n: int = 32, nsteps: int = 10, mach: float = 0.1) -> Case:
    gamma = 1.4
    p0 = 1.0 / (gamma * mach * mach)
    two_pi = 2.0 * math.pi
    Z, Y, X = _grid_xyz(n, n, n, two_pi, two_pi, two_pi)
    rho = np.ones_like(X)
    u = np.sin(X) * np.cos(Y) * np.cos(Z)
    v = -np.cos(X) * np.sin(Y) * np.cos(Z)
    w = np.zeros_like(X)
    p = p0 + (np.cos(2 * X) + np.cos(2 * Y)) * (np.cos(2 * Z) + 2.0) / 16.0
    return Case(name=f"cfg0_tgv_{n}", nx=n, ny=n, nz=n, lx=two_pi, ly=two_pi, lz=two_pi,
                gamma=gamma, rgas=p0, visc_law=VISC_NONE, flux_mode=FLUX_CENTRAL,
                central_order=6, cfl=0.5, nsteps=nsteps, u_ref=math.sqrt(gamma * p0), l_ref=two_pi,
                freestream=(1.0, 0.0, 0.0, 0.0, p0 / (gamma - 1.0)),
                w0=conserved_from_primitive(rho, u, v, w, p, gamma))


# ----------------------------------------------------------------------------------------
# random band-limited solenoidal velocity, E(k) ~ k^4 exp(-2 (k/k0)^2)
# ----------------------------------------------------------------------------------------
def solenoidal_velocity(nx, ny, nz, k0, kmax, seed, dilatational=0.0):
    """Real solenoidal field on [0,2pi)^3 from Gaussian Fourier coefficients on integer
    wavevectors |k| <= kmax projected perpendicular to k, amplitude ~ sqrt(E(k))/k.
    dilatational > 0 keeps that fraction of the component along k (parity tests use it so that the
    shock sensor fires at step 0; the BASELINE configs are purely solenoidal)."""
    import scipy.fft as sfft
    rng = np.random.default_rng(seed)
    K = int(min(kmax, nx // 2 - 1, ny // 2 - 1, nz // 2 - 1))
    kk = np.arange(-K, K + 1)
    KZ, KY, KX = np.meshgrid(kk, kk, kk, indexing="ij")
    kmag = np.sqrt(KX * KX + KY * KY + KZ * KZ).astype(np.float64)
    inside = (kmag > 0) & (kmag <= K)
    amp = np.zeros_like(kmag)
    km = kmag[inside]
    amp[inside] = np.sqrt(km ** 4 * np.exp(-2.0 * (km / k0) ** 2)) / km
    shape = kmag.shape
    c = [(rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) * amp for _ in range(3)]
    ksq = np.where(inside, kmag * kmag, 1.0)
    kdotc = (KX * c[0] + KY * c[1] + KZ * c[2]) / ksq
    kdotc = (1.0 - dilatational) * kdotc
    c = [c[0] - KX * kdotc, c[1] - KY * kdotc, c[2] - KZ * kdotc]
    out = []
    for comp in c:
        # spectrum of Re(sum c e^{ikx}) = (c(k) + conj c(-k)) / 2 ; keep kz >= 0 half
        sym = 0.5 * (comp + np.conj(comp[::-1, ::-1, ::-1]))
        spec = np.zeros((nz, ny, nx // 2 + 1), dtype=np.complex128)
        half = sym[:, :, K:]                     # kx = 0 .. K
        kz_idx = kk % nz
        ky_idx = kk % ny
        spec[np.ix_(kz_idx, ky_idx, np.arange(0, K + 1))] = half
        # numpy's irfftn wants the LAST axis halved: axes order (z, y, x) with x halved
        field = sfft.irfftn(spec, s=(nz, ny, nx), axes=(0, 1, 2), workers=-1) * (nx * ny * nz)
        out.append(field)
    return out  # [u, v, w] each [nz, ny, nx]


def isotropic_turbulence(n=128, mach_t=0.6, k0=4.0, kmax=32, seed=1, nsteps=50,
                         re_lambda=100.0, flux_mode=FLUX_HYBRID, viscous=True,
                         nx=None, ny=None, nz=None, name=None, dilatational=0.0) -> Case:
    """configs 1 and 4: decaying compressible isotropic turbulence in a periodic box."""
    nx = nx or n
    ny = ny or n
    nz = nz or n
    gamma = 1.4
    c0 = math.sqrt(gamma)           # rho0 = T0 = R = 1
    two_pi = 2.0 * math.pi
    u, v, w = solenoidal_velocity(nx, ny, nz, k0, kmax, seed, dilatational)
    rms = math.sqrt(float(np.mean(u * u + v * v + w * w)))
    scale = mach_t * c0 / rms
    u *= scale
    v *= scale
    w *= scale
    rho = np.ones_like(u)
    p = np.ones_like(u)
    uprime = mach_t * c0 / math.sqrt(3.0)
    lam = 2.0 / k0
    mu_ref = uprime * lam / re_lambda
    return Case(name=name or f"iso_{nx}x{ny}x{nz}_mt{mach_t}", nx=nx, ny=ny, nz=nz,
                lx=two_pi, ly=two_pi, lz=two_pi, gamma=gamma, rgas=1.0, prandtl=0.72,
                visc_law=VISC_SUTHERLAND if viscous else VISC_NONE, mu_ref=mu_ref, t_ref=1.0,
                u_ref=c0, l_ref=two_pi, flux_mode=flux_mode, sensor_threshold=0.2,
                central_order=6, weno_order=5, visc_order=6, cfl=0.5, nsteps=nsteps,
                freestream=(1.0, 0.0, 0.0, 0.0, 1.0 / (gamma - 1.0)),
                w0=conserved_from_primitive(rho, u, v, w, p, gamma))


def _band_limited_xz(nx, nz, lx, lz, kmax, rng, ncomp=3):
    """Random real fields f(x, z) with |kx|, |kz| <= kmax modes, unit rms. Shape [ncomp, nz, nx]."""
    x = np.arange(nx) * (2.0 * math.pi / nx)
    z = np.arange(nz) * (2.0 * math.pi / nz)
    out = np.zeros((ncomp, nz, nx))
    ks = np.arange(-kmax, kmax + 1)
    ex = np.exp(1j * np.outer(ks, x))          # [nk, nx]
    ez = np.exp(1j * np.outer(ks, z))          # [nk, nz]
    for c in range(ncomp):
        coef = rng.standard_normal((ks.size, ks.size)) + 1j * rng.standard_normal((ks.size, ks.size))
        coef[kmax, kmax] = 0.0
        f = np.real(ez.T @ coef @ ex)
        out[c] = f / math.sqrt(float(np.mean(f * f)))
    return out


def channel(nx=256, ny=192, nz=128, seed=2, nsteps=50, stretch_b=1.5, mach_b=1.5,
            re_b=3000.0, pert=0.05, flux_mode=FLUX_HYBRID, name=None) -> Case:
    """config 2: supersonic isothermal-wall channel, tanh-stretched y in [-1, 1]."""
    gamma = 1.4
    lx, lz = 6.0 * math.pi, 2.0 * math.pi
    eta = -1.0 + (2.0 * np.arange(ny) + 1.0) / ny
    y = np.tanh(stretch_b * eta) / math.tanh(stretch_b)
    cw = math.sqrt(gamma)           # R = 1, T_w = 1
    ub = mach_b * cw
    mu_w = 1.0 * ub * 1.0 / re_b
    rng = np.random.default_rng(seed)
    modes = _band_limited_xz(nx, nz, lx, lz, 8, rng, 3)            # [3, nz, nx]
    env = (1.0 - y * y) ** 2                                        # [ny]
    prof = 1.5 * ub * (1.0 - y * y)
    u = prof[None, :, None] + pert * ub * env[None, :, None] * modes[0][:, None, :]
    v = pert * ub * env[None, :, None] * modes[1][:, None, :]
    w = pert * ub * env[None, :, None] * modes[2][:, None, :]
    rho = np.ones_like(u)
    p = np.ones_like(u)
    return Case(name=name or f"cfg2_channel_{nx}x{ny}x{nz}", nx=nx, ny=ny, nz=nz, lx=lx, ly=2.0, lz=lz,
                y_nodes=y, y_wall_lo=-1.0, y_wall_hi=1.0,
                bc_y_lo=BC_WALL_ISOTHERMAL, bc_y_hi=BC_WALL_ISOTHERMAL, t_wall_lo=1.0, t_wall_hi=1.0,
                gamma=gamma, rgas=1.0, prandtl=0.72, visc_law=VISC_SUTHERLAND, mu_ref=mu_w, t_ref=1.0,
                u_ref=cw, l_ref=lx, flux_mode=flux_mode, sensor_threshold=0.2, cfl=0.5, nsteps=nsteps,
                freestream=(1.0, 0.0, 0.0, 0.0, 1.0 / (gamma - 1.0)),
                w0=conserved_from_primitive(rho, u, v, w, p, gamma))


def boundary_layer(nx=1024, ny=256, nz=256, seed=3, nsteps=20, mach=2.0, re_delta=5000.0,
                   nblobs=64, blob_amp=0.3, stretch_b=2.0, flux_mode=FLUX_HYBRID, name=None) -> Case:
    """config 3: supersonic flat-plate boundary-layer box (temporal layer, x/z periodic,
    isothermal wall at T_aw below, free-stream fill on top)."""
    gamma, pr = 1.4, 0.72
    delta = 1.0
    lx, ly, lz = 64.0 * delta * nx / 1024.0, 8.0 * delta, 8.0 * delta * nz / 256.0
    eta = (np.arange(ny) + 0.5) / ny
    y = ly * (1.0 - np.tanh(stretch_b * (1.0 - eta)) / math.tanh(stretch_b))
    c_inf = math.sqrt(gamma)        # R = 1, T_inf = 1, rho_inf = 1, p = 1
    U = mach * c_inf
    rfac = math.sqrt(pr)
    t_aw = 1.0 + rfac * 0.5 * (gamma - 1.0) * mach * mach
    zeta = np.minimum(y / delta, 1.0)
    uprof = U * (2.0 * zeta - 2.0 * zeta ** 3 + zeta ** 4)
    tprof = t_aw - rfac * 0.5 * (gamma - 1.0) * mach * mach * (uprof / U) ** 2
    rng = np.random.default_rng(seed)
    modes = _band_limited_xz(nx, nz, lx, lz, 8, rng, 3)
    env = np.where(y < 1.5 * delta, np.sin(math.pi * np.minimum(y / (1.5 * delta), 1.0)) ** 2, 0.0)
    u = uprof[None, :, None] + 0.01 * U * env[None, :, None] * modes[0][:, None, :]
    v = 0.01 * U * env[None, :, None] * modes[1][:, None, :]
    w = 0.01 * U * env[None, :, None] * modes[2][:, None, :]
    # seeded compressive blobs: u' = -A (x - xc)/sigma exp(-|x - xc|^2 / (2 sigma^2))
    dx = lx / nx
    sigma = 4.0 * dx
    xg = np.arange(nx) * dx
    zg = np.arange(nz) * (lz / nz)
    cx = rng.uniform(0.0, lx, nblobs)
    cy = rng.uniform(0.3 * delta, 2.0 * delta, nblobs)
    cz = rng.uniform(0.0, lz, nblobs)
    rad = 5.0 * sigma
    for b in range(nblobs):
        ix = np.nonzero(np.abs((xg - cx[b] + 0.5 * lx) % lx - 0.5 * lx) < rad)[0]
        iy = np.nonzero(np.abs(y - cy[b]) < rad)[0]
        iz = np.nonzero(np.abs((zg - cz[b] + 0.5 * lz) % lz - 0.5 * lz) < rad)[0]
        if ix.size == 0 or iy.size == 0 or iz.size == 0:
            continue
        rx = ((xg[ix] - cx[b] + 0.5 * lx) % lx - 0.5 * lx)[None, None, :]
        ry = (y[iy] - cy[b])[None, :, None]
        rz = ((zg[iz] - cz[b] + 0.5 * lz) % lz - 0.5 * lz)[:, None, None]
        g = blob_amp * U * np.exp(-(rx * rx + ry * ry + rz * rz) / (2.0 * sigma * sigma)) / sigma
        sel = np.ix_(iz, iy, ix)
        u[sel] -= g * rx
        v[sel] -= g * ry
        w[sel] -= g * rz
    p = np.ones_like(u)
    rho = p / (1.0 * tprof[None, :, None] * np.ones_like(u))
    mu_inf = 1.0 * U * delta / re_delta
    e_inf = 1.0 / (gamma - 1.0) + 0.5 * U * U
    return Case(name=name or f"cfg3_bl_{nx}x{ny}x{nz}", nx=nx, ny=ny, nz=nz, lx=lx, ly=ly, lz=lz,
                y_nodes=y, y_wall_lo=0.0, y_wall_hi=ly,
                bc_y_lo=BC_WALL_ISOTHERMAL, bc_y_hi=BC_FREESTREAM, t_wall_lo=t_aw, t_wall_hi=t_aw,
                gamma=gamma, rgas=1.0, prandtl=pr, visc_law=VISC_SUTHERLAND, mu_ref=mu_inf, t_ref=1.0,
                u_ref=c_inf, l_ref=lx, flux_mode=flux_mode, sensor_threshold=0.2, cfl=0.5, nsteps=nsteps,
                freestream=(1.0, U, 0.0, 0.0, e_inf),
                w0=conserved_from_primitive(rho, u, v, w, p, gamma))


def config(index: int, scale: float = 1.0) -> Case:
    """BASELINE.json configs[index]; scale < 1 shrinks the grid (ragged sizes kept) for parity replicas."""
    def s(n, lo=12):
        return max(lo, int(round(n * scale)))
    if index == 0:
        return taylor_green(32 if scale == 1.0 else s(32), nsteps=10)
    if index == 1:
        n = s(128)
        return isotropic_turbulence(n=n, mach_t=0.6, k0=4.0, kmax=32, seed=1, nsteps=50, name=f"cfg1_iso_{n}")
    if index == 2:
        return channel(s(256), s(192), s(128), seed=2, nsteps=50)
    if index == 3:
        return boundary_layer(s(1024), s(256), s(256), seed=3, nsteps=20)
    if index == 4:
        n = s(640)
        return isotropic_turbulence(n=n, mach_t=0.8, k0=8.0, kmax=64, seed=4, nsteps=10, name=f"cfg4_iso_{n}")
    raise ValueError(index)
