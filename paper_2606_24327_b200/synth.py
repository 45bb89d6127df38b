"""Seeded synthetic inputs shaped like the paper's ITG workloads.

This module serves BOTH the CPU oracle and the CUDA path and therefore holds none of the
method's arithmetic: no C1 element, no B-spline evaluation, no equilibrium field, no equations
of motion.  It only draws numbers and writes down closed-form test fields.  The paper's own
decks (Cyclone base case; TCV-X21, L338-342) are not available; these
inputs take their shapes (marker counts L200, N_r 16-32 and n = 6..18 L320, rho* = 1/60 L320,
Eq.(8) profiles L314) and stand in for them.

RNG: stateless counter hash, splitmix64 of (seed, stream, index) -> U(0,1) = (x>>11)*2^-53 + 2^-54;
normals by Box-Muller.  Same numbers on every platform, any order of generation.
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass, field

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = x
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return z ^ (z >> np.uint64(31))


def uniform(seed: int, stream: int, n: int, start: int = 0) -> np.ndarray:
    """n numbers in (0,1), counter-based: element i depends only on (seed, stream, start+i)."""
    idx = np.arange(start, start + n, dtype=np.uint64)
    with np.errstate(over="ignore"):
        key = _splitmix64(np.uint64(seed) * np.uint64(0x100000001B3) + np.uint64(stream))
        x = _splitmix64(idx ^ key)
        x = _splitmix64(x + key)
    return (x >> np.uint64(11)).astype(np.float64) * 2.0**-53 + 2.0**-54


def normal(seed: int, stream: int, n: int, start: int = 0) -> np.ndarray:
    u1 = uniform(seed, 2 * stream, n, start)
    u2 = uniform(seed, 2 * stream + 1, n, start)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


# --------------------------------------------------------------------------- configs
@dataclass
class Config:
    name: str
    R0: float
    a: float
    B0: float
    q: tuple  # (q0, q1, q2): q(r) = q0 + q1 r/a + q2 (r/a)^2
    nr: int
    ntheta: int
    n_planes: int
    n_markers: int
    nsteps: int
    dt: float = 0.05
    seed: int = 0
    structured: bool = False  # cfg 0: exactly BASELINE's 20x10 split quads, no jitter/flip/shuffle
    em: bool = True  # A_par nonzero
    loading: str = "uniform_r"  # "uniform_r" | "uniform_area" | "profile"
    sort_every: int = 0
    # Eq.(8) profile constants (values: DESIGN.md reading R14)
    kappa_n: float = 2.2
    kappa_T: float = 6.9
    w_n: float = 0.3
    w_T: float = 0.3
    rmin_frac: float = 0.05
    phi_period: float = 2.0 * np.pi
    extra: dict = field(default_factory=dict)

    @property
    def qom(self) -> float:  # rho_i(B0) = a/60 (rho* = 1/60, L320)  =>  q_s/m_s = 60/(a B0)
        return 60.0 / (self.a * self.B0)

    @property
    def r0(self) -> float:  # Eq.(8): r0 = a/2 (L316)
        return 0.5 * self.a


_Q1 = (0.86, -0.16, 2.52)
CONFIGS = {
    0: Config("cfg0-tiny", 1.0, 0.36, 1.0, (1.4, 0.0, 0.5), 20, 10, 8, 10_000, 10, seed=0, structured=True,
              loading="uniform_r"),
    1: Config("cfg1-itg-small", 1.67, 0.6, 2.0, _Q1, 28, 90, 16, 1_000_000, 100, seed=1, em=False,
              loading="uniform_area"),
    2: Config("cfg2-em", 1.67, 0.6, 2.0, _Q1, 55, 182, 32, 10_000_000, 50, seed=2, loading="profile", sort_every=10),
    3: Config("cfg3-production", 1.67, 0.6, 2.0, _Q1, 110, 364, 64, 100_000_000, 20, seed=3, loading="profile"),
    4: Config("cfg4-gather-stress", 1.67, 0.6, 2.0, _Q1, 213, 704, 64, 50_000_000, 0, seed=4, loading="profile"),
}


# --------------------------------------------------------------------------- mesh
def make_mesh(cfg: Config):
    """Annulus r in [rmin_frac*a, a], nr x ntheta quads each split in two CCW triangles.

    Unless cfg.structured: interior nodes jittered by <= 0.15 of the local spacing, diagonals
    flipped at random, node and triangle ids shuffled - nothing structured leaks to the library.
    Returns RZ [n_nodes,2] float64, tri [n_tri,3] int32.
    """
    nr, nt, a, R0 = cfg.nr, cfg.ntheta, cfg.a, cfg.R0
    rmin = cfg.rmin_frac * a
    dr, dth = (a - rmin) / nr, 2 * np.pi / nt
    ii, jj = np.meshgrid(np.arange(nr + 1), np.arange(nt), indexing="ij")
    r = rmin + ii * dr
    th = jj * dth
    if not cfg.structured:
        n = (nr + 1) * nt
        jr = (uniform(cfg.seed, 10, n).reshape(nr + 1, nt) - 0.5) * 2 * 0.15 * dr
        jt = (uniform(cfg.seed, 11, n).reshape(nr + 1, nt) - 0.5) * 2 * 0.15 * dth
        jr[0, :] = jr[-1, :] = 0.0  # keep the two boundary circles
        r = r + jr
        th = th + jt
    RZ = np.stack([R0 + r * np.cos(th), r * np.sin(th)], -1).reshape(-1, 2)

    def nid(i, j):
        return i * nt + (j % nt)

    qi, qj = np.meshgrid(np.arange(nr), np.arange(nt), indexing="ij")
    qi, qj = qi.ravel(), qj.ravel()
    A, B, Cc, D = nid(qi, qj), nid(qi + 1, qj), nid(qi + 1, qj + 1), nid(qi, qj + 1)
    if cfg.structured:
        flip = np.zeros(qi.shape[0], dtype=bool)
    else:
        flip = uniform(cfg.seed, 12, qi.shape[0]) < 0.5
    t1 = np.where(flip[:, None], np.stack([A, B, D], -1), np.stack([A, B, Cc], -1))
    t2 = np.where(flip[:, None], np.stack([B, Cc, D], -1), np.stack([A, Cc, D], -1))
    tri = np.stack([t1, t2], 1).reshape(-1, 3)
    if not cfg.structured:
        pn = np.argsort(uniform(cfg.seed, 13, RZ.shape[0]), kind="stable")  # new -> old
        inv = np.empty_like(pn)
        inv[pn] = np.arange(pn.shape[0])
        RZ = RZ[pn]
        tri = inv[tri]
        pt = np.argsort(uniform(cfg.seed, 14, tri.shape[0]), kind="stable")
        tri = tri[pt]
        rot = (uniform(cfg.seed, 15, tri.shape[0]) * 3).astype(np.int64)  # rotate vertex order
        tri = np.take_along_axis(tri, (np.arange(3)[None, :] + rot[:, None]) % 3, axis=1)
    V = RZ[tri]
    area2 = (V[:, 1, 0] - V[:, 0, 0]) * (V[:, 2, 1] - V[:, 0, 1]) - (V[:, 1, 1] - V[:, 0, 1]) * (V[:, 2, 0] - V[:, 0, 0])
    assert (area2 > 0).all(), "mesh generator produced a non-CCW triangle"
    return np.ascontiguousarray(RZ), np.ascontiguousarray(tri.astype(np.int32))


# --------------------------------------------------------------------------- closed-form fields
@dataclass
class Mode:
    amp: float
    m: int
    n: int
    phase: float = 0.0
    kind: str = "sin"  # "sin": sin(pi r/a) ; "gauss": exp(-((r-rs)/width)^2)
    rs: float = 0.0
    width: float = 1.0


def _envelope(md: Mode, r, a):
    if md.kind == "sin":
        k = np.pi / a
        return np.sin(k * r), k * np.cos(k * r), -k * k * np.sin(k * r)
    z = (r - md.rs) / md.width
    e = np.exp(-z * z)
    return e, -2 * z / md.width * e, (4 * z * z - 2) / md.width**2 * e


def mode_field(modes, R, Z, phi, R0, a):
    """Closed form f = sum amp*E(r)*cos(m theta - n phi + phase) and its R,Z derivatives to 2nd order.

    Returns array [..., 6] = f, f_R, f_Z, f_RR, f_RZ, f_ZZ (plain chain rule in polar coordinates)."""
    R, Z, phi = np.broadcast_arrays(np.asarray(R, float), np.asarray(Z, float), np.asarray(phi, float))
    x = R - R0
    r = np.hypot(x, Z)
    th = np.arctan2(Z, x)
    rR, rZ = x / r, Z / r
    tR, tZ = -Z / r**2, x / r**2
    rRR, rRZ, rZZ = Z * Z / r**3, -x * Z / r**3, x * x / r**3
    tRR, tRZ, tZZ = 2 * x * Z / r**4, (Z * Z - x * x) / r**4, -2 * x * Z / r**4
    out = np.zeros(R.shape + (6,))
    for md in modes:
        E, E1, E2 = _envelope(md, r, a)
        ang = md.m * th - md.n * phi + md.phase
        c, s = np.cos(ang), np.sin(ang)
        g_r, g_t = E1 * c, -md.m * E * s
        g_rr, g_rt, g_tt = E2 * c, -md.m * E1 * s, -md.m**2 * E * c
        out[..., 0] += md.amp * E * c
        out[..., 1] += md.amp * (g_r * rR + g_t * tR)
        out[..., 2] += md.amp * (g_r * rZ + g_t * tZ)
        out[..., 3] += md.amp * (g_rr * rR * rR + 2 * g_rt * rR * tR + g_tt * tR * tR + g_r * rRR + g_t * tRR)
        out[..., 4] += md.amp * (g_rr * rR * rZ + g_rt * (rR * tZ + rZ * tR) + g_tt * tR * tZ + g_r * rRZ + g_t * tRZ)
        out[..., 5] += md.amp * (g_rr * rZ * rZ + 2 * g_rt * rZ * tZ + g_tt * tZ * tZ + g_r * rZZ + g_t * tZZ)
    return out


def mode_dphi(modes, R, Z, phi, R0, a):
    """d f / d phi of the same closed form (for discretisation-error reports, never for parity)."""
    R, Z, phi = np.broadcast_arrays(np.asarray(R, float), np.asarray(Z, float), np.asarray(phi, float))
    x = R - R0
    r, th = np.hypot(x, Z), np.arctan2(Z, x)
    out = np.zeros(R.shape)
    for md in modes:
        E, _, _ = _envelope(md, r, a)
        out += md.amp * E * md.n * np.sin(md.m * th - md.n * phi + md.phase)
    return out


def field_dofs(modes, RZ, n_planes, R0, a, phi_period=2 * np.pi, deconvolve=True):
    """Nodal DOFs [n_planes, n_nodes, 6] of the closed form on every toroidal plane.

    The per-plane numbers are B-SPLINE COEFFICIENTS, not samples (reading R3): for a
    single toroidal harmonic n the periodic cubic spline through coefficients c_k takes the value
    c_k*(2+cos(n dphi))/3 at plane k, so each mode's samples are divided by that symbol."""
    dphi = phi_period / n_planes
    phik = np.arange(n_planes) * dphi
    out = np.zeros((n_planes, RZ.shape[0], 6))
    for md in modes:
        sym = (2.0 + np.cos(md.n * dphi)) / 3.0 if deconvolve else 1.0
        # cos(m theta + phase - n phi) = cos(m theta + phase) cos(n phi) + sin(m theta + phase) sin(n phi): the poloidal
        # factors (and their R, Z derivatives) are evaluated once per node, not once per node and plane
        C = mode_field([md], RZ[:, 0], RZ[:, 1], 0.0, R0, a) / sym
        S = mode_field([dataclasses.replace(md, phase=md.phase - 0.5 * np.pi)], RZ[:, 0], RZ[:, 1], 0.0, R0, a) / sym
        for k in range(n_planes):
            out[k] += np.cos(md.n * phik[k]) * C + np.sin(md.n * phik[k]) * S
    return out


def q_of_r(cfg: Config, r):
    x = np.asarray(r) / cfg.a
    return cfg.q[0] + cfg.q[1] * x + cfg.q[2] * x * x


def make_modes(cfg: Config, which: int):
    """cfg 0: one (m,n) = (3,2) mode, 1e-3 sin(pi r/a) for both fields.
    cfg 1-4: 6 modes, n ~ U{5..15}, m = round(n q(r_s)), r_s ~ U[0.3a, 0.7a], gaussian width 0.1a,
    amplitude 1e-3*U(0.5,1.5), phase ~ U[0,2pi); independent draws for Phi (which=0) and A_par (1)."""
    if cfg.structured:
        return [Mode(1e-3, 3, 2, 0.0, "sin")]
    s = 20 + 10 * which
    un = uniform(cfg.seed, s, 6)
    ur = uniform(cfg.seed, s + 1, 6)
    ua = uniform(cfg.seed, s + 2, 6)
    up = uniform(cfg.seed, s + 3, 6)
    modes = []
    for i in range(6):
        n = 5 + int(un[i] * 11)
        rs = (0.3 + 0.4 * ur[i]) * cfg.a
        m = int(round(n * float(q_of_r(cfg, rs))))
        modes.append(Mode(1e-3 * (0.5 + ua[i]), m, n, 2 * np.pi * up[i], "gauss", rs, 0.1 * cfg.a))
    return modes


def make_fields(cfg: Config, RZ):
    """-> (dof_phi, dof_apar) each [n_planes, n_nodes, 6]; dof_apar is all zero when cfg.em is False."""
    dphi = field_dofs(make_modes(cfg, 0), RZ, cfg.n_planes, cfg.R0, cfg.a, cfg.phi_period)
    if cfg.em:
        dap = field_dofs(make_modes(cfg, 1), RZ, cfg.n_planes, cfg.R0, cfg.a, cfg.phi_period)
    else:
        dap = np.zeros_like(dphi)
    return dphi, dap


# --------------------------------------------------------------------------- markers
def _profile(kappa, w, a, R0, r0, r):
    """Eq.(8), PAPER.md L314 -- used here ONLY to shape the loading density / temperature."""
    return np.exp(-kappa * w * (a / R0) * np.tanh((r - r0) / (w * a)))


def make_markers(cfg: Config, n: int | None = None, start: int = 0):
    """Markers [start, start+n) of the config's population (counter-based: any slice is reproducible).

    Returns dict of float64 arrays R, Z, phi, u, w, mu, p.
      r: cfg0 U[0.1a,0.9a]; "uniform_area": uniform in poloidal area on the same interval;
         "profile": density proportional to r*n(r) (inverse CDF on a fixed 4096-point table).
      u = sqrt(T) N(0,1);  mu = T*Exp(1)/B_ref(R) with B_ref = B0 R0/R (the vacuum toroidal field,
      a loading recipe, deliberately not the method's |B|);  w ~ U(-1e-3, 1e-3);  p = 1."""
    n = cfg.n_markers if n is None else n
    a, R0 = cfg.a, cfg.R0
    lo, hi = 0.1 * a, 0.9 * a
    ur = uniform(cfg.seed, 1, n, start)
    if cfg.loading == "uniform_r":
        r = lo + (hi - lo) * ur
    elif cfg.loading == "uniform_area":
        r = np.sqrt(lo * lo + (hi * hi - lo * lo) * ur)
    else:
        g = np.linspace(lo, hi, 4097)
        dens = g * _profile(cfg.kappa_n, cfg.w_n, a, R0, cfg.r0, g)
        cdf = np.concatenate([[0.0], np.cumsum(0.5 * (dens[1:] + dens[:-1]) * np.diff(g))])
        r = np.interp(ur, cdf / cdf[-1], g)
    th = 2 * np.pi * uniform(cfg.seed, 2, n, start)
    ph = cfg.phi_period * uniform(cfg.seed, 3, n, start)
    T = _profile(cfg.kappa_T, cfg.w_T, a, R0, cfg.r0, r) if cfg.loading == "profile" else np.ones(n)
    R = R0 + r * np.cos(th)
    Z = r * np.sin(th)
    u = np.sqrt(T) * normal(cfg.seed, 4, n, start)
    eperp = -np.log(uniform(cfg.seed, 7, n, start))
    mu = T * eperp * R / (cfg.B0 * R0)
    w = (uniform(cfg.seed, 8, n, start) - 0.5) * 2e-3
    return dict(R=R, Z=Z, phi=ph, u=u, w=w, mu=mu, p=np.ones(n))


def equilibrium_args(cfg: Config):
    return dict(R0=cfg.R0, a=cfg.a, B0=cfg.B0, q0=cfg.q[0], q1=cfg.q[1], q2=cfg.q[2], qbar_sqrt=1)


def species_args(cfg: Config):
    return dict(qom=cfg.qom, kappa_n=cfg.kappa_n, kappa_T=cfg.kappa_T, w_n=cfg.w_n, w_T=cfg.w_T, r0=cfg.r0,
                bstar_exact=1, weight_mode=0)
