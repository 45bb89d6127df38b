"""Pins for the oracle's C1 element, toroidal spline, locate and gather (no GPU).

Nothing here re-types the oracle's formulas: each test checks a property the paper / the
mathematics fix (SURVEY.md section 8(c) pins P1-P4, P12-P14, P16).
"""
import dataclasses

import mpmath as mp
import numpy as np
import pytest

from oracle import Oracle
from paper_2606_24327_b200 import synth


def _small_unstructured(seed=5, nr=4, nt=12, P=8):
    cfg = dataclasses.replace(synth.CONFIGS[1], nr=nr, ntheta=nt, n_planes=P, seed=seed, n_markers=2000, em=True)
    RZ, tri = synth.make_mesh(cfg)
    o = Oracle()
    o.equilibrium_set(**synth.equilibrium_args(cfg))
    o.species_set(**synth.species_args(cfg))
    o.mesh_load(RZ, tri, P, cfg.phi_period)
    return cfg, RZ, tri, o


def _rand_poly(rng, deg, x0, y0, scale):
    """Random bivariate polynomial of total degree deg in ((x-x0)/scale, (y-y0)/scale); returns f -> 6 derivs."""
    co = {(i, j): rng.normal() for i in range(deg + 1) for j in range(deg + 1 - i)}

    def f(x, y):
        X, Y = (x - x0) / scale, (y - y0) / scale
        out = []
        for dx, dy in [(0, 0), (1, 0), (0, 1), (2, 0), (1, 1), (0, 2)]:
            s = 0.0
            for (i, j), c in co.items():
                if i < dx or j < dy:
                    continue
                k = c
                for t in range(dx):
                    k *= i - t
                for t in range(dy):
                    k *= j - t
                s = s + k * X ** (i - dx) * Y ** (j - dy)
            out.append(s / scale ** (dx + dy))
        return np.array(out)

    return f


def _interior_points(rng, V, n):
    lam = rng.dirichlet([1, 1, 1], size=n)
    return lam @ V


# P1 ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("which_mesh", ["cfg0", "unstructured"])
def test_P1_reproduces_quartics_not_quintics(cfg0_oracle, which_mesh):
    """L35: the element space contains every polynomial of total degree <= 4 (Bell's reduced quintic);
    a generic quintic is NOT in it (negative control: its edge-normal derivative is quartic)."""
    if which_mesh == "cfg0":
        cfg, RZ, tri, o, _ = cfg0_oracle
    else:
        cfg, RZ, tri, o = _small_unstructured()
    rng = np.random.default_rng(1)
    worst = {4: 0.0, 5: 0.0}
    for deg in (4, 5):
        f = _rand_poly(rng, deg, cfg.R0, 0.0, cfg.a)
        for t in rng.choice(tri.shape[0], 12, replace=False):
            V = RZ[tri[t]]
            dof = np.concatenate([f(*V[v]) for v in range(3)])
            c = o.element_coeffs(t, dof)
            for P in _interior_points(rng, V, 6):
                got = o.poly_eval(t, c, *P)[:3]
                ex = f(*P)[:3]
                scale = np.array([1.0, 1.0 / cfg.a, 1.0 / cfg.a]) * 10.0  # polynomial is O(1..10) on the domain
                worst[deg] = max(worst[deg], np.max(np.abs(got - ex) / scale))
    assert worst[4] < 1e-13, worst
    assert worst[5] > 1e-9, worst  # must NOT be reproduced


# P2 ---------------------------------------------------------------------------------------
def test_P2_C1_across_shared_edges():
    """Random nodal DOFs: value and both gradient components continuous across every shared edge,
    second derivatives are not (negative control)."""
    cfg, RZ, tri, o = _small_unstructured(seed=7)
    rng = np.random.default_rng(2)
    nodal = rng.normal(size=(RZ.shape[0], 6))
    h = cfg.a / 6
    nodal[:, 1:3] /= h
    nodal[:, 3:] /= h * h
    edges = {}
    for t in range(tri.shape[0]):
        for e in range(3):
            a_, b_ = int(tri[t, e]), int(tri[t, (e + 1) % 3])
            edges.setdefault((min(a_, b_), max(a_, b_)), []).append(t)
    shared = [(k, v) for k, v in edges.items() if len(v) == 2]
    assert len(shared) > 50
    jump01, jump2 = 0.0, 0.0
    for (na, nb), (t1, t2) in shared[:80]:
        c1 = o.element_coeffs(t1, nodal[tri[t1]].ravel())
        c2 = o.element_coeffs(t2, nodal[tri[t2]].ravel())
        # fp64 evaluation error of a monomial sum is bounded by eps * sum|c_k m_k|: on thin triangles
        # random (non-smooth) DOFs give coefficients up to ~1e6 in the isotropic local frame
        cmag = max(np.abs(c1).max(), np.abs(c2).max())
        for s in np.linspace(0.0, 1.0, 7):
            P = RZ[na] + s * (RZ[nb] - RZ[na])
            v1, v2 = o.poly_eval(t1, c1, *P), o.poly_eval(t2, c2, *P)
            sc = np.array([1, 1 / h, 1 / h, 1 / h**2, 1 / h**2, 1 / h**2])
            d = np.abs(v1 - v2) / sc
            jump01 = max(jump01, d[:3].max() / (2e-13 + 1e-16 * cmag))
            jump2 = max(jump2, d[3:].max())
    assert jump01 < 1.0, jump01
    assert jump2 > 1e-3, jump2


# P3 ---------------------------------------------------------------------------------------
def test_P3_vertex_dofs_reproduced(cfg0_oracle):
    cfg, RZ, tri, o, _ = cfg0_oracle
    rng = np.random.default_rng(3)
    for t in rng.choice(tri.shape[0], 20, replace=False):
        V = RZ[tri[t]]
        L = max(np.linalg.norm(V[(e + 1) % 3] - V[e]) for e in range(3))
        sc = np.tile([1, 1 / L, 1 / L, 1 / L**2, 1 / L**2, 1 / L**2], 3)  # DOFs of a function varying on scale L
        dof = rng.normal(size=18) * sc
        c = o.element_coeffs(t, dof)
        for v in range(3):
            got = o.poly_eval(t, c, *V[v])
            err = np.abs(got - dof[6 * v:6 * v + 6]) / sc[:6]
            # random (rough) DOFs on aspect-13 triangles: coefficients reach ~1e4 x the value, stored as double
            assert err[:3].max() < 1e-10 and err[3:].max() < 2e-9, (t, v, err)


# P16 --------------------------------------------------------------------------------------
def _mp_reference_value(V, dof18, P):
    """Independent construction in 40-digit arithmetic, affine reference coordinates
    (xi, eta) with v0->(0,0), v1->(1,0), v2->(0,1): DOFs transformed by the Jacobian, constraint
    rows from the physical normal pulled back.  Returns (p, p_R, p_Z) at P."""
    mp.mp.dps = 40
    V = [[mp.mpf(float(x)) for x in v] for v in V]
    J = mp.matrix([[V[1][0] - V[0][0], V[2][0] - V[0][0]], [V[1][1] - V[0][1], V[2][1] - V[0][1]]])
    Ji = J ** -1
    MON = [(i, d - i) for d in range(6) for i in range(d, -1, -1)]

    def dm(i, j, dx, dy, x, y):
        if i < dx or j < dy:
            return mp.mpf(0)
        c = mp.mpf(1)
        for t in range(dx):
            c *= i - t
        for t in range(dy):
            c *= j - t
        return c * x ** (i - dx) * y ** (j - dy)

    L = [(mp.mpf(0), mp.mpf(0)), (mp.mpf(1), mp.mpf(0)), (mp.mpf(0), mp.mpf(1))]
    M = mp.zeros(21, 21)
    rhs = mp.zeros(21, 1)
    r = 0
    for v in range(3):
        f, fR, fZ, fRR, fRZ, fZZ = [mp.mpf(float(x)) for x in dof18[6 * v:6 * v + 6]]
        g = J.T * mp.matrix([fR, fZ])
        H = J.T * mp.matrix([[fRR, fRZ], [fRZ, fZZ]]) * J
        loc = [f, g[0], g[1], H[0, 0], H[0, 1], H[1, 1]]
        for q, (dx, dy) in enumerate([(0, 0), (1, 0), (0, 1), (2, 0), (1, 1), (0, 2)]):
            for k, (i, j) in enumerate(MON):
                M[r, k] = dm(i, j, dx, dy, *L[v])
            rhs[r] = loc[q]
            r += 1
    for e in range(3):
        a_, b_ = V[e], V[(e + 1) % 3]
        tp = mp.matrix([b_[0] - a_[0], b_[1] - a_[1]])
        n = mp.matrix([tp[1], -tp[0]])
        th = Ji * tp  # reference tangent
        nh = Ji * n   # d/dn = n . grad_phys = (Ji n) . grad_ref  (grad_phys = Ji^T grad_ref)
        for k, (i, j) in enumerate(MON):
            if i + j != 5:
                continue
            gx = i * th[0] ** (i - 1) * th[1] ** j if i > 0 else 0
            gy = j * th[0] ** i * th[1] ** (j - 1) if j > 0 else 0
            M[r, k] = nh[0] * gx + nh[1] * gy
        r += 1
    c = mp.lu_solve(M, rhs)
    xi = Ji * mp.matrix([mp.mpf(float(P[0])) - V[0][0], mp.mpf(float(P[1])) - V[0][1]])
    p = sum(c[k] * dm(i, j, 0, 0, xi[0], xi[1]) for k, (i, j) in enumerate(MON))
    gref = mp.matrix([sum(c[k] * dm(i, j, 1, 0, xi[0], xi[1]) for k, (i, j) in enumerate(MON)),
                      sum(c[k] * dm(i, j, 0, 1, xi[0], xi[1]) for k, (i, j) in enumerate(MON))])
    gph = Ji.T * gref
    return float(p), float(gph[0]), float(gph[1])


def test_P16_against_40_digit_independent_construction(cfg0_oracle):
    """The oracle's long-double LU in centroid/longest-edge coordinates agrees with an independent
    40-digit construction in affine reference coordinates to <= 2e-13 of the field scale, including
    on config 0's aspect-13 outer triangles.  This is what makes a 1e-12 parity gate meaningful."""
    cfg, RZ, tri, o, _ = cfg0_oracle
    rng = np.random.default_rng(4)
    kx, ky = 9.0, 7.0

    def d(x, y):
        s, c = np.sin(kx * x + ky * y), np.cos(kx * x + ky * y)
        return [s, kx * c, ky * c, -kx * kx * s, -kx * ky * s, -ky * ky * s]

    V_all = RZ[tri]
    e1 = np.linalg.norm(V_all[:, 1] - V_all[:, 0], axis=1)
    e2 = np.linalg.norm(V_all[:, 2] - V_all[:, 1], axis=1)
    e3 = np.linalg.norm(V_all[:, 0] - V_all[:, 2], axis=1)
    d1, d2 = V_all[:, 1] - V_all[:, 0], V_all[:, 2] - V_all[:, 0]
    area = 0.5 * np.abs(d1[:, 0] * d2[:, 1] - d1[:, 1] * d2[:, 0])
    aspect = np.maximum(np.maximum(e1, e2), e3) ** 2 / (2 * area)
    picks = list(np.argsort(aspect)[-3:]) + list(rng.choice(tri.shape[0], 3, replace=False))
    worst = np.zeros(3)
    for t in picks:
        V = RZ[tri[t]]
        dof = np.concatenate([d(*V[v]) for v in range(3)])
        c = o.element_coeffs(t, dof)
        for P in _interior_points(rng, V, 3):
            ref = np.array(_mp_reference_value(V, dof, P))
            got = o.poly_eval(t, c, *P)[:3]
            worst = np.maximum(worst, np.abs(got - ref) / np.array([1.0, kx, kx]))
    assert aspect.max() > 8
    assert worst.max() < 2e-13, worst


# P4 ---------------------------------------------------------------------------------------
def test_P4_bspline_partition_and_cubic_reproduction(cfg0_oracle):
    """Textbook facts of the uniform cubic B-spline (L35): partition of unity, derivative weights sum
    to zero, knot values (1,4,1,0)/6, and the quasi-interpolant c_k = p(phi_k) - dphi^2 p''(phi_k)/6
    reproduces any cubic away from the periodic wrap."""
    cfg, RZ, tri, o, _ = cfg0_oracle
    P = cfg.n_planes
    dphi = cfg.phi_period / P
    golden = np.loadtxt(__file__.replace("test_oracle_element.py", "golden/bspline_knot_values.txt"), comments="#")
    k, w, dw = o.bspline(3 * dphi)
    assert k == 3
    assert np.allclose(w, golden[0], atol=1e-15)
    assert np.allclose(dw * dphi, golden[1], atol=1e-15)
    rng = np.random.default_rng(5)
    a3, a2, a1, a0 = rng.normal(size=4)
    p = lambda x: ((a3 * x + a2) * x + a1) * x + a0
    p1 = lambda x: (3 * a3 * x + 2 * a2) * x + a1
    p2 = lambda x: 6 * a3 * x + 2 * a2
    phik = np.arange(P) * dphi
    ck = p(phik) - dphi**2 * p2(phik) / 6
    for phi in rng.uniform(1.0 * dphi, (P - 2.0) * dphi, 200):
        k, w, dw = o.bspline(phi)
        assert abs(w.sum() - 1) < 4e-16 and abs(dw.sum()) < 1e-15 / dphi * 4
        assert k == int(np.floor(phi / dphi))
        idx = [(k - 1 + j) % P for j in range(4)]
        assert abs(w @ ck[idx] - p(phi)) < 1e-13 * (1 + abs(p(phi)))
        assert abs(dw @ ck[idx] - p1(phi)) < 1e-12 * (1 + abs(p1(phi)))
    # periodic wrap: phi and phi + period give the same interval and weights; negative phi wraps
    k1, w1, _ = o.bspline(0.3)
    k2, w2, _ = o.bspline(0.3 + cfg.phi_period)
    k3, w3, _ = o.bspline(0.3 - cfg.phi_period)
    assert k1 == k2 == k3 and np.allclose(w1, w2, atol=1e-14) and np.allclose(w1, w3, atol=1e-14)


# P12 --------------------------------------------------------------------------------------
def test_P12_box_grid_equals_brute_force_in_field_values():
    """L89/L125-140 positioning scheme (bounding-box map on an intermediate grid) vs. testing every
    triangle: same field values (triangle ids may differ on shared edges, reading R16)."""
    cfg, RZ, tri, o = _small_unstructured(seed=11, nr=6, nt=20)
    dphi, dap = synth.make_fields(cfg, RZ)
    o.fields_set(0, dphi)
    o.fields_set(1, dap)
    m = synth.make_markers(cfg, 3000)
    # add points on vertices / edge midpoints / outside
    extra = np.concatenate([RZ[:40], 0.5 * (RZ[tri[:40, 0]] + RZ[tri[:40, 1]]), [[cfg.R0, 0.0], [cfg.R0 + 2 * cfg.a, 0.0]]])
    R = np.concatenate([m["R"], extra[:, 0]])
    Z = np.concatenate([m["Z"], extra[:, 1]])
    phi = np.concatenate([m["phi"], np.linspace(0, 6, extra.shape[0])])
    g1, t1 = o.gather(R, Z, phi, brute=False)
    g2, t2 = o.gather(R, Z, phi, brute=True)
    assert ((t1 < 0) == (t2 < 0)).all()
    assert (t1[-2:] == -1).all()  # the hole and far outside
    assert (t1[:3000] >= 0).all()
    sc = np.abs(g2).max(axis=1, keepdims=True)
    assert (np.abs(g1 - g2) / sc).max() < 1e-11
    lam_ok = o.locate(R[:3000], Z[:3000])
    V = RZ[tri[lam_ok]]
    # the located triangle really contains the point (independent check, numpy cross products)
    for a_, b_ in ((0, 1), (1, 2), (2, 0)):
        cr = (V[:, b_, 0] - V[:, a_, 0]) * (Z[:3000] - V[:, a_, 1]) - (V[:, b_, 1] - V[:, a_, 1]) * (R[:3000] - V[:, a_, 0])
        assert (cr >= -1e-14).all()


# P13, P14 ---------------------------------------------------------------------------------
def test_P13_P14_toroidal_symmetries_and_linearity():
    cfg, RZ, tri, o = _small_unstructured(seed=13, nr=5, nt=16, P=8)
    m = synth.make_markers(cfg, 1500)
    R, Z, phi = m["R"], m["Z"], m["phi"]
    # n = 0 field: every plane identical -> gather independent of phi, d/dphi = 0
    md0 = [synth.Mode(1e-3, 2, 0, 0.3, "gauss", 0.5 * cfg.a, 0.2 * cfg.a)]
    d0 = synth.field_dofs(md0, RZ, cfg.n_planes, cfg.R0, cfg.a)
    o.fields_set(0, d0)
    o.fields_set(1, 0 * d0)
    g_a, _ = o.gather(R, Z, phi)
    g_b, _ = o.gather(R, Z, phi + 1.2345)
    sc = np.abs(g_a[:3]).max(axis=1, keepdims=True)
    assert (np.abs(g_a[:3] - g_b[:3]) / sc).max() < 1e-13
    assert np.abs(g_a[3]).max() < 1e-13 * sc[0] / (cfg.phi_period / cfg.n_planes)
    # shift: coefficients rolled by one plane + markers moved by dphi -> identical output
    md = synth.make_modes(cfg, 0)
    d1 = synth.field_dofs(md, RZ, cfg.n_planes, cfg.R0, cfg.a)
    o.fields_set(0, d1)
    g1, _ = o.gather(R, Z, phi)
    o.fields_set(0, np.roll(d1, 1, axis=0))
    g2, _ = o.gather(R, Z, phi + cfg.phi_period / cfg.n_planes)
    sc = np.abs(g1[:4]).max(axis=1, keepdims=True)
    assert (np.abs(g1[:4] - g2[:4]) / sc).max() < 1e-11
    # linearity in the DOFs
    d2 = synth.field_dofs(synth.make_modes(cfg, 1), RZ, cfg.n_planes, cfg.R0, cfg.a)
    o.fields_set(0, d1)
    ga, _ = o.gather(R, Z, phi)
    o.fields_set(0, d2)
    gb, _ = o.gather(R, Z, phi)
    o.fields_set(0, 2.0 * d1 - 3.0 * d2)
    gc, _ = o.gather(R, Z, phi)
    sc = np.abs(gc[:4]).max(axis=1, keepdims=True)
    assert (np.abs(gc[:4] - (2 * ga[:4] - 3 * gb[:4])) / sc).max() < 1e-12


def test_gather_of_global_quartic_is_exact_everywhere():
    """P1 through the whole gather path (locate + spline + element): nodal DOFs of a global quartic on
    all planes (n = 0) -> gather returns the quartic and its gradient at every marker."""
    cfg, RZ, tri, o = _small_unstructured(seed=17, nr=5, nt=14, P=8)
    rng = np.random.default_rng(6)
    f = _rand_poly(rng, 4, cfg.R0, 0.0, cfg.a)
    nod = np.stack([f(*RZ[i]) for i in range(RZ.shape[0])])
    o.fields_set(0, np.broadcast_to(nod, (cfg.n_planes,) + nod.shape).copy())
    o.fields_set(1, np.zeros((cfg.n_planes,) + nod.shape))
    m = synth.make_markers(cfg, 800)
    g, t = o.gather(m["R"], m["Z"], m["phi"])
    ex = np.stack([f(r, z) for r, z in zip(m["R"], m["Z"])])
    assert (t >= 0).all()
    assert np.abs(g[0] - ex[:, 0]).max() < 1e-12 * np.abs(ex[:, 0]).max()
    assert np.abs(g[1] - ex[:, 1]).max() < 1e-12 * np.abs(ex[:, 1]).max()
    assert np.abs(g[2] - ex[:, 2]).max() < 1e-12 * np.abs(ex[:, 2]).max()
    assert np.abs(g[3]).max() < 1e-12 * np.abs(ex[:, 0]).max()
    assert np.abs(g[4:]).max() == 0.0
