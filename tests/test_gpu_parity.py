"""Parity of the CUDA path (through the C-ABI) against the CPU oracle on the same seeded inputs.

Tolerances are north_star's: 1e-12 relative for one gathered field evaluation, 1e-10 for marker state after
10 RK4 steps; norm = max|gpu - oracle| / max|oracle| per output quantity over all compared markers
(reading R18).  Triangle ids are compared only where unique (a point on a shared edge may be
assigned to either neighbour, R16); phi is compared modulo the period.
"""
import dataclasses

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2606_24327_b200 import synth  # noqa: E402

GATHER_TOL = 1e-12
STATE_TOL = 1e-10
KEYS = ("R", "Z", "phi", "u", "w", "mu", "p")


def _make(cfg, n_markers=None, fields=True):
    import torch
    from oracle import Oracle
    from paper_2606_24327_b200.binding import Trimeg

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    RZ, tri = synth.make_mesh(cfg)
    o, g = Oracle(), Trimeg(0)
    for x in (o, g):
        x.equilibrium_set(**synth.equilibrium_args(cfg))
        x.species_set(**synth.species_args(cfg))
        x.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)
    if fields:
        dphi, dap = synth.make_fields(cfg, RZ)
        for x in (o, g):
            x.fields_set(0, dphi)
            x.fields_set(1, dap)
    m = synth.make_markers(cfg, n_markers)
    return RZ, tri, o, g, m


def _dev(m):
    import torch
    return {k: torch.from_numpy(np.ascontiguousarray(v)).cuda() for k, v in m.items()}


def _rel(got, ref, period=None):
    d = np.abs(got - ref)
    if period is not None:
        d = np.minimum(d, np.abs(d - period))
    return d.max() / max(np.abs(ref).max(), 1e-300)


def _check_gather(o, g, R, Z, phi, tol=GATHER_TOL):
    import torch
    ref, tref = o.gather(R, Z, phi)
    out, tout = g.gather(torch.from_numpy(R).cuda(), torch.from_numpy(Z).cuda(), torch.from_numpy(phi).cuda())
    out, tout = out.cpu().numpy(), tout.cpu().numpy()
    assert ((tout < 0) == (tref < 0)).all()
    for q in range(8):
        if np.abs(ref[q]).max() == 0:
            assert np.abs(out[q]).max() == 0
        else:
            assert _rel(out[q], ref[q]) < tol, (q, _rel(out[q], ref[q]))
    return out, tout, ref, tref


def _check_push(o, g, m, cfg, dt, nsteps, variant, sort_every=0, tol=STATE_TOL, sample=None):
    d = _dev(m)
    g.set_push_variant(variant)
    g.set_sort_interval(sort_every)
    g.markers_bind(*[d[k] for k in KEYS])
    g.push_rk4(dt, nsteps)
    res = g.markers_get(host=True)
    idx = np.arange(m["R"].shape[0]) if sample is None else sample
    exp = o.push_rk4(*[m[k][idx] for k in KEYS], dt, nsteps)
    st_gpu, st_ref = res["status"][idx] != 0, exp[5] != 0
    assert (st_gpu == st_ref).all(), f"lost-marker sets differ: {np.flatnonzero(st_gpu != st_ref)[:10]}"
    for q, k in enumerate(("R", "Z", "phi", "u", "w")):
        e = _rel(res[k][idx], exp[q], cfg.phi_period if k == "phi" else None)
        assert e < tol, (k, e, variant)
    return res, exp


# ------------------------------------------------------------------------------------------- gather
def test_gather_cfg0_all_markers():
    """BASELINE configs[0]: 400 triangles (aspect up to 13), 8 planes, 1e4 markers, both fields."""
    cfg = synth.CONFIGS[0]
    RZ, tri, o, g, m = _make(cfg)
    out, tout, ref, tref = _check_gather(o, g, m["R"], m["Z"], m["phi"])
    same = tout == tref
    assert same.mean() > 0.999  # ids agree except possibly on shared edges


def test_gather_edge_cases():
    """Vertices, edge midpoints, the hole, far outside, phi outside [0, 2pi), phi exactly on planes, n = 0, n = 1."""
    import torch
    cfg = synth.CONFIGS[0]
    RZ, tri, o, g, m = _make(cfg, 10)
    P, per = cfg.n_planes, cfg.phi_period
    inner = np.hypot(RZ[:, 0] - cfg.R0, RZ[:, 1]) > 0.06 * cfg.a
    verts = RZ[inner][:60]
    mids = 0.5 * (RZ[tri[:60, 0]] + RZ[tri[:60, 1]])
    pts = np.concatenate([verts, mids, [[cfg.R0, 0.0], [cfg.R0 + 3 * cfg.a, 0.1], [cfg.R0 - 0.5 * cfg.a, 0.5 * cfg.a]]])
    R, Z = np.ascontiguousarray(pts[:, 0]), np.ascontiguousarray(pts[:, 1])
    phi = np.concatenate([np.arange(40) * per / P, np.linspace(-3 * per, 4 * per, R.shape[0] - 40)])
    # interior vertices / edges: the oracle and the GPU may pick different (adjacent) triangles; values agree by C1
    ref, tref = o.gather(R, Z, phi)
    out, tout = g.gather(torch.from_numpy(R).cuda(), torch.from_numpy(Z).cuda(), torch.from_numpy(phi).cuda())
    out, tout = out.cpu().numpy(), tout.cpu().numpy()
    assert tout[-3] == -1 and tout[-2] == -1 and tref[-3] == -1 and tref[-2] == -1
    assert np.abs(out[:, -3:-1]).max() == 0.0
    ok = (tref >= 0) & (tout >= 0)
    assert ok.sum() >= R.shape[0] - 2 - 5  # boundary vertices may fall on either side of the tolerance
    for q in range(8):
        assert _rel(out[q][ok], ref[q][ok]) < 2e-12, (q, _rel(out[q][ok], ref[q][ok]))
    # the reported triangle really contains the point
    V = RZ[tri[tout[ok]]]
    for a_, b_ in ((0, 1), (1, 2), (2, 0)):
        cr = (V[:, b_, 0] - V[:, a_, 0]) * (Z[ok] - V[:, a_, 1]) - (V[:, b_, 1] - V[:, a_, 1]) * (R[ok] - V[:, a_, 0])
        assert (cr >= -1e-12).all()
    # n = 0 and n = 1, HOST memspace
    e = np.empty(0)
    o0, t0 = g.gather(e, e, e)
    assert o0.shape == (8, 0)
    o1, t1 = g.gather(R[:1].copy(), Z[:1].copy(), phi[:1].copy())
    assert _rel(o1[:, 0], ref[:, 0]) < 2e-12


def test_gather_unstructured_em_mesh_ragged_sizes():
    """Jittered/flipped/shuffled 28x90 mesh with 16 planes (config-1 geometry), EM fields; marker counts that are not
    multiples of the block size, spanning many blocks."""
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, n_markers=70_001)
    RZ, tri, o, g, m = _make(cfg)
    _check_gather(o, g, m["R"], m["Z"], m["phi"])
    _check_gather(o, g, m["R"][:257].copy(), m["Z"][:257].copy(), m["phi"][:257].copy())


def test_gather_without_fields_is_zero_and_linear_in_dofs():
    import torch
    cfg = dataclasses.replace(synth.CONFIGS[0], n_markers=500)
    RZ, tri, o, g, m = _make(cfg, fields=False)
    d = _dev(m)
    out, _ = g.gather(d["R"], d["Z"], d["phi"])
    assert float(out.abs().max()) == 0.0
    dphi, dap = synth.make_fields(cfg, RZ)
    g.fields_set(0, dphi)
    a, _ = g.gather(d["R"], d["Z"], d["phi"])
    g.fields_set(0, torch.from_numpy(-2.5 * dphi).cuda())  # DEVICE memspace for the DOFs
    b, _ = g.gather(d["R"], d["Z"], d["phi"])
    assert float((b[:4] + 2.5 * a[:4]).abs().max()) < 1e-12 * float(a[:4].abs().max())
    assert float(b[4:].abs().max()) == 0.0


# ------------------------------------------------------------------------------------------- push
@pytest.mark.parametrize("variant", [0, 1])
def test_push_cfg0_10_steps(variant):
    """BASELINE configs[0] exactly: 1e4 markers, 10 RK4 steps, dt = 0.05; a handful of markers cross the outer
    boundary (status bit) - the lost sets must be identical."""
    cfg = synth.CONFIGS[0]
    RZ, tri, o, g, m = _make(cfg)
    res, exp = _check_push(o, g, m, cfg, cfg.dt, cfg.nsteps, variant)
    assert (exp[5] != 0).sum() > 0  # the case does exercise the lost-marker rule
    # energy (static fields) is conserved by the GPU result as well as by the oracle's (invariant, any size)
    g2, _ = o.gather(res["R"], res["Z"], res["phi"])
    g0, _ = o.gather(m["R"], m["Z"], m["phi"])
    B1 = np.array([o.equil(a, b)["B"] for a, b in zip(res["R"][:500], res["Z"][:500])])
    B0 = np.array([o.equil(a, b)["B"] for a, b in zip(m["R"][:500], m["Z"][:500])])
    E1 = 0.5 * res["u"][:500] ** 2 + m["mu"][:500] * B1 + cfg.qom * (g2[0][:500] - res["u"][:500] * g2[4][:500])
    E0 = 0.5 * m["u"][:500] ** 2 + m["mu"][:500] * B0 + cfg.qom * (g0[0][:500] - m["u"][:500] * g0[4][:500])
    ok = res["status"][:500] == 0
    assert np.median(np.abs(E1 - E0)[ok] / np.abs(E0[ok])) < 1e-5


@pytest.mark.parametrize("variant", [0, 1])
def test_push_unstructured_em_with_resort(variant):
    """Config-1 geometry (unstructured 5040 triangles, 16 planes) with EM fields, 30 011 markers (ragged), 10 steps,
    re-sorted every 3 steps: the sort must not change any marker's trajectory or the caller's ordering."""
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, n_markers=30_011)
    RZ, tri, o, g, m = _make(cfg)
    _check_push(o, g, m, cfg, 0.05, 10, variant, sort_every=3)


@pytest.mark.parametrize("sort_every", [1, 2])
def test_push_sort_fused_into_push(sort_every):
    """Tiled variant with a re-sort every step / every other step: the sort only builds the permutation and the push
    kernel reads the markers through it (and writes the next sort's keys); trajectories, the caller's ordering and
    the lost set must not change.  Also checks markers_get / rhs between pushes (they read the current buffer)."""
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, n_markers=40_013)
    RZ, tri, o, g, m = _make(cfg)
    _check_push(o, g, m, cfg, 0.05, 10, 0, sort_every=sort_every)
    # continue in two further calls (keys carried across calls), then compare against 10 + 3 + 2 oracle steps
    g.push_rk4(0.05, 3)
    mid = g.markers_get(host=True)
    g.push_rk4(0.05, 2)
    res = g.markers_get(host=True)
    exp = o.push_rk4(*[m[k] for k in KEYS], 0.05, 15)
    assert ((res["status"] != 0) == (exp[5] != 0)).all()
    for q, k in enumerate(("R", "Z", "phi", "u", "w")):
        assert _rel(res[k], exp[q], cfg.phi_period if k == "phi" else None) < 2e-10, k
    assert not np.array_equal(mid["R"], res["R"])


@pytest.mark.parametrize("variant", [0, 1])
def test_push_degenerate_cases(variant):
    """n = 1; nsteps = 0 (state unchanged); negative charge; nonlinear weight mode; literal-L53 b*; zero fields."""
    cfg = dataclasses.replace(synth.CONFIGS[0], n_markers=777)
    RZ, tri, o, g, m = _make(cfg)
    one = {k: v[:1].copy() for k, v in m.items()}
    _check_push(o, g, one, cfg, 0.05, 4, variant)
    d = _dev(m)
    g.markers_bind(*[d[k] for k in KEYS])
    g.push_rk4(0.05, 0)
    r0 = g.markers_get(host=True)
    for k in ("R", "Z", "phi", "u", "w"):
        assert np.array_equal(r0[k], m[k])
    sp = synth.species_args(cfg)
    for mod in (dict(qom=-sp["qom"] * 3), dict(weight_mode=1), dict(bstar_exact=0), dict(w_n=0.2, w_T=0.35)):
        s2 = dict(sp, **mod)
        o.species_set(**s2)
        g.species_set(**s2)
        _check_push(o, g, m, cfg, 0.05, 10, variant)
    o.species_set(**sp)
    g.species_set(**sp)
    zero = np.zeros((cfg.n_planes, RZ.shape[0], 6))
    for x in (o, g):
        x.fields_set(0, zero)
        x.fields_set(1, zero)
    _check_push(o, g, m, cfg, 0.05, 10, variant)


def test_rhs_matches_oracle_in_caller_order():
    """trimeg_rhs = the paper's own kernel boundary (L89: five time derivatives per marker)."""
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, nr=10, ntheta=30, n_planes=8, n_markers=5003)
    RZ, tri, o, g, m = _make(cfg)
    d = _dev(m)
    g.markers_bind(*[d[k] for k in KEYS])
    g.sort()
    out = g.rhs(host=True)
    ref, outside = o.rhs(*[m[k] for k in KEYS])
    for q in range(5):
        assert _rel(out[q], ref[q]) < 1e-11, (q, _rel(out[q], ref[q]))


def test_cfg1_full_size_sampled():
    """BASELINE configs[1] at full size (1e6 markers, 5040 triangles, 16 planes) in the launch configuration bench.py
    uses; the oracle checks all markers' gather and a strided 20 000-marker sample of the state after 10 steps."""
    cfg = synth.CONFIGS[1]
    RZ, tri, o, g, m = _make(cfg)
    _check_gather(o, g, m["R"], m["Z"], m["phi"])
    sample = np.arange(0, cfg.n_markers, 50)
    _check_push(o, g, m, cfg, cfg.dt, 10, 0, sample=sample)


def test_cfg3_mesh_two_phase_sorted_every_step():
    """BASELINE configs[3]'s mesh and fields (80 080 triangles, 64 planes, EM) in the configuration bench.py times
    (variant 0, both phases re-sorted every step), with 2e6 of its markers: the oracle checks a strided 4 000-marker
    sample of the state after 5 steps, and every marker's status."""
    cfg = dataclasses.replace(synth.CONFIGS[3], n_markers=2_000_000)
    RZ, tri, o, g, m = _make(cfg)
    sample = np.arange(0, cfg.n_markers, 500)
    res, exp = _check_push(o, g, m, cfg, cfg.dt, 5, 0, sort_every=1, sample=sample)
    st = g.push_stats()
    assert st["sorts"] == 11 and st["retired"] < 0.02 * 11 * cfg.n_markers  # one permutation for the initial k1, two per step; the follow-up path stays rare


# ------------------------------------------------------------------------------------------- errors
def test_error_behaviour():
    import torch
    from paper_2606_24327_b200.binding import Trimeg, TrimegError
    cfg = synth.CONFIGS[0]
    RZ, tri = synth.make_mesh(cfg)
    g = Trimeg(0)
    x = torch.zeros(4, dtype=torch.float64, device="cuda")
    with pytest.raises(TrimegError, match="rc=-2"):
        g.gather(x, x, x)  # no mesh
    with pytest.raises(TrimegError, match="rc=-2"):
        g.species_set(**synth.species_args(cfg))  # needs the equilibrium first
    g.equilibrium_set(**synth.equilibrium_args(cfg))
    g.species_set(**synth.species_args(cfg))
    with pytest.raises(TrimegError, match="rc=-1"):
        g.mesh_load(RZ, tri, 3)  # n_planes < 4
    bad = tri.copy()
    bad[5] = bad[5][::-1]  # clockwise
    with pytest.raises(TrimegError, match="rc=-3"):
        g.mesh_load(RZ, bad, 8)
    bad = tri.copy()
    bad[7, 1] = RZ.shape[0] + 3
    with pytest.raises(TrimegError, match="rc=-3"):
        g.mesh_load(RZ, bad, 8)
    with pytest.raises(TrimegError, match="rc=-2"):
        g.fields_set(0, np.zeros((8, RZ.shape[0], 6)))  # failed loads leave no mesh
    g.mesh_load(RZ, tri, 8)
    with pytest.raises(TrimegError, match="rc=-2"):
        g.push_rk4(0.05, 1)  # no markers
    m = _dev(synth.make_markers(cfg, 64))
    g.markers_bind(*[m[k] for k in KEYS])
    for dt in (0.0, -1.0, float("nan"), float("inf")):
        with pytest.raises(TrimegError, match="rc=-1"):
            g.push_rk4(dt, 1)
    with pytest.raises(TrimegError, match="rc=-1"):
        g.push_rk4(0.05, -1)
    g.push_rk4(0.05, 1)
    g.sync()
