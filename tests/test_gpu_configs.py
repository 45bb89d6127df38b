"""GPU parity on BASELINE configs 2 and 4 as stated, and on the code paths the config tests do not reach
(ragged patch, few planes, Morton numbering, equilibrium re-set, lost-marker rule of both push variants, C-ABI errors).

Same norm and tolerances as tests/test_gpu_parity.py (reading R18): 1e-12 per gathered quantity,
1e-10 per state quantity after 10 RK4 steps.  After 20 steps the bound is 4e-10: the two sides differ by rounding
only, and on these orbits a rounding-level difference grows at most quadratically in the step count over a few
steps (a difference in u shears phi linearly in time, which feeds back through the phi-dependent fields), so
(20 / 10)^2 = 4 times the 10-step bound.
"""
import ctypes as C
import dataclasses

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2606_24327_b200 import synth  # noqa: E402
from test_gpu_parity import GATHER_TOL, KEYS, STATE_TOL, _check_push, _dev, _make, _rel  # noqa: E402


def _compare_state(res, exp, idx, period, tol, what):
    st_gpu, st_ref = res["status"][idx] != 0, exp[5] != 0
    assert (st_gpu == st_ref).all(), f"{what}: lost-marker sets differ at {np.flatnonzero(st_gpu != st_ref)[:10]}"
    errs = {}
    for q, k in enumerate(("R", "Z", "phi", "u", "w")):
        errs[k] = _rel(res[k][idx], exp[q], period if k == "phi" else None)
    assert max(errs.values()) < tol, (what, errs)
    return errs


def test_cfg2_as_stated_profile_loading_sort_every_10():
    """BASELINE configs[2]: 20 020 triangles x 32 planes, EM fields, markers loaded with the Eq.(8) density and
    temperature profiles, re-sorted every 10 steps.  1e6 of its 1e7 markers, 20 steps: both stale decades and the
    re-sort between them are crossed; a strided 10 000-marker sample (including the last marker) against the oracle
    after 10 steps (1e-10) and after 20 steps (4e-10, see the module docstring), all statuses of the sample."""
    cfg = dataclasses.replace(synth.CONFIGS[2], n_markers=1_000_000)
    assert cfg.loading == "profile" and cfg.sort_every == 10 and cfg.n_planes == 32 and 2 * cfg.nr * cfg.ntheta == 20_020
    RZ, tri, o, g, m = _make(cfg)
    sample = np.unique(np.concatenate([np.arange(0, cfg.n_markers, 100), [cfg.n_markers - 1]]))
    d = _dev(m)
    g.set_push_variant(0)
    g.set_sort_interval(cfg.sort_every)
    g.markers_bind(*[d[k] for k in KEYS])
    g.push_rk4(cfg.dt, 10)
    st10 = g.push_stats()
    res10 = g.markers_get(host=True)
    g.push_rk4(cfg.dt, 10)
    st20 = g.push_stats()
    res20 = g.markers_get(host=True)
    ins = [m[k][sample] for k in KEYS]
    e10 = _compare_state(res10, o.push_rk4(*ins, cfg.dt, 10), sample, cfg.phi_period, STATE_TOL, "10 steps")
    e20 = _compare_state(res20, o.push_rk4(*ins, cfg.dt, 20), sample, cfg.phi_period, 4 * STATE_TOL, "20 steps")
    print("cfg2 parity", e10, e20, st10, st20)
    # first call: one order for k1 and one for each phase of step 1, then stale; second call: one re-sort (two orders)
    assert st10["sorts"] == 3 and st20["sorts"] == 2
    assert g.push_variant_used() == 0


def test_cfg4_mesh_gather_random_and_sorted_host_and_device():
    """BASELINE configs[4]'s mesh and fields (299 904 triangles x 64 planes: a 6.95 GB coefficient table, the only case
    whose table offsets exceed 2^32 bytes).  2e6 of its points; the oracle checks a strided 1e5-point sample (including
    the last point) in random order and in cell-sorted order, through DEVICE and HOST buffers."""
    import torch
    cfg = dataclasses.replace(synth.CONFIGS[4], n_markers=2_000_000)
    assert 2 * cfg.nr * cfg.ntheta == 299_904 and cfg.n_planes == 64
    RZ, tri, o, g, m = _make(cfg)
    n = cfg.n_markers
    sample = np.unique(np.concatenate([np.arange(0, n, 20), [n - 1]]))
    ref, tref = o.gather(m["R"][sample], m["Z"][sample], m["phi"][sample])
    # the sample touches the far end of the table
    assert tref.max() > 0.99 * tri.shape[0]

    def check(out, tout, idx, what):
        assert ((tout[idx] < 0) == (tref < 0)).all(), what
        for q in range(8):
            e = _rel(out[q][idx], ref[q])
            assert e < GATHER_TOL, (what, q, e)

    d = _dev({k: m[k] for k in ("R", "Z", "phi")})
    out, tout = g.gather(d["R"], d["Z"], d["phi"])
    out, tout = out.cpu().numpy(), tout.cpu().numpy()
    check(out, tout, sample, "device, random order")
    # cell-sorted order (caller's triangle ids x toroidal interval), HOST buffers
    k = np.minimum((np.mod(m["phi"], cfg.phi_period) / cfg.phi_period * cfg.n_planes).astype(np.int64), cfg.n_planes - 1)
    order = np.argsort(tout.astype(np.int64) * cfg.n_planes + k, kind="stable")
    inv = np.empty_like(order)
    inv[order] = np.arange(n)
    outs, touts = g.gather(np.ascontiguousarray(m["R"][order]), np.ascontiguousarray(m["Z"][order]), np.ascontiguousarray(m["phi"][order]))
    check(outs, touts, inv[sample], "host, cell-sorted order")
    assert np.array_equal(outs[:, inv], out) and np.array_equal(touts[inv], tout)   # the order of the points changes nothing
    del d
    torch.cuda.empty_cache()


@pytest.mark.parametrize("nr,ntheta,n_planes,expect_variant", [(7, 9, 6, 0), (7, 9, 10, 0), (9, 11, 7, 0), (6, 11, 5, 1), (6, 11, 4, 1)])
def test_push_ragged_patch_and_few_planes(nr, ntheta, n_planes, expect_variant):
    """Triangle counts that are not multiples of the patch size (the last patch is padded with unused slots), plane counts
    that are not multiples of the window (n_planes = 6, 7, 10) and plane counts below the tiled kernel's minimum (4, 5:
    the library then runs variant 1 and says so through trimeg_push_variant_used)."""
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, nr=nr, ntheta=ntheta, n_planes=n_planes, n_markers=6007)
    assert (2 * nr * ntheta) % 8 != 0
    RZ, tri, o, g, m = _make(cfg)
    _check_push(o, g, m, cfg, 0.05, 10, 0, sort_every=1)
    assert g.push_variant_used() == expect_variant
    _check_push(o, g, m, cfg, 0.05, 10, 0, sort_every=4)


def test_mesh_before_equilibrium_and_equilibrium_reset_after_species():
    """mesh_load before any equilibrium is known (Morton numbering of the triangles instead of flux-surface numbering), and
    an equilibrium that is replaced AFTER the species was set: the Eq.(8) scalars that depend on a and R0 must follow."""
    from oracle import Oracle
    from paper_2606_24327_b200.binding import Trimeg
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, nr=12, ntheta=40, n_planes=8, n_markers=9001)
    RZ, tri = synth.make_mesh(cfg)
    dphi, dap = synth.make_fields(cfg, RZ)
    m = synth.make_markers(cfg)
    o, g = Oracle(), Trimeg(0)
    g.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)          # no equilibrium yet
    wrong = dict(synth.equilibrium_args(cfg), R0=cfg.R0 * 1.3, a=cfg.a * 0.8)
    g.equilibrium_set(**wrong)
    g.species_set(**synth.species_args(cfg))
    g.equilibrium_set(**synth.equilibrium_args(cfg))             # replaces R0 and a after the species
    o.equilibrium_set(**synth.equilibrium_args(cfg))
    o.species_set(**synth.species_args(cfg))
    o.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)
    for x in (o, g):
        x.fields_set(0, dphi)
        x.fields_set(1, dap)
    _check_push(o, g, m, cfg, 0.05, 10, 0, sort_every=1)
    d = _dev(m)
    g.markers_bind(*[d[k] for k in KEYS])
    out = g.rhs(host=True)
    ref, _ = o.rhs(*[m[k] for k in KEYS])
    assert _rel(out[4], ref[4]) < 1e-11


def test_lost_marker_rule_identical_in_both_variants_near_the_boundary():
    """Markers loaded in a thin shell at the outer boundary (many leave, some end a step just outside without any stage of
    that step outside): both push variants and the oracle must report the same lost set after every step count."""
    cfg = dataclasses.replace(synth.CONFIGS[0], n_markers=4000)
    RZ, tri, o, g, m = _make(cfg)
    r = cfg.a * (0.985 + 0.0149 * synth.uniform(77, 1, cfg.n_markers))
    th = 2 * np.pi * synth.uniform(77, 2, cfg.n_markers)
    m["R"], m["Z"] = cfg.R0 + r * np.cos(th), r * np.sin(th)
    lost = []
    for nsteps in (1, 2, 3, 7):
        per_variant = []
        for variant in (0, 1):
            res, exp = _check_push(o, g, m, cfg, 0.05, nsteps, variant, sort_every=1)
            per_variant.append(res["status"] != 0)
        assert np.array_equal(per_variant[0], per_variant[1])
        lost.append(int(per_variant[0].sum()))
    assert lost[-1] > lost[0] > 0 and lost[-1] < cfg.n_markers


def test_abi_null_pointers_and_bad_memspace():
    """Errors the header promises (include/trimeg.h): null pointers and an unknown memspace return TRIMEG_ERR_BAD_ARG (-1)
    through the raw C-ABI, and leave the context usable."""
    import torch
    from paper_2606_24327_b200.binding import Trimeg, load_library
    lib = load_library()
    cfg = synth.CONFIGS[0]
    RZ, tri = synth.make_mesh(cfg)
    g = Trimeg(0)
    h = g._h
    assert lib.trimeg_create(None, 0, None) == -1
    assert lib.trimeg_equilibrium_set(h, None) == -1
    assert lib.trimeg_species_set(h, None) == -1
    assert lib.trimeg_mesh_load(h, RZ.shape[0], None, tri.shape[0], tri.ctypes.data, 8, 6.28) == -1
    assert lib.trimeg_mesh_load(h, RZ.shape[0], RZ.ctypes.data, tri.shape[0], None, 8, 6.28) == -1
    g.equilibrium_set(**synth.equilibrium_args(cfg))
    g.species_set(**synth.species_args(cfg))
    g.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)
    dof = np.zeros((cfg.n_planes, RZ.shape[0], 6))
    assert lib.trimeg_fields_set(h, 0, None, 0) == -1
    assert lib.trimeg_fields_set(h, 2, dof.ctypes.data, 0) == -1
    assert lib.trimeg_fields_set(h, 0, dof.ctypes.data, 7) == -1
    x = torch.zeros(16, dtype=torch.float64, device="cuda")
    out = torch.zeros((8, 16), dtype=torch.float64, device="cuda")
    p = x.data_ptr()
    assert lib.trimeg_gather(h, 16, None, p, p, out.data_ptr(), None, 1) == -1
    assert lib.trimeg_gather(h, 16, p, p, p, None, None, 1) == -1
    assert lib.trimeg_gather(h, 16, p, p, p, out.data_ptr(), None, 5) == -1
    assert lib.trimeg_gather(h, -1, p, p, p, out.data_ptr(), None, 1) == -1
    scratch = torch.empty(g.scratch_bytes(16), dtype=torch.uint8, device="cuda")
    args = [p] * 7
    assert lib.trimeg_markers_bind(h, 16, *args, 1, None, scratch.numel()) == -1
    assert lib.trimeg_markers_bind(h, 16, None, *args[1:], 1, scratch.data_ptr(), scratch.numel()) == -1
    assert lib.trimeg_markers_bind(h, 16, *args, 3, scratch.data_ptr(), scratch.numel()) == -1
    assert lib.trimeg_markers_bind(h, 16, *args, 1, scratch.data_ptr(), 10) == -5           # scratch too small: OOM code
    assert lib.trimeg_markers_get(h, None, None, None, None, None, None, 9) == -1
    assert lib.trimeg_rhs(h, None, 1) == -1
    assert lib.trimeg_push_stats(h, None) == -1
    assert lib.trimeg_push_variant_used(h, None) == -1
    assert b"" != lib.trimeg_last_error(h)
    # still usable
    mk = _dev(synth.make_markers(cfg, 64))
    g.markers_bind(*[mk[k] for k in KEYS])
    g.push_rk4(0.05, 1)
    g.sync()


def test_push_is_bitwise_reproducible():
    """The phase kernel hands chunks of markers to whichever compute warp is free, so the order of execution differs from
    run to run; the result must not (every marker's arithmetic is its own).  A race on a record, a chunk slot or a staged
    coefficient block would show up here as a run-to-run difference (profiles/r02_sanitizer.md: compute-sanitizer is
    closed on this pool, this test stands in for racecheck)."""
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, n_markers=300_007)
    RZ, tri, o, g, m = _make(cfg)
    d = _dev(m)
    runs = []
    for rep in range(3):
        g.set_push_variant(0)
        g.set_sort_interval(1 if rep < 2 else 3)
        g.markers_bind(*[d[k] for k in KEYS])
        g.push_rk4(0.05, 6)
        runs.append(g.markers_get(host=True))
    for k in ("R", "Z", "phi", "u", "w", "status"):
        assert np.array_equal(runs[0][k], runs[1][k]), k
    # a stale order changes which markers take the follow-up path (same formulas, other rounding): agreement to rounding only
    for k in ("R", "Z", "phi", "u", "w"):
        assert _rel(runs[2][k], runs[0][k], cfg.phi_period if k == "phi" else None) < 1e-12, k
    assert np.array_equal(runs[0]["status"], runs[2]["status"])


@pytest.mark.parametrize("mode", [1, 2])
def test_gather_direct_and_staged_paths(mode):
    """trimeg_gather's two device paths (one thread per point through L1/L2; library-side binning + TMA-staged coefficient
    blocks) against the oracle: config 0 with all markers, the unstructured EM mesh with a ragged count, points outside the
    mesh and in the hole mixed in, phi far outside [0, 2 pi), n = 1 and n = 2 through the staged path."""
    import torch
    cfg = synth.CONFIGS[0]
    RZ, tri, o, g, m = _make(cfg)
    g.set_gather_mode(mode)
    R, Z, phi = m["R"].copy(), m["Z"].copy(), m["phi"].copy()
    R[::97] = cfg.R0 + 2.0 * cfg.a          # outside
    R[5::101] = cfg.R0 + 0.01 * cfg.a       # in the hole
    Z[5::101] = 0.0
    phi[::7] += 5 * cfg.phi_period
    phi[3::11] -= 3 * cfg.phi_period
    ref, tref = o.gather(R, Z, phi)
    out, tout = g.gather(torch.from_numpy(R).cuda(), torch.from_numpy(Z).cuda(), torch.from_numpy(phi).cuda())
    out, tout = out.cpu().numpy(), tout.cpu().numpy()
    assert ((tout < 0) == (tref < 0)).all() and (tref < 0).sum() > 150
    assert np.abs(out[:, tref < 0]).max() == 0.0
    for q in range(8):
        assert _rel(out[q], ref[q]) < GATHER_TOL, (q, _rel(out[q], ref[q]))
    assert (tout == tref).mean() > 0.995
    for n in (1, 2, 33):
        o1, t1 = g.gather(R[:n].copy(), Z[:n].copy(), phi[:n].copy())     # HOST buffers
        for q in range(8):
            assert np.abs(o1[q] - ref[q][:n]).max() <= GATHER_TOL * np.abs(ref[q]).max()
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, n_markers=70_001)
    RZ, tri, o, g, m = _make(cfg)
    g.set_gather_mode(mode)
    ref, tref = o.gather(m["R"], m["Z"], m["phi"])
    d = _dev({k: m[k] for k in ("R", "Z", "phi")})
    out, tout = g.gather(d["R"], d["Z"], d["phi"])
    for q in range(8):
        assert _rel(out[q].cpu().numpy(), ref[q]) < GATHER_TOL
    if mode == 2:
        assert sum(g.gather_kernel_ms().values()) > 0
        g.set_gather_mode(1)
        out1, tout1 = g.gather(d["R"], d["Z"], d["phi"])
        assert torch.equal(tout, tout1) and float((out - out1).abs().max()) <= 1e-13 * float(out1.abs().max())


def test_other_g2p_kernels_match_oracle():
    """trimeg_pullback / trimeg_density_g2p / trimeg_f_interp (readings R22-R24) against the oracle, in
    caller order, on a fresh store and on a store that has been pushed (cell-sorted, stale triangle hints), with markers
    outside the mesh; gradient profiles on (config-2-like loading so that T(r) and n(r) matter)."""
    cfg = dataclasses.replace(synth.CONFIGS[2], nr=12, ntheta=40, n_planes=8, n_markers=20_003)
    RZ, tri, o, g, m = _make(cfg)
    m["R"][::211] = cfg.R0 + 1.2 * cfg.a      # outside
    d = _dev(m)

    def check(state, tag):
        R, Z, phi, u, w = [state[k] for k in ("R", "Z", "phi", "u", "w")]
        for which in (0, 1):
            got = g.density_g2p(which, host=True)
            ref = o.density_g2p(which, R, Z, phi)
            assert np.abs(got - ref).max() <= GATHER_TOL * np.abs(ref).max(), (tag, which)
        got = g.f_interp(host=True)
        ref = o.f_interp(R, Z, phi, u, m["mu"])
        assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max(), tag
        got_dev = g.f_interp().cpu().numpy()
        assert np.array_equal(got_dev, got)
        u1, w1, st1 = o.pullback(R, Z, phi, u, w, m["mu"], m["p"])
        g.pullback()
        res = g.markers_get(host=True)
        assert np.abs(res["u"] - u1).max() <= 1e-13 * np.abs(u1).max(), tag
        assert np.abs(res["w"] - w1).max() <= 1e-12 * np.abs(w1).max(), tag
        assert np.array_equal(res["R"], R) and np.array_equal(res["phi"], phi)
        assert ((res["status"] != 0) >= (st1 != 0)).all()
        return res

    g.markers_bind(*[d[k] for k in KEYS])
    check(m, "fresh store")
    # after a push: records are in cell order with hints of the next evaluation point
    g.markers_bind(*[d[k] for k in KEYS])
    g.set_sort_interval(1)
    g.push_rk4(cfg.dt, 3)
    state = g.markers_get(host=True)
    after = check(state, "pushed store")
    # the pullback invalidated the cached stage: pushing on must equal the oracle pushing the pulled-back state
    g.push_rk4(cfg.dt, 2)
    res = g.markers_get(host=True)
    exp = o.push_rk4(after["R"], after["Z"], after["phi"], after["u"], after["w"], m["mu"], m["p"], cfg.dt, 2, status=after["status"])
    for q, k in enumerate(("R", "Z", "phi", "u", "w")):
        assert _rel(res[k], exp[q], cfg.phi_period if k == "phi" else None) < STATE_TOL, k


def test_deposit_matches_oracle_and_is_the_transpose_of_the_gather():
    """trimeg_deposit (P2G onto the C1 x B-spline basis, reading R25) against the oracle's literal transpose of the gather on
    an unstructured mesh, fresh and pushed stores, both moments; tolerance 1e-11 of the largest entry of each DOF component
    (sums of ~100 contributions per entry in a different order on each side); and the adjoint identity against the
    library's OWN gather with a random DOF vector."""
    import torch
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, nr=8, ntheta=24, n_planes=8, n_markers=6011)
    RZ, tri, o, g, m = _make(cfg)
    m["R"][::301] = cfg.R0 + 1.3 * cfg.a
    d = _dev(m)
    g.markers_bind(*[d[k] for k in KEYS])

    def check(state, tag):
        for quantity, q in ((0, state["w"]), (1, state["w"] * state["u"])):
            ref = o.deposit(state["R"], state["Z"], state["phi"], q)
            got = g.deposit(quantity, host=True)
            for c in range(6):
                assert np.abs(got[:, :, c] - ref[:, :, c]).max() <= 1e-11 * np.abs(ref[:, :, c]).max(), (tag, quantity, c)
            got_dev = g.deposit(quantity).cpu().numpy()
            assert np.abs(got_dev - got).max() <= 1e-12 * np.abs(got).max()
        return got

    check(m, "fresh")
    g.set_sort_interval(1)
    g.push_rk4(cfg.dt, 2)
    state = g.markers_get(host=True)
    b = check(state, "pushed")           # last: quantity 1
    rng = np.random.default_rng(5)
    dof = rng.normal(size=b.shape) * np.array([1.0, 3.0, 3.0, 9.0, 9.0, 9.0])
    g.fields_set(0, dof)
    F, t = g.gather(state["R"], state["Z"], state["phi"])
    q = state["w"] * state["u"]
    assert abs(float((b * dof).sum()) - float((q * F[0]).sum())) < 1e-10 * np.abs(q * F[0]).sum()


@pytest.mark.parametrize("sort_every", [1, 3])
def test_read_only_calls_between_pushes_leave_the_push_unchanged(sort_every):
    """trimeg_rhs stages its results in the inactive record buffer, trimeg_deposit / density / f-interpolation / markers_get read
    the store: none of them may change what the next push computes.  5 steps, all of those calls, 5 more steps = the oracle's
    10 steps (1e-10), for the re-sorting push and for stale-order steps in between."""
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, nr=12, ntheta=36, n_planes=16, n_markers=30_011)
    RZ, tri, o, g, m = _make(cfg)
    d = _dev(m)
    g.set_push_variant(0)
    g.set_sort_interval(sort_every)
    g.markers_bind(*[d[k] for k in KEYS])
    g.push_rk4(cfg.dt, 5)
    rhs_a = g.rhs(host=True)
    g.density_g2p(1); g.f_interp(); g.deposit(0); g.deposit(1)
    mid = g.markers_get()                                   # DEVICE arrays
    rhs_b = g.rhs(host=True)
    assert np.array_equal(rhs_a, rhs_b)
    ref, _ = o.rhs(*[mid[k].cpu().numpy() if k in mid else m[k] for k in KEYS])
    for q in range(5):
        assert _rel(rhs_b[q], ref[q]) < 1e-11, (q, _rel(rhs_b[q], ref[q]))
    g.push_rk4(cfg.dt, 5)
    res = g.markers_get(host=True)
    exp = o.push_rk4(*[m[k] for k in KEYS], cfg.dt, 10)
    _compare_state(res, exp, np.arange(cfg.n_markers), cfg.phi_period, STATE_TOL, f"push / calls / push, sort_every={sort_every}")
    assert g.push_variant_used() == 0


@pytest.mark.parametrize("npts", [1, 4, 8])
def test_gather_gyro_matches_oracle(npts):
    """trimeg_gather_gyro (N-point gyro-average of the gather, reading R26) against the oracle on the unstructured EM mesh:
    ring radii from zero to several elements, rings that leave the mesh through the outer boundary and through the hole,
    HOST and DEVICE buffers.  Tolerance 1e-12 per quantity (the cos / sin of the ring angles differ in the last bit)."""
    import torch
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, n_markers=20_011)
    RZ, tri, o, g, m = _make(cfg)
    R, Z, phi = m["R"], m["Z"], m["phi"]
    rho = 0.08 * cfg.a * synth.uniform(31, 1, R.shape[0])
    rho[::5] = 0.0
    ref, tref = o.gather_gyro(R, Z, phi, rho, npts)
    out, tout = g.gather_gyro(R, Z, phi, rho, npts)
    for q in range(8):
        assert _rel(out[q], ref[q]) < GATHER_TOL, (q, _rel(out[q], ref[q]))
    assert (tout == tref).mean() > 0.999
    d = _dev({"R": R, "Z": Z, "phi": phi, "rho": rho})
    out2, tout2 = g.gather_gyro(d["R"], d["Z"], d["phi"], d["rho"], npts)
    assert np.array_equal(out2.cpu().numpy(), out) and np.array_equal(tout2.cpu().numpy(), tout)
    if npts == 1:
        plain, _ = g.gather(R + rho, Z, phi)
        assert np.abs(out - plain).max() <= 1e-13 * np.abs(plain).max()


def test_numeric_equilibrium_rhs_and_push_match_oracle():
    """Numeric (B-spline) equilibrium, reading R27: a shaped flux function given as tensor-product cubic B-spline coefficients
    (elongated, with a cubic shift term), the same coefficients to the oracle and the library; trimeg_rhs (1e-11) and 10 RK4
    steps (1e-10) against the oracle; the library runs variant 1 with it and says so; switching back to the analytic
    equilibrium restores the tiled path."""
    from oracle import Oracle
    from paper_2606_24327_b200.binding import Trimeg
    from test_oracle_physics import _cubic_exact_coefs
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, nr=10, ntheta=30, n_planes=8, n_markers=7001)
    RZ, tri = synth.make_mesh(cfg)
    dphi, dap = synth.make_fields(cfg, RZ)
    m = synth.make_markers(cfg)
    R0, a, F = cfg.R0, cfg.a, cfg.B0 * cfg.R0
    k = cfg.B0 / (2 * 1.6)                                     # psi ~ B0 r^2 / (2 q) near the axis, q ~ 1.6
    psi = lambda R, Z: k * ((R - R0) ** 2 + Z**2 / 1.4**2) + 0.15 * k / a * (R - R0) ** 3 - 0.1 * k / a * (R - R0) * Z**2
    box = (R0 - 1.3 * a, R0 + 1.3 * a, -1.3 * a, 1.3 * a)
    nR, nZ = 37, 41
    coef = _cubic_exact_coefs(psi, nR, nZ, *box)
    o, g = Oracle(), Trimeg(0)
    for x in (o, g):
        x.equilibrium_set_numeric(nR, nZ, *box, F, R0, a, coef)
        x.species_set(**synth.species_args(cfg))
        x.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)
        x.fields_set(0, dphi)
        x.fields_set(1, dap)
    d = _dev(m)
    g.markers_bind(*[d[k_] for k_ in KEYS])
    out = g.rhs(host=True)
    ref, _ = o.rhs(*[m[k_] for k_ in KEYS])
    for q in range(5):
        assert _rel(out[q], ref[q]) < 1e-11, (q, _rel(out[q], ref[q]))
    _check_push(o, g, m, cfg, 0.05, 10, 0, sort_every=1)
    assert g.push_variant_used() == 1
    fi = g.f_interp(host=True)
    res = g.markers_get(host=True)
    assert np.abs(fi - o.f_interp(res["R"], res["Z"], res["phi"], res["u"], m["mu"])).max() <= 1e-12 * np.abs(fi).max()
    for x in (o, g):
        x.equilibrium_set(**synth.equilibrium_args(cfg))
    _check_push(o, g, m, cfg, 0.05, 10, 0, sort_every=1)
    assert g.push_variant_used() == 0


def test_fields_export_import_round_trip():
    """trimeg_fields_export / trimeg_fields_import (the payload of the one multi-GPU collective): a second context
    that never ran fields_set gathers bit-identical values after importing the first one's table; wrong sizes are refused."""
    import torch
    from paper_2606_24327_b200.binding import Trimeg, TrimegError
    cfg = dataclasses.replace(synth.CONFIGS[1], em=True, nr=8, ntheta=24, n_planes=8, n_markers=3001)
    RZ, tri, o, g, m = _make(cfg)
    d = _dev({k: m[k] for k in ("R", "Z", "phi")})
    ref, _ = g.gather(d["R"], d["Z"], d["phi"])
    buf = g.fields_export()
    assert buf.numel() == g.fields_bytes() > 0
    g2 = Trimeg(0)
    g2.equilibrium_set(**synth.equilibrium_args(cfg))
    g2.species_set(**synth.species_args(cfg))
    g2.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)
    zero, _ = g2.gather(d["R"], d["Z"], d["phi"])
    assert float(zero.abs().max()) == 0.0
    g2.fields_import(buf)
    out, _ = g2.gather(d["R"], d["Z"], d["phi"])
    assert torch.equal(out, ref)
    with pytest.raises(TrimegError, match="rc=-1"):
        g2.fields_import(buf[:-8])
