"""Pins for the oracle's equilibrium, equations of motion, weight equation and RK4 (no GPU).

SURVEY.md section 8(c) pins P5-P11, P15.  Each is a property fixed by the paper's equations
(Eq.(2)-(8), L45-65, L314) or by vector calculus; none re-types the oracle's formulas.
"""
import dataclasses

import numpy as np
import pytest
from scipy.integrate import quad

from oracle import Oracle
from paper_2606_24327_b200 import synth


def _eq(o, R, Z):
    return o.equil(R, Z)


@pytest.fixture(scope="module", params=["cfg0", "cfg1-equilibrium"])
def eq_case(request, cfg0_oracle):
    """(cfg, oracle): config 0 (R0 = B0 = 1) and config 1's equilibrium (R0 = 1.67, B0 = 2, q1 != 0), so that a
    dropped factor of R0, B0 or a cannot hide behind a unit value."""
    if request.param == "cfg0":
        cfg, RZ, tri, o, _ = cfg0_oracle
        return cfg, o
    cfg = dataclasses.replace(synth.CONFIGS[1], nr=4, ntheta=12, n_planes=8, em=True)
    RZ, tri = synth.make_mesh(cfg)
    o = Oracle()
    o.equilibrium_set(**synth.equilibrium_args(cfg))
    o.species_set(**synth.species_args(cfg))
    o.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)
    return cfg, o


# P5 ---------------------------------------------------------------------------------------
def test_P5_field_line_pitch_averages_to_q(eq_case):
    """(1/2pi) oint (B_phi/R)/(B_theta/r) dtheta = q(r): the sqrt(1-eps^2) in qbar (reading R10) is exactly
    what makes the prescribed q(r) the field-line safety factor.  Golden values: q(r) from BASELINE
    config 0, q = 1.4 + 0.5 (r/a)^2."""
    cfg, o = eq_case
    q0, q1, q2 = cfg.q  # BASELINE.json configs[0] / configs[1]
    gold = [(x, q0 + q1 * x + q2 * x * x) for x in (0.25, 0.5, 0.75, 0.9)]
    for r_over_a, q_expected in gold:
        r = r_over_a * cfg.a

        def pitch(th):
            R, Z = cfg.R0 + r * np.cos(th), r * np.sin(th)
            e = _eq(o, R, Z)
            bth = -np.sin(th) * e["B_R"] + np.cos(th) * e["B_Z"]
            return (e["B_phi"] / R) / (bth / r)

        val, _ = quad(pitch, 0, 2 * np.pi, epsabs=1e-13, epsrel=1e-13)
        assert abs(val / (2 * np.pi) - q_expected) < 1e-11, (r_over_a, val / (2 * np.pi), q_expected)
        assert abs(_eq(o, cfg.R0 + r, 0.0)["q"] - q_expected) < 1e-14
        assert pitch(0.3) > 0  # B_theta, B_phi > 0: cos(m theta - n phi) with m ~ nq is field aligned (R11)


# P6 ---------------------------------------------------------------------------------------
def test_P6_divB_gradB_curlb_by_finite_differences(eq_case):
    cfg, o = eq_case
    rng = np.random.default_rng(0)
    h = 1e-5
    for _ in range(10):
        r, th = cfg.a * rng.uniform(0.1, 0.95), rng.uniform(0, 2 * np.pi)
        R, Z = cfg.R0 + r * np.cos(th), r * np.sin(th)
        e = _eq(o, R, Z)
        eRp, eRm, eZp, eZm = _eq(o, R + h, Z), _eq(o, R - h, Z), _eq(o, R, Z + h), _eq(o, R, Z - h)
        d = lambda k, p, m_: (p[k] - m_[k]) / (2 * h)
        # div B = (1/R) d_R (R B_R) + d_Z B_Z  (axisymmetric)
        divB = ((R + h) * eRp["B_R"] - (R - h) * eRm["B_R"]) / (2 * h) / R + d("B_Z", eZp, eZm)
        assert abs(divB) < 1e-8 * e["B"] / cfg.a
        assert abs(d("B", eRp, eRm) - e["gradB_R"]) < 1e-8 * e["B"] / cfg.a
        assert abs(d("B", eZp, eZm) - e["gradB_Z"]) < 1e-8 * e["B"] / cfg.a
        assert e["gradB_phi"] == 0.0
        assert abs(e["b_R"] ** 2 + e["b_phi"] ** 2 + e["b_Z"] ** 2 - 1) < 1e-15
        curl = np.array([-d("b_phi", eZp, eZm),
                         d("b_R", eZp, eZm) - d("b_Z", eRp, eRm),
                         ((R + h) * eRp["b_phi"] - (R - h) * eRm["b_phi"]) / (2 * h) / R])
        got = np.array([e["curlb_R"], e["curlb_phi"], e["curlb_Z"]])
        assert np.abs(curl - got).max() < 1e-8 / cfg.a
        # independent route: curl b = (curl B + b x grad B)/B with curl B = (0, d_Z B_R - d_R B_Z, 0)
        cB = np.array([0.0, d("B_R", eZp, eZm) - d("B_Z", eRp, eRm), 0.0])
        b = np.array([e["b_R"], e["b_phi"], e["b_Z"]])
        gB = np.array([e["gradB_R"], 0.0, e["gradB_Z"]])
        bxg = np.array([b[1] * gB[2] - b[2] * gB[1], b[2] * gB[0] - b[0] * gB[2], b[0] * gB[1] - b[1] * gB[0]])
        assert np.abs((cB + bxg) / e["B"] - got).max() < 1e-8 / cfg.a
        # psi'' is the derivative of psi'
        p1p, p1m = _eq(o, cfg.R0 + r + h, 0.0)["psi1"], _eq(o, cfg.R0 + r - h, 0.0)["psi1"]
        assert abs((p1p - p1m) / (2 * h) - _eq(o, cfg.R0 + r, 0.0)["psi2"]) < 1e-7


# helpers -----------------------------------------------------------------------------------
def _energy(o, cfg, R, Z, phi, u, mu):
    g, _ = o.gather(R, Z, phi)
    B = np.array([o.equil(r, z)["B"] for r, z in zip(R, Z)])
    return 0.5 * u * u + mu * B + cfg.qom * (g[0] - u * g[4])


def _psi_of_r(o, cfg, r):
    return quad(lambda t: o.equil(cfg.R0 + t, 0.0)["psi1"], 0.0, r, epsabs=1e-15, epsrel=1e-14)[0]


def _pphi(o, cfg, R, Z, u):
    out = np.zeros(R.shape[0])
    for i, (r_, z_, u_) in enumerate(zip(R, Z, u)):
        e = o.equil(r_, z_)
        out[i] = cfg.qom * _psi_of_r(o, cfg, e["r"]) + u_ * e["F"] / e["B"]
    return out


def _smooth_case(P=8, n=400, seed=21, zero=False):
    """Small unstructured mesh carrying GLOBAL QUARTIC fields on all planes (inside the element space, n = 0):
    the interpolated field is then a C-infinity function, so RK4 shows its full order."""
    cfg = dataclasses.replace(synth.CONFIGS[0], structured=False, nr=5, ntheta=14, n_planes=P, seed=seed, n_markers=n,
                              R0=1.3, B0=1.7, a=0.4, q=(1.4, 0.1, 0.5))  # no unit-valued parameter
    RZ, tri = synth.make_mesh(cfg)
    o = Oracle()
    o.equilibrium_set(**synth.equilibrium_args(cfg))
    o.species_set(**synth.species_args(cfg))
    o.mesh_load(RZ, tri, P, cfg.phi_period)
    rng = np.random.default_rng(seed)
    nod = np.zeros((2, RZ.shape[0], 6))
    if not zero:
        for f in range(2):
            co = {(i, j): rng.normal() * 2e-3 for i in range(5) for j in range(5 - i)}
            X, Y = (RZ[:, 0] - cfg.R0) / cfg.a, RZ[:, 1] / cfg.a
            for q, (dx, dy) in enumerate([(0, 0), (1, 0), (0, 1), (2, 0), (1, 1), (0, 2)]):
                s = 0.0
                for (i, j), c in co.items():
                    if i < dx or j < dy:
                        continue
                    k = c * np.prod([i - t for t in range(dx)]) * np.prod([j - t for t in range(dy)])
                    s = s + k * X ** (i - dx) * Y ** (j - dy)
                nod[f, :, q] = s / cfg.a ** (dx + dy)
    for f in range(2):
        o.fields_set(f, np.broadcast_to(nod[f], (P,) + nod[f].shape).copy())
    m = synth.make_markers(cfg, n)
    keep = np.hypot(m["R"] - cfg.R0, m["Z"]) < 0.75 * cfg.a  # stay clear of the outer boundary
    m = {k: v[keep] for k, v in m.items()}
    return cfg, o, m


# P7 + P9 -----------------------------------------------------------------------------------
def test_P7_P9_rk4_fourth_order_and_energy_with_smooth_fields():
    """Static fields: E = u^2/2 + mu B + qom (Phi - u A) is an invariant of Eq.(2)-(6) (p_par form, R6), so RK4's
    drift falls 16x per halving of dt; so does the self-convergence error of every state component."""
    cfg, o, m = _smooth_case()
    T = 0.4
    E0 = _energy(o, cfg, m["R"], m["Z"], m["phi"], m["u"], m["mu"])
    res = {}
    for n in (4, 8, 16, 32):
        res[n] = o.push_rk4(m["R"], m["Z"], m["phi"], m["u"], m["w"], m["mu"], m["p"], T / n, n)
        assert (res[n][5] == 0).all()
    drift = {n: np.abs(_energy(o, cfg, *res[n][:4], m["mu"]) - E0).max() for n in res}
    assert drift[4] / drift[8] > 11 and drift[8] / drift[16] > 11, drift
    assert drift[32] < 1e-7 * np.abs(E0).max(), drift
    err = {n: max(np.abs(res[n][q] - res[32][q]).max() for q in (0, 1, 3, 4)) for n in (4, 8, 16)}
    # Richardson: e(4)-ish ratios; (e4-e32)/(e8-e32) -> (16^3-1)/(16^2-1)*... ~ 16.06, (e8-e32)/(e16-e32) ~ 17
    assert 12 < err[4] / err[8] < 20 and 13 < err[8] / err[16] < 21, err


def test_P7_energy_drift_with_genuine_FE_fields(cfg0_oracle):
    """Config 0's helical FE fields (non-axisymmetric, only C1): energy is still an invariant of the flow because
    the gather returns the exact gradient of the interpolant; the drift is tiny and falls with dt (order is
    reduced by the C0 gradient kinks at element edges - not a bug)."""
    cfg, RZ, tri, o, _ = cfg0_oracle
    m = synth.make_markers(cfg, 1500)
    E0 = _energy(o, cfg, m["R"], m["Z"], m["phi"], m["u"], m["mu"])
    d = {}
    for n in (5, 10, 20):
        r = o.push_rk4(m["R"], m["Z"], m["phi"], m["u"], m["w"], m["mu"], m["p"], 0.25 / n, n)
        ok = r[5] == 0
        d[n] = np.median(np.abs(_energy(o, cfg, r[0][ok], r[1][ok], r[2][ok], r[3][ok], m["mu"][ok]) - E0[ok]) / np.abs(E0[ok]))
    assert d[5] < 1e-6 and d[5] / d[10] > 2.5 and d[10] / d[20] > 2.5, d


# P8 ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("charge_sign", [1.0, -1.0])
def test_P8_canonical_toroidal_momentum(charge_sign):
    """Axisymmetric case (zero perturbation): P_phi = qom psi(r) + u F/B is conserved at 4th order with
    b* = B*/B*_par (reading R7).  The literal L53 expression b + (m/q) u curl b / B*_par drifts at a dt-independent
    level - that is how the reading was chosen.  Run for both charge signs (R8)."""
    cfg, o, m = _smooth_case(zero=True, n=120)
    sp = synth.species_args(cfg)
    sp["qom"] *= charge_sign
    cfg = dataclasses.replace(cfg)
    T = 0.4

    def run(bstar_exact, n):
        o.species_set(**{**sp, "bstar_exact": bstar_exact})
        r = o.push_rk4(m["R"], m["Z"], m["phi"], m["u"], m["w"], m["mu"], m["p"], T / n, n)
        qom = sp["qom"]
        P1 = np.array([qom * _psi_of_r(o, cfg, o.equil(a, b)["r"]) + c * o.equil(a, b)["F"] / o.equil(a, b)["B"] for a, b, c in zip(r[0], r[1], r[3])])
        P0 = np.array([qom * _psi_of_r(o, cfg, o.equil(a, b)["r"]) + c * o.equil(a, b)["F"] / o.equil(a, b)["B"] for a, b, c in zip(m["R"], m["Z"], m["u"])])
        return np.abs(P1 - P0) / np.abs(P0).max()

    d4, d8, d16 = run(1, 4), run(1, 8), run(1, 16)
    # order from the median over markers (a few fast, strongly drifting markers are still pre-asymptotic at dt = 0.1)
    assert np.median(d4) / np.median(d8) > 12 and np.median(d8) / np.median(d16) > 12, (np.median(d4), np.median(d8), np.median(d16))
    assert d16.max() < 5e-9, d16.max()
    l4, l16 = run(0, 4), run(0, 16)
    assert np.median(l16) > 1000 * np.median(d16) and 0.5 < np.median(l4) / np.median(l16) < 2.0  # dt-independent drift
    o.species_set(**synth.species_args(cfg))


# P10 --------------------------------------------------------------------------------------
def test_P10_flat_profile_weight_closed_form():
    """kappa_n = kappa_T = 0 (flat n, T = 1) and static fields: Eq.(7) integrates exactly to
    w(t) - w(0) = -(p qom/T) [ (Phi - u A)(t) - (Phi - u A)(0) ]  (dE/dt = 0 and f0 = f0(E))."""
    cfg, o, m = _smooth_case(n=300)
    sp = synth.species_args(cfg)
    sp.update(kappa_n=0.0, kappa_T=0.0)
    o.species_set(**sp)
    p = 0.5 + np.arange(m["R"].shape[0]) % 3  # not all ones
    g0, _ = o.gather(m["R"], m["Z"], m["phi"])
    diffs = []
    for n in (8, 16):
        r = o.push_rk4(m["R"], m["Z"], m["phi"], m["u"], m["w"], m["mu"], p, 0.4 / n, n)
        g1, _ = o.gather(r[0], r[1], r[2])
        pred = -(p * cfg.qom) * ((g1[0] - r[3] * g1[4]) - (g0[0] - m["u"] * g0[4]))
        got = r[4] - m["w"]
        diffs.append(np.abs(got - pred).max() / np.abs(pred).max())
    assert diffs[1] < 1e-6 and diffs[0] / diffs[1] > 10, diffs
    # nonlinear weight mode (p - w): dw/dt = (p - w) * L  =>  ln((p - w)/(p - w0)) = -int L = linear-result/p
    sp2 = dict(sp, weight_mode=1)
    o.species_set(**sp2)
    r2 = o.push_rk4(m["R"], m["Z"], m["phi"], m["u"], m["w"], m["mu"], p, 0.4 / 16, 16)
    o.species_set(**sp)
    r1 = o.push_rk4(m["R"], m["Z"], m["phi"], m["u"], m["w"], m["mu"], p, 0.4 / 16, 16)
    lin = (r1[4] - m["w"]) / p
    assert np.abs(np.log((p - r2[4]) / (p - m["w"])) + lin).max() < 1e-5 * max(np.abs(lin).max(), 1e-3)  # RK4 truncation at dt = 0.025


# P11 --------------------------------------------------------------------------------------
def test_P11_grad_ln_f0_by_finite_differences(eq_case):
    """Eq.(8) profiles (L314) inside a Maxwellian (L63): the analytic gradients used in Eq.(7) equal central
    differences of ln f0; and ln f0(u=0, mu=0) = ln n - 1.5 ln T with n, T from Eq.(8) as printed (L314),
    evaluated here in 30-digit arithmetic with r0 = a/2 (L316)."""
    cfg, o = eq_case
    rng = np.random.default_rng(1)
    h = 1e-6
    for _ in range(12):
        r, th = cfg.a * rng.uniform(0.15, 0.9), rng.uniform(0, 2 * np.pi)
        R, Z, u, mu = cfg.R0 + r * np.cos(th), r * np.sin(th), rng.normal(), rng.exponential()
        g = o.grad_ln_f0(R, Z, u, mu)
        fd = np.array([(o.ln_f0(R + h, Z, u, mu) - o.ln_f0(R - h, Z, u, mu)) / (2 * h),
                       (o.ln_f0(R, Z + h, u, mu) - o.ln_f0(R, Z - h, u, mu)) / (2 * h),
                       (o.ln_f0(R, Z, u + h, mu) - o.ln_f0(R, Z, u - h, mu)) / (2 * h)])
        assert np.abs(g - fd).max() < 2e-8 * max(1.0, np.abs(fd).max()), (g, fd)
    import mpmath as mp
    mp.mp.dps = 30
    for r_over_a in (0.2, 0.5, 0.8):
        H = lambda kap, w: mp.exp(-kap * w * (mp.mpf(cfg.a) / cfg.R0) * mp.tanh((r_over_a * mp.mpf(cfg.a) - mp.mpf(cfg.a) / 2) / (w * mp.mpf(cfg.a))))
        expect = mp.log(H(cfg.kappa_n, cfg.w_n)) - mp.mpf(3) / 2 * mp.log(H(cfg.kappa_T, cfg.w_T))
        val = o.ln_f0(cfg.R0 + r_over_a * cfg.a, 0.0, 0.0, 0.0)
        assert abs(val - float(expect)) < 1e-13


# P15 --------------------------------------------------------------------------------------
def test_P15_infinite_charge_limit_follows_field_lines():
    """qom -> infinity (kappa = m/q -> 0), zero fields, mu = 0: Eq.(2) reduces to dX/dt = u b, so r is constant and
    the toroidal angle advances by int (B_phi/R)/(B_theta/r) dtheta along the orbit (with P5: q(r) per turn)."""
    cfg, o, m = _smooth_case(zero=True, n=60)
    sp = synth.species_args(cfg)
    sp.update(qom=1e13, kappa_n=0.0, kappa_T=0.0)
    o.species_set(**sp)
    mu0 = np.zeros_like(m["mu"])
    u = np.where(np.abs(m["u"]) < 0.3, 0.7, m["u"])
    T, n = 0.6, 24
    r = o.push_rk4(m["R"], m["Z"], m["phi"], u, m["w"], mu0, m["p"], T / n, n)
    r0 = np.hypot(m["R"] - cfg.R0, m["Z"])
    r1 = np.hypot(r[0] - cfg.R0, r[1])
    assert np.abs(r1 - r0).max() < 1e-9 * cfg.a
    assert np.abs(r[3] - u).max() < 1e-12  # no mirror force, no field: u constant
    for i in range(0, r0.shape[0], 7):
        th0, th1 = np.arctan2(m["Z"][i], m["R"][i] - cfg.R0), np.arctan2(r[1][i], r[0][i] - cfg.R0)
        th1 = th0 + np.angle(np.exp(1j * (th1 - th0)))  # short orbit: |dtheta| < pi

        def pitch(th, rr=r0[i]):
            R, Z = cfg.R0 + rr * np.cos(th), rr * np.sin(th)
            e = o.equil(R, Z)
            return (e["B_phi"] / R) / ((-np.sin(th) * e["B_R"] + np.cos(th) * e["B_Z"]) / rr)

        dphi_pred = quad(pitch, th0, th1, epsabs=1e-13, epsrel=1e-13)[0]
        dphi = np.angle(np.exp(1j * (r[2][i] - m["phi"][i])))
        assert abs(dphi - dphi_pred) < 1e-8, (i, dphi, dphi_pred)
    o.species_set(**synth.species_args(cfg))


def test_lost_marker_status_and_zero_field_outside(cfg0_oracle):
    """O9 / reading R15: a marker evaluated outside the mesh keeps moving in the equilibrium with zero perturbed
    field and carries a sticky status flag; markers that stay inside are never flagged."""
    cfg, RZ, tri, o, _ = cfg0_oracle
    R = np.array([cfg.R0 + 0.999 * cfg.a, cfg.R0 + 0.5 * cfg.a])
    Z = np.array([0.0, 0.0])
    phi = np.array([0.1, 0.1])
    u = np.array([0.5, 0.5])
    mu = np.array([3.0, 0.1])  # large mu: grad-B drift pushes the first marker across the outer boundary
    w = np.zeros(2)
    p = np.ones(2)
    out = o.push_rk4(R, Z, phi, u, w, mu, p, 0.05, 40)
    assert out[5][1] == 0
    r_end = np.hypot(out[0][0] - cfg.R0, out[1][0])
    if r_end > cfg.a:
        assert out[5][0] != 0
    d, outside = o.rhs(np.array([cfg.R0 + 1.5 * cfg.a]), np.array([0.0]), phi[:1], u[:1], w[:1], mu[:1], p[:1])
    assert outside[0] == 1 and np.isfinite(d).all() and d[4, 0] == 0.0
    # unconditional form: markers that START outside (beyond the outer boundary; inside the hole of the annulus) are
    # flagged by the very first stage, whatever happens afterwards, while a marker well inside is not; the flag is
    # sticky (a status passed back in is kept, also for a marker that never leaves); and outside the mesh the motion
    # is exactly the equilibrium motion, i.e. what the same oracle gives with both perturbed fields set to zero
    Ro = np.array([cfg.R0 + 1.02 * cfg.a, cfg.R0 + 0.02 * cfg.a, cfg.R0 + 0.5 * cfg.a, cfg.R0 + 1.3 * cfg.a])
    Zo, pho = np.zeros(4), np.full(4, 0.3)
    uo, muo, wo, po = np.full(4, 0.4), np.full(4, 0.2), np.zeros(4), np.ones(4)
    one = o.push_rk4(Ro, Zo, pho, uo, wo, muo, po, 0.05, 1)
    assert list(one[5] != 0) == [True, True, False, True]
    more = o.push_rk4(*one[:5], muo, po, 0.05, 3, status=one[5])
    assert list(more[5] != 0) == [True, True, False, True]
    kept = o.push_rk4(Ro[2:3], Zo[2:3], pho[2:3], uo[2:3], wo[2:3], muo[2:3], po[2:3], 0.05, 2, status=np.array([1], dtype=np.int32))
    assert kept[5][0] != 0
    from oracle import Oracle
    z = Oracle()
    z.equilibrium_set(**synth.equilibrium_args(cfg))
    z.species_set(**synth.species_args(cfg))
    z.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)
    zero = np.zeros((cfg.n_planes, RZ.shape[0], 6))
    z.fields_set(0, zero)
    z.fields_set(1, zero)
    far = o.push_rk4(Ro[3:], Zo[3:], pho[3:], uo[3:], wo[3:], muo[3:], po[3:], 0.05, 5)
    ref = z.push_rk4(Ro[3:], Zo[3:], pho[3:], uo[3:], wo[3:], muo[3:], po[3:], 0.05, 5)
    for q in range(5):
        assert far[q][0] == ref[q][0]
    assert far[4][0] == 0.0  # w stays 0: no perturbed field, no weight drive


# ------------------------------------------------------------------------------------------- O10: the other G2P kernels
def test_other_g2p_kernels_pullback_density_f_interp(cfg0_oracle):
    """Pins P17-P19 for the three grid-to-particle kernels of PAPER.md L97-103 (readings R22-R24).
    P17 pullback: identity where A_par = 0 (here: with a zero A_par field) and outside the mesh (status set); for a spatially
         constant A_par = a0 every marker's u shifts by exactly (q/m) a0 (Eq.(6)) and w by p (q/m) a0 d ln f0/du with
         d ln f0/du from a central difference of ln f0 (an independent route); forth and back (a0, then -a0) restores u and
         leaves w off by exactly -p ((q/m) a0)^2 / T(r), the second-order term the linearisation drops.
    P18 density: equals row 0 / row 4 of the pinned gather, and a0 for the constant field.
    P19 f-interpolation: equals exp(ln f0) at the shifted velocity; with A_par = 0 it is f0(u); ratio of two markers that differ
         only in u is exp(-(u1^2 - u2^2) / 2T)."""
    from oracle import Oracle
    cfg, RZ, tri, o, (dphi, dap) = cfg0_oracle
    m = synth.make_markers(cfg, 400)
    R, Z, phi, u, w, mu, p = [m[k] for k in ("R", "Z", "phi", "u", "w", "mu", "p")]
    qom = cfg.qom
    # constant A_par = a0: nodal value a0, all derivatives zero, every plane (spline coefficients of a constant are the constant)
    a0 = 3.0e-3
    z = Oracle()
    z.equilibrium_set(**synth.equilibrium_args(cfg))
    z.species_set(**synth.species_args(cfg))
    z.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)
    const = np.zeros((cfg.n_planes, RZ.shape[0], 6))
    const[:, :, 0] = a0
    z.fields_set(0, np.zeros_like(const))
    z.fields_set(1, const)
    u1, w1, st = z.pullback(R, Z, phi, u, w, mu, p)
    assert not st.any()
    assert np.abs((u - u1) - qom * a0).max() < 1e-13 * qom * a0 * 10
    h = 1e-5
    dlnf = np.array([(z.ln_f0(a, b, c + h, d) - z.ln_f0(a, b, c - h, d)) / (2 * h) for a, b, c, d in zip(R, Z, u, mu)])
    assert np.abs((w1 - w) - p * qom * a0 * dlnf).max() < 1e-8 * np.abs(w1 - w).max()
    # back with -a0
    const[:, :, 0] = -a0
    z.fields_set(1, const)
    u2, w2, _ = z.pullback(R, Z, phi, u1, w1, mu, p)
    assert np.abs(u2 - u).max() < 1e-14
    T = np.array([-(c) / z.grad_ln_f0(a, b, c, d)[2] for a, b, c, d in zip(R, Z, u, mu)])      # d ln f0/du = -u/T
    assert np.abs((w2 - w) + p * (qom * a0) ** 2 / T).max() < 1e-10 * (qom * a0) ** 2
    # zero A_par: identity; outside the mesh: identity + status
    const[:, :, 0] = 0.0
    z.fields_set(1, const)
    u3, w3, st3 = z.pullback(R, Z, phi, u, w, mu, p)
    assert np.array_equal(u3, u) and np.array_equal(w3, w) and not st3.any()
    Ro = R.copy()
    Ro[:5] = cfg.R0 + 1.5 * cfg.a
    u4, w4, st4 = o.pullback(Ro, Z, phi, u, w, mu, p)
    assert st4[:5].all() and not st4[5:].any() and np.array_equal(u4[:5], u[:5]) and np.array_equal(w4[:5], w[:5])
    assert np.abs(u4[5:] - u[5:]).max() > 0          # the config-0 field does move the others
    # P18
    g, _ = o.gather(R, Z, phi)
    assert np.array_equal(o.density_g2p(0, R, Z, phi), g[0]) and np.array_equal(o.density_g2p(1, R, Z, phi), g[4])
    const[:, :, 0] = a0
    z.fields_set(1, const)
    assert np.abs(z.density_g2p(1, R, Z, phi) - a0).max() < 1e-15
    # P19
    fi = z.f_interp(R, Z, phi, u, mu)
    ref = np.exp([z.ln_f0(a, b, c - qom * a0, d) for a, b, c, d in zip(R, Z, u, mu)])
    assert np.abs(fi - ref).max() <= 1e-15 * ref.max()
    const[:, :, 0] = 0.0
    z.fields_set(1, const)
    f_a = z.f_interp(R, Z, phi, u, mu)
    f_b = z.f_interp(R, Z, phi, 0.5 * u, mu)
    assert np.abs(np.log(f_a / f_b) + (u ** 2 - (0.5 * u) ** 2) / (2 * T)).max() < 1e-11


# ------------------------------------------------------------------------------------------- O11: particle-to-grid
def test_P20_deposit_is_the_transpose_of_the_gather(cfg0_oracle):
    """Pin P20 for the P2G deposition (reading R25).  b = G^T q is fixed by the pinned gather G through the
    adjoint identity  sum_dof b_dof d_dof = sum_p q_p F_d(x_p)  for EVERY DOF vector d: checked for random d (all six
    components, all planes), for d = the constant 1 (total deposited charge = sum of the charges inside the mesh: quintics
    contain constants, B-splines sum to one), and through locality: a marker touches only the three nodes of its triangle
    on the four planes of its toroidal interval, and markers outside the mesh deposit nothing."""
    from oracle import Oracle
    cfg, RZ, tri, o, _ = cfg0_oracle
    m = synth.make_markers(cfg, 300)
    R, Z, phi = m["R"].copy(), m["Z"].copy(), m["phi"]
    R[:4] = cfg.R0 + 1.4 * cfg.a                       # outside
    q = synth.uniform(5, 1, 300) - 0.3
    b = o.deposit(R, Z, phi, q)
    assert b.shape == (cfg.n_planes, RZ.shape[0], 6)
    z = Oracle()
    z.equilibrium_set(**synth.equilibrium_args(cfg))
    z.species_set(**synth.species_args(cfg))
    z.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)
    rng = np.random.default_rng(3)
    scale = np.array([1.0, 5.0, 5.0, 25.0, 25.0, 25.0])          # derivative DOFs in their natural units (1/a powers)
    for trial in range(3):
        d = rng.normal(size=b.shape) * scale
        z.fields_set(0, d)
        F, t = z.gather(R, Z, phi)
        lhs, rhs = float((b * d).sum()), float((q * F[0]).sum())
        assert abs(lhs - rhs) < 1e-11 * np.abs(q * F[0]).sum(), (trial, lhs, rhs)
    one = np.zeros(b.shape)
    one[:, :, 0] = 1.0
    inside = o.locate(R, Z) >= 0
    assert inside.sum() == 296
    assert abs(float((b * one).sum()) - q[inside].sum()) < 1e-12 * np.abs(q).sum()
    # locality of one marker
    i = 10
    b1 = o.deposit(R[i:i + 1], Z[i:i + 1], phi[i:i + 1], np.ones(1))
    k, w, dw = o.bspline(phi[i])
    planes = sorted({(k - 1 + a) % cfg.n_planes for a in range(4)})
    nodes = sorted(tri[o.locate(R[i:i + 1], Z[i:i + 1])[0]])
    nz = np.argwhere(np.abs(b1).max(axis=2) > 0)
    assert sorted(set(nz[:, 0])) == planes and sorted(set(nz[:, 1])) == nodes
    assert np.abs(o.deposit(R[:4], Z[:4], phi[:4], np.ones(4))).max() == 0.0


# ------------------------------------------------------------------------------------------- O12: gyro-average
def test_P21_gyro_average_of_polynomial_fields_has_a_closed_form():
    """Pin P21 for the N-point gyro-average (reading R26).  On fields that are global polynomials of degree <= 4 (inside the
    element space, all planes equal) the ring average is known in closed form for N >= 5 points: with x = R - R0, z = Z,
        <x^2> = x^2 + rho^2/2,  <x z> = x z,  <x^3> = x^3 + 3 x rho^2/2,  <x^2 z^2> = x^2 z^2 + (x^2 + z^2) rho^2/2 + rho^4/8,
    the average of the gradient is the gradient of the average; rho = 0 and N = 1 give the plain gather; an odd-order
    term survives with too few points (N = 2 on x^3 is exact only by symmetry of that ring: negative control with N = 3 on
    x^2 z^2, which needs N >= 5)."""
    cfg, o, m = _smooth_case(P=8, n=300, zero=True)
    RZ, tri = synth.make_mesh(cfg)
    X, Zc = RZ[:, 0] - cfg.R0, RZ[:, 1]
    # Phi = x^2 z^2 + 0.5 x^3 ; A = x z + 2 x^2   (nodal value, gradient, Hessian)
    dP = np.stack([X**2 * Zc**2 + 0.5 * X**3, 2 * X * Zc**2 + 1.5 * X**2, 2 * X**2 * Zc, 2 * Zc**2 + 3 * X, 4 * X * Zc, 2 * X**2], -1)
    dA = np.stack([X * Zc + 2 * X**2, Zc + 4 * X, X, 4 * np.ones_like(X), np.ones_like(X), np.zeros_like(X)], -1)
    o.fields_set(0, np.broadcast_to(dP, (8,) + dP.shape).copy())
    o.fields_set(1, np.broadcast_to(dA, (8,) + dA.shape).copy())
    rr = np.hypot(m["R"] - cfg.R0, m["Z"])
    keep = (rr < 0.6 * cfg.a) & (rr > 0.35 * cfg.a)       # the whole ring (rho <= 0.05 = a/8) stays inside the annulus
    R, Z, phi = m["R"][keep], m["Z"][keep], m["phi"][keep]
    rho = 0.02 + 0.03 * synth.uniform(9, 1, R.shape[0])
    x, z = R - cfg.R0, Z
    for N in (5, 8):
        g, t = o.gather_gyro(R, Z, phi, rho, N)
        expP = x**2 * z**2 + (x**2 + z**2) * rho**2 / 2 + rho**4 / 8 + 0.5 * (x**3 + 1.5 * x * rho**2)
        expPR = 2 * x * z**2 + x * rho**2 + 0.5 * (3 * x**2 + 1.5 * rho**2)
        expPZ = 2 * x**2 * z + z * rho**2
        expA = x * z + 2 * (x**2 + rho**2 / 2)
        for got, exp in ((g[0], expP), (g[1], expPR), (g[2], expPZ), (g[4], expA), (g[5], z + 4 * x), (g[6], x)):
            assert np.abs(got - exp).max() < 1e-12 * max(np.abs(exp).max(), 1e-3), N
        assert np.abs(g[3]).max() < 1e-15 and np.abs(g[7]).max() < 1e-15      # all planes equal: no phi dependence
    g3, _ = o.gather_gyro(R, Z, phi, rho, 3)
    assert np.abs(g3[0] - expP).max() > 1e-9                                   # negative control: three points are too few for x^2 z^2
    plain, tp = o.gather(R, Z, phi)
    g1, t1 = o.gather_gyro(R, Z, phi, 0 * rho, 6)
    assert np.abs(g1 - plain).max() < 1e-14 * np.abs(plain).max() and np.array_equal(t1, tp)      # six equal terms summed and divided by six
    g1b, _ = o.gather_gyro(R + rho, Z, phi, rho, 1)                            # one point: the ring point at angle 0
    pl2, _ = o.gather(R + 2 * rho, Z, phi)
    assert np.abs(g1b - pl2).max() < 1e-14 * np.abs(pl2).max()


# ------------------------------------------------------------------------------------------- O13: numeric equilibrium
def _cubic_exact_coefs(f, nR, nZ, Rmin, Rmax, Zmin, Zmax):
    """B-spline coefficients that reproduce a function that is a cubic in R and a cubic in Z EXACTLY: the textbook
    quasi-interpolant c = f - h^2 f''/6 applied in each direction (exact on cubics), with derivatives by exact finite
    differences of cubics.  Knot i of the coefficient array sits at Rmin + (i - 1) h."""
    hR, hZ = (Rmax - Rmin) / nR, (Zmax - Zmin) / nZ
    Rk = Rmin + (np.arange(nR + 3) - 1) * hR
    Zk = Zmin + (np.arange(nZ + 3) - 1) * hZ
    RR, ZZ = np.meshgrid(Rk, Zk, indexing="ij")
    d2R = lambda g: (g(RR + hR, ZZ) - 2 * g(RR, ZZ) + g(RR - hR, ZZ))          # = h^2 f_RR exactly for cubics
    d2Z = lambda g: (g(RR, ZZ + hZ) - 2 * g(RR, ZZ) + g(RR, ZZ - hZ))
    f0 = f(RR, ZZ)
    fR = d2R(f)
    fZ = d2Z(f)
    fRZ = (f(RR + hR, ZZ + hZ) - 2 * f(RR, ZZ + hZ) + f(RR - hR, ZZ + hZ)) - 2 * fR + (f(RR + hR, ZZ - hZ) - 2 * f(RR, ZZ - hZ) + f(RR - hR, ZZ - hZ))
    return f0 - fR / 6 - fZ / 6 + fRZ / 36


def test_P22_numeric_equilibrium_closed_form_and_convergence_to_the_analytic_one(cfg0_oracle):
    """Pin P22 (reading R27).  (a) a flux function that is cubic in R and in Z is reproduced exactly by the spline, so B, grad B
    and curl b have closed forms: B_R = -psi_Z/R, B_Z = psi_R/R, B_phi = F/R, checked directly, with div B = 0, grad B and
    curl b by central differences of the returned B and b (the P6 checks), at points that straddle knot lines.
    (b) the spline interpolant of the ANALYTIC circular equilibrium's psi converges to the analytic oracle's B, grad B,
    curl b at fourth / second order in the knot spacing (values / second-derivative quantities)."""
    from oracle import Oracle
    from scipy.interpolate import RectBivariateSpline  # noqa: F401  (scipy is only used for (b))
    cfg, RZ, tri, o, _ = cfg0_oracle
    al, be, ga, de, R0, F = 0.8, 1.3, 0.4, -0.6, 1.1, 2.3
    psi = lambda R, Z: al * (R - R0) ** 2 + be * Z**2 + ga * (R - R0) ** 3 + de * (R - R0) * Z**2 + 0.2 * (R - R0) ** 2 * Z**3
    z = Oracle()
    box = (0.6, 1.7, -0.5, 0.6)
    coef = _cubic_exact_coefs(psi, 11, 9, *box)
    z.equilibrium_set_numeric(11, 9, *box, F, R0, 0.4, coef)
    rng = np.random.default_rng(8)
    h = 1e-5
    for _ in range(12):
        R, Z = rng.uniform(0.7, 1.6), rng.uniform(-0.4, 0.5)
        x = R - R0
        pR = 2 * al * x + 3 * ga * x**2 + de * Z**2 + 0.4 * x * Z**3
        pZ = 2 * be * Z + 2 * de * x * Z + 0.6 * x**2 * Z**2
        e = z.equil(R, Z)
        assert abs(e["B_R"] + pZ / R) < 1e-13 and abs(e["B_Z"] - pR / R) < 1e-13 and abs(e["B_phi"] - F / R) < 1e-15
        assert abs(e["B"] - np.sqrt(pR**2 + pZ**2 + F**2) / R) < 1e-13
        eRp, eRm, eZp, eZm = z.equil(R + h, Z), z.equil(R - h, Z), z.equil(R, Z + h), z.equil(R, Z - h)
        d = lambda k, p_, m_: (p_[k] - m_[k]) / (2 * h)
        divB = ((R + h) * eRp["B_R"] - (R - h) * eRm["B_R"]) / (2 * h) / R + d("B_Z", eZp, eZm)
        assert abs(divB) < 1e-8
        assert abs(d("B", eRp, eRm) - e["gradB_R"]) < 1e-8 and abs(d("B", eZp, eZm) - e["gradB_Z"]) < 1e-8
        curl = np.array([-d("b_phi", eZp, eZm), d("b_R", eZp, eZm) - d("b_Z", eRp, eRm),
                         ((R + h) * eRp["b_phi"] - (R - h) * eRm["b_phi"]) / (2 * h) / R])
        assert np.abs(curl - np.array([e["curlb_R"], e["curlb_phi"], e["curlb_Z"]])).max() < 1e-8
    # (b) convergence to the analytic circular equilibrium of config 0
    from scipy.integrate import quad
    from scipy.interpolate import make_interp_spline
    psi1 = lambda r: o.equil(cfg.R0 + r, 0.0)["psi1"]
    rr = np.linspace(0.0, 1.6 * cfg.a, 400)
    pr = np.concatenate([[0.0], np.cumsum([quad(psi1, a_, b_, epsabs=1e-14)[0] for a_, b_ in zip(rr[:-1], rr[1:])])])
    psi_r = make_interp_spline(rr, pr, k=5)
    errs = []
    for n in (24, 48):
        box = (cfg.R0 - 1.2 * cfg.a, cfg.R0 + 1.2 * cfg.a, -1.2 * cfg.a, 1.2 * cfg.a)
        hR = (box[1] - box[0]) / n
        # interpolating spline coefficients through samples at the knots (library routine): not-a-knot is not what the
        # uniform spline space wants at the ends, so fit on an extended grid and keep a window
        Rk = box[0] + (np.arange(n + 3) - 1) * hR
        Zk = box[2] + (np.arange(n + 3) - 1) * hR
        RR, ZZ = np.meshgrid(Rk, Zk, indexing="ij")
        samples = psi_r(np.hypot(RR - cfg.R0, ZZ))
        # solve the tridiagonal (1,4,1)/6 systems in both directions with natural-ish ends (end effects stay at the border)
        M = (np.diag(np.full(n + 3, 4.0)) + np.diag(np.ones(n + 2), 1) + np.diag(np.ones(n + 2), -1)) / 6
        M[0, :3] = [1, -2, 1]; M[-1, -3:] = [1, -2, 1]
        rhs = samples.copy(); rhs[0, :] = 0; rhs[-1, :] = 0
        c1 = np.linalg.solve(M, rhs)
        rhs2 = c1.T.copy(); rhs2[0, :] = 0; rhs2[-1, :] = 0
        coef = np.linalg.solve(M, rhs2).T
        z.equilibrium_set_numeric(n, n, *box, cfg.B0 * cfg.R0, cfg.R0, cfg.a, coef)
        e_max = np.zeros(3)
        for r_, th in [(0.3, 0.4), (0.5, 2.0), (0.7, 4.0), (0.6, 5.5)]:
            R, Z = cfg.R0 + r_ * cfg.a * np.cos(th), r_ * cfg.a * np.sin(th)
            en, ea = z.equil(R, Z), o.equil(R, Z)
            e_max[0] = max(e_max[0], abs(en["B"] - ea["B"]) / ea["B"])
            e_max[1] = max(e_max[1], abs(en["gradB_R"] - ea["gradB_R"]), abs(en["gradB_Z"] - ea["gradB_Z"]))
            e_max[2] = max(e_max[2], abs(en["curlb_phi"] - ea["curlb_phi"]))
        errs.append(e_max)
    print("numeric equilibrium vs analytic, n = 24 / 48:", errs)
    assert errs[1][0] < 2e-6 and errs[0][0] / errs[1][0] > 5          # |B| from first derivatives of psi: third order or better
    assert errs[1][1] < 1e-3 and errs[1][1] < errs[0][1]              # grad B, curl b from second derivatives of the fitted psi: small
    assert errs[1][2] < 1e-3 and errs[1][2] < errs[0][2]              # and decreasing (their rate is set by the crude end conditions of this fit)
