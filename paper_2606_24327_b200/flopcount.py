"""Algorithmic flop count of ONE right-hand-side evaluation of the marker push.

The count is produced by running the documented minimal formulation below once on an operation-counting scalar:
every +, - and * is one flop, a fused multiply-add is two, and each division, square root and exponential is ONE
flop (the Newton steps and polynomials that implement them on the GPU are NOT counted: they are cost, not work).
Negation, comparisons, floor, integer work and loads are free.  `python -m paper_2606_24327_b200.flopcount` prints
the breakdown; bench.py takes FLOP_PER_EVAL / FLOP_PER_PUSH from here instead of a literal.

The formulation (what the kernels in csrc/trimeg_math.cuh compute, in its cheapest form):
  locate    reference coordinates of the point in its triangle = the barycentrics of the inside test
  bspline   interval, fraction, 4 cubic B-spline weights and 4 derivative weights
  gather    2 fields x 4 planes: bivariate quintic value, d/dxi, d/deta by nested Horner with the derivative recurrence
            (38 FMA), weighted sums over the planes, J^-T to the physical gradient
  equil     analytic circular tokamak: B, 1/B, b, grad B, J = (curl B)_phi (5 divisions / reciprocals, 3 square roots)
  rhs       Eq.(2)-(6) in p_par form, b* = B*/B*_par
  weight    Eq.(7) with the Eq.(8) profiles (2 exponentials)
  rk        the stage's share of the RK4 combination for 5 unknowns
It holds none of the method's arithmetic used for results: nothing here is imported by the kernels, the oracle or a test
comparison; it only counts.
"""
from __future__ import annotations

COUNTS = {"add": 0, "mul": 0, "div": 0, "sqrt": 0, "exp": 0}


class S:
    """operation-counting scalar (the value is carried along so that the formulation can be sanity-checked)"""
    __slots__ = ("v",)

    def __init__(self, v):
        self.v = float(v.v if isinstance(v, S) else v)

    @staticmethod
    def _v(x):
        return x.v if isinstance(x, S) else float(x)

    def __add__(self, o):
        COUNTS["add"] += 1
        return S(self.v + S._v(o))

    __radd__ = __add__

    def __sub__(self, o):
        COUNTS["add"] += 1
        return S(self.v - S._v(o))

    def __rsub__(self, o):
        COUNTS["add"] += 1
        return S(S._v(o) - self.v)

    def __mul__(self, o):
        COUNTS["mul"] += 1
        return S(self.v * S._v(o))

    __rmul__ = __mul__

    def __neg__(self):
        return S(-self.v)

    def __truediv__(self, o):
        COUNTS["div"] += 1
        return S(self.v / S._v(o))

    def __rtruediv__(self, o):
        COUNTS["div"] += 1
        return S(S._v(o) / self.v)


def fma(a, b, c):
    COUNTS["mul"] += 1
    COUNTS["add"] += 1
    return S(S._v(a) * S._v(b) + S._v(c))


def sqrt(a):
    COUNTS["sqrt"] += 1
    return S(abs(S._v(a)) ** 0.5)


def exp(a):
    import math
    COUNTS["exp"] += 1
    return S(math.exp(max(-50.0, min(50.0, S._v(a)))))


def _snapshot():
    return dict(COUNTS)


def _since(s0):
    d = {k: COUNTS[k] - s0[k] for k in COUNTS}
    d["flop"] = sum(d.values())
    return d


# ------------------------------------------------------------------------------------------- the formulation
def _locate(R, Z):
    v0x, v0y, a11, a12, a21, a22 = 1.0, 0.1, 3.0, 0.2, -0.4, 2.5
    dx, dy = R - v0x, Z - v0y
    xi = fma(a11, dx, a12 * dy)
    eta = fma(a21, dx, a22 * dy)
    l0 = 1.0 - xi - eta          # third barycentric of the inside test
    return xi, eta, l0


def _bspline(phi):
    inv_dphi, half_inv_dphi, m2_inv_dphi, period, inv_period = 10.0, 5.0, -20.0, 6.28, 1 / 6.28
    pm = fma(-period, int((phi * inv_period).v), phi)      # phi modulo the period (floor is free)
    u = pm * inv_dphi
    s = u - int(u.v)
    t = 1.0 - s
    s2, t2 = s * s, t * t
    s2h, t2h = s2 * half_inv_dphi, t2 * half_inv_dphi
    w = [t2 * t * (1 / 6), fma(s2, fma(0.5, s, -1.0), 2 / 3), fma(t2, fma(0.5, t, -1.0), 2 / 3), s2 * s * (1 / 6)]
    dw = [-t2h, fma(3.0, s2h, m2_inv_dphi * s), -fma(3.0, t2h, m2_inv_dphi * t), s2h]
    return w, dw


def _horner(c, x):
    """value and derivative of sum_i c[i] x^i by Horner with the derivative recurrence: 2 N - 1 FMA for degree N"""
    n = len(c) - 1
    if n == 0:
        return S(c[0]), None
    v = fma(c[n], x, c[n - 1])
    d = S(c[n])
    for i in range(n - 2, -1, -1):
        d = fma(d, x, v)
        v = fma(v, x, c[i])
    return v, d


def _quintic(c, xi, eta):
    """p, p_xi, p_eta of the 21-coefficient quintic, j-major rows a_j(xi) of degree 5 - j: 38 FMA"""
    rows, o = [], 0
    for j in range(6):
        rows.append(c[o:o + 6 - j])
        o += 6 - j
    a5, _ = _horner(rows[5], xi)
    a4, a4x = _horner(rows[4], xi)
    p, py, px = fma(a5, eta, a4), a5, a4x
    for j in (3, 2, 1, 0):
        a, ax = _horner(rows[j], xi)
        py = fma(py, eta, p)
        p = fma(p, eta, a)
        px = fma(px, eta, ax)
    return p, px, py


def _gather(xi, eta, w, dw, u):
    """what the right-hand sides need: A, and g = grad(Phi - u A) as (d_R, raw d_phi, d_Z)"""
    a11, a12, a21, a22 = 3.0, 0.2, -0.4, 2.5
    c = [0.01 * (i + 1) for i in range(21)]
    acc = None
    for j in range(4):
        vals = []
        for f in range(2):
            p, px, py = _quintic(c, xi, eta)
            vals.append((p, px, py))
        if acc is None:   # first plane: products, no accumulate
            acc = [[w[j] * px, w[j] * py, dw[j] * p, w[j] * p] for (p, px, py) in vals]
        else:
            acc = [[fma(w[j], px, a[0]), fma(w[j], py, a[1]), fma(dw[j], p, a[2]), fma(w[j], p, a[3])] for (p, px, py), a in zip(vals, acc)]
    (Px, Py, Pp, _P), (Ax, Ay, Ap, A) = acc
    COUNTS["mul"] -= 1    # Phi itself is not needed by the right-hand sides: its 4 weighted terms are not formed
    COUNTS["add"] -= 3
    COUNTS["mul"] -= 3
    gx, gy, gp = fma(-u, Ax, Px), fma(-u, Ay, Py), fma(-u, Ap, Pp)
    gR = fma(a11, gx, a21 * gy)
    gZ = fma(a12, gx, a22 * gy)
    return gR, gZ, gp, A


def _equil(R, Z):
    R0, B0, F, F2, inv_a, inv_R0sq, q0, q1, q2 = 1.67, 2.0, 3.34, 11.1556, 1 / 0.6, 1 / 1.67 ** 2, 0.86, -0.16, 2.52
    x = R - R0
    r2 = fma(x, x, Z * Z)
    r = sqrt(r2)
    ir = 1.0 / r
    c, s = x * ir, Z * ir
    xa = r * inv_a
    q = fma(xa, fma(q2, xa, q1), q0)
    dq = fma(2.0 * q2, xa, q1) * inv_a
    s2 = fma(-r2, inv_R0sq, 1.0)
    sq = sqrt(s2)
    qb = q * sq
    dqb = fma(dq, sq, -((q * r) * inv_R0sq) / sq)
    iqb = 1.0 / qb
    P = (B0 * r) * iqb
    P1 = fma(-P, dqb, B0) * iqb
    H2 = fma(P, P, F2)
    H = sqrt(H2)
    iH = 1.0 / H
    iR = 1.0 / R
    B = H * iR
    bt = P * iH
    t = (P * P1) * (iH * iR)
    e = dict(B=B, iB=R * iH, iR=iR, bR=-(bt * s), bZ=bt * c, bp=F * iH, gBR=fma(t, c, -(B * iR)), gBZ=t * s,
             J=fma(P * c, iR, -fma(P, ir, P1)) * iR, r=r, c=c, s=s)
    return e


def _rhs(e, u, mu, gR, gZ, gp_raw, A):
    qom, kappa = 60.0, 1 / 60.0
    ku, km = kappa * u, kappa * mu
    kub = ku * e["iB"]
    Bss = fma(kub * e["bp"], e["J"], e["B"])
    iBss = 1.0 / Bss
    SR = fma(kub, e["bp"] * e["gBZ"], e["B"] * e["bR"])
    Sp = fma(kub, fma(e["bZ"], e["gBR"], fma(-e["bR"], e["gBZ"], e["J"])), e["B"] * e["bp"])
    SZ = fma(-kub, e["bp"] * e["gBR"], e["B"] * e["bZ"])
    gp = gp_raw * e["iR"]
    GR, GZ = fma(km, e["gBR"], gR), fma(km, e["gBZ"], gZ)
    cR = fma(e["bp"], GZ, -(e["bZ"] * gp))
    cp = fma(e["bZ"], GR, -(e["bR"] * GZ))
    cZ = fma(e["bR"], gp, -(e["bp"] * GR))
    vpar = fma(-qom, A, u)
    d0 = fma(vpar, SR, cR) * iBss
    d1 = fma(vpar, SZ, cZ) * iBss
    d2 = fma(vpar, Sp, cp) * (iBss * e["iR"])
    qgR, qgp, qgZ = qom * gR, qom * gp, qom * gZ
    Sqg = fma(SR, qgR, fma(Sp, qgp, SZ * qgZ))
    d3 = -(fma(mu, fma(SR, e["gBR"], SZ * e["gBZ"]), Sqg) * iBss)
    return (d0, d1, d2, d3), dict(SR=SR, SZ=SZ, Sqg=Sqg, iBss=iBss, gp=gp)


def _weight(e, x, u, mu, p, gR, gZ, A):
    qom, kn_R0, kT_R0, two_inv_w_a, r0, cT = 60.0, 2.2 / 1.67, 6.9 / 1.67, 2 / (0.3 * 0.6), 0.3, 6.9 * 0.3 * 0.6 / 1.67
    hR = fma(e["bp"], gZ, -(e["bZ"] * x["gp"]))
    hZ = fma(e["bR"], x["gp"], -(e["bp"] * gR))
    qA = qom * A
    eR, eZ = fma(-qA, x["SR"], hR), fma(-qA, x["SZ"], hZ)
    dr = e["r"] - r0
    th = fma(-2.0, 1.0 / (exp(dr * two_inv_w_a) + 1.0), 1.0)       # tanh((r - r0) / (w a)), w_n = w_T
    sech2 = fma(-th, th, 1.0)
    dlnT, dlnn = -kT_R0 * sech2, -kn_R0 * sech2
    iT = exp(cT * th)                                             # 1 / T(r), Eq.(8)
    En = fma(0.5 * u, u, mu * e["B"])
    cr = fma(dlnT, fma(En, iT, -1.5), dlnn)
    muT = mu * iT
    glR, glZ = fma(cr, e["c"], -(muT * e["gBR"])), fma(cr, e["s"], -(muT * e["gBZ"]))
    return -((p * x["iBss"]) * fma(eR, glR, fma(eZ, glZ, x["Sqg"] * (u * iT))))


def _rk(y, d):
    """one stage's share of classical RK4 for 5 unknowns: next evaluation point y_n + c dt k (5 FMA) and the running
    combination acc += b k (5 FMA): 20 flop per stage"""
    h, b = 0.025, 2.0
    nxt = [fma(h, dk, yk) for dk, yk in zip(d, y)]
    acc = [fma(b, dk, yk) for dk, yk in zip(d, y)]
    return nxt, acc


def count():
    """-> dict part -> {add, mul, div, sqrt, exp, flop}, plus 'total'"""
    for k in COUNTS:
        COUNTS[k] = 0
    R, Z, phi, u, w, mu, p = S(1.9), S(0.12), S(1.234), S(0.7), S(1e-4), S(0.4), S(1.0)
    parts = {}
    s0 = _snapshot(); xi, eta, _ = _locate(R, Z); parts["locate"] = _since(s0)
    s0 = _snapshot(); bw, bdw = _bspline(phi); parts["bspline"] = _since(s0)
    s0 = _snapshot(); gR, gZ, gp, A = _gather(xi, eta, bw, bdw, u); parts["gather"] = _since(s0)
    s0 = _snapshot(); e = _equil(R, Z); parts["equil"] = _since(s0)
    s0 = _snapshot(); d4, x = _rhs(e, u, mu, gR, gZ, gp, A); parts["rhs"] = _since(s0)
    s0 = _snapshot(); dw_ = _weight(e, x, u, mu, p, gR, gZ, A); parts["weight"] = _since(s0)
    s0 = _snapshot(); _rk([R, Z, phi, u, w], list(d4) + [dw_]); parts["rk"] = _since(s0)
    tot = {k: sum(v[k] for v in parts.values()) for k in ("add", "mul", "div", "sqrt", "exp", "flop")}
    parts["total"] = tot
    return parts


FLOP_PER_EVAL = count()["total"]["flop"]
FLOP_PER_PUSH = 4 * FLOP_PER_EVAL
SURVEY_FLOP_PER_EVAL = 943   # the survey's own count of its minimal formulation (for comparison only)

if __name__ == "__main__":
    c = count()
    for k, v in c.items():
        print(f"{k:8s} {v['flop']:5d} flop  (add {v['add']}, mul {v['mul']}, div {v['div']}, sqrt {v['sqrt']}, exp {v['exp']})")
    print(f"per RK4 marker-step: 4 x {FLOP_PER_EVAL} = {FLOP_PER_PUSH} flop   (SURVEY.md 8(a): 4 x {SURVEY_FLOP_PER_EVAL} = {4 * SURVEY_FLOP_PER_EVAL})")
