// Device arithmetic of the marker push: toroidal B-spline weights, reduced-quintic evaluation,
// analytic equilibrium, guiding-centre and weight right-hand sides.  fp64 throughout.
// Passages: /root/reference/PAPER.md L35 (C1 element x cubic B-spline), Eq.(2)-(6) L45-55, B*_par L61,
// Eq.(7), Eq.(8) L314.  Formulation notes (what differs from a literal transcription) are in DESIGN.md
// section 6 "Kernel arithmetic".
//
// The routines are templates over the scalar type T (double everywhere in this build; round 2 also tried a two-markers-
// per-lane type with shared coefficient loads).
#pragma once
#include <cstdint>

namespace trimeg {

constexpr int NCOEF = 21;                 // quintic monomials xi^i eta^j, i + j <= 5
constexpr int PLANE_STRIDE = NCOEF * 2;   // doubles per (triangle, plane): [21][field]
constexpr int PLANE_PAD = 1;              // extra toroidal planes in front of the padded coefficient table
// padded table: plane index pp in [0, NPP) holds toroidal plane (pp - 1 - PLANE_PAD) mod P, so the four planes
// k-1..k+2 of interval k are pp = k + PLANE_PAD .. k + PLANE_PAD + 3, contiguous for every k (no wrap in the kernels);
// NPP = (number of 4-interval windows) * 4 + 3 + 2 PLANE_PAD (see trimeg_mesh_load)
constexpr double INSIDE_TOL = -1e-12;

#define TRIMEG_DI __device__ __forceinline__

using ::fma;

struct EquilP {
    double R0, B0, F, F2, inv_a, inv_R0sq, q0, q1, q2;   // F = B0 R0, F2 = F^2
    int qbar_sqrt;
    // kind 1: numeric equilibrium, psi(R, Z) as tensor-product uniform cubic B-spline coefficients psi[nR + 3][nZ + 3] on
    // [Rmin, Rmin + nR hR] x [Zmin, Zmin + nZ hZ] (reading R27); F, F2, R0 as above
    int kind;
    const double* psi;
    int nR, nZ;
    double Rmin, Zmin, inv_hR, inv_hZ;
};
struct SpeciesP {
    double qom, kappa;                 // q/m and m/q
    double kn_R0, kT_R0;               // kappa_n / R0, kappa_T / R0   (d ln H/dr = -(kappa_H/R0) sech^2)
    double two_inv_wn_a, two_inv_wT_a, r0;     // 2/(w_n a), 2/(w_T a): tanh x = 1 - 2/(exp(2x) + 1)
    double cT;                         // kappa_T w_T a / R0 : 1/T = exp(cT tanh)
    double cn;                         // kappa_n w_n a / R0 : n = exp(-cn tanh)
    int same_w, bstar_exact, weight_mode;
};
struct TorP {
    double period, inv_period, inv_dphi, half_inv_dphi, m2_inv_dphi;   // 1/dphi, 1/(2 dphi), -2/dphi
    int P;
};
// per-triangle geometry, 64 B: reference coordinates xi = a11 (R - v0x) + a12 (Z - v0y), eta = a21 (..) + a22 (..)
struct __align__(16) TriGeom {
    double v0x, v0y, a11, a12, a21, a22;
    int nbr[3];   // neighbour across edge 0 (eta = 0), 1 (1 - xi - eta = 0), 2 (xi = 0); -1 = boundary
    int orig;     // caller's triangle index
};
struct BoxGrid {
    double xmin, ymin, inv_dx, inv_dy;
    int nx, ny;
    const int* head;   // [nx*ny + 1]
    const int* list;
};

struct Fields { double P, PR, PZ, Pp, A, AR, AZ, Ap; };   // values, d/dR, d/dZ, raw d/dphi

// ---- reciprocal, reciprocal square root, exp ---------------------------------------------------------
// 1/x and 1/sqrt(x) for normal x (R, q, B, B*_par, r^2 ...): hardware seed (MUFU on the upper 32 bits of x: relative
// error e ~ 2^-20) and ONE third-order correction in FMA form, without the denormal / infinity side path of the library
// routines:  1/x = y0 / (1 - e) = y0 (1 + e + e^2 + O(e^3)),  x^-1/2 = y0 (1 - e)^-1/2 = y0 (1 + e/2 + 3 e^2/8 + O(e^3)),
// truncation <= e^3 ~ 1e-18 relative, below the rounding of the final FMA.
TRIMEG_DI double rcp_nr(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    return fma(y, fma(e, e, e), y);
}
TRIMEG_DI double rsqrt_nr(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x * y, y, 1.0);
    return fma(y * e, fma(e, 0.375, 0.5), y);
}
// exp for the profile terms of Eq.(7)/(8): x = n ln2 + r, |r| <= ln2/2, Taylor polynomial of degree 11 in r (remainder
// <= r^12/12! e^r = 8.8e-15 relative: it enters dw/dt only, whose parity bound is 1e-11 for one evaluation and 1e-10 for the
// weight after 10 steps; measured margin after the change: DESIGN.md section 6), times 2^n built in the exponent field (n
// clamped to +-1000 so that huge arguments saturate to inf / ~0 through an ordinary multiplication instead of wrapping the
// exponent).  The coefficients sit in constant memory so that every DFMA takes its constant as an operand.
__constant__ double c_expk[12] = {1.0, 1.0, 1.0 / 2, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320, 1.0 / 362880,
                                  1.0 / 3628800, 1.0 / 39916800};
__constant__ double c_expr[4] = {1.4426950408889634, 6755399441055744.0, 6.93147180369123816490e-01, 1.90821492927058770002e-10};
TRIMEG_DI double exp_nr(double x) {
    const double t = fma(x, c_expr[0], c_expr[1]);     // round(x / ln2) in the low mantissa bits
    const int n = max(-1000, min(1000, __double2loint(t)));
    const double fn = (double)n;
    double r = fma(-fn, c_expr[2], x);
    r = fma(-fn, c_expr[3], r);
    double p = c_expk[11];
#pragma unroll
    for (int k = 10; k >= 0; --k) p = fma(p, r, c_expk[k]);
    return p * __hiloint2double((n + 1023) << 20, 0);
}

// ---- toroidal uniform periodic cubic B-spline (L35) -------------------------------------------------
// interval index k in [0, P) and fraction s in [0, 1] of phi (any real)
TRIMEG_DI int toroidal_interval(const TorP& tp, double phi, double& s) {
    double pm = fma(-tp.period, floor(phi * tp.inv_period), phi);
    if (pm < 0.0) pm += tp.period;
    if (pm >= tp.period) pm -= tp.period;
    double u = pm * tp.inv_dphi;
    int k = (int)u;
    if (k >= tp.P) k = tp.P - 1;
    s = u - (double)k;
    return k;
}
// w = [(1-s)^3, 3 s^3 - 6 s^2 + 4, 3 t^3 - 6 t^2 + 4, s^3] / 6 with t = 1 - s;  dw = d w / d phi
template <class T>
TRIMEG_DI void bspline_from_s(const TorP& tp, T s, T w[4], T dw[4]) {
    const T t = T(1.0) - s;
    const T s2 = s * s, t2 = t * t;
    const T s2h = s2 * T(tp.half_inv_dphi), t2h = t2 * T(tp.half_inv_dphi);
    w[0] = t2 * t * T(1.0 / 6.0);
    w[3] = s2 * s * T(1.0 / 6.0);
    w[1] = fma(s2, fma(T(0.5), s, T(-1.0)), T(2.0 / 3.0));
    w[2] = fma(t2, fma(T(0.5), t, T(-1.0)), T(2.0 / 3.0));
    dw[0] = -t2h;
    dw[3] = s2h;
    dw[1] = fma(T(3.0), s2h, T(tp.m2_inv_dphi) * s);
    dw[2] = -fma(T(3.0), t2h, T(tp.m2_inv_dphi) * t);
}
// returns the interval k; the four planes are padded-table planes k + PLANE_PAD .. k + PLANE_PAD + 3
TRIMEG_DI int bspline_weights(const TorP& tp, double phi, double w[4], double dw[4]) {
    double s;
    int k = toroidal_interval(tp, phi, s);
    bspline_from_s<double>(tp, s, w, dw);
    return k;
}

// ---- reduced quintic in reference coordinates --------------------------------------------------------
// Coefficients j-major: a_j(xi) = sum_{i<=5-j} c[off_j + i] xi^i, p = sum_j eta^j a_j(xi).
// Two fields interleaved: c[2*idx + f].  38 FMA per field: value, d/dxi, d/deta.
// ld(idx, c0, c1) fetches coefficient idx of field 0 and 1 as doubles.
template <int N, class T, class Ld>
TRIMEG_DI void horner2(Ld ld, int off, T x, T& v0, T& d0, T& v1, T& d1) {
    double c0, c1;
    ld(off + N, c0, c1);
    if (N == 0) { v0 = T(c0); v1 = T(c1); d0 = T(0.0); d1 = T(0.0); return; }
    double e0, e1;
    ld(off + N - 1, e0, e1);
    v0 = fma(T(c0), x, T(e0)); v1 = fma(T(c1), x, T(e1));
    d0 = T(c0); d1 = T(c1);
#pragma unroll
    for (int i = N - 2; i >= 0; --i) {
        ld(off + i, e0, e1);
        d0 = fma(d0, x, v0); d1 = fma(d1, x, v1);
        v0 = fma(v0, x, T(e0)); v1 = fma(v1, x, T(e1));
    }
}

// One plane: acc[0..3] += (w p, w p_xi, w p_eta, dw p) for field 0, acc[4..7] likewise for field 1; the value of field 0
// (acc[0]) only if WITH_P (the right-hand sides never use Phi itself, only its gradient).
// Outer Horner in eta runs j = 5 -> 0 and consumes each a_j(xi), a_j'(xi) as soon as the inner Horner produced it,
// so only the three running sums per field stay live.
template <bool WITH_P, class T, class Ld>
TRIMEG_DI void quintic_pair_accum(Ld ld, T xi, T eta, T w, T dw, T acc[8]) {
    T p0, p1, py0, py1, px0, px1, a0, a1, b0, b1;
    horner2<0>(ld, 20, xi, p0, b0, p1, b1);          // a_5 (constant)
    horner2<1>(ld, 18, xi, a0, px0, a1, px1);        // a_4, a_4'
    py0 = p0; py1 = p1;
    p0 = fma(p0, eta, a0); p1 = fma(p1, eta, a1);
    horner2<2>(ld, 15, xi, a0, b0, a1, b1);
    py0 = fma(py0, eta, p0); py1 = fma(py1, eta, p1); p0 = fma(p0, eta, a0); p1 = fma(p1, eta, a1); px0 = fma(px0, eta, b0); px1 = fma(px1, eta, b1);
    horner2<3>(ld, 11, xi, a0, b0, a1, b1);
    py0 = fma(py0, eta, p0); py1 = fma(py1, eta, p1); p0 = fma(p0, eta, a0); p1 = fma(p1, eta, a1); px0 = fma(px0, eta, b0); px1 = fma(px1, eta, b1);
    horner2<4>(ld, 6, xi, a0, b0, a1, b1);
    py0 = fma(py0, eta, p0); py1 = fma(py1, eta, p1); p0 = fma(p0, eta, a0); p1 = fma(p1, eta, a1); px0 = fma(px0, eta, b0); px1 = fma(px1, eta, b1);
    horner2<5>(ld, 0, xi, a0, b0, a1, b1);
    py0 = fma(py0, eta, p0); py1 = fma(py1, eta, p1); p0 = fma(p0, eta, a0); p1 = fma(p1, eta, a1); px0 = fma(px0, eta, b0); px1 = fma(px1, eta, b1);
    if (WITH_P) acc[0] = fma(w, p0, acc[0]);
    acc[1] = fma(w, px0, acc[1]); acc[2] = fma(w, py0, acc[2]); acc[3] = fma(dw, p0, acc[3]);
    acc[4] = fma(w, p1, acc[4]); acc[5] = fma(w, px1, acc[5]); acc[6] = fma(w, py1, acc[6]); acc[7] = fma(dw, p1, acc[7]);
}

// all four planes; ldp(idx, a, b) fetches pair idx of [4][21] (16-byte aligned pairs); result in reference-gradient form
template <bool WITH_P, class T, class LdPlane>
TRIMEG_DI void gather_cell(LdPlane ldp, T xi, T eta, const T w[4], const T dw[4], T acc[8]) {
#pragma unroll
    for (int q = 0; q < 8; ++q) acc[q] = T(0.0);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        auto ld = [&](int idx, double& a, double& b) { ldp(j * NCOEF + idx, a, b); };
        quintic_pair_accum<WITH_P>(ld, xi, eta, w[j], dw[j], acc);
    }
}
// reference gradient -> physical gradient (grad_phys = J^-T grad_ref)
TRIMEG_DI void to_fields(const TriGeom& g, const double acc[8], Fields& f) {
    f.P = acc[0]; f.PR = fma(g.a11, acc[1], g.a21 * acc[2]); f.PZ = fma(g.a12, acc[1], g.a22 * acc[2]); f.Pp = acc[3];
    f.A = acc[4]; f.AR = fma(g.a11, acc[5], g.a21 * acc[6]); f.AZ = fma(g.a12, acc[5], g.a22 * acc[6]); f.Ap = acc[7];
}

// What the right-hand sides need of the perturbed fields: g = grad(Phi - u A) at fixed u, as (d_R, raw d_phi, d_Z), and A
// itself.  From the gathered reference-frame sums acc[] (quintic_pair_accum) and the triangle's J^-1 = (a11 a12; a21 a22):
// the combination with u is done on the two reference components before the 2x2 transform (7 FMA instead of 11).
template <class T>
struct FieldsG { T gR, gZ, gp, A; };
template <class T>
TRIMEG_DI void to_fields_g(T a11, T a12, T a21, T a22, const T acc[8], T u, FieldsG<T>& f) {
    const T gx = fma(-u, acc[5], acc[1]), gy = fma(-u, acc[6], acc[2]);
    f.gR = fma(a11, gx, a21 * gy);
    f.gZ = fma(a12, gx, a22 * gy);
    f.gp = fma(-u, acc[7], acc[3]);
    f.A = acc[4];
}
TRIMEG_DI void fields_to_g(const Fields& f, double u, FieldsG<double>& g) {
    g.gR = fma(-u, f.AR, f.PR); g.gZ = fma(-u, f.AZ, f.PZ); g.gp = fma(-u, f.Ap, f.Pp); g.A = f.A;
}

// ---- locate -------------------------------------------------------------------------------------------
TRIMEG_DI void ref_coords(const TriGeom& g, double R, double Z, double& xi, double& eta) {
    double dx = R - g.v0x, dy = Z - g.v0y;
    xi = fma(g.a11, dx, g.a12 * dy);
    eta = fma(g.a21, dx, g.a22 * dy);
}
// box-grid lookup (triangle <-> bounding-box map on an nx x ny intermediate grid, flattened
// to head offsets + one list).  Picks the candidate with the largest minimum barycentric; -1 if none is inside.
__device__ inline int locate_box(const BoxGrid& bg, const TriGeom* __restrict__ geom, double R, double Z) {
    int i = (int)floor((R - bg.xmin) * bg.inv_dx), j = (int)floor((Z - bg.ymin) * bg.inv_dy);
    if (i == bg.nx) i = bg.nx - 1;
    if (j == bg.ny) j = bg.ny - 1;
    if (i == -1) i = 0;
    if (j == -1) j = 0;
    if (i < 0 || j < 0 || i >= bg.nx || j >= bg.ny) return -1;
    int b = j * bg.nx + i, best = -1;
    double bestmin = INSIDE_TOL;
    for (int q = bg.head[b]; q < bg.head[b + 1]; ++q) {
        int t = bg.list[q];
        double xi, eta;
        ref_coords(geom[t], R, Z, xi, eta);
        double m = fmin(fmin(xi, eta), 1.0 - xi - eta);
        if (m >= 0.0) return t;     // inside: no other candidate can beat it by more than an edge tie
        if (m >= bestmin) { bestmin = m; best = t; }
    }
    return best;
}
// edge walk from a starting triangle; falls back to the box lookup at a boundary edge or after MAXHOP steps.
// never reports "outside" from the walk alone.
__device__ inline int locate_walk(const BoxGrid& bg, const TriGeom* __restrict__ geom, int start, double R, double Z) {
    constexpr int MAXHOP = 24;
    int t = start;
    if (t >= 0) {
        for (int hop = 0; hop < MAXHOP; ++hop) {
            const TriGeom& g = geom[t];
            double xi, eta;
            ref_coords(g, R, Z, xi, eta);
            double l0 = 1.0 - xi - eta;
            double m = fmin(fmin(xi, eta), l0);
            if (m >= INSIDE_TOL) return t;
            int e = (eta <= xi && eta <= l0) ? 0 : ((l0 <= xi) ? 1 : 2);
            int nb = g.nbr[e];
            if (nb < 0) break;
            t = nb;
        }
    }
    return locate_box(bg, geom, R, Z);
}

// ---- equilibrium (L89) + Eq.(2)-(7) ----------------------------------------------------------------------
// Analytic concentric-circular tokamak, psi'(r) = B0 r / qbar(r) (trimeg.h).  With P = psi', H = sqrt(P^2 + F^2):
//   B = H / R,  b = (-P s, F, P c) / H  in (R, phi, Z)  (c, s = cos, sin of the poloidal angle),
//   grad B = (H' c / R - B / R, 0, H' s / R),  H' = P P' / H,
//   curl B = J e_phi,  J = [P c / R - (P' + P / r)] / R,
//   curl b = (curl B + b x grad B) / B  =>  b . curl b = b_phi J / B.
// (The oracle differentiates the components of b directly; this route is independent of it.)
template <class T>
struct Equil {
    T B, iB, iR, bR, bp, bZ, gBR, gBZ, J, r, c, s;
};
// Numeric equilibrium: B = grad psi x grad phi + F grad phi from the spline's first and second derivatives of psi, through
// the same identities as the analytic one (H = sqrt(|grad psi|^2 + F^2), B = H / R, b = (-psi_Z, F, psi_R) / H,
// grad B = grad H / R - B e_R / R, (curl B)_phi = (psi_R / R - laplace psi) / R).  The oracle differentiates b instead.
TRIMEG_DI void equil_eval_numeric(const EquilP& e, double R, double Z, Equil<double>& o) {
    const double uR = (R - e.Rmin) * e.inv_hR, uZ = (Z - e.Zmin) * e.inv_hZ;
    const int i = max(0, min(e.nR - 1, (int)floor(uR))), j = max(0, min(e.nZ - 1, (int)floor(uZ)));
    double wa[4], da[4], ca[4], wb[4], db[4], cb[4];
    auto pieces = [](double s, double* w, double* d1, double* d2) {
        const double t = 1.0 - s, s2 = s * s, t2 = t * t;
        w[0] = t2 * t * (1.0 / 6.0); w[3] = s2 * s * (1.0 / 6.0);
        w[1] = fma(s2, fma(0.5, s, -1.0), 2.0 / 3.0); w[2] = fma(t2, fma(0.5, t, -1.0), 2.0 / 3.0);
        d1[0] = -0.5 * t2; d1[3] = 0.5 * s2; d1[1] = fma(1.5, s2, -2.0 * s); d1[2] = -fma(1.5, t2, -2.0 * t);
        d2[0] = t; d2[1] = fma(3.0, s, -2.0); d2[2] = fma(3.0, t, -2.0); d2[3] = s;
    };
    pieces(uR - (double)i, wa, da, ca);
    pieces(uZ - (double)j, wb, db, cb);
    double pR = 0, pZ = 0, pRR = 0, pRZ = 0, pZZ = 0;
    const double* base = e.psi + (long long)i * (e.nZ + 3) + j;
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        double v = 0, vz = 0, vzz = 0;     // sums over the Z direction for row a
#pragma unroll
        for (int b = 0; b < 4; ++b) { const double c = __ldg(base + (long long)a * (e.nZ + 3) + b); v = fma(c, wb[b], v); vz = fma(c, db[b], vz); vzz = fma(c, cb[b], vzz); }
        pR = fma(da[a], v, pR); pRR = fma(ca[a], v, pRR); pZ = fma(wa[a], vz, pZ); pRZ = fma(da[a], vz, pRZ); pZZ = fma(wa[a], vzz, pZZ);
    }
    pR *= e.inv_hR; pZ *= e.inv_hZ; pRR *= e.inv_hR * e.inv_hR; pRZ *= e.inv_hR * e.inv_hZ; pZZ *= e.inv_hZ * e.inv_hZ;
    const double H2 = fma(pR, pR, fma(pZ, pZ, e.F2)), iH = rsqrt_nr(H2), H = H2 * iH, iR = rcp_nr(R);
    const double B = H * iR;
    o.B = B; o.iB = R * iH; o.iR = iR;
    o.bR = -(pZ * iH); o.bZ = pR * iH; o.bp = e.F * iH;
    const double HR = fma(pR, pRR, pZ * pRZ) * iH, HZ = fma(pR, pRZ, pZ * pZZ) * iH;
    o.gBR = fma(HR, iR, -(B * iR)); o.gBZ = HZ * iR;
    o.J = fma(pR, iR, -(pRR + pZZ)) * iR;
    const double x = R - e.R0, r2 = fma(x, x, Z * Z), ir = rsqrt_nr(r2);
    o.r = r2 * ir; o.c = x * ir; o.s = Z * ir;
}
// NUM: whether this instantiation may meet a numeric equilibrium (the tiled phase kernel never does: the library runs
// variant 1 then, so its hot loop carries no branch and no extra code for it)
template <class T, bool NUM = false>
TRIMEG_DI void equil_eval(const EquilP& e, T R, T Z, Equil<T>& o) {
    if (NUM && e.kind) { equil_eval_numeric(e, R, Z, o); return; }
    const T x = R - T(e.R0);
    const T r2 = fma(x, x, Z * Z);
    const T ir = rsqrt_nr(r2), r = r2 * ir;
    const T c = x * ir, s = Z * ir;
    const T xa = r * T(e.inv_a);
    const T q = fma(xa, fma(T(e.q2), xa, T(e.q1)), T(e.q0));
    const T dq = fma(T(2.0 * e.q2), xa, T(e.q1)) * T(e.inv_a);
    T qb = q, dqb = dq;
    if (e.qbar_sqrt) {   // qbar = q sqrt(1 - r^2/R0^2)
        const T s2 = fma(-r2, T(e.inv_R0sq), T(1.0));
        const T is = rsqrt_nr(s2), sq = s2 * is;
        qb = q * sq;
        dqb = fma(dq, sq, -(q * r) * (T(e.inv_R0sq) * is));
    }
    const T iqb = rcp_nr(qb);
    const T P = T(e.B0) * r * iqb;                   // psi'
    const T P1 = fma(-P, dqb, T(e.B0)) * iqb;        // psi''
    const T iH = rsqrt_nr(fma(P, P, T(e.F2)));
    const T iR = rcp_nr(R);
    const T H = fma(P, P, T(e.F2)) * iH;
    const T B = H * iR;
    const T bt = P * iH;                             // poloidal component of b
    const T t = (P * P1) * (iH * iR);                // H' / R
    o.B = B; o.iB = R * iH; o.iR = iR;
    o.bR = -(bt * s); o.bZ = bt * c; o.bp = T(e.F) * iH;
    o.gBR = fma(t, c, -(B * iR)); o.gBZ = t * s;
    o.J = fma(P * c, iR, -fma(P, ir, P1)) * iR;
    o.r = r; o.c = c; o.s = s;
}

// time derivatives of (R, Z, phi, u, w) at one phase-space point (gyro-average off, L320; dA^s = 0: p_par form).
//   B*_par = B + kappa u b.curl b  (L61),  S = beta b + kappa u curl b with beta = B (b* = B*/B*_par, reading R7) or
//   beta = B*_par (the literal expression printed at L53), so that in both cases b* = S / B*_par and every product with
//   b* is formed with S and scaled by 1/B*_par once at the end.
// The part of a right-hand-side evaluation that depends on the position only (not on the gathered fields): equilibrium
// and the Eq.(8) profile terms.  Kept separate so that a kernel can issue these long dependent chains (rsqrt, rcp, two
// exponentials) BEFORE the gather and let them overlap with the gather's loads and Horner chains.
template <class T>
struct RhsPre {
    Equil<T> e;
    T dlnT, dlnn, iT;     // d ln T / dr, d ln n / dr, 1 / T(r)
};
template <class T, bool NUM = false>
TRIMEG_DI void rhs_pre(const EquilP& ep, const SpeciesP& sp, T R, T Z, RhsPre<T>& o) {
    equil_eval<T, NUM>(ep, R, Z, o.e);
    const T dr = o.e.r - T(sp.r0);
    const T thT = fma(T(-2.0), rcp_nr(exp_nr(dr * T(sp.two_inv_wT_a)) + T(1.0)), T(1.0));
    T thn = thT;
    if (!sp.same_w) thn = fma(T(-2.0), rcp_nr(exp_nr(dr * T(sp.two_inv_wn_a)) + T(1.0)), T(1.0));   // a real (uniform) branch: as a select the second exponential was always computed
    o.dlnT = T(-sp.kT_R0) * fma(-thT, thT, T(1.0));
    o.dlnn = T(-sp.kn_R0) * fma(-thn, thn, T(1.0));
    o.iT = exp_nr(T(sp.cT) * thT);                                                 // 1/T(r), Eq.(8)
}
// time derivatives of (R, Z, phi, u, w) at one phase-space point (gyro-average off, L320; dA^s = 0: p_par form).
//   B*_par = B + kappa u b.curl b  (L61),  S = beta b + kappa u curl b with beta = B (b* = B*/B*_par, reading R7) or
//   beta = B*_par (the literal expression printed at L53), so that in both cases b* = S / B*_par and every product with
//   b* is formed with S and scaled by 1/B*_par once at the end.
template <class T>
TRIMEG_DI void rhs_post(const SpeciesP& sp, const RhsPre<T>& pre, T u, T w, T mu, T p, const FieldsG<T>& f, T d[5]) {
    const Equil<T>& e = pre.e;
    const T ku = T(sp.kappa) * u, km = T(sp.kappa) * mu;
    const T kub = ku * e.iB;
    const T Bss = fma(kub * e.bp, e.J, e.B);                                       // L61
    const T iBss = rcp_nr(Bss);
    const T beta = sp.bstar_exact ? e.B : Bss;
    // B curl b = (b_phi gB_Z, J + b_Z gB_R - b_R gB_Z, -b_phi gB_R)
    const T SR = fma(kub, e.bp * e.gBZ, beta * e.bR);
    const T Sp = fma(kub, fma(e.bZ, e.gBR, fma(-e.bR, e.gBZ, e.J)), beta * e.bp);
    const T SZ = fma(-kub, e.bp * e.gBR, beta * e.bZ);
    // g = grad(Phi - u A), grad = (d_R, (1/R) d_phi, d_Z)
    const T gR = f.gR, gZ = f.gZ, gp = f.gp * e.iR;
    const T GR = fma(km, e.gBR, gR), GZ = fma(km, e.gBZ, gZ);                      // G = kappa mu grad B + g
    // b x G, right-handed (R, phi, Z)
    const T cR = fma(e.bp, GZ, -(e.bZ * gp)), cp = fma(e.bZ, GR, -(e.bR * GZ)), cZ = fma(e.bR, gp, -(e.bp * GR));
    const T vpar = fma(T(-sp.qom), f.A, u);
    d[0] = fma(vpar, SR, cR) * iBss;                                               // Eq.(2)+(4)
    d[1] = fma(vpar, SZ, cZ) * iBss;
    d[2] = fma(vpar, Sp, cp) * (iBss * e.iR);
    const T qgR = T(sp.qom) * gR, qgp = T(sp.qom) * gp, qgZ = T(sp.qom) * gZ;
    const T Sqg = fma(SR, qgR, fma(Sp, qgp, SZ * qgZ));                            // qom S.g
    d[3] = -(fma(mu, fma(SR, e.gBR, SZ * e.gBZ), Sqg) * iBss);                     // Eq.(3)+(5)
    // Eq.(7): delta-parts of the motion against grad ln f0, f0 Maxwellian with Eq.(8) profiles
    const T hR = fma(e.bp, gZ, -(e.bZ * gp)), hZ = fma(e.bR, gp, -(e.bp * gR));    // (b x g)_R, (b x g)_Z
    const T qA = T(sp.qom) * f.A;
    const T eR = fma(-qA, SR, hR), eZ = fma(-qA, SZ, hZ);                          // Bss * delta Xdot
    const T En = fma(T(0.5) * u, u, mu * e.B);
    const T cr = fma(pre.dlnT, fma(En, pre.iT, T(-1.5)), pre.dlnn);
    const T muT = mu * pre.iT;
    const T glR = fma(cr, e.c, -(muT * e.gBR)), glZ = fma(cr, e.s, -(muT * e.gBZ));
    const T pw = sp.weight_mode ? (p - w) : p;
    d[4] = -((pw * iBss) * fma(eR, glR, fma(eZ, glZ, Sqg * (u * pre.iT))));
}
template <class T, bool NUM = false>
TRIMEG_DI void rhs_eval(const EquilP& ep, const SpeciesP& sp, T R, T Z, T u, T w, T mu, T p, const FieldsG<T>& f, T d[5]) {
    RhsPre<T> pre;
    rhs_pre<T, NUM>(ep, sp, R, Z, pre);
    rhs_post(sp, pre, u, w, mu, p, f, d);
}

// 256-bit global accesses (sm_100: LDG/STG.256): a 32-byte record is one request and one full sector
TRIMEG_DI void ld256(const void* p, double& a, double& b, double& c, double& d) {
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
TRIMEG_DI void st256(void* p, double a, double b, double c, double d) {
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

}  // namespace trimeg
