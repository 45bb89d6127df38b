// Device arithmetic of the marker push: toroidal B-spline weights, reduced-quintic evaluation,
// analytic equilibrium, guiding-centre and weight right-hand sides.  fp64 throughout.
// Passages: /root/reference/PAPER.md L35 (C1 element x cubic B-spline), Eq.(2)-(6) L45-55, B*_par L61,
// Eq.(7), Eq.(8) L314.  Formulation notes (what differs from a literal transcription) are in DESIGN.md
// "Kernel arithmetic": reciprocals are shared, sqrt/div go through rsqrt/rcp + FMA, curl b comes from the
// identity curl b = (curl B + b x grad B)/B, everything else is written in FMA form.
#pragma once
#include <cstdint>

namespace trimeg {

constexpr int NCOEF = 21;                 // quintic monomials xi^i eta^j, i + j <= 5
constexpr int PLANE_STRIDE = NCOEF * 2;   // doubles per (triangle, plane): [21][field]
constexpr int PLANE_PAD = 1;              // extra toroidal planes on each side of the padded coefficient table
// padded table: plane index pp in [0, P + 3 + 2 PLANE_PAD) holds toroidal plane (pp - 1 - PLANE_PAD) mod P, so the four planes
// k-1..k+2 of interval k are pp = k + PLANE_PAD .. k + PLANE_PAD + 3, contiguous for every k (no wrap in the kernels)
constexpr double INSIDE_TOL = -1e-12;

struct EquilP {
    double R0, B0, F, inv_a, inv_R0sq, q0, q1, q2;
    int qbar_sqrt;
};
struct SpeciesP {
    double qom, kappa;                 // q/m and m/q
    double kn_R0, kT_R0;               // kappa_n / R0, kappa_T / R0   (d ln H/dr = -(kappa_H/R0) sech^2)
    double inv_wn_a, inv_wT_a, r0;     // 1/(w_n a), 1/(w_T a)
    double cT;                         // kappa_T w_T a / R0 : T = exp(-cT tanh)
    int same_w, bstar_exact, weight_mode;
};
struct TorP {
    double period, inv_period, inv_dphi, half_inv_dphi;   // 1/dphi, 1/(2 dphi)
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

// 1/x and 1/sqrt(x) for normal positive-or-negative x (R, q, B, B*_par, r^2 ...): hardware seed (MUFU, ~2^-20) and two
// Newton steps in FMA form, without the denormal / infinity side path of the library routines (a branch and a call each).
__device__ __forceinline__ double rcp_nr(double x) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}
__device__ __forceinline__ double rsqrt_nr(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double hx = 0.5 * x;
    double e = fma(-hx * y, y, 0.5);      // (1 - x y^2) / 2
    y = fma(y, e, y);
    e = fma(-hx * y, y, 0.5);
    return fma(y, e, y);
}

// exp and tanh for the profile terms of Eq.(7)/(8) (arguments of order one).  exp: x = n ln2 + r, |r| <= ln2/2, Taylor
// polynomial of degree 13 in r (truncation 0.347^14/14! = 4e-18), 2^n through the exponent field; the coefficients sit in
// constant memory so that every DFMA takes its constant as an operand (the library routines materialise theirs with two
// UMOV each: 110 of the phase kernel's 2 970 instructions per chunk).  tanh x = 1 - 2/(e^{2x} + 1): absolute error ~1e-16,
// which is what sech^2 = 1 - tanh^2 and T = exp(-c tanh) need.
__constant__ double c_expk[14] = {1.0, 1.0, 1.0 / 2, 1.0 / 6, 1.0 / 24, 1.0 / 120, 1.0 / 720, 1.0 / 5040, 1.0 / 40320, 1.0 / 362880,
                                  1.0 / 3628800, 1.0 / 39916800, 1.0 / 479001600, 1.0 / 6227020800.0};
__constant__ double c_expr[4] = {1.4426950408889634, 6755399441055744.0, 6.93147180369123816490e-01, 1.90821492927058770002e-10};
__device__ __forceinline__ double exp_nr(double x) {
    const double t = fma(x, c_expr[0], c_expr[1]);     // round(x / ln2) in the low mantissa bits
    const int n = __double2loint(t);
    const double fn = t - c_expr[1];
    double r = fma(-fn, c_expr[2], x);
    r = fma(-fn, c_expr[3], r);
    double p = c_expk[13];
#pragma unroll
    for (int k = 12; k >= 0; --k) p = fma(p, r, c_expk[k]);
    return __hiloint2double(__double2hiint(p) + n * 1048576, __double2loint(p));
}
__device__ __forceinline__ double tanh_nr(double x) {
    const double E = exp_nr(x + x);
    return fma(-2.0, rcp_nr(E + 1.0), 1.0);
}

// ---- toroidal uniform periodic cubic B-spline (L35) -------------------------------------------------
// interval index k in [0, P) and fraction s in [0, 1] of phi (any real)
__device__ __forceinline__ int toroidal_interval(const TorP& tp, double phi, double& s) {
    double pm = fma(-tp.period, floor(phi * tp.inv_period), phi);
    if (pm < 0.0) pm += tp.period;
    if (pm >= tp.period) pm -= tp.period;
    double u = pm * tp.inv_dphi;
    int k = (int)u;
    if (k >= tp.P) k = tp.P - 1;
    s = u - (double)k;
    return k;
}
__device__ __forceinline__ void bspline_from_s(const TorP& tp, double s, double w[4], double dw[4]) {
    double t = 1.0 - s;
    const double sixth = 1.0 / 6.0;
    double s2 = s * s, t2 = t * t;
    w[0] = t2 * t * sixth;
    w[3] = s2 * s * sixth;
    w[1] = fma(s2, fma(3.0, s, -6.0), 4.0) * sixth;
    w[2] = fma(t2, fma(3.0, t, -6.0), 4.0) * sixth;
    dw[0] = -t2 * tp.half_inv_dphi;
    dw[3] = s2 * tp.half_inv_dphi;
    dw[1] = s * fma(3.0, s, -4.0) * tp.half_inv_dphi;
    dw[2] = -t * fma(3.0, t, -4.0) * tp.half_inv_dphi;
}
// returns the interval k; the four planes are padded-table planes k + PLANE_PAD .. k + PLANE_PAD + 3
__device__ __forceinline__ int bspline_weights(const TorP& tp, double phi, double w[4], double dw[4]) {
    double s;
    int k = toroidal_interval(tp, phi, s);
    bspline_from_s(tp, s, w, dw);
    return k;
}

// ---- reduced quintic in reference coordinates --------------------------------------------------------
// Coefficients j-major: a_j(xi) = sum_{i<=5-j} c[off_j + i] xi^i, p = sum_j eta^j a_j(xi).
// Two fields interleaved: c[2*idx + f].  38 FMA per field: value, d/dxi, d/deta.
template <int N, typename Ld>
__device__ __forceinline__ void horner2(Ld ld, int off, double x, double& v0, double& d0, double& v1, double& d1) {
    // both fields in lock-step; ld(idx, a, b) fetches coefficient idx of field 0 and 1
    double c0, c1;
    ld(off + N, c0, c1);
    if (N == 0) { v0 = c0; v1 = c1; d0 = 0.0; d1 = 0.0; return; }
    double e0, e1;
    ld(off + N - 1, e0, e1);
    v0 = fma(c0, x, e0); v1 = fma(c1, x, e1);
    d0 = c0; d1 = c1;
#pragma unroll
    for (int i = N - 2; i >= 0; --i) {
        ld(off + i, e0, e1);
        d0 = fma(d0, x, v0); d1 = fma(d1, x, v1);
        v0 = fma(v0, x, e0); v1 = fma(v1, x, e1);
    }
}

// acc[0..3] += (w p, w p_xi, w p_eta, dw p) for field 0, acc[4..7] likewise for field 1.
// Outer Horner in eta runs j = 5 -> 0 and consumes each a_j(xi), a_j'(xi) as soon as the inner Horner produced it,
// so only the three running sums per field stay live.
template <typename Ld>
__device__ __forceinline__ void quintic_pair_accum(Ld ld, double xi, double eta, double w, double dw, double acc[8]) {
    double p0, p1, py0, py1, px0, px1, a0, a1, b0, b1;
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
    acc[0] = fma(w, p0, acc[0]); acc[1] = fma(w, px0, acc[1]); acc[2] = fma(w, py0, acc[2]); acc[3] = fma(dw, p0, acc[3]);
    acc[4] = fma(w, p1, acc[4]); acc[5] = fma(w, px1, acc[5]); acc[6] = fma(w, py1, acc[6]); acc[7] = fma(dw, p1, acc[7]);
}

// two planes at once: four independent Horner chains (2 planes x 2 fields) for instruction-level parallelism
template <int N, typename LdA, typename LdB>
__device__ __forceinline__ void horner4(LdA lda, LdB ldb, int off, double x, double v[4], double d[4]) {
    double c[4], e[4];
    lda(off + N, c[0], c[1]); ldb(off + N, c[2], c[3]);
    if (N == 0) {
#pragma unroll
        for (int q = 0; q < 4; ++q) { v[q] = c[q]; d[q] = 0.0; }
        return;
    }
    lda(off + N - 1, e[0], e[1]); ldb(off + N - 1, e[2], e[3]);
#pragma unroll
    for (int q = 0; q < 4; ++q) { v[q] = fma(c[q], x, e[q]); d[q] = c[q]; }
#pragma unroll
    for (int i = N - 2; i >= 0; --i) {
        lda(off + i, e[0], e[1]); ldb(off + i, e[2], e[3]);
#pragma unroll
        for (int q = 0; q < 4; ++q) { d[q] = fma(d[q], x, v[q]); v[q] = fma(v[q], x, e[q]); }
    }
}
template <typename LdA, typename LdB>
__device__ __forceinline__ void quintic_quad_accum(LdA lda, LdB ldb, double xi, double eta, double wa, double dwa, double wb, double dwb, double acc[8]) {
    double p[4], py[4], px[4], a[4], b[4];
    horner4<0>(lda, ldb, 20, xi, p, b);
    horner4<1>(lda, ldb, 18, xi, a, px);
#pragma unroll
    for (int q = 0; q < 4; ++q) { py[q] = p[q]; p[q] = fma(p[q], eta, a[q]); }
    horner4<2>(lda, ldb, 15, xi, a, b);
#pragma unroll
    for (int q = 0; q < 4; ++q) { py[q] = fma(py[q], eta, p[q]); p[q] = fma(p[q], eta, a[q]); px[q] = fma(px[q], eta, b[q]); }
    horner4<3>(lda, ldb, 11, xi, a, b);
#pragma unroll
    for (int q = 0; q < 4; ++q) { py[q] = fma(py[q], eta, p[q]); p[q] = fma(p[q], eta, a[q]); px[q] = fma(px[q], eta, b[q]); }
    horner4<4>(lda, ldb, 6, xi, a, b);
#pragma unroll
    for (int q = 0; q < 4; ++q) { py[q] = fma(py[q], eta, p[q]); p[q] = fma(p[q], eta, a[q]); px[q] = fma(px[q], eta, b[q]); }
    horner4<5>(lda, ldb, 0, xi, a, b);
#pragma unroll
    for (int q = 0; q < 4; ++q) { py[q] = fma(py[q], eta, p[q]); p[q] = fma(p[q], eta, a[q]); px[q] = fma(px[q], eta, b[q]); }
    // q = 0,1: plane A fields 0,1 ; q = 2,3: plane B fields 0,1
    acc[0] = fma(wa, p[0], acc[0]); acc[1] = fma(wa, px[0], acc[1]); acc[2] = fma(wa, py[0], acc[2]); acc[3] = fma(dwa, p[0], acc[3]);
    acc[4] = fma(wa, p[1], acc[4]); acc[5] = fma(wa, px[1], acc[5]); acc[6] = fma(wa, py[1], acc[6]); acc[7] = fma(dwa, p[1], acc[7]);
    acc[0] = fma(wb, p[2], acc[0]); acc[1] = fma(wb, px[2], acc[1]); acc[2] = fma(wb, py[2], acc[2]); acc[3] = fma(dwb, p[2], acc[3]);
    acc[4] = fma(wb, p[3], acc[4]); acc[5] = fma(wb, px[3], acc[5]); acc[6] = fma(wb, py[3], acc[6]); acc[7] = fma(dwb, p[3], acc[7]);
}

// all four planes; ldp(idx, a, b) fetches pair idx of [4][21] (16-byte aligned pairs); result in reference-gradient form
template <typename LdPlane>
__device__ __forceinline__ void gather_cell(LdPlane ldp, double xi, double eta, const double w[4], const double dw[4], double acc[8]) {
#pragma unroll
    for (int q = 0; q < 8; ++q) acc[q] = 0.0;
#ifdef TRIMEG_GATHER_PAIRWISE
#pragma unroll
    for (int j = 0; j < 4; j += 2) {
        auto lda = [&](int idx, double& a, double& b) { ldp(j * NCOEF + idx, a, b); };
        auto ldb = [&](int idx, double& a, double& b) { ldp((j + 1) * NCOEF + idx, a, b); };
        quintic_quad_accum(lda, ldb, xi, eta, w[j], dw[j], w[j + 1], dw[j + 1], acc);
    }
#else
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        auto ld = [&](int idx, double& a, double& b) { ldp(j * NCOEF + idx, a, b); };
        quintic_pair_accum(ld, xi, eta, w[j], dw[j], acc);
    }
#endif
}
// reference gradient -> physical gradient (grad_phys = J^-T grad_ref)
__device__ __forceinline__ void to_fields(const TriGeom& g, const double acc[8], Fields& f) {
    f.P = acc[0]; f.PR = fma(g.a11, acc[1], g.a21 * acc[2]); f.PZ = fma(g.a12, acc[1], g.a22 * acc[2]); f.Pp = acc[3];
    f.A = acc[4]; f.AR = fma(g.a11, acc[5], g.a21 * acc[6]); f.AZ = fma(g.a12, acc[5], g.a22 * acc[6]); f.Ap = acc[7];
}

// ---- locate -------------------------------------------------------------------------------------------
__device__ __forceinline__ void ref_coords(const TriGeom& g, double R, double Z, double& xi, double& eta) {
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
struct Equil {
    double B, invB, bR, bp, bZ, gBR, gBZ, cbR, cbp, cbZ, r, cth, sth;
};
__device__ __forceinline__ void equil_eval(const EquilP& e, double R, double Z, Equil& o) {
    double x = R - e.R0;
    double r2 = fma(x, x, Z * Z);
    double inv_r = rsqrt_nr(r2), r = r2 * inv_r;
    double xa = r * e.inv_a;
    double q = fma(xa, fma(e.q2, xa, e.q1), e.q0);
    double dq = fma(2.0 * e.q2, xa, e.q1) * e.inv_a;
    double qb = q, dqb = dq;
    if (e.qbar_sqrt) {
        double s2 = fma(-r2, e.inv_R0sq, 1.0);
        double inv_s = rsqrt_nr(s2), s = s2 * inv_s;
        double ds = -r * e.inv_R0sq * inv_s;
        qb = q * s;
        dqb = fma(dq, s, q * ds);
    }
    double inv_qb = rcp_nr(qb);
    double p1 = e.B0 * r * inv_qb;                 // psi'
    double p2 = fma(-p1, dqb, e.B0) * inv_qb;      // psi''
    double c = x * inv_r, s_ = Z * inv_r;
    double p1r = p1 * inv_r, D = p2 - p1r;
    double pR = p1 * c, pZ = p1 * s_;
    double pRR = fma(D * c, c, p1r), pRZ = D * c * s_, pZZ = fma(D * s_, s_, p1r);
    double iR = rcp_nr(R);
    double BR = -pZ * iR, BZ = pR * iR, Bp = e.F * iR;
    double BR_R = -(pRZ + BR) * iR, BR_Z = -pZZ * iR;
    double BZ_R = (pRR - BZ) * iR, BZ_Z = pRZ * iR;
    double Bp_R = -Bp * iR;
    double B2 = fma(BR, BR, fma(BZ, BZ, Bp * Bp));
    double iB = rsqrt_nr(B2), B = B2 * iB;
    double gR = fma(BR, BR_R, fma(BZ, BZ_R, Bp * Bp_R)) * iB;
    double gZ = fma(BR, BR_Z, BZ * BZ_Z) * iB;
    double bR = BR * iB, bZ = BZ * iB, bp = Bp * iB;
    double cBp = BR_Z - BZ_R;
    o.B = B; o.invB = iB; o.bR = bR; o.bp = bp; o.bZ = bZ; o.gBR = gR; o.gBZ = gZ;
    o.cbR = bp * gZ * iB;
    o.cbp = (cBp + fma(bZ, gR, -bR * gZ)) * iB;
    o.cbZ = -bp * gR * iB;
    o.r = r; o.cth = c; o.sth = s_;
}

// time derivatives of (R, Z, phi, u, w) at one phase-space point (gyro-average off, L320; dA^s = 0: p_par form)
__device__ __forceinline__ void rhs_eval(const EquilP& ep, const SpeciesP& sp, double R, double Z, double u, double w,
                                         double mu, double p, const Fields& f, double d[5]) {
    Equil e;
    equil_eval(ep, R, Z, e);
    double iR = rcp_nr(R);
    double ku = sp.kappa * u;
    double Bss = fma(ku, fma(e.bR, e.cbR, fma(e.bp, e.cbp, e.bZ * e.cbZ)), e.B);   // L61
    double iBss = rcp_nr(Bss);
    double bsR, bsp, bsZ;
    if (sp.bstar_exact) {
        bsR = fma(ku, e.cbR, e.B * e.bR) * iBss; bsp = fma(ku, e.cbp, e.B * e.bp) * iBss; bsZ = fma(ku, e.cbZ, e.B * e.bZ) * iBss;
    } else {
        double k2 = ku * iBss;
        bsR = fma(k2, e.cbR, e.bR); bsp = fma(k2, e.cbp, e.bp); bsZ = fma(k2, e.cbZ, e.bZ);
    }
    // g = grad(Phi - u A), grad = (d_R, (1/R) d_phi, d_Z)
    double gR = fma(-u, f.AR, f.PR), gp = fma(-u, f.Ap, f.Pp) * iR, gZ = fma(-u, f.AZ, f.PZ);
    double km = sp.kappa * mu;
    double GR = fma(km, e.gBR, gR), Gp = gp, GZ = fma(km, e.gBZ, gZ);
    // b x G, right-handed (R, phi, Z)
    double cR = fma(e.bp, GZ, -e.bZ * Gp), cp = fma(e.bZ, GR, -e.bR * GZ), cZ = fma(e.bR, Gp, -e.bp * GR);
    double vpar = fma(-sp.qom, f.A, u);
    double XR = fma(vpar, bsR, cR * iBss), Xp = fma(vpar, bsp, cp * iBss), XZ = fma(vpar, bsZ, cZ * iBss);   // Eq.(2)+(4)
    double bs_g = fma(bsR, gR, fma(bsp, gp, bsZ * gZ));
    double bs_gB = fma(bsR, e.gBR, bsZ * e.gBZ);
    d[0] = XR; d[1] = XZ; d[2] = Xp * iR;
    d[3] = -fma(mu, bs_gB, sp.qom * bs_g);                                                                  // Eq.(3)+(5)
    // Eq.(7): delta-parts of the motion against grad ln f0, f0 Maxwellian with Eq.(8) profiles
    double hR = fma(e.bp, gZ, -e.bZ * gp), hZ = fma(e.bR, gp, -e.bp * gR);    // (b x g)_R, (b x g)_Z
    double qA = sp.qom * f.A;
    double dXR = fma(hR, iBss, -qA * bsR), dXZ = fma(hZ, iBss, -qA * bsZ);
    double ddu = -sp.qom * bs_g;
    double dr = e.r - sp.r0;
    double thT = tanh_nr(dr * sp.inv_wT_a);
    double thn = sp.same_w ? thT : tanh_nr(dr * sp.inv_wn_a);
    double dlnT = -sp.kT_R0 * fma(-thT, thT, 1.0), dlnn = -sp.kn_R0 * fma(-thn, thn, 1.0);
    double iT = exp_nr(sp.cT * thT);                          // 1/T(r), Eq.(8)
    double En = fma(0.5 * u, u, mu * e.B);
    double cr = fma(dlnT, fma(En, iT, -1.5), dlnn);
    double muT = mu * iT;
    double glR = fma(cr, e.cth, -muT * e.gBR), glZ = fma(cr, e.sth, -muT * e.gBZ);
    double pw = sp.weight_mode ? (p - w) : p;
    d[4] = -pw * fma(dXR, glR, fma(dXZ, glZ, -ddu * u * iT));
}

}  // namespace trimeg
