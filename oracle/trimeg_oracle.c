/*
 * oracle/trimeg_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, double-precision CPU statement of the TRIMEG-C1 marker push
 * (arxiv/paper_2606_24327, /root/reference/PAPER.md; "L<n>" below are PAPER.md
 * lines).  It exists so that the CUDA path has something independent to be
 * compared with.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or constant generator with paper_2606_24327_b200/csrc/.
 *
 * What it computes (the paper's order, DESIGN.md "Readings" R1..R15 where the
 * paper is silent):
 *   O1  C1 element (L15, L35 "C1 continuous finite element basis functions
 *       [10]"; reading R1: Bell reduced quintic, 18 DOF): per triangle a
 *       21x21 system, pivoted LU in long double, one solve per
 *       (triangle, plane, field).
 *   O2  toroidal uniform periodic cubic B-spline (L35).
 *   O3  field at a point = tensor product of O1 and O2 (L35 "interpolated at
 *       each particle position").
 *   O4  locate: triangle <-> bounding-box map on an nx x ny intermediate grid,
 *       flattened to head offsets + one list (L89, L125-140); brute force over
 *       all triangles is kept beside it.
 *   O5  analytic concentric-circular equilibrium (L89 "computes the
 *       equilibrium configuration of the magnetic field"; parameters from
 *       BASELINE.json configs).
 *   O6  guiding-centre equations Eq.(2)-(6), L45-55, B*_par L61, in the
 *       p_par (Hamiltonian) form dA^s = 0 (reading R6).
 *   O7  delta-f weight equation Eq.(7) L65 with Maxwellian f0 and the
 *       Eq.(8) profiles L314.
 *   O8  classical RK4 with frozen fields (north_star; the paper never names
 *       its integrator, L89).
 *   O9  a marker evaluated outside the mesh feels zero perturbed field and
 *       gets a sticky status bit.
 *   O10 the three other grid-to-particle kernels of L97-103 ("pullback
 *       treatment", "density calculation", "distribution-function
 *       interpolation": one sentence each in the paper, "all these kernels rely
 *       on the same G2P function"; readings R22-R24 of DESIGN.md):
 *       pullback = the linearised mixed-variable -> symplectic map of Eq.(1),
 *       (6) with dA^h = A_par:  u <- u - (q/m) A_par,  w <- w + p (q/m) A_par
 *       d ln f0/du (at the old u);  density = the value of one grid field at
 *       every marker;  f-interpolation = f0 (Maxwellian, Eq.(8) profiles, up to
 *       its constant factor) at the marker's position and physical parallel
 *       velocity v_par = u - (q/m) A_par.
 *
 *   O11 particle-to-grid deposition onto the C1 x B-spline basis (L35 "projecting
 *       the quantities stored at the particle locations ... onto the finite
 *       element grid"; L288, L372: what the paper left on the CPU): the
 *       transpose of O3.  b[k][v][c] = sum_p q_p N_{v,c}(R_p, Z_p) B_k(phi_p)
 *       with N_{v,c} the element's nodal basis functions (the interpolant of the
 *       unit DOF vector) and B_k the toroidal spline (reading R25).
 *   O12 N-point gyro-average of the gather (the <...> of Eq.(4)-(6), L49-55; "switched
 *       off" in the paper's runs, L320): the mean of O3 over N points on the gyro-ring
 *       of radius rho in the poloidal plane around the gyrocentre (reading R26).
 *   O13 numeric equilibrium (L87 "equilibrium variables are represented using B-splines", L121, L142-146: the
 *       paper's B-spline library): psi(R, Z) as a tensor-product uniform cubic B-spline on a rectangle, F = R B_phi
 *       constant; B = grad psi x grad phi + F grad phi and everything O5 derives from it (reading R27).
 *
 * Parity unpinned (choices the paper does not fix and nothing external can
 * check): the element family itself (R1), the unit system (R8), linear vs
 * nonlinear weight equation (R13), the domain-exit rule (R15), and WHICH maps the
 * paper's three "other kernels" are (R22-R24: the paper names them in one
 * sentence each; the maps chosen here are pinned as maps, P17-P19).  Everything
 * else is pinned by tests/test_oracle_*.py.
 *
 * Arithmetic: IEEE double everywhere except the element LU and the 21-term polynomial sums
 * (long double, results rounded to double; coefficients are stored as double).
 * No blocking, no fusion, no reordering beyond the formulas as written.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NM 21 /* monomials x^i y^j, i+j<=5 */

typedef struct {
    /* O5 */ double R0, a, B0, q0, q1, q2; int qbar_sqrt, have_eq;
    /* O13 */ int eq_numeric, gnR, gnZ; double gRmin, gRmax, gZmin, gZmax, gF; double *gcoef;
    /* O6/O7 */ double qom, kappa_n, kappa_T, w_n, w_T, r0; int bstar_exact, weight_mode, have_sp;
    /* mesh */ int64_t n_nodes, n_tri; double *RZ; int32_t *tri; int P; double period;
    /* O1 */ long double *LU; int *piv; double *org; double *hh;
    /* O4 */ int nx, ny; double xmin, ymin, dx, dy; int64_t *head; int32_t *list;
    /* fields: coef[which][(t*P+plane)*21 + m] */ double *coef[2];
} orc;

static int mono_i[NM], mono_j[NM], mono_ready = 0;
static void mono_init(void) {
    int k = 0;
    for (int d = 0; d <= 5; d++) for (int i = d; i >= 0; i--) { mono_i[k] = i; mono_j[k] = d - i; k++; }
    mono_ready = 1;
}
static long double ipowl(long double x, int n) { long double r = 1; for (int t = 0; t < n; t++) r *= x; return r; }
/* d^(dx+dy)/dx^dx dy^dy of x^i y^j */
static long double dmono_l(int i, int j, int dx, int dy, long double x, long double y) {
    if (i < dx || j < dy) return 0;
    long double c = 1;
    for (int t = 0; t < dx; t++) c *= (i - t);
    for (int t = 0; t < dy; t++) c *= (j - t);
    return c * ipowl(x, i - dx) * ipowl(y, j - dy);
}

orc *orc_create(void) { if (!mono_ready) mono_init(); return (orc *)calloc(1, sizeof(orc)); }
void orc_destroy(orc *c) {
    if (!c) return;
    free(c->gcoef); free(c->RZ); free(c->tri); free(c->LU); free(c->piv); free(c->org); free(c->hh);
    free(c->head); free(c->list); free(c->coef[0]); free(c->coef[1]); free(c);
}
int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int orc_equilibrium_set(orc *c, double R0, double a, double B0, double q0, double q1, double q2, int qbar_sqrt) {
    c->R0 = R0; c->a = a; c->B0 = B0; c->q0 = q0; c->q1 = q1; c->q2 = q2; c->qbar_sqrt = qbar_sqrt; c->have_eq = 1; c->eq_numeric = 0;
    return 0;
}
/* O13: coef[(nR+3)][(nZ+3)] of psi on [Rmin,Rmax] x [Zmin,Zmax] with nR x nZ intervals, F = R B_phi; R0, a: axis and minor
 * radius for the Eq.(8) profiles (their radial coordinate stays r = |(R - R0, Z)|) */
int orc_equilibrium_set_numeric(orc *c, int nR, int nZ, double Rmin, double Rmax, double Zmin, double Zmax, double F, double R0, double a, const double *coef) {
    if (!c || nR < 1 || nZ < 1 || !(Rmax > Rmin) || !(Zmax > Zmin) || !coef) return -1;
    free(c->gcoef);
    size_t n = (size_t)(nR + 3) * (nZ + 3);
    c->gcoef = (double *)malloc(sizeof(double) * n); memcpy(c->gcoef, coef, sizeof(double) * n);
    c->gnR = nR; c->gnZ = nZ; c->gRmin = Rmin; c->gRmax = Rmax; c->gZmin = Zmin; c->gZmax = Zmax; c->gF = F;
    c->R0 = R0; c->a = a; c->eq_numeric = 1; c->have_eq = 1;
    return 0;
}
int orc_species_set(orc *c, double qom, double kn, double kT, double wn, double wT, double r0, int bstar_exact, int weight_mode) {
    c->qom = qom; c->kappa_n = kn; c->kappa_T = kT; c->w_n = wn; c->w_T = wT; c->r0 = r0;
    c->bstar_exact = bstar_exact; c->weight_mode = weight_mode; c->have_sp = 1;
    return 0;
}

/* ---------------------------------------------------------------- O1 ---- */
/* Build the 21x21 element matrix of triangle t in local coordinates
 * x = (R - org_R)/h, y = (Z - org_Z)/h (org = centroid, h = longest edge):
 * rows 0..17: (p, p_x, p_y, p_xx, p_xy, p_yy) at vertex 0,1,2;
 * rows 18..20: for edge e (vertex e -> e+1), tangent t, normal n=(t_y,-t_x):
 *   the s^4 coefficient of d_n p along the edge, (n . grad p5)(t) = 0,
 *   p5 = degree-5 homogeneous part (normal derivative cubic on each edge => C1). */
static void element_matrix(const orc *c, int64_t t, long double *M, double *org, double *h) {
    const int32_t *tv = c->tri + 3 * t;
    double V[3][2];
    for (int v = 0; v < 3; v++) { V[v][0] = c->RZ[2 * tv[v]]; V[v][1] = c->RZ[2 * tv[v] + 1]; }
    org[0] = (V[0][0] + V[1][0] + V[2][0]) / 3.0; org[1] = (V[0][1] + V[1][1] + V[2][1]) / 3.0;
    double hm = 0;
    for (int e = 0; e < 3; e++) { double ex = V[(e + 1) % 3][0] - V[e][0], ey = V[(e + 1) % 3][1] - V[e][1]; double l = sqrt(ex * ex + ey * ey); if (l > hm) hm = l; }
    *h = hm;
    long double L[3][2];
    for (int v = 0; v < 3; v++) { L[v][0] = ((long double)V[v][0] - org[0]) / hm; L[v][1] = ((long double)V[v][1] - org[1]) / hm; }
    static const int D6[6][2] = {{0, 0}, {1, 0}, {0, 1}, {2, 0}, {1, 1}, {0, 2}};
    memset(M, 0, sizeof(long double) * NM * NM);
    int r = 0;
    for (int v = 0; v < 3; v++) for (int d = 0; d < 6; d++) {
        for (int k = 0; k < NM; k++) M[r * NM + k] = dmono_l(mono_i[k], mono_j[k], D6[d][0], D6[d][1], L[v][0], L[v][1]);
        r++;
    }
    for (int e = 0; e < 3; e++) {
        long double tx = L[(e + 1) % 3][0] - L[e][0], ty = L[(e + 1) % 3][1] - L[e][1], nx = ty, ny = -tx;
        for (int k = 0; k < NM; k++) {
            int i = mono_i[k], j = mono_j[k];
            if (i + j != 5) continue;
            long double gx = i > 0 ? i * ipowl(tx, i - 1) * ipowl(ty, j) : 0;
            long double gy = j > 0 ? j * ipowl(tx, i) * ipowl(ty, j - 1) : 0;
            M[r * NM + k] = nx * gx + ny * gy;
        }
        r++;
    }
}
/* in-place LU with partial pivoting (rows scaled to unit max first); returns -1 if singular */
static int lu_factor(long double *A, int *piv) {
    for (int i = 0; i < NM; i++) piv[i] = i;
    for (int k = 0; k < NM; k++) {
        int p = k; long double best = fabsl(A[k * NM + k]);
        for (int i = k + 1; i < NM; i++) if (fabsl(A[i * NM + k]) > best) { best = fabsl(A[i * NM + k]); p = i; }
        if (best == 0) return -1;
        if (p != k) { for (int j = 0; j < NM; j++) { long double tmp = A[k * NM + j]; A[k * NM + j] = A[p * NM + j]; A[p * NM + j] = tmp; } int tp = piv[k]; piv[k] = piv[p]; piv[p] = tp; }
        for (int i = k + 1; i < NM; i++) {
            long double f = A[i * NM + k] / A[k * NM + k]; A[i * NM + k] = f;
            for (int j = k + 1; j < NM; j++) A[i * NM + j] -= f * A[k * NM + j];
        }
    }
    return 0;
}
static void lu_solve(const long double *A, const int *piv, const long double *b, long double *x) {
    long double y[NM];
    for (int i = 0; i < NM; i++) { long double s = b[piv[i]]; for (int j = 0; j < i; j++) s -= A[i * NM + j] * y[j]; y[i] = s; }
    for (int i = NM - 1; i >= 0; i--) { long double s = y[i]; for (int j = i + 1; j < NM; j++) s -= A[i * NM + j] * x[j]; x[i] = s / A[i * NM + i]; }
}
/* row equilibration happens through the h-scaling of the DOFs; rows 18-20 are O(1) by construction */

static int build_boxes(orc *c);

int orc_mesh_load(orc *c, int64_t n_nodes, const double *RZ, int64_t n_tri, const int32_t *tri, int32_t n_planes, double period) {
    if (!c || !RZ || !tri || n_nodes < 3 || n_tri < 1 || n_planes < 4 || !(period > 0)) return -1;
    free(c->RZ); free(c->tri); free(c->LU); free(c->piv); free(c->org); free(c->hh); free(c->head); free(c->list);
    free(c->coef[0]); free(c->coef[1]); c->coef[0] = c->coef[1] = NULL;
    c->n_nodes = n_nodes; c->n_tri = n_tri; c->P = n_planes; c->period = period;
    c->RZ = (double *)malloc(sizeof(double) * 2 * n_nodes); memcpy(c->RZ, RZ, sizeof(double) * 2 * n_nodes);
    c->tri = (int32_t *)malloc(sizeof(int32_t) * 3 * n_tri); memcpy(c->tri, tri, sizeof(int32_t) * 3 * n_tri);
    for (int64_t t = 0; t < n_tri; t++) {
        const int32_t *tv = tri + 3 * t;
        for (int v = 0; v < 3; v++) if (tv[v] < 0 || tv[v] >= n_nodes) return -3;
        double ax = RZ[2 * tv[1]] - RZ[2 * tv[0]], ay = RZ[2 * tv[1] + 1] - RZ[2 * tv[0] + 1];
        double bx = RZ[2 * tv[2]] - RZ[2 * tv[0]], by = RZ[2 * tv[2] + 1] - RZ[2 * tv[0] + 1];
        if (!(ax * by - ay * bx > 0)) return -3; /* not counter-clockwise / degenerate */
    }
    c->LU = (long double *)malloc(sizeof(long double) * NM * NM * n_tri);
    c->piv = (int *)malloc(sizeof(int) * NM * n_tri);
    c->org = (double *)malloc(sizeof(double) * 2 * n_tri);
    c->hh = (double *)malloc(sizeof(double) * n_tri);
    int bad = 0;
#pragma omp parallel for schedule(static)
    for (int64_t t = 0; t < n_tri; t++) {
        element_matrix(c, t, c->LU + t * NM * NM, c->org + 2 * t, c->hh + t);
        if (lu_factor(c->LU + t * NM * NM, c->piv + t * NM)) bad = 1;
    }
    if (bad) return -3;
    return build_boxes(c);
}

/* DOFs -> 21 monomial coefficients of one triangle, one plane.
 * dof18 = for vertex 0,1,2: (f, f_R, f_Z, f_RR, f_RZ, f_ZZ), physical derivatives (reading R2). */
static void element_solve(const orc *c, int64_t t, const double *dof18, double *coef21) {
    static const int ord[6] = {0, 1, 1, 2, 2, 2};
    long double b[NM], x[NM]; long double h = c->hh[t];
    for (int v = 0; v < 3; v++) for (int d = 0; d < 6; d++) b[6 * v + d] = (long double)dof18[6 * v + d] * ipowl(h, ord[d]);
    b[18] = b[19] = b[20] = 0;
    lu_solve(c->LU + t * NM * NM, c->piv + t * NM, b, x);
    for (int k = 0; k < NM; k++) coef21[k] = (double)x[k];
}
int orc_element_coeffs(orc *c, int64_t t, const double *dof18, double *coef21) {
    if (!c || !c->LU || t < 0 || t >= c->n_tri) return -1;
    element_solve(c, t, dof18, coef21); return 0;
}
/* value, d/dR, d/dZ, d2/dR2, d2/dRdZ, d2/dZ2 of the local polynomial of triangle t at (R,Z) */
static void poly_eval(const orc *c, int64_t t, const double *coef21, double R, double Z, double *out6) {
    /* the 21-term sums are accumulated in long double: in the isotropic local frame a thin triangle can
     * carry coefficients many orders above the value they sum to, and the oracle must not be the
     * less accurate side of a 1e-12 comparison */
    long double h = c->hh[t], x = ((long double)R - c->org[2 * t]) / h, y = ((long double)Z - c->org[2 * t + 1]) / h;
    long double p = 0, px = 0, py = 0, pxx = 0, pxy = 0, pyy = 0;
    for (int k = 0; k < NM; k++) {
        int i = mono_i[k], j = mono_j[k]; long double ck = coef21[k];
        p += ck * ipowl(x, i) * ipowl(y, j);
        if (i >= 1) px += ck * i * ipowl(x, i - 1) * ipowl(y, j);
        if (j >= 1) py += ck * j * ipowl(x, i) * ipowl(y, j - 1);
        if (i >= 2) pxx += ck * i * (i - 1) * ipowl(x, i - 2) * ipowl(y, j);
        if (i >= 1 && j >= 1) pxy += ck * i * j * ipowl(x, i - 1) * ipowl(y, j - 1);
        if (j >= 2) pyy += ck * j * (j - 1) * ipowl(x, i) * ipowl(y, j - 2);
    }
    out6[0] = (double)p; out6[1] = (double)(px / h); out6[2] = (double)(py / h);
    out6[3] = (double)(pxx / (h * h)); out6[4] = (double)(pxy / (h * h)); out6[5] = (double)(pyy / (h * h));
}
int orc_poly_eval(orc *c, int64_t t, const double *coef21, double R, double Z, double *out6) {
    if (!c || !c->LU || t < 0 || t >= c->n_tri) return -1;
    poly_eval(c, t, coef21, R, Z, out6); return 0;
}

int orc_fields_set(orc *c, int which, const double *dof /* [P][n_nodes][6] */) {
    if (!c || !c->LU || which < 0 || which > 1 || !dof) return -1;
    free(c->coef[which]);
    c->coef[which] = (double *)malloc(sizeof(double) * NM * (size_t)c->n_tri * c->P);
    if (!c->coef[which]) return -5;
#pragma omp parallel for schedule(static)
    for (int64_t t = 0; t < c->n_tri; t++) for (int k = 0; k < c->P; k++) {
        double d18[18];
        for (int v = 0; v < 3; v++) memcpy(d18 + 6 * v, dof + ((size_t)k * c->n_nodes + c->tri[3 * t + v]) * 6, sizeof(double) * 6);
        element_solve(c, t, d18, c->coef[which] + ((size_t)t * c->P + k) * NM);
    }
    return 0;
}

/* ---------------------------------------------------------------- O4 ---- */
static void barycentric(const orc *c, int64_t t, double R, double Z, double *lam) {
    const int32_t *tv = c->tri + 3 * t;
    double x0 = c->RZ[2 * tv[0]], y0 = c->RZ[2 * tv[0] + 1], x1 = c->RZ[2 * tv[1]], y1 = c->RZ[2 * tv[1] + 1], x2 = c->RZ[2 * tv[2]], y2 = c->RZ[2 * tv[2] + 1];
    double A2 = (x1 - x0) * (y2 - y0) - (y1 - y0) * (x2 - x0);
    lam[0] = ((x1 - R) * (y2 - Z) - (y1 - Z) * (x2 - R)) / A2;
    lam[1] = ((x2 - R) * (y0 - Z) - (y2 - Z) * (x0 - R)) / A2;
    lam[2] = ((x0 - R) * (y1 - Z) - (y0 - Z) * (x1 - R)) / A2;
}
#define INSIDE_TOL (-1e-12)
static int build_boxes(orc *c) {
    double xmin = 1e300, xmax = -1e300, ymin = 1e300, ymax = -1e300;
    for (int64_t n = 0; n < c->n_nodes; n++) { double x = c->RZ[2 * n], y = c->RZ[2 * n + 1]; if (x < xmin) xmin = x; if (x > xmax) xmax = x; if (y < ymin) ymin = y; if (y > ymax) ymax = y; }
    double wx = xmax - xmin, wy = ymax - ymin;
    int nx = (int)ceil(sqrt((double)c->n_tri * wx / wy)), ny = (int)ceil(sqrt((double)c->n_tri * wy / wx));
    if (nx < 1) nx = 1; if (ny < 1) ny = 1;
    c->nx = nx; c->ny = ny; c->xmin = xmin; c->ymin = ymin; c->dx = wx / nx; c->dy = wy / ny;
    int64_t nb = (int64_t)nx * ny;
    c->head = (int64_t *)calloc(nb + 1, sizeof(int64_t));
    for (int pass = 0; pass < 2; pass++) {
        int64_t *fill = pass ? (int64_t *)calloc(nb, sizeof(int64_t)) : NULL;
        for (int64_t t = 0; t < c->n_tri; t++) {
            const int32_t *tv = c->tri + 3 * t; double bx0 = 1e300, bx1 = -1e300, by0 = 1e300, by1 = -1e300;
            for (int v = 0; v < 3; v++) { double x = c->RZ[2 * tv[v]], y = c->RZ[2 * tv[v] + 1]; if (x < bx0) bx0 = x; if (x > bx1) bx1 = x; if (y < by0) by0 = y; if (y > by1) by1 = y; }
            int i0 = (int)floor((bx0 - xmin) / c->dx) - 1, i1 = (int)floor((bx1 - xmin) / c->dx) + 1, j0 = (int)floor((by0 - ymin) / c->dy) - 1, j1 = (int)floor((by1 - ymin) / c->dy) + 1;
            if (i0 < 0) i0 = 0; if (j0 < 0) j0 = 0; if (i1 > nx - 1) i1 = nx - 1; if (j1 > ny - 1) j1 = ny - 1;
            for (int i = i0; i <= i1; i++) for (int j = j0; j <= j1; j++) {
                int64_t b = (int64_t)j * nx + i;
                if (!pass) c->head[b + 1]++; else c->list[c->head[b] + fill[b]++] = (int32_t)t;
            }
        }
        if (!pass) { for (int64_t b = 0; b < nb; b++) c->head[b + 1] += c->head[b]; c->list = (int32_t *)malloc(sizeof(int32_t) * (c->head[nb] > 0 ? c->head[nb] : 1)); }
        else free(fill);
    }
    return 0;
}
static int64_t locate_one(const orc *c, double R, double Z, int brute) {
    int64_t best = -1; double bestmin = INSIDE_TOL;
    if (brute) {
        for (int64_t t = 0; t < c->n_tri; t++) { double l[3]; barycentric(c, t, R, Z, l); double m = fmin(l[0], fmin(l[1], l[2])); if (m >= bestmin) { bestmin = m; best = t; } }
        return best;
    }
    int i = (int)floor((R - c->xmin) / c->dx), j = (int)floor((Z - c->ymin) / c->dy);
    if (i == c->nx && R <= c->xmin + c->nx * c->dx + 1e-12) i = c->nx - 1;
    if (j == c->ny && Z <= c->ymin + c->ny * c->dy + 1e-12) j = c->ny - 1;
    if (i == -1) i = 0; if (j == -1) j = 0;
    if (i < 0 || j < 0 || i >= c->nx || j >= c->ny) return -1;
    int64_t b = (int64_t)j * c->nx + i;
    for (int64_t q = c->head[b]; q < c->head[b + 1]; q++) { int64_t t = c->list[q]; double l[3]; barycentric(c, t, R, Z, l); double m = fmin(l[0], fmin(l[1], l[2])); if (m >= bestmin) { bestmin = m; best = t; } }
    return best;
}
int orc_locate(orc *c, int64_t n, const double *R, const double *Z, int32_t *tri_out, int brute) {
    if (!c || !c->head) return -1;
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < n; m++) tri_out[m] = (int32_t)locate_one(c, R[m], Z[m], brute);
    return 0;
}

/* ---------------------------------------------------------------- O2 ---- */
/* uniform periodic cubic B-spline: planes k-1..k+2 (mod P), weights w, d/dphi weights dw */
static void bspline(const orc *c, double phi, int *kout, double *w, double *dw) {
    double dphi = c->period / c->P;
    double pm = fmod(phi, c->period); if (pm < 0) pm += c->period;
    double u = pm / dphi; int k = (int)floor(u); double s = u - k;
    if (k >= c->P) { k -= c->P; }
    *kout = k;
    w[0] = (1 - s) * (1 - s) * (1 - s) / 6; w[1] = (3 * s * s * s - 6 * s * s + 4) / 6; w[2] = (-3 * s * s * s + 3 * s * s + 3 * s + 1) / 6; w[3] = s * s * s / 6;
    dw[0] = -(1 - s) * (1 - s) / (2 * dphi); dw[1] = (3 * s * s - 4 * s) / (2 * dphi); dw[2] = (-3 * s * s + 2 * s + 1) / (2 * dphi); dw[3] = s * s / (2 * dphi);
}
int orc_bspline(orc *c, double phi, int *k, double *w4, double *dw4) { if (!c || c->P < 4) return -1; bspline(c, phi, k, w4, dw4); return 0; }

/* ---------------------------------------------------------------- O3 ---- */
/* out4 = F, dF/dR, dF/dZ, dF/dphi (raw) of field `which` at (R,Z,phi) inside triangle t */
static void field_at(const orc *c, int which, int64_t t, double R, double Z, double phi, double *out4) {
    out4[0] = out4[1] = out4[2] = out4[3] = 0;
    if (!c->coef[which] || t < 0) return;
    int k; double w[4], dw[4]; bspline(c, phi, &k, w, dw);
    for (int j = 0; j < 4; j++) {
        int pl = ((k - 1 + j) % c->P + c->P) % c->P; double v[6];
        poly_eval(c, t, c->coef[which] + ((size_t)t * c->P + pl) * NM, R, Z, v);
        out4[0] += w[j] * v[0]; out4[1] += w[j] * v[1]; out4[2] += w[j] * v[2]; out4[3] += dw[j] * v[0];
    }
}
int orc_gather(orc *c, int64_t n, const double *R, const double *Z, const double *phi, double *out /*[8][n]*/, int32_t *tri_out, int brute) {
    if (!c || !c->head) return -1;
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < n; m++) {
        int64_t t = locate_one(c, R[m], Z[m], brute); double f[4];
        for (int which = 0; which < 2; which++) { field_at(c, which, t, R[m], Z[m], phi[m], f); for (int q = 0; q < 4; q++) out[(size_t)(4 * which + q) * n + m] = f[q]; }
        if (tri_out) tri_out[m] = (int32_t)t;
    }
    return 0;
}

/* ---------------------------------------------------------------- O5 ---- */
typedef struct { double r, q, qbar, psi1, psi2; double B[3]; /* R,phi,Z */ double Bmag; double b[3]; double gradB[3]; double curlb[3]; double F; } equil;
/* uniform cubic B-spline pieces on one interval, fraction s in [0,1]: values, first and second derivatives w.r.t. s */
static void cubic_pieces(double s, double *w, double *d1, double *d2) {
    double t = 1 - s;
    w[0] = t * t * t / 6; w[1] = (3 * s * s * s - 6 * s * s + 4) / 6; w[2] = (-3 * s * s * s + 3 * s * s + 3 * s + 1) / 6; w[3] = s * s * s / 6;
    d1[0] = -t * t / 2; d1[1] = (3 * s * s - 4 * s) / 2; d1[2] = (-3 * s * s + 2 * s + 1) / 2; d1[3] = s * s / 2;
    d2[0] = t; d2[1] = 3 * s - 2; d2[2] = -3 * s + 1; d2[3] = s;
}
/* psi_R, psi_Z, psi_RR, psi_RZ, psi_ZZ of the tensor-product spline  psi = sum_ab coef[i+a][j+b] B_a(s) B_b(t)  */
static void psi_spline(const orc *c, double R, double Z, double *p5) {
    double hR = (c->gRmax - c->gRmin) / c->gnR, hZ = (c->gZmax - c->gZmin) / c->gnZ;
    double uR = (R - c->gRmin) / hR, uZ = (Z - c->gZmin) / hZ;
    int i = (int)floor(uR), j = (int)floor(uZ);
    if (i < 0) i = 0; if (i > c->gnR - 1) i = c->gnR - 1;
    if (j < 0) j = 0; if (j > c->gnZ - 1) j = c->gnZ - 1;
    double wa[4], da[4], dda[4], wb[4], db[4], ddb[4];
    cubic_pieces(uR - i, wa, da, dda); cubic_pieces(uZ - j, wb, db, ddb);
    for (int q = 0; q < 5; q++) p5[q] = 0;
    for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) {
        double cf = c->gcoef[(size_t)(i + a) * (c->gnZ + 3) + (j + b)];
        p5[0] += cf * da[a] * wb[b] / hR; p5[1] += cf * wa[a] * db[b] / hZ;
        p5[2] += cf * dda[a] * wb[b] / (hR * hR); p5[3] += cf * da[a] * db[b] / (hR * hZ); p5[4] += cf * wa[a] * ddb[b] / (hZ * hZ);
    }
}
static void equil_eval(const orc *c, double R, double Z, equil *e) {
    if (c->eq_numeric) {   /* O13: the same derivation as below from the spline's derivatives of psi */
        double x = R - c->R0, r = sqrt(x * x + Z * Z), p5[5];
        psi_spline(c, R, Z, p5);
        double pR = p5[0], pZ = p5[1], pRR = p5[2], pRZ = p5[3], pZZ = p5[4], F = c->gF;
        double BR = -pZ / R, BZ = pR / R, Bp = F / R;
        double BR_R = -pRZ / R + pZ / (R * R), BR_Z = -pZZ / R, BZ_R = pRR / R - pR / (R * R), BZ_Z = pRZ / R, Bp_R = -F / (R * R), Bp_Z = 0;
        double B = sqrt(BR * BR + BZ * BZ + Bp * Bp);
        double B_R = (BR * BR_R + BZ * BZ_R + Bp * Bp_R) / B, B_Z = (BR * BR_Z + BZ * BZ_Z + Bp * Bp_Z) / B;
        double bR = BR / B, bp = Bp / B, bZ = BZ / B;
        double bR_Z = BR_Z / B - BR * B_Z / (B * B), bZ_R = BZ_R / B - BZ * B_R / (B * B);
        double bp_R = Bp_R / B - Bp * B_R / (B * B), bp_Z = Bp_Z / B - Bp * B_Z / (B * B);
        (void)BZ_Z;
        e->r = r; e->q = 0; e->qbar = 0; e->psi1 = 0; e->psi2 = 0; e->F = F;
        e->B[0] = BR; e->B[1] = Bp; e->B[2] = BZ; e->Bmag = B; e->b[0] = bR; e->b[1] = bp; e->b[2] = bZ;
        e->gradB[0] = B_R; e->gradB[1] = 0; e->gradB[2] = B_Z;
        e->curlb[0] = -bp_Z; e->curlb[1] = bR_Z - bZ_R; e->curlb[2] = bp_R + bp / R;
        return;
    }
    double x = R - c->R0, r = sqrt(x * x + Z * Z), xa = r / c->a;
    double q = c->q0 + c->q1 * xa + c->q2 * xa * xa, dq = (c->q1 + 2 * c->q2 * xa) / c->a;
    double s = 1, ds = 0;
    if (c->qbar_sqrt) { s = sqrt(1 - (r / c->R0) * (r / c->R0)); ds = -(r / (c->R0 * c->R0)) / s; }
    double qb = q * s, dqb = dq * s + q * ds;
    double p1 = c->B0 * r / qb, p2 = (c->B0 - p1 * dqb) / qb; /* psi', psi'' */
    double F = c->B0 * c->R0;
    /* derivatives of psi(r(R,Z)) */
    double rR = x / r, rZ = Z / r, rRR = Z * Z / (r * r * r), rRZ = -x * Z / (r * r * r), rZZ = x * x / (r * r * r);
    double pR = p1 * rR, pZ = p1 * rZ, pRR = p2 * rR * rR + p1 * rRR, pRZ = p2 * rR * rZ + p1 * rRZ, pZZ = p2 * rZ * rZ + p1 * rZZ;
    double BR = -pZ / R, BZ = pR / R, Bp = F / R;
    double BR_R = -pRZ / R + pZ / (R * R), BR_Z = -pZZ / R, BZ_R = pRR / R - pR / (R * R), BZ_Z = pRZ / R, Bp_R = -F / (R * R), Bp_Z = 0;
    double B = sqrt(BR * BR + BZ * BZ + Bp * Bp);
    double B_R = (BR * BR_R + BZ * BZ_R + Bp * Bp_R) / B, B_Z = (BR * BR_Z + BZ * BZ_Z + Bp * Bp_Z) / B;
    /* unit vector and its derivatives, component by component */
    double bR = BR / B, bp = Bp / B, bZ = BZ / B;
    double bR_R = BR_R / B - BR * B_R / (B * B), bR_Z = BR_Z / B - BR * B_Z / (B * B);
    double bZ_R = BZ_R / B - BZ * B_R / (B * B);
    double bp_R = Bp_R / B - Bp * B_R / (B * B), bp_Z = Bp_Z / B - Bp * B_Z / (B * B);
    e->r = r; e->q = q; e->qbar = qb; e->psi1 = p1; e->psi2 = p2; e->F = F;
    e->B[0] = BR; e->B[1] = Bp; e->B[2] = BZ; e->Bmag = B; e->b[0] = bR; e->b[1] = bp; e->b[2] = bZ;
    e->gradB[0] = B_R; e->gradB[1] = 0; e->gradB[2] = B_Z;
    /* axisymmetric curl in right-handed (R,phi,Z):
     * (curl b)_R = -d_Z b_phi ; (curl b)_phi = d_Z b_R - d_R b_Z ; (curl b)_Z = (1/R) d_R (R b_phi) */
    e->curlb[0] = -bp_Z; e->curlb[1] = bR_Z - bZ_R; e->curlb[2] = bp_R + bp / R;
}
/* out: r,q,qbar,psi',psi'', B_R,B_phi,B_Z, |B|, b(3), gradB(3), curlb(3), F  = 19 doubles */
int orc_equil_eval(orc *c, double R, double Z, double *out19) {
    if (!c || !c->have_eq) return -2;
    equil e; equil_eval(c, R, Z, &e);
    out19[0] = e.r; out19[1] = e.q; out19[2] = e.qbar; out19[3] = e.psi1; out19[4] = e.psi2;
    for (int i = 0; i < 3; i++) { out19[5 + i] = e.B[i]; out19[9 + i] = e.b[i]; out19[12 + i] = e.gradB[i]; out19[15 + i] = e.curlb[i]; }
    out19[8] = e.Bmag; out19[18] = e.F; return 0;
}

/* ------------------------------------------------------------ O6, O7 ---- */
static void cross3(const double *a, const double *c, double *o) { /* right-handed (R,phi,Z) */
    o[0] = a[1] * c[2] - a[2] * c[1]; o[1] = a[2] * c[0] - a[0] * c[2]; o[2] = a[0] * c[1] - a[1] * c[0];
}
static double dot3(const double *a, const double *c) { return a[0] * c[0] + a[1] * c[1] + a[2] * c[2]; }
/* Eq.(8): H(r)/H(r0) = exp[-kappa w (a/R0) tanh((r-r0)/(w a))]; returns H/H(r0) and d ln H/dr */
static double profile(const orc *c, double kappa, double w, double r, double *dlnH) {
    double arg = (r - c->r0) / (w * c->a), th = tanh(arg);
    *dlnH = -(kappa / c->R0) * (1 - th * th);
    return exp(-kappa * w * (c->a / c->R0) * th);
}
/* ln f0 up to a constant: f0 = n/(2 pi T)^{3/2} exp(-(u^2/2 + mu B)/T), L63 "f0 is chosen as the Maxwellian" */
static double ln_f0(const orc *c, double R, double Z, double u, double mu) {
    equil e; equil_eval(c, R, Z, &e); double d; double n = profile(c, c->kappa_n, c->w_n, e.r, &d), T = profile(c, c->kappa_T, c->w_T, e.r, &d);
    return log(n) - 1.5 * log(T) - (0.5 * u * u + mu * e.Bmag) / T;
}
double orc_ln_f0(orc *c, double R, double Z, double u, double mu) { return ln_f0(c, R, Z, u, mu); }
static void grad_ln_f0(const orc *c, const equil *e, double R, double Z, double u, double mu, double *g3 /*R,phi,Z*/, double *du) {
    double dn, dT; (void)profile(c, c->kappa_n, c->w_n, e->r, &dn); double T = profile(c, c->kappa_T, c->w_T, e->r, &dT);
    double E = 0.5 * u * u + mu * e->Bmag; double cr = dn + dT * (E / T - 1.5);
    double x = R - c->R0;
    g3[0] = cr * x / e->r - (mu / T) * e->gradB[0]; g3[1] = 0; g3[2] = cr * Z / e->r - (mu / T) * e->gradB[2];
    *du = -u / T;
}
int orc_grad_ln_f0(orc *c, double R, double Z, double u, double mu, double *out3 /* d_R, d_Z, d_u */) {
    equil e; equil_eval(c, R, Z, &e); double g[3], du; grad_ln_f0(c, &e, R, Z, u, mu, g, &du); out3[0] = g[0]; out3[1] = g[2]; out3[2] = du; return 0;
}
/* time derivatives of (R, Z, phi, u, w); returns 1 if the point is outside the mesh (O9) */
static int rhs_one(const orc *c, double R, double Z, double phi, double u, double w, double mu, double p, double *d5, int brute) {
    equil e; equil_eval(c, R, Z, &e);
    int64_t t = locate_one(c, R, Z, brute);
    double fP[4], fA[4]; field_at(c, 0, t, R, Z, phi, fP); field_at(c, 1, t, R, Z, phi, fA);
    double Phi = fP[0], A = fA[0];
    double gP[3] = {fP[1], fP[3] / R, fP[2]}, gA[3] = {fA[1], fA[3] / R, fA[2]}; /* grad = (d_R, (1/R) d_phi, d_Z) */
    double kap = 1.0 / c->qom;
    double Bss = e.Bmag + kap * u * dot3(e.b, e.curlb);                       /* L61 */
    double bs[3];
    for (int i = 0; i < 3; i++) bs[i] = c->bstar_exact ? (e.Bmag * e.b[i] + kap * u * e.curlb[i]) / Bss : e.b[i] + kap * u * e.curlb[i] / Bss; /* R7 / literal L53 */
    double g[3], G[3], bxG[3], bxg[3];
    for (int i = 0; i < 3; i++) { g[i] = gP[i] - u * gA[i]; G[i] = kap * mu * e.gradB[i] + g[i]; }
    cross3(e.b, G, bxG); cross3(e.b, g, bxg);
    double X[3];
    for (int i = 0; i < 3; i++) X[i] = (u - c->qom * A) * bs[i] + bxG[i] / Bss;  /* Eq.(2)+(4) */
    double udot = -mu * dot3(bs, e.gradB) - c->qom * dot3(bs, g);               /* Eq.(3)+(5) */
    /* Eq.(7) */
    double dX[3]; for (int i = 0; i < 3; i++) dX[i] = bxg[i] / Bss - c->qom * A * bs[i];
    double dudot = -c->qom * dot3(bs, g);
    double gl[3], glu; grad_ln_f0(c, &e, R, Z, u, mu, gl, &glu);
    double pw = c->weight_mode ? (p - w) : p;
    d5[0] = X[0]; d5[1] = X[2]; d5[2] = X[1] / R; d5[3] = udot; d5[4] = -pw * (dot3(dX, gl) + dudot * glu);
    return t < 0;
}
/* --------------------------------------------------------------- O11 ---- */
/* P2G: out[P][n_nodes][6] += q_p * (basis function of every DOF of the marker's triangle, on its four planes).  The basis
 * function of local DOF j is the element's interpolant of the unit vector e_j (one element solve each: slow and literal).
 * Markers outside the mesh deposit nothing.  Serial over markers: the sum is in marker order. */
int orc_deposit(orc *c, int64_t n, const double *R, const double *Z, const double *phi, const double *q, double *out) {
    if (!c || !c->head) return -1;
    memset(out, 0, sizeof(double) * (size_t)c->P * (size_t)c->n_nodes * 6);
    for (int64_t m = 0; m < n; m++) {
        int64_t t = locate_one(c, R[m], Z[m], 0);
        if (t < 0) continue;
        int k; double w[4], dw[4]; bspline(c, phi[m], &k, w, dw);
        for (int j = 0; j < 18; j++) {
            double e[18], coef[NM], v[6];
            for (int i = 0; i < 18; i++) e[i] = (i == j) ? 1.0 : 0.0;
            element_solve(c, t, e, coef);
            poly_eval(c, t, coef, R[m], Z[m], v);
            int node = c->tri[3 * t + j / 6], comp = j % 6;
            for (int a = 0; a < 4; a++) {
                int pl = ((k - 1 + a) % c->P + c->P) % c->P;
                out[((size_t)pl * c->n_nodes + node) * 6 + comp] += q[m] * w[a] * v[0];
            }
        }
    }
    return 0;
}

/* --------------------------------------------------------------- O12 ---- */
/* <F>(R, Z, phi) = (1/N) sum_j F(R + rho cos t_j, Z + rho sin t_j, phi), t_j = 2 pi j / N: the ring in the poloidal plane
 * (the magnetic field is mostly toroidal), all N points on the same toroidal angle; ring points outside the mesh
 * contribute zero (O9).  tri_out = triangle of the gyrocentre itself.  out[8][n] as in orc_gather. */
int orc_gather_gyro(orc *c, int64_t n, const double *R, const double *Z, const double *phi, const double *rho, int npts, double *out, int32_t *tri_out) {
    if (!c || !c->head || npts < 1) return -1;
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < n; m++) {
        double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        for (int j = 0; j < npts; j++) {
            double th = 2.0 * 3.14159265358979323846 * (double)j / (double)npts;
            double Rj = R[m] + rho[m] * cos(th), Zj = Z[m] + rho[m] * sin(th), f[4];
            int64_t t = locate_one(c, Rj, Zj, 0);
            for (int which = 0; which < 2; which++) { field_at(c, which, t, Rj, Zj, phi[m], f); for (int q = 0; q < 4; q++) acc[4 * which + q] += f[q]; }
        }
        for (int q = 0; q < 8; q++) out[(size_t)q * n + m] = acc[q] / (double)npts;
        if (tri_out) tri_out[m] = (int32_t)locate_one(c, R[m], Z[m], 0);
    }
    return 0;
}

/* --------------------------------------------------------------- O10 ---- */
/* L99 "Kernel for pullback treatment ... compute a correction term for the perturbed magnetic potential dA^h for each
 * particle marker": Eq.(6) u = v_par + (q/m)<dA^h>; with dA^h = A_par (R6) the map to the v_par picture is
 * u <- u - (q/m) A_par(R), and the perturbed distribution follows to first order: df <- df + (q/m) A_par df0/du, i.e.
 * w <- w + p (q/m) A_par d ln f0/du evaluated at the OLD u.  Outside the mesh A_par = 0 (O9) and the status bit is set. */
int orc_pullback(orc *c, int64_t n, const double *R, const double *Z, const double *phi, double *u, double *w, const double *mu, const double *p,
                 int32_t *status) {
    if (!c || !c->head) return -1;
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < n; m++) {
        int64_t t = locate_one(c, R[m], Z[m], 0); double f[4];
        field_at(c, 1, t, R[m], Z[m], phi[m], f);
        if (t < 0) { if (status) status[m] |= 1; continue; }
        equil e; equil_eval(c, R[m], Z[m], &e); double gl[3], glu;
        grad_ln_f0(c, &e, R[m], Z[m], u[m], mu[m], gl, &glu);
        double shift = c->qom * f[0];
        w[m] += p[m] * shift * glu;
        u[m] -= shift;
    }
    return 0;
}
/* L100 "Kernel for density calculation": the value of grid field `which` at every marker position (zero outside the mesh) */
int orc_density_g2p(orc *c, int which, int64_t n, const double *R, const double *Z, const double *phi, double *out) {
    if (!c || !c->head || which < 0 || which > 1) return -1;
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < n; m++) {
        int64_t t = locate_one(c, R[m], Z[m], 0); double f[4];
        field_at(c, which, t, R[m], Z[m], phi[m], f);
        out[m] = f[0];
    }
    return 0;
}
/* L101 "Kernel for distribution-function interpolation": f0 (up to its constant factor: n T^-3/2 exp(-E/T), L63) at the
 * marker's position and at its physical parallel velocity v_par = u - (q/m) A_par (Eq.(6)) */
int orc_f_interp(orc *c, int64_t n, const double *R, const double *Z, const double *phi, const double *u, const double *mu, double *out) {
    if (!c || !c->head) return -1;
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < n; m++) {
        int64_t t = locate_one(c, R[m], Z[m], 0); double f[4];
        field_at(c, 1, t, R[m], Z[m], phi[m], f);
        out[m] = exp(ln_f0(c, R[m], Z[m], u[m] - c->qom * f[0], mu[m]));
    }
    return 0;
}

int orc_rhs(orc *c, int64_t n, const double *R, const double *Z, const double *phi, const double *u, const double *w, const double *mu, const double *p, double *out /*[5][n]*/, int32_t *outside) {
    if (!c || !c->have_eq || !c->have_sp || !c->head) return -2;
#pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < n; m++) { double d[5]; int o = rhs_one(c, R[m], Z[m], phi[m], u[m], w[m], mu[m], p[m], d, 0); for (int q = 0; q < 5; q++) out[(size_t)q * n + m] = d[q]; if (outside) outside[m] = o; }
    return 0;
}

/* ---------------------------------------------------------------- O8 ---- */
int orc_push_rk4(orc *c, int64_t n, double *R, double *Z, double *phi, double *u, double *w, const double *mu, const double *p, int32_t *status, double dt, int32_t nsteps) {
    if (!c || !c->have_eq || !c->have_sp || !c->head) return -2;
    if (!(dt > 0) || !isfinite(dt) || nsteps < 0) return -1;
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t m = 0; m < n; m++) {
        double y[5] = {R[m], Z[m], phi[m], u[m], w[m]}; int st = status ? status[m] : 0;
        for (int s = 0; s < nsteps; s++) {
            double k1[5], k2[5], k3[5], k4[5], yt[5];
            st |= rhs_one(c, y[0], y[1], y[2], y[3], y[4], mu[m], p[m], k1, 0);
            for (int q = 0; q < 5; q++) yt[q] = y[q] + 0.5 * dt * k1[q];
            st |= rhs_one(c, yt[0], yt[1], yt[2], yt[3], yt[4], mu[m], p[m], k2, 0);
            for (int q = 0; q < 5; q++) yt[q] = y[q] + 0.5 * dt * k2[q];
            st |= rhs_one(c, yt[0], yt[1], yt[2], yt[3], yt[4], mu[m], p[m], k3, 0);
            for (int q = 0; q < 5; q++) yt[q] = y[q] + dt * k3[q];
            st |= rhs_one(c, yt[0], yt[1], yt[2], yt[3], yt[4], mu[m], p[m], k4, 0);
            for (int q = 0; q < 5; q++) y[q] = y[q] + dt / 6 * (k1[q] + 2 * k2[q] + 2 * k3[q] + k4[q]);
            y[2] = fmod(y[2], c->period); if (y[2] < 0) y[2] += c->period;
        }
        R[m] = y[0]; Z[m] = y[1]; phi[m] = y[2]; u[m] = y[3]; w[m] = y[4]; if (status) status[m] = st;
    }
    return 0;
}
