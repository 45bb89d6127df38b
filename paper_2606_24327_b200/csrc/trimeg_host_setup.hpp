// Host-side one-off setup for trimeg_mesh_load: triangle renumbering, neighbour table, box-grid CSR
// and the reduced-quintic element constants (L35, DESIGN.md "Element in
// reference coordinates").  Plain C++17, long double only for the two small dense inversions.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <unordered_map>
#include <vector>

#ifndef TRIMEG_BOX_REFINE
#define TRIMEG_BOX_REFINE 3.0
#endif
namespace trimeg_host {

// coefficient index of xi^i eta^j in the j-major layout the kernels use
inline int cidx(int i, int j) {
    static const int off[6] = {0, 6, 11, 15, 18, 20};
    return off[j] + i;
}
inline long double dmono(int i, int j, int dx, int dy, long double x, long double y) {
    if (i < dx || j < dy) return 0;
    long double c = 1;
    for (int t = 0; t < dx; t++) c *= (i - t);
    for (int t = 0; t < dy; t++) c *= (j - t);
    return c * std::pow(x, (long double)(i - dx)) * std::pow(y, (long double)(j - dy));
}
// dense inverse by Gauss-Jordan with partial pivoting; returns false if singular
inline bool invert(std::vector<long double>& A, int n) {
    std::vector<long double> I(n * n, 0);
    for (int i = 0; i < n; i++) I[i * n + i] = 1;
    for (int k = 0; k < n; k++) {
        int p = k;
        for (int i = k + 1; i < n; i++) if (fabsl(A[i * n + k]) > fabsl(A[p * n + k])) p = i;
        if (A[p * n + k] == 0) return false;
        if (p != k) for (int j = 0; j < n; j++) { std::swap(A[k * n + j], A[p * n + j]); std::swap(I[k * n + j], I[p * n + j]); }
        long double d = 1 / A[k * n + k];
        for (int j = 0; j < n; j++) { A[k * n + j] *= d; I[k * n + j] *= d; }
        for (int i = 0; i < n; i++) if (i != k) {
            long double f = A[i * n + k];
            if (f == 0) continue;
            for (int j = 0; j < n; j++) { A[i * n + j] -= f * A[k * n + j]; I[i * n + j] -= f * I[k * n + j]; }
        }
    }
    A = I;
    return true;
}

// Element constants, identical for every triangle because the vertex conditions are imposed in the affine
// reference frame (vertices at (0,0), (1,0), (0,1)):
//   Aplus [21][18]: particular solution  c0 = Aplus * d_ref  of the 18 vertex conditions (with the three quintic
//                   coefficients xi^4 eta, xi eta^4, xi^3 eta^2 pinned to zero);
//   Nul   [21][3] : null space of the vertex conditions (the three degree-5 "edge bubbles");
//   Gx,Gy [3][6]  : edge e, quintic monomial m=(5-m, m): the s^4 coefficient of the normal derivative along edge e is
//                   sum_m c5[m] (nh_x Gx[e][m] + nh_y Gy[e][m]) with nh = J^-1 n_phys.
struct ElementConsts {
    double Aplus[21 * 18];
    double Nul[21 * 3];
    double Gx[3 * 6], Gy[3 * 6];
};
inline bool element_consts(ElementConsts& ec) {
    const int n = 21;
    std::vector<long double> M(n * n, 0);
    const long double L[3][2] = {{0, 0}, {1, 0}, {0, 1}};
    const int D6[6][2] = {{0, 0}, {1, 0}, {0, 1}, {2, 0}, {1, 1}, {0, 2}};
    int r = 0;
    for (int v = 0; v < 3; v++) for (int d = 0; d < 6; d++) {
        for (int j = 0; j <= 5; j++) for (int i = 0; i + j <= 5; i++) M[r * n + cidx(i, j)] = dmono(i, j, D6[d][0], D6[d][1], L[v][0], L[v][1]);
        r++;
    }
    M[18 * n + cidx(4, 1)] = 1; M[19 * n + cidx(1, 4)] = 1; M[20 * n + cidx(3, 2)] = 1;
    if (!invert(M, n)) return false;
    for (int i = 0; i < n; i++) {
        for (int k = 0; k < 18; k++) ec.Aplus[i * 18 + k] = (double)M[i * n + k];
        for (int k = 0; k < 3; k++) ec.Nul[i * 3 + k] = (double)M[i * n + 18 + k];
    }
    const long double T[3][2] = {{1, 0}, {-1, 1}, {0, -1}};   // reference edge tangents: v0->v1, v1->v2, v2->v0
    for (int e = 0; e < 3; e++) for (int m = 0; m < 6; m++) {
        int i = 5 - m, j = m;
        long double tx = T[e][0], ty = T[e][1];
        long double gx = i > 0 ? i * std::pow(tx, (long double)(i - 1)) * std::pow(ty, (long double)j) : 0.0L;
        long double gy = j > 0 ? j * std::pow(tx, (long double)i) * std::pow(ty, (long double)(j - 1)) : 0.0L;
        ec.Gx[e * 6 + m] = (double)gx; ec.Gy[e * 6 + m] = (double)gy;
    }
    return true;
}
// per-triangle K [3][6] = (C N5)^-1 C, C [3][6] the edge-constraint rows in the reference frame, N5 [6][3] the quintic
// part of the null space; the element coefficients are c = c0 - Nul * (K * c0_quintic).
inline bool triangle_K(const ElementConsts& ec, const double v[3][2], double K[18]) {
    long double J[2][2] = {{(long double)v[1][0] - v[0][0], (long double)v[2][0] - v[0][0]}, {(long double)v[1][1] - v[0][1], (long double)v[2][1] - v[0][1]}};
    long double det = J[0][0] * J[1][1] - J[0][1] * J[1][0];
    if (!(det > 0)) return false;
    long double Ji[2][2] = {{J[1][1] / det, -J[0][1] / det}, {-J[1][0] / det, J[0][0] / det}};
    long double C[3][6];
    for (int e = 0; e < 3; e++) {
        long double tx = (long double)v[(e + 1) % 3][0] - v[e][0], ty = (long double)v[(e + 1) % 3][1] - v[e][1];
        long double len = sqrtl(tx * tx + ty * ty), nx = ty / len, ny = -tx / len;
        long double hx = Ji[0][0] * nx + Ji[0][1] * ny, hy = Ji[1][0] * nx + Ji[1][1] * ny;
        long double nrm = sqrtl(hx * hx + hy * hy); hx /= nrm; hy /= nrm;   // row scaling is free
        for (int m = 0; m < 6; m++) C[e][m] = hx * ec.Gx[e * 6 + m] + hy * ec.Gy[e * 6 + m];
    }
    std::vector<long double> CN(9, 0);
    for (int e = 0; e < 3; e++) for (int k = 0; k < 3; k++) for (int m = 0; m < 6; m++) CN[e * 3 + k] += C[e][m] * ec.Nul[cidx(5 - m, m) * 3 + k];
    if (!invert(CN, 3)) return false;
    for (int k = 0; k < 3; k++) for (int m = 0; m < 6; m++) {
        long double s = 0;
        for (int e = 0; e < 3; e++) s += CN[k * 3 + e] * C[e][m];
        K[k * 6 + m] = (double)s;
    }
    return true;
}

// spatial order of triangles: Morton code of the centroid on a 2^15 x 2^15 grid
inline uint64_t morton2(uint32_t x, uint32_t y) {
    auto spread = [](uint64_t v) { v &= 0xFFFFFFFFull; v = (v | (v << 16)) & 0x0000FFFF0000FFFFull; v = (v | (v << 8)) & 0x00FF00FF00FF00FFull; v = (v | (v << 4)) & 0x0F0F0F0F0F0F0F0Full; v = (v | (v << 2)) & 0x3333333333333333ull; v = (v | (v << 1)) & 0x5555555555555555ull; return v; };
    return spread(x) | (spread(y) << 1);
}

struct HostMesh {
    std::vector<int32_t> new_of_orig, orig_of_new;   // triangle renumbering
    std::vector<int32_t> tri;                        // [T][3] in new numbering
    std::vector<int32_t> nbr;                        // [T][3], edge e = (v_e, v_{e+1}); -1 boundary
    double xmin, ymin, dx, dy; int nx, ny;
    std::vector<int32_t> head, list;                 // box grid CSR
};
// returns 0 or a negative error code (-3 = bad mesh)
// `axis` (nullable): (R, Z) of the magnetic axis.  With it triangles are numbered along flux surfaces: radial bins one
// element wide (sqrt(2 x mean triangle area)), poloidal angle within a bin, so that consecutive triangles follow the
// poloidal field direction -- the direction markers move in during an RK4 step.  Without it: Morton order.
inline int build_mesh(int64_t n_nodes, const double* RZ, int64_t T, const int32_t* tri_in, const double* axis, HostMesh& hm) {
    double xmin = 1e300, xmax = -1e300, ymin = 1e300, ymax = -1e300;
    for (int64_t n = 0; n < n_nodes; n++) {
        double x = RZ[2 * n], y = RZ[2 * n + 1];
        if (!std::isfinite(x) || !std::isfinite(y)) return -3;
        xmin = std::min(xmin, x); xmax = std::max(xmax, x); ymin = std::min(ymin, y); ymax = std::max(ymax, y);
    }
    for (int64_t t = 0; t < T; t++) {
        const int32_t* tv = tri_in + 3 * t;
        for (int v = 0; v < 3; v++) if (tv[v] < 0 || tv[v] >= n_nodes) return -3;
        double ax = RZ[2 * tv[1]] - RZ[2 * tv[0]], ay = RZ[2 * tv[1] + 1] - RZ[2 * tv[0] + 1];
        double bx = RZ[2 * tv[2]] - RZ[2 * tv[0]], by = RZ[2 * tv[2] + 1] - RZ[2 * tv[0] + 1];
        if (!(ax * by - ay * bx > 0)) return -3;
    }
    double wx = xmax - xmin, wy = ymax - ymin;
    if (!(wx > 0) || !(wy > 0)) return -3;
    // renumber
    std::vector<uint64_t> key(T);
    double area_sum = 0;
    for (int64_t t = 0; t < T; t++) {
        const int32_t* tv = tri_in + 3 * t;
        double ax = RZ[2 * tv[1]] - RZ[2 * tv[0]], ay = RZ[2 * tv[1] + 1] - RZ[2 * tv[0] + 1];
        double bx = RZ[2 * tv[2]] - RZ[2 * tv[0]], by = RZ[2 * tv[2] + 1] - RZ[2 * tv[0] + 1];
        area_sum += 0.5 * (ax * by - ay * bx);
    }
    const double bin_w = std::sqrt(2.0 * area_sum / (double)T);
    for (int64_t t = 0; t < T; t++) {
        const int32_t* tv = tri_in + 3 * t;
        double cx = (RZ[2 * tv[0]] + RZ[2 * tv[1]] + RZ[2 * tv[2]]) / 3, cy = (RZ[2 * tv[0] + 1] + RZ[2 * tv[1] + 1] + RZ[2 * tv[2] + 1]) / 3;
        if (axis) {
            double x = cx - axis[0], y = cy - axis[1];
            double rho = std::sqrt(x * x + y * y), th = std::atan2(y, x);
            if (th < 0) th += 6.283185307179586;
            uint64_t bin = (uint64_t)std::min(4.0e9, rho / bin_w);
            uint64_t ang = (uint64_t)std::min(4294967295.0, th / 6.283185307179586 * 4294967296.0);
            key[t] = (bin << 32) | ang;
        } else {
            uint32_t ix = (uint32_t)std::min(32767.0, (cx - xmin) / wx * 32768.0), iy = (uint32_t)std::min(32767.0, (cy - ymin) / wy * 32768.0);
            key[t] = morton2(ix, iy);
        }
    }
    hm.orig_of_new.resize(T); std::iota(hm.orig_of_new.begin(), hm.orig_of_new.end(), 0);
    std::stable_sort(hm.orig_of_new.begin(), hm.orig_of_new.end(), [&](int32_t a, int32_t b) { return key[a] < key[b]; });
    hm.new_of_orig.resize(T);
    for (int64_t t = 0; t < T; t++) hm.new_of_orig[hm.orig_of_new[t]] = (int32_t)t;
    hm.tri.resize(3 * T);
    for (int64_t t = 0; t < T; t++) for (int v = 0; v < 3; v++) hm.tri[3 * t + v] = tri_in[3 * hm.orig_of_new[t] + v];
    // neighbours through an edge map
    hm.nbr.assign(3 * T, -1);
    std::unordered_map<uint64_t, int64_t> edges;
    edges.reserve((size_t)(3 * T));
    for (int64_t t = 0; t < T; t++) for (int e = 0; e < 3; e++) {
        uint32_t a = (uint32_t)hm.tri[3 * t + e], b = (uint32_t)hm.tri[3 * t + (e + 1) % 3];
        uint64_t k = a < b ? ((uint64_t)a << 32) | b : ((uint64_t)b << 32) | a;
        auto it = edges.find(k);
        if (it == edges.end()) edges.emplace(k, t * 3 + e);
        else {
            int64_t o = it->second;
            if (o < 0) return -3;   // an edge shared by three triangles
            hm.nbr[3 * t + e] = (int32_t)(o / 3); hm.nbr[o] = (int32_t)t; it->second = -1;
        }
    }
    // box grid
    // TRIMEG_BOX_REFINE^2 boxes per triangle of the bounding rectangle; a triangle is listed in the boxes it overlaps (separating-
    // axis test against its three edges, conservative by a small margin), not in all boxes of its bounding box: the candidate
    // lists are what a locate reads (k_gather_keys is bound by those loads, profiles/r02_gather_cfg4.md)
    const double refine = TRIMEG_BOX_REFINE;
    int nx = (int)std::ceil(refine * std::sqrt((double)T * wx / wy)), ny = (int)std::ceil(refine * std::sqrt((double)T * wy / wx));
    nx = std::max(nx, 1); ny = std::max(ny, 1);
    hm.nx = nx; hm.ny = ny; hm.xmin = xmin; hm.ymin = ymin; hm.dx = wx / nx; hm.dy = wy / ny;
    size_t nb = (size_t)nx * ny;
    hm.head.assign(nb + 1, 0);
    std::vector<int32_t> fill;
    for (int pass = 0; pass < 2; pass++) {
        if (pass) fill.assign(nb, 0);
        for (int64_t t = 0; t < T; t++) {
            double bx0 = 1e300, bx1 = -1e300, by0 = 1e300, by1 = -1e300;
            for (int v = 0; v < 3; v++) { double x = RZ[2 * hm.tri[3 * t + v]], y = RZ[2 * hm.tri[3 * t + v] + 1]; bx0 = std::min(bx0, x); bx1 = std::max(bx1, x); by0 = std::min(by0, y); by1 = std::max(by1, y); }
            const double eps = 1e-6;   // in box units: a point on a box boundary may round into either box
            int i0 = std::max(0, (int)std::floor((bx0 - xmin) / hm.dx - eps)), i1 = std::min(nx - 1, (int)std::floor((bx1 - xmin) / hm.dx + eps));
            int j0 = std::max(0, (int)std::floor((by0 - ymin) / hm.dy - eps)), j1 = std::min(ny - 1, (int)std::floor((by1 - ymin) / hm.dy + eps));
            // edge e from vertex e to e+1: outward normal (oriented by the sign of the area) and its offset
            double vx[3], vy[3], enx[3], eny[3], eoff[3];
            for (int v = 0; v < 3; v++) { vx[v] = RZ[2 * hm.tri[3 * t + v]]; vy[v] = RZ[2 * hm.tri[3 * t + v] + 1]; }
            const double area2 = (vx[1] - vx[0]) * (vy[2] - vy[0]) - (vx[2] - vx[0]) * (vy[1] - vy[0]), sg = area2 >= 0.0 ? 1.0 : -1.0;
            for (int e = 0; e < 3; e++) {
                const double ex = vx[(e + 1) % 3] - vx[e], ey = vy[(e + 1) % 3] - vy[e];
                enx[e] = sg * ey; eny[e] = -sg * ex; eoff[e] = enx[e] * vx[e] + eny[e] * vy[e];
            }
            for (int j = j0; j <= j1; j++) for (int i = i0; i <= i1; i++) {
                // the box (grown by eps on every side) lies outside edge e if even its corner nearest to the triangle does
                const double cx0 = xmin + (i - eps) * hm.dx, cx1 = xmin + (i + 1 + eps) * hm.dx, cy0 = ymin + (j - eps) * hm.dy, cy1 = ymin + (j + 1 + eps) * hm.dy;
                bool apart = false;
                for (int e = 0; e < 3 && !apart; e++) {
                    const double dmin = enx[e] * (enx[e] > 0.0 ? cx0 : cx1) + eny[e] * (eny[e] > 0.0 ? cy0 : cy1) - eoff[e];
                    apart = dmin > 1e-9 * (std::fabs(enx[e]) * hm.dx + std::fabs(eny[e]) * hm.dy);
                }
                if (apart) continue;
                size_t b = (size_t)j * nx + i;
                if (!pass) hm.head[b + 1]++; else hm.list[hm.head[b] + fill[b]++] = (int32_t)t;
            }
        }
        if (!pass) { for (size_t b = 0; b < nb; b++) hm.head[b + 1] += hm.head[b]; hm.list.resize(std::max<size_t>(1, hm.head[nb])); }
    }
    return 0;
}

}  // namespace trimeg_host

// ---------------------------------------------------------------------------------------------------------
// Static patches for the tiled push kernel: a patch is a run of TP consecutive triangles in the library's
// numbering; its slot list = own triangles (slots 0..TP-1) followed by a halo of nearby triangles up to SMAX slots.
// Halo choice: candidates are collected ring by ring (triangles sharing a vertex with the set so far) and ranked
// by an anisotropic distance to the nearest own triangle: with the magnetic axis known, the distance along the
// poloidal field direction (tangent to the flux surface) counts 1/aspect of the distance across it, because
// within one RK4 step markers move mainly along the field (parallel streaming) and hardly across it (drifts).
// nbr gives, per slot and edge, the slot across that edge, -1 when that triangle is not staged, -2 when the edge is
// on the mesh boundary.
namespace trimeg_host {
struct HostPatches {
    int TP = 0, SMAX = 0, npatch = 0;
    std::vector<int32_t> slots;    // [npatch][SMAX], -1 = unused
    std::vector<int16_t> nbr;      // [npatch][SMAX][4] (4th = pad)
    std::vector<int32_t> nslots;   // [npatch]
};
inline void build_patches(const HostMesh& hm, const double* RZ, int64_t n_nodes, int64_t T, int TP, int SMAX, const double* axis, double aspect,
                          HostPatches& hp) {
    hp.TP = TP; hp.SMAX = SMAX; hp.npatch = (int)((T + TP - 1) / TP);
    hp.slots.assign((size_t)hp.npatch * SMAX, -1);
    hp.nbr.assign((size_t)hp.npatch * SMAX * 4, -1);
    hp.nslots.assign(hp.npatch, 0);
    // node -> triangles CSR
    std::vector<int32_t> nhead(n_nodes + 1, 0), nlist(3 * T);
    for (int64_t t = 0; t < T; t++) for (int v = 0; v < 3; v++) nhead[hm.tri[3 * t + v] + 1]++;
    for (int64_t n = 0; n < n_nodes; n++) nhead[n + 1] += nhead[n];
    { std::vector<int32_t> f(nhead.begin(), nhead.end() - 1); for (int64_t t = 0; t < T; t++) for (int v = 0; v < 3; v++) nlist[f[hm.tri[3 * t + v]]++] = (int32_t)t; }
    std::vector<double> cx(T), cy(T);
    for (int64_t t = 0; t < T; t++) { cx[t] = (RZ[2 * hm.tri[3 * t]] + RZ[2 * hm.tri[3 * t + 1]] + RZ[2 * hm.tri[3 * t + 2]]) / 3; cy[t] = (RZ[2 * hm.tri[3 * t] + 1] + RZ[2 * hm.tri[3 * t + 1] + 1] + RZ[2 * hm.tri[3 * t + 2] + 1]) / 3; }
    std::vector<int32_t> slot_of(T, -1), mark(T, -1);
    std::vector<int32_t> frontier, next;
    struct Cand { double key; int32_t t; };
    std::vector<Cand> cand;
    const double inv_asp2 = 1.0 / (aspect * aspect);
    for (int p = 0; p < hp.npatch; p++) {
        int64_t t0 = (int64_t)p * TP, t1 = std::min<int64_t>(T, t0 + TP);
        int32_t* sl = &hp.slots[(size_t)p * SMAX];
        int ns = 0;
        for (int64_t t = t0; t < t1; t++) { sl[ns] = (int32_t)t; slot_of[t] = ns; mark[t] = p; ns++; }
        int own = ns;
        // pad unused own slots (last patch) so that own triangles always sit at slot = t - t0
        for (; ns < TP && ns < SMAX; ns++) sl[ns] = -1;
        frontier.assign(sl, sl + own);
        cand.clear();
        for (int ring = 0; ring < 8 && (int)cand.size() < 5 * SMAX && !frontier.empty(); ring++) {
            next.clear();
            for (int32_t t : frontier) for (int v = 0; v < 3; v++) {
                int32_t node = hm.tri[3 * t + v];
                for (int32_t q = nhead[node]; q < nhead[node + 1]; q++) {
                    int32_t o = nlist[q];
                    if (mark[o] == p) continue;
                    mark[o] = p;
                    next.push_back(o);
                    double best = 1e300;
                    for (int64_t h = t0; h < t1; h++) {
                        double dx = cx[o] - cx[h], dy = cy[o] - cy[h], d2;
                        if (axis) {
                            double ex = -(cy[h] - axis[1]), ey = cx[h] - axis[0], en = std::sqrt(ex * ex + ey * ey);
                            if (en > 0) {
                                ex /= en; ey /= en;
                                double dpar = dx * ex + dy * ey, dperp = -dx * ey + dy * ex;
                                d2 = dpar * dpar * inv_asp2 + dperp * dperp;
                            } else d2 = dx * dx + dy * dy;
                        } else d2 = dx * dx + dy * dy;
                        best = std::min(best, d2);
                    }
                    cand.push_back({best, o});
                }
            }
            frontier.swap(next);
        }
        std::sort(cand.begin(), cand.end(), [](const Cand& a, const Cand& b) { return a.key < b.key || (a.key == b.key && a.t < b.t); });
        for (const Cand& c : cand) {
            if (ns >= SMAX) break;
            sl[ns] = c.t; slot_of[c.t] = ns; ns++;
        }
        hp.nslots[p] = ns;
        for (int s = 0; s < ns; s++) {
            int32_t t = sl[s];
            if (t < 0) continue;
            for (int e = 0; e < 3; e++) {
                int32_t nb = hm.nbr[3 * t + e];
                hp.nbr[((size_t)p * SMAX + s) * 4 + e] = nb < 0 ? (int16_t)-2 : (slot_of[nb] >= 0 ? (int16_t)slot_of[nb] : (int16_t)-1);   // -2: mesh boundary, -1: not staged
            }
        }
        for (int s = 0; s < ns; s++) if (sl[s] >= 0) slot_of[sl[s]] = -1;
    }
}
}  // namespace trimeg_host
