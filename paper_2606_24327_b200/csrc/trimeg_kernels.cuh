// Device kernels of the marker push: marker store, setup, gather, the two-phase RK4 push and the counting sort.
// Compiled for sm_100a only.  DESIGN.md "Kernels" describes the split of one RK4 step into two phases.
#pragma once
#include <cuda_runtime.h>

#include "trimeg_math.cuh"
#include "trimeg_tile.cuh"

namespace trimeg {

// ============================================================================================ marker store
// One 128-byte record per marker (array of structures: a marker is always read and written whole, through a sort
// permutation, so one record = one cache line = four full 32-byte sectors).  Two buffers: a phase that re-sorts reads
// buffer A through the permutation and writes buffer B in cell order, so the data movement of the sort costs no pass
// of its own and the next permutation is nearly the identity.  What y and k hold depends on where the step stands:
//   between steps / before phase A:  y = state y_n (R, Z, phi, u, w),       k = k1 = f(y_n)
//   between phase A and phase B:     y = Y = y_n + dt/6 (k1 + 2 k2 + 2 k3),  k = y4 = y_n + dt k3 (stage-4 position)
// tri = triangle (library numbering) of the next phase's first evaluation point, -1 unknown / outside.
struct __align__(16) Rec {
    double y[5];
    double k[5];
    double mu, p;
    int tri, st;
    int id, pad0;            // id = index in the caller's arrays
    double pad[2];
};
static_assert(sizeof(Rec) == 128, "marker record is one 128-byte line");

struct DevTables {
    const TriGeom* geom;     // [T]
    const double* coef;      // [T][P+3+2*PLANE_PAD][21][2]; see PLANE_PAD in trimeg_math.cuh
    BoxGrid bg;
    TorP tor;
    int T;
    long long tri_stride;    // doubles per triangle = (P+3+2*PLANE_PAD)*42
};

// tiled push configuration: patches of 8 triangles + halo (SMAX slots with coefficients, 32 with geometry), windows of 4
// toroidal intervals (+1 each side), ring of NBUF staged blocks, K chunk slots of 32 records, 4 light + 12 compute warps
// per CTA, one CTA per SM.  (TRIMEG_* macros: tuning sweeps only; the shipped build uses the defaults.)
#ifndef TRIMEG_SMAX
#define TRIMEG_SMAX 15
#endif
#ifndef TRIMEG_NBUF
#define TRIMEG_NBUF 3
#endif
#ifndef TRIMEG_NSLOTS
#define TRIMEG_NSLOTS 20
#endif
using Tile = TileCfg<8, TRIMEG_SMAX, 4, TRIMEG_NBUF, TRIMEG_NSLOTS>;
// cell numbering used by the sort: super-cell (patch, window) major, then triangle within the patch, then interval
struct CellMap {
    int P, nwin;
    __host__ __device__ __forceinline__ int cell(int t, int k) const {
        int patch = t / Tile::TP, tl = t - patch * Tile::TP, wdw = k / Tile::WK, kl = k - wdw * Tile::WK;
        return ((patch * nwin + wdw) * Tile::TP + tl) * Tile::WK + kl;
    }
};
// where the sort key of a marker's next evaluation point goes (the counting sort's first pass is fused into the push)
struct KeyOut {
    int* keys;      // [n] cell of the next phase's first evaluation point, indexed like the destination buffer
    int* hist;      // [ncell + 2] histogram of the keys; bin ncell = outside the mesh
    int ncell;
    int enabled;
};

__constant__ double c_Aplus[21 * 18];
__constant__ double c_Nul[21 * 3];

// In memory the eight 16-byte chunks of record i are stored XOR-swizzled by rec_swizzle(i) = i & 7: logical chunk j sits
// at chunk position j ^ rec_swizzle(i) (a record is only ever handled whole, so the swizzle costs nothing; it lets
// row-per-lane shared-memory images of records be read and written 16 bytes per lane without bank conflicts).
__host__ __device__ __forceinline__ int rec_swizzle(long long i) { return (int)i & 7; }
__device__ __forceinline__ void rec_load(const Rec* __restrict__ base, long long i, Rec& r) {
    const double2* s = reinterpret_cast<const double2*>(base + i);
    double2* d = reinterpret_cast<double2*>(&r);
    const int sw = rec_swizzle(i);
#pragma unroll
    for (int j = 0; j < 7; ++j) d[j] = __ldcs(s + (j ^ sw));   // 14 doubles are live; the last chunk is padding
}
__device__ __forceinline__ void rec_store(Rec* __restrict__ base, long long i, const Rec& r) {
    double2* d = reinterpret_cast<double2*>(base + i);
    const double2* s = reinterpret_cast<const double2*>(&r);
    const int sw = rec_swizzle(i);
#pragma unroll
    for (int j = 0; j < 7; ++j) d[j ^ sw] = s[j];
}

// ============================================================================================ setup kernels
// fields_set: nodal DOFs -> per-triangle reference-frame polynomial coefficients, for one field.
// One thread per (triangle, plane).  c = c0 - Nul (K c0_5),  c0 = Aplus d_ref,  d_ref = DOFs pulled back with J.
__global__ void k_fields_set(int T, int P, int which, const int* __restrict__ tri, const double* __restrict__ RZ,
                             const double* __restrict__ Kmat, const double* __restrict__ dof, long long n_nodes, int NPP,
                             double* __restrict__ coef) {
    long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= (long long)T * P) return;
    int t = (int)(gid / P), k = (int)(gid % P);
    int nd[3] = {tri[3 * t], tri[3 * t + 1], tri[3 * t + 2]};
    double x0 = RZ[2 * nd[0]], y0 = RZ[2 * nd[0] + 1];
    double j11 = RZ[2 * nd[1]] - x0, j21 = RZ[2 * nd[1] + 1] - y0, j12 = RZ[2 * nd[2]] - x0, j22 = RZ[2 * nd[2] + 1] - y0;
    double d[18];
#pragma unroll
    for (int v = 0; v < 3; ++v) {
        const double* s = dof + ((long long)k * n_nodes + nd[v]) * 6;
        double f = s[0], fR = s[1], fZ = s[2], fRR = s[3], fRZ = s[4], fZZ = s[5];
        d[6 * v + 0] = f;
        d[6 * v + 1] = j11 * fR + j21 * fZ;                       // J^T grad
        d[6 * v + 2] = j12 * fR + j22 * fZ;
        double hR1 = fRR * j11 + fRZ * j21, hZ1 = fRZ * j11 + fZZ * j21;   // H J (column 1)
        double hR2 = fRR * j12 + fRZ * j22, hZ2 = fRZ * j12 + fZZ * j22;   // H J (column 2)
        d[6 * v + 3] = j11 * hR1 + j21 * hZ1;                     // J^T H J
        d[6 * v + 4] = j11 * hR2 + j21 * hZ2;
        d[6 * v + 5] = j12 * hR2 + j22 * hZ2;
    }
    double c[21];
#pragma unroll
    for (int i = 0; i < 21; ++i) {
        double s = 0.0;
#pragma unroll
        for (int q = 0; q < 18; ++q) s = fma(c_Aplus[i * 18 + q], d[q], s);
        c[i] = s;
    }
    // quintic part: monomial m = (5-m, m) sits at j-major index off[m] + 5 - m
    const int qi[6] = {5, 6 + 4, 11 + 3, 15 + 2, 18 + 1, 20};
    const double* K = Kmat + (long long)t * 18;
    double z[3];
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        double s = 0.0;
#pragma unroll
        for (int m = 0; m < 6; ++m) s = fma(K[r * 6 + m], c[qi[m]], s);
        z[r] = s;
    }
    // toroidal plane k sits at every padded index pp = k + 1 + PLANE_PAD (mod P) inside [0, NPP)
    long long tri_stride = (long long)NPP * PLANE_STRIDE;
    double* base = coef + (long long)t * tri_stride;
    double v[21];
#pragma unroll
    for (int i = 0; i < 21; ++i) v[i] = c[i] - (c_Nul[i * 3] * z[0] + c_Nul[i * 3 + 1] * z[1] + c_Nul[i * 3 + 2] * z[2]);
    for (int pp = (k + 1 + PLANE_PAD) % P; pp < NPP; pp += P) {
#pragma unroll
        for (int i = 0; i < 21; ++i) base[(long long)pp * PLANE_STRIDE + 2 * i + which] = v[i];
    }
}

// SoA caller arrays -> records [first, first + cnt)
__global__ void k_bind(Rec* __restrict__ recs, long long first, long long cnt, const double* R, const double* Z, const double* phi,
                       const double* u, const double* w, const double* mu, const double* p) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= cnt) return;
    Rec r;
    r.y[0] = R[i]; r.y[1] = Z[i]; r.y[2] = phi[i]; r.y[3] = u[i]; r.y[4] = w[i];
#pragma unroll
    for (int q = 0; q < 5; ++q) r.k[q] = 0.0;
    r.mu = mu[i]; r.p = p[i]; r.tri = -1; r.st = 0;
    r.id = (int)(first + i); r.pad0 = 0;
    r.pad[0] = r.pad[1] = 0.0;
    rec_store(recs, first + i, r);
}
// records -> SoA arrays in the caller's order (any may be null), in two steps so that the 8-byte writes are coalesced:
// inv[caller id] = record position (one scattered 4-byte write per marker), then one thread per caller id reads its
// record (a whole line) and writes the arrays in order.
__global__ void k_inv_ids(const Rec* __restrict__ recs, long long n, int* __restrict__ inv) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int2 v = __ldcs(reinterpret_cast<const int2*>(reinterpret_cast<const double2*>(recs + i) + (6 ^ rec_swizzle(i))) + 1);   // (id, pad0)
    inv[v.x] = (int)i;
}
__global__ void k_get(const Rec* __restrict__ recs, const int* __restrict__ inv, long long n, double* R, double* Z, double* phi, double* u, double* w,
                      int* status) {
    long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= n) return;
    Rec r;
    rec_load(recs, inv[o], r);
    if (R) R[o] = r.y[0];
    if (Z) Z[o] = r.y[1];
    if (phi) phi[o] = r.y[2];
    if (u) u[o] = r.y[3];
    if (w) w[o] = r.y[4];
    if (status) status[o] = r.st & 1;
}

// ============================================================================================ gather / global path
struct LdGlobal {   // coefficient pair fetch from the global table (L1/L2)
    const double2* p;
    __device__ __forceinline__ void operator()(int idx, double& a, double& b) const {
        double2 v = __ldg(p + idx);
        a = v.x; b = v.y;
    }
};

__device__ __forceinline__ void gather_at(const DevTables& tb, int t, double R, double Z, double phi, Fields& f) {
    if (t < 0) { f = Fields{0, 0, 0, 0, 0, 0, 0, 0}; return; }
    const TriGeom g = tb.geom[t];
    double xi, eta;
    ref_coords(g, R, Z, xi, eta);
    double w[4], dw[4];
    int kk = bspline_weights(tb.tor, phi, w, dw);
    LdGlobal ld{reinterpret_cast<const double2*>(tb.coef + (long long)t * tb.tri_stride + (long long)(kk + PLANE_PAD) * PLANE_STRIDE)};
    double acc[8];
    gather_cell<true, double>(ld, xi, eta, w, dw, acc);
    to_fields(g, acc, f);
}

#ifndef TRIMEG_GATHER_OCC
#define TRIMEG_GATHER_OCC 4
#endif
__global__ void __launch_bounds__(256, TRIMEG_GATHER_OCC) k_gather(DevTables tb, long long n, const double* __restrict__ R, const double* __restrict__ Z,
                                                const double* __restrict__ phi, double* __restrict__ out, int* __restrict__ tri_out,
                                                const int* __restrict__ flag) {   // flag: null, or the path chosen on the device (1 = this kernel)
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n || (flag && *flag != 1)) return;
    double r = R[m], z = Z[m];
    int t = locate_box(tb.bg, tb.geom, r, z);
    Fields f;
    gather_at(tb, t, r, z, phi[m], f);
    out[m] = f.P; out[n + m] = f.PR; out[2 * n + m] = f.PZ; out[3 * n + m] = f.Pp;
    out[4 * n + m] = f.A; out[5 * n + m] = f.AR; out[6 * n + m] = f.AZ; out[7 * n + m] = f.Ap;
    if (tri_out) tri_out[m] = t < 0 ? -1 : tb.geom[t].orig;
}

// N-point gyro-average of the gather (the <...> of Eq.(4)-(6); switched off in the paper's runs, L320;
// reading R26): mean over npts points of the ring of radius rho in the poloidal plane around (R, Z), same toroidal angle; ring
// points outside the mesh contribute zero.  The ring points of one gyrocentre lie within a few elements of each other, so
// every point after the first is found by an edge walk from its predecessor's triangle.
__global__ void __launch_bounds__(256, 3) k_gather_gyro(DevTables tb, long long n, const double* __restrict__ R, const double* __restrict__ Z,
                                                        const double* __restrict__ phi, const double* __restrict__ rho, int npts, double* __restrict__ out,
                                                        int* __restrict__ tri_out) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned lanes = __ballot_sync(0xffffffffu, m < n);
    if (m >= n) return;
    const double r0 = R[m], z0 = Z[m], ph = phi[m], rh = rho[m];
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int t = -1;
    for (int j = 0; j < npts; ++j) {
        double sn, cs;
        sincospi(2.0 * (double)j / (double)npts, &sn, &cs);
        const double rj = fma(rh, cs, r0), zj = fma(rh, sn, z0);
        t = t >= 0 ? locate_walk(tb.bg, tb.geom, t, rj, zj) : locate_box(tb.bg, tb.geom, rj, zj);
        __syncwarp(lanes);
        Fields f;
        gather_at(tb, t, rj, zj, ph, f);
        acc[0] += f.P; acc[1] += f.PR; acc[2] += f.PZ; acc[3] += f.Pp; acc[4] += f.A; acc[5] += f.AR; acc[6] += f.AZ; acc[7] += f.Ap;
    }
    const double inv = 1.0 / (double)npts;
#pragma unroll
    for (int q = 0; q < 8; ++q) out[(long long)q * n + m] = acc[q] * inv;
    if (tri_out) { const int tc = locate_box(tb.bg, tb.geom, r0, z0); tri_out[m] = tc < 0 ? -1 : tb.geom[tc].orig; }
}

// one right-hand-side evaluation for one marker, fields through L1/L2; updates the triangle hint; returns 1 if outside
// `lanes`: the lanes of the warp that make this call together.  They leave the edge walk after different numbers of hops and
// would otherwise stay diverged through the gather and the right-hand side (the warp then runs that arithmetic once per
// group of lanes: measured 3.0 times per warp in k_deposit before its own reconvergence point was added).
__device__ __forceinline__ int stage_simple(const DevTables& tb, const EquilP& ep, const SpeciesP& sp, int& t, double R, double Z,
                                            double phi, double u, double w, double mu, double p, double d[5], unsigned lanes) {
    t = locate_walk(tb.bg, tb.geom, t, R, Z);
    __syncwarp(lanes);
    Fields f;
    gather_at(tb, t, R, Z, phi, f);
    FieldsG<double> fg;
    fields_to_g(f, u, fg);
    rhs_eval<double, true>(ep, sp, R, Z, u, w, mu, p, fg, d);
    return t < 0;
}

__device__ __forceinline__ double wrap_phi(const TorP& tp, double phi) {
    double ph = fma(-tp.period, floor(phi * tp.inv_period), phi);
    if (ph < 0.0) ph += tp.period;
    if (ph >= tp.period) ph -= tp.period;
    return ph;
}

// ============================================================================================ two-phase RK4 step
// Classical RK4 evaluates f at three places per step: y_n (k1), the half-step points y_n + dt/2 k1 and y_n + dt/2 k2
// (k2, k3), and the full-step points y_n + dt k3 (k4) and y_{n+1} (the next step's k1).  The two half-step points lie
// within O(dt^2) of each other, and so do the two full-step points, but at dt = 0.05 the half- and full-step points of
// the ITG configurations are about one mesh cell apart.  The step is therefore split where the cell changes:
//   phase A (markers ordered by the cell of y_n + dt/2 k1):   k2, k3          -> Y = y_n + dt/6 (k1 + 2 k2 + 2 k3), y4
//   phase B (markers ordered by the cell of y4):              k4, y_{n+1}, k1' = f(y_{n+1})
// so that both evaluations of a phase read the coefficient block of (almost always) one cell and all lanes of a warp
// read the same few cells.  PHASE_INIT computes k1 = f(y_n) for a freshly bound store.
// The arithmetic of a step is the textbook one; only the order in which markers are visited changes.
enum { PHASE_A = 0, PHASE_B = 1, PHASE_INIT = 2 };

// Advances record r through one phase.  eval(y, d) evaluates the right-hand side at y and returns false if it cannot
// (the tiled kernel: evaluation point outside the staged block); then r is left untouched and false is returned.
// next[0..2] = (R, Z, phi) of the following phase's first evaluation point.
template <int PHASE, class Eval>
__device__ __forceinline__ bool phase_step(const TorP& tor, double dt, Rec& r, Eval&& eval, double next[3]) {
    const double h2 = 0.5 * dt, h6 = dt / 6.0;
    double a[5], d[5], y[5];
    // first evaluation point: A: y_n + dt/2 k1;  B: y4;  INIT: (none, only the second evaluation, at y_n)
#pragma unroll
    for (int q = 0; q < 5; ++q) y[q] = PHASE == PHASE_A ? fma(h2, r.k[q], r.y[q]) : (PHASE == PHASE_B ? r.k[q] : r.y[q]);
    // the two evaluations run through ONE copy of the evaluation code (a rolled loop): the kernel body then fits the
    // instruction cache, which two inlined copies did not (profiles/r01c_summary.md, stall_no_instruction)
#pragma unroll 1
    for (int e = (PHASE == PHASE_INIT ? 1 : 0); e < 2; ++e) {
        if (!eval(y, d)) return false;
        if (e == 0) {
#pragma unroll
            for (int q = 0; q < 5; ++q) {
                a[q] = d[q];                                                            // A: k2;  B: k4
                y[q] = PHASE == PHASE_A ? fma(h2, d[q], r.y[q]) : fma(h6, d[q], r.y[q]);  // A: y_n + dt/2 k2;  B: y_{n+1}
            }
            if (PHASE == PHASE_B) y[2] = wrap_phi(tor, y[2]);
        }
    }
    if (PHASE == PHASE_A) {
#pragma unroll
        for (int q = 0; q < 5; ++q) {
            const double acc = fma(2.0, d[q], fma(2.0, a[q], r.k[q])), y0 = r.y[q];
            r.y[q] = fma(h6, acc, y0);                                                  // Y
            r.k[q] = fma(dt, d[q], y0);                                                 // y4 = y_n + dt k3
        }
        next[0] = r.k[0]; next[1] = r.k[1]; next[2] = r.k[2];
    } else {
#pragma unroll
        for (int q = 0; q < 5; ++q) { r.y[q] = y[q]; r.k[q] = d[q]; }                  // y_{n+1} (INIT: y_n), k1 = f(it)
        next[0] = fma(h2, d[0], y[0]); next[1] = fma(h2, d[1], y[1]); next[2] = fma(h2, d[2], y[2]);
    }
    return true;
}

// final store of one record: the record itself and (if enabled) the sort key of its next evaluation point
__device__ __forceinline__ void store_rec(const DevTables& tb, const CellMap& cm, const KeyOut& ko, Rec* recs, long long ri,
                                          Rec& r, int t, const double next[3]) {
    r.tri = t;
    rec_store(recs, ri, r);
    if (ko.enabled) {
        double sf;
        int k = toroidal_interval(tb.tor, next[2], sf);
        int key = t < 0 ? ko.ncell : cm.cell(t, k);
        ko.keys[ri] = key;
        atomicAdd(ko.hist + key, 1);
    }
}

// one phase for one record through the global tables (L1/L2): the follow-up path of the tiled kernel (markers that
// left their staged block, markers outside the mesh), the initial k1, and un-sorted operation
template <int PHASE>
__device__ __forceinline__ void phase_global(const DevTables& tb, const EquilP& ep, const SpeciesP& sp, const CellMap& cm, const KeyOut& ko,
                                             const Rec* src, Rec* dst, long long ri, long long m, double dt, unsigned lanes) {
    Rec r;
    rec_load(src, ri, r);
    int t = r.tri, st = r.st;
    const double mu = r.mu, p = r.p;
    // status bit 0: some RK stage of a finished or running step was evaluated outside the mesh (sticky); bit 1: the cached
    // k1 = f(y_n) was.  That evaluation is the first stage of the NEXT step, so it only counts once that step runs:
    // phase A folds bit 1 into bit 0, markers_get reports bit 0 only (the oracle's and variant 1's rule).
    if (PHASE == PHASE_A && (st & 2)) st = (st | 1) & ~2;
    if (PHASE == PHASE_INIT) st &= ~2;
    int ev = 0;
    auto eval = [&](const double y[5], double d[5]) {
        const int out = stage_simple(tb, ep, sp, t, y[0], y[1], y[2], y[3], y[4], mu, p, d, lanes);
        st |= (PHASE == PHASE_A || (PHASE == PHASE_B && ev == 0)) ? out : 2 * out;
        ++ev;
        return true;
    };
    double next[3];
    phase_step<PHASE>(tb.tor, dt, r, eval, next);
    t = locate_walk(tb.bg, tb.geom, t, next[0], next[1]);
    r.st = st;
    store_rec(tb, cm, ko, dst, m, r, t, next);
}
// positions m = index[i] (or i if index is null) of the cell order for i in [*first (or 0), *count (or n)):
// record src[perm[m]] (or src[m] if perm is null) -> dst[m]
template <int PHASE>
__device__ __forceinline__ void phase_global_range(const DevTables& tb, const EquilP& ep, const SpeciesP& sp, const CellMap& cm, const KeyOut& ko, const Rec* src,
                                                   Rec* dst, const int* __restrict__ perm, const int* __restrict__ index, long long lo, long long hi,
                                                   double dt, int bid, int nblocks) {
    // whole warps go round the loop together (the lanes of the last round that have no record sit it out), so that the lanes
    // with a record can be named for the reconvergence points inside
    const int lane = threadIdx.x & 31;
    for (long long base = lo + (long long)bid * blockDim.x + (threadIdx.x - lane); base < hi; base += (long long)nblocks * blockDim.x) {
        const long long i = base + lane;
        const unsigned lanes = __ballot_sync(0xffffffffu, i < hi);
        if (i < hi) {
            const long long m = index ? (long long)index[i] : i;
            phase_global<PHASE>(tb, ep, sp, cm, ko, src, dst, perm ? (long long)perm[m] : m, m, dt, lanes);
        }
    }
}
template <int PHASE>
__global__ void __launch_bounds__(128) k_phase_global(DevTables tb, EquilP ep, SpeciesP sp, CellMap cm, KeyOut ko, const Rec* src,
                                                      Rec* dst, const int* __restrict__ perm, const int* __restrict__ index,
                                                      const int* __restrict__ first, const int* __restrict__ count, long long n, double dt) {
    const long long lo = first ? (long long)*first : 0, hi = count ? (long long)*count : n;
    phase_global_range<PHASE>(tb, ep, sp, cm, ko, src, dst, perm, index, lo, hi, dt, (int)blockIdx.x, (int)gridDim.x);
}

// first step after a bind: triangle and cell key of every marker's CURRENT position (box-grid locate), so that k1 = f(y_n)
// can be computed by the phase kernel in cell order instead of through the global tables in caller order
__global__ void __launch_bounds__(256) k_locate_keys(DevTables tb, CellMap cm, KeyOut ko, Rec* __restrict__ recs, long long n) {
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    Rec r;
    rec_load(recs, i, r);
    const int t = locate_walk(tb.bg, tb.geom, r.tri, r.y[0], r.y[1]);
    r.tri = t;
    reinterpret_cast<double2*>(recs + i)[6 ^ rec_swizzle(i)] = reinterpret_cast<const double2*>(&r)[6];   // (tri, st, id, pad0)
    double sf;
    const int k = toroidal_interval(tb.tor, r.y[2], sf);
    const int key = t < 0 ? ko.ncell : cm.cell(t, k);
    ko.keys[i] = key;
    atomicAdd(ko.hist + key, 1);
}

// markers whose next evaluation point left the staged geometry of the phase kernel: their records are complete except for
// the triangle of that point (the record holds a hint) and the sort key.  Next point: after phase A the stage-4 position held
// in k, otherwise y + dt/2 k.
template <int PHASE>
__device__ __forceinline__ void fix_keys_range(const DevTables& tb, const CellMap& cm, const KeyOut& ko, Rec* recs, const int* __restrict__ list, int cnt,
                                               long long n, double dt, int bid, int nblocks) {
    for (int i = bid * blockDim.x + threadIdx.x; i < cnt; i += nblocks * blockDim.x) {
        const long long m = list[n - 1 - i];
        Rec r;
        rec_load(recs, m, r);
        const double h2 = 0.5 * dt;
        const double R = PHASE == PHASE_A ? r.k[0] : fma(h2, r.k[0], r.y[0]), Z = PHASE == PHASE_A ? r.k[1] : fma(h2, r.k[1], r.y[1]);
        const double phi = PHASE == PHASE_A ? r.k[2] : fma(h2, r.k[2], r.y[2]);
        const int t = locate_walk(tb.bg, tb.geom, r.tri, R, Z);
        r.tri = t;
        reinterpret_cast<double2*>(recs + m)[6 ^ rec_swizzle(m)] = reinterpret_cast<const double2*>(&r)[6];   // (tri, st, id, pad0)
        if (ko.enabled) {
            double sf;
            const int k = toroidal_interval(tb.tor, phi, sf);
            const int key = t < 0 ? ko.ncell : cm.cell(t, k);
            ko.keys[m] = key;
            atomicAdd(ko.hist + key, 1);
        }
    }
}
template <int PHASE>
__global__ void __launch_bounds__(128) k_fix_keys(DevTables tb, CellMap cm, KeyOut ko, Rec* recs, const int* __restrict__ list, const int* __restrict__ count,
                                                  long long n, double dt) {
    fix_keys_range<PHASE>(tb, cm, ko, recs, list, *count, n, dt, (int)blockIdx.x, (int)gridDim.x);
}
#ifndef TRIMEG_FU_OCC
#define TRIMEG_FU_OCC 4
#endif
// The three follow-ups of a phase in ONE launch (they touch disjoint markers, each alone is a short latency-bound kernel):
// blocks [0, nbA): the markers the tiled kernel retired (list `retired`, *work[4] of them); [nbA, nbA + nbB): the markers
// outside the mesh, sorted behind the last cell (positions from *outside_first); the rest: sort keys of the markers whose
// next evaluation point left the staged geometry (the same list from its end, work[5] of them).  Thread 0 also adds the
// retired count to the statistics.
template <int PHASE>
__global__ void __launch_bounds__(128, TRIMEG_FU_OCC) k_followups(DevTables tb, EquilP ep, SpeciesP sp, CellMap cm, KeyOut ko, const Rec* src, Rec* dst,
                                                   const int* __restrict__ perm, const int* __restrict__ retired, const int* __restrict__ work,
                                                   const int* __restrict__ outside_first, long long n, double dt, unsigned long long* __restrict__ stat,
                                                   int nbA, int nbB) {
    const int b = (int)blockIdx.x;
    if (b == 0 && threadIdx.x == 0) atomicAdd(stat, (unsigned long long)work[4]);
    if (b < nbA + nbB) {
        const bool listed = b < nbA;
        const long long lo = listed ? 0 : (long long)*outside_first, hi = listed ? (long long)work[4] : n;
        phase_global_range<PHASE>(tb, ep, sp, cm, ko, src, dst, perm, listed ? retired : nullptr, lo, hi, dt, listed ? b : b - nbA, listed ? nbA : nbB);
    } else {
        fix_keys_range<PHASE>(tb, cm, ko, dst, retired, work[5], n, dt, b - nbA - nbB, (int)gridDim.x - nbA - nbB);
    }
}

// variant 1: the whole classical RK4 step, one thread per marker, in place, coefficients through L1/L2 (reference for the
// two-phase path; leaves the records' k stale)
__global__ void __launch_bounds__(128) k_push_simple(DevTables tb, EquilP ep, SpeciesP sp, Rec* __restrict__ recs, long long n, double dt) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned lanes = __ballot_sync(0xffffffffu, m < n);
    if (m >= n) return;
    Rec r;
    rec_load(recs, m, r);
    double y0[5], k[5], acc[5], y[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) y0[q] = r.y[q];
    const double mu = r.mu, p = r.p;
    int t = r.tri, st = r.st & ~2;   // variant 1 keeps no cached k1
    st |= stage_simple(tb, ep, sp, t, y0[0], y0[1], y0[2], y0[3], y0[4], mu, p, k, lanes);
#pragma unroll
    for (int q = 0; q < 5; ++q) { acc[q] = k[q]; y[q] = fma(0.5 * dt, k[q], y0[q]); }
    st |= stage_simple(tb, ep, sp, t, y[0], y[1], y[2], y[3], y[4], mu, p, k, lanes);
#pragma unroll
    for (int q = 0; q < 5; ++q) { acc[q] = fma(2.0, k[q], acc[q]); y[q] = fma(0.5 * dt, k[q], y0[q]); }
    st |= stage_simple(tb, ep, sp, t, y[0], y[1], y[2], y[3], y[4], mu, p, k, lanes);
#pragma unroll
    for (int q = 0; q < 5; ++q) { acc[q] = fma(2.0, k[q], acc[q]); y[q] = fma(dt, k[q], y0[q]); }
    st |= stage_simple(tb, ep, sp, t, y[0], y[1], y[2], y[3], y[4], mu, p, k, lanes);
    const double h6 = dt / 6.0;
#pragma unroll
    for (int q = 0; q < 5; ++q) r.y[q] = fma(h6, acc[q] + k[q], y0[q]);
    r.y[2] = wrap_phi(tb.tor, r.y[2]);
    r.tri = t; r.st = st;
    rec_store(recs, m, r);
}

// the paper's own kernel boundary (L89): the five time derivatives at the current state, caller order
__global__ void __launch_bounds__(128) k_rhs(DevTables tb, EquilP ep, SpeciesP sp, const Rec* __restrict__ recs, long long n, double* __restrict__ out,
                                             double* __restrict__ stage) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned lanes = __ballot_sync(0xffffffffu, m < n);
    if (m >= n) return;
    Rec r;
    rec_load(recs, m, r);
    int t = r.tri;
    double d[5];
    stage_simple(tb, ep, sp, t, r.y[0], r.y[1], r.y[2], r.y[3], r.y[4], r.mu, r.p, d, lanes);
#pragma unroll
    // caller order.  Five scattered 8-byte stores per marker cost more than the evaluation (23.5 ms per 1e8 markers against 9.4 ms
    // with coalesced stores: each is a read-modify-write of a sector), so with a staging buffer the five values go out as
    // ONE 64-byte record at the caller's index (two full sectors) and k_rhs_unpack turns the records into the five arrays
    if (stage) {
        st256(stage + 8ll * r.id, d[0], d[1], d[2], d[3]);
        st256(stage + 8ll * r.id + 4, d[4], 0.0, 0.0, 0.0);
    } else {
#pragma unroll
        for (int q = 0; q < 5; ++q) out[(long long)q * n + r.id] = d[q];
    }
}
__global__ void __launch_bounds__(256) k_rhs_unpack(const double* __restrict__ stage, long long n, double* __restrict__ out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double d0, d1, d2, d3, d4, z0, z1, z2;
    ld256(stage + 8ll * i, d0, d1, d2, d3);
    ld256(stage + 8ll * i + 4, d4, z0, z1, z2);
    out[i] = d0; out[n + i] = d1; out[2 * n + i] = d2; out[3 * n + i] = d3; out[4 * n + i] = d4;
}

// ============================================================================================ the other G2P kernels
// "pullback treatment", "density calculation", "distribution-function interpolation" - "all these kernels
// rely on the same G2P function; therefore, they have nearly identical structures".  One thread per marker record, fields
// through L1/L2 (the store is cell-sorted after a push, so neighbouring threads read the same coefficient blocks).
// Readings R22-R24: what each kernel computes is the paper's one sentence made concrete.
__device__ __forceinline__ double profile_th(const SpeciesP& sp, double two_inv_w_a, double r) {   // tanh((r - r0) / (w a))
    return 1.0 - 2.0 / (exp((r - sp.r0) * two_inv_w_a) + 1.0);
}
// pullback (L99, Eq.(1), (6)): u <- u - (q/m) A_par,  w <- w + p (q/m) A_par d ln f0/du at the old u,  d ln f0/du = -u / T(r)
__global__ void __launch_bounds__(128) k_pullback(DevTables tb, EquilP ep, SpeciesP sp, Rec* __restrict__ recs, long long n) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned lanes = __ballot_sync(0xffffffffu, m < n);
    if (m >= n) return;
    Rec r;
    rec_load(recs, m, r);
    const int t = locate_walk(tb.bg, tb.geom, r.tri, r.y[0], r.y[1]);
    __syncwarp(lanes);                       // reconverge after the walk (see stage_simple)
    if (t < 0) { r.st |= 1; }
    else {
        Fields f;
        gather_at(tb, t, r.y[0], r.y[1], r.y[2], f);
        const double x = r.y[0] - ep.R0, rr = sqrt(x * x + r.y[1] * r.y[1]);
        const double iT = exp(sp.cT * profile_th(sp, sp.two_inv_wT_a, rr));
        const double shift = sp.qom * f.A;
        r.y[4] += r.p * shift * (-r.y[3] * iT);
        r.y[3] -= shift;
    }
    rec_store(recs, m, r);   // the triangle hint stays (it belongs to the cached next evaluation point, now invalid anyway)
}
// density (L100): value of grid field `which` at every marker, caller order
__global__ void __launch_bounds__(128) k_density_g2p(DevTables tb, int which, const Rec* __restrict__ recs, long long n, double* __restrict__ out) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned lanes = __ballot_sync(0xffffffffu, m < n);
    if (m >= n) return;
    Rec r;
    rec_load(recs, m, r);
    const int t = locate_walk(tb.bg, tb.geom, r.tri, r.y[0], r.y[1]);
    __syncwarp(lanes);                       // reconverge after the walk (see stage_simple)
    Fields f;
    gather_at(tb, t, r.y[0], r.y[1], r.y[2], f);
    out[r.id] = which ? f.A : f.P;
}
// distribution-function interpolation (L101): f0 = n T^-3/2 exp(-(v^2/2 + mu B)/T) at the marker's position and v = u - (q/m) A_par
__global__ void __launch_bounds__(128) k_f_interp(DevTables tb, EquilP ep, SpeciesP sp, const Rec* __restrict__ recs, long long n, double* __restrict__ out) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned lanes = __ballot_sync(0xffffffffu, m < n);
    if (m >= n) return;
    Rec r;
    rec_load(recs, m, r);
    const int t = locate_walk(tb.bg, tb.geom, r.tri, r.y[0], r.y[1]);
    __syncwarp(lanes);                       // reconverge after the walk (see stage_simple)
    Fields f;
    gather_at(tb, t, r.y[0], r.y[1], r.y[2], f);
    Equil<double> e;
    equil_eval<double, true>(ep, r.y[0], r.y[1], e);
    const double thT = profile_th(sp, sp.two_inv_wT_a, e.r), thn = profile_th(sp, sp.two_inv_wn_a, e.r);
    const double iT = exp(sp.cT * thT), dens = exp(-sp.cn * thn);
    const double v = r.y[3] - sp.qom * f.A;
    out[r.id] = dens * iT * sqrt(iT) * exp(-(0.5 * v * v + r.mu * e.B) * iT);
}

// ============================================================================================ particle-to-grid
// Deposition of the marker charges onto the C1 x B-spline basis ("projecting the quantities stored at the
// particle locations ... onto the finite element grid"; L288, L372; reading R25): the transpose of the gather,
//   b[k][v][c] += q_p B_k(phi_p) N_{v,c}(R_p, Z_p),
// N_{v,c} = the element's nodal basis functions.  With F = m . c (m = the 21 monomials at the point), c = c0 - Nul (K c0_5),
// c0 = Aplus d_ref, d_ref = T_J d (k_fields_set), the 18 basis values are N = T_J^T Aplus^T (m - S^T K^T Nul^T m).
// One thread per marker record: its 18 basis values (times the charge) and 4 toroidal weights go into the warp's rows in
// shared memory.  The 72 contributions of a marker (3 nodes x 6 components x 4 planes) go to addresses that depend on its
// cell (triangle, toroidal interval) only, and the store is in cell order after a push: a warp then holds a few runs of
// markers of the same cell; per run the lanes share the 72 sums (lane l takes outputs l, l + 32, l + 64 and walks over the
// run's rows), ONE atomic per address.  An unsorted store degenerates to runs of one marker, i.e. per-marker atomics.
// (History, per 1e8 markers on config 3: five-step segmented shuffle sums of all 72 values 27.8 ms; sums through shared memory
// 14.7 ms; the moments summed per run and mapped once per run instead of per marker 20.4 ms - fewer instructions, but a
// chain of five dependent warp-wide stages per run; this form, with the per-marker map written out: DESIGN.md section 6.)
constexpr int DEP_STRIDE = 23, DEP_WARPS = 4;      // row: 18 basis values x charge, 4 toroidal weights, pad (odd stride: conflict-free)
__global__ void __launch_bounds__(32 * DEP_WARPS) k_deposit(DevTables tb, int P, int quantity, const Rec* __restrict__ recs, long long n, const int* __restrict__ tri,
                                                 const double* __restrict__ RZ, const double* __restrict__ Kmat, long long n_nodes, double* __restrict__ out) {
    constexpr unsigned FULL = 0xffffffffu;
    __shared__ double s_rows[DEP_WARPS][32][DEP_STRIDE];
    __shared__ int s_meta[DEP_WARPS][32][4];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    double (*rows)[DEP_STRIDE] = s_rows[wid];
    int (*meta)[4] = s_meta[wid];
    const long long ngroups = (n + 31) / 32;
    for (long long grp = (long long)blockIdx.x * DEP_WARPS + wid; grp < ngroups; grp += (long long)gridDim.x * DEP_WARPS) {
        const long long mi = grp * 32 + lane;
        int t = -1, k = 0, key = -1;
        double w[4] = {0.0, 0.0, 0.0, 0.0};
        Rec r;
        if (mi < n) {
            rec_load(recs, mi, r);
            t = locate_walk(tb.bg, tb.geom, r.tri, r.y[0], r.y[1]);
        }
        // the lanes leave the walk after different numbers of hops: without this they stay diverged and the warp runs the
        // arithmetic below once per group of lanes (measured: 3.0 times per warp)
        __syncwarp();
        {
            if (t >= 0) {
                const TriGeom g = tb.geom[t];
                double xi, eta, dw[4];
                ref_coords(g, r.y[0], r.y[1], xi, eta);
                k = bspline_weights(tb.tor, r.y[2], w, dw);
                key = t * P + k;
                const double charge = quantity == 0 ? r.y[4] : r.y[4] * r.y[3];
                // charge x monomials xi^i eta^j at j-major index off_j + i
                double m[21];
                {
                    double xp[6], ep[6];
                    xp[0] = 1.0; ep[0] = charge;
#pragma unroll
                    for (int i = 1; i < 6; ++i) { xp[i] = xp[i - 1] * xi; ep[i] = ep[i - 1] * eta; }
                    int idx = 0;
#pragma unroll
                    for (int j = 0; j < 6; ++j)
#pragma unroll
                        for (int i = 0; i < 6 - j; ++i) m[idx++] = xp[i] * ep[j];
                }
                double y0 = 0.0, y1 = 0.0, y2 = 0.0;
#pragma unroll
                for (int i = 0; i < 21; ++i) { y0 = fma(c_Nul[i * 3], m[i], y0); y1 = fma(c_Nul[i * 3 + 1], m[i], y1); y2 = fma(c_Nul[i * 3 + 2], m[i], y2); }
                const double* K = Kmat + (long long)t * 18;
                // the six degree-5 monomials sit at 5, 10, 14, 17, 19, 20
                m[5] -= fma(y0, K[0], fma(y1, K[6], y2 * K[12]));
                m[10] -= fma(y0, K[1], fma(y1, K[7], y2 * K[13]));
                m[14] -= fma(y0, K[2], fma(y1, K[8], y2 * K[14]));
                m[17] -= fma(y0, K[3], fma(y1, K[9], y2 * K[15]));
                m[19] -= fma(y0, K[4], fma(y1, K[10], y2 * K[16]));
                m[20] -= fma(y0, K[5], fma(y1, K[11], y2 * K[17]));
                const int n0 = tri[3 * t], n1 = tri[3 * t + 1], n2 = tri[3 * t + 2];
                meta[lane][0] = n0; meta[lane][1] = n1; meta[lane][2] = n2;
                const double x0 = RZ[2 * n0], yy0 = RZ[2 * n0 + 1];
                const double j11 = RZ[2 * n1] - x0, j21 = RZ[2 * n1 + 1] - yy0, j12 = RZ[2 * n2] - x0, j22 = RZ[2 * n2 + 1] - yy0;
                const double t11 = j11 * j11, t12 = j11 * j12, t22 = j12 * j12, u11 = 2.0 * j11 * j21, u12 = fma(j11, j22, j21 * j12), u22 = 2.0 * j12 * j22,
                             v11 = j21 * j21, v12 = j21 * j22, v22 = j22 * j22;
#pragma unroll
                for (int v = 0; v < 3; ++v) {
                    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0, a4 = 0.0, a5 = 0.0;      // six independent chains
#pragma unroll
                    for (int i = 0; i < 21; ++i) {
                        a0 = fma(c_Aplus[i * 18 + 6 * v + 0], m[i], a0); a1 = fma(c_Aplus[i * 18 + 6 * v + 1], m[i], a1);
                        a2 = fma(c_Aplus[i * 18 + 6 * v + 2], m[i], a2); a3 = fma(c_Aplus[i * 18 + 6 * v + 3], m[i], a3);
                        a4 = fma(c_Aplus[i * 18 + 6 * v + 4], m[i], a4); a5 = fma(c_Aplus[i * 18 + 6 * v + 5], m[i], a5);
                    }
                    rows[lane][6 * v + 0] = a0;
                    rows[lane][6 * v + 1] = fma(j11, a1, j12 * a2);
                    rows[lane][6 * v + 2] = fma(j21, a1, j22 * a2);
                    rows[lane][6 * v + 3] = fma(t11, a3, fma(t12, a4, t22 * a5));
                    rows[lane][6 * v + 4] = fma(u11, a3, fma(u12, a4, u22 * a5));
                    rows[lane][6 * v + 5] = fma(v11, a3, fma(v12, a4, v22 * a5));
                }
            }
        }
#pragma unroll
        for (int pa = 0; pa < 4; ++pa) rows[lane][18 + pa] = w[pa];
        meta[lane][3] = k;
        const int prevk = __shfl_up_sync(FULL, key, 1);
        unsigned starts = __ballot_sync(FULL, lane == 0 || prevk != key);
        const unsigned inside = __ballot_sync(FULL, key >= 0);
        __syncwarp();
        while (starts) {
            const int b = __ffs(starts) - 1;
            starts &= starts - 1;
            const int e = starts ? __ffs(starts) - 1 : 32;
            if (!((inside >> b) & 1u)) continue;
            const int kk = meta[b][3];
#pragma unroll
            for (int pass = 0; pass < 3; ++pass) {
                const int o = lane + 32 * pass;           // output pa * 18 + (6 v + c)
                if (o < 72) {
                    const int pa = o / 18, q = o - 18 * pa, v = q / 6, c = q - 6 * v;
                    double s0 = 0.0, s1 = 0.0;
                    int pp = b;
                    for (; pp + 1 < e; pp += 2) { s0 = fma(rows[pp][q], rows[pp][18 + pa], s0); s1 = fma(rows[pp + 1][q], rows[pp + 1][18 + pa], s1); }
                    if (pp < e) s0 = fma(rows[pp][q], rows[pp][18 + pa], s0);
                    int pl = kk - 1 + pa;
                    if (pl < 0) pl += P; else if (pl >= P) pl -= P;
                    atomicAdd(out + ((long long)pl * n_nodes + meta[b][v]) * 6 + c, s0 + s1);
                }
            }
        }
        __syncwarp();
    }
}

// ============================================================================================ phase kernel: helpers
// markers that left their staged block during a phase: positions in the cell order, finished by k_phase_global
// and markers whose NEXT evaluation point left the staged geometry (record done, triangle and sort key still to be found by
// k_fix_keys): the same array, filled from its end
struct RetireList {
    int* list;      // [n]
    int* count;     // device counters: [0] retired, [1] keys to fix
    int n;
};

}  // namespace trimeg
#include "trimeg_ws.cuh"
#include "trimeg_gather.cuh"
namespace trimeg {

// ============================================================================================ counting sort by cell
// exclusive scan of int counts, three passes over chunks of SCAN_CHUNK
constexpr int SCAN_THREADS = 512, SCAN_ITEMS = 8, SCAN_CHUNK = SCAN_THREADS * SCAN_ITEMS;
__device__ __forceinline__ int block_exclusive_scan(int v, int* total) {   // SCAN_THREADS threads
    __shared__ int warp_sums[SCAN_THREADS / 32];
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) warp_sums[wid] = x;
    __syncthreads();
    if (wid == 0) {
        int s = lane < SCAN_THREADS / 32 ? warp_sums[lane] : 0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += y; }
        if (lane < SCAN_THREADS / 32) warp_sums[lane] = s;
    }
    __syncthreads();
    int base = wid ? warp_sums[wid - 1] : 0;
    if (total) *total = warp_sums[SCAN_THREADS / 32 - 1];
    __syncthreads();
    return base + x - v;
}
// `skip`: null, or a device flag: the scan is skipped unless *skip == 2 (trimeg_gather's path choice on the device)
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_reduce(const int* __restrict__ in, long long n, int* __restrict__ sums, const int* __restrict__ skip = nullptr) {
    if (skip && *skip != 2) return;
    long long base = (long long)blockIdx.x * SCAN_CHUNK + (long long)threadIdx.x * SCAN_ITEMS;
    int s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) if (base + i < n) s += in[base + i];
    int tot;
    block_exclusive_scan(s, &tot);
    if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_sums(int* __restrict__ sums, int nb, const int* __restrict__ skip = nullptr) {   // single block
    __shared__ int carry;
    if (skip && *skip != 2) return;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nb; b0 += SCAN_THREADS) {
        int i = b0 + threadIdx.x, v = i < nb ? sums[i] : 0, tot;
        int ex = block_exclusive_scan(v, &tot);
        int c = carry;
        if (i < nb) sums[i] = ex + c;
        __syncthreads();
        if (threadIdx.x == 0) carry = c + tot;
        __syncthreads();
    }
}
// writes the exclusive offsets and clears the histogram and the fill counters for the next pass
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(int* __restrict__ in, long long n, const int* __restrict__ sums,
                                                             int* __restrict__ out, int* __restrict__ fill, const int* __restrict__ skip = nullptr) {
    if (skip && *skip != 2) return;
    long long base = (long long)blockIdx.x * SCAN_CHUNK + (long long)threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) { v[i] = base + i < n ? in[base + i] : 0; s += v[i]; }
    int ex = block_exclusive_scan(s, nullptr) + sums[blockIdx.x];
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) {
        if (base + i < n) { out[base + i] = ex; in[base + i] = 0; fill[base + i] = 0; }
        ex += v[i];
    }
}
#ifndef TRIMEG_SORT_PER_THREAD
#define TRIMEG_SORT_PER_THREAD 4
#endif
constexpr int SORT_PER_THREAD = TRIMEG_SORT_PER_THREAD;
// permutation: perm[position in cell order] = record index (4-byte scattered writes)
__global__ void __launch_bounds__(256) k_sort_perm(long long n, const int* __restrict__ keys, const int* __restrict__ offs, int* __restrict__ fill,
                                                   int* __restrict__ perm) {
    // SORT_PER_THREAD records per thread: the chain key -> (offset, fill counter) -> store is three dependent memory round trips,
    // so the kernel's time is set by how many of them a thread keeps in flight (per 1e8 records: 1 per thread 0.85 ms, 4: 0.57, 8: 0.60, 16: 0.75)
    constexpr int W = SORT_PER_THREAD;
    const long long m0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * W;
    if (m0 >= n) return;
    int key[W];
    if (m0 + W <= n) {
#pragma unroll
        for (int q = 0; q < W; q += 4) {
            const int4 k4 = *reinterpret_cast<const int4*>(keys + m0 + q);
            key[q] = k4.x; key[q + 1] = k4.y; key[q + 2] = k4.z; key[q + 3] = k4.w;
        }
    } else {
#pragma unroll
        for (int q = 0; q < W; ++q) key[q] = m0 + q < n ? keys[m0 + q] : -1;
    }
    int off[W], rank[W];
#pragma unroll
    for (int q = 0; q < W; ++q) if (key[q] >= 0) { off[q] = offs[key[q]]; rank[q] = atomicAdd(fill + key[q], 1); }
#pragma unroll
    for (int q = 0; q < W; ++q) if (key[q] >= 0) perm[(long long)off[q] + rank[q]] = (int)(m0 + q);
}
// per phase: acc[0] += markers left to the follow-up kernel
__global__ void k_accumulate_stat(const int* __restrict__ v, unsigned long long* __restrict__ acc) { atomicAdd(acc, (unsigned long long)*v); }

// ============================================================================================ DFMA micro-benchmark
__global__ void __launch_bounds__(512) k_dfma(double* out, int iters, double a, double b) {
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

// the same loop with the operands a real evaluation has: KIND 1: three different register pairs per DFMA (accumulator,
// multiplier, addend); KIND 2: Horner-like, one multiplier shared by the eight chains, addends different.  The values come
// from memory so that nothing folds.
template <int KIND>
__global__ void __launch_bounds__(512) k_dfma_mix(const double* __restrict__ in, double* out, int iters) {
    double x[8], y[8], z[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) { x[q] = in[q] + threadIdx.x; y[q] = in[8 + q] + 1e-13 * threadIdx.x; z[q] = in[16 + q] * (1.0 + threadIdx.x); }   // per-thread values: vector registers
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int q = 0; q < 8; ++q) x[q] = fma(x[q], KIND == 1 ? y[q] : y[0], z[q]);
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x[0] + x[1]) + (x[2] + x[3])) + ((x[4] + x[5]) + (x[6] + x[7]));
}

}  // namespace trimeg
