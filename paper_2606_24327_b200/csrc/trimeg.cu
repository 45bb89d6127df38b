// C-ABI implementation of include/trimeg.h: context, setup kernels, gather, sort and the RK4 push.
// Compiled for sm_100a only.  See DESIGN.md for the data layout and the roofline of each kernel.
#include "../../include/trimeg.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "trimeg_host_setup.hpp"
#include "trimeg_math.cuh"
#include "trimeg_tile.cuh"

using namespace trimeg;

// ============================================================================================ device tables
struct MarkerSoA {           // one of two buffers living in the caller's scratch
    double *R, *Z, *phi, *u, *w, *mu, *p;
    int *tri, *status, *id;
};
struct DevTables {
    const TriGeom* geom;     // [T]
    const double* coef;      // [T][P+3+2*PLANE_PAD][21][2]; see PLANE_PAD in trimeg_math.cuh
    BoxGrid bg;
    TorP tor;
    int T;
    long long tri_stride;    // doubles per triangle = (P+3+2*PLANE_PAD)*42
};

// tiled push configuration: patches of 8 triangles + halo (36 slots), windows of 4 toroidal intervals (+1 each side), ring of 2 staged blocks,
// 16 independent warps per CTA, one CTA per SM
using Tile = TileCfg<8, 36, 4, 16>;
// cell numbering used by the sort: super-cell (patch, window) major, then triangle within the patch, then interval
struct CellMap {
    int P, nwin;
    __host__ __device__ __forceinline__ int cell(int t, int k) const {
        int patch = t / Tile::TP, tl = t - patch * Tile::TP, wdw = k / Tile::WK, kl = k - wdw * Tile::WK;
        return ((patch * nwin + wdw) * Tile::TP + tl) * Tile::WK + kl;
    }
};

__constant__ double c_Aplus[21 * 18];
__constant__ double c_Nul[21 * 3];

// ============================================================================================ setup kernels
// fields_set: nodal DOFs -> per-triangle reference-frame polynomial coefficients, for one field.
// One thread per (triangle, plane).  c = c0 - Nul (K c0_5),  c0 = Aplus d_ref,  d_ref = DOFs pulled back with J.
__global__ void k_fields_set(int T, int P, int which, const int* __restrict__ tri, const double* __restrict__ RZ,
                             const double* __restrict__ Kmat, const double* __restrict__ dof, long long n_nodes,
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
    const int NPP = P + 3 + 2 * PLANE_PAD;
    long long tri_stride = (long long)NPP * PLANE_STRIDE;
    double* base = coef + (long long)t * tri_stride;
    int slots[3];
#pragma unroll
    for (int s = 0; s < 3; ++s) { int pp = k + 1 + PLANE_PAD + (s - 1) * P; slots[s] = (pp >= 0 && pp < NPP) ? pp : -1; }
#pragma unroll
    for (int i = 0; i < 21; ++i) {
        double v = c[i] - (c_Nul[i * 3] * z[0] + c_Nul[i * 3 + 1] * z[1] + c_Nul[i * 3 + 2] * z[2]);
#pragma unroll
        for (int s = 0; s < 3; ++s) if (slots[s] >= 0) base[(long long)slots[s] * PLANE_STRIDE + 2 * i + which] = v;
    }
}

// ============================================================================================ gather / push (simple variant)
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
    gather_cell(ld, xi, eta, w, dw, acc);
    to_fields(g, acc, f);
}

__global__ void __launch_bounds__(256) k_gather(DevTables tb, long long n, const double* __restrict__ R, const double* __restrict__ Z,
                                                const double* __restrict__ phi, double* __restrict__ out, int* __restrict__ tri_out) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    double r = R[m], z = Z[m];
    int t = locate_box(tb.bg, tb.geom, r, z);
    Fields f;
    gather_at(tb, t, r, z, phi[m], f);
    out[m] = f.P; out[n + m] = f.PR; out[2 * n + m] = f.PZ; out[3 * n + m] = f.Pp;
    out[4 * n + m] = f.A; out[5 * n + m] = f.AR; out[6 * n + m] = f.AZ; out[7 * n + m] = f.Ap;
    if (tri_out) tri_out[m] = t < 0 ? -1 : tb.geom[t].orig;
}

// one RK stage evaluation for one marker, fields through L1/L2; updates the triangle hint
__device__ __forceinline__ int stage_simple(const DevTables& tb, const EquilP& ep, const SpeciesP& sp, int& t, double R, double Z,
                                            double phi, double u, double w, double mu, double p, double d[5]) {
    t = locate_walk(tb.bg, tb.geom, t, R, Z);
    Fields f;
    gather_at(tb, t, R, Z, phi, f);
    rhs_eval(ep, sp, R, Z, u, w, mu, p, f, d);
    return t < 0;
}

__global__ void __launch_bounds__(128) k_push_simple(DevTables tb, EquilP ep, SpeciesP sp, MarkerSoA s, long long n, double dt) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    double y0[5] = {s.R[m], s.Z[m], s.phi[m], s.u[m], s.w[m]};
    double mu = s.mu[m], p = s.p[m];
    int t = s.tri[m], st = s.status[m];
    double k[5], acc[5], y[5];
    st |= stage_simple(tb, ep, sp, t, y0[0], y0[1], y0[2], y0[3], y0[4], mu, p, k);
    int t_home = t;
#pragma unroll
    for (int q = 0; q < 5; ++q) { acc[q] = k[q]; y[q] = fma(0.5 * dt, k[q], y0[q]); }
    st |= stage_simple(tb, ep, sp, t, y[0], y[1], y[2], y[3], y[4], mu, p, k);
#pragma unroll
    for (int q = 0; q < 5; ++q) { acc[q] = fma(2.0, k[q], acc[q]); y[q] = fma(0.5 * dt, k[q], y0[q]); }
    st |= stage_simple(tb, ep, sp, t, y[0], y[1], y[2], y[3], y[4], mu, p, k);
#pragma unroll
    for (int q = 0; q < 5; ++q) { acc[q] = fma(2.0, k[q], acc[q]); y[q] = fma(dt, k[q], y0[q]); }
    st |= stage_simple(tb, ep, sp, t, y[0], y[1], y[2], y[3], y[4], mu, p, k);
    const double h6 = dt / 6.0;
#pragma unroll
    for (int q = 0; q < 5; ++q) y[q] = fma(h6, acc[q] + k[q], y0[q]);
    double ph = fma(-tb.tor.period, floor(y[2] * tb.tor.inv_period), y[2]);
    if (ph < 0.0) ph += tb.tor.period;
    if (ph >= tb.tor.period) ph -= tb.tor.period;
    s.R[m] = y[0]; s.Z[m] = y[1]; s.phi[m] = ph; s.u[m] = y[3]; s.w[m] = y[4];
    s.tri[m] = t >= 0 ? t : t_home;
    s.status[m] = st;
}


// queues of retired markers, one per RK stage at which the marker left the staged block (so that the finish kernel's
// remaining-stage loop is warp-uniform); SoA with capacity cap per sub-queue, entry e = stage * cap + slot
struct RetireQueue {
    double* y;      // [5][4 cap] stage position
    double* acc;    // [5][4 cap] weighted sum of the k's so far
    int* m;         // [4 cap] marker index (position in the destination store)
    int* st;        // [4 cap] status so far
    int* count;     // [4] device counters
    int cap;
};
// where the sort key of the updated marker goes (the next step's counting sort is fused into the push)
struct KeyOut {
    int* keys;      // [n] cell of the updated position, indexed like the destination store
    int* hist;      // [ncell + 2] histogram of the keys
    int ncell;
    int enabled;
};
__device__ __forceinline__ double wrap_phi(const TorP& tp, double phi) {
    double ph = fma(-tp.period, floor(phi * tp.inv_period), phi);
    if (ph < 0.0) ph += tp.period;
    if (ph >= tp.period) ph -= tp.period;
    return ph;
}
// final store of one marker: state, triangle of the updated position, status, and (if enabled) its sort key
__device__ __forceinline__ void store_marker(const DevTables& tb, const CellMap& cm, const KeyOut& ko, const MarkerSoA& d, long long j, const double y[5],
                                             double ph, int t, int st) {
    d.R[j] = y[0]; d.Z[j] = y[1]; d.phi[j] = ph; d.u[j] = y[3]; d.w[j] = y[4];
    d.tri[j] = t; d.status[j] = st;
    if (ko.enabled) {
        double sf;
        int k = toroidal_interval(tb.tor, ph, sf);
        int key = t < 0 ? ko.ncell : cm.cell(t, k);
        ko.keys[j] = key;
        atomicAdd(ko.hist + key, 1);
    }
}

// markers outside the mesh (sorted behind the last cell): same arithmetic through the simple path
__global__ void __launch_bounds__(128) k_push_lost(DevTables tb, EquilP ep, SpeciesP sp, MarkerSoA src, MarkerSoA dst, const int* __restrict__ perm,
                                                   KeyOut ko, CellMap cm, const int* __restrict__ first, long long n, double dt) {
    long long m0 = *first;
    for (long long m = m0 + (long long)blockIdx.x * blockDim.x + threadIdx.x; m < n; m += (long long)gridDim.x * blockDim.x) {
        const long long ms = perm ? (long long)perm[m] : m;
        double y0[5] = {src.R[ms], src.Z[ms], src.phi[ms], src.u[ms], src.w[ms]};
        double mu = src.mu[ms], p = src.p[ms];
        int t = src.tri[ms], st = src.status[ms];
        if (perm) { dst.mu[m] = mu; dst.p[m] = p; dst.id[m] = src.id[ms]; }
        double k[5], acc[5], y[5];
        st |= stage_simple(tb, ep, sp, t, y0[0], y0[1], y0[2], y0[3], y0[4], mu, p, k);
#pragma unroll
        for (int q = 0; q < 5; ++q) { acc[q] = k[q]; y[q] = fma(0.5 * dt, k[q], y0[q]); }
        st |= stage_simple(tb, ep, sp, t, y[0], y[1], y[2], y[3], y[4], mu, p, k);
#pragma unroll
        for (int q = 0; q < 5; ++q) { acc[q] = fma(2.0, k[q], acc[q]); y[q] = fma(0.5 * dt, k[q], y0[q]); }
        st |= stage_simple(tb, ep, sp, t, y[0], y[1], y[2], y[3], y[4], mu, p, k);
#pragma unroll
        for (int q = 0; q < 5; ++q) { acc[q] = fma(2.0, k[q], acc[q]); y[q] = fma(dt, k[q], y0[q]); }
        st |= stage_simple(tb, ep, sp, t, y[0], y[1], y[2], y[3], y[4], mu, p, k);
        const double h6 = dt / 6.0;
#pragma unroll
        for (int q = 0; q < 5; ++q) y[q] = fma(h6, acc[q] + k[q], y0[q]);
        const double ph = wrap_phi(tb.tor, y[2]);
        t = locate_walk(tb.bg, tb.geom, t, y[0], y[1]);
        store_marker(tb, cm, ko, dst, m, y, ph, t, st);
    }
}

__global__ void __launch_bounds__(128) k_rhs(DevTables tb, EquilP ep, SpeciesP sp, MarkerSoA s, long long n, double* __restrict__ out) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    int t = s.tri[m];
    double d[5];
    stage_simple(tb, ep, sp, t, s.R[m], s.Z[m], s.phi[m], s.u[m], s.w[m], s.mu[m], s.p[m], d);
    long long o = s.id[m];
#pragma unroll
    for (int q = 0; q < 5; ++q) out[(long long)q * n + o] = d[q];
}


// ============================================================================================ tiled push (variant 0)
// (re)fill ring entry b with the next non-empty super-cell; executed by one whole warp.  The entry's mbarrier completes
// when the TMA bytes have landed (or at once, with sc = -1, when the work list is exhausted).
template <class C>
__device__ __forceinline__ void tile_refill(unsigned char* smem, int b, const DevTables& tb, const TileTables& tt, int* work_counter, int lane) {
    constexpr unsigned FULL = 0xffffffffu;
    double* coef = reinterpret_cast<double*>(smem + C::BLOCK_BYTES * b);
    SlotGeom* sgeom = reinterpret_cast<SlotGeom*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES);
    BlockCtrl* ctl = reinterpret_cast<BlockCtrl*>(smem + C::OFF_CTRL) + b;
    unsigned long long* mbar = reinterpret_cast<unsigned long long*>(smem + C::OFF_CTRL + 64 * C::NBUF) + 2 * b;
    int sc = 0, begin = 0, end = 0;
    for (;;) {
        if (lane == 0) sc = atomicAdd(work_counter, 1);
        sc = __shfl_sync(FULL, sc, 0);
        if (sc >= tt.nsc) { sc = -1; break; }
        begin = tt.offs[(long long)sc * C::CPS]; end = tt.offs[(long long)(sc + 1) * C::CPS];
        if (begin != end) break;
    }
    if (sc < 0) {
        if (lane == 0) { ctl->sc = -1; ctl->left = 0; __threadfence_block(); asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(mbar)) : "memory"); }
        return;
    }
    const int patch = sc / tt.nwin, k0 = (sc - patch * tt.nwin) * C::WK;
    const int ns = tt.nslots[patch];
    const int* pslots = tt.slots + (long long)patch * C::SMAX;
    if (lane == 0) { ctl->sc = sc; ctl->begin = begin; ctl->end = end; ctl->next = begin; ctl->left = 0; ctl->ns = ns; ctl->patch = patch; ctl->k0 = k0; }
    int cnt = 0;
    for (int sl = lane; sl < ns; sl += 32) {
        int t = pslots[sl];
        SlotGeom g;
        if (t >= 0) {
            const TriGeom tg = tb.geom[t];
            g.v0x = tg.v0x; g.v0y = tg.v0y; g.a11 = tg.a11; g.a12 = tg.a12; g.a21 = tg.a21; g.a22 = tg.a22;
            const short* nb = tt.nbr + ((long long)patch * C::SMAX + sl) * 4;
            g.nbr[0] = nb[0]; g.nbr[1] = nb[1]; g.nbr[2] = nb[2]; g.nbr[3] = -1;
            cnt++;
        } else {
            g.v0x = g.v0y = 1e300; g.a11 = g.a12 = g.a21 = g.a22 = 0.0; g.nbr[0] = g.nbr[1] = g.nbr[2] = g.nbr[3] = -1;
        }
        g.tri = t; g.pad = 0;
        sgeom[sl] = g;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(FULL, cnt, o);
    __threadfence_block();
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // earlier generic accesses of this block vs. the async writes
    __syncwarp();
    if (lane == 0) mbar_expect_tx(mbar, (unsigned)(cnt * C::SLOT_DOUBLES * sizeof(double)));
    __syncwarp();
    for (int sl = lane; sl < ns; sl += 32) {
        int t = pslots[sl];
        if (t >= 0)
            tma_bulk_g2s(coef + (size_t)sl * C::SLOT_DOUBLES, tb.coef + (long long)t * tb.tri_stride + (long long)k0 * PLANE_STRIDE,
                         (unsigned)(C::SLOT_DOUBLES * sizeof(double)), mbar);
    }
}

// slot-space edge walk inside the staged block: returns the slot containing (R, Z) or -1 (left the staged set / hop cap)
__device__ __forceinline__ int slot_walk(const SlotGeom* __restrict__ sgeom, int sl, double R, double Z, double& xi, double& eta) {
    if (sl < 0) return -1;
    for (int hop = 0; hop < 16; ++hop) {
        const SlotGeom& g = sgeom[sl];
        double dx = R - g.v0x, dy = Z - g.v0y;
        xi = fma(g.a11, dx, g.a12 * dy);
        eta = fma(g.a21, dx, g.a22 * dy);
        double l0 = 1.0 - xi - eta;
        if (fmin(fmin(xi, eta), l0) >= INSIDE_TOL) return sl;
        int e = (eta <= xi && eta <= l0) ? 0 : ((l0 <= xi) ? 1 : 2);
        sl = g.nbr[e];
        if (sl < 0) return -1;
    }
    return -1;
}

// One RK4 step for the markers of one super-cell after another.  Markers are read from `src` through the sort
// permutation (perm[j] = position in src of the marker that belongs at position j of the cell-sorted order; null =
// src is already in that order and src == dst) and written to dst[j]: the sort's data movement is fused into the push.
template <class C>
__global__ void __launch_bounds__(C::NTHREADS, 1)
k_push_tiled(DevTables tb, TileTables tt, EquilP ep, SpeciesP sp, MarkerSoA src, MarkerSoA dst, const int* __restrict__ perm, RetireQueue rq,
             KeyOut ko, CellMap cm, double dt, int* __restrict__ work_counter) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    BlockCtrl* ctl_all = reinterpret_cast<BlockCtrl*>(smem + C::OFF_CTRL);
    unsigned long long* mbar_all = reinterpret_cast<unsigned long long*>(smem + C::OFF_CTRL + 64 * C::NBUF);
    if (tid == 0) {
        for (int b = 0; b < C::NBUF; ++b) mbar_init(mbar_all + 2 * b, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (wid == 0) {
        for (int b = 0; b < C::NBUF; ++b) tile_refill<C>(smem, b, tb, tt, work_counter, lane);
    }
    const int P = tb.tor.P;
    const double h2 = 0.5 * dt, h6 = dt / 6.0;
    constexpr unsigned FULL = 0xffffffffu;

    // every warp walks the ring in the same order; the last warp to leave an entry refills it (no block-wide barrier)
    for (unsigned it = 0;; ++it) {
        const int b = it % C::NBUF;
        mbar_wait(mbar_all + 2 * b, (it / C::NBUF) & 1);
        BlockCtrl* ctl = ctl_all + b;
        if (ctl->sc < 0) break;
        const double* coef = reinterpret_cast<const double*>(smem + C::BLOCK_BYTES * b);
        const SlotGeom* sgeom = reinterpret_cast<const SlotGeom*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES);
        const int end = ctl->end, patch = ctl->patch, k0 = ctl->k0, ns = ctl->ns;
        int* sh_next = &ctl->next;

        // ---- each warp grabs chunks of 32 markers until the super-cell is drained
        for (;;) {
            int chunk = 0;
            if (lane == 0) chunk = atomicAdd(sh_next, 32);
            chunk = __shfl_sync(FULL, chunk, 0);
            if (chunk >= end) break;
            const int m = chunk + lane;
            bool alive = m < end;   // this lane still integrates a marker
            double y0[5], y[5], acc[5], mu = 0.0, pw = 0.0;
            int st = 0, cur = -1, tri_last = -1;
            if (alive) {
                const long long ms = perm ? (long long)perm[m] : (long long)m;
                y0[0] = src.R[ms]; y0[1] = src.Z[ms]; y0[2] = src.phi[ms]; y0[3] = src.u[ms]; y0[4] = src.w[ms];
                mu = src.mu[ms]; pw = src.p[ms]; st = src.status[ms];
                tri_last = src.tri[ms];
                if (perm) { dst.mu[m] = mu; dst.p[m] = pw; dst.id[m] = src.id[ms]; }
                int sl = tri_last - patch * C::TP;
                if (sl >= 0 && sl < C::TP) cur = sl;
                else {   // drifted since the last sort: look for the triangle in the halo
                    for (int q = C::TP; q < ns; ++q) if (sgeom[q].tri == tri_last) { cur = q; break; }
                }
            } else {
#pragma unroll
                for (int q = 0; q < 5; ++q) y0[q] = 0.0;
            }
#pragma unroll
            for (int q = 0; q < 5; ++q) { y[q] = y0[q]; acc[q] = 0.0; }

#pragma unroll 1
            for (int stage = 0; stage < 4; ++stage) {
                if (alive) {
                    double xi = 0.0, eta = 0.0, sf;
                    int sl = slot_walk(sgeom, cur, y[0], y[1], xi, eta);
                    int k = toroidal_interval(tb.tor, y[2], sf);
                    int dk = k - k0;
                    if (dk > P / 2) dk -= P; else if (dk < -(P / 2)) dk += P;
                    int lk = dk + C::HK;
                    bool in_tile = sl >= 0 && lk >= 0 && lk < C::NW;
                    double d[5];
                    if (in_tile) {
                        // -- gather from the staged block (each lane its own marker)
                        cur = sl;
                        const SlotGeom& g = sgeom[sl];
                        tri_last = g.tri;
                        double w[4], dw[4], g8[8];
                        bspline_from_s(tb.tor, sf, w, dw);
                        LdShared ld{smem_u32(coef + (size_t)sl * C::SLOT_DOUBLES + (size_t)lk * PLANE_STRIDE)};
                        gather_cell(ld, xi, eta, w, dw, g8);
                        Fields fo;
                        fo.P = g8[0]; fo.PR = fma(g.a11, g8[1], g.a21 * g8[2]); fo.PZ = fma(g.a12, g8[1], g.a22 * g8[2]); fo.Pp = g8[3];
                        fo.A = g8[4]; fo.AR = fma(g.a11, g8[5], g.a21 * g8[6]); fo.AZ = fma(g.a12, g8[5], g.a22 * g8[6]); fo.Ap = g8[7];
                        rhs_eval(ep, sp, y[0], y[1], y[3], y[4], mu, pw, fo, d);
                    } else {
                        // left the staged block: retire (the follow-up kernel finishes this step from here)
                        int slot = atomicAdd(rq.count + stage, 1);
                        if (slot < rq.cap) {
                            const size_t e = (size_t)stage * rq.cap + slot, tot = 4 * (size_t)rq.cap;
#pragma unroll
                            for (int q = 0; q < 5; ++q) { rq.y[q * tot + e] = y[q]; rq.acc[q * tot + e] = acc[q]; }
                            rq.m[e] = m;
                            rq.st[e] = st;
                            alive = false;
                        } else {   // queue full (pathological): evaluate in place through the global tables
                            int t = tri_last;
                            st |= stage_simple(tb, ep, sp, t, y[0], y[1], y[2], y[3], y[4], mu, pw, d);
                            if (t >= 0) tri_last = t;
                        }
                    }
                    if (alive) {
                        const double wgt = (stage == 0 || stage == 3) ? 1.0 : 2.0;
                        const double hs = stage == 2 ? dt : h2;
#pragma unroll
                        for (int q = 0; q < 5; ++q) { acc[q] = fma(wgt, d[q], acc[q]); y[q] = fma(hs, d[q], y0[q]); }
                    }
                }
            }
            if (alive) {
#pragma unroll
                for (int q = 0; q < 5; ++q) y[q] = fma(h6, acc[q], y0[q]);
                const double ph = wrap_phi(tb.tor, y[2]);
                // triangle of the updated position: staged walk, else the global walk (rare)
                double xi, eta;
                int sl = slot_walk(sgeom, cur, y[0], y[1], xi, eta);
                int t = sl >= 0 ? sgeom[sl].tri : locate_walk(tb.bg, tb.geom, tri_last, y[0], y[1]);
                store_marker(tb, cm, ko, dst, m, y, ph, t, st);
            }
        }
        // leave the entry; the last warp out refills it with the next super-cell
        __syncwarp();
        int last = 0;
        if (lane == 0) { __threadfence_block(); last = atomicAdd(&ctl->left, 1) == C::NWARPS - 1; }
        last = __shfl_sync(FULL, last, 0);
        if (last) { __threadfence_block(); tile_refill<C>(smem, b, tb, tt, work_counter, lane); }
    }
}

// finish the step of the retired markers through the global tables (same arithmetic as the simple path).
// Sub-queue q holds the markers that left at stage q; each is padded to whole warps so that the stage loop is warp-uniform.
__global__ void __launch_bounds__(128) k_push_finish(DevTables tb, EquilP ep, SpeciesP sp, MarkerSoA src, MarkerSoA dst, const int* __restrict__ perm,
                                                     RetireQueue rq, KeyOut ko, CellMap cm, double dt) {
    int cnt[4], start[5];
    start[0] = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) { cnt[q] = min(rq.count[q], rq.cap); start[q + 1] = start[q] + ((cnt[q] + 31) & ~31); }
    const double h2 = 0.5 * dt, h6 = dt / 6.0;
    const size_t tot = 4 * (size_t)rq.cap;
    for (int v = blockIdx.x * blockDim.x + threadIdx.x; v < start[4]; v += gridDim.x * blockDim.x) {
        const int q = v >= start[3] ? 3 : (v >= start[2] ? 2 : (v >= start[1] ? 1 : 0));
        const int i = v - start[q];
        if (i >= cnt[q]) continue;
        const size_t e = (size_t)q * rq.cap + i;
        const int m = rq.m[e];
        int st = rq.st[e];
        const long long ms = perm ? (long long)perm[m] : (long long)m;
        int t = src.tri[ms];
        double y0[5] = {src.R[ms], src.Z[ms], src.phi[ms], src.u[ms], src.w[ms]};
        const double mu = src.mu[ms], p = src.p[ms];
        double y[5], acc[5], d[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) { y[c] = rq.y[c * tot + e]; acc[c] = rq.acc[c * tot + e]; }
        for (int stage = q; stage < 4; ++stage) {
            st |= stage_simple(tb, ep, sp, t, y[0], y[1], y[2], y[3], y[4], mu, p, d);
            const double wgt = (stage == 0 || stage == 3) ? 1.0 : 2.0;
            const double hs = stage == 2 ? dt : h2;
#pragma unroll
            for (int c = 0; c < 5; ++c) { acc[c] = fma(wgt, d[c], acc[c]); y[c] = fma(hs, d[c], y0[c]); }
        }
#pragma unroll
        for (int c = 0; c < 5; ++c) y[c] = fma(h6, acc[c], y0[c]);
        const double ph = wrap_phi(tb.tor, y[2]);
        t = locate_walk(tb.bg, tb.geom, t, y[0], y[1]);
        store_marker(tb, cm, ko, dst, m, y, ph, t, st);
    }
}

// ============================================================================================ marker store / sort
__global__ void k_bind(MarkerSoA s, long long n, const double* R, const double* Z, const double* phi, const double* u,
                       const double* w, const double* mu, const double* p) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    s.R[m] = R[m]; s.Z[m] = Z[m]; s.phi[m] = phi[m]; s.u[m] = u[m]; s.w[m] = w[m]; s.mu[m] = mu[m]; s.p[m] = p[m];
    s.tri[m] = -1; s.status[m] = 0; s.id[m] = (int)m;
}
__global__ void k_unsort(MarkerSoA s, long long n, double* R, double* Z, double* phi, double* u, double* w, int* status) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    long long o = s.id[m];
    if (R) R[o] = s.R[m];
    if (Z) Z[o] = s.Z[m];
    if (phi) phi[o] = s.phi[m];
    if (u) u[o] = s.u[m];
    if (w) w[o] = s.w[m];
    if (status) status[o] = s.status[m];
}
// cell key = tri * P + toroidal interval; markers outside the mesh go to the last cell (T*P)
__global__ void __launch_bounds__(256) k_sort_keys(DevTables tb, CellMap cm, int ncell, MarkerSoA s, long long n, int* __restrict__ keys, int* __restrict__ hist) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    int t = locate_walk(tb.bg, tb.geom, s.tri[m], s.R[m], s.Z[m]);
    double sf;
    int k = toroidal_interval(tb.tor, s.phi[m], sf);
    int key = t < 0 ? ncell : cm.cell(t, k);
    s.tri[m] = t;
    keys[m] = key;
    atomicAdd(hist + key, 1);
}
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
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_reduce(const int* __restrict__ in, long long n, int* __restrict__ sums) {
    long long base = (long long)blockIdx.x * SCAN_CHUNK + (long long)threadIdx.x * SCAN_ITEMS;
    int s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) if (base + i < n) s += in[base + i];
    int tot;
    block_exclusive_scan(s, &tot);
    if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_sums(int* __restrict__ sums, int nb) {   // single block
    __shared__ int carry;
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
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(const int* __restrict__ in, long long n, const int* __restrict__ sums,
                                                             int* __restrict__ out) {
    long long base = (long long)blockIdx.x * SCAN_CHUNK + (long long)threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS], s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) { v[i] = base + i < n ? in[base + i] : 0; s += v[i]; }
    int ex = block_exclusive_scan(s, nullptr) + sums[blockIdx.x];
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) { if (base + i < n) out[base + i] = ex; ex += v[i]; }
}
// permutation: perm[new position] = old position (4-byte scattered writes), then a gather with coalesced writes
__global__ void __launch_bounds__(256) k_sort_perm(long long n, const int* __restrict__ keys, const int* __restrict__ offs, int* __restrict__ fill,
                                                   int* __restrict__ perm) {
    long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= n) return;
    int key = keys[m];
    long long pos = (long long)offs[key] + atomicAdd(fill + key, 1);
    perm[pos] = (int)m;
}
__global__ void __launch_bounds__(256) k_sort_gather(MarkerSoA a, MarkerSoA b, long long n, const int* __restrict__ perm) {
    long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    long long m = perm[j];
    b.R[j] = a.R[m]; b.Z[j] = a.Z[m]; b.phi[j] = a.phi[m]; b.u[j] = a.u[m]; b.w[j] = a.w[m];
    b.mu[j] = a.mu[m]; b.p[j] = a.p[m]; b.tri[j] = a.tri[m]; b.status[j] = a.status[m]; b.id[j] = a.id[m];
}
// per step: acc[0] += marker-stage evaluations left to the follow-up kernel, acc[1] += markers retired (4 threads, one per sub-queue)
__global__ void k_accumulate_stat(const int* __restrict__ v, int cap, unsigned long long* __restrict__ acc) {
    unsigned long long c = (unsigned long long)min(v[threadIdx.x], cap);
    atomicAdd(acc, c * (4 - threadIdx.x));
    atomicAdd(acc + 1, c);
}

// ============================================================================================ DFMA micro-benchmark
__global__ void __launch_bounds__(512) k_dfma(double* out, int iters, double a, double b) {
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

// ============================================================================================ context
struct trimeg_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int num_sms = 148;
    std::string err;
    bool have_eq = false, have_sp = false, have_mesh = false, have_markers = false;
    EquilP ep{};
    SpeciesP sp{};
    trimeg_equil eq_in{};
    // mesh
    int T = 0, P = 0;
    long long n_nodes = 0;
    double period = 0;
    TriGeom* d_geom = nullptr;
    int *d_tri = nullptr, *d_head = nullptr, *d_list = nullptr, *d_new_of_orig = nullptr;
    double *d_RZ = nullptr, *d_K = nullptr, *d_coef = nullptr;
    DevTables tb{};
    // markers
    long long n = 0;
    MarkerSoA buf[2]{};
    int cur = 0;
    int *d_keys = nullptr, *d_perm = nullptr;   // in scratch
    int *d_hist = nullptr, *d_offs = nullptr, *d_fill = nullptr, *d_sums = nullptr;   // library-owned, [T*P+2]
    long long ncell = 0;
    bool sorted = false;
    bool keys_valid = false;    // d_keys / d_hist describe the current store (written by the last push step)
    int sort_every = 0;
    // retire queues (in scratch)
    RetireQueue rq{};
    // per-kernel timing of the last step of trimeg_push_rk4 (events on the context's stream)
    cudaEvent_t ev[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    bool ev_valid = false;
    long long steps_since_sort = 0;
    int variant = 0;
    long long stats[4] = {0, 0, 0, 0};
    // tiled kernel tables
    int *d_pslots = nullptr, *d_pnslots = nullptr, *d_work = nullptr;
    short* d_pnbr = nullptr;
    unsigned long long* d_stats = nullptr;
    TileTables tt{};
    CellMap cm{};
    bool tiled_ok = false;
};

static int fail(trimeg_ctx* c, int code, const char* fmt, ...) {
    if (c) {
        char buf[512];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        c->err = buf;
    }
    return code;
}
#define CU(call)                                                                                          \
    do {                                                                                                  \
        cudaError_t e__ = (call);                                                                         \
        if (e__ != cudaSuccess) {                                                                         \
            int code__ = (e__ == cudaErrorMemoryAllocation) ? TRIMEG_ERR_OOM : TRIMEG_ERR_CUDA;           \
            return fail(ctx, code__, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e__), __FILE__, __LINE__); \
        }                                                                                                 \
    } while (0)
#define KCHECK() CU(cudaGetLastError())

static inline unsigned blocks_for(long long n, int threads) { return (unsigned)((n + threads - 1) / threads); }
static inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

static void free_mesh(trimeg_ctx* c) {
    cudaFree(c->d_geom); cudaFree(c->d_tri); cudaFree(c->d_head); cudaFree(c->d_list); cudaFree(c->d_new_of_orig);
    cudaFree(c->d_RZ); cudaFree(c->d_K); cudaFree(c->d_coef);
    cudaFree(c->d_hist); cudaFree(c->d_offs); cudaFree(c->d_fill); cudaFree(c->d_sums);
    cudaFree(c->d_pslots); cudaFree(c->d_pnslots); cudaFree(c->d_pnbr); cudaFree(c->d_work); cudaFree(c->d_stats);
    c->d_pslots = c->d_pnslots = c->d_work = nullptr; c->d_pnbr = nullptr; c->d_stats = nullptr;
    c->d_geom = nullptr; c->d_tri = c->d_head = c->d_list = c->d_new_of_orig = nullptr;
    c->d_RZ = c->d_K = c->d_coef = nullptr;
    c->d_hist = c->d_offs = c->d_fill = c->d_sums = nullptr;
    c->have_mesh = false; c->have_markers = false;
}

extern "C" {

int trimeg_create(trimeg_ctx** out, int device, void* cuda_stream) {
    if (!out) return TRIMEG_ERR_BAD_ARG;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) return TRIMEG_ERR_CUDA;
    if (cudaSetDevice(device) != cudaSuccess) return TRIMEG_ERR_CUDA;
    trimeg_ctx* c = new (std::nothrow) trimeg_ctx;
    if (!c) return TRIMEG_ERR_OOM;
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, device);
    trimeg_host::ElementConsts ec;
    if (!trimeg_host::element_consts(ec)) { delete c; return TRIMEG_ERR_BAD_STATE; }
    if (cudaMemcpyToSymbol(c_Aplus, ec.Aplus, sizeof ec.Aplus) != cudaSuccess || cudaMemcpyToSymbol(c_Nul, ec.Nul, sizeof ec.Nul) != cudaSuccess) {
        delete c;
        return TRIMEG_ERR_CUDA;
    }
    for (auto& e : c->ev) if (cudaEventCreate(&e) != cudaSuccess) { delete c; return TRIMEG_ERR_CUDA; }
    *out = c;
    return TRIMEG_OK;
}

int trimeg_destroy(trimeg_ctx* ctx) {
    if (!ctx) return TRIMEG_ERR_BAD_ARG;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    for (auto& e : ctx->ev) if (e) cudaEventDestroy(e);
    free_mesh(ctx);
    delete ctx;
    return TRIMEG_OK;
}

int trimeg_sync(trimeg_ctx* ctx) {
    if (!ctx) return TRIMEG_ERR_BAD_ARG;
    CU(cudaStreamSynchronize(ctx->stream));
    return TRIMEG_OK;
}

const char* trimeg_last_error(const trimeg_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int trimeg_equilibrium_set(trimeg_ctx* ctx, const trimeg_equil* eq) {
    if (!ctx || !eq) return fail(ctx, TRIMEG_ERR_BAD_ARG, "equilibrium_set: null argument");
    if (!(eq->R0 > 0) || !(eq->a > 0) || !(eq->a < eq->R0) || !std::isfinite(eq->B0) || eq->B0 == 0 || !std::isfinite(eq->q0 + eq->q1 + eq->q2))
        return fail(ctx, TRIMEG_ERR_BAD_ARG, "equilibrium_set: need 0 < a < R0, finite nonzero B0, finite q");
    ctx->eq_in = *eq;
    EquilP& e = ctx->ep;
    e.R0 = eq->R0; e.B0 = eq->B0; e.F = eq->B0 * eq->R0; e.inv_a = 1.0 / eq->a; e.inv_R0sq = 1.0 / (eq->R0 * eq->R0);
    e.q0 = eq->q0; e.q1 = eq->q1; e.q2 = eq->q2; e.qbar_sqrt = eq->qbar_sqrt ? 1 : 0;
    ctx->have_eq = true;
    return TRIMEG_OK;
}

int trimeg_species_set(trimeg_ctx* ctx, const trimeg_species* s) {
    if (!ctx || !s) return fail(ctx, TRIMEG_ERR_BAD_ARG, "species_set: null argument");
    if (!ctx->have_eq) return fail(ctx, TRIMEG_ERR_BAD_STATE, "species_set: call trimeg_equilibrium_set first (profiles use a and R0)");
    if (!std::isfinite(s->qom) || s->qom == 0 || !(s->w_n > 0) || !(s->w_T > 0) || !std::isfinite(s->kappa_n + s->kappa_T + s->r0))
        return fail(ctx, TRIMEG_ERR_BAD_ARG, "species_set: need finite nonzero qom, w_n > 0, w_T > 0");
    const trimeg_equil& eq = ctx->eq_in;
    SpeciesP& p = ctx->sp;
    p.qom = s->qom; p.kappa = 1.0 / s->qom;
    p.kn_R0 = s->kappa_n / eq.R0; p.kT_R0 = s->kappa_T / eq.R0;
    p.inv_wn_a = 1.0 / (s->w_n * eq.a); p.inv_wT_a = 1.0 / (s->w_T * eq.a); p.r0 = s->r0;
    p.cT = s->kappa_T * s->w_T * eq.a / eq.R0;
    p.same_w = (s->w_n == s->w_T) ? 1 : 0;
    p.bstar_exact = s->bstar_exact ? 1 : 0; p.weight_mode = s->weight_mode ? 1 : 0;
    ctx->have_sp = true;
    return TRIMEG_OK;
}

int trimeg_mesh_load(trimeg_ctx* ctx, int64_t n_nodes, const double* RZ, int64_t n_tri, const int32_t* tri, int32_t n_planes, double phi_period) {
    if (!ctx || !RZ || !tri) return fail(ctx, TRIMEG_ERR_BAD_ARG, "mesh_load: null argument");
    if (n_nodes < 3 || n_tri < 1 || n_planes < 4 || !(phi_period > 0) || !std::isfinite(phi_period))
        return fail(ctx, TRIMEG_ERR_BAD_ARG, "mesh_load: need n_nodes >= 3, n_tri >= 1, n_planes >= 4, phi_period > 0");
    if ((double)n_tri * n_planes + 2 > 2.0e9 || n_nodes > 2000000000LL) return fail(ctx, TRIMEG_ERR_BAD_ARG, "mesh_load: n_tri * n_planes exceeds int32 cell ids");
    CU(cudaSetDevice(ctx->device));
    CU(cudaStreamSynchronize(ctx->stream));
    free_mesh(ctx);
    trimeg_host::HostMesh hm;
    // with the equilibrium known, number triangles along flux surfaces and shape the patch halos along the poloidal field
    const double axis[2] = {ctx->eq_in.R0, 0.0};
    const double* axis_p = ctx->have_eq ? axis : nullptr;
    int rc = trimeg_host::build_mesh(n_nodes, RZ, n_tri, tri, axis_p, hm);
    if (rc) return fail(ctx, TRIMEG_ERR_BAD_MESH, "mesh_load: vertex index out of range, non-finite node, clockwise/degenerate triangle or non-manifold edge");
    trimeg_host::ElementConsts ec;
    trimeg_host::element_consts(ec);
    const int T = (int)n_tri;
    std::vector<TriGeom> geom(T);
    std::vector<double> K((size_t)T * 18);
    for (int t = 0; t < T; ++t) {
        double v[3][2];
        for (int q = 0; q < 3; ++q) { v[q][0] = RZ[2 * hm.tri[3 * t + q]]; v[q][1] = RZ[2 * hm.tri[3 * t + q] + 1]; }
        long double j11 = (long double)v[1][0] - v[0][0], j21 = (long double)v[1][1] - v[0][1], j12 = (long double)v[2][0] - v[0][0], j22 = (long double)v[2][1] - v[0][1];
        long double det = j11 * j22 - j12 * j21;
        TriGeom& g = geom[t];
        g.v0x = v[0][0]; g.v0y = v[0][1];
        g.a11 = (double)(j22 / det); g.a12 = (double)(-j12 / det); g.a21 = (double)(-j21 / det); g.a22 = (double)(j11 / det);
        for (int e = 0; e < 3; ++e) g.nbr[e] = hm.nbr[3 * t + e];
        g.orig = hm.orig_of_new[t];
        if (!trimeg_host::triangle_K(ec, v, &K[(size_t)t * 18])) return fail(ctx, TRIMEG_ERR_BAD_MESH, "mesh_load: degenerate triangle %d", g.orig);
    }
    ctx->T = T; ctx->P = n_planes; ctx->n_nodes = n_nodes; ctx->period = phi_period;
    const long long tri_stride = (long long)(n_planes + 3 + 2 * PLANE_PAD) * PLANE_STRIDE;
    const size_t coef_bytes = (size_t)T * tri_stride * sizeof(double);
    trimeg_host::HostPatches hp;
    trimeg_host::build_patches(hm, RZ, n_nodes, T, Tile::TP, Tile::SMAX, axis_p, 3.0, hp);
    const int nwin = (n_planes + Tile::WK - 1) / Tile::WK;
    ctx->cm.P = n_planes; ctx->cm.nwin = nwin;
    ctx->ncell = (long long)hp.npatch * nwin * Tile::CPS;
    if ((double)hp.npatch * nwin * Tile::CPS + 2 > 2.0e9) return fail(ctx, TRIMEG_ERR_BAD_ARG, "mesh_load: too many cells for int32 ids");
    ctx->tiled_ok = (n_planes % Tile::WK == 0) && (n_planes >= Tile::NW);
    CU(cudaMalloc(&ctx->d_geom, sizeof(TriGeom) * T));
    CU(cudaMalloc(&ctx->d_tri, sizeof(int) * 3 * T));
    CU(cudaMalloc(&ctx->d_head, sizeof(int) * hm.head.size()));
    CU(cudaMalloc(&ctx->d_list, sizeof(int) * hm.list.size()));
    CU(cudaMalloc(&ctx->d_new_of_orig, sizeof(int) * T));
    CU(cudaMalloc(&ctx->d_RZ, sizeof(double) * 2 * n_nodes));
    CU(cudaMalloc(&ctx->d_K, sizeof(double) * 18 * T));
    CU(cudaMalloc(&ctx->d_coef, coef_bytes));
    size_t ncnt = (size_t)ctx->ncell + 2;
    CU(cudaMalloc(&ctx->d_hist, sizeof(int) * ncnt));
    CU(cudaMalloc(&ctx->d_offs, sizeof(int) * ncnt));
    CU(cudaMalloc(&ctx->d_fill, sizeof(int) * ncnt));
    CU(cudaMalloc(&ctx->d_sums, sizeof(int) * (ncnt / SCAN_CHUNK + 2)));
    CU(cudaMalloc(&ctx->d_pslots, sizeof(int) * hp.slots.size()));
    CU(cudaMalloc(&ctx->d_pnslots, sizeof(int) * hp.nslots.size()));
    CU(cudaMalloc(&ctx->d_pnbr, sizeof(short) * hp.nbr.size()));
    CU(cudaMalloc(&ctx->d_work, sizeof(int) * 8));
    CU(cudaMalloc(&ctx->d_stats, sizeof(unsigned long long) * 4));
    CU(cudaMemcpyAsync(ctx->d_pslots, hp.slots.data(), sizeof(int) * hp.slots.size(), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_pnslots, hp.nslots.data(), sizeof(int) * hp.nslots.size(), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_pnbr, hp.nbr.data(), sizeof(short) * hp.nbr.size(), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_stats, 0, sizeof(unsigned long long) * 4, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_offs, 0, sizeof(int) * ncnt, ctx->stream));
    ctx->tt.slots = ctx->d_pslots; ctx->tt.nbr = ctx->d_pnbr; ctx->tt.nslots = ctx->d_pnslots; ctx->tt.offs = ctx->d_offs;
    ctx->tt.npatch = hp.npatch; ctx->tt.nwin = nwin; ctx->tt.nsc = hp.npatch * nwin;
    CU(cudaFuncSetAttribute(k_push_tiled<Tile>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tile::BYTES));
    CU(cudaMemcpyAsync(ctx->d_geom, geom.data(), sizeof(TriGeom) * T, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_tri, hm.tri.data(), sizeof(int) * 3 * T, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_head, hm.head.data(), sizeof(int) * hm.head.size(), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_list, hm.list.data(), sizeof(int) * hm.list.size(), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_new_of_orig, hm.new_of_orig.data(), sizeof(int) * T, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_RZ, RZ, sizeof(double) * 2 * n_nodes, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_K, K.data(), sizeof(double) * 18 * T, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_coef, 0, coef_bytes, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));   // host vectors go out of scope
    DevTables& tb = ctx->tb;
    tb.geom = ctx->d_geom; tb.coef = ctx->d_coef; tb.T = T; tb.tri_stride = tri_stride;
    tb.bg.xmin = hm.xmin; tb.bg.ymin = hm.ymin; tb.bg.inv_dx = 1.0 / hm.dx; tb.bg.inv_dy = 1.0 / hm.dy;
    tb.bg.nx = hm.nx; tb.bg.ny = hm.ny; tb.bg.head = ctx->d_head; tb.bg.list = ctx->d_list;
    tb.tor.period = phi_period; tb.tor.inv_period = 1.0 / phi_period; tb.tor.P = n_planes;
    tb.tor.inv_dphi = (double)n_planes / phi_period; tb.tor.half_inv_dphi = 0.5 * (double)n_planes / phi_period;
    ctx->have_mesh = true;
    return TRIMEG_OK;
}

int trimeg_fields_set(trimeg_ctx* ctx, int which, const double* dof, int memspace) {
    if (!ctx || !dof || which < 0 || which > 1 || (memspace != TRIMEG_HOST && memspace != TRIMEG_DEVICE))
        return fail(ctx, TRIMEG_ERR_BAD_ARG, "fields_set: bad argument");
    if (!ctx->have_mesh) return fail(ctx, TRIMEG_ERR_BAD_STATE, "fields_set: call trimeg_mesh_load first");
    CU(cudaSetDevice(ctx->device));
    const double* d_dof = dof;
    double* tmp = nullptr;
    size_t bytes = sizeof(double) * 6 * (size_t)ctx->n_nodes * ctx->P;
    if (memspace == TRIMEG_HOST) {
        CU(cudaMalloc(&tmp, bytes));
        cudaError_t e = cudaMemcpyAsync(tmp, dof, bytes, cudaMemcpyHostToDevice, ctx->stream);
        if (e != cudaSuccess) { cudaFree(tmp); return fail(ctx, TRIMEG_ERR_CUDA, "fields_set: H2D copy failed: %s", cudaGetErrorString(e)); }
        d_dof = tmp;
    }
    long long work = (long long)ctx->T * ctx->P;
    k_fields_set<<<blocks_for(work, 128), 128, 0, ctx->stream>>>(ctx->T, ctx->P, which, ctx->d_tri, ctx->d_RZ, ctx->d_K, d_dof, ctx->n_nodes, ctx->d_coef);
    cudaError_t e = cudaGetLastError();
    if (tmp) { cudaStreamSynchronize(ctx->stream); cudaFree(tmp); }
    if (e != cudaSuccess) return fail(ctx, TRIMEG_ERR_CUDA, "fields_set kernel: %s", cudaGetErrorString(e));
    return TRIMEG_OK;
}

int trimeg_gather(trimeg_ctx* ctx, int64_t n, const double* R, const double* Z, const double* phi, double* out, int32_t* tri_out, int memspace) {
    if (!ctx || n < 0 || (n > 0 && (!R || !Z || !phi || !out)) || (memspace != TRIMEG_HOST && memspace != TRIMEG_DEVICE))
        return fail(ctx, TRIMEG_ERR_BAD_ARG, "gather: bad argument");
    if (!ctx->have_mesh) return fail(ctx, TRIMEG_ERR_BAD_STATE, "gather: call trimeg_mesh_load first");
    if (n == 0) return TRIMEG_OK;
    CU(cudaSetDevice(ctx->device));
    if (memspace == TRIMEG_DEVICE) {
        k_gather<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(ctx->tb, n, R, Z, phi, out, tri_out);
        KCHECK();
        return TRIMEG_OK;
    }
    double* d = nullptr;
    int* dt = nullptr;
    CU(cudaMalloc(&d, sizeof(double) * 11 * (size_t)n));
    if (cudaMalloc(&dt, sizeof(int) * (size_t)n) != cudaSuccess) { cudaFree(d); return fail(ctx, TRIMEG_ERR_OOM, "gather: out of device memory"); }
    cudaError_t e = cudaSuccess;
    auto step = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    step(cudaMemcpyAsync(d, R, sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream));
    step(cudaMemcpyAsync(d + n, Z, sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream));
    step(cudaMemcpyAsync(d + 2 * n, phi, sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream));
    if (e == cudaSuccess) { k_gather<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(ctx->tb, n, d, d + n, d + 2 * n, d + 3 * n, dt); step(cudaGetLastError()); }
    step(cudaMemcpyAsync(out, d + 3 * n, sizeof(double) * 8 * n, cudaMemcpyDeviceToHost, ctx->stream));
    if (tri_out) step(cudaMemcpyAsync(tri_out, dt, sizeof(int) * n, cudaMemcpyDeviceToHost, ctx->stream));
    step(cudaStreamSynchronize(ctx->stream));
    cudaFree(d); cudaFree(dt);
    if (e != cudaSuccess) return fail(ctx, TRIMEG_ERR_CUDA, "gather: %s", cudaGetErrorString(e));
    return TRIMEG_OK;
}

// scratch layout: two MarkerSoA buffers (7 doubles + 3 ints per marker each) + keys
// retire queues: four sub-queues of cap entries each (10 doubles + 2 ints per entry); cap = n/32 per stage (>= 1024)
static int retire_cap(long long n) { return (int)std::max<long long>(1024, n / 32); }
static size_t retire_bytes(int cap) { return align256((size_t)4 * cap * (10 * sizeof(double) + 2 * sizeof(int))); }
static size_t soa_bytes(long long n) { return 7 * align256(sizeof(double) * (size_t)n) + 3 * align256(sizeof(int) * (size_t)n); }
size_t trimeg_scratch_bytes(const trimeg_ctx* ctx, int64_t n) {
    if (!ctx || n <= 0) return 0;
    return 2 * soa_bytes(n) + 2 * align256(sizeof(int) * (size_t)n) + retire_bytes(retire_cap(n)) + 256;
}
static void carve(MarkerSoA& s, char*& p, long long n) {
    double** dp[7] = {&s.R, &s.Z, &s.phi, &s.u, &s.w, &s.mu, &s.p};
    for (auto q : dp) { *q = (double*)p; p += align256(sizeof(double) * (size_t)n); }
    int** ip[3] = {&s.tri, &s.status, &s.id};
    for (auto q : ip) { *q = (int*)p; p += align256(sizeof(int) * (size_t)n); }
}

// counting sort by cell, in three parts: keys + histogram of the current store (skipped when the last push step
// already produced them), offsets + permutation, and the data movement (fused into the tiled push, or k_sort_gather)
static int sort_keys(trimeg_ctx* ctx) {
    const long long n = ctx->n, ncnt = ctx->ncell + 2;   // cells + lost bin + end sentinel
    CU(cudaMemsetAsync(ctx->d_hist, 0, sizeof(int) * ncnt, ctx->stream));
    k_sort_keys<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(ctx->tb, ctx->cm, (int)ctx->ncell, ctx->buf[ctx->cur], n, ctx->d_keys, ctx->d_hist);
    KCHECK();
    ctx->stats[0] += 1;
    return TRIMEG_OK;
}
static int sort_perm(trimeg_ctx* ctx) {
    const long long n = ctx->n, ncnt = ctx->ncell + 2;
    CU(cudaMemsetAsync(ctx->d_fill, 0, sizeof(int) * ncnt, ctx->stream));
    int nb = (int)((ncnt + SCAN_CHUNK - 1) / SCAN_CHUNK);
    k_scan_reduce<<<nb, SCAN_THREADS, 0, ctx->stream>>>(ctx->d_hist, ncnt, ctx->d_sums);
    KCHECK();
    k_scan_sums<<<1, SCAN_THREADS, 0, ctx->stream>>>(ctx->d_sums, nb);
    KCHECK();
    k_scan_apply<<<nb, SCAN_THREADS, 0, ctx->stream>>>(ctx->d_hist, ncnt, ctx->d_sums, ctx->d_offs);
    KCHECK();
    k_sort_perm<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(n, ctx->d_keys, ctx->d_offs, ctx->d_fill, ctx->d_perm);
    KCHECK();
    ctx->stats[0] += 4;
    ctx->stats[3] += 1;
    return TRIMEG_OK;
}
static int do_sort(trimeg_ctx* ctx) {   // full sort with a separate gather pass
    int rc = ctx->keys_valid ? TRIMEG_OK : sort_keys(ctx);
    if (rc) return rc;
    rc = sort_perm(ctx);
    if (rc) return rc;
    k_sort_gather<<<blocks_for(ctx->n, 256), 256, 0, ctx->stream>>>(ctx->buf[ctx->cur], ctx->buf[ctx->cur ^ 1], ctx->n, ctx->d_perm);
    KCHECK();
    ctx->cur ^= 1;
    ctx->sorted = true;
    ctx->keys_valid = false;
    ctx->steps_since_sort = 0;
    ctx->stats[0] += 1;
    return TRIMEG_OK;
}

int trimeg_markers_bind(trimeg_ctx* ctx, int64_t n, const double* R, const double* Z, const double* phi, const double* u, const double* w,
                        const double* mu, const double* p, int memspace, void* scratch, size_t scratch_bytes) {
    if (!ctx || n <= 0 || !R || !Z || !phi || !u || !w || !mu || !p || !scratch || (memspace != TRIMEG_HOST && memspace != TRIMEG_DEVICE))
        return fail(ctx, TRIMEG_ERR_BAD_ARG, "markers_bind: bad argument");
    if (n > 2000000000LL) return fail(ctx, TRIMEG_ERR_BAD_ARG, "markers_bind: n exceeds int32 marker ids");
    if (!ctx->have_mesh) return fail(ctx, TRIMEG_ERR_BAD_STATE, "markers_bind: call trimeg_mesh_load first");
    if (scratch_bytes < trimeg_scratch_bytes(ctx, n)) return fail(ctx, TRIMEG_ERR_OOM, "markers_bind: scratch too small (%zu < %zu)", scratch_bytes, trimeg_scratch_bytes(ctx, n));
    CU(cudaSetDevice(ctx->device));
    char* ptr = (char*)(((uintptr_t)scratch + 255) & ~(uintptr_t)255);
    carve(ctx->buf[0], ptr, n);
    carve(ctx->buf[1], ptr, n);
    ctx->d_keys = (int*)ptr;
    ctx->d_perm = (int*)(ptr + align256(sizeof(int) * (size_t)n));
    {
        char* q = ptr + 2 * align256(sizeof(int) * (size_t)n);
        RetireQueue& rq = ctx->rq;
        rq.cap = retire_cap(n);
        rq.y = (double*)q; rq.acc = rq.y + 5 * 4 * (size_t)rq.cap;
        rq.m = (int*)(rq.acc + 5 * 4 * (size_t)rq.cap); rq.st = rq.m + 4 * (size_t)rq.cap;
        rq.count = ctx->d_work + 4;
    }
    ctx->n = n; ctx->cur = 0; ctx->sorted = false; ctx->keys_valid = false; ctx->steps_since_sort = 0;
    if (memspace == TRIMEG_HOST) {   // stage through the second buffer
        MarkerSoA& b = ctx->buf[1];
        const double* src[7] = {R, Z, phi, u, w, mu, p};
        double* dst[7] = {b.R, b.Z, b.phi, b.u, b.w, b.mu, b.p};
        for (int q = 0; q < 7; ++q) CU(cudaMemcpyAsync(dst[q], src[q], sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream));
        k_bind<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(ctx->buf[0], n, b.R, b.Z, b.phi, b.u, b.w, b.mu, b.p);
    } else {
        k_bind<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(ctx->buf[0], n, R, Z, phi, u, w, mu, p);
    }
    KCHECK();
    ctx->have_markers = true;
    return TRIMEG_OK;
}

int trimeg_markers_get(trimeg_ctx* ctx, double* R, double* Z, double* phi, double* u, double* w, int32_t* status, int memspace) {
    if (!ctx || (memspace != TRIMEG_HOST && memspace != TRIMEG_DEVICE)) return fail(ctx, TRIMEG_ERR_BAD_ARG, "markers_get: bad argument");
    if (!ctx->have_markers) return fail(ctx, TRIMEG_ERR_BAD_STATE, "markers_get: no markers bound");
    CU(cudaSetDevice(ctx->device));
    const long long n = ctx->n;
    MarkerSoA& s = ctx->buf[ctx->cur];
    if (memspace == TRIMEG_DEVICE) {
        k_unsort<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(s, n, R, Z, phi, u, w, status);
        KCHECK();
        return TRIMEG_OK;
    }
    // HOST: un-sort into the inactive buffer (free between sorts), then copy out
    MarkerSoA& b = ctx->buf[ctx->cur ^ 1];
    k_unsort<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(s, n, R ? b.R : nullptr, Z ? b.Z : nullptr, phi ? b.phi : nullptr, u ? b.u : nullptr,
                                                           w ? b.w : nullptr, status ? b.status : nullptr);
    KCHECK();
    if (R) CU(cudaMemcpyAsync(R, b.R, sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream));
    if (Z) CU(cudaMemcpyAsync(Z, b.Z, sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream));
    if (phi) CU(cudaMemcpyAsync(phi, b.phi, sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream));
    if (u) CU(cudaMemcpyAsync(u, b.u, sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream));
    if (w) CU(cudaMemcpyAsync(w, b.w, sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream));
    if (status) CU(cudaMemcpyAsync(status, b.status, sizeof(int) * n, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return TRIMEG_OK;
}

int trimeg_sort(trimeg_ctx* ctx) {
    if (!ctx) return TRIMEG_ERR_BAD_ARG;
    if (!ctx->have_markers) return fail(ctx, TRIMEG_ERR_BAD_STATE, "sort: no markers bound");
    CU(cudaSetDevice(ctx->device));
    return do_sort(ctx);
}

int trimeg_set_sort_interval(trimeg_ctx* ctx, int32_t every_n_steps) {
    if (!ctx || every_n_steps < 0) return fail(ctx, TRIMEG_ERR_BAD_ARG, "set_sort_interval: need every_n_steps >= 0");
    ctx->sort_every = every_n_steps;
    return TRIMEG_OK;
}

int trimeg_set_push_variant(trimeg_ctx* ctx, int32_t variant) {
    if (!ctx || variant < 0 || variant > 1) return fail(ctx, TRIMEG_ERR_BAD_ARG, "set_push_variant: 0 or 1");
    ctx->variant = variant;
    return TRIMEG_OK;
}

int trimeg_push_rk4(trimeg_ctx* ctx, double dt, int32_t nsteps) {
    if (!ctx || !(dt > 0) || !std::isfinite(dt) || nsteps < 0) return fail(ctx, TRIMEG_ERR_BAD_ARG, "push_rk4: need finite dt > 0 and nsteps >= 0");
    if (!ctx->have_mesh || !ctx->have_eq || !ctx->have_sp || !ctx->have_markers)
        return fail(ctx, TRIMEG_ERR_BAD_STATE, "push_rk4: mesh, equilibrium, species and markers must be set first");
    CU(cudaSetDevice(ctx->device));
    ctx->stats[0] = ctx->stats[1] = ctx->stats[2] = ctx->stats[3] = 0;
    CU(cudaMemsetAsync(ctx->d_stats, 0, sizeof(unsigned long long) * 4, ctx->stream));
    const long long n = ctx->n;
    ctx->ev_valid = false;
    for (int s = 0; s < nsteps; ++s) {
        const bool need_sort = !ctx->sorted || (ctx->sort_every > 0 && ctx->steps_since_sort >= ctx->sort_every);
        const bool timed = (s == nsteps - 1);
        if (timed) CU(cudaEventRecord(ctx->ev[0], ctx->stream));
        if (ctx->variant == 0 && ctx->tiled_ok) {
            // the sort only builds the permutation; the push reads the markers through it and writes the other buffer
            const int* perm = nullptr;
            if (need_sort) {
                int rc = ctx->keys_valid ? TRIMEG_OK : sort_keys(ctx);
                if (rc) return rc;
                rc = sort_perm(ctx);
                if (rc) return rc;
                perm = ctx->d_perm;
                ctx->sorted = true;
                ctx->steps_since_sort = 0;
            }
            MarkerSoA& src = ctx->buf[ctx->cur];
            MarkerSoA& dst = need_sort ? ctx->buf[ctx->cur ^ 1] : ctx->buf[ctx->cur];
            KeyOut ko;
            ko.keys = ctx->d_keys; ko.hist = ctx->d_hist; ko.ncell = (int)ctx->ncell;
            ko.enabled = (ctx->sort_every > 0 && ctx->steps_since_sort + 1 >= ctx->sort_every) ? 1 : 0;
            if (ko.enabled) CU(cudaMemsetAsync(ctx->d_hist, 0, sizeof(int) * (ctx->ncell + 2), ctx->stream));
            CU(cudaMemsetAsync(ctx->d_work, 0, 8 * sizeof(int), ctx->stream));
            if (timed) CU(cudaEventRecord(ctx->ev[1], ctx->stream));
            k_push_tiled<Tile><<<ctx->num_sms, Tile::NTHREADS, Tile::BYTES, ctx->stream>>>(ctx->tb, ctx->tt, ctx->ep, ctx->sp, src, dst, perm, ctx->rq, ko, ctx->cm, dt, ctx->d_work);
            KCHECK();
            if (timed) CU(cudaEventRecord(ctx->ev[2], ctx->stream));
            k_push_finish<<<ctx->num_sms * 8, 128, 0, ctx->stream>>>(ctx->tb, ctx->ep, ctx->sp, src, dst, perm, ctx->rq, ko, ctx->cm, dt);
            KCHECK();
            k_accumulate_stat<<<1, 4, 0, ctx->stream>>>(ctx->rq.count, ctx->rq.cap, ctx->d_stats + 1);
            KCHECK();
            // markers outside the mesh sit behind the last cell: push them through the simple path
            k_push_lost<<<148 * 4, 128, 0, ctx->stream>>>(ctx->tb, ctx->ep, ctx->sp, src, dst, perm, ko, ctx->cm, ctx->d_offs + ctx->ncell, n, dt);
            KCHECK();
            if (timed) CU(cudaEventRecord(ctx->ev[3], ctx->stream));
            if (need_sort) ctx->cur ^= 1;
            ctx->keys_valid = ko.enabled != 0;
            ctx->stats[0] += 4;
        } else {
            if (need_sort) {
                int rc = do_sort(ctx);
                if (rc) return rc;
            }
            if (timed) { CU(cudaEventRecord(ctx->ev[1], ctx->stream)); }
            k_push_simple<<<blocks_for(n, 128), 128, 0, ctx->stream>>>(ctx->tb, ctx->ep, ctx->sp, ctx->buf[ctx->cur], n, dt);
            KCHECK();
            if (timed) { CU(cudaEventRecord(ctx->ev[2], ctx->stream)); CU(cudaEventRecord(ctx->ev[3], ctx->stream)); }
            ctx->keys_valid = false;
            ctx->stats[0] += 1;
        }
        if (timed) ctx->ev_valid = true;
        ctx->steps_since_sort += 1;
    }
    return TRIMEG_OK;
}

int trimeg_push_kernel_ms(trimeg_ctx* ctx, double out[3]) {
    if (!ctx || !out) return fail(ctx, TRIMEG_ERR_BAD_ARG, "push_kernel_ms: null argument");
    if (!ctx->ev_valid) return fail(ctx, TRIMEG_ERR_BAD_STATE, "push_kernel_ms: no step has been pushed");
    CU(cudaSetDevice(ctx->device));
    CU(cudaEventSynchronize(ctx->ev[3]));
    for (int i = 0; i < 3; ++i) {
        float ms = 0;
        CU(cudaEventElapsedTime(&ms, ctx->ev[i], ctx->ev[i + 1]));
        out[i] = ms;
    }
    return TRIMEG_OK;
}

int trimeg_rhs(trimeg_ctx* ctx, double* out, int memspace) {
    if (!ctx || !out || (memspace != TRIMEG_HOST && memspace != TRIMEG_DEVICE)) return fail(ctx, TRIMEG_ERR_BAD_ARG, "rhs: bad argument");
    if (!ctx->have_mesh || !ctx->have_eq || !ctx->have_sp || !ctx->have_markers)
        return fail(ctx, TRIMEG_ERR_BAD_STATE, "rhs: mesh, equilibrium, species and markers must be set first");
    CU(cudaSetDevice(ctx->device));
    const long long n = ctx->n;
    double* d = out;
    if (memspace == TRIMEG_HOST) CU(cudaMalloc(&d, sizeof(double) * 5 * (size_t)n));
    k_rhs<<<blocks_for(n, 128), 128, 0, ctx->stream>>>(ctx->tb, ctx->ep, ctx->sp, ctx->buf[ctx->cur], n, d);
    cudaError_t e = cudaGetLastError();
    if (memspace == TRIMEG_HOST) {
        if (e == cudaSuccess) e = cudaMemcpyAsync(out, d, sizeof(double) * 5 * n, cudaMemcpyDeviceToHost, ctx->stream);
        cudaError_t e2 = cudaStreamSynchronize(ctx->stream);
        if (e == cudaSuccess) e = e2;
        cudaFree(d);
    }
    if (e != cudaSuccess) return fail(ctx, TRIMEG_ERR_CUDA, "rhs: %s", cudaGetErrorString(e));
    return TRIMEG_OK;
}

int trimeg_bench_dfma(trimeg_ctx* ctx, double* tflops) {
    if (!ctx || !tflops) return fail(ctx, TRIMEG_ERR_BAD_ARG, "bench_dfma: null argument");
    CU(cudaSetDevice(ctx->device));
    const int nb = ctx->num_sms * 2, th = 512, iters = 40000;
    double* d = nullptr;
    CU(cudaMalloc(&d, sizeof(double) * (size_t)nb * th));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    k_dfma<<<nb, th, 0, ctx->stream>>>(d, 1000, 1.0000001, 1e-9);
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, ctx->stream);
        k_dfma<<<nb, th, 0, ctx->stream>>>(d, iters, 1.0000001, 1e-9);
        cudaEventRecord(e1, ctx->stream);
        cudaEventSynchronize(e1);
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaError_t e = cudaGetLastError();
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    if (e != cudaSuccess) return fail(ctx, TRIMEG_ERR_CUDA, "bench_dfma: %s", cudaGetErrorString(e));
    *tflops = 2.0 * 8 * (double)iters * nb * th / (best * 1e-3) * 1e-12;
    return TRIMEG_OK;
}

int trimeg_push_stats(trimeg_ctx* ctx, int64_t out[4]) {
    if (!ctx || !out) return TRIMEG_ERR_BAD_ARG;
    for (int i = 0; i < 4; ++i) out[i] = ctx->stats[i];
    if (ctx->d_stats) {   // slow-path evaluations are counted on the device
        unsigned long long h[4] = {0, 0, 0, 0};
        CU(cudaSetDevice(ctx->device));
        CU(cudaMemcpyAsync(h, ctx->d_stats, sizeof h, cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        out[1] = (int64_t)h[1];
        out[2] = (int64_t)h[2];
    }
    return TRIMEG_OK;
}

}  // extern "C"
