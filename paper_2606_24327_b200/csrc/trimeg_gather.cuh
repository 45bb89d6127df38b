// Staged grid-to-particle gather for many points in any order (trimeg_gather; BASELINE configs[4]).
//
// One field evaluation reads 8 x 168 B of coefficients per point; through L1/L2 with the points in caller order that is
// 7x the algorithmic HBM traffic on config 4 (profiles/r01c_gather_cfg4.md).  Here the library bins the points itself:
//   1. k_gather_keys     caller order: box-grid locate (L89, L125-140), toroidal interval -> bin key, histogram (the atomic's
//                        return value is the point's rank within its bin).  A bin is a (triangle, window of GW intervals):
//                        the staged kernel does not care about the order within it, and 8x fewer counters than cells stay
//                        in L2;
//   2. scan              (the push's counting-sort kernels) -> bin offsets;
//   3. k_gather_scatter  caller order: position = offset + rank; 32-byte point record written there (a full sector),
//                        position kept per caller index;
//   4. k_gather_staged   persistent CTAs, one super-cell (GT triangles x GW toroidal intervals) at a time, dealt out
//                        round-robin: its coefficient block, geometry and point records arrive by TMA bulk copies (two
//                        stages, 'landed' / 'consumed' mbarriers, no CTA-wide barrier), warps evaluate its points from
//                        shared memory and write 64-byte result records in bin order (coalesced).  Bound by shared-memory
//                        bandwidth (1 344 B of coefficients per point, ~4 wavefronts per LDS.128);
//   5. k_gather_unsort   caller order: result record (fetched by a lane pair as one 64-byte request) -> the caller's eight
//                        arrays (coalesced writes), triangle id.
// HBM bytes per point: 36 + 68 + (96 + coefficients) + 140, against 92 + coefficients algorithmic; DESIGN.md section 6,
// profiles/r02_gather_cfg4.md.
#pragma once

namespace trimeg {

// tuning knobs of the staged kernel (python -m paper_2606_24327_b200.build --defs "-DTRIMEG_GT=8 ..."): triangles per
// super-cell, threads per CTA, CTAs per SM, TMA stages
#ifndef TRIMEG_GT
#define TRIMEG_GT 4
#endif
#ifndef TRIMEG_GTHREADS
#define TRIMEG_GTHREADS 96
#endif
#ifndef TRIMEG_GOCC
#define TRIMEG_GOCC 6
#endif
#ifndef TRIMEG_GNST
#define TRIMEG_GNST 2
#endif
constexpr int GT = TRIMEG_GT, GW = 8;                       // triangles x toroidal intervals per gather super-cell
constexpr int GNPL = GW + 3;                        // staged planes per triangle
constexpr int GSLOT = GNPL * PLANE_STRIDE;          // doubles per staged triangle
#ifndef TRIMEG_GKEY_CELL
#define TRIMEG_GKEY_CELL 0
#endif
// bins per super-cell: one per (triangle, window) - the order of a triangle's points within the window does not matter to the
// staged kernel, and 8x fewer counters keep the histogram L2-resident - or, as a tuning build, one per cell
constexpr int GCELLS = TRIMEG_GKEY_CELL ? GT * GW : GT;
constexpr int GTHREADS = TRIMEG_GTHREADS;

struct GatherMap {   // bin numbering of the gather: super-cell (patch, window) major, then triangle (then interval)
    int nwin;
    __host__ __device__ __forceinline__ int cell(int t, int k) const {
        const int patch = t / GT, tl = t - patch * GT, w = k / GW, kl = k - w * GW;
        return TRIMEG_GKEY_CELL ? ((patch * nwin + w) * GT + tl) * GW + kl : (patch * nwin + w) * GT + tl;
    }
};
struct __align__(32) GPoint { double R, Z, phi; int id, tri; };   // one point in cell order (32 B = one sector)
static_assert(sizeof(GPoint) == 32, "GPoint");
// 256-bit global accesses (sm_100: LDG/STG.256): a 32-byte record is one request and one full sector
TRIMEG_DI void ld256(const void* p, double& a, double& b, double& c, double& d) {
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
TRIMEG_DI void st256(void* p, double a, double b, double c, double d) {
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// Which path?  A strided sample of runs of 32 consecutive points: if most neighbours share a cell the caller's order is
// already clustered and the direct kernel (coefficients through L1/L2) is the faster one; otherwise the points are binned.
// flag[0] = 1 direct, 2 staged; every kernel of either path returns at once if the flag names the other path, so the choice
// costs no host round trip.
constexpr int GPROBE_RUNS = 2048;
__global__ void __launch_bounds__(32) k_gather_probe(DevTables tb, GatherMap gm, long long n, const double* __restrict__ R, const double* __restrict__ Z,
                                                     const double* __restrict__ phi, int* __restrict__ cnt) {
    const long long nruns = n / 32;
    const long long run = (long long)blockIdx.x * (nruns / gridDim.x > 0 ? nruns / gridDim.x : 1);
    const long long i = run * 32 + threadIdx.x;
    int key = -2 - (int)threadIdx.x;
    if (i < n) {
        const int t = locate_box(tb.bg, tb.geom, R[i], Z[i]);
        double s;
        const int k = toroidal_interval(tb.tor, phi[i], s);
        key = t < 0 ? -1 : gm.cell(t, k);
    }
    const int up = __shfl_down_sync(0xffffffffu, key, 1);
    const unsigned same = __ballot_sync(0xffffffffu, threadIdx.x < 31 && up == key);
    if (threadIdx.x == 0) { atomicAdd(cnt, __popc(same)); atomicAdd(cnt + 1, 31); }
}
__global__ void k_gather_decide(int mode, const int* __restrict__ cnt, int* __restrict__ flag) {
    // clustered if more than 30 % of the sampled neighbours share a cell (cell-sorted input: ~60 % at 2.6 points per cell;
    // random input: ~0)
    flag[0] = mode == 1 ? 1 : (mode == 2 ? 2 : (10 * cnt[0] > 3 * cnt[1] ? 1 : 2));
}

__global__ void __launch_bounds__(256) k_gather_keys(DevTables tb, GatherMap gm, long long n, const double* __restrict__ R, const double* __restrict__ Z,
                                                     const double* __restrict__ phi, int ncell, int* __restrict__ keys, int* __restrict__ tris,
                                                     int* __restrict__ ranks, int* __restrict__ hist, const int* __restrict__ flag) {
    if (*flag != 2) return;      // fixed grid + grid-stride loop: the path not taken costs microseconds, not a 5e7-thread launch
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int t = locate_box(tb.bg, tb.geom, R[i], Z[i]);
        double s;
        const int k = toroidal_interval(tb.tor, phi[i], s);
        const int key = t < 0 ? ncell : gm.cell(t, k);
        keys[i] = key;
        tris[i] = t;
        ranks[i] = atomicAdd(hist + key, 1);      // the old count is this point's rank within its cell: the scatter needs no second atomic
    }
}

__global__ void __launch_bounds__(256) k_gather_scatter(long long n, const double* __restrict__ R, const double* __restrict__ Z, const double* __restrict__ phi,
                                                        const int* __restrict__ keys, const int* __restrict__ tris, const int* __restrict__ offs,
                                                        GPoint* __restrict__ pts, int* __restrict__ inv, const int* __restrict__ flag) {
    if (*flag != 2) return;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int key = keys[i];
        const int pos = offs[key] + inv[i];      // inv[] comes in holding the rank within the cell and leaves holding the position
        st256(pts + pos, R[i], Z[i], phi[i], __hiloint2double(tris[i], (int)i));     // (id, tri) in the low and high word
        inv[i] = pos;
    }
}

// shared memory of one CTA: GNST stages of { coefficients [GT][GSLOT], geometry [GT] }, then control.  The kernel is bound by
// the latency of one super-cell's round (wait, evaluate, barrier), not by bytes, so many small CTAs beat few large ones:
// measured on config 4 (profiles/r02_gather_cfg4.md), 8 triangles x 256 threads x 2 CTAs/SM x 3 stages 3.70 ms,
// 4 triangles x 96 threads x 6 CTAs/SM x 2 stages 3.01 ms (the default; ~83 points per super-cell there fill 96 lanes to 87 %).
constexpr int GNST = TRIMEG_GNST;
constexpr int GPCAP = GTHREADS;                     // point records staged with a super-cell (the first pass of its evaluation)
struct GatherSmem {
    static constexpr size_t COEF = sizeof(double) * GT * GSLOT;
    static constexpr size_t OFF_PTS = COEF + sizeof(TriGeom) * GT;
    static constexpr size_t STAGE = OFF_PTS + sizeof(GPoint) * GPCAP;
    static constexpr size_t OFF_CTRL = GNST * STAGE;      // per stage: 'landed' mbarrier (8 B), unit, begin, end (ints), pad, 'consumed' mbarrier (8 B)
    static constexpr size_t BYTES = OFF_CTRL + GNST * 32;
};

__global__ void __launch_bounds__(GTHREADS, TRIMEG_GOCC)
k_gather_staged(DevTables tb, GatherMap gm, int nunits, int NPP, const int* __restrict__ offs, const GPoint* __restrict__ pts,
                double* __restrict__ res, int* __restrict__ work_counter, const int* __restrict__ flag) {
    extern __shared__ __align__(128) unsigned char smem[];
    if (*flag != 2) return;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    auto bar_of = [&](int s) { return reinterpret_cast<unsigned long long*>(smem + GatherSmem::OFF_CTRL + 32 * s); };
    auto ctl_of = [&](int s) { return reinterpret_cast<int*>(smem + GatherSmem::OFF_CTRL + 32 * s + 8); };
    auto done_of = [&](int s) { return reinterpret_cast<unsigned long long*>(smem + GatherSmem::OFF_CTRL + 32 * s + 24); };
    constexpr int NW = GTHREADS / 32;
    if (tid == 0) {
        for (int q = 0; q < GNST; ++q) { mbar_init(bar_of(q), 1); mbar_init(done_of(q), NW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    // warp 0 stages.  Super-cells are dealt out round-robin (CTA b takes b, b + grid, ...: ~700 per CTA on config 4, so the load
    // evens out) and the point range of the NEXT one is loaded while the current one is being issued, so that staging is
    // issue-only: no global round trip sits between the end of a round and the next round's copies.  (With a work counter
    // and the geometry copied by the warp itself, warp 0 came 2-3 us late to every round's barrier: 38 % of the kernel's
    // stall samples were the other warps waiting there, profiles/r02_gather_cfg4.md.)
    static_assert(sizeof(TriGeom) == 64, "geometry records are copied in bulk");
    int nu = blockIdx.x, nbeg = 0, nend = 0;               // warp 0: the next super-cell and its point range
    auto fetch = [&]() { if (nu < nunits) { nbeg = offs[(long long)nu * GCELLS]; nend = offs[(long long)(nu + 1) * GCELLS]; } };
    if (wid == 0) fetch();
    auto stage = [&](int s, unsigned use) {                  // use: how often stage s has been filled before
        if (use > 0) mbar_wait(done_of(s), (use - 1) & 1);    // every warp is done with its previous contents
        while (nu < nunits && nbeg == nend) { nu += gridDim.x; fetch(); }        // empty super-cells are skipped
        const int u = nu < nunits ? nu : -1, begin = nbeg, end = nend;
        nu += gridDim.x; fetch();
        int* ctl = ctl_of(s);
        if (lane == 0) { ctl[0] = u; ctl[1] = begin; ctl[2] = end; }
        if (u < 0) { __syncwarp(); if (lane == 0) mbar_arrive(bar_of(s)); return; }
        const int patch = u / gm.nwin, w = u - patch * gm.nwin;
        const int pp0 = w * GW + PLANE_PAD, npl = min(GNPL, NPP - pp0);
        const int t = patch * GT + lane;
        const int cnt = min(GT, tb.T - patch * GT);
        const bool has = lane < cnt;
        unsigned char* st = smem + GatherSmem::STAGE * s;
        const unsigned bytes = (unsigned)(npl * PLANE_STRIDE * sizeof(double));
        // the super-cell's first GPCAP point records come with it: the evaluation starts from shared memory
        const unsigned pbytes = (unsigned)(min(end - begin, GPCAP) * (int)sizeof(GPoint));
        const unsigned gbytes = (unsigned)(cnt * (int)sizeof(TriGeom));
        if (lane == 0) mbar_expect_tx(bar_of(s), cnt * bytes + pbytes + gbytes);
        __syncwarp();
        if (has) tma_bulk_g2s(reinterpret_cast<double*>(st) + (size_t)lane * GSLOT, tb.coef + (long long)t * tb.tri_stride + (long long)pp0 * PLANE_STRIDE, bytes, bar_of(s));
        if (lane == 0) {
            tma_bulk_g2s(st + GatherSmem::COEF, tb.geom + (long long)patch * GT, gbytes, bar_of(s));
            tma_bulk_g2s(st + GatherSmem::OFF_PTS, pts + begin, pbytes, bar_of(s));
        }
    };
    // No CTA-wide barrier per round: a warp that is done with a stage says so on the stage's 'consumed' barrier and goes on to
    // the next stage, so the warps may drift apart by up to GNST - 1 rounds.  A super-cell with more points than threads
    // gives some warp a second pass; with a barrier per round the other warps stood idle for it (28 % of all stall samples),
    // now they work ahead, and the lane numbering rotates by one warp per round so that the extra pass is not always warp 0's.
    if (wid == 0) { for (int q = 0; q < GNST - 1; ++q) stage(q, 0); }
    for (unsigned it = 0;; ++it) {
        const int s = it % GNST;
        if (wid == 0) stage((it + GNST - 1) % GNST, (it + GNST - 1) / GNST);
        mbar_wait(bar_of(s), (it / GNST) & 1);
        const int* ctl = ctl_of(s);
        const int u = ctl[0], begin = ctl[1], end = ctl[2];
        if (u < 0) break;
        const int patch = u / gm.nwin, w = u - patch * gm.nwin;
        const double* coef = reinterpret_cast<const double*>(smem + GatherSmem::STAGE * s);
        const TriGeom* geom = reinterpret_cast<const TriGeom*>(smem + GatherSmem::STAGE * s + GatherSmem::COEF);
        const int rot = tid + 32 * (int)(it % NW), vt = rot >= GTHREADS ? rot - GTHREADS : rot;
        for (int pos = begin + vt; pos < end; pos += GTHREADS) {
            GPoint p;
            {
                double it;
                if (pos - begin < GPCAP) {
                    const double2* sp = reinterpret_cast<const double2*>(smem + GatherSmem::STAGE * s + GatherSmem::OFF_PTS) + 2 * (pos - begin);
                    const double2 a = sp[0], b = sp[1];
                    p.R = a.x; p.Z = a.y; p.phi = b.x; it = b.y;
                } else {
                    ld256(pts + pos, p.R, p.Z, p.phi, it);
                }
                p.id = __double2loint(it); p.tri = __double2hiint(it);
            }
            const int tl = p.tri - patch * GT;
            const TriGeom& g = geom[tl];
            double xi, eta, bw[4], dw[4], acc[8];
            ref_coords(g, p.R, p.Z, xi, eta);
            const int k = bspline_weights(tb.tor, p.phi, bw, dw);
            LdShared ld{smem_u32(coef + (size_t)tl * GSLOT + (size_t)(k - w * GW) * PLANE_STRIDE)};
            gather_cell<true, double>(ld, xi, eta, bw, dw, acc);
            Fields f;
            to_fields(g, acc, f);
            st256(res + 8ll * pos, f.P, f.PR, f.PZ, f.Pp);
            st256(res + 8ll * pos + 4, f.A, f.AR, f.AZ, f.Ap);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(done_of(s));            // this warp is done with stage s
    }
}

__global__ void __launch_bounds__(256) k_gather_unsort(long long n, const int* __restrict__ tris, const int* __restrict__ inv, const double* __restrict__ res,
                                                       const int* __restrict__ orig, double* __restrict__ out, int* __restrict__ tri_out,
                                                       const int* __restrict__ flag) {
    if (*flag != 2) return;
    // A warp takes 32 consecutive caller indices.  Each 64-byte result record is fetched by a PAIR of lanes (one 32-byte
    // half each, so the pair's two accesses are one 64-byte request), 16 records per load instruction; the halves are then
    // handed to the lane that writes the point (coalesced stores into the caller's eight arrays).
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, half = lane & 1, pl = lane >> 1;
    const long long nround = (n + 31) / 32 * 32;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nround; i += (long long)gridDim.x * blockDim.x) {
        int t = -1, pos = 0;
        if (i < n) { t = tris[i]; pos = inv[i]; }
        double q[2][4];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int ts = __shfl_sync(FULL, t, 16 * h + pl), ps = __shfl_sync(FULL, pos, 16 * h + pl);
            q[h][0] = q[h][1] = q[h][2] = q[h][3] = 0.0;
            if (ts >= 0) ld256(res + 8ll * ps + 4 * half, q[h][0], q[h][1], q[h][2], q[h][3]);
        }
        const int src = 2 * (lane & 15);
#pragma unroll
        for (int f = 0; f < 8; ++f) {
            const double v0 = __shfl_sync(FULL, q[0][f & 3], src + (f >> 2)), v1 = __shfl_sync(FULL, q[1][f & 3], src + (f >> 2));
            if (i < n) out[(long long)f * n + i] = lane < 16 ? v0 : v1;
        }
        if (tri_out && i < n) tri_out[i] = t < 0 ? -1 : orig[t];
    }
}

}  // namespace trimeg
