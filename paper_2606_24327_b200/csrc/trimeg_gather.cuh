// Staged grid-to-particle gather for many points in any order (trimeg_gather; BASELINE configs[4]).
//
// One field evaluation reads 8 x 168 B of coefficients per point; through L1/L2 with the points in caller order that is
// 7x the algorithmic HBM traffic on config 4 (profiles/r01c_gather_cfg4.md).  Here the library bins the points itself:
//   1. k_gather_keys     caller order: box-grid locate (L89, L125-140), toroidal interval -> bin key, histogram (the atomic's
//                        return value is the point's rank within its bin).  A bin is a (triangle, window of GW intervals):
//                        the staged kernel does not care about the order within it, and 8x fewer counters than cells stay
//                        in L2;
//   2. scan              (the push's counting-sort kernels) -> bin offsets;
//   3. k_gather_scatter  caller order: position = offset + rank; 32-byte point record (with the caller's index) written there
//                        (a full sector);
//   4. k_gather_staged   persistent CTAs, one super-cell (GT triangles x GW toroidal intervals) at a time, dealt out
//                        round-robin: its coefficient block, geometry and point records arrive by TMA bulk copies (two
//                        stages, 'landed' / 'consumed' mbarriers, no CTA-wide barrier), warps evaluate its points from
//                        shared memory and write each 64-byte result record at the CALLER's index (two full sectors,
//                        scattered).  Bound by shared-memory bandwidth (1 344 B of coefficients per point, ~4 wavefronts
//                        per LDS.128);
//   5. k_gather_unsort   caller order: result record (read in order) -> the caller's eight arrays, triangle id.
// HBM bytes per point: 36 + 64 + (96 + coefficients) + 136, against 92 + coefficients algorithmic; DESIGN.md section 6,
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
                                                        GPoint* __restrict__ pts, const int* __restrict__ ranks, const int* __restrict__ flag) {
    if (*flag != 2) return;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int key = keys[i];
        const int pos = offs[key] + ranks[i];    // rank within the bin: the value the histogram atomic of k_gather_keys returned
        st256(pts + pos, R[i], Z[i], phi[i], __hiloint2double(tris[i], (int)i));     // (id, tri) in the low and high word
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
            // the result record goes to the CALLER's index (two full sectors, scattered), so that the last pass reads its input
            // in order: 3.0 + 1.1 ms against 2.9 + 1.8 ms with records in bin order and a random-read un-sort (config 4)
            st256(res + 8ll * p.id, f.P, f.PR, f.PZ, f.Pp);
            st256(res + 8ll * p.id + 4, f.A, f.AR, f.AZ, f.Ap);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(done_of(s));            // this warp is done with stage s
    }
}

__global__ void __launch_bounds__(256) k_gather_unsort(long long n, const int* __restrict__ tris, const double* __restrict__ res,
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
        if (i < n) { t = tris[i]; pos = (int)i; }
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

// ---------------------------------------------------------------------------------------------------------------------
// Points the caller has already clustered by cell (BASELINE configs[4], second run): no binning, no un-sorting, results written
// straight into the caller's arrays.  The direct kernel (k_gather) reads every coefficient pair with one LDG.128 whose 32
// lanes sit in ~12 different cells: 12 L1 tag look-ups per instruction, 84 instructions per point - it is bound by the L1
// tag stage (profiles/r02_gather_cfg4.md).  Here every WARP works on its own: it takes 32 consecutive points, locates them,
// finds the runs of equal (triangle, window) among its lanes, has the coefficient block of each of the first RW_SLOTS runs
// copied into its private shared-memory slots by TMA (3.7 KB per run, its own mbarrier), and evaluates from shared memory;
// lanes of further runs read through L1/L2.  No CTA-wide synchronisation: ~20 warps per SM, each at its own point of the
// load -> locate -> copy -> evaluate -> store sequence, cover one another's latencies.
#ifdef TRIMEG_WAITSTATS
#define RW_CLK(c) const long long c = clock64()
#define RW_ACC(c0, c1, c2, c3, c4) do { if (lane == 0) { unsigned long long* gw = g_wait[blockIdx.x % 160]; atomicAdd(gw + 30, (unsigned long long)(c1 - c0)); \
    atomicAdd(gw + 31, (unsigned long long)(c2 - c1)); atomicAdd(gw + 32, (unsigned long long)(c3 - c2)); atomicAdd(gw + 33, (unsigned long long)(c4 - c3)); atomicAdd(gw + 34, 1ull); } } while (0)
#else
#define RW_CLK(c) do {} while (0)
#define RW_ACC(c0, c1, c2, c3, c4) do {} while (0)
#endif
#ifndef TRIMEG_RW_SLOTS
#define TRIMEG_RW_SLOTS 3
#endif
#ifndef TRIMEG_RW_WARPS
#define TRIMEG_RW_WARPS 4
#endif
#ifndef TRIMEG_RW_OCC
#define TRIMEG_RW_OCC 4
#endif
constexpr int RW_SLOTS = TRIMEG_RW_SLOTS, RW_WARPS = TRIMEG_RW_WARPS;
struct GatherRunsSmem {
    static constexpr size_t WARP = sizeof(double) * RW_SLOTS * GSLOT;      // coefficient slots of one warp
    static constexpr size_t OFF_BAR = RW_WARPS * WARP;
    static constexpr size_t BYTES = OFF_BAR + 8 * RW_WARPS;
};
// (The same kernel fed with the library's own bin-ordered records, as the evaluation step of the staged path, was measured too:
// 3.2 ms against k_gather_staged's 2.9 ms on config 4 - the super-cell kernel stays.)
__global__ void __launch_bounds__(32 * RW_WARPS, TRIMEG_RW_OCC)
k_gather_runs(DevTables tb, GatherMap gm, int NPP, long long n, const double* __restrict__ R, const double* __restrict__ Z, const double* __restrict__ phi,
              double* __restrict__ out, int* __restrict__ tri_out, int* __restrict__ work_counter, const int* __restrict__ flag) {
    extern __shared__ __align__(128) unsigned char smem[];
    if (flag && *flag != 1) return;
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    double* slots = reinterpret_cast<double*>(smem + GatherRunsSmem::WARP * wid);
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(smem + GatherRunsSmem::OFF_BAR) + wid;
    if (lane == 0) { mbar_init(bar, 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
    __syncwarp();
    const long long ngroups = (n + 31) / 32;
    // software pipeline: while the copies of group g are in flight the warp locates the points of its next group (loaded one
    // iteration earlier) and loads those of the one after, so a group costs max(copy, locate) + evaluation instead of
    // load + locate + copy + evaluation (measured per group before: 1 200 + 7 000 + 500 + 4 300 cycles, the 7 000 being the
    // dependent chain point -> box -> list -> geometry)
    // groups are handed out in chunks of RW_CHUNK consecutive ones off a work counter (the next chunk is claimed while the
    // current one is worked on): consecutive groups keep the same-triangle hint useful and the locate's loads in L1, the
    // counter evens out the warps (with a static split the slowest warp set the kernel's time: SMs 60 % busy on average)
    constexpr int RW_CHUNK = 32;
    auto claim = [&]() { int c = 0; if (lane == 0) c = atomicAdd(work_counter, 1); return (long long)__shfl_sync(FULL, c, 0) * RW_CHUNK; };
    long long gpos = claim(), gnext = claim(), gstop = min(ngroups, gpos + RW_CHUNK);
    auto next_group = [&]() -> long long {
        if (gpos >= gstop) {
            if (gpos >= ngroups) return ngroups;
            gpos = gnext; gstop = min(ngroups, gpos + RW_CHUNK); gnext = claim();
            if (gpos >= ngroups) return ngroups;
        }
        return gpos++;
    };
    auto load = [&](long long grp, double& r, double& z, double& ph) {
        const long long i = grp * 32 + lane;
        r = 0; z = 0; ph = 0;
        if (grp < ngroups && i < n) { r = R[i]; z = Z[i]; ph = phi[i]; }
    };
    // the previous group of this warp ended in triangle `hint`; in clustered input most of the next points lie in it too, so one
    // test against it (one address for the whole warp, an L1 hit) replaces the box lookup's chain of dependent loads
    // (measured: 5 900 of a group's 10 300 cycles) for them
    auto locate = [&](long long grp, double r, double z, int hint) {
        if (!(grp < ngroups && grp * 32 + lane < n)) return -1;
#ifdef TRIMEG_RW_NOLOCATE
        if (hint >= 0) return hint;
#endif
        if (hint >= 0) {                            // one test (the caller's triangle numbering need not be spatial: no walk)
            double xi, eta;
            ref_coords(tb.geom[hint], r, z, xi, eta);
            if (fmin(fmin(xi, eta), 1.0 - xi - eta) >= 0.0) return hint;
        }
        return locate_box(tb.bg, tb.geom, r, z);
    };
    auto last_of = [&](int t) {                      // triangle of the warp's last located lane, -1 if none
        const unsigned m = __ballot_sync(FULL, t >= 0);
        return m ? __shfl_sync(FULL, t, 31 - __clz(m)) : -1;
    };
    double r, z, ph, rn, zn, phn;
    long long grp = next_group(), grp1 = next_group();
    load(grp, r, z, ph);
    load(grp1, rn, zn, phn);
    int t = locate(grp, r, z, -1);
    for (unsigned round = 0; grp < ngroups; ++round) {
        const long long i = grp * 32 + lane;
        double s;
        RW_CLK(c0);
        const int k = toroidal_interval(tb.tor, ph, s);
        const int w = k / GW, pp0 = w * GW + PLANE_PAD;
        const int bid = t >= 0 ? t * gm.nwin + w : -1;
        const int prev = __shfl_up_sync(FULL, bid, 1);
        const bool head = bid >= 0 && (lane == 0 || prev != bid);
        const unsigned hm = __ballot_sync(FULL, head);
        const int run = __popc(hm & (0xffffffffu >> (31 - lane))) - 1;     // heads at or before this lane; -1: leading points outside the mesh
        const unsigned bytes = (unsigned)(min(GNPL, NPP - pp0) * PLANE_STRIDE * (int)sizeof(double));
        const bool issue = head && run < RW_SLOTS;
        unsigned tot = issue ? bytes : 0u;
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) tot += __shfl_xor_sync(FULL, tot, o);
        fence_async_smem();                    // this warp's reads of its slots (previous group) come before the copies that overwrite them
        if (lane == 0) mbar_expect_tx(bar, tot);
        __syncwarp();
        if (issue) tma_bulk_g2s(slots + (size_t)run * GSLOT, tb.coef + (long long)t * tb.tri_stride + (long long)pp0 * PLANE_STRIDE, bytes, bar);
        double rf, zf, phf;
        RW_CLK(c1);
        const long long grp2 = next_group();
        load(grp2, rf, zf, phf);
        RW_CLK(c1a);
        const int tn = locate(grp1, rn, zn, last_of(t));
        RW_CLK(c2);
#ifdef TRIMEG_WAITSTATS
        if (lane == 0) atomicAdd(g_wait[blockIdx.x % 160] + 35, (unsigned long long)(c1a - c1));
#endif
        Fields f = Fields{0, 0, 0, 0, 0, 0, 0, 0};
        int orig = -1;
        mbar_wait(bar, round & 1);
        RW_CLK(c3);
        if (t >= 0) {
            const TriGeom g = tb.geom[t];
            double xi, eta, acc[8], bw[4], dw[4];
            ref_coords(g, r, z, xi, eta);
            bspline_from_s<double>(tb.tor, s, bw, dw);
            if (run < RW_SLOTS) {
#ifdef TRIMEG_RW_NOEVAL
                const double2 v = *reinterpret_cast<const double2*>(slots + (size_t)run * GSLOT + (size_t)(k - w * GW) * PLANE_STRIDE);
                for (int q = 0; q < 8; ++q) acc[q] = v.x * xi + v.y * eta + bw[q & 3] + dw[q & 3];
#else
                LdShared ld{smem_u32(slots + (size_t)run * GSLOT + (size_t)(k - w * GW) * PLANE_STRIDE)};
                gather_cell<true, double>(ld, xi, eta, bw, dw, acc);
#endif
            } else {
                LdGlobal ld{reinterpret_cast<const double2*>(tb.coef + (long long)t * tb.tri_stride + (long long)(k + PLANE_PAD) * PLANE_STRIDE)};
                gather_cell<true, double>(ld, xi, eta, bw, dw, acc);
            }
            to_fields(g, acc, f);
            orig = g.orig;
        }
        if (i < n) {
            out[i] = f.P; out[n + i] = f.PR; out[2 * n + i] = f.PZ; out[3 * n + i] = f.Pp;
            out[4 * n + i] = f.A; out[5 * n + i] = f.AR; out[6 * n + i] = f.AZ; out[7 * n + i] = f.Ap;
            if (tri_out) tri_out[i] = orig;
        }
        RW_CLK(c4);
        RW_ACC(c0, c1, c2, c3, c4);
        r = rn; z = zn; ph = phn; t = tn;
        rn = rf; zn = zf; phn = phf;
        grp = grp1; grp1 = grp2;
        __syncwarp();
    }
}

}  // namespace trimeg
