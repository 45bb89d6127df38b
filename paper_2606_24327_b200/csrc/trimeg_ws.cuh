// Warp-specialised phase kernel (included by trimeg_kernels.cuh after the tile helpers).
//
// One persistent CTA per SM, 16 warps in four warp-groups:
//   warp 0    "stager"     : takes super-cells off the work list, waits until a ring entry is free, fills it (slot geometry,
//                            lane layout of its 32 cells, TMA bulk copies of the coefficient blocks);
//   warps 1-2 "publishers" : once an entry has landed, cut its lanes into chunks of 32 (cells padded to even sizes, see
//                            BlockCtrl) and, for each, copy the chunk's records into a free chunk slot (cp.async through the
//                            sort permutation; completion is signalled on the slot's mbarrier by cp.async.mbarrier.arrive);
//   warp 3    "prefetcher" : follows the stager's work list through a small mailbox and pulls the marker records of every
//                            super-cell into L2 (prefetch.global.L2 through the sort permutation) several ring entries before
//                            the publishers copy them: the chunk slots then only have to cover an L2 latency, not HBM's;
//   warps 4-15 "compute"   : take chunk slots in ticket order, pull their record into registers, evaluate the phase, put
//                            the record back into its slot row, send the chunk off as one bulk store, free the slot and
//                            count the chunk done on its ring entry.
// The light warp-group hands registers to the compute groups (setmaxnreg: 40 / 152 of a 128-register launch).
// A ring entry is refilled when all chunks cut from it are done AND both publishers have read its control block.
#pragma once

namespace trimeg {

// Tuning / debugging builds only (never shipped): -DTRIMEG_WAITSTATS accumulates the cycles each role spends waiting
// (compute warps binned by the chunk count of their ring entry), -DTRIMEG_WATCHDOG replaces every barrier wait by one that
// gives up after ~1 s, records who waited on what (g_dbg) and lets the kernel end (this is how the slot/ticket aliasing
// deadlock fixed in this file was found; profiles/r02_sanitizer.md).
#if defined(TRIMEG_WAITSTATS) || defined(TRIMEG_WATCHDOG)
__device__ unsigned long long g_wait[160][160];   // [block][counter]: per-block, so that the counters do not contend
__device__ int g_abort;
__device__ unsigned long long g_dbg[64];
#endif
#ifdef TRIMEG_WAITSTATS
#define WS_T0() const long long ws_t0__ = clock64()
#define WS_ADD(i) do { if ((threadIdx.x & 31) == 0) atomicAdd(&g_wait[blockIdx.x][i], (unsigned long long)(clock64() - ws_t0__)); } while (0)
#else
#define WS_T0() do {} while (0)
#define WS_ADD(i) do {} while (0)
#endif
#ifdef TRIMEG_WATCHDOG
TRIMEG_DI bool mbar_wait_wd(void* bar, unsigned parity, int code, int aux) {
    const long long t0 = clock64();
    bool recorded = false;
    for (unsigned spin = 0;; ++spin) {
        unsigned ok;
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
        if (ok) return true;
        if ((spin & 255) == 255) {
            const long long el = clock64() - t0;
            if (!recorded && el > 2000000000ll) {
                recorded = true;
                if ((threadIdx.x & 31) == 0) {
                    const unsigned long long slot = atomicAdd(&g_dbg[0], 1ull);
                    if (slot < 15) { g_dbg[4 * slot + 4] = code; g_dbg[4 * slot + 5] = blockIdx.x; g_dbg[4 * slot + 6] = threadIdx.x >> 5; g_dbg[4 * slot + 7] = (unsigned long long)aux; }
                }
            }
            if (el > 3000000000ll) *(volatile int*)&g_abort = 1;
            if (*(volatile int*)&g_abort) return false;
        }
    }
}
#define MBW(bar, parity, code, aux) do { if (!mbar_wait_wd(bar, parity, code, aux)) return; } while (0)
#define WS_ABORTED() (*(volatile int*)&g_abort)
TRIMEG_DI bool mbar_wait_any(void* bar, unsigned parity, int code, int aux) { return mbar_wait_wd(bar, parity, code, aux); }
#else
#define MBW(bar, parity, code, aux) mbar_wait(bar, parity)
#define WS_ABORTED() false
TRIMEG_DI bool mbar_wait_any(void* bar, unsigned parity, int, int) { mbar_wait(bar, parity); return true; }
#endif

// stager, part 1: take the next non-empty super-cell off the work list and pull everything its ring entry needs out of
// global memory into registers (lane l holds slot l and cell l).  Done BEFORE a ring entry is free, so that only
// shared-memory writes and the TMA issue remain once it is.  Returns false when the work list is exhausted.
struct StageWork { int sc, patch, k0, ns, t, off, off_end, incl, npad; double ox, oy; SlotGeom g; };
template <class C>
TRIMEG_DI bool ws_fetch(const DevTables& tb, const TileTables& tt, int* work_counter, int lane, StageWork& w) {
    constexpr unsigned FULL = 0xffffffffu;
    static_assert(C::CPS == 32, "one cell per lane");
    int sc = 0;
    for (;;) {
        if (lane == 0) sc = atomicAdd(work_counter, 1);
        sc = __shfl_sync(FULL, sc, 0);
        if (sc >= tt.nsc) return false;
        const int o = tt.offs[(long long)sc * C::CPS + lane], o1 = tt.offs[(long long)sc * C::CPS + lane + 1];
        int incl = (o1 - o + 1) & ~1;                    // lanes of this cell (even), then inclusive prefix sum over the cells
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const int y = __shfl_up_sync(FULL, incl, d); if (lane >= d) incl += y; }
        w.npad = __shfl_sync(FULL, incl, 31);
        w.off = o; w.incl = incl; w.off_end = __shfl_sync(FULL, o1, 31);
        if (w.npad > 0) break;
    }
    w.sc = sc;
    w.patch = sc / tt.nwin; w.k0 = (sc - w.patch * tt.nwin) * C::WK;
    w.ns = tt.nslots[w.patch];
    w.t = -1;
    SlotGeom& g = w.g;
    // an unused slot fails every inside test (xi = eta = -1) and leads nowhere
    g.a11 = g.a12 = g.a21 = g.a22 = 0.0; g.c1 = g.c2 = -1.0;
    g.nbr[0] = g.nbr[1] = g.nbr[2] = g.nbr[3] = -1; g.pad[0] = g.pad[1] = 0;
    TriGeom tg;
    tg.v0x = tg.v0y = 0.0;
    if (lane < w.ns) {
        w.t = tt.slots[(long long)w.patch * C::SGEOM + lane];
        if (w.t >= 0) tg = tb.geom[w.t];
    }
    // origin of the affine forms: vertex 0 of the patch's first triangle (slot 0 always holds an own triangle)
    w.ox = __shfl_sync(FULL, tg.v0x, 0); w.oy = __shfl_sync(FULL, tg.v0y, 0);
    if (w.t >= 0) {
        g.a11 = tg.a11; g.a12 = tg.a12; g.a21 = tg.a21; g.a22 = tg.a22;
        const double ex = w.ox - tg.v0x, ey = w.oy - tg.v0y;      // a few element sizes: no cancellation in c
        g.c1 = fma(tg.a11, ex, tg.a12 * ey);
        g.c2 = fma(tg.a21, ex, tg.a22 * ey);
        const short* nb = tt.nbr + ((long long)w.patch * C::SGEOM + lane) * 4;
        g.nbr[0] = nb[0]; g.nbr[1] = nb[1]; g.nbr[2] = nb[2];
    }
    return true;
}
// stager, part 2: fill the (free) ring entry b from registers and start the TMA bulk copies of its coefficient blocks
template <class C>
TRIMEG_DI void ws_commit(unsigned char* smem, int b, const DevTables& tb, const StageWork& w, int lane) {
    constexpr unsigned FULL = 0xffffffffu;
    double* coef = reinterpret_cast<double*>(smem + C::BLOCK_BYTES * b);
    SlotGeom* sgeom = reinterpret_cast<SlotGeom*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES);
    BlockCtrl* ctl = reinterpret_cast<BlockCtrl*>(smem + C::OFF_CTRL + C::CTRL_BYTES * b);
    unsigned long long* full = reinterpret_cast<unsigned long long*>(smem + C::OFF_BAR) + 2 * b;
    if (lane == 0) {
        ctl->sc = w.sc; ctl->patch = w.patch; ctl->k0 = w.k0; ctl->ns = w.ns; ctl->npad = w.npad;
        ctl->nchunks = (w.npad + 31) >> 5;
        ctl->ox = w.ox; ctl->oy = w.oy;
        *reinterpret_cast<volatile int*>(&ctl->done) = 0;
        ctl->cell_off[32] = w.off_end;
    }
    ctl->cell_off[lane] = w.off;
    ctl->pad_incl[lane] = w.incl;
    sgeom[lane] = w.g;
    reinterpret_cast<int*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES + C::GEOM_BYTES)[lane] = w.t;
    const bool has_coef = w.t >= 0 && lane < C::SMAX;
    const int cnt = __popc(__ballot_sync(FULL, has_coef));
    __threadfence_block();
    fence_async_smem();   // earlier generic accesses of this block vs. the async writes
    __syncwarp();
    if (lane == 0) mbar_expect_tx(full, (unsigned)(cnt * C::SLOT_DOUBLES * sizeof(double)));
    __syncwarp();
    if (has_coef)
        tma_bulk_g2s(coef + (size_t)lane * C::SLOT_DOUBLES, tb.coef + (long long)w.t * tb.tri_stride + (long long)w.k0 * PLANE_STRIDE,
                     (unsigned)(C::SLOT_DOUBLES * sizeof(double)), full);
}

// Edge walk inside the staged block from slot sl for the point (dR, dZ) (relative to the patch origin): returns the slot
// containing it or a negative code: -1 left the staged set (or hop cap), -2 crossed the mesh boundary.  On success
// xi, eta are the point's reference coordinates in that triangle and j[] its J^-1 (the walk's own numbers: one
// shared-memory round trip per hop, nothing to recompute afterwards).
TRIMEG_DI int slot_walk(const SlotGeom* __restrict__ sgeom, int sl, double dR, double dZ, double& xi, double& eta, double j[4]) {
    if (sl < 0) return -1;
    const unsigned base = smem_u32(sgeom);
#pragma unroll 1
    for (int hop = 0; hop < 16; ++hop) {
        const unsigned ad = base + 64u * (unsigned)sl;
        double c1, c2, nn, pp;
        lds128(ad, j[0], j[1]); lds128(ad + 16, j[2], j[3]); lds128(ad + 32, c1, c2); lds128(ad + 48, nn, pp);
        xi = fma(j[0], dR, fma(j[1], dZ, c1));
        eta = fma(j[2], dR, fma(j[3], dZ, c2));
        const double l0 = (1.0 - xi) - eta;
        if (xi >= INSIDE_TOL && eta >= INSIDE_TOL && l0 >= INSIDE_TOL) return sl;
        const int nlo = __double2loint(nn), nhi = __double2hiint(nn);
        sl = (eta <= xi && eta <= l0) ? (short)nlo : ((l0 <= xi) ? (nlo >> 16) : (short)nhi);
        if (sl < 0) return sl;
    }
    return -1;
}

// toroidal interval and fraction for phi inside [0, period) without the modulo (the general routine otherwise): the state's
// phi is wrapped once per step, so the evaluation points of a step stay within a fraction of an interval of that range
TRIMEG_DI int interval_fast(const TorP& tp, double phi, double& s) {
    const double u = phi * tp.inv_dphi, kf = floor(u);
    const int k = __double2int_rz(kf);
    if ((unsigned)k < (unsigned)tp.P) { s = u - kf; return k; }
    return toroidal_interval(tp, phi, s);
}

template <class C, int PHASE>
__global__ void __launch_bounds__(C::NTHREADS, 1)
k_phase_ws(DevTables tb, TileTables tt, EquilP ep, SpeciesP sp, const Rec* src, Rec* dst, const int* __restrict__ perm,
           RetireList rq, KeyOut ko, CellMap cm, double dt, int* __restrict__ work_counter) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    unsigned long long* blk_bar = reinterpret_cast<unsigned long long*>(smem + C::OFF_BAR);      // [b][0] full, [b][1] seen
    ChunkDesc* desc = reinterpret_cast<ChunkDesc*>(smem + C::OFF_DESC);
    unsigned long long* chunk_bar = reinterpret_cast<unsigned long long*>(smem + C::OFF_CBAR);   // [s][0] full, [s][1] empty
    unsigned char* ltab = smem + C::OFF_LTAB;                                                    // [s][lane] record row, 0xff = idle lane
    int* cons_head = reinterpret_cast<int*>(smem + C::OFF_HEAD);
    int* pfq = reinterpret_cast<int*>(smem + C::OFF_PFQ);                                        // [PFQ][2] (begin, end), then the sequence number
    volatile int* pf_seq = pfq + 2 * C::PFQ;
    constexpr unsigned FULL = 0xffffffffu;
    auto ctl_of = [&](int b) { return reinterpret_cast<BlockCtrl*>(smem + C::OFF_CTRL + C::CTRL_BYTES * b); };
    if (tid == 0) {
        for (int b = 0; b < C::NBUF; ++b) { mbar_init(blk_bar + 2 * b, 1); mbar_init(blk_bar + 2 * b + 1, C::NPUB); }
        for (int s = 0; s < C::K; ++s) { mbar_init(chunk_bar + 2 * s, 64); mbar_init(chunk_bar + 2 * s + 1, 1); }   // full: per lane one plain + one copy-completion arrival
        *cons_head = 0;
        *pf_seq = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (wid < C::NLIGHT) {
        reg_dealloc<C::REG_LIGHT>();
        if (wid == 0) {
            // ------------------------------------------------------------------ stager
            StageWork w;
            int posted = 0;
            auto post = [&](bool have_) {   // tell the prefetcher which records come next (begin = -1: no more work)
                const int begin = __shfl_sync(FULL, w.off, 0);
                if (C::NPUB + 1 >= C::NLIGHT) {   // no prefetcher warp
                    return;
                }
                if (lane == 0) {
                    pfq[2 * (posted % C::PFQ)] = have_ ? begin : -1; pfq[2 * (posted % C::PFQ) + 1] = w.off_end;
                    __threadfence_block();
                    *pf_seq = posted + 1;
                }
                ++posted;
            };
            bool have = ws_fetch<C>(tb, tt, work_counter, lane, w);
            post(have);
            for (unsigned it = 0;; ++it) {
                const int b = it % C::NBUF;
                if (it >= (unsigned)C::NBUF) {
                    WS_T0();
                    // previous occupant: both publishers have read its control block, and all chunks cut from it are done
                    MBW(blk_bar + 2 * b + 1, (it / C::NBUF - 1) & 1, 1, (int)it);
                    BlockCtrl* ctl = ctl_of(b);
                    if (lane == 0) {
                        const int need = ctl->nchunks;
#ifdef TRIMEG_WATCHDOG
                        const long long t0 = clock64();
                        while (*reinterpret_cast<volatile int*>(&ctl->done) < need) {
                            __nanosleep(64);
                            if (*(volatile int*)&g_abort) break;
                            if (clock64() - t0 > 2000000000ll) {
                                const unsigned long long slot = atomicAdd(&g_dbg[0], 1ull);
                                if (slot < 15) { g_dbg[4 * slot + 4] = 2; g_dbg[4 * slot + 5] = blockIdx.x; g_dbg[4 * slot + 6] = ((unsigned long long)need << 32) | (unsigned)*reinterpret_cast<volatile int*>(&ctl->done); g_dbg[4 * slot + 7] = it; }
                                *(volatile int*)&g_abort = 1;
                                break;
                            }
                        }
#else
                        while (*reinterpret_cast<volatile int*>(&ctl->done) < need) __nanosleep(64);
#endif
                    }
                    __syncwarp();
                    WS_ADD(0);
                    if (WS_ABORTED()) return;
                }
                if (!have) {   // end of work: the entry carries sc = -1 and its barrier completes at once
                    if (lane == 0) {
                        ctl_of(b)->sc = -1;
                        __threadfence_block();
                        mbar_arrive(blk_bar + 2 * b);
                    }
                    break;
                }
                ws_commit<C>(smem, b, tb, w, lane);
                have = ws_fetch<C>(tb, tt, work_counter, lane, w);   // the next entry's global loads overlap the compute warps' work
                post(have);
            }
        } else if (wid <= C::NPUB) {
            // ------------------------------------------------------------------ publishers: warp pid takes the tickets t with t % NPUB == pid
            const unsigned pid = wid - 1;
            unsigned ticket = 0;
            auto slot_acquire = [&](unsigned t) {   // wait until the previous user of the slot has been copied out
                const unsigned s = t % C::K, g = t / C::K;
                WS_T0();
                if (g >= 1) { if (!mbar_wait_any(chunk_bar + 2 * s + 1, (g - 1) & 1, 3, (int)t)) return -1; }
                WS_ADD(3);
                return (int)s;
            };
            for (unsigned it = 0;; ++it) {
                const int b = it % C::NBUF;
                { WS_T0(); MBW(blk_bar + 2 * b, (it / C::NBUF) & 1, 4, (int)it); WS_ADD(2); }
                const BlockCtrl* ctl = ctl_of(b);
                const int sc = ctl->sc;
                int c_off = 0, c_end = 0, c_incl = 0, npad = 0;
                if (sc >= 0) { c_off = ctl->cell_off[lane]; c_end = ctl->cell_off[lane + 1]; c_incl = ctl->pad_incl[lane]; npad = ctl->npad; }
                __syncwarp();
                if (lane == 0) mbar_arrive(blk_bar + 2 * b + 1);   // control block read: the stager may refill once the chunks are done
                if (sc < 0) break;
                // the chunks of this entry carry tickets ticket .. ticket + nch - 1; ours are those of parity pid
                const unsigned t0 = ticket, nch = (unsigned)(npad + 31) >> 5;
                ticket = t0 + nch;
                // lane position g of the entry -> cell (binary search in the inclusive prefix sums held one per lane) -> marker;
                // returns the chunk's first record, sets its record count, this lane's row (0xff: idle lane) and the source
                // record of row `lane` (the permutation entry: a global load that stays in flight while the previous chunk is
                // being copied)
                auto layout = [&](unsigned t, int& nrec, int& rowl, int& pr) {
                    const int g = 32 * (int)(t - t0) + lane;
                    int cell = 0;
#pragma unroll
                    for (int st = 16; st >= 1; st >>= 1) { const int v = __shfl_sync(FULL, c_incl, cell + st - 1); if (v <= g) cell += st; }
                    cell = min(cell, 31);
                    const int o = __shfl_sync(FULL, c_off, cell), oe = __shfl_sync(FULL, c_end, cell), pin = __shfl_sync(FULL, c_incl, cell);
                    const int m = o + (g - (pin - ((oe - o + 1) & ~1)));      // position within the (padded) cell
                    const bool valid = g < npad && m < oe;                  // the pad lane of an odd cell is idle
                    const unsigned vmask = __ballot_sync(FULL, valid);     // lane 0 is always valid (cells start on even lanes)
                    const int m_first = __shfl_sync(FULL, m, 0);
                    nrec = __shfl_sync(FULL, m, 31 - __clz(vmask)) - m_first + 1;
                    rowl = valid ? (m - m_first) : 0xff;
                    pr = m_first + lane;
                    if (perm && lane < nrec) pr = perm[pr];
                    return m_first;
                };
                // software pipeline of depth 3: the permutation entries of a chunk are loaded (global memory: several microseconds
                // under load) three of this publisher's chunks before its records are copied
                unsigned t = t0 + (pid + C::NPUB - t0 % C::NPUB) % C::NPUB;
                int mq0 = 0, nq0 = 0, rq0 = 0, pq0 = 0, mq1 = 0, nq1 = 0, rq1 = 0, pq1 = 0, mq2 = 0, nq2 = 0, rq2 = 0, pq2 = 0;
                if (t < t0 + nch) mq0 = layout(t, nq0, rq0, pq0);
                if (t + C::NPUB < t0 + nch) mq1 = layout(t + C::NPUB, nq1, rq1, pq1);
                if (t + 2 * C::NPUB < t0 + nch) mq2 = layout(t + 2 * C::NPUB, nq2, rq2, pq2);
                for (; t < t0 + nch; t += C::NPUB) {
                    const int m_first = mq0, nrec = nq0, rowl = rq0, pr = pq0;
                    mq0 = mq1; nq0 = nq1; rq0 = rq1; pq0 = pq1;
                    mq1 = mq2; nq1 = nq2; rq1 = rq2; pq1 = pq2;
                    { WS_T0(); if (t + 3 * C::NPUB < t0 + nch) mq2 = layout(t + 3 * C::NPUB, nq2, rq2, pq2); WS_ADD(8); }
                    const int s = slot_acquire(t);
                    if (s < 0) return;
                    if (lane == 0) { desc[s].m0 = m_first; desc[s].nrec = nrec; desc[s].b = b; desc[s].ticket = (int)t; }
                    ltab[s * 32 + lane] = (unsigned char)rowl;
                    // descriptor and lane table are published by a plain (release) arrival of every lane: no fence here - a
                    // membar would also wait for the copies still in flight and for the next chunk's permutation loads, i.e.
                    // for a global-memory latency per chunk (that made the publishers the bottleneck: profiles/r02_summary.md)
                    __syncwarp();
                    mbar_arrive(chunk_bar + 2 * s);
                    WS_T0();
                    const unsigned ib = smem_u32(smem + C::OFF_STAGE + (size_t)s * C::WSTAGE);
                    const int ch = lane & 7, q = lane >> 3;
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        const int r = 4 * k + q;                                   // row of the chunk slot = record m_first + r of dst
                        const int ri = __shfl_sync(FULL, pr, r);
                        if (r < nrec) {
                            // logical 16-byte chunk j of a record sits at position j ^ rec_swizzle(index): source position ch
                            const int j = ch ^ rec_swizzle(ri);
                            const unsigned d = ib + r * 128 + 16 * (j ^ rec_swizzle(m_first + r));
                            const char* gp = reinterpret_cast<const char*>(src + ri) + 16 * ch;
                            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gp) : "memory");
                        }
                    }
                    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(chunk_bar + 2 * s)) : "memory");
                    WS_ADD(9);
                }
            }
            // one end-of-work ticket per compute warp
            for (int q = 0; q < C::NCOMP; ++q, ++ticket) {
                if (ticket % C::NPUB != pid) continue;
                const int s = slot_acquire(ticket);
                if (s < 0) return;
                if (lane == 0) { desc[s].m0 = -1; desc[s].ticket = (int)ticket; }
                __syncwarp();
                mbar_arrive(chunk_bar + 2 * s);
                mbar_arrive(chunk_bar + 2 * s);
            }
        } else if (wid < C::NLIGHT) {
            // ------------------------------------------------------------------ prefetcher (a hint only: nothing waits for it)
            for (int n = 0;; ++n) {
                while (*pf_seq <= n) { __nanosleep(200); if (WS_ABORTED()) return; }
                __threadfence_block();
                const int begin = pfq[2 * (n % C::PFQ)], end = pfq[2 * (n % C::PFQ) + 1];
                if (begin < 0) break;
#ifndef TRIMEG_NO_PREFETCH
                for (int i = begin + lane; i < end; i += 32)
#else
                for (int i = begin + lane; i < begin; i += 32)
#endif
                {
                    const int ri = perm ? perm[i] : i;
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(src + ri));
                }
            }
        }
    } else {
        reg_alloc<C::REG_COMP>();
        // ------------------------------------------------------------------ compute warps
        const int P = tb.tor.P;
        unsigned t_next = 0;
        if (lane == 0) t_next = (unsigned)atomicAdd(cons_head, 1);
        for (;;) {
            const unsigned t = __shfl_sync(FULL, t_next, 0);
            const unsigned s = t % C::K, gen = t / C::K;
#ifdef TRIMEG_WAITSTATS
            const long long ws_it0 = clock64();
            long long ws_wait = 0;
#endif
            // A compute warp holds up to two tickets (the one it works on and the next), so more tickets can be outstanding
            // than there are chunk slots: a warp may reach its wait while the slot's PREVIOUS generation has not been published
            // yet, and a parity wait cannot tell "two phases behind" from "done".  The descriptor's ticket number can.
            { WS_T0();
              for (;;) {
                  MBW(chunk_bar + 2 * s, gen & 1, 5, (int)t);
                  if (*reinterpret_cast<volatile int*>(&desc[s].ticket) == (int)t) break;
                  __nanosleep(100);
              }
              WS_ADD(4);
#ifdef TRIMEG_WAITSTATS
              ws_wait = clock64() - ws_t0__;
#endif
            }
            const int m0 = desc[s].m0, nrec = desc[s].nrec, b = desc[s].b;
            if (m0 < 0) break;
            const int rowi = ltab[s * 32 + lane];
            const bool valid = rowi != 0xff;
            const int m = m0 + rowi;
            const unsigned row = smem_u32(smem + C::OFF_STAGE + (size_t)s * C::WSTAGE) + rowi * 128;
            const int sw = rec_swizzle(m);
            // next ticket now, so that its latency hides behind the arithmetic (volatile asm: as a plain atomicAdd the
            // compiler sinks it to the end of the iteration, next to the other lane-0 work, and its latency is exposed)
            if (lane == 0) asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(t_next) : "r"(smem_u32(cons_head)) : "memory");

            const double* coef = reinterpret_cast<const double*>(smem + C::BLOCK_BYTES * b);
            const SlotGeom* sgeom = reinterpret_cast<const SlotGeom*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES);
            const int* stri = reinterpret_cast<const int*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES + C::GEOM_BYTES);
            BlockCtrl* ctl = ctl_of(b);
            const int patch = ctl->patch, k0 = ctl->k0, ns = ctl->ns;
            const double ox = ctl->ox, oy = ctl->oy;
            if (valid) {
                // The record STAYS in its row of the chunk slot (16-byte chunks: 0 = y0 y1, 1 = y2 y3, 2 = y4 k0, 3 = k1 k2,
                // 4 = k3 k4, 5 = mu p, 6 = tri st | id pad0); every use re-reads what it needs, so that the gather (the
                // register-hungry part) runs with only the evaluation point live.  The row is not written before the phase
                // has succeeded: a retired marker's row goes out as it came in.
                auto ldr = [&](int j, double& x, double& y) { lds128(row + 16 * (j ^ sw), x, y); };
                double ti, ii;
                ldr(6, ti, ii);
                int st = __double2hiint(ti), slot = -1;
                const int tri0 = __double2loint(ti);
                if (PHASE == PHASE_A && (st & 2)) st = (st | 1) & ~2;   // the cached k1 = f(y_n) was evaluated outside: that stage belongs to this step
                if (PHASE == PHASE_INIT) st &= ~2;                       // k1 is being recomputed
                {
                    const int sl = tri0 - patch * C::TP;
                    if (sl >= 0 && sl < C::TP) slot = sl;
                    else {   // not sorted since it moved: look for the triangle in the halo
                        for (int q = C::TP; q < ns; ++q) if (stri[q] == tri0) { slot = q; break; }
                    }
                }
                auto eval = [&](const double y[5], double d[5]) {
#ifdef TRIMEG_NOEVAL   // tuning builds only: the record pipeline without the arithmetic
                    d[0] = d[1] = d[2] = d[3] = d[4] = 0.0;
                    return true;
#endif
                    double xi, eta, jj[4], sf;
                    const int sl = slot_walk(sgeom, slot, y[0] - ox, y[1] - oy, xi, eta, jj);
                    const int k = interval_fast(tb.tor, y[2], sf);
                    int dk = k - k0;
                    if (dk > P / 2) dk -= P; else if (dk < -(P / 2)) dk += P;
                    const int lk = dk + C::HK;
                    if (!(sl >= 0 && sl < C::SMAX && lk >= 0 && lk < C::NW)) return false;   // slots >= SMAX carry geometry only
                    slot = sl;
                    double w[4], dw[4], g8[8];
                    bspline_from_s<double>(tb.tor, sf, w, dw);
                    LdShared ld{smem_u32(coef + (size_t)sl * C::SLOT_DOUBLES + (size_t)lk * PLANE_STRIDE)};
                    gather_cell<false, double>(ld, xi, eta, w, dw, g8);
                    FieldsG<double> f;
                    to_fields_g<double>(jj[0], jj[1], jj[2], jj[3], g8, y[3], f);
                    double mu, pw;
                    ldr(5, mu, pw);
                    rhs_eval<double>(ep, sp, y[0], y[1], y[3], y[4], mu, pw, f, d);
                    return true;
                };
                const double h2 = 0.5 * dt, h6 = dt / 6.0;
                double y[5], d[5], a[5], next[3];
                bool ok;
                auto ld_y = [&](double v[5]) { double t; ldr(0, v[0], v[1]); ldr(1, v[2], v[3]); ldr(2, v[4], t); };
                auto ld_k = [&](double v[5]) { double t; ldr(2, t, v[0]); ldr(3, v[1], v[2]); ldr(4, v[3], v[4]); };
                if (PHASE == PHASE_A) {
                    double yn[5], k1[5];
                    ld_y(yn); ld_k(k1);
#pragma unroll
                    for (int q = 0; q < 5; ++q) y[q] = fma(h2, k1[q], yn[q]);
                } else if (PHASE == PHASE_B) ld_k(y);          // y4
                else ld_y(y);                                  // y_n
                // the two evaluations run through ONE copy of the evaluation code (a rolled loop: instruction cache)
#pragma unroll 1
                for (int e = (PHASE == PHASE_INIT ? 1 : 0); e < 2; ++e) {
                    ok = eval(y, d);
                    if (!ok) break;
                    if (e == 0) {
                        double yn[5];
                        ld_y(yn);                              // A: y_n;  B: Y = y_n + dt/6 (k1 + 2 k2 + 2 k3)
#pragma unroll
                        for (int q = 0; q < 5; ++q) {
                            a[q] = d[q];                                                        // A: k2
                            y[q] = PHASE == PHASE_A ? fma(h2, d[q], yn[q]) : fma(h6, d[q], yn[q]);  // A: y_n + dt/2 k2;  B: y_{n+1}
                        }
                        if (PHASE == PHASE_B) y[2] = wrap_phi(tb.tor, y[2]);
                    }
                }
                if (ok) {
                    double ny[5], nk[5];
                    if (PHASE == PHASE_A) {
                        double yn[5], k1[5];
                        ld_y(yn); ld_k(k1);
#pragma unroll
                        for (int q = 0; q < 5; ++q) {
                            ny[q] = fma(h6, fma(2.0, d[q], fma(2.0, a[q], k1[q])), yn[q]);     // Y
                            nk[q] = fma(dt, d[q], yn[q]);                                      // y4 = y_n + dt k3
                        }
                        next[0] = nk[0]; next[1] = nk[1]; next[2] = nk[2];
                    } else {
#pragma unroll
                        for (int q = 0; q < 5; ++q) { ny[q] = y[q]; nk[q] = d[q]; }            // y_{n+1} (INIT: y_n), k1 = f(it)
                        next[0] = fma(h2, d[0], y[0]); next[1] = fma(h2, d[1], y[1]); next[2] = fma(h2, d[2], y[2]);
                    }
                    // triangle of the next phase's first evaluation point: staged walk; a point that left the staged geometry is
                    // located through the global tables by k_fix_keys (the record keeps the last triangle as its hint)
                    double xi, eta, jj[4];
                    const int sl = slot_walk(sgeom, slot, next[0] - ox, next[1] - oy, xi, eta, jj);
                    int tn;
                    if (sl >= 0) {
                        tn = stri[sl];
                        if (ko.enabled) {
                            double sf;
                            const int k = interval_fast(tb.tor, next[2], sf);
                            const int key = cm.cell(tn, k);
                            ko.keys[m] = key;
                            atomicAdd(ko.hist + key, 1);
                        }
                    } else {
                        tn = stri[slot];
                        rq.list[rq.n - 1 - atomicAdd(rq.count + 1, 1)] = m;
                    }
                    // the record goes back into its row of the chunk slot ...
                    auto str = [&](int j, double x, double yv) { sts128(row + 16 * (j ^ sw), x, yv); };
                    str(0, ny[0], ny[1]); str(1, ny[2], ny[3]); str(2, ny[4], nk[0]); str(3, nk[1], nk[2]); str(4, nk[3], nk[4]);
                    str(6, __hiloint2double(st, tn), ii);
                } else {
                    // the follow-up kernel redoes this phase through the global tables from the untouched record (its row is
                    // left as it came in and goes to dst[m] with the rest of the chunk)
                    rq.list[atomicAdd(rq.count, 1)] = m;
                }
            }
            // ... and the chunk leaves as ONE bulk copy (32 scattered 128-byte lines would cost 224 LSU wavefronts as STG.128)
#ifdef TRIMEG_WAITSTATS
            const long long ws_tail0 = clock64();
#endif
            fence_async_smem();
            __syncwarp();
            if (lane == 0) {
                tma_bulk_s2g(dst + m0, smem + C::OFF_STAGE + (size_t)s * C::WSTAGE, (unsigned)(nrec * 128));
                bulk_commit();
                __threadfence_block();
                atomicAdd(&ctl->done, 1);            // one more chunk of this ring entry done
                bulk_wait_read0();                   // the copy has read the slot:
                mbar_arrive(chunk_bar + 2 * s + 1);  // it may be refilled
#ifdef TRIMEG_WAITSTATS
                atomicAdd(&g_wait[blockIdx.x][6], (unsigned long long)(clock64() - ws_tail0));
                atomicAdd(&g_wait[blockIdx.x][5], (unsigned long long)(clock64() - ws_it0));
                atomicAdd(&g_wait[blockIdx.x][7], 1ull);
                const int bin = min(ctl->nchunks, 47);
                atomicAdd(&g_wait[blockIdx.x][16 + bin], (unsigned long long)ws_wait);          // cycles waiting for the chunk
                atomicAdd(&g_wait[blockIdx.x][64 + bin], (unsigned long long)(clock64() - ws_it0));
                atomicAdd(&g_wait[blockIdx.x][112 + bin], 1ull);
#endif
            }
        }
    }
}

}  // namespace trimeg
