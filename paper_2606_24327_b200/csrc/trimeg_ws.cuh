// Warp-specialised phase kernel, two markers per lane (included by trimeg_kernels.cuh after the tile helpers).
//
// One persistent CTA per SM, 16 warps in four warp-groups:
//   warp 0    "stager"     : takes super-cells off the work list, waits until a ring entry is free, fills it (slot geometry,
//                            pair layout of its 32 cells, TMA bulk copies of the coefficient blocks);
//   warps 1-2 "publishers" : once an entry has landed, cut its markers into chunks of 32 PAIRS (two markers of the same cell
//                            per lane; an odd cell leaves one half-empty pair) and, for each chunk, copy its <= 64 records
//                            into a free chunk slot (cp.async through the sort permutation, completion on the slot's mbarrier);
//   warp 3                 : spare (only takes part in the register hand-over);
//   warps 4-7 "locators"   : take computed chunks in ticket order, find the triangle of every marker's NEXT evaluation point
//                            (edge walk in the staged geometry), write the next sort key and its histogram count, and send the
//                            chunk off as one bulk store.  This latency-bound bookkeeping would otherwise sit between the FP64
//                            sections of the compute warps;
//   warps 8-15 "compute"   : take chunk slots in ticket order; each lane evaluates the phase for its two markers in lock-step
//                            (type D2): one LDS.128 of a coefficient pair feeds 2 fields x 2 markers, and the FP64 pipe sees two
//                            independent dependency chains per warp.  The records go back into their slot rows.
// The light warps hand their registers to the compute groups (setmaxnreg: 40 / 216 of a 128-register launch).
// A ring entry is refilled when all chunks cut from it have left AND both publishers have read its control block.
#pragma once

namespace trimeg {

// stager, part 1: take the next non-empty super-cell off the work list and pull everything its ring entry needs out of
// global memory into registers (lane l holds slot l and cell l).  Done BEFORE a ring entry is free, so that only
// shared-memory writes and the TMA issue remain once it is.  Returns false when the work list is exhausted.
struct StageWork { int sc, patch, k0, ns, t, off, off_end, incl, npairs; SlotGeom g; };
template <class C>
TRIMEG_DI bool ws_fetch(const DevTables& tb, const TileTables& tt, int* work_counter, int lane, StageWork& w) {
    constexpr unsigned FULL = 0xffffffffu;
    int sc = 0;
    for (;;) {
        if (lane == 0) sc = atomicAdd(work_counter, 1);
        sc = __shfl_sync(FULL, sc, 0);
        if (sc >= tt.nsc) return false;
        const int o = tt.offs[(long long)sc * C::CPS + lane], o1 = tt.offs[(long long)sc * C::CPS + lane + 1];
        int incl = (o1 - o + 1) >> 1;                    // pairs of this lane's cell, then inclusive prefix sum over the cells
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const int y = __shfl_up_sync(FULL, incl, d); if (lane >= d) incl += y; }
        w.npairs = __shfl_sync(FULL, incl, 31);
        w.off = o; w.incl = incl; w.off_end = __shfl_sync(FULL, o1, 31);
        if (w.npairs > 0) break;
    }
    w.sc = sc;
    w.patch = sc / tt.nwin; w.k0 = (sc - w.patch * tt.nwin) * C::WK;
    w.ns = tt.nslots[w.patch];
    w.t = -1;
    SlotGeom& g = w.g;
    // an unused slot fails every inside test (all barycentrics = -1) and leads nowhere
    g.v0x = g.v0y = 0.0; g.a11 = g.a12 = g.a21 = g.a22 = 0.0; g.c1 = g.c2 = -1.0; g.l0a = g.l0b = 0.0; g.l0c = -1.0;
    g.nbr[0] = g.nbr[1] = g.nbr[2] = g.nbr[3] = -1;
    if (lane < w.ns) {
        w.t = tt.slots[(long long)w.patch * C::SGEOM + lane];
        if (w.t >= 0) {
            const TriGeom tg = tb.geom[w.t];
            g.v0x = tg.v0x; g.v0y = tg.v0y; g.a11 = tg.a11; g.a12 = tg.a12; g.a21 = tg.a21; g.a22 = tg.a22;
            g.c1 = -fma(tg.a11, tg.v0x, tg.a12 * tg.v0y);
            g.c2 = -fma(tg.a21, tg.v0x, tg.a22 * tg.v0y);
            g.l0a = -(tg.a11 + tg.a21); g.l0b = -(tg.a12 + tg.a22); g.l0c = 1.0 - g.c1 - g.c2;
            const short* nb = tt.nbr + ((long long)w.patch * C::SGEOM + lane) * 4;
            g.nbr[0] = nb[0]; g.nbr[1] = nb[1]; g.nbr[2] = nb[2];
        }
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
        ctl->sc = w.sc; ctl->patch = w.patch; ctl->k0 = w.k0; ctl->ns = w.ns; ctl->npairs = w.npairs;
        ctl->nchunks = (w.npairs + 31) >> 5;
        *reinterpret_cast<volatile int*>(&ctl->done) = 0;
        ctl->cell_off[32] = w.off_end;
    }
    ctl->cell_off[lane] = w.off;
    ctl->pair_incl[lane] = w.incl;
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

// Edge walk of the two markers of a lane inside the staged block, in lock-step (one copy of the code, two independent
// dependency chains).  out = slot containing the point, or a negative code: -1 left the staged set (or hop cap), -2 crossed
// the mesh boundary; xi, eta are valid where out >= 0.
TRIMEG_DI void slot_walk2(const SlotGeom* __restrict__ sgeom, int slA, int slB, D2 R, D2 Z, int& outA, int& outB, D2& xi, D2& eta) {
    bool doneA = slA < 0, doneB = slB < 0;
    int curA = max(slA, 0), curB = max(slB, 0);
    outA = -1; outB = -1;
#pragma unroll 1
    for (int hop = 0; hop < 16; ++hop) {
        const SlotGeom& gA = sgeom[curA];
        const SlotGeom& gB = sgeom[curB];
        const D2 l1 = fma(D2(gA.a11, gB.a11), R, fma(D2(gA.a12, gB.a12), Z, D2(gA.c1, gB.c1)));
        const D2 l2 = fma(D2(gA.a21, gB.a21), R, fma(D2(gA.a22, gB.a22), Z, D2(gA.c2, gB.c2)));
        const D2 l0 = fma(D2(gA.l0a, gB.l0a), R, fma(D2(gA.l0b, gB.l0b), Z, D2(gA.l0c, gB.l0c)));
        const int2 nA = *reinterpret_cast<const int2*>(gA.nbr), nB = *reinterpret_cast<const int2*>(gB.nbr);   // all three neighbours at once
        if (!doneA) {
            if (l1.a >= INSIDE_TOL && l2.a >= INSIDE_TOL && l0.a >= INSIDE_TOL) { doneA = true; outA = curA; }
            else {
                const int nb = (l2.a <= l1.a && l2.a <= l0.a) ? (short)nA.x : ((l0.a <= l1.a) ? (nA.x >> 16) : (short)nA.y);
                if (nb < 0) { doneA = true; outA = nb; } else curA = nb;
            }
        }
        if (!doneB) {
            if (l1.b >= INSIDE_TOL && l2.b >= INSIDE_TOL && l0.b >= INSIDE_TOL) { doneB = true; outB = curB; }
            else {
                const int nb = (l2.b <= l1.b && l2.b <= l0.b) ? (short)nB.x : ((l0.b <= l1.b) ? (nB.x >> 16) : (short)nB.y);
                if (nb < 0) { doneB = true; outB = nb; } else curB = nb;
            }
        }
        if (doneA && doneB) break;
    }
    // coordinates for the evaluation, cancellation-free
    const SlotGeom& gA = sgeom[max(outA, 0)];
    const SlotGeom& gB = sgeom[max(outB, 0)];
    const D2 dx = R - D2(gA.v0x, gB.v0x), dy = Z - D2(gA.v0y, gB.v0y);
    xi = fma(D2(gA.a11, gB.a11), dx, D2(gA.a12, gB.a12) * dy);
    eta = fma(D2(gA.a21, gB.a21), dx, D2(gA.a22, gB.a22) * dy);
}

// the same for one marker, result only (locator warps: few registers)
TRIMEG_DI int slot_walk1(const SlotGeom* __restrict__ sgeom, int sl, double R, double Z) {
    if (sl < 0) return -1;
#pragma unroll 1
    for (int hop = 0; hop < 16; ++hop) {
        const SlotGeom& g = sgeom[sl];
        const double l1 = fma(g.a11, R, fma(g.a12, Z, g.c1)), l2 = fma(g.a21, R, fma(g.a22, Z, g.c2)), l0 = fma(g.l0a, R, fma(g.l0b, Z, g.l0c));
        const int2 n = *reinterpret_cast<const int2*>(g.nbr);
        if (l1 >= INSIDE_TOL && l2 >= INSIDE_TOL && l0 >= INSIDE_TOL) return sl;
        sl = (l2 <= l1 && l2 <= l0) ? (short)n.x : ((l0 <= l1) ? (n.x >> 16) : (short)n.y);
        if (sl < 0) return sl;
    }
    return -1;
}

template <class C, int PHASE>
__global__ void __launch_bounds__(C::NTHREADS, 1)
k_phase_ws(DevTables tb, TileTables tt, EquilP ep, SpeciesP sp, const Rec* src, Rec* dst, const int* __restrict__ perm,
           RetireList rq, KeyOut ko, CellMap cm, double dt, int* __restrict__ work_counter) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    unsigned long long* blk_bar = reinterpret_cast<unsigned long long*>(smem + C::OFF_BAR);      // [b][0] full, [b][1] seen
    ChunkDesc* desc = reinterpret_cast<ChunkDesc*>(smem + C::OFF_DESC);
    unsigned char* ltab = smem + C::OFF_LTAB;
    unsigned long long* chunk_bar = reinterpret_cast<unsigned long long*>(smem + C::OFF_CBAR);   // [s][0] full, [s][1] computed, [s][2] empty
    unsigned char* lflag = smem + C::OFF_LFLAG;
    int* cons_head = reinterpret_cast<int*>(smem + C::OFF_HEAD);
    constexpr unsigned FULL = 0xffffffffu;
    auto ctl_of = [&](int b) { return reinterpret_cast<BlockCtrl*>(smem + C::OFF_CTRL + C::CTRL_BYTES * b); };
    if (tid == 0) {
        for (int b = 0; b < C::NBUF; ++b) { mbar_init(blk_bar + 2 * b, 1); mbar_init(blk_bar + 2 * b + 1, 1); }
        for (int s = 0; s < C::K; ++s) { mbar_init(chunk_bar + 3 * s, 32); mbar_init(chunk_bar + 3 * s + 1, 1); mbar_init(chunk_bar + 3 * s + 2, 1); }
        *cons_head = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (wid < C::NLIGHT) {
        reg_dealloc<C::REG_LIGHT>();
        if (wid == 0) {
            // ------------------------------------------------------------------ stager
            StageWork w;
            bool have = ws_fetch<C>(tb, tt, work_counter, lane, w);
            for (unsigned it = 0;; ++it) {
                const int b = it % C::NBUF;
                if (it >= (unsigned)C::NBUF) {
                    // previous occupant: the publisher has read its control block, and all chunks cut from it have left
                    mbar_wait(blk_bar + 2 * b + 1, (it / C::NBUF - 1) & 1);
                    BlockCtrl* ctl = ctl_of(b);
                    if (lane == 0) {
                        const int need = ctl->nchunks;
                        while (*reinterpret_cast<volatile int*>(&ctl->done) < need) __nanosleep(64);
                    }
                    __syncwarp();
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
            }
        } else if (wid == 1) {
            // ------------------------------------------------------------------ publisher: chunks in ticket order.  The layout and the
            // permutation entries of chunk i + 1 are fetched before chunk i is copied in, so that their latency is hidden.
            unsigned ticket = 0;
            auto slot_acquire = [&](unsigned t) {   // wait until the previous user of the slot has been copied out
                const unsigned s = t % C::K, g = t / C::K;
                if (g >= 1) mbar_wait(chunk_bar + 3 * s + 2, (g - 1) & 1);
                return (int)s;
            };
            // a chunk whose layout is known and whose permutation entries are in flight
            int p_have = 0, p_mfirst = 0, p_nrec = 0, p_b = 0, p_pr0 = 0, p_pr1 = 0;
            unsigned char p_lt = 0;
            unsigned p_t = 0;
            auto emit = [&]() {
                const int s = slot_acquire(p_t);
                if (lane == 0) { desc[s].m_first = p_mfirst; desc[s].nrec = p_nrec; desc[s].b = p_b; }
                ltab[s * 32 + lane] = p_lt;
                __threadfence_block();
                __syncwarp();
                const unsigned ib = smem_u32(smem + C::OFF_STAGE + (size_t)s * C::WSTAGE);
                const int ch = lane & 7, q = lane >> 3;
#pragma unroll
                for (int k = 0; k < 16; ++k) {
                    const int r = 4 * k + q;                                   // row of the chunk slot = record m_first + r of dst
                    const int ri = __shfl_sync(FULL, k < 8 ? p_pr0 : p_pr1, r & 31);
                    if (r < p_nrec) {
                        // logical 16-byte chunk j of a record sits at position j ^ rec_swizzle(index): source position ch
                        const int j = ch ^ rec_swizzle(ri);
                        const unsigned d = ib + r * 128 + 16 * (j ^ rec_swizzle(p_mfirst + r));
                        const char* gp = reinterpret_cast<const char*>(src + ri) + 16 * ch;
                        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gp) : "memory");
                    }
                }
                asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(chunk_bar + 3 * s)) : "memory");
                p_have = 0;
            };
            for (unsigned it = 0;; ++it) {
                const int b = it % C::NBUF;
                if (p_have) emit();   // never hold a chunk back while waiting for the next ring entry
                mbar_wait(blk_bar + 2 * b, (it / C::NBUF) & 1);
                const BlockCtrl* ctl = ctl_of(b);
                const int sc = ctl->sc;
                int c_off = 0, c_end = 0, c_incl = 0, npairs = 0;
                if (sc >= 0) { c_off = ctl->cell_off[lane]; c_end = ctl->cell_off[lane + 1]; c_incl = ctl->pair_incl[lane]; npairs = ctl->npairs; }
                __syncwarp();
                if (lane == 0) mbar_arrive(blk_bar + 2 * b + 1);   // control block read: the stager may refill once the chunks are done
                if (sc < 0) break;
                const unsigned t0 = ticket, nch = (unsigned)(npairs + 31) >> 5;
                ticket = t0 + nch;
                for (unsigned t = t0; t < t0 + nch; ++t) {
                    // pair g of the entry -> cell (binary search in the inclusive prefix sums held one per lane) -> marker positions
                    const int g = 32 * (int)(t - t0) + lane;
                    const bool valid = g < npairs;
                    int cell = 0;
#pragma unroll
                    for (int st = 16; st >= 1; st >>= 1) { const int v = __shfl_sync(FULL, c_incl, cell + st - 1); if (v <= g) cell += st; }
                    cell = min(cell, 31);
                    const int o = __shfl_sync(FULL, c_off, cell), oe = __shfl_sync(FULL, c_end, cell), pin = __shfl_sync(FULL, c_incl, cell);
                    const int first_pair = pin - ((oe - o + 1) >> 1);
                    const int mA = o + 2 * (g - first_pair);
                    const int hasB = (valid && mA + 1 < oe) ? 1 : 0;
                    const int m_first = __shfl_sync(FULL, mA, 0);
                    const int last_lane = min(31, npairs - 32 * (int)(t - t0) - 1);
                    const int nrec = __shfl_sync(FULL, mA + hasB, last_lane) - m_first + 1;
                    // source records of rows lane and lane + 32
                    int pr0 = m_first + lane, pr1 = m_first + 32 + lane;
                    if (perm) { if (lane < nrec) pr0 = perm[pr0]; if (lane + 32 < nrec) pr1 = perm[pr1]; }
                    if (p_have) emit();   // the previous chunk goes in while this one's permutation entries are in flight
                    p_have = 1; p_t = t; p_mfirst = m_first; p_nrec = nrec; p_b = b; p_pr0 = pr0; p_pr1 = pr1;
                    p_lt = valid ? (unsigned char)(0x80 | (hasB << 6) | (mA - m_first)) : (unsigned char)0;
                }
            }
            // one end-of-work ticket per compute warp
            for (int q = 0; q < C::NCOMP; ++q, ++ticket) {
                const int s = slot_acquire(ticket);
                if (lane == 0) { desc[s].m_first = -1; __threadfence_block(); }
                __syncwarp();
                mbar_arrive(chunk_bar + 3 * s);
            }
        } else {
            // ------------------------------------------------------------------ locators: warp j takes the tickets t with t % NLOC == j
            const double h2 = 0.5 * dt;
            for (unsigned t = wid - 2;; t += C::NLOC) {
                const unsigned s = t % C::K, gen = t / C::K;
                mbar_wait(chunk_bar + 3 * s + 1, gen & 1);
                const int m_first = desc[s].m_first, nrec = desc[s].nrec, b = desc[s].b;
                if (m_first < 0) break;
                const int lt = ltab[s * 32 + lane], lf = lflag[s * 32 + lane];
                const SlotGeom* sgeom = reinterpret_cast<const SlotGeom*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES);
                const int* stri = reinterpret_cast<const int*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES + C::GEOM_BYTES);
                const BlockCtrl* ctl = ctl_of(b);
                const int patch = ctl->patch, ns = ctl->ns;
                const unsigned slot_base = smem_u32(smem + C::OFF_STAGE + (size_t)s * C::WSTAGE);
    #pragma unroll 1
                for (int x = 0; x < 2; ++x) {                         // the lane's first, then its second marker (one copy of the code)
                    if (!((lf >> x) & 1)) continue;                   // nothing to locate: no marker, or retired
                    const int row = (lt & 63) + x, m = m_first + row;
                    const unsigned ad = slot_base + row * 128;
                    const int sw = rec_swizzle(m);
                    // next evaluation point: after phase A the stage-4 position held in k, otherwise y + dt/2 k
                    double R, Z, phi, y4, k0, k1, k2, ti, ii;
                    lds128(ad + 16 * (2 ^ sw), y4, k0); lds128(ad + 16 * (3 ^ sw), k1, k2); lds128(ad + 16 * (6 ^ sw), ti, ii);
                    if (PHASE == PHASE_A) { R = k0; Z = k1; phi = k2; }
                    else {
                        double y0, y1, y2, y3;
                        lds128(ad + 16 * (0 ^ sw), y0, y1); lds128(ad + 16 * (1 ^ sw), y2, y3);
                        R = fma(h2, k0, y0); Z = fma(h2, k1, y1); phi = fma(h2, k2, y2);
                    }
                    const int tri0 = __double2loint(ti);              // triangle of the last evaluation point (written by the compute warp)
                    int sl = tri0 - patch * C::TP;
                    if (sl < 0 || sl >= C::TP) {
                        sl = -1;
                        for (int q = C::TP; q < ns; ++q) if (stri[q] == tri0) { sl = q; break; }
                    }
                    sl = slot_walk1(sgeom, sl, R, Z);
                    int tn = tri0;
                    if (sl < 0) {   // the point left the staged geometry: k_fix_keys locates it through the global tables (hint: last triangle)
                        rq.list[rq.n - 1 - atomicAdd(rq.count + 1, 1)] = m;
                    } else {
                        tn = stri[sl];
                        if (ko.enabled) {
                            double sf;
                            const int k = toroidal_interval(tb.tor, phi, sf);
                            const int key = cm.cell(tn, k);
                            ko.keys[m] = key;
                            atomicAdd(ko.hist + key, 1);
                        }
                        sts128(ad + 16 * (6 ^ sw), __hiloint2double(__double2hiint(ti), tn), ii);
                    }
                }
                // the chunk leaves as ONE bulk copy
                fence_async_smem();
                __syncwarp();
                if (lane == 0) {
                    tma_bulk_s2g(dst + m_first, smem + C::OFF_STAGE + (size_t)s * C::WSTAGE, (unsigned)(nrec * 128));
                    bulk_commit();
                    __threadfence_block();
                    atomicAdd(&ctl_of(b)->done, 1);      // one more chunk of this ring entry done
                    bulk_wait_read0();                   // the copy has read the slot:
                    mbar_arrive(chunk_bar + 3 * s + 2);  // it may be refilled
                }
            }
        }
    } else {
        reg_alloc<C::REG_COMP>();
        // ------------------------------------------------------------------ compute warps
        const int P = tb.tor.P;
        const double h2 = 0.5 * dt, h6 = dt / 6.0;
        unsigned t_next = 0;
        if (lane == 0) t_next = (unsigned)atomicAdd(cons_head, 1);
        for (;;) {
            const unsigned t = __shfl_sync(FULL, t_next, 0);
            const unsigned s = t % C::K, gen = t / C::K;
            mbar_wait(chunk_bar + 3 * s, gen & 1);
            const int m_first = desc[s].m_first, b = desc[s].b;
            if (m_first < 0) {   // end of work: pass the ticket on so that its locator stops too
                if (lane == 0) mbar_arrive(chunk_bar + 3 * s + 1);
                break;
            }
            const int lt = ltab[s * 32 + lane];
            // next ticket now, so that its latency hides behind the arithmetic
            if (lane == 0) asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(t_next) : "r"(smem_u32(cons_head)) : "memory");
            // lanes without a pair (tail of a super-cell) shadow row 0 and have no side effects; a lane without a second
            // marker evaluates its first one twice
            const bool validA = (lt & 0x80) != 0, validB = (lt & 0x40) != 0;
            const int rowA = lt & 63, rowB = rowA + (validB ? 1 : 0);
            const int mA = m_first + rowA, mB = m_first + rowB;
            const unsigned slot_base = smem_u32(smem + C::OFF_STAGE + (size_t)s * C::WSTAGE);
            const unsigned adA = slot_base + rowA * 128, adB = slot_base + rowB * 128;
            const int swA = rec_swizzle(mA), swB = rec_swizzle(mB);
            auto ld2 = [&](int j, D2& x, D2& y) { lds128(adA + 16 * (j ^ swA), x.a, y.a); lds128(adB + 16 * (j ^ swB), x.b, y.b); };
            const double* coef = reinterpret_cast<const double*>(smem + C::BLOCK_BYTES * b);
            const SlotGeom* sgeom = reinterpret_cast<const SlotGeom*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES);
            const int* stri = reinterpret_cast<const int*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES + C::GEOM_BYTES);
            const BlockCtrl* ctl = ctl_of(b);
            const int patch = ctl->patch, k0 = ctl->k0, ns = ctl->ns;

            // ---- record -> first evaluation point
            D2 y[5], mu, pw;
            int triA, stA, idA, triB, stB, idB;
            {
                D2 r0, r1, r2, r3, r4, k0_, k1_, k2_, k3_, k4_;
                ld2(0, r0, r1); ld2(1, r2, r3); ld2(2, r4, k0_); ld2(3, k1_, k2_); ld2(4, k3_, k4_); ld2(5, mu, pw);
                D2 ti, ii;
                ld2(6, ti, ii);
                triA = __double2loint(ti.a); stA = __double2hiint(ti.a); idA = __double2loint(ii.a);
                triB = __double2loint(ti.b); stB = __double2hiint(ti.b); idB = __double2loint(ii.b);
                if (PHASE == PHASE_A) {        // y_n + dt/2 k1
                    y[0] = fma(D2(h2), k0_, r0); y[1] = fma(D2(h2), k1_, r1); y[2] = fma(D2(h2), k2_, r2); y[3] = fma(D2(h2), k3_, r3); y[4] = fma(D2(h2), k4_, r4);
                } else if (PHASE == PHASE_B) { // y4
                    y[0] = k0_; y[1] = k1_; y[2] = k2_; y[3] = k3_; y[4] = k4_;
                } else {                       // y_n
                    y[0] = r0; y[1] = r1; y[2] = r2; y[3] = r3; y[4] = r4;
                }
            }
            if (PHASE == PHASE_A) {   // the cached k1 = f(y_n) was evaluated outside the mesh: that stage belongs to this step
                if (stA & 2) stA = (stA | 1) & ~2;
                if (stB & 2) stB = (stB | 1) & ~2;
            }
            if (PHASE == PHASE_INIT) { stA &= ~2; stB &= ~2; }   // k1 is being recomputed
            // staged slot of the triangle hint
            auto slot_of = [&](int tri) {
                int sl = tri - patch * C::TP;
                if (sl >= 0 && sl < C::TP) return sl;
                for (int q = C::TP; q < ns; ++q) if (stri[q] == tri) return q;   // not sorted since it moved: look in the halo
                return -1;
            };
            int slotA = slot_of(triA), slotB = slot_of(triB);
            bool retA = false, retB = false;

            // one right-hand-side evaluation for both markers of the lane.  A point outside the staged block retires its
            // marker (the marker then shadows a valid location: its results are never stored).
            auto eval = [&](const D2 yy[5], D2 d[5]) {
                D2 xi, eta, sf;
                int slA, slB;
                slot_walk2(sgeom, slotA, slotB, yy[0], yy[1], slA, slB, xi, eta);
                const int kA = toroidal_interval(tb.tor, yy[2].a, sf.a), kB = toroidal_interval(tb.tor, yy[2].b, sf.b);
                int dkA = kA - k0, dkB = kB - k0;
                if (dkA > P / 2) dkA -= P; else if (dkA < -(P / 2)) dkA += P;
                if (dkB > P / 2) dkB -= P; else if (dkB < -(P / 2)) dkB += P;
                int lkA = dkA + C::HK, lkB = dkB + C::HK;
                if (slA >= 0 && slA < C::SMAX && lkA >= 0 && lkA < C::NW) slotA = slA; else { retA = true; slA = 0; lkA = C::HK; }   // slots >= SMAX carry geometry only
                if (slB >= 0 && slB < C::SMAX && lkB >= 0 && lkB < C::NW) slotB = slB; else { retB = true; slB = 0; lkB = C::HK; }
                const unsigned baseA = smem_u32(coef + (size_t)slA * C::SLOT_DOUBLES + (size_t)lkA * PLANE_STRIDE);
                const unsigned baseB = smem_u32(coef + (size_t)slB * C::SLOT_DOUBLES + (size_t)lkB * PLANE_STRIDE);
                // both markers through marker A's cell (one coefficient load feeds both); where a pair has split (the two
                // points lie in different cells: a few percent of the second evaluations of a phase), marker B again alone
                D2 acc[8];
                gather_cell_rolled<false, D2, LdShared>(baseA, xi, eta, sf, tb.tor.inv_dphi, acc);
                const bool split = baseA != baseB;
                if (__any_sync(FULL, split)) {
                    if (split) {
                        double ab[8];
                        gather_cell_rolled<false, double, LdShared>(baseB, xi.b, eta.b, sf.b, tb.tor.inv_dphi, ab);
#pragma unroll
                        for (int q = 1; q < 8; ++q) acc[q].b = ab[q];
                    }
                }
                const SlotGeom& gA = sgeom[slA];
                const SlotGeom& gB = sgeom[slB];
                FieldsG<D2> f;
                to_fields_g<D2>(D2(gA.a11, gB.a11), D2(gA.a12, gB.a12), D2(gA.a21, gB.a21), D2(gA.a22, gB.a22), acc, yy[3], f);
                // equilibrium and right-hand sides: one marker at a time through ONE copy of the code (registers and
                // instruction cache; three warps per scheduler supply the FP64 pipe's parallelism here)
#pragma unroll 1
                for (int x = 0; x < 2; ++x) {
                    FieldsG<double> fx;
                    fx.gR = x ? f.gR.b : f.gR.a; fx.gZ = x ? f.gZ.b : f.gZ.a; fx.gp = x ? f.gp.b : f.gp.a; fx.A = x ? f.A.b : f.A.a;
                    double dx[5];
                    rhs_eval<double>(ep, sp, x ? yy[0].b : yy[0].a, x ? yy[1].b : yy[1].a, x ? yy[3].b : yy[3].a, x ? yy[4].b : yy[4].a,
                                     x ? mu.b : mu.a, x ? pw.b : pw.a, fx, dx);
#pragma unroll
                    for (int q = 0; q < 5; ++q) { if (x) d[q].b = dx[q]; else d[q].a = dx[q]; }
                }
            };

            D2 d[5], S[5];
            if (PHASE == PHASE_INIT) {
                eval(y, d);                                   // k1 = f(y_n)
            } else {
#pragma unroll 1
                for (int e = 0; e < 2; ++e) {                 // ONE copy of the evaluation code (instruction cache)
                    eval(y, d);
                    if (e == 0) {
                        D2 r0, r1, r2, r3, r4, k0_, k1_, k2_, k3_, k4_;
                        ld2(0, r0, r1); ld2(1, r2, r3); ld2(2, r4, k0_);
                        if (PHASE == PHASE_A) {               // d = k2: S = k1 + 2 k2, next point y_n + dt/2 k2
                            ld2(3, k1_, k2_); ld2(4, k3_, k4_);
                            S[0] = fma(D2(2.0), d[0], k0_); S[1] = fma(D2(2.0), d[1], k1_); S[2] = fma(D2(2.0), d[2], k2_);
                            S[3] = fma(D2(2.0), d[3], k3_); S[4] = fma(D2(2.0), d[4], k4_);
                            y[0] = fma(D2(h2), d[0], r0); y[1] = fma(D2(h2), d[1], r1); y[2] = fma(D2(h2), d[2], r2);
                            y[3] = fma(D2(h2), d[3], r3); y[4] = fma(D2(h2), d[4], r4);
                        } else {                              // d = k4: y_{n+1} = Y + dt/6 k4, phi wrapped; next point y_{n+1}
                            y[0] = fma(D2(h6), d[0], r0); y[1] = fma(D2(h6), d[1], r1); y[2] = fma(D2(h6), d[2], r2);
                            y[3] = fma(D2(h6), d[3], r3); y[4] = fma(D2(h6), d[4], r4);
                            y[2] = D2(wrap_phi(tb.tor, y[2].a), wrap_phi(tb.tor, y[2].b));
                        }
                    }
                }
            }
            // ---- new record contents and the next phase's first evaluation point
            D2 ny[5], nk[5];
            if (PHASE == PHASE_A) {       // Y = y_n + dt/6 (k1 + 2 k2 + 2 k3), y4 = y_n + dt k3
                D2 r0, r1, r2, r3, r4, k0_;
                ld2(0, r0, r1); ld2(1, r2, r3); ld2(2, r4, k0_);
                const D2 y0[5] = {r0, r1, r2, r3, r4};
#pragma unroll
                for (int q = 0; q < 5; ++q) { ny[q] = fma(D2(h6), fma(D2(2.0), d[q], S[q]), y0[q]); nk[q] = fma(D2(dt), d[q], y0[q]); }
            } else {                      // y_{n+1} (INIT: y_n) and k1 = f(it)
#pragma unroll
                for (int q = 0; q < 5; ++q) { ny[q] = y[q]; nk[q] = d[q]; }
            }
            // the records go back into their rows, with the triangle of the last evaluation point as the hint for the locator
            // (a retired marker's row is left as it came in: the follow-up kernel redoes its phase through the global tables)
            {
                const bool wA = validA && !retA, wB = validB && !retB;
                if (validA && retA) rq.list[atomicAdd(rq.count, 1)] = mA;
                if (validB && retB) rq.list[atomicAdd(rq.count, 1)] = mB;
                const int tlA = stri[max(slotA, 0)], tlB = stri[max(slotB, 0)];
                auto stp = [&](int j, D2 x, D2 yv) {
                    if (wA) sts128(adA + 16 * (j ^ swA), x.a, yv.a);
                    if (wB) sts128(adB + 16 * (j ^ swB), x.b, yv.b);
                };
                stp(0, ny[0], ny[1]); stp(1, ny[2], ny[3]); stp(2, ny[4], nk[0]); stp(3, nk[1], nk[2]); stp(4, nk[3], nk[4]);
                stp(6, D2(__hiloint2double(stA, tlA), __hiloint2double(stB, tlB)), D2(__hiloint2double(0, idA), __hiloint2double(0, idB)));
                lflag[s * 32 + lane] = (unsigned char)((wA ? 1 : 0) | (wB ? 2 : 0));
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(chunk_bar + 3 * s + 1);   // computed: over to the locator
        }
    }
}

}  // namespace trimeg
