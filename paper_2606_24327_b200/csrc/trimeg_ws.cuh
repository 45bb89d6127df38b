// Warp-specialised phase kernel (included by trimeg_kernels.cuh after the tile helpers).
//
// One persistent CTA per SM, 16 warps in four warp-groups:
//   warp 0    "stager"     : takes super-cells off the work list, waits until a ring entry is free, fills it (slot geometry
//                            + TMA bulk copies of the coefficient blocks);
//   warps 1-2 "publishers" : once an entry has landed, cut its marker range into chunks of 32 and, for each, copy the
//                            32 records into a free chunk slot (cp.async through the sort permutation; completion is
//                            signalled on the slot's mbarrier by cp.async.mbarrier.arrive);
//   warp 3                 : spare (only takes part in the register hand-over);
//   warps 4-15 "compute"   : take chunk slots in ticket order, pull their record into registers, evaluate the phase, put
//                            the record back into its slot row, send the chunk off as one bulk store, free the slot and
//                            count the chunk done on its ring entry.
// The light warp-group hands registers to the compute groups (setmaxnreg: 40 / 152 of a 128-register launch).
// A ring entry is refilled when all chunks cut from it are done AND both publishers have read its control block.
// (Round 2 also tried two markers per lane with shared coefficient loads and separate locator warps: profiles/r02_*.)
#pragma once

namespace trimeg {

// stager, part 1: take the next non-empty super-cell off the work list and pull everything its ring entry needs out of
// global memory into registers (lane sl holds slot sl).  Done BEFORE a ring entry is free, so that only shared-memory
// writes and the TMA issue remain once it is.  Returns false when the work list is exhausted.
struct StageWork { int sc, begin, end, patch, k0, ns, t; SlotGeom g; };
template <class C>
TRIMEG_DI bool ws_fetch(const DevTables& tb, const TileTables& tt, int* work_counter, int lane, StageWork& w) {
    constexpr unsigned FULL = 0xffffffffu;
    int sc = 0, begin = 0, end = 0;
    for (;;) {
        if (lane == 0) sc = atomicAdd(work_counter, 1);
        sc = __shfl_sync(FULL, sc, 0);
        if (sc >= tt.nsc) return false;
        begin = tt.offs[(long long)sc * C::CPS]; end = tt.offs[(long long)(sc + 1) * C::CPS];
        if (begin != end) break;
    }
    w.sc = sc; w.begin = begin; w.end = end;
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
    BlockCtrl* ctl = reinterpret_cast<BlockCtrl*>(smem + C::OFF_CTRL) + b;
    unsigned long long* full = reinterpret_cast<unsigned long long*>(smem + C::OFF_BAR) + 2 * b;
    if (lane == 0) {
        ctl->sc = w.sc; ctl->begin = w.begin; ctl->end = w.end; ctl->patch = w.patch; ctl->k0 = w.k0; ctl->ns = w.ns;
        ctl->nchunks = (w.end - w.begin + 31) >> 5;
        *reinterpret_cast<volatile int*>(&ctl->done) = 0;
    }
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

// Edge walk inside the staged block: returns the slot containing (R, Z) or a negative code: -1 left the staged set (or hop
// cap), -2 crossed the mesh boundary.  The inside test uses the affine form of the barycentrics (SlotGeom); all three
// neighbours come with the same loads, so a hop costs one shared-memory round trip and two dependent FMAs.
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
// reference coordinates for the polynomial evaluation, in the cancellation-free form
TRIMEG_DI void slot_coords(const SlotGeom& g, double R, double Z, double& xi, double& eta) {
    const double dx = R - g.v0x, dy = Z - g.v0y;
    xi = fma(g.a11, dx, g.a12 * dy);
    eta = fma(g.a21, dx, g.a22 * dy);
}

template <class C, int PHASE>
__global__ void __launch_bounds__(C::NTHREADS, 1)
k_phase_ws(DevTables tb, TileTables tt, EquilP ep, SpeciesP sp, const Rec* src, Rec* dst, const int* __restrict__ perm,
           RetireList rq, KeyOut ko, CellMap cm, double dt, int* __restrict__ work_counter) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    BlockCtrl* ctl_all = reinterpret_cast<BlockCtrl*>(smem + C::OFF_CTRL);
    unsigned long long* blk_bar = reinterpret_cast<unsigned long long*>(smem + C::OFF_BAR);      // [b][0] full, [b][1] seen
    ChunkDesc* desc = reinterpret_cast<ChunkDesc*>(smem + C::OFF_DESC);
    unsigned long long* chunk_bar = reinterpret_cast<unsigned long long*>(smem + C::OFF_CBAR);   // [s][0] full, [s][1] empty
    int* cons_head = reinterpret_cast<int*>(smem + C::OFF_HEAD);
    constexpr unsigned FULL = 0xffffffffu;
    if (tid == 0) {
        for (int b = 0; b < C::NBUF; ++b) { mbar_init(blk_bar + 2 * b, 1); mbar_init(blk_bar + 2 * b + 1, C::NPUB); }
        for (int s = 0; s < C::K; ++s) { mbar_init(chunk_bar + 2 * s, 32); mbar_init(chunk_bar + 2 * s + 1, 1); }
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
                    // previous occupant: both publishers have read its control block, and all chunks cut from it are done
                    mbar_wait(blk_bar + 2 * b + 1, (it / C::NBUF - 1) & 1);
                    BlockCtrl* ctl = ctl_all + b;
                    if (lane == 0) {
                        const int need = ctl->nchunks;
                        while (*reinterpret_cast<volatile int*>(&ctl->done) < need) __nanosleep(64);
                    }
                    __syncwarp();
                }
                if (!have) {   // end of work: the entry carries sc = -1 and its barrier completes at once
                    if (lane == 0) {
                        ctl_all[b].sc = -1;
                        __threadfence_block();
                        mbar_arrive(blk_bar + 2 * b);
                    }
                    break;
                }
                ws_commit<C>(smem, b, tb, w, lane);
                have = ws_fetch<C>(tb, tt, work_counter, lane, w);   // the next entry's global loads overlap the compute warps' work
            }
        } else if (wid <= C::NPUB) {
            // ------------------------------------------------------------------ publishers: warp pid takes the tickets t with t % NPUB == pid
            const unsigned pid = wid - 1;
            unsigned ticket = 0;
            auto slot_acquire = [&](unsigned t) {   // wait until the previous user of the slot has been copied out
                const unsigned s = t % C::K, g = t / C::K;
                if (g >= 1) mbar_wait(chunk_bar + 2 * s + 1, (g - 1) & 1);
                return (int)s;
            };
            for (unsigned it = 0;; ++it) {
                const int b = it % C::NBUF;
                mbar_wait(blk_bar + 2 * b, (it / C::NBUF) & 1);
                const BlockCtrl* ctl = ctl_all + b;
                const int sc = ctl->sc, begin = ctl->begin, end = ctl->end;
                __syncwarp();
                if (lane == 0) mbar_arrive(blk_bar + 2 * b + 1);   // control block read: the stager may refill once the chunks are done
                if (sc < 0) break;
                // the chunks of this entry carry tickets ticket .. ticket + nch - 1; ours are those of parity pid
                const unsigned t0 = ticket, nch = (unsigned)(end - begin + 31) >> 5;
                unsigned t = t0 + (pid + C::NPUB - t0 % C::NPUB) % C::NPUB;
                ticket = t0 + nch;
                int pr_next = 0;
                if (t < t0 + nch) { const int q = begin + 32 * (int)(t - t0) + lane; if (q < end) pr_next = perm ? perm[q] : q; }
                for (; t < t0 + nch; t += C::NPUB) {
                    const int c0 = begin + 32 * (int)(t - t0);
                    const int pr = pr_next;
                    const int n0 = c0 + 32 * C::NPUB + lane;
                    if (n0 < end) pr_next = perm ? perm[n0] : n0;      // our next chunk's permutation entries: in flight during this one
                    const int s = slot_acquire(t);
                    if (lane == 0) { desc[s].m0 = c0; desc[s].end = end; desc[s].b = b; __threadfence_block(); }
                    __syncwarp();
                    const int nvalid = min(32, end - c0);
                    const unsigned ib = smem_u32(smem + C::OFF_STAGE + (size_t)s * C::WSTAGE);
                    const int ch = lane & 7, g = lane >> 3;
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        const int r = 4 * k + g;                                   // row of the chunk slot = record c0 + r of dst
                        const int ri = __shfl_sync(FULL, pr, r);
                        if (r < nvalid) {
                            // logical 16-byte chunk j of a record sits at position j ^ rec_swizzle(index): source position ch
                            const int j = ch ^ rec_swizzle(ri);
                            const unsigned d = ib + r * 128 + 16 * (j ^ rec_swizzle(c0 + r));
                            const char* gp = reinterpret_cast<const char*>(src + ri) + 16 * ch;
                            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gp) : "memory");
                        }
                    }
                    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(chunk_bar + 2 * s)) : "memory");
                }
            }
            // one end-of-work ticket per compute warp
            for (int q = 0; q < C::NCOMP; ++q, ++ticket) {
                if (ticket % C::NPUB != pid) continue;
                const int s = slot_acquire(ticket);
                if (lane == 0) { desc[s].m0 = -1; __threadfence_block(); }
                __syncwarp();
                mbar_arrive(chunk_bar + 2 * s);
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
            mbar_wait(chunk_bar + 2 * s, gen & 1);
            const int m0 = desc[s].m0, end = desc[s].end, b = desc[s].b;
            if (m0 < 0) break;
            const int m = m0 + lane;
            const bool valid = m < end;
            const unsigned row = smem_u32(smem + C::OFF_STAGE + (size_t)s * C::WSTAGE) + lane * 128;
            const int sw = rec_swizzle(m);
            Rec r;
            if (valid) {
                double* rd = reinterpret_cast<double*>(&r);
#pragma unroll
                for (int j = 0; j < 7; ++j) lds128(row + 16 * (j ^ sw), rd[2 * j], rd[2 * j + 1]);
            }
            // next ticket now, so that its latency hides behind the arithmetic (volatile asm: as a plain atomicAdd the
            // compiler sinks it to the end of the iteration, next to the other lane-0 work, and its latency is exposed)
            if (lane == 0) asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(t_next) : "r"(smem_u32(cons_head)) : "memory");

            const double* coef = reinterpret_cast<const double*>(smem + C::BLOCK_BYTES * b);
            const SlotGeom* sgeom = reinterpret_cast<const SlotGeom*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES);
            const int* stri = reinterpret_cast<const int*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES + C::GEOM_BYTES);
            BlockCtrl* ctl = ctl_all + b;
            const int patch = ctl->patch, k0 = ctl->k0, ns = ctl->ns;
            if (valid) {
                const double mu = r.mu, pw = r.p;
                int st = r.st, slot = -1;
                if (PHASE == PHASE_A && (st & 2)) st = (st | 1) & ~2;   // the cached k1 = f(y_n) was evaluated outside: that stage belongs to this step
                if (PHASE == PHASE_INIT) st &= ~2;                       // k1 is being recomputed
                {
                    const int sl = r.tri - patch * C::TP;
                    if (sl >= 0 && sl < C::TP) slot = sl;
                    else {   // not sorted since it moved: look for the triangle in the halo
                        for (int q = C::TP; q < ns; ++q) if (stri[q] == r.tri) { slot = q; break; }
                    }
                }
                auto eval = [&](const double y[5], double d[5]) {
                    const int sl = slot_walk1(sgeom, slot, y[0], y[1]);
                    double sf;
                    const int k = toroidal_interval(tb.tor, y[2], sf);
                    int dk = k - k0;
                    if (dk > P / 2) dk -= P; else if (dk < -(P / 2)) dk += P;
                    const int lk = dk + C::HK;
                    if (!(sl >= 0 && sl < C::SMAX && lk >= 0 && lk < C::NW)) return false;   // slots >= SMAX carry geometry only
                    slot = sl;
                    const SlotGeom& gg = sgeom[sl];
                    double xi, eta, w[4], dw[4], g8[8];
                    slot_coords(gg, y[0], y[1], xi, eta);
                    bspline_from_s<double>(tb.tor, sf, w, dw);
                    LdShared ld{smem_u32(coef + (size_t)sl * C::SLOT_DOUBLES + (size_t)lk * PLANE_STRIDE)};
                    gather_cell<false, double>(ld, xi, eta, w, dw, g8);
                    FieldsG<double> f;
                    to_fields_g<double>(gg.a11, gg.a12, gg.a21, gg.a22, g8, y[3], f);
                    rhs_eval<double>(ep, sp, y[0], y[1], y[3], y[4], mu, pw, f, d);
                    return true;
                };
                double next[3];
                if (phase_step<PHASE>(tb.tor, dt, r, eval, next)) {
                    // triangle of the next phase's first evaluation point: staged walk; a point that left the staged geometry is
                    // located through the global tables by k_fix_keys (the record keeps the last triangle as its hint)
                    const int sl = slot_walk1(sgeom, slot, next[0], next[1]);
                    r.st = st;
                    if (sl >= 0) {
                        const int tn = stri[sl];
                        r.tri = tn;
                        if (ko.enabled) {
                            double sf;
                            const int k = toroidal_interval(tb.tor, next[2], sf);
                            const int key = cm.cell(tn, k);
                            ko.keys[m] = key;
                            atomicAdd(ko.hist + key, 1);
                        }
                    } else {
                        r.tri = stri[slot];
                        rq.list[rq.n - 1 - atomicAdd(rq.count + 1, 1)] = m;
                    }
                    // the record goes back into its row of the chunk slot ...
                    const double* rs = reinterpret_cast<const double*>(&r);
#pragma unroll
                    for (int j = 0; j < 7; ++j) if (j != 5) sts128(row + 16 * (j ^ sw), rs[2 * j], rs[2 * j + 1]);
                } else {
                    // the follow-up kernel redoes this phase through the global tables from the untouched record (its row is
                    // left as it came in and goes to dst[m] with the rest of the chunk)
                    rq.list[atomicAdd(rq.count, 1)] = m;
                }
            }
            // ... and the chunk leaves as ONE bulk copy (32 scattered 128-byte lines would cost 224 LSU wavefronts as STG.128)
            fence_async_smem();
            __syncwarp();
            if (lane == 0) {
                tma_bulk_s2g(dst + m0, smem + C::OFF_STAGE + (size_t)s * C::WSTAGE, (unsigned)(min(32, end - m0) * 128));
                bulk_commit();
                __threadfence_block();
                atomicAdd(&ctl->done, 1);            // one more chunk of this ring entry done
                bulk_wait_read0();                   // the copy has read the slot:
                mbar_arrive(chunk_bar + 2 * s + 1);  // it may be refilled
            }
        }
    }
}

}  // namespace trimeg
