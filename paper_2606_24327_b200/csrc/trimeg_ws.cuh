// Warp-specialised phase kernel (included by trimeg_kernels.cuh after the tile helpers).
//
// Measured on the plain tiled kernel (profiles/r01c_summary.md): with 16 warps per SM every warp spent more time in the
// per-chunk skeleton (ring waits, permutation load, record copies, block refills: 8.7 ms per pass with the arithmetic
// compiled out) than in the arithmetic itself (6.6 ms), and the two added up instead of overlapping.  Here the skeleton
// is taken off the compute warps:
//   warp 0  "stager"    : takes super-cells off the work list, waits until a ring entry is free, fills it (slot geometry
//                         + TMA bulk copies of the coefficient blocks);
//   warps 1-2 "publishers": once an entry has landed, cuts its marker range into chunks of 32 and, for each, copies the
//                         32 records into a free chunk slot (cp.async through the sort permutation; completion is
//                         signalled on the slot's mbarrier by cp.async.mbarrier.arrive);
//   warps 3.. "compute" : take chunk slots in ticket order, pull their record into registers, evaluate the phase, put
//                         the record back into its slot row, send the chunk off as one bulk store, free the slot and
//                         count the chunk done on its ring entry.
// A ring entry is refilled when all chunks cut from it are done, not when every warp has walked past it.
#pragma once

namespace trimeg {

struct ChunkDesc { int m0, end, b, pad; };   // m0 < 0: no more work

template <class C>
struct WsLayout {
#ifndef TRIMEG_NSLOTS
#define TRIMEG_NSLOTS 20
#endif
    static constexpr int K = TRIMEG_NSLOTS;                              // chunk slots (4 KB each): one per compute warp + look-ahead
    static constexpr int NPUB = 2;                                       // publisher warps (tickets of parity pid)
    static constexpr int NCONS = C::NWARPS - 1 - NPUB;
    static_assert(K % NPUB == 0, "a chunk slot is always served by the same publisher warp (an odd K hung on the GPU)");
    static constexpr size_t OFF_DESC = C::OFF_STAGE + C::WSTAGE * K;
    static constexpr size_t OFF_FULL = OFF_DESC + 16 * K;
    static constexpr size_t OFF_EMPTY = OFF_FULL + 8 * K;
    static constexpr size_t OFF_HEAD = OFF_EMPTY + 8 * K;
    static constexpr size_t BYTES = OFF_HEAD + 64;
};

__device__ __forceinline__ void mbar_arrive(void* bar) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory"); }

// stager, part 1: take the next non-empty super-cell off the work list and pull everything its ring entry needs out of
// global memory into registers (lane sl holds slot sl).  Done BEFORE a ring entry is free, so that only shared-memory
// writes and the TMA issue remain once it is.  Returns false when the work list is exhausted.
struct StageWork { int sc, begin, end, patch, k0, ns, t; SlotGeom g; };
template <class C>
__device__ __forceinline__ bool ws_fetch(const DevTables& tb, const TileTables& tt, int* work_counter, int lane, StageWork& w) {
    static_assert(C::SMAX <= C::SGEOM && C::SGEOM <= 32, "one slot per lane");
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
    g.v0x = g.v0y = 1e300; g.a11 = g.a12 = g.a21 = g.a22 = 0.0; g.nbr[0] = g.nbr[1] = g.nbr[2] = g.nbr[3] = -1;
    if (lane < w.ns) {
        w.t = tt.slots[(long long)w.patch * C::SGEOM + lane];
        if (w.t >= 0) {
            const TriGeom tg = tb.geom[w.t];
            g.v0x = tg.v0x; g.v0y = tg.v0y; g.a11 = tg.a11; g.a12 = tg.a12; g.a21 = tg.a21; g.a22 = tg.a22;
            const short* nb = tt.nbr + ((long long)w.patch * C::SGEOM + lane) * 4;
            g.nbr[0] = nb[0]; g.nbr[1] = nb[1]; g.nbr[2] = nb[2];
        }
    }
    g.tri = w.t; g.pad = 0;
    return true;
}
// stager, part 2: fill the (free) ring entry b from registers and start the TMA bulk copies of its coefficient blocks
template <class C>
__device__ __forceinline__ void ws_commit(unsigned char* smem, int b, const DevTables& tb, const StageWork& w, int lane) {
    constexpr unsigned FULL = 0xffffffffu;
    double* coef = reinterpret_cast<double*>(smem + C::BLOCK_BYTES * b);
    SlotGeom* sgeom = reinterpret_cast<SlotGeom*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES);
    BlockCtrl* ctl = reinterpret_cast<BlockCtrl*>(smem + C::OFF_CTRL) + b;
    unsigned long long* mbar = reinterpret_cast<unsigned long long*>(smem + C::OFF_CTRL + 64 * C::NBUF) + 2 * b;
    if (lane == 0) {
        ctl->sc = w.sc; ctl->begin = w.begin; ctl->end = w.end; ctl->next = w.begin; ctl->ns = w.ns; ctl->patch = w.patch; ctl->k0 = w.k0;
        ctl->pad[0] = (w.end - w.begin + 31) >> 5;                    // chunks that will be cut from this entry
        *reinterpret_cast<volatile int*>(&ctl->left) = 0;             // chunks done
    }
    if (lane < w.ns) sgeom[lane] = w.g;
    const bool has_coef = w.t >= 0 && lane < C::SMAX;
    const int cnt = __popc(__ballot_sync(FULL, has_coef));
    __threadfence_block();
    fence_async_smem();   // earlier generic accesses of this block vs. the async writes
    __syncwarp();
    if (lane == 0) mbar_expect_tx(mbar, (unsigned)(cnt * C::SLOT_DOUBLES * sizeof(double)));
    __syncwarp();
    if (has_coef)
        tma_bulk_g2s(coef + (size_t)lane * C::SLOT_DOUBLES, tb.coef + (long long)w.t * tb.tri_stride + (long long)w.k0 * PLANE_STRIDE,
                     (unsigned)(C::SLOT_DOUBLES * sizeof(double)), mbar);
}

#ifdef TRIMEG_MAXNREG
#define TRIMEG_WS_BOUNDS __maxnreg__(TRIMEG_MAXNREG)
#else
#define TRIMEG_WS_BOUNDS __launch_bounds__(C::NTHREADS, 1)
#endif
template <class C, int PHASE>
__global__ void TRIMEG_WS_BOUNDS
k_phase_ws(DevTables tb, TileTables tt, EquilP ep, SpeciesP sp, const Rec* __restrict__ src, Rec* __restrict__ dst, const int* __restrict__ perm,
           RetireList rq, KeyOut ko, CellMap cm, double dt, int* __restrict__ work_counter) {
    using L = WsLayout<C>;
    extern __shared__ __align__(128) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    BlockCtrl* ctl_all = reinterpret_cast<BlockCtrl*>(smem + C::OFF_CTRL);
    unsigned long long* blk_bar = reinterpret_cast<unsigned long long*>(smem + C::OFF_CTRL + 64 * C::NBUF);   // stride 2
    ChunkDesc* desc = reinterpret_cast<ChunkDesc*>(smem + L::OFF_DESC);
    unsigned long long* full_bar = reinterpret_cast<unsigned long long*>(smem + L::OFF_FULL);
    unsigned long long* empty_bar = reinterpret_cast<unsigned long long*>(smem + L::OFF_EMPTY);
    int* cons_head = reinterpret_cast<int*>(smem + L::OFF_HEAD);
    constexpr unsigned FULL = 0xffffffffu;
    if (tid == 0) {
        for (int b = 0; b < C::NBUF; ++b) mbar_init(blk_bar + 2 * b, 1);
        for (int s = 0; s < L::K; ++s) { mbar_init(full_bar + s, 32); mbar_init(empty_bar + s, 1); }
        *cons_head = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (wid == 0) {
        // ------------------------------------------------------------------ stager
        StageWork w;
        bool have = ws_fetch<C>(tb, tt, work_counter, lane, w);
        for (unsigned it = 0;; ++it) {
            const int b = it % C::NBUF;
            if (it >= (unsigned)C::NBUF) {   // previous occupant: all chunks cut from it are done
                BlockCtrl* ctl = ctl_all + b;
                if (lane == 0) {
                    const int need = ctl->pad[0];
#ifdef TRIMEG_WAITSTATS
                    const long long w0 = clock64();
#endif
                    while (*reinterpret_cast<volatile int*>(&ctl->left) < need) __nanosleep(64);
#ifdef TRIMEG_WAITSTATS
                    atomicAdd(rq.count + 2, (int)((clock64() - w0) >> 10));
#endif
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
    } else if (wid <= L::NPUB) {
        // ------------------------------------------------------------------ publishers: warp pid takes the tickets t with t % NPUB == pid
        const unsigned pid = wid - 1;
        unsigned ticket = 0;
        auto slot_acquire = [&](unsigned t) {   // wait until the previous user of the slot has pulled its records out
            const unsigned s = t % L::K, g = t / L::K;
            if (g >= 1) mbar_wait(empty_bar + s, (g - 1) & 1);
            return (int)s;
        };
        for (unsigned it = 0;; ++it) {
            const int b = it % C::NBUF;
#ifdef TRIMEG_WAITSTATS
            const long long w0 = clock64();
#endif
            mbar_wait(blk_bar + 2 * b, (it / C::NBUF) & 1);
#ifdef TRIMEG_WAITSTATS
            if (lane == 0) atomicAdd(rq.count + 3, (int)((clock64() - w0) >> 10));
#endif
            const BlockCtrl* ctl = ctl_all + b;
            if (ctl->sc < 0) break;
            const int begin = ctl->begin, end = ctl->end;
            // the chunks of this entry carry tickets ticket .. ticket + nch - 1; ours are those of parity pid
            const unsigned t0 = ticket, nch = (unsigned)(end - begin + 31) >> 5;
            unsigned t = t0 + (pid + L::NPUB - t0 % L::NPUB) % L::NPUB;
            ticket = t0 + nch;
            int pr_next = 0;
            if (t < t0 + nch) { const int q = begin + 32 * (int)(t - t0) + lane; if (q < end) pr_next = perm ? perm[q] : q; }
            for (; t < t0 + nch; t += L::NPUB) {
                const int c0 = begin + 32 * (int)(t - t0);
                const int pr = pr_next;
                const int n0 = c0 + 32 * L::NPUB + lane;
                if (n0 < end) pr_next = perm ? perm[n0] : n0;      // our next chunk's permutation entries: in flight during this one
                const int s = slot_acquire(t);
                if (lane == 0) { desc[s].m0 = c0; desc[s].end = end; desc[s].b = b; __threadfence_block(); }
                __syncwarp();
                const int nvalid = min(32, end - c0);
                const unsigned ib = smem_u32(smem + C::OFF_STAGE + (size_t)s * C::WSTAGE);
                const int ch = lane & 7, g = lane >> 3;
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const int R = 4 * k + g;
                    const int ri = __shfl_sync(FULL, pr, R);
                    if (R < nvalid) {
                        const unsigned d = ib + R * 128 + 16 * ((ch ^ (ri & 7)) ^ (R & 7));
                        const char* gp = reinterpret_cast<const char*>(src + ri) + 16 * ch;
                        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gp) : "memory");
                    }
                }
                asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(full_bar + s)) : "memory");
            }
        }
        // one end-of-work ticket per compute warp
        for (int q = 0; q < L::NCONS; ++q, ++ticket) {
            if (ticket % L::NPUB != pid) continue;
            const int s = slot_acquire(ticket);
            if (lane == 0) { desc[s].m0 = -1; __threadfence_block(); }
            __syncwarp();
            mbar_arrive(full_bar + s);
        }
    } else {
        // ------------------------------------------------------------------ compute warps
        const int P = tb.tor.P;
        unsigned t_next = 0;
        if (lane == 0) t_next = (unsigned)atomicAdd(cons_head, 1);
        for (;;) {
            const unsigned t = __shfl_sync(FULL, t_next, 0);
            const unsigned s = t % L::K, g = t / L::K;
#ifdef TRIMEG_WAITSTATS
            const long long w0 = clock64();
#endif
            mbar_wait(full_bar + s, g & 1);
#ifdef TRIMEG_WAITSTATS
            if (lane == 0) atomicAdd(rq.count + 1, (int)((clock64() - w0) >> 10));
#endif
            const int m0 = desc[s].m0, end = desc[s].end, b = desc[s].b;
            if (m0 < 0) break;
            const int m = m0 + lane;
            const bool valid = m < end;
            Rec r;
            if (valid) {
                const unsigned a = smem_u32(smem + C::OFF_STAGE + (size_t)s * C::WSTAGE) + lane * 128;
                double* rd = reinterpret_cast<double*>(&r);
#pragma unroll
                for (int j = 0; j < 7; ++j) lds128(a + 16 * (j ^ (lane & 7)), rd[2 * j], rd[2 * j + 1]);
            }
            // next ticket now, so that its latency hides behind the arithmetic (volatile asm: as a plain atomicAdd the
            // compiler sinks it to the end of the iteration, next to the other lane-0 work, and its latency is exposed)
            if (lane == 0) asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(t_next) : "r"(smem_u32(cons_head)) : "memory");

            const double* coef = reinterpret_cast<const double*>(smem + C::BLOCK_BYTES * b);
            const SlotGeom* sgeom = reinterpret_cast<const SlotGeom*>(smem + C::BLOCK_BYTES * b + C::COEF_BYTES);
            BlockCtrl* ctl = ctl_all + b;
            const int patch = ctl->patch, k0 = ctl->k0, ns = ctl->ns;
            if (valid) {
                const double mu = r.mu, pw = r.p;
                int st = r.st, slot = -1, tri_last = r.tri;
                {
                    int sl = tri_last - patch * C::TP;
                    if (sl >= 0 && sl < C::TP) slot = sl;
                    else {   // not sorted since it moved: look for the triangle in the halo
                        for (int q = C::TP; q < ns; ++q) if (sgeom[q].tri == tri_last) { slot = q; break; }
                    }
                }
                auto eval = [&](const double y[5], double d[5]) {
                    double xi = 0.0, eta = 0.0, sf;
                    const int sl = slot_walk(sgeom, slot, y[0], y[1], xi, eta);
                    const int k = toroidal_interval(tb.tor, y[2], sf);
                    int dk = k - k0;
                    if (dk > P / 2) dk -= P; else if (dk < -(P / 2)) dk += P;
                    const int lk = dk + C::HK;
                    if (!(sl >= 0 && sl < C::SMAX && lk >= 0 && lk < C::NW)) return false;   // slots >= SMAX carry geometry only
                    slot = sl;
                    const SlotGeom& gg = sgeom[sl];
                    tri_last = gg.tri;
                    double w[4], dw[4], g8[8];
                    bspline_from_s(tb.tor, sf, w, dw);
                    LdShared ld{smem_u32(coef + (size_t)sl * C::SLOT_DOUBLES + (size_t)lk * PLANE_STRIDE)};
                    gather_cell(ld, xi, eta, w, dw, g8);
                    Fields fo;
                    fo.P = g8[0]; fo.PR = fma(gg.a11, g8[1], gg.a21 * g8[2]); fo.PZ = fma(gg.a12, g8[1], gg.a22 * g8[2]); fo.Pp = g8[3];
                    fo.A = g8[4]; fo.AR = fma(gg.a11, g8[5], gg.a21 * g8[6]); fo.AZ = fma(gg.a12, g8[5], gg.a22 * g8[6]); fo.Ap = g8[7];
                    rhs_eval(ep, sp, y[0], y[1], y[3], y[4], mu, pw, fo, d);
                    return true;
                };
                double next[3];
                if (phase_step<PHASE>(tb.tor, dt, r, eval, next)) {
                    // triangle of the next phase's first evaluation point: staged walk, else the global walk
                    // (binning by the last staged triangle instead was tried: 8.6 % of the markers then start the next
                    // phase outside their patch's halo and retire)
                    double xi, eta;
                    const int sl = slot_walk(sgeom, slot, next[0], next[1], xi, eta);
                    const int tn = sl >= 0 ? sgeom[sl].tri : locate_walk(tb.bg, tb.geom, tri_last, next[0], next[1]);
                    r.st = st; r.tri = tn;
                    if (ko.enabled) {
                        double sf;
                        const int k = toroidal_interval(tb.tor, next[2], sf);
                        const int key = tn < 0 ? ko.ncell : cm.cell(tn, k);
                        ko.keys[m] = key;
                        atomicAdd(ko.hist + key, 1);
                    }
                } else {
                    // the follow-up kernel redoes this phase through the global tables; r is unchanged and goes to dst[m] as it
                    // is (when the phase works in place, dst[m] is also what the follow-up kernel reads)
                    rq.list[atomicAdd(rq.count, 1)] = m;
                }
                // the record goes back into its row of the chunk slot, now in the swizzle of its position in dst ...
                const unsigned a = smem_u32(smem + C::OFF_STAGE + (size_t)s * C::WSTAGE) + lane * 128;
                const double* rs = reinterpret_cast<const double*>(&r);
#pragma unroll
                for (int j = 0; j < 7; ++j) sts128(a + 16 * (j ^ (m & 7)), rs[2 * j], rs[2 * j + 1]);
            }
            // ... and the chunk leaves as ONE bulk copy (32 scattered 128-byte lines would cost 224 LSU wavefronts as STG.128)
            fence_async_smem();
            __syncwarp();
            if (lane == 0) {
                tma_bulk_s2g(dst + m0, smem + C::OFF_STAGE + (size_t)s * C::WSTAGE, (unsigned)(min(32, end - m0) * 128));
                bulk_commit();
                __threadfence_block();
                atomicAdd(&ctl->left, 1);        // one more chunk of this ring entry done
                bulk_wait_read0();               // the copy has read the slot:
                mbar_arrive(empty_bar + s);      // it may be refilled
            }
        }
    }
}

}  // namespace trimeg
