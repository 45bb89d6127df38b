// Shared-memory tiling of the phase kernel: layout constants, slot geometry and the PTX helpers
// (mbarrier, TMA bulk copy, shared-memory vector access, register re-allocation).
//
// Why tiles: one field evaluation reads 8 x 21 coefficients = 1344 B per marker.  Through L1 with one address per lane
// that is >= 336 L1 cycles per warp against 338 DFMA = 169 issue cycles of FP64 work.  So the coefficient blocks of a
// patch of TP triangles plus a halo (SMAX slots), for a window of WK toroidal intervals plus HK on either side, are
// staged per super-cell with 1-D TMA bulk copies (cp.async.bulk + mbarrier), and markers are visited in cell order so
// that the lanes of a warp read the same few blocks.  A marker whose evaluation point leaves the staged set RETIRES to a
// list that a follow-up kernel finishes through the global tables, so that no warp waits on a divergent slow lane.
#pragma once
#include "trimeg_math.cuh"

namespace trimeg {

struct TileTables {
    const int* slots;        // [npatch][SGEOM] global triangle per slot, -1 unused
    const short* nbr;        // [npatch][SGEOM][4] slot across edge e, -1 = not staged, -2 = mesh boundary
    const int* nslots;       // [npatch]
    const int* offs;         // [ncell + 1] exclusive offsets of the cell-sorted marker store
    int npatch, nwin, nsc;   // super-cells = npatch * nwin
};

// tuning switches of the phase kernel (the shipped build uses the defaults; python -m paper_2606_24327_b200.build --defs ...)
#ifndef TRIMEG_NCOMP
#define TRIMEG_NCOMP 12
#endif
#ifndef TRIMEG_REG_COMP
#define TRIMEG_REG_COMP 152
#endif
#ifndef TRIMEG_NPUB
#define TRIMEG_NPUB 2
#endif
template <int TP_, int SMAX_, int WK_, int NBUF_, int K_>
struct TileCfg {
    static constexpr int TP = TP_, SMAX = SMAX_, WK = WK_, HK = PLANE_PAD;
    // 16 warps: one light warp-group (stager, NPUB publishers, prefetcher if NPUB = 2) and NCOMP / 4 compute warp-groups
    static constexpr int NLIGHT = 4, NPUB = TRIMEG_NPUB, NCOMP = TRIMEG_NCOMP;
    static constexpr int NWARPS = NLIGHT + NCOMP, NTHREADS = 32 * NWARPS;
    // register hand-over (setmaxnreg): 16 warps launch with 128 registers; the light warps drop to 56, the compute warps
    // take 24 more each (4 x 56 + 12 x 152 = 2048 = 16 x 128)
    static constexpr int REG_LIGHT = 56, REG_COMP = TRIMEG_REG_COMP;
    static_assert(NLIGHT * REG_LIGHT + NCOMP * REG_COMP <= NWARPS * (65536 / (32 * NWARPS) / 8 * 8), "setmaxnreg: the roles' registers must fit the launch allocation (else the kernel hangs)");
    static constexpr int NPL = WK + 2 * HK + 3;      // staged planes per slot
    static constexpr int NW = WK + 2 * HK;           // toroidal intervals covered
    static constexpr int CPS = TP * WK;              // cells per super-cell
    static constexpr int SLOT_DOUBLES = NPL * PLANE_STRIDE;
    static constexpr int NBUF = NBUF_;               // ring of staged blocks
    static constexpr int K = K_;                     // chunk slots: one per compute warp + look-ahead
    static_assert(K % NPUB == 0, "a chunk slot is always served by the same publisher warp (an odd K hung on the GPU)");
    // slot GEOMETRY (64 B per slot) is staged for SGEOM slots, coefficients only for the first SMAX of them: the walk that
    // locates the next phase's first evaluation point needs no coefficients and stays in shared memory further out
    static constexpr int SGEOM = 32;
    static_assert(SMAX <= SGEOM, "one slot per lane of the stager");
    // shared memory carve-up (bytes): NBUF x { coefficients, slot geometry, slot triangles }, control, chunk slots
    static constexpr size_t COEF_BYTES = sizeof(double) * SMAX * SLOT_DOUBLES;
    static constexpr size_t GEOM_BYTES = 64 * SGEOM;
    static constexpr size_t BLOCK_BYTES = COEF_BYTES + GEOM_BYTES + 4 * SGEOM;
    static constexpr size_t CTRL_BYTES = 320;                                // BlockCtrl per ring entry
    static constexpr size_t OFF_CTRL = BLOCK_BYTES * NBUF;
    static constexpr size_t OFF_BAR = OFF_CTRL + CTRL_BYTES * NBUF;          // per ring entry: full, seen (8 B each)
    static constexpr size_t OFF_DESC = OFF_BAR + 16 * NBUF;                  // per chunk slot: ChunkDesc (16 B)
    static constexpr size_t OFF_CBAR = OFF_DESC + 16 * K;                    // per chunk slot: full, empty (8 B each)
    static constexpr size_t OFF_LTAB = OFF_CBAR + 16 * K;                    // per chunk slot: lane -> record row (32 B)
    static constexpr size_t OFF_HEAD = OFF_LTAB + 32 * K;                    // ticket counter (16 B), then the prefetch mailbox
    static constexpr int PFQ = 8;                                            // mailbox entries (begin, end) + sequence number
    static constexpr size_t OFF_PFQ = OFF_HEAD + 16;
    static constexpr int CHUNK = 32;                                         // lanes (<= marker records) per chunk slot
    static constexpr size_t WSTAGE = CHUNK * 128;
    static constexpr size_t OFF_STAGE = (OFF_PFQ + 8 * PFQ + 16 + 127) / 128 * 128;
    static constexpr size_t BYTES = OFF_STAGE + WSTAGE * K;
    static_assert(BLOCK_BYTES % 16 == 0 && OFF_CTRL % 16 == 0, "TMA destinations and control blocks are 16-byte aligned");
    static_assert(BYTES <= 227 * 1024, "shared memory per CTA");
};
// Control block of one ring entry (one super-cell = TP triangles x WK toroidal intervals = 32 cells).
// Lanes of a chunk are laid out over the cells PADDED TO EVEN sizes: an LDS.128 whose lane pairs (2i, 2i+1) read the same
// address takes 2 shared-memory cycles, one with a pair split across two cells takes 4 (measured, profiles/r02b_lds.md), so
// every cell starts on an even lane; an odd cell leaves one lane idle.
struct __align__(16) BlockCtrl {
    int sc, patch, k0, ns;
    int nchunks;     // chunks that will be cut from this entry
    int done;        // chunks finished (compute warps count up)
    int npad;        // lanes of the entry = sum of the padded cell sizes
    int pad0;
    double ox, oy;   // origin of the slot geometry's affine forms (a vertex of the patch)
    int cell_off[33];   // offsets of the 32 cells in the cell-sorted store, and the end
    int pad_incl[32];   // inclusive prefix sums of the padded cell sizes
};
static_assert(sizeof(BlockCtrl) <= 320, "BlockCtrl");
struct ChunkDesc { int m0, nrec, b, ticket; };   // records m0 .. m0 + nrec - 1 of the destination (m0 < 0: no more work); ticket the slot was filled for

// Geometry of one staged slot, 64 B: the barycentrics as affine forms of the position RELATIVE TO THE PATCH ORIGIN,
//   xi = a11 dR + a12 dZ + c1,  eta = a21 dR + a22 dZ + c2,  (dR, dZ) = (R, Z) - (ox, oy),  1 - xi - eta the third.
// With the origin a vertex of the patch, |c| is a few units and the forms carry no cancellation (the same numbers serve
// the inside test of the edge walk and the polynomial evaluation); all three neighbours come with one load.
struct __align__(16) SlotGeom {
    double a11, a12, a21, a22;    // J^-1
    double c1, c2;
    short nbr[4];                 // slot across edge 0 (eta = 0), 1 (1 - xi - eta = 0), 2 (xi = 0): -1 not staged, -2 mesh boundary
    int pad[2];
};
static_assert(sizeof(SlotGeom) == 64, "SlotGeom");

TRIMEG_DI unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
TRIMEG_DI void mbar_init(void* bar, int count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count)); }
TRIMEG_DI void mbar_expect_tx(void* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
TRIMEG_DI void mbar_arrive(void* bar) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory"); }
TRIMEG_DI void mbar_wait(void* bar, unsigned parity) {
    asm volatile(
        "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
TRIMEG_DI void tma_bulk_g2s(void* dst, const void* src, unsigned bytes, void* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src), "r"(bytes),
                 "r"(smem_u32(bar))
                 : "memory");
}
// shared -> global bulk copy (bytes: multiple of 16); completion is tracked by the issuing thread's bulk async-group
TRIMEG_DI void tma_bulk_s2g(void* dst, const void* src, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}
TRIMEG_DI void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
TRIMEG_DI void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
TRIMEG_DI void sts128(unsigned addr, double a, double b) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(a), "d"(b) : "memory");
}
TRIMEG_DI void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
TRIMEG_DI void lds128(unsigned addr, double& a, double& b) {
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(a), "=d"(b) : "r"(addr));
}
// warp-group register re-allocation (sm_90a+): the producer group gives registers up, the compute groups take them
template <int N> TRIMEG_DI void reg_dealloc() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> TRIMEG_DI void reg_alloc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }

struct LdShared {   // coefficient pair fetch from the staged block
    unsigned base;  // shared-space byte address of the cell's first plane
    TRIMEG_DI void operator()(int idx, double& a, double& b) const {
        asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(a), "=d"(b) : "r"(base + 16u * (unsigned)idx));
    }
};

}  // namespace trimeg
