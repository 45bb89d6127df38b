// Shared-memory tiling of the phase kernel: layout constants, slot geometry and the PTX helpers
// (mbarrier, TMA bulk copy, shared-memory vector access).
//
// Why tiles: one field evaluation reads 8 x 21 coefficients = 1344 B per marker.  Through L1 with one address per lane
// that is >= 336 L1 cycles per warp against 338 DFMA = 169 issue cycles of FP64 work (measured: the L1-path kernel is
// 2x slower even when every lane of a warp sits in the same cell).  So the coefficient blocks of a patch of TP triangles
// plus a halo (SMAX slots), for a window of WK toroidal intervals plus HK on either side, are staged per super-cell with
// 1-D TMA bulk copies (cp.async.bulk + mbarrier), and markers are visited in cell order so that the lanes of a warp read
// the same few blocks.  A marker whose evaluation point leaves the staged set RETIRES to a list that a follow-up kernel
// finishes through the global tables, so that no warp waits on a divergent slow lane.
#pragma once
#include "trimeg_math.cuh"

namespace trimeg {

struct TileTables {
    const int* slots;        // [npatch][SMAX] global triangle per slot, -1 unused
    const short* nbr;        // [npatch][SMAX][4] slot across edge e, -1 = not staged / boundary
    const int* nslots;       // [npatch]
    const int* offs;         // [ncell + 1] exclusive offsets of the cell-sorted marker store
    int npatch, nwin, nsc;   // super-cells = npatch * nwin
};

template <int TP_, int SMAX_, int WK_, int NWARPS_, int NBUF_>
struct TileCfg {
    static constexpr int TP = TP_, SMAX = SMAX_, WK = WK_, HK = PLANE_PAD, NWARPS = NWARPS_, NTHREADS = 32 * NWARPS_;
    static constexpr int NPL = WK + 2 * HK + 3;      // staged planes per slot
    static constexpr int NW = WK + 2 * HK;           // toroidal intervals covered
    static constexpr int CPS = TP * WK;              // cells per super-cell
    static constexpr int SLOT_DOUBLES = NPL * PLANE_STRIDE;
    static constexpr int NBUF = NBUF_;               // ring of staged blocks
    // shared memory carve-up (bytes): NBUF x { coefficients, slot geometry }, then the control words
    static constexpr size_t COEF_BYTES = sizeof(double) * SMAX * SLOT_DOUBLES;
    // slot GEOMETRY (64 B per slot) is staged for SGEOM slots, coefficients only for the first SMAX of them: the walk that
    // locates the next phase's first evaluation point needs no coefficients and stays in shared memory further out
#ifndef TRIMEG_SGEOM
#define TRIMEG_SGEOM 32
#endif
    static constexpr int SGEOM = TRIMEG_SGEOM;
    static constexpr size_t BLOCK_BYTES = COEF_BYTES + 64 * SGEOM;
    static constexpr size_t OFF_CTRL = BLOCK_BYTES * NBUF;
    // chunk slots: 32 marker records of 128 B (XOR-swizzled rows), filled by cp.async; NWARPS slots
    static constexpr size_t WSTAGE = 32 * 128;
    static constexpr size_t OFF_STAGE = (OFF_CTRL + 64 * NBUF + 16 * NBUF + 127) / 128 * 128;
    static constexpr size_t BYTES = OFF_STAGE + WSTAGE * NWARPS;
};
struct BlockCtrl {   // 64 B per ring entry; left = chunks done, pad[0] = chunks cut from the entry
    int sc, begin, end, next, left, ns, patch, k0;
    int pad[8];
};

struct __align__(16) SlotGeom {   // 64 B
    double v0x, v0y, a11, a12, a21, a22;
    short nbr[4];
    int tri, pad;
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void* bar, int count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count)); }
__device__ __forceinline__ void mbar_expect_tx(void* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(void* bar, unsigned parity) {
    asm volatile(
        "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_bulk_g2s(void* dst, const void* src, unsigned bytes, void* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src), "r"(bytes),
                 "r"(smem_u32(bar))
                 : "memory");
}
// shared -> global bulk copy (bytes: multiple of 16); completion is tracked by the issuing thread's bulk async-group
__device__ __forceinline__ void tma_bulk_s2g(void* dst, const void* src, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void sts128(unsigned addr, double a, double b) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(a), "d"(b) : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void lds128(unsigned addr, double& a, double& b) {
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(a), "=d"(b) : "r"(addr));
}

struct LdShared {   // coefficient pair fetch from the staged block
    unsigned base;  // shared-space byte address of the cell's first plane
    __device__ __forceinline__ void operator()(int idx, double& a, double& b) const {
        asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(a), "=d"(b) : "r"(base + 16u * (unsigned)idx));
    }
};

}  // namespace trimeg
