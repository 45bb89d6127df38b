// Tiled RK4 push: cell-coherent gather through shared memory.
//
// Why: one field evaluation reads 8 x 21 coefficients = 1344 B per marker.  Through L1 with one address per lane
// that costs >= 1344*32/128 = 336 L1 cycles per warp (measured: 16-32 B/clk/SM delivered when lanes diverge), against
// 338 DFMA = 169 issue cycles per SM of FP64 work.  Shared memory delivers 256 B/clk/SM when consecutive lanes read
// the same address (measured), i.e. 168 cycles per warp -- if the lanes of a warp sit in the same few cells.  RK
// stages 2-4 are evaluated at displaced positions (at dt = 0.05 most markers leave their home triangle), so lanes
// are re-grouped by cell before every gather:
//   owner lane (holds the marker's RK state in registers)      gather lane (rank i of the warp in cell order)
//     locate by edge walk in the staged patch, B-spline cell
//     warp bitonic sort of (cell, lane) keys           ---->   reads (xi, eta, s) of the i-th marker in cell order,
//                                                              evaluates 2 fields x 4 planes with near-broadcast LDS.128,
//     reads 8 field values back, equilibrium + RHS     <----   writes physical-gradient results to the owner's row
// Everything between two stagings is warp-synchronous (no block barrier): the 16 warps of the CTA run independently
// and hide each other's latencies.
// The coefficient blocks of a patch of TP triangles plus a halo (SMAX slots), for a window of WK toroidal intervals
// plus HK on either side, are staged per super-cell with 1-D TMA bulk copies (cp.async.bulk + mbarrier).
// A marker whose stage position leaves the staged set RETIRES: it parks (marker index, stage, y_stage, k-sum) in a
// global queue and a follow-up kernel finishes its step through the global tables, so that no warp ever waits on
// a divergent slow lane.
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
    static constexpr size_t BLOCK_BYTES = COEF_BYTES + 64 * SMAX;
    static constexpr size_t OFF_CTRL = BLOCK_BYTES * NBUF;
    static constexpr size_t OFF_WBAR = OFF_CTRL + 64 * NBUF + 16 * NBUF;          // one mbarrier per warp (record loads)
    // per-warp marker staging: the 32 records of the next chunk (cp.async), 128 B each, XOR-swizzled rows
    static constexpr size_t WSTAGE = 32 * 128;
    static constexpr size_t OFF_STAGE = (OFF_WBAR + 8 * NWARPS + 127) / 128 * 128;
    static constexpr size_t BYTES = OFF_STAGE + WSTAGE * NWARPS;
};
struct BlockCtrl {   // 64 B per ring entry
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
// 16 <= bytes, multiple of 16; completion is tracked by the issuing thread's bulk async-group
__device__ __forceinline__ void tma_bulk_s2g(void* dst, const void* src, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void lds128(unsigned addr, double& a, double& b) {
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(a), "=d"(b) : "r"(addr));
}
__device__ __forceinline__ void sts128(unsigned addr, double a, double b) {
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(a), "d"(b) : "memory");
}

struct LdShared {   // coefficient pair fetch from the staged block
    unsigned base;  // shared-space byte address of the cell's first plane
    __device__ __forceinline__ void operator()(int idx, double& a, double& b) const {
        asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(a), "=d"(b) : "r"(base + 16u * (unsigned)idx));
    }
};

}  // namespace trimeg
