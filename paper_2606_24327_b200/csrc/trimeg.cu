// C-ABI implementation of include/trimeg.h: context, mesh/field setup, marker store, gather, sort and the RK4 push.
// Compiled for sm_100a only.  See DESIGN.md for the data layout and the roofline of each kernel.
#include "../../include/trimeg.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "trimeg_host_setup.hpp"
#include "trimeg_kernels.cuh"

using namespace trimeg;

// ============================================================================================ context
struct trimeg_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int num_sms = 148;
    std::string err;
    bool have_eq = false, have_sp = false, have_mesh = false, have_markers = false;
    EquilP ep{};
    double* d_psi = nullptr;     // numeric equilibrium: spline coefficients of psi (library-owned)
    SpeciesP sp{};
    trimeg_equil eq_in{};
    trimeg_species sp_in{};
    int NPP = 0;                 // planes of the padded coefficient table
    // mesh
    int T = 0, P = 0;
    long long n_nodes = 0;
    double period = 0;
    TriGeom* d_geom = nullptr;
    int *d_tri = nullptr, *d_head = nullptr, *d_list = nullptr;
    double *d_RZ = nullptr, *d_K = nullptr, *d_coef = nullptr;
    DevTables tb{};
    // markers (all in the caller's scratch)
    long long n = 0;
    Rec* recs[2] = {nullptr, nullptr};         // ping-pong: a phase that re-sorts reads recs[cur] and writes recs[cur ^ 1]
    int cur = 0;
    int *d_keys = nullptr, *d_perm = nullptr, *d_retired = nullptr;
    int *d_hist = nullptr, *d_offs = nullptr, *d_fill = nullptr, *d_sums = nullptr;   // library-owned, [ncell + 2]
    long long ncell = 0;
    // state of the two-phase step
    bool k1_valid = false;      // records hold k = f(y) of the current state and tri / keys of y + key_dt/2 k
    bool keys_valid = false;    // d_keys / d_hist describe the next phase's first evaluation points
    bool order_valid = false;   // d_perm / d_offs hold some complete cell order of the records (possibly stale)
    bool force_sort = false;
    double key_dt = 0.0;
    int sort_every = 1;
    long long steps_since_sort = 0;
    int variant = 0;
    long long stats[4] = {0, 0, 0, 0};
    // per-kernel timing of the last (up to EV_STEPS) steps of the last trimeg_push_rk4 call (events on the context's stream)
    static constexpr int EV_STEPS = 32;
    cudaEvent_t ev[EV_STEPS][8] = {};
    int ev_steps = 0;            // steps of the last call that carry events
    // tiled kernel tables
    int *d_pslots = nullptr, *d_pnslots = nullptr, *d_work = nullptr;
    short* d_pnbr = nullptr;
    unsigned long long* d_stats = nullptr;
    TileTables tt{};
    CellMap cm{};
    bool tiled_ok = false;
    // staged gather (trimeg_gather with many points): its own cell numbering and counting-sort arrays, a grow-only workspace
    GatherMap gm{};
    long long g_ncell = 0;
    int g_nunits = 0;
    int *d_orig = nullptr, *d_ghist = nullptr, *d_goffs = nullptr, *d_gfill = nullptr, *d_gsums = nullptr, *d_gwork = nullptr;
    void* d_gws = nullptr;
    size_t gws_bytes = 0;
    unsigned char* noalloc_ws = nullptr;   // device address of g_noalloc_scratch on this context's device (trimeg_create)
    int gather_mode = 0;        // 0 automatic (staged for n >= GATHER_STAGED_MIN), 1 always direct, 2 always staged
    double gather_ms[5] = {0, 0, 0, 0, 0};   // device time of the last staged gather: keys, scan, scatter, staged, unsort
    cudaEvent_t gev[7] = {};
};
static constexpr long long GATHER_STAGED_MIN = 1 << 16;

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

// ---- trimeg_gather_noalloc: the staged gather with its per-call scratch in a static device array instead of the grow-only
// cudaMalloc'ed workspace, for callers that must not allocate (CUDA graph capture, serving loops).  Layout: a 256-byte header
// (work counter, path flag, two spare words) followed by the five arrays gather_device carves from its workspace, sized for
// TRIMEG_GATHER_NOALLOC_MAX points.  Every GPU that loads the library holds these 13.5 MiB until the process exits; every
// call on a device shares them (calls that overlap on the GPU race).
constexpr size_t noalloc_align256(size_t x) { return (x + 255) & ~(size_t)255; }
constexpr size_t NOALLOC_N = TRIMEG_GATHER_NOALLOC_MAX;
constexpr size_t NOALLOC_HEADER = 256;
constexpr size_t NOALLOC_BYTES = NOALLOC_HEADER + 3 * noalloc_align256(sizeof(int) * NOALLOC_N) + noalloc_align256(sizeof(GPoint) * NOALLOC_N) +
                                 noalloc_align256(sizeof(double) * 8 * NOALLOC_N);
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_BYTES];
// In host code the name g_noalloc_scratch is only a stand-in for the symbol: its device address is looked up once per device
// (with that device current) and kept here.
static std::mutex g_noalloc_mutex;
static void* g_noalloc_addr[64] = {};
static cudaError_t noalloc_scratch_address(int device, void** out) {
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (device < 0 || device >= 64) return cudaErrorInvalidDevice;
    if (!g_noalloc_addr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);     // the device of the calling thread: trimeg_create has set it
        if (e != cudaSuccess) return e;
        g_noalloc_addr[device] = p;
    }
    *out = g_noalloc_addr[device];
    return cudaSuccess;
}

static void free_mesh(trimeg_ctx* c) {
    cudaFree(c->d_geom); cudaFree(c->d_tri); cudaFree(c->d_head); cudaFree(c->d_list);
    cudaFree(c->d_RZ); cudaFree(c->d_K); cudaFree(c->d_coef);
    cudaFree(c->d_hist); cudaFree(c->d_offs); cudaFree(c->d_fill); cudaFree(c->d_sums);
    cudaFree(c->d_pslots); cudaFree(c->d_pnslots); cudaFree(c->d_pnbr); cudaFree(c->d_work); cudaFree(c->d_stats);
    cudaFree(c->d_orig); cudaFree(c->d_ghist); cudaFree(c->d_goffs); cudaFree(c->d_gfill); cudaFree(c->d_gsums); cudaFree(c->d_gwork); cudaFree(c->d_gws);
    c->d_orig = c->d_ghist = c->d_goffs = c->d_gfill = c->d_gsums = c->d_gwork = nullptr; c->d_gws = nullptr; c->gws_bytes = 0;
    c->d_pslots = c->d_pnslots = c->d_work = nullptr; c->d_pnbr = nullptr; c->d_stats = nullptr;
    c->d_geom = nullptr; c->d_tri = c->d_head = c->d_list = nullptr;
    c->d_RZ = c->d_K = c->d_coef = nullptr;
    c->d_hist = c->d_offs = c->d_fill = c->d_sums = nullptr;
    c->have_mesh = false; c->have_markers = false;
}
// anything the cached k1 / keys depend on has changed
static void invalidate_step_state(trimeg_ctx* c) { c->k1_valid = false; c->keys_valid = false; }

// device form of the species: Eq.(8) scalars from the raw species and the current equilibrium (a, R0)
static void derive_species(trimeg_ctx* ctx) {
    const trimeg_equil& eq = ctx->eq_in;
    const trimeg_species* s = &ctx->sp_in;
    SpeciesP& p = ctx->sp;
    p.qom = s->qom; p.kappa = 1.0 / s->qom;
    p.kn_R0 = s->kappa_n / eq.R0; p.kT_R0 = s->kappa_T / eq.R0;
    p.two_inv_wn_a = 2.0 / (s->w_n * eq.a); p.two_inv_wT_a = 2.0 / (s->w_T * eq.a); p.r0 = s->r0;
    p.cT = s->kappa_T * s->w_T * eq.a / eq.R0;
    p.cn = s->kappa_n * s->w_n * eq.a / eq.R0;
    p.same_w = (s->w_n == s->w_T) ? 1 : 0;
    p.bstar_exact = s->bstar_exact ? 1 : 0; p.weight_mode = s->weight_mode ? 1 : 0;
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
    if (noalloc_scratch_address(device, (void**)&c->noalloc_ws) != cudaSuccess) { delete c; return TRIMEG_ERR_CUDA; }
    for (auto& st : c->ev) for (auto& e : st) if (cudaEventCreate(&e) != cudaSuccess) { delete c; return TRIMEG_ERR_CUDA; }
    for (auto& e : c->gev) if (cudaEventCreate(&e) != cudaSuccess) { delete c; return TRIMEG_ERR_CUDA; }
    *out = c;
    return TRIMEG_OK;
}

int trimeg_destroy(trimeg_ctx* ctx) {
    if (!ctx) return TRIMEG_ERR_BAD_ARG;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    for (auto& st : ctx->ev) for (auto& e : st) if (e) cudaEventDestroy(e);
    for (auto& e : ctx->gev) if (e) cudaEventDestroy(e);
    cudaFree(ctx->d_psi);
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
    e.R0 = eq->R0; e.B0 = eq->B0; e.F = eq->B0 * eq->R0; e.F2 = e.F * e.F; e.inv_a = 1.0 / eq->a; e.inv_R0sq = 1.0 / (eq->R0 * eq->R0);
    e.q0 = eq->q0; e.q1 = eq->q1; e.q2 = eq->q2; e.qbar_sqrt = eq->qbar_sqrt ? 1 : 0;
    e.kind = 0; e.psi = nullptr;
    ctx->have_eq = true;
    if (ctx->have_sp) derive_species(ctx);   // the profile scalars of Eq.(8) depend on a and R0
    invalidate_step_state(ctx);
    return TRIMEG_OK;
}

int trimeg_equilibrium_set_numeric(trimeg_ctx* ctx, const trimeg_equil_grid* g, const double* psi_coef) {
    if (!ctx || !g || !psi_coef) return fail(ctx, TRIMEG_ERR_BAD_ARG, "equilibrium_set_numeric: null argument");
    if (g->nR < 1 || g->nZ < 1 || !(g->Rmax > g->Rmin) || !(g->Zmax > g->Zmin) || !(g->Rmin > 0) || !std::isfinite(g->F) || g->F == 0 || !(g->R0 > 0) ||
        !(g->a > 0) || (long long)(g->nR + 3) * (g->nZ + 3) > 100000000LL)
        return fail(ctx, TRIMEG_ERR_BAD_ARG, "equilibrium_set_numeric: need nR, nZ >= 1, 0 < Rmin < Rmax, Zmin < Zmax, finite nonzero F, R0 > 0, a > 0");
    CU(cudaSetDevice(ctx->device));
    CU(cudaStreamSynchronize(ctx->stream));
    cudaFree(ctx->d_psi); ctx->d_psi = nullptr;
    const size_t bytes = sizeof(double) * (size_t)(g->nR + 3) * (g->nZ + 3);
    CU(cudaMalloc(&ctx->d_psi, bytes));
    CU(cudaMemcpy(ctx->d_psi, psi_coef, bytes, cudaMemcpyHostToDevice));
    ctx->eq_in = trimeg_equil{};
    ctx->eq_in.R0 = g->R0; ctx->eq_in.a = g->a; ctx->eq_in.B0 = g->F / g->R0;
    EquilP& e = ctx->ep;
    e = EquilP{};
    e.R0 = g->R0; e.B0 = g->F / g->R0; e.F = g->F; e.F2 = g->F * g->F; e.inv_a = 1.0 / g->a; e.inv_R0sq = 1.0 / (g->R0 * g->R0);
    e.kind = 1; e.psi = ctx->d_psi; e.nR = g->nR; e.nZ = g->nZ; e.Rmin = g->Rmin; e.Zmin = g->Zmin;
    e.inv_hR = g->nR / (g->Rmax - g->Rmin); e.inv_hZ = g->nZ / (g->Zmax - g->Zmin);
    ctx->have_eq = true;
    if (ctx->have_sp) derive_species(ctx);
    invalidate_step_state(ctx);
    return TRIMEG_OK;
}

int trimeg_species_set(trimeg_ctx* ctx, const trimeg_species* s) {
    if (!ctx || !s) return fail(ctx, TRIMEG_ERR_BAD_ARG, "species_set: null argument");
    if (!ctx->have_eq) return fail(ctx, TRIMEG_ERR_BAD_STATE, "species_set: call trimeg_equilibrium_set first (profiles use a and R0)");
    if (!std::isfinite(s->qom) || s->qom == 0 || !(s->w_n > 0) || !(s->w_T > 0) || !std::isfinite(s->kappa_n + s->kappa_T + s->r0))
        return fail(ctx, TRIMEG_ERR_BAD_ARG, "species_set: need finite nonzero qom, w_n > 0, w_T > 0");
    ctx->sp_in = *s;
    derive_species(ctx);
    ctx->have_sp = true;
    invalidate_step_state(ctx);
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
    // padded coefficient table: whole windows of Tile::WK intervals, so that the staged plane range of the last window
    // (which may be partly empty when n_planes is not a multiple of WK) stays inside the triangle's run
    const int nwin = (n_planes + Tile::WK - 1) / Tile::WK;
    ctx->NPP = nwin * Tile::WK + 3 + 2 * PLANE_PAD;
    const long long tri_stride = (long long)ctx->NPP * PLANE_STRIDE;
    const size_t coef_bytes = (size_t)T * tri_stride * sizeof(double);
    trimeg_host::HostPatches hp;
    trimeg_host::build_patches(hm, RZ, n_nodes, T, Tile::TP, Tile::SGEOM, axis_p, 3.0, hp);
    ctx->cm.P = n_planes; ctx->cm.nwin = nwin;
    ctx->ncell = (long long)hp.npatch * nwin * Tile::CPS;
    if ((double)hp.npatch * nwin * Tile::CPS + 2 > 2.0e9) return fail(ctx, TRIMEG_ERR_BAD_ARG, "mesh_load: too many cells for int32 ids");
    ctx->tiled_ok = n_planes >= Tile::NW;   // fewer planes: the window's wrapped intervals would alias (variant 1 is used instead)
    CU(cudaMalloc(&ctx->d_geom, sizeof(TriGeom) * T));
    CU(cudaMalloc(&ctx->d_tri, sizeof(int) * 3 * T));
    CU(cudaMalloc(&ctx->d_head, sizeof(int) * hm.head.size()));
    CU(cudaMalloc(&ctx->d_list, sizeof(int) * hm.list.size()));
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
    {   // staged gather: cells = (patch of GT triangles) x (window of GW intervals) x GT x GW
        const int gnwin = (n_planes + GW - 1) / GW, gnpatch = (T + GT - 1) / GT;
        ctx->gm.nwin = gnwin;
        ctx->g_nunits = gnpatch * gnwin;
        ctx->g_ncell = (long long)ctx->g_nunits * GCELLS;
        if ((double)ctx->g_nunits * GCELLS + 2 > 2.0e9) return fail(ctx, TRIMEG_ERR_BAD_ARG, "mesh_load: too many cells for int32 ids");
        const size_t gcnt = (size_t)ctx->g_ncell + 2;
        CU(cudaMalloc(&ctx->d_orig, sizeof(int) * T));
        CU(cudaMalloc(&ctx->d_ghist, sizeof(int) * gcnt));
        CU(cudaMalloc(&ctx->d_goffs, sizeof(int) * gcnt));
        CU(cudaMalloc(&ctx->d_gfill, sizeof(int) * gcnt));
        CU(cudaMalloc(&ctx->d_gsums, sizeof(int) * (gcnt / SCAN_CHUNK + 2)));
        CU(cudaMalloc(&ctx->d_gwork, sizeof(int) * 4));
        CU(cudaMemcpyAsync(ctx->d_orig, hm.orig_of_new.data(), sizeof(int) * T, cudaMemcpyHostToDevice, ctx->stream));
        CU(cudaMemsetAsync(ctx->d_ghist, 0, sizeof(int) * gcnt, ctx->stream));
        CU(cudaMemsetAsync(ctx->d_gfill, 0, sizeof(int) * gcnt, ctx->stream));
        CU(cudaFuncSetAttribute(k_gather_staged, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GatherSmem::BYTES));
        CU(cudaFuncSetAttribute(k_gather_runs, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)GatherRunsSmem::BYTES));
        // all of the SM's L1/shared array as shared memory for the kernels whose CTAs per SM are set by it
        CU(cudaFuncSetAttribute(k_gather_runs, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        CU(cudaFuncSetAttribute(k_gather_staged, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    }
    CU(cudaMemcpyAsync(ctx->d_pslots, hp.slots.data(), sizeof(int) * hp.slots.size(), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_pnslots, hp.nslots.data(), sizeof(int) * hp.nslots.size(), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_pnbr, hp.nbr.data(), sizeof(short) * hp.nbr.size(), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_stats, 0, sizeof(unsigned long long) * 4, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_offs, 0, sizeof(int) * ncnt, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_hist, 0, sizeof(int) * ncnt, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_fill, 0, sizeof(int) * ncnt, ctx->stream));
    ctx->tt.slots = ctx->d_pslots; ctx->tt.nbr = ctx->d_pnbr; ctx->tt.nslots = ctx->d_pnslots; ctx->tt.offs = ctx->d_offs;
    ctx->tt.npatch = hp.npatch; ctx->tt.nwin = nwin; ctx->tt.nsc = hp.npatch * nwin;
    CU(cudaFuncSetAttribute(k_phase_ws<Tile, PHASE_A>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tile::BYTES));
    CU(cudaFuncSetAttribute(k_phase_ws<Tile, PHASE_B>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tile::BYTES));
    CU(cudaFuncSetAttribute(k_phase_ws<Tile, PHASE_INIT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Tile::BYTES));
    CU(cudaMemcpyAsync(ctx->d_geom, geom.data(), sizeof(TriGeom) * T, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_tri, hm.tri.data(), sizeof(int) * 3 * T, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_head, hm.head.data(), sizeof(int) * hm.head.size(), cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->d_list, hm.list.data(), sizeof(int) * hm.list.size(), cudaMemcpyHostToDevice, ctx->stream));
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
    tb.tor.m2_inv_dphi = -2.0 * (double)n_planes / phi_period;
    ctx->have_mesh = true;
    invalidate_step_state(ctx);
    ctx->order_valid = false;
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
    k_fields_set<<<blocks_for(work, 128), 128, 0, ctx->stream>>>(ctx->T, ctx->P, which, ctx->d_tri, ctx->d_RZ, ctx->d_K, d_dof, ctx->n_nodes, ctx->NPP, ctx->d_coef);
    cudaError_t e = cudaGetLastError();
    if (tmp) { cudaStreamSynchronize(ctx->stream); cudaFree(tmp); }
    if (e != cudaSuccess) return fail(ctx, TRIMEG_ERR_CUDA, "fields_set kernel: %s", cudaGetErrorString(e));
    invalidate_step_state(ctx);   // the cached k1 was evaluated with the old fields
    return TRIMEG_OK;
}

size_t trimeg_fields_bytes(const trimeg_ctx* ctx) {
    if (!ctx || !ctx->have_mesh) return 0;
    return (size_t)ctx->T * (size_t)ctx->NPP * PLANE_STRIDE * sizeof(double);
}

// the coefficient table as one opaque block of DEVICE memory: lets N ranks run fields_set on one of them and hand the result
// to the others with one collective; the layout is private to this library version
int trimeg_fields_export(trimeg_ctx* ctx, void* dst_device, size_t bytes) {
    if (!ctx || !dst_device) return fail(ctx, TRIMEG_ERR_BAD_ARG, "fields_export: null argument");
    if (!ctx->have_mesh) return fail(ctx, TRIMEG_ERR_BAD_STATE, "fields_export: call trimeg_mesh_load first");
    if (bytes != trimeg_fields_bytes(ctx)) return fail(ctx, TRIMEG_ERR_BAD_ARG, "fields_export: need exactly %zu bytes", trimeg_fields_bytes(ctx));
    CU(cudaSetDevice(ctx->device));
    CU(cudaMemcpyAsync(dst_device, ctx->d_coef, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    return TRIMEG_OK;
}

int trimeg_fields_import(trimeg_ctx* ctx, const void* src_device, size_t bytes) {
    if (!ctx || !src_device) return fail(ctx, TRIMEG_ERR_BAD_ARG, "fields_import: null argument");
    if (!ctx->have_mesh) return fail(ctx, TRIMEG_ERR_BAD_STATE, "fields_import: call trimeg_mesh_load first");
    if (bytes != trimeg_fields_bytes(ctx)) return fail(ctx, TRIMEG_ERR_BAD_ARG, "fields_import: need exactly %zu bytes", trimeg_fields_bytes(ctx));
    CU(cudaSetDevice(ctx->device));
    CU(cudaMemcpyAsync(ctx->d_coef, src_device, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    invalidate_step_state(ctx);   // the cached k1 was evaluated with the old fields
    return TRIMEG_OK;
}

// DEVICE pointers; the staged path for many points (trimeg_gather.cuh), the direct kernel otherwise
static int gather_device(trimeg_ctx* ctx, long long n, const double* R, const double* Z, const double* phi, double* out, int32_t* tri_out) {
    if (ctx->gather_mode == 1 || (ctx->gather_mode == 0 && n < GATHER_STAGED_MIN)) {
        k_gather<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(ctx->tb, n, R, Z, phi, out, tri_out, nullptr);
        KCHECK();
        return TRIMEG_OK;
    }
    if (n > 2000000000LL) return fail(ctx, TRIMEG_ERR_BAD_ARG, "gather: n exceeds int32 point ids");
    // workspace (library-owned, grows on demand, kept for the next call): keys, triangles, positions, point and result records
    const size_t need = 3 * align256(sizeof(int) * (size_t)n) + align256(sizeof(GPoint) * (size_t)n) + align256(sizeof(double) * 8 * (size_t)n);
    if (need > ctx->gws_bytes) {
        CU(cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->d_gws); ctx->d_gws = nullptr; ctx->gws_bytes = 0;
        CU(cudaMalloc(&ctx->d_gws, need));
        ctx->gws_bytes = need;
    }
    char* ptr = (char*)ctx->d_gws;
    int* keys = (int*)ptr; ptr += align256(sizeof(int) * (size_t)n);
    int* tris = (int*)ptr; ptr += align256(sizeof(int) * (size_t)n);
    int* inv = (int*)ptr; ptr += align256(sizeof(int) * (size_t)n);
    GPoint* pts = (GPoint*)ptr; ptr += align256(sizeof(GPoint) * (size_t)n);
    double* res = (double*)ptr;
    const long long gcnt = ctx->g_ncell + 2;
    const int nb = (int)((gcnt + SCAN_CHUNK - 1) / SCAN_CHUNK);
    const unsigned sgrid = (unsigned)std::min<long long>(blocks_for(n, 256), (long long)ctx->num_sms * 32);   // grid-stride kernels of the staged path
    // d_gwork: [0] work counter of the staged kernel, [1] path flag (1 direct, 2 staged), [2..3] probe counters
    int* flag = ctx->d_gwork + 1;
    CU(cudaMemsetAsync(ctx->d_gwork, 0, sizeof(int) * 4, ctx->stream));
    if (ctx->gather_mode == 0) {
        const int runs = (int)std::min<long long>(GPROBE_RUNS, std::max<long long>(1, n / 32));
        k_gather_probe<<<runs, 32, 0, ctx->stream>>>(ctx->tb, ctx->gm, n, R, Z, phi, ctx->d_gwork + 2);
        KCHECK();
    }
    k_gather_decide<<<1, 1, 0, ctx->stream>>>(ctx->gather_mode, ctx->d_gwork + 2, flag);
    KCHECK();
    CU(cudaEventRecord(ctx->gev[0], ctx->stream));
    k_gather_keys<<<sgrid, 256, 0, ctx->stream>>>(ctx->tb, ctx->gm, n, R, Z, phi, (int)ctx->g_ncell, keys, tris, inv, ctx->d_ghist, flag);
    KCHECK();
    CU(cudaEventRecord(ctx->gev[1], ctx->stream));
    k_scan_reduce<<<nb, SCAN_THREADS, 0, ctx->stream>>>(ctx->d_ghist, gcnt, ctx->d_gsums, flag);
    k_scan_sums<<<1, SCAN_THREADS, 0, ctx->stream>>>(ctx->d_gsums, nb, flag);
    k_scan_apply<<<nb, SCAN_THREADS, 0, ctx->stream>>>(ctx->d_ghist, gcnt, ctx->d_gsums, ctx->d_goffs, ctx->d_gfill, flag);   // also clears histogram and fill
    KCHECK();
    CU(cudaEventRecord(ctx->gev[2], ctx->stream));
    k_gather_scatter<<<sgrid, 256, 0, ctx->stream>>>(n, R, Z, phi, keys, tris, ctx->d_goffs, pts, inv, flag);
    KCHECK();
    CU(cudaEventRecord(ctx->gev[3], ctx->stream));
    k_gather_staged<<<ctx->num_sms * TRIMEG_GOCC, GTHREADS, GatherSmem::BYTES, ctx->stream>>>(ctx->tb, ctx->gm, ctx->g_nunits, ctx->NPP, ctx->d_goffs, pts, res, ctx->d_gwork, flag);
    KCHECK();
    CU(cudaEventRecord(ctx->gev[4], ctx->stream));
    k_gather_unsort<<<sgrid, 256, 0, ctx->stream>>>(n, tris, res, ctx->d_orig, out, tri_out, flag);
    KCHECK();
    CU(cudaEventRecord(ctx->gev[5], ctx->stream));
    k_gather_runs<<<ctx->num_sms * TRIMEG_RW_OCC, 32 * RW_WARPS, GatherRunsSmem::BYTES, ctx->stream>>>(ctx->tb, ctx->gm, ctx->NPP, n, R, Z, phi, out, tri_out, ctx->d_gwork, flag);
    KCHECK();
    CU(cudaEventRecord(ctx->gev[6], ctx->stream));
    ctx->gather_ms[0] = -1.0;   // events recorded: trimeg_gather_kernel_ms reads them
    return TRIMEG_OK;
}

int trimeg_gather(trimeg_ctx* ctx, int64_t n, const double* R, const double* Z, const double* phi, double* out, int32_t* tri_out, int memspace) {
    if (!ctx || n < 0 || (n > 0 && (!R || !Z || !phi || !out)) || (memspace != TRIMEG_HOST && memspace != TRIMEG_DEVICE))
        return fail(ctx, TRIMEG_ERR_BAD_ARG, "gather: bad argument");
    if (!ctx->have_mesh) return fail(ctx, TRIMEG_ERR_BAD_STATE, "gather: call trimeg_mesh_load first");
    if (n == 0) return TRIMEG_OK;
    CU(cudaSetDevice(ctx->device));
    if (memspace == TRIMEG_DEVICE) return gather_device(ctx, n, R, Z, phi, out, tri_out);
    double* d = nullptr;
    int* dt = nullptr;
    CU(cudaMalloc(&d, sizeof(double) * 11 * (size_t)n));
    if (cudaMalloc(&dt, sizeof(int) * (size_t)n) != cudaSuccess) { cudaFree(d); return fail(ctx, TRIMEG_ERR_OOM, "gather: out of device memory"); }
    cudaError_t e = cudaSuccess;
    auto step = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    step(cudaMemcpyAsync(d, R, sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream));
    step(cudaMemcpyAsync(d + n, Z, sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream));
    step(cudaMemcpyAsync(d + 2 * n, phi, sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream));
    int rc = TRIMEG_OK;
    if (e == cudaSuccess) rc = gather_device(ctx, n, d, d + n, d + 2 * n, d + 3 * n, dt);
    if (rc == TRIMEG_OK) {
        step(cudaMemcpyAsync(out, d + 3 * n, sizeof(double) * 8 * n, cudaMemcpyDeviceToHost, ctx->stream));
        if (tri_out) step(cudaMemcpyAsync(tri_out, dt, sizeof(int) * n, cudaMemcpyDeviceToHost, ctx->stream));
    }
    step(cudaStreamSynchronize(ctx->stream));
    cudaFree(d); cudaFree(dt);
    if (rc != TRIMEG_OK) return rc;
    if (e != cudaSuccess) return fail(ctx, TRIMEG_ERR_CUDA, "gather: %s", cudaGetErrorString(e));
    return TRIMEG_OK;
}

// The staged path of gather_device with every per-call buffer inside the static array: no cudaMalloc, no cudaFree, no event, no
// synchronisation; kernels, one cudaMemsetAsync.  (The histogram / offset tables it also uses belong to the mesh and were
// allocated by trimeg_mesh_load.)
int trimeg_gather_noalloc(trimeg_ctx* ctx, int64_t n, const double* R, const double* Z, const double* phi, double* out, int32_t* tri_out) {
    if (!ctx || n < 0 || (n > 0 && (!R || !Z || !phi || !out))) return fail(ctx, TRIMEG_ERR_BAD_ARG, "gather_noalloc: bad argument");
    if (n > (int64_t)NOALLOC_N)
        return fail(ctx, TRIMEG_ERR_BAD_ARG, "gather_noalloc: n = %lld exceeds TRIMEG_GATHER_NOALLOC_MAX = %lld points (the size of the static scratch array); use trimeg_gather",
                    (long long)n, (long long)NOALLOC_N);
    if (!ctx->have_mesh) return fail(ctx, TRIMEG_ERR_BAD_STATE, "gather_noalloc: call trimeg_mesh_load first");
    if (!ctx->noalloc_ws) return fail(ctx, TRIMEG_ERR_BAD_STATE, "gather_noalloc: static scratch address unknown");
    if (n == 0) return TRIMEG_OK;
    CU(cudaSetDevice(ctx->device));
    unsigned char* ptr = ctx->noalloc_ws;
    int* work = (int*)ptr; ptr += NOALLOC_HEADER;          // [0] work counter of the staged kernel, [1] path flag
    int* keys = (int*)ptr; ptr += noalloc_align256(sizeof(int) * NOALLOC_N);
    int* tris = (int*)ptr; ptr += noalloc_align256(sizeof(int) * NOALLOC_N);
    int* inv = (int*)ptr; ptr += noalloc_align256(sizeof(int) * NOALLOC_N);
    GPoint* pts = (GPoint*)ptr; ptr += noalloc_align256(sizeof(GPoint) * NOALLOC_N);
    double* res = (double*)ptr;
    const long long gcnt = ctx->g_ncell + 2;
    const int nb = (int)((gcnt + SCAN_CHUNK - 1) / SCAN_CHUNK);
    const unsigned sgrid = (unsigned)std::min<long long>(blocks_for(n, 256), (long long)ctx->num_sms * 32);
    int* flag = work + 1;
    // the array keeps the last call's contents: the header must start at zero (work counter); keys, triangles, ranks, point and
    // result records are written for every index below n before they are read
    CU(cudaMemsetAsync(work, 0, NOALLOC_HEADER, ctx->stream));
    k_gather_decide<<<1, 1, 0, ctx->stream>>>(2, work + 2, flag);
    KCHECK();
    k_gather_keys<<<sgrid, 256, 0, ctx->stream>>>(ctx->tb, ctx->gm, n, R, Z, phi, (int)ctx->g_ncell, keys, tris, inv, ctx->d_ghist, flag);
    KCHECK();
    k_scan_reduce<<<nb, SCAN_THREADS, 0, ctx->stream>>>(ctx->d_ghist, gcnt, ctx->d_gsums, flag);
    k_scan_sums<<<1, SCAN_THREADS, 0, ctx->stream>>>(ctx->d_gsums, nb, flag);
    k_scan_apply<<<nb, SCAN_THREADS, 0, ctx->stream>>>(ctx->d_ghist, gcnt, ctx->d_gsums, ctx->d_goffs, ctx->d_gfill, flag);   // also clears histogram and fill
    KCHECK();
    k_gather_scatter<<<sgrid, 256, 0, ctx->stream>>>(n, R, Z, phi, keys, tris, ctx->d_goffs, pts, inv, flag);
    KCHECK();
    k_gather_staged<<<ctx->num_sms * TRIMEG_GOCC, GTHREADS, GatherSmem::BYTES, ctx->stream>>>(ctx->tb, ctx->gm, ctx->g_nunits, ctx->NPP, ctx->d_goffs, pts, res, work, flag);
    KCHECK();
    k_gather_unsort<<<sgrid, 256, 0, ctx->stream>>>(n, tris, res, ctx->d_orig, out, tri_out, flag);
    KCHECK();
    return TRIMEG_OK;
}

int trimeg_gather_gyro(trimeg_ctx* ctx, int64_t n, const double* R, const double* Z, const double* phi, const double* rho, int32_t npts, double* out,
                       int32_t* tri_out, int memspace) {
    if (!ctx || n < 0 || npts < 1 || npts > 64 || (n > 0 && (!R || !Z || !phi || !rho || !out)) || (memspace != TRIMEG_HOST && memspace != TRIMEG_DEVICE))
        return fail(ctx, TRIMEG_ERR_BAD_ARG, "gather_gyro: bad argument (1 <= npts <= 64)");
    if (!ctx->have_mesh) return fail(ctx, TRIMEG_ERR_BAD_STATE, "gather_gyro: call trimeg_mesh_load first");
    if (n == 0) return TRIMEG_OK;
    CU(cudaSetDevice(ctx->device));
    if (memspace == TRIMEG_DEVICE) {
        k_gather_gyro<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(ctx->tb, n, R, Z, phi, rho, npts, out, tri_out);
        KCHECK();
        return TRIMEG_OK;
    }
    double* d = nullptr;
    int* dt = nullptr;
    CU(cudaMalloc(&d, sizeof(double) * 12 * (size_t)n));
    if (cudaMalloc(&dt, sizeof(int) * (size_t)n) != cudaSuccess) { cudaFree(d); return fail(ctx, TRIMEG_ERR_OOM, "gather_gyro: out of device memory"); }
    cudaError_t e = cudaSuccess;
    auto step = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    const double* src[4] = {R, Z, phi, rho};
    for (int q = 0; q < 4; ++q) step(cudaMemcpyAsync(d + q * n, src[q], sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream));
    if (e == cudaSuccess) { k_gather_gyro<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(ctx->tb, n, d, d + n, d + 2 * n, d + 3 * n, npts, d + 4 * n, dt); step(cudaGetLastError()); }
    step(cudaMemcpyAsync(out, d + 4 * n, sizeof(double) * 8 * n, cudaMemcpyDeviceToHost, ctx->stream));
    if (tri_out) step(cudaMemcpyAsync(tri_out, dt, sizeof(int) * n, cudaMemcpyDeviceToHost, ctx->stream));
    step(cudaStreamSynchronize(ctx->stream));
    cudaFree(d); cudaFree(dt);
    if (e != cudaSuccess) return fail(ctx, TRIMEG_ERR_CUDA, "gather_gyro: %s", cudaGetErrorString(e));
    return TRIMEG_OK;
}

int trimeg_set_gather_mode(trimeg_ctx* ctx, int32_t mode) {
    if (!ctx || mode < 0 || mode > 2) return fail(ctx, TRIMEG_ERR_BAD_ARG, "set_gather_mode: 0 automatic, 1 direct, 2 staged");
    ctx->gather_mode = mode;
    return TRIMEG_OK;
}

int trimeg_gather_kernel_ms(trimeg_ctx* ctx, double out[6]) {
    if (!ctx || !out) return fail(ctx, TRIMEG_ERR_BAD_ARG, "gather_kernel_ms: null argument");
    if (ctx->gather_ms[0] != -1.0) return fail(ctx, TRIMEG_ERR_BAD_STATE, "gather_kernel_ms: no staged gather has run");
    CU(cudaSetDevice(ctx->device));
    CU(cudaEventSynchronize(ctx->gev[6]));
    for (int i = 0; i < 6; ++i) {
        float ms = 0;
        CU(cudaEventElapsedTime(&ms, ctx->gev[i], ctx->gev[i + 1]));
        out[i] = ms;
    }
    return TRIMEG_OK;
}

// scratch layout: two buffers of n 128-byte records, then keys, permutation and retire list (n ints each).  The
// inactive record buffer doubles as the staging area of HOST-memspace bind / get.
static size_t int_bytes(long long n) { return align256(sizeof(int) * (size_t)n); }
size_t trimeg_scratch_bytes(const trimeg_ctx* ctx, int64_t n) {
    if (!ctx || n <= 0) return 0;
    return 2 * align256(sizeof(Rec) * (size_t)n) + 3 * int_bytes(n) + 256;
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
    ctx->recs[0] = (Rec*)ptr; ptr += align256(sizeof(Rec) * (size_t)n);
    ctx->recs[1] = (Rec*)ptr; ptr += align256(sizeof(Rec) * (size_t)n);
    ctx->d_keys = (int*)ptr;
    ctx->d_perm = (int*)(ptr + int_bytes(n));
    ctx->d_retired = (int*)(ptr + 2 * int_bytes(n));
    ctx->n = n; ctx->cur = 0;
    ctx->order_valid = false; ctx->force_sort = false; ctx->steps_since_sort = 0;
    invalidate_step_state(ctx);
    CU(cudaMemsetAsync(ctx->d_hist, 0, sizeof(int) * (ctx->ncell + 2), ctx->stream));
    if (memspace == TRIMEG_HOST) {   // stage the seven arrays in the second record buffer
        double* st = (double*)ctx->recs[1];
        const double* src[7] = {R, Z, phi, u, w, mu, p};
        for (int q = 0; q < 7; ++q) CU(cudaMemcpyAsync(st + q * n, src[q], sizeof(double) * n, cudaMemcpyHostToDevice, ctx->stream));
        k_bind<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(ctx->recs[0], 0, n, st, st + n, st + 2 * n, st + 3 * n, st + 4 * n, st + 5 * n, st + 6 * n);
    } else {
        k_bind<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(ctx->recs[0], 0, n, R, Z, phi, u, w, mu, p);
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
    const Rec* recs = ctx->recs[ctx->cur];
    // the retire list is free between phases: it holds the caller id -> record position map
    k_inv_ids<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(recs, n, ctx->d_retired);
    KCHECK();
    if (memspace == TRIMEG_DEVICE) {
        k_get<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(recs, ctx->d_retired, n, R, Z, phi, u, w, status);
        KCHECK();
        return TRIMEG_OK;
    }
    // HOST: un-sort into the inactive record buffer (free between steps), then copy out
    double* st = (double*)ctx->recs[ctx->cur ^ 1];
    int* sti = (int*)(st + 5 * n);
    k_get<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(recs, ctx->d_retired, n, R ? st : nullptr, Z ? st + n : nullptr, phi ? st + 2 * n : nullptr, u ? st + 3 * n : nullptr,
                                                        w ? st + 4 * n : nullptr, status ? sti : nullptr);
    KCHECK();
    double* dst[5] = {R, Z, phi, u, w};
    for (int q = 0; q < 5; ++q) if (dst[q]) CU(cudaMemcpyAsync(dst[q], st + q * n, sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream));
    if (status) CU(cudaMemcpyAsync(status, sti, sizeof(int) * n, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return TRIMEG_OK;
}

int trimeg_sort(trimeg_ctx* ctx) {
    if (!ctx) return TRIMEG_ERR_BAD_ARG;
    if (!ctx->have_markers) return fail(ctx, TRIMEG_ERR_BAD_STATE, "sort: no markers bound");
    ctx->force_sort = true;   // the cell order is rebuilt by the next push step
    return TRIMEG_OK;
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

}  // extern "C"

// counting sort, second half: histogram -> offsets (clearing histogram and fill counters), keys -> permutation
static int build_order(trimeg_ctx* ctx) {
    const long long n = ctx->n, ncnt = ctx->ncell + 2;   // cells + outside bin + end sentinel
    int nb = (int)((ncnt + SCAN_CHUNK - 1) / SCAN_CHUNK);
    k_scan_reduce<<<nb, SCAN_THREADS, 0, ctx->stream>>>(ctx->d_hist, ncnt, ctx->d_sums);
    KCHECK();
    k_scan_sums<<<1, SCAN_THREADS, 0, ctx->stream>>>(ctx->d_sums, nb);
    KCHECK();
    k_scan_apply<<<nb, SCAN_THREADS, 0, ctx->stream>>>(ctx->d_hist, ncnt, ctx->d_sums, ctx->d_offs, ctx->d_fill);
    KCHECK();
    k_sort_perm<<<blocks_for((n + SORT_PER_THREAD - 1) / SORT_PER_THREAD, 256), 256, 0, ctx->stream>>>(n, ctx->d_keys, ctx->d_offs, ctx->d_fill, ctx->d_perm);
    KCHECK();
    ctx->order_valid = true;
    ctx->stats[0] += 4;
    ctx->stats[3] += 1;
    return TRIMEG_OK;
}

template <int PHASE>
static int run_phase(trimeg_ctx* ctx, double dt, bool sort_now, bool keys_out, cudaEvent_t* ev) {
    if (sort_now) {
        int rc = build_order(ctx);
        if (rc) return rc;
    }
    KeyOut ko;
    ko.keys = ctx->d_keys; ko.hist = ctx->d_hist; ko.ncell = (int)ctx->ncell; ko.enabled = keys_out ? 1 : 0;
    RetireList rq{ctx->d_retired, ctx->d_work + 4, (int)ctx->n};
    CU(cudaMemsetAsync(ctx->d_work, 0, 8 * sizeof(int), ctx->stream));
    // a phase that re-sorts moves the records into the other buffer in cell order; otherwise it works in place in the stale order
    const Rec* src = ctx->recs[ctx->cur];
    Rec* dst = ctx->recs[sort_now ? ctx->cur ^ 1 : ctx->cur];
    const int* perm = sort_now ? ctx->d_perm : nullptr;
    if (ev) CU(cudaEventRecord(ev[0], ctx->stream));
    k_phase_ws<Tile, PHASE><<<ctx->num_sms, Tile::NTHREADS, Tile::BYTES, ctx->stream>>>(ctx->tb, ctx->tt, ctx->ep, ctx->sp, src, dst, perm, rq, ko, ctx->cm, dt,
                                                                                           ctx->d_work);
    KCHECK();
    if (ev) CU(cudaEventRecord(ev[1], ctx->stream));
    // follow-ups in one launch: markers that left their staged block and markers outside the mesh (sorted behind the last cell)
    // through the global tables, sort keys of the markers whose next point left the staged geometry, statistics
    {
        const int nbA = ctx->num_sms * 12, nbB = ctx->num_sms * 2, nbC = ctx->num_sms * 12;
        k_followups<PHASE><<<nbA + nbB + nbC, 128, 0, ctx->stream>>>(ctx->tb, ctx->ep, ctx->sp, ctx->cm, ko, src, dst, perm, ctx->d_retired, ctx->d_work,
                                                                     ctx->d_offs + ctx->ncell, ctx->n, dt, ctx->d_stats + 1, nbA, nbB);
        KCHECK();
    }
    if (sort_now) ctx->cur ^= 1;
    if (ev) CU(cudaEventRecord(ev[2], ctx->stream));
    ctx->stats[0] += 2;
    return TRIMEG_OK;
}

extern "C" {

int trimeg_push_rk4(trimeg_ctx* ctx, double dt, int32_t nsteps) {
    if (!ctx || !(dt > 0) || !std::isfinite(dt) || nsteps < 0) return fail(ctx, TRIMEG_ERR_BAD_ARG, "push_rk4: need finite dt > 0 and nsteps >= 0");
    if (!ctx->have_mesh || !ctx->have_eq || !ctx->have_sp || !ctx->have_markers)
        return fail(ctx, TRIMEG_ERR_BAD_STATE, "push_rk4: mesh, equilibrium, species and markers must be set first");
    CU(cudaSetDevice(ctx->device));
    ctx->stats[0] = ctx->stats[1] = ctx->stats[2] = ctx->stats[3] = 0;
    CU(cudaMemsetAsync(ctx->d_stats, 0, sizeof(unsigned long long) * 4, ctx->stream));
    const long long n = ctx->n;
    ctx->ev_steps = 0;
    for (int s = 0; s < nsteps; ++s) {
        const bool timed = (nsteps - s <= trimeg_ctx::EV_STEPS);
        cudaEvent_t* const sev = ctx->ev[timed ? ctx->ev_steps : 0];
        if (ctx->variant == 0 && ctx->tiled_ok && !ctx->ep.kind) {
            const bool need_sort = ctx->force_sort || !ctx->order_valid || (ctx->sort_every > 0 && ctx->steps_since_sort >= ctx->sort_every);
            if (!ctx->k1_valid || ctx->key_dt != dt || (need_sort && !ctx->keys_valid)) {
                // k1 = f(y_n) and the keys of the half-step points, through the global tables (first step after a bind, or after
                // fields / species / dt changed)
                KeyOut ko;
                ko.keys = ctx->d_keys; ko.hist = ctx->d_hist; ko.ncell = (int)ctx->ncell; ko.enabled = need_sort ? 1 : 0;
                CU(cudaMemsetAsync(ctx->d_hist, 0, sizeof(int) * (ctx->ncell + 2), ctx->stream));
                Rec* recs = ctx->recs[ctx->cur];
                if (need_sort) {
                    // bin by the cell of y_n itself, then let the phase kernel compute k1 in that order (it also writes the
                    // keys of the half-step points for phase A)
                    ko.enabled = 1;
                    k_locate_keys<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(ctx->tb, ctx->cm, ko, recs, n);
                    KCHECK();
                    int rc = run_phase<PHASE_INIT>(ctx, dt, true, true, nullptr);
                    if (rc) return rc;
                } else {
                    k_phase_global<PHASE_INIT><<<blocks_for(n, 128), 128, 0, ctx->stream>>>(ctx->tb, ctx->ep, ctx->sp, ctx->cm, ko, recs, recs, nullptr, nullptr,
                                                                                            nullptr, nullptr, n, dt);
                    KCHECK();
                }
                ctx->k1_valid = true; ctx->key_dt = dt; ctx->keys_valid = need_sort;
                ctx->stats[0] += 1;
            }
            const long long next_since = need_sort ? 1 : ctx->steps_since_sort + 1;
            const bool next_sorts = ctx->sort_every > 0 && next_since >= ctx->sort_every;
            if (timed) CU(cudaEventRecord(sev[0], ctx->stream));
            int rc = run_phase<PHASE_A>(ctx, dt, need_sort, need_sort, timed ? sev + 1 : nullptr);
            if (rc) return rc;
            if (timed) CU(cudaEventRecord(sev[4], ctx->stream));
            rc = run_phase<PHASE_B>(ctx, dt, need_sort, next_sorts, timed ? sev + 5 : nullptr);
            if (rc) return rc;
            ctx->keys_valid = next_sorts;
            ctx->steps_since_sort = next_since;
            ctx->force_sort = false;
        } else {
            if (timed) { CU(cudaEventRecord(sev[0], ctx->stream)); CU(cudaEventRecord(sev[1], ctx->stream)); }
            k_push_simple<<<blocks_for(n, 128), 128, 0, ctx->stream>>>(ctx->tb, ctx->ep, ctx->sp, ctx->recs[ctx->cur], n, dt);
            KCHECK();
            if (timed) for (int q = 2; q < 8; ++q) CU(cudaEventRecord(sev[q], ctx->stream));
            invalidate_step_state(ctx);
            ctx->stats[0] += 1;
        }
        if (timed) ++ctx->ev_steps;
    }
    return TRIMEG_OK;
}

#ifndef TRIMEG_BUILD_DEFS
#define TRIMEG_BUILD_DEFS ""
#endif
const char* trimeg_build_info(void) { return TRIMEG_BUILD_DEFS; }

int trimeg_push_variant_used(trimeg_ctx* ctx, int32_t* out) {
    if (!ctx || !out) return fail(ctx, TRIMEG_ERR_BAD_ARG, "push_variant_used: null argument");
    if (!ctx->have_mesh) return fail(ctx, TRIMEG_ERR_BAD_STATE, "push_variant_used: call trimeg_mesh_load first");
    *out = (ctx->variant == 0 && ctx->tiled_ok && !ctx->ep.kind) ? 0 : 1;
    return TRIMEG_OK;
}

int trimeg_push_kernel_ms(trimeg_ctx* ctx, double out[3]) {
    if (!ctx || !out) return fail(ctx, TRIMEG_ERR_BAD_ARG, "push_kernel_ms: null argument");
    if (ctx->ev_steps <= 0) return fail(ctx, TRIMEG_ERR_BAD_STATE, "push_kernel_ms: no step has been pushed");
    CU(cudaSetDevice(ctx->device));
    CU(cudaEventSynchronize(ctx->ev[ctx->ev_steps - 1][7]));
    // events: 0 step start | 1 A tiled start, 2 A tiled end, 3 A follow-ups end | 4 B start | 5 B tiled start, 6 B tiled end, 7 B follow-ups end
    const int span[3][2][2] = {{{0, 1}, {4, 5}}, {{1, 2}, {5, 6}}, {{2, 3}, {6, 7}}};
    for (int i = 0; i < 3; ++i) {
        double tot = 0;
        for (int st = 0; st < ctx->ev_steps; ++st)
            for (int h = 0; h < 2; ++h) {
                float ms = 0;
                CU(cudaEventElapsedTime(&ms, ctx->ev[st][span[i][h][0]], ctx->ev[st][span[i][h][1]]));
                tot += ms;
            }
        out[i] = tot / ctx->ev_steps;   // mean per step over the timed steps of the last call
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
    // staged through the inactive record buffer (free between steps; 64 of its 128 bytes per marker)
    double* stage = (double*)ctx->recs[ctx->cur ^ 1];
    k_rhs<<<blocks_for(n, 128), 128, 0, ctx->stream>>>(ctx->tb, ctx->ep, ctx->sp, ctx->recs[ctx->cur], n, d, stage);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) { k_rhs_unpack<<<blocks_for(n, 256), 256, 0, ctx->stream>>>(stage, n, d); e = cudaGetLastError(); }
    if (memspace == TRIMEG_HOST) {
        if (e == cudaSuccess) e = cudaMemcpyAsync(out, d, sizeof(double) * 5 * n, cudaMemcpyDeviceToHost, ctx->stream);
        cudaError_t e2 = cudaStreamSynchronize(ctx->stream);
        if (e == cudaSuccess) e = e2;
        cudaFree(d);
    }
    if (e != cudaSuccess) return fail(ctx, TRIMEG_ERR_CUDA, "rhs: %s", cudaGetErrorString(e));
    return TRIMEG_OK;
}

// the three other grid-to-particle kernels (readings R22-R24)
int trimeg_pullback(trimeg_ctx* ctx) {
    if (!ctx) return TRIMEG_ERR_BAD_ARG;
    if (!ctx->have_mesh || !ctx->have_eq || !ctx->have_sp || !ctx->have_markers)
        return fail(ctx, TRIMEG_ERR_BAD_STATE, "pullback: mesh, equilibrium, species and markers must be set first");
    CU(cudaSetDevice(ctx->device));
    k_pullback<<<blocks_for(ctx->n, 128), 128, 0, ctx->stream>>>(ctx->tb, ctx->ep, ctx->sp, ctx->recs[ctx->cur], ctx->n);
    KCHECK();
    invalidate_step_state(ctx);   // u and w changed: the cached k1 = f(y_n) no longer belongs to the state
    return TRIMEG_OK;
}

static int per_marker_scalar(trimeg_ctx* ctx, int kind, int which, double* out, int memspace, const char* what) {
    if (!ctx || !out || (memspace != TRIMEG_HOST && memspace != TRIMEG_DEVICE) || which < 0 || which > 1) return fail(ctx, TRIMEG_ERR_BAD_ARG, "%s: bad argument", what);
    if (!ctx->have_mesh || !ctx->have_eq || !ctx->have_sp || !ctx->have_markers)
        return fail(ctx, TRIMEG_ERR_BAD_STATE, "%s: mesh, equilibrium, species and markers must be set first", what);
    CU(cudaSetDevice(ctx->device));
    const long long n = ctx->n;
    double* d = out;
    if (memspace == TRIMEG_HOST) CU(cudaMalloc(&d, sizeof(double) * (size_t)n));
    if (kind == 0) k_density_g2p<<<blocks_for(n, 128), 128, 0, ctx->stream>>>(ctx->tb, which, ctx->recs[ctx->cur], n, d);
    else k_f_interp<<<blocks_for(n, 128), 128, 0, ctx->stream>>>(ctx->tb, ctx->ep, ctx->sp, ctx->recs[ctx->cur], n, d);
    cudaError_t e = cudaGetLastError();
    if (memspace == TRIMEG_HOST) {
        if (e == cudaSuccess) e = cudaMemcpyAsync(out, d, sizeof(double) * n, cudaMemcpyDeviceToHost, ctx->stream);
        cudaError_t e2 = cudaStreamSynchronize(ctx->stream);
        if (e == cudaSuccess) e = e2;
        cudaFree(d);
    }
    if (e != cudaSuccess) return fail(ctx, TRIMEG_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
    return TRIMEG_OK;
}
int trimeg_density_g2p(trimeg_ctx* ctx, int which, double* out, int memspace) { return per_marker_scalar(ctx, 0, which, out, memspace, "density_g2p"); }
int trimeg_f_interp(trimeg_ctx* ctx, double* out, int memspace) { return per_marker_scalar(ctx, 1, 0, out, memspace, "f_interp"); }

// particle-to-grid: the transpose of the gather (reading R25)
int trimeg_deposit(trimeg_ctx* ctx, int quantity, double* dof_out, int memspace) {
    if (!ctx || !dof_out || quantity < 0 || quantity > 1 || (memspace != TRIMEG_HOST && memspace != TRIMEG_DEVICE)) return fail(ctx, TRIMEG_ERR_BAD_ARG, "deposit: bad argument");
    if (!ctx->have_mesh || !ctx->have_markers) return fail(ctx, TRIMEG_ERR_BAD_STATE, "deposit: mesh and markers must be set first");
    CU(cudaSetDevice(ctx->device));
    const size_t bytes = sizeof(double) * 6 * (size_t)ctx->n_nodes * ctx->P;
    double* d = dof_out;
    if (memspace == TRIMEG_HOST) CU(cudaMalloc(&d, bytes));
    cudaError_t e = cudaMemsetAsync(d, 0, bytes, ctx->stream);
    if (e == cudaSuccess) {
        k_deposit<<<(unsigned)std::min<long long>(blocks_for(ctx->n, 32 * DEP_WARPS), (long long)ctx->num_sms * 16), 32 * DEP_WARPS, 0, ctx->stream>>>(ctx->tb, ctx->P, quantity, ctx->recs[ctx->cur], ctx->n, ctx->d_tri, ctx->d_RZ, ctx->d_K, ctx->n_nodes, d);
        e = cudaGetLastError();
    }
    if (memspace == TRIMEG_HOST) {
        if (e == cudaSuccess) e = cudaMemcpyAsync(dof_out, d, bytes, cudaMemcpyDeviceToHost, ctx->stream);
        cudaError_t e2 = cudaStreamSynchronize(ctx->stream);
        if (e == cudaSuccess) e = e2;
        cudaFree(d);
    }
    if (e != cudaSuccess) return fail(ctx, TRIMEG_ERR_CUDA, "deposit: %s", cudaGetErrorString(e));
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

int trimeg_bench_dfma_mix(trimeg_ctx* ctx, int32_t kind, double* tflops) {
    if (!ctx || !tflops || kind < 1 || kind > 2) return fail(ctx, TRIMEG_ERR_BAD_ARG, "bench_dfma_mix: kind 1 (three register operands) or 2 (shared multiplier)");
    CU(cudaSetDevice(ctx->device));
    const int nb = ctx->num_sms * 2, th = 512, iters = 40000;
    double *d = nullptr, *in = nullptr;
    CU(cudaMalloc(&d, sizeof(double) * (size_t)nb * th));
    if (cudaMalloc(&in, sizeof(double) * 24) != cudaSuccess) { cudaFree(d); return fail(ctx, TRIMEG_ERR_OOM, "bench_dfma_mix: out of device memory"); }
    double h[24];
    for (int q = 0; q < 8; ++q) { h[q] = 1.0 + q; h[8 + q] = 1.0000001 + 1e-9 * q; h[16 + q] = 1e-9 * (1 + q); }
    cudaMemcpyAsync(in, h, sizeof h, cudaMemcpyHostToDevice, ctx->stream);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 6; ++rep) {     // the first is the warm-up
        cudaEventRecord(e0, ctx->stream);
        if (kind == 1) k_dfma_mix<1><<<nb, th, 0, ctx->stream>>>(in, d, iters);
        else k_dfma_mix<2><<<nb, th, 0, ctx->stream>>>(in, d, iters);
        cudaEventRecord(e1, ctx->stream);
        cudaEventSynchronize(e1);
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaError_t e = cudaGetLastError();
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d); cudaFree(in);
    if (e != cudaSuccess) return fail(ctx, TRIMEG_ERR_CUDA, "bench_dfma_mix: %s", cudaGetErrorString(e));
    *tflops = 2.0 * 8 * (double)iters * nb * th / (best * 1e-3) * 1e-12;
    return TRIMEG_OK;
}

int trimeg_push_stats(trimeg_ctx* ctx, int64_t out[4]) {
    if (!ctx || !out) return TRIMEG_ERR_BAD_ARG;
    for (int i = 0; i < 4; ++i) out[i] = ctx->stats[i];
    if (ctx->d_stats) {   // markers left to the follow-up kernel are counted on the device, per phase
        unsigned long long h[4] = {0, 0, 0, 0};
        CU(cudaSetDevice(ctx->device));
        CU(cudaMemcpyAsync(h, ctx->d_stats, sizeof h, cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        out[1] = (int64_t)(2 * h[1]);   // each follow-up marker-phase is two right-hand-side evaluations
        out[2] = (int64_t)h[1];
    }
    return TRIMEG_OK;
}

}  // extern "C"

#if defined(TRIMEG_WAITSTATS) || defined(TRIMEG_WATCHDOG)
// tuning / debugging builds only (see trimeg_ws.cuh); not part of include/trimeg.h
extern "C" int trimeg_debug_wait(unsigned long long out[160], int reset) {
    if (cudaDeviceSynchronize() != cudaSuccess) return -4;
    static unsigned long long h[160][160];
    if (cudaMemcpyFromSymbol(h, trimeg::g_wait, sizeof h) != cudaSuccess) return -4;
    for (int i = 0; i < 160; ++i) { out[i] = 0; for (int b = 0; b < 160; ++b) out[i] += h[b][i]; }
    if (reset) { memset(h, 0, sizeof h); cudaMemcpyToSymbol(trimeg::g_wait, h, sizeof h); }
    return 0;
}
extern "C" int trimeg_debug_dbg(unsigned long long out[64]) {
    cudaError_t e = cudaDeviceSynchronize();
    if (cudaMemcpyFromSymbol(out, trimeg::g_dbg, sizeof(unsigned long long) * 64) != cudaSuccess) return -4;
    return e == cudaSuccess ? 0 : -4;
}
#endif
