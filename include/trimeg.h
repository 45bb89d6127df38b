/*
 * trimeg.h -- C-ABI of the B200-native TRIMEG-C1 marker push (arxiv/paper_2606_24327).
 *
 * The library computes, for every marker of a gyrokinetic particle-in-cell run, the paper's
 * "particle push" (section 3.2): locate the marker in the unstructured poloidal
 * triangle mesh and its toroidal interval, interpolate the perturbed fields dPhi, dA_par and their
 * gradients with the C1 finite element x toroidal cubic B-spline representation (L35), evaluate the
 * equilibrium field, and advance the gyrocentre equations Eq.(2)-(6) (L45-55) and the delta-f weight
 * equation Eq.(7) (L65) -- here fused into a 4-stage Runge-Kutta step on the device.
 *
 * Conventions
 *   - plain C, no exceptions cross this boundary; every call returns 0 or a negative trimeg_status.
 *   - all floating point is IEEE double; indices are int32; sizes int64.
 *   - "memspace" says where a caller buffer lives: TRIMEG_HOST (pageable or pinned host memory) or
 *     TRIMEG_DEVICE (memory of the context's CUDA device).  The caller owns every buffer it passes;
 *     the library copies what it keeps, except the marker scratch (see trimeg_markers_bind).
 *   - all work is enqueued on the CUDA stream given at trimeg_create and is asynchronous with
 *     respect to the host unless the call returns data into HOST memory (then it synchronises).
 *   - coordinates are right-handed cylindrical (R, phi, Z); marker state is stored (R, Z, phi, u, w).
 *   - there is no CPU fallback: without a CUDA device trimeg_create fails with TRIMEG_ERR_CUDA.
 */
#ifndef TRIMEG_H
#define TRIMEG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    TRIMEG_OK = 0,
    TRIMEG_ERR_BAD_ARG = -1,   /* null pointer, non-positive size, dt <= 0 or not finite, n_planes < 4 ... */
    TRIMEG_ERR_BAD_STATE = -2, /* call order: e.g. fields_set before mesh_load, push before markers_bind */
    TRIMEG_ERR_BAD_MESH = -3,  /* vertex index out of range, clockwise or degenerate triangle */
    TRIMEG_ERR_CUDA = -4,      /* a CUDA runtime call failed; see trimeg_last_error */
    TRIMEG_ERR_OOM = -5        /* device allocation failed or the bound scratch is too small */
} trimeg_status;

enum { TRIMEG_HOST = 0, TRIMEG_DEVICE = 1 };
enum { TRIMEG_FIELD_PHI = 0, TRIMEG_FIELD_APAR = 1 };

typedef struct trimeg_ctx trimeg_ctx;

/* Create a context on CUDA device `device`; `cuda_stream` is a cudaStream_t (0/NULL = legacy default
 * stream), typically torch.cuda.current_stream().cuda_stream.  *out is set only on success. */
int trimeg_create(trimeg_ctx** out, int device, void* cuda_stream);
int trimeg_destroy(trimeg_ctx* ctx);
/* Block the host until everything enqueued on the context's stream has finished. */
int trimeg_sync(trimeg_ctx* ctx);
/* Human-readable text of the last error on this context ("" if none); valid until the next call. */
const char* trimeg_last_error(const trimeg_ctx* ctx);

/* Analytic concentric-circular tokamak equilibrium ("computes the equilibrium configuration of
 * the magnetic field"; the paper's numeric B-spline equilibrium L87/L121 is replaced by the closed form the
 * BASELINE configs give):  B = grad(psi) x grad(phi) + B0 R0 grad(phi),  psi'(r) = B0 r / qbar(r),
 * q(r) = q0 + q1 r/a + q2 (r/a)^2,  qbar = q sqrt(1 - r^2/R0^2) if qbar_sqrt else q,  r^2 = (R-R0)^2 + Z^2. */
typedef struct {
    double R0, a, B0, q0, q1, q2;
    int32_t qbar_sqrt;
} trimeg_equil;
int trimeg_equilibrium_set(trimeg_ctx* ctx, const trimeg_equil* eq);

/* Numeric equilibrium ("equilibrium variables are represented using B-splines", L121, L142-146: the paper's
 * B-spline library; reading R27): the poloidal flux psi(R, Z) as a tensor-product uniform cubic B-spline,
 *   psi = sum_{a,b=0..3} psi_coef[i + a][j + b] B_a(s) B_b(t),  i = floor((R - Rmin) / hR), s its fraction (likewise j, t in Z),
 * psi_coef[nR + 3][nZ + 3] in HOST memory (copied), hR = (Rmax - Rmin) / nR; outside the rectangle the edge polynomial is
 * continued.  B = grad psi x grad phi + F grad phi with constant F = R B_phi; R0 and a only serve the Eq.(8) profiles (their
 * radial coordinate stays r = |(R - R0, Z)|) and the triangle numbering.  Replaces a previous equilibrium of either kind.
 * With a numeric equilibrium trimeg_push_rk4 runs variant 1 (one thread per marker); trimeg_push_variant_used says so.
 * Errors: BAD_ARG, CUDA, OOM. */
typedef struct {
    int32_t nR, nZ;
    double Rmin, Rmax, Zmin, Zmax;
    double F, R0, a;
} trimeg_equil_grid;
int trimeg_equilibrium_set_numeric(trimeg_ctx* ctx, const trimeg_equil_grid* grid, const double* psi_coef);

/* Species and equilibrium profiles.  qom = q_s/m_s in the normalised units of Eq.(2)-(6) (sign = charge sign);
 * Eq.(8) (L314): H(r)/H(r0) = exp[-kappa_H w_H (a/R0) tanh((r - r0)/(w_H a))] for H = n, T.
 * bstar_exact = 1: bstar = Bstar / Bstar_par with Bstar = B + (m/q) u curl b (default); 0: the literal expression printed at L53.
 * weight_mode = 0: dw/dt = -p [...] (linear delta-f, default); 1: dw/dt = -(p - w) [...]. */
typedef struct {
    double qom;
    double kappa_n, kappa_T, w_n, w_T, r0;
    int32_t bstar_exact;
    int32_t weight_mode;
} trimeg_species;
int trimeg_species_set(trimeg_ctx* ctx, const trimeg_species* sp);

/* Poloidal mesh + toroidal grid (L35; positioning tables L89, L125-140 are built here, once).
 * RZ: HOST [n_nodes][2] node coordinates; tri: HOST [n_tri][3] vertex indices, counter-clockwise.
 * n_planes >= 4 uniform planes over [0, phi_period) (periodic).  Replaces any previous mesh and drops fields.
 * Errors: BAD_ARG, BAD_MESH (index out of range, non-CCW/degenerate triangle), OOM, CUDA. */
int trimeg_mesh_load(trimeg_ctx* ctx, int64_t n_nodes, const double* RZ, int64_t n_tri, const int32_t* tri,
                     int32_t n_planes, double phi_period);

/* Nodal degrees of freedom of one perturbed field (L35 "field variables on the grid"):
 * dof [n_planes][n_nodes][6] = (f, f_R, f_Z, f_RR, f_RZ, f_ZZ) per node, physical derivatives; per-plane
 * values are toroidal B-spline coefficients.  Converted on the device to per-triangle polynomial
 * coefficients.  A field never set is zero.  Errors: BAD_ARG, BAD_STATE (no mesh), OOM, CUDA. */
int trimeg_fields_set(trimeg_ctx* ctx, int which, const double* dof, int memspace);

/* Grid-to-particle interpolation at arbitrary points (the paper's G2P function, L35, L103):
 * out [8][n] = Phi, dPhi/dR, dPhi/dZ, dPhi/dphi, Apar, dApar/dR, dApar/dZ, dApar/dphi (d/dphi is the raw
 * angle derivative, not divided by R).  tri_out (nullable) [n]: index of the containing triangle in the
 * caller's numbering, -1 = outside the mesh (outputs are then zero).  R, Z, phi, out, tri_out all live in
 * `memspace`.  Errors: BAD_ARG, BAD_STATE (no mesh), CUDA. */
int trimeg_gather(trimeg_ctx* ctx, int64_t n, const double* R, const double* Z, const double* phi, double* out,
                  int32_t* tri_out, int memspace);

/* The per-triangle coefficient table that trimeg_fields_set builds (both fields), as one opaque block: its size in bytes
 * (0 without a mesh), a copy of it into / out of caller-owned DEVICE memory (enqueued on the context's stream).  For the one
 * collective of a multi-GPU run (mesh and fields replicated on every rank): one rank runs
 * trimeg_fields_set, exports, the block is broadcast (NCCL), the other ranks import.  The layout is private to this build
 * of the library and to the mesh it was loaded with (same mesh_load arguments on every rank).
 * Errors: BAD_ARG (null, wrong size), BAD_STATE (no mesh), CUDA. */
size_t trimeg_fields_bytes(const trimeg_ctx* ctx);
int trimeg_fields_export(trimeg_ctx* ctx, void* dst_device, size_t bytes);
int trimeg_fields_import(trimeg_ctx* ctx, const void* src_device, size_t bytes);

/* trimeg_gather for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): same operation, same arguments and results as trimeg_gather with DEVICE buffers, always through the staged
 * path (library-side binning, TMA-staged coefficient blocks), but every per-call buffer lives in ONE
 * static device array inside the library (13.5 MiB, held by every GPU that loads the library until the process exits), so the
 * call issues kernels and one cudaMemsetAsync on the context's stream and nothing else: no cudaMalloc / cudaFree, no events,
 * no synchronisation.  n <= TRIMEG_GATHER_NOALLOC_MAX points per call; more is refused with BAD_ARG and a message naming
 * the limit (split the points, or use trimeg_gather).  R, Z, phi, out [8][n], tri_out (nullable) are DEVICE pointers owned by
 * the caller.  All contexts on a device share the array and it keeps the last call's contents: calls are safe one after the
 * other on one stream (or otherwise ordered on the GPU); two calls that OVERLAP on the GPU (different streams or contexts
 * of the same device without ordering) race and give wrong results.  Errors: BAD_ARG, BAD_STATE (no mesh), CUDA. */
#define TRIMEG_GATHER_NOALLOC_MAX 131072
int trimeg_gather_noalloc(trimeg_ctx* ctx, int64_t n, const double* R, const double* Z, const double* phi, double* out,
                          int32_t* tri_out);

/* N-point gyro-average of the gather (the <...> of Eq.(4)-(6); off in the paper's runs, L320; DESIGN.md
 * reading R26): out[q][i] = mean over j = 0 .. npts-1 of the gathered quantity q at (R_i + rho_i cos(2 pi j / npts),
 * Z_i + rho_i sin(2 pi j / npts), phi_i); ring points outside the mesh contribute zero; rho_i >= 0 is the gyro-radius of
 * point i in the units of R, Z; 1 <= npts <= 64.  out and tri_out (triangle of the gyrocentre itself, nullable) as in
 * trimeg_gather.  Errors: BAD_ARG, BAD_STATE (no mesh), CUDA, OOM. */
int trimeg_gather_gyro(trimeg_ctx* ctx, int64_t n, const double* R, const double* Z, const double* phi, const double* rho,
                       int32_t npts, double* out, int32_t* tri_out, int memspace);

/* How trimeg_gather runs on the device.  Two paths: the direct kernel (one thread per point, coefficients through L1/L2:
 * fastest when the caller's points are already clustered by cell) and the staged path (the library bins the points by cell,
 * stages the coefficient blocks in shared memory by TMA and un-sorts the results; csrc/trimeg_gather.cuh: 4x faster on
 * points in random order).  0 (default): direct below 65536 points, otherwise chosen on the device from a sample of the
 * points (share of neighbours in the same cell); 1 forces the direct kernel, 2 the staged path.  The staged path keeps a
 * library-owned DEVICE workspace of 108 bytes per point (grow-only, freed by mesh_load / destroy).  Results do not depend
 * on the mode beyond rounding.  Errors: BAD_ARG. */
int trimeg_set_gather_mode(trimeg_ctx* ctx, int32_t mode);
/* Device time (CUDA events on the context's stream; blocks until they completed) of the last gather of >= 65536 points that
 * was not forced onto the direct kernel, milliseconds: [0] locate + keys + histogram, [1] scan, [2] scatter into cell order,
 * [3] staged evaluation, [4] un-sort into the caller's arrays, [5] direct kernel (the path not taken returns at once).
 * Errors: BAD_ARG, BAD_STATE (no such gather yet), CUDA. */
int trimeg_gather_kernel_ms(trimeg_ctx* ctx, double out[6]);

/* Bytes of DEVICE scratch trimeg_markers_bind needs for n markers (0 on error): 268 bytes per marker (two buffers of
 * 128-byte records for the re-sorting phases + sort key, permutation and follow-up list, 4 bytes each): 26.8 GB at 1e8
 * markers.  This is twice the structure-of-arrays budget of SURVEY.md 8(a) (a1); DESIGN.md section 5 says why. */
size_t trimeg_scratch_bytes(const trimeg_ctx* ctx, int64_t n);

/* Hand n markers to the library (L89: R, Z, phi, v_par, w per marker; mu and p are constants of the motion).
 * The seven arrays [n] live in `memspace` and are read once (copied into the library's marker store
 * (one 128-byte record per marker), which lives in `scratch`: DEVICE memory owned by the caller that must stay valid until the next
 * bind/destroy; with TRIMEG_HOST inputs the call returns after the copies are enqueued from the caller's
 * buffers, so those must stay valid until trimeg_sync).  Marker status is reset to 0.
 * Errors: BAD_ARG, BAD_STATE (no mesh), OOM (scratch too small), CUDA. */
int trimeg_markers_bind(trimeg_ctx* ctx, int64_t n, const double* R, const double* Z, const double* phi,
                        const double* u, const double* w, const double* mu, const double* p, int memspace,
                        void* scratch, size_t scratch_bytes);

/* Current marker state in the caller's original order.  Any pointer may be null (skipped).
 * status bit 0: some RK stage was evaluated outside the mesh (zero perturbed field was used). */
int trimeg_markers_get(trimeg_ctx* ctx, double* R, double* Z, double* phi, double* u, double* w, int32_t* status,
                       int memspace);

/* Ordering of the marker store by cell (triangle x toroidal interval).  trimeg_push_rk4 (variant 0) runs every RK4 step
 * as two phases, each in the cell order of ITS evaluation points; every phase writes the next
 * phase's cell keys and their histogram, a scan and a scatter turn them into a permutation, and the next phase reads its
 * markers through it (the sort has no data pass of its own).  set_sort_interval(n): rebuild both orders every n-th step
 * (default 1 = every step; 0 = only when needed, i.e. once after bind); between re-sorts the phases run in the stale
 * order and markers that drifted out of their staged block take a slower follow-up path (results do not change).
 * trimeg_sort: force a rebuild at the next step.  Caller order is never affected. */
int trimeg_sort(trimeg_ctx* ctx);
int trimeg_set_sort_interval(trimeg_ctx* ctx, int32_t every_n_steps);

/* Advance all bound markers by nsteps classical RK4 steps of size dt with the fields frozen (north_star;
 * the paper returns the five time derivatives to the host instead, L89).  phi is wrapped into
 * [0, phi_period) after every step.  Errors: BAD_ARG (dt <= 0 or not finite, nsteps < 0), BAD_STATE
 * (mesh, equilibrium, species or markers missing), CUDA. */
int trimeg_push_rk4(trimeg_ctx* ctx, double dt, int32_t nsteps);

/* One evaluation of the right-hand side for the bound markers in the caller's order -- the paper's own kernel
 * boundary (L89: "time derivatives of R, Z, phi, v_par and the marker weights w").  out [5][n] in `memspace`. */
int trimeg_rhs(trimeg_ctx* ctx, double* out, int memspace);

/* Select the push kernel: 0 = two-phase warp-specialised kernel (cell-coherent gather through shared memory, default),
 * 1 = simple (whole RK4 step, one thread per marker, coefficients through L1/L2).  Both compute the same thing. */
int trimeg_set_push_variant(trimeg_ctx* ctx, int32_t variant);

/* Which push kernel trimeg_push_rk4 will actually run with the loaded mesh: *out = 0 (two-phase kernel) or 1 (simple).
 * Variant 0 needs n_planes >= 6 (a staged window of 4 toroidal intervals plus one on either side must not alias under
 * the periodic wrap); with fewer planes variant 1 runs whatever trimeg_set_push_variant selected.
 * Errors: BAD_ARG, BAD_STATE (no mesh). */
int trimeg_push_variant_used(trimeg_ctx* ctx, int32_t* out);

/* Diagnostics used by the benchmark: achieved FP64 FMA throughput of this device in TFLOP/s
 * (a register-only DFMA loop; the roofline's measured "alu" peak). */
int trimeg_bench_dfma(trimeg_ctx* ctx, double* tflops);
/* The same loop with the register operands of real arithmetic: kind 1 = accumulator, multiplier and addend are three
 * different register pairs in every DFMA; kind 2 = Horner-like, one multiplier shared by eight chains with different addends.
 * (trimeg_bench_dfma's loop takes multiplier and addend from two fixed registers.)  Errors: BAD_ARG, OOM, CUDA. */
int trimeg_bench_dfma_mix(trimeg_ctx* ctx, int32_t kind, double* tflops);
/* The three other grid-to-particle kernels of the paper ("pullback treatment", "density calculation",
 * "distribution-function interpolation"; "all these kernels rely on the same G2P function").  The paper gives each one
 * sentence; what they compute here is DESIGN.md readings R22-R24.  All work on the bound marker store.
 *  - trimeg_pullback: the linearised map from the p_par (Hamiltonian, dA^h = A_par) to the v_par (symplectic) picture,
 *    Eq.(1), (6): for every marker  u <- u - (q/m) A_par(R, Z, phi),  w <- w + p (q/m) A_par d ln f0/du (at the old u;
 *    d ln f0/du = -u / T(r) for the Maxwellian of L63 with the Eq.(8) temperature).  A marker outside the mesh is left
 *    unchanged and gets its status bit.  In place; invalidates the cached stage of the push.
 *  - trimeg_density_g2p: out[i] = value of grid field `which` (0 or 1) at marker i (0 outside the mesh), caller order.
 *  - trimeg_f_interp: out[i] = n(r) T(r)^-3/2 exp(-(v^2/2 + mu B)/T(r)) at marker i with v = u - (q/m) A_par (Eq.(6)):
 *    the equilibrium distribution f0 up to its constant factor, at the marker's physical parallel velocity.
 * out: n doubles in `memspace`.  Errors: BAD_ARG, BAD_STATE (mesh, equilibrium, species, markers), CUDA. */
int trimeg_pullback(trimeg_ctx* ctx);
int trimeg_density_g2p(trimeg_ctx* ctx, int which, double* out, int memspace);
int trimeg_f_interp(trimeg_ctx* ctx, double* out, int memspace);

/* Particle-to-grid deposition onto the C1 x B-spline basis ("projecting the quantities stored at the particle
 * locations ... onto the finite element grid"; what the paper left on the CPU, L288, L372): the transpose of the gather.
 * dof_out[n_planes][n_nodes][6] (the layout of trimeg_fields_set's `dof`, in `memspace`) is zeroed and receives
 *   sum over the bound markers of  q_p * B_k(phi_p) * N_{v,c}(R_p, Z_p),
 * N_{v,c} the nodal basis functions of the element containing the marker, B_k the toroidal cubic B-spline, and the marker
 * charge q_p = w (quantity 0: density moment) or w u_par (quantity 1: parallel-current moment).  Markers outside the mesh
 * deposit nothing.  Sums are accumulated with floating-point atomics: the result is reproducible to rounding, not bitwise.
 * Errors: BAD_ARG, BAD_STATE (mesh, markers), CUDA, OOM. */
int trimeg_deposit(trimeg_ctx* ctx, int quantity, double* dof_out, int memspace);

/* The -D options this library was built with beyond the defaults ("" for the shipped configuration). */
const char* trimeg_build_info(void);
/* Counters of the last trimeg_push_rk4 call: [0] kernel launches, [1] right-hand-side evaluations that took the
 * slow (out-of-block) path in the follow-up kernel, [2] marker-phases that left their staged block (summed over
 * phases and steps), [3] permutations built. */
int trimeg_push_stats(trimeg_ctx* ctx, int64_t out[4]);
/* Device time (CUDA events on the context's stream; blocks until they have completed) per RK4 step, averaged over the
 * (up to 32) last steps of the last trimeg_push_rk4 call, in milliseconds: [0] sort kernels of a step (scan, permutation; both phases), [1] the
 * two launches of the phase kernel (the roofline's "dominant kernel"; divide by 2 for one launch), [2] the follow-up
 * kernels (markers that left their staged block, markers outside the mesh).  Errors: BAD_ARG, BAD_STATE (nothing pushed yet), CUDA. */
int trimeg_push_kernel_ms(trimeg_ctx* ctx, double out[3]);

#ifdef __cplusplus
}
#endif
#endif /* TRIMEG_H */
