/*
 * semb200.h — C ABI of libsemb200.so: the B200-native (sm_100a, fp64) spectral-element
 * Poisson/Helmholtz hot path of arxiv/paper_2501_13240 (NekRS runs of Rayleigh-Benard convection).
 *
 * The call list follows BASELINE.json:north_star — mesh/setup(E, N, coords, boundary tags),
 * apply_axhelm, gather_scatter, pcg_solve, export_field — and the paper's hand-off protocol
 * (§3.1, Listing 2: register device pointers once, set state/cycle and
 * state/time and publish per analysis step, close at exit; PAPER.md:L128 zero-copy; L171-177 the
 * consumer must know which memory space a pointer lives in).
 *
 * Conventions
 *   - Every function returns int: 0 = SEMB_OK, < 0 an error, > 0 a status with valid outputs.
 *   - "device" pointers are CUDA device memory of the current device, OWNED BY THE CALLER, never
 *     freed or retained beyond the call unless the call says so (semb_publish_field retains the
 *     pointer, not the memory).  "host" pointers are ordinary host memory.
 *   - Mesh-derived arrays are owned by the handle until semb_destroy.
 *   - All work is enqueued on the caller's stream (a cudaStream_t passed as void*; NULL = default
 *     stream).  Only semb_setup, the solvers (semb_pcg_solve, semb_step_solve, semb_boussinesq_step: to poll the stop flag),
 *     semb_estimate_lmax, the first use of a multigrid hierarchy / Schwarz smoother / geometry class / flow metrics (one-off
 *     setup work) and the *_host calls synchronise.
 *   - Layout ("(ijk) ordering on [-1,1]^3"): local node l = e*Np + k*n1*n1 + j*n1 + i,
 *     n1 = N+1, Np = n1^3, i fastest; n = E*Np local nodes; all fields fp64, indices int32.
 *   - There is no CPU fallback: with no CUDA device every compute call returns SEMB_ECUDA.
 */
#ifndef SEMB200_H
#define SEMB200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define SEMB_API __attribute__((visibility("default")))
#else
#define SEMB_API
#endif

#define SEMB_OK          0
#define SEMB_MAXIT       1   /* pcg_solve: maxit reached, outputs valid                     */
#define SEMB_EINVAL     -1   /* bad argument                                                */
#define SEMB_ENOMEM     -2   /* allocation failed                                           */
#define SEMB_ECUDA      -3   /* CUDA runtime error (see semb_last_error)                    */
#define SEMB_EGEOM      -4   /* non-positive Jacobian (semb_last_error names the element)   */
#define SEMB_EBREAKDOWN -5   /* PCG breakdown: p.Ap <= 0 or not finite                      */
#define SEMB_EMATCH     -6   /* coordinate matching is not an equivalence at this tolerance */
#define SEMB_ENOTFOUND  -7   /* export_field: no such field                                 */

#define SEMB_MAX_N      10   /* PAPER.md:L204 §4.1: polynomial order p <= 10                */

typedef struct semb_mesh* semb_handle;

/* Optional allocator for every device buffer the library owns (so that e.g. torch's caching
 * allocator owns all memory).  NULL => cudaMalloc/cudaFree. */
typedef struct {
    void* (*alloc)(size_t bytes, void* user);
    void  (*free)(void* ptr, void* user);
    void*  user;
} semb_allocator;

/* ---- basis (host) ------------------------------------------------------------------------
 * GLL nodes xi[N+1], weights rho[N+1] and the derivative matrix D[(N+1)*(N+1)], D[i*n1+j] =
 * l'_j(xi_i) (PAPER.md:L85 GLL quadrature; L100 "(p+1)x(p+1) operator matrices identical for
 * all elements").  The diagonal is minus the off-diagonal row sum (reading R2).
 * Host pointers; any may be NULL.  1 <= N <= SEMB_MAX_N else SEMB_EINVAL. */
SEMB_API int semb_gll(int N, double* xi, double* rho, double* D);

/* ---- setup (PAPER.md:L85, L100 chain rule for deformed elements, L102 inter-element exchange) --
 * x, y, z     device [n]   node coordinates, layout above.
 * face_tag    HOST   [E*6] faces r-,r+,s-,s+,t-,t+ ; 0 = none/interior/periodic, 1..31 = user id.
 * period      HOST   [3]   0 = not periodic, else the period length in that direction.
 * gid_or_null device [n]   optional caller-supplied global ids (int32, any labels >= 0 that are
 *                          equal exactly on coincident nodes); skips coordinate matching.  The
 *                          library still renumbers to canonical first-touch ids.
 * Computes (device, handle-owned): geometric factors G_rr,G_rs,G_rt,G_ss,G_st,G_tt,B per node,
 * canonical global ids, gather lists, inverse multiplicity.  Synchronises the stream.
 * Errors: SEMB_EINVAL, SEMB_ENOMEM, SEMB_ECUDA, SEMB_EGEOM, SEMB_EMATCH (*out = NULL on error). */
SEMB_API int semb_setup(int64_t E, int N, const double* x, const double* y, const double* z,
               const int32_t* face_tag, const double* period, const int32_t* gid_or_null,
               const semb_allocator* alloc_or_null, void* stream, semb_handle* out);

/* Frees everything the handle owns ("close").  NULL is a no-op. */
SEMB_API int semb_destroy(semb_handle h);

/* Message of the last error on this handle (or of the last failed semb_setup if h == NULL).
 * The string is owned by the library. */
SEMB_API const char* semb_last_error(semb_handle h);

typedef struct {
    int64_t E; int32_t N; int32_t n1; int64_t Np; int64_t n;
    int64_t n_unique;      /* number of global nodes                                        */
    int64_t n_shared;      /* local nodes whose global node has >= 2 copies                 */
    int64_t n_gs;          /* global nodes with >= 2 copies                                  */
    double  tol;           /* matching tolerance used (1e-8 * smallest node spacing)        */
    const int32_t* gid;       /* device [n]  canonical global ids                            */
    const double*  geo;       /* device [E][7][Np]: G_rr,G_rs,G_rt,G_ss,G_st,G_tt,B          */
    const double*  invmult;   /* device [n]  1 / multiplicity                                */
    const int32_t* gs_offsets;/* device [n_gs+1] CSR offsets into gs_ids                     */
    const int32_t* gs_ids;    /* device [n_shared] local ids, classes by gid, members ascending */
} semb_info;
SEMB_API int semb_mesh_info(semb_handle h, semb_info* out);

/* ---- the local operator (north_star: per element w = D^T G D u + lambda B u) ----
 * u, w   device [nfields][n], w != u.  lambda == 0 and no coefficient fields selects the
 *        6-factor Poisson kernel (64 B/node), otherwise the 7-factor Helmholtz kernel (72 B/node).
 * lambda0_or_null, lambda1_or_null  device [n]: per-node coefficients, w = D^T(lambda0 G)D u +
 *        lambda1 B u (reading R3); with lambda1 == NULL the scalar lambda multiplies B.
 * Element-local: no assembly, no mask.  Asynchronous on stream. */
SEMB_API int semb_apply_axhelm(semb_handle h, double lambda, const double* lambda0_or_null,
                      const double* lambda1_or_null, const double* u, double* w, int nfields,
                      void* stream);

/* ---- geometry representation read by semb_apply_axhelm and by every fp64 operator application of the solvers
 * (SURVEY.md §8 f-3 "on-the-fly geometric factors ... mixed-precision geo storage"; PAPER.md:L100 fixes only the chain
 * rule; the paper's box meshes are vertically stretched Cartesian element maps, i.e. affine bricks).
 * The operator is unchanged (reading R23); what changes is what is streamed from memory per application:
 *   SEMB_GEO_STORED     (default) G(6)+B per node in fp64                                  48 (56) B/node
 *   SEMB_GEO_F32        the same factors rounded to float once, widened on load, fp64 arithmetic:
 *                       w = D^T fl32(G) D u + lambda fl32(B) u exactly                     24 (28) B/node
 *   SEMB_GEO_AFFINE     every element a parallelepiped: 7 constants per element            64 B/element
 *   SEMB_GEO_TRILINEAR  every element the trilinear image of its 8 corner nodes: 24 coefficients per element, Jacobian,
 *                       cofactors and J recomputed per node                                 192 B/element
 * tol: largest admissible distance of any node from the affine / trilinear map of its element's corners, relative to the
 * largest |coordinate| of the mesh; <= 0 => 16 eps (coordinates that ARE that map up to their own rounding).
 * dev_out_or_null HOST [2]: the measured deviations (trilinear, affine).  Returns SEMB_EGEOM and leaves the mode
 * unchanged when the mesh is not in the class.  Coefficient fields (lambda0 / lambda1) need SEMB_GEO_STORED.
 * Synchronises the stream the first time a class is measured. */
#define SEMB_GEO_STORED     0
#define SEMB_GEO_F32        1
#define SEMB_GEO_AFFINE     2
#define SEMB_GEO_TRILINEAR  3
SEMB_API int semb_set_geometry_mode(semb_handle h, int mode, double tol, double* dev_out_or_null, void* stream);

/* ---- direct-stiffness summation QQ^T -------------------------------------
 * w device [nfields][n], in place: every copy of a global node receives the sum of all copies,
 * summed in ascending local index (deterministic, no atomics). */
SEMB_API int semb_gather_scatter(semb_handle h, double* w, int nfields, void* stream);

/* w[l] = 0 at every local node whose global node lies on a face whose tag t has bit t set in
 * dirichlet_tags (PAPER.md:L238 isothermal / no-slip plates). */
SEMB_API int semb_apply_mask(semb_handle h, uint32_t dirichlet_tags, double* w, int nfields, void* stream);

/* b = M QQ^T (B o f): right-hand side from nodal values f (device [n]); b device [n], b != f. */
SEMB_API int semb_assemble_rhs(semb_handle h, uint32_t dirichlet_tags, const double* f, double* b, void* stream);

/* out = M QQ^T A_L (M v): the assembled masked operator (v, out device [n], out != v). */
SEMB_API int semb_apply_operator(semb_handle h, double lambda, uint32_t dirichlet_tags, const double* v,
                        double* out, void* stream);

/* dinv_out device [n] = 1 / (QQ^T diag(D^T G D + lambda B)), 1 at masked nodes (Jacobi). */
SEMB_API int semb_jacobi_diag(semb_handle h, double lambda, uint32_t dirichlet_tags, double* dinv_out, void* stream);

/* ---- PCG (the pressure Poisson solve; north_star: Jacobi / Chebyshev-Jacobi PCG) ----- */
typedef struct {
    double   lambda;          /* operator D^T G D + lambda B                                     */
    uint32_t dirichlet_tags;  /* bit t set => faces tagged t are Dirichlet (homogeneous)         */
    int32_t  precond;         /* 3 = p-multigrid V-cycle (mg_* fields); 0 none, 1 Jacobi, 2 Chebyshev-Jacobi                            */
    int32_t  cheb_degree;     /* k operator applications per preconditioner application          */
    double   cheb_lmax;       /* upper bound of spec(D^-1 A); <= 0 => 10-step Lanczos x 1.1      */
    double   rtol, atol;      /* stop when ||r|| <= max(rtol ||b||, atol) (unique-node 2-norm)   */
    int32_t  maxit;
    int32_t  x0_is_zero;      /* 1: ignore the contents of x and start from 0                    */
    int32_t  check_every;     /* iterations enqueued between host polls of the stop flag; <= 0 => 16.
                                 The iteration count returned is exact regardless.               */
    int32_t  profile;         /* 1: bracket every axhelm launch of the loop with CUDA events on the stream
                                 (no synchronisation added) and report their mean in stats.axhelm_ms     */
    /* precond == 3: p-multigrid V-cycle (§2.2 "p-multigrid ... Chebyshev-accelerated ... smoothers";
     * DESIGN.md reading R19).  Level l re-discretises the same elements at order mg_orders[l] (mg_orders[0] = N,
     * strictly decreasing, >= 1), coordinates interpolated from level 0; transfer = Lagrange interpolation of the
     * coarse basis at the fine GLL nodes and its transpose on unique nodes; smoother = Chebyshev-Jacobi of degree
     * mg_smooth_degree before and after the coarse correction, of degree mg_coarse_degree alone on the last level;
     * mg_lmax[l] <= 0 => estimated (10-step Lanczos x 1.1 from the level's M QQ^T u, u ~ U[-1,1) seeded per level)
     * and cached in the handle. */
    int32_t  mg_nlevels;      /* 2..8; 0 with precond == 3 => orders N, 5, 3, 1 (N > 7), N, 3, 1 (N > 3) or N, 1 */
    int32_t  mg_orders[8];
    int32_t  mg_smooth_degree, mg_coarse_degree;     /* <= 0 => 1 and 32 (measured best compromise) */
    double   mg_lmax[8];
    int32_t  mg_smoother_kind; /* 4: Chebyshev polynomial of the FOURTH kind (needs only lmax); else the
                                  first-kind recurrence on [0.1, 1] lmax of reading R9                          */
    int32_t  pad_;
    double   mg_coarse_lmin_frac; /* first-kind smoother of the LAST level runs on [frac, 1] lmax; <= 0 => 0.01.  A smaller
                                     fraction with a higher mg_coarse_degree (<= 64) makes it act as a coarse solver      */
    int32_t  null_mean;       /* 1: the operator has the constants as null space (lambda = 0 and no Dirichlet node: the
                                 all-Neumann pressure problem of a closed cell): solve A x = b - mean(b)
                                 and return the solution of zero mean, mean(v) = <v,1> / n_unique over unique nodes
                                 (reading R20).  SEMB_EINVAL if the tag set selects any Dirichlet node. */
    int32_t  mg_fp32;         /* 1: the V-cycle keeps its vectors and geometric factors in FP32 (the
                                 preconditioner runs in FP32 "to save on memory bandwidth") and computes in float (only
                                 the class sums of the gather-scatter accumulate in fp64); the PCG around the cycle, its
                                 residual and its solution stay fp64
                                 (reading R21: same iteration counts, fp64 true residual <= 2e-10)          */
    int32_t  mg_schwarz;      /* 1: every level of order >= 2 except the last is smoothed by the fourth-kind Chebyshev polynomial
                                 (degree mg_smooth_degree) in S A, S the overlapping Schwarz smoother of PAPER.md:L102 -- element
                                 closures as subdomains, fast-diagonalisation subdomain solves (reading R26); lambda_max(S A)
                                 estimated by 10 preconditioned Lanczos steps x 1.1 and cached.  0: Chebyshev-Jacobi (R19) */
    int32_t  pad2_;
} semb_pcg_opts;

typedef struct {
    int32_t iters;            /* iterations performed                                            */
    int32_t status;           /* same as the return value                                        */
    double  b_norm, r0_norm, r_norm, lmax_used;
    double* hist_host_or_null;/* in: host buffer [hist_len] for ||r_it||, it = 0..; may be NULL   */
    int32_t hist_len;
    int32_t profiled;         /* number of axhelm launches that were timed (opts.profile)            */
    double  axhelm_ms;        /* mean device time of those launches, milliseconds                    */
    int64_t launches;         /* kernels this call launched                                          */
} semb_pcg_stats;

/* b device [n]: assembled, masked right-hand side.  x device [n]: in = initial guess (continuous,
 * zero at Dirichlet nodes) unless x0_is_zero, out = solution.  Returns SEMB_OK (converged),
 * SEMB_MAXIT, SEMB_EBREAKDOWN, or an error.  Synchronises only to poll the stop flag. */
SEMB_API int semb_pcg_solve(semb_handle h, const semb_pcg_opts* opts, const double* b, double* x,
                   semb_pcg_stats* stats, void* stream);

/* One time step's worth of solves (BASELINE.json configs[4]: per step one pressure Poisson solve and the three
 * velocity and one temperature Helmholtz solves implied by the diffusion terms of PAPER.md:L194-196 Eq. 1-2), run
 * back to back on `stream` in the order given.  Each item is an independent semb_pcg_solve with its own
 * lambda, Dirichlet tag set, preconditioner and tolerances; masks and Jacobi diagonals are cached in the handle
 * per (tags, lambda), so repeated steps pay no setup.  items HOST [nsolves]; b, x device [n] each, caller-owned;
 * stats HOST [nsolves] or NULL.  Returns the first error (< 0; later items are not run), else SEMB_MAXIT if any
 * solve stopped at maxit, else SEMB_OK. */
typedef struct {
    semb_pcg_opts opts;
    const double* b;          /* device [n] assembled, masked right-hand side            */
    double*       x;          /* device [n] in: initial guess (see opts.x0_is_zero), out */
} semb_solve_item;
SEMB_API int semb_step_solve(semb_handle h, int nsolves, const semb_solve_item* items, semb_pcg_stats* stats,
                    void* stream);

/* 1.1 x the largest Ritz value of D^-1/2 A D^-1/2 after `steps` Lanczos steps from the continuous,
 * masked start vector v0 (device [n]). */
SEMB_API int semb_estimate_lmax(semb_handle h, double lambda, uint32_t dirichlet_tags, const double* v0,
                       int steps, double* lmax_out, void* stream);

/* z = one p-multigrid V-cycle applied to r (device [n] each, z != r; r continuous and masked) for the operator
 * (opts->lambda, opts->dirichlet_tags) with the levels opts->mg_* describe.  lmax_used_or_null HOST [nlevels]:
 * the bounds the smoothers used.  The coarse levels are built on first use and owned by the handle. */
SEMB_API int semb_mg_vcycle(semb_handle h, const semb_pcg_opts* opts, const double* r, double* z,
                   double* lmax_used_or_null, void* stream);
/* Transfer between levels `level` and `level + 1` of the same hierarchy: restrict_ == 0: out (level, [n_level]) =
 * M P in (level + 1); restrict_ != 0: out (level + 1) = M QQ^T J^T (invmult o in) (level).  Device pointers;
 * sizes: semb_mg_level_size. */
SEMB_API int semb_mg_transfer(semb_handle h, const semb_pcg_opts* opts, int level, int restrict_, const double* in,
                     double* out, void* stream);
/* local nodes of level `level` (E * (mg_orders[level] + 1)^3), or < 0 on error */
SEMB_API int64_t semb_mg_level_size(semb_handle h, const semb_pcg_opts* opts, int level);

/* z = Chebyshev-Jacobi(k) preconditioner applied to r (device [n] each, z != r). */
SEMB_API int semb_cheb_jacobi(semb_handle h, double lambda, uint32_t dirichlet_tags, int k, double lmax,
                     const double* r, double* z, void* stream);

/* out = S r, the Schwarz smoother of reading R26 for the operator (lambda, dirichlet_tags) on the handle's own mesh (order >= 2):
 * S r = M QQ^T [ w o A~_e^-1 (w o r) ], w = sqrt(1 / multiplicity).  r, out device [n], r continuous and masked, out != r. */
SEMB_API int semb_schwarz_apply(semb_handle h, double lambda, uint32_t dirichlet_tags, const double* r, double* out, void* stream);

/* ---- in-situ hand-off ---------------------------------------- */
#define SEMB_F64          1
#define SEMB_MEM_HOST     0
#define SEMB_MEM_DEVICE   1

typedef struct {
    const char* name;    /* owned by the handle                                    */
    void*       ptr;     /* for a registered field: exactly the pointer registered */
    int32_t     dtype;   /* SEMB_F64                                               */
    int32_t     memspace;/* SEMB_MEM_DEVICE                    */
    int64_t     count, stride;   /* elements; stride in elements                   */
    int64_t     cycle;   /* state/cycle of the last publish_state  */
    double      time;    /* state/time                            */
} semb_field_desc;

/* Register a device array under a name once.  Names "velocity_x|y|z" additionally
 * define the derived field "velocity_magnitude" (library-owned buffer, allocated here, not later). */
SEMB_API int semb_publish_field(semb_handle h, const char* name, double* dev_ptr, int64_t count);
/* Per analysis step: records cycle/time and refreshes, with one kernel on stream, those derived fields
 * that a consumer has asked for through semb_export_field before (none otherwise: nothing unused is paid for).
 * Steps that do no analysis simply do not call it.  A derived field's buffer is current from the first publish_state AFTER
 * its first export_field on. */
SEMB_API int semb_publish_state(semb_handle h, int64_t cycle, double time, void* stream);
/* No copy, no allocation, no synchronisation, no launch. */
SEMB_API int semb_export_field(semb_handle h, const char* name, semb_field_desc* out);
/* In-device consumer: min, max and an nbins histogram of the field over [lo, hi] (values outside go
 * to the end bins); bin = min(nbins-1, floor((v - lo) * (nbins / (hi - lo)))).
 * minmax_dev device [2], hist_dev device [nbins] (uint64).  Results stay on the device.
 * lo < hi: ONE pass over the field (min, max and counts together, 8 B/node).  If lo >= hi the range [min, max] found by a
 * first pass is used (two passes). */
SEMB_API int semb_field_minmax_hist(const semb_field_desc* f, int nbins, double lo, double hi,
                           double* minmax_dev, uint64_t* hist_dev, void* stream);

/* The same statistics of the magnitude of a vector field given by its three exported components, |v| = sqrt(fma(vz, vz,
 * fma(vy, vy, vx vx))) (reading R11) computed ON THE FLY: nothing is written, 24 B/node per pass.  One pass when
 * lo < hi, two when the range is to be found.  The three descriptors must agree in count and stride. */
SEMB_API int semb_vector_magnitude_minmax_hist(const semb_field_desc* vx, const semb_field_desc* vy, const semb_field_desc* vz,
                                      int nbins, double lo, double hi, double* minmax_dev, uint64_t* hist_dev, void* stream);

/* The same consumer for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): semb_field_minmax_hist with identical arguments and bit-identical results, but the call allocates NOTHING -- no
 * cudaMalloc, cudaFree, cudaMemset or allocating library routine -- and the outputs are written once, with their final values, by
 * the last thread block to finish.  Its accumulators (order-encoded min / max words, 64-bit bin counters, completion ticket) live
 * in one file-scope device array of 8 + SEMB_NOALLOC_MAX_BINS 64-bit words = 32 832 bytes, which every GPU that loads the
 * library holds until the process exits.  Limit: nbins <= SEMB_NOALLOC_MAX_BINS, else SEMB_EINVAL (the message names the limit).
 * Every call SHARES that array: each call clears it with a launch of its own first, so calls ordered on one stream (or by events)
 * are independent, but calls that OVERLAP on the GPU -- different streams or host threads with no ordering -- race on it and give
 * wrong counts.  One array per device: calls on different GPUs do not interact.  Asynchronous on stream (3-4 launches). */
#define SEMB_NOALLOC_MAX_BINS 4096
SEMB_API int semb_field_minmax_hist_noalloc(const semb_field_desc* f, int nbins, double lo, double hi,
                                   double* minmax_dev, uint64_t* hist_dev, void* stream);
/* Message of the last error of semb_field_minmax_hist_noalloc on the calling thread ("" if none).  Owned by the library. */
SEMB_API const char* semb_noalloc_last_error(void);

/* ---- in-situ IMAGE consumer (§5.3: the overview scene = "two slices on the walls,
 * two vertical slices in the background and an isocontour", 4096 pixels on the longest side, 2048 on the other).
 * The paper renders with ASCENT / VTK-m; no graphics API exists here, so the primitives are CUDA kernels on the mesh of
 * hexahedral SUB-CELLS between neighbouring GLL nodes, trilinear inside a cell (reading R24), fed by the
 * descriptors of semb_export_field.  Sub-cell id = e*N^3 + (k*N + j)*N + i.
 *
 * View: pixel (px, py) has the centre origin + ((px + 0.5) du) u + ((py + 0.5) dv) v, u and v unit vectors; w = u x v is the
 * viewing direction and (X - origin).w the depth of a point; depth_lo < depth_hi bound the scene along w (iso-surface only).
 * Colour map: s = clamp((val - lo) / (hi - lo), 0, 1) (ncolors - 1), linear between control points m = floor(s) and m + 1,
 * channel = floor(c + 0.5), alpha 255; packed r | g << 8 | b << 16 | a << 24.
 * key_dev device [width*height] uint64 (caller-owned scratch that doubles as output), rgba_dev device [width*height] or NULL.
 * Asynchronous on stream; nothing is allocated; images are reproducible bit for bit (atomicMin on order-independent keys). */
typedef struct {
    int32_t width, height;
    double  origin[3], u[3], v[3];
    double  du, dv;
    double  depth_lo, depth_hi;
} semb_image_view;

typedef struct {
    double   lo, hi;
    int32_t  ncolors;          /* 2..16 control points */
    uint8_t  rgb[16][3];
    uint32_t background;       /* packed RGBA of pixels nothing covers */
} semb_colormap;

/* rgba_dev[l] = colour of val_dev[l] (device arrays of n entries). */
SEMB_API int semb_colormap_apply(const semb_colormap* cm, const double* val_dev, int64_t n, uint32_t* rgba_dev, void* stream);

/* Planar slice: the image plane itself cuts the mesh.  Every sub-cell whose corners lie on both sides of the plane (or on
 * it) claims the pixels whose centres it contains (Newton inversion of its trilinear map: <= 12 steps, step <= 1e-10, inside
 * = |r|, |s|, |t| <= 1 + 1e-9); where several cells contain a centre the smallest id wins.  key = cell id << 32 | RGBA, cell
 * id 0xffffffff where nothing was hit. */
SEMB_API int semb_image_slice(semb_handle h, const semb_field_desc* field, const semb_image_view* view, const semb_colormap* cmap,
                     uint64_t* key_dev, uint32_t* rgba_dev, void* stream);

/* Iso-surface {field = iso} seen orthographically along w: marching tetrahedra (6 per sub-cell around the diagonal corner
 * 0 - corner 7, corner q = a + 2b + 4c) on the linear interpolant, flat shading 0.25 + 0.75 |n . light| (light HOST [3], unit)
 * of the colour the map gives to color_or_null's value (NULL: to iso), nearest surface per pixel.
 * key = depth quantised to 2^-32 of [depth_lo, depth_hi] << 32 | RGBA, depth 0xffffffff where nothing was hit. */
SEMB_API int semb_image_isosurface(semb_handle h, const semb_field_desc* field, double iso, const semb_field_desc* color_or_null,
                          const semb_image_view* view, const semb_colormap* cmap, const double* light, uint64_t* key_dev,
                          uint32_t* rgba_dev, void* stream);

/* ---- the rest of a Boussinesq time step around the solves (Eqs. (1)-(3), L238, L272).
 * The paper states the equations only; the discrete step is DESIGN.md reading R25:  nu = sqrt(Pr/Ra), kappa = 1/sqrt(Ra Pr),
 * theta = T - (1 - z); order 1 on the first step (beta0 = 1, b = [1], a = [1]), then BDF2 / EXT2 (3/2, [2, -1/2], [2, -1]):
 *   (i)   N_c = -(u.grad)u_c + delta_cz T + f_c,  N_theta = -(u.grad)theta + u_z + f_theta  (collocation, per element);
 *         omega = curl u;  omega_bar = QQ^T(B omega) / QQ^T(B);  C = curl omega_bar
 *   (ii)  u~ = sum_k b_k u^(n+1-k) + dt sum_k a_k N^(n+1-k);  g = u~/dt - nu sum_k a_k C^(n+1-k);
 *         A p = QQ^T wdiv(g), all Neumann, zero mean (null_mean), started from p^n
 *   (iii) (A + beta0/(nu dt) B) u_c^(n+1) = M QQ^T B (u~_c - dt dp/dx_c) / (nu dt), started from u_c^n; the same for theta with kappa.
 * Building blocks, each element-local and asynchronous on stream (arrays device [n]): */
/* collocation gradient of a nodal field: g_b = sum_a (dr_a/dx_b) dphi/dr_a (discontinuous across elements) */
SEMB_API int semb_gradient(semb_handle h, const double* phi, double* gx, double* gy, double* gz, void* stream);
/* weak divergence, the transpose of the gradient in the GLL inner product: out_i = int grad(phi_i) . g  (unassembled) */
SEMB_API int semb_weak_divergence(semb_handle h, const double* gx, const double* gy, const double* gz, double* out, void* stream);
/* step (i): N4 device [4][n] = N_x, N_y, N_z, N_theta; omega3 device [3][n] = the averaged vorticity omega_bar.
 * forcing_or_null HOST array of 4 device pointers (each may be NULL). */
SEMB_API int semb_flow_explicit_terms(semb_handle h, const double* ux, const double* uy, const double* uz, const double* theta,
                             const double* const* forcing_or_null, double* N4, double* omega3, void* stream);

typedef struct {
    double   Ra, Pr, dt;
    uint32_t tags_u, tags_T;      /* Dirichlet tag sets of the velocity (no-slip walls) and of theta (isothermal plates) */
    double   rtol;                /* of every solve; <= 0 => 1e-10 */
    int32_t  precond_p, precond_u;/* semb_pcg_opts.precond of the pressure solve (0 => 3, p-multigrid) and of the Helmholtz solves (0 => 1, Jacobi) */
    int32_t  mg_fp32, maxit;      /* maxit <= 0 => 20000 */
    int32_t  mg_schwarz, pad_;    /* 1: the p-multigrid solves smooth with the Chebyshev-Schwarz smoother (semb_pcg_opts.mg_schwarz) */
    const double* forcing[4];     /* optional body forces f_x, f_y, f_z, f_theta at time level n, device [n] each, or NULL */
} semb_flow_opts;

typedef struct {                  /* every array device [n], caller-owned */
    double* u[3]; double* theta; double* p;      /* in: level n (p: initial guess of the solve); out: level n+1 */
    double* u1[3]; double* theta1;               /* in: level n-1;            out: level n                      */
    double* N1[4];                               /* in: explicit terms of level n-1; out: of level n            */
    double* C1[3];                               /* in: curl curl u of level n-1;    out: of level n            */
    int64_t step_index;                          /* 0 on the first call (histories are then ignored); incremented */
} semb_flow_state;

typedef struct { int32_t iters[5], status[5]; } semb_flow_stats;    /* pressure, u_x, u_y, u_z, theta */

/* One time step.  Returns the worst status of the five solves (SEMB_OK, SEMB_MAXIT) or an error.  The metrics (72 B/node)
 * and 21 work vectors are allocated on the first call and owned by the handle. */
SEMB_API int semb_boussinesq_step(semb_handle h, const semb_flow_opts* opts, semb_flow_state* state, semb_flow_stats* stats_or_null,
                         void* stream);

/* ---- convenience: the same calls with HOST buffers (copies inside; used for end-to-end timing) */
SEMB_API int semb_apply_axhelm_host(semb_handle h, double lambda, const double* u_host, double* w_host);
/* pcg_solve with b and x in HOST memory (pinned memory makes the copies asynchronous): b is copied to the
 * device, the solve runs, x is copied back; the device staging buffers belong to the handle. */
SEMB_API int semb_pcg_solve_host(semb_handle h, const semb_pcg_opts* opts, const double* b_host, double* x_host,
                                 semb_pcg_stats* stats, void* stream);

/* Blocking copy of `bytes` bytes from device memory (e.g. a semb_info view) to host memory. */
SEMB_API int semb_read_device(const void* dev, void* host, size_t bytes);

/* Measurement aid, not part of the method ("a measured read-heavy stream ceiling"): dst[l] = sum over
 * c < nread of src[c*n + l], a pure stream with nread : 1 read : write mix (axhelm's is 7 : 1).  src device [nread*n],
 * dst device [n], both 16-byte aligned, n even, 1 <= nread <= 8.  Asynchronous on stream.  bench.py times it to state
 * what HBM delivers for that mix next to the 1 : 1 copy bandwidth. */
SEMB_API int semb_stream_probe(const double* src, double* dst, int64_t n, int nread, void* stream);

/* Library version and the compute capability it was built for ("sm_100a"). */
SEMB_API const char* semb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SEMB200_H */
