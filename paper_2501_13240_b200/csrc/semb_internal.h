// Internal declarations of libsemb200.so (not part of the ABI).  CUDA C++ for sm_100a only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <map>
#include <string>
#include <utility>
#include <vector>

#include "../../include/semb200.h"

#define SEMB_MAXN1 (SEMB_MAX_N + 1)

// Device-resident scalars of the Krylov loop (alpha, beta, ... never visit the host; north_star:
// "fused PCG vector updates and dot-product reductions").  One copy lives in device memory, a pinned host
// mirror receives it when the host polls the stop flag.
struct semb_scalars {
    double rho_old, rho_new, pAp, alpha, beta, rr, rz, rnorm, bnorm, r0norm, target, rtol, atol, aux, shift;
    int32_t iter, done, status, maxit, x_pending, pad_;
    uint32_t ticket[8];
};

struct semb_mask_entry {
    int32_t* list = nullptr;   // device: local ids of Dirichlet nodes, ascending
    int64_t  count = 0;
};

#define SEMB_DINV_CACHE 8
#define SEMB_FLOW_WORK 21      // N(4) omega(3) curl-curl(3) u~(3) g(3) b_p(1) grad p(3) rhs(1)
struct semb_dinv_entry { uint32_t tags; double lambda; double* d; uint64_t stamp; };

struct semb_field_entry {
    std::string name;
    double* ptr = nullptr;
    int64_t count = 0;
    bool derived = false;
    bool wanted = false;       // derived fields: a consumer has asked for the pointer, so publish_state keeps the buffer current
};

struct semb_mg;
struct semb_schwarz;
struct semb_coarse;

struct semb_mesh {
    int64_t E = 0; int N = 0, n1 = 0; int64_t Np = 0, n = 0;
    int64_t n_unique = 0, n_shared = 0, n_gs = 0;
    double tol = 0.0;
    bool has_alloc = false; semb_allocator alloc{};
    double xi[SEMB_MAXN1], rho[SEMB_MAXN1], D[SEMB_MAXN1 * SEMB_MAXN1];   // host copies
    // handle-owned device arrays
    double*  xyz = nullptr;        // [3][n] copy of the node coordinates (coarse multigrid levels are built from it)
    double   period[3] = {0.0, 0.0, 0.0};
    double*  geo = nullptr;        // [E][7][Np]  canonical layout (semb_info.geo)
    double*  geoK = nullptr;       // kernel-native layout of the same data (axhelm.cu), may alias geo
    // geometry representation the fp64 axhelm launches read (semb_set_geometry_mode; geomode.cu)
    int      geo_mode = 0;         // SEMB_GEO_STORED | _F32 | _AFFINE | _TRILINEAR
    float*   geoF = nullptr;       // [E][7][Np] float copy of geo (mode 1)
    double*  geoC = nullptr;       // [E][8]  affine element constants (mode 2)
    double*  geoT = nullptr;       // [E][3][8] trilinear coefficients (mode 3)
    double   geo_dev[2] = {-1.0, -1.0};   // measured: max deviation of the nodes from the trilinear / affine map of the corners, relative to max |coordinate|
    int32_t* gid = nullptr;        // [n]
    double*  invmult = nullptr;    // [n]
    int32_t* gs_off = nullptr;     // [n_gs+1]
    int32_t* gs_ids = nullptr;     // [n_shared]
    int32_t* gs_code = nullptr;    // [n] gather-form code per node (setup.cu: k_gs_code)
    int32_t* gs_hi = nullptr;      // [n_gs_hi] indices (into gs_off) of the classes with >= 3 members
    int64_t  n_gs_hi = 0;
    std::vector<int32_t> face_tag; // host [E*6]
    int32_t* face_tag_dev = nullptr;
    std::map<uint32_t, semb_mask_entry> masks;
    // Jacobi diagonals: the lambda-independent assembled parts diagA = QQ^T diag(D^T G D), diagB = QQ^T B are built
    // once; 1 / (diagA + lambda diagB) (1 at masked nodes) is kept for the SEMB_DINV_CACHE most recently used
    // (tags, lambda) pairs only, so a variable time step (lambda = c / dt) neither leaks memory nor re-runs the setup.
    double* diagA = nullptr; double* diagB = nullptr;
    std::vector<semb_dinv_entry> dinvs; uint64_t dinv_clock = 0;
    // flow operators of the Boussinesq step (flow.cu), built on first use
    double* flow_met = nullptr;         // [E][9][Np] dr_a/dx_b
    double* flow_D = nullptr;           // D on the device
    double* flow_work = nullptr;        // [SEMB_FLOW_WORK][n]
    const double** flow_tab = nullptr;  // device pointer tables (8 slots x 16)
    // solver workspace
    double* work = nullptr; int64_t work_vecs = 0;
    double* partials = nullptr;         // block partial sums [4][SEMB_MAX_BLOCKS]
    double* ax_dot = nullptr;           // per-element partials of p.Ap written by axhelm [E]
    bool defer_dot_finish = false;      // small-mesh PCG: the partials are summed by k_iter_small, not by k_ax_dot_finish
    semb_scalars* scal = nullptr;       // device
    semb_scalars* scal_host = nullptr;  // pinned mirror
    double* hist_dev = nullptr; int hist_cap = 0;
    // persistent small-mesh PCG (pcg_persist.cu): remote-copy lists of the shared nodes, Dirichlet flags of the last tag set, per-block partials + barrier
    int32_t* pp_noff = nullptr; int32_t* pp_rlist = nullptr; int pp_maxcnt = 0;
    unsigned char* pp_msk = nullptr; double* pp_part = nullptr; uint32_t pp_msk_tags = 0; bool pp_msk_valid = false;
    double* stage = nullptr;            // device staging of the *_host entry points [2][n]
    int64_t launches = 0;               // kernels launched through this handle (bench.py reports it)
    std::vector<cudaEvent_t> prof_ev;   // event pairs around axhelm launches (opts.profile)
    std::vector<semb_mg*> mgs;          // p-multigrid hierarchies built so far (mg.cu), owned
    std::vector<semb_schwarz*> schwarz; // Schwarz subdomain data of this (level) mesh per Dirichlet tag set (schwarz.cu), owned
    semb_coarse* coarse = nullptr;      // assembled operator of this mesh when it is the order-1 last level of a multigrid hierarchy (coarse.cu), owned
    // export
    std::vector<semb_field_entry> fields;
    int64_t cycle = 0; double time = 0.0;
    std::string err;
};

// Widening of a stored value (double, or float on the fp32-storage multigrid levels) to the fp64 the kernels compute
// in.  Measured and rejected: doing the float -> double widening with integer operations instead of F2F.F64.F32 made
// the fp32 V-cycle 8 % SLOWER than the plain cast (cfg3: 23.2 vs 19.1 ms per iteration; fp64 storage: 21.7 ms).
#ifdef __CUDACC__
__device__ __forceinline__ double semb_wide(double v) { return v; }
__device__ __forceinline__ double semb_wide(float f) { return (double)f; }
#endif

// ---- helpers -------------------------------------------------------------------------------
int  semb_sm_count();      // multiProcessorCount of the current device (cached per process; 148 on B200): streaming grids are sized from it
int  semb_fail(semb_mesh* h, int code, const char* fmt, ...);
void* semb_dev_alloc(semb_mesh* h, size_t bytes);
void  semb_dev_free(semb_mesh* h, void* p);

#define SEMB_CUDA(h, call)                                                                     \
    do { cudaError_t e_ = (call);                                                              \
         if (e_ != cudaSuccess) return semb_fail((h), SEMB_ECUDA, "%s:%d %s: %s", __FILE__,    \
                                                 __LINE__, #call, cudaGetErrorString(e_)); } while (0)

#define SEMB_MAX_BLOCKS 4096   // upper bound on the grid of any kernel that writes block partials

// ---- basis.cpp
void semb_basis_host(int N, double* xi, double* rho, double* D);

// ---- setup.cu
int semb_setup_geo(semb_mesh* h, const double* x, const double* y, const double* z, cudaStream_t s);
int semb_setup_numbering(semb_mesh* h, const double* x, const double* y, const double* z,
                         const double* period, const int32_t* gid_in, cudaStream_t s);
int semb_get_mask(semb_mesh* h, uint32_t tags, semb_mask_entry* out, cudaStream_t s);
// Jacobi / unpreconditioned PCG iterations of a small mesh in ONE cooperative launch, from the state k_pcg_init left (r, scal).
// Returns 1 if launched (scal->done is then set by the kernel), 0 if the mesh is not eligible, < 0 on error.
int semb_pcg_persist_run(semb_mesh* h, double lambda, const semb_mask_entry& m, uint32_t tags, const double* dinv, double* r, double* x, double* p,
                         double* q, double* hist, int hist_cap, cudaStream_t s);
int semb_get_dinv(semb_mesh* h, double lambda, uint32_t tags, double** out, cudaStream_t s);
int semb_diag_local(semb_mesh* h, double lambda, double* d, cudaStream_t s);

// ---- axhelm.cu
int semb_axhelm_upload_basis(semb_mesh* h);
int semb_axhelm_prepare_geo(semb_mesh* h, cudaStream_t s);
// dot_partials != NULL: also writes per-block partial sums of sum_l u_l w_l and (last block) their total
// into *dot_total (device).
// scal != NULL (PCG): the kernel early-exits when scal->done, and its last block leaves
// scal->pAp = sum_l u_l w_l and scal->alpha = scal->rho_new / scal->pAp (breakdown -> status, done).
int semb_axhelm_launch(semb_mesh* h, double lambda, const double* lam0, const double* lam1,
                       const double* u, double* w, int nfields, semb_scalars* scal, cudaStream_t s);

int semb_axhelm_pcg_launch(semb_mesh* h, double lambda, const double* zsrc, const double* dinv, double* p, double* x,
                           double* q, semb_scalars* scal, cudaStream_t s);

int64_t semb_axhelm_dot_count(semb_mesh* h);       // number of per-block partials the PCG-fused launch writes into h->ax_dot
int semb_axhelm_scaled_launch(semb_mesh* h, double lambda, const double* r, const double* dinv, double scale, double* d,
                              double* Ad, semb_scalars* scal, cudaStream_t s);

int semb_axhelm_launch_f(semb_mesh* h, double lambda, const float* geo, const float* u, float* w, semb_scalars* scal, cudaStream_t s);
int semb_axhelm_scaled_launch_f(semb_mesh* h, double lambda, const float* geo, const float* r, const float* dinv, double scale, float* d,
                                float* Ad, semb_scalars* scal, cudaStream_t s);

// ---- gs.cu
int semb_gs_launch(semb_mesh* h, double* w, int nfields, cudaStream_t s);
// QQ^T restricted to the classes with >= 3 members (the rest is done in gather form by the consumer, pcg.cu)
int semb_gs_hi_launch(semb_mesh* h, double* w, const semb_scalars* scal, cudaStream_t s);
int semb_mask_launch(semb_mesh* h, const semb_mask_entry& m, double* w, int nfields, cudaStream_t s);
int semb_gs_launch_f(semb_mesh* h, float* w, cudaStream_t s);
int semb_gs_hi_launch_f(semb_mesh* h, float* w, const semb_scalars* scal, cudaStream_t s);
int semb_mask_launch_f(semb_mesh* h, const semb_mask_entry& m, float* w, cudaStream_t s);

// ---- pcg.cu
int semb_pcg_run(semb_mesh* h, const semb_pcg_opts* o, const double* b, double* x, semb_pcg_stats* st,
                 cudaStream_t s);
int semb_lanczos_run(semb_mesh* h, double lambda, uint32_t tags, const double* v0, int steps, double* lmax,
                     cudaStream_t s);
int semb_cheb_run(semb_mesh* h, double lambda, uint32_t tags, int k, double lmax, const double* r, double* z,
                  cudaStream_t s);
int semb_operator_run(semb_mesh* h, double lambda, const semb_mask_entry& m, const double* v, double* out,
                      cudaStream_t s);
int semb_ensure_work(semb_mesh* h, int64_t vecs);
#define SEMB_MAX_CHEB 64
struct semb_cheb_coef { double itheta; double c1[SEMB_MAX_CHEB], c2[SEMB_MAX_CHEB]; };
// kind 4: fourth-kind polynomial (lmax only); else first kind on [lmin_frac, 1] lmax (lmin_frac <= 0 => 0.1, reading R9)
semb_cheb_coef semb_cheb_coefficients(int k, double lmax, int kind = 1, double lmin_frac = 0.1);
// z = Cheb_k(r) on h;  res, d, Ad: work vectors [n].  in_pcg: also leave rho = <r,z> and beta in scal.
int semb_cheb_apply(semb_mesh* h, double lambda, const semb_mask_entry& m, const double* dinv, int k, const semb_cheb_coef& c,
                    const double* r, double* z, double* res, double* d, double* Ad, semb_scalars* scal, bool in_pcg, cudaStream_t s,
                    bool zacc = false);       // zacc: z += Cheb_k(r) instead of z = Cheb_k(r) (k >= 1)
// res = r - M QQ^T A_L z  (z continuous and masked; tmp: scratch [n])
int semb_residual_launch(semb_mesh* h, double lambda, const semb_mask_entry& m, const double* z, const double* r, double* res,
                         double* tmp, semb_scalars* scal, cudaStream_t s);
int semb_residual_launch_f(semb_mesh* h, double lambda, const float* geo, const semb_mask_entry& m, const float* z, const float* r,
                           float* res, float* tmp, semb_scalars* scal, cudaStream_t s);
int semb_cheb_apply_f(semb_mesh* h, double lambda, const float* geo, const semb_mask_entry& m, const float* dinv, int k,
                      const semb_cheb_coef& c, const float* r, float* z, float* res, float* d, float* Ad, semb_scalars* scal,
                      cudaStream_t s, bool zacc);
int semb_dot_rz_launch(semb_mesh* h, const double* r, const double* z, semb_scalars* scal, cudaStream_t s);

// ---- mg.cu: p-multigrid V-cycle
struct semb_mg_ctx { semb_mg* mg; double lambda; uint32_t tags; int k_smooth, k_coarse, kind, fp32; double coarse_frac; double lmax[8];
                     int schwarz; semb_schwarz* sz[8]; double sz_lmax[8]; };
int semb_mg_orders(semb_mesh* h, const semb_pcg_opts* o, int* nlev_out, int* orders);
int semb_mg_prepare(semb_mesh* h, const semb_pcg_opts* o, semb_mg_ctx* ctx, cudaStream_t s);
int semb_mg_vcycle_run(semb_mesh* h, const semb_mg_ctx& ctx, int level, const double* r, double* z, semb_scalars* scal, cudaStream_t s);
int semb_mg_transfer_run(semb_mesh* h, const semb_mg_ctx& ctx, int level, int restrict_, const double* in, double* out, cudaStream_t s);
int64_t semb_mg_level_n(const semb_mg_ctx& ctx, int level);
void semb_mg_destroy_all(semb_mesh* h);

// ---- coarse.cu: the order-1 last level on its assembled operator (one launch per Chebyshev step)
void semb_coarse_free(semb_mesh* L);
int semb_coarse_get(semb_mesh* L, semb_coarse** out, cudaStream_t s);       // *out = NULL: not eligible, stay matrix-free
int semb_coarse_cheb(semb_mesh* L, semb_coarse* c, double lambda, uint32_t tags, const semb_mask_entry& m, const double* dinv, int k,
                     const semb_cheb_coef& cf, const double* r, double* z, semb_scalars* scal, cudaStream_t s);
int semb_coarse_cheb_f(semb_mesh* L, semb_coarse* c, double lambda, uint32_t tags, const semb_mask_entry& m, const float* dinv, int k,
                       const semb_cheb_coef& cf, const float* r, float* z, semb_scalars* scal, cudaStream_t s);

// ---- schwarz.cu: overlapping Schwarz smoother of the multigrid levels (reading R26)
void semb_schwarz_free(semb_mesh* L);
int semb_schwarz_get(semb_mesh* L, uint32_t tags, bool want_float, semb_schwarz** out, cudaStream_t s);
int semb_schwarz_lmax(semb_mesh* L, semb_schwarz* zd, double lambda, const semb_mask_entry& m, const double* v0, int steps, double* const* work,
                      double* lmax, cudaStream_t s);
int semb_schwarz_apply_run(semb_mesh* L, uint32_t tags, double lambda, const double* r, double* out, cudaStream_t s);
// z (+)= W_k-Chebyshev (fourth kind) in S A applied to r; res, d, sr, t: work vectors of the level
int semb_schwarz_cheb4(semb_mesh* L, semb_schwarz* zd, double lambda, const semb_mask_entry& m, int k, double lmax, const double* r, double* z,
                       double* res, double* d, double* sr, double* t, semb_scalars* scal, cudaStream_t s, bool zacc);
int semb_schwarz_cheb4_f(semb_mesh* L, semb_schwarz* zd, double lambda, const float* geo, const semb_mask_entry& m, int k, double lmax, const float* r,
                         float* z, float* res, float* d, float* sr, float* t, semb_scalars* scal, cudaStream_t s, bool zacc);

// ---- flow.cu
int semb_flow_prepare(semb_mesh* h, cudaStream_t s);

// ---- export.cu
int semb_vmag_launch(const double* vx, const double* vy, const double* vz, double* out, int64_t n, cudaStream_t s);
int semb_minmax_hist_launch(const double* v, const double* v1, const double* v2, int64_t n, int64_t stride, int nbins, double lo, double hi,
                            double* minmax_dev, uint64_t* hist_dev, cudaStream_t s);
