// C ABI entry points of libsemb200.so (include/semb200.h): argument checks, handle bookkeeping, dispatch.
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include "semb_internal.h"

static std::string g_setup_error;

int semb_fail(semb_mesh* h, int code, const char* fmt, ...)
{
    char buf[512];
    va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof(buf), fmt, ap); va_end(ap);
    if (h) h->err = buf; else g_setup_error = buf;
    return code;
}

int semb_sm_count()
{
    static int sms = 0;
    if (sms <= 0) {
        int dev = 0, v = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) sms = v;
        else { cudaGetLastError(); return 148; }
    }
    return sms;
}

void* semb_dev_alloc(semb_mesh* h, size_t bytes)
{
    if (bytes == 0) bytes = 8;
    if (h && h->has_alloc) return h->alloc.alloc(bytes, h->alloc.user);
    void* p = nullptr;
    if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return p;
}

void semb_dev_free(semb_mesh* h, void* p)
{
    if (!p) return;
    if (h && h->has_alloc) h->alloc.free(p, h->alloc.user); else cudaFree(p);
}

extern "C" {

int semb_read_device(const void* dev, void* host, size_t bytes)
{
    if (!dev || !host) return SEMB_EINVAL;
    return cudaMemcpy(host, dev, bytes, cudaMemcpyDeviceToHost) == cudaSuccess ? SEMB_OK : SEMB_ECUDA;
}

const char* semb_version(void) { return "semb200 0.1 (sm_100a, fp64)"; }

int semb_gll(int N, double* xi, double* rho, double* D)
{
    if (N < 1 || N > SEMB_MAX_N) return SEMB_EINVAL;
    semb_basis_host(N, xi, rho, D);
    return SEMB_OK;
}

const char* semb_last_error(semb_handle h) { return h ? h->err.c_str() : g_setup_error.c_str(); }

int semb_destroy(semb_handle h)
{
    if (!h) return SEMB_OK;
    cudaDeviceSynchronize();
    semb_mg_destroy_all(h);
    semb_schwarz_free(h);
    semb_coarse_free(h);
    semb_dev_free(h, h->xyz);
    semb_dev_free(h, h->geo); semb_dev_free(h, h->gid); semb_dev_free(h, h->invmult); semb_dev_free(h, h->gs_code); semb_dev_free(h, h->gs_hi);
    if (h->geoK && h->geoK != h->geo) semb_dev_free(h, h->geoK);
    semb_dev_free(h, h->geoF); semb_dev_free(h, h->geoC); semb_dev_free(h, h->geoT);
    semb_dev_free(h, h->flow_met); semb_dev_free(h, h->flow_D); semb_dev_free(h, h->flow_work); semb_dev_free(h, (void*)h->flow_tab);
    semb_dev_free(h, h->gs_off); semb_dev_free(h, h->gs_ids); semb_dev_free(h, h->face_tag_dev);
    for (auto& kv : h->masks) semb_dev_free(h, kv.second.list);
    for (auto& en : h->dinvs) semb_dev_free(h, en.d);
    semb_dev_free(h, h->diagA); semb_dev_free(h, h->diagB);
    semb_dev_free(h, h->work); semb_dev_free(h, h->partials); semb_dev_free(h, h->ax_dot); semb_dev_free(h, h->scal); semb_dev_free(h, h->hist_dev); semb_dev_free(h, h->stage);
    semb_dev_free(h, h->pp_noff); semb_dev_free(h, h->pp_rlist); semb_dev_free(h, h->pp_msk); semb_dev_free(h, h->pp_part);
    if (h->scal_host) cudaFreeHost(h->scal_host);
    for (cudaEvent_t ev : h->prof_ev) cudaEventDestroy(ev);
    for (auto& f : h->fields) if (f.derived) semb_dev_free(h, f.ptr);
    delete h;
    return SEMB_OK;
}

int semb_setup(int64_t E, int N, const double* x, const double* y, const double* z, const int32_t* face_tag,
               const double* period, const int32_t* gid_or_null, const semb_allocator* a, void* stream,
               semb_handle* out)
{
    if (out) *out = nullptr;
    if (!out || E < 1 || N < 1 || N > SEMB_MAX_N || !x || !y || !z || !face_tag || !period)
        return semb_fail(nullptr, SEMB_EINVAL, "semb_setup: bad argument (E=%lld N=%d)", (long long)E, N);
    const int64_t Np = (int64_t)(N + 1) * (N + 1) * (N + 1);
    if (E * Np >= ((int64_t)1 << 31)) return semb_fail(nullptr, SEMB_EINVAL, "semb_setup: E*(N+1)^3 must be < 2^31");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return semb_fail(nullptr, SEMB_ECUDA, "semb_setup: no CUDA device (there is no CPU fallback)");
    }
    semb_mesh* h = new semb_mesh();
    h->E = E; h->N = N; h->n1 = N + 1; h->Np = Np; h->n = E * Np;
    if (a && a->alloc && a->free) { h->has_alloc = true; h->alloc = *a; }
    cudaStream_t s = (cudaStream_t)stream;
    semb_basis_host(N, h->xi, h->rho, h->D);
    h->face_tag.assign(face_tag, face_tag + E * 6);
    h->fields.reserve(64);        // descriptors hand out name pointers: never reallocate
    int rc = SEMB_OK;
    do {
        h->face_tag_dev = (int32_t*)semb_dev_alloc(h, sizeof(int32_t) * (size_t)E * 6);
        if (!h->face_tag_dev) { rc = semb_fail(h, SEMB_ENOMEM, "face tags"); break; }
        if (cudaMemcpyAsync(h->face_tag_dev, face_tag, sizeof(int32_t) * (size_t)E * 6, cudaMemcpyHostToDevice, s) != cudaSuccess) {
            rc = semb_fail(h, SEMB_ECUDA, "face tag upload: %s", cudaGetErrorString(cudaGetLastError())); break;
        }
        h->xyz = (double*)semb_dev_alloc(h, sizeof(double) * 3 * (size_t)h->n);
        if (!h->xyz) { rc = semb_fail(h, SEMB_ENOMEM, "coordinates"); break; }
        {
            const double* src[3] = { x, y, z };
            bool ok = true;
            for (int c = 0; c < 3; ++c)
                ok = ok && cudaMemcpyAsync(h->xyz + c * h->n, src[c], sizeof(double) * (size_t)h->n, cudaMemcpyDeviceToDevice, s) == cudaSuccess;
            if (!ok) { rc = semb_fail(h, SEMB_ECUDA, "coordinate copy: %s", cudaGetErrorString(cudaGetLastError())); break; }
            for (int c = 0; c < 3; ++c) h->period[c] = period[c];
        }
        if ((rc = semb_axhelm_upload_basis(h))) break;
        if ((rc = semb_setup_geo(h, x, y, z, s))) break;
        if ((rc = semb_setup_numbering(h, x, y, z, period, gid_or_null, s))) break;
        if ((rc = semb_axhelm_prepare_geo(h, s))) break;
        if ((rc = semb_ensure_work(h, 0))) break;
        if (cudaStreamSynchronize(s) != cudaSuccess) { rc = semb_fail(h, SEMB_ECUDA, "setup sync: %s", cudaGetErrorString(cudaGetLastError())); break; }
    } while (0);
    if (rc) { g_setup_error = h->err; semb_destroy(h); return rc; }
    *out = h;
    return SEMB_OK;
}

int semb_mesh_info(semb_handle h, semb_info* o)
{
    if (!h || !o) return SEMB_EINVAL;
    o->E = h->E; o->N = h->N; o->n1 = h->n1; o->Np = h->Np; o->n = h->n;
    o->n_unique = h->n_unique; o->n_shared = h->n_shared; o->n_gs = h->n_gs; o->tol = h->tol;
    o->gid = h->gid; o->geo = h->geo; o->invmult = h->invmult; o->gs_offsets = h->gs_off; o->gs_ids = h->gs_ids;
    return SEMB_OK;
}

int semb_apply_axhelm(semb_handle h, double lambda, const double* lam0, const double* lam1, const double* u,
                      double* w, int nfields, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!u || !w || u == w || nfields < 1) return semb_fail(h, SEMB_EINVAL, "apply_axhelm: bad argument");
    return semb_axhelm_launch(h, lambda, lam0, lam1, u, w, nfields, nullptr, (cudaStream_t)stream);
}

int semb_gather_scatter(semb_handle h, double* w, int nfields, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!w || nfields < 1) return semb_fail(h, SEMB_EINVAL, "gather_scatter: bad argument");
    return semb_gs_launch(h, w, nfields, (cudaStream_t)stream);
}

int semb_apply_mask(semb_handle h, uint32_t tags, double* w, int nfields, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!w || nfields < 1) return semb_fail(h, SEMB_EINVAL, "apply_mask: bad argument");
    semb_mask_entry m;
    int rc = semb_get_mask(h, tags, &m, (cudaStream_t)stream); if (rc) return rc;
    return semb_mask_launch(h, m, w, nfields, (cudaStream_t)stream);
}

__global__ void k_mass_times(int64_t n, int64_t Np, const double* __restrict__ geo, const double* __restrict__ f, double* __restrict__ b)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e = l / Np, loc = l - e * Np;
        b[l] = geo[e * 7 * Np + 6 * Np + loc] * f[l];
    }
}

int semb_assemble_rhs(semb_handle h, uint32_t tags, const double* f, double* b, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!f || !b || f == b) return semb_fail(h, SEMB_EINVAL, "assemble_rhs: bad argument");
    cudaStream_t s = (cudaStream_t)stream;
    semb_mask_entry m;
    int rc = semb_get_mask(h, tags, &m, s); if (rc) return rc;
    int64_t blocks = (h->n + 1023) / 1024; if (blocks > semb_sm_count() * 8) blocks = semb_sm_count() * 8;
    k_mass_times<<<(unsigned)blocks, 256, 0, s>>>(h->n, h->Np, h->geo, f, b);
    SEMB_CUDA(h, cudaGetLastError());
    rc = semb_gs_launch(h, b, 1, s); if (rc) return rc;
    return semb_mask_launch(h, m, b, 1, s);
}

int semb_apply_operator(semb_handle h, double lambda, uint32_t tags, const double* v, double* out, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!v || !out || v == out) return semb_fail(h, SEMB_EINVAL, "apply_operator: bad argument");
    semb_mask_entry m;
    int rc = semb_get_mask(h, tags, &m, (cudaStream_t)stream); if (rc) return rc;
    return semb_operator_run(h, lambda, m, v, out, (cudaStream_t)stream);
}

int semb_jacobi_diag(semb_handle h, double lambda, uint32_t tags, double* dinv_out, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!dinv_out) return semb_fail(h, SEMB_EINVAL, "jacobi_diag: bad argument");
    double* d;
    int rc = semb_get_dinv(h, lambda, tags, &d, (cudaStream_t)stream); if (rc) return rc;
    SEMB_CUDA(h, cudaMemcpyAsync(dinv_out, d, sizeof(double) * (size_t)h->n, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return SEMB_OK;
}

int semb_pcg_solve(semb_handle h, const semb_pcg_opts* o, const double* b, double* x, semb_pcg_stats* st, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!o || !b || !x || b == x) return semb_fail(h, SEMB_EINVAL, "pcg_solve: bad argument");
    const int rc = semb_pcg_run(h, o, b, x, st, (cudaStream_t)stream);
    if (st) st->status = rc;
    return rc;
}

int semb_step_solve(semb_handle h, int nsolves, const semb_solve_item* items, semb_pcg_stats* stats, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (nsolves < 0 || (nsolves > 0 && !items)) return semb_fail(h, SEMB_EINVAL, "step_solve: bad argument");
    int worst = SEMB_OK;
    for (int i = 0; i < nsolves; ++i) {
        const int rc = semb_pcg_solve(h, &items[i].opts, items[i].b, items[i].x, stats ? &stats[i] : nullptr, stream);
        if (rc < 0) return rc;
        if (rc > worst) worst = rc;
    }
    return worst;
}

int semb_estimate_lmax(semb_handle h, double lambda, uint32_t tags, const double* v0, int steps, double* lmax_out, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!v0 || !lmax_out) return semb_fail(h, SEMB_EINVAL, "estimate_lmax: bad argument");
    int rc = semb_ensure_work(h, 4); if (rc) return rc;
    return semb_lanczos_run(h, lambda, tags, v0, steps, lmax_out, (cudaStream_t)stream);
}

int semb_mg_vcycle(semb_handle h, const semb_pcg_opts* o, const double* r, double* z, double* lmax_used, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!o || !r || !z || r == z) return semb_fail(h, SEMB_EINVAL, "mg_vcycle: bad argument");
    semb_mg_ctx ctx;
    int rc = semb_mg_prepare(h, o, &ctx, (cudaStream_t)stream); if (rc) return rc;
    if (lmax_used) for (int l = 0; l < 8 && semb_mg_level_n(ctx, l) >= 0; ++l) lmax_used[l] = ctx.lmax[l];
    return semb_mg_vcycle_run(h, ctx, 0, r, z, nullptr, (cudaStream_t)stream);
}

int semb_mg_transfer(semb_handle h, const semb_pcg_opts* o, int level, int restrict_, const double* in, double* out, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!o || !in || !out || in == out) return semb_fail(h, SEMB_EINVAL, "mg_transfer: bad argument");
    semb_mg_ctx ctx;
    int rc = semb_mg_prepare(h, o, &ctx, (cudaStream_t)stream); if (rc) return rc;
    return semb_mg_transfer_run(h, ctx, level, restrict_, in, out, (cudaStream_t)stream);
}

int64_t semb_mg_level_size(semb_handle h, const semb_pcg_opts* o, int level)
{
    if (!h || !o) return SEMB_EINVAL;
    int nlev = 0, orders[8];
    const int rc = semb_mg_orders(h, o, &nlev, orders); if (rc) return rc;       // validates; builds nothing
    if (level < 0 || level >= nlev) return semb_fail(h, SEMB_EINVAL, "mg_level_size: level %d of %d", level, nlev);
    const int64_t n1 = orders[level] + 1;
    return h->E * n1 * n1 * n1;
}

int semb_schwarz_apply(semb_handle h, double lambda, uint32_t tags, const double* r, double* out, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!r || !out || r == out) return semb_fail(h, SEMB_EINVAL, "schwarz_apply: bad argument");
    return semb_schwarz_apply_run(h, tags, lambda, r, out, (cudaStream_t)stream);
}

int semb_cheb_jacobi(semb_handle h, double lambda, uint32_t tags, int k, double lmax, const double* r, double* z, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!r || !z || r == z) return semb_fail(h, SEMB_EINVAL, "cheb_jacobi: bad argument");
    return semb_cheb_run(h, lambda, tags, k, lmax, r, z, (cudaStream_t)stream);
}

// ---- export --------------------------------------------------------------------------------
static semb_field_entry* find_field(semb_mesh* h, const char* name)
{
    for (auto& f : h->fields) if (f.name == name) return &f;
    return nullptr;
}

int semb_publish_field(semb_handle h, const char* name, double* dev_ptr, int64_t count)
{
    if (!h) return SEMB_EINVAL;
    if (!name || !dev_ptr || count < 1) return semb_fail(h, SEMB_EINVAL, "publish_field: bad argument");
    if (!strcmp(name, "velocity_magnitude")) return semb_fail(h, SEMB_EINVAL, "publish_field: velocity_magnitude is derived");
    semb_field_entry* f = find_field(h, name);
    if (f) { f->ptr = dev_ptr; f->count = count; }
    else {
        if (h->fields.size() + 2 > h->fields.capacity()) return semb_fail(h, SEMB_EINVAL, "publish_field: too many fields");
        semb_field_entry e; e.name = name; e.ptr = dev_ptr; e.count = count; h->fields.push_back(e);
    }
    // the derived field's buffer is allocated here, once, so that publish_state / export_field never allocate
    semb_field_entry *vx = find_field(h, "velocity_x"), *vy = find_field(h, "velocity_y"), *vz = find_field(h, "velocity_z");
    if (vx && vy && vz && vx->count == vy->count && vx->count == vz->count && !find_field(h, "velocity_magnitude")) {
        semb_field_entry e; e.name = "velocity_magnitude"; e.count = vx->count; e.derived = true;
        e.ptr = (double*)semb_dev_alloc(h, sizeof(double) * (size_t)e.count);
        if (!e.ptr) return semb_fail(h, SEMB_ENOMEM, "velocity_magnitude buffer");
        h->fields.push_back(e);
    }
    return SEMB_OK;
}

int semb_publish_state(semb_handle h, int64_t cycle, double time, void* stream)
{
    if (!h) return SEMB_EINVAL;
    h->cycle = cycle; h->time = time;
    semb_field_entry* vm = find_field(h, "velocity_magnitude");
    if (vm && vm->wanted) {           // refreshed only once a consumer has asked for the pointer (pay for nothing unused)
        semb_field_entry *vx = find_field(h, "velocity_x"), *vy = find_field(h, "velocity_y"), *vz = find_field(h, "velocity_z");
        if (semb_vmag_launch(vx->ptr, vy->ptr, vz->ptr, vm->ptr, vm->count, (cudaStream_t)stream))
            return semb_fail(h, SEMB_ECUDA, "velocity_magnitude kernel: %s", cudaGetErrorString(cudaGetLastError()));
    }
    return SEMB_OK;
}

int semb_export_field(semb_handle h, const char* name, semb_field_desc* out)
{
    if (!h || !name || !out) return SEMB_EINVAL;
    semb_field_entry* f = find_field(h, name);
    if (!f) return SEMB_ENOTFOUND;
    if (f->derived && !f->wanted) {
        // first request of a derived field: from now on publish_state refreshes it; the content is current from the NEXT
        // publish_state on (this call itself launches nothing)
        f->wanted = true;
    }
    out->name = f->name.c_str(); out->ptr = f->ptr; out->dtype = SEMB_F64; out->memspace = SEMB_MEM_DEVICE;
    out->count = f->count; out->stride = 1; out->cycle = h->cycle; out->time = h->time;
    return SEMB_OK;
}

int semb_field_minmax_hist(const semb_field_desc* f, int nbins, double lo, double hi, double* minmax_dev,
                           uint64_t* hist_dev, void* stream)
{
    if (!f || !f->ptr || !minmax_dev || !hist_dev) return SEMB_EINVAL;
    if (f->memspace != SEMB_MEM_DEVICE || f->dtype != SEMB_F64) return SEMB_EINVAL;
    return semb_minmax_hist_launch((const double*)f->ptr, nullptr, nullptr, f->count, f->stride, nbins, lo, hi, minmax_dev, hist_dev,
                                   (cudaStream_t)stream);
}

int semb_vector_magnitude_minmax_hist(const semb_field_desc* fx, const semb_field_desc* fy, const semb_field_desc* fz, int nbins,
                                      double lo, double hi, double* minmax_dev, uint64_t* hist_dev, void* stream)
{
    if (!fx || !fy || !fz || !fx->ptr || !fy->ptr || !fz->ptr || !minmax_dev || !hist_dev) return SEMB_EINVAL;
    for (const semb_field_desc* f : {fx, fy, fz})
        if (f->memspace != SEMB_MEM_DEVICE || f->dtype != SEMB_F64 || f->count != fx->count || f->stride != fx->stride) return SEMB_EINVAL;
    return semb_minmax_hist_launch((const double*)fx->ptr, (const double*)fy->ptr, (const double*)fz->ptr, fx->count, fx->stride, nbins,
                                   lo, hi, minmax_dev, hist_dev, (cudaStream_t)stream);
}

int semb_apply_axhelm_host(semb_handle h, double lambda, const double* u_host, double* w_host)
{
    if (!h) return SEMB_EINVAL;
    if (!u_host || !w_host) return semb_fail(h, SEMB_EINVAL, "apply_axhelm_host: bad argument");
    int rc = semb_ensure_work(h, 2); if (rc) return rc;
    const size_t bytes = sizeof(double) * (size_t)h->n;
    SEMB_CUDA(h, cudaMemcpy(h->work, u_host, bytes, cudaMemcpyHostToDevice));
    rc = semb_axhelm_launch(h, lambda, nullptr, nullptr, h->work, h->work + h->n, 1, nullptr, 0); if (rc) return rc;
    SEMB_CUDA(h, cudaMemcpy(w_host, h->work + h->n, bytes, cudaMemcpyDeviceToHost));
    return SEMB_OK;
}

int semb_pcg_solve_host(semb_handle h, const semb_pcg_opts* o, const double* b_host, double* x_host,
                        semb_pcg_stats* st, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!o || !b_host || !x_host) return semb_fail(h, SEMB_EINVAL, "pcg_solve_host: bad argument");
    cudaStream_t s = (cudaStream_t)stream;
    const size_t bytes = sizeof(double) * (size_t)h->n;
    if (!h->stage) {
        h->stage = (double*)semb_dev_alloc(h, 2 * bytes);
        if (!h->stage) return semb_fail(h, SEMB_ENOMEM, "host-call staging buffers");
    }
    double *b = h->stage, *x = h->stage + h->n;
    SEMB_CUDA(h, cudaMemcpyAsync(b, b_host, bytes, cudaMemcpyHostToDevice, s));
    if (!o->x0_is_zero) SEMB_CUDA(h, cudaMemcpyAsync(x, x_host, bytes, cudaMemcpyHostToDevice, s));
    const int rc = semb_pcg_run(h, o, b, x, st, s);
    if (st) st->status = rc;
    if (rc < 0) return rc;
    SEMB_CUDA(h, cudaMemcpyAsync(x_host, x, bytes, cudaMemcpyDeviceToHost, s));
    SEMB_CUDA(h, cudaStreamSynchronize(s));
    return rc;
}

}  // extern "C"
