// The rest of a Boussinesq time step around the Poisson / Helmholtz solves (Eqs. (1)-(3):
//   du/dt + u.grad u = -grad p + T z^ + sqrt(Pr/Ra) lap u,   dT/dt + u.grad T = lap T / sqrt(Ra Pr),   div u = 0,
// PAPER.md:L238 no-slip isothermal plates, L272 start from u = 0, T = 1 - z).  The paper states the equations, not the time
// discretisation; reading R25 fixes it: BDF2 / EXT2 (order 1 on the first step), collocation advection and
// buoyancy, a pressure Poisson equation in weak form whose right-hand side carries the extrapolated curl-curl of the velocity
// (so that the natural boundary condition is the consistent one and the step is second order), all-Neumann pressure with the
// mean projection of reading R20, then one Helmholtz solve per velocity component and one for theta = T - (1 - z).
//
// Kernels here: the collocation gradient (one block per element, the element's fields and D in shared memory), the fused
// explicit-terms kernel (4 gradients -> advection, buoyancy, vorticity), curl, weak divergence (transpose of the gradient in
// the GLL inner product) and the streaming combinations; the solves are semb_pcg_run of pcg.cu.
#include <math.h>

#include "semb_internal.h"

// dr_a/dx_b (a = r,s,t rows; b = x,y,z) at index 3a + b: met[E][9][Np], the inverse of the Jacobian d(x,y,z)/d(r,s,t)
__global__ void k_flow_metrics(int n1, int64_t n, const double* __restrict__ xyz, const double* __restrict__ Dg, double* __restrict__ met)
{
    extern __shared__ double sm[];
    const int Np = n1 * n1 * n1;
    double* sD = sm; double* sx = sD + n1 * n1; double* sy = sx + Np; double* sz = sy + Np;
    const int64_t e = blockIdx.x;
    for (int t = threadIdx.x; t < n1 * n1; t += blockDim.x) sD[t] = Dg[t];
    for (int t = threadIdx.x; t < Np; t += blockDim.x) { sx[t] = xyz[e * Np + t]; sy[t] = xyz[n + e * Np + t]; sz[t] = xyz[2 * n + e * Np + t]; }
    __syncthreads();
    double* m = met + e * 9 * (int64_t)Np;
    for (int l = threadIdx.x; l < Np; l += blockDim.x) {
        const int i = l % n1, j = (l / n1) % n1, k = l / (n1 * n1);
        double xr = 0, xs = 0, xt = 0, yr = 0, ys = 0, yt = 0, zr = 0, zs = 0, zt = 0;
        for (int q = 0; q < n1; ++q) {
            const int ir = k * n1 * n1 + j * n1 + q, is = k * n1 * n1 + q * n1 + i, it = q * n1 * n1 + j * n1 + i;
            const double dr = sD[i * n1 + q], ds = sD[j * n1 + q], dt = sD[k * n1 + q];
            xr += dr * sx[ir]; xs += ds * sx[is]; xt += dt * sx[it];
            yr += dr * sy[ir]; ys += ds * sy[is]; yt += dt * sy[it];
            zr += dr * sz[ir]; zs += ds * sz[is]; zt += dt * sz[it];
        }
        const double J = xr * (ys * zt - yt * zs) - xs * (yr * zt - yt * zr) + xt * (yr * zs - ys * zr), iJ = 1.0 / J;
        m[0 * Np + l] = (ys * zt - yt * zs) * iJ;  m[1 * Np + l] = -(xs * zt - xt * zs) * iJ; m[2 * Np + l] = (xs * yt - xt * ys) * iJ;
        m[3 * Np + l] = -(yr * zt - yt * zr) * iJ; m[4 * Np + l] = (xr * zt - xt * zr) * iJ;  m[5 * Np + l] = -(xr * yt - xt * yr) * iJ;
        m[6 * Np + l] = (yr * zs - ys * zr) * iJ;  m[7 * Np + l] = -(xr * zs - xs * zr) * iJ; m[8 * Np + l] = (xr * ys - xs * yr) * iJ;
    }
}

// reference derivatives of one field held in shared memory S[Np] at node (i, j, k)
__device__ __forceinline__ void flow_dref(int n1, const double* __restrict__ sD, const double* __restrict__ S, int i, int j, int k,
                                          double& pr, double& ps, double& pt)
{
    pr = 0.0; ps = 0.0; pt = 0.0;
    for (int q = 0; q < n1; ++q) {
        pr += sD[i * n1 + q] * S[k * n1 * n1 + j * n1 + q];
        ps += sD[j * n1 + q] * S[k * n1 * n1 + q * n1 + i];
        pt += sD[k * n1 + q] * S[q * n1 * n1 + j * n1 + i];
    }
}

#define FLOW_PHYS(m, Np, l, pr, ps, pt, gx, gy, gz)                                             \
    gx = m[0 * Np + l] * pr + m[3 * Np + l] * ps + m[6 * Np + l] * pt;                          \
    gy = m[1 * Np + l] * pr + m[4 * Np + l] * ps + m[7 * Np + l] * pt;                          \
    gz = m[2 * Np + l] * pr + m[5 * Np + l] * ps + m[8 * Np + l] * pt

// NF fields at once (in[f], f < NF); MODEK 0: gradients out[3f + b]; MODEK 1 (NF = 3): curl, out[0..2]
template <int NF, int MODEK>
__global__ void __launch_bounds__(128)
k_flow_grad(int n1, const double* __restrict__ met, const double* __restrict__ Dg, const double* const* __restrict__ in,
            double* const* __restrict__ out)
{
    extern __shared__ double sm[];
    const int Np = n1 * n1 * n1;
    double* sD = sm; double* S = sD + n1 * n1;
    const int64_t e = blockIdx.x;
    for (int t = threadIdx.x; t < n1 * n1; t += blockDim.x) sD[t] = Dg[t];
    for (int f = 0; f < NF; ++f)
        for (int t = threadIdx.x; t < Np; t += blockDim.x) S[f * Np + t] = in[f][e * Np + t];
    __syncthreads();
    const double* m = met + e * 9 * (int64_t)Np;
    for (int l = threadIdx.x; l < Np; l += blockDim.x) {
        const int i = l % n1, j = (l / n1) % n1, k = l / (n1 * n1);
        double g[NF][3];
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            double pr, ps, pt;
            flow_dref(n1, sD, S + f * Np, i, j, k, pr, ps, pt);
            FLOW_PHYS(m, Np, l, pr, ps, pt, g[f][0], g[f][1], g[f][2]);
        }
        if (MODEK == 0) {
#pragma unroll
            for (int f = 0; f < NF; ++f) { out[3 * f][e * Np + l] = g[f][0]; out[3 * f + 1][e * Np + l] = g[f][1]; out[3 * f + 2][e * Np + l] = g[f][2]; }
        } else {
            out[0][e * Np + l] = g[NF - 1][1] - g[1][2];
            out[1][e * Np + l] = g[0][2] - g[NF - 1][0];
            out[2][e * Np + l] = g[1][0] - g[0][1];
        }
    }
}

// explicit terms of step (i): in = ux, uy, uz, theta; out = N_x, N_y, N_z, N_theta, omega_x, omega_y, omega_z (premultiplied by
// the mass factor B when bw != NULL, ready for the mass-weighted average); z = node heights; f = optional forcing [4]
__global__ void __launch_bounds__(128)
k_flow_explicit(int n1, int64_t n, const double* __restrict__ met, const double* __restrict__ Dg, const double* __restrict__ zc,
                const double* __restrict__ geo, const double* const* __restrict__ in, const double* const* __restrict__ f,
                double* const* __restrict__ out)
{
    extern __shared__ double sm[];
    const int Np = n1 * n1 * n1;
    double* sD = sm; double* S = sD + n1 * n1;
    const int64_t e = blockIdx.x;
    for (int t = threadIdx.x; t < n1 * n1; t += blockDim.x) sD[t] = Dg[t];
    for (int c = 0; c < 4; ++c)
        for (int t = threadIdx.x; t < Np; t += blockDim.x) S[c * Np + t] = in[c][e * Np + t];
    __syncthreads();
    const double* m = met + e * 9 * (int64_t)Np;
    const double* B = geo + e * 7 * (int64_t)Np + 6 * (int64_t)Np;
    for (int l = threadIdx.x; l < Np; l += blockDim.x) {
        const int i = l % n1, j = (l / n1) % n1, k = l / (n1 * n1);
        double g[4][3];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            double pr, ps, pt;
            flow_dref(n1, sD, S + c * Np, i, j, k, pr, ps, pt);
            FLOW_PHYS(m, Np, l, pr, ps, pt, g[c][0], g[c][1], g[c][2]);
        }
        const double ux = S[l], uy = S[Np + l], uz = S[2 * Np + l], th = S[3 * Np + l];
        const int64_t gl = e * Np + l;
        const double T = th + (1.0 - zc[gl]);
        double N[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) N[c] = -(ux * g[c][0] + uy * g[c][1] + uz * g[c][2]);
        N[2] += T; N[3] += uz;
        if (f) {
#pragma unroll
            for (int c = 0; c < 4; ++c) if (f[c]) N[c] += f[c][gl];
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) out[c][gl] = N[c];
        const double b = B[l];
        out[4][gl] = b * (g[2][1] - g[1][2]);
        out[5][gl] = b * (g[0][2] - g[2][0]);
        out[6][gl] = b * (g[1][0] - g[0][1]);
    }
}

// out_i = sum_a sum_m D_mi [B (dr_a/dx . g)](m, ..): the transpose of the collocation gradient in the GLL inner product
__global__ void __launch_bounds__(128)
k_flow_wdiv(int n1, const double* __restrict__ met, const double* __restrict__ geo, const double* __restrict__ Dg,
            const double* __restrict__ gx, const double* __restrict__ gy, const double* __restrict__ gz, double* __restrict__ out)
{
    extern __shared__ double sm[];
    const int Np = n1 * n1 * n1;
    double* sD = sm; double* fr = sD + n1 * n1; double* fs = fr + Np; double* ft = fs + Np;
    const int64_t e = blockIdx.x;
    for (int t = threadIdx.x; t < n1 * n1; t += blockDim.x) sD[t] = Dg[t];
    const double* m = met + e * 9 * (int64_t)Np;
    const double* B = geo + e * 7 * (int64_t)Np + 6 * (int64_t)Np;
    for (int l = threadIdx.x; l < Np; l += blockDim.x) {
        const double a = gx[e * Np + l], b = gy[e * Np + l], c = gz[e * Np + l], w = B[l];
        fr[l] = w * (m[0 * Np + l] * a + m[1 * Np + l] * b + m[2 * Np + l] * c);
        fs[l] = w * (m[3 * Np + l] * a + m[4 * Np + l] * b + m[5 * Np + l] * c);
        ft[l] = w * (m[6 * Np + l] * a + m[7 * Np + l] * b + m[8 * Np + l] * c);
    }
    __syncthreads();
    for (int l = threadIdx.x; l < Np; l += blockDim.x) {
        const int i = l % n1, j = (l / n1) % n1, k = l / (n1 * n1);
        double s = 0.0;
        for (int q = 0; q < n1; ++q)
            s += sD[q * n1 + i] * fr[k * n1 * n1 + j * n1 + q] + sD[q * n1 + j] * fs[k * n1 * n1 + q * n1 + i] + sD[q * n1 + k] * ft[q * n1 * n1 + j * n1 + i];
        out[e * Np + l] = s;
    }
}

// ---- streaming combinations of the step ------------------------------------------------------------------------
struct flow_coef { double b0, b1, a0, a1, dt, nu; };

// v = v / w  (mass-weighted average after QQ^T: w = QQ^T B)
__global__ void k_flow_divide(int64_t n, int nf, double* __restrict__ v, const double* __restrict__ w)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n * nf; l += (int64_t)gridDim.x * blockDim.x) v[l] /= w[l % n];
}

// u~ = b0 u + b1 u1 + dt (a0 N + a1 N1);  g = u~ / dt - nu (a0 C + a1 C1);  histories: u1 <- u, N1 <- N, C1 <- C
__global__ void k_flow_tilde(int64_t n, flow_coef k, const double* __restrict__ u, double* __restrict__ u1, const double* __restrict__ N,
                             double* __restrict__ N1, const double* __restrict__ C, double* __restrict__ C1, double* __restrict__ ut,
                             double* __restrict__ g)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const double uu = u[l], nn = N[l], cc = C[l];
        const double t = k.b0 * uu + k.b1 * u1[l] + k.dt * (k.a0 * nn + k.a1 * N1[l]);
        ut[l] = t;
        g[l] = t / k.dt - k.nu * (k.a0 * cc + k.a1 * C1[l]);
        u1[l] = uu; N1[l] = nn; C1[l] = cc;
    }
}
// rhs = B (u~ - dt dp) / (nu dt)       (dp == NULL: the theta equation, rhs = B theta~ / (kappa dt) with nu := kappa)
__global__ void k_flow_rhs(int64_t n, int64_t Np, const double* __restrict__ geo, double dt, double nu, const double* __restrict__ ut,
                           const double* __restrict__ dp, double* __restrict__ rhs)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e = l / Np;
        const double B = geo[e * 7 * Np + 6 * Np + (l - e * Np)];
        const double v = dp ? ut[l] - dt * dp[l] : ut[l];
        rhs[l] = B * (v / (nu * dt));
    }
}
// theta~ = b0 th + b1 th1 + dt (a0 N + a1 N1);  histories th1 <- th, N1 <- N
__global__ void k_flow_tilde_theta(int64_t n, flow_coef k, const double* __restrict__ th, double* __restrict__ th1, const double* __restrict__ N,
                                   double* __restrict__ N1, double* __restrict__ tt)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const double a = th[l], nn = N[l];
        tt[l] = k.b0 * a + k.b1 * th1[l] + k.dt * (k.a0 * nn + k.a1 * N1[l]);
        th1[l] = a; N1[l] = nn;
    }
}

// ---- host side -----------------------------------------------------------------------------------------------
static unsigned flow_grid(int64_t n) { int64_t b = (n + 1023) / 1024, cap = (int64_t)semb_sm_count() * 8; return (unsigned)(b < 1 ? 1 : (b > cap ? cap : b)); }

// metrics, the basis on the device, pointer tables and work vectors: built on first use, owned by the handle
int semb_flow_prepare(semb_mesh* h, cudaStream_t s)
{
    if (h->flow_met) return SEMB_OK;
    if (!h->xyz) return semb_fail(h, SEMB_EINVAL, "flow: the handle holds no coordinates");
    const int n1 = h->n1; const int64_t Np = h->Np;
    double* met = (double*)semb_dev_alloc(h, sizeof(double) * 9 * (size_t)h->n);
    double* D = (double*)semb_dev_alloc(h, sizeof(double) * n1 * n1);
    double* work = (double*)semb_dev_alloc(h, sizeof(double) * SEMB_FLOW_WORK * (size_t)h->n);
    const double** tab = (const double**)semb_dev_alloc(h, sizeof(double*) * 16 * 8);
    if (!met || !D || !work || !tab) {
        semb_dev_free(h, met); semb_dev_free(h, D); semb_dev_free(h, work); semb_dev_free(h, (void*)tab);
        return semb_fail(h, SEMB_ENOMEM, "flow: metrics and work vectors (%zu bytes)", sizeof(double) * (9 + SEMB_FLOW_WORK) * (size_t)h->n);
    }
    cudaError_t e = cudaMemcpyAsync(D, h->D, sizeof(double) * n1 * n1, cudaMemcpyHostToDevice, s);
    const size_t smem = sizeof(double) * (n1 * n1 + 3 * Np);
    if (e == cudaSuccess) {
        k_flow_metrics<<<(unsigned)h->E, 128, smem, s>>>(n1, h->n, h->xyz, D, met);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) {
        semb_dev_free(h, met); semb_dev_free(h, D); semb_dev_free(h, work); semb_dev_free(h, (void*)tab);
        return semb_fail(h, SEMB_ECUDA, "flow: metrics: %s", cudaGetErrorString(e));
    }
    h->flow_met = met; h->flow_D = D; h->flow_work = work; h->flow_tab = tab;
    return SEMB_OK;
}

// uploads a small table of device pointers into slot `slot` (16 entries each) of the handle's pointer table
static const double** flow_table(semb_mesh* h, int slot, const double* const* p, int count, cudaStream_t s)
{
    const double** dst = h->flow_tab + 16 * slot;
    cudaMemcpyAsync((void*)dst, p, sizeof(double*) * count, cudaMemcpyHostToDevice, s);
    return dst;
}

int semb_flow_gradient_run(semb_mesh* h, const double* phi, double* gx, double* gy, double* gz, cudaStream_t s)
{
    int rc = semb_flow_prepare(h, s); if (rc) return rc;
    const double* in[1] = {phi}; const double* out[3] = {gx, gy, gz};
    const double** din = flow_table(h, 0, in, 1, s); const double** dout = flow_table(h, 1, out, 3, s);
    k_flow_grad<1, 0><<<(unsigned)h->E, 128, sizeof(double) * (h->n1 * h->n1 + h->Np), s>>>(h->n1, h->flow_met, h->flow_D, din, (double* const*)dout);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

int semb_flow_curl_run(semb_mesh* h, const double* vx, const double* vy, const double* vz, double* cx, double* cy, double* cz, cudaStream_t s)
{
    int rc = semb_flow_prepare(h, s); if (rc) return rc;
    const double* in[3] = {vx, vy, vz}; const double* out[3] = {cx, cy, cz};
    const double** din = flow_table(h, 2, in, 3, s); const double** dout = flow_table(h, 3, out, 3, s);
    k_flow_grad<3, 1><<<(unsigned)h->E, 128, sizeof(double) * (h->n1 * h->n1 + 3 * h->Np), s>>>(h->n1, h->flow_met, h->flow_D, din, (double* const*)dout);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

int semb_flow_wdiv_run(semb_mesh* h, const double* gx, const double* gy, const double* gz, double* out, cudaStream_t s)
{
    int rc = semb_flow_prepare(h, s); if (rc) return rc;
    k_flow_wdiv<<<(unsigned)h->E, 128, sizeof(double) * (h->n1 * h->n1 + 3 * h->Np), s>>>(h->n1, h->flow_met, h->geo, h->flow_D, gx, gy, gz, out);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

// N [4][n] and B-weighted vorticity [3][n] into out7 ([7][n] contiguous)
static int flow_explicit_run(semb_mesh* h, const double* ux, const double* uy, const double* uz, const double* th, const double* const* f,
                             double* out7, cudaStream_t s)
{
    const double* in[4] = {ux, uy, uz, th};
    const double* out[7]; for (int c = 0; c < 7; ++c) out[c] = out7 + c * h->n;
    const double** din = flow_table(h, 4, in, 4, s); const double** dout = flow_table(h, 5, out, 7, s);
    const double** df = nullptr;
    if (f && (f[0] || f[1] || f[2] || f[3])) df = flow_table(h, 6, f, 4, s);
    const size_t smem = sizeof(double) * (h->n1 * h->n1 + 4 * h->Np);
    static bool attr = false;
    if (!attr) { cudaFuncSetAttribute(k_flow_explicit, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024); attr = true; }
    k_flow_explicit<<<(unsigned)h->E, 128, smem, s>>>(h->n1, h->n, h->flow_met, h->flow_D, h->xyz + 2 * h->n, h->geo, din, df, (double* const*)dout);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

extern "C" int semb_gradient(semb_handle h, const double* phi, double* gx, double* gy, double* gz, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!phi || !gx || !gy || !gz) return semb_fail(h, SEMB_EINVAL, "gradient: bad argument");
    return semb_flow_gradient_run(h, phi, gx, gy, gz, (cudaStream_t)stream);
}

extern "C" int semb_weak_divergence(semb_handle h, const double* gx, const double* gy, const double* gz, double* out, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!gx || !gy || !gz || !out || out == gx || out == gy || out == gz) return semb_fail(h, SEMB_EINVAL, "weak_divergence: bad argument");
    return semb_flow_wdiv_run(h, gx, gy, gz, out, (cudaStream_t)stream);
}

extern "C" int semb_flow_explicit_terms(semb_handle h, const double* ux, const double* uy, const double* uz, const double* theta,
                                        const double* const* forcing_or_null, double* N4, double* omega3, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!ux || !uy || !uz || !theta || !N4 || !omega3) return semb_fail(h, SEMB_EINVAL, "flow_explicit_terms: bad argument");
    cudaStream_t s = (cudaStream_t)stream;
    int rc = semb_flow_prepare(h, s); if (rc) return rc;
    double* w = h->flow_work;                                   // [7][n]
    rc = flow_explicit_run(h, ux, uy, uz, theta, forcing_or_null, w, s); if (rc) return rc;
    SEMB_CUDA(h, cudaMemcpyAsync(N4, w, sizeof(double) * 4 * (size_t)h->n, cudaMemcpyDeviceToDevice, s));
    // the averaged vorticity of step (i): QQ^T (B omega) / QQ^T B
    double* dA; rc = semb_get_dinv(h, 0.0, 0, &dA, s); if (rc) return rc;      // makes sure diagB = QQ^T B exists
    rc = semb_gs_launch(h, w + 4 * h->n, 3, s); if (rc) return rc;
    k_flow_divide<<<flow_grid(3 * h->n), 256, 0, s>>>(h->n, 3, w + 4 * h->n, h->diagB);
    SEMB_CUDA(h, cudaMemcpyAsync(omega3, w + 4 * h->n, sizeof(double) * 3 * (size_t)h->n, cudaMemcpyDeviceToDevice, s));
    return SEMB_OK;
}

extern "C" int semb_boussinesq_step(semb_handle h, const semb_flow_opts* o, semb_flow_state* st, semb_flow_stats* stats, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (!o || !st) return semb_fail(h, SEMB_EINVAL, "boussinesq_step: bad argument");
    if (!(o->Ra > 0.0) || !(o->Pr > 0.0) || !(o->dt > 0.0)) return semb_fail(h, SEMB_EINVAL, "boussinesq_step: Ra, Pr, dt must be positive");
    double* const must[] = {st->u[0], st->u[1], st->u[2], st->theta, st->p, st->u1[0], st->u1[1], st->u1[2], st->theta1,
                            st->N1[0], st->N1[1], st->N1[2], st->N1[3], st->C1[0], st->C1[1], st->C1[2]};
    for (double* q : must) if (!q) return semb_fail(h, SEMB_EINVAL, "boussinesq_step: the state holds a NULL array");
    cudaStream_t s = (cudaStream_t)stream;
    int rc = semb_flow_prepare(h, s); if (rc) return rc;
    const int64_t n = h->n;
    const double nu = sqrt(o->Pr / o->Ra), ka = 1.0 / sqrt(o->Ra * o->Pr), dt = o->dt;
    const bool first = st->step_index == 0;
    const flow_coef kc = first ? flow_coef{1.0, 0.0, 1.0, 0.0, dt, nu} : flow_coef{2.0, -0.5, 2.0, -1.0, dt, nu};
    const double beta0 = first ? 1.0 : 1.5;
    double* w = h->flow_work;                                   // [SEMB_FLOW_WORK][n]
    double *Nn = w, *om = w + 4 * n, *Cc = w + 7 * n, *ut = w + 10 * n, *g = w + 13 * n, *bp = w + 16 * n, *gp = w + 17 * n, *rhs = w + 20 * n;
    // (i) explicit terms, averaged vorticity, its curl
    rc = flow_explicit_run(h, st->u[0], st->u[1], st->u[2], st->theta, o->forcing, Nn, s); if (rc) return rc;
    double* dA; rc = semb_get_dinv(h, 0.0, 0, &dA, s); if (rc) return rc;      // diagB = QQ^T B
    rc = semb_gs_launch(h, om, 3, s); if (rc) return rc;
    k_flow_divide<<<flow_grid(3 * n), 256, 0, s>>>(n, 3, om, h->diagB);
    rc = semb_flow_curl_run(h, om, om + n, om + 2 * n, Cc, Cc + n, Cc + 2 * n, s); if (rc) return rc;
    // (ii) u~, g, pressure right-hand side and solve
    for (int c = 0; c < 3; ++c)
        k_flow_tilde<<<flow_grid(n), 256, 0, s>>>(n, kc, st->u[c], st->u1[c], Nn + c * n, st->N1[c], Cc + c * n, st->C1[c], ut + c * n, g + c * n);
    rc = semb_flow_wdiv_run(h, g, g + n, g + 2 * n, bp, s); if (rc) return rc;
    rc = semb_gs_launch(h, bp, 1, s); if (rc) return rc;
    h->launches += 5;
    semb_pcg_opts po{};
    po.lambda = 0.0; po.dirichlet_tags = 0; po.precond = o->precond_p ? o->precond_p : 3; po.cheb_degree = 2; po.rtol = o->rtol > 0.0 ? o->rtol : 1e-10;
    po.maxit = o->maxit > 0 ? o->maxit : 20000; po.x0_is_zero = 0; /* started from p^n (zero on the first step) */ po.null_mean = 1; po.mg_fp32 = o->mg_fp32; po.mg_schwarz = o->mg_schwarz; po.mg_smoother_kind = o->mg_schwarz ? 4 : 1;
    semb_pcg_stats ps{};
    rc = semb_pcg_run(h, &po, bp, st->p, &ps, s);
    if (stats) { stats->iters[0] = ps.iters; stats->status[0] = rc; }
    if (rc < 0) return rc;
    int worst = rc;
    // (iii) velocity and temperature
    rc = semb_flow_gradient_run(h, st->p, gp, gp + n, gp + 2 * n, s); if (rc) return rc;
    semb_mask_entry mu, mt;
    rc = semb_get_mask(h, o->tags_u, &mu, s); if (rc) return rc;
    rc = semb_get_mask(h, o->tags_T, &mt, s); if (rc) return rc;
    semb_pcg_opts ho{};
    ho.precond = o->precond_u ? o->precond_u : 1; ho.cheb_degree = 2; ho.rtol = po.rtol; ho.maxit = po.maxit; ho.x0_is_zero = 0; ho.mg_fp32 = o->mg_fp32; ho.mg_schwarz = o->mg_schwarz; ho.mg_smoother_kind = o->mg_schwarz ? 4 : 1;
    for (int c = 0; c < 3; ++c) {
        k_flow_rhs<<<flow_grid(n), 256, 0, s>>>(n, h->Np, h->geo, dt, nu, ut + c * n, gp + c * n, rhs);
        rc = semb_gs_launch(h, rhs, 1, s); if (rc) return rc;
        rc = semb_mask_launch(h, mu, rhs, 1, s); if (rc) return rc;
        ho.lambda = beta0 / (nu * dt); ho.dirichlet_tags = o->tags_u;
        rc = semb_pcg_run(h, &ho, rhs, st->u[c], &ps, s);
        if (stats) { stats->iters[1 + c] = ps.iters; stats->status[1 + c] = rc; }
        if (rc < 0) return rc;
        if (rc > worst) worst = rc;
    }
    k_flow_tilde_theta<<<flow_grid(n), 256, 0, s>>>(n, kc, st->theta, st->theta1, Nn + 3 * n, st->N1[3], ut);
    k_flow_rhs<<<flow_grid(n), 256, 0, s>>>(n, h->Np, h->geo, dt, ka, ut, nullptr, rhs);
    rc = semb_gs_launch(h, rhs, 1, s); if (rc) return rc;
    rc = semb_mask_launch(h, mt, rhs, 1, s); if (rc) return rc;
    ho.lambda = beta0 / (ka * dt); ho.dirichlet_tags = o->tags_T;
    rc = semb_pcg_run(h, &ho, rhs, st->theta, &ps, s);
    if (stats) { stats->iters[4] = ps.iters; stats->status[4] = rc; }
    if (rc < 0) return rc;
    if (rc > worst) worst = rc;
    h->launches += 6;
    st->step_index += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return worst;
}
