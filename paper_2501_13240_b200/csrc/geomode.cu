// Geometry representations of the axhelm kernels ("on-the-fly geometric factors ... store 8
// vertices/element for trilinear elements and recompute G", "mixed-precision geo storage").  PAPER.md:L100 §2.2 fixes
// only that deformed elements go through the chain rule; §4: the paper's own Gamma = 4 meshes are
// Cartesian boxes whose element map is stretched vertically -- every element an axis-aligned brick, i.e. AFFINE.
//
// semb_set_geometry_mode measures how far the node coordinates of every element are from the trilinear (and from
// the affine) map of its 8 corner nodes and, when the mesh is in the class the mode needs, builds that mode's data:
//   1  float copy of the stored factors                               (exactly representable widening on load)
//   2  per element (1/J) C_a.C_b (6) and J from the affine map        (64 B per element instead of 48-56 B per node)
//   3  per element the 8 x 3 trilinear coefficients                   (192 B per element)
// The operator is the same one (reading R23): modes 2 and 3 re-evaluate the same factors from the same
// coordinates in another order, so they differ from the stored ones by the conditioning bound of reading R22.
#include <math.h>
#include <string.h>

#include "semb_internal.h"

__device__ __forceinline__ unsigned long long gm_enc(double v)      // v >= 0: the bit pattern is order preserving
{
    return (unsigned long long)__double_as_longlong(v);
}

// One block per element.  tri[e][c][8]: x_c = c0 + c1 r + c2 s + c3 t + c4 rs + c5 rt + c6 st + c7 rst from the 8 corner
// nodes; red[0] = max over nodes and coordinates of |x_c(node) - trilinear map|, red[1] = the same against the affine
// part c0 + c1 r + c2 s + c3 t alone, red[2] = max |coordinate|.
__global__ void __launch_bounds__(128)
k_trilinear_fit(int n1, const double* __restrict__ xyz, int64_t n, const double* __restrict__ xig, double* __restrict__ tri,
                unsigned long long* __restrict__ red)
{
    __shared__ double c[3][8], xi[SEMB_MAXN1], sred[3][4];
    const int Np = n1 * n1 * n1, N = n1 - 1;
    const int64_t e = blockIdx.x;
    if (threadIdx.x < n1) xi[threadIdx.x] = xig[threadIdx.x];
    if (threadIdx.x < 24) {
        const int cc = threadIdx.x / 8, q = threadIdx.x % 8;        // coefficient q of coordinate cc
        double s = 0.0;
        for (int v = 0; v < 8; ++v) {
            const int vi = v & 1, vj = (v >> 1) & 1, vk = v >> 2;
            const double r = vi ? 1.0 : -1.0, sg = vj ? 1.0 : -1.0, t = vk ? 1.0 : -1.0;
            const double wgt[8] = {1.0, r, sg, t, r * sg, r * t, sg * t, r * sg * t};
            s += wgt[q] * xyz[cc * n + e * Np + (vk * N) * n1 * n1 + (vj * N) * n1 + vi * N];
        }
        c[cc][q] = 0.125 * s;
        tri[e * 24 + threadIdx.x] = 0.125 * s;
    }
    __syncthreads();
    double dt = 0.0, da = 0.0, mx = 0.0;
    for (int l = threadIdx.x; l < Np; l += blockDim.x) {
        const int i = l % n1, j = (l / n1) % n1, k = l / (n1 * n1);
        const double r = xi[i], s = xi[j], t = xi[k];
        for (int cc = 0; cc < 3; ++cc) {
            const double X = xyz[cc * n + e * Np + l];
            const double aff = c[cc][0] + c[cc][1] * r + c[cc][2] * s + c[cc][3] * t;
            const double trl = aff + c[cc][4] * r * s + c[cc][5] * r * t + c[cc][6] * s * t + c[cc][7] * r * s * t;
            dt = fmax(dt, fabs(X - trl)); da = fmax(da, fabs(X - aff)); mx = fmax(mx, fabs(X));
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        dt = fmax(dt, __shfl_xor_sync(0xffffffffu, dt, o)); da = fmax(da, __shfl_xor_sync(0xffffffffu, da, o));
        mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if ((threadIdx.x & 31) == 0) { sred[0][threadIdx.x >> 5] = dt; sred[1][threadIdx.x >> 5] = da; sred[2][threadIdx.x >> 5] = mx; }
    __syncthreads();
    if (threadIdx.x < 3) {
        double v = fmax(fmax(sred[threadIdx.x][0], sred[threadIdx.x][1]), fmax(sred[threadIdx.x][2], sred[threadIdx.x][3]));
        atomicMax(&red[threadIdx.x], gm_enc(v));
    }
}

// affine constants from the linear part of the map: x_r = (c1 of x, y, z) etc.; cofactors C_r = x_s x x_t, ...
__global__ void k_affine_constants(int64_t E, const double* __restrict__ tri, double* __restrict__ gc)
{
    const int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e >= E) return;
    const double* c = tri + e * 24;
    const double xr = c[1], xs = c[2], xt = c[3], yr = c[9], ys = c[10], yt = c[11], zr = c[17], zs = c[18], zt = c[19];
    const double rx = ys * zt - yt * zs, ry = zs * xt - zt * xs, rz = xs * yt - xt * ys;
    const double sx = yt * zr - yr * zt, sy = zt * xr - zr * xt, sz = xt * yr - xr * yt;
    const double tx = yr * zs - ys * zr, ty = zr * xs - zs * xr, tz = xr * ys - xs * yr;
    const double J = xr * rx + yr * ry + zr * rz, iJ = 1.0 / J;
    double* g = gc + e * 8;
    g[0] = (rx * rx + ry * ry + rz * rz) * iJ; g[1] = (rx * sx + ry * sy + rz * sz) * iJ; g[2] = (rx * tx + ry * ty + rz * tz) * iJ;
    g[3] = (sx * sx + sy * sy + sz * sz) * iJ; g[4] = (sx * tx + sy * ty + sz * tz) * iJ; g[5] = (tx * tx + ty * ty + tz * tz) * iJ;
    g[6] = J; g[7] = 0.0;
}

__global__ void k_to_float(int64_t n, const double* __restrict__ in, float* __restrict__ out)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) out[l] = (float)in[l];
}

extern "C" int semb_set_geometry_mode(semb_handle h, int mode, double tol, double* dev_out, void* stream)
{
    if (!h) return SEMB_EINVAL;
    if (mode < 0 || mode > 3) return semb_fail(h, SEMB_EINVAL, "set_geometry_mode: mode %d", mode);
    cudaStream_t s = (cudaStream_t)stream;
    if (tol <= 0.0) tol = 16.0 * 2.220446049250313e-16;
    if (mode >= 2 || dev_out) {
        if (!h->xyz) return semb_fail(h, SEMB_EINVAL, "set_geometry_mode: the handle holds no coordinates");
        if (!h->geoT) {
            // the fit: coefficients + measured deviations, once per handle
            double* tri = (double*)semb_dev_alloc(h, sizeof(double) * 24 * (size_t)h->E);
            double* aux = (double*)semb_dev_alloc(h, sizeof(double) * (SEMB_MAXN1 + 4));
            if (!tri || !aux) { semb_dev_free(h, tri); semb_dev_free(h, aux); return semb_fail(h, SEMB_ENOMEM, "set_geometry_mode: coefficients"); }
            unsigned long long* red = (unsigned long long*)(aux + SEMB_MAXN1);
            unsigned long long r3[3] = {0, 0, 0};
            cudaError_t e = cudaMemcpyAsync(aux, h->xi, sizeof(double) * h->n1, cudaMemcpyHostToDevice, s);
            if (e == cudaSuccess) e = cudaMemsetAsync(red, 0, 3 * sizeof(unsigned long long), s);
            if (e == cudaSuccess) {
                k_trilinear_fit<<<(unsigned)h->E, 128, 0, s>>>(h->n1, h->xyz, h->n, aux, tri, red);
                e = cudaGetLastError();
            }
            if (e == cudaSuccess) e = cudaMemcpyAsync(r3, red, sizeof(r3), cudaMemcpyDeviceToHost, s);
            if (e == cudaSuccess) e = cudaStreamSynchronize(s);
            semb_dev_free(h, aux);
            if (e != cudaSuccess) { semb_dev_free(h, tri); return semb_fail(h, SEMB_ECUDA, "set_geometry_mode: %s", cudaGetErrorString(e)); }
            double v[3];
            memcpy(v, r3, sizeof(v));
            const double scale = v[2] > 0.0 ? v[2] : 1.0;
            h->geo_dev[0] = v[0] / scale; h->geo_dev[1] = v[1] / scale;
            h->geoT = tri;
        }
        if (dev_out) { dev_out[0] = h->geo_dev[0]; dev_out[1] = h->geo_dev[1]; }
    }
    if (mode == 3 && !(h->geo_dev[0] <= tol))
        return semb_fail(h, SEMB_EGEOM, "set_geometry_mode: the elements are not trilinear (deviation %.3e of the coordinate scale, tolerance %.3e)", h->geo_dev[0], tol);
    if (mode == 2) {
        if (!(h->geo_dev[1] <= tol))
            return semb_fail(h, SEMB_EGEOM, "set_geometry_mode: the elements are not affine (deviation %.3e of the coordinate scale, tolerance %.3e)", h->geo_dev[1], tol);
        if (!h->geoC) {
            h->geoC = (double*)semb_dev_alloc(h, sizeof(double) * 8 * (size_t)h->E);
            if (!h->geoC) return semb_fail(h, SEMB_ENOMEM, "set_geometry_mode: affine constants");
            k_affine_constants<<<(unsigned)((h->E + 127) / 128), 128, 0, s>>>(h->E, h->geoT, h->geoC);
            SEMB_CUDA(h, cudaGetLastError());
        }
    }
    if (mode == 1 && !h->geoF) {
        const int64_t ng = 7 * h->n;
        h->geoF = (float*)semb_dev_alloc(h, sizeof(float) * (size_t)ng);
        if (!h->geoF) return semb_fail(h, SEMB_ENOMEM, "set_geometry_mode: float factors");
        int64_t b = (ng + 1023) / 1024; if (b > semb_sm_count() * 8) b = semb_sm_count() * 8;
        k_to_float<<<(unsigned)b, 256, 0, s>>>(ng, h->geo, h->geoF);
        SEMB_CUDA(h, cudaGetLastError());
    }
    h->geo_mode = mode;
    return SEMB_OK;
}
