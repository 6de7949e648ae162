// Overlapping Schwarz smoother of the p-multigrid levels (§2.2: "p-multigrid that uses
// 4th-kind Chebyshev-acceleration of overlapping Schwarz smoothers"; the paper gives no formulas, reading R26).
//
// Subdomain = the closure of one element (its (N+1)^3 nodes; neighbours overlap in their shared faces).  Subdomain operator =
// the separable approximation  B_t x B_s x A_r + B_t x A_s x B_r + A_t x B_s x B_r + lambda B_t x B_s x B_r  of the assembled
// operator restricted to the element's nodes, built per direction from a 1-D GLL element of the element's mean edge length
// plus the end entries of the neighbour across each face (whose length arrives through one gather-scatter of the interior
// face nodes); Dirichlet faces drop their end node.  It is inverted by fast diagonalisation,
//     A~^-1 = (S_t x S_s x S_r) [Lam_r (+) Lam_s (+) Lam_t + lambda]^-1 (S_t x S_s x S_r)^T,   A_d S_d = B_d S_d Lam_d,
// with the small symmetric eigenproblems solved on the device at setup by cyclic Jacobi rotations (one thread each).
//     S r = M QQ^T [ w o A~^-1 (w o r) ],  w = sqrt(1 / multiplicity)
// is symmetric positive semi-definite; the level smoother is the fourth-kind Chebyshev polynomial in S A.
#include <math.h>

#include <vector>

#include "axhelm_kernels.cuh"      // ax_tile<n1>: the conflict-free shared-memory layouts of the element tile
#include "semb_internal.h"

#ifndef SEMB_SZ_LINE
#define SEMB_SZ_LINE 1
#endif

struct semb_schwarz {             // per (level mesh, Dirichlet tag set); owned by the level mesh
    uint32_t tags = 0;
    double* S = nullptr;          // [E][3][n1][n1]  S_d[node][mode]
    double* lam = nullptr;        // [E][3][n1]
    double* w = nullptr;          // [n] sqrt(invmult)
    float* Sf = nullptr; float* lamf = nullptr; float* wf = nullptr;     // float copies for the FP32-storage levels
    std::vector<std::pair<double, double>> lmax;                          // (lambda, estimated lambda_max(S A))
};

// ---- setup ---------------------------------------------------------------------------------------------------
// len[e][3]: mean straight length of the four edges in direction r, s, t;  F: that length on the interior nodes of the faces
__global__ void k_sz_lengths(int n1, int64_t n, const double* __restrict__ xyz, double* __restrict__ len, double* __restrict__ F)
{
    const int64_t e = blockIdx.x;
    const int N = n1 - 1, Np = n1 * n1 * n1;
    __shared__ double l[3];
    if (threadIdx.x < 3) {
        const int d = threadIdx.x;
        double s = 0.0;
        for (int a = 0; a <= N; a += N) for (int b = 0; b <= N; b += N) {
            int lo, hi;
            if (d == 0) { lo = a * n1 * n1 + b * n1; hi = lo + N; }
            else if (d == 1) { lo = a * n1 * n1 + b; hi = lo + N * n1; }
            else { lo = a * n1 + b; hi = lo + N * n1 * n1; }
            double q = 0.0;
            for (int c = 0; c < 3; ++c) { const double v = xyz[c * n + e * Np + hi] - xyz[c * n + e * Np + lo]; q += v * v; }
            s += sqrt(q);
        }
        l[d] = 0.25 * s;
        len[e * 3 + d] = 0.25 * s;
    }
    __syncthreads();
    for (int t = threadIdx.x; t < Np; t += blockDim.x) {
        const int i = t % n1, j = (t / n1) % n1, k = t / (n1 * n1);
        const bool ii = i > 0 && i < N, jj = j > 0 && j < N, kk = k > 0 && k < N;
        double v = 0.0;
        if ((i == 0 || i == N) && jj && kk) v = l[0];
        else if ((j == 0 || j == N) && ii && kk) v = l[1];
        else if ((k == 0 || k == N) && ii && jj) v = l[2];
        F[e * Np + t] = v;
    }
}

// One thread per (element, direction): the 1-D generalised eigenproblem A S = B S Lam, S^T B S = I, by cyclic Jacobi on
// B^-1/2 A B^-1/2 restricted to the free nodes.  Kh = D^T diag(rho) D (row-major n1 x n1), rho: GLL weights.
__global__ void k_sz_eigen(int64_t E, int n1, const double* __restrict__ Kh, const double* __restrict__ rho, const double* __restrict__ len,
                           const double* __restrict__ Fs, const double* __restrict__ invmult, const int32_t* __restrict__ face_tag, uint32_t tags,
                           double* __restrict__ Sout, double* __restrict__ lamout)
{
    const int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (q >= E * 3) return;
    const int64_t e = q / 3; const int d = (int)(q % 3);
    const int N = n1 - 1, Np = n1 * n1 * n1;
    double A[SEMB_MAXN1 * SEMB_MAXN1], V[SEMB_MAXN1 * SEMB_MAXN1], B[SEMB_MAXN1];
    int idx[SEMB_MAXN1];
    const double l = len[e * 3 + d];
    for (int a = 0; a < n1; ++a) { B[a] = 0.5 * l * rho[a]; for (int b = 0; b < n1; ++b) A[a * n1 + b] = (2.0 / l) * Kh[a * n1 + b]; }
    bool freeN[2] = {true, true};
    for (int side = 0; side < 2; ++side) {
        const int f = 2 * d + side, node = side ? N : 0;
        const int pi_ = (d == 0) ? (1 * n1 * n1 + 1 * n1 + node) : (d == 1) ? (1 * n1 * n1 + node * n1 + 1) : (node * n1 * n1 + 1 * n1 + 1);
        const int32_t tag = face_tag[e * 6 + f];
        if (tag > 0 && tag < 32 && ((tags >> tag) & 1u)) freeN[side] = false;
        else if (invmult[e * Np + pi_] < 0.75) {                       // two copies: an interior face
            const double ln = Fs[e * Np + pi_] - l;
            A[node * n1 + node] += (2.0 / ln) * Kh[N * n1 + N];
            B[node] += 0.5 * ln * rho[N];
        }
    }
    int nf = 0;
    for (int a = 0; a < n1; ++a) if ((a > 0 || freeN[0]) && (a < N || freeN[1])) idx[nf++] = a;
    // C = B^-1/2 A B^-1/2 on the free nodes (stored in A's top-left nf x nf with stride n1), V = I
    for (int a = 0; a < nf; ++a) for (int b = 0; b < nf; ++b) V[a * n1 + b] = (a == b) ? 1.0 : 0.0;
    for (int a = 0; a < nf; ++a) for (int b = 0; b < nf; ++b) {
        const double v = A[idx[a] * n1 + idx[b]] / sqrt(B[idx[a]] * B[idx[b]]);
        A[a * n1 + b] = v;                                             // idx is ascending with idx[a] >= a: entries are read before they are overwritten
    }
    for (int sweep = 0; sweep < 30; ++sweep) {
        double off = 0.0, dg = 0.0;
        for (int a = 0; a < nf; ++a) { dg += A[a * n1 + a] * A[a * n1 + a]; for (int b = a + 1; b < nf; ++b) off += A[a * n1 + b] * A[a * n1 + b]; }
        if (off <= 1e-30 * dg) break;
        for (int p = 0; p < nf - 1; ++p) for (int r = p + 1; r < nf; ++r) {
            const double apr = A[p * n1 + r];
            if (apr == 0.0) continue;
            const double theta = (A[r * n1 + r] - A[p * n1 + p]) / (2.0 * apr);
            const double t = (theta >= 0.0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
            const double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
            for (int k = 0; k < nf; ++k) {                              // columns p, r
                const double akp = A[k * n1 + p], akr = A[k * n1 + r];
                A[k * n1 + p] = c * akp - s * akr; A[k * n1 + r] = s * akp + c * akr;
            }
            for (int k = 0; k < nf; ++k) {                              // rows p, r
                const double apk = A[p * n1 + k], ark = A[r * n1 + k];
                A[p * n1 + k] = c * apk - s * ark; A[r * n1 + k] = s * apk + c * ark;
            }
            for (int k = 0; k < nf; ++k) {
                const double vkp = V[k * n1 + p], vkr = V[k * n1 + r];
                V[k * n1 + p] = c * vkp - s * vkr; V[k * n1 + r] = s * vkp + c * vkr;
            }
        }
    }
    double* So = Sout + (e * 3 + d) * (int64_t)(n1 * n1); double* lo = lamout + (e * 3 + d) * (int64_t)n1;
    for (int a = 0; a < n1 * n1; ++a) So[a] = 0.0;
    for (int m = 0; m < n1; ++m) lo[m] = 1.0;                          // dummy modes of dropped nodes: zero eigenvector, harmless eigenvalue
    for (int m = 0; m < nf; ++m) {
        lo[m] = A[m * n1 + m];
        for (int a = 0; a < nf; ++a) So[idx[a] * n1 + m] = V[a * n1 + m] / sqrt(B[idx[a]]);
    }
}

__global__ void k_sz_sqrt(int64_t n, const double* __restrict__ in, double* __restrict__ out)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) out[l] = sqrt(in[l]);
}
template <typename TI, typename TO>
__global__ void k_sz_convert(int64_t n, const TI* __restrict__ in, TO* __restrict__ out)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) out[l] = (TO)in[l];
}

// ---- apply: out = w o A~^-1 (w o r), one block per element, six one-dimensional passes through shared memory ----------
template <typename ST>
__global__ void __launch_bounds__(128)
k_sz_apply(int n1, double lambda, const ST* __restrict__ Sm, const ST* __restrict__ lamv, const ST* __restrict__ w, const ST* __restrict__ r,
           ST* __restrict__ out, const semb_scalars* __restrict__ scal)
{
    typedef ST CT;
    extern __shared__ unsigned char smraw[];
    if (scal && *(volatile const int32_t*)&scal->done) return;
    const int Np = n1 * n1 * n1, n2 = n1 * n1;
    CT* A = (CT*)smraw; CT* B = A + Np; CT* S = B + Np; CT* L = S + 3 * n2;      // S[d][node][mode], L[d][mode]
    const int64_t e = blockIdx.x;
    for (int t = threadIdx.x; t < 3 * n2; t += blockDim.x) S[t] = Sm[e * 3 * n2 + t];
    for (int t = threadIdx.x; t < 3 * n1; t += blockDim.x) L[t] = lamv[e * 3 * n1 + t];
    for (int t = threadIdx.x; t < Np; t += blockDim.x) A[t] = w[e * Np + t] * r[e * Np + t];
    __syncthreads();
    const CT* Sr = S; const CT* Ss = S + n2; const CT* St = S + 2 * n2;
    // forward: (S_t x S_s x S_r)^T
    for (int t = threadIdx.x; t < Np; t += blockDim.x) {               // B[k][j][a] = sum_i Sr[i][a] A[k][j][i]
        const int a = t % n1, kj = t / n1;
        CT s = (CT)0;
        for (int i = 0; i < n1; ++i) s += Sr[i * n1 + a] * A[kj * n1 + i];
        B[t] = s;
    }
    __syncthreads();
    for (int t = threadIdx.x; t < Np; t += blockDim.x) {               // A[k][b][a] = sum_j Ss[j][b] B[k][j][a]
        const int a = t % n1, b = (t / n1) % n1, k = t / n2;
        CT s = (CT)0;
        for (int j = 0; j < n1; ++j) s += Ss[j * n1 + b] * B[k * n2 + j * n1 + a];
        A[t] = s;
    }
    __syncthreads();
    const CT lh = (CT)lambda;
    CT big = lh;                                                       // largest denominator of the block: threshold of the pseudo-inverse
    for (int d = 0; d < 3; ++d) { CT mx = (CT)0; for (int q = 0; q < n1; ++q) mx = fmax(mx, L[d * n1 + q]); big += mx; }
    const CT tiny = big * (CT)(sizeof(CT) == 8 ? 1e-12 : 1e-5);
    for (int t = threadIdx.x; t < Np; t += blockDim.x) {               // B[c][b][a] = sum_k St[k][c] A[k][b][a], then the diagonal inverse
        const int ba = t % n2, c = t / n2, a = ba % n1, b = ba / n1;
        CT s = (CT)0;
        for (int k = 0; k < n1; ++k) s += St[k * n1 + c] * A[k * n2 + ba];
        const CT den = L[2 * n1 + c] + L[n1 + b] + L[a] + lh;
        B[t] = (den > tiny) ? s / den : (CT)0;
    }
    __syncthreads();
    // backward: S_t x S_s x S_r
    for (int t = threadIdx.x; t < Np; t += blockDim.x) {               // A[k][b][a] = sum_c St[k][c] B[c][b][a]
        const int ba = t % n2, k = t / n2;
        CT s = (CT)0;
        for (int c = 0; c < n1; ++c) s += St[k * n1 + c] * B[c * n2 + ba];
        A[t] = s;
    }
    __syncthreads();
    for (int t = threadIdx.x; t < Np; t += blockDim.x) {               // B[k][j][a] = sum_b Ss[j][b] A[k][b][a]
        const int a = t % n1, j = (t / n1) % n1, k = t / n2;
        CT s = (CT)0;
        for (int b = 0; b < n1; ++b) s += Ss[j * n1 + b] * A[k * n2 + b * n1 + a];
        B[t] = s;
    }
    __syncthreads();
    for (int t = threadIdx.x; t < Np; t += blockDim.x) {               // out[k][j][i] = w sum_a Sr[i][a] B[k][j][a]
        const int i = t % n1, kj = t / n1;
        CT s = (CT)0;
        for (int a = 0; a < n1; ++a) s += Sr[i * n1 + a] * B[kj * n1 + a];
        out[e * Np + t] = w[e * Np + t] * s;
    }
}

// ---- apply, production form: one thread per LINE, as in the axhelm kernel (axhelm_kernels.cuh).  Thread (a, b) of an element owns
// the t-line (i=a, j=b, k=*), an r-line and an s-line; a line is transformed in registers by the element's own n1 x n1 matrix,
// whose rows come from shared memory as 128-bit BROADCAST loads (every thread of the block reads the same row), and shared memory
// otherwise only transposes the tile between the three line orientations (32-bit tiles for the FP32 levels, the swizzled
// conflict-free layout for n1 = 8).  Passes: r, s forward; t forward, diagonal inverse, t backward in registers; s, r backward.
#ifndef SEMB_SZ_LPT8
#define SEMB_SZ_LPT8 2
#endif
#ifndef SEMB_SZ_LPT10
#define SEMB_SZ_LPT10 2
#endif
#ifndef SEMB_SZ_EPB10
#define SEMB_SZ_EPB10 3
#endif
#ifndef SEMB_SZ_EPB8
#define SEMB_SZ_EPB8 2
#endif
template <int n1, typename ST> struct sz_cfg {
    static constexpr int VL = 16 / (int)sizeof(ST);                       // elements per 128-bit load
    static constexpr int RL = (n1 + VL - 1) / VL * VL;                    // padded row length
    // LPT lines per thread (n1 = 8, 10): one broadcast matrix-row load feeds LPT multiply-adds, which halves the kernel's
    // largest share of shared-memory wavefronts; the lines of a thread are (a, b) and (a, b + n1/2).  Measured on B200 (40 M nodes,
    // V-cycle on fp32 levels with Schwarz smoothing / fp64 apply): N = 9 6.84 -> 6.61 ms / 0.79 -> 0.77 ms, N = 7 5.70 -> 5.64 ms /
    // 0.70 -> 0.65 ms; elements per block 5 | 3 | 2 at n1 = 10: 6.74 | 6.61 | 6.73 ms.
    static constexpr int LPT = (n1 == 8) ? SEMB_SZ_LPT8 : (n1 == 10) ? SEMB_SZ_LPT10 : 1;
    static constexpr int TPE = n1 * n1 / LPT;                             // threads per element
    static constexpr int EPB = (n1 <= 3) ? 14 : (n1 == 4) ? 8 : (n1 <= 6) ? 3 : (LPT == 1) ? 1
                             : (sizeof(ST) == 4) ? (n1 == 10 ? SEMB_SZ_EPB10 : SEMB_SZ_EPB8) : 2;
};

// y_l = M x_l for the LPT lines of a thread
template <int n1, typename ST, int LPT>
__device__ __forceinline__ void sz_line(const ST* __restrict__ M, const ST (&x)[LPT][sz_cfg<n1, ST>::RL], ST (&y)[LPT][n1])
{
    constexpr int RL = sz_cfg<n1, ST>::RL, VL = sz_cfg<n1, ST>::VL;
#pragma unroll
    for (int o = 0; o < n1; ++o) {
        ST acc[LPT];
#pragma unroll
        for (int l = 0; l < LPT; ++l) acc[l] = (ST)0;
#pragma unroll
        for (int q = 0; q < RL; q += VL) {
            if (sizeof(ST) == 4) {
                const float4 m4 = *reinterpret_cast<const float4*>(reinterpret_cast<const float*>(M) + o * RL + q);
#pragma unroll
                for (int l = 0; l < LPT; ++l) acc[l] += (ST)m4.x * x[l][q] + (ST)m4.y * x[l][q + 1] + (ST)m4.z * x[l][q + 2] + (ST)m4.w * x[l][q + 3];
            } else {
                const double2 m2 = *reinterpret_cast<const double2*>(reinterpret_cast<const double*>(M) + o * RL + q);
#pragma unroll
                for (int l = 0; l < LPT; ++l) acc[l] += (ST)m2.x * x[l][q] + (ST)m2.y * x[l][q + 1];
            }
        }
#pragma unroll
        for (int l = 0; l < LPT; ++l) y[l][o] = acc[l];
    }
}

template <int n1, typename ST>
__global__ void __launch_bounds__(sz_cfg<n1, ST>::TPE * sz_cfg<n1, ST>::EPB)
k_sz_line(int64_t E, double lambda, const ST* __restrict__ Sm, const ST* __restrict__ lamv, const ST* __restrict__ w, const ST* __restrict__ r,
          ST* __restrict__ out, const semb_scalars* __restrict__ scal)
{
    using T = ax_tile<n1>;
    using C = sz_cfg<n1, ST>;
    constexpr int n2 = n1 * n1, Np = n2 * n1, RL = C::RL, EPB = C::EPB, LPT = C::LPT, TPE = C::TPE, BS = n1 / LPT;
    constexpr bool W32 = sizeof(ST) == 4;
#define SZ_I(k, j, i) (W32 ? T::idx32(k, j, i) : T::idx(k, j, i))
    __shared__ __align__(16) ST tileA[EPB * T::size];
    __shared__ __align__(16) ST mat[EPB][3][2][n1 * RL];                  // [direction][0: S^T (forward), 1: S (backward)][row][padded column]
    __shared__ ST lam[EPB][3][n1];
    if (scal && *(volatile const int32_t*)&scal->done) return;
    const int el = (EPB > 1) ? threadIdx.x / TPE : 0, tl = (EPB > 1) ? threadIdx.x - el * TPE : threadIdx.x;
    int64_t e = blockIdx.x * (int64_t)EPB + el;
    const bool valid = e < E;
    if (!valid) e = E - 1;
    ST* __restrict__ Su = tileA + el * T::size;
    const int a = tl % n1, b = tl / n1;                                   // the thread's lines: second index b + l * BS
    // the element's matrices: S_d[node][mode] -> forward rows [mode][node], backward rows [node][mode], zero padded
    for (int t = tl; t < 3 * n1 * RL; t += TPE) {
        const int d = t / (n1 * RL), row = (t / RL) % n1, col = t % RL;
        const bool in = col < n1;
        mat[el][d][0][row * RL + col] = in ? Sm[(e * 3 + d) * n2 + col * n1 + row] : (ST)0;
        mat[el][d][1][row * RL + col] = in ? Sm[(e * 3 + d) * n2 + row * n1 + col] : (ST)0;
    }
    for (int t = tl; t < 3 * n1; t += TPE) lam[el][t / n1][t % n1] = lamv[e * 3 * n1 + t];
    ST wv[LPT][n1];
#pragma unroll
    for (int l = 0; l < LPT; ++l) {
#pragma unroll
        for (int k = 0; k < n1; ++k) {
            const int64_t g = e * Np + k * n2 + (b + l * BS) * n1 + a;
            wv[l][k] = w[g];
            Su[SZ_I(k, b + l * BS, a)] = wv[l][k] * r[g];
        }
    }
    __syncthreads();
    ST x[LPT][RL], y[LPT][n1];
#pragma unroll
    for (int l = 0; l < LPT; ++l) {
#pragma unroll
        for (int q = n1; q < RL; ++q) x[l][q] = (ST)0;
    }
    // one pass: read the thread's LPT lines, contract, write back.  ORI 0: r-line (i = *, j = a, k = b_l), 1: s-line (i = a, j = *, k = b_l)
#define SZ_PASS(ORI, M)                                                                                            \
    {                                                                                                              \
        _Pragma("unroll") for (int l = 0; l < LPT; ++l) {                                                          \
            _Pragma("unroll") for (int q = 0; q < n1; ++q) x[l][q] = (ORI == 0) ? Su[SZ_I(b + l * BS, a, q)] : Su[SZ_I(b + l * BS, q, a)]; \
        }                                                                                                          \
        sz_line<n1, ST, LPT>(M, x, y);                                                                             \
        _Pragma("unroll") for (int l = 0; l < LPT; ++l) {                                                          \
            _Pragma("unroll") for (int q = 0; q < n1; ++q) {                                                       \
                if (ORI == 0) Su[SZ_I(b + l * BS, a, q)] = y[l][q]; else Su[SZ_I(b + l * BS, q, a)] = y[l][q];     \
            }                                                                                                      \
        }                                                                                                          \
        __syncthreads();                                                                                           \
    }
    SZ_PASS(0, mat[el][0][0])
    SZ_PASS(1, mat[el][1][0])
    // t: forward, diagonal inverse, backward on the thread's own t-lines (i = a, j = b_l, k = *); modes (a, b_l) of r and s
#pragma unroll
    for (int l = 0; l < LPT; ++l) {
#pragma unroll
        for (int k = 0; k < n1; ++k) x[l][k] = Su[SZ_I(k, b + l * BS, a)];
    }
    sz_line<n1, ST, LPT>(mat[el][2][0], x, y);
    {
        ST big = (ST)lambda;
#pragma unroll
        for (int d = 0; d < 3; ++d) { ST mx = (ST)0; for (int q = 0; q < n1; ++q) mx = fmax(mx, lam[el][d][q]); big += mx; }
        const ST tiny = big * (ST)(W32 ? 1e-5 : 1e-12);
#pragma unroll
        for (int l = 0; l < LPT; ++l) {
            const ST lab = lam[el][0][a] + lam[el][1][b + l * BS] + (ST)lambda;
#pragma unroll
            for (int c = 0; c < n1; ++c) { const ST den = lam[el][2][c] + lab; x[l][c] = (den > tiny) ? y[l][c] / den : (ST)0; }
        }
    }
    sz_line<n1, ST, LPT>(mat[el][2][1], x, y);
#pragma unroll
    for (int l = 0; l < LPT; ++l) {
#pragma unroll
        for (int k = 0; k < n1; ++k) Su[SZ_I(k, b + l * BS, a)] = y[l][k];
    }
    __syncthreads();
    SZ_PASS(1, mat[el][1][1])
    SZ_PASS(0, mat[el][0][1])
#undef SZ_PASS
#pragma unroll
    for (int l = 0; l < LPT; ++l) {
#pragma unroll
        for (int k = 0; k < n1; ++k) if (valid) out[e * Np + k * n2 + (b + l * BS) * n1 + a] = wv[l][k] * Su[SZ_I(k, b + l * BS, a)];
    }
#undef SZ_I
}

template <int n1, typename ST>
static void sz_line_launch(semb_mesh* L, double lambda, const ST* S, const ST* lam, const ST* w, const ST* v, ST* out, semb_scalars* scal, cudaStream_t s)
{
    constexpr int EPB = sz_cfg<n1, ST>::EPB;
    k_sz_line<n1, ST><<<(unsigned)((L->E + EPB - 1) / EPB), sz_cfg<n1, ST>::TPE * EPB, 0, s>>>(L->E, lambda, S, lam, w, v, out, scal);
}

// d = c1 d + c2 sr (first: d = c2 sr);  z = z + d (zset: z = d)
template <typename ST>
__global__ void k_sz_update(int64_t n, double c1, double c2, const ST* __restrict__ sr, ST* __restrict__ d, ST* __restrict__ z, int first, int zset,
                            const semb_scalars* __restrict__ scal)
{
    if (scal && *(volatile const int32_t*)&scal->done) return;
    const ST k1 = (ST)c1, k2 = (ST)c2;
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const ST dn = first ? k2 * sr[l] : k1 * d[l] + k2 * sr[l];
        d[l] = dn;
        z[l] = zset ? dn : z[l] + dn;
    }
}
template <typename ST>
__global__ void k_sz_axpy(int64_t n, double a, const ST* __restrict__ x, const ST* __restrict__ y, ST* __restrict__ out, const semb_scalars* __restrict__ scal)
{
    if (scal && *(volatile const int32_t*)&scal->done) return;
    const ST k = (ST)a;
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) out[l] = y[l] + k * x[l];
}

// Gather form of QQ^T for a vector that is consumed once (as in pcg.cu): code -1 = no copy; <= -2: one partner at local index
// -(code + 2); >= 3: the class was summed in place by k_gs_hi.  Four nodes per thread in lock-step keep four partner loads in flight.
template <typename ST>
__device__ __forceinline__ void sz_gather4(const ST* __restrict__ v, const int32_t* __restrict__ code, int64_t l0, int64_t n, int64_t stride, ST (&val)[4])
{
    int32_t c[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { const int64_t l = l0 + u * stride; c[u] = (l < n) ? code[l] : -1; }
    ST own[4], pv[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { const int64_t l = l0 + u * stride; own[u] = (l < n) ? v[l] : (ST)0; pv[u] = (c[u] <= -2) ? v[-(c[u] + 2)] : (ST)0; }
#pragma unroll
    for (int u = 0; u < 4; ++u) val[u] = own[u] + pv[u];
}
// d = c1 d + c2 QQ^T sr (first: d = c2 QQ^T sr);  z = z + d (zset: z = d)
template <typename ST>
__global__ void __launch_bounds__(256)
k_sz_update_g(int64_t n, double c1, double c2, const ST* __restrict__ sr, const int32_t* __restrict__ code, ST* __restrict__ d, ST* __restrict__ z,
              int first, int zset, const semb_scalars* __restrict__ scal)
{
    if (scal && *(volatile const int32_t*)&scal->done) return;
    const ST k1 = (ST)c1, k2 = (ST)c2;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t l0 = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l0 < n; l0 += 4 * stride) {
        ST sv[4];
        sz_gather4<ST>(sr, code, l0, n, stride, sv);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int64_t l = l0 + u * stride;
            if (l < n) { const ST dn = first ? k2 * sv[u] : k1 * d[l] + k2 * sv[u]; d[l] = dn; z[l] = zset ? dn : z[l] + dn; }
        }
    }
}
// out = y - QQ^T x
template <typename ST>
__global__ void __launch_bounds__(256)
k_sz_resid_g(int64_t n, const ST* __restrict__ x, const int32_t* __restrict__ code, const ST* __restrict__ y, ST* __restrict__ out,
             const semb_scalars* __restrict__ scal)
{
    if (scal && *(volatile const int32_t*)&scal->done) return;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t l0 = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l0 < n; l0 += 4 * stride) {
        ST sv[4];
        sz_gather4<ST>(x, code, l0, n, stride, sv);
#pragma unroll
        for (int u = 0; u < 4; ++u) { const int64_t l = l0 + u * stride; if (l < n) out[l] = y[l] - sv[u]; }
    }
}

static unsigned sz_grid(int64_t n) { int64_t b = (n + 1023) / 1024, cap = (int64_t)semb_sm_count() * 8; return (unsigned)(b < 1 ? 1 : (b > cap ? cap : b)); }

void semb_schwarz_free(semb_mesh* L)
{
    for (semb_schwarz* z : L->schwarz) {
        semb_dev_free(L, z->S); semb_dev_free(L, z->lam); semb_dev_free(L, z->w); semb_dev_free(L, z->Sf); semb_dev_free(L, z->lamf); semb_dev_free(L, z->wf);
        delete z;
    }
    L->schwarz.clear();
}

// subdomain data of level mesh L for the Dirichlet tag set `tags` (built once, cached in L)
int semb_schwarz_get(semb_mesh* L, uint32_t tags, bool want_float, semb_schwarz** out, cudaStream_t s)
{
    if (L->N < 2) return semb_fail(L, SEMB_EINVAL, "Schwarz smoother needs order >= 2");
    semb_schwarz* z = nullptr;
    for (semb_schwarz* c : L->schwarz) if (c->tags == tags) z = c;
    const int n1 = L->n1; const int64_t E = L->E, n = L->n;
    if (!z) {
        if (!L->xyz) return semb_fail(L, SEMB_EINVAL, "Schwarz smoother: the level holds no coordinates");
        z = new semb_schwarz(); z->tags = tags;
        double Kh[SEMB_MAXN1 * SEMB_MAXN1];
        for (int a = 0; a < n1; ++a) for (int b = 0; b < n1; ++b) {
            double v = 0.0;
            for (int m = 0; m < n1; ++m) v += L->D[m * n1 + a] * L->rho[m] * L->D[m * n1 + b];
            Kh[a * n1 + b] = v;
        }
        z->S = (double*)semb_dev_alloc(L, sizeof(double) * 3 * n1 * n1 * (size_t)E);
        z->lam = (double*)semb_dev_alloc(L, sizeof(double) * 3 * n1 * (size_t)E);
        z->w = (double*)semb_dev_alloc(L, sizeof(double) * (size_t)n);
        double* tmp = (double*)semb_dev_alloc(L, sizeof(double) * ((size_t)n + 3 * (size_t)E + n1 * n1 + n1));
        int rc = (z->S && z->lam && z->w && tmp) ? SEMB_OK : semb_fail(L, SEMB_ENOMEM, "Schwarz smoother data");
        if (!rc) {
            double *F = tmp, *len = tmp + n, *dK = len + 3 * E, *drho = dK + n1 * n1;
            cudaError_t e = cudaMemcpyAsync(dK, Kh, sizeof(double) * n1 * n1, cudaMemcpyHostToDevice, s);
            if (e == cudaSuccess) e = cudaMemcpyAsync(drho, L->rho, sizeof(double) * n1, cudaMemcpyHostToDevice, s);
            if (e == cudaSuccess) { k_sz_lengths<<<(unsigned)E, 128, 0, s>>>(n1, n, L->xyz, len, F); e = cudaGetLastError(); }
            if (e != cudaSuccess) rc = semb_fail(L, SEMB_ECUDA, "Schwarz setup: %s", cudaGetErrorString(e));
            if (!rc) rc = semb_gs_launch(L, F, 1, s);
            if (!rc) {
                k_sz_eigen<<<(unsigned)((3 * E + 63) / 64), 64, 0, s>>>(E, n1, dK, drho, len, F, L->invmult, L->face_tag_dev, tags, z->S, z->lam);
                k_sz_sqrt<<<sz_grid(n), 256, 0, s>>>(n, L->invmult, z->w);
                e = cudaGetLastError();
                if (e == cudaSuccess) e = cudaStreamSynchronize(s);
                if (e != cudaSuccess) rc = semb_fail(L, SEMB_ECUDA, "Schwarz eigenproblems: %s", cudaGetErrorString(e));
            }
        }
        semb_dev_free(L, tmp);
        if (rc) { semb_dev_free(L, z->S); semb_dev_free(L, z->lam); semb_dev_free(L, z->w); delete z; return rc; }
        L->schwarz.push_back(z);
    }
    if (want_float && !z->Sf) {
        const int64_t ns = 3 * n1 * n1 * E, nl = 3 * n1 * E;
        z->Sf = (float*)semb_dev_alloc(L, sizeof(float) * (size_t)ns); z->lamf = (float*)semb_dev_alloc(L, sizeof(float) * (size_t)nl);
        z->wf = (float*)semb_dev_alloc(L, sizeof(float) * (size_t)n);
        if (!z->Sf || !z->lamf || !z->wf) return semb_fail(L, SEMB_ENOMEM, "Schwarz smoother data (fp32)");
        k_sz_convert<double, float><<<sz_grid(ns), 256, 0, s>>>(ns, z->S, z->Sf);
        k_sz_convert<double, float><<<sz_grid(nl), 256, 0, s>>>(nl, z->lam, z->lamf);
        k_sz_convert<double, float><<<sz_grid(n), 256, 0, s>>>(n, z->w, z->wf);
        SEMB_CUDA(L, cudaGetLastError());
    }
    *out = z;
    return SEMB_OK;
}

// ---- the level operations in the storage type ---------------------------------------------------------------
static inline const double* sz_S(const semb_schwarz* z, double) { return z->S; }
static inline const float* sz_S(const semb_schwarz* z, float) { return z->Sf; }
static inline const double* sz_lam(const semb_schwarz* z, double) { return z->lam; }
static inline const float* sz_lam(const semb_schwarz* z, float) { return z->lamf; }
static inline const double* sz_w(const semb_schwarz* z, double) { return z->w; }
static inline const float* sz_w(const semb_schwarz* z, float) { return z->wf; }
static inline int sz_gs(semb_mesh* L, double* v, cudaStream_t s) { return semb_gs_launch(L, v, 1, s); }
static inline int sz_gs(semb_mesh* L, float* v, cudaStream_t s) { return semb_gs_launch_f(L, v, s); }
static inline int sz_mask(semb_mesh* L, const semb_mask_entry& m, double* v, cudaStream_t s) { return semb_mask_launch(L, m, v, 1, s); }
static inline int sz_mask(semb_mesh* L, const semb_mask_entry& m, float* v, cudaStream_t s) { return semb_mask_launch_f(L, m, v, s); }
static inline int sz_gs_hi(semb_mesh* L, double* v, semb_scalars* scal, cudaStream_t s) { return semb_gs_hi_launch(L, v, scal, s); }
static inline int sz_gs_hi(semb_mesh* L, float* v, semb_scalars* scal, cudaStream_t s) { return semb_gs_hi_launch_f(L, v, scal, s); }
static inline int sz_axhelm(semb_mesh* L, double lambda, const double*, const double* u, double* w, semb_scalars* scal, cudaStream_t s)
{ (void)scal; return semb_axhelm_launch(L, lambda, nullptr, nullptr, u, w, 1, nullptr, s); }
static inline int sz_axhelm(semb_mesh* L, double lambda, const float* geo, const float* u, float* w, semb_scalars* scal, cudaStream_t s)
{ return semb_axhelm_launch_f(L, lambda, geo, u, w, scal, s); }

// out = S v = M QQ^T [w o A~^-1 (w o v)];  local_only: stop before QQ^T (the consumer applies it in gather form after k_gs_hi)
template <typename ST>
static int sz_apply(semb_mesh* L, const semb_schwarz* z, double lambda, const semb_mask_entry& m, const ST* v, ST* out, semb_scalars* scal, cudaStream_t s,
                    bool local_only = false)
{
    const int n1 = L->n1;
    const ST *S = sz_S(z, ST()), *lm = sz_lam(z, ST()), *w = sz_w(z, ST());
    switch (SEMB_SZ_LINE ? n1 : 0) {
        case 3:  sz_line_launch<3, ST>(L, lambda, S, lm, w, v, out, scal, s); break;
        case 4:  sz_line_launch<4, ST>(L, lambda, S, lm, w, v, out, scal, s); break;
        case 5:  sz_line_launch<5, ST>(L, lambda, S, lm, w, v, out, scal, s); break;
        case 6:  sz_line_launch<6, ST>(L, lambda, S, lm, w, v, out, scal, s); break;
        case 7:  sz_line_launch<7, ST>(L, lambda, S, lm, w, v, out, scal, s); break;
        case 8:  sz_line_launch<8, ST>(L, lambda, S, lm, w, v, out, scal, s); break;
        case 9:  sz_line_launch<9, ST>(L, lambda, S, lm, w, v, out, scal, s); break;
        case 10: sz_line_launch<10, ST>(L, lambda, S, lm, w, v, out, scal, s); break;
        case 11: sz_line_launch<11, ST>(L, lambda, S, lm, w, v, out, scal, s); break;
        default: {                       // the plain six-pass kernel (run-time order; kept as the A/B reference: -DSEMB_SZ_LINE=0)
            const size_t smem = sizeof(ST) * (2 * (size_t)L->Np + 3 * n1 * n1 + 3 * n1);
            k_sz_apply<ST><<<(unsigned)L->E, 128, smem, s>>>(n1, lambda, S, lm, w, v, out, scal);
        }
    }
    L->launches += 1;
    if (local_only) {
        int rc = sz_mask(L, m, out, s); if (rc) return rc;
        return sz_gs_hi(L, out, scal, s);
    }
    int rc = sz_gs(L, out, s); if (rc) return rc;
    return sz_mask(L, m, out, s);
}

// z (+)= fourth-kind Chebyshev polynomial of degree k in S A applied to r.  sr, d, t: work vectors; res: work (holds r - A z_k)
template <typename ST>
static int sz_cheb4(semb_mesh* L, const semb_schwarz* zd, double lambda, const ST* geo, const semb_mask_entry& m, int k, double lmax,
                    const ST* r, ST* z, ST* res, ST* d, ST* sr, ST* t, semb_scalars* scal, cudaStream_t s, bool zacc)
{
    const int64_t n = L->n;
    // every assembled vector of the recurrence is consumed exactly once, so QQ^T is applied in gather form by the consumer
    // (k_gs_hi for the edge / corner classes, the face partner inside the streaming kernel) instead of a read-modify-write pass
    int rc = sz_apply<ST>(L, zd, lambda, m, r, sr, scal, s, true); if (rc) return rc;
    k_sz_update_g<ST><<<sz_grid(n), 256, 0, s>>>(n, 0.0, 4.0 / (3.0 * lmax), sr, L->gs_code, d, z, 1, zacc ? 0 : 1, scal);
    const ST* rin = r;
    for (int i = 1; i <= k; ++i) {
        rc = sz_axhelm(L, lambda, geo, d, t, scal, s); if (rc) return rc;             // t = A_L d
        rc = sz_mask(L, m, t, s); if (rc) return rc;
        rc = sz_gs_hi(L, t, scal, s); if (rc) return rc;
        k_sz_resid_g<ST><<<sz_grid(n), 256, 0, s>>>(n, t, L->gs_code, rin, res, scal);  // res = res - QQ^T A_L d
        rin = res;
        rc = sz_apply<ST>(L, zd, lambda, m, res, sr, scal, s, true); if (rc) return rc;
        k_sz_update_g<ST><<<sz_grid(n), 256, 0, s>>>(n, (2.0 * i - 1.0) / (2.0 * i + 3.0), (8.0 * i + 4.0) / ((2.0 * i + 3.0) * lmax), sr, L->gs_code, d, z, 0, 0, scal);
        L->launches += 2;
    }
    L->launches += 1;
    SEMB_CUDA(L, cudaGetLastError());
    return SEMB_OK;
}

int semb_schwarz_cheb4(semb_mesh* L, semb_schwarz* zd, double lambda, const semb_mask_entry& m, int k, double lmax, const double* r, double* z,
                       double* res, double* d, double* sr, double* t, semb_scalars* scal, cudaStream_t s, bool zacc)
{
    return sz_cheb4<double>(L, zd, lambda, nullptr, m, k, lmax, r, z, res, d, sr, t, scal, s, zacc);
}
int semb_schwarz_cheb4_f(semb_mesh* L, semb_schwarz* zd, double lambda, const float* geo, const semb_mask_entry& m, int k, double lmax, const float* r,
                         float* z, float* res, float* d, float* sr, float* t, semb_scalars* scal, cudaStream_t s, bool zacc)
{
    return sz_cheb4<float>(L, zd, lambda, geo, m, k, lmax, r, z, res, d, sr, t, scal, s, zacc);
}
int semb_schwarz_apply_run(semb_mesh* L, uint32_t tags, double lambda, const double* r, double* out, cudaStream_t s)
{
    semb_schwarz* zd; semb_mask_entry m;
    int rc = semb_schwarz_get(L, tags, false, &zd, s); if (rc) return rc;
    rc = semb_get_mask(L, tags, &m, s); if (rc) return rc;
    return sz_apply<double>(L, zd, lambda, m, r, out, nullptr, s);
}

// <a, b> over unique nodes, on the host (setup only)
__global__ void k_sz_dot(int64_t n, const double* __restrict__ a, const double* __restrict__ b, const double* __restrict__ invmult, double* __restrict__ out)
{
    __shared__ double red[256];
    double s = 0.0;
    for (int64_t l = threadIdx.x; l < n; l += blockDim.x) s += a[l] * b[l] * invmult[l];
    red[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) { if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o]; __syncthreads(); }
    if (threadIdx.x == 0) *out = red[0];
}
__global__ void k_sz_dot_blocks(int64_t n, const double* __restrict__ a, const double* __restrict__ b, const double* __restrict__ invmult, double* __restrict__ part)
{
    __shared__ double red[256];
    double s = 0.0;
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) s += a[l] * b[l] * invmult[l];
    red[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) { if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o]; __syncthreads(); }
    if (threadIdx.x == 0) part[blockIdx.x] = red[0];
}
static int sz_dot(semb_mesh* L, const double* a, const double* b, double* scratch, double* host, cudaStream_t s)
{
    const unsigned g = sz_grid(L->n);
    k_sz_dot_blocks<<<g, 256, 0, s>>>(L->n, a, b, L->invmult, scratch);
    double part[2048];
    SEMB_CUDA(L, cudaMemcpyAsync(part, scratch, sizeof(double) * g, cudaMemcpyDeviceToHost, s));
    SEMB_CUDA(L, cudaStreamSynchronize(s));
    double t = 0.0;
    for (unsigned i = 0; i < g; ++i) t += part[i];
    *host = t;
    return SEMB_OK;
}

double semb_tridiag_lmax(int m, const double* a, const double* b);

// 1.1 x the largest Ritz value of S A after `steps` steps of the preconditioned conjugate-gradient (Lanczos) recurrence from v0
// (work: 5 vectors of the level).  Cached per lambda in the Schwarz data.
int semb_schwarz_lmax(semb_mesh* L, semb_schwarz* zd, double lambda, const semb_mask_entry& m, const double* v0, int steps, double* const* work,
                      double* lmax, cudaStream_t s)
{
    for (auto& kv : zd->lmax) if (kv.first == lambda) { *lmax = kv.second; return SEMB_OK; }
    const int64_t n = L->n;
    double *r = work[0], *z = work[1], *p = work[2], *q = work[3], *scr = work[4];
    SEMB_CUDA(L, cudaMemcpyAsync(r, v0, sizeof(double) * (size_t)n, cudaMemcpyDeviceToDevice, s));
    int rc = sz_apply<double>(L, zd, lambda, m, r, z, nullptr, s); if (rc) return rc;
    double rho, pq, al[64], be[64];
    rc = sz_dot(L, r, z, scr, &rho, s); if (rc) return rc;
    SEMB_CUDA(L, cudaMemcpyAsync(p, z, sizeof(double) * (size_t)n, cudaMemcpyDeviceToDevice, s));
    int cnt = 0;
    if (steps > 64) steps = 64;
    for (int j = 0; j < steps; ++j) {
        rc = semb_axhelm_launch(L, lambda, nullptr, nullptr, p, q, 1, nullptr, s); if (rc) return rc;
        rc = semb_mask_launch(L, m, q, 1, s); if (rc) return rc;
        rc = semb_gs_launch(L, q, 1, s); if (rc) return rc;
        rc = sz_dot(L, p, q, scr, &pq, s); if (rc) return rc;
        const double a = rho / pq;
        k_sz_axpy<double><<<sz_grid(n), 256, 0, s>>>(n, -a, q, r, r, nullptr);
        rc = sz_apply<double>(L, zd, lambda, m, r, z, nullptr, s); if (rc) return rc;
        double rho_new;
        rc = sz_dot(L, r, z, scr, &rho_new, s); if (rc) return rc;
        const double b = rho_new / rho;
        al[cnt] = a; be[cnt] = b; ++cnt;
        if (!(rho_new > 1e-28 * fabs(rho))) break;
        k_sz_axpy<double><<<sz_grid(n), 256, 0, s>>>(n, b, p, z, p, nullptr);         // p = z + b p
        rho = rho_new;
    }
    double td[64], te[64];
    for (int j = 0; j < cnt; ++j) {
        td[j] = 1.0 / al[j] + (j > 0 ? be[j - 1] / al[j - 1] : 0.0);
        if (j + 1 < cnt) te[j] = sqrt(be[j]) / al[j];
    }
    *lmax = 1.1 * semb_tridiag_lmax(cnt, td, te);
    zd->lmax.push_back(std::make_pair(lambda, *lmax));
    return SEMB_OK;
}
