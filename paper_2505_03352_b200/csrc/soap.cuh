// soap.cuh -- SOAP optimizer step, Eqs. (12)-(13) (readings S21-S23), on one [mx,my] matrix of control variables.
// Optimizer glue around the hot path, run once per design iteration: small dense fp32 products (mx, my ~ 250..1024) whose
// accuracy matters (they rotate moments that are compared at 1e-5) -- plain FFMA tiles, no tensor cores, no library GEMM.
//   Eq. (12)  L <- b2 L + (1-b2) G G^T,  R <- b2 R + (1-b2) G^T G                      two k_gemm launches
//   Eq. (13)  M <- b1 M + (1-b1) G (Eq. (10), S21);  G' = Q_L^T G Q_R;  M' = Q_L^T M Q_R  k_soap_moment + four k_gemm launches
//             V' <- b2 V' + (1-b2) G'^2;  N' = Mhat'/sqrt(Vhat' + eps) (S22)            k_soap_rotated
//             C <- C - eta Q_L N' Q_R^T                                                 two k_gemm launches (alpha = -eta, beta = 1)
// The eigenvectors Q_L, Q_R come from a library eigensolver (epsgrad.cu: cuSOLVER syevd, loaded on first use).
#pragma once
#include "common.cuh"

namespace epsgrad {

constexpr int GM_T = 64, GM_K = 16, GM_THREADS = 256;

// C[m,n] = alpha op(A) op(B) + beta C, row-major, op = transpose when TA / TB.  op(A) is [m,k], op(B) is [k,n].
// 64x64 tile per CTA, 4x4 outputs per thread, k in steps of 16 through shared memory; k is summed in increasing order.
template <bool TA, bool TB>
__global__ void __launch_bounds__(GM_THREADS) k_gemm(const float *__restrict__ A, const float *__restrict__ B, float *C,
                                                     int m, int n, int k, int lda, int ldb, int ldc, float alpha, float beta)
{
    __shared__ float As[GM_K][GM_T + 4];      // As[kk][i] = op(A)[i0 + i, k0 + kk]
    __shared__ float Bs[GM_K][GM_T + 4];      // Bs[kk][j] = op(B)[k0 + kk, j0 + j]
    const int tid = threadIdx.x, i0 = blockIdx.y * GM_T, j0 = blockIdx.x * GM_T;
    const int ti = (tid >> 4) << 2, tj = (tid & 15) << 2;
    float acc[4][4] = {};
    for (int k0 = 0; k0 < k; k0 += GM_K) {
        for (int e = tid; e < GM_T * GM_K; e += GM_THREADS) {
            // the fastest-varying index of each load follows the operand's contiguous axis
            int i, kk;
            if (TA) { i = e % GM_T; kk = e / GM_T; } else { kk = e % GM_K; i = e / GM_K; }
            const int gi = i0 + i, gk = k0 + kk;
            As[kk][i] = (gi < m && gk < k) ? (TA ? A[(size_t)gk * lda + gi] : A[(size_t)gi * lda + gk]) : 0.0f;
            int j, kb;
            if (TB) { kb = e % GM_K; j = e / GM_K; } else { j = e % GM_T; kb = e / GM_T; }
            const int gj = j0 + j, gkb = k0 + kb;
            Bs[kb][j] = (gj < n && gkb < k) ? (TB ? B[(size_t)gj * ldb + gkb] : B[(size_t)gkb * ldb + gj]) : 0.0f;
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < GM_K; ++kk) {
            const float4 a = *reinterpret_cast<const float4 *>(&As[kk][ti]);
            const float4 b = *reinterpret_cast<const float4 *>(&Bs[kk][tj]);
            const float av[4] = {a.x, a.y, a.z, a.w}, bv[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
            for (int x = 0; x < 4; ++x)
#pragma unroll
                for (int y = 0; y < 4; ++y) acc[x][y] = fmaf(av[x], bv[y], acc[x][y]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int x = 0; x < 4; ++x)
#pragma unroll
        for (int y = 0; y < 4; ++y) {
            const int gi = i0 + ti + x, gj = j0 + tj + y;
            if (gi < m && gj < n) {
                float *c = C + (size_t)gi * ldc + gj;
                *c = beta == 0.0f ? alpha * acc[x][y] : fmaf(alpha, acc[x][y], beta * *c);
            }
        }
}

// M <- b1 M + (1-b1) G   (Eq. (10), original basis; S21)
__global__ void __launch_bounds__(256) k_soap_moment(float *M, const float *G, size_t n, float b1, float omb1)
{
    const size_t k = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (k < n) M[k] = fmaf(b1, M[k], omb1 * G[k]);
}

// V' <- b2 V' + (1-b2) G'^2;  N' = (M'/c1)/sqrt(V'/c2 + eps), written over G'   (Eq. (13); S22).  IEEE division and root.
__global__ void __launch_bounds__(256) k_soap_rotated(float *Vp, float *Gp, const float *Mp, size_t n,
                                                      float b2, float omb2, float inv_c1, float inv_c2, float eps)
{
    const size_t k = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (k >= n) return;
    const float g = Gp[k];
    const float v = fmaf(b2, Vp[k], omb2 * g * g);
    Vp[k] = v;
    Gp[k] = (Mp[k] * inv_c1) / sqrtf(fmaf(v, inv_c2, eps));
}

// out = in^T for an n x n matrix (the eigensolver is column-major: its output read row-major has the eigenvectors in rows)
__global__ void __launch_bounds__(256) k_transpose(const float *in, float *out, int n)
{
    __shared__ float t[32][33];
    const int bx = blockIdx.x * 32, by = blockIdx.y * 32, tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int r = ty; r < 32; r += 8)
        if (by + r < n && bx + tx < n) t[r][tx] = in[(size_t)(by + r) * n + bx + tx];
    __syncthreads();
    for (int r = ty; r < 32; r += 8)
        if (bx + r < n && by + tx < n) out[(size_t)(bx + r) * n + by + tx] = t[tx][r];
}

// Adam, Eqs. (10)-(11), one step in place on n control variables: M = b1 M + (1-b1) G, V = b2 V + (1-b2) G^2,
// C -= lr (M/c1) / (sqrt(V/c2) + eps) with the bias corrections c1 = 1 - b1^i, c2 = 1 - b2^i formed on the host in float64.
// IEEE division and square root (no approximations): the update is compared with the float64 oracle at 1e-6.
__global__ void __launch_bounds__(256) k_adam(float *C, float *M, float *V, const float *G, size_t n,
                                              float b1, float b2, float omb1, float omb2, float inv_c1, float inv_c2, float lr, float eps)
{
    const size_t k = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (k >= n) return;
    const float g = G[k];
    const float m = fmaf(b1, M[k], omb1 * g);          // omb = 1 - b, rounded once from float64 (1.0f - 0.999f is off by 5e-5)
    const float v = fmaf(b2, V[k], omb2 * g * g);
    M[k] = m;
    V[k] = v;
    C[k] -= lr * (m * inv_c1) / (sqrtf(v * inv_c2) + eps);
}

}  // namespace epsgrad
