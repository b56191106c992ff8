// filter.cuh -- Eq. (2) as a polyphase stencil and its transpose.
//
// Mask pixel p = m*a0 + f (phase f in [0,m)) sits at X_p = (p+1/2)/s; control node a at
// x_a = u(a+1/2) (S3).  With a = a0 + t:  X_p - x_a = (f+1/2)/s - u/2 - u t, so the weight
// depends on (phase, tap) only: a table built on the host in float64.
//   forward  Phi'[p,q] = invden[p,q] * sum_{tx,ty} W[tx][ty][fx][fy] * c'[a0+tx-T][b0+ty-T]
//   reverse  dC[a,b]   = sum_{tx,ty,fx,fy} W[tx][ty][fx][fy] * v[m(a-tx+T)+fx][m(b-ty+T)+fy]
// c' = C - eta0 inside the control grid and 0 outside (centred accumulation: beta
// amplifies the fp32 rounding of Phi); v already carries invden.
// The conic basis is not separable: 2-D table, one thread per control pixel holding its
// m x m mask pixels in registers.  The per-axis-truncated Gaussian (S11) is separable:
// two 1-D passes through a temporary in global memory.
#pragma once
#include "common.cuh"

namespace epsgrad {

struct FilterParams {
    const float *C;        // [B,mx,my]
    float *phi;            // [B,px,py]   centred filter output
    const float *w;        // conic: [NT][NT][m][m]; separable: [NT][m]
    const int *tyrange;    // conic: [NT][2] first / last ty with a non-zero weight for this tx
    Normaliser nrm;
    int mx, my, px, py, T, NT;
    float eta0;
};

// ---------------------------------------------------------------- conic, forward
// grid (ceil(my/TB), ceil(mx/TA), B), block TA*TB threads; thread (la,lb) <-> control pixel.
template <int M, int TA, int TB>
__global__ void __launch_bounds__(TA *TB) k_filter_conic(const FilterParams P)
{
    extern __shared__ __align__(16) float sm[];
    const int T = P.T, NT = P.NT;
    const int CW = TB + 2 * T + 1;                 // pitch of the c' tile (odd-ish: no conflicts needed, reads are row-contiguous)
    float *w_s = sm;                               // NT*NT*M*M
    float *c_s = w_s + NT * NT * M * M;            // (TA+2T) * CW
    int *ty_s = reinterpret_cast<int *>(c_s + (TA + 2 * T) * CW);   // 2*NT
    const int tid = threadIdx.x, nthr = TA * TB;
    const int a_base = blockIdx.y * TA, b_base = blockIdx.x * TB, b = blockIdx.z;

    for (int i = tid; i < NT * NT * M * M; i += nthr) w_s[i] = P.w[i];
    for (int i = tid; i < 2 * NT; i += nthr) ty_s[i] = P.tyrange[i];
    const float *Cb = P.C + (size_t)b * P.mx * P.my;
    for (int i = tid; i < (TA + 2 * T) * (TB + 2 * T); i += nthr) {
        const int r = i / (TB + 2 * T), c = i - r * (TB + 2 * T);
        const int a = a_base - T + r, bb = b_base - T + c;
        float v = 0.0f;
        if (a >= 0 && a < P.mx && bb >= 0 && bb < P.my) v = Cb[(size_t)a * P.my + bb] - P.eta0;
        c_s[r * CW + c] = v;
    }
    __syncthreads();

    const int la = tid / TB, lb = tid - la * TB;
    const int a0 = a_base + la, b0 = b_base + lb;
    float acc[M][M];
#pragma unroll
    for (int i = 0; i < M; ++i)
#pragma unroll
        for (int j = 0; j < M; ++j) acc[i][j] = 0.0f;

    for (int tx = 0; tx < NT; ++tx) {
        const int ty0 = ty_s[2 * tx], ty1 = ty_s[2 * tx + 1];
        const float *crow = c_s + (la + tx) * CW + lb;
        for (int ty = ty0; ty <= ty1; ++ty) {
            const float cv = crow[ty];
            float wt[M * M];
            lds_vec<M * M>(w_s + (tx * NT + ty) * (M * M), wt);      // warp-uniform address: broadcast
#pragma unroll
            for (int i = 0; i < M; ++i)
#pragma unroll
                for (int j = 0; j < M; ++j) acc[i][j] = fmaf(wt[i * M + j], cv, acc[i][j]);
        }
    }
    if (a0 >= P.mx || b0 >= P.my) return;
    float *out = P.phi + (size_t)b * P.px * P.py;
    const int nix = P.nrm.ix(a0, 0), niy = P.nrm.iy(b0, 0);   // all m x m pixels of a control pixel share its border class
#pragma unroll
    for (int i = 0; i < M; ++i) {
        const int p = M * a0 + i;
        float *row = out + (size_t)p * P.py + M * b0;
#pragma unroll
        for (int j = 0; j < M; j += 2) {
            float2 o;
            o.x = acc[i][j] * P.nrm.at_index(nix + i, niy + j);
            o.y = acc[i][j + 1] * P.nrm.at_index(nix + i, niy + j + 1);
            *reinterpret_cast<float2 *>(row + j) = o;
        }
    }
}

// ---------------------------------------------------------------- conic, transpose (gather)
struct FilterTParams {
    const float *v;        // [B,px,py]  mask cotangent, invden applied
    float *dC;             // [B,mx,my]
    const float *w;        // as FilterParams
    const int *tyrange;
    int mx, my, px, py, T, NT;
};

// One warp per row of TB control pixels; SP lanes share a control pixel, each taking M/SP of its m phase
// rows, and reduce with xor-shuffles (4x the parallelism of one thread per pixel: the grid is only
// (mx/8) x (my/TB) CTAs).  Lane = sp*TB + lb keeps a quarter-warp on 8 neighbouring pixels, so the
// M-float reads of v are contiguous across lanes (no bank conflicts).
template <int M> struct FilterTShape {
    static constexpr int SP = (M % 4 == 0) ? 4 : 2;     // lanes per control pixel
    static constexpr int TB = 32 / SP, TA = 8, NTHR = 32 * TA, ROWS = M / SP;
};

// grid (ceil(my/TB), ceil(mx/TA), B)
template <int M>
__global__ void __launch_bounds__(FilterTShape<M>::NTHR) k_filterT_conic(const FilterTParams P)
{
    using S = FilterTShape<M>;
    constexpr int TA = S::TA, TB = S::TB, ROWS = S::ROWS, nthr = S::NTHR;
    extern __shared__ __align__(16) float sm[];
    const int T = P.T, NT = P.NT;
    const int VH = M * (TA + 2 * T), VW = M * (TB + 2 * T);   // v tile
    float *w_s = sm;                               // NT*NT*M*M
    float *v_s = w_s + NT * NT * M * M;            // VH*VW
    int *ty_s = reinterpret_cast<int *>(v_s + VH * VW);
    const int tid = threadIdx.x;
    const int a_base = blockIdx.y * TA, b_base = blockIdx.x * TB, b = blockIdx.z;

    for (int i = tid; i < NT * NT * M * M; i += nthr) w_s[i] = P.w[i];
    for (int i = tid; i < 2 * NT; i += nthr) ty_s[i] = P.tyrange[i];
    const float *vb = P.v + (size_t)b * P.px * P.py;
    const int p_base = M * (a_base - T), q_base = M * (b_base - T);
    for (int i = tid; i < VH * VW; i += nthr) {
        const int r = i / VW, c = i - r * VW;
        const int p = p_base + r, q = q_base + c;
        float x = 0.0f;
        if (p >= 0 && p < P.px && q >= 0 && q < P.py) x = vb[(size_t)p * P.py + q];
        v_s[i] = x;
    }
    __syncthreads();

    const int la = tid >> 5, lane = tid & 31, sp = lane / TB, lb = lane - sp * TB;
    const int a = a_base + la, bb = b_base + lb;
    float part[M];                                 // independent partial sums: no serial FMA chain
#pragma unroll
    for (int j = 0; j < M; ++j) part[j] = 0.0f;
    for (int tx = 0; tx < NT; ++tx) {
        const int ty0 = ty_s[2 * tx], ty1 = ty_s[2 * tx + 1];
        // forward used node a = a0 + (tx-T)  ->  source block a0 = a - (tx-T); local block la + 2T - tx
        const float *vrow = v_s + (M * (la + 2 * T - tx) + sp * ROWS) * VW;
        for (int ty = ty0; ty <= ty1; ++ty) {
            const float *vt = vrow + M * (lb + 2 * T - ty);
            float wt[ROWS * M];
            lds_vec<ROWS * M>(w_s + (tx * NT + ty) * (M * M) + sp * ROWS * M, wt);
#pragma unroll
            for (int i = 0; i < ROWS; ++i) {
                float vv[M];
                lds_vec<M>(vt + i * VW, vv);
#pragma unroll
                for (int j = 0; j < M; ++j) part[j] = fmaf(wt[i * M + j], vv[j], part[j]);
            }
        }
    }
    float acc = 0.0f;
#pragma unroll
    for (int j = 0; j < M; ++j) acc += part[j];
#pragma unroll
    for (int off = TB; off < 32; off <<= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
    if (sp == 0 && a < P.mx && bb < P.my) P.dC[((size_t)b * P.mx + a) * P.my + bb] = acc;
}

}  // namespace epsgrad
