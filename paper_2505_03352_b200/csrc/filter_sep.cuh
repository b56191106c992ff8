// filter_sep.cuh -- Eq. (2) for a separable basis (Gaussian truncated per axis, S11):
// W(dx,dy) = w1(dx) w1(dy), so the polyphase stencil factors into a pass along y and a
// pass along x (32+32 taps instead of 1024 at sigma = 10, R = 32).
//   up_y   : C   [B,mx,my] -> tmp [B,mx,py]   tmp[a][m b0+f]  = sum_t w1[t][f] c'[a][b0+t-T]
//   up_x   : tmp [B,mx,py] -> Phi'[B,px,py]   Phi'[m a0+f][q] = invden * sum_t w1[t][f] tmp[a0+t-T][q]
//   down_x : v   [B,px,py] -> tmpT[B,mx,py]   tmpT[a][q] = sum_{t,f} w1[t][f] v[m(a-t+T)+f][q]
//   down_y : tmpT[B,mx,py] -> dC  [B,mx,my]   dC[a][b]   = sum_{t,f} w1[t][f] tmpT[a][m(b-t+T)+f]
#pragma once
#include "common.cuh"

namespace epsgrad {

struct SepParams {
    const float *in;
    float *out;
    const float *w1;       // [NT][m]
    Normaliser nrm;        // used by up_x only
    int mx, my, px, py, T, NT;
    float eta0;            // used by up_y only
};

constexpr int SEP_THREADS = 256;

// grid (ceil(my/32), ceil(mx/8), B); thread <-> (a, b0): M outputs along y
template <int M>
__global__ void __launch_bounds__(SEP_THREADS) k_sep_up_y(const SepParams P)
{
    extern __shared__ __align__(16) float sm[];
    constexpr int TA = 8, TB = 32;
    const int T = P.T, NT = P.NT, CW = TB + 2 * T;
    float *w_s = sm;                   // NT*M
    float *c_s = w_s + NT * M;         // TA*CW
    const int tid = threadIdx.x;
    const int a_base = blockIdx.y * TA, b_base = blockIdx.x * TB, b = blockIdx.z;
    for (int i = tid; i < NT * M; i += SEP_THREADS) w_s[i] = P.w1[i];
    const float *Cb = P.in + (size_t)b * P.mx * P.my;
    for (int i = tid; i < TA * CW; i += SEP_THREADS) {
        const int r = i / CW, c = i - r * CW;
        const int a = a_base + r, bb = b_base - T + c;
        c_s[i] = (a < P.mx && bb >= 0 && bb < P.my) ? Cb[(size_t)a * P.my + bb] - P.eta0 : 0.0f;
    }
    __syncthreads();
    const int la = tid / TB, lb = tid - la * TB;
    const int a = a_base + la, b0 = b_base + lb;
    float acc[M];
#pragma unroll
    for (int f = 0; f < M; ++f) acc[f] = 0.0f;
    const float *crow = c_s + la * CW + lb;
    for (int t = 0; t < NT; ++t) {
        const float cv = crow[t];
#pragma unroll
        for (int f = 0; f < M; ++f) acc[f] = fmaf(w_s[t * M + f], cv, acc[f]);
    }
    if (a >= P.mx || b0 >= P.my) return;
    float *o = P.out + ((size_t)b * P.mx + a) * P.py + M * b0;
#pragma unroll
    for (int f = 0; f < M; f += 2) *reinterpret_cast<float2 *>(o + f) = make_float2(acc[f], acc[f + 1]);
}

// grid (ceil(py/128), ceil(mx/8), B); thread <-> (a0, q) x 4: M outputs along x
template <int M>
__global__ void __launch_bounds__(SEP_THREADS) k_sep_up_x(const SepParams P)
{
    extern __shared__ __align__(16) float sm[];
    constexpr int TA = 8, TQ = 128;
    const int T = P.T, NT = P.NT, RH = TA + 2 * T;
    float *w_s = sm;                   // NT*M
    float *t_s = w_s + NT * M;         // RH*TQ
    const int tid = threadIdx.x;
    const int a_base = blockIdx.y * TA, q_base = blockIdx.x * TQ, b = blockIdx.z;
    for (int i = tid; i < NT * M; i += SEP_THREADS) w_s[i] = P.w1[i];
    const float *tb = P.in + (size_t)b * P.mx * P.py;
    for (int i = tid; i < RH * TQ; i += SEP_THREADS) {
        const int r = i / TQ, c = i - r * TQ;
        const int a = a_base - T + r, q = q_base + c;
        t_s[i] = (a >= 0 && a < P.mx && q < P.py) ? tb[(size_t)a * P.py + q] : 0.0f;
    }
    __syncthreads();
    float *ob = P.out + (size_t)b * P.px * P.py;
    for (int it = tid; it < TA * TQ; it += SEP_THREADS) {
        const int la = it / TQ, lq = it - la * TQ;
        const int a0 = a_base + la, q = q_base + lq;
        float acc[M];
#pragma unroll
        for (int f = 0; f < M; ++f) acc[f] = 0.0f;
        for (int t = 0; t < NT; ++t) {
            const float x = t_s[(la + t) * TQ + lq];
#pragma unroll
            for (int f = 0; f < M; ++f) acc[f] = fmaf(w_s[t * M + f], x, acc[f]);
        }
        if (a0 < P.mx && q < P.py) {
#pragma unroll
            for (int f = 0; f < M; ++f) {
                const int p = M * a0 + f;
                ob[(size_t)p * P.py + q] = acc[f] * P.nrm.at(p, q);
            }
        }
    }
}

// grid (ceil(py/64), ceil(mx/8), B); thread <-> (a, q) x 2
template <int M>
__global__ void __launch_bounds__(SEP_THREADS) k_sep_down_x(const SepParams P)
{
    extern __shared__ __align__(16) float sm[];
    constexpr int TA = 8, TQ = 64;
    const int T = P.T, NT = P.NT, RH = M * (TA + 2 * T);
    float *w_s = sm;                   // NT*M
    float *v_s = w_s + NT * M;         // RH*TQ
    const int tid = threadIdx.x;
    const int a_base = blockIdx.y * TA, q_base = blockIdx.x * TQ, b = blockIdx.z;
    for (int i = tid; i < NT * M; i += SEP_THREADS) w_s[i] = P.w1[i];
    const float *vb = P.in + (size_t)b * P.px * P.py;
    const int p_base = M * (a_base - T);
    for (int i = tid; i < RH * TQ; i += SEP_THREADS) {
        const int r = i / TQ, c = i - r * TQ;
        const int p = p_base + r, q = q_base + c;
        v_s[i] = (p >= 0 && p < P.px && q < P.py) ? vb[(size_t)p * P.py + q] : 0.0f;
    }
    __syncthreads();
    float *ob = P.out + (size_t)b * P.mx * P.py;
    for (int it = tid; it < TA * TQ; it += SEP_THREADS) {
        const int la = it / TQ, lq = it - la * TQ;
        const int a = a_base + la, q = q_base + lq;
        float acc = 0.0f;
        for (int t = 0; t < NT; ++t) {
            const float *vr = v_s + (M * (la + 2 * T - t)) * TQ + lq;
#pragma unroll
            for (int f = 0; f < M; ++f) acc = fmaf(w_s[t * M + f], vr[f * TQ], acc);
        }
        if (a < P.mx && q < P.py) ob[(size_t)a * P.py + q] = acc;
    }
}

// grid (ceil(my/32), ceil(mx/8), B); thread <-> (a, b)
template <int M>
__global__ void __launch_bounds__(SEP_THREADS) k_sep_down_y(const SepParams P)
{
    extern __shared__ __align__(16) float sm[];
    constexpr int TA = 8, TB = 32;
    const int T = P.T, NT = P.NT, VW = M * (TB + 2 * T);
    float *w_s = sm;                   // NT*M
    float *v_s = w_s + NT * M;         // TA*VW
    const int tid = threadIdx.x;
    const int a_base = blockIdx.y * TA, b_base = blockIdx.x * TB, b = blockIdx.z;
    for (int i = tid; i < NT * M; i += SEP_THREADS) w_s[i] = P.w1[i];
    const float *tb = P.in + (size_t)b * P.mx * P.py;
    const int q_base = M * (b_base - T);
    for (int i = tid; i < TA * VW; i += SEP_THREADS) {
        const int r = i / VW, c = i - r * VW;
        const int a = a_base + r, q = q_base + c;
        v_s[i] = (a < P.mx && q >= 0 && q < P.py) ? tb[(size_t)a * P.py + q] : 0.0f;
    }
    __syncthreads();
    const int la = tid / TB, lb = tid - la * TB;
    const int a = a_base + la, bb = b_base + lb;
    if (a >= P.mx || bb >= P.my) return;
    float acc = 0.0f;
    const float *vr = v_s + la * VW;
    for (int t = 0; t < NT; ++t) {
        const float *vt = vr + M * (lb + 2 * T - t);
#pragma unroll
        for (int f = 0; f < M; ++f) acc = fmaf(w_s[t * M + f], vt[f], acc);
    }
    P.out[((size_t)b * P.mx + a) * P.my + bb] = acc;
}

}  // namespace epsgrad
