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

// The two passes along x read and write whole mask rows, so a thread owns one mask column q (coalesced across the warp) and
// register-blocks SEPX_NBA consecutive control rows: an input value loaded once from L2 feeds SEPX_NBA * M FMAs, the
// weights come from a zero-padded shared table as one 16-byte broadcast per (row, output) -- no staging of the input, no
// bounds tests in the inner loop.  (The first version staged an 8-row tile with a 2T-row halo in shared memory: 5x
// redundant loads and 1.25 shared-memory reads per FMA; 656 + 1003 us on the Wide-batch config.)
constexpr int SEPX_NBA = 16, SEPX_THREADS = 128;

__host__ __device__ inline size_t sepx_smem_floats(int NT, int M) { return (size_t)(NT + 2 * (SEPX_NBA - 1) + 4) * M; }

// weights w1[t][0..M) for t in [-(NBA-1), NT+NBA-1), zero outside [0,NT)
template <int M>
__device__ __forceinline__ void sepx_load_weights(const SepParams &P, float *w_pad)
{
    const int n = (P.NT + 2 * (SEPX_NBA - 1) + 4) * M;        // 4 spare entries for the row unrolling of up_x
    for (int i = threadIdx.x; i < n; i += SEPX_THREADS) {
        const int t = i / M - (SEPX_NBA - 1);
        w_pad[i] = (t >= 0 && t < P.NT) ? P.w1[t * M + (i % M)] : 0.0f;
    }
    __syncthreads();
}

// up_x: grid (ceil(py/128), ceil(mx/NBA), B), 128 threads; Phi'[M a0 + f][q] = invden * sum_t w1[t][f] tmp[a0 + t - T][q]
template <int M>
__global__ void __launch_bounds__(SEPX_THREADS) k_sep_up_x(const SepParams P)
{
    static_assert(M % 2 == 0, "even phases");
    extern __shared__ __align__(16) float w_pad[];
    constexpr int NBA = SEPX_NBA;
    sepx_load_weights<M>(P, w_pad);
    const int T = P.T;
    const int q = blockIdx.x * SEPX_THREADS + threadIdx.x, a_base = blockIdx.y * NBA, b = blockIdx.z;
    if (q >= P.py) return;
    const float *tb = P.in + (size_t)b * P.mx * P.py + q;
    float acc[NBA][M];
#pragma unroll
    for (int ja = 0; ja < NBA; ++ja)
#pragma unroll
        for (int f = 0; f < M; ++f) acc[ja][f] = 0.0f;
    // input row r = a_base - T + rr feeds output a_base + ja through tap t = rr - ja
    const int r_lo = max(a_base - T, 0), r_hi = min(a_base + NBA - 1 + T, P.mx - 1);
    for (int r0 = r_lo; r0 <= r_hi; r0 += 4) {
        float x[4];                                            // four input rows in flight
#pragma unroll
        for (int u = 0; u < 4; ++u) x[u] = r0 + u <= r_hi ? tb[(size_t)(r0 + u) * P.py] : 0.0f;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            // rows past r_hi carry x = 0 and read weights inside the padded table (r_hi + 3 - (a_base - T) + NBA - 1 < NT + 2 NBA)
            const float *wr = w_pad + (size_t)(r0 + u - (a_base - T) + NBA - 1) * M;   // entry of ja = 0; ja steps back M floats
#pragma unroll
            for (int ja = 0; ja < NBA; ++ja) {
                float wv[M];
                lds_vec<M>(wr - ja * M, wv);
#pragma unroll
                for (int f = 0; f < M; ++f) acc[ja][f] = fmaf(wv[f], x[u], acc[ja][f]);
            }
        }
    }
    float *ob = P.out + (size_t)b * P.px * P.py + q;
    const int niy = P.nrm.iy_of(q);
#pragma unroll
    for (int ja = 0; ja < NBA; ++ja) {
        const int a0 = a_base + ja;
        if (a0 >= P.mx) break;
#pragma unroll
        for (int f = 0; f < M; ++f) {
            const int p = M * a0 + f;
            ob[(size_t)p * P.py] = acc[ja][f] * P.nrm.at_index(P.nrm.ix(a0, f), niy);
        }
    }
}

// down_x: grid (ceil(py/128), ceil(mx/NBA), B), 128 threads; tmpT[a][q] = sum_{t,f} w1[t][f] v[M (a - t + T) + f][q]
template <int M>
__global__ void __launch_bounds__(SEPX_THREADS) k_sep_down_x(const SepParams P)
{
    extern __shared__ __align__(16) float w_pad[];
    constexpr int NBA = SEPX_NBA;
    sepx_load_weights<M>(P, w_pad);
    const int T = P.T;
    const int q = blockIdx.x * SEPX_THREADS + threadIdx.x, a_base = blockIdx.y * NBA, b = blockIdx.z;
    if (q >= P.py) return;
    const float *vb = P.in + (size_t)b * P.px * P.py + q;
    float acc[NBA];
#pragma unroll
    for (int ja = 0; ja < NBA; ++ja) acc[ja] = 0.0f;
    // source block a' (mask rows M a' .. M a' + M - 1) reaches output a = a_base + ja through tap t = a - a' + T = ja - rr + NBA-1 + ... (below)
    const int s_lo = max(a_base - T, 0), s_hi = min(a_base + NBA - 1 + T, P.mx - 1);
    for (int ap = s_lo; ap <= s_hi; ++ap) {
        float x[M];
#pragma unroll
        for (int f = 0; f < M; ++f) x[f] = vb[(size_t)(M * ap + f) * P.py];
        // t = a_base + ja - ap + T; padded index t + NBA - 1
        const float *wr = w_pad + (size_t)(a_base - ap + T + NBA - 1) * M;       // entry of ja = 0; ja steps forward M floats
#pragma unroll
        for (int ja = 0; ja < NBA; ++ja) {
            float wv[M];
            lds_vec<M>(wr + ja * M, wv);
#pragma unroll
            for (int f = 0; f < M; ++f) acc[ja] = fmaf(wv[f], x[f], acc[ja]);
        }
    }
    float *ob = P.out + (size_t)b * P.mx * P.py + q;
#pragma unroll
    for (int ja = 0; ja < NBA; ++ja)
        if (a_base + ja < P.mx) ob[(size_t)(a_base + ja) * P.py] = acc[ja];
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
