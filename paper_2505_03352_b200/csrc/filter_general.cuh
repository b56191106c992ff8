// filter_general.cuh -- Eq. (2) and its transpose for a NON-INTEGER number of Yee cells per control pixel
// (epsgrad_config_t nx_cells / ny_cells; Fig. 4: 36 x 36 control variables on 210 x 210 cells, 5.83 cells per pixel).
// Control node a sits at x_a = ux (a + 1/2), ux = Nx/Mx (S3); mask pixel p at X_p = (p + 1/2)/s.  Without an integer ratio the
// weights have no (phase, tap) structure to tabulate, so both kernels evaluate the basis on the fly -- coordinates in float64
// (exact), the basis itself in float32:
//   forward  Phi'[p,q] = sum_ab W(X_p - x_a, Y_q - y_b) (C[a,b] - eta0) / sum_ab W(...)       one thread per mask pixel; it also
//            leaves 1/sum_ab W on a mask-sized plane, which the reverse pass reads through Normaliser::plane_py (S2);
//   reverse  dC[a,b] = sum_pq W(X_p - x_a, Y_q - y_b) v[p,q]                                  one warp per control node
//            (gather, fixed summation order: deterministic; v already carries 1/sum W).
// A coverage path, not a tuned one: the BASELINE configs have 2 cells per control pixel and take filter4.cuh / filter_sep.cuh.
#pragma once
#include "common.cuh"

namespace epsgrad {

constexpr int FG_THREADS = 256;

struct FilterGenParams {
    const float *C;        // [B,mx,my]                        (forward)
    float *phi;            // [B,px,py] centred filter output  (forward)
    float *invden;         // [px,py] 1 / sum W                (forward: written; 1 everywhere when normalize = 0)
    const float *v;        // [B,px,py] mask cotangent / den   (reverse)
    float *dC;             // [B,mx,my]                        (reverse)
    int mx, my, px, py, s;
    int kind, normalize;   // EPSGRAD_FILTER_*; density-filter form (S2)
    double ux, uy;         // Yee cells per control pixel along x, y
    float R, inv_R, inv_2s2, eta0;
};

// S1 / S11: conic max(0, 1 - r/R); Gaussian exp(-r^2 / 2 sigma^2) inside the square |dx|, |dy| <= R
__device__ __forceinline__ float fg_basis(const FilterGenParams &P, float dx, float dy)
{
    if (P.kind == 0) return fmaxf(0.0f, 1.0f - sqrtf(dx * dx + dy * dy) * P.inv_R);
    if (fabsf(dx) > P.R || fabsf(dy) > P.R) return 0.0f;
    return expf(-(dx * dx + dy * dy) * P.inv_2s2);
}

// control nodes that can reach coordinate X: |X - u (a + 1/2)| <= R, one node of slack on either side, clamped
__device__ __forceinline__ void fg_node_range(double X, double R, double u, int M, int &lo, int &hi)
{
    lo = max(0, (int)floor((X - R) / u - 0.5) - 1);
    hi = min(M - 1, (int)ceil((X + R) / u - 0.5) + 1);
}

// grid (ceil(px*py / FG_THREADS), B)
__global__ void __launch_bounds__(FG_THREADS) k_filter_general(const FilterGenParams P)
{
    const size_t n_mask = (size_t)P.px * P.py, i = (size_t)blockIdx.x * FG_THREADS + threadIdx.x;
    if (i >= n_mask) return;
    const int b = blockIdx.y, p = (int)(i / P.py), q = (int)(i - (size_t)p * P.py);
    const double X = (p + 0.5) / P.s, Y = (q + 0.5) / P.s;
    int alo, ahi, blo, bhi;
    fg_node_range(X, (double)P.R, P.ux, P.mx, alo, ahi);
    fg_node_range(Y, (double)P.R, P.uy, P.my, blo, bhi);
    const float *Cb = P.C + (size_t)b * P.mx * P.my;
    float num = 0.0f, den = 0.0f;
    for (int a = alo; a <= ahi; ++a) {
        const float dx = (float)(X - P.ux * (a + 0.5));
        for (int bb = blo; bb <= bhi; ++bb) {
            const float w = fg_basis(P, dx, (float)(Y - P.uy * (bb + 0.5)));
            num = fmaf(w, Cb[(size_t)a * P.my + bb] - P.eta0, num);      // centred: beta multiplies the rounding of Phi
            den += w;
        }
    }
    const float inv = P.normalize ? 1.0f / den : 1.0f;
    P.phi[(size_t)b * n_mask + i] = num * inv;
    if (b == 0) P.invden[i] = inv;
}

// grid (ceil(mx*my / (FG_THREADS / 32)), B): one WARP per control node -- its window of mask pixels ((2 R s + 3)^2, 35 x 35 for
// Fig. 4) is split over the lanes and the 32 partial sums are added in a fixed butterfly order (deterministic).  One thread per
// node left 1296 threads with 1225 dependent evaluations each: 246 us for Fig. 4's 36 x 36 nodes.
__global__ void __launch_bounds__(FG_THREADS) k_filterT_general(const FilterGenParams P)
{
    const int n_ctrl = P.mx * P.my, lane = threadIdx.x & 31, i = blockIdx.x * (FG_THREADS / 32) + (threadIdx.x >> 5);
    if (i >= n_ctrl) return;                       // whole warps leave
    const int b = blockIdx.y, a = i / P.my, bb = i - a * P.my;
    const double xa = P.ux * (a + 0.5), yb = P.uy * (bb + 0.5), R = (double)P.R;
    // mask pixels within reach: |(p + 1/2)/s - x_a| <= R, one pixel of slack, clamped (the basis is zero beyond its support)
    const int plo = max(0, (int)floor((xa - R) * P.s - 0.5) - 1), phi_ = min(P.px - 1, (int)ceil((xa + R) * P.s - 0.5) + 1);
    const int qlo = max(0, (int)floor((yb - R) * P.s - 0.5) - 1), qhi = min(P.py - 1, (int)ceil((yb + R) * P.s - 0.5) + 1);
    const int nq = qhi - qlo + 1, n_win = (phi_ - plo + 1) * nq;
    const float *vb = P.v + (size_t)b * P.px * P.py;
    const double inv_s = 1.0 / P.s;                // a multiplication per pixel instead of a float64 division (1 ulp of float64 apart at most)
    float acc = 0.0f;
    for (int k = lane; k < n_win; k += 32) {
        const int kp = k / nq, p = plo + kp, q = qlo + (k - kp * nq);
        acc = fmaf(fg_basis(P, (float)((p + 0.5) * inv_s - xa), (float)((q + 0.5) * inv_s - yb)), vb[(size_t)p * P.py + q], acc);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) P.dC[(size_t)b * n_ctrl + i] = acc;
}

}  // namespace epsgrad
