// morph.cuh -- morphological filters of the design mask, Eqs. (4)-(5), forward and transposed.
//   dilate  y = (1/alpha) log sum K_m exp(alpha x)              erode  y = 1 - (1/alpha) log sum K_m exp(alpha (1 - x))
// K_m = 1 inside a circle of diameter d, normalised to unit sum over the pixels inside the region (G5, S18), finite
// sums on the mask grid as in Eq. (8).  With a signed alpha both are ONE formula,
//   y_i = (1/a) log( (1/N_i) sum_{j in disk(i)} exp(a x_j) ),      a = +alpha: dilate,  a = -alpha: erode,
// and so is the transpose (the disk is symmetric, N cancels out of d y_i / d x_j = exp(a x_j) / S_i):
//   xbar_j = sum_{i in disk(j)} ybar_i exp(a (x_j - y_i)) / N_i    (exponent bounded by log N: no overflow).
// Both directions are the same skeleton -- stage f(pixel) for a tile plus a halo of R pixels (0 outside the region), sum it
// over the disk, finish per pixel -- so one kernel serves the four forward and the four transposed operations of the chain
// "dilate, erode, erode, dilate" (S17), with the neighbouring pointwise steps folded in at the chain ends:
//   first forward op  stages exp(a rho0) with rho0 = projection (Eq. (3)/(6) form, S9) of the filter output, and keeps rho0;
//   last forward op   writes y - 1/2, the centred input of the second projection, Eq. (6);
//   last transposed op multiplies by the slope of the first projection and by 1/den (S2): the mask cotangent v of filterT.
// Between the ops of the chain the masks are kept in "z-space": op k stores z_k = (1/N) sum exp(a_k x) instead of
// y_k = log(z_k)/a_k, because the next op only needs exp(a_{k+1} y_k) = z_k^(a_{k+1}/a_k) = z_k or 1/z_k (|a| = alpha for all
// four ops), and the transposed ops only exp(-a_k y_k) = 1/z_k: six of the eight launches run without exp or log, and the
// log/exp round trip's rounding disappears.  Only the chain's first input (rho0) and last output (rho~) are real masks.
// A thread owns four neighbouring pixels of a row: the part of a disk row that their four windows share is summed once
// (plain adds: no sliding-window subtraction, the staged values span e^-20..e^20).  Bound: shared-memory reads and FADD issue; L2-resident.
#pragma once
#include "common.cuh"
#include "sizes.cuh"
#include "reduce.cuh"

namespace epsgrad {


struct MorphParams {
    const float *x;        // [B,px,py] input of the forward op: first op: centred filter output Phi'; later ops: z of the previous op
    const float *y;        // transposed op: output of the forward op: z of this op; last op of the chain: the centred mask y - 1/2
    const float *ybar;     // transposed op: cotangent of y
    float *out;            // forward: z of this op (last op: y - 1/2); transposed: xbar (first op of the chain: v)
    float *rho0;           // first forward op: keeps rho0 = projection(Phi') for the transposed pass
    float *dbeta_part;     // first op, transposed: nullptr, or one partial sum of d F/d beta per CTA (first projection; reduce.cuh)
    const int *hl;         // [2R+1] half-lengths of the disk rows
    const float *invn;     // [(2R+1)^2] 1/N by border class (rows, columns)
    Normaliser nrm;        // first op of the chain, transposed: 1/den of Eq. (2)
    int px, py, R;
    int transposed, first, last;
    int x_inv;             // ops after the first: exp(a x) = 1/z_prev (the sign of alpha flipped) instead of z_prev
    float a;               // signed alpha
    float beta, eta_r;     // first projection (first op only)
};

__host__ __device__ inline size_t morph_smem_floats(int R) { return (size_t)(MO_T + 2 * R) * (MO_T + 2 * R + 1) + 2 * R + 1; }

// border class of pixel p along an axis of n pixels (n >= 2R+1): distance to the nearer edge, capped at R
__device__ __forceinline__ int morph_class(int p, int n, int R)
{
    if (p < R) return p;
    const int d = n - 1 - p;
    return d < R ? 2 * R - d : R;
}

// grid (ceil(py/32), ceil(px/32), B)
__global__ void __launch_bounds__(MO_THREADS) k_morph(const __grid_constant__ MorphParams P)
{
    extern __shared__ __align__(16) float sm[];
    const int R = P.R, W = MO_T + 2 * R, pitch = W + 1;
    float *f_s = sm;                                       // [W][pitch]
    int *hl_s = reinterpret_cast<int *>(f_s + W * pitch);  // [2R+1]
    const int tid = threadIdx.x, b = blockIdx.z;
    const int p0 = blockIdx.y * MO_T, q0 = blockIdx.x * MO_T;
    const size_t plane = (size_t)b * P.px * P.py;
    const float a = P.a;
    const int NI = 2 * R + 1;

    for (int k = tid; k < NI; k += MO_THREADS) hl_s[k] = P.hl[k];
    // ---- stage f over the tile + halo (flat index, advanced without divisions)
    {
        int lp = tid / W, lq = tid - lp * W;
        const int dlp = MO_THREADS / W, dlq = MO_THREADS - dlp * W;
        for (int it = tid; it < W * W; it += MO_THREADS) {
            const int p = p0 - R + lp, q = q0 - R + lq;
            float f = 0.0f;
            if (p >= 0 && p < P.px && q >= 0 && q < P.py) {
                const size_t idx = plane + (size_t)p * P.py + q;
                if (!P.transposed) {
                    float xv = P.x[idx];
                    if (P.first) {
                        // rho0 = 1/2 (1 + tanh(beta (Phi - eta))) = 1/(1 + exp(-2t))
                        const float t = P.beta * (xv - P.eta_r);
                        xv = fast_rcp(1.0f + __expf(-2.0f * t));
                        if (lp >= R && lp < R + MO_T && lq >= R && lq < R + MO_T) P.rho0[idx] = xv;
                        f = __expf(a * xv);
                    } else {
                        f = P.x_inv ? fast_rcp(xv) : xv;          // exp(a y_prev) = z_prev^(+-1)
                    }
                } else {
                    // exp(-a y) = 1/z of this op; the last op kept the real mask (centred): one exponential
                    const float iz = P.last ? __expf(-a * (P.y[idx] + 0.5f)) : fast_rcp(P.y[idx]);
                    f = P.ybar[idx] * iz * P.invn[morph_class(p, P.px, R) * NI + morph_class(q, P.py, R)];
                }
            }
            f_s[lp * pitch + lq] = f;
            lp += dlp; lq += dlq;
            if (lq >= W) { lq -= W; ++lp; }
        }
    }
    __syncthreads();

    // ---- disk sums: thread -> row r, columns 4 c4 .. 4 c4 + 3
    const int r = tid >> 3, c4 = (tid & 7) << 2;
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    for (int dp = -R; dp <= R; ++dp) {
        const int h = hl_s[dp + R];
        const float *row = f_s + (r + R + dp) * pitch + c4 + R - h;     // first element of the run of pixel c4
        const int n = 2 * h + 1;
        if (n >= 4) {
            // the four windows [u, u+n) share the elements 3 .. n-1: sum them once, then add each window's own three
            float c = 0.f;
            for (int k = 3; k < n; ++k) c += row[k];
            const float v0 = row[0], v1 = row[1], v2 = row[2], w0 = row[n], w1 = row[n + 1], w2 = row[n + 2];
            acc[0] += c + ((v0 + v1) + v2);
            acc[1] += c + ((v1 + v2) + w0);
            acc[2] += c + ((v2 + w0) + w1);
            acc[3] += c + ((w0 + w1) + w2);
        } else {
#pragma unroll
            for (int u = 0; u < 4; ++u)
                for (int k = 0; k < n; ++k) acc[u] += row[u + k];
        }
    }
    // ---- finish per pixel
    const int p = p0 + r;
    const float inv_a = 1.0f / a;
    float db = 0.f;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int q = q0 + c4 + u;
        if (p >= P.px || q >= P.py) continue;
        const size_t idx = plane + (size_t)p * P.py + q;
        if (!P.transposed) {
            const float invn = P.invn[morph_class(p, P.px, R) * NI + morph_class(q, P.py, R)];
            const float z = acc[u] * invn;
            P.out[idx] = P.last ? __logf(z) * inv_a - 0.5f : z;
        } else {
            const float xv = P.first ? P.rho0[idx] : P.x[idx];
            float o = acc[u] * (P.first ? __expf(a * xv) : (P.x_inv ? fast_rcp(xv) : xv));     // exp(a x) as in the forward staging
            if (P.first) {
                // first op of the chain: projection^T in the overflow-free analytic form, then 1/den (S2);
                // the same cotangent gives the first projection's share of d F/d beta: Phibar (Phi - eta)/beta
                const float phi = P.x[idx];
                o *= project_slope(phi, P.beta, P.eta_r);
                db = fmaf(o, phi - P.eta_r, db);
                o *= P.nrm.at(p, q);
            }
            P.out[idx] = o;
        }
    }
    if (P.dbeta_part) {                                        // block-uniform; first transposed op only
        const float sdb = block_sum(db, f_s);                  // f_s is dead past block_sum's first barrier
        if (tid == 0) P.dbeta_part[(size_t)b * gridDim.y * gridDim.x + blockIdx.y * gridDim.x + blockIdx.x] = sdb / P.beta;
    }
}

}  // namespace epsgrad
