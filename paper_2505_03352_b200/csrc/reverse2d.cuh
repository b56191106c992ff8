// reverse2d.cuh -- R2..R5 of the reverse pass in gather form, one tile kernel:
// from the z-reduced cotangent gbar [B,5,nx,ny] to the mask cotangent
//   v[p,q] = Phibar[p,q] / den[p,q]
// that the transposed filter (R6) gathers.  The forward residuals are recomputed from
// the centred filter output Phi' (cheap: the 2-D chain is ALU-light and L2-resident).
//   R2  Eq. (7)^T:  q = 1/eps2d, qbar = -gbar/q^2, Hbar = n^2 qbar,
//                            Abar = -(1-n^2) qbar/A^2, n2bar = (H - 1/A) qbar
//   R3  normals^T:  gbar_c, gbar_o from n2bar; Dbar = Sobel^T with the replicate
//                            padding folded back at the borders; Abar += Dbar/deps
//   R4  averages^T: each mask pixel gathers from the E_x, E_y, E_z cells
//                            whose footprint holds it (clamped last pixel counted s/2+1 times)
//   R5  mixing^T, projection^T: rhobar = deps (ebar - rbar/e^2),
//                            Phibar = rhobar * (beta/2) sech^2 t   (stable form)
// Dependency cone of a TI x TJ tile: cotangents on a 1-cell ring (E_x/E_y owners), their
// Sobel^T on a 2-cell ring, forward A,H on a 3-cell ring (+ the half-cell shift).
#pragma once
#include "common.cuh"

namespace epsgrad {

struct Rev2dParams {
    const float *phi;      // [B,px,py]
    const float *gbar;     // [B,5,nx,ny]
    float *v;              // [B,px,py]
    Normaliser nrm;
    int nx, ny, px, py, s;
    float beta, eta_r, eps_clad, deps, delta;
    float w_lo, w_hi;      // fractional z-face weights of eps_zz (0 if that face cell is absent)
};

constexpr int REV_TI = 16, REV_TJ = 16, REV_THREADS = 256;
constexpr int REV_CI = REV_TI + 5, REV_CJ = REV_TJ + 5;

__host__ __device__ inline size_t rev_smem_floats(int s)
{
    const int MP = s * REV_CI + s / 2, MQ = s * REV_CJ + s / 2;
    return (size_t)2 * MP * MQ + 14 * REV_CI * REV_CJ + REV_TI * REV_TJ + (size_t)s * (REV_TI + REV_TJ);
}

// d eps_zz / d eps2d_z on a face cell of weight w:  w (eps_zz/v)^2, eps_zz/v = 1/(w + (1-w) v/eps_clad)
__device__ __forceinline__ float face_factor(float w, float v, float inv_ec)
{
    const float f = fast_rcp(w + (1.0f - w) * v * inv_ec);
    return w * f * f;
}

// grid (ceil(ny/TJ), ceil(nx/TI), B).  S > 0: compile-time subpixel count; S = 0: runtime P.s.
template <int S>
__global__ void __launch_bounds__(REV_THREADS) k_reverse2d(const Rev2dParams P)
{
    extern __shared__ __align__(16) float sm[];
    constexpr int TI = REV_TI, TJ = REV_TJ, NTH = REV_THREADS, CI = REV_CI, CJ = REV_CJ, NC = CI * CJ;
    const int s = S > 0 ? S : P.s, hs = s >> 1;
    const int MP = s * CI + hs, MQ = s * CJ + hs;
    float *e_s = sm;
    float *r_s = e_s + MP * MQ;
    float *A[2], *H[2], *Hb[2], *Ab[2], *Gx[2], *Gy[2], *AbF[2];
    float *ptr = r_s + MP * MQ;
    for (int c = 0; c < 2; ++c) {
        A[c] = ptr; H[c] = ptr + NC; Hb[c] = ptr + 2 * NC; Ab[c] = ptr + 3 * NC;
        Gx[c] = ptr + 4 * NC; Gy[c] = ptr + 5 * NC; AbF[c] = ptr + 6 * NC;
        ptr += 7 * NC;
    }
    float *AbZ = ptr;                  // [TI*TJ]
    int *nidx = reinterpret_cast<int *>(AbZ + TI * TJ);   // normaliser table row of each tile mask row, then column of each mask column

    const int tid = threadIdx.x;
    const int i0 = blockIdx.y * TI, j0 = blockIdx.x * TJ, b = blockIdx.z;
    const int oi = i0 - 3, oj = j0 - 3;            // cell origin of the staged arrays
    const int nx = P.nx, ny = P.ny, ncol = nx * ny;
    const float inv_s2 = 1.0f / (float)(s * s), inv_deps = 1.0f / P.deps, inv_ec = 1.0f / P.eps_clad;
    const float *phib = P.phi + (size_t)b * P.px * P.py;
    const float *gb = P.gbar + (size_t)b * 5 * ncol;
    // tile whose 3-cell ring lies inside the region: no clamping, no folded border terms (block-uniform)
    const bool inner = i0 >= 3 && j0 >= 3 && i0 + TI + 2 <= nx - 1 && j0 + TJ + 2 <= ny - 1;

    for (int k = tid; k < s * (TI + TJ); k += NTH) {
        const int along_x = k < s * TI;
        const int pix = along_x ? s * i0 + k : s * j0 + (k - s * TI);
        nidx[k] = along_x ? P.nrm.ix_of(min(pix, P.px - 1)) : P.nrm.iy_of(min(pix, P.py - 1));
    }
    // ---- A: mask tile e, r (replicate)
    {
        const int p_base = s * oi, q_base = s * oj;
        for (int i = tid; i < MP * MQ; i += NTH) {
            const int lp = i / MQ, lq = i - lp * MQ;
            const int p = clampi(p_base + lp, 0, P.px - 1), q = clampi(q_base + lq, 0, P.py - 1);
            const float e = project_mix(phib[p * P.py + q], P.beta, P.eta_r, P.eps_clad, P.deps);
            e_s[i] = e;
            r_s[i] = fast_rcp(e);
        }
    }
    __syncthreads();

    // ---- B: forward averages A_c, H_c (c = x,y) on the 3-cell ring
    for (int i = tid; i < NC; i += NTH) {
        const int ci = i / CJ, cj = i - ci * CJ;
        const int lp0 = s * ci, lq0 = s * cj;
        float ax = 0.f, hx = 0.f, ay = 0.f, hy = 0.f;
        for (int a = 0; a < s; ++a)
            for (int bb = 0; bb < s; ++bb) {
                const int ix = (lp0 + hs + a) * MQ + lq0 + bb;
                const int iy = (lp0 + a) * MQ + lq0 + hs + bb;
                ax += e_s[ix]; hx += r_s[ix];
                ay += e_s[iy]; hy += r_s[iy];
            }
        A[0][i] = ax * inv_s2; H[0][i] = hx * inv_s2;
        A[1][i] = ay * inv_s2; H[1][i] = hy * inv_s2;
    }
    __syncthreads();

    // ---- C: R2 + first half of R3 on the 2-cell ring: Hbar, Abar, gxbar, gybar per component
    {
        constexpr int RI = TI + 3, RJ = TJ + 3;           // cells ci in [1, TI+3], cj in [1, TJ+3]
        for (int it = tid; it < 2 * RI * RJ; it += NTH) {
            const int c = it / (RI * RJ), rem = it - c * (RI * RJ);
            const int ci = 1 + rem / RJ, cj = 1 + rem % RJ, i_ = ci * CJ + cj;
            const int i = oi + ci, j = oj + cj;
            float hb = 0.f, ab = 0.f, gxb = 0.f, gyb = 0.f;
            if (inner || (i >= 0 && i < nx && j >= 0 && j < ny)) {
                const float *Ac = A[c];
                float gx, gy;
                if (inner) {
                    const float *q0 = Ac + i_ - CJ, *q1 = Ac + i_, *q2 = Ac + i_ + CJ;
                    const float a00 = q0[-1], a01 = q0[0], a02 = q0[1], a10 = q1[-1], a12 = q1[1];
                    const float a20 = q2[-1], a21 = q2[0], a22 = q2[1];
                    gx = ((a20 - a00) + 2.0f * (a21 - a01) + (a22 - a02)) * 0.125f;
                    gy = ((a02 - a00) + 2.0f * (a12 - a10) + (a22 - a20)) * 0.125f;
                } else {
                    gx = 0.f; gy = 0.f;
#pragma unroll
                    for (int di = -1; di <= 1; ++di)
#pragma unroll
                        for (int dj = -1; dj <= 1; ++dj) {
                            const int ni = clampi(i + di, 0, nx - 1) - oi, nj = clampi(j + dj, 0, ny - 1) - oj;
                            const float d = Ac[ni * CJ + nj];
                            gx = fmaf((float)(di * (2 - (dj < 0 ? -dj : dj))) * 0.125f, d, gx);
                            gy = fmaf((float)(dj * (2 - (di < 0 ? -di : di))) * 0.125f, d, gy);
                        }
                }
                gx *= inv_deps; gy *= inv_deps;
                const float gc = c == 0 ? gx : gy, go = c == 0 ? gy : gx;
                const float rS = fast_rcp(gc * gc + go * go + P.delta);
                const float n2 = gc * gc * rS;
                const float ra = fast_rcp(Ac[i_]), h = H[c][i_];
                const float e2d = fast_rcp(n2 * h + (1.0f - n2) * ra);       // eps2d_c = 1/q
                const float G = gb[c * ncol + i * ny + j];
                const float qbar = -G * e2d * e2d;
                hb = n2 * qbar;
                ab = -(1.0f - n2) * qbar * ra * ra;
                const float n2bar = (h - ra) * qbar;
                const float k2 = 2.0f * n2bar * gc * rS * rS;
                const float gcb = k2 * (go * go + P.delta), gob = -k2 * gc * go;
                gxb = c == 0 ? gcb : gob;
                gyb = c == 0 ? gob : gcb;
            }
            Hb[c][i_] = hb; Ab[c][i_] = ab; Gx[c][i_] = gxb; Gy[c][i_] = gyb;
        }
    }
    __syncthreads();

    // ---- D: Sobel^T with the replicate padding folded back (second half of R3); z component
    {
        constexpr int RI = TI + 1, RJ = TJ + 1;           // cells ci in [2, TI+2], cj in [2, TJ+2]
        for (int it = tid; it < 2 * RI * RJ; it += NTH) {
            const int c = it / (RI * RJ), rem = it - c * (RI * RJ);
            const int ci = 2 + rem / RJ, cj = 2 + rem % RJ, i_ = ci * CJ + cj;
            const int ii = oi + ci, jj = oj + cj;
            float out = 0.f;
            if (inner || (ii >= 0 && ii < nx && jj >= 0 && jj < ny)) {
                float dbar = 0.f;
                const float *gxs = Gx[c], *gys = Gy[c];
                if (inner || (ii >= 1 && ii <= nx - 2 && jj >= 1 && jj <= ny - 2)) {
                    // interior: the cell (ii-di, jj-dj) reached (ii,jj) through its stencil entry (di,dj)
#pragma unroll
                    for (int di = -1; di <= 1; ++di)
#pragma unroll
                        for (int dj = -1; dj <= 1; ++dj) {
                            const int src = i_ - di * CJ - dj;
                            const float kx = (float)(di * (2 - (dj < 0 ? -dj : dj))) * 0.125f;
                            const float ky = (float)(dj * (2 - (di < 0 ? -di : di))) * 0.125f;
                            dbar = fmaf(kx, gxs[src], fmaf(ky, gys[src], dbar));
                        }
                } else {
                    // border: sources (i,di) with clamp(i+di) == ii: i = ii-di in range, plus the folded terms
                    for (int cx = 0; cx < 5; ++cx) {
                        int di, i;
                        if (cx < 3) { di = cx - 1; i = ii - di; if (i < 0 || i >= nx) continue; }
                        else if (cx == 3) { if (ii != 0) continue; di = -1; i = 0; }
                        else { if (ii != nx - 1) continue; di = 1; i = nx - 1; }
                        for (int cy = 0; cy < 5; ++cy) {
                            int dj, j;
                            if (cy < 3) { dj = cy - 1; j = jj - dj; if (j < 0 || j >= ny) continue; }
                            else if (cy == 3) { if (jj != 0) continue; dj = -1; j = 0; }
                            else { if (jj != ny - 1) continue; dj = 1; j = ny - 1; }
                            const int src = (i - oi) * CJ + (j - oj);
                            const float kx = (float)(di * (2 - (dj < 0 ? -dj : dj))) * 0.125f;
                            const float ky = (float)(dj * (2 - (di < 0 ? -di : di))) * 0.125f;
                            dbar = fmaf(kx, gxs[src], fmaf(ky, gys[src], dbar));
                        }
                    }
                }
                out = Ab[c][i_] + dbar * inv_deps;
            }
            AbF[c][i_] = out;
        }
    }
    for (int it = tid; it < TI * TJ; it += NTH) {
        const int ti = it / TJ, tj = it - ti * TJ;
        const int i = i0 + ti, j = j0 + tj;
        float out = 0.f;
        if (i < nx && j < ny) {
            float az = 0.f;
            const int lp0 = s * (ti + 3), lq0 = s * (tj + 3);
            for (int a = 0; a < s; ++a)
                for (int bb = 0; bb < s; ++bb) az += e_s[(lp0 + a) * MQ + lq0 + bb];
            az *= inv_s2;                                   // eps2d_z
            const int cell = i * ny + j;
            out = gb[2 * ncol + cell];
            if (P.w_lo > 0.f) out = fmaf(face_factor(P.w_lo, az, inv_ec), gb[3 * ncol + cell], out);
            if (P.w_hi > 0.f) out = fmaf(face_factor(P.w_hi, az, inv_ec), gb[4 * ncol + cell], out);
        }
        AbZ[it] = out;
    }
    __syncthreads();

    // ---- E: R4 + R5 per mask pixel of the tile
    const int TP = s * TI, TQ = s * TJ;
    float *vb = P.v + (size_t)b * P.px * P.py;
    for (int it = tid; it < TP * TQ; it += NTH) {
        const int tp = it / TQ, tq = it - tp * TQ;
        const int p = s * i0 + tp, q = s * j0 + tq;
        if (p >= P.px || q >= P.py) continue;
        const int iz = p / s, jz = q / s;
        float ebar = AbZ[(iz - i0) * TJ + (jz - j0)], rbar = 0.f;
        if (p >= hs) {                                       // E_x owner
            const int ix = (p - hs) / s;
            const float mlt = p == P.px - 1 ? (float)(1 + hs) : 1.0f;
            const int idx = (ix - oi) * CJ + (jz - oj);
            ebar = fmaf(mlt, AbF[0][idx], ebar);
            rbar = fmaf(mlt, Hb[0][idx], rbar);
        }
        if (q >= hs) {                                       // E_y owner
            const int jy = (q - hs) / s;
            const float mlt = q == P.py - 1 ? (float)(1 + hs) : 1.0f;
            const int idx = (iz - oi) * CJ + (jy - oj);
            ebar = fmaf(mlt, AbF[1][idx], ebar);
            rbar = fmaf(mlt, Hb[1][idx], rbar);
        }
        const float r = r_s[(tp + 3 * s) * MQ + tq + 3 * s];           // 1/e
        const float rhobar = P.deps * inv_s2 * (ebar - rbar * r * r);
        const float slope = project_slope(phib[p * P.py + q], P.beta, P.eta_r);
        vb[p * P.py + q] = rhobar * slope * P.nrm.at_index(nidx[tp], nidx[TP + tq]);
    }
}

}  // namespace epsgrad
