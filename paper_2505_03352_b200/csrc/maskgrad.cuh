// maskgrad.cuh -- R2..R5 in gather form: from the z-reduced cotangent G (zreduce.cuh) and the per-cell
// coefficients the forward 2-D kernel left (fwd2d.cuh) to the mask cotangent  v[p,q] = Phibar[p,q] / den[p,q]  that the
// transposed filter (R6) gathers.
//   R2/R3a Eq. (7)^T and normals^T are linear in G and local to the cell: Hbar_c = hbk_c G_c, Abar_c = abk_c G_c,
//       gxbar_c = gxk_c G_c, gybar_c = gyk_c G_c (c = x,y); Abar_z = G_zfull + flo G_zlo + fhi G_zhi -- formed while staging
//   R3b Dbar_c = Sobel^T(gxbar_c, gybar_c) with the replicate padding folded back at the borders (S5);
//       AbarF_c = Abar_c + Dbar_c / deps
//   R4  averages^T: each mask pixel gathers from the E_x, E_y, E_z cells whose footprint holds it
//       (the clamped last pixel is counted s/2+1 times)
//   R5  mixing^T, projection^T: rhobar = deps (ebar - rbar/e^2), Phibar = rhobar (beta/2) sech^2 t,
//       sech^2 in the overflow-free form (the paper's custom tanh derivative rule)
// One CTA per TI x TJ cells (s TI x s TJ mask pixels); owners of a tile's pixels lie on [i0-1, i0+TI-1], their
// Sobel^T sources on [i0-2, i0+TI].
#pragma once
#include "common.cuh"
#include "sizes.cuh"
#include "reduce.cuh"

namespace epsgrad {

struct MaskGradParams {
    const float *phi;      // [B,px,py] centred input of the last projection: Phi' or, with morphological filters, rho~ - 1/2
    const float *gbar;     // [B,5,nx,ny]  z-reduced cotangent: x, y, z-full, z-lower-face, z-upper-face
    const float *coef;     // [B,10,nx,ny] [hbk, abk, gxk, gyk] for c = x, for c = y, flo, fhi
    float *v;              // [B,px,py]
    float *dbeta_part;     // nullptr, or one partial sum of d F/d beta per CTA: [B][gridDim.y * gridDim.x] (reduce.cuh)
    Normaliser nrm;
    int nx, ny, px, py, s;
    int use_den;           // 1: v carries 1/den of Eq. (2); 0: the morphological filters^T follow and the last one applies it
    float beta, eta_r, eps_clad, deps;
};



// One tile of TI x TJ cells by a CTA of MG_THREADS threads; sm: maskgrad_smem_floats(s) floats; part_idx: the tile's slot in
// dbeta_part ([B][tile rows][tiles per row]).  No barrier at entry or exit.  CG: G, the coefficients and Phi' are read through L2 (ld.global.cg) -- for the
// persistent kernel (mega.cuh), where other CTAs of the same launch produce them.  S > 0: compile-time subpixel count; S = 0: runtime P.s.
template <int S, bool CG>
__device__ __forceinline__ void tile_maskgrad(const MaskGradParams &P, int bx, int by, int b, int part_idx, float *sm)
{
    constexpr int TI = MG_TI, TJ = MG_TJ, NTH = MG_THREADS, CI = MG_CI, CJ = MG_CJ, NC = CI * CJ;
    const int s = S > 0 ? S : P.s, hs = s >> 1;
    float *R = sm;                     // [8][NC] staged residual planes: Hb, Ab, Gx, Gy for c = x then c = y
    float *AbF = sm + 8 * NC;          // [2][NC]
    float *AbZ = sm + 10 * NC;         // [TI*TJ]
    int *nidx = reinterpret_cast<int *>(AbZ + TI * TJ);   // normaliser table row of each tile mask row, then column of each mask column

    const int tid = threadIdx.x;
    const int i0 = by * TI, j0 = bx * TJ;
    const int oi = i0 - 2, oj = j0 - 2;            // cell origin of the staged arrays
    const int nx = P.nx, ny = P.ny, ncol = nx * ny;
    const float inv_s2 = 1.0f / (float)(s * s), inv_deps = 1.0f / P.deps;
    const float *gb = P.gbar + (size_t)b * 5 * ncol, *cb = P.coef + (size_t)b * 10 * ncol;
    // tile whose 2-cell ring lies strictly inside the region: no folded border terms (block-uniform)
    const bool inner = i0 >= 3 && j0 >= 3 && i0 + TI + 1 <= nx - 1 && j0 + TJ + 1 <= ny - 1;

    for (int k = tid; k < s * (TI + TJ); k += NTH) {
        const int along_x = k < s * TI;
        const int pix = along_x ? s * i0 + k : s * j0 + (k - s * TI);
        nidx[k] = along_x ? P.nrm.ix_of(min(pix, P.px - 1)) : P.nrm.iy_of(min(pix, P.py - 1));
    }
    // staging: a warp per row of the (TI+3) x (TJ+3) cell block, a lane per cell; R2/R3a products formed on the way
    static_assert(CJ <= 32, "one lane per staged column");
    for (int ci = tid >> 5; ci < CI; ci += NTH / 32) {
        const int cj = tid & 31, i = oi + ci, j = oj + cj;
        if (cj < CJ) {
            float r8[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            if (i >= 0 && i < nx && j >= 0 && j < ny) {
                const int cell = i * ny + j;
                const float gx = ld_plane<CG>(gb + cell), gy = ld_plane<CG>(gb + ncol + cell);
#pragma unroll
                for (int o = 0; o < 4; ++o) {
                    r8[o] = ld_plane<CG>(cb + (size_t)o * ncol + cell) * gx;
                    r8[4 + o] = ld_plane<CG>(cb + (size_t)(4 + o) * ncol + cell) * gy;
                }
            }
#pragma unroll
            for (int o = 0; o < 8; ++o) R[o * NC + ci * CJ + cj] = r8[o];
        }
    }
    for (int it = tid; it < TI * TJ; it += NTH) {
        const int ti = it / TJ, tj = it - ti * TJ, i = i0 + ti, j = j0 + tj;
        float az = 0.f;
        if (i < nx && j < ny) {
            const int cell = i * ny + j;
            az = fmaf(ld_plane<CG>(cb + (size_t)8 * ncol + cell), ld_plane<CG>(gb + (size_t)3 * ncol + cell),
                      fmaf(ld_plane<CG>(cb + (size_t)9 * ncol + cell), ld_plane<CG>(gb + (size_t)4 * ncol + cell), ld_plane<CG>(gb + (size_t)2 * ncol + cell)));
        }
        AbZ[it] = az;
    }
    __syncthreads();

    // ---- Sobel^T with the replicate padding folded back, on the owner cells [i0-1, i0+TI-1] x [j0-1, j0+TJ-1]
    {
        constexpr int RI = TI + 1, RJ = TJ + 1;           // ci in [1, TI+1], cj in [1, TJ+1]
        for (int it = tid; it < 2 * RI * RJ; it += NTH) {
            const int c = it / (RI * RJ), rem = it - c * (RI * RJ);
            const int ci = 1 + rem / RJ, cj = 1 + rem % RJ, i_ = ci * CJ + cj;
            const int ii = oi + ci, jj = oj + cj;
            float out = 0.f;
            if (inner || (ii >= 0 && ii < nx && jj >= 0 && jj < ny)) {
                float dbar = 0.f;
                const float *gxs = R + (4 * c + 2) * NC, *gys = R + (4 * c + 3) * NC;
                if (inner || (ii >= 1 && ii <= nx - 2 && jj >= 1 && jj <= ny - 2)) {
                    // interior: the cell (ii-di, jj-dj) reached (ii,jj) through its stencil entry (di,dj)
#pragma unroll
                    for (int di = -1; di <= 1; ++di)
#pragma unroll
                        for (int dj = -1; dj <= 1; ++dj) {
                            const int src = i_ - di * CJ - dj;
                            const float kx = (float)(di * (2 - (dj < 0 ? -dj : dj))) * 0.125f;
                            const float ky = (float)(dj * (2 - (di < 0 ? -di : di))) * 0.125f;
                            if (di != 0) dbar = fmaf(kx, gxs[src], dbar);        // the zero taps fold away (unrolled)
                            if (dj != 0) dbar = fmaf(ky, gys[src], dbar);
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
                out = R[(4 * c + 1) * NC + i_] + dbar * inv_deps;
            }
            AbF[c * NC + i_] = out;
        }
    }
    __syncthreads();

    // ---- R4 + R5 per mask pixel of the tile
    const int TP = s * TI, TQ = s * TJ;
    const float *phib = P.phi + (size_t)b * P.px * P.py;
    float *vb = P.v + (size_t)b * P.px * P.py;
    if constexpr (S == 2) {
        // s = 2: a thread per cell owns its 2 x 2 pixels.  Rows p = 2i, 2i+1 have E_x owners i-1 and i, columns q = 2j, 2j+1
        // have E_y owners j-1 and j: nine shared-memory values serve the four pixels; 8-byte loads and stores.
        static_assert(TI * TJ == NTH, "one thread per cell");
        const int ti = tid / TJ, tj = tid - ti * TJ, i = i0 + ti, j = j0 + tj;
        float db = 0.f;                                             // sum of Phibar (x - eta) over this thread's pixels
        if (i < nx && j < ny) {
        const int c0 = (ti + 2) * CJ + tj + 2;                      // the cell in the staged arrays
        const float az = AbZ[tid];
        float ex[2], hx[2], ey[2], hy[2];                           // owner values per pixel row a / column c, multiplicity folded in
        ex[0] = i >= 1 ? AbF[c0 - CJ] : 0.f;  hx[0] = i >= 1 ? R[c0 - CJ] : 0.f;
        ey[0] = j >= 1 ? AbF[NC + c0 - 1] : 0.f;  hy[0] = j >= 1 ? R[4 * NC + c0 - 1] : 0.f;
        const float mx = i == nx - 1 ? 2.0f : 1.0f, my = j == ny - 1 ? 2.0f : 1.0f;   // the clamped last pixel is owned twice
        ex[1] = mx * AbF[c0];  hx[1] = mx * R[c0];
        ey[1] = my * AbF[NC + c0];  hy[1] = my * R[4 * NC + c0];
        const int p = 2 * i, q = 2 * j;
        const float2 ph0 = ld_plane2<CG>(reinterpret_cast<const float2 *>(phib + p * P.py + q));
        const float2 ph1 = ld_plane2<CG>(reinterpret_cast<const float2 *>(phib + (p + 1) * P.py + q));
        const float phv[2][2] = {{ph0.x, ph0.y}, {ph1.x, ph1.y}};
        const int nq0 = nidx[TP + 2 * tj], nq1 = nidx[TP + 2 * tj + 1];
        const float k0 = P.deps * inv_s2 * 2.0f * P.beta;
#pragma unroll
        for (int a = 0; a < 2; ++a) {
            const int np = nidx[2 * ti + a];
            float o[2];
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                // one exponential serves rho and its slope: e2 = exp(-2|t|), rho = 1/(1+e2) or e2/(1+e2), slope = 2 beta e2/(1+e2)^2
                const float t = P.beta * (phv[a][c] - P.eta_r);
                const float e2 = __expf(-2.0f * fabsf(t));
                const float d = fast_rcp(1.0f + e2);
                const float r = fast_rcp(fmaf(P.deps, t >= 0.f ? d : e2 * d, P.eps_clad));   // 1/e
                const float ebar = az + ex[a] + ey[c], rbar = hx[a] + hy[c];
                const float pb = k0 * e2 * d * d * (ebar - rbar * r * r);          // Phibar
                db = fmaf(pb, phv[a][c] - P.eta_r, db);
                o[c] = pb * (P.use_den ? P.nrm.at_index(np, c == 0 ? nq0 : nq1) : 1.0f);
            }
            *reinterpret_cast<float2 *>(vb + (p + a) * P.py + q) = make_float2(o[0], o[1]);
        }
        }
        if (P.dbeta_part) {                                         // block-uniform
            const float sdb = block_sum(db, reinterpret_cast<float *>(nidx));      // nidx is dead for every thread past block_sum's first barrier
            if (tid == 0) P.dbeta_part[part_idx] = sdb / P.beta;
        }
    } else {
    float db = 0.f;
    for (int base = tid; base < TP * TQ; base += 4 * NTH) {
        float ph[4];                                           // filter output of four pixels in flight
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int it = base + u * NTH, tp = it / TQ, tq = it - tp * TQ;
            const int p = s * i0 + tp, q = s * j0 + tq;
            if (it < TP * TQ && p < P.px && q < P.py) ph[u] = ld_plane<CG>(phib + p * P.py + q);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int it = base + u * NTH, tp = it / TQ, tq = it - tp * TQ;
            const int p = s * i0 + tp, q = s * j0 + tq;
            if (it >= TP * TQ || p >= P.px || q >= P.py) continue;
            const int iz = p / s, jz = q / s;
            float ebar = AbZ[(iz - i0) * TJ + (jz - j0)], rbar = 0.f;
            if (p >= hs) {                                       // E_x owner
                const int ix = (p - hs) / s;
                const float mlt = p == P.px - 1 ? (float)(1 + hs) : 1.0f;
                const int idx = (ix - oi) * CJ + (jz - oj);
                ebar = fmaf(mlt, AbF[idx], ebar);
                rbar = fmaf(mlt, R[idx], rbar);
            }
            if (q >= hs) {                                       // E_y owner
                const int jy = (q - hs) / s;
                const float mlt = q == P.py - 1 ? (float)(1 + hs) : 1.0f;
                const int idx = (iz - oi) * CJ + (jy - oj);
                ebar = fmaf(mlt, AbF[NC + idx], ebar);
                rbar = fmaf(mlt, R[4 * NC + idx], rbar);
            }
            // one exponential serves rho and its slope: a = exp(-2|t|), rho = 1/(1+a) or a/(1+a), slope = 2 beta a/(1+a)^2
            const float t = P.beta * (ph[u] - P.eta_r);
            const float a = __expf(-2.0f * fabsf(t));
            const float d = fast_rcp(1.0f + a);
            const float rho = t >= 0.f ? d : a * d;
            const float r = fast_rcp(fmaf(P.deps, rho, P.eps_clad));   // 1/e
            const float slope = 2.0f * P.beta * a * d * d;
            const float rhobar = P.deps * inv_s2 * (ebar - rbar * r * r);
            db = fmaf(rhobar * slope, ph[u] - P.eta_r, db);
            vb[p * P.py + q] = rhobar * slope * (P.use_den ? P.nrm.at_index(nidx[tp], nidx[TP + tq]) : 1.0f);
        }
    }
    if (P.dbeta_part) {
        const float sdb = block_sum(db, reinterpret_cast<float *>(nidx));
        if (tid == 0) P.dbeta_part[part_idx] = sdb / P.beta;
    }
    }
}

// grid (ceil(ny/TJ), ceil(nx/TI), B)
template <int S>
__global__ void __launch_bounds__(MG_THREADS, 8) k_maskgrad(const __grid_constant__ MaskGradParams P)
{
    extern __shared__ __align__(16) float sm[];
    pdl_launch();
    pdl_wait();
    tile_maskgrad<S, false>(P, blockIdx.x, blockIdx.y, blockIdx.z, (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x, sm);
}

}  // namespace epsgrad
