// fwd2d.cuh -- F2..F5 of the chain on the 2-D grid, one CTA per TI x TJ Yee cells:
//   projection + mixing (Eq. (3)/(6)) -> cell averages on the half-cell shifted footprints
//   (Eq. (8)) -> Sobel normals -> Eq. (7), plus Eq. (7) with n = z_hat on the
//   (at most two) fractional face cells of E_z (S7).
// It leaves, per Yee column, the five values the z-extrusion (extrude.cuh) needs -- eps2d_x, eps2d_y, eps2d_z and
// eps_zz on the lower / upper face cell -- and, when a reverse pass follows, the ten coefficients of R2 and of the
// first half of R3: those steps are linear in the z-reduced cotangent G, which enters only at the cell itself,
//   Hbar_c = hbk_c G_c,  Abar_c = abk_c G_c,  gxbar_c = gxk_c G_c,  gybar_c = gyk_c G_c   (c = x, y)
//   Abar_z = G_zfull + flo G_zlo + fhi G_zhi
// with  q = 1/eps2d, qbar = -G/q^2, Hbar = n^2 qbar, Abar = -(1-n^2) qbar/A^2, n2bar = (H - 1/A) qbar (Eq. (7)^T)
// and the cotangents of the Sobel gradients from n2bar (normals^T).  The mask kernel (maskgrad.cuh) multiplies.
// Everything here is L2-resident (4 B read per mask pixel, 60 B written per cell); the kernel is ALU/latency bound.
#pragma once
#include "common.cuh"
#include "sizes.cuh"

namespace epsgrad {


struct Fwd2dParams {
    const float *phi;      // [B,px,py] centred filter output
    float *e2d;            // [B,5,nx,ny] or nullptr
    float *coef;           // [B,10,nx,ny] or nullptr
    float *eps2d;          // [B,3,nx,ny] or nullptr (stage tap)
    int nx, ny, px, py, s;
    float beta, eta_r, eps_clad, deps, delta;
    float w_lo, w_hi;      // fractional z-face weights of eps_zz (0 if that face cell is absent)
};


// d eps_zz / d eps2d_z on a face cell of weight w:  w (eps_zz/v)^2, eps_zz/v = 1/(w + (1-w) v/eps_clad)
__device__ __forceinline__ float face_factor(float w, float v, float inv_ec)
{
    const float f = fast_rcp(w + (1.0f - w) * v * inv_ec);
    return w * f * f;
}

// Sobel gradient of the staged average A at local cell (ci,cj) of a [.][CJ] array whose origin is cell (oi,oj);
// replicate padding at the region border (S5) unless the whole ring is inside (`inner`).
template <int CJ>
__device__ __forceinline__ void sobel_at(const float *A, int ci, int cj, int i, int j, int oi, int oj, int nx, int ny,
                                         bool inner, float &gx, float &gy)
{
    // one formula for both cases (differences of opposite neighbours first: exact for nearly equal values), so that a cell gets
    // the same bits whether its tile touches the border of the region or not; only the addressing differs
    const float *q1 = A + ci * CJ + cj;
    float a00, a01, a02, a10, a12, a20, a21, a22;
    if (inner) {
        const float *q0 = q1 - CJ, *q2 = q1 + CJ;
        a00 = q0[-1]; a01 = q0[0]; a02 = q0[1]; a10 = q1[-1]; a12 = q1[1]; a20 = q2[-1]; a21 = q2[0]; a22 = q2[1];
    } else {
        const float *q0 = q1 + (clampi(i - 1, 0, nx - 1) - i) * CJ, *q2 = q1 + (clampi(i + 1, 0, nx - 1) - i) * CJ;
        const int cm = clampi(j - 1, 0, ny - 1) - j, cp = clampi(j + 1, 0, ny - 1) - j;
        a00 = q0[cm]; a01 = q0[0]; a02 = q0[cp]; a10 = q1[cm]; a12 = q1[cp]; a20 = q2[cm]; a21 = q2[0]; a22 = q2[cp];
    }
    gx = ((a20 - a00) + 2.0f * (a21 - a01) + (a22 - a02)) * 0.125f;
    gy = ((a02 - a00) + 2.0f * (a12 - a10) + (a22 - a20)) * 0.125f;
}

// One tile of TI x TJ cells by a CTA of F2_THREADS threads; sm: fwd2d_smem_floats(s) floats.  No barrier at entry or exit:
// the caller separates calls that reuse sm.  CG: Phi' is read through L2 (ld.global.cg) -- for the persistent kernel (mega.cuh),
// where other CTAs of the same launch produce it.  S > 0: compile-time subpixel count (index divisions fold to shifts); S = 0: runtime P.s.
template <int S, bool CG>
__device__ __forceinline__ void tile_fwd2d(const Fwd2dParams &P, int bx, int by, int b, float *sm)
{
    constexpr int TI = F2_TI, TJ = F2_TJ, NTH = F2_THREADS;
    constexpr int CI = TI + 2, CJ = TJ + 2;
    const int s = S > 0 ? S : P.s, hs = s >> 1;
    const int MP = s * CI + hs, MQ = s * CJ + hs;
    float *e_s = sm;
    float *r_s = e_s + MP * MQ;
    float *Ax = r_s + MP * MQ;
    float *Hx = Ax + CI * CJ;
    float *Ay = Hx + CI * CJ;
    float *Hy = Ay + CI * CJ;

    const int tid = threadIdx.x;
    const int i0 = by * TI, j0 = bx * TJ;
    const int nx = P.nx, ny = P.ny, ncol = nx * ny;
    const float inv_s2 = 1.0f / (float)(s * s);

    // ---- stage 1: mask tile (replicate outside the region, S5): e and r = 1/e; loads batched four deep.  The flat index
    // advances by NTH without divisions; tiles whose ring lies inside the mask skip the clamps (block-uniform).
    {
        const float *phib = P.phi + (size_t)b * P.px * P.py;
        const int p_base = s * (i0 - 1), q_base = s * (j0 - 1);
        const bool inside = p_base >= 0 && q_base >= 0 && p_base + MP <= P.px && q_base + MQ <= P.py;
        const int dlp = NTH / MQ, dlq = NTH - dlp * MQ;
        int lp = tid / MQ, lq = tid - lp * MQ;
        for (int base = tid; base < MP * MQ; base += 4 * NTH) {
            float ph[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (base + u * NTH < MP * MQ) {
                    const int p = inside ? p_base + lp : clampi(p_base + lp, 0, P.px - 1);
                    const int q = inside ? q_base + lq : clampi(q_base + lq, 0, P.py - 1);
                    ph[u] = ld_plane<CG>(phib + p * P.py + q);
                }
                lp += dlp; lq += dlq;
                if (lq >= MQ) { lq -= MQ; ++lp; }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int i = base + u * NTH;
                if (i < MP * MQ) {
                    const float e = project_mix(ph[u], P.beta, P.eta_r, P.eps_clad, P.deps);
                    e_s[i] = e;
                    r_s[i] = fast_rcp(e);
                }
            }
        }
    }
    __syncthreads();

    // ---- stage 2: <e>, <1/e> on the E_x and E_y footprints for the tile + 1-cell ring
    for (int i = tid; i < CI * CJ; i += NTH) {
        const int ci = i / CJ, cj = i - ci * CJ;
        const int lp0 = s * ci, lq0 = s * cj;
        float ax = 0.f, hx = 0.f, ay = 0.f, hy = 0.f;
        for (int a = 0; a < s; ++a)
            for (int bb = 0; bb < s; ++bb) {
                const int ix = (lp0 + hs + a) * MQ + lq0 + bb;       // E_x: half a cell toward +x
                const int iy = (lp0 + a) * MQ + lq0 + hs + bb;       // E_y: half a cell toward +y
                ax += e_s[ix]; hx += r_s[ix];
                ay += e_s[iy]; hy += r_s[iy];
            }
        Ax[i] = ax * inv_s2; Hx[i] = hx * inv_s2;
        Ay[i] = ay * inv_s2; Hy[i] = hy * inv_s2;
    }
    __syncthreads();

    // ---- stage 3 (one thread per cell): Sobel normals of D_c = (A_c - eps_clad)/deps, Eq. (7); eps2d_z = <e>_z
    const float inv_deps = 1.0f / P.deps, inv_ec = 1.0f / P.eps_clad;
    const bool inner = i0 >= 1 && j0 >= 1 && i0 + TI <= nx - 1 && j0 + TJ <= ny - 1;   // 1-cell ring inside the region
    const int ii = tid / TJ, jj = tid - ii * TJ;
    const int i = i0 + ii, j = j0 + jj, ic = (ii + 1) * CJ + jj + 1;
    if (i >= nx || j >= ny) return;
    const int cellg = i * ny + j;
    float *ed = P.e2d ? P.e2d + (size_t)b * F2_NE2D * ncol + cellg : nullptr;
    float *cf = P.coef ? P.coef + (size_t)b * F2_NCOEF * ncol + cellg : nullptr;
    float *tap = P.eps2d ? P.eps2d + (size_t)b * 3 * ncol + cellg : nullptr;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        const float *A = c == 0 ? Ax : Ay, *H = c == 0 ? Hx : Hy;
        float gx, gy;
        sobel_at<CJ>(A, ii + 1, jj + 1, i, j, i0 - 1, j0 - 1, nx, ny, inner, gx, gy);
        gx *= inv_deps; gy *= inv_deps;
        const float gc = c == 0 ? gx : gy, go = c == 0 ? gy : gx;
        const float rS = fast_rcp(gc * gc + go * go + P.delta);
        const float n2 = gc * gc * rS;
        const float ra = fast_rcp(A[ic]), h = H[ic];
        const float e2 = fast_rcp(n2 * h + (1.0f - n2) * ra);        // eps2d_c = 1/q  (Eq. (7))
        if (ed) ed[(size_t)c * ncol] = e2;
        if (tap) tap[(size_t)c * ncol] = e2;
        if (cf) {
            const float q2 = e2 * e2;                                 // qbar = -q2 G
            const float k2 = -2.0f * (h - ra) * q2 * gc * rS * rS;    // n2bar = -(h - 1/A) q2 G
            const float gck = k2 * (go * go + P.delta), gok = -k2 * gc * go;
            cf[(size_t)(4 * c + 0) * ncol] = -n2 * q2;
            cf[(size_t)(4 * c + 1) * ncol] = (1.0f - n2) * q2 * ra * ra;
            cf[(size_t)(4 * c + 2) * ncol] = c == 0 ? gck : gok;
            cf[(size_t)(4 * c + 3) * ncol] = c == 0 ? gok : gck;
        }
    }
    float az = 0.f;
    {
        const int lp0 = s * (ii + 1), lq0 = s * (jj + 1);
        for (int a = 0; a < s; ++a)
            for (int bb = 0; bb < s; ++bb) az += e_s[(lp0 + a) * MQ + lq0 + bb];
        az *= inv_s2;
    }
    if (tap) tap[(size_t)2 * ncol] = az;
    if (ed) {
        // Eq. (7) with n = z_hat on the fractional face cells of E_z (S7): once per column
        const float rz = fast_rcp(az);
        ed[(size_t)2 * ncol] = az;
        ed[(size_t)3 * ncol] = P.w_lo > 0.f ? fast_rcp(P.w_lo * rz + (1.0f - P.w_lo) * inv_ec) : 0.f;
        ed[(size_t)4 * ncol] = P.w_hi > 0.f ? fast_rcp(P.w_hi * rz + (1.0f - P.w_hi) * inv_ec) : 0.f;
    }
    if (cf) {
        cf[(size_t)8 * ncol] = P.w_lo > 0.f ? face_factor(P.w_lo, az, inv_ec) : 0.f;
        cf[(size_t)9 * ncol] = P.w_hi > 0.f ? face_factor(P.w_hi, az, inv_ec) : 0.f;
    }
}

// grid (ceil(ny/TJ), ceil(nx/TI), B)
template <int S>
__global__ void __launch_bounds__(F2_THREADS, 8) k_fwd2d(const __grid_constant__ Fwd2dParams P)
{
    extern __shared__ __align__(16) float sm[];
    pdl_launch();
    pdl_wait();
    tile_fwd2d<S, false>(P, blockIdx.x, blockIdx.y, blockIdx.z, sm);
}

}  // namespace epsgrad
