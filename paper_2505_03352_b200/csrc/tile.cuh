// tile.cuh -- the two HBM streams of the path in ONE tile kernel.
// One CTA owns TI x TJ Yee columns of one design and runs, for them,
//   F2-F5  projection + mixing (Eq. (3)/(6)) -> cell averages on the half-cell shifted
//          footprints (Eq. (8)) -> Sobel normals -> Eq. (7)
//   F6     z-extrusion with fractional faces (S7,S8): 16-byte streaming stores, 12 B per Yee cell
//   R1     Eq. (1) cotangent G3 = -2 Re(E_F (.) E_A) (S10) of every field pair and its
//          z-reduction with the extrusion weights; only the 16-byte chunks of a z column that hold slab
//          cells are read (64-byte L2 fills), by asynchronous copies into shared memory that are issued
//          before the 2-D chain runs and consumed after the eps stores have been issued
//   R2 + first half of R3   Eq. (7)^T and normals^T per cell: everything they need -- A_c, H_c
//          on the one-cell ring, the Sobel gradients -- is still in shared memory from F3/F4, and the
//          cotangent enters only at the cell itself, so no halo of field reads is needed.
// It leaves nine per-cell planes (Hbar_c, Abar_c, gxbar_c, gybar_c for c = x,y and Abar_z) for the mask
// kernel (maskgrad.cuh), which applies Sobel^T, averages^T, mixing^T and projection^T.
// The forward store stream and the field read stream of different resident CTAs overlap; the 2-D
// arithmetic hides under them.  eps == nullptr skips F6, n_pairs == 0 skips R1-R3.
#pragma once
#include "common.cuh"

namespace epsgrad {

constexpr int TILE_TI = 8, TILE_TJ = 16, TILE_THREADS = 256, TILE_MAX_PAIRS = 8;
constexpr int TILE_STAGE_CELLS = 64;     // cells whose windows (13 chunks per field: 4 + 4 + 5 for the paper slab) fit the staging buffer
constexpr int TILE_NRES = 9;      // residual planes: [Hb, Ab, Gx, Gy] for c = x, the same for c = y, Abar_z

struct TileParams {
    const float *phi;      // [B,px,py] centred filter output
    float *eps;            // [B,3,nx,ny,nz] or nullptr
    float *eps2d;          // [B,3,nx,ny] or nullptr (stage tap)
    float *gtap;           // [B,5,nx,ny] or nullptr (stage tap): z-reduced cotangent planes x, y, z-full, z-lower, z-upper
    float *res;            // [B,9,nx,ny] or nullptr: reverse residual planes
    const float4 *ef[TILE_MAX_PAIRS];
    const float4 *ea[TILE_MAX_PAIRS];
    const float *zw;       // [7][nz] z tables (epsgrad.cu): wxy, wz, z-full, z-lower-face, z-upper-face indicators,
                           //          eps_clad (1 - wxy), eps_clad [wz == 0]
    int n_pairs, accumulate;
    int nx, ny, nz, px, py, s;
    int ch0[2], nch[2];         // chunk window (chunk = 2 cells = 16 B) for {x,y} and {z}
    int chs[2];                 // log2 of the lanes per column of the copy loop: 2^chs >= nch
    int ncp;                    // cells staged per pass of R1 (<= TI*TJ): the staging buffer holds ncp (2 nch[0] + nch[1]) chunks per field
    int sparse;                 // windows <= 128 B per column: 64-byte L2 fills
    float beta, eta_r, eps_clad, deps, delta;
    float w_lo, w_hi;      // fractional z-face weights of eps_zz (0 if that face cell is absent)
};

// floats of the 2-D part (16-byte multiple), and cells per R1 pass for windows of `rows` chunks per cell
__host__ __device__ inline size_t tile_smem_floats(int s, int nz)
{
    const int CI = TILE_TI + 2, CJ = TILE_TJ + 2;
    const int MP = s * CI + s / 2, MQ = s * CJ + s / 2;
    const size_t n = (size_t)2 * MP * MQ + 4 * CI * CJ + 10 * TILE_TI * TILE_TJ + 7 * (size_t)nz;
    return (n + 3) / 4 * 4;
}
__host__ __device__ inline int tile_cells_per_pass(int rows)
{
    const int ncell = TILE_TI * TILE_TJ, cap = TILE_STAGE_CELLS * 13;
    int n = cap / (rows > 0 ? rows : 1);
    if (n >= 32) n &= ~31;                 // whole warps of cells
    return n > ncell ? ncell : n;
}

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
    if (inner) {
        const float *q1 = A + ci * CJ + cj, *q0 = q1 - CJ, *q2 = q1 + CJ;
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
                const float d = A[ni * CJ + nj];
                gx = fmaf((float)(di * (2 - (dj < 0 ? -dj : dj))) * 0.125f, d, gx);
                gy = fmaf((float)(dj * (2 - (di < 0 ? -di : di))) * 0.125f, d, gy);
            }
    }
}

// 16-byte asynchronous copy global -> shared (LDGSTS): no register staging, completion by cp.async groups.
// SPARSE windows ask for 64-byte L2 fills (the default fill is the whole 128-byte line; common.cuh ld_stream).
template <bool SPARSE>
__device__ __forceinline__ void cp_async16(float4 *smem, const float4 *g)
{
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    if (SPARSE) asm volatile("cp.async.cg.shared.global.L2::64B [%0], [%1], 16;" :: "r"(sa), "l"(g) : "memory");
    else asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(sa), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async4(float *smem, const float *g)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" :: "r"((unsigned)__cvta_generic_to_shared(smem)), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_wait_but_last() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// R1, issue side: start the copies of the z windows of cells [cell0, cell0+nc) of the tile, all three components,
// fields E_F and E_A of pair p, into the staging buffer.  Buffer layout per field: [chunk row][cell], chunk rows
// = nch[0] rows of x, nch[0] rows of y, nch[1] rows of z (reads of consecutive cells are conflict-free).
// Consecutive threads take consecutive chunks of a column, then the next column: a warp covers 32/nch windows.
template <bool SPARSE>
__device__ __forceinline__ void zwindow_issue(const TileParams &P, float4 *buf, int p, int cell0, int nc, int b, int i0, int j0)
{
    constexpr int TJ = TILE_TJ, NTH = TILE_THREADS;
    const int nzc = P.nz >> 1, rows = 2 * P.nch[0] + P.nch[1];
    float4 *bf = buf, *ba = buf + rows * P.ncp;
    int row0 = 0;
    for (int c = 0; c < 3; ++c) {
        const int grp = c == 2, nch = P.nch[grp], ch0 = P.ch0[grp], sh = P.chs[grp];
        // 2^sh >= nch lanes per column (a power of two: no divisions); lanes beyond the window idle
        const int ch = threadIdx.x & ((1 << sh) - 1), lstep = NTH >> sh;
        if (ch < nch) {
            const size_t plane = ((size_t)b * 3 + c) * P.nx * P.ny * nzc + ch0 + ch;
            const float4 *pf = P.ef[p] + plane, *pa = P.ea[p] + plane;
            float4 *df = bf + (row0 + ch) * P.ncp, *da = ba + (row0 + ch) * P.ncp;
            for (int lc = threadIdx.x >> sh; lc < nc; lc += lstep) {
                const int cell = cell0 + lc, ii = cell / TJ, jj = cell - ii * TJ;
                if (i0 + ii < P.nx && j0 + jj < P.ny) {
                    const unsigned off = (unsigned)((i0 + ii) * P.ny + (j0 + jj)) * (unsigned)nzc;
                    cp_async16<SPARSE>(df + lc, pf + off);
                    cp_async16<SPARSE>(da + lc, pa + off);
                }
            }
        }
        row0 += nch;
    }
    cp_async_commit();
}

// R1, consume side: Eq. (1) cotangent -2 Re(E_F E_A) of the staged windows times the extrusion weights, summed over z.
// Item (c, lc) -> acc[0] (x, y or z-full), acc[1], acc[2] (z lower / upper face).
__device__ __forceinline__ void zwindow_reduce(const TileParams &P, const float *zw, const float4 *buf, int c, int lc,
                                               bool live, float acc[3])
{
    if (!live) return;
    const int grp = c == 2, nch = P.nch[grp], ch0 = P.ch0[grp], nz = P.nz;
    const int rows = 2 * P.nch[0] + P.nch[1], row0 = c * P.nch[0];
    const float4 *bf = buf + row0 * P.ncp + lc, *ba = bf + rows * P.ncp;
    for (int ch = 0; ch < nch; ++ch) {
        const float4 f = bf[ch * P.ncp], a = ba[ch * P.ncp];
        const int k = 2 * (ch0 + ch);
        const float g0 = -2.0f * (f.x * a.x - f.y * a.y);
        const float g1 = -2.0f * (f.z * a.z - f.w * a.w);
        if (grp == 0) {
            acc[0] = fmaf(zw[k], g0, fmaf(zw[k + 1], g1, acc[0]));
        } else {
#pragma unroll
            for (int o = 0; o < 3; ++o) acc[o] = fmaf(zw[(2 + o) * nz + k], g0, fmaf(zw[(2 + o) * nz + k + 1], g1, acc[o]));
        }
    }
}

// grid (ceil(ny/TJ), ceil(nx/TI), B).  S > 0: compile-time subpixel count (index divisions fold to shifts); S = 0: runtime P.s.
template <int S, bool SPARSE>
__global__ void __launch_bounds__(TILE_THREADS, 4) k_tile(const __grid_constant__ TileParams P)
{
    extern __shared__ __align__(16) float sm[];
    constexpr int TI = TILE_TI, TJ = TILE_TJ, NTH = TILE_THREADS, NCELL = TI * TJ;
    constexpr int CI = TI + 2, CJ = TJ + 2;
    const int s = S > 0 ? S : P.s, hs = s >> 1;
    const int MP = s * CI + hs, MQ = s * CJ + hs;
    float *e_s = sm;
    float *r_s = e_s + MP * MQ;
    float *Ax = r_s + MP * MQ;
    float *Hx = Ax + CI * CJ;
    float *Ay = Hx + CI * CJ;
    float *Hy = Ay + CI * CJ;
    float *e2 = Hy + CI * CJ;          // [5][NCELL]: eps2d_x, eps2d_y, eps2d_z, eps_zz on the lower / upper face cell
    float *G = e2 + 5 * NCELL;         // [5][NCELL]: z-reduced cotangent x, y, z-full, z-lower-face, z-upper-face
    float *zw = G + 5 * NCELL;         // [7][nz]
    float4 *stage = reinterpret_cast<float4 *>(sm + tile_smem_floats(s, P.nz));   // R1 staging: 2 fields x rows x ncp chunks

    const int tid = threadIdx.x;
    const int i0 = blockIdx.y * TI, j0 = blockIdx.x * TJ, b = blockIdx.z;
    const int nx = P.nx, ny = P.ny, nz = P.nz, ncol = nx * ny;
    const float inv_s2 = 1.0f / (float)(s * s);
    const bool rev = P.n_pairs > 0;

    // asynchronous copies first: the z tables (group 0), then the field windows of pair 0 (group 1, R1), which travel
    // while the 2-D chain runs and the eps stores are issued
    for (int k = tid; k < 7 * nz; k += NTH) cp_async4(zw + k, P.zw + k);
    cp_async_commit();
    if (rev) zwindow_issue<SPARSE>(P, stage, 0, 0, P.ncp, b, i0, j0);

    // ---- stage 1: mask tile (replicate outside the region, S5): e and r = 1/e; loads batched four deep
    {
        const float *phib = P.phi + (size_t)b * P.px * P.py;
        const int p_base = s * (i0 - 1), q_base = s * (j0 - 1);
        for (int base = tid; base < MP * MQ; base += 4 * NTH) {
            float ph[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int i = base + u * NTH;
                if (i < MP * MQ) {
                    const int lp = i / MQ, lq = i - lp * MQ;
                    const int p = clampi(p_base + lp, 0, P.px - 1), q = clampi(q_base + lq, 0, P.py - 1);
                    ph[u] = phib[p * P.py + q];
                }
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
    const bool in_region = tid < NCELL && i < nx && j < ny;
    float az = 0.f;
    if (in_region) {
        float out[3];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const float *A = c == 0 ? Ax : Ay, *H = c == 0 ? Hx : Hy;
            float gx, gy;
            sobel_at<CJ>(A, ii + 1, jj + 1, i, j, i0 - 1, j0 - 1, nx, ny, inner, gx, gy);
            gx *= inv_deps; gy *= inv_deps;
            const float gc = c == 0 ? gx : gy;
            const float n2 = gc * gc * fast_rcp(gx * gx + gy * gy + P.delta);
            out[c] = fast_rcp(n2 * H[ic] + (1.0f - n2) * fast_rcp(A[ic]));
        }
        {
            const int lp0 = s * (ii + 1), lq0 = s * (jj + 1);
            for (int a = 0; a < s; ++a)
                for (int bb = 0; bb < s; ++bb) az += e_s[(lp0 + a) * MQ + lq0 + bb];
            az *= inv_s2;
            out[2] = az;
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            e2[c * NCELL + tid] = out[c];
            if (P.eps2d) P.eps2d[(((size_t)b * 3 + c) * nx + i) * ny + j] = out[c];
        }
        // Eq. (7) with n = z_hat on the (at most two) fractional face cells of E_z (S7): once per column
        const float rz = fast_rcp(az);
        e2[3 * NCELL + tid] = P.w_lo > 0.f ? fast_rcp(P.w_lo * rz + (1.0f - P.w_lo) * inv_ec) : 0.f;
        e2[4 * NCELL + tid] = P.w_hi > 0.f ? fast_rcp(P.w_hi * rz + (1.0f - P.w_hi) * inv_ec) : 0.f;
    }
    if (rev) cp_async_wait_but_last(); else cp_async_wait_all();       // the z tables have landed (group 0)
    __syncthreads();

    // ---- stage 4: z-extrusion, 16-byte streaming stores.  Every output is affine in the staged per-column values:
    //   eps_cc[k] = eps_clad (1 - wxy_k) + wxy_k eps2d_c          (c = x, y)
    //   eps_zz[k] = eps_clad [wz_k = 0] + [wz_k = 1] eps2d_z + [k = lower face] v_lo + [k = upper face] v_hi
    if (P.eps) {
        const int TIv = min(TI, nx - i0), TJv = min(TJ, ny - j0);
        const int nz4 = nz >> 2;
        const float *w_xy = zw, *b_xy = zw + 5 * nz, *b_z = zw + 6 * nz, *i_f = zw + 2 * nz, *i_l = zw + 3 * nz, *i_h = zw + 4 * nz;
        const int cpp = NTH / nz4;                       // columns covered by one pass of the CTA
        if (NTH % nz4 == 0 && cpp % TJ == 0) {
            // a thread keeps its 4 z cells and its tile column cj for the whole tile (weights live in registers) and walks
            // down the rows: no index arithmetic per store
            const int kc = tid % nz4, k = kc << 2, cq = tid / nz4, cj = cq % TJ, ci0 = cq / TJ, rstep = cpp / TJ;
            if (cj < TJv) {
                const int row_stride = ny * nz;
                {
                    float wx[4], bx[4];
#pragma unroll
                    for (int x = 0; x < 4; ++x) { wx[x] = w_xy[k + x]; bx[x] = b_xy[k + x]; }
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        float *dst = P.eps + ((((size_t)b * 3 + c) * nx + i0 + ci0) * ny + j0 + cj) * nz + k;   // row offsets fit 32 bits
                        const float *vp = e2 + c * NCELL + ci0 * TJ + cj;
#pragma unroll
                        for (int r = 0; r < TI; ++r) {
                            if (ci0 + r * rstep < TIv) {
                                const float v = vp[r * rstep * TJ];
                                float4 o;
                                o.x = fmaf(wx[0], v, bx[0]); o.y = fmaf(wx[1], v, bx[1]);
                                o.z = fmaf(wx[2], v, bx[2]); o.w = fmaf(wx[3], v, bx[3]);
                                __stcs(reinterpret_cast<float4 *>(dst + r * rstep * row_stride), o);
                            }
                        }
                    }
                }
                {
                    float bz[4], zf[4], zl[4], zh[4];
#pragma unroll
                    for (int x = 0; x < 4; ++x) { bz[x] = b_z[k + x]; zf[x] = i_f[k + x]; zl[x] = i_l[k + x]; zh[x] = i_h[k + x]; }
                    float *dst = P.eps + ((((size_t)b * 3 + 2) * nx + i0 + ci0) * ny + j0 + cj) * nz + k;
                    const float *vp = e2 + 2 * NCELL + ci0 * TJ + cj;
#pragma unroll
                    for (int r = 0; r < TI; ++r) {
                        if (ci0 + r * rstep < TIv) {
                            const float v = vp[r * rstep * TJ], vl = vp[NCELL + r * rstep * TJ], vh = vp[2 * NCELL + r * rstep * TJ];
                            float4 o;
                            o.x = fmaf(zf[0], v, fmaf(zl[0], vl, fmaf(zh[0], vh, bz[0])));
                            o.y = fmaf(zf[1], v, fmaf(zl[1], vl, fmaf(zh[1], vh, bz[1])));
                            o.z = fmaf(zf[2], v, fmaf(zl[2], vl, fmaf(zh[2], vh, bz[2])));
                            o.w = fmaf(zf[3], v, fmaf(zl[3], vl, fmaf(zh[3], vh, bz[3])));
                            __stcs(reinterpret_cast<float4 *>(dst + r * rstep * row_stride), o);
                        }
                    }
                }
            }
        } else {
            for (int c = 0; c < 3; ++c) {
                float *base = P.eps + ((((size_t)b * 3 + c) * nx + i0) * ny + j0) * nz;
                const float *vc = e2 + c * NCELL;
                for (int f = tid; f < TIv * TJ * nz4; f += NTH) {
                    const int cell = f / nz4, k = (f - cell * nz4) << 2;
                    const int ci = cell / TJ, cj = cell - ci * TJ;
                    if (cj >= TJv) continue;
                    const float v = vc[cell], vl = e2[3 * NCELL + cell], vh = e2[4 * NCELL + cell];
                    float o[4];
#pragma unroll
                    for (int x = 0; x < 4; ++x)
                        o[x] = c < 2 ? fmaf(w_xy[k + x], v, b_xy[k + x])
                                     : fmaf(i_f[k + x], v, fmaf(i_l[k + x], vl, fmaf(i_h[k + x], vh, b_z[k + x])));
                    __stcs(reinterpret_cast<float4 *>(base + ((size_t)ci * ny + cj) * nz + k), make_float4(o[0], o[1], o[2], o[3]));
                }
            }
        }
    }
    if (!rev) return;

    // ---- R1: Eq. (1) product and z-reduction of the staged field windows, all pairs, into G.
    // Warp item = (component, 32 cells of the pass): warp-uniform component, conflict-free reads; a warp owns items w and w + NTH/32.
    for (int cell0 = 0; cell0 < NCELL; cell0 += P.ncp) {
        const int nc = min(P.ncp, NCELL - cell0), ncw = (nc + 31) >> 5, nitem = 3 * ncw;
        const int warp = tid >> 5, lane = tid & 31;
        float acc[2][3] = {{0.f, 0.f, 0.f}, {0.f, 0.f, 0.f}};
        for (int p = 0; p < P.n_pairs; ++p) {
            if (cell0 > 0 || p > 0) {
                __syncthreads();                     // every thread is done reading the previous windows
                zwindow_issue<SPARSE>(P, stage, p, cell0, nc, b, i0, j0);
            }
            cp_async_wait_all();
            __syncthreads();
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int item = warp + u * (NTH / 32);
                if (item < nitem) {
                    const int c = item / ncw, lc = (item - c * ncw) * 32 + lane, cell = cell0 + lc, ci = cell / TJ;
                    zwindow_reduce(P, zw, stage, c, lc, lc < nc && i0 + ci < nx && j0 + (cell - ci * TJ) < ny, acc[u]);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int item = warp + u * (NTH / 32);
            if (item < nitem) {
                const int c = item / ncw, lc = (item - c * ncw) * 32 + lane, cell = cell0 + lc;
                if (lc < nc) {
                    if (c < 2) G[c * NCELL + cell] = acc[u][0];
                    else { G[2 * NCELL + cell] = acc[u][0]; G[3 * NCELL + cell] = acc[u][1]; G[4 * NCELL + cell] = acc[u][2]; }
                }
            }
        }
    }
    __syncthreads();
    if (!in_region) return;
    const int cellg = i * ny + j;
    if (P.gtap) {
        float *gt = P.gtap + (size_t)b * 5 * ncol + cellg;
#pragma unroll
        for (int o = 0; o < 5; ++o) gt[(size_t)o * ncol] = P.accumulate ? gt[(size_t)o * ncol] + G[o * NCELL + tid] : G[o * NCELL + tid];
    }
    if (!P.res) return;

    // ---- R2 + first half of R3 (one thread per cell):  q = 1/eps2d, qbar = -G/q^2, Hbar = n^2 qbar,
    //      Abar = -(1-n^2) qbar/A^2, n2bar = (H - 1/A) qbar -> cotangents of the Sobel gradients
    float *rs = P.res + (size_t)b * TILE_NRES * ncol + cellg;
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
        const float e2d = fast_rcp(n2 * h + (1.0f - n2) * ra);       // eps2d_c = 1/q
        const float qbar = -G[c * NCELL + tid] * e2d * e2d;
        const float hb = n2 * qbar;
        const float ab = -(1.0f - n2) * qbar * ra * ra;
        const float n2bar = (h - ra) * qbar;
        const float k2 = 2.0f * n2bar * gc * rS * rS;
        const float gcb = k2 * (go * go + P.delta), gob = -k2 * gc * go;
        float o4[4] = {hb, ab, c == 0 ? gcb : gob, c == 0 ? gob : gcb};
#pragma unroll
        for (int o = 0; o < 4; ++o) {
            float *dst = rs + (size_t)(4 * c + o) * ncol;
            *dst = P.accumulate ? *dst + o4[o] : o4[o];
        }
    }
    {
        float out = G[2 * NCELL + tid];
        if (P.w_lo > 0.f) out = fmaf(face_factor(P.w_lo, az, inv_ec), G[3 * NCELL + tid], out);
        if (P.w_hi > 0.f) out = fmaf(face_factor(P.w_hi, az, inv_ec), G[4 * NCELL + tid], out);
        float *dst = rs + (size_t)8 * ncol;
        *dst = P.accumulate ? *dst + out : out;
    }
}

}  // namespace epsgrad
