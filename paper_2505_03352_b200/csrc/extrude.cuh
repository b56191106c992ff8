// extrude.cuh -- F6: z-extrusion of the 2-D stage to the slab [z_lo, z_hi] with fractional faces (S7, S8).
// Pure store stream: 12 B per Yee cell written with 16-byte streaming stores, 20 B per Yee column read (L2-resident
// planes left by fwd2d.cuh).  Every output is affine in the per-column values:
//   eps_cc[k] = eps_clad (1 - wxy_k) + wxy_k eps2d_c                                         (c = x, y)
//   eps_zz[k] = eps_clad [wz_k = 0] + [wz_k = 1] eps2d_z + [k = lower face] v_lo + [k = upper face] v_hi
// where v_lo, v_hi are Eq. (7) with n = z_hat on the face cells (computed once per column by fwd2d).
// The stream is written the way a plain fill is: a CTA owns one component and one block of consecutive columns, and CTAs
// are dispatched component by component, so the CTAs resident at any time write one contiguous, advancing window of eps
// (a plain fill of the buffer takes 28.8 us; this kernel 34-35 us; 36.5 us when every CTA walks its own three component
// planes).  nz/4 threads share a column, each keeping its
// four z cells and their table entries in registers; a warp store covers 32/(nz/4) neighbouring columns = 512
// contiguous bytes; the block's plane values are staged once in shared memory (coalesced) and read as broadcasts.
#pragma once
#include "common.cuh"

namespace epsgrad {

// the eps store: 16 bytes, streaming (st.global.cs).  EPSGRAD_EPS_STORE selects the alternatives that were timed against it
// (DESIGN.md 5.6): 1 = .cg, 2 = .wt (write-through), 3 = L2 evict-first policy, 4 = L2 evict-last policy.
#ifndef EPSGRAD_EPS_STORE
#define EPSGRAD_EPS_STORE 0
#endif
__device__ __forceinline__ void st_eps(float4 *p, const float4 v)
{
#if EPSGRAD_EPS_STORE == 0
    __stcs(p, v);
#elif EPSGRAD_EPS_STORE == 1
    __stcg(p, v);
#elif EPSGRAD_EPS_STORE == 2
    __stwt(p, v);
#else
    unsigned long long pol;
#if EPSGRAD_EPS_STORE == 3
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
#else
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
#endif
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol) : "memory");
#endif
}

constexpr int EX_THREADS = 256, EX_PASSES = 16, EX_CTAS_PER_SM = 8;

struct ExtrudeParams {
    const float *e2d;      // [B,5,ncol]: eps2d_x, eps2d_y, eps2d_z, eps_zz lower face, eps_zz upper face
    float *eps;            // [B,3,ncol,nz], or the simulation domain's array when embedded (cm)
    ColumnMap cm;          // where the columns sit in eps (16-byte pieces = 4 cells)
    const float *zw;       // [7][nz] z tables (epsgrad.cu)
    int ncol, nz;          // columns written (the whole region, or the rows of an x-slab: epsgrad_plan_set_slab)
    int pstride;           // columns per plane of e2d (the whole region)
    int nblk;              // column blocks per component plane
    int cpb;               // columns per block (extrude_cols_per_block)
    int sh4;               // log2(nz/4) when nz/4 is a power of two <= EX_THREADS (fast path), else -1
};

__host__ __device__ inline int extrude_cols_per_block(int nz)
{
    const int nz4 = nz >> 2;
    return EX_THREADS % nz4 == 0 ? (EX_THREADS / nz4) * EX_PASSES : 64;
}

// Columns [col0, col0 + ncb) (ncb <= cpb) of component c of design b by a CTA of EX_THREADS threads; vsm: 3 cpb floats of shared
// memory (plane values of the block).  No barrier at entry or exit.  CG: the plane values are read through L2 (ld.global.cg) -- for
// the persistent kernel (mega.cuh), where other CTAs of the same launch produce them.
template <bool CG>
__device__ __forceinline__ void block_extrude(const ExtrudeParams &P, int c, int col0, int ncb, int b, float *vsm)
{
    const int tid = threadIdx.x, nz = P.nz, nz4 = nz >> 2;
    const int cpb = P.cpb;
    const float *ed = P.e2d + (size_t)b * 5 * P.pstride;
    float4 *out = reinterpret_cast<float4 *>(P.eps) + P.cm.plane(b, c);
    // stage: c = x, y need their own plane; c = z needs planes 2 (full cells), 3 and 4 (face cells)
    const int npl = c == 2 ? 3 : 1;
    for (int o = 0; o < npl; ++o)
        for (int lc = tid; lc < ncb; lc += EX_THREADS) vsm[o * cpb + lc] = ld_plane<CG>(ed + (size_t)(c + o) * P.pstride + col0 + lc);
    if (P.sh4 >= 0 && !P.cm.embedded) {
        // region-sized eps: the block is one contiguous run; a thread walks it with a constant stride (few instructions per
        // store: the kernel's issue slots are what the 2-D work beside it needs)
        const int kq = tid & (nz4 - 1), k = kq << 2, cq = tid >> P.sh4, cpp = EX_THREADS >> P.sh4;
        float4 *dst = out + (size_t)(col0 + cq) * nz4 + kq;
        const size_t stride = (size_t)cpp * nz4;
        const float *vp = vsm + cq;
        if (c < 2) {
            float wx[4], bx[4];
#pragma unroll
            for (int x = 0; x < 4; ++x) { wx[x] = __ldg(P.zw + k + x); bx[x] = __ldg(P.zw + 5 * nz + k + x); }
            __syncthreads();
            if (ncb == cpb) {
#pragma unroll
                for (int pass = 0; pass < EX_PASSES; ++pass) {
                    const float v = vp[pass * cpp];
                    st_eps(dst + pass * stride, make_float4(fmaf(wx[0], v, bx[0]), fmaf(wx[1], v, bx[1]), fmaf(wx[2], v, bx[2]), fmaf(wx[3], v, bx[3])));
                }
            } else {
                for (int lc = cq; lc < ncb; lc += cpp, dst += stride) {
                    const float v = vsm[lc];
                    st_eps(dst, make_float4(fmaf(wx[0], v, bx[0]), fmaf(wx[1], v, bx[1]), fmaf(wx[2], v, bx[2]), fmaf(wx[3], v, bx[3])));
                }
            }
        } else {
            float bz[4], zf[4], zl[4], zh[4];
#pragma unroll
            for (int x = 0; x < 4; ++x) {
                bz[x] = __ldg(P.zw + 6 * nz + k + x); zf[x] = __ldg(P.zw + 2 * nz + k + x);
                zl[x] = __ldg(P.zw + 3 * nz + k + x); zh[x] = __ldg(P.zw + 4 * nz + k + x);
            }
            __syncthreads();
            for (int lc = cq; lc < ncb; lc += cpp, dst += stride) {
                const float v = vsm[lc], vl = vsm[cpb + lc], vh = vsm[2 * cpb + lc];
                float4 o;
                o.x = fmaf(zf[0], v, fmaf(zl[0], vl, fmaf(zh[0], vh, bz[0])));
                o.y = fmaf(zf[1], v, fmaf(zl[1], vl, fmaf(zh[1], vh, bz[1])));
                o.z = fmaf(zf[2], v, fmaf(zl[2], vl, fmaf(zh[2], vh, bz[2])));
                o.w = fmaf(zf[3], v, fmaf(zl[3], vl, fmaf(zh[3], vh, bz[3])));
                st_eps(dst, o);
            }
        }
    } else if (P.sh4 >= 0) {
        const int kq = tid & (nz4 - 1), k = kq << 2, cq = tid >> P.sh4, cpp = EX_THREADS >> P.sh4;
        float4 *dst = out + kq;
        if (c < 2) {
            float wx[4], bx[4];
#pragma unroll
            for (int x = 0; x < 4; ++x) { wx[x] = __ldg(P.zw + k + x); bx[x] = __ldg(P.zw + 5 * nz + k + x); }
            __syncthreads();
#pragma unroll
            for (int pass = 0; pass < EX_PASSES; ++pass) {
                const int lc = cq + pass * cpp;
                if (lc < ncb) {
                    const float v = vsm[lc];
                    float4 o;
                    o.x = fmaf(wx[0], v, bx[0]); o.y = fmaf(wx[1], v, bx[1]);
                    o.z = fmaf(wx[2], v, bx[2]); o.w = fmaf(wx[3], v, bx[3]);
                    st_eps(dst + P.cm.col(col0 + lc), o);
                }
            }
        } else {
            float bz[4], zf[4], zl[4], zh[4];
#pragma unroll
            for (int x = 0; x < 4; ++x) {
                bz[x] = __ldg(P.zw + 6 * nz + k + x); zf[x] = __ldg(P.zw + 2 * nz + k + x);
                zl[x] = __ldg(P.zw + 3 * nz + k + x); zh[x] = __ldg(P.zw + 4 * nz + k + x);
            }
            __syncthreads();
#pragma unroll
            for (int pass = 0; pass < EX_PASSES; ++pass) {
                const int lc = cq + pass * cpp;
                if (lc < ncb) {
                    const float v = vsm[lc], vl = vsm[cpb + lc], vh = vsm[2 * cpb + lc];
                    float4 o;
                    o.x = fmaf(zf[0], v, fmaf(zl[0], vl, fmaf(zh[0], vh, bz[0])));
                    o.y = fmaf(zf[1], v, fmaf(zl[1], vl, fmaf(zh[1], vh, bz[1])));
                    o.z = fmaf(zf[2], v, fmaf(zl[2], vl, fmaf(zh[2], vh, bz[2])));
                    o.w = fmaf(zf[3], v, fmaf(zl[3], vl, fmaf(zh[3], vh, bz[3])));
                    st_eps(dst + P.cm.col(col0 + lc), o);
                }
            }
        }
    } else {
        // nz/4 does not divide the CTA: flat loop over the 16-byte pieces of the block
        const float *w_xy = P.zw, *b_xy = P.zw + 5 * nz, *b_z = P.zw + 6 * nz, *i_f = P.zw + 2 * nz, *i_l = P.zw + 3 * nz, *i_h = P.zw + 4 * nz;
        __syncthreads();
        for (int f = tid; f < ncb * nz4; f += EX_THREADS) {
            const int lc = f / nz4, k = (f - lc * nz4) << 2;
            const float v = vsm[lc];
            float o[4];
#pragma unroll
            for (int x = 0; x < 4; ++x)
                o[x] = c < 2 ? fmaf(w_xy[k + x], v, b_xy[k + x])
                             : fmaf(i_f[k + x], v, fmaf(i_l[k + x], vsm[cpb + lc], fmaf(i_h[k + x], vsm[2 * cpb + lc], b_z[k + x])));
            st_eps(out + P.cm.col(col0 + lc) + (k >> 2), make_float4(o[0], o[1], o[2], o[3]));
        }
    }
}

// grid (nblk, 3, B): x fastest, so CTAs are dispatched component by component; dynamic shared memory 3 cpb floats
__global__ void __launch_bounds__(EX_THREADS, EX_CTAS_PER_SM) k_extrude(const __grid_constant__ ExtrudeParams P)
{
    extern __shared__ float vsm[];                            // plane values of the block: [3][cpb]
    pdl_launch();
    pdl_wait();
    const int col0 = blockIdx.x * P.cpb;
    block_extrude<false>(P, blockIdx.y, col0, min(P.cpb, P.ncol - col0), blockIdx.z, vsm);
}

}  // namespace epsgrad
