// zreduce.cuh -- R1 of the reverse pass: Eq. (1) cotangent and its z-reduction.
//   G3 = -2 Re(E_F (.) E_A) = -2 (Re E_F Re E_A - Im E_F Im E_A)           (S10)
//   G[x|y][i,j] = sum_k wxy_k G3[c,i,j,k]                   (transpose of the z-extrusion)
//   eps_zz,k = 1/(wz_k/eps2d_z + (1-wz_k)/eps_clad): its derivative w.r.t. eps2d_z is 1 on full cells (wz_k = 1) and
//   depends on eps2d_z only on the (at most two) fractional face cells, so the z component is reduced to three
//   planes -- full cells, lower face, upper face -- and the mask kernel applies the face factors.  This keeps the
//   field stream independent of the 2-D chain: the kernel depends on nothing but the fields.
// Only the 16-byte chunks (2 complex64 cells) of a z column that hold slab cells are read ("|Omega_D";
// d eps/dC = 0 elsewhere); `dense` plans read every chunk.  A CTA owns one component and ZR_COLS consecutive columns, and
// CTAs are dispatched component by component: the resident CTAs read one advancing window of one component plane of E_F
// and of E_A (measured: 37 us; 48 us when every CTA reads its columns in all three component planes).  A
// CTA starts asynchronous 16-byte copies (LDGSTS) of every window of both fields into shared memory -- no register
// staging, one pass of address arithmetic, up to 5 CTAs x 40 KB in flight per SM -- then each thread multiplies and
// reduces one column out of shared memory.  Sparse windows ask for 64-byte L2 fills: the default fill is the whole
// 128-byte line, and 64 B is the smallest granule the part offers, so a window that straddles a line
// boundary costs 128 B of DRAM traffic per column, component and field instead of 256 B.
#pragma once
#include <cuda.h>          // CUtensorMap (type only: the encoder is fetched through cudaGetDriverEntryPoint)
#include "common.cuh"

namespace epsgrad {

constexpr int ZR_THREADS = 256, ZR_COLS = 256, ZR_MAX_PAIRS = 8;
constexpr int ZR_STAGE_CHUNKS = ZR_COLS * 5;    // staging capacity per field in 16-byte chunks (paper slab: 4 or 5 per column)

struct ZredParams {
    const float4 *ef[ZR_MAX_PAIRS];
    const float4 *ea[ZR_MAX_PAIRS];
    float *gbar;           // [B,5,ncol]: planes x, y, z-full, z-lower-face, z-upper-face
    const float *zw;       // [7][nz] z tables (epsgrad.cu); rows 0 (wxy) and 2..4 (z-full / lower / upper indicators) are used
    int n_pairs, accumulate;
    int ncol, nz, nblk;    // columns read (the whole region, or the rows of an x-slab); nblk = ceil(ncol / ZR_COLS) column blocks per plane
    int pstride;           // columns per plane of gbar (the whole region)
    int ch0[2], nch[2];    // chunk window (chunk = 2 cells = 16 B) for {x,y} and {z}
    int chs[2];            // log2 of the lanes per column of the copy loop: 2^chs >= nch
    ColumnMap cm;          // where the columns sit in E_F / E_A (16-byte pieces = 2 cells)
    int ncp[2];            // columns staged per pass (<= ZR_COLS): ncp (nch | 1) <= ZR_STAGE_CHUNKS
    int choff;             // chunk the stored columns start at: 0, or the first chunk of the union window for packed fields
    int evict_first;       // field fills carry an L2 evict-first policy: they recycle each other's lines instead of pushing out the
                           // dirty eps lines of the step before
};

__host__ __device__ inline int zred_cols_per_pass(int nch, int max_cols = ZR_COLS, int stage_chunks = ZR_STAGE_CHUNKS)
{
    int n = stage_chunks / (nch | 1);
    if (n >= 32) n &= ~31;                 // whole warps of columns
    return n > max_cols ? max_cols : n;
}

// 16-byte asynchronous copy global -> shared (LDGSTS): completion by cp.async groups.
__device__ __forceinline__ unsigned long long policy_evict_first()
{
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// pol: 0, or an L2 cache policy (createpolicy) for the fill
template <bool SPARSE>
__device__ __forceinline__ void cp_async16(float4 *smem, const float4 *g, unsigned long long pol = 0)
{
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    if (pol) {
        if (SPARSE) asm volatile("cp.async.cg.shared.global.L2::cache_hint.L2::64B [%0], [%1], 16, %2;" :: "r"(sa), "l"(g), "l"(pol) : "memory");
        else asm volatile("cp.async.cg.shared.global.L2::cache_hint [%0], [%1], 16, %2;" :: "r"(sa), "l"(g), "l"(pol) : "memory");
        return;
    }
    if (SPARSE) asm volatile("cp.async.cg.shared.global.L2::64B [%0], [%1], 16;" :: "r"(sa), "l"(g) : "memory");
    else asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(sa), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Issue side: copies of the z windows of columns [col0, col0+nc) of component c of design b, fields E_F and E_A of pair p.
// Buffer layout per field: [column][nch | 1] chunks: a column's window stays contiguous, so a returning 32-byte sector
// lands in one shared-memory write (a [chunk][column] layout splits it in two and costs 25 % of the kernel, measured),
// and the odd pitch makes the per-column reads of consecutive threads conflict-free.  2^chs >= nch lanes per column (a
// power of two: no divisions), so a warp instruction covers 32 >> chs neighbouring windows; lanes beyond the window idle.
// HOSTSRC: the fields live in pinned host memory (epsgrad_plan_set_host_direct): plain 16-byte loads, four columns in
// flight per thread, then shared-memory stores -- over PCIe these run 3x faster than LDGSTS (measured), and the bus, not
// the SM, is the limit.
template <bool SPARSE, bool HOSTSRC>
__device__ __forceinline__ void zwindow_issue(const ZredParams &P, float4 *buf, int p, int b, int c, int col0, int nc)
{
    const int grp = c == 2, nch = P.nch[grp], sh = P.chs[grp], ncp = P.ncp[grp];
    const int ch = threadIdx.x & ((1 << sh) - 1), lstep = ZR_THREADS >> sh;
    const unsigned long long pol = P.evict_first ? policy_evict_first() : 0ull;
    if (ch < nch) {
        const size_t first = P.cm.plane(b, c) + (P.ch0[grp] - P.choff) + ch;
        const float4 *pf = P.ef[p] + first, *pa = P.ea[p] + first;
        const int pitch = nch | 1;
        float4 *df = buf + ch, *da = df + pitch * ncp;
        if (HOSTSRC) {
            for (int lc0 = threadIdx.x >> sh; lc0 < nc; lc0 += 4 * lstep) {
                float4 f[4], a[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int lc = lc0 + u * lstep;
                    if (lc < nc) { const size_t o = P.cm.col(col0 + lc); f[u] = ld_stream<false>(pf + o); a[u] = ld_stream<false>(pa + o); }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int lc = lc0 + u * lstep;
                    if (lc < nc) { df[lc * pitch] = f[u]; da[lc * pitch] = a[u]; }
                }
            }
        } else {
            if (!P.cm.embedded) {
                // region-sized fields: constant strides, few instructions per copy
                const int lc0 = threadIdx.x >> sh;
                const size_t o0 = (size_t)(col0 + lc0) * P.cm.col_pitch, ostep = (size_t)lstep * P.cm.col_pitch;
                pf += o0; pa += o0; df += lc0 * pitch; da += lc0 * pitch;
                const int sstep = lstep * pitch;
                for (int lc = lc0; lc < nc; lc += lstep, pf += ostep, pa += ostep, df += sstep, da += sstep) {
                    cp_async16<SPARSE>(df, pf, pol);
                    cp_async16<SPARSE>(da, pa, pol);
                }
            } else {
                for (int lc = threadIdx.x >> sh; lc < nc; lc += lstep) {
                    const size_t o = P.cm.col(col0 + lc);
                    cp_async16<SPARSE>(df + lc * pitch, pf + o, pol);
                    cp_async16<SPARSE>(da + lc * pitch, pa + o, pol);
                }
            }
        }
    }
    cp_async_commit();
}

// Columns [colb, colb + ncb) (ncb <= ZR_COLS) of component c of design b by a CTA of ZR_THREADS threads; stage: 2 fields x ncp x
// (nch | 1) chunks of shared memory.  In two halves, so that a caller can do other work while the first copies are in flight
// (mega.cuh): _begin starts the copies of the first pass of the first pair; _finish waits, reduces and runs the remaining
// passes and pairs.  No barrier at entry or exit: the caller separates calls that reuse `stage`.
template <bool SPARSE, bool HOSTSRC>
__device__ __forceinline__ void block_zreduce_begin(const ZredParams &P, int c, int colb, int ncb, int b, float4 *stage)
{
    zwindow_issue<SPARSE, HOSTSRC>(P, stage, 0, b, c, colb, min(P.ncp[c == 2], ncb));
}

template <bool SPARSE, bool HOSTSRC>
__device__ __forceinline__ void block_zreduce_finish(const ZredParams &P, int c, int colb, int ncb, int b, float4 *stage)
{
    const int tid = threadIdx.x;
    const int grp = c == 2, nch = P.nch[grp], ch0 = P.ch0[grp], ncp = P.ncp[grp], nz = P.nz;
    // a thread reduces one column; the extrusion weights (2 cells per chunk; three rows for component z) are warp-uniform
    // cached loads
    for (int c0 = 0; c0 < ncb; c0 += ncp) {
        const int nc = min(ncp, ncb - c0);
        float acc[3] = {0.f, 0.f, 0.f};
        for (int p = 0; p < P.n_pairs; ++p) {
            if (c0 > 0 || p > 0) {
                __syncthreads();                     // every thread is done reading the previous windows
                zwindow_issue<SPARSE, HOSTSRC>(P, stage, p, b, c, colb + c0, nc);
            }
            cp_async_wait_all();
            __syncthreads();
            if (tid < nc) {
                const int pitch = nch | 1;
                const float4 *bf = stage + tid * pitch, *ba = bf + pitch * ncp;
                for (int ch = 0; ch < nch; ++ch) {
                    const float4 f = bf[ch], a = ba[ch];
                    const int k = 2 * (ch0 + ch);
                    const float g0 = -2.0f * (f.x * a.x - f.y * a.y);       // Eq. (1): -2 Re(E_F E_A), plain product (S10)
                    const float g1 = -2.0f * (f.z * a.z - f.w * a.w);
                    if (grp == 0) {
                        acc[0] = fmaf(__ldg(P.zw + k), g0, fmaf(__ldg(P.zw + k + 1), g1, acc[0]));
                    } else {
#pragma unroll
                        for (int o = 0; o < 3; ++o)
                            acc[o] = fmaf(__ldg(P.zw + (2 + o) * nz + k), g0, fmaf(__ldg(P.zw + (2 + o) * nz + k + 1), g1, acc[o]));
                    }
                }
            }
        }
        if (tid < nc) {
            float *dst = P.gbar + (size_t)b * 5 * P.pstride + colb + c0 + tid;
            const int nout = grp ? 3 : 1;
            for (int o = 0; o < nout; ++o) {
                float *d = dst + (size_t)(grp ? 2 + o : c) * P.pstride;
                *d = P.accumulate ? *d + acc[o] : acc[o];
            }
        }
    }
}

template <bool SPARSE, bool HOSTSRC>
__device__ __forceinline__ void block_zreduce(const ZredParams &P, int c, int colb, int ncb, int b, float4 *stage)
{
    block_zreduce_begin<SPARSE, HOSTSRC>(P, c, colb, ncb, b, stage);
    block_zreduce_finish<SPARSE, HOSTSRC>(P, c, colb, ncb, b, stage);
}

// grid (nblk, 3, B): x fastest, so CTAs are dispatched component by component; dynamic shared memory: 2 fields x ncp x (nch | 1) chunks
template <bool SPARSE, bool HOSTSRC>
__global__ void __launch_bounds__(ZR_THREADS, 5) k_zreduce(const __grid_constant__ ZredParams P)
{
    extern __shared__ __align__(16) float4 stage[];
    const int colb = blockIdx.x * ZR_COLS;
    block_zreduce<SPARSE, HOSTSRC>(P, blockIdx.y, colb, min(ZR_COLS, P.ncol - colb), blockIdx.z, stage);
}

// ---------------------------------------------------------------- TMA variant
// The same reduction with the windows fetched by the tensor memory accelerator: per pass and field ONE bulk tensor copy
// (cp.async.bulk.tensor.2d, box {ZR_TMA_W floats of z} x {256 columns}, L2 promotion 64 B) issued by one thread and tracked
// by an mbarrier, instead of ~3000 LDGSTS instructions per CTA.  Measured at paper scale: 39 us against 37 us for the
// LDGSTS kernel (both DRAM bound), and no better beside the 2-D kernels of the two-stream schedule (the hypothesis that the
// LDGSTS stream's pressure on the SM's memory pipe is what slows them down did not hold), so it is an option
// (epsgrad_plan_set_tma), off by default.  Region-sized (not embedded), device-resident fields with sparse windows only.
// Fields as a 2-D tensor: rows = z columns (B*3*ncol of them), inner dimension = 2 nz floats.  Both window groups use one
// box width ZR box = 4 * max(nch[0] | 1, nch[1] | 1) floats starting at the group's first chunk (a box that sticks out of
// the column is zero-filled by the hardware); the odd chunk pitch keeps the per-column reads conflict-free.
struct ZredTmaParams {
    alignas(64) CUtensorMap mf[ZR_MAX_PAIRS];
    alignas(64) CUtensorMap ma[ZR_MAX_PAIRS];
    float *gbar;
    const float *zw;
    int n_pairs, accumulate;
    int ncol, nz;
    int ch0[2], nch[2];
    int wb;                // box width in 16-byte chunks
};

__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}

__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned phase)
{
    asm volatile(
        "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}\n"
        :: "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(phase) : "memory");
}
__device__ __forceinline__ void tma_load_2d(void *smem, const CUtensorMap *map, unsigned long long *bar, int x, int y)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
                 :: "r"((unsigned)__cvta_generic_to_shared(smem)), "l"(map), "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(x), "r"(y) : "memory");
}

// grid (n_cta, 1, B): persistent CTAs, each walking the (component, column block) items n_cta apart, component by component
// (items of one component are consecutive, so the resident CTAs still read one advancing window); n_cta is chosen on the
// host as a few CTAs per SM, which leaves shared memory, threads and registers of every SM to the 2-D kernels of the other
// stream.  Dynamic shared memory: 2 fields x 256 columns x wb chunks (+ 128 bytes of alignment slack).
__global__ void __launch_bounds__(ZR_THREADS, 5) k_zreduce_tma(const __grid_constant__ ZredTmaParams P)
{
    extern __shared__ unsigned char smraw[];
    __shared__ __align__(8) unsigned long long bar;
    float4 *stage = reinterpret_cast<float4 *>((reinterpret_cast<uintptr_t>(smraw) + 127) & ~(uintptr_t)127);
    const int tid = threadIdx.x, b = blockIdx.y;
    const int nz = P.nz, wb = P.wb, nblk = (P.ncol + ZR_COLS - 1) / ZR_COLS;
    float4 *sf = stage, *sa = stage + ZR_COLS * wb;
    const unsigned box_bytes = (unsigned)ZR_COLS * wb * 16u;
    if (tid == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned phase = 0;
    for (int item = blockIdx.x; item < 3 * nblk; item += gridDim.x) {
        const int c = item / nblk, blk = item - c * nblk;
        const int grp = c == 2, nch = P.nch[grp], ch0 = P.ch0[grp];
        const int colb = blk * ZR_COLS, ncb = min(ZR_COLS, P.ncol - colb);
        const int row0 = (b * 3 + c) * P.ncol + colb;        // < 2^31 by validate()
        float acc[3] = {0.f, 0.f, 0.f};
        for (int p = 0; p < P.n_pairs; ++p) {
            __syncthreads();                                 // every thread is done reading the previous windows
            if (tid == 0) {
                mbar_expect_tx(&bar, 2u * box_bytes);        // rows or floats outside the tensor are zero-filled and still counted
                tma_load_2d(sf, &P.mf[p], &bar, 4 * ch0, row0);
                tma_load_2d(sa, &P.ma[p], &bar, 4 * ch0, row0);
            }
            mbar_wait(&bar, phase);
            phase ^= 1u;
            if (tid < ncb) {
                const float4 *bf = sf + tid * wb, *ba = sa + tid * wb;
                for (int ch = 0; ch < nch; ++ch) {
                    const float4 f = bf[ch], a = ba[ch];
                    const int k = 2 * (ch0 + ch);
                    const float g0 = -2.0f * (f.x * a.x - f.y * a.y);       // Eq. (1): -2 Re(E_F E_A), plain product (S10)
                    const float g1 = -2.0f * (f.z * a.z - f.w * a.w);
                    if (grp == 0) {
                        acc[0] = fmaf(__ldg(P.zw + k), g0, fmaf(__ldg(P.zw + k + 1), g1, acc[0]));
                    } else {
#pragma unroll
                        for (int o = 0; o < 3; ++o)
                            acc[o] = fmaf(__ldg(P.zw + (2 + o) * nz + k), g0, fmaf(__ldg(P.zw + (2 + o) * nz + k + 1), g1, acc[o]));
                    }
                }
            }
        }
        if (tid < ncb) {
            float *dst = P.gbar + (size_t)b * 5 * P.ncol + colb + tid;
            const int nout = grp ? 3 : 1;
            for (int o = 0; o < nout; ++o) {
                float *d = dst + (size_t)(grp ? 2 + o : c) * P.ncol;
                *d = P.accumulate ? *d + acc[o] : acc[o];
            }
        }
    }
}

}  // namespace epsgrad
