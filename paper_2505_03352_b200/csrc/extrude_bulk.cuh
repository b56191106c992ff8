// extrude_bulk.cuh -- F6 as a thin persistent store stream: the z-extrusion of extrude.cuh with the eps
// columns assembled in shared memory and written by bulk asynchronous copies (cp.async.bulk.global.shared::cta, SASS
// UBLKCP) instead of per-thread 16-byte stores.
//
// Outside the slab every cell of a z column is eps_clad (the layout is extruded to the device layer only), so of
// the nz/4 16-byte pieces of a column only the ones that hold slab cells (2-3 of 16 at paper scale) change from column to
// column.  A CTA keeps EXB_NBUF column blocks [EXB_COLS][nz] in shared memory, filled once with the constant part; per
// work item it rewrites only the window pieces of its columns (the same affine forms as extrude.cuh: bitwise the same
// results) and one thread hands the block to the copy engine.  Per 512-byte column this is 3 shared-memory stores instead
// of 16 global stores with their address arithmetic: the kernel issues ~1/10 of the instructions of k_extrude and needs
// few warps and registers, which leaves the SM's issue slots and load/store pipe to the 2-D kernels that run beside it
// on the auxiliary stream.
// Work items (component c, column block) are walked component by component, gridDim.x apart, so that the CTAs resident at
// any time write one advancing window of one component plane (as a plain fill does).
// Region-sized or x-slab eps only (columns of a plane are one contiguous run); embedded plans keep k_extrude.
#pragma once
#include "common.cuh"
#include "extrude.cuh"

namespace epsgrad {

constexpr int EXB_THREADS = 256, EXB_NBUF = 4;

struct ExtrudeBulkParams {
    const float *e2d;      // [B,5,pstride]: eps2d_x, eps2d_y, eps2d_z, eps_zz lower face, eps_zz upper face
    float *eps;            // [B,3,ncol,nz]
    const float *zw;       // [7][nz] z tables (epsgrad.cu)
    int ncol, nz, pstride; // columns written per plane; cells per column; columns per plane of e2d
    int cols;              // columns per work item: cols * nz * 4 bytes per bulk copy (a multiple of 16)
    int nblk;              // column blocks per component plane
    int q0, nq;            // first 16-byte piece and number of pieces of the union of the x|y and z slab windows
    float eps_clad;
};

__device__ __forceinline__ void bulk_store(void *gdst, const void *ssrc, unsigned bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 :: "l"(gdst), "r"((unsigned)__cvta_generic_to_shared(ssrc)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" :: "n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// grid (n_cta, 1, B), EXB_THREADS threads; dynamic shared memory EXB_NBUF * cols * nz floats
__global__ void __launch_bounds__(EXB_THREADS) k_extrude_bulk(const __grid_constant__ ExtrudeBulkParams P)
{
    extern __shared__ __align__(128) float exb_sm[];
    const int tid = threadIdx.x, b = blockIdx.z, nz = P.nz, nz4 = nz >> 2, cols = P.cols;
    const int blk_floats = cols * nz;
    // constant part: eps_clad everywhere (the window pieces are rewritten for every item)
    {
        const float4 cl = make_float4(P.eps_clad, P.eps_clad, P.eps_clad, P.eps_clad);
        float4 *s4 = reinterpret_cast<float4 *>(exb_sm);
        for (int i = tid; i < EXB_NBUF * cols * nz4; i += EXB_THREADS) s4[i] = cl;
    }
    const float *ed = P.e2d + (size_t)b * 5 * P.pstride;
    float *outb = P.eps + (size_t)b * 3 * P.ncol * nz;
    const int n_items = 3 * P.nblk, nq = P.nq, nwork = cols * nq;     // window pieces per item
    // this thread's (column, piece) pairs of an item: w = tid + r * EXB_THREADS, column lc = w / nq, piece q0 + w % nq
    constexpr int MAXR = 4;                                          // cols * nq <= MAXR * EXB_THREADS (host checks)
    int slot = 0;
    float v[MAXR], vl[MAXR], vh[MAXR];                               // prefetched plane values of the next item
    auto fetch = [&](int item) {
        const int c = item / P.nblk, col0 = (item - c * P.nblk) * cols;
#pragma unroll
        for (int r = 0; r < MAXR; ++r) {
            const int w = tid + r * EXB_THREADS, lc = w / nq, col = col0 + lc;
            v[r] = vl[r] = vh[r] = 0.f;
            if (w < nwork && col < P.ncol) {
                v[r] = __ldg(ed + (size_t)c * P.pstride + col);
                if (c == 2) { vl[r] = __ldg(ed + (size_t)3 * P.pstride + col); vh[r] = __ldg(ed + (size_t)4 * P.pstride + col); }
            }
        }
    };
    int item = blockIdx.x;
    if (item < n_items) fetch(item);
    __syncthreads();
    for (; item < n_items; item += gridDim.x) {
        const int c = item / P.nblk, col0 = (item - c * P.nblk) * cols, ncb = min(cols, P.ncol - col0);
        float *buf = exb_sm + slot * blk_floats;
        // the copy that last read this buffer (EXB_NBUF items ago) must be done reading it
        if (tid == 0) bulk_wait_read<EXB_NBUF - 1>();
        __syncthreads();
#pragma unroll
        for (int r = 0; r < MAXR; ++r) {
            const int w = tid + r * EXB_THREADS;
            if (w < nwork) {
                const int lc = w / nq, q = P.q0 + (w - lc * nq), k = q << 2;
                float4 o;
                if (c < 2) {
                    o.x = fmaf(__ldg(P.zw + k), v[r], __ldg(P.zw + 5 * nz + k));
                    o.y = fmaf(__ldg(P.zw + k + 1), v[r], __ldg(P.zw + 5 * nz + k + 1));
                    o.z = fmaf(__ldg(P.zw + k + 2), v[r], __ldg(P.zw + 5 * nz + k + 2));
                    o.w = fmaf(__ldg(P.zw + k + 3), v[r], __ldg(P.zw + 5 * nz + k + 3));
                } else {
                    float t[4];
#pragma unroll
                    for (int x = 0; x < 4; ++x)
                        t[x] = fmaf(__ldg(P.zw + 2 * nz + k + x), v[r],
                                    fmaf(__ldg(P.zw + 3 * nz + k + x), vl[r], fmaf(__ldg(P.zw + 4 * nz + k + x), vh[r], __ldg(P.zw + 6 * nz + k + x))));
                    o = make_float4(t[0], t[1], t[2], t[3]);
                }
                reinterpret_cast<float4 *>(buf)[lc * nz4 + q] = o;
            }
        }
        const int next = item + gridDim.x;
        if (next < n_items) fetch(next);                             // in flight while the copy below is issued
        fence_async_smem();                                          // generic-proxy writes -> visible to the copy engine
        __syncthreads();
        if (tid == 0) {
            bulk_store(outb + ((size_t)c * P.ncol + col0) * nz, buf, (unsigned)(ncb * nz * 4));
            bulk_commit();
        }
        slot = slot + 1 == EXB_NBUF ? 0 : slot + 1;
    }
    if (tid == 0) bulk_wait_all();                                   // shared memory must outlive the reads; global writes complete
}

}  // namespace epsgrad
