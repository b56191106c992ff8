// zreduce_pipe.cuh -- R1 (Eq. (1) cotangent + z-reduction, zreduce.cuh) as a thin persistent read stream:
// one CTA per SM, the slab windows of E_F and E_A fetched by the tensor memory accelerator through a ring of
// a few shared-memory stages with full / empty mbarriers, so that the copies of the next stages are in flight while the
// consumer warps multiply and reduce the current one.
//   producer: one elected thread; per (item, pair) it waits for the stage to be empty, arms the full barrier with the byte
//             count and issues two bulk tensor copies (cp.async.bulk.tensor.2d, SASS UTMALDG; L2 promotion 64 B: the
//             smallest fill this part offers), box = {window floats} x {ZP_COLS columns};
//   consumers: ZP_COLS threads, one z column each: wait full, Eq. (1) product (plain, S10) and weighted sum over the
//             window out of shared memory, arrive on empty; after the last pair of an item they store the reduced
//             cotangent planes (coalesced).
// Against k_zreduce (LDGSTS, 5 CTAs x 40 KB per SM) the kernel holds 160 threads and its stages (~100 KB) per SM and issues
// no per-column load instructions, which leaves the SM's warp slots, shared memory and load/store pipe to the 2-D kernels
// of the auxiliary stream.  Same arithmetic in the same order as k_zreduce: bitwise equal results.
// Fields as a 2-D tensor: rows = z columns (B*3*ncol), inner dimension = 2 nz floats (region-sized or x-slab arrays).
#pragma once
#include "zreduce.cuh"

namespace epsgrad {

constexpr int ZP_COLS = 128, ZP_MAX_STAGE = 12, ZP_CONSUMERS = ZP_COLS, ZP_THREADS = ZP_CONSUMERS + 32;

struct ZredPipeParams {
    alignas(64) CUtensorMap mf[ZR_MAX_PAIRS];
    alignas(64) CUtensorMap ma[ZR_MAX_PAIRS];
    float *gbar;           // [B,5,pstride]
    const float *zw;       // [7][nz]
    int n_pairs, accumulate;
    int ncol, nz, pstride; // columns read per plane (region or x-slab rows), cells per column, columns per plane of gbar
    int ch0[2], nch[2];    // chunk window (chunk = 2 cells = 16 B) for {x,y} and {z}
    int wb;                // box width in 16-byte chunks (odd: conflict-free column reads)
    int nblk;              // column blocks per plane
    int nstage;            // stages of the shared-memory ring (2..ZP_MAX_STAGE)
};

__host__ __device__ inline size_t zpipe_smem_bytes(int wb, int nstage)
{
    return (size_t)nstage * 2 * ZP_COLS * wb * 16 + 128 /* alignment slack */ + 2 * ZP_MAX_STAGE * 8;
}

// grid (n_cta, 1, B): persistent CTAs, each walking the (component, column block) items n_cta apart, component by component
__global__ void __launch_bounds__(ZP_THREADS) k_zreduce_pipe(const __grid_constant__ ZredPipeParams P)
{
    extern __shared__ unsigned char zp_raw[];
    unsigned char *base = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(zp_raw) + 127) & ~(uintptr_t)127);
    const int wb = P.wb, NS = P.nstage;
    const unsigned stage_bytes = 2u * ZP_COLS * wb * 16u;
    unsigned long long *full = reinterpret_cast<unsigned long long *>(base + (size_t)NS * stage_bytes);
    unsigned long long *empty = full + ZP_MAX_STAGE;
    const int tid = threadIdx.x, b = blockIdx.z, nz = P.nz, nblk = P.nblk, n_items = 3 * nblk;

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, ZP_CONSUMERS); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (tid >= ZP_CONSUMERS) {
        // ---- producer warp: one thread issues every copy
        if (tid == ZP_CONSUMERS) {
            int s = 0; unsigned ph = 0;
            for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
                const int c = item / nblk, blk = item - c * nblk, grp = c == 2;
                const int row0 = (b * 3 + c) * P.ncol + blk * ZP_COLS, x0 = 4 * P.ch0[grp];
                for (int p = 0; p < P.n_pairs; ++p) {
                    mbar_wait(empty + s, ph ^ 1u);               // first round: passes at once (fresh barrier, parity trick)
                    unsigned char *sf = base + (size_t)s * stage_bytes;
                    mbar_expect_tx(full + s, stage_bytes);       // out-of-tensor rows / floats are zero-filled and still counted
                    tma_load_2d(sf, &P.mf[p], full + s, x0, row0);
                    tma_load_2d(sf + stage_bytes / 2, &P.ma[p], full + s, x0, row0);
                    if (++s == NS) { s = 0; ph ^= 1u; }
                }
            }
        }
        return;
    }

    // ---- consumers: thread <-> column
    int s = 0; unsigned ph = 0;
    for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
        const int c = item / nblk, blk = item - c * nblk, grp = c == 2;
        const int nch = P.nch[grp], ch0 = P.ch0[grp];
        const int colb = blk * ZP_COLS, ncb = min(ZP_COLS, P.ncol - colb);
        float acc[3] = {0.f, 0.f, 0.f};
        for (int p = 0; p < P.n_pairs; ++p) {
            mbar_wait(full + s, ph);
            const float4 *bf = reinterpret_cast<const float4 *>(base + (size_t)s * stage_bytes) + tid * wb, *ba = bf + ZP_COLS * wb;
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
            mbar_arrive(empty + s);                              // this thread is done reading the stage
            if (++s == NS) { s = 0; ph ^= 1u; }
        }
        if (tid < ncb) {
            float *dst = P.gbar + (size_t)b * 5 * P.pstride + colb + tid;
            const int nout = grp ? 3 : 1;
            for (int o = 0; o < nout; ++o) {
                float *d = dst + (size_t)(grp ? 2 + o : c) * P.pstride;
                *d = P.accumulate ? *d + acc[o] : acc[o];
            }
        }
    }
}

}  // namespace epsgrad
