// stream.cuh -- the two HBM streams of eps_forward_vjp in ONE launch.
// k_forward (12 B written per Yee cell) and k_zreduce (slab sectors of E_F, E_A read) are
// independent once the filter has run.  Launched back to back each leaves HBM idle part of the
// time: every forward CTA starts with its 2-D stage (no stores yet), reads and writes never mix,
// and each launch pays its own ramp and tail.  Here a single 1-D grid carries both kinds of CTA,
// interleaved by index in proportion to their counts (Bresenham), so the block scheduler keeps
// both streams in flight: the read stream covers the forward tiles' 2-D stages and the write
// stream's dirty-line write-back overlaps the reads instead of trailing into the next kernel.
#pragma once
#include "forward.cuh"
#include "zreduce.cuh"

namespace epsgrad {

struct StreamParams {
    FwdParams F;
    ZredParams Z;
    int fx, fy, nf;          // forward tiles: fx * fy per design, nf = fx * fy * B in total
    int nbz[2];              // zreduce blocks per plane for {x,y} and {z}
    int nz_blocks;           // zreduce blocks in total: B * (2 nbz[0] + nbz[1])
};

static_assert(FWD_THREADS == ZR_THREADS, "one block size for both roles");

// grid (nf + nz_blocks), dynamic shared memory = fwd_smem_floats
template <int S, int ZR_UNROLL, bool SPARSE>
__global__ void __launch_bounds__(FWD_THREADS, 4) k_stream(const __grid_constant__ StreamParams P)
{
    extern __shared__ __align__(16) float sm[];
    const unsigned long long total = (unsigned long long)P.nf + P.nz_blocks, i = blockIdx.x;
    const int f_before = (int)(i * P.nf / total), f_after = (int)((i + 1) * P.nf / total);
    if (f_after > f_before) {                                    // this block is forward tile f_before
        const int per = P.fx * P.fy, bz = f_before / per, r = f_before - bz * per;
        forward_tile<S>(P.F, sm, r % P.fx, r / P.fx, bz);
    } else {                                                     // zreduce block number i - f_after
        const int z = (int)i - f_after, per = 2 * P.nbz[0] + P.nbz[1];
        const int b = z / per, r = z - b * per;
        const int c = r < P.nbz[0] ? 0 : (r < 2 * P.nbz[0] ? 1 : 2);
        zreduce_block<ZR_UNROLL, SPARSE>(P.Z, r - c * P.nbz[0], c, b);
    }
}

}  // namespace epsgrad
