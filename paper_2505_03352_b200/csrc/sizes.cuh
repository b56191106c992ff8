// sizes.cuh -- tile shapes, plane counts and shared-memory budgets that both the plan (plan.cu: workspace carve-up, limits) and
// the kernels need.  Constants only: no kernel lives here, so host-only translation units can include it.
#pragma once
#include <cstddef>

namespace epsgrad {

// 2-D stage (fwd2d.cuh): one CTA per F2_TI x F2_TJ Yee cells
constexpr int F2_TI = 16, F2_TJ = 16, F2_THREADS = 256;
constexpr int F2_NE2D = 5;        // planes: eps2d_x, eps2d_y, eps2d_z, eps_zz on the lower face cell, on the upper face cell
constexpr int F2_NCOEF = 10;      // planes: [hbk, abk, gxk, gyk] for c = x, the same for c = y, flo, fhi

__host__ __device__ inline size_t fwd2d_smem_floats(int s)
{
    const int CI = F2_TI + 2, CJ = F2_TJ + 2;
    const int MP = s * CI + s / 2, MQ = s * CJ + s / 2;
    return (size_t)2 * MP * MQ + 4 * CI * CJ;
}

// mask cotangent (maskgrad.cuh): one CTA per MG_TI x MG_TJ cells
constexpr int MG_TI = 16, MG_TJ = 16, MG_THREADS = 256;
constexpr int MG_CI = MG_TI + 3, MG_CJ = MG_TJ + 3;        // staged cells: [i0-2, i0+TI] x [j0-2, j0+TJ]

__host__ __device__ inline size_t maskgrad_smem_floats(int s)
{
    return (size_t)10 * MG_CI * MG_CJ + MG_TI * MG_TJ + (size_t)s * (MG_TI + MG_TJ);
}

// morphological filters (morph.cuh): MO_T x MO_T mask pixels per CTA, disk radius up to MO_MAX_R pixels
constexpr int MO_T = 32, MO_THREADS = 256, MO_MAX_R = 16;

// u(beta) partial sums (reduce.cuh)
constexpr int UB_THREADS = 256, UB_PER_THREAD = 16;

// tensor-core filter (filter_tc.cuh): 128 = 4 phases x 32 mask columns (8 control columns) by FTC_N control rows per tile
constexpr int FTC_WORKERS = 512, FTC_THREADS = FTC_WORKERS + 64, FTC_TB = 8, FTC_M = 128;   // + the weight-producer warp and the MMA warp
constexpr int FTC_N_RESIDENT = 64, FTC_N_STREAM = 256, FTC_STAGES = 3;   // control rows per tile; stages of the streamed weights' ring
__host__ __device__ constexpr int ftc_k(int NT) { return ((FTC_TB + NT - 1) + 7) / 8 * 8; }          // FTC_TB + 2T rounded up to 8
__host__ __device__ constexpr size_t ftc_a_floats(int NT) { return (size_t)2 * NT * ftc_k(NT) * FTC_M; }   // hi and lo tables
__host__ __device__ constexpr size_t ftc_smem_bytes(int NT, int N, bool stream)
{
    return ((stream ? (size_t)FTC_STAGES * 2 * ftc_k(NT) * FTC_M : ftc_a_floats(NT)) + (size_t)4 * ftc_k(NT) * (N + NT - 1)) * 4 + 128;
}
// tensor-core transposed filter (filterT_tc.cuh): k-steps of 8 of the K = 16 (8 + 2T) values; weight slabs [KS][hi, lo][2][128][4]
__host__ __device__ constexpr int ftt_kq(int NT) { return 4 * (FTC_TB + NT - 1); }            // mask columns a block of 8 control columns reads
__host__ __device__ constexpr int ftt_ksteps(int NT) { return 4 * ftt_kq(NT) / 8; }
__host__ __device__ constexpr size_t ftt_a_floats(int NT) { return (size_t)ftt_ksteps(NT) * 2 * 2 * FTC_M * 4; }
constexpr int FTT_GROUP = 4, FTT_RING = 2, FTT_MAXN = 256;   // k-steps per group (the unit of the rings: 32 KB of weights, 65 KB of data); groups per ring
__host__ __device__ constexpr unsigned ftt_b_step_floats() { return 2 * 2 * (FTT_MAXN * 4 + 16); }   // a data slab: [hi, lo][2 chunks][256 rows + 64 bytes][4 floats]
__host__ __device__ constexpr size_t ftt_smem_bytes(int NT)
{
    // the read-out buffer E [8 NT][FTT_MAXN + 1] reuses the data ring (idle between the last MMA of a tile and the first slab of the next)
    return (size_t)FTT_RING * FTT_GROUP * ((size_t)2 * 2 * FTC_M * 16 + (size_t)ftt_b_step_floats() * 4) + 128;
}

// low 13 mantissa bits cleared: exactly representable as tf32 whatever the unit does with the bits it does not read
__host__ __device__ inline float tf32_trunc(float x)
{
#ifdef __CUDA_ARCH__
    return __uint_as_float(__float_as_uint(x) & 0xffffe000u);
#else
    union { float f; unsigned u; } v; v.f = x; v.u &= 0xffffe000u; return v.f;
#endif
}

// persistent dataflow kernel (mega.cuh): Yee rows per band, phases, ints before the per-band counters of the schedule buffer
constexpr int MK_BAND = 16;
enum { PH_F1 = 0, PH_F2, PH_X, PH_M, PH_T, PH_Z, PH_N };    // the compute list's phases in within-step order, then the field blocks
constexpr int MK_SCHED_HEAD = 8;

}  // namespace epsgrad
