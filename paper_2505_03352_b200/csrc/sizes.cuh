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

// persistent dataflow kernel (mega.cuh): Yee rows per band, phases, ints before the per-band counters of the schedule buffer
constexpr int MK_BAND = 16;
enum { PH_F1 = 0, PH_F2, PH_X, PH_M, PH_T, PH_Z, PH_N };    // the compute list's phases in within-step order, then the field blocks
constexpr int MK_SCHED_HEAD = 8;

}  // namespace epsgrad
