// filter4.cuh -- fast paths of the conic polyphase stencil (filter.cuh) for m = u*s = 4 and a
// compile-time tap count NTC = 2T+1 in {5, 9, 13} (R = 4, 8, 12 cells at u = 2).
//
// Both directions use the same decomposition:
//   - 4 lanes per group of NB = 4 neighbouring control pixels along y; lane `sp` owns phase row
//     fx = sp of those pixels (4 phase columns fy), so 16 (forward) / 16 (reverse) independent
//     accumulators per lane and 4x the warps of a thread-per-pixel mapping;
//   - per tap row tx the lane first pulls the NTC weight vectors W[tx][*][sp][0..3] into registers
//     (warp-wide that is one 64-byte broadcast each), then sweeps the NTC+3 source columns, each
//     loaded value feeding up to NB outputs:  shared-memory wavefronts per FMA drop from 1.25
//     (reverse) / 0.31 (forward) to 0.40 / 0.15 -- the earlier kernels were shared-memory bound
//     (profiles/r1a_ncu_full_summary.md).
// Forward reads c' (control resolution, scalar, conflict-free); reverse reads the v tile staged with
// one padding block after every 4 (block c at float offset 4(c + c/4)): lanes of a quarter-warp then
// hit 8 distinct 16-byte bank groups.
#pragma once
#include "filter.cuh"

namespace epsgrad {

constexpr int F4_NB = 4, F4_TA = 4, F4_TB = 8 * F4_NB, F4_THREADS = 32 * F4_TA;

constexpr int F4_G = 3, F4F_THREADS = F4_THREADS * F4_G;     // forward: tap rows split over F4_G warp groups (see the transpose below)

// 16-byte asynchronous copy with zero fill: src_bytes = 16 copies, 0 writes zeros (the source address is not read)
__device__ __forceinline__ void f4_cp_async16_zfill(float *smem, const float *g, int src_bytes)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;"
                 :: "r"((unsigned)__cvta_generic_to_shared(smem)), "l"(g), "r"(src_bytes) : "memory");
}

// the weight table W[NTC][NTC][4][4] into shared memory by asynchronous copies (not committed: the caller's next
// cp.async.commit_group / wait_group covers them)
template <int NTC>
__device__ __forceinline__ void f4_stage_weights(float *w_s, const float *w, int nthr)
{
    for (int i = threadIdx.x; i < NTC * NTC * 4; i += nthr) f4_cp_async16_zfill(w_s + 4 * i, w + 4 * i, 16);
}

__host__ __device__ inline size_t filter4_smem_floats(int NT)
{
    const int T = (NT - 1) / 2;
    return (size_t)NT * NT * 16 + (size_t)(F4_TA + 2 * T) * (F4_TB + 2 * T + 1) + (size_t)F4_G * F4_THREADS * 16;
}

// One tile of 4 x 32 control pixels (16 x 128 mask pixels) by a CTA of 32*F4_TA*G threads: warp <-> (tap-row group g,
// control row la), lane = sp*8 + lb.  w_s: the weight table [NTC][NTC][4][4] in shared memory (16-byte aligned; filled by
// the caller, barrier included in here); scratch: (TA+2T)*CW + 3 + G*F4_THREADS*16 floats.
template <int NTC, int G>
__device__ __forceinline__ void tile_filter_conic4(const FilterParams &P, int bx, int by, int b, const float *w_s, float *scratch)
{
    constexpr int T = (NTC - 1) / 2, TA = F4_TA, TB = F4_TB, NB = F4_NB, CW = TB + 2 * T + 1;
    constexpr int TXPG = (NTC + G - 1) / G, NTHR = F4_THREADS * G;
    float *c_s = scratch;                          // [(TA+2T)][CW]
    float *part = c_s + (TA + 2 * T) * CW;         // [G][jb][j][F4_THREADS] partial sums
    part += (4 - (((uintptr_t)part >> 2) & 3)) & 3;                     // 16-byte aligned (one float4 of slack is in the budget)
    const int tid = threadIdx.x;
    const int a_base = by * TA, b_base = bx * TB;

    const float *Cb = P.C + (size_t)b * P.mx * P.my;
    for (int r = tid >> 5; r < TA + 2 * T; r += NTHR / 32) {
        const int a = a_base - T + r;
        for (int c = tid & 31; c < TB + 2 * T; c += 32) {
            const int bb = b_base - T + c;
            float v = 0.0f;
            if (a >= 0 && a < P.mx && bb >= 0 && bb < P.my) v = Cb[(size_t)a * P.my + bb] - P.eta0;
            c_s[r * CW + c] = v;
        }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");      // the caller's copies of the weight table, if any
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    __syncthreads();

    const int warp = tid >> 5, g = warp / TA, la = warp - g * TA, lane = tid & 31, sp = lane >> 3, lb = lane & 7;
    float acc[NB][4];
#pragma unroll
    for (int jb = 0; jb < NB; ++jb)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[jb][j] = 0.0f;

    const int tx0 = g * TXPG, tx1 = min(tx0 + TXPG, NTC);
#pragma unroll 1
    for (int tx = tx0; tx < tx1; ++tx) {
        float wr[NTC][4];
#pragma unroll
        for (int ty = 0; ty < NTC; ++ty) lds_vec<4>(w_s + ((tx * NTC + ty) * 4 + sp) * 4, wr[ty]);
        const float *crow = c_s + (la + tx) * CW + NB * lb;
#pragma unroll
        for (int k = 0; k < NTC + NB - 1; ++k) {       // source column b0 + jb + ty - T, k = jb + ty
            const float cv = crow[k];
#pragma unroll
            for (int jb = 0; jb < NB; ++jb) {
                const int ty = k - jb;
                if (ty >= 0 && ty < NTC) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) acc[jb][j] = fmaf(wr[ty][j], cv, acc[jb][j]);
                }
            }
        }
    }
    // partial sums meet in shared memory: slot (la, lane) of group g, one float4 per jb; consecutive lanes, consecutive float4
    const int slot = la * 32 + lane;
#pragma unroll
    for (int jb = 0; jb < NB; ++jb)
        reinterpret_cast<float4 *>(part)[(g * NB + jb) * F4_THREADS + slot] = make_float4(acc[jb][0], acc[jb][1], acc[jb][2], acc[jb][3]);
    __syncthreads();
    // (jb, slot) pairs over all threads: sum the groups, apply the normaliser, store
    for (int it = tid; it < NB * F4_THREADS; it += NTHR) {
        const int jb = it / F4_THREADS, sl = it - jb * F4_THREADS;
        const int la2 = sl >> 5, ln = sl & 31, sp2 = ln >> 3, lb2 = ln & 7;
        const int a0 = a_base + la2, b0 = b_base + NB * lb2 + jb;
        float4 o = reinterpret_cast<const float4 *>(part)[jb * F4_THREADS + sl];
#pragma unroll
        for (int gg = 1; gg < G; ++gg) {
            const float4 t = reinterpret_cast<const float4 *>(part)[(gg * NB + jb) * F4_THREADS + sl];
            o.x += t.x; o.y += t.y; o.z += t.z; o.w += t.w;
        }
        if (a0 >= P.mx || b0 >= P.my) continue;
        const int nix = P.nrm.ix(a0, sp2), niy = P.nrm.iy(b0, 0);
        o.x *= P.nrm.at_index(nix, niy);
        o.y *= P.nrm.at_index(nix, niy + 1);
        o.z *= P.nrm.at_index(nix, niy + 2);
        o.w *= P.nrm.at_index(nix, niy + 3);
        *reinterpret_cast<float4 *>(P.phi + ((size_t)b * P.px + 4 * a0 + sp2) * P.py + 4 * b0) = o;
    }
}

// grid (ceil(my/32), ceil(mx/4), B), 384 threads
template <int NTC>
__global__ void __launch_bounds__(F4F_THREADS) k_filter_conic4(const FilterParams P)
{
    extern __shared__ __align__(16) float sm[];
    f4_stage_weights<NTC>(sm, P.w, F4F_THREADS);
    pdl_launch();
    pdl_wait();                                    // Phi' may still be read by the kernel before (the previous call's reverse pass)
    tile_filter_conic4<NTC, F4_G>(P, blockIdx.x, blockIdx.y, blockIdx.z, sm, sm + NTC * NTC * 16);
}

// ---------------------------------------------------------------- transpose
// The tap rows tx are split over F4T_G warp groups (each warp of a group owns one control row of the tile), so a CTA
// carries F4T_G * F4_TA warps instead of F4_TA: the kernel is latency bound (one wave of ~500 CTAs), and the extra warps
// are what hides the shared-memory and FMA latencies.  Partial sums meet in shared memory.  The v tile is staged with
// 16-byte asynchronous copies (zero-filled outside the mask), all in flight at once.
constexpr int F4T_G = 3, F4T_THREADS = 32 * F4_TA * F4T_G;

__host__ __device__ inline int filterT4_pitch(int T) { const int nb = F4_TB + 2 * T; return 4 * (nb + (nb + 3) / 4); }
__host__ __device__ inline size_t filterT4_smem_floats(int NT)
{
    const int T = (NT - 1) / 2;
    return (size_t)NT * NT * 16 + (size_t)4 * (F4_TA + 2 * T) * filterT4_pitch(T) + (size_t)F4T_G * F4_TA * F4_TB;
}


// rows of the v tile a CTA stages per pass when the NTC tap rows are processed in PASSES passes
__host__ __device__ constexpr int filterT4_tile_rows(int NTC, int PASSES) { return 4 * (F4_TA + (NTC + PASSES - 1) / PASSES - 1); }

// One tile of 4 x 32 control pixels by a CTA of 32*F4_TA*G threads.  w_s: the weight table in shared memory (filled by the
// caller before the call; the barrier after the v tile has landed covers it); scratch: filterT4_tile_rows * pitch + G*TA*TB floats,
// 16-byte aligned.  The tap rows are processed in PASSES passes, each staging only the v rows its tap rows reach (PASSES = 1: the
// whole (TA+2T)-row tile at once; more passes: less shared memory, one more load phase each); within a pass the tap rows are
// split over the G warp groups.  The v tile is read through L2 (cp.async.cg).
template <int NTC, int G, int PASSES>
__device__ __forceinline__ void tile_filterT_conic4(const FilterTParams &P, int bx, int by, int b, const float *w_s, float *scratch)
{
    constexpr int T = (NTC - 1) / 2, TA = F4_TA, TB = F4_TB, NB = F4_NB;
    constexpr int TXPP = (NTC + PASSES - 1) / PASSES;              // tap rows per pass
    constexpr int TXPG = (TXPP + G - 1) / G, NTHR = F4_THREADS * G;   // tap rows per warp group within a pass
    constexpr int VH = filterT4_tile_rows(NTC, PASSES), VB = TB + 2 * T;       // v tile: rows, blocks of 4 floats per row
    const int pitch = filterT4_pitch(T);
    float *v_s = scratch;                          // [VH][pitch], block c at 4(c + c/4)
    float *part = v_s + VH * pitch;                // [G][TA][TB] partial sums
    const int tid = threadIdx.x;
    const int a_base = by * TA, b_base = bx * TB;
    const float *vb = P.v + (size_t)b * P.px * P.py;
    const int q_base = 4 * (b_base - T);
    const int warp = tid >> 5, g = warp / TA, la = warp - g * TA, lane = tid & 31, sp = lane >> 3, lb = lane & 7;
    float acc[NB][4];
#pragma unroll
    for (int jb = 0; jb < NB; ++jb)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[jb][j] = 0.0f;

#pragma unroll 1
    for (int pass = 0; pass < PASSES; ++pass) {
        const int txa = pass * TXPP, txb = min(txa + TXPP, NTC);          // tap rows of this pass
        // forward used node a = a0 + (tx-T): source block row a - (tx-T), local la + 2T - tx in [2T - (txb-1), TA-1 + 2T - txa]
        const int row_lo = 2 * T - (txb - 1), nrow = 4 * (TA + txb - txa - 1);
        const int p_base = 4 * (a_base - T + row_lo);
        if (PASSES > 1 && pass > 0) __syncthreads();                       // every warp is done with the previous pass's rows
        for (int r = tid >> 5; r < nrow; r += NTHR / 32) {
            const int p = p_base + r;
            const bool rin = p >= 0 && p < P.px;
            for (int c = tid & 31; c < VB; c += 32) {
                const int q = q_base + 4 * c;
                const bool in = rin && q >= 0 && q < P.py;
                f4_cp_async16_zfill(v_s + r * pitch + 4 * (c + (c >> 2)), in ? vb + (size_t)p * P.py + q : vb, in ? 16 : 0);
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncthreads();

        const int tx0 = txa + g * TXPG, tx1 = min(tx0 + TXPG, txb);
#pragma unroll 1
        for (int tx = tx0; tx < tx1; ++tx) {
            float wr[NTC][4];
#pragma unroll
            for (int ty = 0; ty < NTC; ++ty) lds_vec<4>(w_s + ((tx * NTC + ty) * 4 + sp) * 4, wr[ty]);
            const float *vrow = v_s + (4 * (la + 2 * T - tx - row_lo) + sp) * pitch;
#pragma unroll
            for (int k = 0; k < NTC + NB - 1; ++k) {       // source block column NB*lb + k;  k = jb + 2T - ty
                const int c = NB * lb + k;
                float vv[4];
                lds_vec<4>(vrow + 4 * (c + (c >> 2)), vv);
#pragma unroll
                for (int jb = 0; jb < NB; ++jb) {
                    const int ty = jb + 2 * T - k;
                    if (ty >= 0 && ty < NTC) {
#pragma unroll
                        for (int j = 0; j < 4; ++j) acc[jb][j] = fmaf(wr[ty][j], vv[j], acc[jb][j]);
                    }
                }
            }
        }
    }
#pragma unroll
    for (int jb = 0; jb < NB; ++jb) {
        float s = (acc[jb][0] + acc[jb][1]) + (acc[jb][2] + acc[jb][3]);
        s += __shfl_xor_sync(0xffffffffu, s, 8);
        s += __shfl_xor_sync(0xffffffffu, s, 16);
        if (sp == 0) part[(g * TA + la) * TB + NB * lb + jb] = s;
    }
    __syncthreads();
    if (tid < TA * TB) {
        const int a = a_base + tid / TB, bb = b_base + tid % TB;
        float s = 0.0f;
#pragma unroll
        for (int gg = 0; gg < G; ++gg) s += part[gg * TA * TB + tid];
        if (a < P.mx && bb < P.my) P.dC[((size_t)b * P.mx + a) * P.my + bb] = s;
    }
}

// grid (ceil(my/32), ceil(mx/4), B), 384 threads
template <int NTC>
__global__ void __launch_bounds__(F4T_THREADS) k_filterT_conic4(const FilterTParams P)
{
    extern __shared__ __align__(16) float sm[];
    f4_stage_weights<NTC>(sm, P.w, F4T_THREADS);      // the table is the plan's: staged while the mask cotangent is still being written
    pdl_launch();
    pdl_wait();
    tile_filterT_conic4<NTC, F4T_G, 1>(P, blockIdx.x, blockIdx.y, blockIdx.z, sm, sm + NTC * NTC * 16);
}

}  // namespace epsgrad
