// mega.cuh -- the whole path (F1..F6, R1..R6) as ONE persistent dataflow kernel.
//
// The six kernels of a step are cut into work items -- filter tiles (F1), 2-D-stage tiles (F2), eps column blocks (X = F6),
// field column blocks (Z = R1), mask-cotangent tiles (M = R2-R5), transposed-filter tiles (T = R6) -- that are grouped in
// BANDS of 16 Yee rows (8 control rows, 32 mask rows).  An item of band b depends only on items of bands b-1..b+1 of the
// phase(s) before it:
//      F2[b] <- F1[b-1..b+1]     X[b] <- F2[b]     M[b] <- F2[b-1..b+1], Z[b-1..b+1]     T[b] <- M[b-1..b+1]
// (filter reach 4T <= 32 mask rows; half-cell shift, averages and Sobel ring <= 2 cells).  Every phase counts its finished
// items per band in global memory; an item starts when the counters of the bands it needs are complete.
// Items are handed out from two ticket lists (atomicAdd), both sorted by pipeline step  tau = band + lag[phase]:
//      compute list:  F1[t], F2[t-lag_F2], X[t-lag_X], M[t-lag_M], T[t-lag_T]
//      field list:    Z[t]                                       (no inputs but the fields: can always start)
// and every dependence points to a smaller tau.  Every CTA runs the same loop: take a field block and START its asynchronous
// copies (LDGSTS into its own staging buffer); take a compute item, wait for its bands, run it -- the copies land meanwhile --;
// then multiply and reduce the field block.  While a compute item's bands are incomplete the CTA finishes and starts more
// field blocks instead of idling.  This cannot deadlock: a CTA never blocks while it holds work it could run; the earliest
// unfinished compute item has all its inputs (they have a smaller tau) or needs field blocks, which every waiting CTA
// works on; and it is either held by a CTA (which then runs it) or the next ticket, which the next free CTA takes.
// What it buys over six launches: no launch ramps and tails between phases; DRAM latency of the field reads is hidden behind
// the ALU work of the same CTA; and every intermediate (Phi', eps2d, coefficients, G, v) is consumed a few bands after it was
// produced, from L2, at any problem size.
// Same tile arithmetic as the stand-alone kernels, except the summation order over the filter's tap rows (two warp groups).
#pragma once
#include "filter4.cuh"
#include "fwd2d.cuh"
#include "extrude.cuh"
#include "zreduce.cuh"
#include "maskgrad.cuh"

namespace epsgrad {

constexpr int MK_THREADS = 256, MK_G = 2;                   // CTA size; tap-row groups of the filter tiles (MK_BAND: sizes.cuh)
constexpr int MK_TPASS = 2;                                  // passes of a transposed-filter tile over its tap rows (shared memory)
constexpr int MK_ZCOLS = 128;                                // z columns per field block (20 KB of staging at 5 chunks per column)
constexpr int MK_NCOMPUTE = 5;

static_assert(F4_THREADS * MK_G == MK_THREADS && F2_THREADS == MK_THREADS && MG_THREADS == MK_THREADS &&
              ZR_THREADS == MK_THREADS && EX_THREADS == MK_THREADS, "one CTA size for every role");
static_assert(F2_TI == MK_BAND && MG_TI == MK_BAND && 2 * 4 * F4_TA == 2 * MK_BAND, "a band is one 2-D tile row and two filter tile rows");
static_assert(MK_ZCOLS <= ZR_COLS, "a thread per column in the reduction");

struct MegaParams {
    FilterParams f1; Fwd2dParams f2; ExtrudeParams ex; ZredParams zr; MaskGradParams mg; FilterTParams ft;
    int *sched;                     // [0] compute-list ticket, [1] field-block ticket, [MK_SCHED_HEAD + ph*B*nb + d*nb + b] finished items
    int B, nb;                      // designs; bands per design
    int full[PH_N], last[PH_N];     // items of a phase in a full band / in the last band of a design (0, 0: phase off)
    int lag[PH_N];                  // band b of phase ph belongs to pipeline step b + lag[ph]
    int nbx1, nbx2;                 // tiles per tile row: (transposed) filter (32 control columns); 2-D stage / mask cotangent (16 cells)
    int zblk[2], xblk[2];           // column blocks per component in a full band / in the last band
    int w_floats, scratch_floats;   // shared memory: filter weight table, the compute items' scratch, then the field staging
    unsigned long long *prof;       // nullptr, or [2*PH_N + 4] sums over all CTAs: cycles per phase, items per phase, tickets, total, waiting for bands, releases
};

__host__ __device__ inline int mk_prefix(const MegaParams &P, int ph, int k)      // items of phase ph in bands [0, k)
{
    if (k <= 0) return 0;
    return k < P.nb ? k * P.full[ph] : (P.nb - 1) * P.full[ph] + P.last[ph];
}
__host__ __device__ inline int mk_count(const MegaParams &P, int ph, int b) { return b == P.nb - 1 ? P.last[ph] : P.full[ph]; }

__host__ __device__ inline int mk_step_start(const MegaParams &P, int t)   // compute items in steps [0, t) of one design
{
    int s = 0;
    for (int ph = 0; ph < MK_NCOMPUTE; ++ph) {
        int kb = t - P.lag[ph];
        if (kb > P.nb) kb = P.nb;
        s += mk_prefix(P, ph, kb);
    }
    return s;
}

__device__ __forceinline__ int ld_acquire(const int *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// Are the bands that item (ph, d, b) reads complete?  Called by warp 0; lanes 0-2 look at bands b-1..b+1 of the first
// producer phase, lanes 3-5 at those of the second one (M only).  Non-blocking; the verdict is warp-uniform.
__device__ __forceinline__ bool mk_ready(const MegaParams &P, const int *done, int ph, int d, int b, int lane)
{
    bool ok = true;
    if (lane < 6) {
        int dp = -1;
        if (lane < 3) dp = ph == PH_F2 ? PH_F1 : (ph == PH_X ? PH_F2 : (ph == PH_M ? PH_F2 : (ph == PH_T ? PH_M : -1)));
        else if (ph == PH_M) dp = PH_Z;
        const int bb = b + (lane % 3) - 1;
        if (dp >= 0 && bb >= 0 && bb < P.nb && (ph != PH_X || bb == b))
            ok = ld_acquire(done + (dp * P.B + d) * P.nb + bb) >= mk_count(P, dp, bb);
    }
    return __all_sync(0xffffffffu, ok);
}

// grid (n_cta), MK_THREADS threads; dynamic shared memory: weight table + compute scratch + field staging
template <int NTC, bool SPARSE>
__global__ void __launch_bounds__(MK_THREADS, 4) k_mega(const __grid_constant__ MegaParams P)
{
    extern __shared__ __align__(16) float sm[];
    __shared__ int s_c[4], s_z[4], s_flag;
    float *w_s = sm, *scratch = sm + P.w_floats;
    float4 *zstage = reinterpret_cast<float4 *>(scratch + P.scratch_floats);
    const int tid = threadIdx.x, lane = tid & 31;
    int *done = P.sched + MK_SCHED_HEAD;

    f4_stage_weights<NTC>(w_s, P.f1.w, MK_THREADS);
    asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group 0;" ::: "memory");

    const int c_per_design = mk_step_start(P, 1 << 28), z_per_design = mk_prefix(P, PH_Z, P.nb);
    const int c_total = c_per_design * P.B, z_total = z_per_design * P.B;
    bool c_exh = c_total == 0, z_exh = z_total == 0, zpend = false;
    int cur_t = 0, cur_d = 0;                                  // decode cursor of the compute list (thread 0)
    int zc = 0, zd = 0, zb = 0, zcolb = 0, zncb = 0;           // the field block in flight

    __shared__ long long s_prof[2 * PH_N + 8];                 // thread 0's cycle accounting (P.prof only)
    if (P.prof && tid == 0) {
        for (int q = 0; q < 2 * PH_N + 8; ++q) s_prof[q] = 0;
        s_prof[2 * PH_N + 1] = clock64();
    }
    auto account = [&](int slot, long long t0, int items) {    // slot: phase; 2*PH_N: tickets; 2*PH_N+2: waiting for bands; +3: release
        if (P.prof && tid == 0) { s_prof[slot] += clock64() - t0; if (items) s_prof[PH_N + slot] += items; }
    };

    auto publish = [&](int ph, int d, int b) {                 // after a barrier that follows the item's global writes
        if (tid == 0)
            asm volatile("red.release.gpu.global.add.s32 [%0], 1;" :: "l"(done + (ph * P.B + d) * P.nb + b) : "memory");
    };
    auto z_decode_begin = [&]() {                              // s_z holds a fresh ticket (or -1): start its copies
        const int n = s_z[0];
        if (n < 0) return;
        zd = n / z_per_design;
        int r = n - zd * z_per_design;
        zb = r / P.full[PH_Z];                                 // every band but the last has full[] blocks
        if (zb >= P.nb) zb = P.nb - 1;
        r -= zb * P.full[PH_Z];
        const int nblk = P.zblk[zb == P.nb - 1];
        zc = r / nblk;
        const int blk = r - zc * nblk;
        const int col0 = zb * MK_BAND * P.f2.ny, cend = min(P.f2.nx, (zb + 1) * MK_BAND) * P.f2.ny;
        zcolb = col0 + blk * MK_ZCOLS;
        zncb = min(MK_ZCOLS, cend - zcolb);
        block_zreduce_begin<SPARSE, false>(P.zr, zc, zcolb, zncb, zd, zstage);
        zpend = true;
    };
    auto z_finish = [&]() {
        const long long t0 = clock64();
        block_zreduce_finish<SPARSE, false>(P.zr, zc, zcolb, zncb, zd, zstage);
        __syncthreads();
        publish(PH_Z, zd, zb);
        zpend = false;
        account(PH_Z, t0, 1);
    };

    for (;;) {
        const long long t_a = clock64();
        // ---- tickets: a field block to prefetch (lane 0) and a compute item (lane 1), taken in parallel
        if (tid < 32) {
            int zn = -1, cn = -1;
            if (lane == 0 && !zpend && !z_exh) { zn = atomicAdd(P.sched + 1, 1); if (zn >= z_total) zn = -1; }
            if (lane == 1 && !c_exh) { cn = atomicAdd(P.sched + 0, 1); if (cn >= c_total) cn = -1; }
            if (lane == 0) s_z[0] = zn;
            if (lane == 1) {
                int ph = -1, d = 0, b = 0, idx = 0;
                if (cn >= 0) {
                    d = cn / c_per_design;
                    int r = cn - d * c_per_design;
                    int t = cur_d == d ? cur_t : 0;
                    while (r >= mk_step_start(P, t + 1)) ++t;
                    cur_t = t; cur_d = d;
                    r -= mk_step_start(P, t);
                    for (int q = 0; q < MK_NCOMPUTE; ++q) {
                        const int bb = t - P.lag[q];
                        if (bb < 0 || bb >= P.nb) continue;
                        const int cnt = mk_count(P, q, bb);
                        if (r < cnt) { ph = q; b = bb; idx = r; break; }
                        r -= cnt;
                    }
                }
                s_c[0] = ph; s_c[1] = d; s_c[2] = b; s_c[3] = idx;
            }
        }
        __syncthreads();
        account(2 * PH_N, t_a, 0);
        const long long t_z = clock64();
        if (!zpend && !z_exh) { if (s_z[0] < 0) z_exh = true; else z_decode_begin(); }
        const int ph = c_exh ? -1 : s_c[0], d = s_c[1], b = s_c[2], idx = s_c[3];
        if (ph < 0) c_exh = true;
        account(2 * PH_N + 4, t_z, 0);
        if (ph >= 0) {
            // ---- wait for the item's bands; meanwhile finish / start field blocks
            for (;;) {
                const long long t_w = clock64();
                if (tid < 32) {
                    bool r = mk_ready(P, done, ph, d, b, lane);
                    if (!r && z_exh && !zpend)
                        while (!(r = mk_ready(P, done, ph, d, b, lane))) __nanosleep(200);    // nothing else to do
                    if (lane == 0) s_flag = r;
                }
                __syncthreads();
                account(2 * PH_N + 2, t_w, 0);
                if (s_flag) break;
                if (zpend) z_finish();
                else {
                    if (tid == 0) { int zn = atomicAdd(P.sched + 1, 1); s_z[0] = zn < z_total ? zn : -1; }
                    __syncthreads();
                    if (s_z[0] < 0) z_exh = true; else z_decode_begin();
                }
                __syncthreads();
            }
            const long long t_b = clock64();
            switch (ph) {
            case PH_F1: {
                const int tr = idx / P.nbx1;
                tile_filter_conic4<NTC, MK_G>(P.f1, idx - tr * P.nbx1, 2 * b + tr, d, w_s, scratch);
            } break;
            case PH_F2: tile_fwd2d<2, true>(P.f2, idx, b, d, scratch); break;
            case PH_M: tile_maskgrad<2, true>(P.mg, idx, b, d, (d * P.nb + b) * P.nbx2 + idx, scratch); break;
            case PH_T: {
                const int tr = idx / P.nbx1;
                tile_filterT_conic4<NTC, MK_G, MK_TPASS>(P.ft, idx - tr * P.nbx1, 2 * b + tr, d, w_s, scratch);
            } break;
            case PH_X: {
                const int nblk = P.xblk[b == P.nb - 1];
                const int c = idx / nblk, blk = idx - c * nblk;
                const int col0 = b * MK_BAND * P.f2.ny, cend = min(P.f2.nx, (b + 1) * MK_BAND) * P.f2.ny;
                const int colb = col0 + blk * P.ex.cpb;
                block_extrude<true>(P.ex, c, colb, min(P.ex.cpb, cend - colb), d, scratch);
            } break;
            }
            __syncthreads();                                   // the item's global writes are ordered before the release
            account(ph, t_b, 1);
            const long long t_p = clock64();
            publish(ph, d, b);
            account(2 * PH_N + 3, t_p, 0);
        }
        if (zpend) z_finish();
        if (c_exh && z_exh) break;
        const long long t_e = clock64();
        __syncthreads();                                       // s_c / s_z are rewritten by the next round
        account(2 * PH_N + 5, t_e, 0);
    }
    if (P.prof && tid == 0) {
        for (int q = 0; q < 2 * PH_N + 8; ++q)
            if (q != 2 * PH_N + 1) atomicAdd(P.prof + q, (unsigned long long)s_prof[q]);
        atomicAdd(P.prof + 2 * PH_N + 1, (unsigned long long)(clock64() - s_prof[2 * PH_N + 1]));
    }
}

}  // namespace epsgrad
