// filterT_tc.cuh -- the transposed filter (R6: dF/dC = filter^T v) on the tensor cores (tcgen05, TMEM), DESIGN.md 5.11.
//
// The transpose consumes 16 mask pixels per control pixel it produces, so the mapping of filter_tc.cuh (outputs on M) does not
// fit: here the INPUT row-groups are the N side and every one of them is multiplied with all the taps it feeds,
//   D[(tx, beta), n] = sum_{fx, qq} A[(tx, beta), (fx, qq)] * v[4 a' + fx, 4 (bb - T) + qq],        a' = a_in0 + n,
//   A[(tx, beta), (fx, qq)] = W[tx][beta + 2T - qq/4][fx][qq % 4]   (0 outside the NT taps),
// for a block of 8 control columns bb .. bb+7 (qq over its 4 (8 + 2T) mask columns) and N input control rows: one GEMM with
// M = 8 NT rows (104 at R = 12, padded to 128), K = 16 (8 + 2T) (320), followed by an overlap-add over the tap rows,
//   dC[a, bb + beta] = sum_tx D[(tx, beta), a - tx + T - a_in0],
// done out of shared memory in a fixed order (deterministic: no atomics).  A tile produces N - 2T output rows.
// Both operands stream through rings whose unit is a GROUP of 4 k-steps (8 of the K values each; 2 groups per ring): the
// weights by one 32 KB bulk copy per group (from the plan's table, two tf32 terms), the data by the 16 worker warps -- a group
// is 32 consecutive mask columns of a mask row, so 8 lanes fetch a whole 128-byte line; each value is split into two tf32
// terms on the way into shared memory.  Per group the issuing thread waits for the two slabs, issues 12 MMAs (hi*hi + hi*lo +
// lo*hi per k-step, as in filter_tc.cuh) and commits once per ring; the workers wait, store, fence and arrive once.
// K-major operands without swizzle, [2 chunks][rows][4 floats].
// What bounds it (measured by switching parts off, profiles/r2_experiments.md): SHARED-MEMORY BANDWIDTH.  Per group the tensor
// cores read 12 x (4 KB of A + 16 N bytes of B) ~ 130 KB, the workers store 64 KB and the bulk copy writes 32 KB: ~225 KB at
// 128 B/clk is ~1800 cycles against ~1350 for the MMAs alone (without the workers' stores the kernel runs in 69 us instead of
// 110 at 1000 x 1000, R = 12).  Two things that cost more before they were found: (1) fence.proxy.async compiles to
// MEMBAR.ALL.CTA + FENCE.VIEW.ASYNC and the MEMBAR waits for the warp's outstanding global loads too, so a prefetch issued
// before the fence is waited for at the fence: the next group's loads are issued after it; (2) one commit / wait / arrive per
// k-step kept the issuing thread busier than the MMAs it issued.
#pragma once
#include "filter_tc.cuh"

namespace epsgrad {

struct FilterTTcParams {
    const float *v;        // [B,px,py] mask cotangent / den
    float *dC;             // [B,mx,my]
    const float *a_tab;    // [KS][2 (hi, lo)][2 chunks][128][4]: the weight slabs of the k-steps
    int mx, my, px, py;
    int n_in, n_out;       // input row-groups staged per tile (a multiple of 16, <= 256) and output rows per tile (n_in - 2T)
    int tiles_x, tiles_y, n_tiles;     // column blocks of 8, row blocks of n_out, times B
    unsigned long long *dbg;           // nullptr, or cycle sums over the CTAs: [8] MMA thread waiting for weights, [9] for data, [10] MMA thread total,
                                       // [11] worker 0 waiting for a free data stage, [12] for the accumulator, [13] read-out, [14] overlap-add, [15] worker 0 total
};

// grid (min(n_tiles, #SM)), FTC_THREADS threads
template <int NTC>
__global__ void __launch_bounds__(FTC_THREADS, 1) k_filterT_tc(const FilterTTcParams P)
{
    constexpr int T = (NTC - 1) / 2, KQ = ftt_kq(NTC), KS = ftt_ksteps(NTC), G = FTT_GROUP, NG = KS / G, NR = FTT_RING, ROWS = 8 * NTC;
    constexpr unsigned A_STEP = 2 * 2 * FTC_M * 4;                  // floats of a k-step's weights: [hi, lo][2 chunks][128][4]
    constexpr unsigned B_STEP = ftt_b_step_floats();                // floats of a k-step's data:    [hi, lo][2 chunks][n_in <= 256 (+ 4: see LBOF)][4]
    constexpr unsigned A_GROUP = G * A_STEP, B_GROUP = G * B_STEP;
    static_assert(KS % G == 0, "whole groups");
    extern __shared__ unsigned char ftt_raw[];
    float *As = reinterpret_cast<float *>((reinterpret_cast<uintptr_t>(ftt_raw) + 127) & ~(uintptr_t)127);   // [NR][A_GROUP]
    float *Bs = As + NR * A_GROUP;                                  // [NR][B_GROUP]
    float *E = Bs;                                                  // [ROWS][n_in + 1]: the accumulator, for the overlap-add; reuses the data ring,
                                                                    // which is idle from the last MMA of a tile (d_full) to the first slab of the next
    static_assert((size_t)ROWS * (FTT_MAXN + 1) <= (size_t)NR * B_GROUP, "E fits in the data ring");
    __shared__ __align__(8) unsigned long long a_full[NR], a_empty[NR], b_full[NR], b_empty[NR], d_full;
    __shared__ unsigned tmem_slot;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int my_tiles = blockIdx.x < P.n_tiles ? (P.n_tiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    const int N = P.n_in;
    const unsigned LBOF = (unsigned)N * 4 + 16;    // floats between the two 16-byte chunks of a k-step: 64 bytes of padding put them in different banks

    if (tid == 0) {
        for (int s = 0; s < NR; ++s) { mbar_init(a_full + s, 1); mbar_init(a_empty + s, 1); mbar_init(b_full + s, FTC_WORKERS / 32); mbar_init(b_empty + s, 1); }
        mbar_init(&d_full, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"((unsigned)__cvta_generic_to_shared(&tmem_slot)), "r"((unsigned)FTT_MAXN) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    pdl_launch();
    pdl_wait();                                    // v is the kernel before's output
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem = tmem_slot;

    if (warp == FTC_WORKERS / 32) {
        // ---- weight producer (one thread): one bulk copy per group of k-steps (the table is [ks][hi, lo][2][128][4]: groups are contiguous)
        if (lane == 0) {
            int s = 0; unsigned ph = 0;
            for (int it = 0; it < my_tiles; ++it)
                for (int g = 0; g < NG; ++g) {
                    mbar_wait(a_empty + s, ph ^ 1u);
                    mbar_expect_tx(a_full + s, A_GROUP * 4u);
                    bulk_load(As + (size_t)s * A_GROUP, P.a_tab + (size_t)g * A_GROUP, A_GROUP * 4u, a_full + s);
                    if (++s == NR) { s = 0; ph ^= 1u; }
                }
        }
    } else if (warp == FTC_WORKERS / 32 + 1) {
        // ---- MMA issuer (one thread): 3 G MMAs per group, then one commit per ring
        if (lane == 0) {
            const unsigned idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((unsigned)(N >> 3) << 17) | ((unsigned)(FTC_M >> 4) << 24);
            const unsigned long long a0d = umma_desc(As, FTC_M * 16, 128), b0d = umma_desc(Bs, LBOF * 4, 128);
            constexpr unsigned long long A_GR = ((unsigned long long)A_GROUP * 4) >> 4, B_GR = ((unsigned long long)B_GROUP * 4) >> 4;
            constexpr unsigned long long A_ST = ((unsigned long long)A_STEP * 4) >> 4, B_ST = ((unsigned long long)B_STEP * 4) >> 4;
            constexpr unsigned long long A_LO = ((unsigned long long)(2 * FTC_M * 4) * 4) >> 4;
            const unsigned long long B_LO = ((unsigned long long)(2 * LBOF) * 4) >> 4;
            int s = 0; unsigned ph = 0;
            long long wa = 0, wb = 0; const long long m0 = P.dbg ? clock64() : 0;
            for (int it = 0; it < my_tiles; ++it) {
                // the accumulator's previous tile has been read out: the workers' first data slab of this tile follows their read-out
                for (int g = 0; g < NG; ++g) {
                    if (P.dbg) {
                        const long long c0 = clock64(); mbar_wait(a_full + s, ph);
                        const long long c1 = clock64(); mbar_wait(b_full + s, ph);
                        wa += c1 - c0; wb += clock64() - c1;
                    } else {
                        mbar_wait(a_full + s, ph);
                        mbar_wait(b_full + s, ph);
                    }
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                    for (int u = 0; u < G; ++u) {
                        const unsigned long long ah = a0d + (unsigned long long)s * A_GR + u * A_ST, al = ah + A_LO;
                        const unsigned long long bh = b0d + (unsigned long long)s * B_GR + u * B_ST, bl = bh + B_LO;
                        umma_tf32(tmem, ah, bh, idesc, (g | u) != 0);
                        umma_tf32(tmem, ah, bl, idesc, 1u);
                        umma_tf32(tmem, al, bh, idesc, 1u);
                    }
                    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                                 :: "r"((unsigned)__cvta_generic_to_shared(a_empty + s)) : "memory");
                    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                                 :: "r"((unsigned)__cvta_generic_to_shared(b_empty + s)) : "memory");
                    if (++s == NR) { s = 0; ph ^= 1u; }
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                             :: "r"((unsigned)__cvta_generic_to_shared(&d_full)) : "memory");
            }
            if (P.dbg) { atomicAdd(P.dbg + 8, (unsigned long long)wa); atomicAdd(P.dbg + 9, (unsigned long long)wb); atomicAdd(P.dbg + 10, (unsigned long long)(clock64() - m0)); }
        }
    } else {
        // ---- workers: feed the data slabs of a tile, then read the accumulator out and overlap-add it
        // A group of 4 k-steps is 32 consecutive mask columns (128 bytes) of a mask row: 8 lanes load them with one request
        // (lane = (row, k-step, half)); a warp feeds 16 input row-groups, 4 per load.
        static_assert(FTT_GROUP == 4 && FTC_WORKERS / 32 * 16 == FTT_MAXN, "8 lanes per 128-byte line, 16 row-groups per warp");
        const int u_l = (lane & 7) >> 1, h = lane & 1, n0w = 16 * warp + (lane >> 3);
        const bool feeds = 16 * warp < N;          // n_in is a multiple of 16: a warp's 16 row-groups are all staged or all beyond n_in
        int s = 0; unsigned ph = 0;
        long long we = 0, wd = 0, tr = 0, to = 0, tf = 0, ta = 0; const long long w0 = P.dbg ? clock64() : 0;
        const int per_b = P.tiles_x * P.tiles_y;
        // The 16 worker warps share the SM's issue slots with each other: the loop below is kept to ~100 instructions per group
        // (addresses by increments, no divisions), or the tensor cores wait for their operands.
        // Load j of a group reads input row-group n0w + 4 j; the lane's k-step ks = G g + u_l is phase row fx = ks / (KQ/8) and
        // mask columns q0 + 8 kk .. + 3 with kk = ks % (KQ/8), q0 = 4 (bb - T) + 4 h.
        long long off0 = 0;                        // element offset of (row-group n0w, fx = 0, column q0) in v; may point outside (then masked)
        int okm = 0, q0 = 0, kk = 0, fx = 0;
        auto setup = [&](int tile) {
            const int b = tile / per_b, rem = tile - b * per_b, by = rem / P.tiles_x, bx = rem - by * P.tiles_x;
            const int a_in0 = by * P.n_out - T;
            q0 = 4 * (bx * FTC_TB - T) + 4 * h;
            off0 = (long long)b * P.px * P.py + (long long)(4 * (a_in0 + n0w)) * P.py + q0;
            okm = 0;
#pragma unroll
            for (int j = 0; j < G; ++j) {
                const int ap = a_in0 + n0w + 4 * j;
                if (tile < P.n_tiles && feeds && ap >= 0 && ap < P.mx) okm |= 1 << j;
            }
            kk = u_l; fx = 0;
        };
        float4 pre[G];
        auto loads = [&]() {
            const int col = q0 + 8 * kk;
            const bool cok = col >= 0 && col < P.py;
            const float *p = P.v + (off0 + (long long)fx * P.py + 8 * kk);
#pragma unroll
            for (int j = 0; j < G; ++j)
                pre[j] = (cok && ((okm >> j) & 1)) ? __ldcg(reinterpret_cast<const float4 *>(p + (size_t)j * 16 * P.py)) : make_float4(0.f, 0.f, 0.f, 0.f);
        };
        setup(blockIdx.x);
        loads();
        float *const dst0 = Bs + (size_t)u_l * B_STEP + (size_t)h * LBOF + (size_t)n0w * 4;
        for (int it = 0; it < my_tiles; ++it) {
            const int tile = blockIdx.x + it * gridDim.x;
            const int b = tile / per_b, rem = tile - b * per_b;
            const int by = rem / P.tiles_x, bx = rem - by * P.tiles_x;
            const int a_out0 = by * P.n_out, bb = bx * FTC_TB;
            // The fence that makes a slab visible to the tensor cores (SASS: MEMBAR.ALL.CTA + FENCE.VIEW.ASYNC) also waits for the
            // warp's outstanding global loads: the loads of the next group are issued AFTER it, and land while the warp waits for
            // the ring slot to be free again.
#pragma unroll 1
            for (int g = 0; g < NG; ++g) {
                if (P.dbg) { const long long c0 = clock64(); mbar_wait(b_empty + s, ph ^ 1u); we += clock64() - c0; }
                else mbar_wait(b_empty + s, ph ^ 1u);                // the MMAs that read this slot are done
                if (feeds) {
                    float *d = dst0 + (size_t)s * B_GROUP;
#pragma unroll
                    for (int j = 0; j < G; ++j) {
                        const float4 x = pre[j];
                        float4 hi, lo;
                        hi.x = tf32_trunc(x.x); hi.y = tf32_trunc(x.y); hi.z = tf32_trunc(x.z); hi.w = tf32_trunc(x.w);
                        lo.x = tf32_trunc(x.x - hi.x); lo.y = tf32_trunc(x.y - hi.y); lo.z = tf32_trunc(x.z - hi.z); lo.w = tf32_trunc(x.w - hi.w);
                        *reinterpret_cast<float4 *>(d + j * 16) = hi;
                        *reinterpret_cast<float4 *>(d + j * 16 + 2 * LBOF) = lo;
                    }
                }
                const long long f0 = P.dbg ? clock64() : 0;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                const long long f1 = P.dbg ? clock64() : 0;
                __syncwarp();
                if (lane == 0) mbar_arrive(b_full + s);              // one arrival per warp
                if (P.dbg) { tf += f1 - f0; ta += clock64() - f1; }
                if (g + 1 < NG) {                                    // next group of this tile ...
                    kk += G;
                    if (kk >= KQ / 8) { kk -= KQ / 8; ++fx; }
                } else setup(tile + (int)gridDim.x);                 // ... or the first one of the next tile
                loads();
                if (++s == NR) { s = 0; ph ^= 1u; }
            }
            // ---- read-out: TMEM lane = (tx, beta) row, columns = input row-groups; into E, then the overlap-add over tx
            const long long r0 = P.dbg ? clock64() : 0;
            mbar_wait(&d_full, (unsigned)it & 1u);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const long long r1 = P.dbg ? clock64() : 0;
            {
                const int quad = warp & 3, part = warp >> 2, row = quad * 32 + lane;
                constexpr int NPART = FTC_WORKERS / 128;
                const int pitch = N + 1;
                for (int n0 = part * 16; n0 < N; n0 += 16 * NPART) {
                    unsigned vv[16];
                    const unsigned taddr = tmem + ((unsigned)(quad * 32) << 16) + (unsigned)n0;
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                                 : "=r"(vv[0]), "=r"(vv[1]), "=r"(vv[2]), "=r"(vv[3]), "=r"(vv[4]), "=r"(vv[5]), "=r"(vv[6]), "=r"(vv[7]),
                                   "=r"(vv[8]), "=r"(vv[9]), "=r"(vv[10]), "=r"(vv[11]), "=r"(vv[12]), "=r"(vv[13]), "=r"(vv[14]), "=r"(vv[15])
                                 : "r"(taddr) : "memory");
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    if (row < ROWS) {
#pragma unroll
                        for (int i = 0; i < 16; ++i) E[row * pitch + n0 + i] = __uint_as_float(vv[i]);
                    }
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                ftc_worker_sync();                 // E complete; the accumulator may be overwritten by the next tile's MMAs
                const long long r2 = P.dbg ? clock64() : 0;
                float *dCb = P.dC + (size_t)b * P.mx * P.my;
                for (int o = tid; o < P.n_out * 8; o += FTC_WORKERS) {     // lanes <-> consecutive rows: conflict-free reads (odd pitch)
                    const int beta = o / P.n_out, i = o - beta * P.n_out, a = a_out0 + i, bc = bb + beta;
                    if (a < P.mx && bc < P.my) {
                        const float *e = E + beta * pitch + i + 2 * T;
                        float acc = 0.0f;
#pragma unroll
                        for (int tx = 0; tx < NTC; ++tx) acc += e[tx * (8 * pitch - 1)];
                        dCb[(size_t)a * P.my + bc] = acc;
                    }
                }
                ftc_worker_sync();                 // E may be overwritten
                if (P.dbg) { wd += r1 - r0; tr += r2 - r1; to += clock64() - r2; }
            }
        }
        if (P.dbg && tid == 0) {
            atomicAdd(P.dbg + 11, (unsigned long long)we); atomicAdd(P.dbg + 12, (unsigned long long)wd); atomicAdd(P.dbg + 13, (unsigned long long)tr);
            atomicAdd(P.dbg + 14, (unsigned long long)to); atomicAdd(P.dbg + 15, (unsigned long long)(clock64() - w0));
            atomicAdd(P.dbg + 16, (unsigned long long)tf); atomicAdd(P.dbg + 17, (unsigned long long)ta);
        }
    }
    __syncthreads();
    if (warp == 1)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"((unsigned)FTT_MAXN) : "memory");
}

}  // namespace epsgrad
