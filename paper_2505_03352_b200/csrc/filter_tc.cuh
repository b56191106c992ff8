// filter_tc.cuh -- Eq. (2) on the 5th-generation tensor cores (tcgen05, accumulators in tensor memory).
//
// For m = 4 mask pixels per control pixel the conic filter of filter4.cuh is, per tap row tx, a banded product along y:
//   Phi'[4 a0 + fx, 4 b0 + fy] = invden * sum_tx sum_j  A_tx[(fx, b0 - bb, fy), j] * C'[a0 + tx - T, bb - T + j]
// with A_tx[(fx, beta, fy), j] = W[tx][j - beta][fx][fy] (0 outside the NT taps), bb the first control column of a block of
// FTC_TB = 8 columns and j running over its FTC_TB + 2T input columns.  For a block of FTC_N control rows that is a GEMM
//   D[128 x FTC_N] += A_tx[128 x K] * B_tx[K x FTC_N],      B_tx[j, n] = C'[a_base + n + tx - T, bb - T + j],
// summed over the NT tap rows: M = 4 phases x 32 mask columns, N = control rows, K = FTC_TB + 2T rounded up to 8.  The band
// makes the product K / NT = 1.8 x denser than the stencil (R = 8), which the tensor cores absorb many times over.
// Accuracy: kind::tf32 keeps 10 mantissa bits, so both operands are split into two tf32 terms (x = hi + lo exactly up to
// 2^-21 |x|) and three products are accumulated in float32: hi*hi + hi*lo + lo*hi; the dropped lo*lo term is 2^-22 relative.
// The weight split is built on the host from the float64 table; the C' split is done while staging.
// Layout: both operands K-major without swizzle, as [K/4 chunks][rows][4 floats]: rows of a chunk are 16 bytes apart (stride
// between 8-row core matrices = 128 B), so the B operand of tap row tx is the staged tile shifted by tx rows: one staged C'
// tile serves all NT tap rows through the start address of its descriptor.
// One CTA per SM, warp-specialised (below): the eight worker warps read TMEM as warp = phase row fx and half of the control
// rows, lane = mask column, and store 128 contiguous bytes of Phi' per control row.
#pragma once
#include "filter.cuh"
#include "filter4.cuh"
#include "sizes.cuh"
#include "zreduce.cuh"        // mbarrier helpers

namespace epsgrad {

struct FilterTcParams {
    const float *C;        // [B,mx,my]
    float *phi;            // [B,px,py] centred filter output
    const float *a_tab;    // [2 (hi, lo)][NT][K/4][128][4]: the banded weight matrices, split into two tf32 terms
    Normaliser nrm;
    int mx, my, px, py;
    int tiles_x, tiles_y, n_tiles;     // column blocks of 8, row blocks of FTC_N, times B
    float eta0;
    unsigned long long *dbg;   // nullptr, or cycle sums over the CTAs: [0] staging, [1] wait for the accumulator, [2] read-out + stores, [3] MMA warp waiting for a tile, [4] MMA issue, [5] tiles
};

// shared-memory matrix descriptor (K-major, no swizzle): start, leading (between the two 4-float chunks of a K step) and stride
// (between 8-row core matrices) byte offsets, all in 16-byte units; version 1 (sm_100)
__device__ __forceinline__ unsigned long long umma_desc(const void *smem, unsigned lbo_bytes, unsigned sbo_bytes)
{
    const unsigned a = (unsigned)__cvta_generic_to_shared(smem);
    return (unsigned long long)((a >> 4) & 0x3fffu) | ((unsigned long long)((lbo_bytes >> 4) & 0x3fffu) << 16) |
           ((unsigned long long)((sbo_bytes >> 4) & 0x3fffu) << 32) | (1ull << 46);
}

__device__ __forceinline__ void umma_tf32(unsigned tmem_d, unsigned long long adesc, unsigned long long bdesc, unsigned idesc, unsigned accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}\n"
                 :: "r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}

// barrier of the FTC_WORKERS threads that stage, issue and store (the producer warp is not part of it)
__device__ __forceinline__ void ftc_worker_sync() { asm volatile("bar.sync 1, %0;" :: "n"(FTC_WORKERS) : "memory"); }

// one bulk asynchronous copy global -> shared, completion (byte count) on an mbarrier
__device__ __forceinline__ void bulk_load(void *smem, const void *gsrc, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gsrc), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}

// grid (min(n_tiles, #SM)), FTC_THREADS threads, ftc_smem_bytes(NTC, N, STREAM) of dynamic shared memory.
// N: control rows per tile (= TMEM columns per accumulator; there are two).  STREAM = false: all NT weight matrices stay in
// shared memory (NT <= 9: 147 KB at R = 8).  STREAM = true: they pass through a ring of FTC_STAGES tap-row stages (24 KB each at
// R = 12) and a tile is N = 256 rows, so that the 320 KB of weights are re-read from L2 once per 2048 control pixels.
// Warp roles: 8 worker warps stage C' of tile i+1 and then read and store the accumulator of tile i; one thread of warp 8 feeds
// the weight ring (bulk copies); one thread of warp 9 issues the MMAs of tile i+1 into the other accumulator.  Hand-offs by
// mbarriers: b_full (tile staged), d_full (tcgen05.commit: accumulator complete), d_empty (accumulator read out), a_full / a_empty.
template <int NTC, int N, bool STREAM>
__global__ void __launch_bounds__(FTC_THREADS, 1) k_filter_tc(const FilterTcParams P)
{
    constexpr int T = (NTC - 1) / 2, K = ftc_k(NTC), RB = N + 2 * T;
    constexpr unsigned TX_FLOATS = K * FTC_M;                       // one tap row's matrix (hi or lo)
    constexpr unsigned A_BYTES = (unsigned)(ftc_a_floats(NTC) * 4);
    constexpr int NST = STREAM ? FTC_STAGES : 1;
    extern __shared__ unsigned char ftc_raw[];
    float *A = reinterpret_cast<float *>((reinterpret_cast<uintptr_t>(ftc_raw) + 127) & ~(uintptr_t)127);
    // resident: [2][NTC][K/4][128][4]; streamed: [FTC_STAGES][2][K/4][128][4]
    float *Bs = A + (STREAM ? (size_t)FTC_STAGES * 2 * TX_FLOATS : ftc_a_floats(NTC));      // [2 buffers][hi, lo][K/4][RB][4]
    __shared__ __align__(8) unsigned long long a_full[NST], a_empty[NST], b_full[2], d_full[2], d_empty[2];
    __shared__ unsigned tmem_slot;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int my_tiles = blockIdx.x < P.n_tiles ? (P.n_tiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;

    if (tid == 0) {
        for (int s = 0; s < NST; ++s) { mbar_init(a_full + s, 1); mbar_init(a_empty + s, 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(b_full + s, 1); mbar_init(d_full + s, 1); mbar_init(d_empty + s, 1); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        if (!STREAM) {
            // the weight matrices: copies by the bulk-copy engine, in flight while the first tile is staged (the table is the plan's)
            mbar_expect_tx(a_full, A_BYTES);
            constexpr unsigned PIECE = 32768;
            for (unsigned o = 0; o < A_BYTES; o += PIECE)
                bulk_load(reinterpret_cast<unsigned char *>(A) + o, reinterpret_cast<const unsigned char *>(P.a_tab) + o,
                          A_BYTES - o < PIECE ? A_BYTES - o : PIECE, a_full);
        }
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"((unsigned)__cvta_generic_to_shared(&tmem_slot)), "r"((unsigned)(2 * N)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    pdl_launch();
    pdl_wait();                                    // Phi' may still be read by the kernel before (the previous call's reverse pass)
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();                               // barriers initialised, TMEM address written
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tmem = tmem_slot;

    if (warp == FTC_WORKERS / 32) {
        // ---- weight producer (one thread): the tap-row matrices of every tile of this CTA through the ring
        if (STREAM && lane == 0) {
            int s = 0; unsigned ph = 0;
            const float *src_hi = P.a_tab, *src_lo = P.a_tab + ftc_a_floats(NTC) / 2;
            for (int it = 0; it < my_tiles; ++it)
                for (int tx = 0; tx < NTC; ++tx) {
                    mbar_wait(a_empty + s, ph ^ 1u);
                    float *dst = A + (size_t)s * 2 * TX_FLOATS;
                    mbar_expect_tx(a_full + s, 2u * TX_FLOATS * 4u);
                    // every CTA streams the same table at the same time: each starts at a different piece of the tap row, so that
                    // the copies of the SMs do not sweep the L2 slices in lockstep
                    constexpr unsigned NP = 8, PIECE = 2u * TX_FLOATS * 4u / NP, HALF = TX_FLOATS * 4u;
                    static_assert(HALF % PIECE == 0 && PIECE % 16 == 0, "pieces do not straddle the hi / lo halves");
                    for (unsigned q = 0; q < NP; ++q) {
                        const unsigned o = ((q + blockIdx.x) % NP) * PIECE;      // byte offset within [hi | lo] of this tap row
                        const unsigned char *src = o < HALF ? reinterpret_cast<const unsigned char *>(src_hi + (size_t)tx * TX_FLOATS) + o
                                                            : reinterpret_cast<const unsigned char *>(src_lo + (size_t)tx * TX_FLOATS) + (o - HALF);
                        bulk_load(reinterpret_cast<unsigned char *>(dst) + o, src, PIECE, a_full + s);
                    }
                    if (++s == NST) { s = 0; ph ^= 1u; }
                }
        }
    } else if (warp == FTC_WORKERS / 32 + 1) {
        // ---- MMA issuer (one thread)
        if (lane == 0) {
            // instruction descriptor: D = F32, A = B = TF32, both K-major, N, M
            constexpr unsigned idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((unsigned)(N >> 3) << 17) | ((unsigned)(FTC_M >> 4) << 24);
            int a_s = 0; unsigned a_ph = 0;
            if (!STREAM && my_tiles > 0) mbar_wait(a_full, 0);
            for (int it = 0; it < my_tiles; ++it) {
                const int buf = it & 1;
                const unsigned ph = (unsigned)(it >> 1) & 1u;
                const long long m0 = clock64();
                mbar_wait(b_full + buf, ph);           // the tile is staged
                mbar_wait(d_empty + buf, ph ^ 1u);     // the accumulator's previous tile has been read out (first use: passes)
                const long long m1 = clock64();
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const float *Bh = Bs + (size_t)buf * 2 * K * RB, *Bl = Bh + K * RB;
                const unsigned td = tmem + (unsigned)(buf * N);
                // descriptors differ in their start address only (bits 0-13, in 16-byte units; shared memory is < 256 KB, so the
                // field never carries): one add per operand and MMA instead of rebuilding them
                const unsigned long long bh0 = umma_desc(Bh, RB * 16, 128), bl0 = umma_desc(Bl, RB * 16, 128);
                const unsigned long long a0d = umma_desc(A, FTC_M * 16, 128);
                constexpr unsigned long long A_KSTEP = (2ull * FTC_M * 4 * 4) >> 4, B_KSTEP = (2ull * RB * 4 * 4) >> 4;   // two 4-float chunks
                constexpr unsigned long long A_TX = ((unsigned long long)TX_FLOATS * 4) >> 4, A_LO = ((unsigned long long)(ftc_a_floats(NTC) / 2) * 4) >> 4;
#pragma unroll 1
                for (int tx = 0; tx < NTC; ++tx) {
                    // resident: hi of tap row tx at tx * TX_FLOATS, lo at half the table + that; streamed: stage a_s holds [hi | lo]
                    const unsigned long long ahd = a0d + (STREAM ? (unsigned long long)a_s * 2 * A_TX : (unsigned long long)tx * A_TX);
                    const unsigned long long ald = ahd + (STREAM ? A_TX : A_LO);
                    const unsigned long long bhd = bh0 + (unsigned long long)tx, bld = bl0 + (unsigned long long)tx;      // tx rows of 16 bytes
                    if (STREAM) {
                        mbar_wait(a_full + a_s, a_ph);
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    }
#pragma unroll
                    for (int kk = 0; kk < K / 8; ++kk) {
                        umma_tf32(td, ahd + kk * A_KSTEP, bhd + kk * B_KSTEP, idesc, (tx | kk) != 0);
                        umma_tf32(td, ahd + kk * A_KSTEP, bld + kk * B_KSTEP, idesc, 1u);
                        umma_tf32(td, ald + kk * A_KSTEP, bhd + kk * B_KSTEP, idesc, 1u);
                    }
                    if (STREAM) {                      // the stage is free once these MMAs have read it
                        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                                     :: "r"((unsigned)__cvta_generic_to_shared(a_empty + a_s)) : "memory");
                        if (++a_s == NST) { a_s = 0; a_ph ^= 1u; }
                    }
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];"
                             :: "r"((unsigned)__cvta_generic_to_shared(d_full + buf)) : "memory");
                if (P.dbg) { atomicAdd(P.dbg + 3, (unsigned long long)(m1 - m0)); atomicAdd(P.dbg + 4, (unsigned long long)(clock64() - m1)); }
            }
        }
    } else {
        // ---- workers: stage tile it, then read out and store tile it - 1 (while the tensor core works on tile it)
        // warps w, w + 4, w + 8, .. share TMEM lanes 32 fx .. 32 fx + 31 and split the control rows: a warp has one store in flight at
        // a time (~120 cycles per 128-byte row segment, measured), so the read-out scales with the number of warps doing it
        constexpr int NPART = FTC_WORKERS / 128;
        const int fx = warp & 3, part = warp >> 2, beta = lane >> 2, fy = lane & 3;
        for (int it = 0; it <= my_tiles; ++it) {
            const long long t0 = clock64();
            if (it < my_tiles) {
                const int tile = blockIdx.x + it * gridDim.x;
                const int per_b = P.tiles_x * P.tiles_y, b = tile / per_b, rem = tile - b * per_b;
                const int by = rem / P.tiles_x, bx = rem - by * P.tiles_x;
                const int a_base = by * N, bb = bx * FTC_TB;
                // C' of the tile, split into two tf32 terms: row r <-> control row a_base - T + r, j <-> column bb - T + j.  The
                // buffer was last read by the MMAs of tile it - 2, which completed before that tile's read-out began.
                float *Bh = Bs + (size_t)(it & 1) * 2 * K * RB, *Bl = Bh + K * RB;
                const float *Cb = P.C + (size_t)b * P.mx * P.my;
                constexpr int U = 8;                   // loads in flight per thread
                for (int base = tid; base < RB * K; base += U * FTC_WORKERS) {
                    float v[U];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const int idx = base + u * FTC_WORKERS, r = idx / K, j = idx - r * K;
                        const int a = a_base - T + r, bc = bb - T + j;
                        v[u] = 0.0f;
                        if (idx < RB * K && j < FTC_TB + 2 * T && a >= 0 && a < P.mx && bc >= 0 && bc < P.my) v[u] = Cb[(size_t)a * P.my + bc] - P.eta0;
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const int idx = base + u * FTC_WORKERS, r = idx / K, j = idx - r * K;
                        if (idx < RB * K) {
                            const float hi = tf32_trunc(v[u]), lo = tf32_trunc(v[u] - hi);
                            const int o = ((j >> 2) * RB + r) * 4 + (j & 3);
                            Bh[o] = hi; Bl[o] = lo;
                        }
                    }
                }
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the tensor core's reads
                ftc_worker_sync();
                if (tid == 0) mbar_arrive(b_full + (it & 1));
            }
            const long long t1 = clock64();
            if (P.dbg && tid == 0) atomicAdd(P.dbg + 0, (unsigned long long)(t1 - t0));
            if (it > 0) {
                const int jt = it - 1, buf = jt & 1;
                const int tile = blockIdx.x + jt * gridDim.x;
                const int per_b = P.tiles_x * P.tiles_y, b = tile / per_b, rem = tile - b * per_b;
                const int by = rem / P.tiles_x, bx = rem - by * P.tiles_x;
                const int a_base = by * N, bb = bx * FTC_TB;
                // warp <-> phase row fx (TMEM lanes 32 fx .. 32 fx + 31) and half of the control rows, lane <-> mask column
                const int b0 = bb + beta;
                const bool col_ok = b0 < P.my;
                const int niy = col_ok ? P.nrm.iy(b0, fy) : 0;
                const float inv_in = P.nrm.at_index(T * 4 + fx, niy);      // normaliser away from the first / last T control rows
                float *out = P.phi + (size_t)b * P.px * P.py + (size_t)4 * bb + lane;
                mbar_wait(d_full + buf, (unsigned)(jt >> 1) & 1u);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const long long t2 = clock64();
#pragma unroll 1
                for (int n0 = part * (N / NPART); n0 < (part + 1) * (N / NPART); n0 += 16) {
                    unsigned v[16];
                    const unsigned taddr = tmem + ((unsigned)(fx * 32) << 16) + (unsigned)(buf * N + n0);
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                                   "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                                 : "r"(taddr) : "memory");
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    float *orow = out + (size_t)(4 * (a_base + n0) + fx) * P.py;
#pragma unroll
                    for (int i = 0; i < 16; ++i, orow += (size_t)4 * P.py) {
                        const int a0 = a_base + n0 + i;
                        if (col_ok && a0 < P.mx) {
                            const float inv = (a0 >= T && a0 < P.mx - T) ? inv_in : P.nrm.at_index(P.nrm.ix(a0, fx), niy);
                            __stcg(orow, __uint_as_float(v[i]) * inv);      // L2: the 2-D stage reads Phi' from there
                        }
                    }
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                ftc_worker_sync();                     // every worker has read its part of the accumulator
                if (tid == 0) mbar_arrive(d_empty + buf);
                if (P.dbg && tid == 0) {
                    const long long t3 = clock64();
                    atomicAdd(P.dbg + 1, (unsigned long long)(t2 - t1)); atomicAdd(P.dbg + 2, (unsigned long long)(t3 - t2)); atomicAdd(P.dbg + 5, 1ull);
                }
            }
        }
    }
    if (!STREAM && my_tiles == 0 && tid == 0) mbar_wait(a_full, 0);       // shared memory must outlive the copies into it
    __syncthreads();
    if (warp == 1)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"((unsigned)(2 * N)) : "memory");
}

}  // namespace epsgrad
