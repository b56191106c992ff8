// extrude_window.cuh -- F6 restricted to the z cells that depend on the design (epsgrad_plan_set_eps_window_only).
//
// Outside the slab every cell of a z column is eps_clad whatever C and beta are (the layout is extruded to the device
// layer only), so once an eps array holds the result of ONE full call, a later call only has to rewrite the slab window of
// every column: the union of the x|y and z windows (extrude_bulk.cuh), rounded outwards to whole 32-byte sectors so that no
// store needs a read-modify-write of a partly written sector (paper scale: cells 24..39 of 64, 64 of 256 bytes per column).
// A thread per (column, 16-byte piece); the same affine forms in the same order as extrude.cuh: inside the window the bits are
// those of the full kernel, outside it nothing is touched.  Region-sized, x-slab and embedded arrays (ColumnMap).
#pragma once
#include "extrude.cuh"

namespace epsgrad {

constexpr int EW_THREADS = 256;

struct ExtrudeWindowParams {
    ExtrudeParams e;
    int q0, nq;            // first 16-byte piece (4 cells) and number of pieces of the window; both even
};

// grid (ceil(ncol * nq / EW_THREADS), 3, B)
__global__ void __launch_bounds__(EW_THREADS) k_extrude_window(const __grid_constant__ ExtrudeWindowParams W)
{
    pdl_launch();
    pdl_wait();
    const ExtrudeParams &P = W.e;
    const int c = blockIdx.y, b = blockIdx.z, nz = P.nz, nq = W.nq;
    const unsigned w = blockIdx.x * EW_THREADS + threadIdx.x;             // (column, piece) pair; ncol * nq < 2^31 (host checks)
    const int col = (int)(w / (unsigned)nq), q = W.q0 + (int)(w - (unsigned)col * (unsigned)nq), k = q << 2;
    if (col >= P.ncol) return;
    const float *ed = P.e2d + (size_t)b * 5 * P.pstride + col;
    float4 *out = reinterpret_cast<float4 *>(P.eps) + P.cm.plane(b, c) + P.cm.col(col) + q;
    const float *zw = P.zw;
    float4 o;
    if (c < 2) {
        const float v = __ldg(ed + (size_t)c * P.pstride);
        o.x = fmaf(__ldg(zw + k), v, __ldg(zw + 5 * nz + k));
        o.y = fmaf(__ldg(zw + k + 1), v, __ldg(zw + 5 * nz + k + 1));
        o.z = fmaf(__ldg(zw + k + 2), v, __ldg(zw + 5 * nz + k + 2));
        o.w = fmaf(__ldg(zw + k + 3), v, __ldg(zw + 5 * nz + k + 3));
    } else {
        const float v = __ldg(ed + (size_t)2 * P.pstride), vl = __ldg(ed + (size_t)3 * P.pstride), vh = __ldg(ed + (size_t)4 * P.pstride);
        float t[4];
#pragma unroll
        for (int x = 0; x < 4; ++x)
            t[x] = fmaf(__ldg(zw + 2 * nz + k + x), v, fmaf(__ldg(zw + 3 * nz + k + x), vl, fmaf(__ldg(zw + 4 * nz + k + x), vh, __ldg(zw + 6 * nz + k + x))));
        o = make_float4(t[0], t[1], t[2], t[3]);
    }
    st_eps(out, o);
}

}  // namespace epsgrad
