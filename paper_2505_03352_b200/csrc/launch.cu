// launch.cu -- kernel launches, the schedules (serial, two-stream, persistent) and the device entry points of the C ABI
// (include/epsgrad.h).  The only translation unit that includes the kernels of the path.
#include "plan.cuh"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <utility>

#include "common.cuh"
#include "filter.cuh"
#include "filter4.cuh"
#include "filter_sep.cuh"
#include "filter_general.cuh"
#include "filter_tc.cuh"
#include "filterT_tc.cuh"
#include "fwd2d.cuh"
#include "extrude.cuh"
#include "extrude_bulk.cuh"
#include "extrude_window.cuh"
#include "zreduce.cuh"
#include "zreduce_pipe.cuh"
#include "scalar3d.cuh"
#include "maskgrad.cuh"
#include "mega.cuh"
#include "morph.cuh"
#include "reduce.cuh"

namespace epsgrad {

// Opt a kernel in to `bytes` of dynamic shared memory: once per plan and kernel (the attribute is per device, as the plan is),
// not at every launch.
template <typename K>
int set_smem(epsgrad_plan *P, K kernel, size_t bytes)
{
    if (bytes <= 48 * 1024) return EPSGRAD_OK;
    const void *fn = (const void *)kernel;
    for (int i = 0; i < P->n_smem_set; ++i)
        if (P->smem_fn[i] == fn) {
            if (P->smem_bytes[i] >= bytes) return EPSGRAD_OK;
            if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess) { cudaGetLastError(); return EPSGRAD_ECUDA; }
            P->smem_bytes[i] = bytes;
            return EPSGRAD_OK;
        }
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    if (P->n_smem_set < EPSGRAD_MAX_SMEM_KERNELS) { P->smem_fn[P->n_smem_set] = fn; P->smem_bytes[P->n_smem_set] = bytes; ++P->n_smem_set; }
    return EPSGRAD_OK;
}

// Launch with the programmatic-dependent-launch attribute when the operation before it on `st` was a kernel of this call that
// releases its dependents early (common.cuh pdl_launch / pdl_wait): the plan remembers that stream in pdl_stream.
template <typename... KArgs, typename... Args>
cudaError_t launch_k(epsgrad_plan *P, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = P->use_pdl && P->pdl_valid && P->pdl_stream == st ? 1 : 0;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
    P->pdl_stream = st; P->pdl_valid = 1; P->pdl_mark = 1;
    return e;
}
// any other operation on a stream (event record / wait, copy, a kernel without pdl_launch) ends the chain
inline void pdl_break(epsgrad_plan *P) { P->pdl_valid = 0; }

__global__ void k_stamp(unsigned long long *slot)
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    *slot = t;
}

// timeline on: a one-thread kernel that stores the device clock runs at this point of stream `st`
void stamp(epsgrad_plan *P, const char *what, cudaStream_t st)
{
    if (!P->d_tl || P->n_tl >= 2 * EPSGRAD_MAX_KERNELS) return;
    P->tlname[P->n_tl] = what;
    k_stamp<<<1, 1, 0, st>>>(P->d_tl + P->n_tl++);
}

void begin_call(epsgrad_plan *P, cudaStream_t st)
{
    P->last_launches = 0;
    P->n_tl = 0;
    P->pdl_valid = P->pdl_mark = 0;
    if (P->prof) cudaEventRecord(P->ev[0], st);
}

int check_launch(epsgrad_plan *P, const char *name, cudaStream_t st)
{
    // a kernel launched without launch_k, the profiling events and the timeline stamps all end a dependent-launch chain
    if (!P->pdl_mark || P->prof || P->d_tl) P->pdl_valid = 0;
    P->pdl_mark = 0;
    const int idx = P->last_launches++;
    if (idx < EPSGRAD_MAX_KERNELS) {
        P->kname[idx] = name;
        if (P->prof) cudaEventRecord(P->ev[idx + 1], st);
    }
    stamp(P, name, st);
    return cudaGetLastError() == cudaSuccess ? EPSGRAD_OK : EPSGRAD_ECUDA;
}

Normaliser make_nrm(const epsgrad_plan *P)
{
    Normaliser n;
    n.tab = P->d_invden; n.mx = P->cfg.mx; n.my = P->cfg.my; n.m = P->m; n.T = P->T;
    n.KX = P->KX; n.KY = P->KY; n.separable = P->separable;
    n.plane_py = 0;
    if (P->general) { n.tab = ws_invden(P); n.plane_py = P->py; }      // the plane k_filter_general wrote (every call runs F1 first)
    return n;
}


FilterParams fill_filter(const epsgrad_plan *P, const float *C, float *phi)
{
    FilterParams fp;
    fp.C = C; fp.phi = phi; fp.w = P->d_w; fp.tyrange = P->d_tyrange; fp.nrm = make_nrm(P);
    fp.mx = P->cfg.mx; fp.my = P->cfg.my; fp.px = P->px; fp.py = P->py; fp.T = P->T; fp.NT = P->NT; fp.eta0 = P->eta0;
    return fp;
}

FilterTParams fill_filterT(const epsgrad_plan *P, const float *v, float *dC)
{
    FilterTParams fp;
    fp.v = v; fp.dC = dC; fp.w = P->d_w; fp.tyrange = P->d_tyrange;
    fp.mx = P->cfg.mx; fp.my = P->cfg.my; fp.px = P->px; fp.py = P->py; fp.T = P->T; fp.NT = P->NT;
    return fp;
}

// ---- F1: C -> centred Phi on the mask
template <int M>
int launch_filter_m(epsgrad_plan *P, const float *C, float *phi, cudaStream_t st)
{
    const int B = P->cfg.batch, mx = P->cfg.mx, my = P->cfg.my, T = P->T, NT = P->NT;
    if (!P->separable) {
        constexpr int TA = 8, TB = 16;
        const FilterParams fp = fill_filter(P, C, phi);
        // tensor cores (filter_tc.cuh): always when asked for (use_tc = 1); by default (2) where they measured faster than the
        // FFMA stencil -- enough tiles to amortise the per-CTA set-up (weights, TMEM): R = 12 from ~500 x 500 control pixels
        // (27 against 47 us; 55 against 158 us at 1000 x 1000), R <= 8 from ~375 x 375 (14.5 against 20.5 us; a tie at 250 x 250)
        bool tc = M == 4 && P->use_tc && P->d_atc && (NT == 5 || NT == 9 || NT == 13);
        if (tc && P->use_tc == 2) {
            const bool big = NT == 13;
            const int nt = cdiv(my, FTC_TB) * cdiv(mx, big ? FTC_N_STREAM : FTC_N_RESIDENT) * B;
            tc = big ? 2 * nt >= P->n_sm : 2 * nt >= 3 * P->n_sm;
        }
        if (tc) {
            FilterTcParams tp;
            tp.C = C; tp.phi = phi; tp.a_tab = P->d_atc; tp.nrm = fp.nrm;
            tp.mx = mx; tp.my = my; tp.px = P->px; tp.py = P->py; tp.eta0 = P->eta0;
            tp.dbg = P->d_mprof;          // cycle accounting, when epsgrad_plan_fused_profile is on
            const bool stream = NT == 13 || P->tune[7] == 1;          // R = 12: the weight matrices do not fit in shared memory
            const int Nt = stream ? FTC_N_STREAM : FTC_N_RESIDENT;
            tp.tiles_x = cdiv(my, FTC_TB); tp.tiles_y = cdiv(mx, Nt); tp.n_tiles = tp.tiles_x * tp.tiles_y * B;
            const size_t smem_tc = ftc_smem_bytes(NT, Nt, stream);
            const int grid_tc = std::min(tp.n_tiles, P->n_sm);
            int rct = EPSGRAD_OK;
#define EPSGRAD_TC_LAUNCH(NTC_, N_, S_)                                                         \
            do {                                                                                \
                rct = set_smem(P, k_filter_tc<NTC_, N_, S_>, smem_tc);                          \
                if (!rct) k_filter_tc<NTC_, N_, S_><<<grid_tc, FTC_THREADS, smem_tc, st>>>(tp);  \
            } while (0)
            if (NT == 13) EPSGRAD_TC_LAUNCH(13, FTC_N_STREAM, true);
            else if (NT == 9 && stream) EPSGRAD_TC_LAUNCH(9, FTC_N_STREAM, true);
            else if (NT == 9) EPSGRAD_TC_LAUNCH(9, FTC_N_RESIDENT, false);
            else if (stream) EPSGRAD_TC_LAUNCH(5, FTC_N_STREAM, true);
            else EPSGRAD_TC_LAUNCH(5, FTC_N_RESIDENT, false);
#undef EPSGRAD_TC_LAUNCH
            if (rct) return rct;
            return check_launch(P, "filter", st);
        }
        if (M == 4 && (NT == 5 || NT == 9 || NT == 13)) {      // fast path (filter4.cuh)
            auto kern = NT == 5 ? k_filter_conic4<5> : (NT == 9 ? k_filter_conic4<9> : k_filter_conic4<13>);
            const size_t smem4 = (filter4_smem_floats(NT) + 4) * 4;
            int rc4 = set_smem(P, kern, smem4);
            if (rc4) return rc4;
            launch_k(P, kern, dim3(cdiv(my, F4_TB), cdiv(mx, F4_TA), B), dim3(F4F_THREADS), smem4, st, fp);
            return check_launch(P, "filter", st);
        }
        const size_t smem = ((size_t)NT * NT * M * M + (size_t)(TA + 2 * T) * (TB + 2 * T + 1) + 2 * NT) * 4;
        if (smem > 200 * 1024) return EPSGRAD_EUNSUPPORTED;
        int rc = set_smem(P, k_filter_conic<M, TA, TB>, smem);
        if (rc) return rc;
        k_filter_conic<M, TA, TB><<<dim3(cdiv(my, TB), cdiv(mx, TA), B), TA * TB, smem, st>>>(fp);
        return check_launch(P, "filter", st);
    }
    SepParams sp;
    sp.w1 = P->d_w; sp.nrm = make_nrm(P);
    sp.mx = mx; sp.my = my; sp.px = P->px; sp.py = P->py; sp.T = T; sp.NT = NT; sp.eta0 = P->eta0;
    {
        sp.in = C; sp.out = ws_tmp(P);
        const size_t smem = ((size_t)NT * M + (size_t)8 * (32 + 2 * T)) * 4;
        int rc = set_smem(P, k_sep_up_y<M>, smem);
        if (rc) return rc;
        k_sep_up_y<M><<<dim3(cdiv(my, 32), cdiv(mx, 8), B), SEP_THREADS, smem, st>>>(sp);
        if ((rc = check_launch(P, "filter_up_y", st))) return rc;
    }
    {
        sp.in = ws_tmp(P); sp.out = phi;
        const size_t smem = sepx_smem_floats(NT, M) * 4;
        if (smem > 200 * 1024) return EPSGRAD_EUNSUPPORTED;
        int rc = set_smem(P, k_sep_up_x<M>, smem);
        if (rc) return rc;
        k_sep_up_x<M><<<dim3(cdiv(P->py, SEPX_THREADS), cdiv(mx, SEPX_NBA), B), SEPX_THREADS, smem, st>>>(sp);
        return check_launch(P, "filter_up_x", st);
    }
}

// ---- R6: mask cotangent v -> dF/dC
template <int M>
int launch_filterT_conic(epsgrad_plan *P, const float *v, float *dC, cudaStream_t st)
{
    using S = FilterTShape<M>;
    const int T = P->T, NT = P->NT;
    const FilterTParams fp = fill_filterT(P, v, dC);
    // tensor cores (filterT_tc.cuh): when asked for (use_tc = 1); by default (2) where they measured faster than the FFMA kernel:
    // R = 12 from ~500 x 500 control pixels (44 against 58 us; 112 against 203 us at 1000 x 1000), R <= 8 at 1000 x 1000
    // (87 against 125 us; within 2 us of each other at 375 and 500, slower at 250)
    bool tc = M == 4 && P->use_tc && P->d_att && (NT == 5 || NT == 9 || NT == 13);
    if (tc) {
        FilterTTcParams tp;
        tp.v = v; tp.dC = dC; tp.a_tab = P->d_att;
        tp.mx = fp.mx; tp.my = fp.my; tp.px = fp.px; tp.py = fp.py; tp.dbg = P->d_mprof;
        const int nb = cdiv(fp.mx, FTT_MAXN - 2 * T);                      // row blocks; rows per block rounded so that n_in % 16 == 0
        tp.n_in = std::min(FTT_MAXN, (cdiv(fp.mx, nb) + 2 * T + 15) / 16 * 16);
        tp.n_out = tp.n_in - 2 * T;
        tp.tiles_x = cdiv(fp.my, FTC_TB); tp.tiles_y = cdiv(fp.mx, tp.n_out); tp.n_tiles = tp.tiles_x * tp.tiles_y * P->cfg.batch;
        if (P->use_tc == 2) tc = NT == 13 ? tp.n_tiles >= P->n_sm : 2 * tp.n_tiles >= 3 * P->n_sm;
        if (tc) {
            auto kern = NT == 5 ? k_filterT_tc<5> : (NT == 9 ? k_filterT_tc<9> : k_filterT_tc<13>);
            const size_t smem_t = ftt_smem_bytes(NT);
            int rct = set_smem(P, kern, smem_t);
            if (rct) return rct;
            kern<<<std::min(tp.n_tiles, P->n_sm), FTC_THREADS, smem_t, st>>>(tp);
            return check_launch(P, "filterT", st);
        }
    }
    if (M == 4 && (NT == 5 || NT == 9 || NT == 13)) {          // fast path (filter4.cuh)
        auto kern = NT == 5 ? k_filterT_conic4<5> : (NT == 9 ? k_filterT_conic4<9> : k_filterT_conic4<13>);
        const size_t smem4 = filterT4_smem_floats(NT) * 4;
        int rc4 = set_smem(P, kern, smem4);
        if (rc4) return rc4;
        launch_k(P, kern, dim3(cdiv(fp.my, F4_TB), cdiv(fp.mx, F4_TA), P->cfg.batch), dim3(F4T_THREADS), smem4, st, fp);
        return check_launch(P, "filterT", st);
    }
    const size_t smem = ((size_t)NT * NT * M * M + (size_t)M * (S::TA + 2 * T) * M * (S::TB + 2 * T) + 2 * NT) * 4;
    if (smem > 200 * 1024) return EPSGRAD_EUNSUPPORTED;
    int rc = set_smem(P, k_filterT_conic<M>, smem);
    if (rc) return rc;
    k_filterT_conic<M><<<dim3(cdiv(fp.my, S::TB), cdiv(fp.mx, S::TA), P->cfg.batch), S::NTHR, smem, st>>>(fp);
    return check_launch(P, "filterT", st);
}

template <int M>
int launch_filterT_m(epsgrad_plan *P, const float *v, float *dC, cudaStream_t st)
{
    if (!P->separable)
        return launch_filterT_conic<M>(P, v, dC, st);
    const int B = P->cfg.batch, mx = P->cfg.mx, my = P->cfg.my, T = P->T, NT = P->NT;
    SepParams sp;
    sp.w1 = P->d_w; sp.nrm = make_nrm(P);
    sp.mx = mx; sp.my = my; sp.px = P->px; sp.py = P->py; sp.T = T; sp.NT = NT; sp.eta0 = 0.0f;
    {
        sp.in = v; sp.out = ws_tmp(P);
        const size_t smem = sepx_smem_floats(NT, M) * 4;
        if (smem > 200 * 1024) return EPSGRAD_EUNSUPPORTED;
        int rc = set_smem(P, k_sep_down_x<M>, smem);
        if (rc) return rc;
        k_sep_down_x<M><<<dim3(cdiv(P->py, SEPX_THREADS), cdiv(mx, SEPX_NBA), B), SEPX_THREADS, smem, st>>>(sp);
        if ((rc = check_launch(P, "filterT_down_x", st))) return rc;
    }
    {
        sp.in = ws_tmp(P); sp.out = dC;
        const size_t smem = ((size_t)NT * M + (size_t)8 * M * (32 + 2 * T)) * 4;
        if (smem > 200 * 1024) return EPSGRAD_EUNSUPPORTED;
        int rc = set_smem(P, k_sep_down_y<M>, smem);
        if (rc) return rc;
        k_sep_down_y<M><<<dim3(cdiv(my, 32), cdiv(mx, 8), B), SEP_THREADS, smem, st>>>(sp);
        return check_launch(P, "filterT_down_y", st);
    }
}

FilterGenParams fill_filter_general(const epsgrad_plan *P)
{
    FilterGenParams fp;
    std::memset(&fp, 0, sizeof(fp));
    fp.mx = P->cfg.mx; fp.my = P->cfg.my; fp.px = P->px; fp.py = P->py; fp.s = P->cfg.subpixel;
    fp.kind = P->cfg.filter_kind; fp.normalize = P->cfg.filter_normalize;
    fp.ux = (double)P->nx / P->cfg.mx; fp.uy = (double)P->ny / P->cfg.my;
    fp.R = (float)P->cfg.filter_radius; fp.inv_R = (float)(1.0 / P->cfg.filter_radius);
    fp.inv_2s2 = P->cfg.filter_kind == EPSGRAD_FILTER_GAUSSIAN ? (float)(1.0 / (2.0 * P->cfg.filter_sigma * P->cfg.filter_sigma)) : 0.0f;
    fp.eta0 = P->eta0;
    return fp;
}

int launch_filter(epsgrad_plan *P, const float *C, float *phi, cudaStream_t st)
{
    if (P->general) {
        FilterGenParams fp = fill_filter_general(P);
        fp.C = C; fp.phi = phi; fp.invden = ws_invden(P);
        if (P->cfg.batch > 65535) return EPSGRAD_EUNSUPPORTED;
        const size_t n_mask = (size_t)P->px * P->py;
        k_filter_general<<<dim3((unsigned)((n_mask + FG_THREADS - 1) / FG_THREADS), P->cfg.batch), FG_THREADS, 0, st>>>(fp);
        return check_launch(P, "filter", st);
    }
    switch (P->m) {
    case 2: return launch_filter_m<2>(P, C, phi, st);
    case 4: return launch_filter_m<4>(P, C, phi, st);
    case 6: return launch_filter_m<6>(P, C, phi, st);
    case 8: return launch_filter_m<8>(P, C, phi, st);
    }
    return EPSGRAD_EUNSUPPORTED;
}

int launch_filterT(epsgrad_plan *P, const float *v, float *dC, cudaStream_t st)
{
    if (P->general) {
        FilterGenParams fp = fill_filter_general(P);
        fp.v = v; fp.dC = dC;
        if (P->cfg.batch > 65535) return EPSGRAD_EUNSUPPORTED;
        k_filterT_general<<<dim3(cdiv(P->cfg.mx * P->cfg.my, FG_THREADS / 32), P->cfg.batch), FG_THREADS, 0, st>>>(fp);
        return check_launch(P, "filterT", st);
    }
    switch (P->m) {
    case 2: return launch_filterT_m<2>(P, v, dC, st);
    case 4: return launch_filterT_m<4>(P, v, dC, st);
    case 6: return launch_filterT_m<6>(P, v, dC, st);
    case 8: return launch_filterT_m<8>(P, v, dC, st);
    }
    return EPSGRAD_EUNSUPPORTED;
}

// ---- F2..F5: the 2-D chain; e2d / coef / eps2d may be null
Fwd2dParams fill_fwd2d(const epsgrad_plan *P, const float *phi, float beta, float *e2d, float *coef, float *eps2d)
{
    Fwd2dParams fp;
    fp.phi = phi; fp.e2d = e2d; fp.coef = coef; fp.eps2d = eps2d;
    fp.nx = P->nx; fp.ny = P->ny; fp.px = P->px; fp.py = P->py; fp.s = P->cfg.subpixel;
    fp.beta = beta; fp.eta_r = P->eta_r; fp.eps_clad = P->eps_clad; fp.deps = P->deps; fp.delta = P->delta;
    if (P->morph_R > 0) { fp.phi = ws_mc(P); fp.eta_r = 0.0f; }     // Eq. (6) on the filtered mask, centred at 1/2
    fp.w_lo = P->w_lo; fp.w_hi = P->w_hi;
    return fp;
}

int launch_fwd2d(epsgrad_plan *P, const float *phi, float beta, float *e2d, float *coef, float *eps2d, cudaStream_t st)
{
    const Fwd2dParams fp = fill_fwd2d(P, phi, beta, e2d, coef, eps2d);
    const size_t smem = fwd2d_smem_floats(fp.s) * 4;
    auto kern = fp.s == 2 ? k_fwd2d<2> : (fp.s == 4 ? k_fwd2d<4> : k_fwd2d<0>);
    int rc = set_smem(P, kern, smem);
    if (rc) return rc;
    launch_k(P, kern, dim3(cdiv(P->ny, F2_TJ), cdiv(P->nx, F2_TI), P->cfg.batch), dim3(F2_THREADS), smem, st, fp);
    return check_launch(P, "fwd2d", st);
}

// Column addressing of eps (cells_per_piece = 4) or of a field (2) in 16-byte pieces (common.cuh ColumnMap)
ColumnMap make_colmap(const epsgrad_plan *P, int cells_per_piece)
{
    ColumnMap cm;
    const epsgrad_embedding_t &e = P->emb;
    cm.ny = P->ny;
    if (e.nx_full > 0) {
        cm.embedded = 1;
        cm.col_pitch = (unsigned)(e.nz_full / cells_per_piece);
        cm.row_pitch = (size_t)e.ny_full * cm.col_pitch;
        cm.plane_pitch = (size_t)e.nx_full * cm.row_pitch;
        cm.base = (size_t)e.i0 * cm.row_pitch + (size_t)e.j0 * cm.col_pitch + (size_t)(e.k0 / cells_per_piece);
    } else {
        cm.embedded = 0;
        cm.col_pitch = (unsigned)(P->cfg.nz / cells_per_piece);
        cm.row_pitch = (size_t)P->ny * cm.col_pitch;
        cm.plane_pitch = (size_t)(P->slab_nx > 0 ? P->slab_nx : P->nx) * cm.row_pitch;
        cm.base = 0;
    }
    return cm;
}

// ---- F6: the eps store stream
ExtrudeParams fill_extrude(const epsgrad_plan *P, const float *e2d, float *eps)
{
    ExtrudeParams ep;
    ep.e2d = e2d; ep.eps = eps; ep.zw = P->d_zw; ep.ncol = P->nx * P->ny; ep.nz = P->cfg.nz;
    ep.pstride = ep.ncol;
    if (P->slab_nx > 0) { ep.ncol = P->slab_nx * P->ny; ep.e2d += (size_t)P->slab_x0 * P->ny; }     // the slab's rows are one run of columns
    ep.cm = make_colmap(P, 4);
    ep.cpb = extrude_cols_per_block(ep.nz);
    ep.nblk = cdiv(ep.ncol, ep.cpb);
    const int nz4 = ep.nz >> 2;
    ep.sh4 = -1;
    if (EX_THREADS % nz4 == 0)
        for (int sft = 0; sft <= 8; ++sft)
            if ((1 << sft) == nz4) ep.sh4 = sft;
    return ep;
}

int launch_extrude(epsgrad_plan *P, const float *e2d, float *eps, cudaStream_t st)
{
    if (P->cfg.batch > 65535) return EPSGRAD_EUNSUPPORTED;
    if (P->cfg.nz % 4) {
        // columns that are not whole 16-byte pieces: one thread per cell (scalar3d.cuh)
        if (P->emb.nx_full > 0) return EPSGRAD_EUNSUPPORTED;
        ExtrudeScalarParams sp;
        sp.e2d = e2d; sp.eps = eps; sp.zw = P->d_zw; sp.nz = P->cfg.nz;
        sp.pstride = P->nx * P->ny; sp.ncol = sp.pstride;
        if (P->slab_nx > 0) { sp.ncol = P->slab_nx * P->ny; sp.e2d += (size_t)P->slab_x0 * P->ny; }
        const size_t n = (size_t)sp.ncol * sp.nz;
        k_extrude_scalar<<<dim3((unsigned)((n + SC_THREADS - 1) / SC_THREADS), 3, P->cfg.batch), SC_THREADS, 0, st>>>(sp);
        return check_launch(P, "extrude", st);
    }
    const ExtrudeParams ep = fill_extrude(P, e2d, eps);
    if (P->eps_window_only) {
        // only the z cells that depend on the design (extrude_window.cuh): the union of the slab windows, in whole 32-byte sectors
        ExtrudeWindowParams wp;
        wp.e = ep;
        int lo = ep.nz, hi = -1;
        for (int g = 0; g < 2; ++g)
            if (P->nch[g] > 0) { lo = std::min(lo, 2 * P->ch0[g]); hi = std::max(hi, 2 * (P->ch0[g] + P->nch[g]) - 1); }
        if (hi < lo) return EPSGRAD_OK;                          // no cell of any column depends on the design
        const int nz4 = ep.nz / 4;
        wp.q0 = (lo / 4) & ~1;
        wp.nq = std::min(nz4, (std::min(hi, ep.nz - 1) / 4 + 2) & ~1) - wp.q0;
        if ((double)ep.ncol * wp.nq > 2.0e9) return EPSGRAD_EUNSUPPORTED;
        const unsigned nblk = (unsigned)(((size_t)ep.ncol * wp.nq + EW_THREADS - 1) / EW_THREADS);
        launch_k(P, k_extrude_window, dim3(nblk, 3, P->cfg.batch), dim3(EW_THREADS), 0, st, wp);
        return check_launch(P, "extrude", st);
    }
    if (P->use_bulk && P->emb.nx_full == 0) {
        // thin persistent store stream (extrude_bulk.cuh): columns of a plane are one contiguous run
        ExtrudeBulkParams bp;
        bp.e2d = ep.e2d; bp.eps = eps; bp.zw = P->d_zw; bp.ncol = ep.ncol; bp.nz = ep.nz; bp.pstride = ep.pstride;
        bp.eps_clad = P->eps_clad;
        int lo = ep.nz, hi = -1;                                  // union of the two slab windows in 16-byte pieces of eps (4 cells)
        for (int g = 0; g < 2; ++g)
            if (P->nch[g] > 0) { lo = std::min(lo, 2 * P->ch0[g]); hi = std::max(hi, 2 * (P->ch0[g] + P->nch[g]) - 1); }
        bp.q0 = hi >= lo ? lo / 4 : 0;
        bp.nq = hi >= lo ? std::min(hi, ep.nz - 1) / 4 - bp.q0 + 1 : 0;
        const int blk_bytes = P->tune[0] > 0 ? P->tune[0] : 16384;
        int cols = blk_bytes / (ep.nz * 4);
        if (bp.nq > 0 && cols * bp.nq > 4 * EXB_THREADS) cols = 4 * EXB_THREADS / bp.nq;
        if (cols >= 1) {
            bp.cols = cols;
            bp.nblk = cdiv(bp.ncol, cols);
            const size_t smem_b = (size_t)EXB_NBUF * cols * ep.nz * 4;
            int rcb = set_smem(P, k_extrude_bulk, smem_b);
            if (rcb) return rcb;
            const int per_sm = P->tune[1] > 0 ? P->tune[1] : 2;
            const int n_items = 3 * bp.nblk, n_want = std::max(1, per_sm * P->n_sm / P->cfg.batch);
            k_extrude_bulk<<<dim3(std::min(n_items, n_want), 1, P->cfg.batch), EXB_THREADS, smem_b, st>>>(bp);
            return check_launch(P, "extrude", st);
        }
    }
    const size_t smem = (size_t)3 * ep.cpb * 4;
    int rc = set_smem(P, k_extrude, smem);
    if (rc) return rc;
    launch_k(P, k_extrude, dim3(ep.nblk, 3, P->cfg.batch), dim3(EX_THREADS), smem, st, ep);
    return check_launch(P, "extrude", st);
}

// ---- R1: the field read stream; more than ZR_MAX_PAIRS pairs are chained through accumulating launches
// first chunk and number of chunks of the union of the two slab windows (x|y and z) of a field column
void window_union(const epsgrad_plan *P, int *first, int *count)
{
    int lo = P->cfg.nz / 2, hi = 0;
    for (int g = 0; g < 2; ++g)
        if (P->nch[g] > 0) { lo = std::min(lo, P->ch0[g]); hi = std::max(hi, P->ch0[g] + P->nch[g]); }
    *first = hi > lo ? lo : 0;
    *count = hi > lo ? hi - lo : 0;
}

extern "C" int epsgrad_plan_set_eps_window_only(epsgrad_plan_t *P, int enable)
{
    if (!P) return EPSGRAD_EINVAL;
    if (enable && P->cfg.nz % 4) return EPSGRAD_EUNSUPPORTED;
    P->eps_window_only = enable != 0;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_packed_fields(epsgrad_plan_t *P, int enable)
{
    if (!P) return EPSGRAD_EINVAL;
    if (enable && (P->emb.nx_full > 0 || P->slab_nx > 0 || P->dense || P->cfg.nz % 4)) return EPSGRAD_EUNSUPPORTED;
    P->packed_fields = enable != 0;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_packed_window(const epsgrad_plan_t *P, int *first_cell, int *n_cells)
{
    if (!P || !first_cell || !n_cells) return EPSGRAD_EINVAL;
    int u0 = 0, un = 0;
    window_union(P, &u0, &un);
    *first_cell = 2 * u0;                  // 16-byte chunks of two complex64 cells
    *n_cells = 2 * un;
    return EPSGRAD_OK;
}

// everything of ZredParams but the field pointers; smem: bytes of staging a CTA needs; sparse: windows worth 64-byte fills
int fill_zreduce(const epsgrad_plan *P, float *gbar, bool packed, ZredParams &zp, size_t &smem, bool &sparse, int &maxnch,
                 int max_cols = ZR_COLS, int stage_chunks = ZR_STAGE_CHUNKS)
{
    zp.gbar = gbar; zp.zw = P->d_zw; zp.ncol = P->nx * P->ny; zp.nz = P->cfg.nz;
    zp.evict_first = P->tune[5] == 1;      // the launch decides for knob value 0 (launch_zreduce)
    zp.pstride = zp.ncol;
    if (P->slab_nx > 0) {
        zp.ncol = P->slab_nx * P->ny;
        zp.gbar += (size_t)P->slab_x0 * P->ny;
    }
    zp.cm = make_colmap(P, 2);
    int u0 = 0, un = 0;
    zp.choff = 0;
    if (packed) {
        window_union(P, &u0, &un);
        zp.cm.embedded = 0;
        zp.cm.col_pitch = (unsigned)un;
        zp.cm.row_pitch = (size_t)P->ny * un;
        zp.cm.plane_pitch = (size_t)P->nx * zp.cm.row_pitch;
        zp.cm.base = 0;
        zp.choff = u0;
    }
    maxnch = 1;
    for (int g = 0; g < 2; ++g) {
        zp.ch0[g] = P->dense ? 0 : P->ch0[g];
        zp.nch[g] = P->dense ? P->cfg.nz / 2 : P->nch[g];
        if (zp.nch[g] > maxnch) maxnch = zp.nch[g];
        zp.chs[g] = 0;
        while ((1 << zp.chs[g]) < zp.nch[g]) ++zp.chs[g];
        if (zp.chs[g] > 8) return EPSGRAD_EUNSUPPORTED;     // window wider than one CTA pass (nz > 512)
    }
    smem = 0;
    for (int g = 0; g < 2; ++g) {
        zp.ncp[g] = zred_cols_per_pass(zp.nch[g], max_cols, stage_chunks);
        if (zp.ncp[g] < 1) return EPSGRAD_EUNSUPPORTED;
        const size_t need = (size_t)2 * (zp.nch[g] | 1) * zp.ncp[g] * 16;
        if (need > smem) smem = need;
    }
    zp.nblk = cdiv(zp.ncol, ZR_COLS);
    // windows of at most 128 bytes per column: ask for 64-byte fills
    sparse = maxnch * 16 <= 128 && zp.nz * 8 > 128 && !packed;     // packed windows are one dense stream
    return EPSGRAD_OK;
}

// packed: EF / EA hold only the union window of every column, [B,3,ncol][count] chunks (the host entry point's gather)
int launch_zreduce(epsgrad_plan *P, int n_pairs, const void *const *EF, const void *const *EA, float *gbar, cudaStream_t st,
                   bool host_src, bool packed)
{
    ZredParams zp;
    size_t smem = 0;
    bool sparse = false;
    int maxnch = 1;
    if (P->packed_fields && !host_src && !P->cur_host_src) {      // device fields on the slab window only (epsgrad_plan_set_packed_fields)
        if (P->emb.nx_full > 0 || P->slab_nx > 0 || P->dense || P->cfg.nz % 4) return EPSGRAD_EUNSUPPORTED;
        packed = true;
    }
    // x-slab: only the slab's rows have fields; the cotangent of every other column of the region is zero
    if (P->slab_nx > 0 &&
        cudaMemsetAsync(gbar, 0, (size_t)P->cfg.batch * 5 * P->nx * P->ny * sizeof(float), st) != cudaSuccess) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    int widest = 0;                                               // slab window in 16-byte chunks
    for (int g = 0; g < 2; ++g) widest = std::max(widest, P->dense ? P->cfg.nz / 2 : P->nch[g]);
    if (P->cfg.nz % 4 || (widest > 256 && P->emb.nx_full == 0 && !packed && !host_src && !P->cur_host_src)) {
        // field columns that are not whole 16-byte chunks, or a window wider than one CTA pass of the vector kernel (512
        // cells): one thread per column, 8-byte loads (scalar3d.cuh)
        if (P->emb.nx_full > 0 || packed || host_src || P->cur_host_src) return EPSGRAD_EUNSUPPORTED;
        if (P->cfg.batch > 65535) return EPSGRAD_EUNSUPPORTED;
        ZredScalarParams sp;
        sp.gbar = gbar; sp.zw = P->d_zw; sp.nz = P->cfg.nz;
        sp.pstride = P->nx * P->ny; sp.ncol = sp.pstride;
        if (P->slab_nx > 0) { sp.ncol = P->slab_nx * P->ny; sp.gbar += (size_t)P->slab_x0 * P->ny; }
        for (int g = 0; g < 2; ++g) {
            sp.k0[g] = P->dense ? 0 : 2 * P->ch0[g];
            sp.k1[g] = P->dense ? sp.nz : std::min(sp.nz, 2 * (P->ch0[g] + P->nch[g]));
        }
        for (int p0 = 0; p0 < n_pairs; p0 += ZR_MAX_PAIRS) {
            const int np = std::min(ZR_MAX_PAIRS, n_pairs - p0);
            for (int p = 0; p < ZR_MAX_PAIRS; ++p) {
                sp.ef[p] = (const float2 *)(p < np ? EF[p0 + p] : nullptr);
                sp.ea[p] = (const float2 *)(p < np ? EA[p0 + p] : nullptr);
            }
            sp.n_pairs = np; sp.accumulate = p0 > 0;
            k_zreduce_scalar<<<dim3(cdiv(sp.ncol, SC_THREADS), 3, P->cfg.batch), SC_THREADS, 0, st>>>(sp);
            int rcs = check_launch(P, "zreduce", st);
            if (rcs) return rcs;
        }
        return EPSGRAD_OK;
    }
    int rcf = fill_zreduce(P, gbar, packed, zp, smem, sparse, maxnch);
    if (rcf) return rcf;
    // L2 evict-first fills: they keep the field stream from pushing the previous step's dirty eps lines (at most
    // one L2 of them) out under itself -- 104 -> 96 us per step at paper scale.  That cost is fixed, so it only matters for
    // streams of a few L2 sizes; on the multi-GB streams of Large / Wide batch the policy costs ~1 % instead, so by default it
    // is on up to 4 GB of field columns per launch (knob 5: 1 always, 2 never).
    if (P->tune[5] == 0) zp.evict_first = (double)P->cfg.batch * 3.0 * zp.ncol * zp.nz * 16.0 * std::min(n_pairs, ZR_MAX_PAIRS) <= 4.0e9;
    host_src = host_src || P->cur_host_src;
    if (!host_src && !packed && P->use_tma == 2 && P->tma_encode && P->emb.nx_full == 0 && maxnch <= 24) {
        // thin persistent read stream (zreduce_pipe.cuh): TMA boxes {window, ZP_COLS columns} through a ring of stages
        typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                     const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                     CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
        EncodeFn enc = (EncodeFn)P->tma_encode;
        ZredPipeParams pp;
        pp.gbar = zp.gbar; pp.zw = P->d_zw; pp.ncol = zp.ncol; pp.nz = zp.nz; pp.pstride = zp.pstride;
        for (int g = 0; g < 2; ++g) { pp.ch0[g] = zp.ch0[g]; pp.nch[g] = zp.nch[g]; }
        pp.wb = maxnch | 1;
        pp.nblk = cdiv(zp.ncol, ZP_COLS);
        const cuuint64_t dims[2] = {(cuuint64_t)zp.nz * 2, (cuuint64_t)P->cfg.batch * 3 * zp.ncol};
        const cuuint64_t strides[1] = {(cuuint64_t)zp.nz * 8};
        const cuuint32_t box[2] = {(cuuint32_t)pp.wb * 4, (cuuint32_t)ZP_COLS}, es[2] = {1, 1};
        const int stage_b = 2 * ZP_COLS * pp.wb * 16;
        pp.nstage = P->tune[2] > 0 ? P->tune[2] : std::max(2, std::min(8, 100 * 1024 / stage_b));
        if (pp.nstage > ZP_MAX_STAGE) pp.nstage = ZP_MAX_STAGE;
        const size_t smem_p = zpipe_smem_bytes(pp.wb, pp.nstage);
        if (smem_p > 220 * 1024) return EPSGRAD_EUNSUPPORTED;
        int rcp = set_smem(P, k_zreduce_pipe, smem_p);
        if (rcp) return rcp;
        const CUtensorMapL2promotion promo = sparse ? CU_TENSOR_MAP_L2_PROMOTION_L2_64B : CU_TENSOR_MAP_L2_PROMOTION_L2_128B;
        const int n_items = 3 * pp.nblk, n_want = std::max(1, (P->tune[3] > 0 ? P->tune[3] : 1) * P->n_sm / P->cfg.batch);
        const dim3 grid_p(std::min(n_items, n_want), 1, P->cfg.batch);
        if (P->cfg.batch > 65535) return EPSGRAD_EUNSUPPORTED;
        for (int p0 = 0; p0 < n_pairs; p0 += ZR_MAX_PAIRS) {
            const int np = n_pairs - p0 < ZR_MAX_PAIRS ? n_pairs - p0 : ZR_MAX_PAIRS;
            for (int p = 0; p < np; ++p) {
                if (enc(&pp.mf[p], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void *>(EF[p0 + p]), dims, strides, box, es,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS ||
                    enc(&pp.ma[p], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void *>(EA[p0 + p]), dims, strides, box, es,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
                    return EPSGRAD_ECUDA;
            }
            for (int p = np; p < ZR_MAX_PAIRS; ++p) { pp.mf[p] = pp.mf[0]; pp.ma[p] = pp.ma[0]; }
            pp.n_pairs = np; pp.accumulate = p0 > 0;
            k_zreduce_pipe<<<grid_p, ZP_THREADS, smem_p, st>>>(pp);
            rcp = check_launch(P, "zreduce", st);
            if (rcp) return rcp;
        }
        return EPSGRAD_OK;
    }
    if (sparse && !host_src && P->use_tma == 1 && P->emb.nx_full == 0 && P->slab_nx == 0) {
        // TMA variant (zreduce.cuh): one 2-D tensor map per field, rows = z columns, box = {window, 256 columns}
        typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                     const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                     CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
        EncodeFn enc = (EncodeFn)P->tma_encode;
        ZredTmaParams tp;
        tp.gbar = gbar; tp.zw = P->d_zw; tp.ncol = zp.ncol; tp.nz = zp.nz;
        for (int g = 0; g < 2; ++g) { tp.ch0[g] = zp.ch0[g]; tp.nch[g] = zp.nch[g]; }
        tp.wb = (zp.nch[0] | 1) > (zp.nch[1] | 1) ? (zp.nch[0] | 1) : (zp.nch[1] | 1);
        const cuuint64_t dims[2] = {(cuuint64_t)zp.nz * 2, (cuuint64_t)P->cfg.batch * 3 * zp.ncol};
        const cuuint64_t strides[1] = {(cuuint64_t)zp.nz * 8};
        const cuuint32_t box[2] = {(cuuint32_t)tp.wb * 4, (cuuint32_t)ZR_COLS}, es[2] = {1, 1};
        const size_t smem_t = (size_t)2 * ZR_COLS * tp.wb * 16 + 128;
        int rct = set_smem(P, k_zreduce_tma, smem_t);
        if (rct) return rct;
        const int per_sm = 5;                                   // resident set: 5 CTAs x 40 KB of windows in flight per SM
        const int n_items = 3 * cdiv(zp.ncol, ZR_COLS), n_want = per_sm * P->n_sm / P->cfg.batch;
        const dim3 grid_t(n_items < n_want || n_want < 1 ? n_items : n_want, P->cfg.batch);
        if (P->cfg.batch > 65535) return EPSGRAD_EUNSUPPORTED;
        for (int p0 = 0; p0 < n_pairs; p0 += ZR_MAX_PAIRS) {
            const int np = n_pairs - p0 < ZR_MAX_PAIRS ? n_pairs - p0 : ZR_MAX_PAIRS;
            for (int p = 0; p < np; ++p) {
                if (enc(&tp.mf[p], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void *>(EF[p0 + p]), dims, strides, box, es,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_64B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS ||
                    enc(&tp.ma[p], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void *>(EA[p0 + p]), dims, strides, box, es,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_64B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
                    return EPSGRAD_ECUDA;
            }
            for (int p = np; p < ZR_MAX_PAIRS; ++p) { tp.mf[p] = tp.mf[0]; tp.ma[p] = tp.ma[0]; }
            tp.n_pairs = np; tp.accumulate = p0 > 0;
            k_zreduce_tma<<<grid_t, ZR_THREADS, smem_t, st>>>(tp);
            rct = check_launch(P, "zreduce", st);
            if (rct) return rct;
        }
        return EPSGRAD_OK;
    }
    auto kern = host_src ? k_zreduce<false, true> : (sparse ? k_zreduce<true, false> : k_zreduce<false, false>);
    int rc = set_smem(P, kern, smem);
    if (rc) return rc;
    if (P->cfg.batch > 65535) return EPSGRAD_EUNSUPPORTED;
    const dim3 grid(zp.nblk, 3, P->cfg.batch);
    for (int p0 = 0; p0 < n_pairs; p0 += ZR_MAX_PAIRS) {
        const int np = n_pairs - p0 < ZR_MAX_PAIRS ? n_pairs - p0 : ZR_MAX_PAIRS;
        for (int p = 0; p < ZR_MAX_PAIRS; ++p) {
            zp.ef[p] = (const float4 *)(p < np ? EF[p0 + p] : nullptr);
            zp.ea[p] = (const float4 *)(p < np ? EA[p0 + p] : nullptr);
        }
        zp.n_pairs = np; zp.accumulate = p0 > 0;
        kern<<<grid, ZR_THREADS, smem, st>>>(zp);
        rc = check_launch(P, "zreduce", st);
        if (rc) return rc;
    }
    return EPSGRAD_OK;
}

// ---- Eqs. (4)-(5): "dilate, erode, erode, dilate" (S17) between the first projection and Eq. (6)
int launch_morph_one(epsgrad_plan *P, const MorphParams &mp, cudaStream_t st, const char *name)
{
    const size_t smem = morph_smem_floats(P->morph_R) * 4;
    int rc = set_smem(P, k_morph, smem);
    if (rc) return rc;
    k_morph<<<dim3(cdiv(P->py, MO_T), cdiv(P->px, MO_T), P->cfg.batch), MO_THREADS, smem, st>>>(mp);
    return check_launch(P, name, st);
}

MorphParams morph_base(const epsgrad_plan *P, float beta)
{
    MorphParams mp;
    std::memset(&mp, 0, sizeof(mp));
    mp.hl = P->d_hl; mp.invn = P->d_invn; mp.nrm = make_nrm(P);
    mp.px = P->px; mp.py = P->py; mp.R = P->morph_R;
    mp.beta = beta; mp.eta_r = P->eta_r;
    return mp;
}

// forward: Phi' -> rho0 (kept in m[0]) -> z_1 (m[1]) -> z_2 (m[2]) -> z_3 (m[3]) -> rho~ - 1/2 (mc); z-space: morph.cuh
int launch_morph_forward(epsgrad_plan *P, const float *phi, float beta, cudaStream_t st)
{
    static const float sign[4] = {1.f, -1.f, -1.f, 1.f};
    for (int k = 0; k < 4; ++k) {
        MorphParams mp = morph_base(P, beta);
        mp.x = k == 0 ? phi : ws_m(P, k);
        mp.out = k == 3 ? ws_mc(P) : ws_m(P, k + 1);
        mp.rho0 = ws_m(P, 0);
        mp.first = k == 0; mp.last = k == 3; mp.transposed = 0;
        mp.x_inv = k > 0 && sign[k] != sign[k - 1];
        mp.a = sign[k] * P->morph_alpha;
        int rc = launch_morph_one(P, mp, st, "morph");
        if (rc) return rc;
    }
    return EPSGRAD_OK;
}

// transposed: cotangent of rho~ (cot) -> ... -> v (the last op applies projection^T and 1/den); buffers alternate
int launch_morph_reverse(epsgrad_plan *P, const float *phi, float beta, float *v, cudaStream_t st)
{
    static const float sign[4] = {1.f, -1.f, -1.f, 1.f};
    float *src = v, *dst = ws_cot(P);                  // maskgrad left the cotangent of rho~ in v; four ops later the result is back in v
    for (int k = 3; k >= 0; --k) {
        MorphParams mp = morph_base(P, beta);
        mp.x = k == 0 ? phi : ws_m(P, k);
        mp.y = k == 3 ? ws_mc(P) : ws_m(P, k + 1);
        mp.ybar = src;
        mp.out = dst;
        mp.rho0 = ws_m(P, 0);
        mp.first = k == 0; mp.last = k == 3; mp.transposed = 1;
        mp.x_inv = k > 0 && sign[k] != sign[k - 1];
        mp.dbeta_part = k == 0 && P->cur_dbeta ? ws_part(P) + (size_t)P->cfg.batch * P->n_part_mg : nullptr;   // [B][n_part_mo]
        mp.a = sign[k] * P->morph_alpha;
        int rc = launch_morph_one(P, mp, st, "morphT");
        if (rc) return rc;
        float *t = src; src = dst; dst = t;
    }
    return EPSGRAD_OK;
}

// d F/d beta: add the per-CTA partial sums maskgrad (and, with the filters on, the last morph^T op) left
int launch_dbeta_sum(epsgrad_plan *P, cudaStream_t st)
{
    if (!P->cur_dbeta) return EPSGRAD_OK;
    const float *pa = ws_part(P);
    k_sum_partials<<<P->cfg.batch, 256, 0, st>>>(pa, P->n_part_mg, pa + (size_t)P->cfg.batch * P->n_part_mg, P->n_part_mo, 1.0f, P->cur_dbeta);
    return check_launch(P, "dbeta", st);
}

// F1 and, when they are on, the first projection and the morphological filters
int launch_front(epsgrad_plan *P, const float *C, float beta, cudaStream_t st)
{
    int rc = launch_filter(P, C, ws_phi(P), st);
    if (!rc && P->morph_R > 0) rc = launch_morph_forward(P, ws_phi(P), beta, st);
    return rc;
}

// ---- R2..R5
MaskGradParams fill_maskgrad(const epsgrad_plan *P, const float *phi, float beta, const float *gbar, const float *coef, float *v)
{
    MaskGradParams mp;
    mp.phi = phi; mp.gbar = gbar; mp.coef = coef; mp.v = v; mp.nrm = make_nrm(P);
    mp.nx = P->nx; mp.ny = P->ny; mp.px = P->px; mp.py = P->py; mp.s = P->cfg.subpixel;
    mp.beta = beta; mp.eta_r = P->eta_r; mp.eps_clad = P->eps_clad; mp.deps = P->deps;
    mp.use_den = 1;
    mp.dbeta_part = P->cur_dbeta ? ws_part(P) : nullptr;               // [B][n_part_mg]
    if (P->morph_R > 0) { mp.phi = ws_mc(P); mp.eta_r = 0.0f; mp.use_den = 0; }   // v holds the cotangent of rho~: the filters^T follow
    return mp;
}

int launch_maskgrad(epsgrad_plan *P, const float *phi, float beta, const float *gbar, const float *coef, float *v, cudaStream_t st)
{
    const MaskGradParams mp = fill_maskgrad(P, phi, beta, gbar, coef, v);
    const size_t smem = maskgrad_smem_floats(mp.s) * 4;
    auto kern = mp.s == 2 ? k_maskgrad<2> : (mp.s == 4 ? k_maskgrad<4> : k_maskgrad<0>);
    int rc = set_smem(P, kern, smem);
    if (rc) return rc;
    launch_k(P, kern, dim3(cdiv(P->ny, MG_TJ), cdiv(P->nx, MG_TI), P->cfg.batch), dim3(MG_THREADS), smem, st, mp);
    return check_launch(P, "maskgrad", st);
}

int check_common(epsgrad_plan *P, const float *C, float beta)
{
    if (!P || !aligned16(C) || !(beta > 0.0f) || !std::isfinite(beta)) return EPSGRAD_EINVAL;
    if (!P->ws) return EPSGRAD_ENOWORKSPACE;
    return EPSGRAD_OK;
}

int check_pairs(int n_pairs, const void *const *EF, const void *const *EA)
{
    if (n_pairs < 1 || !EF || !EA) return EPSGRAD_EINVAL;
    for (int p = 0; p < n_pairs; ++p)
        if (!aligned16(EF[p]) || !aligned16(EA[p])) return EPSGRAD_EINVAL;
    return EPSGRAD_OK;
}


// ---- the whole step as one persistent dataflow kernel (mega.cuh)
bool mega_applies(const epsgrad_plan *P, int n_pairs)
{
    return P->use_mega == 1 && P->d_sched && P->cfg.nz % 4 == 0 && !P->cur_dbeta && P->slab_nx == 0 && !P->packed_fields && !P->eps_window_only && !P->cur_host_src && !P->prof && n_pairs <= ZR_MAX_PAIRS;
}

template <int NTC>
int launch_mega_nt(epsgrad_plan *P, MegaParams &mp, bool sparse, size_t smem, cudaStream_t st)
{
    auto kern = sparse ? k_mega<NTC, true> : k_mega<NTC, false>;
    int rc = set_smem(P, kern, smem);
    if (rc) return rc;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, MK_THREADS, smem) != cudaSuccess || per_sm < 1) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    if (P->tune[4] > 0 && P->tune[4] < per_sm) per_sm = P->tune[4];
    const int grid = per_sm * P->n_sm;
    if (cudaMemsetAsync(P->d_sched, 0, P->sched_bytes, st) != cudaSuccess) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    kern<<<grid, MK_THREADS, smem, st>>>(mp);
    return check_launch(P, "chain", st);
}

// phases: which steps this launch runs (bit PH_*); the others' outputs are taken as complete (an earlier launch made them)
int launch_mega(epsgrad_plan *P, const float *C, float beta, int n_pairs, const void *const *EF, const void *const *EA,
                float *eps, float *dFdC, cudaStream_t st, unsigned phases = 0x3f)
{
    MegaParams mp;
    std::memset(&mp, 0, sizeof(mp));
    const int T = P->T, NT = P->NT, nx = P->nx, ny = P->ny, mx = P->cfg.mx, my = P->cfg.my;
    mp.f1 = fill_filter(P, C, ws_phi(P));
    mp.f2 = fill_fwd2d(P, ws_phi(P), beta, eps ? ws_e2d(P) : nullptr, dFdC ? ws_coef(P) : nullptr, nullptr);
    mp.sched = P->d_sched;
    mp.prof = P->d_mprof;
    mp.B = P->cfg.batch;
    mp.nb = cdiv(nx, MK_BAND);
    mp.nbx1 = cdiv(my, F4_TB);
    mp.nbx2 = cdiv(ny, F2_TJ);
    mp.w_floats = NT * NT * 16;
    const int ntr = cdiv(mx, F4_TA), rows_last = nx - (mp.nb - 1) * MK_BAND;
    size_t scratch = std::max((size_t)((F4_TA + 2 * T) * (F4_TB + 2 * T + 1) + 4 + MK_G * F4_THREADS * 16) * 4,
                              fwd2d_smem_floats(2) * 4);
    size_t zsmem = 0;
    mp.full[PH_F1] = 2 * mp.nbx1;            mp.last[PH_F1] = (ntr - 2 * (mp.nb - 1)) * mp.nbx1;
    mp.full[PH_F2] = mp.last[PH_F2] = mp.nbx2;
    bool sparse = false;
    if (eps) {
        mp.ex = fill_extrude(P, ws_e2d(P), eps);
        mp.xblk[0] = cdiv(MK_BAND * ny, mp.ex.cpb); mp.xblk[1] = cdiv(rows_last * ny, mp.ex.cpb);
        mp.full[PH_X] = 3 * mp.xblk[0];      mp.last[PH_X] = 3 * mp.xblk[1];
        scratch = std::max(scratch, (size_t)3 * mp.ex.cpb * 4);
    }
    if (dFdC) {
        int maxnch = 1;
        int rc = fill_zreduce(P, ws_gbar(P), false, mp.zr, zsmem, sparse, maxnch, MK_ZCOLS, MK_ZCOLS * 5);
        if (rc) return rc;
        for (int p = 0; p < ZR_MAX_PAIRS; ++p) {
            mp.zr.ef[p] = (const float4 *)(p < n_pairs ? EF[p] : nullptr);
            mp.zr.ea[p] = (const float4 *)(p < n_pairs ? EA[p] : nullptr);
        }
        mp.zr.n_pairs = n_pairs; mp.zr.accumulate = 0;
        mp.zblk[0] = cdiv(MK_BAND * ny, MK_ZCOLS); mp.zblk[1] = cdiv(rows_last * ny, MK_ZCOLS);
        mp.full[PH_Z] = 3 * mp.zblk[0];      mp.last[PH_Z] = 3 * mp.zblk[1];
        mp.mg = fill_maskgrad(P, ws_phi(P), beta, ws_gbar(P), ws_coef(P), ws_v(P));
        mp.full[PH_M] = mp.last[PH_M] = mp.nbx2;
        mp.ft = fill_filterT(P, ws_v(P), dFdC);
        mp.full[PH_T] = mp.full[PH_F1];      mp.last[PH_T] = mp.last[PH_F1];
        scratch = std::max(scratch, maskgrad_smem_floats(2) * 4);
        scratch = std::max(scratch, ((size_t)filterT4_tile_rows(NT, MK_TPASS) * filterT4_pitch(T) + (size_t)MK_G * F4_TA * F4_TB) * 4);
    }
    scratch = align_up(scratch, 16);
    mp.scratch_floats = (int)(scratch / 4);
    // pipeline step of band b: tau = b + lag; every dependence points to a smaller tau (mega.cuh)
    // An item runs for several steps' worth of tickets (a step of 16 rows is ~190 tickets for ~600 CTAs), so the lag between a
    // phase and its consumer is a few steps: the consumer's bands are then complete when its ticket comes up.
    const int L = P->tune[6] > 0 ? P->tune[6] : 7;
    mp.lag[PH_Z] = 0; mp.lag[PH_F1] = 0; mp.lag[PH_F2] = L; mp.lag[PH_X] = 2 * L; mp.lag[PH_M] = 2 * L; mp.lag[PH_T] = 3 * L;
    for (int ph = 0; ph < PH_N; ++ph)
        if (!(phases >> ph & 1)) mp.full[ph] = mp.last[ph] = 0;
    if (!(phases >> PH_Z & 1)) zsmem = 0;
    const size_t smem = (size_t)mp.w_floats * 4 + scratch + zsmem;
    if (smem > 200 * 1024) return EPSGRAD_EUNSUPPORTED;
    switch (NT) {
    case 5: return launch_mega_nt<5>(P, mp, sparse, smem, st);
    case 9: return launch_mega_nt<9>(P, mp, sparse, smem, st);
    case 13: return launch_mega_nt<13>(P, mp, sparse, smem, st);
    }
    return EPSGRAD_EUNSUPPORTED;
}

// The whole path.  eps == nullptr skips F6, dFdC == nullptr skips R1-R6.
// Dependencies: fwd2d <- filter;  extrude <- fwd2d;  maskgrad <- zreduce, fwd2d;  filterT <- maskgrad;  zreduce <- nothing.
// Two HBM-bound kernels (zreduce: field reads; extrude: eps stores) and four small L2-resident ones.  Running the two
// HBM streams at once gains nothing (measured: DRAM is the shared limit); hiding the small kernels under
// them does.  With overlap on, the small kernels go to the plan's auxiliary stream, which has the highest priority so
// that their CTAs are placed ahead of the pending CTAs of the big kernels: filter -> fwd2d run there beside zreduce,
// then maskgrad -> filterT beside extrude (which follows zreduce on the caller's stream).  The call joins the auxiliary
// stream back before returning: to the caller everything is ordered on `stream`, there is no host synchronisation, and
// the call stays CUDA-graph capturable.
int run_chain(epsgrad_plan *P, const float *C, float beta, int n_pairs, const void *const *EF,
              const void *const *EA, float *eps, float *dFdC, cudaStream_t st)
{
    int rc = EPSGRAD_OK;
    if (mega_applies(P, n_pairs)) return launch_mega(P, C, beta, n_pairs, EF, EA, eps, dFdC, st);
    if (!dFdC || !P->overlap || P->prof) {
        rc = launch_front(P, C, beta, st);
        if (!rc) rc = launch_fwd2d(P, ws_phi(P), beta, eps ? ws_e2d(P) : nullptr, dFdC ? ws_coef(P) : nullptr, nullptr, st);
        if (!rc && dFdC) rc = launch_zreduce(P, n_pairs, EF, EA, ws_gbar(P), st);
        if (!rc && eps) rc = launch_extrude(P, ws_e2d(P), eps, st);
        if (!rc && dFdC) rc = launch_maskgrad(P, ws_phi(P), beta, ws_gbar(P), ws_coef(P), ws_v(P), st);
        if (!rc && dFdC && P->morph_R > 0) rc = launch_morph_reverse(P, ws_phi(P), beta, ws_v(P), st);
        if (!rc && dFdC) rc = launch_filterT(P, ws_v(P), dFdC, st);
        if (!rc && dFdC) rc = launch_dbeta_sum(P, st);
        return rc;
    }
    cudaStream_t ax = P->aux;
    stamp(P, "begin", st);
    // (event records and waits sit between most kernels of the two streams: only filter -> 2-D stage and mask cotangent ->
    // transposed filter are adjacent launches, and those two pairs chain by programmatic dependent launch)
    if (cudaEventRecord(P->ev_fork, st) != cudaSuccess || cudaStreamWaitEvent(ax, P->ev_fork, 0) != cudaSuccess) {
        cudaGetLastError();
        return EPSGRAD_ECUDA;
    }
    const bool chains = P->use_mega == 2 && P->d_sched && P->cfg.nz % 4 == 0 && !P->cur_dbeta && P->slab_nx == 0;   // the 2-D chains as two persistent kernels
    if (chains) rc = launch_mega(P, C, beta, n_pairs, EF, EA, eps, dFdC, ax, 1u << PH_F1 | 1u << PH_F2);
    else rc = launch_front(P, C, beta, ax);
    if (!rc) rc = launch_zreduce(P, n_pairs, EF, EA, ws_gbar(P), st);
    pdl_break(P);
    if (!rc && cudaEventRecord(P->ev_r, st) != cudaSuccess) rc = EPSGRAD_ECUDA;
    if (!rc && !chains) rc = launch_fwd2d(P, ws_phi(P), beta, eps ? ws_e2d(P) : nullptr, ws_coef(P), nullptr, ax);
    pdl_break(P);
    if (!rc && cudaEventRecord(P->ev_2d, ax) != cudaSuccess) rc = EPSGRAD_ECUDA;
    if (!rc && cudaStreamWaitEvent(ax, P->ev_r, 0) != cudaSuccess) rc = EPSGRAD_ECUDA;
    if (!rc && chains) rc = launch_mega(P, C, beta, n_pairs, EF, EA, eps, dFdC, ax, 1u << PH_M | 1u << PH_T);
    if (!rc && !chains) rc = launch_maskgrad(P, ws_phi(P), beta, ws_gbar(P), ws_coef(P), ws_v(P), ax);
    if (!rc && eps) {
        if (cudaStreamWaitEvent(st, P->ev_2d, 0) != cudaSuccess) rc = EPSGRAD_ECUDA;
        if (!rc) rc = launch_extrude(P, ws_e2d(P), eps, st);
    }
    if (!rc && P->morph_R > 0) rc = launch_morph_reverse(P, ws_phi(P), beta, ws_v(P), ax);
    if (!rc && !chains) rc = launch_filterT(P, ws_v(P), dFdC, ax);
    if (!rc) rc = launch_dbeta_sum(P, ax);
    // always join, even on error, so that the auxiliary stream never outlives the call
    if (cudaEventRecord(P->ev_join, ax) != cudaSuccess || cudaStreamWaitEvent(st, P->ev_join, 0) != cudaSuccess) {
        cudaGetLastError();
        if (!rc) rc = EPSGRAD_ECUDA;
    }
    return rc;
}

}  // namespace epsgrad

using namespace epsgrad;

// ------------------------------------------------------------------------------------ hot path
extern "C" int eps_forward(epsgrad_plan_t *P, const float *C, float beta, float *eps, void *stream)
{
    int rc = check_common(P, C, beta);
    if (rc) return rc;
    if (!aligned16(eps)) return EPSGRAD_EINVAL;
    DeviceGuard g(P->device);
    cudaStream_t st = (cudaStream_t)stream;
    begin_call(P, st);
    return run_chain(P, C, beta, 0, nullptr, nullptr, eps, nullptr, st);
}

extern "C" int eps_vjp(epsgrad_plan_t *P, const float *C, float beta, int n_pairs,
                       const void *const *EF, const void *const *EA, float *dFdC, void *stream)
{
    int rc = check_common(P, C, beta);
    if (!rc) rc = check_pairs(n_pairs, EF, EA);
    if (rc) return rc;
    if (!aligned16(dFdC)) return EPSGRAD_EINVAL;
    DeviceGuard g(P->device);
    cudaStream_t st = (cudaStream_t)stream;
    begin_call(P, st);
    return run_chain(P, C, beta, n_pairs, EF, EA, nullptr, dFdC, st);
}

extern "C" int eps_vjp_beta(epsgrad_plan_t *P, const float *C, float beta, int n_pairs,
                            const void *const *EF, const void *const *EA, float *dFdC, float *dFdbeta, void *stream)
{
    int rc = check_common(P, C, beta);
    if (!rc) rc = check_pairs(n_pairs, EF, EA);
    if (rc) return rc;
    if (!aligned16(dFdC) || !dFdbeta) return EPSGRAD_EINVAL;
    DeviceGuard g(P->device);
    cudaStream_t st = (cudaStream_t)stream;
    begin_call(P, st);
    P->cur_dbeta = dFdbeta;
    rc = run_chain(P, C, beta, n_pairs, EF, EA, nullptr, dFdC, st);
    P->cur_dbeta = nullptr;
    return rc;
}

extern "C" int eps_unbinarity(epsgrad_plan_t *P, const float *C, float beta, float *u, void *stream)
{
    int rc = check_common(P, C, beta);
    if (rc) return rc;
    if (!u) return EPSGRAD_EINVAL;
    DeviceGuard g(P->device);
    cudaStream_t st = (cudaStream_t)stream;
    begin_call(P, st);
    rc = launch_front(P, C, beta, st);
    if (rc) return rc;
    const size_t n_mask = (size_t)P->px * P->py;
    const bool morph = P->morph_R > 0;
    k_unbinarity<<<dim3(P->n_part_ub, P->cfg.batch), UB_THREADS, 0, st>>>(morph ? ws_mc(P) : ws_phi(P), n_mask, beta,
                                                                         morph ? 0.0f : P->eta_r, ws_part(P));
    rc = check_launch(P, "unbinarity", st);
    if (rc) return rc;
    k_sum_partials<<<P->cfg.batch, 256, 0, st>>>(ws_part(P), P->n_part_ub, nullptr, 0, (float)(1.0 / (double)n_mask), u);
    return check_launch(P, "unbinarity_sum", st);
}

extern "C" int eps_forward_vjp(epsgrad_plan_t *P, const float *C, float beta, int n_pairs,
                               const void *const *EF, const void *const *EA,
                               float *eps, float *dFdC, void *stream)
{
    int rc = check_common(P, C, beta);
    if (!rc) rc = check_pairs(n_pairs, EF, EA);
    if (rc) return rc;
    if (!aligned16(eps) || !aligned16(dFdC)) return EPSGRAD_EINVAL;
    DeviceGuard g(P->device);
    cudaStream_t st = (cudaStream_t)stream;
    begin_call(P, st);
    return run_chain(P, C, beta, n_pairs, EF, EA, eps, dFdC, st);
}

// ------------------------------------------------------------------------------------ stage taps
extern "C" int epsgrad_stage_filter(epsgrad_plan_t *P, const float *C, float *phi_centred, void *stream)
{
    int rc = check_common(P, C, 1.0f);
    if (rc) return rc;
    if (!aligned16(phi_centred)) return EPSGRAD_EINVAL;
    DeviceGuard g(P->device);
    begin_call(P, (cudaStream_t)stream);
    return launch_filter(P, C, phi_centred, (cudaStream_t)stream);
}

extern "C" int epsgrad_stage_eps2d(epsgrad_plan_t *P, const float *C, float beta, float *eps2d, void *stream)
{
    int rc = check_common(P, C, beta);
    if (rc) return rc;
    if (!aligned16(eps2d)) return EPSGRAD_EINVAL;
    DeviceGuard g(P->device);
    cudaStream_t st = (cudaStream_t)stream;
    begin_call(P, st);
    rc = launch_front(P, C, beta, st);
    if (!rc) rc = launch_fwd2d(P, ws_phi(P), beta, nullptr, nullptr, eps2d, st);
    return rc;
}

extern "C" int epsgrad_stage_zreduce(epsgrad_plan_t *P, int n_pairs, const void *const *EF,
                                     const void *const *EA, float *gbar, void *stream)
{
    if (!P) return EPSGRAD_EINVAL;
    int rc = check_pairs(n_pairs, EF, EA);
    if (rc) return rc;
    if (!aligned16(gbar)) return EPSGRAD_EINVAL;
    DeviceGuard g(P->device);
    begin_call(P, (cudaStream_t)stream);
    return launch_zreduce(P, n_pairs, EF, EA, gbar, (cudaStream_t)stream);
}
