// epsgrad.cu -- C ABI (include/epsgrad.h), plan / table construction and kernel launches.
// Product code for sm_100a; shares nothing with oracle/.
#include "../../include/epsgrad.h"

#include <cmath>
#include <dlfcn.h>
#include <mutex>
#include <cusolverDn.h>   // types and prototypes only: the library is loaded on first use (dlopen), never linked
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "common.cuh"
#include "filter.cuh"
#include "filter4.cuh"
#include "filter_sep.cuh"
#include "fwd2d.cuh"
#include "extrude.cuh"
#include "extrude_bulk.cuh"
#include "zreduce.cuh"
#include "zreduce_pipe.cuh"
#include "maskgrad.cuh"
#include "mega.cuh"
#include "morph.cuh"
#include "reduce.cuh"
#include "soap.cuh"

using namespace epsgrad;

#define EPSGRAD_VERSION 100   /* 0.1.0 */
#define EPSGRAD_MAX_KERNELS 24

struct epsgrad_plan {
    epsgrad_config_t cfg;
    int device, n_sm;
    int nx, ny, px, py, m;
    int T, NT, KX, KY;
    int separable;
    // device tables (one allocation)
    void *d_tables;
    float *d_w;                // conic [NT][NT][m][m] | separable [NT][m]
    int *d_tyrange;            // conic [NT][2]
    float *d_invden;           // conic [KX*m][KY*m] | separable [KX*m] + [KY*m]
    float *d_zw;               // [7][nz]: wxy, wz, z-full / lower-face / upper-face indicators, eps_clad(1-wxy), eps_clad[wz=0]
    // z windows (chunks of 2 cells) for {x,y} and {z}; face weights
    int ch0[2], nch[2];
    float w_lo, w_hi;
    // morphological filters (Eqs. (4)-(5)): disk radius in mask pixels (0 = off), alpha, device tables
    int morph_R;
    float morph_alpha;
    int *d_hl;                 // [2R+1] half-lengths of the disk rows
    float *d_invn;             // [(2R+1)^2] 1/N by border class
    size_t off_m[4], off_mc, off_cot;
    // beta-related outputs (NEXT-2): per-CTA partial sums, the d F/d beta output of the call in flight
    size_t off_part; int n_part_mg, n_part_mo, n_part_ub;
    float *cur_dbeta;
    // embedding of the design region in the caller's simulation-domain arrays (epsgrad_plan_set_embedding); emb.nx_full = 0: none
    epsgrad_embedding_t emb;
    int use_tma;               // field windows by TMA bulk tensor copies where possible (epsgrad_plan_set_tma): 1 single-stage, 2 pipelined
    int use_bulk;              // eps columns written by bulk copies from shared memory (epsgrad_plan_set_bulk_stores)
    int tune[8];               // measurement knobs (epsgrad_plan_set_tuning)
    int use_mega;              // the whole step as one persistent dataflow kernel where the configuration allows (epsgrad_plan_set_fused)
    int *d_sched;              // its ticket and per-band completion counters
    unsigned long long *d_mprof;   // optional cycle accounting of the persistent kernel (epsgrad_plan_fused_profile)
    size_t sched_bytes;
    void *tma_encode;          // cuTensorMapEncodeTiled, fetched through the runtime (no link against libcuda)
    int slab_x0, slab_nx;                   // x-slab: the caller's arrays hold Yee rows [slab_x0, slab_x0 + slab_nx) only; 0, 0 = off
    int dense, host_direct, cur_host_src;   // cur_host_src: the fields of the call in flight are pinned host memory
    // scalars
    float eta0, eta_r, eps_clad, deps, delta;
    // caller-owned buffers
    void *ws; size_t ws_bytes;
    void *stg; size_t stg_bytes;
    // workspace carve-up (byte offsets)
    size_t off_phi, off_v, off_gbar, off_e2d, off_coef, off_tmp, ws_need;
    int last_launches;
    uint64_t last_h2d, last_d2h;
    // optional per-kernel timing (epsgrad_plan_set_profiling)
    int prof;
    cudaEvent_t ev[EPSGRAD_MAX_KERNELS + 1];
    // two-stream schedule: the field stream (zreduce) runs beside filter -> fwd2d, the 2-D reverse chain beside the eps stores
    int overlap;
    cudaStream_t aux;
    cudaEvent_t ev_fork, ev_r, ev_2d, ev_join;
    const char *kname[EPSGRAD_MAX_KERNELS];
    // optional device-clock stamps between the kernels of both streams (epsgrad_plan_set_timeline)
    unsigned long long *d_tl;
    int n_tl;
    const char *tlname[2 * EPSGRAD_MAX_KERNELS];
};

struct DeviceGuardC {
    int prev;
    explicit DeviceGuardC(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuardC() { if (prev >= 0) cudaSetDevice(prev); }
};

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

static double basis(const epsgrad_config_t &c, double dx, double dy)
{
    if (c.filter_kind == EPSGRAD_FILTER_CONIC) {                   // S1: max(0, 1 - r/R)
        const double w = 1.0 - std::sqrt(dx * dx + dy * dy) / c.filter_radius;
        return w > 0.0 ? w : 0.0;
    }
    if (std::fabs(dx) > c.filter_radius || std::fabs(dy) > c.filter_radius) return 0.0;   // S11
    return std::exp(-(dx * dx + dy * dy) / (2.0 * c.filter_sigma * c.filter_sigma));
}

static double basis1(const epsgrad_config_t &c, double d)       // separable factor (Gaussian only)
{
    if (std::fabs(d) > c.filter_radius) return 0.0;
    return std::exp(-d * d / (2.0 * c.filter_sigma * c.filter_sigma));
}

// representative control index of border class k (inverse of border_class)
static int class_rep(int k, int M, int T, int K)
{
    if (K == M) return k;
    return k <= T ? k : M - 1 - (2 * T - k);
}

static double overlap(double a0, double a1, double b0, double b1)
{
    const double lo = a0 > b0 ? a0 : b0, hi = a1 < b1 ? a1 : b1;
    return hi > lo ? hi - lo : 0.0;
}

static int validate(const epsgrad_config_t *c)
{
    if (!c) return EPSGRAD_EINVAL;
    if (c->batch < 1 || c->mx < 1 || c->my < 1 || c->upsample < 1 || c->nz < 1) return EPSGRAD_EINVAL;
    if (c->subpixel < 2 || (c->subpixel & 1)) return EPSGRAD_EINVAL;
    if (!(c->z_hi > c->z_lo)) return EPSGRAD_EINVAL;
    if (!(c->filter_radius > 0.0)) return EPSGRAD_EINVAL;
    if (c->filter_kind != EPSGRAD_FILTER_CONIC && c->filter_kind != EPSGRAD_FILTER_GAUSSIAN) return EPSGRAD_EINVAL;
    if (c->filter_kind == EPSGRAD_FILTER_GAUSSIAN && !(c->filter_sigma > 0.0)) return EPSGRAD_EINVAL;
    if (!(c->eps_core > 0.0) || !(c->eps_clad > 0.0) || c->eps_core == c->eps_clad) return EPSGRAD_EINVAL;
    if (!(c->normal_delta >= 1e-30) || !std::isfinite(c->normal_delta)) return EPSGRAD_EINVAL;   // 0 / denormal: n^2 = 0/0 on flat cells
    if (!std::isfinite(c->eta) || !std::isfinite(c->z_lo) || !std::isfinite(c->z_hi)) return EPSGRAD_EINVAL;
    if (!(c->morph_diameter >= 0.0)) return EPSGRAD_EINVAL;
    if (c->morph_diameter > 0.0) {
        if (!(c->morph_alpha > 0.0)) return EPSGRAD_EINVAL;
        const int R = (int)std::floor(0.5 * c->morph_diameter * c->subpixel);
        if (R > MO_MAX_R) return EPSGRAD_EUNSUPPORTED;
        if (c->subpixel * c->upsample * c->mx < 2 * R + 1 || c->subpixel * c->upsample * c->my < 2 * R + 1) return EPSGRAD_EUNSUPPORTED;
    }
    const int m = c->upsample * c->subpixel;
    if (m != 2 && m != 4 && m != 6 && m != 8) return EPSGRAD_EUNSUPPORTED;
    if (c->nz % 4) return EPSGRAD_EUNSUPPORTED;
    const double cells = (double)c->batch * 3.0 * c->upsample * c->mx * c->upsample * c->my;
    if (cells * c->subpixel * c->subpixel > 2.0e9) return EPSGRAD_EUNSUPPORTED;   // 32-bit plane indices
    return EPSGRAD_OK;
}

// ------------------------------------------------------------------------------------ plan
extern "C" int epsgrad_plan_create(const epsgrad_config_t *cfg, int device, epsgrad_plan_t **out)
{
    if (!out) return EPSGRAD_EINVAL;
    int rc = validate(cfg);
    if (rc) return rc;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return EPSGRAD_ECUDA;
    }
    epsgrad_plan *P = new (std::nothrow) epsgrad_plan();
    if (!P) return EPSGRAD_ENOMEM;
    std::memset(P, 0, sizeof(*P));
    P->cfg = *cfg;
    P->device = device;
    if (cudaDeviceGetAttribute(&P->n_sm, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || P->n_sm < 1) { cudaGetLastError(); P->n_sm = 148; }
    const int u = cfg->upsample, s = cfg->subpixel, m = u * s;
    P->m = m;
    P->nx = u * cfg->mx; P->ny = u * cfg->my;
    P->px = s * P->nx;   P->py = s * P->ny;
    P->separable = cfg->filter_kind == EPSGRAD_FILTER_GAUSSIAN;
    // taps: X_p - x_a = delta_f - u t, |delta_f| < u/2  =>  |t| <= floor((R + u/2)/u)
    const int T = (int)std::floor((cfg->filter_radius + 0.5 * u) / u);
    const int NT = 2 * T + 1;
    P->T = T; P->NT = NT;
    P->KX = cfg->mx >= NT ? NT : cfg->mx;
    P->KY = cfg->my >= NT ? NT : cfg->my;
    P->eta0 = cfg->filter_normalize ? (float)cfg->eta : 0.0f;
    P->eta_r = (float)(cfg->eta - (double)P->eta0);
    P->eps_clad = (float)cfg->eps_clad;
    P->deps = (float)(cfg->eps_core - cfg->eps_clad);
    P->delta = (float)cfg->normal_delta;

    // ---- filter tables (float64 on the host, rounded once to fp32)
    std::vector<double> d1(m);                       // delta_f = (f + 1/2)/s - u/2
    for (int f = 0; f < m; ++f) d1[f] = (f + 0.5) / s - 0.5 * u;
    std::vector<float> w;
    std::vector<int> tyr(2 * NT, 0);
    std::vector<float> invden;
    bool uncovered = false;                          // a mask pixel out of reach of every control pixel: den = 0 in Eq. (2)/S2
    if (!P->separable) {
        w.assign((size_t)NT * NT * m * m, 0.0f);
        for (int tx = 0; tx < NT; ++tx) {
            int lo = NT, hi = -1;
            for (int ty = 0; ty < NT; ++ty) {
                bool any = false;
                for (int fx = 0; fx < m; ++fx)
                    for (int fy = 0; fy < m; ++fy) {
                        const double v = basis(*cfg, d1[fx] - (double)u * (tx - T), d1[fy] - (double)u * (ty - T));
                        w[(((size_t)tx * NT + ty) * m + fx) * m + fy] = (float)v;
                        any |= v != 0.0;
                    }
                if (any) { if (ty < lo) lo = ty; hi = ty; }
            }
            tyr[2 * tx] = lo; tyr[2 * tx + 1] = hi;   // empty row: lo > hi
        }
        const int RX = P->KX * m, RY = P->KY * m;
        invden.assign((size_t)RX * RY, 1.0f);
        if (cfg->filter_normalize)
            for (int kx = 0; kx < P->KX; ++kx)
                for (int ky = 0; ky < P->KY; ++ky) {
                    const int a0 = class_rep(kx, cfg->mx, T, P->KX), b0 = class_rep(ky, cfg->my, T, P->KY);
                    for (int fx = 0; fx < m; ++fx)
                        for (int fy = 0; fy < m; ++fy) {
                            double den = 0.0;
                            for (int tx = 0; tx < NT; ++tx) {
                                const int a = a0 + tx - T;
                                if (a < 0 || a >= cfg->mx) continue;
                                for (int ty = 0; ty < NT; ++ty) {
                                    const int b = b0 + ty - T;
                                    if (b < 0 || b >= cfg->my) continue;
                                    den += (double)w[(((size_t)tx * NT + ty) * m + fx) * m + fy];
                                }
                            }
                            if (!(den > 0.0)) uncovered = true;
                            invden[(size_t)(kx * m + fx) * RY + ky * m + fy] = (float)(1.0 / den);
                        }
                }
    } else {
        w.assign((size_t)NT * m, 0.0f);
        for (int t = 0; t < NT; ++t)
            for (int f = 0; f < m; ++f) w[(size_t)t * m + f] = (float)basis1(*cfg, d1[f] - (double)u * (t - T));
        const int RX = P->KX * m, RY = P->KY * m;
        invden.assign((size_t)RX + RY, 1.0f);
        if (cfg->filter_normalize)
            for (int ax = 0; ax < 2; ++ax) {
                const int K = ax ? P->KY : P->KX, M = ax ? cfg->my : cfg->mx;
                for (int k = 0; k < K; ++k) {
                    const int a0 = class_rep(k, M, T, K);
                    for (int f = 0; f < m; ++f) {
                        double den = 0.0;
                        for (int t = 0; t < NT; ++t) {
                            const int a = a0 + t - T;
                            if (a >= 0 && a < M) den += (double)w[(size_t)t * m + f];
                        }
                        if (!(den > 0.0)) uncovered = true;
                        invden[(ax ? RX : 0) + k * m + f] = (float)(1.0 / den);
                    }
                }
            }
    }

    if (uncovered) { delete P; return EPSGRAD_EINVAL; }    // the density filter would divide 0 by 0 there (R < u/sqrt(2))

    // ---- z tables (S7, S8): wxy_k = |[k,k+1] ^ slab|, wz_k = |[k+1/2,k+3/2] ^ slab|
    const int nz = cfg->nz;
    std::vector<float> zw((size_t)7 * nz, 0.0f);
    int kmin[2] = {nz, nz}, kmax[2] = {-1, -1};
    int n_face = 0;
    for (int k = 0; k < nz; ++k) {
        const double wxy = overlap(k, k + 1.0, cfg->z_lo, cfg->z_hi);
        const double wz = overlap(k + 0.5, k + 1.5, cfg->z_lo, cfg->z_hi);
        zw[k] = (float)wxy;
        zw[nz + k] = (float)wz;
        zw[5 * nz + k] = (float)(cfg->eps_clad * (1.0 - wxy));
        zw[6 * nz + k] = wz > 0.0 ? 0.0f : (float)cfg->eps_clad;
        if (wxy > 0.0) { if (k < kmin[0]) kmin[0] = k; kmax[0] = k; }
        if (wz > 0.0) {
            if (k < kmin[1]) kmin[1] = k;
            kmax[1] = k;
            if ((float)wz == 1.0f) zw[2 * nz + k] = 1.0f;
            else if (n_face == 0) { zw[3 * nz + k] = 1.0f; P->w_lo = (float)wz; ++n_face; }
            else if (n_face == 1) { zw[4 * nz + k] = 1.0f; P->w_hi = (float)wz; ++n_face; }
            else { delete P; return EPSGRAD_EINVAL; }   // cannot happen for an interval slab
        }
    }
    for (int g = 0; g < 2; ++g) {
        if (kmax[g] < 0) { P->ch0[g] = 0; P->nch[g] = 0; }
        else { P->ch0[g] = kmin[g] / 2; P->nch[g] = kmax[g] / 2 - P->ch0[g] + 1; }
    }

    // ---- shared-memory budget of the transposed conic filter (v tile + weight table)
    if (!P->separable) {
        const int sp = m % 4 == 0 ? 4 : 2, tb = 32 / sp, ta = 8;
        const size_t need = ((size_t)NT * NT * m * m + (size_t)m * (ta + 2 * T) * m * (tb + 2 * T) + 2 * NT) * 4;
        if (need > 200 * 1024) { delete P; return EPSGRAD_EUNSUPPORTED; }
    }
    if (fwd2d_smem_floats(s) * 4 > 200 * 1024 || maskgrad_smem_floats(s) * 4 > 200 * 1024) { delete P; return EPSGRAD_EUNSUPPORTED; }

    // ---- upload
    int prev = 0;
    cudaGetDevice(&prev);
    cudaSetDevice(device);
    const size_t b_w = align_up(w.size() * 4, 256), b_ty = align_up(tyr.size() * 4, 256);
    const size_t b_id = align_up(invden.size() * 4, 256), b_zw = align_up(zw.size() * 4, 256);
    cudaError_t ce = cudaMalloc(&P->d_tables, b_w + b_ty + b_id + b_zw);
    if (ce == cudaSuccess) {
        char *base = (char *)P->d_tables;
        P->d_w = (float *)base;
        P->d_tyrange = (int *)(base + b_w);
        P->d_invden = (float *)(base + b_w + b_ty);
        P->d_zw = (float *)(base + b_w + b_ty + b_id);
        ce = cudaMemcpy(P->d_w, w.data(), w.size() * 4, cudaMemcpyHostToDevice);
        if (ce == cudaSuccess) ce = cudaMemcpy(P->d_tyrange, tyr.data(), tyr.size() * 4, cudaMemcpyHostToDevice);
        if (ce == cudaSuccess) ce = cudaMemcpy(P->d_invden, invden.data(), invden.size() * 4, cudaMemcpyHostToDevice);
        if (ce == cudaSuccess) ce = cudaMemcpy(P->d_zw, zw.data(), zw.size() * 4, cudaMemcpyHostToDevice);
    }
    cudaSetDevice(prev);
    if (ce != cudaSuccess) {
        cudaGetLastError();
        if (P->d_tables) cudaFree(P->d_tables);
        delete P;
        return EPSGRAD_ECUDA;
    }

    // ---- morphological disk: K_m = 1 for dp^2 + dq^2 <= (d s / 2)^2, unit sum over the in-region pixels (S18)
    if (cfg->morph_diameter > 0.0) {
        const double rp = 0.5 * cfg->morph_diameter * s;
        const int R = (int)std::floor(rp), NI = 2 * R + 1;
        P->morph_R = R;
        P->morph_alpha = (float)cfg->morph_alpha;
        std::vector<int> hl(NI);
        for (int dp = -R; dp <= R; ++dp) hl[dp + R] = (int)std::floor(std::sqrt(rp * rp - (double)dp * dp) + 1e-9);
        std::vector<float> invn((size_t)NI * NI);
        for (int cp = 0; cp < NI; ++cp)
            for (int cq = 0; cq < NI; ++cq) {
                // class c < R: c pixels from the low edge; c > R: 2R - c pixels from the high edge; R: interior
                const int lo_p = cp < R ? cp : R, hi_p = cp > R ? 2 * R - cp : R;
                const int lo_q = cq < R ? cq : R, hi_q = cq > R ? 2 * R - cq : R;
                int n = 0;
                for (int dp = -lo_p; dp <= hi_p; ++dp)
                    for (int dq = -lo_q; dq <= hi_q; ++dq)
                        if ((double)(dp * dp + dq * dq) <= rp * rp) ++n;
                invn[(size_t)cp * NI + cq] = (float)(1.0 / n);
            }
        int prevd = 0;
        cudaGetDevice(&prevd);
        cudaSetDevice(device);
        bool okm = cudaMalloc(&P->d_hl, NI * sizeof(int)) == cudaSuccess &&
                   cudaMalloc(&P->d_invn, invn.size() * sizeof(float)) == cudaSuccess &&
                   cudaMemcpy(P->d_hl, hl.data(), NI * sizeof(int), cudaMemcpyHostToDevice) == cudaSuccess &&
                   cudaMemcpy(P->d_invn, invn.data(), invn.size() * sizeof(float), cudaMemcpyHostToDevice) == cudaSuccess;
        cudaSetDevice(prevd);
        if (!okm) { cudaGetLastError(); epsgrad_plan_destroy(P); return EPSGRAD_ECUDA; }
    }

    // ---- auxiliary stream and fork/join events (no timing) for the two-stream schedule
    {
        int prev2 = 0;
        cudaGetDevice(&prev2);
        cudaSetDevice(device);
        // highest priority: the small kernels it carries must get SM slots ahead of the pending CTAs of the HBM-bound kernels
        int prio_least = 0, prio_greatest = 0;
        cudaDeviceGetStreamPriorityRange(&prio_least, &prio_greatest);
        bool ok = cudaStreamCreateWithPriority(&P->aux, cudaStreamNonBlocking, prio_greatest) == cudaSuccess &&
                  cudaEventCreateWithFlags(&P->ev_fork, cudaEventDisableTiming) == cudaSuccess &&
                  cudaEventCreateWithFlags(&P->ev_r, cudaEventDisableTiming) == cudaSuccess &&
                  cudaEventCreateWithFlags(&P->ev_2d, cudaEventDisableTiming) == cudaSuccess &&
                  cudaEventCreateWithFlags(&P->ev_join, cudaEventDisableTiming) == cudaSuccess;
        cudaSetDevice(prev2);
        if (!ok) { cudaGetLastError(); epsgrad_plan_destroy(P); return EPSGRAD_ECUDA; }
        P->overlap = 1;
        P->host_direct = 2;
        {
            cudaDriverEntryPointQueryResult qres;
            void *fn = nullptr;
            if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess) { cudaGetLastError(); fn = nullptr; }
            P->tma_encode = fn;
            P->use_tma = 0;              // measured: 39 us against 37 us for the LDGSTS kernel at paper scale
        }
    }

    // ---- workspace carve-up
    const size_t n_mask = (size_t)cfg->batch * P->px * P->py, n_cell = (size_t)cfg->batch * P->nx * P->ny;
    size_t off = 0;
    P->off_phi = off;  off += align_up(n_mask * 4, 256);
    P->off_v = off;    off += align_up(n_mask * 4, 256);
    P->off_gbar = off; off += align_up(n_cell * 5 * 4, 256);
    P->off_e2d = off;  off += align_up(n_cell * F2_NE2D * 4, 256);
    P->off_coef = off; off += align_up(n_cell * F2_NCOEF * 4, 256);
    if (P->morph_R > 0) {
        for (int k = 0; k < 4; ++k) { P->off_m[k] = off; off += align_up(n_mask * 4, 256); }
        P->off_mc = off;  off += align_up(n_mask * 4, 256);
        P->off_cot = off; off += align_up(n_mask * 4, 256);
    }
    P->n_part_mg = ((P->ny + MG_TJ - 1) / MG_TJ) * ((P->nx + MG_TI - 1) / MG_TI);
    P->n_part_mo = P->morph_R > 0 ? ((P->py + MO_T - 1) / MO_T) * ((P->px + MO_T - 1) / MO_T) : 0;
    P->n_part_ub = (int)(((size_t)P->px * P->py + UB_THREADS * UB_PER_THREAD - 1) / (UB_THREADS * UB_PER_THREAD));
    {
        const size_t a = (size_t)P->n_part_mg + P->n_part_mo, b = (size_t)P->n_part_ub;
        P->off_part = off; off += align_up((size_t)cfg->batch * (a > b ? a : b) * 4, 256);
    }
    P->off_tmp = off;  off += P->separable ? align_up((size_t)cfg->batch * cfg->mx * P->py * 4, 256) : 0;
    P->ws_need = off;
    // ---- persistent dataflow kernel (mega.cuh): conic fast path with 4 mask pixels per control pixel, s = 2, no morphological filters
    if (!P->separable && m == 4 && s == 2 && (NT == 5 || NT == 9 || NT == 13) && P->morph_R == 0) {
        const int nb = (P->nx + MK_BAND - 1) / MK_BAND;
        P->sched_bytes = ((size_t)MK_SCHED_HEAD + (size_t)PH_N * cfg->batch * nb) * sizeof(int);
        int prev3 = 0;
        cudaGetDevice(&prev3);
        cudaSetDevice(device);
        const bool oks = cudaMalloc(&P->d_sched, P->sched_bytes) == cudaSuccess;
        cudaSetDevice(prev3);
        if (!oks) { cudaGetLastError(); P->d_sched = nullptr; epsgrad_plan_destroy(P); return EPSGRAD_ECUDA; }
        P->use_mega = 0;         // measured slower than the separate kernels on every config: an option, off by default
    }
    *out = P;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_destroy(epsgrad_plan_t *P)
{
    if (!P) return EPSGRAD_EINVAL;
    if (P->d_tables) cudaFree(P->d_tables);
    if (P->d_tl) cudaFree(P->d_tl);
    if (P->d_hl) cudaFree(P->d_hl);
    if (P->d_invn) cudaFree(P->d_invn);
    if (P->d_sched) cudaFree(P->d_sched);
    if (P->d_mprof) cudaFree(P->d_mprof);
    if (P->aux) cudaStreamDestroy(P->aux);
    if (P->ev_fork) cudaEventDestroy(P->ev_fork);
    if (P->ev_r) cudaEventDestroy(P->ev_r);
    if (P->ev_2d) cudaEventDestroy(P->ev_2d);
    if (P->ev_join) cudaEventDestroy(P->ev_join);
    if (P->ev[0])
        for (int i = 0; i <= EPSGRAD_MAX_KERNELS; ++i) cudaEventDestroy(P->ev[i]);
    delete P;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_profiling(epsgrad_plan_t *P, int enable)
{
    if (!P) return EPSGRAD_EINVAL;
    if (enable && !P->ev[0]) {
        int prev = 0;
        cudaGetDevice(&prev);
        cudaSetDevice(P->device);
        bool ok = true;
        for (int i = 0; i <= EPSGRAD_MAX_KERNELS && ok; ++i) ok = cudaEventCreate(&P->ev[i]) == cudaSuccess;
        cudaSetDevice(prev);
        if (!ok) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    }
    P->prof = enable != 0;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_last_kernel_times(epsgrad_plan_t *P, int max_n, float *ms, const char **names)
{
    if (!P || max_n < 0 || (max_n > 0 && (!ms || !names))) return EPSGRAD_EINVAL;
    int n = P->last_launches < EPSGRAD_MAX_KERNELS ? P->last_launches : EPSGRAD_MAX_KERNELS;
    if (n > max_n) n = max_n;
    for (int i = 0; i < n; ++i) {
        names[i] = P->kname[i];
        ms[i] = -1.0f;
        if (P->prof) {
            if (cudaEventSynchronize(P->ev[i + 1]) != cudaSuccess ||
                cudaEventElapsedTime(&ms[i], P->ev[i], P->ev[i + 1]) != cudaSuccess) {
                cudaGetLastError();
                return EPSGRAD_ECUDA;
            }
        }
    }
    return n;
}

extern "C" size_t epsgrad_workspace_bytes(const epsgrad_plan_t *P) { return P ? P->ws_need : 0; }

extern "C" int epsgrad_plan_set_workspace(epsgrad_plan_t *P, void *p, size_t bytes)
{
    if (!P || !p || ((uintptr_t)p & 255)) return EPSGRAD_EINVAL;
    if (bytes < P->ws_need) return EPSGRAD_ENOWORKSPACE;
    P->ws = p; P->ws_bytes = bytes;
    return EPSGRAD_OK;
}

static size_t n_eps(const epsgrad_plan_t *P) { return (size_t)P->cfg.batch * 3 * P->nx * P->ny * P->cfg.nz; }
static size_t n_ctrl(const epsgrad_plan_t *P) { return (size_t)P->cfg.batch * P->cfg.mx * P->cfg.my; }

extern "C" size_t epsgrad_staging_bytes(const epsgrad_plan_t *P, int n_pairs)
{
    if (!P || n_pairs < 0) return 0;
    return 2 * align_up(n_ctrl(P) * 4, 256) + align_up(n_eps(P) * 4, 256) + (size_t)2 * n_pairs * align_up(n_eps(P) * 8, 256);
}

extern "C" int epsgrad_plan_set_staging(epsgrad_plan_t *P, void *p, size_t bytes)
{
    if (!P || !p || ((uintptr_t)p & 255)) return EPSGRAD_EINVAL;
    P->stg = p; P->stg_bytes = bytes;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_dense_reads(epsgrad_plan_t *P, int dense)
{
    if (!P) return EPSGRAD_EINVAL;
    P->dense = dense != 0;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_embedding(epsgrad_plan_t *P, const epsgrad_embedding_t *e)
{
    if (!P) return EPSGRAD_EINVAL;
    if (!e) { std::memset(&P->emb, 0, sizeof(P->emb)); return EPSGRAD_OK; }
    if (e->nx_full < 1 || e->ny_full < 1 || e->nz_full < 1 || e->i0 < 0 || e->j0 < 0 || e->k0 < 0) return EPSGRAD_EINVAL;
    if (e->i0 + P->nx > e->nx_full || e->j0 + P->ny > e->ny_full || e->k0 + P->cfg.nz > e->nz_full) return EPSGRAD_EINVAL;
    if (e->nz_full % 4 || e->k0 % 4) return EPSGRAD_EUNSUPPORTED;          // 16-byte pieces of eps (4 cells) and of the fields (2 cells)
    if ((double)P->cfg.batch * 3.0 * e->nx_full * e->ny_full > 2.0e9) return EPSGRAD_EUNSUPPORTED;
    if (P->slab_nx > 0) return EPSGRAD_EUNSUPPORTED;                        // one addressing option at a time
    P->emb = *e;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_tma(epsgrad_plan_t *P, int enable)
{
    if (!P) return EPSGRAD_EINVAL;
    if (enable && !P->tma_encode) return EPSGRAD_EUNSUPPORTED;
    P->use_tma = enable < 0 ? 0 : (enable > 2 ? 2 : enable);
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_bulk_stores(epsgrad_plan_t *P, int enable)
{
    if (!P) return EPSGRAD_EINVAL;
    P->use_bulk = enable != 0;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_fused(epsgrad_plan_t *P, int enable)
{
    if (!P) return EPSGRAD_EINVAL;
    if (enable && !P->d_sched) return EPSGRAD_EUNSUPPORTED;
    P->use_mega = enable < 0 ? 0 : (enable > 2 ? 2 : enable);
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_fused_profile(epsgrad_plan_t *P, int enable, uint64_t *out20)
{
    if (!P) return EPSGRAD_EINVAL;
    DeviceGuardC g(P->device);
    const size_t bytes = (2 * PH_N + 8) * sizeof(unsigned long long);
    if (out20 && P->d_mprof) {
        if (cudaDeviceSynchronize() != cudaSuccess || cudaMemcpy(out20, P->d_mprof, bytes, cudaMemcpyDeviceToHost) != cudaSuccess) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    }
    if (enable && !P->d_mprof) {
        if (cudaMalloc(&P->d_mprof, bytes) != cudaSuccess) { cudaGetLastError(); P->d_mprof = nullptr; return EPSGRAD_ECUDA; }
    }
    if (P->d_mprof) cudaMemset(P->d_mprof, 0, bytes);
    if (!enable && P->d_mprof) { cudaFree(P->d_mprof); P->d_mprof = nullptr; }
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_tuning(epsgrad_plan_t *P, int knob, int value)
{
    if (!P || knob < 0 || knob >= 8) return EPSGRAD_EINVAL;
    P->tune[knob] = value;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_slab(epsgrad_plan_t *P, int x_first, int x_count)
{
    if (!P) return EPSGRAD_EINVAL;
    if (x_first == 0 && x_count == 0) { P->slab_x0 = P->slab_nx = 0; return EPSGRAD_OK; }
    if (x_first < 0 || x_count < 1 || x_first + x_count > P->nx) return EPSGRAD_EINVAL;
    if (P->emb.nx_full > 0) return EPSGRAD_EUNSUPPORTED;         // one addressing option at a time
    P->slab_x0 = x_first; P->slab_nx = x_count;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_host_direct(epsgrad_plan_t *P, int enable)
{
    if (!P) return EPSGRAD_EINVAL;
    P->host_direct = enable < 0 ? 0 : (enable > 2 ? 2 : enable);
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_overlap(epsgrad_plan_t *P, int enable)
{
    if (!P) return EPSGRAD_EINVAL;
    P->overlap = enable != 0;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_timeline(epsgrad_plan_t *P, int enable)
{
    if (!P) return EPSGRAD_EINVAL;
    if (enable && !P->d_tl) {
        DeviceGuardC g(P->device);
        if (cudaMalloc(&P->d_tl, 2 * EPSGRAD_MAX_KERNELS * sizeof(unsigned long long)) != cudaSuccess) { cudaGetLastError(); P->d_tl = nullptr; return EPSGRAD_ECUDA; }
    } else if (!enable && P->d_tl) {
        cudaFree(P->d_tl);
        P->d_tl = nullptr;
    }
    P->n_tl = 0;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_read_timeline(epsgrad_plan_t *P, int max_n, uint64_t *ns, const char **names)
{
    if (!P || max_n < 0 || (max_n > 0 && (!ns || !names))) return EPSGRAD_EINVAL;
    if (!P->d_tl) return 0;
    const int n = P->n_tl < max_n ? P->n_tl : max_n;
    DeviceGuardC g(P->device);
    if (cudaDeviceSynchronize() != cudaSuccess ||
        cudaMemcpy(ns, P->d_tl, n * sizeof(unsigned long long), cudaMemcpyDeviceToHost) != cudaSuccess) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    for (int i = 0; i < n; ++i) names[i] = P->tlname[i];
    return n;
}

extern "C" int epsgrad_plan_last_launches(const epsgrad_plan_t *P) { return P ? P->last_launches : 0; }

extern "C" int epsgrad_plan_last_copy_bytes(const epsgrad_plan_t *P, uint64_t *h2d, uint64_t *d2h)
{
    if (!P) return EPSGRAD_EINVAL;
    if (h2d) *h2d = P->last_h2d;
    if (d2h) *d2h = P->last_d2h;
    return EPSGRAD_OK;
}

extern "C" const char *epsgrad_status_string(int st)
{
    switch (st) {
    case EPSGRAD_OK: return "ok";
    case EPSGRAD_EINVAL: return "invalid argument";
    case EPSGRAD_EUNSUPPORTED: return "unsupported configuration";
    case EPSGRAD_ENOWORKSPACE: return "workspace or staging buffer missing or too small";
    case EPSGRAD_ECUDA: return "CUDA runtime error";
    case EPSGRAD_ENOMEM: return "host allocation failed";
    default: return "unknown status";
    }
}

extern "C" int epsgrad_version(void) { return EPSGRAD_VERSION; }

// ------------------------------------------------------------------------------------ launches
namespace {

inline int cdiv(int a, int b) { return (a + b - 1) / b; }

template <typename K>
int set_smem(K kernel, size_t bytes)
{
    if (bytes > 48 * 1024 &&
        cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess) {
        cudaGetLastError();
        return EPSGRAD_ECUDA;
    }
    return EPSGRAD_OK;
}

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
    if (P->prof) cudaEventRecord(P->ev[0], st);
}

int check_launch(epsgrad_plan *P, const char *name, cudaStream_t st)
{
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
    return n;
}

float *ws_phi(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_phi); }
float *ws_v(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_v); }
float *ws_m(const epsgrad_plan *P, int k) { return (float *)((char *)P->ws + P->off_m[k]); }
float *ws_mc(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_mc); }
float *ws_cot(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_cot); }
float *ws_part(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_part); }
float *ws_gbar(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_gbar); }
float *ws_e2d(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_e2d); }
float *ws_coef(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_coef); }
float *ws_tmp(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_tmp); }

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
        if (M == 4 && (NT == 5 || NT == 9 || NT == 13)) {      // fast path (filter4.cuh)
            auto kern = NT == 5 ? k_filter_conic4<5> : (NT == 9 ? k_filter_conic4<9> : k_filter_conic4<13>);
            const size_t smem4 = (filter4_smem_floats(NT) + 4) * 4;
            int rc4 = set_smem(kern, smem4);
            if (rc4) return rc4;
            kern<<<dim3(cdiv(my, F4_TB), cdiv(mx, F4_TA), B), F4F_THREADS, smem4, st>>>(fp);
            return check_launch(P, "filter", st);
        }
        const size_t smem = ((size_t)NT * NT * M * M + (size_t)(TA + 2 * T) * (TB + 2 * T + 1) + 2 * NT) * 4;
        if (smem > 200 * 1024) return EPSGRAD_EUNSUPPORTED;
        int rc = set_smem(k_filter_conic<M, TA, TB>, smem);
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
        int rc = set_smem(k_sep_up_y<M>, smem);
        if (rc) return rc;
        k_sep_up_y<M><<<dim3(cdiv(my, 32), cdiv(mx, 8), B), SEP_THREADS, smem, st>>>(sp);
        if ((rc = check_launch(P, "filter_up_y", st))) return rc;
    }
    {
        sp.in = ws_tmp(P); sp.out = phi;
        const size_t smem = sepx_smem_floats(NT, M) * 4;
        if (smem > 200 * 1024) return EPSGRAD_EUNSUPPORTED;
        int rc = set_smem(k_sep_up_x<M>, smem);
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
    if (M == 4 && (NT == 5 || NT == 9 || NT == 13)) {          // fast path (filter4.cuh)
        auto kern = NT == 5 ? k_filterT_conic4<5> : (NT == 9 ? k_filterT_conic4<9> : k_filterT_conic4<13>);
        const size_t smem4 = filterT4_smem_floats(NT) * 4;
        int rc4 = set_smem(kern, smem4);
        if (rc4) return rc4;
        kern<<<dim3(cdiv(fp.my, F4_TB), cdiv(fp.mx, F4_TA), P->cfg.batch), F4T_THREADS, smem4, st>>>(fp);
        return check_launch(P, "filterT", st);
    }
    const size_t smem = ((size_t)NT * NT * M * M + (size_t)M * (S::TA + 2 * T) * M * (S::TB + 2 * T) + 2 * NT) * 4;
    if (smem > 200 * 1024) return EPSGRAD_EUNSUPPORTED;
    int rc = set_smem(k_filterT_conic<M>, smem);
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
        int rc = set_smem(k_sep_down_x<M>, smem);
        if (rc) return rc;
        k_sep_down_x<M><<<dim3(cdiv(P->py, SEPX_THREADS), cdiv(mx, SEPX_NBA), B), SEPX_THREADS, smem, st>>>(sp);
        if ((rc = check_launch(P, "filterT_down_x", st))) return rc;
    }
    {
        sp.in = ws_tmp(P); sp.out = dC;
        const size_t smem = ((size_t)NT * M + (size_t)8 * M * (32 + 2 * T)) * 4;
        if (smem > 200 * 1024) return EPSGRAD_EUNSUPPORTED;
        int rc = set_smem(k_sep_down_y<M>, smem);
        if (rc) return rc;
        k_sep_down_y<M><<<dim3(cdiv(my, 32), cdiv(mx, 8), B), SEP_THREADS, smem, st>>>(sp);
        return check_launch(P, "filterT_down_y", st);
    }
}

int launch_filter(epsgrad_plan *P, const float *C, float *phi, cudaStream_t st)
{
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
    int rc = set_smem(kern, smem);
    if (rc) return rc;
    kern<<<dim3(cdiv(P->ny, F2_TJ), cdiv(P->nx, F2_TI), P->cfg.batch), F2_THREADS, smem, st>>>(fp);
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
    const ExtrudeParams ep = fill_extrude(P, e2d, eps);
    if (P->cfg.batch > 65535) return EPSGRAD_EUNSUPPORTED;
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
            int rcb = set_smem(k_extrude_bulk, smem_b);
            if (rcb) return rcb;
            const int per_sm = P->tune[1] > 0 ? P->tune[1] : 2;
            const int n_items = 3 * bp.nblk, n_want = std::max(1, per_sm * P->n_sm / P->cfg.batch);
            k_extrude_bulk<<<dim3(std::min(n_items, n_want), 1, P->cfg.batch), EXB_THREADS, smem_b, st>>>(bp);
            return check_launch(P, "extrude", st);
        }
    }
    const size_t smem = (size_t)3 * ep.cpb * 4;
    int rc = set_smem(k_extrude, smem);
    if (rc) return rc;
    k_extrude<<<dim3(ep.nblk, 3, P->cfg.batch), EX_THREADS, smem, st>>>(ep);
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

// everything of ZredParams but the field pointers; smem: bytes of staging a CTA needs; sparse: windows worth 64-byte fills
int fill_zreduce(const epsgrad_plan *P, float *gbar, bool packed, ZredParams &zp, size_t &smem, bool &sparse, int &maxnch,
                 int max_cols = ZR_COLS, int stage_chunks = ZR_STAGE_CHUNKS)
{
    zp.gbar = gbar; zp.zw = P->d_zw; zp.ncol = P->nx * P->ny; zp.nz = P->cfg.nz;
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
                   bool host_src = false, bool packed = false)
{
    ZredParams zp;
    size_t smem = 0;
    bool sparse = false;
    int maxnch = 1;
    // x-slab: only the slab's rows have fields; the cotangent of every other column of the region is zero
    if (P->slab_nx > 0 &&
        cudaMemsetAsync(gbar, 0, (size_t)P->cfg.batch * 5 * P->nx * P->ny * sizeof(float), st) != cudaSuccess) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    int rcf = fill_zreduce(P, gbar, packed, zp, smem, sparse, maxnch);
    if (rcf) return rcf;
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
        int rcp = set_smem(k_zreduce_pipe, smem_p);
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
        int rct = set_smem(k_zreduce_tma, smem_t);
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
    int rc = set_smem(kern, smem);
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
    int rc = set_smem(k_morph, smem);
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
    int rc = set_smem(kern, smem);
    if (rc) return rc;
    kern<<<dim3(cdiv(P->ny, MG_TJ), cdiv(P->nx, MG_TI), P->cfg.batch), MG_THREADS, smem, st>>>(mp);
    return check_launch(P, "maskgrad", st);
}

bool aligned16(const void *p) { return p && !((uintptr_t)p & 15); }

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

struct DeviceGuard {
    int prev;
    explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// ---- the whole step as one persistent dataflow kernel (mega.cuh)
bool mega_applies(const epsgrad_plan *P, int n_pairs)
{
    return P->use_mega == 1 && P->d_sched && !P->cur_dbeta && P->slab_nx == 0 && !P->cur_host_src && !P->prof && n_pairs <= ZR_MAX_PAIRS;
}

template <int NTC>
int launch_mega_nt(epsgrad_plan *P, MegaParams &mp, bool sparse, size_t smem, cudaStream_t st)
{
    auto kern = sparse ? k_mega<NTC, true> : k_mega<NTC, false>;
    int rc = set_smem(kern, smem);
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
    if (cudaEventRecord(P->ev_fork, st) != cudaSuccess || cudaStreamWaitEvent(ax, P->ev_fork, 0) != cudaSuccess) {
        cudaGetLastError();
        return EPSGRAD_ECUDA;
    }
    const bool chains = P->use_mega == 2 && P->d_sched && !P->cur_dbeta && P->slab_nx == 0;   // the 2-D chains as two persistent kernels
    if (chains) rc = launch_mega(P, C, beta, n_pairs, EF, EA, eps, dFdC, ax, 1u << PH_F1 | 1u << PH_F2);
    else rc = launch_front(P, C, beta, ax);
    if (!rc) rc = launch_zreduce(P, n_pairs, EF, EA, ws_gbar(P), st);
    if (!rc && cudaEventRecord(P->ev_r, st) != cudaSuccess) rc = EPSGRAD_ECUDA;
    if (!rc && !chains) rc = launch_fwd2d(P, ws_phi(P), beta, eps ? ws_e2d(P) : nullptr, ws_coef(P), nullptr, ax);
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

}  // namespace

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

extern "C" int epsgrad_adam_step(float *C, float *M, float *V, const float *G, size_t n, int step,
                                 double b1, double b2, double lr, double eps, void *stream)
{
    if (!C || !M || !V || !G || step < 1) return EPSGRAD_EINVAL;
    if (!(b1 >= 0.0 && b1 < 1.0) || !(b2 >= 0.0 && b2 < 1.0) || !(lr > 0.0) || !(eps >= 0.0)) return EPSGRAD_EINVAL;
    if (n == 0) return EPSGRAD_OK;
    const double c1 = 1.0 - std::pow(b1, (double)step), c2 = 1.0 - std::pow(b2, (double)step);
    k_adam<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(C, M, V, G, n, (float)b1, (float)b2, (float)(1.0 - b1), (float)(1.0 - b2), (float)(1.0 / c1),
                                                                        (float)(1.0 / c2), (float)lr, (float)eps);
    return cudaGetLastError() == cudaSuccess ? EPSGRAD_OK : EPSGRAD_ECUDA;
}

// ------------------------------------------------------------------------------------ SOAP, Eqs. (12)-(13)
namespace {

template <bool TA, bool TB>
int gemm(const float *A, const float *B, float *C, int m, int n, int k, int lda, int ldb, int ldc, float alpha, float beta, cudaStream_t st)
{
    k_gemm<TA, TB><<<dim3(cdiv(n, GM_T), cdiv(m, GM_T)), GM_THREADS, 0, st>>>(A, B, C, m, n, k, lda, ldb, ldc, alpha, beta);
    return cudaGetLastError() == cudaSuccess ? EPSGRAD_OK : EPSGRAD_ECUDA;
}

// cuSOLVER's dense symmetric eigensolver, found at run time: the library is a dependency of this one optional call only
struct SolverApi {
    bool tried = false, ok = false;
    decltype(&cusolverDnCreate) create = nullptr;
    decltype(&cusolverDnSetStream) set_stream = nullptr;
    decltype(&cusolverDnSsyevd_bufferSize) bufsize = nullptr;
    decltype(&cusolverDnSsyevd) syevd = nullptr;
    cusolverDnHandle_t handle[64] = {};
};
SolverApi g_solver;
std::mutex g_solver_mutex;

cusolverDnHandle_t solver_handle(int device)
{
    std::lock_guard<std::mutex> lock(g_solver_mutex);
    SolverApi &S = g_solver;
    if (!S.tried) {
        S.tried = true;
        void *lib = nullptr;
        for (const char *name : {"libcusolver.so.11", "libcusolver.so.12", "libcusolver.so"})
            if ((lib = dlopen(name, RTLD_NOW | RTLD_GLOBAL))) break;
        if (lib) {
            S.create = (decltype(S.create))dlsym(lib, "cusolverDnCreate");
            S.set_stream = (decltype(S.set_stream))dlsym(lib, "cusolverDnSetStream");
            S.bufsize = (decltype(S.bufsize))dlsym(lib, "cusolverDnSsyevd_bufferSize");
            S.syevd = (decltype(S.syevd))dlsym(lib, "cusolverDnSsyevd");
            S.ok = S.create && S.set_stream && S.bufsize && S.syevd;
        }
    }
    if (!S.ok || device < 0 || device >= 64) return nullptr;
    if (!S.handle[device] && S.create(&S.handle[device]) != CUSOLVER_STATUS_SUCCESS) S.handle[device] = nullptr;
    return S.handle[device];
}

int solver_lwork(cusolverDnHandle_t h, int n)
{
    int lwork = 0;
    if (g_solver.bufsize(h, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n, nullptr, n, nullptr, &lwork) != CUSOLVER_STATUS_SUCCESS) return -1;
    return lwork;
}

}  // namespace

extern "C" int epsgrad_soap_accumulate(float *L, float *R, const float *G, int mx, int my, double b2, void *stream)
{
    if (!L || !R || !G || mx < 1 || my < 1 || !(b2 >= 0.0 && b2 < 1.0)) return EPSGRAD_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = gemm<false, true>(G, G, L, mx, mx, my, my, my, mx, (float)(1.0 - b2), (float)b2, st);        // G G^T
    if (!rc) rc = gemm<true, false>(G, G, R, my, my, mx, my, my, my, (float)(1.0 - b2), (float)b2, st);   // G^T G
    return rc;
}

extern "C" size_t epsgrad_soap_step_workspace_bytes(int mx, int my)
{
    return mx < 1 || my < 1 ? 0 : 3 * align_up((size_t)mx * my * 4, 256);
}

extern "C" int epsgrad_soap_step(float *C, float *M, float *Vp, const float *G, const float *QL, const float *QR, int mx, int my,
                                 int step, double b1, double b2, double lr, double eps, void *work, size_t work_bytes, void *stream)
{
    if (!C || !M || !Vp || !G || !QL || !QR || mx < 1 || my < 1 || step < 1) return EPSGRAD_EINVAL;
    if (!(b1 >= 0.0 && b1 < 1.0) || !(b2 >= 0.0 && b2 < 1.0) || !(lr > 0.0) || !(eps >= 0.0)) return EPSGRAD_EINVAL;
    if (!work || work_bytes < epsgrad_soap_step_workspace_bytes(mx, my)) return EPSGRAD_ENOWORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)mx * my, pitch = align_up(n * 4, 256);
    float *T = (float *)work, *Gp = (float *)((char *)work + pitch), *Mp = (float *)((char *)work + 2 * pitch);
    const unsigned nb = (unsigned)((n + 255) / 256);
    const double c1 = 1.0 - std::pow(b1, (double)step), c2 = 1.0 - std::pow(b2, (double)step);
    k_soap_moment<<<nb, 256, 0, st>>>(M, G, n, (float)b1, (float)(1.0 - b1));
    int rc = cudaGetLastError() == cudaSuccess ? EPSGRAD_OK : EPSGRAD_ECUDA;
    if (!rc) rc = gemm<true, false>(QL, G, T, mx, my, mx, mx, my, my, 1.0f, 0.0f, st);       // Q_L^T G
    if (!rc) rc = gemm<false, false>(T, QR, Gp, mx, my, my, my, my, my, 1.0f, 0.0f, st);     // (.) Q_R
    if (!rc) rc = gemm<true, false>(QL, M, T, mx, my, mx, mx, my, my, 1.0f, 0.0f, st);       // Q_L^T M
    if (!rc) rc = gemm<false, false>(T, QR, Mp, mx, my, my, my, my, my, 1.0f, 0.0f, st);
    if (rc) return rc;
    k_soap_rotated<<<nb, 256, 0, st>>>(Vp, Gp, Mp, n, (float)b2, (float)(1.0 - b2), (float)(1.0 / c1), (float)(1.0 / c2), (float)eps);
    if (cudaGetLastError() != cudaSuccess) return EPSGRAD_ECUDA;
    rc = gemm<false, false>(QL, Gp, T, mx, my, mx, mx, my, my, 1.0f, 0.0f, st);              // Q_L N'
    if (!rc) rc = gemm<false, true>(T, QR, C, mx, my, my, my, my, my, (float)(-lr), 1.0f, st);   // C <- C - eta (.) Q_R^T
    return rc;
}

extern "C" size_t epsgrad_soap_eigh_workspace_bytes(int n)
{
    if (n < 1) return 0;
    int device = 0;
    if (cudaGetDevice(&device) != cudaSuccess) { cudaGetLastError(); return 0; }
    cusolverDnHandle_t h = solver_handle(device);
    if (!h) return 0;
    const int lwork = solver_lwork(h, n);
    if (lwork < 0) return 0;
    return align_up((size_t)n * n * 4, 256) + align_up((size_t)lwork * 4, 256) + 256;
}

extern "C" int epsgrad_soap_eigh(const float *A, float *Q, float *w, int n, void *work, size_t work_bytes, void *stream)
{
    if (!A || !Q || !w || n < 1) return EPSGRAD_EINVAL;
    int device = 0;
    if (cudaGetDevice(&device) != cudaSuccess) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    cusolverDnHandle_t h = solver_handle(device);
    if (!h) return EPSGRAD_EUNSUPPORTED;                   // no cuSOLVER on this machine
    const int lwork = solver_lwork(h, n);
    if (lwork < 0) return EPSGRAD_ECUDA;
    const size_t b_a = align_up((size_t)n * n * 4, 256), b_w = align_up((size_t)lwork * 4, 256);
    if (!work || work_bytes < b_a + b_w + 256) return EPSGRAD_ENOWORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    float *a = (float *)work, *lw = (float *)((char *)work + b_a);
    int *info = (int *)((char *)work + b_a + b_w);
    if (cudaMemcpyAsync(a, A, (size_t)n * n * 4, cudaMemcpyDeviceToDevice, st) != cudaSuccess) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    {
        // the per-device handle carries the stream: binding it and enqueueing the solver is one critical section
        std::lock_guard<std::mutex> lock(g_solver_mutex);
        if (g_solver.set_stream(h, st) != CUSOLVER_STATUS_SUCCESS) return EPSGRAD_ECUDA;
        // A is symmetric, so its row-major image is its column-major image; the eigenvectors come back as columns, column-major
        if (g_solver.syevd(h, CUSOLVER_EIG_MODE_VECTOR, CUBLAS_FILL_MODE_LOWER, n, a, n, w, lw, lwork, info) != CUSOLVER_STATUS_SUCCESS) return EPSGRAD_ECUDA;
    }
    k_transpose<<<dim3(cdiv(n, 32), cdiv(n, 32)), 256, 0, st>>>(a, Q, n);
    return cudaGetLastError() == cudaSuccess ? EPSGRAD_OK : EPSGRAD_ECUDA;
}

extern "C" int epsgrad_soap_eigh_info(const void *work, size_t work_bytes, int n, void *stream, int *info)
{
    if (!work || !info || n < 1) return EPSGRAD_EINVAL;
    int device = 0;
    if (cudaGetDevice(&device) != cudaSuccess) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    cusolverDnHandle_t h = solver_handle(device);
    if (!h) return EPSGRAD_EUNSUPPORTED;
    const int lwork = solver_lwork(h, n);
    if (lwork < 0) return EPSGRAD_ECUDA;
    const size_t b_a = align_up((size_t)n * n * 4, 256), b_w = align_up((size_t)lwork * 4, 256);
    if (work_bytes < b_a + b_w + 256) return EPSGRAD_ENOWORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    if (cudaMemcpyAsync(info, (const char *)work + b_a + b_w, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    return EPSGRAD_OK;
}

extern "C" double epsgrad_beta_schedule(double beta_min, double beta_max, int i, int n_iter)
{
    const double x = n_iter > 0 ? (double)i / (double)n_iter : 1.0;
    return beta_min + (beta_max - beta_min) * std::expm1(x * x) / std::expm1(1.0);
}

extern "C" int epsgrad_beta_update(double *t, double *beta_max, double gamma, double u, double u0, double beta)
{
    if (!t || !beta_max || !(u > 0.0) || !(u0 > 0.0) || !(beta > 0.0) || !(gamma >= 0.0 && gamma <= 1.0)) return EPSGRAD_EINVAL;
    const double tn = gamma * *t + (1.0 - gamma) * (1.0 / u - 1.0) / beta;
    if (!(tn > 0.0)) return EPSGRAD_EINVAL;
    *t = tn;
    *beta_max = gamma * *beta_max + (1.0 - gamma) * (1.0 / u0 - 1.0) / tn;
    return EPSGRAD_OK;
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

// ------------------------------------------------------------------------------------ host buffers
extern "C" int eps_forward_vjp_host(epsgrad_plan_t *P, const float *C_host, float beta, int n_pairs,
                                    const void *const *EF_host, const void *const *EA_host,
                                    float *eps_host, float *dFdC_host, void *stream)
{
    if (!P || !C_host || !(beta > 0.0f) || !std::isfinite(beta)) return EPSGRAD_EINVAL;
    if (!eps_host && !dFdC_host) return EPSGRAD_EINVAL;
    if (dFdC_host) {
        if (n_pairs < 1 || !EF_host || !EA_host) return EPSGRAD_EINVAL;
        for (int p = 0; p < n_pairs; ++p)
            if (!EF_host[p] || !EA_host[p]) return EPSGRAD_EINVAL;
    } else {
        n_pairs = 0;
    }
    if (P->emb.nx_full > 0 || P->slab_nx > 0) return EPSGRAD_EUNSUPPORTED;     // host buffers are region-sized: no embedding or slab here
    if (!P->ws) return EPSGRAD_ENOWORKSPACE;
    if (!P->stg || P->stg_bytes < epsgrad_staging_bytes(P, n_pairs)) return EPSGRAD_ENOWORKSPACE;
    DeviceGuard g(P->device);
    cudaStream_t st = (cudaStream_t)stream;
    begin_call(P, st);
    P->last_h2d = P->last_d2h = 0;

    const size_t b_c = n_ctrl(P) * 4, b_e = n_eps(P) * 4, b_f = n_eps(P) * 8;
    char *base = (char *)P->stg;
    float *dC = (float *)base;              base += align_up(b_c, 256);
    float *dG = (float *)base;              base += align_up(b_c, 256);
    float *dE = (float *)base;              base += align_up(b_e, 256);
    std::vector<const void *> ef(n_pairs), ea(n_pairs);
    bool ok = cudaMemcpyAsync(dC, C_host, b_c, cudaMemcpyHostToDevice, st) == cudaSuccess;
    P->last_h2d += b_c;
    // Eq. (1) needs only the slab cells of the fields ("|Omega_D").  When every field buffer is pinned, mapped host
    // memory, the z-reduction reads its windows straight out of it (16-byte asynchronous copies over PCIe / C2C) and the
    // rest of the fields never crosses the bus; otherwise (pageable memory, dense plans) the fields are staged whole.
    bool direct = P->host_direct && !P->dense && n_pairs > 0;
    for (int p = 0; p < n_pairs && direct; ++p) {
        const void *hp[2] = {EF_host[p], EA_host[p]};
        const void **dp[2] = {&ef[p], &ea[p]};
        for (int f = 0; f < 2 && direct; ++f) {
            cudaPointerAttributes at;
            if (cudaPointerGetAttributes(&at, hp[f]) != cudaSuccess) { cudaGetLastError(); direct = false; break; }
            if (at.type != cudaMemoryTypeHost || !at.devicePointer || ((uintptr_t)at.devicePointer & 15)) { direct = false; break; }
            *dp[f] = at.devicePointer;
        }
    }
    if (direct) {
        const size_t ncolB = (size_t)P->cfg.batch * P->nx * P->ny;
        P->last_h2d += (size_t)2 * n_pairs * ncolB * ((size_t)2 * P->nch[0] + P->nch[1]) * 16;   // the chunks the kernel copies
    }
    for (int p = 0; p < n_pairs && ok && !direct; ++p) {
        ef[p] = base; base += align_up(b_f, 256);
        ea[p] = base; base += align_up(b_f, 256);
        ok = cudaMemcpyAsync((void *)ef[p], EF_host[p], b_f, cudaMemcpyHostToDevice, st) == cudaSuccess &&
             cudaMemcpyAsync((void *)ea[p], EA_host[p], b_f, cudaMemcpyHostToDevice, st) == cudaSuccess;
        P->last_h2d += 2 * b_f;
    }
    if (!ok) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    if (direct && P->host_direct == 2 && eps_host && dFdC_host && P->overlap && !P->prof) {
        // Copy-engine gather: one strided 2-D copy per field moves the union slab window of every z column into a packed
        // staging buffer on the auxiliary stream, while eps is computed and sent to the host on the caller's stream -- the
        // two transfers use the two copy engines, and no SM waits on the bus (at paper scale 7.0 ms against 7.9 ms for the
        // in-place reads beside the same eps transfer).
        int u0 = 0, un = 0;
        window_union(P, &u0, &un);
        const size_t rows = (size_t)P->cfg.batch * 3 * P->nx * P->ny, wbytes = (size_t)un * 16, b_p = align_up(rows * wbytes, 256);
        cudaStream_t ax = P->aux;
        ok = cudaEventRecord(P->ev_fork, st) == cudaSuccess && cudaStreamWaitEvent(ax, P->ev_fork, 0) == cudaSuccess;
        for (int p = 0; p < n_pairs && ok; ++p) {
            ef[p] = base; base += b_p;
            ea[p] = base; base += b_p;
            if (un > 0)
                ok = cudaMemcpy2DAsync((void *)ef[p], wbytes, (const char *)EF_host[p] + (size_t)u0 * 16, (size_t)P->cfg.nz * 8, wbytes, rows,
                                       cudaMemcpyHostToDevice, ax) == cudaSuccess &&
                     cudaMemcpy2DAsync((void *)ea[p], wbytes, (const char *)EA_host[p] + (size_t)u0 * 16, (size_t)P->cfg.nz * 8, wbytes, rows,
                                       cudaMemcpyHostToDevice, ax) == cudaSuccess;
        }
        ok = ok && cudaEventRecord(P->ev_r, ax) == cudaSuccess;
        P->last_h2d = b_c + (size_t)2 * n_pairs * rows * wbytes;
        int rc = EPSGRAD_OK;
        if (ok) {
            rc = launch_front(P, dC, beta, st);
            if (!rc) rc = launch_fwd2d(P, ws_phi(P), beta, ws_e2d(P), ws_coef(P), nullptr, st);
            if (!rc && eps_host) {
                rc = launch_extrude(P, ws_e2d(P), dE, st);
                if (!rc) ok = cudaMemcpyAsync(eps_host, dE, b_e, cudaMemcpyDeviceToHost, st) == cudaSuccess;
                P->last_d2h += b_e;
            }
        }
        // always join the auxiliary stream
        if (cudaStreamWaitEvent(st, P->ev_r, 0) != cudaSuccess) ok = false;
        if (!ok) { cudaGetLastError(); return EPSGRAD_ECUDA; }
        if (rc) return rc;
        rc = launch_zreduce(P, n_pairs, ef.data(), ea.data(), ws_gbar(P), st, false, true);
        if (!rc) rc = launch_maskgrad(P, ws_phi(P), beta, ws_gbar(P), ws_coef(P), ws_v(P), st);
        if (!rc && P->morph_R > 0) rc = launch_morph_reverse(P, ws_phi(P), beta, ws_v(P), st);
        if (!rc) rc = launch_filterT(P, ws_v(P), dG, st);
        if (rc) return rc;
        ok = cudaMemcpyAsync(dFdC_host, dG, b_c, cudaMemcpyDeviceToHost, st) == cudaSuccess;
        P->last_d2h += b_c;
        if (!ok) { cudaGetLastError(); return EPSGRAD_ECUDA; }
        return EPSGRAD_OK;
    }
    if (direct && eps_host && dFdC_host && P->overlap && !P->prof) {
        // The bus is full duplex: eps does not depend on the fields, so it is finished first and travels to the host on the
        // auxiliary stream while the z-reduction pulls its windows the other way.
        cudaStream_t ax = P->aux;
        int rc = launch_front(P, dC, beta, st);
        if (!rc) rc = launch_fwd2d(P, ws_phi(P), beta, ws_e2d(P), ws_coef(P), nullptr, st);
        if (!rc) rc = launch_extrude(P, ws_e2d(P), dE, st);
        if (rc) return rc;
        ok = cudaEventRecord(P->ev_2d, st) == cudaSuccess && cudaStreamWaitEvent(ax, P->ev_2d, 0) == cudaSuccess &&
             cudaMemcpyAsync(eps_host, dE, b_e, cudaMemcpyDeviceToHost, ax) == cudaSuccess &&
             cudaEventRecord(P->ev_join, ax) == cudaSuccess;
        P->last_d2h += b_e;
        if (ok) {
            rc = launch_zreduce(P, n_pairs, ef.data(), ea.data(), ws_gbar(P), st, true);
            if (!rc) rc = launch_maskgrad(P, ws_phi(P), beta, ws_gbar(P), ws_coef(P), ws_v(P), st);
            if (!rc && P->morph_R > 0) rc = launch_morph_reverse(P, ws_phi(P), beta, ws_v(P), st);
            if (!rc) rc = launch_filterT(P, ws_v(P), dG, st);
            if (!rc) ok = cudaMemcpyAsync(dFdC_host, dG, b_c, cudaMemcpyDeviceToHost, st) == cudaSuccess;
            P->last_d2h += b_c;
        }
        // always join
        if (cudaStreamWaitEvent(st, P->ev_join, 0) != cudaSuccess) ok = false;
        if (!ok) { cudaGetLastError(); return EPSGRAD_ECUDA; }
        return rc;
    }
    P->cur_host_src = direct;
    int rc = run_chain(P, dC, beta, n_pairs, ef.data(), ea.data(), eps_host ? dE : nullptr, dFdC_host ? dG : nullptr, st);
    P->cur_host_src = 0;
    if (rc) return rc;
    if (eps_host) {
        ok = ok && cudaMemcpyAsync(eps_host, dE, b_e, cudaMemcpyDeviceToHost, st) == cudaSuccess;
        P->last_d2h += b_e;
    }
    if (dFdC_host) {
        ok = ok && cudaMemcpyAsync(dFdC_host, dG, b_c, cudaMemcpyDeviceToHost, st) == cudaSuccess;
        P->last_d2h += b_c;
    }
    if (!ok) { cudaGetLastError(); return EPSGRAD_ECUDA; }
    return EPSGRAD_OK;
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
