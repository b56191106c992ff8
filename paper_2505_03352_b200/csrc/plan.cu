// plan.cu -- epsgrad_plan_t: validation of the configuration, the filter / normaliser / z tables (float64 on the host,
// rounded once), the workspace carve-up and the plan's options (include/epsgrad.h).  Host code only.
#include "plan.cuh"
#include "sizes.cuh"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

using namespace epsgrad;

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

// explicit cell counts that are not upsample x the control grid: Eq. (2) by the general kernels (filter_general.cuh)
static bool is_general(const epsgrad_config_t *c)
{
    return (c->nx_cells > 0 || c->ny_cells > 0) && !(c->nx_cells == c->upsample * c->mx && c->ny_cells == c->upsample * c->my);
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
    }
    if (c->nx_cells < 0 || c->ny_cells < 0 || (c->nx_cells > 0) != (c->ny_cells > 0)) return EPSGRAD_EINVAL;
    if (c->nx_cells > 0 && (c->nx_cells < c->mx || c->ny_cells < c->my)) return EPSGRAD_EINVAL;      // at least one cell per control pixel
    const int nx = c->nx_cells > 0 ? c->nx_cells : c->upsample * c->mx, ny = c->nx_cells > 0 ? c->ny_cells : c->upsample * c->my;
    if (c->morph_diameter > 0.0) {
        const int R = (int)std::floor(0.5 * c->morph_diameter * c->subpixel);
        if (c->subpixel * nx < 2 * R + 1 || c->subpixel * ny < 2 * R + 1) return EPSGRAD_EUNSUPPORTED;
    }
    const int m = c->upsample * c->subpixel;
    if (!is_general(c) && m != 2 && m != 4 && m != 6 && m != 8) return EPSGRAD_EUNSUPPORTED;
    if (c->subpixel > 8) return EPSGRAD_EUNSUPPORTED;
    const double cells = (double)c->batch * 3.0 * nx * ny;
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
    // general plans (non-integer cells per control pixel) never use the phase tables below: they are built for one cell per
    // pixel, only so that every table pointer of the plan is valid
    P->general = is_general(cfg);
    const int u = P->general ? 1 : cfg->upsample, s = cfg->subpixel, m = u * s;
    P->m = m;
    P->nx = cfg->nx_cells > 0 ? cfg->nx_cells : u * cfg->mx;
    P->ny = cfg->nx_cells > 0 ? cfg->ny_cells : u * cfg->my;
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

    if (uncovered && !P->general) { delete P; return EPSGRAD_EINVAL; }    // the density filter would divide 0 by 0 there (R < u/sqrt(2))

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

    if (P->general) {
        // coverage of the normalised Eq. (2) (S2): the mask pixel farthest from the control nodes, axis by axis (the grid is a product)
        double far[2] = {0.0, 0.0};
        for (int ax = 0; ax < 2; ++ax) {
            const int M = ax ? cfg->my : cfg->mx, N = ax ? P->ny : P->nx;
            const double uu = (double)N / M;
            for (int p = 0; p < s * N; ++p) {
                const double X = (p + 0.5) / s;
                int a = (int)std::floor(X / uu);
                a = a < 0 ? 0 : (a > M - 1 ? M - 1 : a);
                double dmin = std::fabs(X - uu * (a + 0.5));
                if (a > 0) dmin = std::min(dmin, std::fabs(X - uu * (a - 0.5)));
                if (a < M - 1) dmin = std::min(dmin, std::fabs(X - uu * (a + 1.5)));
                far[ax] = std::max(far[ax], dmin);
            }
        }
        const double R = cfg->filter_radius;
        uncovered = cfg->filter_normalize && (P->separable ? (far[0] > R || far[1] > R) : !(std::sqrt(far[0] * far[0] + far[1] * far[1]) < R));
        if (uncovered) { delete P; return EPSGRAD_EINVAL; }
    }

    // ---- shared-memory budget of the transposed conic filter (v tile + weight table)
    if (!P->separable && !P->general) {
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

    // ---- tensor-core filter (filter_tc.cuh): per tap row tx the banded matrix A_tx[(fx, beta, fy), j] = W[tx][j - beta][fx][fy],
    // split into two tf32 terms (hi + lo = the float32 weight up to 2^-21), in the K-major chunk layout the MMA descriptors name
    if (!P->separable && !P->general && m == 4 && (NT == 5 || NT == 9 || NT == 13)) {
        const int K = ftc_k(NT), KC = K / 4;
        std::vector<float> atc(ftc_a_floats(NT), 0.0f);
        const size_t half = atc.size() / 2;
        for (int tx = 0; tx < NT; ++tx)
            for (int fx = 0; fx < 4; ++fx)
                for (int beta = 0; beta < FTC_TB; ++beta)
                    for (int fy = 0; fy < 4; ++fy)
                        for (int j = 0; j < K; ++j) {
                            const int ty = j - beta, row = fx * 32 + beta * 4 + fy;
                            if (ty < 0 || ty >= NT) continue;
                            const float wv = w[(((size_t)tx * NT + ty) * m + fx) * m + fy];
                            const float hi = tf32_trunc(wv), lo = tf32_trunc(wv - hi);
                            const size_t o = (((size_t)tx * KC + (j >> 2)) * FTC_M + row) * 4 + (j & 3);
                            atc[o] = hi; atc[half + o] = lo;
                        }
        int prevt = 0;
        cudaGetDevice(&prevt);
        cudaSetDevice(device);
        const bool okt = cudaMalloc(&P->d_atc, atc.size() * 4) == cudaSuccess &&
                         cudaMemcpy(P->d_atc, atc.data(), atc.size() * 4, cudaMemcpyHostToDevice) == cudaSuccess;
        cudaSetDevice(prevt);
        // the transpose (filterT_tc.cuh): A[(tx, beta), (fx, qq)] = W[tx][beta + 2T - qq/4][fx][qq % 4], in k-step slabs of 8 (fx, qq) values
        const int KQ = ftt_kq(NT), KS = ftt_ksteps(NT);
        std::vector<float> att(ftt_a_floats(NT), 0.0f);
        for (int ks = 0; ks < KS; ++ks) {
            const int fx = ks / (KQ / 8), q8 = 8 * (ks - fx * (KQ / 8));
            for (int c = 0; c < 2; ++c)
                for (int tx = 0; tx < NT; ++tx)
                    for (int beta = 0; beta < FTC_TB; ++beta)
                        for (int e = 0; e < 4; ++e) {
                            const int qq = q8 + 4 * c + e, ty = beta + 2 * T - (qq >> 2), fy = qq & 3, row = tx * FTC_TB + beta;
                            if (ty < 0 || ty >= NT) continue;
                            const float wv = w[(((size_t)tx * NT + ty) * m + fx) * m + fy];
                            const float hi = tf32_trunc(wv), lo = tf32_trunc(wv - hi);
                            const size_t o = ((size_t)ks * 2 * 2 + c) * FTC_M * 4 + (size_t)row * 4 + e;      // [ks][hi][c][row][e]; lo one [2][128][4] further
                            att[o] = hi; att[o + 2 * FTC_M * 4] = lo;
                        }
        }
        cudaSetDevice(device);
        const bool oka = cudaMalloc(&P->d_att, att.size() * 4) == cudaSuccess &&
                         cudaMemcpy(P->d_att, att.data(), att.size() * 4, cudaMemcpyHostToDevice) == cudaSuccess;
        cudaSetDevice(prevt);
        if (!okt || !oka) { cudaGetLastError(); epsgrad_plan_destroy(P); return EPSGRAD_ECUDA; }
        P->use_tc = 2;           // where it measured faster (launch.cu)
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
        P->use_pdl = 1;
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
    P->off_tmp = off;  off += P->separable && !P->general ? align_up((size_t)cfg->batch * cfg->mx * P->py * 4, 256) : 0;
    P->off_invden = off; off += P->general ? align_up((size_t)P->px * P->py * 4, 256) : 0;     // 1 / sum W on the mask (filter_general.cuh)
    P->ws_need = off;
    // ---- persistent dataflow kernel (mega.cuh): conic fast path with 4 mask pixels per control pixel, s = 2, no morphological filters
    if (!P->separable && !P->general && m == 4 && s == 2 && (NT == 5 || NT == 9 || NT == 13) && P->morph_R == 0) {
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
    if (P->d_atc) cudaFree(P->d_atc);
    if (P->d_att) cudaFree(P->d_att);
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
    if (dense && P->packed_fields) return EPSGRAD_EUNSUPPORTED;            // packed fields have no cells outside the window to read
    P->dense = dense != 0;
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_embedding(epsgrad_plan_t *P, const epsgrad_embedding_t *e)
{
    if (!P) return EPSGRAD_EINVAL;
    if (!e) { std::memset(&P->emb, 0, sizeof(P->emb)); return EPSGRAD_OK; }
    if (e->nx_full < 1 || e->ny_full < 1 || e->nz_full < 1 || e->i0 < 0 || e->j0 < 0 || e->k0 < 0) return EPSGRAD_EINVAL;
    if (e->i0 + P->nx > e->nx_full || e->j0 + P->ny > e->ny_full || e->k0 + P->cfg.nz > e->nz_full) return EPSGRAD_EINVAL;
    if (e->nz_full % 4 || e->k0 % 4 || P->cfg.nz % 4) return EPSGRAD_EUNSUPPORTED;   // 16-byte pieces of eps (4 cells) and of the fields (2 cells)
    if ((double)P->cfg.batch * 3.0 * e->nx_full * e->ny_full > 2.0e9) return EPSGRAD_EUNSUPPORTED;
    if (P->slab_nx > 0 || P->packed_fields) return EPSGRAD_EUNSUPPORTED;   // one addressing option at a time
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

extern "C" int epsgrad_plan_set_tensor_cores(epsgrad_plan_t *P, int enable)
{
    if (!P) return EPSGRAD_EINVAL;
    if (enable && !P->d_atc) return EPSGRAD_EUNSUPPORTED;
    P->use_tc = enable < 0 ? 0 : (enable > 2 ? 2 : enable);
    return EPSGRAD_OK;
}

extern "C" int epsgrad_plan_set_pdl(epsgrad_plan_t *P, int enable)
{
    if (!P) return EPSGRAD_EINVAL;
    P->use_pdl = enable != 0;
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
    DeviceGuard g(P->device);
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
    if (P->emb.nx_full > 0 || P->general || P->packed_fields) return EPSGRAD_EUNSUPPORTED;   // one addressing option at a time; slabs are cut along control rows
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
        DeviceGuard g(P->device);
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
    DeviceGuard g(P->device);
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

