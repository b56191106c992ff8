/*
 * epsgrad_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, float64 CPU restatement of the parametrization chain
 *     C  ->  eps_hat on the Yee grid          (paper Sec. 3, Eqs. (2),(3)/(6),(7),(8))
 * and of its reverse pass
 *     dF/dC = -2 Re( (d eps_hat / dC)^T . (E_F (.) E_A) )     (paper Eq. (1))
 * of arxiv 2505.03352 ("Accelerated inverse design of passive Si photonics").
 * Citations "P:L<n>" are line numbers of the paper text; "S<n>" are
 * the readings of silent/ambiguous points listed in DESIGN.md section 3.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.  It shares no code,
 * header, table or helper with the CUDA path (paper_2505_03352_b200/csrc) and
 * is never tuned: every stage is the defining loop, written in the paper's
 * order; reverse stages are the literal scatter-transposes of the forward
 * loops (serial, so that they need no atomics).  OpenMP is used only on loops
 * whose iterations write disjoint outputs.
 *
 * Parity pins: tests/test_oracle_*.py (closed forms, hand-made masks, library
 * special cases, brute force, adjoint identity, finite differences, a float64
 * autograd restatement).  Unpinned: absolute eps values on random inputs are
 * not printed anywhere in the paper; they are pinned through the stage checks.
 *
 * Geometry (cell units; S3).  Design region [0,nx] x [0,ny].  Control node a
 * sits at x_a = ux*(a+1/2) with ux = nx/mx.  Mask pixel p has its centre at
 * X_p = (p+1/2)/s, s mask pixels per Yee cell, mask size px = s*nx.  Yee node
 * i owns the block x in [i,i+1]; E_z sits on the node in the xy plane, E_x is
 * half a cell toward +x, E_y half a cell toward +y.  In z, E_x/E_y have the
 * footprint [k,k+1] and E_z has [k+1/2,k+3/2].  The slab is [z_lo,z_hi].
 * All arrays are row-major with the last index fastest.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t mx, my;          /* control grid                                      */
    int32_t nx, ny, nz;      /* Yee grid of the design region                     */
    int32_t s;               /* mask pixels per Yee cell per axis (even; S4)      */
    int32_t filter_kind;     /* 0 conic, 1 Gaussian with per-axis truncation (S11)*/
    int32_t normalize;       /* 1: density filter, renormalised at borders (S2)   */
    double  radius, sigma;   /* in Yee cells (S3)                                 */
    double  z_lo, z_hi;      /* slab extent in cell units (S8)                    */
    double  eta;             /* 0.5 -> Eq. (6) form, 0 -> Eq. (3) form (S9)       */
    double  eps_core, eps_clad;
    double  delta;           /* guard in the normal normalisation (S6)            */
    double  morph_diam;      /* d of Eqs. (4)-(5) in Yee cells; 0 = filters off   */
    double  morph_alpha;     /* alpha of Eqs. (4)-(5) (App. B: 20)                */
} orc_cfg;

static int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* ------------------------------------------------------------------ */
/* Step 1. Basis function b(dx,dy) of Eq. (2) (S1, S11).    */
/* ------------------------------------------------------------------ */
double orc_weight(const orc_cfg *g, double dx, double dy)
{
    if (g->filter_kind == 0) {                      /* conic: max(0, 1 - d/R) */
        double w = 1.0 - sqrt(dx * dx + dy * dy) / g->radius;
        return w > 0.0 ? w : 0.0;
    }
    /* Gaussian, truncated per axis at |d| <= R (square support, S11) */
    if (fabs(dx) > g->radius || fabs(dy) > g->radius) return 0.0;
    return exp(-(dx * dx + dy * dy) / (2.0 * g->sigma * g->sigma));
}

/* range of control nodes that can have non-zero weight at coordinate X */
static void node_range(double X, double R, double u, int m, int *lo, int *hi)
{
    int a0 = (int)floor((X - R) / u - 0.5) - 1;
    int a1 = (int)ceil((X + R) / u - 0.5) + 1;
    *lo = clampi(a0, 0, m - 1);
    *hi = clampi(a1, 0, m - 1);
}

/* ------------------------------------------------------------------ */
/* Step 2. Level-set / density expansion, Eq. (2), evaluated  */
/* at the mask pixel centres; normalised form (S2):                   */
/*   Phi[p,q] = sum_ab W(X_p-x_a, Y_q-y_b) C[a,b] / sum_ab W(...)     */
/* den[] (may be NULL) receives the normaliser (1 if !normalize).     */
/* ------------------------------------------------------------------ */
void orc_filter(const orc_cfg *g, const double *C, double *Phi, double *den_out)
{
    const int px = g->s * g->nx, py = g->s * g->ny;
    const double ux = (double)g->nx / g->mx, uy = (double)g->ny / g->my;
#pragma omp parallel for schedule(static)
    for (int p = 0; p < px; ++p) {
        double X = (p + 0.5) / g->s;
        int alo, ahi;
        node_range(X, g->radius, ux, g->mx, &alo, &ahi);
        for (int q = 0; q < py; ++q) {
            double Y = (q + 0.5) / g->s;
            int blo, bhi;
            node_range(Y, g->radius, uy, g->my, &blo, &bhi);
            double num = 0.0, den = 0.0;
            for (int a = alo; a <= ahi; ++a)
                for (int b = blo; b <= bhi; ++b) {
                    double w = orc_weight(g, X - ux * (a + 0.5), Y - uy * (b + 0.5));
                    num += w * C[(size_t)a * g->my + b];
                    den += w;
                }
            if (!g->normalize) den = 1.0;
            Phi[(size_t)p * py + q] = num / den;
            if (den_out) den_out[(size_t)p * py + q] = den;
        }
    }
}

/* transpose of orc_filter: Cbar[a,b] += W * Phibar[p,q] / den[p,q]   (scatter) */
void orc_filter_T(const orc_cfg *g, const double *Phibar, double *Cbar)
{
    const int px = g->s * g->nx, py = g->s * g->ny;
    const double ux = (double)g->nx / g->mx, uy = (double)g->ny / g->my;
    memset(Cbar, 0, sizeof(double) * (size_t)g->mx * g->my);
    for (int p = 0; p < px; ++p) {
        double X = (p + 0.5) / g->s;
        int alo, ahi;
        node_range(X, g->radius, ux, g->mx, &alo, &ahi);
        for (int q = 0; q < py; ++q) {
            double Y = (q + 0.5) / g->s;
            int blo, bhi;
            node_range(Y, g->radius, uy, g->my, &blo, &bhi);
            double den = 0.0;
            for (int a = alo; a <= ahi; ++a)
                for (int b = blo; b <= bhi; ++b)
                    den += orc_weight(g, X - ux * (a + 0.5), Y - uy * (b + 0.5));
            if (!g->normalize) den = 1.0;
            double v = Phibar[(size_t)p * py + q] / den;
            for (int a = alo; a <= ahi; ++a)
                for (int b = blo; b <= bhi; ++b)
                    Cbar[(size_t)a * g->my + b] +=
                        orc_weight(g, X - ux * (a + 0.5), Y - uy * (b + 0.5)) * v;
        }
    }
}

/* ------------------------------------------------------------------ */
/* Step 3a. Projection, Eq. (3)/(6) (S9):                  */
/*   rho = 1/2 (1 + tanh(beta (Phi - eta)))                            */
/* ------------------------------------------------------------------ */
void orc_project(int64_t n, const double *Phi, double beta, double eta, double *rho)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) rho[i] = 0.5 * (1.0 + tanh(beta * (Phi[i] - eta)));
}

/* analytic derivative: d rho / d Phi = (beta/2) / cosh^2(beta (Phi-eta)) */
void orc_project_T(int64_t n, const double *Phi, double beta, double eta,
                   const double *rhobar, double *Phibar)
{
    for (int64_t i = 0; i < n; ++i) {
        double c = cosh(beta * (Phi[i] - eta));
        Phibar[i] = rhobar[i] * (0.5 * beta) / (c * c);   /* c = inf -> 0 */
    }
}

/* eps_hat is differentiable in beta too: d rho / d beta = (Phi - eta)/2 / cosh^2(beta (Phi - eta));
 * returns sum_i rhobar_i d rho_i / d beta. */
double orc_project_dbeta(int64_t n, const double *Phi, double beta, double eta, const double *rhobar)
{
    double acc = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        double c = cosh(beta * (Phi[i] - eta));
        acc += rhobar[i] * 0.5 * (Phi[i] - eta) / (c * c);
    }
    return acc;
}

/* ------------------------------------------------------------------ */
/* Step 3b. Mixing rule: e = rho eps_core + (1-rho) eps_clad;  */
/* r = 1/e is the integrand of <eps^-1> in Eq. (7).                    */
/* ------------------------------------------------------------------ */
void orc_mix(const orc_cfg *g, int64_t n, const double *rho, double *e, double *r)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        e[i] = rho[i] * g->eps_core + (1.0 - rho[i]) * g->eps_clad;
        r[i] = 1.0 / e[i];
    }
}

/* rhobar += (eps_core-eps_clad) * (ebar - rbar / e^2) */
void orc_mix_T(const orc_cfg *g, int64_t n, const double *e, const double *ebar,
               const double *rbar, double *rhobar)
{
    for (int64_t i = 0; i < n; ++i)
        rhobar[i] += (g->eps_core - g->eps_clad) * (ebar[i] - rbar[i] / (e[i] * e[i]));
}

/* ------------------------------------------------------------------ */
/* Step 4. Cell averages, Eq. (8) as finite sums on the     */
/* high-resolution mask: shift by half an FDTD cell and down-sample    */
/* (P:L95).  comp 0 = E_x (shift +s/2 in p), 1 = E_y (shift +s/2 in    */
/* q), 2 = E_z (no shift).  Pixel indices are clamped (replicate, S5). */
/* ------------------------------------------------------------------ */
void orc_average(const orc_cfg *g, const double *f, int comp, double *out)
{
    const int s = g->s, px = s * g->nx, py = s * g->ny;
    const int sp = comp == 0 ? s / 2 : 0, sq = comp == 1 ? s / 2 : 0;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < g->nx; ++i)
        for (int j = 0; j < g->ny; ++j) {
            double acc = 0.0;
            for (int a = 0; a < s; ++a)
                for (int b = 0; b < s; ++b) {
                    int p = clampi(s * i + sp + a, 0, px - 1);
                    int q = clampi(s * j + sq + b, 0, py - 1);
                    acc += f[(size_t)p * py + q];
                }
            out[(size_t)i * g->ny + j] = acc / (double)(s * s);
        }
}

/* fbar[p,q] += outbar[i,j] / s^2 for every (a,b) of the footprint (scatter) */
void orc_average_T(const orc_cfg *g, const double *outbar, int comp, double *fbar)
{
    const int s = g->s, px = s * g->nx, py = s * g->ny;
    const int sp = comp == 0 ? s / 2 : 0, sq = comp == 1 ? s / 2 : 0;
    for (int i = 0; i < g->nx; ++i)
        for (int j = 0; j < g->ny; ++j) {
            double v = outbar[(size_t)i * g->ny + j] / (double)(s * s);
            for (int a = 0; a < s; ++a)
                for (int b = 0; b < s; ++b) {
                    int p = clampi(s * i + sp + a, 0, px - 1);
                    int q = clampi(s * j + sq + b, 0, py - 1);
                    fbar[(size_t)p * py + q] += v;
                }
        }
}

/* ------------------------------------------------------------------ */
/* Step 5. Sobel operators on the design at FDTD resolution,   */
/* replicate padding (S5), scaled by 1/8 so that a unit ramp has g=1:  */
/*   gx[i,j] = sum_{di,dj} di (2-|dj|)/8 D[i+di, j+dj],  gy: di <-> dj */
/* ------------------------------------------------------------------ */
void orc_sobel(const orc_cfg *g, const double *D, double *gx, double *gy)
{
#pragma omp parallel for schedule(static)
    for (int i = 0; i < g->nx; ++i)
        for (int j = 0; j < g->ny; ++j) {
            double ax = 0.0, ay = 0.0;
            for (int di = -1; di <= 1; ++di)
                for (int dj = -1; dj <= 1; ++dj) {
                    int ii = clampi(i + di, 0, g->nx - 1), jj = clampi(j + dj, 0, g->ny - 1);
                    double d = D[(size_t)ii * g->ny + jj];
                    ax += di * (2 - abs(dj)) / 8.0 * d;
                    ay += dj * (2 - abs(di)) / 8.0 * d;
                }
            gx[(size_t)i * g->ny + j] = ax;
            gy[(size_t)i * g->ny + j] = ay;
        }
}

/* Dbar[clamp(i+di), clamp(j+dj)] += coefficient * gbar[i,j]  (scatter) */
void orc_sobel_T(const orc_cfg *g, const double *gxbar, const double *gybar, double *Dbar)
{
    for (int i = 0; i < g->nx; ++i)
        for (int j = 0; j < g->ny; ++j) {
            double bx = gxbar[(size_t)i * g->ny + j], by = gybar[(size_t)i * g->ny + j];
            for (int di = -1; di <= 1; ++di)
                for (int dj = -1; dj <= 1; ++dj) {
                    int ii = clampi(i + di, 0, g->nx - 1), jj = clampi(j + dj, 0, g->ny - 1);
                    Dbar[(size_t)ii * g->ny + jj] +=
                        di * (2 - abs(dj)) / 8.0 * bx + dj * (2 - abs(di)) / 8.0 * by;
                }
        }
}

/* ------------------------------------------------------------------ */
/* Step 6. Sub-pixel smoothing, Eq. (7), in the 2-D stage with */
/* n = (n_x, n_y, 0) (S7) and one normal per component from that       */
/* component's own shifted density (S6):                               */
/*   n_c^2 = g_c^2 / (g_x^2 + g_y^2 + delta),                          */
/*   eps2d_c = 1 / (n_c^2 H_c + (1 - n_c^2) / A_c)   (c = x, y)        */
/*   eps2d_z = A_z                                                     */
/* comp selects which of (gx, gy) is g_c.  n2_out may be NULL.         */
/* ------------------------------------------------------------------ */
void orc_eq7(const orc_cfg *g, int comp, const double *A, const double *H,
             const double *gx, const double *gy, double *eps2d, double *n2_out)
{
    const int64_t n = (int64_t)g->nx * g->ny;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        if (comp == 2) { eps2d[i] = A[i]; if (n2_out) n2_out[i] = 0.0; continue; }
        double gc = comp == 0 ? gx[i] : gy[i];
        double n2 = gc * gc / (gx[i] * gx[i] + gy[i] * gy[i] + g->delta);
        eps2d[i] = 1.0 / (n2 * H[i] + (1.0 - n2) / A[i]);
        if (n2_out) n2_out[i] = n2;
    }
}

/* reverse of orc_eq7 for c = x,y: from eps2dbar to Abar, Hbar, gxbar, gybar (all overwritten) */
void orc_eq7_T(const orc_cfg *g, int comp, const double *A, const double *H,
               const double *gx, const double *gy, const double *eps2dbar,
               double *Abar, double *Hbar, double *gxbar, double *gybar)
{
    const int64_t n = (int64_t)g->nx * g->ny;
    for (int64_t i = 0; i < n; ++i) {
        if (comp == 2) { Abar[i] = eps2dbar[i]; Hbar[i] = gxbar[i] = gybar[i] = 0.0; continue; }
        double gc = comp == 0 ? gx[i] : gy[i], go = comp == 0 ? gy[i] : gx[i];
        double S = gc * gc + go * go + g->delta;
        double n2 = gc * gc / S;
        double q = n2 * H[i] + (1.0 - n2) / A[i];          /* eps2d = 1/q           */
        double qbar = -eps2dbar[i] / (q * q);
        Hbar[i] = n2 * qbar;
        Abar[i] = -(1.0 - n2) * qbar / (A[i] * A[i]);
        double n2bar = (H[i] - 1.0 / A[i]) * qbar;
        /* n2 = gc^2/S: d/dgc = 2 gc (go^2+delta)/S^2, d/dgo = -2 gc^2 go/S^2 */
        double gcbar = n2bar * 2.0 * gc * (go * go + g->delta) / (S * S);
        double gobar = -n2bar * 2.0 * gc * gc * go / (S * S);
        if (comp == 0) { gxbar[i] = gcbar; gybar[i] = gobar; }
        else           { gybar[i] = gcbar; gxbar[i] = gobar; }
    }
}

/* ------------------------------------------------------------------ */
/* Step 7. z-extrusion with fractional fill at the faces:      */
/* overlap of the component's z-footprint with the slab, then Eq. (7)  */
/* once more with n = z_hat at the horizontal faces (S7, S8):          */
/*   eps_cc[i,j,k] = eps_clad + wxy_k (eps2d_c - eps_clad),  c = x,y   */
/*   eps_zz[i,j,k] = 1 / (wz_k / eps2d_z + (1 - wz_k) / eps_clad)      */
/* ------------------------------------------------------------------ */
static double overlap(double a0, double a1, double b0, double b1)
{
    double lo = a0 > b0 ? a0 : b0, hi = a1 < b1 ? a1 : b1;
    return hi > lo ? hi - lo : 0.0;
}

void orc_zweights(const orc_cfg *g, double *wxy, double *wz)
{
    for (int k = 0; k < g->nz; ++k) {
        wxy[k] = overlap(k, k + 1.0, g->z_lo, g->z_hi);
        wz[k]  = overlap(k + 0.5, k + 1.5, g->z_lo, g->z_hi);
    }
}

void orc_extrude(const orc_cfg *g, const double *eps2d, double *eps)
{
    const int64_t ncell = (int64_t)g->nx * g->ny;
    double *wxy = malloc(sizeof(double) * g->nz), *wz = malloc(sizeof(double) * g->nz);
    orc_zweights(g, wxy, wz);
    for (int c = 0; c < 3; ++c) {
#pragma omp parallel for schedule(static)
        for (int64_t ij = 0; ij < ncell; ++ij) {
            double v = eps2d[c * ncell + ij];
            double *col = eps + ((size_t)c * ncell + ij) * g->nz;
            for (int k = 0; k < g->nz; ++k)
                col[k] = c < 2 ? g->eps_clad + wxy[k] * (v - g->eps_clad)
                               : 1.0 / (wz[k] / v + (1.0 - wz[k]) / g->eps_clad);
        }
    }
    free(wxy); free(wz);
}

/* eps2dbar[c,i,j] = sum_k epsbar[c,i,j,k] * d eps[c,i,j,k] / d eps2d[c,i,j] */
void orc_extrude_T(const orc_cfg *g, const double *eps2d, const double *epsbar, double *eps2dbar)
{
    const int64_t ncell = (int64_t)g->nx * g->ny;
    double *wxy = malloc(sizeof(double) * g->nz), *wz = malloc(sizeof(double) * g->nz);
    orc_zweights(g, wxy, wz);
    for (int c = 0; c < 3; ++c) {
#pragma omp parallel for schedule(static)
        for (int64_t ij = 0; ij < ncell; ++ij) {
            double v = eps2d[c * ncell + ij], acc = 0.0;
            const double *col = epsbar + ((size_t)c * ncell + ij) * g->nz;
            for (int k = 0; k < g->nz; ++k) {
                if (c < 2) acc += wxy[k] * col[k];
                else {
                    double ez = 1.0 / (wz[k] / v + (1.0 - wz[k]) / g->eps_clad);
                    acc += col[k] * ez * ez * wz[k] / (v * v);
                }
            }
            eps2dbar[c * ncell + ij] = acc;
        }
    }
    free(wxy); free(wz);
}

/* ------------------------------------------------------------------ */
/* Morphological filters, Eqs. (4)-(5), on the mask grid.   */
/*   dilate  y = (1/alpha) log  sum K_m exp(alpha x)                   */
/*   erode   y = 1 - (1/alpha) log sum K_m exp(alpha (1 - x))          */
/* K_m = 1 inside a circle of diameter d: the mask pixels whose */
/* centre offset (dp,dq) has dp^2 + dq^2 <= (d s / 2)^2, d in cells.   */
/* K_m is normalised to unit sum over the pixels that lie inside the   */
/* region (G5, S18): otherwise dilate(c) != c.  Finite sums replace    */
/* the integrals, as in Eq. (8).                               */
/* ------------------------------------------------------------------ */
void orc_morph(const orc_cfg *g, const double *x, int erode, double *y)
{
    const int px = g->s * g->nx, py = g->s * g->ny;
    const double rp = 0.5 * g->morph_diam * g->s, al = g->morph_alpha;
    const int R = (int)floor(rp);
#pragma omp parallel for schedule(static)
    for (int p = 0; p < px; ++p)
        for (int q = 0; q < py; ++q) {
            double S = 0.0;
            int N = 0;
            for (int dp = -R; dp <= R; ++dp)
                for (int dq = -R; dq <= R; ++dq) {
                    if ((double)(dp * dp + dq * dq) > rp * rp) continue;
                    const int pp = p + dp, qq = q + dq;
                    if (pp < 0 || pp >= px || qq < 0 || qq >= py) continue;
                    const double v = x[(size_t)pp * py + qq];
                    S += exp(al * (erode ? 1.0 - v : v));
                    ++N;
                }
            const double l = log(S / (double)N) / al;
            y[(size_t)p * py + q] = erode ? 1.0 - l : l;
        }
}

/* transpose of orc_morph at x: xbar += J^T ybar (scatter form, serial).
 * d y[p,q] / d x[p',q'] = exp(alpha x') / S[p,q] (dilate), exp(alpha (1-x')) / S[p,q] (erode). */
void orc_morph_T(const orc_cfg *g, const double *x, int erode, const double *ybar, double *xbar)
{
    const int px = g->s * g->nx, py = g->s * g->ny;
    const double rp = 0.5 * g->morph_diam * g->s, al = g->morph_alpha;
    const int R = (int)floor(rp);
    for (int p = 0; p < px; ++p)
        for (int q = 0; q < py; ++q) {
            double S = 0.0;
            for (int dp = -R; dp <= R; ++dp)
                for (int dq = -R; dq <= R; ++dq) {
                    if ((double)(dp * dp + dq * dq) > rp * rp) continue;
                    const int pp = p + dp, qq = q + dq;
                    if (pp < 0 || pp >= px || qq < 0 || qq >= py) continue;
                    const double v = x[(size_t)pp * py + qq];
                    S += exp(al * (erode ? 1.0 - v : v));
                }
            const double yb = ybar[(size_t)p * py + q];
            for (int dp = -R; dp <= R; ++dp)
                for (int dq = -R; dq <= R; ++dq) {
                    if ((double)(dp * dp + dq * dq) > rp * rp) continue;
                    const int pp = p + dp, qq = q + dq;
                    if (pp < 0 || pp >= px || qq < 0 || qq >= py) continue;
                    const double v = x[(size_t)pp * py + qq];
                    xbar[(size_t)pp * py + qq] += yb * exp(al * (erode ? 1.0 - v : v)) / S;
                }
        }
}

/* ------------------------------------------------------------------ */
/* Whole forward chain, steps 1-7 in order.  C is the fp32 buffer the  */
/* GPU sees, converted to double.  eps: [3,nx,ny,nz] double.           */
/* eps2d_out: optional [3,nx,ny].                                      */
/* ------------------------------------------------------------------ */
typedef struct {
    double *Phi, *rho, *e, *r;          /* mask arrays [px*py]                */
    double *mx[5];                      /* morphological chain: rho0, dilate, erode, erode, dilate (S17) */
    double *A[3], *H[3], *D[3];         /* cell averages per component        */
    double *gx[2], *gy[2];              /* Sobel gradients of D_x, D_y        */
    double *eps2d;                      /* [3,nx,ny]                          */
} orc_work;

static void work_alloc(const orc_cfg *g, orc_work *w)
{
    size_t nm = (size_t)g->s * g->nx * g->s * g->ny, nc = (size_t)g->nx * g->ny;
    w->Phi = malloc(8 * nm); w->rho = malloc(8 * nm); w->e = malloc(8 * nm); w->r = malloc(8 * nm);
    for (int k = 0; k < 5; ++k) w->mx[k] = g->morph_diam > 0.0 ? malloc(8 * nm) : NULL;
    for (int c = 0; c < 3; ++c) { w->A[c] = malloc(8 * nc); w->H[c] = malloc(8 * nc); w->D[c] = malloc(8 * nc); }
    for (int c = 0; c < 2; ++c) { w->gx[c] = malloc(8 * nc); w->gy[c] = malloc(8 * nc); }
    w->eps2d = malloc(8 * 3 * nc);
}

static void work_free(orc_work *w)
{
    free(w->Phi); free(w->rho); free(w->e); free(w->r);
    for (int k = 0; k < 5; ++k) free(w->mx[k]);
    for (int c = 0; c < 3; ++c) { free(w->A[c]); free(w->H[c]); free(w->D[c]); }
    for (int c = 0; c < 2; ++c) { free(w->gx[c]); free(w->gy[c]); }
    free(w->eps2d);
}

static void forward_2d(const orc_cfg *g, const float *C32, double beta, orc_work *w)
{
    const int64_t nm = (int64_t)g->s * g->nx * g->s * g->ny, nc = (int64_t)g->nx * g->ny;
    double *C = malloc(8 * (size_t)g->mx * g->my);
    for (int64_t i = 0; i < (int64_t)g->mx * g->my; ++i) C[i] = (double)C32[i];
    orc_filter(g, C, w->Phi, NULL);                                 /* steps 1-2 */
    free(C);
    if (g->morph_diam > 0.0) {
        /* P:L64-74 (S17): first projection, then "dilate and erode and erode and dilate" (close, then open),
         * then the second projection, Eq. (6), with its threshold 1/2 */
        static const int is_erode[4] = {0, 1, 1, 0};
        orc_project(nm, w->Phi, beta, g->eta, w->mx[0]);
        for (int k = 0; k < 4; ++k) orc_morph(g, w->mx[k], is_erode[k], w->mx[k + 1]);
        orc_project(nm, w->mx[4], beta, 0.5, w->rho);
    } else
        orc_project(nm, w->Phi, beta, g->eta, w->rho);              /* step 3    */
    orc_mix(g, nm, w->rho, w->e, w->r);
    for (int c = 0; c < 3; ++c) {                                   /* step 4    */
        orc_average(g, w->e, c, w->A[c]);
        orc_average(g, w->r, c, w->H[c]);
        orc_average(g, w->rho, c, w->D[c]);
    }
    for (int c = 0; c < 2; ++c) orc_sobel(g, w->D[c], w->gx[c], w->gy[c]);   /* step 5 */
    for (int c = 0; c < 3; ++c)                                     /* step 6    */
        orc_eq7(g, c, w->A[c], w->H[c], c < 2 ? w->gx[c] : NULL, c < 2 ? w->gy[c] : NULL,
                w->eps2d + c * nc, NULL);
}

int orc_forward(const orc_cfg *g, const float *C32, double beta, double *eps, double *eps2d_out)
{
    orc_work w;
    work_alloc(g, &w);
    forward_2d(g, C32, beta, &w);
    if (eps2d_out) memcpy(eps2d_out, w.eps2d, 8 * 3 * (size_t)g->nx * g->ny);
    if (eps) orc_extrude(g, w.eps2d, eps);                          /* step 7    */
    work_free(&w);
    return 0;
}

/* every intermediate of the 2-D stage, for the stage-by-stage pins; any pointer may be NULL */
int orc_forward_stages(const orc_cfg *g, const float *C32, double beta,
                       double *Phi, double *rho, double *e, double *r,
                       double *A, double *H, double *D,      /* [3,nx,ny] each */
                       double *gx, double *gy,               /* [2,nx,ny] each */
                       double *eps2d)                        /* [3,nx,ny]      */
{
    const size_t nm = (size_t)g->s * g->nx * g->s * g->ny, nc = (size_t)g->nx * g->ny;
    orc_work w;
    work_alloc(g, &w);
    forward_2d(g, C32, beta, &w);
    if (Phi) memcpy(Phi, w.Phi, 8 * nm);
    if (rho) memcpy(rho, w.rho, 8 * nm);
    if (e) memcpy(e, w.e, 8 * nm);
    if (r) memcpy(r, w.r, 8 * nm);
    for (int c = 0; c < 3; ++c) {
        if (A) memcpy(A + c * nc, w.A[c], 8 * nc);
        if (H) memcpy(H + c * nc, w.H[c], 8 * nc);
        if (D) memcpy(D + c * nc, w.D[c], 8 * nc);
    }
    for (int c = 0; c < 2; ++c) {
        if (gx) memcpy(gx + c * nc, w.gx[c], 8 * nc);
        if (gy) memcpy(gy + c * nc, w.gy[c], 8 * nc);
    }
    if (eps2d) memcpy(eps2d, w.eps2d, 8 * 3 * nc);
    work_free(&w);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Reverse chain for a real cotangent on eps reduced to the 2-D stage: */
/* eps2dbar [3,nx,ny] -> dF/dC [mx,my].  Stages in reverse order, each */
/* the transpose of its forward loop.                                  */
/* ------------------------------------------------------------------ */
static void reverse_2d(const orc_cfg *g, double beta, const orc_work *w,
                       const double *eps2dbar, double *dFdC, double *dFdbeta)
{
    const size_t nm = (size_t)g->s * g->nx * g->s * g->ny, nc = (size_t)g->nx * g->ny;
    double *ebar = calloc(nm, 8), *rbar = calloc(nm, 8), *rhobar = calloc(nm, 8);
    double *Abar = malloc(8 * nc), *Hbar = malloc(8 * nc), *Dbar = malloc(8 * nc);
    double *gxbar = malloc(8 * nc), *gybar = malloc(8 * nc), *Phibar = malloc(8 * nm);
    for (int c = 0; c < 3; ++c) {
        orc_eq7_T(g, c, w->A[c], w->H[c], c < 2 ? w->gx[c] : NULL, c < 2 ? w->gy[c] : NULL,
                  eps2dbar + c * nc, Abar, Hbar, gxbar, gybar);     /* step 6^T */
        memset(Dbar, 0, 8 * nc);
        if (c < 2) orc_sobel_T(g, gxbar, gybar, Dbar);              /* step 5^T */
        orc_average_T(g, Abar, c, ebar);                            /* step 4^T */
        orc_average_T(g, Hbar, c, rbar);
        orc_average_T(g, Dbar, c, rhobar);
    }
    orc_mix_T(g, (int64_t)nm, w->e, ebar, rbar, rhobar);            /* step 3^T */
    if (g->morph_diam > 0.0) {
        static const int is_erode[4] = {0, 1, 1, 0};
        double *cur = malloc(8 * nm), *nxt = malloc(8 * nm);
        if (dFdbeta) *dFdbeta = orc_project_dbeta((int64_t)nm, w->mx[4], beta, 0.5, rhobar);
        orc_project_T((int64_t)nm, w->mx[4], beta, 0.5, rhobar, cur);
        for (int k = 3; k >= 0; --k) {
            memset(nxt, 0, 8 * nm);
            orc_morph_T(g, w->mx[k], is_erode[k], cur, nxt);
            double *t = cur; cur = nxt; nxt = t;
        }
        if (dFdbeta) *dFdbeta += orc_project_dbeta((int64_t)nm, w->Phi, beta, g->eta, cur);   /* both projections use beta (S17) */
        orc_project_T((int64_t)nm, w->Phi, beta, g->eta, cur, Phibar);
        free(cur); free(nxt);
    } else {
        if (dFdbeta) *dFdbeta = orc_project_dbeta((int64_t)nm, w->Phi, beta, g->eta, rhobar);
        orc_project_T((int64_t)nm, w->Phi, beta, g->eta, rhobar, Phibar);
    }
    orc_filter_T(g, Phibar, dFdC);                                  /* step 2^T */
    free(ebar); free(rbar); free(rhobar); free(Abar); free(Hbar); free(Dbar);
    free(gxbar); free(gybar); free(Phibar);
}

/* VJP with an arbitrary real cotangent epsbar [3,nx,ny,nz]. */
int orc_vjp_real_beta(const orc_cfg *g, const float *C32, double beta, const double *epsbar, double *dFdC, double *dFdbeta);
int orc_vjp_real(const orc_cfg *g, const float *C32, double beta, const double *epsbar, double *dFdC)
{
    return orc_vjp_real_beta(g, C32, beta, epsbar, dFdC, NULL);
}

/* the same with d F / d beta = epsbar . d eps_hat / d beta; dFdbeta may be NULL */
int orc_vjp_real_beta(const orc_cfg *g, const float *C32, double beta, const double *epsbar, double *dFdC, double *dFdbeta)
{
    orc_work w;
    work_alloc(g, &w);
    forward_2d(g, C32, beta, &w);
    double *e2bar = malloc(8 * 3 * (size_t)g->nx * g->ny);
    orc_extrude_T(g, w.eps2d, epsbar, e2bar);                       /* step 7^T */
    reverse_2d(g, beta, &w, e2bar, dFdC, dFdbeta);
    free(e2bar);
    work_free(&w);
    return 0;
}

/*
 * Eq. (1): dF/dC = -2 Re( (d eps/dC)^T (E_F (.) E_A) ), summed over
 * the field pairs.  The product is the plain element-wise complex product, no
 * conjugate (S10).  Fields are complex64 [3,nx,ny,nz], interleaved
 * (re,im) floats, converted to double.
 */
int orc_vjp_beta(const orc_cfg *g, const float *C32, double beta, int n_pairs,
                 const float *const *EF, const float *const *EA, double *dFdC, double *dFdbeta);
int orc_vjp(const orc_cfg *g, const float *C32, double beta, int n_pairs,
            const float *const *EF, const float *const *EA, double *dFdC)
{
    return orc_vjp_beta(g, C32, beta, n_pairs, EF, EA, dFdC, NULL);
}

int orc_vjp_beta(const orc_cfg *g, const float *C32, double beta, int n_pairs,
                 const float *const *EF, const float *const *EA, double *dFdC, double *dFdbeta)
{
    const size_t n3 = 3 * (size_t)g->nx * g->ny * g->nz;
    double *G3 = calloc(n3, 8);
    for (int p = 0; p < n_pairs; ++p) {
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < (int64_t)n3; ++i) {
            double ar = EF[p][2 * i], ai = EF[p][2 * i + 1];
            double br = EA[p][2 * i], bi = EA[p][2 * i + 1];
            G3[i] += -2.0 * (ar * br - ai * bi);
        }
    }
    int rc = orc_vjp_real_beta(g, C32, beta, G3, dFdC, dFdbeta);
    free(G3);
    return rc;
}

/* ------------------------------------------------------------------ */
/* "Unbinarity" u(beta), the relative number of gray pixels.  */
/* Reading S20: the measure of non-discreteness, the mean over the     */
/* design mask of 4 rho (1 - rho) (1 for rho = 1/2, 0 for a binary     */
/* pixel), rho being the final projected mask.                          */
/* ------------------------------------------------------------------ */
double orc_unbinarity(const orc_cfg *g, const float *C32, double beta)
{
    const int64_t nm = (int64_t)g->s * g->nx * g->s * g->ny;
    orc_work w;
    work_alloc(g, &w);
    forward_2d(g, C32, beta, &w);
    double acc = 0.0;
    for (int64_t i = 0; i < nm; ++i) acc += 4.0 * w.rho[i] * (1.0 - w.rho[i]);
    work_free(&w);
    return acc / (double)nm;
}

/* Eq. (14): beta_i = beta_min + (beta_max - beta_min) (exp((i/N)^2) - 1)/(e - 1) */
double orc_beta_schedule(double beta_min, double beta_max, int i, int n_iter)
{
    const double x = (double)i / (double)n_iter;
    return beta_min + (beta_max - beta_min) * (exp(x * x) - 1.0) / (exp(1.0) - 1.0);
}

/* Eq. (15): t <- gamma t + (1-gamma)(1/u - 1)/beta;  beta_max <- gamma beta_max + (1-gamma)(1/u0 - 1)/t */
void orc_beta_update(double *t, double *beta_max, double gamma, double u, double u0, double beta)
{
    *t = gamma * *t + (1.0 - gamma) * (1.0 / u - 1.0) / beta;
    *beta_max = gamma * *beta_max + (1.0 - gamma) * (1.0 / u0 - 1.0) / *t;
}

/* ------------------------------------------------------------------ */
/* Adam, Eqs. (10)-(11), one step i >= 1, in place:       */
/*   M = b1 M + (1-b1) G,  V = b2 V + (1-b2) G^2,                      */
/*   Mh = M/(1-b1^i),  Vh = V/(1-b2^i),  C = C - lr Mh/(sqrt(Vh)+eps)  */
/* ------------------------------------------------------------------ */
void orc_adam_step(int64_t n, double *C, double *M, double *V, const double *G,
                   int i, double b1, double b2, double lr, double eps)
{
    const double c1 = 1.0 - pow(b1, (double)i), c2 = 1.0 - pow(b2, (double)i);
    for (int64_t k = 0; k < n; ++k) {
        M[k] = b1 * M[k] + (1.0 - b1) * G[k];
        V[k] = b2 * V[k] + (1.0 - b2) * G[k] * G[k];
        C[k] -= lr * (M[k] / c1) / (sqrt(V[k] / c2) + eps);
    }
}

int orc_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        n = omp_get_num_threads();
    }
#endif
    return n;
}
