/* Sanitizer run of the oracle ("oracle built with -fsanitize=address,undefined in a test target").
 * TEST INFRASTRUCTURE.  Built and run by tests/test_oracle_sanitize.py:
 *   gcc -O1 -g -fsanitize=address,undefined -fno-sanitize-recover=undefined -o sanitize_main sanitize_main.c -lm
 * It includes the oracle's source (single-threaded: no OpenMP) and drives every entry point on small, ragged grids --
 * borders everywhere, grid smaller than the filter, slab faces inside one cell, morphological filters on -- so that any
 * out-of-bounds index, uninitialised read that ASan can see, or undefined arithmetic aborts the program.  It checks no
 * values (the pins in tests/ do); it prints a checksum so that the work cannot be optimised away. */
#include "epsgrad_oracle.c"
#include <stdio.h>

static double run(int mx, int my, int u, int s, int nz, double z_lo, double z_hi, int kind, double radius, double sigma,
                  double morph, double beta)
{
    orc_cfg g;
    memset(&g, 0, sizeof(g));
    g.mx = mx; g.my = my; g.nx = u * mx; g.ny = u * my; g.nz = nz; g.s = s;
    g.filter_kind = kind; g.normalize = 1; g.radius = radius; g.sigma = sigma;
    g.z_lo = z_lo; g.z_hi = z_hi; g.eta = 0.5; g.eps_core = 12.11; g.eps_clad = 2.085; g.delta = 1e-12;
    g.morph_diam = morph; g.morph_alpha = 20.0;
    const size_t nc = (size_t)mx * my, n3 = 3 * (size_t)g.nx * g.ny * g.nz;
    float *C = malloc(nc * sizeof(float));
    float *ef = malloc(2 * n3 * sizeof(float)), *ea = malloc(2 * n3 * sizeof(float));
    double *eps = malloc(n3 * sizeof(double)), *grad = malloc(nc * sizeof(double));
    unsigned long long st = 88172645463325252ULL + (unsigned long long)(mx * 131 + my);
    for (size_t i = 0; i < nc; ++i) { st ^= st << 13; st ^= st >> 7; st ^= st << 17; C[i] = (float)((st >> 11) * (1.0 / 9007199254740992.0)); }
    for (size_t i = 0; i < 2 * n3; ++i) { st ^= st << 13; st ^= st >> 7; st ^= st << 17; ef[i] = (float)((st >> 11) * (2.0 / 9007199254740992.0) - 1.0); ea[i] = ef[i] * 0.5f + 0.25f; }
    const float *pf[2] = {ef, ea}, *pa[2] = {ea, ef};
    double db = 0.0, sum = 0.0;
    orc_forward(&g, C, beta, eps, NULL);
    orc_vjp_beta(&g, C, beta, 2, pf, pa, grad, &db);
    sum += orc_unbinarity(&g, C, beta) + db;
    for (size_t i = 0; i < n3; ++i) sum += eps[i];
    for (size_t i = 0; i < nc; ++i) sum += grad[i];
    free(C); free(ef); free(ea); free(eps); free(grad);
    return sum;
}

int main(void)
{
    double sum = 0.0;
    sum += run(7, 5, 2, 2, 8, 2.25, 5.75, 0, 3.0, 1.0, 0.0, 8.0);      /* ragged, conic */
    sum += run(3, 4, 2, 2, 8, 3.6, 3.9, 0, 8.0, 1.0, 0.0, 16.0);       /* grid smaller than the filter; slab inside one cell */
    sum += run(1, 9, 3, 2, 12, 0.0, 12.0, 0, 2.5, 1.0, 0.0, 4.0);      /* a single control row; slab fills z */
    sum += run(6, 7, 1, 4, 4, 0.5, 3.5, 1, 5.0, 1.5, 0.0, 6.0);        /* Gaussian, s = 4 */
    sum += run(9, 8, 2, 2, 8, 2.25, 5.75, 0, 3.0, 1.0, 2.5, 12.0);     /* morphological filters on */
    sum += run(5, 5, 1, 8, 8, 2.0, 6.0, 0, 2.0, 1.0, 1.5, 20.0);       /* s = 8 with the filters on */
    double C[6] = {0.1, 0.2, 0.3, 0.4, 0.5, 0.6}, M[6] = {0}, V[6] = {0}, G[6] = {1, -2, 3, -4, 5, -6};
    orc_adam_step(6, C, M, V, G, 1, 0.9, 0.999, 1e-3, 1e-8);
    double t = 1.0, bm = 60.0;
    orc_beta_update(&t, &bm, 0.95, 0.2, 0.01, 12.0);
    sum += C[0] + t + bm + orc_beta_schedule(10.0, 150.0, 3, 10);
    printf("checksum %.17g\n", sum);
    return 0;
}
