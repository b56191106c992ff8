// optimizer.cu -- the optimizer side of the design loop (include/epsgrad.h): Adam, Eqs. (10)-(11); SOAP, Eqs. (12)-(13), with the
// eigensolver (cuSOLVER syevd, the library's one library step) found at run time; the beta schedule, Eqs. (14)-(15).
#include "plan.cuh"

#include <cmath>
#include <dlfcn.h>
#include <mutex>
#include <cusolverDn.h>   // types and prototypes only: the library is loaded on first use (dlopen), never linked

#include "soap.cuh"

using namespace epsgrad;

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

