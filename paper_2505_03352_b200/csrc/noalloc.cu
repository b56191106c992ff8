// noalloc.cu -- eps_unbinarity_static: u(beta) (S20) of a mask the caller holds, for callers that may not allocate
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// The two-stage sum of eps_unbinarity (reduce.cuh: per-CTA partial sums, then one CTA per design adds them in a fixed
// order) needs scratch for the partial sums.  The plan's entry point keeps them in the caller-provided workspace; this one
// keeps them in a FILE-SCOPE DEVICE ARRAY of a fixed size, so it needs no workspace, no plan allocation and calls no
// cudaMalloc / cudaFree / allocating library routine: only two kernel launches.
//   - EPSGRAD_STATIC_PARTIALS floats (16 KB), resident on every GPU that loads the library until the process exits.
//   - In host code the array's NAME is a host-side stand-in, not a device address: its device address is taken once per
//     device with cudaGetSymbolAddress (with that device current) and that pointer is what the kernels get.
//   - Every call, from every plan and stream, shares the array.  A call first writes every slot it later reads, so the
//     contents a previous call left do not matter and nothing has to be cleared; but two calls that OVERLAP on the GPU
//     (different streams, or graph branches) race on it: callers serialise them.
// Same arithmetic in the same order as k_unbinarity / k_sum_partials: bitwise the same u.
#include <mutex>

#include "plan.cuh"
#include "common.cuh"
#include "sizes.cuh"

namespace epsgrad {

constexpr int EPSGRAD_STATIC_PARTIALS = 4096;          // floats: B * ceil(px py / 4096) must not exceed this (16.7 M mask pixels)
constexpr int NA_MAX_DEVICES = 64;

static __device__ __align__(256) float g_static_partials[EPSGRAD_STATIC_PARTIALS];

// sum over the CTA, valid in thread 0 (the order of reduce.cuh's block_sum)
__device__ __forceinline__ float na_block_sum(float v, float *scratch)
{
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    __syncthreads();
    if (lane == 0) scratch[warp] = v;
    __syncthreads();
    float s = 0.f;
    if (warp == 0) {
        s = lane < nw ? scratch[lane] : 0.f;
        for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    }
    return s;
}

// partial sums of sech^2(beta (x - eta_r)) = 4 rho (1 - rho) over the mask of design blockIdx.y; grid (n_part, B)
__global__ void __launch_bounds__(UB_THREADS) k_unbinarity_static(const float *x, size_t n_mask, float beta, float eta_r, float *part)
{
    __shared__ float scratch[32];
    const float *xb = x + (size_t)blockIdx.y * n_mask;
    const size_t base = (size_t)blockIdx.x * (UB_THREADS * UB_PER_THREAD) + threadIdx.x;
    float v = 0.f;
#pragma unroll 4
    for (int k = 0; k < UB_PER_THREAD; ++k) {
        const size_t i = base + (size_t)k * UB_THREADS;
        if (i < n_mask) {
            const float a = __expf(-2.0f * fabsf(beta * (xb[i] - eta_r)));     // sech^2 t = 4a/(1+a)^2, a = exp(-2|t|)
            const float d = fast_rcp(1.0f + a);
            v += 4.0f * a * d * d;
        }
    }
    const float s = na_block_sum(v, scratch);
    if (threadIdx.x == 0) part[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = s;
}

// u[b] = scale * sum_i part[b * n + i]; grid B, 256 threads
__global__ void __launch_bounds__(256) k_sum_static(const float *part, int n, float scale, float *u)
{
    __shared__ float scratch[32];
    float v = 0.f;
    for (int i = threadIdx.x; i < n; i += 256) v += part[(size_t)blockIdx.x * n + i];
    const float s = na_block_sum(v, scratch);
    if (threadIdx.x == 0) u[blockIdx.x] = scale * s;
}

// device address of the scratch array on `device` (current): looked up once per device
static std::mutex g_na_mutex;
static float *g_na_ptr[NA_MAX_DEVICES];

static int static_partials_ptr(int device, float **out)
{
    if (device < 0 || device >= NA_MAX_DEVICES) return EPSGRAD_EUNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[device]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_partials) != cudaSuccess || !p) { cudaGetLastError(); return EPSGRAD_ECUDA; }
        g_na_ptr[device] = static_cast<float *>(p);
    }
    *out = g_na_ptr[device];
    return EPSGRAD_OK;
}

}  // namespace epsgrad

using namespace epsgrad;

extern "C" int epsgrad_static_scratch_partials(void) { return EPSGRAD_STATIC_PARTIALS; }

extern "C" int eps_unbinarity_static(const epsgrad_plan_t *P, const float *phi, float beta, float *u, void *stream)
{
    if (!P || !phi || !u || !(beta > 0.0f) || !std::isfinite(beta)) return EPSGRAD_EINVAL;
    if (P->morph_R > 0) return EPSGRAD_EUNSUPPORTED;                   // the last projection's input is then not the filter output
    const size_t n_mask = (size_t)P->px * P->py;
    const size_t n_part = (n_mask + (size_t)UB_THREADS * UB_PER_THREAD - 1) / ((size_t)UB_THREADS * UB_PER_THREAD);
    if (n_part * (size_t)P->cfg.batch > (size_t)EPSGRAD_STATIC_PARTIALS || P->cfg.batch > 65535) return EPSGRAD_EUNSUPPORTED;
    DeviceGuard g(P->device);
    float *part = nullptr;
    int rc = static_partials_ptr(P->device, &part);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    k_unbinarity_static<<<dim3((unsigned)n_part, P->cfg.batch), UB_THREADS, 0, st>>>(phi, n_mask, beta, P->eta_r, part);
    if (cudaGetLastError() != cudaSuccess) return EPSGRAD_ECUDA;
    k_sum_static<<<P->cfg.batch, 256, 0, st>>>(part, (int)n_part, (float)(1.0 / (double)n_mask), u);
    return cudaGetLastError() == cudaSuccess ? EPSGRAD_OK : EPSGRAD_ECUDA;
}
