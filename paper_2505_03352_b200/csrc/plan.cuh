// plan.cuh -- the plan (epsgrad_plan_t of include/epsgrad.h) and the host-side launch layer's interface, shared by the
// translation units of the library: plan.cu (validation, tables, options), launch.cu (kernel launches, the schedules, the
// device entry points), hostpath.cu (the host-buffer entry point), optimizer.cu (Adam, SOAP, beta schedule).
// Host code only; no kernel is declared or defined here.
#pragma once
#include "../../include/epsgrad.h"

#include <cuda_runtime.h>
#include <cstddef>
#include <cstdint>

#define EPSGRAD_VERSION 100   /* 0.1.0 */
#define EPSGRAD_MAX_KERNELS 24
#define EPSGRAD_MAX_SMEM_KERNELS 48
#define EPSGRAD_MAX_HOST_PAIRS 64     /* field pairs per eps_forward_vjp_host call */

struct epsgrad_plan {
    epsgrad_config_t cfg;
    int device, n_sm;
    int nx, ny, px, py, m;
    int T, NT, KX, KY;
    int separable;
    int general;               // explicit cell counts, non-integer cells per control pixel: Eq. (2) by filter_general.cuh
    // device tables (one allocation)
    void *d_tables;
    float *d_w;                // conic [NT][NT][m][m] | separable [NT][m]
    int *d_tyrange;            // conic [NT][2]
    float *d_atc;              // tensor-core filter (filter_tc.cuh): banded weight matrices [2 (hi, lo)][NT][K/4][128][4], or nullptr
    float *d_att;              // transposed tensor-core filter (filterT_tc.cuh): weight slabs of the k-steps, two tf32 terms
    int use_tc;                // Eq. (2) forward on the tensor cores where d_atc exists (epsgrad_plan_set_tensor_cores)
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
    int eps_window_only;       // eps_forward rewrites only the slab window of every z column (epsgrad_plan_set_eps_window_only)
    int packed_fields;         // device E_F / E_A hold only the union slab window of every z column (epsgrad_plan_set_packed_fields)
    int use_tma;               // field windows by TMA bulk tensor copies where possible (epsgrad_plan_set_tma): 1 single-stage, 2 pipelined
    int use_pdl;               // programmatic dependent launch between consecutive kernels of a stream (epsgrad_plan_set_pdl)
    int pdl_valid, pdl_mark; cudaStream_t pdl_stream;     // the last operation of the call in flight was a kernel on pdl_stream that releases its dependents early
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
    size_t off_phi, off_v, off_gbar, off_e2d, off_coef, off_tmp, off_invden, ws_need;
    int last_launches;
    // kernels already opted in to their dynamic shared memory on this plan's device (launch.cu set_smem)
    const void *smem_fn[EPSGRAD_MAX_SMEM_KERNELS]; size_t smem_bytes[EPSGRAD_MAX_SMEM_KERNELS]; int n_smem_set;
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

namespace epsgrad {

struct DeviceGuard {
    int prev;
    explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline int cdiv(int a, int b) { return (a + b - 1) / b; }
inline bool aligned16(const void *p) { return p && !((uintptr_t)p & 15); }
inline size_t n_eps(const epsgrad_plan *P) { return (size_t)P->cfg.batch * 3 * P->nx * P->ny * P->cfg.nz; }
inline size_t n_ctrl(const epsgrad_plan *P) { return (size_t)P->cfg.batch * P->cfg.mx * P->cfg.my; }

// workspace planes
inline float *ws_phi(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_phi); }
inline float *ws_v(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_v); }
inline float *ws_m(const epsgrad_plan *P, int k) { return (float *)((char *)P->ws + P->off_m[k]); }
inline float *ws_mc(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_mc); }
inline float *ws_cot(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_cot); }
inline float *ws_part(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_part); }
inline float *ws_gbar(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_gbar); }
inline float *ws_e2d(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_e2d); }
inline float *ws_coef(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_coef); }
inline float *ws_tmp(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_tmp); }
inline float *ws_invden(const epsgrad_plan *P) { return (float *)((char *)P->ws + P->off_invden); }

// ---- launch layer (launch.cu).  Every function enqueues on `st` and returns an EPSGRAD_* status.
void begin_call(epsgrad_plan *P, cudaStream_t st);
int launch_front(epsgrad_plan *P, const float *C, float beta, cudaStream_t st);                       // F1 (+ morphological filters)
int launch_filter(epsgrad_plan *P, const float *C, float *phi, cudaStream_t st);
int launch_fwd2d(epsgrad_plan *P, const float *phi, float beta, float *e2d, float *coef, float *eps2d, cudaStream_t st);
int launch_extrude(epsgrad_plan *P, const float *e2d, float *eps, cudaStream_t st);
int launch_zreduce(epsgrad_plan *P, int n_pairs, const void *const *EF, const void *const *EA, float *gbar, cudaStream_t st,
                   bool host_src = false, bool packed = false);
int launch_maskgrad(epsgrad_plan *P, const float *phi, float beta, const float *gbar, const float *coef, float *v, cudaStream_t st);
int launch_morph_reverse(epsgrad_plan *P, const float *phi, float beta, float *v, cudaStream_t st);
int launch_filterT(epsgrad_plan *P, const float *v, float *dC, cudaStream_t st);
int run_chain(epsgrad_plan *P, const float *C, float beta, int n_pairs, const void *const *EF, const void *const *EA,
              float *eps, float *dFdC, cudaStream_t st);
// first chunk and number of chunks of the union of the two slab windows (x|y and z) of a field column
void window_union(const epsgrad_plan *P, int *first, int *count);

}  // namespace epsgrad
