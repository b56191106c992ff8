/*
 * epsgrad.h -- C ABI of the B200-native parametrization chain  C -> eps_hat  on the
 * Yee grid and of its reverse pass (arxiv 2505.03352, "Accelerated inverse design of
 * passive Si photonics").  "P:L<n>" = line n of the paper text; "S<n>" =
 * the readings of silent / ambiguous points listed in DESIGN.md section 3.
 *
 * What the library computes
 *   forward (Fig. 2/3):
 *     Eq. (2)  Phi  = sum_ab C_ab b(x-x_a, y-y_b)   on a mask with `subpixel` pixels per
 *              Yee cell (normalised density-filter form by default, S2)
 *     Eq. (3)/(6)  rho = 1/2 (1 + tanh(beta (Phi - eta)))
 *     Eq. (4)/(5)  optional morphological dilate / erode of rho, then Eq. (6)
 *     mixing   eps = rho eps_core + (1-rho) eps_clad
 *     Eq. (8)  cell averages <eps>, <1/eps> on the half-cell-shifted E_x/E_y/E_z
 *              footprints (finite sums on the mask)
 *     normals  Sobel operators at FDTD resolution, normalised
 *     Eq. (7)  eps_ii^-1 = n_i^2 <eps^-1> + (1-n_i^2) <eps>^-1
 *     z-extrusion to the slab [z_lo, z_hi] with fractional faces              P:L45 (S7, S8)
 *   reverse (Eq. (1); "VJP ... with arbitrary field"):
 *     dF/dC = -2 Re( (d eps_hat/dC)^T (E_F (.) E_A) ),  summed over field pairs;
 *     the product is the plain element-wise complex product.
 *
 * Conventions
 *   - All arrays are dense, row-major, last index fastest (component first).
 *       C     [B, Mx, My]             float32
 *       eps   [B, 3, Nx, Ny, Nz]      float32   (eps_xx, eps_yy, eps_zz), Nx = upsample*Mx
 *       E_F/A [B, 3, Nx, Ny, Nz]      complex64, interleaved (re, im) float32
 *       dFdC  [B, Mx, My]             float32, OVERWRITTEN with the sum over the pairs
 *   - Device entry points take DEVICE pointers (16-byte aligned) and enqueue all work on
 *     `stream` (a cudaStream_t passed as void*; NULL = the legacy default stream).  They
 *     never synchronise the host, never allocate, and never write an input.
 *   - *_host entry points take HOST pointers (pinned memory recommended), stage through
 *     the plan's staging buffer (epsgrad_plan_set_staging), enqueue H2D copies, the same
 *     kernels, and D2H copies on `stream`, and return without synchronising.  Pinned field
 *     buffers are read in place, slab windows only (epsgrad_plan_set_host_direct).
 *   - The caller owns every data buffer, the workspace and the staging buffer.  The
 *     library owns the plan: a host struct plus a few KB of device tables (filter
 *     weights, border normalisers, z weights) allocated in epsgrad_plan_create.
 *   - Every function returns an int status: 0 = EPSGRAD_OK, negative = error (below).
 *     No exceptions, no abort.  Asynchronous faults surface at the caller's next sync.
 *   - There is no CPU path.  Without a CUDA device plan creation fails with EPSGRAD_ECUDA.
 *   - A plan carries per-call state (launch accounting, the schedule's events): use one plan
 *     from one host thread at a time; different plans are independent.
 */
#ifndef EPSGRAD_H_
#define EPSGRAD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define EPSGRAD_OK             0
#define EPSGRAD_EINVAL        -1   /* null / misaligned pointer, bad size, beta <= 0, eps <= 0, a normalised filter whose
                                      support leaves a mask pixel without any control pixel (R <= (u - 1/s)/sqrt(2)), ... */
#define EPSGRAD_EUNSUPPORTED  -2   /* upsample*subpixel not in {2,4,6,8} (unless nx_cells, ny_cells are given), tables too large (conic filter: taps x
                                      phases beyond 200 KB of shared memory, e.g. R = 12 cells at 8 mask pixels per control pixel),
                                      morphological disk radius > 16 mask pixels or wider than the mask */
#define EPSGRAD_ENOWORKSPACE  -3   /* workspace / staging buffer missing or too small */
#define EPSGRAD_ECUDA         -4   /* CUDA runtime error (no device, launch failure) */
#define EPSGRAD_ENOMEM        -5   /* host allocation failed */

#define EPSGRAD_FILTER_CONIC     0 /* b = max(0, 1 - r/R)                              (S1)  */
#define EPSGRAD_FILTER_GAUSSIAN  1 /* b = exp(-r^2/2 sigma^2), |dx|,|dy| <= R per axis (S11) */

#define EPSGRAD_MAX_PAIRS 8        /* field pairs fused into one z-reduction launch; more are chained */

typedef struct epsgrad_plan epsgrad_plan_t;   /* opaque, library-owned */

/* Position of the design region inside a simulation domain (cells); see epsgrad_plan_set_embedding. */
typedef struct {
    int32_t nx_full, ny_full, nz_full;   /* the solver's grid                                         */
    int32_t i0, j0, k0;                  /* first cell of the design region in it (k0 % 4 == 0)       */
} epsgrad_embedding_t;

/* Geometry, filter and materials of a batch of B identical design regions (cell units). */
typedef struct {
    int32_t batch;            /* B >= 1 independent designs                                  */
    int32_t mx, my;           /* control grid (Eq. (2) nodes, pixel-centred; S3)             */
    int32_t upsample;         /* u: Yee cells per control pixel, Nx = u*Mx, Ny = u*My        */
    int32_t subpixel;         /* s: mask pixels per Yee cell per axis, even (S4; default 2)  */
    int32_t nz;               /* Yee cells in z (multiples of 4 take the 16-byte paths; any other nz a scalar one) */
    int32_t filter_kind;      /* EPSGRAD_FILTER_*                                            */
    int32_t filter_normalize; /* 1: density filter, renormalised at borders (S2); 0: raw Eq. (2) */
    int32_t nx_cells, ny_cells; /* 0, 0: Nx = upsample*Mx, Ny = upsample*My.  Otherwise the Yee cells of the design region, any
                                 numbers >= Mx, My: control node a sits at x_a = (Nx/Mx)(a + 1/2), a non-integer number of cells per
                                 control pixel (Fig. 4: 36 x 36 control variables on 210 x 210 cells).  Such plans run
                                 Eq. (2) and its transpose with weights evaluated on the fly (filter_general.cuh) and `upsample`
                                 is ignored; no x-slab, no persistent kernel for them                              */
    double  z_lo, z_hi;       /* slab extent in cell units, may be fractional (S8)           */
    double  filter_radius;    /* R in Yee cells                                              */
    double  filter_sigma;     /* Gaussian sigma in Yee cells                                 */
    double  eta;              /* projection threshold: 0.5 -> Eq. (6), 0 -> Eq. (3) (S9)     */
    double  eps_core, eps_clad;
    double  normal_delta;     /* guard in n_c^2 = g_c^2/(|g|^2 + delta) (S6).  Recommended (the binding's default) 1e-8: in
                                 float32 the Sobel differences of a flat mask carry noise^2 ~ 1e-14, so a guard near it turns
                                 rounding noise into normals.  Must be >= 1e-30: EPSGRAD_EINVAL below (0 and
                                 denormals would give n^2 = 0/0 on every flat cell) */
    double  morph_diameter;   /* d of Eqs. (4)-(5) in Yee cells (minimum feature size); 0 = morphological
                                 filters off.  On: rho0 = projection(Phi), "dilate, erode, erode, dilate" (
                                 S17) with the disk K_m normalised over the in-region pixels (S18), then Eq. (6) */
    double  morph_alpha;      /* alpha of Eqs. (4)-(5) (App. B: 20); used when morph_diameter > 0                */
} epsgrad_config_t;

/* ---- plan -------------------------------------------------------------------------- */
/* Validates cfg, builds the tables on `device`.  *out is set only on success.           */
int epsgrad_plan_create(const epsgrad_config_t *cfg, int device, epsgrad_plan_t **out);
int epsgrad_plan_destroy(epsgrad_plan_t *plan);

/* Scratch the device entry points need (filter output Phi, 2-D stage and reverse coefficient planes,
 * reduced cotangent, mask cotangent, separable-filter temporaries).  The caller allocates it (e.g. a torch
 * uint8 tensor) and keeps it alive and unshared while calls of this plan are in flight. */
size_t epsgrad_workspace_bytes(const epsgrad_plan_t *plan);
int    epsgrad_plan_set_workspace(epsgrad_plan_t *plan, void *dev_ptr, size_t bytes);

/* Device staging for the *_host entry points: C, dFdC, eps and n_pairs field pairs.     */
size_t epsgrad_staging_bytes(const epsgrad_plan_t *plan, int n_pairs);
int    epsgrad_plan_set_staging(epsgrad_plan_t *plan, void *dev_ptr, size_t bytes);

/* Reverse-pass field reads (P:L27 restricts Eq. (1) to Omega_D; in z only the slab cells
 * have d eps/dC != 0).  0 (default): read only the 16-byte chunks of each z column that
 * hold slab cells.  1: read every z cell (weights are zero outside the slab).  Results
 * are identical; this is a measurement switch.                                           */
int epsgrad_plan_set_dense_reads(epsgrad_plan_t *plan, int dense);

/* Two-stream schedule (default on).  The path has two HBM-bound kernels -- the Eq. (1) field reads, which depend
 * on nothing, and the eps stores -- and four small L2-resident ones.  Calls that compute dF/dC fork the plan's auxiliary
 * (high-priority) stream from `stream` (event) and run the small kernels there: filter -> 2-D chain beside the field reads,
 * then the 2-D reverse chain and the transposed filter beside the eps stores; the two HBM-bound kernels stay on `stream`,
 * which the auxiliary stream joins (event) before the call returns: to the caller everything is
 * still ordered on `stream`, with no host synchronisation, and the calls remain CUDA-graph capturable.  0 = one stream,
 * strictly serial (also used while per-kernel profiling is on).  Results are bitwise identical.                        */
int epsgrad_plan_set_overlap(epsgrad_plan_t *plan, int enable);

/* Number of kernel launches the last eps_* call of this plan enqueued (for accounting). */
int epsgrad_plan_last_launches(const epsgrad_plan_t *plan);

/* Per-kernel timing for roofline accounting.  When enabled, every eps_* / stage call also
 * records a CUDA event on `stream` before its first and after each of its kernels (at most
 * 24).  epsgrad_plan_last_kernel_times waits (host-blocking: the one exception to "never
 * synchronises") for the last call's events and returns the number n of kernels it
 * launched, writing ms[i] = device time between the events around kernel i (it includes
 * the launch gap before it) and names[i] = a static string naming the kernel; ms[i] = -1
 * when profiling was off.  Negative return = error.                                     */
int epsgrad_plan_set_profiling(epsgrad_plan_t *plan, int enable);
int epsgrad_plan_last_kernel_times(epsgrad_plan_t *plan, int max_n, float *ms, const char **names);

/* Timeline of one call (diagnostic; default off).  When enabled, a one-thread kernel that stores the device clock
 * (%globaltimer, ns) is enqueued at the start of a two-stream call and after each kernel on that kernel's stream (up to
 * 48 stamps), so the stamps show when each kernel of either stream ended.  epsgrad_plan_read_timeline synchronises the
 * device (host-blocking) and returns the number n of stamps of the last call with their names ("begin" or the kernel
 * whose end they mark).  The extra kernels perturb the schedule slightly; not for timed runs.                          */
int epsgrad_plan_set_timeline(epsgrad_plan_t *plan, int enable);
int epsgrad_plan_read_timeline(epsgrad_plan_t *plan, int max_n, uint64_t *ns, const char **names);

/* ---- the hot path (device pointers) -------------------------------------------------- */
/* eps_hat(C, beta): the whole forward chain.  beta > 0 (it changes every
 * iteration, Eq. (14), hence a call argument).                                    */
int eps_forward(epsgrad_plan_t *plan, const float *C, float beta, float *eps, void *stream);

/* Eq. (1): dFdC = -2 Re((d eps/dC)^T (E_F (.) E_A)) summed over n_pairs >= 1
 * pairs.  EF, EA: HOST arrays of n_pairs DEVICE pointers to complex64 [B,3,Nx,Ny,Nz].
 * A real cotangent w can be fed as E_F = -w/2 + 0i, E_A = 1 + 0i.
 * A z window of the field reads (the slab's cells; the whole column for dense plans) wider
 * than 512 cells takes the scalar kernel (region-sized or x-slab device arrays; embedded
 * or host-resident fields: EPSGRAD_EUNSUPPORTED).                                      */
int eps_vjp(epsgrad_plan_t *plan, const float *C, float beta, int n_pairs,
            const void *const *EF, const void *const *EA, float *dFdC, void *stream);

/* eps_vjp plus d F/d beta: eps_hat(C, beta) is differentiable with respect to the projection strength too;
 * dFdbeta: DEVICE array of B floats, dFdbeta[b] = -2 Re( (d eps_hat_b/d beta)^T (E_F (.) E_A) ) summed over the pairs.  With the
 * morphological filters on both projections contribute (S17).  Deterministic (two-stage sums, no atomics).               */
int eps_vjp_beta(epsgrad_plan_t *plan, const float *C, float beta, int n_pairs,
                 const void *const *EF, const void *const *EA, float *dFdC, float *dFdbeta, void *stream);

/* "Unbinarity" u(beta), the relative number of gray pixels of the design, read as the measure of non-discreteness
 * (S20): the mean over the design mask of 4 rho (1 - rho), rho the final projected mask; u: DEVICE array of B floats.   */
int eps_unbinarity(epsgrad_plan_t *plan, const float *C, float beta, float *u, void *stream);

/* The same u(beta) for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): of a mask the caller already holds -- phi: DEVICE array [B, s Nx, s Ny], the centred filter output
 * (what epsgrad_stage_filter writes) -- with the partial sums of the two-stage reduction in a file-scope device array of the
 * library instead of the plan's workspace.  The call needs no workspace and calls no cudaMalloc / cudaFree / allocating
 * library routine: two kernel launches on `stream`.  Bitwise the same u as eps_unbinarity (same sums in the same order).
 * LIMIT: the array holds epsgrad_static_scratch_partials() = 4096 floats (16 KB, resident on every GPU that loads the library
 * until exit): B * ceil(s Nx * s Ny / 4096) must not exceed it (16.7 M mask pixels in all; paper scale uses 245), else
 * EPSGRAD_EUNSUPPORTED -- as with the morphological filters on (the last projection's input is then not the filter output).
 * Every call, whatever its plan or stream, SHARES the array: a call writes every slot before it reads it, so what an earlier
 * call left does not matter, but calls that overlap on the GPU (different streams) race -- serialise them.              */
int eps_unbinarity_static(const epsgrad_plan_t *plan, const float *phi, float beta, float *u, void *stream);
int epsgrad_static_scratch_partials(void);

/* The paper's update rule for the projection strength (host scalars).  Eq. (14), P:L150:
 *   beta_i = beta_min + (beta_max - beta_min) (exp((i/N)^2) - 1)/(e - 1);
 * Eq. (15), moving averages with decay gamma that steer beta_max so that u reaches u0 at the last iteration:
 *   t <- gamma t + (1-gamma)(1/u - 1)/beta,   beta_max <- gamma beta_max + (1-gamma)(1/u0 - 1)/t.
 * epsgrad_beta_update returns EPSGRAD_EINVAL (and changes nothing) for u, u0, beta <= 0, gamma outside [0,1] or t <= 0.   */
double epsgrad_beta_schedule(double beta_min, double beta_max, int i, int n_iter);
int    epsgrad_beta_update(double *t, double *beta_max, double gamma, double u, double u0, double beta);

/* Adam, Eqs. (10)-(11): one step `step` >= 1, in place, on n control variables (DEVICE pointers; M, V the
 * moment buffers, zero before step 1; G the gradient of Eq. (1)).  Defaults of App. B: b1 .9, b2 .999, lr .001.
 *   M = b1 M + (1-b1) G,  V = b2 V + (1-b2) G^2,  C -= lr (M/(1-b1^step)) / (sqrt(V/(1-b2^step)) + eps)                     */
int epsgrad_adam_step(float *C, float *M, float *V, const float *G, size_t n, int step,
                      double b1, double b2, double lr, double eps, void *stream);

/* SOAP, Eqs. (12)-(13) (readings S21-S23 in DESIGN.md), on ONE [mx,my] matrix of control variables (a batch:
 * one set of buffers and calls per design).  All pointers DEVICE, row-major float32:
 *   C, M, G [mx,my]   control variables, first moment of Eq. (10) in the original basis (zero before step 1), gradient;
 *   Vp [mx,my]        second moment in the rotated basis (zero before step 1);
 *   L [mx,mx], R [my,my]   the accumulators of Eq. (12) (zero before step 1);
 *   QL [mx,mx], QR [my,my] their orthonormal eigenvectors as COLUMNS, Q[r][j] = component r of eigenvector j.
 * One optimizer iteration is: epsgrad_soap_accumulate; epsgrad_soap_eigh on L and on R (every iteration or every few: the
 * caller's choice, S23); epsgrad_soap_step.
 *   epsgrad_soap_accumulate   L <- b2 L + (1-b2) G G^T,  R <- b2 R + (1-b2) G^T G                              (Eq. (12))
 *   epsgrad_soap_eigh         Q, w <- eigenvectors / ascending eigenvalues [n] of the symmetric A [n,n] (A is not
 *                             written).  The library's one LIBRARY step (cuSOLVER syevd), loaded with dlopen on first use:
 *                             EPSGRAD_EUNSUPPORTED (and workspace_bytes = 0) when cuSOLVER is not on the machine.  Uses the
 *                             current device; the per-device solver handle is bound to `stream` and the solver enqueued
 *                             under one lock, so host threads may call it concurrently.  Eigenvector signs are the solver's:
 *                             they do not change the update (S23).  The solver's status word stays in `work`:
 *   epsgrad_soap_eigh_info    copies it to *info and synchronises `stream` (host-blocking): 0 = converged, i > 0 = i
 *                             off-diagonal elements of the tridiagonal form did not converge (Q is then not to be used).
 *   epsgrad_soap_step         M <- b1 M + (1-b1) G;  G' = QL^T G QR;  M' = QL^T M QR;  V' <- b2 V' + (1-b2) G'^2;
 *                             N' = (M'/(1-b1^step)) / sqrt(V'/(1-b2^step) + eps)  (eps inside the root, as printed);
 *                             C <- C - lr QL N' QR^T                                                           (Eq. (13))
 *                             Range of eps in float32: on the first steps L ~ G G^T and R ~ G^T G, so G' is diagonal up to
 *                             rounding and every other entry of N' is noise/sqrt(noise^2 + eps) with noise ~ 1e-7 |G|: the
 *                             update agrees with float64 (1e-4) for eps >= ~1e-2 mean(G^2) (what tests/test_gpu_soap.py and
 *                             test_gpu_loop.py use); at App. B's "small number" 1e-8 with |G| ~ 1 the
 *                             off-diagonal entries of the first update are wrong by ~1e-3 each.
 * `work` is caller-owned device scratch of at least the matching *_workspace_bytes.  Errors: EPSGRAD_EINVAL (null pointer,
 * size < 1, step < 1, b outside [0,1), lr <= 0, eps < 0), EPSGRAD_ENOWORKSPACE, EPSGRAD_ECUDA.  No host synchronisation.   */
int    epsgrad_soap_accumulate(float *L, float *R, const float *G, int mx, int my, double b2, void *stream);
size_t epsgrad_soap_eigh_workspace_bytes(int n);
int    epsgrad_soap_eigh(const float *A, float *Q, float *w, int n, void *work, size_t work_bytes, void *stream);
int    epsgrad_soap_eigh_info(const void *work, size_t work_bytes, int n, void *stream, int *info);
size_t epsgrad_soap_step_workspace_bytes(int mx, int my);
int    epsgrad_soap_step(float *C, float *M, float *Vp, const float *G, const float *QL, const float *QR, int mx, int my,
                         int step, double b1, double b2, double lr, double eps, void *work, size_t work_bytes, void *stream);

/* Both in one call; the filter output (Phi) is computed once and shared.                */
int eps_forward_vjp(epsgrad_plan_t *plan, const float *C, float beta, int n_pairs,
                    const void *const *EF, const void *const *EA,
                    float *eps, float *dFdC, void *stream);

/* ---- the same calls on HOST buffers (end-to-end path; copies included) --------------- */
/* eps_host / dFdC_host may be NULL to skip that output (and its work).  At most 64 pairs per call (EPSGRAD_EUNSUPPORTED beyond). */
int eps_forward_vjp_host(epsgrad_plan_t *plan, const float *C_host, float beta, int n_pairs,
                         const void *const *EF_host, const void *const *EA_host,
                         float *eps_host, float *dFdC_host, void *stream);
/* Embedding in a simulation domain (Eq. (1) restricts the fields to Omega_D; Fig. 4: a 210x210-cell design
 * region in a 430x450x64 model).  After this call the DEVICE entry points take eps, E_F and E_A as the solver's full arrays
 * [B, 3, nx_full, ny_full, nz_full]: the fields are read, and eps is written, only inside the block
 * [i0, i0+Nx) x [j0, j0+Ny) x [k0, k0+Nz); the rest of eps is not touched (it belongs to the solver).  z_lo, z_hi stay relative
 * to k0.  NULL switches back to region-sized arrays.  Needs nz_full % 4 == 0 and k0 % 4 == 0 (16-byte pieces), else
 * EPSGRAD_EUNSUPPORTED; a block that sticks out of the domain is EPSGRAD_EINVAL.  epsgrad_stage_zreduce follows the embedding
 * (its fields are the solver's arrays); the *_host entry points keep region-sized buffers and return EPSGRAD_EUNSUPPORTED
 * while an embedding is set.                                                                                              */
int epsgrad_plan_set_embedding(epsgrad_plan_t *plan, const epsgrad_embedding_t *embedding);

/* x-slab of a region shared by several GPUs (default off).  The plan's region is this rank's rows of a larger
 * design plus a halo wide enough for the dependency cone (filter radius + 3 cells on either side), but the
 * caller's eps / E_F / E_A hold only the rows it owns: [B,3,x_count,Ny,Nz] = Yee rows [x_first, x_first + x_count) of the
 * region.  eps is written and the fields are read on those rows only; every other row of the region contributes nothing to
 * dFdC, which stays region-sized (partial: the ranks' gradients add; the halo parts overlap the neighbours' controls).
 * (0, 0) switches back.  EPSGRAD_EINVAL for a range outside the region; EPSGRAD_EUNSUPPORTED together with an embedding and
 * in the *_host entry points.                                                                                              */
int epsgrad_plan_set_slab(epsgrad_plan_t *plan, int x_first, int x_count);

/* Fields on the design region only (Eq. (1) is restricted to Omega_D, and in z the design region is the slab).  After
 * epsgrad_plan_set_packed_fields(plan, 1) the DEVICE entry points take every E_F / E_A as [B, 3, Nx, Ny, n_cells] complex64:
 * the z cells [first_cell, first_cell + n_cells) of each column, contiguous -- the union of the slab windows of the x|y and z
 * components, rounded to 16-byte pieces (two cells), as epsgrad_plan_packed_window returns them (paper scale: cells 26..35 of
 * 64).  This is what a solver holds when it accumulates its frequency-domain fields on Omega_D only; the field stream then
 * reads one dense array (80 instead of 512 bytes per column, no half-used fills).  Same arithmetic in the same order as with
 * full columns: bitwise the same dFdC.  eps is unaffected (full columns).  EPSGRAD_EUNSUPPORTED together with an embedding, an
 * x-slab, dense reads or nz % 4 != 0, and in the *_host entry point (which gathers the windows itself).                      */
int epsgrad_plan_set_packed_fields(epsgrad_plan_t *plan, int enable);

/* eps on the design region only (the layout is extruded to the device layer; every cell of a z column outside the slab
 * is eps_clad whatever C and beta are).  After epsgrad_plan_set_eps_window_only(plan, 1) the DEVICE entry points rewrite only
 * the z cells of every column that depend on the design -- the union of the slab windows of the three components, rounded
 * outwards to whole 32-byte sectors (paper scale: cells 24..39 of 64) -- and touch nothing else of `eps`.  The caller's eps
 * array must therefore already hold the result of ONE earlier full call (enable = 0) of the same plan geometry: a design loop
 * makes its first eps_forward a full one and every later one a window one (48 instead of 192 MB stored per call at paper
 * scale).  Inside the window the bits are those of the full call.  EPSGRAD_EUNSUPPORTED when nz % 4 != 0 and in the *_host
 * entry point (its eps buffer is written whole).  Works with an embedding and with x-slabs.                              */
int epsgrad_plan_set_eps_window_only(epsgrad_plan_t *plan, int enable);
int epsgrad_plan_packed_window(const epsgrad_plan_t *plan, int *first_cell, int *n_cells);

/* How the device-resident field windows are fetched.  0: by 16-byte asynchronous copies (LDGSTS), 5 CTAs per SM.
 * 1: by the tensor memory accelerator, one bulk tensor copy per field and 256 columns, one stage per CTA (region-sized
 * fields with sparse windows only; other cases fall back).  2: thin persistent read stream -- one CTA per SM, TMA copies
 * through a ring of shared-memory stages with full / empty mbarriers (region-sized or x-slab fields; embedded, packed and
 * host-resident fields fall back to 0).  Same bytes, bitwise the same results; a measurement switch.
 * EPSGRAD_EUNSUPPORTED when TMA descriptors cannot be built on this driver.                                               */
int epsgrad_plan_set_tma(epsgrad_plan_t *plan, int mode);

/* Eq. (2) and its transpose on the tensor cores (tcgen05.mma kind::tf32, accumulators in tensor memory; both operands split
 * into two tf32 terms and three products accumulated in float32; filter_tc.cuh, filterT_tc.cuh).  Applies to the conic filter
 * with upsample * subpixel = 4 and R <= 12 cells (EPSGRAD_EUNSUPPORTED when set on another plan).  Mode 2 (default on such
 * plans): where each kernel measured faster than its FFMA stencil, i.e. on control grids with enough tiles for every SM --
 * the filter from ~500 x 500 control pixels at R = 12 (55 us against 158 us at 1000 x 1000) and from ~375 x 375 at R <= 8
 * (52 against 97 us at 1000 x 1000); its transpose from ~500 x 500 at R = 12 (112 against 203 us at 1000 x 1000) and at
 * 1000 x 1000 for R <= 8 (87 against 125 us).  1: wherever they apply; 0: never (filter4.cuh).  The tensor core's float32
 * accumulation is coarser than FFMA's: measured against the oracle, eps errors grow from 7e-7 to 3.3e-6 at beta = 64
 * (tolerance 1e-5); dF/dC differs from the FFMA kernel's by <= 2.5e-6 of its largest entry (tolerance 1e-4).              */
int epsgrad_plan_set_tensor_cores(epsgrad_plan_t *plan, int enable);

/* Programmatic dependent launch (default on).  Consecutive kernels of a stream -- filter -> 2-D stage (-> eps stores in
 * eps_forward), mask cotangent -> transposed filter -- are launched with the programmatic-stream-serialization attribute: the
 * next kernel's CTAs are scheduled, and stage their tables, while the previous kernel drains, and wait (griddepcontrol.wait)
 * before they read what it wrote.  Bitwise the same results; 0 = plain stream order.  CUDA-graph capturable either way.   */
int epsgrad_plan_set_pdl(epsgrad_plan_t *plan, int enable);

/* How eps is written.  0: per-thread 16-byte streaming stores (k_extrude).  1: thin persistent store stream -- the columns
 * are assembled in shared memory (only the slab pieces change from column to column) and written by bulk asynchronous copies
 * (region-sized or x-slab eps; embedded plans fall back to 0).  Bitwise the same results; a measurement switch.           */
int epsgrad_plan_set_bulk_stores(epsgrad_plan_t *plan, int enable);

/* One persistent dataflow kernel for the whole call (default on where it applies).  The six steps of the path are cut into
 * tiles and column blocks grouped in bands of 16 Yee rows; one launch of co-resident CTAs takes them from two ticket lists
 * (the two HBM streams; the 2-D work) and runs each as soon as the bands it depends on are complete, so that the ALU-bound
 * 2-D tiles execute on the same SMs while the memory-bound blocks wait for DRAM, there are no launch ramps between steps, and
 * every intermediate is consumed from L2 a few bands after it was produced, at any problem size.  Applies to the conic filter
 * with upsample * subpixel = 4, subpixel = 2, R <= 12 cells, morphological filters off, up to EPSGRAD_MAX_PAIRS pairs, device
 * buffers, no x-slab, no eps_vjp_beta; every other call runs the step as separate kernels (0 forces that everywhere).
 * EPSGRAD_EUNSUPPORTED when enabled on a plan it does not apply to.  Results equal the separate kernels' except for the
 * summation order of the filter taps (two partial sums per pixel instead of three).                                      */
int epsgrad_plan_set_fused(epsgrad_plan_t *plan, int enable);

/* Cycle accounting of the persistent kernel (diagnostic; default off).  enable != 0 allocates and clears 20 device counters that
 * every CTA of the following fused calls adds to: [0..5] SM cycles spent in the items of each of the six phases (F1, F2, X, M, T,
 * Z), [6..11] the number of items of each phase, [12] cycles spent taking and decoding tickets (and starting field copies),
 * [13] total CTA cycles, [14] cycles spent waiting for bands, [15] cycles in the release that publishes an item, [16] cycles starting field copies, [17] cycles in the barrier that ends a round, [18..19] reserved.  out20 != NULL:
 * synchronises the device (host-blocking) and returns the counters accumulated so far before clearing them.               */
int epsgrad_plan_fused_profile(epsgrad_plan_t *plan, int enable, uint64_t *out20);

/* Measurement knobs of the two stream kernels (0 = the default of each): knob 0 = bytes per bulk store, 1 = store-stream
 * CTAs per SM, 2 = stages of the read stream's ring, 3 = read-stream CTAs per SM; 4 = CTAs per SM of the persistent kernel, 6 = pipeline lag (steps) between a phase of the persistent kernel and its consumer; 5 = L2 evict-first policy of the field fills (0: on for field arrays up to 4 GB per launch, the default; 1: always; 2: never); 7 = force streamed tensor-core weights.  EPSGRAD_EINVAL for a
 * knob outside 0..7.  Values are clamped to what the kernels support; results never depend on them.                      */
int epsgrad_plan_set_tuning(epsgrad_plan_t *plan, int knob, int value);

/* Field transfer of the *_host entry points (mode; default 2).  Eq. (1) needs only the slab cells of the fields (P:L27:
 * only Omega_D enters the gradient), so when every field buffer is pinned, mapped host memory (and the plan is not in
 * dense-read mode) the rest of the fields never crosses the bus:
 *   1: the Eq. (1) reduction reads its slab windows straight out of host memory;
 *   2: as 1 for calls that return the gradient only; calls that also return eps gather the union slab window of every z
 *      column into the staging buffer with one strided copy per field on the copy engine, beside the eps transfer in the
 *      other direction (4 % faster than 1 at paper scale);
 *   0: every field is copied whole into the staging buffer first (also the fallback for buffers that are not pinned).
 * Results are identical in all modes.                                                                                    */
int epsgrad_plan_set_host_direct(epsgrad_plan_t *plan, int enable);
/* bytes the last *_host call copied host->device and device->host                       */
int epsgrad_plan_last_copy_bytes(const epsgrad_plan_t *plan, uint64_t *h2d, uint64_t *d2h);

/* ---- stage taps (device pointers; for stage-by-stage parity tests) ------------------- */
/* Phi - eta0 on the mask [B, s*Nx, s*Ny] (eta0 = eta if filter_normalize else 0).       */
int epsgrad_stage_filter(epsgrad_plan_t *plan, const float *C, float *phi_centred, void *stream);
/* eps2d [B,3,Nx,Ny]: the 2-D stage before z-extrusion (steps 1-6).                      */
int epsgrad_stage_eps2d(epsgrad_plan_t *plan, const float *C, float beta, float *eps2d, void *stream);
/* z-reduced cotangent [B,5,Nx,Ny]: planes x, y, z(full cells), z(lower face), z(upper face). */
int epsgrad_stage_zreduce(epsgrad_plan_t *plan, int n_pairs, const void *const *EF,
                          const void *const *EA, float *gbar, void *stream);

const char *epsgrad_status_string(int status);
/* library version: major*10000 + minor*100 + patch */
int epsgrad_version(void);

#ifdef __cplusplus
}
#endif
#endif /* EPSGRAD_H_ */
