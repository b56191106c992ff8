// hostpath.cu -- eps_forward_vjp_host: the path on HOST buffers (include/epsgrad.h), copies included.  Host code only: it
// stages through the plan's staging buffer and calls the launch layer (plan.cuh).
#include "plan.cuh"

#include <cmath>

using namespace epsgrad;

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
    if (n_pairs > EPSGRAD_MAX_HOST_PAIRS) return EPSGRAD_EUNSUPPORTED;
    if (P->emb.nx_full > 0 || P->slab_nx > 0 || P->packed_fields || P->eps_window_only) return EPSGRAD_EUNSUPPORTED;     // host buffers are region-sized, full z columns: no embedding, slab or packed windows here
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
    const void *ef[EPSGRAD_MAX_HOST_PAIRS], *ea[EPSGRAD_MAX_HOST_PAIRS];     // device-side addresses of the pairs
    bool ok = cudaMemcpyAsync(dC, C_host, b_c, cudaMemcpyHostToDevice, st) == cudaSuccess;
    P->last_h2d += b_c;
    // Eq. (1) needs only the slab cells of the fields ("|Omega_D").  When every field buffer is pinned, mapped host
    // memory, the z-reduction reads its windows straight out of it (16-byte asynchronous copies over PCIe / C2C) and the
    // rest of the fields never crosses the bus; otherwise (pageable memory, dense plans) the fields are staged whole.
    bool direct = P->host_direct && !P->dense && n_pairs > 0 && P->cfg.nz % 4 == 0;   // odd columns: staged whole (scalar3d.cuh)
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
        rc = launch_zreduce(P, n_pairs, ef, ea, ws_gbar(P), st, false, true);
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
            rc = launch_zreduce(P, n_pairs, ef, ea, ws_gbar(P), st, true);
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
    int rc = run_chain(P, dC, beta, n_pairs, ef, ea, eps_host ? dE : nullptr, dFdC_host ? dG : nullptr, st);
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

