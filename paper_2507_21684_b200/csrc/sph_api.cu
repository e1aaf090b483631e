// sph_api.cu -- context life cycle, error reporting and the host-buffer end-to-end entry point of include/sph.h.
#include "sph_internal.cuh"

#include <new>

extern "C" int sph_create(sph_ctx **out, int device, int64_t n_max)
{
    if (!out || n_max < 0) return SPH_E_INVALID;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) {
        (void)cudaGetLastError();
        return SPH_E_CUDA;                  // no CUDA device: there is no CPU fallback
    }
    SPH_CUDA_TRY(cudaSetDevice(device));
    sph_ctx *ctx = new (std::nothrow) sph_ctx();
    if (!ctx) return SPH_E_NOMEM;
    ctx->device = device;
    ctx->n_hint = n_max;
    if (cudaMallocHost((void **)&ctx->h_pinned, 64 * sizeof(int64_t)) != cudaSuccess) {
        (void)cudaGetLastError();
        delete ctx;
        return SPH_E_NOMEM;
    }
    *out = ctx;
    return SPH_OK;
}

extern "C" int sph_destroy(sph_ctx *ctx)
{
    if (!ctx) return SPH_E_INVALID;
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    DevBuf *bufs[] = {&ctx->key_a, &ctx->key_b, &ctx->idx_a, &ctx->idx_b, &ctx->hist, &ctx->perm, &ctx->inv_perm,
                      &ctx->key_sorted, &ctx->pos_s, &ctx->cell_start, &ctx->cell_end, &ctx->stats, &ctx->cnt,
                      &ctx->row_ptr, &ctx->col, &ctx->col16, &ctx->scan_tmp, &ctx->maskbuf, &ctx->tile_words, &ctx->tile_mask_base, &ctx->fstats, &ctx->tstate, &ctx->fctl, &ctx->tile_tabs, &ctx->d_pos, &ctx->d_va, &ctx->d_mom, &ctx->d_g4, &ctx->d_lr, &ctx->d_dx4, &ctx->d_gb4, &ctx->d_rb, &ctx->d_rc, &ctx->d_rd, &ctx->d_re, &ctx->d_x2, &ctx->d_vb, &ctx->d_ab, &ctx->d_part, &ctx->tile_orders[0].buf, &ctx->tile_orders[1].buf, &ctx->tile_orders[2].buf, &ctx->tile_orders[3].buf, &ctx->s0, &ctx->s1, &ctx->s2, &ctx->s3, &ctx->c0buf,
                      &ctx->out4, &ctx->m_s, &ctx->kind_s, &ctx->partials, &ctx->eos, &ctx->hx, &ctx->hv, &ctx->hrho,
                      &ctx->hm, &ctx->hh, &ctx->hkind, &ctx->hlam, &ctx->hmu, &ctx->ho_drho, &ctx->ho_acc, &ctx->ho_xb,
                      &ctx->ho_vb, &ctx->ho_rb, &ctx->ho_pb, &ctx->ho_dens};
    for (DevBuf *b : bufs) b->release();
    for (auto &b : ctx->rk) b.release();
    if (ctx->h_pinned) cudaFreeHost(ctx->h_pinned);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->ev_in) cudaEventDestroy(ctx->ev_in);
    if (ctx->ev_out) cudaEventDestroy(ctx->ev_out);
    for (int c = 0; c < 4; ++c)
        if (ctx->ev_final[c]) cudaEventDestroy(ctx->ev_final[c]);
    if (ctx->ev_final_x) cudaEventDestroy(ctx->ev_final_x);
    for (const ProfRec &r : ctx->prof.live) {
        cudaEventDestroy(r.a);
        cudaEventDestroy(r.b);
    }
    for (cudaEvent_t e : ctx->prof.pool) cudaEventDestroy(e);
    (void)cudaGetLastError();
    delete ctx;
    return SPH_OK;
}

extern "C" int sph_check(sph_ctx *ctx)
{
    if (!ctx) return SPH_E_INVALID;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    SPH_CUDA_TRY(cudaStreamSynchronize(ctx->last_stream));
    if (!ctx->stats.p) return SPH_OK;
    uint32_t flag = 0;
    SPH_CUDA_TRY(cudaMemcpy(&flag, ctx->stats.p, 4, cudaMemcpyDeviceToHost));
    return flag ? SPH_E_DOMAIN : SPH_OK;
}

#ifdef SPH_BOUNDS
unsigned int sph_bounds_read_fused();
unsigned int sph_bounds_read_pairs_tile();
#endif
// violations counted by the checked accesses of a -DSPH_BOUNDS build since the library was loaded; -1 in a normal build
extern "C" int sph_debug_bounds_violations(sph_ctx *ctx, int64_t *count)
{
    if (!ctx || !count) return SPH_E_INVALID;
#ifdef SPH_BOUNDS
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    SPH_CUDA_TRY(cudaDeviceSynchronize());
    *count = (int64_t)sph_bounds_read_fused() + (int64_t)sph_bounds_read_pairs_tile();
#else
    *count = -1;
#endif
    return SPH_OK;
}

extern "C" const char *sph_strerror(int code)
{
    switch (code) {
    case SPH_OK: return "ok";
    case SPH_E_INVALID: return "invalid argument";
    case SPH_E_DOMAIN: return "domain error (cell size / periodic cells / position outside a bounded axis)";
    case SPH_E_STATE: return "call order violated";
    case SPH_E_NOMEM: return "out of memory";
    case SPH_E_CUDA: return "CUDA runtime error (or no CUDA device: this library has no CPU fallback)";
    case SPH_E_TOO_LARGE: return "size beyond the fixed capacity of an allocation-free entry point";
    default: return "unknown error";
    }
}

extern "C" int sph_get_info(sph_ctx *ctx, int32_t ncell[3], int64_t *n, int64_t *nnz, int64_t *launches)
{
    if (!ctx) return SPH_E_INVALID;
    if (ncell)
        for (int k = 0; k < 3; ++k) ncell[k] = ctx->geom.ncell[k];
    if (n) *n = ctx->n;
    if (nnz) *nnz = ctx->lists_ready ? ctx->nnz : 0;
    if (launches) *launches = ctx->launches;
    return SPH_OK;
}

extern "C" int sph_get_layout(sph_ctx *ctx, int32_t *mode, int32_t *tile_edge, int64_t *halo_max, int64_t *rows_max)
{
    if (!ctx) return SPH_E_INVALID;
    if (!ctx->lists_ready) return SPH_E_STATE;
    if (mode) *mode = ctx->tile_mode ? 2 : 1;
    if (tile_edge) *tile_edge = ctx->tile_mode ? ctx->tg.B : 0;
    if (halo_max) *halo_max = ctx->tile_mode ? (int64_t)ctx->tile_Mmax : 0;
    if (rows_max) *rows_max = ctx->tile_mode ? (int64_t)ctx->tile_Tmax : 0;
    return SPH_OK;
}

extern "C" int sph_forward_backward_host(sph_ctx *ctx, const sph_domain *dom, const sph_params *par, float search_scale,
                                         int64_t n, const float *x, const float *v, const float *rho, const float *m,
                                         const float *h, const uint8_t *kind, const float *drho_bar, const float *acc_bar,
                                         float *drho_dt, float *acc, float *x_bar, float *v_bar, float *rho_bar,
                                         float *params_bar, int64_t *nnz_out)
{
    if (!ctx || !dom || !par || n <= 0 || !x || !v || !rho || !m || !h || !kind || !drho_bar || !acc_bar) return SPH_E_INVALID;
    if (dom->dim != 2 && dom->dim != 3) return SPH_E_INVALID;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = nullptr;
    const size_t nv = (size_t)n * dom->dim * 4, ns = (size_t)n * 4;
    SPH_TRY(ctx->hx.reserve(nv));  SPH_TRY(ctx->hv.reserve(nv));  SPH_TRY(ctx->hrho.reserve(ns));
    SPH_TRY(ctx->hm.reserve(ns));  SPH_TRY(ctx->hh.reserve(ns));  SPH_TRY(ctx->hkind.reserve((size_t)n));
    SPH_TRY(ctx->hlam.reserve(ns)); SPH_TRY(ctx->hmu.reserve(nv));
    SPH_TRY(ctx->ho_drho.reserve(ns)); SPH_TRY(ctx->ho_acc.reserve(nv)); SPH_TRY(ctx->ho_xb.reserve(nv));
    SPH_TRY(ctx->ho_vb.reserve(nv)); SPH_TRY(ctx->ho_rb.reserve(ns)); SPH_TRY(ctx->ho_pb.reserve(64));
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->hx.p, x, nv, cudaMemcpyHostToDevice, st));
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->hv.p, v, nv, cudaMemcpyHostToDevice, st));
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->hrho.p, rho, ns, cudaMemcpyHostToDevice, st));
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->hm.p, m, ns, cudaMemcpyHostToDevice, st));
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->hh.p, h, ns, cudaMemcpyHostToDevice, st));
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->hkind.p, kind, (size_t)n, cudaMemcpyHostToDevice, st));
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->hlam.p, drho_bar, ns, cudaMemcpyHostToDevice, st));
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->hmu.p, acc_bar, nv, cudaMemcpyHostToDevice, st));
    SPH_TRY(sph_build_cells(ctx, dom, ctx->hx.as<float>(), ctx->hh.as<float>(), n, (sph_stream_t)st));
    SPH_TRY(sph_neighbors(ctx, search_scale, nnz_out, (sph_stream_t)st));
    SPH_TRY(sph_rhs(ctx, par, ctx->hx.as<float>(), ctx->hv.as<float>(), ctx->hrho.as<float>(), ctx->hm.as<float>(),
                    ctx->hkind.as<uint8_t>(), ctx->ho_drho.as<float>(), ctx->ho_acc.as<float>(), (sph_stream_t)st));
    SPH_TRY(sph_rhs_vjp(ctx, par, ctx->hx.as<float>(), ctx->hv.as<float>(), ctx->hrho.as<float>(), ctx->hm.as<float>(),
                        ctx->hkind.as<uint8_t>(), ctx->hlam.as<float>(), ctx->hmu.as<float>(), ctx->ho_xb.as<float>(),
                        ctx->ho_vb.as<float>(), ctx->ho_rb.as<float>(), ctx->ho_pb.as<float>(), (sph_stream_t)st));
    if (drho_dt) SPH_CUDA_TRY(cudaMemcpyAsync(drho_dt, ctx->ho_drho.p, ns, cudaMemcpyDeviceToHost, st));
    if (acc) SPH_CUDA_TRY(cudaMemcpyAsync(acc, ctx->ho_acc.p, nv, cudaMemcpyDeviceToHost, st));
    if (x_bar) SPH_CUDA_TRY(cudaMemcpyAsync(x_bar, ctx->ho_xb.p, nv, cudaMemcpyDeviceToHost, st));
    if (v_bar) SPH_CUDA_TRY(cudaMemcpyAsync(v_bar, ctx->ho_vb.p, nv, cudaMemcpyDeviceToHost, st));
    if (rho_bar) SPH_CUDA_TRY(cudaMemcpyAsync(rho_bar, ctx->ho_rb.p, ns, cudaMemcpyDeviceToHost, st));
    if (params_bar) SPH_CUDA_TRY(cudaMemcpyAsync(params_bar, ctx->ho_pb.p, 40, cudaMemcpyDeviceToHost, st));
    SPH_CUDA_TRY(cudaStreamSynchronize(st));
    return sph_check(ctx);
}

extern "C" int sph_step_host(sph_ctx *ctx, const sph_domain *dom, const sph_domain *dom_rk, const sph_params *par,
                             float dt, float skin, int64_t n, float *x, float *v, float *rho, const float *m,
                             const float *h, const uint8_t *kind, const float *drho_bar, const float *acc_bar,
                             float *density, float *drho_dt, float *acc, float *x_bar, float *v_bar, float *rho_bar,
                             float *params_bar, int64_t *nnz_out)
{
    if (!ctx || !dom || !dom_rk || !par || n <= 0 || !x || !v || !rho || !m || !h || !kind || !drho_bar || !acc_bar)
        return SPH_E_INVALID;
    if ((dom->dim != 2 && dom->dim != 3) || dom_rk->dim != dom->dim) return SPH_E_INVALID;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    cudaStream_t st = nullptr;
    sph_stream_t ss = (sph_stream_t)st;
    const size_t nv = (size_t)n * dom->dim * 4, ns = (size_t)n * 4;
    SPH_TRY(ctx->hx.reserve(nv));  SPH_TRY(ctx->hv.reserve(nv));  SPH_TRY(ctx->hrho.reserve(ns));
    SPH_TRY(ctx->hm.reserve(ns));  SPH_TRY(ctx->hh.reserve(ns));  SPH_TRY(ctx->hkind.reserve((size_t)n));
    SPH_TRY(ctx->hlam.reserve(ns)); SPH_TRY(ctx->hmu.reserve(nv));
    SPH_TRY(ctx->ho_drho.reserve(ns)); SPH_TRY(ctx->ho_acc.reserve(nv)); SPH_TRY(ctx->ho_xb.reserve(nv));
    SPH_TRY(ctx->ho_vb.reserve(nv)); SPH_TRY(ctx->ho_rb.reserve(ns)); SPH_TRY(ctx->ho_pb.reserve(64));
    SPH_TRY(ctx->ho_dens.reserve(ns));
    float *dx = ctx->hx.as<float>(), *dv = ctx->hv.as<float>(), *dr = ctx->hrho.as<float>(), *dm = ctx->hm.as<float>();
    float *dh = ctx->hh.as<float>();
    uint8_t *dk = ctx->hkind.as<uint8_t>();
    // Copies off the critical path run on a second (non-blocking) stream: the cotangents and v, rho, m, kind arrive while
    // the cells and lists are built from x and h; the seven results of the first half leave while sph_rk_step runs.
    if (!ctx->copy_stream) {
        SPH_CUDA_TRY(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        SPH_CUDA_TRY(cudaEventCreateWithFlags(&ctx->ev_in, cudaEventDisableTiming));
        SPH_CUDA_TRY(cudaEventCreateWithFlags(&ctx->ev_out, cudaEventDisableTiming));
    }
    cudaStream_t cs = ctx->copy_stream;
    SPH_CUDA_TRY(cudaStreamSynchronize(st));                      // the staging buffers of the previous call are free
    SPH_CUDA_TRY(cudaMemcpyAsync(dx, x, nv, cudaMemcpyHostToDevice, st));
    SPH_CUDA_TRY(cudaMemcpyAsync(dh, h, ns, cudaMemcpyHostToDevice, st));
    SPH_CUDA_TRY(cudaMemcpyAsync(dm, m, ns, cudaMemcpyHostToDevice, cs));
    SPH_CUDA_TRY(cudaMemcpyAsync(dv, v, nv, cudaMemcpyHostToDevice, cs));
    SPH_CUDA_TRY(cudaMemcpyAsync(dr, rho, ns, cudaMemcpyHostToDevice, cs));
    SPH_CUDA_TRY(cudaMemcpyAsync(dk, kind, (size_t)n, cudaMemcpyHostToDevice, cs));
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->hlam.p, drho_bar, ns, cudaMemcpyHostToDevice, cs));
    SPH_CUDA_TRY(cudaMemcpyAsync(ctx->hmu.p, acc_bar, nv, cudaMemcpyHostToDevice, cs));
    SPH_CUDA_TRY(cudaEventRecord(ctx->ev_in, cs));
    int64_t nnz0 = 0;
    // whatever path leaves this function, a later sph_rk_step must not take lists prepared here for its own
    struct PreparedGuard {
        sph_ctx *c;
        ~PreparedGuard() { c->rk_lists_prepared = false; c->rk_final_chunks = 1; }
    } prepared_guard{ctx};
    SPH_TRY(sph_build_cells(ctx, dom, dx, dh, n, ss));
    SPH_TRY(sph_neighbors(ctx, 1.0f, &nnz0, ss));
    SPH_CUDA_TRY(cudaStreamWaitEvent(st, ctx->ev_in, 0));
    SPH_TRY(sph_density(ctx, dm, ctx->ho_dens.as<float>(), ss));
    SPH_TRY(sph_rhs(ctx, par, dx, dv, dr, dm, dk, ctx->ho_drho.as<float>(), ctx->ho_acc.as<float>(), ss));
    SPH_TRY(sph_rhs_vjp(ctx, par, dx, dv, dr, dm, dk, ctx->hlam.as<float>(), ctx->hmu.as<float>(), ctx->ho_xb.as<float>(),
                        ctx->ho_vb.as<float>(), ctx->ho_rb.as<float>(), ctx->ho_pb.as<float>(), ss));
    SPH_CUDA_TRY(cudaEventRecord(ctx->ev_out, st));
    // the lists of the RK4 step first: their build reads a few words back, and those read-backs must not queue behind
    // the 100 MB of results in the device-to-host copy engine
    SPH_TRY(sph_rk_prepare_lists(ctx, dom_rk, skin, dx, dh, n, st));
    SPH_CUDA_TRY(cudaStreamWaitEvent(cs, ctx->ev_out, 0));
    if (density) SPH_CUDA_TRY(cudaMemcpyAsync(density, ctx->ho_dens.p, ns, cudaMemcpyDeviceToHost, cs));
    if (drho_dt) SPH_CUDA_TRY(cudaMemcpyAsync(drho_dt, ctx->ho_drho.p, ns, cudaMemcpyDeviceToHost, cs));
    if (acc) SPH_CUDA_TRY(cudaMemcpyAsync(acc, ctx->ho_acc.p, nv, cudaMemcpyDeviceToHost, cs));
    if (x_bar) SPH_CUDA_TRY(cudaMemcpyAsync(x_bar, ctx->ho_xb.p, nv, cudaMemcpyDeviceToHost, cs));
    if (v_bar) SPH_CUDA_TRY(cudaMemcpyAsync(v_bar, ctx->ho_vb.p, nv, cudaMemcpyDeviceToHost, cs));
    if (rho_bar) SPH_CUDA_TRY(cudaMemcpyAsync(rho_bar, ctx->ho_rb.p, ns, cudaMemcpyDeviceToHost, cs));
    if (params_bar) SPH_CUDA_TRY(cudaMemcpyAsync(params_bar, ctx->ho_pb.p, 40, cudaMemcpyDeviceToHost, cs));
    // the advanced state leaves in ranges of caller indices, each as soon as its part of the final update is done
    constexpr int kFinalChunks = 4;
    for (int c = 0; c < kFinalChunks; ++c)
        if (!ctx->ev_final[c]) SPH_CUDA_TRY(cudaEventCreateWithFlags(&ctx->ev_final[c], cudaEventDisableTiming));
    if (!ctx->ev_final_x) SPH_CUDA_TRY(cudaEventCreateWithFlags(&ctx->ev_final_x, cudaEventDisableTiming));
    ctx->rk_final_chunks = kFinalChunks;
    const int rc_rk = sph_rk_step(ctx, dom_rk, par, dt, skin, n, dx, dv, dr, dm, dh, dk, ss);
    SPH_TRY(rc_rk);
    if (nnz_out) {
        nnz_out[0] = nnz0;
        nnz_out[1] = ctx->nnz;
    }
    // the new positions were complete before the last right-hand side started: they leave while it runs
    SPH_CUDA_TRY(cudaStreamWaitEvent(cs, ctx->ev_final_x, 0));
    SPH_CUDA_TRY(cudaMemcpyAsync(x, dx, nv, cudaMemcpyDeviceToHost, cs));
    for (int c = 0; c < kFinalChunks; ++c) {
        const int64_t i0 = n * c / kFinalChunks, i1 = n * (c + 1) / kFinalChunks;
        SPH_CUDA_TRY(cudaStreamWaitEvent(cs, ctx->ev_final[c], 0));
        if (i1 <= i0) continue;
        const size_t ov = (size_t)i0 * dom->dim, cv = (size_t)(i1 - i0) * dom->dim * 4, cs1 = (size_t)(i1 - i0) * 4;
        SPH_CUDA_TRY(cudaMemcpyAsync(v + ov, dv + ov, cv, cudaMemcpyDeviceToHost, cs));
        SPH_CUDA_TRY(cudaMemcpyAsync(rho + i0, dr + i0, cs1, cudaMemcpyDeviceToHost, cs));
    }
    SPH_CUDA_TRY(cudaStreamSynchronize(st));
    SPH_CUDA_TRY(cudaStreamSynchronize(cs));
    return sph_check(ctx);
}

// ------------------------------------------------------------------------------------------ profiling
extern "C" int sph_profile_enable(sph_ctx *ctx, int on)
{
    if (!ctx) return SPH_E_INVALID;
    ctx->prof.on = on != 0;
    return SPH_OK;
}

extern "C" int sph_profile_read(sph_ctx *ctx, double *ms_sum, int64_t *launches)
{
    if (!ctx) return SPH_E_INVALID;
    SPH_CUDA_TRY(cudaSetDevice(ctx->device));
    SPH_CUDA_TRY(cudaDeviceSynchronize());
    Profiler &pf = ctx->prof;
    for (const ProfRec &r : pf.live) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess) pf.ms[r.cls] += (double)ms;
        else (void)cudaGetLastError();
        pf.pool.push_back(r.a);
        pf.pool.push_back(r.b);
    }
    pf.live.clear();
    for (int k = 0; k < SPH_K_NCLASS; ++k) {
        if (ms_sum) ms_sum[k] = pf.ms[k];
        if (launches) launches[k] = pf.count[k];
        pf.ms[k] = 0.0;
        pf.count[k] = 0;
    }
    return SPH_OK;
}

extern "C" int sph_set_option(sph_ctx *ctx, int key, int value)
{
    if (!ctx) return SPH_E_INVALID;
    switch (key) {
    case SPH_OPT_PAIR_GROUP:
        if (value != 0 && value != 4 && value != 8 && value != 16 && value != 32) return SPH_E_INVALID;
        ctx->opt_group = value;
        return SPH_OK;
    case SPH_OPT_LIST_MODE:
        if (value < 0 || value > 2) return SPH_E_INVALID;
        ctx->opt_list_mode = value;
        return SPH_OK;
    case SPH_OPT_PAIR_WARPS:
        if (value != 0 && value != 4 && value != 8 && value != 10 && value != 12 && value != 16 && value != 20 && value != 24)
            return SPH_E_INVALID;
        ctx->opt_warps = value;
        return SPH_OK;
    case SPH_OPT_RK_EXTRA_SKIN:
        if (value < -1 || value > 2000) return SPH_E_INVALID;
        ctx->opt_rk_extra_permille = value;
        return SPH_OK;
    case SPH_OPT_FILL_MASKS:
        ctx->opt_fill_masks = value != 0;
        return SPH_OK;
    case SPH_OPT_TILE_EDGE:
        if (value != 0 && value != 1 && value != 2 && value != 4) return SPH_E_INVALID;
        ctx->opt_tile_edge = value;
        return SPH_OK;
    case SPH_OPT_BUILD_FUSED:
        ctx->opt_build_fused = value != 0;
        return SPH_OK;
    case SPH_OPT_STAGE_BULK:
        ctx->opt_stage_bulk = value != 0;
        return SPH_OK;
    case SPH_OPT_TILE_TABLES:
        ctx->opt_tile_tables = value != 0;
        return SPH_OK;
    case SPH_OPT_VJP_SPLIT:
        ctx->opt_vjp_split = value != 0;
        return SPH_OK;
    case SPH_OPT_UNIFORM_MASS_PATH:
        ctx->opt_no_um = value == 0;
        return SPH_OK;
    default:
        return SPH_E_INVALID;
    }
}
