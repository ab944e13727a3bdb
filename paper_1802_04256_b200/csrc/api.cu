// C ABI of librpim (include/rpim.h): argument checks, workspace ownership, stage sequencing.
#include <cmath>
#include <cstring>
#include <new>

#include "common.cuh"

namespace {

// DESIGN.md R5: coefficients and tables of the reproducible power function, evaluated on the
// host in the library's own code (the oracle has its own, independent copy of this recipe).
void fill_shape_params(double alpha_c, double d_c, double q, ShapeParams& P) {
    P.inv_dc = 1.0 / d_c;
    P.ac2 = alpha_c * alpha_c;
    P.twoq = 2.0 * q;
    const double a = q - 1.0;
    P.pw.b[0] = 1.0;
    for (int j = 1; j <= 9; ++j) P.pw.b[j] = (P.pw.b[j - 1] * (a - (double)(j - 1))) / (double)j;
    for (int i = 0; i < 32; ++i) {
        const double c = 1.0 + (double)(2 * i + 1) / 64.0;
        P.pw.invc[i] = 1.0 / c;
        P.pw.E[i] = (double)powl((long double)P.pw.invc[i], -(long double)a);
    }
    for (int e = -64; e <= 63; ++e) P.pw.F[e + 64] = (double)powl(2.0L, (long double)e * (long double)a);
}

void free_all(rpim_ctx* c) {
    ws_free(c, &c->d_cell_of); ws_free(c, &c->d_cell_start); ws_free(c, &c->d_cell_cursor);
    ws_free(c, &c->d_node_order); ws_free(c, &c->d_sorted_xyz); ws_free(c, &c->d_support);
    ws_free(c, &c->d_inc_count); ws_free(c, &c->d_inc_ptr); ws_free(c, &c->d_inc_q); ws_free(c, &c->d_inc_j);
    ws_free(c, &c->d_blen); ws_free(c, &c->d_brow_ptr); ws_free(c, &c->d_bcol); ws_free(c, &c->d_bdiag);
    ws_free(c, &c->d_stage); ws_free(c, &c->d_singular); ws_free(c, &c->d_scratch);
    ws_free(c, &c->d_mask_ptr); ws_free(c, &c->d_masks);
    c->have_masks = false;
    ws_free(c, &c->d_gpos); ws_free(c, &c->d_gmeta);
    ws_free(c, &c->d_tile_ptr); ws_free(c, &c->d_tdesc);
    c->have_tiles = false; c->tg_C = 0;
    ws_free(c, &c->h2d_nodes); ws_free(c, &c->h2d_qpts);
    ws_free(c, &c->hb_qw); ws_free(c, &c->hb_vals); ws_free(c, &c->hb_f); ws_free(c, &c->hb_ub);
    ws_free(c, &c->hb_bn); ws_free(c, &c->hb_bm); ws_free(c, &c->hb_rp); ws_free(c, &c->hb_ci);
    { int64_t* t = (int64_t*)c->d_scan_tmp; ws_free(c, &t); c->d_scan_tmp = nullptr; c->scan_tmp_elems = 0; }
    // blocks still registered as live here have no owner (a temporary lost on an error path): release them too
    for (auto& b : c->ws_sizes) { cudaFree(b.first); c->ws_bytes -= b.second; }
    c->ws_sizes.clear();
    ws_release_cache(c);
    c->have_pattern = c->have_shape = false;
}

}  // namespace

extern "C" {

int rpim_create(rpim_ctx** out_ctx, int device, void* cuda_stream) {
    if (!out_ctx) return RPIM_ERR_INVALID_ARG;
    *out_ctx = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0 || device < 0 || device >= ndev) {
        cudaGetLastError();
        return RPIM_ERR_CUDA;
    }
    rpim_ctx* c = new (std::nothrow) rpim_ctx();
    if (!c) return RPIM_ERR_ALLOC;
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    if (cudaSetDevice(device) != cudaSuccess) { delete c; return RPIM_ERR_CUDA; }
    if (cudaMalloc((void**)&c->d_flags, NUM_FLAGS * sizeof(long long)) != cudaSuccess) { delete c; return RPIM_ERR_ALLOC; }
    cudaMemset(c->d_flags, 0, NUM_FLAGS * sizeof(long long));
    for (auto& e : c->ev) cudaEventCreate(&e);
    *out_ctx = c;
    return RPIM_OK;
}

int rpim_destroy(rpim_ctx* ctx) {
    if (!ctx) return RPIM_OK;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    free_all(ctx);
    if (ctx->d_flags) cudaFree(ctx->d_flags);
    for (auto& e : ctx->ev) if (e) cudaEventDestroy(e);
    for (auto& e : ctx->phase_events) cudaEventDestroy(e);
    if (ctx->side_stream) { cudaStreamSynchronize(ctx->side_stream); cudaStreamDestroy(ctx->side_stream); }
    for (auto& e : ctx->side_ev) if (e) cudaEventDestroy(e);
    delete ctx;
    return RPIM_OK;
}

const char* rpim_last_error(const rpim_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }
int64_t rpim_workspace_bytes(const rpim_ctx* ctx) { return ctx ? ctx->ws_bytes : 0; }
int64_t rpim_launch_count(const rpim_ctx* ctx) { return ctx ? ctx->launches : 0; }

int rpim_set_reduction(rpim_ctx* ctx, int mode) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (mode < 0 || mode > 3) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "reduction mode must be 0 (auto), 1 (rows), 2 (panels) or 3 (long rows)");
    ctx->reduce_mode = mode;
    return RPIM_OK;
}

int rpim_set_panel_shape(rpim_ctx* ctx, int rows_per_tile, int warps_per_group, int rows_per_group, int ring_stages,
                         int staging, int tile_desc) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    const bool ok = (rows_per_tile == 0 || (rows_per_tile >= 2 && rows_per_tile <= 8 && !(rows_per_tile & 1))) &&
                    (warps_per_group >= 0 && warps_per_group <= 4) && (rows_per_group >= 0 && rows_per_group <= 2) &&
                    (ring_stages == 0 || (ring_stages >= 2 && ring_stages <= 8)) && (staging >= 0 && staging <= 2) &&
                    (tile_desc >= 0 && tile_desc <= 2);
    if (!ok)
        RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "rpim_set_panel_shape: rows_per_tile in {0,2,4,6,8}, warps_per_group 0..4, "
                  "rows_per_group 0..2, ring_stages 0 or 2..8, staging 0..2, tile_desc 0..2");
    ctx->ov_T = rows_per_tile; ctx->ov_CW = warps_per_group; ctx->ov_R = rows_per_group;
    ctx->ov_nstage = ring_stages; ctx->ov_grad = staging; ctx->ov_tdesc = tile_desc;
    return RPIM_OK;
}

int rpim_set_modulus_scale(rpim_ctx* ctx, const double* d_escale) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!ctx->have_pattern) RPIM_FAIL(ctx, RPIM_ERR_STATE, "rpim_set_modulus_scale before rpim_build_pattern");
    ctx->d_escale = d_escale;
    return RPIM_OK;
}

int rpim_reduction_used(const rpim_ctx* ctx) { return ctx && ctx->have_pattern ? (ctx->have_tiles ? 2 : 1) : 0; }

int rpim_reduction_params(const rpim_ctx* ctx, int out[10]) {
    if (!ctx || !out) return RPIM_ERR_INVALID_ARG;
    const bool t = ctx->have_pattern && ctx->have_tiles;
    out[0] = rpim_reduction_used(ctx);
    out[1] = t ? ctx->tg_C : 0;
    out[2] = t ? ctx->tg_T : 0;
    out[3] = t ? ctx->tg_CW : 0;
    out[4] = t ? ctx->tg_nstage : 0;
    out[5] = t ? ctx->max_ulen : 0;
    out[6] = ctx->have_pattern ? ctx->max_blen : 0;
    out[7] = (int)(100.0 * ctx->tg_mean_union + 0.5);
    out[8] = t ? ctx->tg_R : 0;
    out[9] = t && ctx->tg_grad_only ? 1 : 0;
    return RPIM_OK;
}

int rpim_build_pattern(rpim_ctx* ctx, const double* d_nodes, int64_t N, const double* d_qpts, int64_t Nq, int k,
                       int index_bits, int64_t* out_nnz, int* out_index_bits) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!d_nodes || !d_qpts || N <= 0 || Nq <= 0) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "null pointer or empty input");
    if (k < 4 || k > RPIM_MAX_K || k > N) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "k = %d must satisfy 4 <= k <= min(N, %d)", k, RPIM_MAX_K);
    if (index_bits != 0 && index_bits != 32 && index_bits != 64 && index_bits != RPIM_INDEX_MIXED)
        RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "index_bits must be 0, 32, 64 or RPIM_INDEX_MIXED (%d)", RPIM_INDEX_MIXED);
    if (N > 700000000 || Nq * (int64_t)k > 0x7fffffff00LL || Nq > 0x7fffffff) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "problem too large for 32-bit node / point ids");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    ctx->have_pattern = ctx->have_shape = ctx->have_masks = false;
    ws_free(ctx, &ctx->d_stage);
    ws_free(ctx, &ctx->d_singular);
    ctx->d_nodes = d_nodes; ctx->d_qpts = d_qpts; ctx->N = N; ctx->Nq = Nq; ctx->k = k;
    ctx->d_escale = nullptr;
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_flags, 0, NUM_FLAGS * sizeof(long long), st));
    int rc;
    if ((rc = ws_alloc(ctx, &ctx->d_support, Nq * k))) return rc;
    cudaEventRecord(ctx->ev[0], st);
    if ((rc = rpim_stage_grid_knn(ctx, d_qpts, Nq, k, ctx->d_support, true))) return rc;
    cudaEventRecord(ctx->ev[1], st);
    if ((rc = rpim_stage_incidence(ctx))) return rc;
    cudaEventRecord(ctx->ev[2], st);
    // the reduction's integer preprocessing: point groups first (they decide between the tiled and the
    // row-owner kernel, and so whether slot masks are built with the block rows), row tiles last
    if ((rc = rpim_stage_groups(ctx))) return rc;
    if ((rc = rpim_stage_block_pattern(ctx))) return rc;
    if (ctx->tg_C == 0 && (rc = rpim_stage_slot_masks(ctx))) return rc;
    if ((rc = rpim_stage_tiles(ctx))) return rc;
    cudaEventRecord(ctx->ev[3], st);
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    for (int i = 0; i < 3; ++i) {
        cudaEventElapsedTime(&ctx->phase_ms[i], ctx->ev[i], ctx->ev[i + 1]);
        ctx->phase_total_ms[i] += ctx->phase_ms[i];
    }
    ctx->phase_calls[0]++;
    const int64_t nnz = 9 * ctx->nnzb;
    int bits = index_bits ? index_bits : (nnz > 0x7fffffffLL ? 64 : 32);
    if (bits == 32 && nnz > 0x7fffffffLL) RPIM_FAIL(ctx, RPIM_ERR_INDEX_OVERFLOW, "nnz = %lld does not fit 32-bit indices", (long long)nnz);
    ctx->index_bits = bits;
    ctx->have_pattern = true;
    if (out_nnz) *out_nnz = nnz;
    if (out_index_bits) *out_index_bits = bits;
    return RPIM_OK;
}

namespace {
// number of points whose support row differs between two tables
__global__ void support_diff_kernel(const int32_t* __restrict__ a, const int32_t* __restrict__ b, int64_t Nq, int k,
                                    unsigned long long* __restrict__ changed) {
    const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool d = false;
    if (q < Nq)
        for (int j = 0; j < k; ++j) d = d || a[q * k + j] != b[q * k + j];
    const unsigned m = __ballot_sync(0xffffffffu, d);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(changed, (unsigned long long)__popc(m));
}
}  // namespace

int rpim_update_nodes(rpim_ctx* ctx, const double* d_nodes, const double* d_qpts, int64_t* out_changed_points,
                      int* out_pattern_rebuilt, int64_t* out_nnz) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!ctx->have_pattern) RPIM_FAIL(ctx, RPIM_ERR_STATE, "rpim_update_nodes before rpim_build_pattern");
    if (!d_nodes) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "null pointer");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const int64_t Nq = ctx->Nq;
    const int k = ctx->k;
    ctx->d_nodes = d_nodes;
    if (d_qpts) ctx->d_qpts = d_qpts;
    ctx->have_shape = false;            // staged shape functions belong to the old coordinates
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_flags, 0, NUM_FLAGS * sizeof(long long), st));
    int rc;
    cudaEventRecord(ctx->ev[0], st);
    bool rebuild = true;
    int64_t moved = 0;
    if ((rc = rpim_stage_grid_refresh(ctx, &rebuild, &moved))) { ctx->have_pattern = false; return rc; }
    int32_t* d_new = nullptr;
    if ((rc = ws_alloc(ctx, &d_new, Nq * k))) { ctx->have_pattern = false; return rc; }
    // from here on the grid and d_nodes are the new ones: every failure gives d_new back and drops the pattern
    auto drop = [&]() { ws_free(ctx, &d_new); ctx->have_pattern = false; };
    cudaError_t e0 = cudaMemsetAsync(ctx->d_flags + FLAG_KNN_CAP, 0, sizeof(long long), st);
    if (e0 != cudaSuccess) { drop(); RPIM_FAIL(ctx, RPIM_ERR_CUDA, "rpim_update_nodes: memset failed: %s", cudaGetErrorString(e0)); }
    if ((rc = rpim_stage_grid_knn(ctx, ctx->d_qpts, Nq, k, d_new, rebuild))) { drop(); return rc; }
    unsigned long long* d_changed = (unsigned long long*)ctx->d_scratch;
    e0 = cudaMemsetAsync(d_changed, 0, sizeof(unsigned long long), st);
    if (e0 != cudaSuccess) { drop(); RPIM_FAIL(ctx, RPIM_ERR_CUDA, "rpim_update_nodes: memset failed: %s", cudaGetErrorString(e0)); }
    support_diff_kernel<<<(unsigned)((Nq + 255) / 256), 256, 0, st>>>(ctx->d_support, d_new, Nq, k, d_changed);
    ctx->launches++;
    unsigned long long changed = 0;
    long long capf = 0;
    cudaEventRecord(ctx->ev[1], st);
    cudaError_t e = cudaMemcpyAsync(&changed, d_changed, sizeof(changed), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&capf, ctx->d_flags + FLAG_KNN_CAP, sizeof(capf), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess || capf) {
        ws_free(ctx, &d_new);
        ctx->have_pattern = false;
        if (capf) RPIM_FAIL(ctx, RPIM_ERR_CAPACITY, "kNN: %lld points found fewer than k nodes (k > N?)", capf);
        RPIM_FAIL(ctx, RPIM_ERR_CUDA, "rpim_update_nodes failed: %s", cudaGetErrorString(e));
    }
    cudaEventElapsedTime(&ctx->phase_ms[0], ctx->ev[0], ctx->ev[1]);
    ctx->phase_ms[1] = ctx->phase_ms[2] = 0.f;
    if (out_changed_points) *out_changed_points = (int64_t)changed;
    if (out_pattern_rebuilt) *out_pattern_rebuilt = changed != 0;
    if (changed == 0) {
        // supports unchanged: incidence lists, block pattern, slot maps, point groups and row tiles all stand
        ws_free(ctx, &d_new);
    } else {
        ws_free(ctx, &ctx->d_support);
        ctx->d_support = d_new;
        ctx->have_pattern = ctx->have_masks = false;
        cudaEventRecord(ctx->ev[1], st);
        if ((rc = rpim_stage_incidence(ctx))) return rc;
        cudaEventRecord(ctx->ev[2], st);
        if ((rc = rpim_stage_groups(ctx))) return rc;
        if ((rc = rpim_stage_block_pattern(ctx))) return rc;
        if (ctx->tg_C == 0 && (rc = rpim_stage_slot_masks(ctx))) return rc;
        if ((rc = rpim_stage_tiles(ctx))) return rc;
        cudaEventRecord(ctx->ev[3], st);
        CUDA_TRY(ctx, cudaStreamSynchronize(st));
        cudaEventElapsedTime(&ctx->phase_ms[1], ctx->ev[1], ctx->ev[2]);
        cudaEventElapsedTime(&ctx->phase_ms[2], ctx->ev[2], ctx->ev[3]);
        const int64_t nnz = 9 * ctx->nnzb;
        if (ctx->index_bits == 32 && nnz > 0x7fffffffLL)
            RPIM_FAIL(ctx, RPIM_ERR_INDEX_OVERFLOW, "nnz = %lld no longer fits the 32-bit indices chosen by rpim_build_pattern", (long long)nnz);
        ctx->have_pattern = true;
    }
    if (out_nnz) *out_nnz = 9 * ctx->nnzb;
    return RPIM_OK;
}

int rpim_get_pattern(rpim_ctx* ctx, void* d_row_ptr, void* d_col_idx, int32_t* d_support) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!ctx->have_pattern) RPIM_FAIL(ctx, RPIM_ERR_STATE, "rpim_get_pattern before rpim_build_pattern");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    int rc;
    if ((rc = rpim_stage_emit_pattern(ctx, d_row_ptr, d_col_idx))) return rc;
    if (d_support)
        CUDA_TRY(ctx, cudaMemcpyAsync(d_support, ctx->d_support, (size_t)ctx->Nq * ctx->k * sizeof(int32_t),
                                      cudaMemcpyDeviceToDevice, ctx->stream));
    return RPIM_OK;
}

int rpim_assemble(rpim_ctx* ctx, const double* d_qw, double E, double nu, double alpha_c, double d_c, double q,
                  const double body[3], double* d_vals, double* d_f, int64_t* out_singular) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!ctx->have_pattern) RPIM_FAIL(ctx, RPIM_ERR_STATE, "rpim_assemble before rpim_build_pattern");
    if (!d_qw || !body || !d_vals || !d_f) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "null pointer");
    if (!(d_c > 0.0) || !(alpha_c > 0.0) || !std::isfinite(q) || !std::isfinite(E) || !(nu > -1.0 && nu < 0.5))
        RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "need d_c > 0, alpha_c > 0, finite q and E, -1 < nu < 0.5");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    fill_shape_params(alpha_c, d_c, q, ctx->sp);
    ctx->have_sp = true;
    int rc;
    // (whole groups of RPIM_GROUP_POINTS points: the panel reduction copies a group's staged rows in one piece)
    if (!ctx->d_stage && (rc = ws_alloc(ctx, &ctx->d_stage, ((ctx->Nq + RPIM_GROUP_POINTS - 1) / RPIM_GROUP_POINTS) * RPIM_GROUP_POINTS * 4 * (int64_t)ctx->k))) return rc;
    if (!ctx->d_singular && (rc = ws_alloc(ctx, &ctx->d_singular, ctx->Nq))) return rc;
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_flags + FLAG_SINGULAR, 0, sizeof(long long), st));
    // a triple of pooled events per call so that a caller can sum kernel times over many calls
    cudaEvent_t pe[3] = {nullptr, nullptr, nullptr};
    if (ctx->phase_events_used + 3 <= 3 * 4096) {
        while (ctx->phase_events.size() < ctx->phase_events_used + 3) {
            cudaEvent_t e;
            CUDA_TRY(ctx, cudaEventCreate(&e));
            ctx->phase_events.push_back(e);
        }
        for (int i = 0; i < 3; ++i) pe[i] = ctx->phase_events[ctx->phase_events_used + i];
        ctx->phase_events_used += 3;
    }
    cudaEventRecord(ctx->ev[4], st);
    if (pe[0]) cudaEventRecord(pe[0], st);
    if ((rc = rpim_stage_shape(ctx, ctx->d_qpts, ctx->d_support, ctx->Nq, ctx->d_stage, ctx->d_singular))) return rc;
    cudaEventRecord(ctx->ev[5], st);
    if (pe[1]) cudaEventRecord(pe[1], st);
    const double lambda = E * nu / ((1.0 + nu) * (1.0 - 2.0 * nu));
    const double mu = E / (2.0 * (1.0 + nu));
    rc = ctx->have_tiles ? rpim_stage_accumulate_panels(ctx, d_qw, lambda, mu, body, d_vals, d_f)
                         : rpim_stage_accumulate(ctx, d_qw, lambda, mu, body, d_vals, d_f);
    if (rc) return rc;
    cudaEventRecord(ctx->ev[6], st);
    if (pe[2]) cudaEventRecord(pe[2], st);
    ctx->phase_calls[1]++;
    ctx->have_shape = true;
    if (out_singular) {
        long long ns = 0;
        CUDA_TRY(ctx, cudaMemcpyAsync(&ns, ctx->d_flags + FLAG_SINGULAR, sizeof(ns), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(ctx, cudaStreamSynchronize(st));
        *out_singular = ns;
    }
    return RPIM_OK;
}

int rpim_add_point_loads(rpim_ctx* ctx, const double* d_pts, const double* d_w, const double* d_t, int64_t M,
                         double* d_f) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!ctx->have_pattern || !ctx->have_sp) RPIM_FAIL(ctx, RPIM_ERR_STATE, "rpim_add_point_loads before rpim_assemble");
    if (M < 0 || (M > 0 && (!d_pts || !d_w || !d_t || !d_f))) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "null pointer");
    if (M == 0) return RPIM_OK;
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    int32_t* d_sup = nullptr;
    double* d_stage = nullptr;
    uint8_t* d_sing = nullptr;
    int rc = RPIM_OK;
    // the capacity and singular-point counters are this call's own: clear them first
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_flags + FLAG_KNN_CAP, 0, sizeof(long long), st));
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_flags + FLAG_SINGULAR, 0, sizeof(long long), st));
    if ((rc = ws_alloc(ctx, &d_sup, M * ctx->k)) == RPIM_OK && (rc = ws_alloc(ctx, &d_stage, M * 4 * (int64_t)ctx->k)) == RPIM_OK &&
        (rc = ws_alloc(ctx, &d_sing, M)) == RPIM_OK) {
        if ((rc = rpim_stage_grid_knn(ctx, d_pts, M, ctx->k, d_sup, false)) == RPIM_OK &&
            (rc = rpim_stage_shape(ctx, d_pts, d_sup, M, d_stage, d_sing)) == RPIM_OK)
            rc = rpim_stage_point_loads(ctx, d_sup, d_stage, d_w, d_t, M, d_f);
    }
    cudaError_t e = cudaStreamSynchronize(st);
    long long capf = 0, nsing = 0;
    cudaMemcpy(&capf, ctx->d_flags + FLAG_KNN_CAP, sizeof(capf), cudaMemcpyDeviceToHost);
    cudaMemcpy(&nsing, ctx->d_flags + FLAG_SINGULAR, sizeof(nsing), cudaMemcpyDeviceToHost);
    cudaMemsetAsync(ctx->d_flags + FLAG_KNN_CAP, 0, sizeof(long long), st);   // reported: do not poison later calls
    cudaMemsetAsync(ctx->d_flags + FLAG_SINGULAR, 0, sizeof(long long), st);
    ws_free(ctx, &d_sup);
    ws_free(ctx, &d_stage);
    ws_free(ctx, &d_sing);
    if (rc) return rc;
    if (e != cudaSuccess) RPIM_FAIL(ctx, RPIM_ERR_CUDA, "point loads failed: %s", cudaGetErrorString(e));
    if (capf) RPIM_FAIL(ctx, RPIM_ERR_CAPACITY, "kNN capacity exceeded for %lld load points", capf);
    if (nsing)
        RPIM_FAIL(ctx, RPIM_ERR_SINGULAR_POINT, "%lld of %lld load points have a singular moment matrix (their k nearest "
                  "nodes are degenerate, e.g. coplanar): their traction was NOT added", nsing, (long long)M);
    return RPIM_OK;
}

int rpim_apply_penalty(rpim_ctx* ctx, const int64_t* d_bc_nodes, const uint8_t* d_bc_mask, const double* d_u_bar,
                       int64_t m, double alpha, int alpha_is_relative, double* d_vals, double* d_f,
                       double* out_alpha_used) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!ctx->have_pattern) RPIM_FAIL(ctx, RPIM_ERR_STATE, "rpim_apply_penalty before rpim_build_pattern");
    if (m < 0 || !d_vals || !d_f || (m > 0 && (!d_bc_nodes || !d_u_bar))) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "null pointer");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    return rpim_stage_penalty(ctx, d_bc_nodes, d_bc_mask, d_u_bar, m, alpha, alpha_is_relative, d_vals, d_f,
                              out_alpha_used);
}

namespace {
__global__ void split_stage_kernel(const double* __restrict__ stage, int64_t M, int k, double* __restrict__ phi,
                                   double* __restrict__ dphi) {
    const int64_t total = M * 4 * (int64_t)k;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        const int64_t q = e / (4 * k);
        const int r = (int)(e % (4 * k));
        const int c = r / k, j = r - c * k;       // staged layout: [q][phi, d/dx, d/dy, d/dz][j]
        if (c == 0) { if (phi) phi[q * k + j] = stage[e]; }
        else if (dphi) dphi[(q * 3 + (c - 1)) * (int64_t)k + j] = stage[e];
    }
}
}  // namespace

namespace {
// Sustained FP64 multiply-add rate: eight independent fma chains per thread, no memory traffic.
__global__ void __launch_bounds__(1024) fp64_probe_kernel(int iters, double seed, double* __restrict__ sink) {
    double a0 = seed + threadIdx.x, a1 = a0 + 1.0, a2 = a0 + 2.0, a3 = a0 + 3.0;
    double a4 = a0 + 4.0, a5 = a0 + 5.0, a6 = a0 + 6.0, a7 = a0 + 7.0;
    const double m = 1.0 - 1e-9, c = 1e-9;
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    const double t = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (t == 123.456) sink[0] = t;   // never true: keeps the chains alive
}
}  // namespace

int rpim_probe_fp64(rpim_ctx* ctx, double* out_tflops, double* out_ms) {
    if (!ctx || !out_tflops) return RPIM_ERR_INVALID_ARG;
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->device);
    double* d_sink = nullptr;
    int rc = ws_alloc(ctx, &d_sink, 8);
    if (rc) return rc;
    const int iters = 4096, blocks = sms * 2, threads = 1024;
    cudaEvent_t e0, e1;
    CUDA_TRY(ctx, cudaEventCreate(&e0));
    CUDA_TRY(ctx, cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {   // the first launch warms up; best of the next three
        cudaEventRecord(e0, ctx->stream);
        fp64_probe_kernel<<<blocks, threads, 0, ctx->stream>>>(iters, 1.0 + rep, d_sink);
        cudaEventRecord(e1, ctx->stream);
        ctx->launches++;
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); ws_free(ctx, &d_sink); RPIM_FAIL(ctx, RPIM_ERR_CUDA, "fp64 probe failed: %s", cudaGetErrorString(e)); }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    ws_free(ctx, &d_sink);
    const double flops = 2.0 * 8.0 * (double)iters * (double)blocks * (double)threads;
    *out_tflops = flops / ((double)best * 1e-3) / 1e12;
    if (out_ms) *out_ms = best;
    return RPIM_OK;
}

namespace {
// Sustained rate of the FP64 tensor-core path that exists on sm_100a (mma.sync m8n8k4, the legacy warp-level
// instruction; tcgen05 has no FP64 kind): eight independent accumulator chains per warp, no memory traffic.
__global__ void __launch_bounds__(1024) dmma_probe_kernel(int iters, double seed, double* __restrict__ sink) {
    double c[8][2];
#pragma unroll
    for (int j = 0; j < 8; ++j) { c[j][0] = seed + j; c[j][1] = seed - j; }
    const double a = 1.0 - 1e-9 * (double)(threadIdx.x & 3), b = 1e-9 * (double)(1 + (threadIdx.x & 7));
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 8; ++j)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                         : "+d"(c[j][0]), "+d"(c[j][1]) : "d"(a), "d"(b));
    }
    double t = 0.0;
#pragma unroll
    for (int j = 0; j < 8; ++j) t += c[j][0] + c[j][1];
    if (t == 123.456) sink[0] = t;   // never true: keeps the chains alive
}
}  // namespace

int rpim_probe_fp64_dmma(rpim_ctx* ctx, double* out_tflops, double* out_ms) {
    if (!ctx || !out_tflops) return RPIM_ERR_INVALID_ARG;
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->device);
    double* d_sink = nullptr;
    int rc = ws_alloc(ctx, &d_sink, 8);
    if (rc) return rc;
    const int iters = 2048, blocks = sms * 2, threads = 1024;
    cudaEvent_t e0, e1;
    CUDA_TRY(ctx, cudaEventCreate(&e0));
    CUDA_TRY(ctx, cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {   // the first launch warms up; best of the next three
        cudaEventRecord(e0, ctx->stream);
        dmma_probe_kernel<<<blocks, threads, 0, ctx->stream>>>(iters, 1.0 + rep, d_sink);
        cudaEventRecord(e1, ctx->stream);
        ctx->launches++;
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); ws_free(ctx, &d_sink); RPIM_FAIL(ctx, RPIM_ERR_CUDA, "fp64 mma probe failed: %s", cudaGetErrorString(e)); }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    ws_free(ctx, &d_sink);
    // one m8n8k4 = 8 x 8 x 4 multiply-adds per warp
    const double flops = 2.0 * 256.0 * 8.0 * (double)iters * (double)blocks * (double)(threads / 32);
    *out_tflops = flops / ((double)best * 1e-3) / 1e12;
    if (out_ms) *out_ms = best;
    return RPIM_OK;
}

int rpim_get_shape(rpim_ctx* ctx, double* d_phi, double* d_dphi, uint8_t* d_singular) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!ctx->have_shape) RPIM_FAIL(ctx, RPIM_ERR_STATE, "rpim_get_shape before rpim_assemble");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    if (d_phi || d_dphi) {
        const int64_t total = ctx->Nq * 4 * (int64_t)ctx->k;
        split_stage_kernel<<<(unsigned)std::min<int64_t>((total + 255) / 256, 148 * 32), 256, 0, ctx->stream>>>(
            ctx->d_stage, ctx->Nq, ctx->k, d_phi, d_dphi);
        KERNEL_CHECK(ctx);
    }
    if (d_singular)
        CUDA_TRY(ctx, cudaMemcpyAsync(d_singular, ctx->d_singular, (size_t)ctx->Nq, cudaMemcpyDeviceToDevice, ctx->stream));
    return RPIM_OK;
}

int rpim_last_phase_ms(rpim_ctx* ctx, float out_ms[5]) {
    if (!ctx || !out_ms) return RPIM_ERR_INVALID_ARG;
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    if (ctx->have_shape) {
        cudaEventElapsedTime(&ctx->phase_ms[3], ctx->ev[4], ctx->ev[5]);
        cudaEventElapsedTime(&ctx->phase_ms[4], ctx->ev[5], ctx->ev[6]);
    }
    for (int i = 0; i < 5; ++i) out_ms[i] = ctx->phase_ms[i];
    return RPIM_OK;
}

int rpim_phase_totals(rpim_ctx* ctx, double out_ms[5], int64_t out_calls[2], int reset) {
    if (!ctx || !out_ms) return RPIM_ERR_INVALID_ARG;
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    double shape = 0.0, reduce = 0.0;
    for (size_t i = 0; i + 2 < ctx->phase_events_used + 0 && i + 2 < ctx->phase_events.size() + 0; i += 3) {
        float a = 0.f, b = 0.f;
        if (cudaEventElapsedTime(&a, ctx->phase_events[i], ctx->phase_events[i + 1]) == cudaSuccess) shape += a;
        if (cudaEventElapsedTime(&b, ctx->phase_events[i + 1], ctx->phase_events[i + 2]) == cudaSuccess) reduce += b;
    }
    cudaGetLastError();
    for (int i = 0; i < 3; ++i) out_ms[i] = ctx->phase_total_ms[i];
    out_ms[3] = shape;
    out_ms[4] = reduce;
    if (out_calls) { out_calls[0] = ctx->phase_calls[0]; out_calls[1] = ctx->phase_calls[1]; }
    if (reset) {
        ctx->phase_events_used = 0;
        for (int i = 0; i < 5; ++i) ctx->phase_total_ms[i] = 0.0;
        ctx->phase_calls[0] = ctx->phase_calls[1] = 0;
    }
    return RPIM_OK;
}

// ------------------------------------------------------------------ host-buffer (end-to-end) entry points
int rpim_host_pattern(rpim_ctx* ctx, const double* h_nodes, int64_t N, const double* h_qpts, int64_t Nq, int k,
                      int index_bits, int64_t* out_nnz, int* out_index_bits) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!h_nodes || !h_qpts || N <= 0 || Nq <= 0) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "null pointer or empty input");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    int rc;
    if ((rc = ws_alloc(ctx, &ctx->h2d_nodes, 3 * N))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->h2d_qpts, 3 * Nq))) return rc;
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h2d_nodes, h_nodes, (size_t)3 * N * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h2d_qpts, h_qpts, (size_t)3 * Nq * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    return rpim_build_pattern(ctx, ctx->h2d_nodes, N, ctx->h2d_qpts, Nq, k, index_bits, out_nnz, out_index_bits);
}

int rpim_host_assemble(rpim_ctx* ctx, const double* h_qw, double E, double nu, double alpha_c, double d_c, double q,
                       const double body[3], const int64_t* h_bc_nodes, const uint8_t* h_bc_mask,
                       const double* h_u_bar, int64_t m, double alpha, int alpha_is_relative, void* h_row_ptr,
                       void* h_col_idx, double* h_vals, double* h_f, int64_t* out_singular, double* out_alpha_used) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!ctx->have_pattern) RPIM_FAIL(ctx, RPIM_ERR_STATE, "rpim_host_assemble before rpim_host_pattern");
    if (!h_qw || !h_vals || !h_f || m < 0 || (m > 0 && (!h_bc_nodes || !h_u_bar))) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "null pointer");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const int64_t nnz = 9 * ctx->nnzb, n3 = 3 * ctx->N;
    // width of a row_ptr entry / of a col_idx entry (RPIM_INDEX_MIXED: 64-bit offsets, 32-bit column ids)
    const size_t iw = ctx->index_bits == 32 ? 4 : 8, iwc = ctx->index_bits == 64 ? 8 : 4;
    // device buffers of the call live in the context's workspace (cached across calls: no cudaMalloc / cudaFree
    // per step); the index arrays go back to the host on a side stream while the values are assembled
    int rc = RPIM_OK;
    if ((rc = ws_alloc(ctx, &ctx->hb_qw, ctx->Nq))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->hb_vals, std::max<int64_t>(nnz, 1)))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->hb_f, n3))) return rc;
    if (m > 0) {
        if ((rc = ws_alloc(ctx, &ctx->hb_bn, m))) return rc;
        if ((rc = ws_alloc(ctx, &ctx->hb_ub, 3 * m))) return rc;
        if (h_bc_mask && (rc = ws_alloc(ctx, &ctx->hb_bm, m))) return rc;
    }
    if (h_row_ptr && (rc = ws_alloc(ctx, &ctx->hb_rp, (int64_t)((n3 + 1) * iw)))) return rc;
    if (h_col_idx && (rc = ws_alloc(ctx, &ctx->hb_ci, (int64_t)(std::max<int64_t>(nnz, 1) * iwc)))) return rc;
    if (!ctx->side_stream) {
        CUDA_TRY(ctx, cudaStreamCreateWithFlags(&ctx->side_stream, cudaStreamNonBlocking));
        CUDA_TRY(ctx, cudaEventCreateWithFlags(&ctx->side_ev[0], cudaEventDisableTiming));
        CUDA_TRY(ctx, cudaEventCreateWithFlags(&ctx->side_ev[1], cudaEventDisableTiming));
    }
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->hb_qw, h_qw, (size_t)ctx->Nq * sizeof(double), cudaMemcpyHostToDevice, st));
    if (m > 0) {
        CUDA_TRY(ctx, cudaMemcpyAsync(ctx->hb_bn, h_bc_nodes, (size_t)m * sizeof(int64_t), cudaMemcpyHostToDevice, st));
        CUDA_TRY(ctx, cudaMemcpyAsync(ctx->hb_ub, h_u_bar, (size_t)3 * m * sizeof(double), cudaMemcpyHostToDevice, st));
        if (h_bc_mask) CUDA_TRY(ctx, cudaMemcpyAsync(ctx->hb_bm, h_bc_mask, (size_t)m, cudaMemcpyHostToDevice, st));
    }
    if ((rc = rpim_get_pattern(ctx, h_row_ptr ? ctx->hb_rp : nullptr, h_col_idx ? ctx->hb_ci : nullptr, nullptr))) return rc;
    CUDA_TRY(ctx, cudaEventRecord(ctx->side_ev[0], st));
    CUDA_TRY(ctx, cudaStreamWaitEvent(ctx->side_stream, ctx->side_ev[0], 0));
    if (h_row_ptr) CUDA_TRY(ctx, cudaMemcpyAsync(h_row_ptr, ctx->hb_rp, (size_t)(n3 + 1) * iw, cudaMemcpyDeviceToHost, ctx->side_stream));
    if (h_col_idx) CUDA_TRY(ctx, cudaMemcpyAsync(h_col_idx, ctx->hb_ci, (size_t)nnz * iwc, cudaMemcpyDeviceToHost, ctx->side_stream));
    CUDA_TRY(ctx, cudaEventRecord(ctx->side_ev[1], ctx->side_stream));
    rc = rpim_assemble(ctx, ctx->hb_qw, E, nu, alpha_c, d_c, q, body, ctx->hb_vals, ctx->hb_f, out_singular);
    if (rc == RPIM_OK)
        rc = rpim_apply_penalty(ctx, m > 0 ? ctx->hb_bn : nullptr, (m > 0 && h_bc_mask) ? ctx->hb_bm : nullptr,
                                m > 0 ? ctx->hb_ub : nullptr, m, alpha, alpha_is_relative, ctx->hb_vals, ctx->hb_f,
                                out_alpha_used);
    if (rc == RPIM_OK) {
        cudaError_t e = cudaMemcpyAsync(h_vals, ctx->hb_vals, (size_t)nnz * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(h_f, ctx->hb_f, (size_t)n3 * sizeof(double), cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) { ctx->err = std::string("device to host copy failed: ") + cudaGetErrorString(e); rc = RPIM_ERR_CUDA; }
    }
    // join the side stream into the main one and drain both, also on failure (the host arrays are the caller's)
    cudaStreamWaitEvent(st, ctx->side_ev[1], 0);
    cudaError_t e1 = cudaStreamSynchronize(st);
    if (rc == RPIM_OK && e1 != cudaSuccess) RPIM_FAIL(ctx, RPIM_ERR_CUDA, "rpim_host_assemble failed: %s", cudaGetErrorString(e1));
    return rc;
}

}  // extern "C"
