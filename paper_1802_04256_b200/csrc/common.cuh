// Internal declarations of librpim (sm_100a).  Not part of the C ABI (include/rpim.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/rpim.h"

#define RPIM_WARP 32
#define RPIM_GROUP_POINTS 8      // quadrature points per group of the panel reduction (groups.cu)
#define RPIM_PANEL_MAX_UNION_RATIO 2.0   // automatic choice: panel kernel when mean |U_g| <= ratio * k (the group's points share their supports)

// device-side error / counter slots (ctx->d_flags, int64 each)
enum { FLAG_KNN_CAP = 0, FLAG_PAT_CAP = 1, FLAG_BC_BAD = 2, FLAG_SINGULAR = 3, FLAG_INC_CAP = 4, FLAG_OVF_ROWS = 5, FLAG_OVF_Q = 6, FLAG_INC_LONG = 7, FLAG_ROW_TICKET = 8, FLAG_INC_LONG2 = 9, FLAG_TILE_CAP = 10, FLAG_OVF_Q2 = 11, NUM_FLAGS = 16 };

struct GridParams {
    double lo[3];
    double cell;      // cell edge
    double inv_cell;  // 1.0 / cell
    int nc[3];
    int64_t ncell;
};

// Reproducible power t^(q-1): tables and coefficients (R5), filled on the host.
struct PowTables {
    double b[10];
    double invc[32];
    double E[32];
    double F[128];
};

struct ShapeParams {
    double inv_dc, ac2, twoq;
    PowTables pw;
};

struct rpim_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    int64_t launches = 0;
    int64_t ws_bytes = 0;
    std::unordered_map<void*, int64_t> ws_sizes;          // live blocks -> capacity in bytes
    std::vector<std::pair<void*, int64_t>> ws_cache;      // parked blocks (freed, reusable)

    // problem
    const double* d_nodes = nullptr;
    const double* d_qpts = nullptr;
    int64_t N = 0, Nq = 0;
    int k = 0;
    bool have_pattern = false, have_shape = false;
    int index_bits = 64;
    int64_t nnzb = 0;   // number of 3x3 blocks
    int max_blen = 0;   // longest block row
    int max_inc = 0;    // longest incidence list

    // cell grid
    GridParams grid{};
    int* d_cell_of = nullptr;        // N
    int64_t* d_cell_start = nullptr; // ncell + 1
    int* d_cell_cursor = nullptr;    // ncell
    int* d_node_order = nullptr;     // N   (node ids in cell order)
    double* d_sorted_xyz = nullptr;  // 3 x N (SoA, cell order)

    // supports and incidence
    int32_t* d_support = nullptr;    // Nq x k
    int* d_inc_count = nullptr;      // N
    int64_t* d_inc_ptr = nullptr;    // N + 1
    int32_t* d_inc_q = nullptr;      // Nq*k  (point id, ascending per node)
    uint8_t* d_inc_j = nullptr;      // Nq*k  (position of the node in that point's support)

    // block pattern
    int* d_blen = nullptr;           // N
    int64_t* d_brow_ptr = nullptr;   // N + 1
    int32_t* d_bcol = nullptr;       // nnzb
    int* d_bdiag = nullptr;          // N (slot of the diagonal block in its row)

    // precomputed slot maps of the reduction (optional: skipped when they would not fit):
    // for incident point p of block row I, ceil(L_I / 32) words; bit s = column slot s of the row
    // is a support node of the point
    bool have_masks = false;
    int mask_stride = 0;             // > 0: words per incident point, row I at inc_ptr[I] * stride; 0: d_mask_ptr, ceil(L_I/32)
    int64_t* d_mask_ptr = nullptr;   // N + 1 (word offset of row I)
    unsigned* d_masks = nullptr;

    // panel reduction (groups.cu, reduce_panels.cu): point groups, their unions, row tiles
    int reduce_mode = 0;             // 0 = automatic, 1 = row-owner kernel, 2 = panel kernel whenever it fits, 3 = long-row kernel
    bool have_tiles = false;
    int tg_C = 0;                    // 32-lane chunks per group union (0: panel path not applicable)
    int tg_T = 0;                    // block rows per tile (even)
    int tg_nstage = 0;               // stages of the group ring
    int tg_CW = 0;                   // consumer warps per row group
    bool tg_grad_only = false;       // the groups' staged rows travel as a 2-D tensor copy of the gradient rows only
    int tg_R = 2;                    // block rows per row group (2: a pair shares the gradient loads; 1: twice the warps)
    // rpim_set_panel_shape: forced launch shape of the panel reduction (0 = automatic), read by rpim_stage_tiles
    int ov_T = 0, ov_CW = 0, ov_R = 0, ov_nstage = 0, ov_grad = 0 /*1 tensor copy, 2 plain*/, ov_tdesc = 0 /*1 warp, 2 thread*/;
    int max_ulen = 0;                // most upper block columns (diagonal included) of a row
    double tg_mean_union = 0.0;      // mean |U_g| of the last statistics pass
    int64_t ntiles = 0;
    uint8_t* d_gpos = nullptr;       // Nq x k: position of (point, support node) in its group's union
    // G group records of rpim_panel_meta_bytes(C): [32 C x 8 bytes: support position of union entry u in the
    // group's point p, 0xFF = absent][32 C ints: sorted union of the group's supports, padded with -1]
    // [8 doubles: quadrature weights, written by rpim_assemble]
    unsigned char* d_gmeta = nullptr;
    int64_t* d_tile_ptr = nullptr;   // ntiles + 1
    unsigned* d_tdesc = nullptr;     // tile descriptors, 1 + T/2 words each

    // staged shape functions: Nq x 4 x k  (per point four rows of k: phi, dphi/dx, dphi/dy, dphi/dz in support order)
    double* d_stage = nullptr;
    uint8_t* d_singular = nullptr;   // Nq
    ShapeParams sp{};
    const double* d_escale = nullptr;   // optional per-point modulus scale (caller-owned), R8b
    bool have_sp = false;

    // misc
    long long* d_flags = nullptr;    // NUM_FLAGS
    double* d_scratch = nullptr;     // small reductions (>= 4096 doubles)
    void* d_scan_tmp = nullptr;      // scan block sums
    int64_t scan_tmp_elems = 0;

    cudaEvent_t ev[8] = {};
    float phase_ms[5] = {0, 0, 0, 0, 0};
    // per-call event triples (begin shape, end shape = begin reduce, end reduce) since the last reset
    std::vector<cudaEvent_t> phase_events;
    size_t phase_events_used = 0;
    double phase_total_ms[5] = {0, 0, 0, 0, 0};   // accumulated pattern-stage times (measured at sync points)
    int64_t phase_calls[2] = {0, 0};              // build_pattern calls, assemble calls since reset

    // device buffers of the host-buffer entry points
    double *h2d_nodes = nullptr, *h2d_qpts = nullptr;
    double *hb_qw = nullptr, *hb_vals = nullptr, *hb_f = nullptr, *hb_ub = nullptr;
    int64_t* hb_bn = nullptr;
    uint8_t *hb_bm = nullptr, *hb_rp = nullptr, *hb_ci = nullptr;
    cudaStream_t side_stream = nullptr;   // device -> host copy of the index arrays, overlapped with the assembly
    cudaEvent_t side_ev[2] = {nullptr, nullptr};
};

#define RPIM_FAIL(ctx, code, ...)                          \
    do {                                                   \
        char _b[512];                                      \
        snprintf(_b, sizeof(_b), __VA_ARGS__);             \
        (ctx)->err = _b;                                   \
        return (code);                                     \
    } while (0)

#define CUDA_TRY(ctx, expr)                                                                     \
    do {                                                                                        \
        cudaError_t _e = (expr);                                                                \
        if (_e != cudaSuccess)                                                                  \
            RPIM_FAIL(ctx, (_e == cudaErrorMemoryAllocation ? RPIM_ERR_ALLOC : RPIM_ERR_CUDA),  \
                      "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
    } while (0)

#define KERNEL_CHECK(ctx)                                                                       \
    do {                                                                                        \
        (ctx)->launches++;                                                                      \
        cudaError_t _e = cudaGetLastError();                                                    \
        if (_e != cudaSuccess)                                                                  \
            RPIM_FAIL(ctx, RPIM_ERR_CUDA, "kernel launch failed: %s (%s:%d)",                   \
                      cudaGetErrorString(_e), __FILE__, __LINE__);                              \
    } while (0)

// Workspace allocator with a per-context cache: a freed block is parked and handed out again to
// the next request it fits (capacity within 2x of the request), so that repeated
// rpim_build_pattern / rpim_assemble calls on same-sized problems never reach cudaMalloc/cudaFree
// (both synchronise the device).  ws_release_cache really frees the parked blocks.
inline void ws_release_cache(rpim_ctx* ctx) {
    for (auto& b : ctx->ws_cache) { cudaFree(b.first); ctx->ws_bytes -= b.second; }
    ctx->ws_cache.clear();
}
template <typename T>
void ws_free(rpim_ctx* ctx, T** p) {
    if (*p) {
        auto it = ctx->ws_sizes.find((void*)*p);
        if (it != ctx->ws_sizes.end()) {
            ctx->ws_cache.emplace_back((void*)*p, it->second);
            ctx->ws_sizes.erase(it);
        } else {
            cudaFree(*p);
        }
    }
    *p = nullptr;
}
template <typename T>
int ws_alloc(rpim_ctx* ctx, T** p, int64_t count) {
    if (count <= 0) count = 1;
    const int64_t need = count * (int64_t)sizeof(T);
    if (*p) {   // already large enough (and not wastefully so): keep it
        auto it = ctx->ws_sizes.find((void*)*p);
        if (it != ctx->ws_sizes.end() && it->second >= need && it->second <= 2 * need + 4096) return RPIM_OK;
    }
    ws_free(ctx, p);
    int best = -1;
    for (int i = 0; i < (int)ctx->ws_cache.size(); ++i) {
        const int64_t cap = ctx->ws_cache[i].second;
        if (cap >= need && cap <= 2 * need + 4096 && (best < 0 || cap < ctx->ws_cache[best].second)) best = i;
    }
    if (best >= 0) {
        *p = (T*)ctx->ws_cache[best].first;
        ctx->ws_sizes[(void*)*p] = ctx->ws_cache[best].second;
        ctx->ws_cache.erase(ctx->ws_cache.begin() + best);
        return RPIM_OK;
    }
    cudaError_t e = cudaMalloc((void**)p, (size_t)need);
    if (e != cudaSuccess) {   // give the parked blocks back to the driver and retry once
        cudaGetLastError();
        cudaStreamSynchronize(ctx->stream);
        ws_release_cache(ctx);
        e = cudaMalloc((void**)p, (size_t)need);
    }
    if (e != cudaSuccess) {
        *p = nullptr;
        cudaGetLastError();
        RPIM_FAIL(ctx, RPIM_ERR_ALLOC, "device allocation of %lld bytes failed: %s", (long long)need,
                  cudaGetErrorString(e));
    }
    ctx->ws_sizes[(void*)*p] = need;
    ctx->ws_bytes += need;
    return RPIM_OK;
}

// ---- stages implemented in the other translation units
int rpim_scan_i32_to_i64(rpim_ctx* ctx, const int* d_in, int64_t* d_out, int64_t n);  // exclusive, writes n+1
int rpim_stage_grid_knn(rpim_ctx* ctx, const double* d_pts, int64_t M, int k, int32_t* d_support, bool build_grid);
int rpim_stage_grid_refresh(rpim_ctx* ctx, bool* out_rebuild, int64_t* out_moved);
int rpim_stage_incidence(rpim_ctx* ctx);
int rpim_stage_block_pattern(rpim_ctx* ctx);
int rpim_stage_slot_masks(rpim_ctx* ctx);
int rpim_stage_groups(rpim_ctx* ctx);   // after the support search: decides ctx->tg_C
int rpim_stage_tiles(rpim_ctx* ctx);    // after incidence + block pattern: decides ctx->have_tiles
int rpim_stage_accumulate_panels(rpim_ctx* ctx, const double* d_qw, double lambda, double mu, const double body[3],
                                double* d_vals, double* d_f);
int rpim_stage_emit_pattern(rpim_ctx* ctx, void* d_row_ptr, void* d_col_idx);
int rpim_stage_shape(rpim_ctx* ctx, const double* d_pts, const int32_t* d_support, int64_t M, double* d_stage,
                     uint8_t* d_singular);
int rpim_stage_shape_rows(rpim_ctx* ctx, const double* d_pts, const int32_t* d_support, int64_t M, double* d_stage,
                          uint8_t* d_singular);   // 1 = no specialised kernel for ctx->k
int rpim_stage_accumulate(rpim_ctx* ctx, const double* d_qw, double lambda, double mu, const double body[3],
                          double* d_vals, double* d_f);
int rpim_stage_point_loads(rpim_ctx* ctx, const int32_t* d_support, const double* d_stage, const double* d_w,
                           const double* d_t, int64_t M, double* d_f);
int rpim_stage_penalty(rpim_ctx* ctx, const int64_t* d_bc_nodes, const uint8_t* d_bc_mask, const double* d_u_bar,
                       int64_t m, double alpha, int relative, double* d_vals, double* d_f, double* out_alpha);

// Dynamic shared memory of reduce_panels_kernel<CW, T / 2> (reduce_panels.cu) for rows of up to Ucap upper
// block columns (diagonal included): byte offsets of its areas, identical on host and device.
struct PanelSmem {
    int LS;            // accumulator / column-list stride in block columns (Ucap rounded up to even)
    int hlog;          // log2 of the per-row table size (power of two >= 1.5 Ucap)
    unsigned stage_bytes;
    unsigned off_acc, off_bcol, off_hash, off_aw, off_stage, off_bar, off_rowo, total;
};
// bytes of a group's record: [jinv: 32 C x 8][union node ids: 32 C ints][weights: 8 doubles]
inline unsigned rpim_panel_meta_bytes(int C) { return 32u * C * 12u + RPIM_GROUP_POINTS * 8u; }
// the group's staged rows travel as a 2-D tensor copy of the three gradient rows per point when their 24 k bytes
// are a 16-byte multiple and fit a copy box (else as one plain bulk copy of the whole rows, phi included)
inline bool rpim_panel_grad_only(int k) { return (k & 1) == 0 && 3 * k <= 256; }
inline PanelSmem rpim_panel_smem(int C, int CW, int R, int T, int k, int Ucap, int nstage, bool grad_only) {
    PanelSmem L;
    L.LS = (Ucap + 1) & ~1;
    L.hlog = 6;
    while (2 * (1 << L.hlog) < 3 * Ucap) ++L.hlog;   // load factor <= 2/3 at the longest row, ~ 0.45 typically
    auto up16 = [](unsigned v) { return (v + 15u) & ~15u; };
    auto up128 = [](unsigned v) { return (v + 127u) & ~127u; };
    L.stage_bytes = up128((unsigned)(RPIM_GROUP_POINTS * (grad_only ? 3 : 4) * k * 8) + rpim_panel_meta_bytes(C) + 32u);
    unsigned o = 0;
    L.off_acc = o; o = up16(o + (unsigned)T * 9u * L.LS * 8u);
    L.off_bcol = o; o = up16(o + (unsigned)T * L.LS * 4u);
    L.off_hash = o; o = up16(o + (unsigned)T * (2u << L.hlog));
    L.off_aw = o; o = up16(o + (unsigned)(T / R) * CW * RPIM_GROUP_POINTS * 6u * 8u);
    L.off_stage = up128(o); o = up16(L.off_stage + (unsigned)nstage * L.stage_bytes);
    L.off_bar = o; o = up16(o + 2u * nstage * 8u);
    L.off_rowo = o; o = up16(o + (unsigned)T * 16u);
    L.total = o;
    return L;
}

// ---- small device helpers
__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }

// In-place ascending bitonic sort of n (power of two) 64-bit keys in shared memory by one warp.
__device__ __forceinline__ void warp_bitonic_u64(unsigned long long* key, int n) {
    const int lane = lane_id();
    for (int size = 2; size <= n; size <<= 1) {
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            __syncwarp();
            for (int t = lane; t < (n >> 1); t += 32) {
                int lo = 2 * t - (t & (stride - 1));
                int hi = lo + stride;
                bool up = ((lo & size) == 0);
                unsigned long long a = key[lo], b = key[hi];
                if ((a > b) == up) { key[lo] = b; key[hi] = a; }
            }
        }
    }
    __syncwarp();
}

// Same for (key, value) pairs ordered by (key, value).
__device__ __forceinline__ void warp_bitonic_u64_i32(unsigned long long* key, int* val, int n) {
    const int lane = lane_id();
    for (int size = 2; size <= n; size <<= 1) {
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            __syncwarp();
            for (int t = lane; t < (n >> 1); t += 32) {
                int lo = 2 * t - (t & (stride - 1));
                int hi = lo + stride;
                bool up = ((lo & size) == 0);
                unsigned long long a = key[lo], b = key[hi];
                int va = val[lo], vb = val[hi];
                bool gt = (a > b) || (a == b && va > vb);
                if (gt == up) { key[lo] = b; key[hi] = a; val[lo] = vb; val[hi] = va; }
            }
        }
    }
    __syncwarp();
}

__device__ __forceinline__ void warp_bitonic_i32(int* key, int n) {
    const int lane = lane_id();
    for (int size = 2; size <= n; size <<= 1) {
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            __syncwarp();
            for (int t = lane; t < (n >> 1); t += 32) {
                int lo = 2 * t - (t & (stride - 1));
                int hi = lo + stride;
                bool up = ((lo & size) == 0);
                int a = key[lo], b = key[hi];
                if ((a > b) == up) { key[lo] = b; key[hi] = a; }
            }
        }
    }
    __syncwarp();
}

__host__ __device__ __forceinline__ int next_pow2(int v) {
    int p = 1;
    while (p < v) p <<= 1;
    return p;
}
