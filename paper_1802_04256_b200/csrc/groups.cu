// Point groups and row tiles: the integer preprocessing of the panel reduction (reduce_panels.cu,
// step a6).  Built by rpim_build_pattern next to the CSR pattern; depends on the supports only.
//
//   group g   = the GB = 8 consecutive quadrature points 8g .. 8g+7 (the Gauss points of one background
//               cell when a cell carries 8 of them: their supports nearly coincide)
//   U_g       = sorted union of the supports of the group's points (32 C entries, padded with -1)
//   gpos      = position of every (point, support node) in U_g                       (one byte each)
//   gjinv     = per union entry eight bytes: byte p = support position of U_g[u] in the group's point p,
//               0xFF when that point does not hold the node
//   tile t    = the T consecutive block rows T t .. T t + T-1 (T even, <= 8)
//   tdesc     = per tile the ascending list of the groups incident to any of its rows; per (tile, group)
//               1 + T/2 words: the group id, then per row 16 bits: position u_r of the row's node in
//               U_g (low byte) and the mask of the group's points whose support contains that node (high
//               byte; 0 = the row is not incident to the group)
//
// The panel path applies when the groups fit (max |U_g| <= 128) and two rows' accumulators fit in shared
// memory; otherwise the row-owner kernel of accumulate.cu runs.
#include <cstdlib>

#include "common.cuh"

namespace {

constexpr int GB = RPIM_GROUP_POINTS;
constexpr int GSORT = 1024;     // >= GB * RPIM_MAX_K = 992 ids sorted per group
constexpr int GU_MAX = 128;     // longest union the reduction handles (4 chunks of 32 lanes)
constexpr int GW = 4;           // warps per block
constexpr int TMAX = 8;         // most block rows per tile

// One warp per group.  FILL = false: only |U_g| statistics (max, sum).  FILL = true: U_g, gpos, gu_mask.
template <bool FILL>
__global__ void __launch_bounds__(GW * 32)
group_union_kernel(int64_t Nq, int k, int C, int64_t gstep, const int32_t* __restrict__ support, int* __restrict__ max_len,
                   unsigned long long* __restrict__ sum_len,
                   uint8_t* __restrict__ gpos, unsigned char* __restrict__ gmeta) {
    __shared__ int buf_s[GW][GSORT];
    __shared__ int ul_s[GW][GU_MAX];
    __shared__ __align__(16) uint8_t ji_s[GW][GU_MAX * GB];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int* buf = buf_s[wid];
    int* ul = ul_s[wid];
    uint8_t* ji = ji_s[wid];
    const int64_t G = (Nq + GB - 1) / GB;
    const int gcap = 32 * C;
    // gstep > 1: a sample (every gstep-th group), statistics only
    for (int64_t gs = (int64_t)blockIdx.x * GW + wid; gs * gstep < G; gs += (int64_t)gridDim.x * GW) {
        const int64_t g = gs * gstep;
        const int64_t q0 = g * GB;
        const int nb = (int)min((int64_t)GB, Nq - q0);
        const int n = nb * k;
        const int32_t* src = support + q0 * k;
        const int np = next_pow2(n);
        __syncwarp();
        for (int i = lane; i < np; i += 32) buf[i] = (i < n) ? src[i] : 0x7FFFFFFF;
        __syncwarp();
        warp_bitonic_i32(buf, np);
        int total = 0;
        for (int i0 = 0; i0 < n; i0 += 32) {
            const int i = i0 + lane;
            const bool fresh = i < n && (i == 0 || buf[i] != buf[i - 1]);
            const unsigned m = __ballot_sync(0xffffffffu, fresh);
            const int pos = total + __popc(m & ((1u << lane) - 1u));
            if (fresh && pos < GU_MAX) ul[pos] = buf[i];
            total += __popc(m);
        }
        __syncwarp();
        if constexpr (!FILL) {
            if (lane == 0) {
                atomicMax(max_len, total);
                atomicAdd(sum_len, (unsigned long long)total);
            }
        } else {
            // total <= gcap: the host chose C from the statistics pass
            unsigned char* rec = gmeta + g * (int64_t)(gcap * 12 + GB * 8);   // rpim_panel_meta_bytes(C)
            int* gu_nodes = reinterpret_cast<int*>(rec + gcap * 8);
            for (int u = lane; u < gcap; u += 32) gu_nodes[u] = (u < total) ? ul[u] : -1;
            for (int u = lane; u < GU_MAX * GB / 4; u += 32) reinterpret_cast<unsigned*>(ji)[u] = 0xFFFFFFFFu;
            __syncwarp();
            for (int i = lane; i < n; i += 32) {
                const int node = src[i];
                int lo = 0, hi = total - 1;
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (ul[mid] < node) lo = mid + 1; else hi = mid;
                }
                gpos[q0 * k + i] = (uint8_t)lo;
                const int p = i / k;
                ji[lo * GB + p] = (uint8_t)(i - p * k);
            }
            __syncwarp();
            uint4* dst = reinterpret_cast<uint4*>(rec);
            for (int e = lane; e < gcap * GB / 16; e += 32) dst[e] = reinterpret_cast<const uint4*>(ji)[e];
        }
    }
}

// One thread per tile: merge of the T rows' incidence lists (ascending point ids) by point group.
template <bool FILL>
__global__ void __launch_bounds__(128)
tile_desc_thread_kernel(int64_t N, int64_t ntiles, int T, int k, const int64_t* __restrict__ inc_ptr,
                 const int32_t* __restrict__ inc_q, const uint8_t* __restrict__ inc_j,
                 const uint8_t* __restrict__ gpos, int* __restrict__ count, const int64_t* __restrict__ tile_ptr,
                 unsigned* __restrict__ tdesc) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntiles) return;
    const int DW = 1 + T / 2;
    int64_t c[TMAX], e[TMAX];
    int gq[TMAX];   // group of the next entry of row r (INT_MAX: list exhausted)
#pragma unroll
    for (int r = 0; r < TMAX; ++r) {
        const int64_t I = t * T + r;
        c[r] = e[r] = 0;
        if (r < T && I < N) { c[r] = inc_ptr[I]; e[r] = inc_ptr[I + 1]; }
        gq[r] = (c[r] < e[r]) ? inc_q[c[r]] / GB : 0x7FFFFFFF;
    }
    int n = 0;
    unsigned* dst = FILL ? tdesc + tile_ptr[t] * DW : nullptr;
    while (true) {
        int g = gq[0];
#pragma unroll
        for (int r = 1; r < TMAX; ++r) g = min(g, gq[r]);
        if (g == 0x7FFFFFFF) break;
        unsigned half[TMAX];
#pragma unroll
        for (int r = 0; r < TMAX; ++r) half[r] = 0u;
#pragma unroll
        for (int r = 0; r < TMAX; ++r) {
            if (gq[r] != g) continue;
            unsigned m = 0u, u = 0u;
            while (true) {
                const int q = inc_q[c[r]];
                m |= 1u << (q - g * GB);
                if (FILL) u = gpos[(int64_t)q * k + inc_j[c[r]]];
                ++c[r];
                if (c[r] >= e[r]) { gq[r] = 0x7FFFFFFF; break; }
                const int gn = inc_q[c[r]] / GB;
                if (gn != g) { gq[r] = gn; break; }
            }
            half[r] = u | (m << 8);
        }
        if (FILL) {
            dst[(int64_t)n * DW] = (unsigned)g;
#pragma unroll
            for (int w = 0; w < TMAX / 2; ++w)
                if (1 + w < DW) dst[(int64_t)n * DW + 1 + w] = half[2 * w] | (half[2 * w + 1] << 16);
        }
        ++n;
    }
    if (!FILL) count[t] = n;
}


// One warp per tile: the T rows' incidence lists (ascending point ids) cut into runs of one point group each
// (lane-parallel, 32 entries at a time), the (group, row, union position, point mask) items sorted by group in
// shared memory, one descriptor per distinct group.  FILL = false counts the descriptors of a tile, FILL = true
// writes them.  A tile with more than TD_ITEMS items or TD_GROUPS groups raises FLAG_PAT_CAP's neighbour
// FLAG_TILE_CAP: the caller then takes the thread-per-tile kernel above.  (One thread per tile has the parallelism only
// when there are hundreds of thousands of tiles; one warp per tile is 2.3x faster at `slope`, 7.8k tiles, and slower
// at `stress`, 341k tiles, where its 26 KB of shared memory per warp leave 8 warps per SM.)
constexpr int TD_ITEMS = 2048;   // (row, group) items of a tile (runs cut by a 32-entry boundary count twice)
constexpr int TD_GROUPS = 512;   // distinct groups of a tile
constexpr int TD_WARPS = 4;
constexpr int TD_DWMAX = 1 + TMAX / 2;

template <bool FILL>
__global__ void __launch_bounds__(TD_WARPS * 32)
tile_desc_warp_kernel(int64_t N, int64_t ntiles, int T, int k, const int64_t* __restrict__ inc_ptr,
                 const int32_t* __restrict__ inc_q, const uint8_t* __restrict__ inc_j,
                 const uint8_t* __restrict__ gpos, int* __restrict__ count, const int64_t* __restrict__ tile_ptr,
                 unsigned* __restrict__ tdesc, long long* __restrict__ flags) {
    constexpr unsigned FULLW = 0xffffffffu;
    extern __shared__ __align__(16) unsigned char td_smem[];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned long long* items = reinterpret_cast<unsigned long long*>(td_smem) + (size_t)wid * TD_ITEMS;
    unsigned* desc = reinterpret_cast<unsigned*>(td_smem + (size_t)TD_WARPS * TD_ITEMS * 8) + (size_t)wid * TD_GROUPS * TD_DWMAX;   // (FILL only)
    const int DW = 1 + T / 2;
    const unsigned lt = (1u << lane) - 1u;
    for (int64_t t = (int64_t)blockIdx.x * TD_WARPS + wid; t < ntiles; t += (int64_t)gridDim.x * TD_WARPS) {
        __syncwarp();
        int n = 0;
        for (int r = 0; r < T; ++r) {
            const int64_t I = t * T + r;
            if (I >= N) break;
            const int64_t pa = inc_ptr[I];
            const int np = (int)(inc_ptr[I + 1] - pa);
            for (int t0 = 0; t0 < np; t0 += 32) {
                const int i = t0 + lane;
                const int q = i < np ? inc_q[pa + i] : -1;
                const int g = q >= 0 ? q / GB : -1;
                const unsigned bit = q >= 0 ? 1u << (q % GB) : 0u;
                const int gp = __shfl_up_sync(FULLW, g, 1);
                const bool head = q >= 0 && (lane == 0 || g != gp);
                unsigned m = bit;
#pragma unroll
                for (int d = 1; d < GB; ++d) {
                    const int gd = __shfl_down_sync(FULLW, g, d);
                    const unsigned bd = __shfl_down_sync(FULLW, bit, d);
                    if (lane + d < 32 && gd == g) m |= bd;
                }
                const unsigned heads = __ballot_sync(FULLW, head);
                const int pos = n + __popc(heads & lt);
                if (head && pos < TD_ITEMS) {
                    // every point of the group that holds the row's node holds it at the same union position
                    const unsigned u = FILL ? gpos[(int64_t)q * k + inc_j[pa + i]] : 0u;
                    items[pos] = ((unsigned long long)(unsigned)g << 32) | ((unsigned)r << 16) | (m << 8) | u;   // low 16 bits: the row's descriptor half
                }
                n += __popc(heads);
            }
        }
        if (n > TD_ITEMS) {
            if (lane == 0) atomicAdd((unsigned long long*)&flags[FLAG_TILE_CAP], 1ull);
            if (!FILL && lane == 0) count[t] = 0;
            continue;
        }
        const int npow = next_pow2(max(n, 1));
        for (int i = n + lane; i < npow; i += 32) items[i] = ~0ull;
        __syncwarp();
        warp_bitonic_u64(items, npow);
        // distinct groups: item i opens a descriptor when its group differs from the previous item's
        int ng = 0;
        const int64_t out0 = FILL ? tile_ptr[t] : 0;
        if (FILL) {
            const int cap = min((int)(tile_ptr[t + 1] - out0), TD_GROUPS) * DW;
            for (int i = lane; i < cap; i += 32) desc[i] = 0u;
            __syncwarp();
        }
        for (int i0 = 0; i0 < n; i0 += 32) {
            const int i = i0 + lane;
            const unsigned long long v = i < n ? items[i] : ~0ull;
            const unsigned g = (unsigned)(v >> 32);
            const unsigned gprev = (i > 0 && i < n) ? (unsigned)(items[i - 1] >> 32) : 0xFFFFFFFFu;
            const bool head = i < n && (i == 0 || g != gprev);
            const unsigned heads = __ballot_sync(FULLW, head);
            if (FILL && i < n) {
                const int d = ng + __popc(heads & (lt | (1u << lane))) - 1;   // descriptor of this item's group
                if (d < TD_GROUPS) {
                    if (head) desc[d * DW] = g;
                    const unsigned r = (unsigned)(v >> 16) & 0xFFFFu, half = (unsigned)v & 0xFFFFu;
                    atomicOr(&desc[d * DW + 1 + (r >> 1)], half << (16 * (r & 1)));
                }
            }
            ng += __popc(heads);
        }
        if (ng > TD_GROUPS) {
            if (lane == 0) atomicAdd((unsigned long long*)&flags[FLAG_TILE_CAP], 1ull);
            if (!FILL && lane == 0) count[t] = 0;
            continue;
        }
        if (!FILL) {
            if (lane == 0) count[t] = ng;
        } else {
            __syncwarp();
            unsigned* dst = tdesc + out0 * DW;
            for (int i = lane; i < ng * DW; i += 32) dst[i] = desc[i];
        }
    }
}

}  // namespace

// After the support search: unions of the point groups; decides whether the panel reduction applies
// (ctx->tg_C > 0) and, if so, leaves gpos and the group records in the workspace.
int rpim_stage_groups(rpim_ctx* ctx) {
    cudaStream_t st = ctx->stream;
    ctx->tg_C = 0;
    ctx->have_tiles = false;
    ctx->tg_mean_union = 0.0;
    if (ctx->reduce_mode == 1 || ctx->reduce_mode == 3) return RPIM_OK;
    const int64_t Nq = ctx->Nq, G = (Nq + GB - 1) / GB;
    const int k = ctx->k;
    int* d_max = (int*)ctx->d_scratch;
    unsigned long long* d_sum = (unsigned long long*)(ctx->d_scratch + 1);
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_scratch, 0, 2 * sizeof(double), st));
    const unsigned nb = (unsigned)std::min<int64_t>((G + GW - 1) / GW, 148 * 16);
    int h_max = 0;
    unsigned long long h_sum = 0;
    if (ctx->reduce_mode == 0 && G > 16384) {
        // automatic choice on a large problem: a sample of about 4096 groups first; unions far over the bar
        // (one point per cell: mean |U_g| ~ 3 k) settle it without the full pass
        const int64_t gstep = G / 4096, Gs = (G + gstep - 1) / gstep;
        group_union_kernel<false><<<(unsigned)((Gs + GW - 1) / GW), GW * 32, 0, st>>>(Nq, k, 0, gstep, ctx->d_support, d_max, d_sum,
                                                                                   nullptr, nullptr);
        KERNEL_CHECK(ctx);
        CUDA_TRY(ctx, cudaMemcpyAsync(&h_sum, d_sum, sizeof(h_sum), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(ctx, cudaStreamSynchronize(st));
        ctx->tg_mean_union = (double)h_sum / (double)Gs;
        if (ctx->tg_mean_union > 1.25 * RPIM_PANEL_MAX_UNION_RATIO * k) return RPIM_OK;
        CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_scratch, 0, 2 * sizeof(double), st));
        h_sum = 0;
    }
    group_union_kernel<false><<<nb, GW * 32, 0, st>>>(Nq, k, 0, 1, ctx->d_support, d_max, d_sum, nullptr, nullptr);
    KERNEL_CHECK(ctx);
    CUDA_TRY(ctx, cudaMemcpyAsync(&h_max, d_max, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaMemcpyAsync(&h_sum, d_sum, sizeof(h_sum), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    ctx->tg_mean_union = (double)h_sum / (double)G;
    if (h_max > GU_MAX) return RPIM_OK;
    // automatic choice: the panel kernel pays when a group's points share most of their supports
    if (ctx->reduce_mode == 0 && ctx->tg_mean_union > RPIM_PANEL_MAX_UNION_RATIO * k) return RPIM_OK;
    int C = (h_max + 31) / 32;
    if (C < 2) C = 2;
    int rc;
    if ((rc = ws_alloc(ctx, &ctx->d_gpos, Nq * k))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_gmeta, G * (int64_t)rpim_panel_meta_bytes(C)))) return rc;
    group_union_kernel<true><<<nb, GW * 32, 0, st>>>(Nq, k, C, 1, ctx->d_support, nullptr, nullptr, ctx->d_gpos, ctx->d_gmeta);
    KERNEL_CHECK(ctx);
    ctx->tg_C = C;
    return RPIM_OK;
}

namespace {
// most upper block columns (diagonal included) of a block row
__global__ void max_ulen_kernel(int64_t N, const int* __restrict__ blen, const int* __restrict__ bdiag, int* __restrict__ out) {
    int m = 0;
    for (int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; I < N; I += (int64_t)gridDim.x * blockDim.x)
        if (blen[I] > 0) m = max(m, blen[I] - bdiag[I]);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, d));
    if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, m);
}
}  // namespace

// After incidence + block pattern: rows per tile and ring depth from the shared-memory budget, tile descriptors.
int rpim_stage_tiles(rpim_ctx* ctx) {
    cudaStream_t st = ctx->stream;
    ctx->have_tiles = false;
    if (ctx->tg_C == 0) return RPIM_OK;
    const int64_t N = ctx->N;
    int* d_max = (int*)ctx->d_scratch;
    CUDA_TRY(ctx, cudaMemsetAsync(d_max, 0, sizeof(int), st));
    max_ulen_kernel<<<(unsigned)std::min<int64_t>((N + 255) / 256, 1024), 256, 0, st>>>(N, ctx->d_blen, ctx->d_bdiag, d_max);
    KERNEL_CHECK(ctx);
    CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->max_ulen, d_max, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    const int Ucap = std::max(ctx->max_ulen, 1);
    // Launch shape of reduce_panels_kernel.  Measured on B200: one block row per consumer
    // warp group and two warps per group (13 warps at T = 6) beat row pairs with three warps (10 warps) by 7 % at
    // `stress`; the most rows per tile (8, 6, 4, 2) that leave room for a ring of five stages (else four, three),
    // then the deepest ring (<= 8).  rpim_set_panel_shape overrides any of them (tuning and tests; validated there).
    int CW = ctx->ov_CW ? ctx->ov_CW : 2;
    int R = ctx->ov_R ? ctx->ov_R : 1;
    if (R == 1 && CW > 3) CW = 3;
    const unsigned budget = 227u * 1024u;
    // rows per tile and ring depth for one way of staging the groups' rows
    auto choose = [&](bool grad_only, int& T, int& nstage) {
        T = 0;
        nstage = 0;
        // (a deep ring decouples the consumer warps: at `stress` 6 rows with 6 stages beat 8 rows with 3 by 36 %)
        if (Ucap <= 1024)
            for (int need = 5; need >= 3 && T == 0; --need)
                for (int t = TMAX; t >= 2 && T == 0; t -= 2)
                    if (rpim_panel_smem(ctx->tg_C, CW, R, t, ctx->k, Ucap, need, grad_only).total <= budget) T = t;
        if (ctx->ov_T && Ucap <= 1024) T = ctx->ov_T;   // (the row-length guard holds for a forced T as well)
        if (T == 0) return;
        for (nstage = 8; nstage > 2 && rpim_panel_smem(ctx->tg_C, CW, R, T, ctx->k, Ucap, nstage, grad_only).total > budget; --nstage) {}
        if (ctx->ov_nstage) nstage = ctx->ov_nstage;
        if (rpim_panel_smem(ctx->tg_C, CW, R, T, ctx->k, Ucap, nstage, grad_only).total > budget) T = 0;
    };
    // Whole staged rows by one plain bulk copy, or the gradient rows only by a 2-D tensor copy (three quarters of
    // the bytes, but eight row transfers inside the request: slower at `slope`, where the plain ring is already
    // six deep).  The tensor copy is taken when it buys rows per tile or ring depth.
    int T = 0, nstage = 0;
    bool grad_only = false;
    choose(false, T, nstage);
    if (rpim_panel_grad_only(ctx->k)) {
        int Tg = 0, ng = 0;
        choose(true, Tg, ng);
        if (Tg > T || (Tg == T && ng > nstage)) { T = Tg; nstage = ng; grad_only = true; }
    }
    if (ctx->ov_grad) {
        const bool want = ctx->ov_grad == 1;
        if (want != grad_only && (!want || rpim_panel_grad_only(ctx->k))) { grad_only = want; choose(grad_only, T, nstage); }
    }
    if (T == 0) { ctx->tg_C = 0; return RPIM_OK; }   // rows too long to keep two of them on chip
    const int64_t ntiles = (N + T - 1) / T;
    const int DW = 1 + T / 2;
    int rc;
    int* d_cnt = nullptr;
    if ((rc = ws_alloc(ctx, &d_cnt, ntiles))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_tile_ptr, ntiles + 1))) { ws_free(ctx, &d_cnt); return rc; }
    // descriptors: one warp per tile when the tiles are few (a thread per tile would leave the GPU empty), else --
    // or when a tile overflows the warp kernel's shared-memory lists -- one thread per tile
    const unsigned nbw = (unsigned)std::min<int64_t>((ntiles + TD_WARPS - 1) / TD_WARPS, 148 * 16);
    const unsigned nbt = (unsigned)((ntiles + 127) / 128);
    const size_t td_smem_cnt = (size_t)TD_WARPS * TD_ITEMS * 8;                                  // the count pass keeps no descriptors
    const size_t td_smem = (size_t)TD_WARPS * (TD_ITEMS * 8 + TD_GROUPS * TD_DWMAX * 4);
    bool by_warp = ntiles <= 65536;
    if (ctx->ov_tdesc) by_warp = ctx->ov_tdesc == 1;   // rpim_set_panel_shape: tests
    if (by_warp) {
        CUDA_TRY(ctx, cudaFuncSetAttribute(tile_desc_warp_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)td_smem_cnt));
        CUDA_TRY(ctx, cudaFuncSetAttribute(tile_desc_warp_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)td_smem));
        CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_flags + FLAG_TILE_CAP, 0, sizeof(long long), st));
        tile_desc_warp_kernel<false><<<nbw, TD_WARPS * 32, td_smem_cnt, st>>>(N, ntiles, T, ctx->k, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_inc_j,
                                                                             ctx->d_gpos, d_cnt, nullptr, nullptr, ctx->d_flags);
        ctx->launches++;
        long long tile_cap = 0;
        cudaError_t e = cudaMemcpyAsync(&tile_cap, ctx->d_flags + FLAG_TILE_CAP, sizeof(long long), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { ws_free(ctx, &d_cnt); RPIM_FAIL(ctx, RPIM_ERR_CUDA, "tile descriptor count failed: %s", cudaGetErrorString(e)); }
        if (tile_cap) by_warp = false;
    }
    if (!by_warp) {
        tile_desc_thread_kernel<false><<<nbt, 128, 0, st>>>(N, ntiles, T, ctx->k, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_inc_j,
                                                            ctx->d_gpos, d_cnt, nullptr, nullptr);
        ctx->launches++;
    }
    if (cudaGetLastError() != cudaSuccess) { ws_free(ctx, &d_cnt); RPIM_FAIL(ctx, RPIM_ERR_CUDA, "tile descriptor count launch failed"); }
    rc = rpim_scan_i32_to_i64(ctx, d_cnt, ctx->d_tile_ptr, ntiles);
    ws_free(ctx, &d_cnt);
    if (rc) return rc;
    int64_t total = 0;
    CUDA_TRY(ctx, cudaMemcpyAsync(&total, ctx->d_tile_ptr + ntiles, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    if ((rc = ws_alloc(ctx, &ctx->d_tdesc, std::max<int64_t>(total, 1) * DW))) return rc;
    if (by_warp)
        tile_desc_warp_kernel<true><<<nbw, TD_WARPS * 32, td_smem, st>>>(N, ntiles, T, ctx->k, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_inc_j,
                                                                        ctx->d_gpos, nullptr, ctx->d_tile_ptr, ctx->d_tdesc, ctx->d_flags);
    else
        tile_desc_thread_kernel<true><<<nbt, 128, 0, st>>>(N, ntiles, T, ctx->k, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_inc_j,
                                                           ctx->d_gpos, nullptr, ctx->d_tile_ptr, ctx->d_tdesc);
    KERNEL_CHECK(ctx);
    ctx->tg_T = T;
    ctx->tg_CW = CW;
    ctx->tg_R = R;
    ctx->tg_grad_only = grad_only;
    ctx->tg_nstage = nstage;
    ctx->ntiles = ntiles;
    ctx->have_tiles = true;
    return RPIM_OK;
}
