// Step a2 (R2): node -> point incidence lists, block-CSR pattern (union of
// supp x supp), scalar CSR emission.  Integer work only; every list is sorted, so the
// result does not depend on the order in which threads happen to run.
#include "common.cuh"

namespace {

// ------------------------------------------------------------------ incidence (transpose of the support table)
__global__ void inc_count_kernel(const int32_t* __restrict__ support, int64_t total, int* __restrict__ count) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x)
        atomicAdd(&count[support[e]], 1);
}

__global__ void inc_fill_kernel(const int32_t* __restrict__ support, int64_t total, int k,
                                const int64_t* __restrict__ inc_ptr, int* __restrict__ cursor,
                                int32_t* __restrict__ inc_q, uint8_t* __restrict__ inc_j) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        int node = support[e];
        int p = atomicAdd(&cursor[node], 1);
        int64_t dst = inc_ptr[node] + p;
        inc_q[dst] = (int32_t)(e / k);
        inc_j[dst] = (uint8_t)(e % k);
    }
}

constexpr int INC_CAP = 4096;   // longest incidence list sorted on chip
constexpr int INC_WARPS = 4;

// one warp per node: sort its list ascending by point id (the position byte rides along)
__global__ void __launch_bounds__(INC_WARPS * 32)
inc_sort_kernel(int64_t N, const int64_t* __restrict__ inc_ptr, int32_t* __restrict__ inc_q,
                uint8_t* __restrict__ inc_j, long long* __restrict__ flags) {
    extern __shared__ unsigned char smem_raw[];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned long long* key = (unsigned long long*)smem_raw + (size_t)wid * INC_CAP;
    for (int64_t I = (int64_t)blockIdx.x * INC_WARPS + wid; I < N; I += (int64_t)gridDim.x * INC_WARPS) {
        const int64_t a = inc_ptr[I];
        const int len = (int)(inc_ptr[I + 1] - a);
        if (len <= 1) continue;
        if (len > INC_CAP) {
            if (lane == 0) atomicAdd((unsigned long long*)&flags[FLAG_INC_CAP], 1ull);
            continue;
        }
        const int np = next_pow2(len);
        for (int i = lane; i < np; i += 32)
            key[i] = (i < len) ? (((unsigned long long)(unsigned)inc_q[a + i] << 8) | inc_j[a + i])
                               : 0xFFFFFFFFFFFFFFFFull;
        __syncwarp();
        warp_bitonic_u64(key, np);
        for (int i = lane; i < len; i += 32) {
            inc_q[a + i] = (int32_t)(key[i] >> 8);
            inc_j[a + i] = (uint8_t)(key[i] & 0xFF);
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------ block rows: union of the supports of incident points
constexpr int PAT_HASH = 4096;          // open-addressing table per warp (power of two)
constexpr int PAT_MAXROW = 2048;        // longest block row handled
constexpr int PAT_WARPS = 4;

__device__ __forceinline__ unsigned pat_hash(int key) { return ((unsigned)key * 2654435761u) >> 20; }   // 12 bits

// returns the number of distinct columns of block row I (all lanes), leaving them in `table`;
// PAT_MAXROW + 1 if the row does not fit
__device__ __forceinline__ int row_union(int* table, int64_t I, const int64_t* __restrict__ inc_ptr,
                                         const int32_t* __restrict__ inc_q, const int32_t* __restrict__ support,
                                         int k) {
    const int lane = lane_id();
    for (int i = lane; i < PAT_HASH; i += 32) table[i] = -1;
    __syncwarp();
    int fresh = 0;
    bool overflow = false;
    const int64_t a = inc_ptr[I], b = inc_ptr[I + 1];
    for (int64_t p = a; p < b; ++p) {
        const int32_t* s = support + (int64_t)inc_q[p] * k;
        for (int j = lane; j < k; j += 32) {
            int key = s[j];
            unsigned h = pat_hash(key) & (PAT_HASH - 1);
            for (int probes = 0;; ++probes) {
                if (probes >= PAT_HASH) { overflow = true; break; }
                int old = atomicCAS(&table[h], -1, key);
                if (old == -1) { ++fresh; break; }
                if (old == key) break;
                h = (h + 1) & (PAT_HASH - 1);
            }
        }
        // every 8 points (<= 8 * RPIM_MAX_K new keys) stop if the row is already too long, so the
        // table never fills up: 2048 + 992 < PAT_HASH
        if (((p - a) & 7) == 7) {
            int tot = fresh;
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, d);
            if (tot > PAT_MAXROW || __any_sync(0xffffffffu, overflow)) return PAT_MAXROW + 1;
        }
    }
    if (__any_sync(0xffffffffu, overflow)) return PAT_MAXROW + 1;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) fresh += __shfl_xor_sync(0xffffffffu, fresh, d);
    __syncwarp();
    return fresh;
}

__global__ void __launch_bounds__(PAT_WARPS * 32)
brow_count_kernel(int64_t N, const int64_t* __restrict__ inc_ptr, const int32_t* __restrict__ inc_q,
                  const int32_t* __restrict__ support, int k, int* __restrict__ blen, long long* __restrict__ flags) {
    extern __shared__ int pat_smem[];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int* table = pat_smem + (size_t)wid * PAT_HASH;
    for (int64_t I = (int64_t)blockIdx.x * PAT_WARPS + wid; I < N; I += (int64_t)gridDim.x * PAT_WARPS) {
        const int L = row_union(table, I, inc_ptr, inc_q, support, k);
        if (L > PAT_MAXROW && lane == 0) atomicAdd((unsigned long long*)&flags[FLAG_PAT_CAP], 1ull);
        if (lane == 0) blen[I] = min(L, PAT_MAXROW);
        __syncwarp();
    }
}

__global__ void __launch_bounds__(PAT_WARPS * 32)
brow_fill_kernel(int64_t N, const int64_t* __restrict__ inc_ptr, const int32_t* __restrict__ inc_q,
                 const int32_t* __restrict__ support, int k, const int64_t* __restrict__ brow_ptr,
                 int32_t* __restrict__ bcol, int* __restrict__ bdiag) {
    extern __shared__ int pat_smem[];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int* table = pat_smem + (size_t)wid * PAT_HASH;
    int* list = pat_smem + (size_t)PAT_WARPS * PAT_HASH + (size_t)wid * PAT_MAXROW;
    for (int64_t I = (int64_t)blockIdx.x * PAT_WARPS + wid; I < N; I += (int64_t)gridDim.x * PAT_WARPS) {
        const int L = row_union(table, I, inc_ptr, inc_q, support, k);
        if (L > PAT_MAXROW) continue;   // reported by the count pass
        // compact the table into the list
        int base = 0;
        for (int i0 = 0; i0 < PAT_HASH; i0 += 32) {
            int v = table[i0 + lane];
            unsigned m = __ballot_sync(0xffffffffu, v >= 0);
            if (v >= 0) list[base + __popc(m & ((1u << lane) - 1))] = v;
            base += __popc(m);
        }
        const int np = next_pow2(L);
        for (int i = L + lane; i < np; i += 32) list[i] = 0x7FFFFFFF;
        __syncwarp();
        warp_bitonic_i32(list, np);
        const int64_t o = brow_ptr[I];
        for (int i = lane; i < L; i += 32) {
            int c = list[i];
            bcol[o + i] = c;
            if (c == (int)I) bdiag[I] = i;
        }
        __syncwarp();
    }
}

__global__ void max_i32_kernel(const int* __restrict__ v, int64_t n, int* __restrict__ out) {
    int m = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        m = max(m, v[i]);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, d));
    if ((threadIdx.x & 31) == 0) atomicMax(out, m);
}

// ------------------------------------------------------------------ scalar CSR emission (3x3 expansion)
template <typename IdxT>
__global__ void emit_rowptr_kernel(int64_t N, const int64_t* __restrict__ brow_ptr, IdxT* __restrict__ row_ptr) {
    int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (I > N) return;
    if (I == N) { row_ptr[3 * N] = (IdxT)(9 * brow_ptr[N]); return; }
    const int64_t o = brow_ptr[I], L = brow_ptr[I + 1] - o;
#pragma unroll
    for (int a = 0; a < 3; ++a) row_ptr[3 * I + a] = (IdxT)(9 * o + a * 3 * L);
}

template <typename IdxT>
__global__ void __launch_bounds__(256)
emit_colidx_kernel(int64_t N, const int64_t* __restrict__ brow_ptr, const int32_t* __restrict__ bcol,
                   IdxT* __restrict__ col_idx) {
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int64_t I = (int64_t)blockIdx.x * 8 + wid; I < N; I += (int64_t)gridDim.x * 8) {
        const int64_t o = brow_ptr[I];
        const int L = (int)(brow_ptr[I + 1] - o);
        for (int a = 0; a < 3; ++a) {
            IdxT* dst = col_idx + 9 * o + (int64_t)a * 3 * L;
            for (int i = lane; i < 3 * L; i += 32) dst[i] = (IdxT)(3 * (int64_t)bcol[o + i / 3] + i % 3);
        }
    }
}

}  // namespace

int rpim_stage_incidence(rpim_ctx* ctx) {
    cudaStream_t st = ctx->stream;
    const int64_t N = ctx->N, total = ctx->Nq * ctx->k;
    int rc;
    if ((rc = ws_alloc(ctx, &ctx->d_inc_count, N))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_inc_ptr, N + 1))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_inc_q, total))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_inc_j, total))) return rc;
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_inc_count, 0, N * sizeof(int), st));
    const unsigned nb = (unsigned)std::min<int64_t>((total + 255) / 256, 148 * 32);
    inc_count_kernel<<<nb, 256, 0, st>>>(ctx->d_support, total, ctx->d_inc_count);
    KERNEL_CHECK(ctx);
    if ((rc = rpim_scan_i32_to_i64(ctx, ctx->d_inc_count, ctx->d_inc_ptr, N))) return rc;
    // longest list (for capacity checks and launch sizing later)
    int* d_max = (int*)ctx->d_scratch;
    CUDA_TRY(ctx, cudaMemsetAsync(d_max, 0, sizeof(int), st));
    max_i32_kernel<<<(unsigned)std::min<int64_t>((N + 255) / 256, 1024), 256, 0, st>>>(ctx->d_inc_count, N, d_max);
    KERNEL_CHECK(ctx);
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_inc_count, 0, N * sizeof(int), st));
    inc_fill_kernel<<<nb, 256, 0, st>>>(ctx->d_support, total, ctx->k, ctx->d_inc_ptr, ctx->d_inc_count,
                                        ctx->d_inc_q, ctx->d_inc_j);
    KERNEL_CHECK(ctx);
    const size_t smem = (size_t)INC_WARPS * INC_CAP * sizeof(unsigned long long);
    CUDA_TRY(ctx, cudaFuncSetAttribute(inc_sort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    inc_sort_kernel<<<(unsigned)std::min<int64_t>((N + INC_WARPS - 1) / INC_WARPS, 148 * 16), INC_WARPS * 32, smem,
                      st>>>(N, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_inc_j, ctx->d_flags);
    KERNEL_CHECK(ctx);
    CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->max_inc, d_max, sizeof(int), cudaMemcpyDeviceToHost, st));
    return RPIM_OK;
}

int rpim_stage_block_pattern(rpim_ctx* ctx) {
    cudaStream_t st = ctx->stream;
    const int64_t N = ctx->N;
    int rc;
    if ((rc = ws_alloc(ctx, &ctx->d_blen, N))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_brow_ptr, N + 1))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_bdiag, N))) return rc;
    const unsigned nb = (unsigned)std::min<int64_t>((N + PAT_WARPS - 1) / PAT_WARPS, 148 * 16);
    const size_t smem_cnt = (size_t)PAT_WARPS * PAT_HASH * sizeof(int);
    const size_t smem_fill = smem_cnt + (size_t)PAT_WARPS * PAT_MAXROW * sizeof(int);
    CUDA_TRY(ctx, cudaFuncSetAttribute(brow_count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cnt));
    CUDA_TRY(ctx, cudaFuncSetAttribute(brow_fill_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_fill));
    brow_count_kernel<<<nb, PAT_WARPS * 32, smem_cnt, st>>>(N, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_support, ctx->k,
                                                     ctx->d_blen, ctx->d_flags);
    KERNEL_CHECK(ctx);
    if ((rc = rpim_scan_i32_to_i64(ctx, ctx->d_blen, ctx->d_brow_ptr, N))) return rc;
    int* d_max = (int*)ctx->d_scratch;
    CUDA_TRY(ctx, cudaMemsetAsync(d_max, 0, sizeof(int), st));
    max_i32_kernel<<<(unsigned)std::min<int64_t>((N + 255) / 256, 1024), 256, 0, st>>>(ctx->d_blen, N, d_max);
    KERNEL_CHECK(ctx);
    long long h_flags[NUM_FLAGS];
    CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->nnzb, ctx->d_brow_ptr + N, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->max_blen, d_max, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaMemcpyAsync(h_flags, ctx->d_flags, sizeof(h_flags), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    if (h_flags[FLAG_KNN_CAP])
        RPIM_FAIL(ctx, RPIM_ERR_CAPACITY, "kNN: %lld points need more than the on-chip candidate capacity (or k > N)",
                  h_flags[FLAG_KNN_CAP]);
    if (h_flags[FLAG_INC_CAP])
        RPIM_FAIL(ctx, RPIM_ERR_CAPACITY, "incidence: %lld nodes belong to more than %d supports", h_flags[FLAG_INC_CAP],
                  INC_CAP);
    if (h_flags[FLAG_PAT_CAP])
        RPIM_FAIL(ctx, RPIM_ERR_CAPACITY, "pattern: %lld block rows are longer than %d", h_flags[FLAG_PAT_CAP],
                  PAT_MAXROW);
    if ((rc = ws_alloc(ctx, &ctx->d_bcol, ctx->nnzb))) return rc;
    brow_fill_kernel<<<nb, PAT_WARPS * 32, smem_fill, st>>>(N, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_support, ctx->k,
                                                    ctx->d_brow_ptr, ctx->d_bcol, ctx->d_bdiag);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}

int rpim_stage_emit_pattern(rpim_ctx* ctx, void* d_row_ptr, void* d_col_idx) {
    cudaStream_t st = ctx->stream;
    const int64_t N = ctx->N;
    const unsigned nbr = (unsigned)((N + 1 + 255) / 256);
    const unsigned nbc = (unsigned)std::min<int64_t>((N + 7) / 8, 148 * 32);
    if (ctx->index_bits == 32) {
        if (d_row_ptr) { emit_rowptr_kernel<int32_t><<<nbr, 256, 0, st>>>(N, ctx->d_brow_ptr, (int32_t*)d_row_ptr); KERNEL_CHECK(ctx); }
        if (d_col_idx) { emit_colidx_kernel<int32_t><<<nbc, 256, 0, st>>>(N, ctx->d_brow_ptr, ctx->d_bcol, (int32_t*)d_col_idx); KERNEL_CHECK(ctx); }
    } else {
        if (d_row_ptr) { emit_rowptr_kernel<int64_t><<<nbr, 256, 0, st>>>(N, ctx->d_brow_ptr, (int64_t*)d_row_ptr); KERNEL_CHECK(ctx); }
        if (d_col_idx) { emit_colidx_kernel<int64_t><<<nbc, 256, 0, st>>>(N, ctx->d_brow_ptr, ctx->d_bcol, (int64_t*)d_col_idx); KERNEL_CHECK(ctx); }
    }
    return RPIM_OK;
}
