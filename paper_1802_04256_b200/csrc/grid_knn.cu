// Step a1 (R1): exact k-nearest-neighbour support search on a uniform cell grid.
// Integer / exact-order work: the result is unique (keys (d2, node id) are distinct), so the
// cell size, scan order and thread mapping below are free implementation choices.
#include <cfloat>
#include <cmath>

#include "common.cuh"

// ------------------------------------------------------------------ exclusive scan int32 -> int64
namespace {
constexpr int SCAN_THREADS = 1024;
constexpr int SCAN_ITEMS = 4;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

__global__ void scan_tile_kernel(const int* __restrict__ in, int64_t* __restrict__ out, int64_t n,
                                 int64_t* __restrict__ tile_sum) {
    __shared__ int64_t warp_tot[32];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    int64_t v[SCAN_ITEMS];
    int64_t s = 0;
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i) {
        int64_t x = (base + i < n) ? (int64_t)in[base + i] : 0;
        v[i] = s;
        s += x;
    }
    // warp inclusive scan of s
    int64_t inc = s;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int64_t t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) warp_tot[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int64_t w = warp_tot[lane];
        int64_t winc = w;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int64_t t = __shfl_up_sync(0xffffffffu, winc, d);
            if (lane >= d) winc += t;
        }
        warp_tot[lane] = winc - w;   // exclusive
        if (lane == 31) tile_sum[blockIdx.x] = winc;
    }
    __syncthreads();
    const int64_t off = warp_tot[wid] + (inc - s);
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i)
        if (base + i < n) out[base + i] = off + v[i];
}

__global__ void scan_sums_kernel(int64_t* tile_sum, int64_t ntiles) {
    // single block, sequential over chunks of blockDim.x with a running carry
    __shared__ int64_t buf[1024];
    __shared__ int64_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int64_t c0 = 0; c0 < ntiles; c0 += blockDim.x) {
        int64_t i = c0 + threadIdx.x;
        int64_t x = (i < ntiles) ? tile_sum[i] : 0;
        buf[threadIdx.x] = x;
        __syncthreads();
        for (int d = 1; d < (int)blockDim.x; d <<= 1) {
            int64_t t = (threadIdx.x >= (unsigned)d) ? buf[threadIdx.x - d] : 0;
            __syncthreads();
            buf[threadIdx.x] += t;
            __syncthreads();
        }
        if (i < ntiles) tile_sum[i] = carry + buf[threadIdx.x] - x;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry += buf[threadIdx.x];
        __syncthreads();
    }
    if (threadIdx.x == 0) tile_sum[ntiles] = carry;   // grand total
}

__global__ void scan_add_kernel(int64_t* __restrict__ out, int64_t n, const int64_t* __restrict__ tile_sum,
                                int64_t ntiles) {
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    const int64_t add = tile_sum[blockIdx.x];
#pragma unroll
    for (int i = 0; i < SCAN_ITEMS; ++i)
        if (base + i < n) out[base + i] += add;
    if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = tile_sum[ntiles];
}
}  // namespace

int rpim_scan_i32_to_i64(rpim_ctx* ctx, const int* d_in, int64_t* d_out, int64_t n) {
    const int64_t ntiles = (n + SCAN_TILE - 1) / SCAN_TILE;
    if (ctx->scan_tmp_elems < ntiles + 1) {
        int64_t* p = (int64_t*)ctx->d_scan_tmp;
        int rc = ws_alloc(ctx, &p, ntiles + 1);
        ctx->d_scan_tmp = p;
        if (rc) return rc;
        ctx->scan_tmp_elems = ntiles + 1;
    }
    int64_t* tmp = (int64_t*)ctx->d_scan_tmp;
    if (n == 0) {
        CUDA_TRY(ctx, cudaMemsetAsync(d_out, 0, sizeof(int64_t), ctx->stream));
        return RPIM_OK;
    }
    scan_tile_kernel<<<(unsigned)ntiles, SCAN_THREADS, 0, ctx->stream>>>(d_in, d_out, n, tmp);
    KERNEL_CHECK(ctx);
    scan_sums_kernel<<<1, 1024, 0, ctx->stream>>>(tmp, ntiles);
    KERNEL_CHECK(ctx);
    scan_add_kernel<<<(unsigned)ntiles, SCAN_THREADS, 0, ctx->stream>>>(d_out, n, tmp, ntiles);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}

// ------------------------------------------------------------------ bounding box + cell binning
namespace {
__global__ void bbox_partial_kernel(const double* __restrict__ nodes, int64_t N, double* __restrict__ part) {
    double lo[3] = {DBL_MAX, DBL_MAX, DBL_MAX}, hi[3] = {-DBL_MAX, -DBL_MAX, -DBL_MAX};
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double v = nodes[3 * i + c];
            lo[c] = fmin(lo[c], v);
            hi[c] = fmax(hi[c], v);
        }
    __shared__ double s[6][256];
#pragma unroll
    for (int c = 0; c < 3; ++c) { s[c][threadIdx.x] = lo[c]; s[3 + c][threadIdx.x] = hi[c]; }
    __syncthreads();
    for (int d = blockDim.x >> 1; d > 0; d >>= 1) {
        if ((int)threadIdx.x < d)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                s[c][threadIdx.x] = fmin(s[c][threadIdx.x], s[c][threadIdx.x + d]);
                s[3 + c][threadIdx.x] = fmax(s[3 + c][threadIdx.x], s[3 + c][threadIdx.x + d]);
            }
        __syncthreads();
    }
    if (threadIdx.x < 6) part[blockIdx.x * 6 + threadIdx.x] = s[threadIdx.x][0];
}

__global__ void bbox_final_kernel(double* part, int nparts) {
    // one warp; result in part[0..5]
    const int lane = threadIdx.x;
    double lo[3] = {DBL_MAX, DBL_MAX, DBL_MAX}, hi[3] = {-DBL_MAX, -DBL_MAX, -DBL_MAX};
    for (int b = lane; b < nparts; b += 32)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            lo[c] = fmin(lo[c], part[b * 6 + c]);
            hi[c] = fmax(hi[c], part[b * 6 + 3 + c]);
        }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            lo[c] = fmin(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], d));
            hi[c] = fmax(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], d));
        }
    __syncwarp();
    if (lane == 0)
#pragma unroll
        for (int c = 0; c < 3; ++c) { part[c] = lo[c]; part[3 + c] = hi[c]; }
}

__device__ __forceinline__ void cell_coords(const GridParams& g, double x, double y, double z, int* c) {
    double p[3] = {x, y, z};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        int v = (int)floor((p[a] - g.lo[a]) * g.inv_cell);
        c[a] = min(max(v, 0), g.nc[a] - 1);
    }
}

__global__ void cell_count_kernel(GridParams g, const double* __restrict__ nodes, int64_t N,
                                  int* __restrict__ cell_of, int* __restrict__ count) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int c[3];
    cell_coords(g, nodes[3 * i], nodes[3 * i + 1], nodes[3 * i + 2], c);
    int id = c[0] + g.nc[0] * (c[1] + g.nc[1] * c[2]);
    cell_of[i] = id;
    atomicAdd(&count[id], 1);
}

__global__ void cell_fill_kernel(const double* __restrict__ nodes, int64_t N, const int* __restrict__ cell_of,
                                 const int64_t* __restrict__ cell_start, int* __restrict__ cursor,
                                 int* __restrict__ node_order) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    int id = cell_of[i];
    int p = atomicAdd(&cursor[id], 1);
    node_order[cell_start[id] + p] = (int)i;
}

// make the order inside every cell deterministic (ascending node id) and gather coordinates
__global__ void cell_sort_gather_kernel(const double* __restrict__ nodes, int64_t ncell,
                                        const int64_t* __restrict__ cell_start, int* __restrict__ node_order,
                                        double* __restrict__ sx, double* __restrict__ sy, double* __restrict__ sz) {
    int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    int64_t a = cell_start[c], b = cell_start[c + 1];
    for (int64_t i = a + 1; i < b; ++i) {   // insertion sort, cells hold a handful of nodes
        int v = node_order[i];
        int64_t j = i - 1;
        while (j >= a && node_order[j] > v) { node_order[j + 1] = node_order[j]; --j; }
        node_order[j + 1] = v;
    }
    for (int64_t i = a; i < b; ++i) {
        int64_t id = node_order[i];
        sx[i] = nodes[3 * id];
        sy[i] = nodes[3 * id + 1];
        sz[i] = nodes[3 * id + 2];
    }
}

// moving nodes (rpim_update_nodes): how many nodes left their cell of the existing grid (or the grid's box)
__global__ void cell_moved_kernel(GridParams g, const double* __restrict__ nodes, int64_t N,
                                  const int* __restrict__ cell_of, unsigned long long* __restrict__ moved) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool m = false;
    if (i < N) {
        const double p[3] = {nodes[3 * i], nodes[3 * i + 1], nodes[3 * i + 2]};
        int c[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int v = (int)floor((p[a] - g.lo[a]) * g.inv_cell);
            m = m || v < 0 || v >= g.nc[a] || !(p[a] == p[a]);
            c[a] = min(max(v, 0), g.nc[a] - 1);
        }
        m = m || (c[0] + g.nc[0] * (c[1] + g.nc[1] * c[2])) != cell_of[i];
    }
    const unsigned b = __ballot_sync(0xffffffffu, m);
    if ((threadIdx.x & 31) == 0 && b) atomicAdd(moved, (unsigned long long)__popc(b));
}

// same cells, new coordinates: refresh the cell-ordered SoA copy
__global__ void cell_regather_kernel(const double* __restrict__ nodes, int64_t N, const int* __restrict__ node_order,
                                     double* __restrict__ sx, double* __restrict__ sy, double* __restrict__ sz) {
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int64_t id = node_order[i];
    sx[i] = nodes[3 * id];
    sy[i] = nodes[3 * id + 1];
    sz[i] = nodes[3 * id + 2];
}

// ------------------------------------------------------------------ the search: one warp per query point
// CAP = candidates held on chip per query.  The first launch uses the smallest capacity that
// fits the expected candidate count (more resident warps); queries that need more are appended
// to an overflow list and redone by the KNN_CAP_MAX instantiation; the LAST tier has no limit (streaming
// selection: the buffer is sorted and cut back to the best k whenever it fills up).
constexpr int KNN_CAP_MAX = 2048;

template <int CAP, int WARPS, bool LAST>
__global__ void __launch_bounds__(WARPS * 32)
knn_kernel(GridParams g, const double* __restrict__ sx, const double* __restrict__ sy,
           const double* __restrict__ sz, const int* __restrict__ node_order,
           const int64_t* __restrict__ cell_start, const double* __restrict__ pts, int64_t M, int k, int R0,
           const int32_t* __restrict__ qlist, const long long* __restrict__ nq_ptr,
           int32_t* __restrict__ ovf_list, int ovf_flag, int32_t* __restrict__ support, long long* __restrict__ flags) {
    extern __shared__ unsigned char smem_raw[];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned long long* key = (unsigned long long*)smem_raw + (size_t)wid * CAP;
    int* val = (int*)((unsigned long long*)smem_raw + (size_t)WARPS * CAP) + (size_t)wid * CAP;
    const int64_t nq = qlist ? (int64_t)*nq_ptr : M;

    for (int64_t qi = (int64_t)blockIdx.x * WARPS + wid; qi < nq; qi += (int64_t)gridDim.x * WARPS) {
        const int64_t q = qlist ? qlist[qi] : qi;
        const double xq = pts[3 * q], yq = pts[3 * q + 1], zq = pts[3 * q + 2];
        int cq[3];
        cell_coords(g, xq, yq, zq, cq);
        int R = R0;
        int npad = 0;
        bool fail = false, overflow = false;
        while (true) {
            int a[3], b[3];
            bool whole = true;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                a[c] = max(cq[c] - R, 0);
                b[c] = min(cq[c] + R, g.nc[c] - 1);
                if (a[c] > 0 || b[c] < g.nc[c] - 1) whole = false;
            }
            const int ny = b[1] - a[1] + 1, nz = b[2] - a[2] + 1;
            const int nrows = ny * nz;
            // count candidates (cells of one x-row are contiguous in cell order)
            int cnt = 0;
            for (int r = lane; r < nrows; r += 32) {
                int y = a[1] + r % ny, z = a[2] + r / ny;
                int64_t c0 = a[0] + (int64_t)g.nc[0] * (y + (int64_t)g.nc[1] * z);
                int64_t c1 = c0 + (b[0] - a[0]);
                cnt += (int)(cell_start[c1 + 1] - cell_start[c0]);
            }
            cnt = __reduce_add_sync(0xffffffffu, cnt);
            if (cnt < k) {
                if (whole) { fail = true; break; }
                ++R;
                continue;
            }
            if (cnt > CAP && !LAST) { overflow = true; break; }
            // gather candidates with their squared distances (R1: no fma, fixed association).  The last tier has no
            // capacity limit: when the buffer is full it is sorted and only the best k are kept (streaming selection
            // under the same total order (d^2, node id): the result does not depend on where the buffer filled up)
            int base = 0;
            for (int r = 0; r < nrows; ++r) {
                int y = a[1] + r % ny, z = a[2] + r / ny;
                int64_t c0 = a[0] + (int64_t)g.nc[0] * (y + (int64_t)g.nc[1] * z);
                int64_t s0 = cell_start[c0], s1 = cell_start[c0 + (b[0] - a[0]) + 1];
                while (s0 < s1) {
                    const int take = (int)min((int64_t)(CAP - base), s1 - s0);
                    for (int64_t p = s0 + lane; p < s0 + take; p += 32) {
                        double dx = __dsub_rn(sx[p], xq), dy = __dsub_rn(sy[p], yq), dz = __dsub_rn(sz[p], zq);
                        double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
                        key[base + (int)(p - s0)] = (unsigned long long)__double_as_longlong(d2);
                        val[base + (int)(p - s0)] = node_order[p];
                    }
                    base += take;
                    s0 += take;
                    if (base == CAP && (s0 < s1 || r + 1 < nrows)) {   // (only the last tier gets here: cnt > CAP)
                        __syncwarp();
                        warp_bitonic_u64_i32(key, val, CAP);
                        base = k;
                    }
                }
            }
            npad = next_pow2(base);
            for (int i = base + lane; i < npad; i += 32) { key[i] = 0xFFFFFFFFFFFFFFFFull; val[i] = 0x7FFFFFFF; }
            __syncwarp();
            warp_bitonic_u64_i32(key, val, npad);
            if (whole) break;
            // distance from the query to the part of space not covered by the scanned cells
            double bound = DBL_MAX;
            const double xyz[3] = {xq, yq, zq};
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                if (a[c] > 0) bound = fmin(bound, xyz[c] - (g.lo[c] + a[c] * g.cell));
                if (b[c] < g.nc[c] - 1) bound = fmin(bound, (g.lo[c] + (b[c] + 1) * g.cell) - xyz[c]);
            }
            bound -= 1e-9 * g.cell;   // margin for rounding in the cell assignment
            double dk = __longlong_as_double((long long)key[k - 1]);
            if (bound > 0.0 && dk < bound * bound) break;
            ++R;
        }
        if (overflow && !LAST) {
            if (lane == 0) {
                const unsigned long long slot = atomicAdd((unsigned long long*)&flags[ovf_flag], 1ull);
                ovf_list[slot] = (int32_t)q;
            }
            __syncwarp();
            continue;
        }
        if (fail || overflow) {
            if (lane == 0) atomicAdd((unsigned long long*)&flags[FLAG_KNN_CAP], 1ull);
            for (int j = lane; j < k; j += 32) support[q * k + j] = 0;
            __syncwarp();
            continue;
        }
        // the k winners, ascending by node id
        const int kp = next_pow2(k);
        for (int j = k + lane; j < kp; j += 32) val[j] = 0x7FFFFFFF;
        __syncwarp();
        warp_bitonic_i32(val, kp);
        for (int j = lane; j < k; j += 32) support[q * k + j] = val[j];
        __syncwarp();
    }
}

// ------------------------------------------------------------------ the search, fast form: candidates in registers
// One warp per query, at most 32 * EPL candidates (EPL per lane) from at most 32 x-rows of cells.
// Instead of sorting the candidates the warp SELECTS the k smallest under the order (d^2, node id):
// bisection on the bit pattern of d^2 (monotone for d^2 >= 0) with a warp-wide count per step,
// stopping as soon as exactly k candidates lie at or below the trial value; exact ties at the k-th
// distance (regular grids, R1) are resolved by a second bisection on the node id.  Only the
// k winners are sorted (ascending node id).  Queries that need more cells or candidates go to the
// overflow list and are redone by knn_kernel<KNN_CAP_MAX>.  Same result, bit for bit.
template <int EPL, int WARPS>
__global__ void __launch_bounds__(WARPS * 32)
knn_select_kernel(GridParams g, const double* __restrict__ sx, const double* __restrict__ sy,
                  const double* __restrict__ sz, const int* __restrict__ node_order,
                  const int64_t* __restrict__ cell_start, const double* __restrict__ pts, int64_t M, int k, int R0,
                  int32_t* __restrict__ ovf_list, int32_t* __restrict__ support, long long* __restrict__ flags) {
    constexpr unsigned FULLW = 0xffffffffu;
    constexpr unsigned long long KINF = 0xFFFFFFFFFFFFFFFFull;
    __shared__ int win_s[WARPS][128];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int* win = win_s[wid];
    const unsigned lt = (1u << lane) - 1u;

    for (int64_t q = (int64_t)blockIdx.x * WARPS + wid; q < M; q += (int64_t)gridDim.x * WARPS) {
        const double xq = pts[3 * q], yq = pts[3 * q + 1], zq = pts[3 * q + 2];
        int cq[3];
        cell_coords(g, xq, yq, zq, cq);
        int R = R0;
        bool fail = false, overflow = false;
        unsigned long long key[EPL];
        int id[EPL];
        unsigned sel = 0;   // bit e: candidate e of this lane is one of the k winners
        while (true) {
            int a[3], b[3];
            bool whole = true;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                a[c] = max(cq[c] - R, 0);
                b[c] = min(cq[c] + R, g.nc[c] - 1);
                if (a[c] > 0 || b[c] < g.nc[c] - 1) whole = false;
            }
            const int ny = b[1] - a[1] + 1, nz = b[2] - a[2] + 1;
            const int nrows = ny * nz;
            if (nrows > 32) { overflow = true; break; }
            // lane r: x-row r of cells (contiguous in cell order) -> first sorted node and length
            int s0 = 0, len = 0;
            if (lane < nrows) {
                const int y = a[1] + lane % ny, z = a[2] + lane / ny;
                const int64_t c0 = a[0] + (int64_t)g.nc[0] * (y + (int64_t)g.nc[1] * z);
                const int64_t st = cell_start[c0];
                s0 = (int)st;
                len = (int)(cell_start[c0 + (b[0] - a[0]) + 1] - st);
            }
            int incl = len;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int up = __shfl_up_sync(FULLW, incl, d);
                if (lane >= d) incl += up;
            }
            const int cnt = __shfl_sync(FULLW, incl, 31);
            if (cnt < k) {
                if (whole) { fail = true; break; }
                ++R;
                continue;
            }
            if (cnt > 32 * EPL) { overflow = true; break; }
            const int off = incl - len;
            // non-empty rows compacted to lanes 0..: lane c holds (first node - offset) of the c-th non-empty row
            const unsigned nonempty = __ballot_sync(FULLW, len > 0);
            const int src = __fns(nonempty, 0, lane + 1);
            const int bs = __shfl_sync(FULLW, s0 - off, src & 31);
            // candidate c = 32 e + lane: row = number of row starts at or before c, minus one
            int pre = 0;
#pragma unroll
            for (int e = 0; e < EPL; ++e) {
                const unsigned word = __reduce_or_sync(FULLW, (len > 0 && (off >> 5) == e) ? (1u << (off & 31)) : 0u);
                const int c = 32 * e + lane;
                const int crow = pre + __popc(word & (lt | (1u << lane))) - 1;
                const int p = __shfl_sync(FULLW, bs, crow & 31) + c;
                pre += __popc(word);
                if (c < cnt) {
                    // R1: no fma, fixed association
                    const double dx = __dsub_rn(sx[p], xq), dy = __dsub_rn(sy[p], yq), dz = __dsub_rn(sz[p], zq);
                    const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
                    key[e] = (unsigned long long)__double_as_longlong(d2);
                    id[e] = node_order[p];
                } else {
                    key[e] = KINF;
                    id[e] = 0x7FFFFFFF;
                }
            }
            // ---- select: smallest T with count(key <= T) >= k
            unsigned long long kmax = 0;
#pragma unroll
            for (int e = 0; e < EPL; ++e)
                if (key[e] != KINF && key[e] > kmax) kmax = key[e];
            {
                unsigned hi32 = __reduce_max_sync(FULLW, (unsigned)(kmax >> 32));
                unsigned lo32 = __reduce_max_sync(FULLW, ((unsigned)(kmax >> 32) == hi32) ? (unsigned)kmax : 0u);
                kmax = ((unsigned long long)hi32 << 32) | lo32;
            }
            // ... and the smallest one: the bracket [kmin, kmax] spans a few binades instead of all of them
            unsigned long long kmin = KINF;
#pragma unroll
            for (int e = 0; e < EPL; ++e)
                if (key[e] < kmin) kmin = key[e];
            {
                unsigned hi32 = __reduce_min_sync(FULLW, (unsigned)(kmin >> 32));
                unsigned lo32 = __reduce_min_sync(FULLW, ((unsigned)(kmin >> 32) == hi32) ? (unsigned)kmin : 0xffffffffu);
                kmin = ((unsigned long long)hi32 << 32) | lo32;
            }
            unsigned long long lo = kmin, hi = kmax, T = 0;
            int c_le = 0;
            bool found = false;
            for (int it = 0; it < 24 && !found; ++it) {
                const unsigned long long mid = lo + ((hi - lo) >> 1);
                int c = 0;
#pragma unroll
                for (int e = 0; e < EPL; ++e) c += (key[e] <= mid) ? 1 : 0;
                c = __reduce_add_sync(FULLW, c);
                if (c == k) { T = mid; c_le = c; found = true; }
                else if (c > k) hi = mid;
                else lo = mid + 1;
                if (!found && lo == hi) {
                    T = lo; found = true;
                    int cc = 0;
#pragma unroll
                    for (int e = 0; e < EPL; ++e) cc += (key[e] <= T) ? 1 : 0;
                    c_le = __reduce_add_sync(FULLW, cc);
                }
            }
            while (!found) {   // step through the distinct values left in [lo, hi]
                unsigned long long v = KINF;
#pragma unroll
                for (int e = 0; e < EPL; ++e)
                    if (key[e] >= lo && key[e] < v) v = key[e];
                const unsigned vh = __reduce_min_sync(FULLW, (unsigned)(v >> 32));
                const unsigned vl = __reduce_min_sync(FULLW, ((unsigned)(v >> 32) == vh) ? (unsigned)v : 0xffffffffu);
                v = ((unsigned long long)vh << 32) | vl;
                int c = 0;
#pragma unroll
                for (int e = 0; e < EPL; ++e) c += (key[e] <= v) ? 1 : 0;
                c = __reduce_add_sync(FULLW, c);
                if (c >= k) { T = v; c_le = c; found = true; }
                else lo = v + 1;
            }
            sel = 0;
            if (c_le == k) {
#pragma unroll
                for (int e = 0; e < EPL; ++e) sel |= (key[e] <= T) ? (1u << e) : 0u;
            } else {
                // exact ties at the k-th distance: all of key < T, and of key == T the `need` smallest ids
                int c = 0;
#pragma unroll
                for (int e = 0; e < EPL; ++e) c += (key[e] < T) ? 1 : 0;
                const int need = k - __reduce_add_sync(FULLW, c);
                unsigned ilo = 0, ihi = 0x7FFFFFFEu, IT = 0;
                while (true) {   // node ids are distinct: some trial value separates exactly `need` of them
                    const unsigned mid = ilo + ((ihi - ilo) >> 1);
                    int ci = 0;
#pragma unroll
                    for (int e = 0; e < EPL; ++e) ci += (key[e] == T && (unsigned)id[e] <= mid) ? 1 : 0;
                    ci = __reduce_add_sync(FULLW, ci);
                    if (ci == need) { IT = mid; break; }
                    if (ci > need) ihi = mid; else ilo = mid + 1;
                }
#pragma unroll
                for (int e = 0; e < EPL; ++e)
                    sel |= (key[e] < T || (key[e] == T && (unsigned)id[e] <= IT)) ? (1u << e) : 0u;
            }
            if (whole) break;
            // distance from the query to the part of space not covered by the scanned cells
            double bound = DBL_MAX;
            const double xyz[3] = {xq, yq, zq};
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                if (a[c] > 0) bound = fmin(bound, xyz[c] - (g.lo[c] + a[c] * g.cell));
                if (b[c] < g.nc[c] - 1) bound = fmin(bound, (g.lo[c] + (b[c] + 1) * g.cell) - xyz[c]);
            }
            bound -= 1e-9 * g.cell;   // margin for rounding in the cell assignment
            // the k-th distance = largest selected key
            unsigned long long km = 0;
#pragma unroll
            for (int e = 0; e < EPL; ++e)
                if (((sel >> e) & 1u) && key[e] > km) km = key[e];
            const unsigned kh = __reduce_max_sync(FULLW, (unsigned)(km >> 32));
            const unsigned kl = __reduce_max_sync(FULLW, ((unsigned)(km >> 32) == kh) ? (unsigned)km : 0u);
            const double dk = __longlong_as_double((long long)(((unsigned long long)kh << 32) | kl));
            if (bound > 0.0 && dk < bound * bound) break;
            ++R;
        }
        if (overflow) {
            if (lane == 0) {
                const unsigned long long slot = atomicAdd((unsigned long long*)&flags[FLAG_OVF_Q], 1ull);
                ovf_list[slot] = (int32_t)q;
            }
            __syncwarp();
            continue;
        }
        if (fail) {
            if (lane == 0) atomicAdd((unsigned long long*)&flags[FLAG_KNN_CAP], 1ull);
            for (int j = lane; j < k; j += 32) support[q * k + j] = 0;
            __syncwarp();
            continue;
        }
        // the k winners -> shared memory (any order), then ascending by node id
        int base = 0;
#pragma unroll
        for (int e = 0; e < EPL; ++e) {
            const bool s = (sel >> e) & 1u;
            const unsigned m = __ballot_sync(FULLW, s);
            if (s) win[base + __popc(m & lt)] = id[e];
            base += __popc(m);
        }
        const int kp = next_pow2(k);
        for (int j = k + lane; j < kp; j += 32) win[j] = 0x7FFFFFFF;
        __syncwarp();
        warp_bitonic_i32(win, kp);
        for (int j = lane; j < k; j += 32) support[q * k + j] = win[j];
        __syncwarp();
    }
}

template <int EPL, int WARPS>
int launch_knn_select(rpim_ctx* ctx, const double* d_pts, int64_t M, int k, int32_t* ovf_list, int32_t* d_support,
                      int64_t blocks_cap) {
    const int64_t N = ctx->N;
    const int64_t blocks = std::min<int64_t>((M + WARPS - 1) / WARPS, blocks_cap);
    knn_select_kernel<EPL, WARPS><<<(unsigned)blocks, WARPS * 32, 0, ctx->stream>>>(
        ctx->grid, ctx->d_sorted_xyz, ctx->d_sorted_xyz + N, ctx->d_sorted_xyz + 2 * N, ctx->d_node_order,
        ctx->d_cell_start, d_pts, M, k, 2, ovf_list, d_support, ctx->d_flags);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}

// qflag: the counter of the query list (when qlist is given); oflag: the counter of the overflow list this launch appends to
template <int CAP, int WARPS, bool LAST>
int launch_knn(rpim_ctx* ctx, const double* d_pts, int64_t M, int k, int R0, const int32_t* qlist, int qflag, int32_t* ovf_list,
               int oflag, int32_t* d_support, int64_t blocks_cap) {
    const int64_t N = ctx->N;
    auto kern = knn_kernel<CAP, WARPS, LAST>;
    const size_t smem = (size_t)WARPS * CAP * (sizeof(unsigned long long) + sizeof(int));
    CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int64_t blocks = qlist ? blocks_cap : std::min<int64_t>((M + WARPS - 1) / WARPS, blocks_cap);
    kern<<<(unsigned)blocks, WARPS * 32, smem, ctx->stream>>>(
        ctx->grid, ctx->d_sorted_xyz, ctx->d_sorted_xyz + N, ctx->d_sorted_xyz + 2 * N, ctx->d_node_order,
        ctx->d_cell_start, d_pts, M, k, R0, qlist, ctx->d_flags + qflag, ovf_list, oflag, d_support, ctx->d_flags);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}
}  // namespace

// Incremental cell-grid update for moved nodes (ctx->d_nodes already points at the new coordinates): when
// no node left its cell only the cell-ordered coordinates are refreshed, otherwise *out_rebuild = true and
// the caller rebuilds the grid (rpim_stage_grid_knn with build_grid).  Synchronises.
int rpim_stage_grid_refresh(rpim_ctx* ctx, bool* out_rebuild, int64_t* out_moved) {
    cudaStream_t st = ctx->stream;
    const int64_t N = ctx->N;
    unsigned long long* d_moved = (unsigned long long*)ctx->d_scratch;
    CUDA_TRY(ctx, cudaMemsetAsync(d_moved, 0, sizeof(unsigned long long), st));
    const unsigned nb = (unsigned)((N + 255) / 256);
    cell_moved_kernel<<<nb, 256, 0, st>>>(ctx->grid, ctx->d_nodes, N, ctx->d_cell_of, d_moved);
    KERNEL_CHECK(ctx);
    unsigned long long moved = 0;
    CUDA_TRY(ctx, cudaMemcpyAsync(&moved, d_moved, sizeof(moved), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    *out_moved = (int64_t)moved;
    *out_rebuild = moved != 0;
    if (moved == 0) {
        cell_regather_kernel<<<nb, 256, 0, st>>>(ctx->d_nodes, N, ctx->d_node_order, ctx->d_sorted_xyz,
                                                 ctx->d_sorted_xyz + N, ctx->d_sorted_xyz + 2 * N);
        KERNEL_CHECK(ctx);
    }
    return RPIM_OK;
}

int rpim_stage_grid_knn(rpim_ctx* ctx, const double* d_pts, int64_t M, int k, int32_t* d_support, bool build_grid) {
    cudaStream_t st = ctx->stream;
    const int64_t N = ctx->N;
    if (build_grid) {
        int rc;
        if ((rc = ws_alloc(ctx, &ctx->d_scratch, 8192))) return rc;
        bbox_partial_kernel<<<256, 256, 0, st>>>(ctx->d_nodes, N, ctx->d_scratch);
        KERNEL_CHECK(ctx);
        bbox_final_kernel<<<1, 32, 0, st>>>(ctx->d_scratch, 256);
        KERNEL_CHECK(ctx);
        double bb[6];
        CUDA_TRY(ctx, cudaMemcpyAsync(bb, ctx->d_scratch, sizeof(bb), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(ctx, cudaStreamSynchronize(st));
        for (int c = 0; c < 6; ++c)
            if (!std::isfinite(bb[c])) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "node coordinates are not finite");
        double ext[3], emax = 0.0;
        for (int c = 0; c < 3; ++c) { ext[c] = bb[3 + c] - bb[c]; emax = std::fmax(emax, ext[c]); }
        if (!(emax > 0.0)) emax = 1.0;
        double vol = 1.0;
        for (int c = 0; c < 3; ++c) vol *= std::fmax(ext[c], 1e-9 * emax);
        const double h_avg = std::cbrt(vol / (double)N);
        const double r_k = std::cbrt(3.0 * k / (4.0 * 3.14159265358979323846)) * h_avg;
        GridParams g;
        g.cell = 1.08 * r_k / 2.0;   // two rings of cells cover the expected support radius
        int64_t ncell;
        while (true) {
            ncell = 1;
            for (int c = 0; c < 3; ++c) {
                g.nc[c] = (int)std::fmin(2000.0, std::floor(ext[c] / g.cell) + 1.0);
                ncell *= g.nc[c];
            }
            if (ncell <= 4 * N + 64) break;
            g.cell *= 1.26;
        }
        g.inv_cell = 1.0 / g.cell;
        for (int c = 0; c < 3; ++c) g.lo[c] = bb[c];
        g.ncell = ncell;
        ctx->grid = g;
        if ((rc = ws_alloc(ctx, &ctx->d_cell_of, N))) return rc;
        if ((rc = ws_alloc(ctx, &ctx->d_cell_start, ncell + 1))) return rc;
        if ((rc = ws_alloc(ctx, &ctx->d_cell_cursor, ncell))) return rc;
        if ((rc = ws_alloc(ctx, &ctx->d_node_order, N))) return rc;
        if ((rc = ws_alloc(ctx, &ctx->d_sorted_xyz, 3 * N))) return rc;
        CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_cell_cursor, 0, ncell * sizeof(int), st));
        const unsigned nb = (unsigned)((N + 255) / 256);
        cell_count_kernel<<<nb, 256, 0, st>>>(g, ctx->d_nodes, N, ctx->d_cell_of, ctx->d_cell_cursor);
        KERNEL_CHECK(ctx);
        if ((rc = rpim_scan_i32_to_i64(ctx, ctx->d_cell_cursor, ctx->d_cell_start, ncell))) return rc;
        CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_cell_cursor, 0, ncell * sizeof(int), st));
        cell_fill_kernel<<<nb, 256, 0, st>>>(ctx->d_nodes, N, ctx->d_cell_of, ctx->d_cell_start, ctx->d_cell_cursor,
                                             ctx->d_node_order);
        KERNEL_CHECK(ctx);
        cell_sort_gather_kernel<<<(unsigned)((ncell + 127) / 128), 128, 0, st>>>(
            ctx->d_nodes, ncell, ctx->d_cell_start, ctx->d_node_order, ctx->d_sorted_xyz, ctx->d_sorted_xyz + N,
            ctx->d_sorted_xyz + 2 * N);
        KERNEL_CHECK(ctx);
    }
    if (M == 0) return RPIM_OK;
    // expected candidates in the first (2 R0 + 1)^3 = 125 cells, with a margin for density fluctuations
    const GridParams& g = ctx->grid;
    const double per_cell = (double)N / (double)g.ncell;
    const double expect = 125.0 * per_cell * 1.25;
    const int cap = expect <= 256 ? 256 : expect <= 512 ? 512 : expect <= 1024 ? 1024 : KNN_CAP_MAX;
    // Tiers: the capacity the mean density asks for; its overflow list redone with the largest capacity; what still
    // does not fit (a 5 x 5 x 5 ring of cells holding more than KNN_CAP_MAX nodes: local density ~ 14 x the mean,
    // graded clouds) redone from the query's own cell outwards (R0 = 0) -- the ring only grows until the k-th
    // distance is covered, so the dense spots need far fewer cells.  Same result in every tier, bit for bit.
    int rc = RPIM_OK;
    int32_t *d_ovf = nullptr, *d_ovf2 = nullptr;
    if ((rc = ws_alloc(ctx, &d_ovf, M)) || (rc = ws_alloc(ctx, &d_ovf2, M))) { ws_free(ctx, &d_ovf); return rc; }
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_flags + FLAG_OVF_Q, 0, sizeof(long long), st));
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_flags + FLAG_OVF_Q2, 0, sizeof(long long), st));
    if (cap == KNN_CAP_MAX) {
        rc = launch_knn<KNN_CAP_MAX, 4, false>(ctx, d_pts, M, k, 2, nullptr, FLAG_OVF_Q, d_ovf2, FLAG_OVF_Q2, d_support, 148 * 64);
    } else {
        if (cap == 256) rc = launch_knn_select<8, 8>(ctx, d_pts, M, k, d_ovf, d_support, 148 * 64);
        else if (cap == 512) rc = launch_knn_select<16, 8>(ctx, d_pts, M, k, d_ovf, d_support, 148 * 64);
        else rc = launch_knn<1024, 4, false>(ctx, d_pts, M, k, 2, nullptr, FLAG_OVF_Q, d_ovf, FLAG_OVF_Q, d_support, 148 * 64);
        if (rc == RPIM_OK)
            rc = launch_knn<KNN_CAP_MAX, 4, false>(ctx, d_pts, M, k, 2, d_ovf, FLAG_OVF_Q, d_ovf2, FLAG_OVF_Q2, d_support, 148 * 2);
    }
    if (rc == RPIM_OK) rc = launch_knn<KNN_CAP_MAX, 4, true>(ctx, d_pts, M, k, 0, d_ovf2, FLAG_OVF_Q2, nullptr, FLAG_OVF_Q2, d_support, 148 * 2);
    ws_free(ctx, &d_ovf2);
    ws_free(ctx, &d_ovf);   // parked in the workspace cache (later reuse is ordered by the stream)
    return rc;
}
