// rpim_apply_penalty_static (include/rpim.h): the penalty stage (step a7, R10) for callers
// that must not allocate device memory.
//
// rpim_apply_penalty needs three pieces of scratch memory: the per-CTA partial maxima of the diagonal, one bit per
// node to find ids that are listed twice, and a counter of rejected ids.  It takes them from the context's
// workspace, which reaches cudaMalloc whenever no parked block fits.  Here the same three pieces live in ONE
// file-scope device array of fixed size, part of the library image: nothing is allocated, by this file or by
// anything it calls.  The price is a hard limit on the number of nodes (RPIM_STATIC_PENALTY_MAX_NODES), about
// half a MiB of device memory on every GPU that loads librpim until the process exits, and one array shared by all
// contexts on a device (calls that overlap on the GPU race on it).
//
// The kernels below are this file's own copies of the penalty kernels in accumulate.cu with the scratch pointers
// replaced; the arithmetic (an exact maximum, alpha * max, one add per constrained diagonal and load entry) is the
// same, so the two entry points give bitwise equal K and f.
#include <cstddef>
#include <mutex>

#include "common.cuh"

namespace {

constexpr int64_t kMaxNodes = RPIM_STATIC_PENALTY_MAX_NODES;
constexpr int kParts = 592;                          // CTAs of the diagonal-maximum pass (4 per SM)

// Layout of the scratch array.  `alpha` and `bad` are read back by the host in one copy, so they sit together.
struct PenaltyScratch {
    double alpha;                                    // alpha actually applied (written by ps_alpha_kernel)
    unsigned long long bad;                          // boundary ids rejected by ps_check_kernel
    double part[kParts];                             // per-CTA maxima of the diagonal
    unsigned seen[(kMaxNodes + 31) / 32];            // one bit per node: id already met in the boundary list
};

// The scratch memory itself.  In HOST code the name `g_penalty_scratch` is only a handle of the symbol, not a device
// address: handing it to a kernel would fault (or, where the GPU can reach host memory, quietly use the wrong
// memory).  Host code therefore goes through scratch_for_device() below, which asks the runtime for the address.
static __device__ __align__(256) unsigned char g_penalty_scratch[sizeof(PenaltyScratch)];

// Device address of the array on each device, filled once per device on first use.
constexpr int kMaxDevices = 64;
PenaltyScratch* g_scratch_addr[kMaxDevices] = {};
std::mutex g_scratch_mutex;

// Set-up, once per device, with that device current (the caller has just done cudaSetDevice): every device has
// its own copy of the array at its own address.
cudaError_t scratch_for_device(int device, PenaltyScratch** out) {
    if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_penalty_scratch);
        if (e != cudaSuccess) return e;
        g_scratch_addr[device] = (PenaltyScratch*)p;
    }
    *out = g_scratch_addr[device];
    return cudaSuccess;
}

// Pass 1: the array keeps whatever the previous call left in it, so clear what has to start at zero (the seen
// bits of this problem's nodes and the counter), and take each CTA's maximum of the diagonal entries of K.
__global__ void ps_clear_and_diag_max_kernel(int64_t N, const int64_t* __restrict__ brow_ptr,
                                             const int* __restrict__ bdiag, const double* __restrict__ vals,
                                             PenaltyScratch* __restrict__ s) {
    const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t nthreads = (int64_t)gridDim.x * blockDim.x;
    const int64_t words = (N + 31) / 32;
    for (int64_t wd = tid; wd < words; wd += nthreads) s->seen[wd] = 0u;
    if (tid == 0) s->bad = 0ull;
    double m = 0.0;
    for (int64_t I = tid; I < N; I += nthreads) {
        const int64_t o = brow_ptr[I];
        const int64_t L = brow_ptr[I + 1] - o;
        if (L == 0) continue;
        const int64_t d = bdiag[I];
#pragma unroll
        for (int a = 0; a < 3; ++a) m = fmax(m, vals[9 * o + a * 3 * L + 3 * d + a]);
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, d));
    __shared__ double sm[32];
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x < 32) {
        m = (threadIdx.x < (blockDim.x >> 5)) ? sm[threadIdx.x] : 0.0;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, d));
        if (threadIdx.x == 0) s->part[blockIdx.x] = m;
    }
}

// Pass 2 (one warp): alpha_used = alpha * max_d K_dd, or alpha itself.
__global__ void ps_alpha_kernel(PenaltyScratch* __restrict__ s, int nparts, double alpha, int relative) {
    double m = 0.0;
    for (int b = threadIdx.x; b < nparts; b += 32) m = fmax(m, s->part[b]);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, d));
    if (threadIdx.x == 0) s->alpha = relative ? alpha * m : alpha;
}

// Pass 3: the boundary list is valid when every id is in range, has a matrix row and is listed once.
__global__ void ps_check_kernel(int64_t N, const int64_t* __restrict__ bc_nodes, int64_t m,
                                const int64_t* __restrict__ brow_ptr, PenaltyScratch* __restrict__ s) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    const int64_t I = bc_nodes[i];
    bool bad = I < 0 || I >= N || brow_ptr[I + 1] == brow_ptr[I];
    if (!bad) bad = (atomicOr(&s->seen[I >> 5], 1u << (I & 31)) >> (I & 31)) & 1u;
    if (bad) atomicAdd(&s->bad, 1ull);
}

// Pass 4 (only after the host has seen bad == 0): K_dd += alpha_used, f_d += alpha_used * u_bar_d.
__global__ void ps_apply_kernel(const int64_t* __restrict__ bc_nodes, const uint8_t* __restrict__ bc_mask,
                                const double* __restrict__ ubar, int64_t m, const PenaltyScratch* __restrict__ s,
                                const int64_t* __restrict__ brow_ptr, const int* __restrict__ bdiag,
                                double* __restrict__ vals, double* __restrict__ f) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    const int64_t I = bc_nodes[i];
    const double a = s->alpha;
    const int mask = bc_mask ? bc_mask[i] : 7;
    const int64_t o = brow_ptr[I], L = brow_ptr[I + 1] - o, d = bdiag[I];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (!((mask >> c) & 1)) continue;
        vals[9 * o + c * 3 * L + 3 * d + c] += a;
        f[3 * I + c] += a * ubar[3 * i + c];
    }
}

}  // namespace

extern "C" {

int64_t rpim_apply_penalty_static_max_nodes(void) { return kMaxNodes; }

int rpim_apply_penalty_static(rpim_ctx* ctx, const int64_t* d_bc_nodes, const uint8_t* d_bc_mask,
                              const double* d_u_bar, int64_t m, double alpha, int alpha_is_relative, double* d_vals,
                              double* d_f, double* out_alpha_used) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!ctx->have_pattern) RPIM_FAIL(ctx, RPIM_ERR_STATE, "rpim_apply_penalty_static before rpim_build_pattern");
    if (m < 0 || !d_vals || !d_f || (m > 0 && (!d_bc_nodes || !d_u_bar))) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "null pointer");
    if (ctx->N > kMaxNodes)
        RPIM_FAIL(ctx, RPIM_ERR_CAPACITY,
                  "rpim_apply_penalty_static: %lld nodes exceed the built-in scratch array's limit of %lld "
                  "(RPIM_STATIC_PENALTY_MAX_NODES); use rpim_apply_penalty, which allocates its scratch memory",
                  (long long)ctx->N, (long long)kMaxNodes);
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    PenaltyScratch* s = nullptr;
    {
        const cudaError_t e = scratch_for_device(ctx->device, &s);
        if (e != cudaSuccess)
            RPIM_FAIL(ctx, RPIM_ERR_CUDA, "cudaGetSymbolAddress of the penalty scratch array failed on device %d: %s",
                      ctx->device, cudaGetErrorString(e));
    }
    cudaStream_t st = ctx->stream;
    ps_clear_and_diag_max_kernel<<<kParts, 256, 0, st>>>(ctx->N, ctx->d_brow_ptr, ctx->d_bdiag, d_vals, s);
    KERNEL_CHECK(ctx);
    ps_alpha_kernel<<<1, 32, 0, st>>>(s, kParts, alpha, alpha_is_relative);
    KERNEL_CHECK(ctx);
    if (m > 0) {
        ps_check_kernel<<<(unsigned)((m + 127) / 128), 128, 0, st>>>(ctx->N, d_bc_nodes, m, ctx->d_brow_ptr, s);
        KERNEL_CHECK(ctx);
    }
    struct { double alpha; unsigned long long bad; } head = {0.0, 0ull};   // first 16 bytes of PenaltyScratch
    static_assert(offsetof(PenaltyScratch, bad) == 8 && offsetof(PenaltyScratch, part) == 16, "head layout");
    CUDA_TRY(ctx, cudaMemcpyAsync(&head, s, sizeof(head), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    if (out_alpha_used) *out_alpha_used = head.alpha;
    if (head.bad)
        RPIM_FAIL(ctx, RPIM_ERR_BC_NODE_INVALID,
                  "%llu boundary node ids are out of range, listed more than once or have no matrix row; nothing applied",
                  head.bad);
    if (m > 0) {
        ps_apply_kernel<<<(unsigned)((m + 127) / 128), 128, 0, st>>>(d_bc_nodes, d_bc_mask, d_u_bar, m, s,
                                                                     ctx->d_brow_ptr, ctx->d_bdiag, d_vals, d_f);
        KERNEL_CHECK(ctx);
    }
    return RPIM_OK;
}

}  // extern "C"
