// Stage 3 of the paper ("solve the system ... then the stresses"), SURVEY 8(f)
// NEXT-1: block-Jacobi-preconditioned (3x3 nodal blocks) conjugate gradients on the assembled, penalised K (symmetric
// positive definite, R10/A2) and stress recovery sigma = D B u at the quadrature points.
//
// K is used in the layout rpim_assemble writes (block row I: three scalar rows of 3 L entries at
// 9 * brow_ptr[I]) together with the context's block columns, so a product reads 8 bytes of values
// and 4/9 byte of index per stored entry -- half of what a scalar int64 CSR product would move.
// Every reduction (dot products, row sums) has a fixed order: the iterates are bitwise reproducible.
#include <algorithm>
#include <cmath>
#include <string>

#include "common.cuh"

namespace {

constexpr int SV_THREADS = 256;
constexpr int SV_PARTS = 1184;   // blocks of the vector kernels = partial sums per dot product (148 SM x 8)

// scalars of the iteration (device resident, no host round trip per step)
enum { S_RZ = 0, S_PAP = 1, S_ALPHA = 2, S_BETA = 3, S_RR = 4, S_BREAK = 5, S_NUM = 8 };

__device__ __forceinline__ double block_sum(double v, double* sh) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sh[w] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += sh[i];
    return t;   // valid in thread 0
}

// y = K x, one warp per block row; optionally partial sums of x . y per block of rows
__global__ void __launch_bounds__(SV_THREADS)
bspmv_kernel(int64_t N, const int64_t* __restrict__ brow_ptr, const int32_t* __restrict__ bcol,
             const double* __restrict__ vals, const double* __restrict__ x, double* __restrict__ y,
             double* __restrict__ part_xy) {
    __shared__ double sh[SV_THREADS / 32];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double dot = 0.0;   // lane 0 of each warp accumulates x . y of its rows
    for (int64_t I = (int64_t)blockIdx.x * (SV_THREADS / 32) + wid; I < N; I += (int64_t)gridDim.x * (SV_THREADS / 32)) {
        const int64_t o = brow_ptr[I];
        const int L = (int)(brow_ptr[I + 1] - o);
        const double* v0 = vals + 9 * o;
        double a0 = 0.0, a1 = 0.0, a2 = 0.0;
        for (int s = lane; s < L; s += 32) {
            const int64_t J = bcol[o + s];
            const double x0 = x[3 * J], x1 = x[3 * J + 1], x2 = x[3 * J + 2];
            const double* r0 = v0 + 3 * s;
            const double* r1 = r0 + 3 * L;
            const double* r2 = r1 + 3 * L;
            a0 = fma(r0[2], x2, fma(r0[1], x1, fma(r0[0], x0, a0)));
            a1 = fma(r1[2], x2, fma(r1[1], x1, fma(r1[0], x0, a1)));
            a2 = fma(r2[2], x2, fma(r2[1], x1, fma(r2[0], x0, a2)));
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            a0 += __shfl_xor_sync(0xffffffffu, a0, d);
            a1 += __shfl_xor_sync(0xffffffffu, a1, d);
            a2 += __shfl_xor_sync(0xffffffffu, a2, d);
        }
        if (lane == 0) {
            y[3 * I] = a0; y[3 * I + 1] = a1; y[3 * I + 2] = a2;
            if (part_xy) dot += (x[3 * I] * a0 + x[3 * I + 1] * a1) + x[3 * I + 2] * a2;
        }
    }
    if (part_xy) {
        __syncthreads();
        if (lane == 0) sh[wid] = dot;
        __syncthreads();
        if (threadIdx.x == 0) {
            double t = 0.0;
            for (int i = 0; i < SV_THREADS / 32; ++i) t += sh[i];
            part_xy[blockIdx.x] = t;
        }
    }
}

// inverse of the 3x3 diagonal block of every node (block Jacobi), 9 doubles per node, row-major.
// A block that is not positive definite falls back to its positive diagonal entries; nodes without
// entries (in no support) get 0: their unknowns stay 0.
__global__ void diag_inv_kernel(int64_t N, const int64_t* __restrict__ brow_ptr, const int* __restrict__ bdiag,
                                const double* __restrict__ vals, double* __restrict__ dinv) {
    const int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (I >= N) return;
    const int64_t o = brow_ptr[I], L = brow_ptr[I + 1] - o;
    double m[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    if (L > 0)
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int b = 0; b < 3; ++b) m[a][b] = vals[9 * o + a * 3 * L + 3 * (int64_t)bdiag[I] + b];
    const double c00 = m[1][1] * m[2][2] - m[1][2] * m[2][1];
    const double c01 = m[1][2] * m[2][0] - m[1][0] * m[2][2];
    const double c02 = m[1][0] * m[2][1] - m[1][1] * m[2][0];
    const double det = (m[0][0] * c00 + m[0][1] * c01) + m[0][2] * c02;
    double inv[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    const bool spd = m[0][0] > 0.0 && c00 > 0.0 && det > 0.0 && isfinite(det);   // leading minors (Sylvester, from the last row up)
    if (spd) {
        const double rd = 1.0 / det;
        inv[0] = c00 * rd;
        inv[1] = (m[0][2] * m[2][1] - m[0][1] * m[2][2]) * rd;
        inv[2] = (m[0][1] * m[1][2] - m[0][2] * m[1][1]) * rd;
        inv[3] = c01 * rd;
        inv[4] = (m[0][0] * m[2][2] - m[0][2] * m[2][0]) * rd;
        inv[5] = (m[0][2] * m[1][0] - m[0][0] * m[1][2]) * rd;
        inv[6] = c02 * rd;
        inv[7] = (m[0][1] * m[2][0] - m[0][0] * m[2][1]) * rd;
        inv[8] = (m[0][0] * m[1][1] - m[0][1] * m[1][0]) * rd;
    } else {
#pragma unroll
        for (int a = 0; a < 3; ++a) inv[4 * a] = (m[a][a] > 0.0) ? 1.0 / m[a][a] : 0.0;
    }
#pragma unroll
    for (int e = 0; e < 9; ++e) dinv[9 * I + e] = inv[e];
}

__device__ __forceinline__ void apply_block(const double* __restrict__ d, double r0, double r1, double r2, double& z0,
                                            double& z1, double& z2) {
    z0 = fma(d[2], r2, fma(d[1], r1, d[0] * r0));
    z1 = fma(d[5], r2, fma(d[4], r1, d[3] * r0));
    z2 = fma(d[8], r2, fma(d[7], r1, d[6] * r0));
}

// r = f - y, z = Dinv r, p = z; partial sums of r.z and r.r (one thread per node, contiguous slice per block)
__global__ void __launch_bounds__(SV_THREADS)
pcg_init_kernel(int64_t N, const double* __restrict__ f, const double* __restrict__ y, const double* __restrict__ dinv,
                double* __restrict__ r, double* __restrict__ z, double* __restrict__ p, double* __restrict__ part_rz,
                double* __restrict__ part_rr) {
    __shared__ double sh[SV_THREADS / 32];
    double rz = 0.0, rr = 0.0;
    const int64_t per = (N + gridDim.x - 1) / gridDim.x;   // contiguous slice per block: fixed summation order
    const int64_t lo = per * blockIdx.x, hi = min(N, lo + per);
    for (int64_t I = lo + threadIdx.x; I < hi; I += SV_THREADS) {
        const double r0 = f[3 * I] - y[3 * I], r1 = f[3 * I + 1] - y[3 * I + 1], r2 = f[3 * I + 2] - y[3 * I + 2];
        double z0, z1, z2;
        apply_block(dinv + 9 * I, r0, r1, r2, z0, z1, z2);
        r[3 * I] = r0; r[3 * I + 1] = r1; r[3 * I + 2] = r2;
        z[3 * I] = z0; z[3 * I + 1] = z1; z[3 * I + 2] = z2;
        p[3 * I] = z0; p[3 * I + 1] = z1; p[3 * I + 2] = z2;
        rz = fma(r2, z2, fma(r1, z1, fma(r0, z0, rz)));
        rr = fma(r2, r2, fma(r1, r1, fma(r0, r0, rr)));
    }
    const double t0 = block_sum(rz, sh);
    const double t1 = block_sum(rr, sh);
    if (threadIdx.x == 0) { part_rz[blockIdx.x] = t0; part_rr[blockIdx.x] = t1; }
}

// one block: fixed-order sum of the partials, then the scalar recurrences
// mode 0: rz = sum(a), rr = sum(b)            (after init)
// mode 1: pAp = sum(a), alpha = rz / pAp      (after the product)
// mode 2: rz' = sum(a), rr = sum(b), beta = rz' / rz, rz = rz'
__global__ void pcg_scalar_kernel(int mode, const double* __restrict__ pa, const double* __restrict__ pb, int nparts,
                                  double* __restrict__ sc) {
    __shared__ double sh[SV_THREADS / 32];
    double a = 0.0, b = 0.0;
    for (int i = threadIdx.x; i < nparts; i += SV_THREADS) { a += pa[i]; if (pb) b += pb[i]; }
    const double ta = block_sum(a, sh);
    const double tb = block_sum(b, sh);
    if (threadIdx.x == 0) {
        if (mode == 0) { sc[S_RZ] = ta; sc[S_RR] = tb; sc[S_BREAK] = 0.0; }
        else if (mode == 1) {
            // p^T K p must be positive for a definite K; anything else (semi-definite K from singular points or
            // unconstrained components, overflow) is a breakdown: freeze the iterate and raise the flag
            const bool ok = ta > 0.0 && ta < 1.7976931348623157e308 && (sc[S_BREAK] == 0.0);
            sc[S_PAP] = ta;
            sc[S_ALPHA] = ok ? sc[S_RZ] / ta : 0.0;
            if (!ok && sc[S_RR] != 0.0) sc[S_BREAK] = 1.0;   // (r = 0 exactly is convergence, not a breakdown)
        }
        else { sc[S_BETA] = (sc[S_RZ] != 0.0) ? ta / sc[S_RZ] : 0.0; sc[S_RZ] = ta; sc[S_RR] = tb; }
    }
}

// x += alpha p, r -= alpha Ap, z = Dinv r; partial sums of r.z and r.r (one thread per node)
__global__ void __launch_bounds__(SV_THREADS)
pcg_update_kernel(int64_t N, const double* __restrict__ sc, const double* __restrict__ p, const double* __restrict__ Ap,
                  const double* __restrict__ dinv, double* __restrict__ x, double* __restrict__ r,
                  double* __restrict__ z, double* __restrict__ part_rz, double* __restrict__ part_rr) {
    __shared__ double sh[SV_THREADS / 32];
    const double alpha = sc[S_ALPHA];
    double rz = 0.0, rr = 0.0;
    const int64_t per = (N + gridDim.x - 1) / gridDim.x;
    const int64_t lo = per * blockIdx.x, hi = min(N, lo + per);
    for (int64_t I = lo + threadIdx.x; I < hi; I += SV_THREADS) {
        double rn[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int64_t i = 3 * I + c;
            x[i] = fma(alpha, p[i], x[i]);
            rn[c] = fma(-alpha, Ap[i], r[i]);
            r[i] = rn[c];
        }
        double z0, z1, z2;
        apply_block(dinv + 9 * I, rn[0], rn[1], rn[2], z0, z1, z2);
        z[3 * I] = z0; z[3 * I + 1] = z1; z[3 * I + 2] = z2;
        rz = fma(rn[2], z2, fma(rn[1], z1, fma(rn[0], z0, rz)));
        rr = fma(rn[2], rn[2], fma(rn[1], rn[1], fma(rn[0], rn[0], rr)));
    }
    const double t0 = block_sum(rz, sh);
    const double t1 = block_sum(rr, sh);
    if (threadIdx.x == 0) { part_rz[blockIdx.x] = t0; part_rr[blockIdx.x] = t1; }
}

__global__ void pcg_direction_kernel(int64_t n, const double* __restrict__ sc, const double* __restrict__ z,
                                     double* __restrict__ p) {
    const double beta = sc[S_BETA];
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        p[i] = fma(beta, p[i], z[i]);
}

__global__ void __launch_bounds__(SV_THREADS)
norm2_kernel(int64_t n, const double* __restrict__ v, double* __restrict__ part) {
    __shared__ double sh[SV_THREADS / 32];
    double s = 0.0;
    const int64_t per = (n + gridDim.x - 1) / gridDim.x;
    const int64_t lo = per * blockIdx.x, hi = min(n, lo + per);
    for (int64_t i = lo + threadIdx.x; i < hi; i += SV_THREADS) s = fma(v[i], v[i], s);
    const double t = block_sum(s, sh);
    if (threadIdx.x == 0) part[blockIdx.x] = t;
}

// sigma (Voigt xx yy zz xy yz zx) = D eps, eps = sum_I B_I u_I with the staged gradients; one warp per point
__global__ void __launch_bounds__(SV_THREADS)
stress_kernel(int64_t Nq, int k, const int32_t* __restrict__ support, const double* __restrict__ stage,
              const double* __restrict__ u, const double* __restrict__ escale, double lambda0, double mu0, double* __restrict__ sigma) {
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int64_t q = (int64_t)blockIdx.x * (SV_THREADS / 32) + wid; q < Nq; q += (int64_t)gridDim.x * (SV_THREADS / 32)) {
        double e[6] = {0, 0, 0, 0, 0, 0};   // exx eyy ezz gxy gyz gzx (engineering shear)
        for (int j = lane; j < k; j += 32) {
            const int64_t J = support[q * k + j];
            const double* g = stage + q * 4 * k + j;   // staged layout [q][phi, d/dx, d/dy, d/dz][k]
            const double gx = g[k], gy = g[2 * k], gz = g[3 * k];
            const double ux = u[3 * J], uy = u[3 * J + 1], uz = u[3 * J + 2];
            e[0] = fma(gx, ux, e[0]);
            e[1] = fma(gy, uy, e[1]);
            e[2] = fma(gz, uz, e[2]);
            e[3] = fma(gx, uy, fma(gy, ux, e[3]));
            e[4] = fma(gy, uz, fma(gz, uy, e[4]));
            e[5] = fma(gx, uz, fma(gz, ux, e[5]));
        }
#pragma unroll
        for (int c = 0; c < 6; ++c)
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) e[c] += __shfl_xor_sync(0xffffffffu, e[c], d);
        if (lane == 0) {
            const double sc = escale ? escale[q] : 1.0;   // R8b: the point's modulus scale
            const double lambda = escale ? lambda0 * sc : lambda0, mu = escale ? mu0 * sc : mu0;
            const double tr = (e[0] + e[1]) + e[2];
            double* s = sigma + 6 * q;
            s[0] = fma(2.0 * mu, e[0], lambda * tr);
            s[1] = fma(2.0 * mu, e[1], lambda * tr);
            s[2] = fma(2.0 * mu, e[2], lambda * tr);
            s[3] = mu * e[3]; s[4] = mu * e[4]; s[5] = mu * e[5];
        }
    }
}

}  // namespace

extern "C" {

int rpim_matvec(rpim_ctx* ctx, const double* d_vals, const double* d_x, double* d_y) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!ctx->have_pattern) RPIM_FAIL(ctx, RPIM_ERR_STATE, "rpim_matvec before rpim_build_pattern");
    if (!d_vals || !d_x || !d_y) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "null pointer");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    const unsigned nb = (unsigned)std::min<int64_t>((ctx->N + 7) / 8, 148 * 16);
    bspmv_kernel<<<nb, SV_THREADS, 0, ctx->stream>>>(ctx->N, ctx->d_brow_ptr, ctx->d_bcol, d_vals, d_x, d_y, nullptr);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}

int rpim_solve_pcg(rpim_ctx* ctx, const double* d_vals, const double* d_f, double* d_u, double rel_tol, int max_iter,
                   int* out_iters, double* out_rel_resid) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!ctx->have_pattern) RPIM_FAIL(ctx, RPIM_ERR_STATE, "rpim_solve_pcg before rpim_build_pattern");
    if (!d_vals || !d_f || !d_u || !(rel_tol > 0.0) || max_iter < 0) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "null pointer, rel_tol <= 0 or max_iter < 0");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const int64_t N = ctx->N, n = 3 * N;
    double* w = nullptr;   // r | z | p | Ap | Dinv (9 per node) | partials a | partials b | scalars
    int rc;
    if ((rc = ws_alloc(ctx, &w, 7 * n + 2 * SV_PARTS + S_NUM))) return rc;
    double *r = w, *z = w + n, *p = w + 2 * n, *Ap = w + 3 * n, *dinv = w + 4 * n;
    double *pa = w + 7 * n, *pb = pa + SV_PARTS, *sc = pb + SV_PARTS;
    const unsigned nbm = (unsigned)std::min<int64_t>((N + 7) / 8, SV_PARTS);
    const unsigned nbv = (unsigned)std::min<int64_t>((n + SV_THREADS - 1) / SV_THREADS, SV_PARTS);
    const unsigned nbn = (unsigned)std::min<int64_t>((N + SV_THREADS - 1) / SV_THREADS, SV_PARTS);   // node-wise kernels
    auto fail = [&](int code) { ws_free(ctx, &w); return code; };
#define SOLVE_LAUNCH_CHECK()                                                         \
    do {                                                                             \
        ctx->launches++;                                                             \
        cudaError_t _e = cudaGetLastError();                                         \
        if (_e != cudaSuccess) {                                                     \
            ctx->err = std::string("kernel launch failed: ") + cudaGetErrorString(_e); \
            return fail(RPIM_ERR_CUDA);                                              \
        }                                                                            \
    } while (0)
    diag_inv_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(N, ctx->d_brow_ptr, ctx->d_bdiag, d_vals, dinv);
    SOLVE_LAUNCH_CHECK();
    // ||f||^2 (the tolerance is relative to it)
    norm2_kernel<<<nbv, SV_THREADS, 0, st>>>(n, d_f, pa);
    SOLVE_LAUNCH_CHECK();
    pcg_scalar_kernel<<<1, SV_THREADS, 0, st>>>(0, pa, nullptr, (int)nbv, sc);
    SOLVE_LAUNCH_CHECK();
    double h_sc[S_NUM];
    if (cudaMemcpyAsync(h_sc, sc, sizeof(h_sc), cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) {
        ctx->err = "device to host copy failed";
        return fail(RPIM_ERR_CUDA);
    }
    const double ff = h_sc[S_RZ];
    int it = 0;
    double rel = 0.0;
    bool breakdown = false;
    if (!std::isfinite(ff)) {
        // a NaN or Inf in the load vector is not "f = 0": report it instead of a converged solve (d_u untouched)
        if (out_iters) *out_iters = 0;
        if (out_rel_resid) *out_rel_resid = ff;
        ctx->err = "rpim_solve_pcg: the load vector is not finite (||f||^2 is NaN or Inf)";
        return fail(RPIM_ERR_BREAKDOWN);
    }
    if (ff == 0.0) {
        // f = 0: the solution of the definite system is u = 0, whatever the initial guess was
        if (cudaMemsetAsync(d_u, 0, (size_t)n * sizeof(double), st) != cudaSuccess) { ctx->err = "memset failed"; return fail(RPIM_ERR_CUDA); }
    } else {
        bspmv_kernel<<<nbm, SV_THREADS, 0, st>>>(N, ctx->d_brow_ptr, ctx->d_bcol, d_vals, d_u, Ap, nullptr);
        SOLVE_LAUNCH_CHECK();
        pcg_init_kernel<<<nbn, SV_THREADS, 0, st>>>(N, d_f, Ap, dinv, r, z, p, pa, pb);
        SOLVE_LAUNCH_CHECK();
        pcg_scalar_kernel<<<1, SV_THREADS, 0, st>>>(0, pa, pb, (int)nbn, sc);
        SOLVE_LAUNCH_CHECK();
        const int check = 25;   // iterations between two looks at the residual (one small copy each)
        while (true) {
            if (cudaMemcpyAsync(h_sc, sc, sizeof(h_sc), cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) {
                ctx->err = "device to host copy failed";
                return fail(RPIM_ERR_CUDA);
            }
            rel = std::sqrt(h_sc[S_RR] / ff);
            breakdown = h_sc[S_BREAK] != 0.0;
            if (!(rel > rel_tol) || it >= max_iter || breakdown) break;   // also leaves on NaN
            const int todo = std::min(check, max_iter - it);
            for (int s = 0; s < todo; ++s) {
                bspmv_kernel<<<nbm, SV_THREADS, 0, st>>>(N, ctx->d_brow_ptr, ctx->d_bcol, d_vals, p, Ap, pa);
                SOLVE_LAUNCH_CHECK();
                pcg_scalar_kernel<<<1, SV_THREADS, 0, st>>>(1, pa, nullptr, (int)nbm, sc);
                SOLVE_LAUNCH_CHECK();
                pcg_update_kernel<<<nbn, SV_THREADS, 0, st>>>(N, sc, p, Ap, dinv, d_u, r, z, pa, pb);
                SOLVE_LAUNCH_CHECK();
                pcg_scalar_kernel<<<1, SV_THREADS, 0, st>>>(2, pa, pb, (int)nbn, sc);
                SOLVE_LAUNCH_CHECK();
                pcg_direction_kernel<<<nbv, SV_THREADS, 0, st>>>(n, sc, z, p);
                SOLVE_LAUNCH_CHECK();
            }
            it += todo;
        }
        // what is reported is the TRUE residual ||f - K u|| / ||f|| of the returned iterate, not the
        // recurrence value the loop watched (the two drift apart over thousands of iterations)
        bspmv_kernel<<<nbm, SV_THREADS, 0, st>>>(N, ctx->d_brow_ptr, ctx->d_bcol, d_vals, d_u, Ap, nullptr);
        SOLVE_LAUNCH_CHECK();
        pcg_init_kernel<<<nbn, SV_THREADS, 0, st>>>(N, d_f, Ap, dinv, r, z, p, pa, pb);
        SOLVE_LAUNCH_CHECK();
        pcg_scalar_kernel<<<1, SV_THREADS, 0, st>>>(0, pa, pb, (int)nbn, sc);
        SOLVE_LAUNCH_CHECK();
        if (cudaMemcpyAsync(h_sc, sc, sizeof(h_sc), cudaMemcpyDeviceToHost, st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) {
            ctx->err = "device to host copy failed";
            return fail(RPIM_ERR_CUDA);
        }
        rel = std::sqrt(h_sc[S_RR] / ff);
    }
#undef SOLVE_LAUNCH_CHECK
    ws_free(ctx, &w);
    if (out_iters) *out_iters = it;
    if (out_rel_resid) *out_rel_resid = rel;
    if (breakdown || !(rel == rel))
        RPIM_FAIL(ctx, RPIM_ERR_BREAKDOWN, "conjugate gradients broke down within %d iterations (p^T K p <= 0 or not finite: K is "
                  "not positive definite -- singular points, unconstrained rigid-body modes?); relative residual %.3e", it, rel);
    return RPIM_OK;
}

int rpim_recover_stress(rpim_ctx* ctx, const double* d_u, double E, double nu, double* d_sigma) {
    if (!ctx) return RPIM_ERR_INVALID_ARG;
    if (!ctx->have_shape) RPIM_FAIL(ctx, RPIM_ERR_STATE, "rpim_recover_stress before rpim_assemble");
    if (!d_u || !d_sigma || !(nu > -1.0 && nu < 0.5)) RPIM_FAIL(ctx, RPIM_ERR_INVALID_ARG, "null pointer or nu outside (-1, 0.5)");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    const double lambda = E * nu / ((1.0 + nu) * (1.0 - 2.0 * nu));
    const double mu = E / (2.0 * (1.0 + nu));
    const unsigned nb = (unsigned)std::min<int64_t>((ctx->Nq + 7) / 8, 148 * 16);
    stress_kernel<<<nb, SV_THREADS, 0, ctx->stream>>>(ctx->Nq, ctx->k, ctx->d_support, ctx->d_stage, d_u, ctx->d_escale, lambda, mu,
                                                      d_sigma);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}

}  // extern "C"
