// Steps a3 + a4 (R3-R7): per point, build the (k+4)x(k+4) multiquadric + linear
// moment system in local dimensionless coordinates, factor it with the structured symmetric
// elimination (four 2x2 pivots {anchor node, polynomial term}, then 1x1 pivots in order on the
// definite Schur complement) and solve the four right-hand sides -> phi, dphi/dx, dphi/dy, dphi/dz.
//
// Bit-level contract: only IEEE add / mul / fma / 1.0/x in the order DESIGN.md R3-R7 states; every
// matrix element's update chain is one fma per pivot in ascending pivot order, so the mapping of
// elements to lanes is free.  The file is compiled with -fmad=false: a*b+c is never contracted,
// fused operations are written as fma().
//
// This translation unit holds the generic kernel (any 4 <= k <= RPIM_MAX_K): one warp per point,
// lower triangle packed in shared memory.
#include "common.cuh"

namespace {

struct PowSmem {
    double b[10];
    double invc[32];
    double E[32];
    double F[128];
};

__device__ __forceinline__ double pow_qm1(double t, const PowSmem& T) {
    const long long bits = __double_as_longlong(t);
    const int e = (int)((unsigned long long)bits >> 52) - 1023;   // sign bit set -> e >= 1025
    if (e < -64 || e > 63) return __longlong_as_double(0x7ff8000000000000LL);
    const int i = (int)((bits >> 47) & 31);
    const double m = __longlong_as_double((bits & 0x000FFFFFFFFFFFFFLL) | 0x3FF0000000000000LL);
    const double r = fma(m, T.invc[i], -1.0);
    double p = T.b[9];
#pragma unroll
    for (int j = 8; j >= 0; --j) p = fma(p, r, T.b[j]);
    return (T.F[e + 64] * T.E[i]) * p;
}

__device__ __forceinline__ int tri(int u, int v) { return u * (u + 1) / 2 + v; }

// flattened lower-triangle index e -> (u, v), v <= u
__device__ __forceinline__ void tri_unflatten(int e, int& u, int& v) {
    int r = (int)((sqrtf(8.0f * (float)e + 1.0f) - 1.0f) * 0.5f);
    while (r * (r + 1) / 2 > e) --r;
    while ((r + 1) * (r + 2) / 2 <= e) ++r;
    u = r;
    v = e - r * (r + 1) / 2;
}

__host__ __device__ inline size_t shape_smem_doubles_per_warp(int k) {
    const int n = k + 4;
    return (size_t)n * (n + 1) / 2   // A
           + 4 * (size_t)n           // Y
           + 3 * (size_t)k           // X
           + 4 * (size_t)k           // W
           + 3 * (size_t)n           // vcol0, vcol1 / lbuf0, lbuf1 share: v0, v1, l0
           + 2 * (size_t)n           // l1, rinv
           + (size_t)(n + 1) / 2 + 8;  // pos (ints) + scalars
}

__global__ void __launch_bounds__(128)
shape_generic_kernel(const double* __restrict__ nodes, const double* __restrict__ pts,
                     const int32_t* __restrict__ support, int64_t M, int k, ShapeParams SP,
                     double* __restrict__ stage, uint8_t* __restrict__ singular, long long* __restrict__ flags) {
    extern __shared__ double smem_d[];
    __shared__ PowSmem PW;
    const int nwarps = blockDim.x >> 5;
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < 10; i += blockDim.x) PW.b[i] = SP.pw.b[i];
    for (int i = threadIdx.x; i < 32; i += blockDim.x) { PW.invc[i] = SP.pw.invc[i]; PW.E[i] = SP.pw.E[i]; }
    for (int i = threadIdx.x; i < 128; i += blockDim.x) PW.F[i] = SP.pw.F[i];
    __syncthreads();

    const int n = k + 4;
    const int T = n * (n + 1) / 2;
    double* base = smem_d + (size_t)wid * shape_smem_doubles_per_warp(k);
    double* A = base;
    double* Y = A + T;
    double* X = Y + 4 * n;      // X[c*k + i]
    double* W = X + 3 * k;      // W[4*i + m]
    double* v0 = W + 4 * k;
    double* v1 = v0 + n;
    double* l0 = v1 + n;
    double* l1 = l0 + n;
    double* rinv = l1 + n;
    int* pos = (int*)(rinv + n);

    for (int64_t q = (int64_t)blockIdx.x * nwarps + wid; q < M; q += (int64_t)gridDim.x * nwarps) {
        const int32_t* s = support + q * k;
        const double xq = pts[3 * q], yq = pts[3 * q + 1], zq = pts[3 * q + 2];
        double* out = stage + q * 4 * (int64_t)k;
        bool bad = false;

        // ---- R3: local dimensionless coordinates; W = [1 X Y Z]
        double wmax = 1.0;
        for (int i = lane; i < k; i += 32) {
            const int64_t id = s[i];
            const double x = (nodes[3 * id] - xq) * SP.inv_dc;
            const double y = (nodes[3 * id + 1] - yq) * SP.inv_dc;
            const double z = (nodes[3 * id + 2] - zq) * SP.inv_dc;
            X[i] = x; X[k + i] = y; X[2 * k + i] = z;
            W[4 * i] = 1.0; W[4 * i + 1] = x; W[4 * i + 2] = y; W[4 * i + 3] = z;
            wmax = fmax(wmax, fmax(fabs(x), fmax(fabs(y), fabs(z))));
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) wmax = fmax(wmax, __shfl_xor_sync(0xffffffffu, wmax, d));
        __syncwarp();

        // ---- R6: anchors by partial pivoting on W
        unsigned used = 0;   // bit sl set: node lane + 32*sl is an anchor
        int anchor[4];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            double bv = -1.0;
            int bi = 0x7FFFFFFF;
            for (int i = lane, sl = 0; i < k; i += 32, ++sl) {
                if (used & (1u << sl)) continue;
                const double v = fabs(W[4 * i + m]);
                if (v > bv) { bv = v; bi = i; }
            }
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                const double ov = __shfl_xor_sync(0xffffffffu, bv, d);
                const int oi = __shfl_xor_sync(0xffffffffu, bi, d);
                if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
            }
            if (!(bv > 1e-12 * wmax)) { bad = true; break; }
            anchor[m] = bi;
            if ((bi & 31) == lane) used |= 1u << (bi >> 5);
            const double ri = 1.0 / W[4 * bi + m];
            double wa[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) wa[j] = W[4 * bi + j];
            __syncwarp();
            for (int i = lane, sl = 0; i < k; i += 32, ++sl) {
                if (used & (1u << sl)) continue;
                const double f = W[4 * i + m] * ri;
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (j > m) W[4 * i + j] = fma(-f, wa[j], W[4 * i + j]);
            }
            __syncwarp();
        }
        if (bad) {
            for (int i = lane; i < 4 * k; i += 32) out[i] = 0.0;
            if (lane == 0) { singular[q] = 1; atomicAdd((unsigned long long*)&flags[FLAG_SINGULAR], 1ull); }
            __syncwarp();
            continue;
        }

        // ---- positions: [a0, poly0, a1, poly1, a2, poly2, a3, poly3, other nodes ascending]
        if (lane < 4) { pos[2 * lane] = anchor[lane]; pos[2 * lane + 1] = -1 - lane; }
        {
            int basecnt = 8;
            for (int i0 = 0, sl = 0; i0 < k; i0 += 32, ++sl) {
                const int i = i0 + lane;
                const bool keep = (i < k) && !(used & (1u << sl));
                const unsigned msk = __ballot_sync(0xffffffffu, keep);
                if (keep) pos[basecnt + __popc(msk & ((1u << lane) - 1))] = i;
                basecnt += __popc(msk);
            }
        }
        __syncwarp();

        // ---- R4: matrix (lower triangle) and right-hand sides
        double gmax = 0.0;
        for (int e = lane; e < T; e += 32) {
            int u, v;
            tri_unflatten(e, u, v);
            const int pu = pos[u], pv = pos[v];
            double val;
            if (pu >= 0 && pv >= 0) {
                const double dx = X[pu] - X[pv], dy = X[k + pu] - X[k + pv], dz = X[2 * k + pu] - X[2 * k + pv];
                const double t = fma(dz, dz, fma(dy, dy, dx * dx)) + SP.ac2;
                val = t * pow_qm1(t, PW);
                gmax = fmax(gmax, fabs(val));
                if (!(val == val)) gmax = __longlong_as_double(0x7ff8000000000000LL);
            } else if (pu >= 0) {
                const int m = -1 - pv;
                val = (m == 0) ? 1.0 : X[(m - 1) * k + pu];
            } else if (pv >= 0) {
                const int m = -1 - pu;
                val = (m == 0) ? 1.0 : X[(m - 1) * k + pv];
            } else {
                val = 0.0;
            }
            A[e] = val;
        }
        for (int u = lane; u < n; u += 32) {
            const int pu = pos[u];
            double y0 = 0.0, y1 = 0.0, y2 = 0.0, y3 = 0.0;
            if (pu >= 0) {
                const double x = X[pu], y = X[k + pu], z = X[2 * k + pu];
                const double t = fma(z, z, fma(y, y, x * x)) + SP.ac2;
                const double Pw = pow_qm1(t, PW);
                y0 = t * Pw;
                const double sc = SP.twoq * Pw;
                y1 = sc * (-x); y2 = sc * (-y); y3 = sc * (-z);
            } else {
                const int m = -1 - pu;
                y0 = (m == 0) ? 1.0 : 0.0; y1 = (m == 1) ? 1.0 : 0.0; y2 = (m == 2) ? 1.0 : 0.0; y3 = (m == 3) ? 1.0 : 0.0;
            }
            Y[4 * u] = y0; Y[4 * u + 1] = y1; Y[4 * u + 2] = y2; Y[4 * u + 3] = y3;
        }
        {   // NaN-propagating max
            bool isn = !(gmax == gmax);
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) gmax = fmax(gmax, __shfl_xor_sync(0xffffffffu, gmax, d));
            if (__any_sync(0xffffffffu, isn) || !(gmax < 1.7e308)) bad = true;
        }
        __syncwarp();

        // ---- R7 (a): four 2x2 pivots
        double rb[4], al[4];
#pragma unroll 1
        for (int m = 0; m < 4 && !bad; ++m) {
            const int i0 = 2 * m, i1 = 2 * m + 1;
            const double alpha = A[tri(i0, i0)], beta = A[tri(i1, i0)];
            if (!(fabs(beta) > 1e-12 * wmax)) { bad = true; break; }
            const double rbeta = 1.0 / beta;
            rb[m] = rbeta; al[m] = alpha;
            for (int u = i1 + 1 + lane; u < n; u += 32) {
                const double w0 = A[tri(u, i0)], w1 = A[tri(u, i1)];
                const double L0 = w1 * rbeta;
                const double L1 = fma(-alpha, L0, w0) * rbeta;
                v0[u] = w0; v1[u] = w1; l0[u] = L0; l1[u] = L1;
            }
            __syncwarp();
            const int mm = n - 1 - i1;   // trailing rows
            for (int e = lane; e < mm * (mm + 1) / 2; e += 32) {
                int du, dv;
                tri_unflatten(e, du, dv);
                const int u = i1 + 1 + du, v = i1 + 1 + dv;
                const int idx = tri(u, v);
                A[idx] = fma(-l1[u], v1[v], fma(-l0[u], v0[v], A[idx]));
            }
            for (int e = lane; e < mm * 4; e += 32) {
                const int u = i1 + 1 + (e >> 2), r = e & 3;
                Y[4 * u + r] = fma(-l1[u], Y[4 * i1 + r], fma(-l0[u], Y[4 * i0 + r], Y[4 * u + r]));
            }
            for (int u = i1 + 1 + lane; u < n; u += 32) { A[tri(u, i0)] = l0[u]; A[tri(u, i1)] = l1[u]; }
            __syncwarp();
        }
        // ---- R7 (b): 1x1 pivots in order
#pragma unroll 1
        for (int c = 8; c < n && !bad; ++c) {
            const double d = A[tri(c, c)];
            if (!(fabs(d) > 1e-14 * gmax)) { bad = true; break; }
            const double ri = 1.0 / d;
            if (lane == 0) rinv[c] = ri;
            for (int u = c + 1 + lane; u < n; u += 32) {
                const double w = A[tri(u, c)];
                v0[u] = w;
                l0[u] = w * ri;
            }
            __syncwarp();
            const int mm = n - 1 - c;
            for (int e = lane; e < mm * (mm + 1) / 2; e += 32) {
                int du, dv;
                tri_unflatten(e, du, dv);
                const int u = c + 1 + du, v = c + 1 + dv;
                const int idx = tri(u, v);
                A[idx] = fma(-l0[u], v0[v], A[idx]);
            }
            for (int e = lane; e < mm * 4; e += 32) {
                const int u = c + 1 + (e >> 2), r = e & 3;
                Y[4 * u + r] = fma(-l0[u], Y[4 * c + r], Y[4 * u + r]);
            }
            for (int u = c + 1 + lane; u < n; u += 32) A[tri(u, c)] = l0[u];
            __syncwarp();
        }
        if (bad) {
            for (int i = lane; i < 4 * k; i += 32) out[i] = 0.0;
            if (lane == 0) { singular[q] = 1; atomicAdd((unsigned long long*)&flags[FLAG_SINGULAR], 1ull); }
            __syncwarp();
            continue;
        }
        // ---- back substitution: w = D^-1 y, then x = L^-T w (axpy form, u descending)
        for (int e = lane; e < (n - 8) * 4; e += 32) {
            const int c = 8 + (e >> 2), r = e & 3;
            Y[4 * c + r] = Y[4 * c + r] * rinv[c];
        }
        if (lane < 16) {
            const int m = lane >> 2, r = lane & 3;
            const int i0 = 2 * m, i1 = 2 * m + 1;
            // rb / al live in registers indexed by m: select without dynamic indexing
            const double rbm = (m == 0) ? rb[0] : (m == 1) ? rb[1] : (m == 2) ? rb[2] : rb[3];
            const double alm = (m == 0) ? al[0] : (m == 1) ? al[1] : (m == 2) ? al[2] : al[3];
            const double z0 = Y[4 * i1 + r] * rbm;
            const double z1 = fma(-alm, z0, Y[4 * i0 + r]) * rbm;
            Y[4 * i0 + r] = z0;
            Y[4 * i1 + r] = z1;
        }
        __syncwarp();
#pragma unroll 1
        for (int u = n - 1; u >= 1; --u) {
            const int vmax = (u < 8) ? ((u >> 1) * 2 - 1) : (u - 1);
            const double yu0 = Y[4 * u], yu1 = Y[4 * u + 1], yu2 = Y[4 * u + 2], yu3 = Y[4 * u + 3];
            for (int v = lane; v <= vmax; v += 32) {
                const double l = A[tri(u, v)];
                Y[4 * v] = fma(-l, yu0, Y[4 * v]);
                Y[4 * v + 1] = fma(-l, yu1, Y[4 * v + 1]);
                Y[4 * v + 2] = fma(-l, yu2, Y[4 * v + 2]);
                Y[4 * v + 3] = fma(-l, yu3, Y[4 * v + 3]);
            }
            __syncwarp();
        }
        // ---- outputs in support order; derivatives back to physical coordinates
        bool finite = true;
        for (int u = lane; u < n; u += 32) {
            const int pu = pos[u];
            if (pu < 0) continue;
            const double p0 = Y[4 * u], g1 = Y[4 * u + 1] * SP.inv_dc, g2 = Y[4 * u + 2] * SP.inv_dc,
                         g3 = Y[4 * u + 3] * SP.inv_dc;
            finite = finite && isfinite(p0) && isfinite(g1) && isfinite(g2) && isfinite(g3);
            out[pu] = p0; out[k + pu] = g1; out[2 * k + pu] = g2; out[3 * k + pu] = g3;   // staged layout [q][phi, d/dx, d/dy, d/dz][k]
        }
        if (__any_sync(0xffffffffu, !finite)) {
            __syncwarp();
            for (int i = lane; i < 4 * k; i += 32) out[i] = 0.0;
            if (lane == 0) { singular[q] = 1; atomicAdd((unsigned long long*)&flags[FLAG_SINGULAR], 1ull); }
        } else if (lane == 0) {
            singular[q] = 0;
        }
        __syncwarp();
    }
}

}  // namespace

int rpim_stage_shape(rpim_ctx* ctx, const double* d_pts, const int32_t* d_support, int64_t M, double* d_stage,
                     uint8_t* d_singular) {
    if (M == 0) return RPIM_OK;
    const int k = ctx->k;
    {   // register-resident kernels for the support sizes of the BASELINE.json configs (shape_rows.cu)
        const int rc = rpim_stage_shape_rows(ctx, d_pts, d_support, M, d_stage, d_singular);
        if (rc <= 0) return rc;
    }
    const size_t per_warp = shape_smem_doubles_per_warp(k) * sizeof(double);
    int warps = 4;
    while (warps > 1 && per_warp * warps > 100 * 1024) warps >>= 1;
    const size_t smem = per_warp * warps;
    CUDA_TRY(ctx, cudaFuncSetAttribute(shape_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int64_t blocks = (M + warps - 1) / warps;
    const int64_t cap = 148LL * (int64_t)std::max<size_t>(1, (220 * 1024) / (smem + 2048));
    if (blocks > cap * 4) blocks = cap * 4;
    shape_generic_kernel<<<(unsigned)blocks, warps * 32, smem, ctx->stream>>>(
        ctx->d_nodes, d_pts, d_support, M, k, ctx->sp, d_stage, d_singular, ctx->d_flags);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}
