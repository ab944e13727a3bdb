// Steps a3 + a4 (R3-R7), register-resident kernels for the support sizes of the
// BASELINE.json configs.  Same operation-level contract as the generic kernel in shape.cu
// (every element's update chain is one fma per pivot in ascending pivot order), different
// decomposition:
//
//   * a group of G lanes (16 or 32) owns one quadrature point, so a warp works on 32/G points;
//   * the multiquadric entries are evaluated on a flattened, balanced list of node pairs and
//     parked in shared memory as a packed strictly-lower triangle in SUPPORT order;
//   * matrix rows live in registers, row-cyclic over the lanes of the group: lane g owns the
//     free rows g, g+G, ... (free = support nodes that are not anchors, ascending), and lanes
//     0..7 additionally own the eight head rows [a0, poly0, ..., a3, poly3];
//   * the four 2x2 pivots and then the 1x1 pivots run right-looking: the pivot column is
//     published through shared memory, every lane updates its own rows with independent fmas;
//   * multipliers overwrite the packed triangle in place and feed the axpy-form back substitution.
//
// All loops are unrolled at compile time (K is a template parameter) so that register arrays are
// indexed statically.  Lanes whose row index falls beyond the last free row duplicate the last
// row (same values to the same addresses), which removes every bounds predicate.
#include <type_traits>

#include "pow_qm1.cuh"

namespace {

constexpr unsigned FULL = 0xffffffffu;

template <int K, int G>
struct Cfg {
    static constexpr int N = K + 4;                      // moment system size
    static constexpr int M = K - 4;                      // free rows
    static constexpr int NSLOT = (M + G - 1) / G;        // free row slots per lane
    static constexpr int NT = (K + G - 1) / G;           // support slots per lane
    static constexpr int PPW = 32 / G;                   // points per warp
    static constexpr int NITEM = (K + 1) * K / 2;        // strictly-lower pairs of K nodes + the point
    static constexpr int NTRI = K * (K + 1) / 2;         // stored matrix entries (lower triangle with diagonal)
    // per-point shared memory, in doubles
    static constexpr int OFF_SL = 0;
    static constexpr int OFF_X = OFF_SL + ((NTRI + 1) & ~1);  // (K+1) x 4 local coordinates (last = the point)
    static constexpr int OFF_Y = OFF_X + 4 * (K + 1);         // K x 4 right-hand sides
    static constexpr int OFF_W = OFF_Y + 4 * K;               // N x 8 (w0, w1) per 2x2 pivot, position order
    static constexpr int OFF_L = OFF_W + 8 * N;               // N x 8 (L0, L1) per 2x2 pivot, position order
    static constexpr int CSTR = (M + 4 + 1) & ~1;
    // 2 x CSTR pivot column / solution broadcast of the 1x1 stage.  It reuses the (w0, w1) area, which
    // is dead once the free-free rows have been loaded (a __syncwarp separates the two uses): at
    // k = 60 this is what lets two CTAs share an SM.
    static constexpr int OFF_C = OFF_W;
    static_assert(2 * CSTR <= 8 * N, "broadcast area fits the (w0, w1) area");
    static constexpr int OFF_H = OFF_L + 8 * N;               // 4 pivots x 2 rows x 4 head right-hand sides
    static constexpr int RAW = OFF_H + 32;
    static constexpr int PER_POINT = ((RAW + 15) & ~15) + 8;  // = 8 mod 16: the groups of a warp hit different banks
    static constexpr int TAB_DOUBLES = ((NITEM + 3) / 4 + 1) & ~1;
};

// Node order used on chip ("nu order"): the four anchors first (nu = m), then the free nodes in
// ascending support order (nu = 4 + u).  The packed lower triangle, the coordinates and the
// right-hand sides are all indexed by nu, so every address below is lane base + compile-time offset.
__host__ __device__ constexpr int tri_row(int i) { return (i * (i + 1)) / 2; }

__device__ __forceinline__ int skipmap(int u, const int (&b)[4]) {
    int i = u;
    i += (i >= b[0]);
    i += (i >= b[1]);
    i += (i >= b[2]);
    i += (i >= b[3]);
    return i;
}

// compile-time loop: f(std::integral_constant<int, I>) for I = B, B+S, ... while I != E
template <int B, int E, int S = 1, typename F>
__device__ __forceinline__ void static_for(F&& f) {
    if constexpr (B != E) {
        f(std::integral_constant<int, B>{});
        static_for<B + S, E, S>(f);
    }
}

__device__ __forceinline__ void st2(double* p, double a, double b) { *reinterpret_cast<double2*>(p) = make_double2(a, b); }
__device__ __forceinline__ double2 ld2(const double* p) { return *reinterpret_cast<const double2*>(p); }

template <int K, int G, int WARPS>
__global__ void __launch_bounds__(WARPS * 32)
shape_rows_kernel(const double* __restrict__ nodes, const double* __restrict__ pts,
                  const int32_t* __restrict__ support, int64_t Mpts, const __grid_constant__ ShapeParams SP,
                  double* __restrict__ stage, uint8_t* __restrict__ singular, long long* __restrict__ flags) {
    using C = Cfg<K, G>;
    constexpr int N = C::N, M = C::M, NSLOT = C::NSLOT, NT = C::NT, PPW = C::PPW;
    constexpr int HS = NSLOT;   // index of the head slot in the per-slot arrays

    extern __shared__ __align__(16) double smem[];
    PowSmem& PW = *reinterpret_cast<PowSmem*>(smem);
    unsigned short* tab = reinterpret_cast<unsigned short*>(smem + 192);
    pow_smem_fill(PW, SP.pw);
    for (int e = threadIdx.x; e < C::NITEM; e += blockDim.x) {
        int r = (int)((sqrtf(8.0f * (float)e + 1.0f) - 1.0f) * 0.5f);
        while (r * (r + 1) / 2 > e) --r;
        while ((r + 1) * (r + 2) / 2 <= e) ++r;
        tab[e] = (unsigned short)(((r + 1) << 8) | (e - r * (r + 1) / 2));   // pair (i = r+1, j), j < i
    }
    __syncthreads();

    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane & (G - 1), grp = lane / G;
    double* P = smem + 192 + C::TAB_DOUBLES + (size_t)(wid * PPW + grp) * C::PER_POINT;
    double* SL = P + C::OFF_SL;
    double* Xs = P + C::OFF_X;
    double* Yb = P + C::OFF_Y;
    double* Wp = P + C::OFF_W;
    double* Lp = P + C::OFF_L;
    double* Cb = P + C::OFF_C;
    double* Yh = P + C::OFF_H;

    const double inv_dc = SP.inv_dc, ac2 = SP.ac2, twoq = SP.twoq;
    const double* pb = SP.pw.b;
    const double Rdiag = ac2 * pow_qm1(ac2, PW, pb);

    const int64_t stride = (int64_t)gridDim.x * WARPS * PPW;
    for (int64_t q0 = ((int64_t)blockIdx.x * WARPS + wid) * PPW; q0 < Mpts; q0 += stride) {
        int64_t q = q0 + grp;
        const bool live = q < Mpts;
        if (!live) q = Mpts - 1;
        const int32_t* sup = support + q * K;
        const double xq = pts[3 * q], yq = pts[3 * q + 1], zq = pts[3 * q + 2];
        bool bad = false;

        // ---- R3: local dimensionless coordinates, W = [1 X Y Z] (registers, support slots)
        double W[NT][4], X3[NT][3];
        unsigned used = 0;
        double wmax = 1.0;
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            const int i = g + G * t;
            if (i < K) {
                const int64_t id = sup[i];
                const double x = (nodes[3 * id] - xq) * inv_dc;
                const double y = (nodes[3 * id + 1] - yq) * inv_dc;
                const double z = (nodes[3 * id + 2] - zq) * inv_dc;
                X3[t][0] = x; X3[t][1] = y; X3[t][2] = z;
                W[t][0] = 1.0; W[t][1] = x; W[t][2] = y; W[t][3] = z;
                wmax = fmax(wmax, fmax(fabs(x), fmax(fabs(y), fabs(z))));
            } else {
                X3[t][0] = X3[t][1] = X3[t][2] = 0.0;
                W[t][0] = W[t][1] = W[t][2] = W[t][3] = 0.0;
                used |= 1u << t;
            }
        }
#pragma unroll
        for (int d = G / 2; d > 0; d >>= 1) wmax = fmax(wmax, __shfl_xor_sync(FULL, wmax, d));

        // ---- R6: anchors by partial pivoting on W
        int anc[4];
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            double bv = -1.0;
            int bi = 0x7FFFFFFF;
#pragma unroll
            for (int t = 0; t < NT; ++t) {
                const double v = fabs(W[t][m]);
                if (!((used >> t) & 1u) && v > bv) { bv = v; bi = g + G * t; }
            }
#pragma unroll
            for (int d = G / 2; d > 0; d >>= 1) {
                const double ov = __shfl_xor_sync(FULL, bv, d);
                const int oi = __shfl_xor_sync(FULL, bi, d);
                if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
            }
            if (!(bv > 1e-12 * wmax)) bad = true;
            if (bi >= K) bi = m;   // keep the indices valid after a failure (the result is discarded)
            anc[m] = bi;
            const int ol = bi & (G - 1), ot = bi / G;
            double wb[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (j < m) continue;
                double v = 0.0;
#pragma unroll
                for (int t = 0; t < NT; ++t)
                    if (t == ot) v = W[t][j];
                wb[j] = __shfl_sync(FULL, v, ol, G);
            }
            if (ol == g) used |= 1u << ot;
            const double ri = __drcp_rn(wb[m]);
#pragma unroll
            for (int t = 0; t < NT; ++t) {
                if ((used >> t) & 1u) continue;
                const double f = W[t][m] * ri;
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (j > m) W[t][j] = fma(-f, wb[j], W[t][j]);
            }
        }
        int bs[4] = {anc[0], anc[1], anc[2], anc[3]};   // ascending copy for the free-row map
#define RPIM_CSWAP(a, b) { const int lo_ = min(bs[a], bs[b]), hi_ = max(bs[a], bs[b]); bs[a] = lo_; bs[b] = hi_; }
        RPIM_CSWAP(0, 1) RPIM_CSWAP(2, 3) RPIM_CSWAP(0, 2) RPIM_CSWAP(1, 3) RPIM_CSWAP(1, 2)
#undef RPIM_CSWAP

        // ---- coordinates in nu order; diagonal of the multiquadric block
#pragma unroll
        for (int t = 0; t < NT; ++t) {
            const int i = g + G * t;
            if (i < K) {
                int nu = 4 + i - (i > bs[0]) - (i > bs[1]) - (i > bs[2]) - (i > bs[3]);
#pragma unroll
                for (int m = 0; m < 4; ++m)
                    if (i == anc[m]) nu = m;
                st2(Xs + 4 * nu, X3[t][0], X3[t][1]);
                Xs[4 * nu + 2] = X3[t][2];
                SL[tri_row(i) + i] = Rdiag;
            }
        }
        if (g == 0) { st2(Xs + 4 * K, 0.0, 0.0); Xs[4 * K + 2] = 0.0; }
        __syncwarp();

        // ---- R4: multiquadric entries (pairs of nodes) and right-hand sides (node, point)
        double gmax = Rdiag;
#pragma unroll 2
        for (int e0 = 0; e0 < C::NITEM; e0 += G) {
            const int e = e0 + g;
            if (e < C::NITEM) {
                const unsigned tb = tab[e];
                const int i = tb >> 8, j = tb & 255;
                const double2 aij = ld2(Xs + 4 * j);
                const double az = Xs[4 * j + 2];
                double dx, dy, dz;
                if (i < K) {
                    const double2 bij = ld2(Xs + 4 * i);
                    dx = bij.x - aij.x; dy = bij.y - aij.y; dz = Xs[4 * i + 2] - az;
                } else {
                    dx = -aij.x; dy = -aij.y; dz = -az;
                }
                const double t = fma(dz, dz, fma(dy, dy, dx * dx)) + ac2;
                const double Pw = pow_qm1(t, PW, pb);
                const double val = t * Pw;
                if (i < K) {
                    SL[e + i] = val;               // tri_row(i) + j
                    gmax = fmax(gmax, fabs(val));
                } else {
                    const double sc = twoq * Pw;
                    st2(Yb + 4 * j, val, sc * dx);
                    st2(Yb + 4 * j + 2, sc * dy, sc * dz);
                }
            }
        }
#pragma unroll
        for (int d = G / 2; d > 0; d >>= 1) gmax = fmax(gmax, __shfl_xor_sync(FULL, gmax, d));
        if (!(gmax < 1.7976931348623157e308)) bad = true;
        __syncwarp();

        // ---- rows owned by this lane: free slots 0..NSLOT-1 and the head slot
        int urow[NSLOT];
        double* SLr[NSLOT];      // row base of the lane's free rows in the packed triangle
        double h[NSLOT + 1][8], Y[NSLOT + 1][4];
        double L0[NSLOT][4], L1[NSLOT][4];
#pragma unroll
        for (int s = 0; s < NSLOT; ++s) {
            const int u = min(g + G * s, M - 1);
            urow[s] = u;
            SLr[s] = SL + tri_row(4 + u);
            const double* xr = Xs + 4 * (4 + u);
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                h[s][2 * m] = SLr[s][m];
                h[s][2 * m + 1] = (m == 0) ? 1.0 : xr[m - 1];
            }
            const double2 y01 = ld2(Yb + 4 * (4 + u)), y23 = ld2(Yb + 4 * (4 + u) + 2);
            Y[s][0] = y01.x; Y[s][1] = y01.y; Y[s][2] = y23.x; Y[s][3] = y23.y;
        }
        const int hp = min(g, 7);            // head position of this lane
        const int hm = hp >> 1;
        const bool hpoly = hp & 1;
        {
#pragma unroll
            for (int m = 0; m < 4; ++m) {
                double v0 = 0.0, v1 = 0.0;
                if (hpoly) {
                    if (m <= hm) v0 = (hm == 0) ? 1.0 : Xs[4 * m + hm - 1];        // polynomial hm at anchor m
                } else if (m < hm) {
                    v0 = SL[tri_row(hm) + m];
                    v1 = (m == 0) ? 1.0 : Xs[4 * hm + m - 1];
                } else if (m == hm) {
                    v0 = Rdiag;
                }
                h[HS][2 * m] = v0; h[HS][2 * m + 1] = v1;
            }
            if (hpoly) {
#pragma unroll
                for (int r = 0; r < 4; ++r) Y[HS][r] = (r == hm) ? 1.0 : 0.0;
            } else {
                const double2 y01 = ld2(Yb + 4 * hm), y23 = ld2(Yb + 4 * hm + 2);
                Y[HS][0] = y01.x; Y[HS][1] = y01.y; Y[HS][2] = y23.x; Y[HS][3] = y23.y;
            }
        }

        // ---- R7 (a): four 2x2 pivots {anchor m, polynomial m}
        double rb[4], al[4];
        static_for<0, 4>([&](auto m_) {
            constexpr int m = decltype(m_)::value;
#pragma unroll
            for (int s = 0; s < NSLOT; ++s) st2(Wp + 8 * (8 + urow[s]) + 2 * m, h[s][2 * m], h[s][2 * m + 1]);
            if (hp >= 2 * m) {
                st2(Wp + 8 * hp + 2 * m, h[HS][2 * m], h[HS][2 * m + 1]);
                if (hp <= 2 * m + 1) {
                    double* dst = Yh + 8 * m + 4 * (hp & 1);
                    st2(dst, Y[HS][0], Y[HS][1]);
                    st2(dst + 2, Y[HS][2], Y[HS][3]);
                }
            }
            __syncwarp();
            const double alpha = Wp[8 * (2 * m) + 2 * m], beta = Wp[8 * (2 * m + 1) + 2 * m];
            if (!(fabs(beta) > 1e-12 * wmax)) bad = true;
            const double rbeta = __drcp_rn(beta);
            rb[m] = rbeta; al[m] = alpha;
            const double2 a01 = ld2(Yh + 8 * m), a23 = ld2(Yh + 8 * m + 2);
            const double2 b01 = ld2(Yh + 8 * m + 4), b23 = ld2(Yh + 8 * m + 6);
            double2 wj[8];
#pragma unroll
            for (int j = 0; j < 8; ++j)
                if (j >= 2 * m + 2) wj[j] = ld2(Wp + 8 * j + 2 * m);
#pragma unroll
            for (int s = 0; s < NSLOT; ++s) {
                const double w0 = h[s][2 * m], w1 = h[s][2 * m + 1];
                const double l0 = w1 * rbeta;
                const double l1 = fma(-alpha, l0, w0) * rbeta;
                L0[s][m] = l0; L1[s][m] = l1;
                Y[s][0] = fma(-l1, b01.x, fma(-l0, a01.x, Y[s][0]));
                Y[s][1] = fma(-l1, b01.y, fma(-l0, a01.y, Y[s][1]));
                Y[s][2] = fma(-l1, b23.x, fma(-l0, a23.x, Y[s][2]));
                Y[s][3] = fma(-l1, b23.y, fma(-l0, a23.y, Y[s][3]));
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (j >= 2 * m + 2) h[s][j] = fma(-l1, wj[j].y, fma(-l0, wj[j].x, h[s][j]));
                st2(Lp + 8 * (8 + urow[s]) + 2 * m, l0, l1);
            }
            if (hp > 2 * m + 1) {
                const double w0 = h[HS][2 * m], w1 = h[HS][2 * m + 1];
                const double l0 = w1 * rbeta;
                const double l1 = fma(-alpha, l0, w0) * rbeta;
                Y[HS][0] = fma(-l1, b01.x, fma(-l0, a01.x, Y[HS][0]));
                Y[HS][1] = fma(-l1, b01.y, fma(-l0, a01.y, Y[HS][1]));
                Y[HS][2] = fma(-l1, b23.x, fma(-l0, a23.x, Y[HS][2]));
                Y[HS][3] = fma(-l1, b23.y, fma(-l0, a23.y, Y[HS][3]));
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (j >= 2 * m + 2) h[HS][j] = fma(-l1, wj[j].y, fma(-l0, wj[j].x, h[HS][j]));
                st2(Lp + 8 * hp + 2 * m, l0, l1);
            }
        });
        __syncwarp();

        // ---- load the free-free rows into registers and apply the four 2x2 pivots to them
        double a[NSLOT][M];
        static_for<0, M>([&](auto v_) {
            constexpr int v = decltype(v_)::value;
            const double2 w01 = ld2(Wp + 8 * (8 + v)), w23 = ld2(Wp + 8 * (8 + v) + 2);
            const double2 w45 = ld2(Wp + 8 * (8 + v) + 4), w67 = ld2(Wp + 8 * (8 + v) + 6);
#pragma unroll
            for (int s = 0; s < NSLOT; ++s) {
                if (G * s + G - 1 < v) continue;   // every row of the slot lies above column v
                double x = SLr[s][4 + v];
                x = fma(-L1[s][0], w01.y, fma(-L0[s][0], w01.x, x));
                x = fma(-L1[s][1], w23.y, fma(-L0[s][1], w23.x, x));
                x = fma(-L1[s][2], w45.y, fma(-L0[s][2], w45.x, x));
                x = fma(-L1[s][3], w67.y, fma(-L0[s][3], w67.x, x));
                a[s][v] = x;
            }
        });

        // ---- R7 (b): 1x1 pivots in order, right-looking
        __syncwarp();   // every lane has read its (w0, w1) values: the area becomes the broadcast buffer
        double rsave[NSLOT];
#pragma unroll
        for (int s = 0; s < NSLOT; ++s) rsave[s] = 0.0;
        static_for<0, M>([&](auto c_) {
            constexpr int c = decltype(c_)::value;
            double* cb = Cb + (c & 1) * C::CSTR;
            constexpr int sc = c / G;   // slot of row c
            const bool own = (urow[sc] == c);
#pragma unroll
            for (int s = 0; s < NSLOT; ++s) {
                if (G * s + G - 1 < c) continue;
                cb[urow[s]] = a[s][c];
            }
            if (own) {
                st2(cb + C::CSTR - 4, Y[sc][0], Y[sc][1]);
                st2(cb + C::CSTR - 2, Y[sc][2], Y[sc][3]);
            }
            __syncwarp();
            const double d = cb[c];
            const double2 yc01 = ld2(cb + C::CSTR - 4), yc23 = ld2(cb + C::CSTR - 2);
            if (!(fabs(d) > 1e-14 * gmax)) bad = true;
            const double rinv = __drcp_rn(d);
            if (own) rsave[sc] = rinv;
            double l[NSLOT];
#pragma unroll
            for (int s = 0; s < NSLOT; ++s) {
                if (G * s + G - 1 <= c) continue;   // no row of the slot lies below row c
                l[s] = a[s][c] * rinv;
                if (urow[s] > c) {
                    SLr[s][4 + c] = l[s];
                    Y[s][0] = fma(-l[s], yc01.x, Y[s][0]);
                    Y[s][1] = fma(-l[s], yc01.y, Y[s][1]);
                    Y[s][2] = fma(-l[s], yc23.x, Y[s][2]);
                    Y[s][3] = fma(-l[s], yc23.y, Y[s][3]);
                }
            }
#pragma unroll
            for (int v = c + 1; v < M; ++v) {
                const double cv = cb[v];
#pragma unroll
                for (int s = 0; s < NSLOT; ++s) {
                    if (G * s + G - 1 <= c || v > G * s + G - 1) continue;
                    a[s][v] = fma(-l[s], cv, a[s][v]);
                }
            }
        });

        // ---- back substitution: w = D^-1 y, then x = L^-T w in axpy form, positions descending
#pragma unroll
        for (int s = 0; s < NSLOT; ++s)
#pragma unroll
            for (int r = 0; r < 4; ++r) Y[s][r] = Y[s][r] * rsave[s];
        {
            const double rbm = (hm == 0) ? rb[0] : (hm == 1) ? rb[1] : (hm == 2) ? rb[2] : rb[3];
            const double alm = (hm == 0) ? al[0] : (hm == 1) ? al[1] : (hm == 2) ? al[2] : al[3];
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const double mine = Y[HS][r];
                const double other = __shfl_xor_sync(FULL, mine, 1);
                // anchor row (even): z0 = Y[poly] * rb; polynomial row (odd): z1 = fma(-alpha, z0, Y[anchor]) * rb
                const double z0 = (hpoly ? mine : other) * rbm;
                const double z1 = fma(-alm, z0, hpoly ? other : mine) * rbm;
                Y[HS][r] = hpoly ? z1 : z0;
            }
        }
        __syncwarp();
        const double* SLc[NSLOT];   // column base: L[u][own row] = SLc[s][tri_row(4 + u)]
#pragma unroll
        for (int s = 0; s < NSLOT; ++s) SLc[s] = SL + 4 + urow[s];
        const double* Lph = Lp + hp;
        static_for<N - 1, 1, -1>([&](auto p_) {
            constexpr int p = decltype(p_)::value;
            double* xb = Cb + (p & 1) * C::CSTR;
            if (p >= 8) {
                constexpr int sp = (p >= 8) ? (p - 8) / G : 0;
                if (urow[sp] == p - 8) { st2(xb, Y[sp][0], Y[sp][1]); st2(xb + 2, Y[sp][2], Y[sp][3]); }
            } else if (g == p) {
                st2(xb, Y[HS][0], Y[HS][1]); st2(xb + 2, Y[HS][2], Y[HS][3]);
            }
            __syncwarp();
            const double2 x01 = ld2(xb), x23 = ld2(xb + 2);
            if (p >= 8) {
                constexpr int u = p - 8;
#pragma unroll
                for (int s = 0; s < NSLOT; ++s) {
                    if (G * s >= u) continue;   // no row of the slot lies above row u
                    const double lv = SLc[s][tri_row(4 + u)];
                    if (urow[s] < u) {
                        Y[s][0] = fma(-lv, x01.x, Y[s][0]);
                        Y[s][1] = fma(-lv, x01.y, Y[s][1]);
                        Y[s][2] = fma(-lv, x23.x, Y[s][2]);
                        Y[s][3] = fma(-lv, x23.y, Y[s][3]);
                    }
                }
            }
            {
                constexpr int vmax = (p >= 8) ? 7 : ((p >> 1) * 2 - 1);
                const double lv = Lph[8 * p];
                if (hp <= vmax) {
                    Y[HS][0] = fma(-lv, x01.x, Y[HS][0]);
                    Y[HS][1] = fma(-lv, x01.y, Y[HS][1]);
                    Y[HS][2] = fma(-lv, x23.x, Y[HS][2]);
                    Y[HS][3] = fma(-lv, x23.y, Y[HS][3]);
                }
            }
        });

        // ---- outputs in support order (staged layout [q][phi, d/dx, d/dy, d/dz][K]); derivatives back to physical coordinates
        double* out = stage + q * 4 * (int64_t)K;
        bool finite = true;
#pragma unroll
        for (int s = 0; s < NSLOT; ++s) {
            const int ir = skipmap(urow[s], bs);
            const double p0 = Y[s][0], g1 = Y[s][1] * inv_dc, g2 = Y[s][2] * inv_dc, g3 = Y[s][3] * inv_dc;
            finite = finite && isfinite(p0) && isfinite(g1) && isfinite(g2) && isfinite(g3);
            if (live) { out[ir] = p0; out[K + ir] = g1; out[2 * K + ir] = g2; out[3 * K + ir] = g3; }
        }
        if (!hpoly) {
            const int ia = (hm == 0) ? anc[0] : (hm == 1) ? anc[1] : (hm == 2) ? anc[2] : anc[3];
            const double p0 = Y[HS][0], g1 = Y[HS][1] * inv_dc, g2 = Y[HS][2] * inv_dc, g3 = Y[HS][3] * inv_dc;
            finite = finite && isfinite(p0) && isfinite(g1) && isfinite(g2) && isfinite(g3);
            if (live) { out[ia] = p0; out[K + ia] = g1; out[2 * K + ia] = g2; out[3 * K + ia] = g3; }
        }
        const unsigned gmask = (G == 32) ? FULL : (0xffffu << (16 * grp));
        const bool fail = ((__ballot_sync(FULL, bad || !finite) & gmask) != 0u);
        __syncwarp();
        if (live) {
            if (fail) {
                for (int i = g; i < 4 * K; i += G) out[i] = 0.0;
                if (g == 0) { singular[q] = 1; atomicAdd((unsigned long long*)&flags[FLAG_SINGULAR], 1ull); }
            } else if (g == 0) {
                singular[q] = 0;
            }
        }
        __syncwarp();
    }
}

template <int K, int G, int WARPS>
int launch_rows(rpim_ctx* ctx, const double* d_pts, const int32_t* d_support, int64_t M, double* d_stage,
                uint8_t* d_singular) {
    using C = Cfg<K, G>;
    auto kern = shape_rows_kernel<K, G, WARPS>;
    const size_t smem = (192 + C::TAB_DOUBLES + (size_t)WARPS * C::PPW * C::PER_POINT) * sizeof(double);
    CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 1;
    CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, WARPS * 32, smem));
    if (per_sm < 1) per_sm = 1;
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->device);
    const int64_t per_block = (int64_t)WARPS * C::PPW;
    int64_t blocks = (M + per_block - 1) / per_block;
    const int64_t wave = (int64_t)sms * per_sm;
    if (blocks > wave) blocks = wave;      // persistent: one resident wave, grid-stride over the points
    kern<<<(unsigned)blocks, WARPS * 32, smem, ctx->stream>>>(ctx->d_nodes, d_pts, d_support, M, ctx->sp, d_stage,
                                                              d_singular, ctx->d_flags);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}

}  // namespace

// Returns RPIM_OK when a register-resident kernel exists for ctx->k and was launched,
// 1 when the caller has to use the generic kernel, or a negative rpim_status.
int rpim_stage_shape_rows(rpim_ctx* ctx, const double* d_pts, const int32_t* d_support, int64_t M, double* d_stage,
                          uint8_t* d_singular) {
    switch (ctx->k) {
        case 27: return launch_rows<27, 16, 4>(ctx, d_pts, d_support, M, d_stage, d_singular);
        case 30: return launch_rows<30, 16, 4>(ctx, d_pts, d_support, M, d_stage, d_singular);
        case 40: return launch_rows<40, 32, 4>(ctx, d_pts, d_support, M, d_stage, d_singular);
        case 60: return launch_rows<60, 32, 4>(ctx, d_pts, d_support, M, d_stage, d_singular);
        default: return 1;
    }
}
