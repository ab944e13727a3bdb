// =====================================================================================
// RPIM ORACLE  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// A plain, slow, single-threaded CPU implementation of the data-parallel hot path of
// meshfree RPIM (GeoMFree3D, arXiv 1802.04256): support search, CSR pattern, moment
// matrix, shape functions, w*B^T*D*B assembly, body-force / traction loads, penalty BCs.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may build, load or call this file.  It shares no code, header, table generator or
// helper with the CUDA library (paper_1802_04256_b200/csrc); the two are written
// independently from the readings listed in DESIGN.md ("Readings of the paper").
//
// What the paper fixes (PAPER.md = /root/reference/PAPER.md at build time of this repo):
//   * the method is the Radial Point Interpolation Method of Liu (refs [23,24])
//   * stage 1 assembles the global stiffness matrix from independent per-unit element
//     matrices, stage 2 enforces displacement BCs by the penalty
//     function method, stage 3 solves.
// The paper prints no formula; every formula below is the standard RPIM definition with
// the parameters BASELINE.json fixes, and every choice the paper leaves open is the
// numbered reading R1..R12 of DESIGN.md.  Each function cites the reading it follows.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): brute-force kNN, pattern invariants,
// pow vs powl, partition of unity / linear reproduction / Kronecker delta, dense
// long-double solve of the plainly-built moment matrix (orc_shape_dense_ref, which uses
// neither pow_qm1 nor the LDL^T below), symmetry of K, rigid-body null space, energy
// identity on linear fields, load resultants, cantilever closed form, penalty exactness;
// K and f end to end against the definition in long double (orc_assemble_dense_ref: plain G,
// powl, partial-pivoting LU, literal B and D, long-double sums).
// No function in this file is "parity unpinned".
//
// Floating point: fp64, compiled with -ffp-contract=off so that a*b+c is never fused
// unless written as fma().  Build: see oracle/build.py.
// =====================================================================================
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

namespace {

// ------------------------------------------------------------------------------------
// R5: reproducible evaluation of t^(q-1).
//   a      = q - 1.0
//   b_0    = 1, b_j = (b_{j-1} * (a - (j-1))) / j          j = 1..9   (binomial series)
//   c_i    = 1 + (2i+1)/64, invc_i = 1.0 / c_i             i = 0..31
//   E_i    = RN( invc_i^(-a) )      (long-double powl, rounded to double)
//   F_e    = RN( 2^(e*a) )          e = -64..63
//   t = m * 2^e, m in [1,2), i = top 5 mantissa bits, r = fma(m, invc_i, -1)
//   t^a   ~= (F_e * E_i) * Horner_fma(b_9..b_0; r)
// Domain: normal positive t with 2^-64 <= t < 2^64, anything else gives NaN.
// ------------------------------------------------------------------------------------
struct PowTab {
    double a;
    double b[10];
    double invc[32];
    double E[32];
    double F[128];
};

void pow_setup(double q, PowTab& T) {
    T.a = q - 1.0;
    T.b[0] = 1.0;
    for (int j = 1; j <= 9; ++j) T.b[j] = (T.b[j - 1] * (T.a - (double)(j - 1))) / (double)j;
    for (int i = 0; i < 32; ++i) {
        double c = 1.0 + (double)(2 * i + 1) / 64.0;
        T.invc[i] = 1.0 / c;
        T.E[i] = (double)powl((long double)T.invc[i], -(long double)T.a);
    }
    for (int e = -64; e <= 63; ++e)
        T.F[e + 64] = (double)powl(2.0L, (long double)e * (long double)T.a);
}

inline double pow_qm1(double t, const PowTab& T) {
    uint64_t bits;
    std::memcpy(&bits, &t, 8);
    int64_t e = (int64_t)(bits >> 52) - 1023;  // sign bit set -> e >= 1025 -> rejected
    if (e < -64 || e > 63) return std::numeric_limits<double>::quiet_NaN();
    int i = (int)((bits >> 47) & 31u);
    uint64_t mb = (bits & 0x000FFFFFFFFFFFFFull) | 0x3FF0000000000000ull;
    double m;
    std::memcpy(&m, &mb, 8);
    double r = std::fma(m, T.invc[i], -1.0);
    double p = T.b[9];
    for (int j = 8; j >= 0; --j) p = std::fma(p, r, T.b[j]);
    return (T.F[e + 64] * T.E[i]) * p;
}

struct ShapeParams {
    double inv_dc;   // 1.0 / d_c
    double ac2;      // alpha_c * alpha_c   (dimensionless shape parameter squared)
    double q;
    double twoq;     // 2.0 * q
    PowTab pw;
};

void shape_setup(double alpha_c, double d_c, double q, ShapeParams& P) {
    P.inv_dc = 1.0 / d_c;
    P.ac2 = alpha_c * alpha_c;
    P.q = q;
    P.twoq = 2.0 * q;
    pow_setup(q, P.pw);
}

// ------------------------------------------------------------------------------------
// R3-R7: RPIM shape functions at one point.
//   moment system  G [a; b] = [r; p],   G = [[R0, P], [P^T, 0]]  ((k+4) x (k+4)),
//   R0_ij = (|X_i - X_j|^2 + ac2)^q, P_i = [1, X_i, Y_i, Z_i], local dimensionless
//   coordinates X_i = (x_i - x_q) * inv_dc   (BASELINE.json north_star: "(k+4)x(k+4)
//   RPIM moment matrix (multiquadric RBF plus linear polynomial)"; configs[0]:
//   "R = (r^2 + (4.0*h)^2)^1.03").
// Solve (R6/R7): structured symmetric elimination
//   (1) anchors a_0..a_3 by Gaussian elimination with partial pivoting on [1 X Y Z];
//   (2) unknown order [a_0, poly0, a_1, poly1, a_2, poly2, a_3, poly3, other nodes asc.];
//   (3) four 2x2 pivots {node a_m, poly m} (the (poly,poly) entry is exactly zero),
//       then 1x1 pivots in order on the remaining (definite) Schur complement;
//   (4) every update is a single fma in ascending pivot order, multipliers are
//       value * reciprocal, reciprocals are IEEE 1.0/x.
// Output: phi[k], dphi[3][k] (derivatives w.r.t. physical x, y, z), in support order.
// Returns 0, or 1 if the point is singular (outputs zeroed).
// ------------------------------------------------------------------------------------
int shape_point(const double* nodes, const int32_t* supp, int k, const double* xq,
                const ShapeParams& SP, double* phi, double* dphi, std::vector<double>& work) {
    const int n = k + 4;
    for (int i = 0; i < k; ++i) phi[i] = 0.0;
    for (int i = 0; i < 3 * k; ++i) dphi[i] = 0.0;

    std::vector<double> X(3 * (size_t)k);
    for (int i = 0; i < k; ++i)
        for (int c = 0; c < 3; ++c)
            X[3 * i + c] = (nodes[3 * (size_t)supp[i] + c] - xq[c]) * SP.inv_dc;

    // ---- (1) anchors: partial pivoting on W = [1 X Y Z]
    std::vector<double> W(4 * (size_t)k);
    double wmax = 0.0;
    for (int i = 0; i < k; ++i) {
        W[4 * i] = 1.0;
        for (int c = 0; c < 3; ++c) W[4 * i + 1 + c] = X[3 * i + c];
        for (int c = 0; c < 4; ++c) wmax = std::max(wmax, std::fabs(W[4 * i + c]));
    }
    int anchor[4];
    std::vector<char> used(k, 0);
    for (int m = 0; m < 4; ++m) {
        int best = -1;
        double bv = -1.0;
        for (int i = 0; i < k; ++i) {
            if (used[i]) continue;
            double v = std::fabs(W[4 * i + m]);
            if (v > bv) { bv = v; best = i; }   // strict > : ties keep the smallest i
        }
        if (best < 0 || !(bv > 1e-12 * wmax)) return 1;
        anchor[m] = best;
        used[best] = 1;
        double rinv = 1.0 / W[4 * best + m];
        for (int i = 0; i < k; ++i) {
            if (used[i]) continue;
            double f = W[4 * i + m] * rinv;
            for (int j = m + 1; j < 4; ++j) W[4 * i + j] = std::fma(-f, W[4 * best + j], W[4 * i + j]);
        }
    }

    // ---- (2) positions: pos -> local node index (>= 0) or poly index (-1 - m)
    std::vector<int> pos(n);
    for (int m = 0; m < 4; ++m) { pos[2 * m] = anchor[m]; pos[2 * m + 1] = -1 - m; }
    {
        int u = 8;
        for (int i = 0; i < k; ++i) if (!used[i]) pos[u++] = i;
    }

    // ---- build A (lower triangle used) and the 4 right-hand sides
    work.assign((size_t)n * n + (size_t)n * 4, 0.0);
    double* A = work.data();
    double* Y = A + (size_t)n * n;
    auto polyval = [&](int node, int m) -> double { return m == 0 ? 1.0 : X[3 * node + (m - 1)]; };
    double gmax = 0.0;
    for (int u = 0; u < n; ++u) {
        for (int v = 0; v <= u; ++v) {
            int pu = pos[u], pv = pos[v];
            double val;
            if (pu >= 0 && pv >= 0) {
                double dx = X[3 * pu] - X[3 * pv];
                double dy = X[3 * pu + 1] - X[3 * pv + 1];
                double dz = X[3 * pu + 2] - X[3 * pv + 2];
                double t = std::fma(dz, dz, std::fma(dy, dy, dx * dx)) + SP.ac2;
                val = t * pow_qm1(t, SP.pw);
                gmax = std::max(gmax, std::fabs(val));
            } else if (pu >= 0) {
                val = polyval(pu, -1 - pv);
            } else if (pv >= 0) {
                val = polyval(pv, -1 - pu);
            } else {
                val = 0.0;
            }
            A[(size_t)u * n + v] = val;
        }
    }
    for (int u = 0; u < n; ++u) {
        int pu = pos[u];
        if (pu >= 0) {
            double x = X[3 * pu], y = X[3 * pu + 1], z = X[3 * pu + 2];
            double t = std::fma(z, z, std::fma(y, y, x * x)) + SP.ac2;
            double Pw = pow_qm1(t, SP.pw);
            Y[4 * u] = t * Pw;
            double s = SP.twoq * Pw;
            Y[4 * u + 1] = s * (-x);
            Y[4 * u + 2] = s * (-y);
            Y[4 * u + 3] = s * (-z);
        } else {
            int m = -1 - pu;
            Y[4 * u + m] = 1.0;   // p(x_q) = [1,0,0,0]; d p / d X_a = e_a
        }
    }
    if (!(gmax == gmax) || !(gmax < std::numeric_limits<double>::infinity())) return 1;

    // ---- (3a) 2x2 pivots
    double rb[4], al[4];
    for (int m = 0; m < 4; ++m) {
        const int i0 = 2 * m, i1 = 2 * m + 1;
        double alpha = A[(size_t)i0 * n + i0];
        double beta = A[(size_t)i1 * n + i0];
        if (!(std::fabs(beta) > 1e-12 * wmax)) return 1;
        double rbeta = 1.0 / beta;
        rb[m] = rbeta;
        al[m] = alpha;
        // multipliers first (they need the un-updated columns i0, i1)
        for (int u = i1 + 1; u < n; ++u) {
            double w0 = A[(size_t)u * n + i0], w1 = A[(size_t)u * n + i1];
            double L0 = w1 * rbeta;
            double L1 = std::fma(-alpha, L0, w0) * rbeta;
            // trailing update uses (L0,L1) of row u and (w0,w1) of column index v
            // (rows v < u still hold their original w0,w1 because they are overwritten below
            //  only after the row loop has passed them: keep copies)
            Y[4 * u + 0] = std::fma(-L1, Y[4 * i1 + 0], std::fma(-L0, Y[4 * i0 + 0], Y[4 * u + 0]));
            Y[4 * u + 1] = std::fma(-L1, Y[4 * i1 + 1], std::fma(-L0, Y[4 * i0 + 1], Y[4 * u + 1]));
            Y[4 * u + 2] = std::fma(-L1, Y[4 * i1 + 2], std::fma(-L0, Y[4 * i0 + 2], Y[4 * u + 2]));
            Y[4 * u + 3] = std::fma(-L1, Y[4 * i1 + 3], std::fma(-L0, Y[4 * i0 + 3], Y[4 * u + 3]));
            // stash multipliers in the (unused) upper triangle so the lower part keeps w0,w1
            A[(size_t)i0 * n + u] = L0;
            A[(size_t)i1 * n + u] = L1;
        }
        for (int u = i1 + 1; u < n; ++u) {
            double L0 = A[(size_t)i0 * n + u], L1 = A[(size_t)i1 * n + u];
            for (int v = i1 + 1; v <= u; ++v) {
                double w0v = A[(size_t)v * n + i0], w1v = A[(size_t)v * n + i1];
                A[(size_t)u * n + v] = std::fma(-L1, w1v, std::fma(-L0, w0v, A[(size_t)u * n + v]));
            }
        }
        for (int u = i1 + 1; u < n; ++u) {   // now overwrite the columns with the multipliers
            A[(size_t)u * n + i0] = A[(size_t)i0 * n + u];
            A[(size_t)u * n + i1] = A[(size_t)i1 * n + u];
        }
    }
    // ---- (3b) 1x1 pivots
    std::vector<double> rinv(n, 0.0);
    for (int c = 8; c < n; ++c) {
        double d = A[(size_t)c * n + c];
        if (!(std::fabs(d) > 1e-14 * gmax)) return 1;
        double ri = 1.0 / d;
        rinv[c] = ri;
        for (int u = c + 1; u < n; ++u) {
            double l = A[(size_t)u * n + c] * ri;
            for (int v = c + 1; v <= u; ++v)
                A[(size_t)u * n + v] = std::fma(-l, A[(size_t)v * n + c], A[(size_t)u * n + v]);
            for (int r = 0; r < 4; ++r) Y[4 * u + r] = std::fma(-l, Y[4 * c + r], Y[4 * u + r]);
            A[(size_t)c * n + u] = l;   // stash in the upper triangle
        }
        for (int u = c + 1; u < n; ++u) A[(size_t)u * n + c] = A[(size_t)c * n + u];
    }
    // ---- (4) back substitution: w = D^-1 y, then x = L^-T w in axpy form, u descending
    for (int c = 8; c < n; ++c)
        for (int r = 0; r < 4; ++r) Y[4 * c + r] = Y[4 * c + r] * rinv[c];
    for (int m = 0; m < 4; ++m) {
        const int i0 = 2 * m, i1 = 2 * m + 1;
        for (int r = 0; r < 4; ++r) {
            double z0 = Y[4 * i1 + r] * rb[m];
            double z1 = std::fma(-al[m], z0, Y[4 * i0 + r]) * rb[m];
            Y[4 * i0 + r] = z0;
            Y[4 * i1 + r] = z1;
        }
    }
    for (int u = n - 1; u >= 1; --u) {
        // x_u is final here; positions inside the same 2x2 block are not coupled through L
        int vmax = (u < 8) ? ((u / 2) * 2 - 1) : (u - 1);
        for (int v = 0; v <= vmax; ++v) {
            double l = A[(size_t)u * n + v];
            for (int r = 0; r < 4; ++r) Y[4 * v + r] = std::fma(-l, Y[4 * u + r], Y[4 * v + r]);
        }
    }
    for (int u = 0; u < n; ++u) {
        int pu = pos[u];
        if (pu < 0) continue;
        phi[pu] = Y[4 * u];
        dphi[0 * k + pu] = Y[4 * u + 1] * SP.inv_dc;
        dphi[1 * k + pu] = Y[4 * u + 2] * SP.inv_dc;
        dphi[2 * k + pu] = Y[4 * u + 3] * SP.inv_dc;
    }
    for (int i = 0; i < k; ++i) {
        bool ok = std::isfinite(phi[i]) && std::isfinite(dphi[i]) && std::isfinite(dphi[k + i]) &&
                  std::isfinite(dphi[2 * k + i]);
        if (!ok) {
            for (int j = 0; j < k; ++j) phi[j] = 0.0;
            for (int j = 0; j < 3 * k; ++j) dphi[j] = 0.0;
            return 1;
        }
    }
    return 0;
}

// ------------------------------------------------------------------------------------
// R1: support = the k nearest field nodes under the order (d2, node id),
// d2 = (dx*dx + dy*dy) + dz*dz with dx = x_node - x_q, every operation rounded to
// nearest, no fma; the list is stored ascending by node id.
// ------------------------------------------------------------------------------------
struct DistId {
    double d2;
    int32_t id;
};
inline bool dist_less(const DistId& a, const DistId& b) {
    return a.d2 < b.d2 || (a.d2 == b.d2 && a.id < b.id);
}
inline double dist2(const double* p, const double* q) {
    double dx = p[0] - q[0], dy = p[1] - q[1], dz = p[2] - q[2];
    return (dx * dx + dy * dy) + dz * dz;
}

void knn_brute(const double* nodes, int64_t N, const double* qpts, int64_t Nq, int k, int32_t* support) {
    std::vector<DistId> c((size_t)N);
    for (int64_t q = 0; q < Nq; ++q) {
        for (int64_t i = 0; i < N; ++i) c[i] = {dist2(nodes + 3 * i, qpts + 3 * q), (int32_t)i};
        std::nth_element(c.begin(), c.begin() + (k - 1), c.end(), dist_less);
        std::vector<int32_t> ids(k);
        for (int j = 0; j < k; ++j) ids[j] = c[j].id;
        std::sort(ids.begin(), ids.end());
        std::copy(ids.begin(), ids.end(), support + (size_t)q * k);
    }
}

// Exact cell-grid search (the oracle's own; validated against knn_brute in the tests).
void knn_grid(const double* nodes, int64_t N, const double* qpts, int64_t Nq, int k, int32_t* support) {
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int64_t i = 0; i < N; ++i)
        for (int c = 0; c < 3; ++c) {
            lo[c] = std::min(lo[c], nodes[3 * i + c]);
            hi[c] = std::max(hi[c], nodes[3 * i + c]);
        }
    double vol = 1.0;
    for (int c = 0; c < 3; ++c) vol *= std::max(hi[c] - lo[c], 1e-300);
    double s = std::cbrt(vol / (double)N) * 1.5;   // about 3.4 nodes per cell
    int nc[3];
    for (int c = 0; c < 3; ++c) nc[c] = std::max(1, (int)std::floor((hi[c] - lo[c]) / s) + 1);
    auto cell_of = [&](const double* p, int* ci) {
        for (int c = 0; c < 3; ++c) {
            int v = (int)std::floor((p[c] - lo[c]) / s);
            ci[c] = std::min(std::max(v, 0), nc[c] - 1);
        }
    };
    int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
    std::vector<int64_t> start((size_t)ncell + 1, 0);
    std::vector<int32_t> order((size_t)N);
    std::vector<int64_t> cid((size_t)N);
    for (int64_t i = 0; i < N; ++i) {
        int ci[3];
        cell_of(nodes + 3 * i, ci);
        cid[i] = ci[0] + (int64_t)nc[0] * (ci[1] + (int64_t)nc[1] * ci[2]);
        start[cid[i] + 1]++;
    }
    for (int64_t c = 0; c < ncell; ++c) start[c + 1] += start[c];
    {
        std::vector<int64_t> cur(start.begin(), start.end() - 1);
        for (int64_t i = 0; i < N; ++i) order[cur[cid[i]]++] = (int32_t)i;
    }
    std::vector<DistId> cand;
    for (int64_t q = 0; q < Nq; ++q) {
        const double* xq = qpts + 3 * q;
        int cq[3];
        cell_of(xq, cq);
        for (int R = 1;; ++R) {
            int a[3], b[3];
            bool whole = true;
            for (int c = 0; c < 3; ++c) {
                a[c] = std::max(cq[c] - R, 0);
                b[c] = std::min(cq[c] + R, nc[c] - 1);
                if (a[c] > 0 || b[c] < nc[c] - 1) whole = false;
            }
            cand.clear();
            for (int z = a[2]; z <= b[2]; ++z)
                for (int y = a[1]; y <= b[1]; ++y)
                    for (int x = a[0]; x <= b[0]; ++x) {
                        int64_t c = x + (int64_t)nc[0] * (y + (int64_t)nc[1] * z);
                        for (int64_t p = start[c]; p < start[c + 1]; ++p) {
                            int32_t id = order[p];
                            cand.push_back({dist2(nodes + 3 * (int64_t)id, xq), id});
                        }
                    }
            if ((int64_t)cand.size() < k) {
                if (whole) break;   // k > N: caller error
                continue;
            }
            std::nth_element(cand.begin(), cand.begin() + (k - 1), cand.end(), dist_less);
            double dk = cand[k - 1].d2;
            // distance from x_q to the part of space not covered by the scanned cells
            double bound = std::numeric_limits<double>::infinity();
            for (int c = 0; c < 3; ++c) {
                if (a[c] > 0) bound = std::min(bound, xq[c] - (lo[c] + a[c] * s));
                if (b[c] < nc[c] - 1) bound = std::min(bound, (lo[c] + (b[c] + 1) * s) - xq[c]);
            }
            bound -= 1e-9 * s;   // margin for rounding in the cell assignment
            if (whole || (bound > 0.0 && dk < bound * bound)) break;
        }
        std::vector<int32_t> ids(k);
        for (int j = 0; j < k; ++j) ids[j] = cand[j].id;
        std::sort(ids.begin(), ids.end());
        std::copy(ids.begin(), ids.end(), support + (size_t)q * k);
    }
}

}  // namespace

extern "C" {

// R5: the scalar power function, exposed for the pow pin.  Returns t^(q-1).
double orc_pow_qm1(double t, double q) {
    PowTab T;
    pow_setup(q, T);
    return pow_qm1(t, T);
}

// R1.  method 0 = brute force, 1 = cell grid.  support: Nq x k int32, ascending ids.
int orc_knn(const double* nodes, int64_t N, const double* qpts, int64_t Nq, int k, int method,
            int32_t* support) {
    if (k < 1 || k > N) return -1;
    if (method == 0) knn_brute(nodes, N, qpts, Nq, k, support);
    else knn_grid(nodes, N, qpts, Nq, k, support);
    return 0;
}

// R2: scalar CSR pattern = 3x3 expansion of the union over points of supp x supp, rows
// sorted ascending; DOF id = 3*node + component.  Two calls: count (row_ptr, 3N+1
// entries, nnz = row_ptr[3N]) and fill.
static void block_columns(const int32_t* support, int64_t Nq, int k, int64_t N,
                          std::vector<int64_t>& inc_ptr, std::vector<int64_t>& inc) {
    inc_ptr.assign((size_t)N + 1, 0);
    for (int64_t e = 0; e < Nq * k; ++e) inc_ptr[support[e] + 1]++;
    for (int64_t I = 0; I < N; ++I) inc_ptr[I + 1] += inc_ptr[I];
    inc.resize((size_t)(Nq * k));
    std::vector<int64_t> cur(inc_ptr.begin(), inc_ptr.end() - 1);
    for (int64_t q = 0; q < Nq; ++q)
        for (int j = 0; j < k; ++j) inc[cur[support[q * k + j]]++] = q;
}
static void row_of(const int32_t* support, int k, const std::vector<int64_t>& inc_ptr,
                   const std::vector<int64_t>& inc, int64_t I, std::vector<int32_t>& v) {
    v.clear();
    for (int64_t p = inc_ptr[I]; p < inc_ptr[I + 1]; ++p) {
        const int32_t* s = support + (size_t)inc[p] * k;
        v.insert(v.end(), s, s + k);
    }
    std::sort(v.begin(), v.end());
    v.erase(std::unique(v.begin(), v.end()), v.end());
}

int orc_pattern_count(const int32_t* support, int64_t Nq, int k, int64_t N, int64_t* row_ptr) {
    std::vector<int64_t> inc_ptr, inc;
    block_columns(support, Nq, k, N, inc_ptr, inc);
    std::vector<int32_t> v;
    row_ptr[0] = 0;
    for (int64_t I = 0; I < N; ++I) {
        row_of(support, k, inc_ptr, inc, I, v);
        int64_t L = (int64_t)v.size();
        for (int a = 0; a < 3; ++a) row_ptr[3 * I + a + 1] = row_ptr[3 * I + a] + 3 * L;
    }
    return 0;
}

int orc_pattern_fill(const int32_t* support, int64_t Nq, int k, int64_t N, const int64_t* row_ptr,
                     int64_t* col_idx) {
    std::vector<int64_t> inc_ptr, inc;
    block_columns(support, Nq, k, N, inc_ptr, inc);
    std::vector<int32_t> v;
    for (int64_t I = 0; I < N; ++I) {
        row_of(support, k, inc_ptr, inc, I, v);
        for (int a = 0; a < 3; ++a) {
            int64_t p = row_ptr[3 * I + a];
            for (size_t s = 0; s < v.size(); ++s)
                for (int b = 0; b < 3; ++b) col_idx[p++] = 3 * (int64_t)v[s] + b;
            if (p != row_ptr[3 * I + a + 1]) return -2;
        }
    }
    return 0;
}

// R3-R7: shape functions of M points.  phi: M x k, dphi: M x 3 x k.  singular: M bytes.
int orc_shape(const double* nodes, const double* pts, const int32_t* support, int64_t M, int k,
              double alpha_c, double d_c, double q, double* phi, double* dphi, uint8_t* singular) {
    ShapeParams SP;
    shape_setup(alpha_c, d_c, q, SP);
    std::vector<double> work;
    for (int64_t p = 0; p < M; ++p) {
        int s = shape_point(nodes, support + (size_t)p * k, k, pts + 3 * p, SP, phi + (size_t)p * k,
                            dphi + (size_t)p * 3 * k, work);
        if (singular) singular[p] = (uint8_t)s;
    }
    return 0;
}

// Pin for orc_shape: the DEFINITION, in long double, with none of the machinery above.
// Builds G = [[R0, P],[P^T, 0]] in GLOBAL coordinates with R0_ij = powl(r_ij^2 + (alpha_c d_c)^2, q),
// solves the 4 right-hand sides by textbook partial-pivoting LU in long double.
int orc_shape_dense_ref(const double* nodes, const double* pts, const int32_t* support, int64_t M,
                        int k, double alpha_c, double d_c, double q, double* phi, double* dphi) {
    typedef long double ld;
    const int n = k + 4;
    std::vector<ld> A((size_t)n * n), B((size_t)n * 4);
    for (int64_t p = 0; p < M; ++p) {
        const int32_t* s = support + (size_t)p * k;
        const double* xq = pts + 3 * p;
        ld c2 = (ld)alpha_c * (ld)d_c * (ld)alpha_c * (ld)d_c;
        std::fill(A.begin(), A.end(), (ld)0);
        std::fill(B.begin(), B.end(), (ld)0);
        for (int i = 0; i < k; ++i) {
            const double* xi = nodes + 3 * (size_t)s[i];
            for (int j = 0; j < k; ++j) {
                const double* xj = nodes + 3 * (size_t)s[j];
                ld r2 = 0;
                for (int c = 0; c < 3; ++c) r2 += ((ld)xi[c] - (ld)xj[c]) * ((ld)xi[c] - (ld)xj[c]);
                A[(size_t)i * n + j] = powl(r2 + c2, (ld)q);
            }
            A[(size_t)i * n + k] = 1;
            A[(size_t)k * n + i] = 1;
            ld r2 = 0;
            for (int c = 0; c < 3; ++c) {
                A[(size_t)i * n + k + 1 + c] = (ld)xi[c];
                A[(size_t)(k + 1 + c) * n + i] = (ld)xi[c];
                r2 += ((ld)xq[c] - (ld)xi[c]) * ((ld)xq[c] - (ld)xi[c]);
            }
            B[(size_t)i * 4] = powl(r2 + c2, (ld)q);
            for (int c = 0; c < 3; ++c)   // d/dx_c (r^2 + c2)^q = 2 q (x_c - x_i,c) (r^2+c2)^(q-1)
                B[(size_t)i * 4 + 1 + c] = 2 * (ld)q * ((ld)xq[c] - (ld)xi[c]) * powl(r2 + c2, (ld)q - 1);
        }
        B[(size_t)k * 4] = 1;
        for (int c = 0; c < 3; ++c) {
            B[(size_t)(k + 1 + c) * 4] = (ld)xq[c];
            B[(size_t)(k + 1 + c) * 4 + 1 + c] = 1;
        }
        for (int c = 0; c < n; ++c) {
            int piv = c;
            for (int i = c + 1; i < n; ++i)
                if (fabsl(A[(size_t)i * n + c]) > fabsl(A[(size_t)piv * n + c])) piv = i;
            if (piv != c) {
                for (int j = 0; j < n; ++j) std::swap(A[(size_t)c * n + j], A[(size_t)piv * n + j]);
                for (int j = 0; j < 4; ++j) std::swap(B[(size_t)c * 4 + j], B[(size_t)piv * 4 + j]);
            }
            for (int i = c + 1; i < n; ++i) {
                ld l = A[(size_t)i * n + c] / A[(size_t)c * n + c];
                for (int j = c; j < n; ++j) A[(size_t)i * n + j] -= l * A[(size_t)c * n + j];
                for (int j = 0; j < 4; ++j) B[(size_t)i * 4 + j] -= l * B[(size_t)c * 4 + j];
            }
        }
        for (int c = n - 1; c >= 0; --c)
            for (int j = 0; j < 4; ++j) {
                ld v = B[(size_t)c * 4 + j];
                for (int i = c + 1; i < n; ++i) v -= A[(size_t)c * n + i] * B[(size_t)i * 4 + j];
                B[(size_t)c * 4 + j] = v / A[(size_t)c * n + c];
            }
        for (int i = 0; i < k; ++i) {
            phi[(size_t)p * k + i] = (double)B[(size_t)i * 4];
            for (int c = 0; c < 3; ++c) dphi[((size_t)p * 3 + c) * k + i] = (double)B[(size_t)i * 4 + 1 + c];
        }
    }
    return 0;
}

// R8: element stiffness w * B^T D B with the literal strain-displacement matrix B (6 x 3k,
// Voigt order xx, yy, zz, xy, yz, zx, engineering shear) and the isotropic D; body-force
// load f_{3I+c} += (w * phi_I) * b_c.  Points are accumulated in the given order with plain
// fp64 adds.  Rows are restricted to nodes [node_lo, node_hi); row_ptr / col_idx describe
// exactly those rows (row_ptr has 3*(node_hi-node_lo)+1 entries and starts at 0); vals and f
// are zeroed here.  BASELINE.json north_star: "form B (6x3k) and w*B^T*D*B, and reduce the
// result into a global CSR matrix over 3N DOFs".
// (escale: optional per-point modulus scale of DESIGN.md R8b, E_q = E * escale[q], one Poisson ratio: the
// stiffness contribution of point q is weighted by w[q] * escale[q], the load by w[q]; NULL = none)
static int assemble_impl(const double* nodes, const double* pts, const double* w, const double* escale, const int32_t* support,
                         int64_t M, int k, double E, double nu, double alpha_c, double d_c, double q,
                         const double* body, int64_t node_lo, int64_t node_hi, const int64_t* row_ptr,
                         const int64_t* col_idx, double* vals, double* f, int64_t* n_singular) {
    ShapeParams SP;
    shape_setup(alpha_c, d_c, q, SP);
    const double lam = E * nu / ((1.0 + nu) * (1.0 - 2.0 * nu));
    const double mu = E / (2.0 * (1.0 + nu));
    double D[6][6] = {};
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) D[i][j] = lam;
        D[i][i] = lam + 2.0 * mu;
        D[3 + i][3 + i] = mu;
    }
    const int64_t nrows = 3 * (node_hi - node_lo);
    std::fill(vals, vals + row_ptr[nrows], 0.0);
    std::fill(f, f + nrows, 0.0);
    std::vector<double> phi(k), dphi(3 * (size_t)k), work, B(6 * 3 * (size_t)k), DB(6 * 3 * (size_t)k);
    int64_t nsing = 0;
    for (int64_t p = 0; p < M; ++p) {
        const int32_t* s = support + (size_t)p * k;
        bool touches = false;
        for (int i = 0; i < k; ++i) touches |= (s[i] >= node_lo && s[i] < node_hi);
        if (!touches) continue;
        if (shape_point(nodes, s, k, pts + 3 * p, SP, phi.data(), dphi.data(), work)) { ++nsing; continue; }
        const double wk = escale ? w[p] * escale[p] : w[p];
        const int nc = 3 * k;
        std::fill(B.begin(), B.end(), 0.0);
        for (int i = 0; i < k; ++i) {
            double gx = dphi[i], gy = dphi[k + i], gz = dphi[2 * k + i];
            B[0 * nc + 3 * i + 0] = gx;
            B[1 * nc + 3 * i + 1] = gy;
            B[2 * nc + 3 * i + 2] = gz;
            B[3 * nc + 3 * i + 0] = gy; B[3 * nc + 3 * i + 1] = gx;
            B[4 * nc + 3 * i + 1] = gz; B[4 * nc + 3 * i + 2] = gy;
            B[5 * nc + 3 * i + 0] = gz; B[5 * nc + 3 * i + 2] = gx;
        }
        for (int r = 0; r < 6; ++r)
            for (int c = 0; c < nc; ++c) {
                double acc = 0.0;
                for (int t = 0; t < 6; ++t) acc += D[r][t] * B[t * nc + c];
                DB[r * nc + c] = acc;
            }
        for (int i = 0; i < k; ++i) {
            int64_t I = s[i];
            if (I < node_lo || I >= node_hi) continue;
            for (int a = 0; a < 3; ++a) {
                const int64_t row = 3 * (I - node_lo) + a;
                const int64_t* cb = col_idx + row_ptr[row];
                const int64_t len = row_ptr[row + 1] - row_ptr[row];
                for (int j = 0; j < k; ++j)
                    for (int b = 0; b < 3; ++b) {
                        double acc = 0.0;
                        for (int t = 0; t < 6; ++t) acc += B[t * nc + 3 * i + a] * DB[t * nc + 3 * j + b];
                        const int64_t col = 3 * (int64_t)s[j] + b;
                        const int64_t* it = std::lower_bound(cb, cb + len, col);
                        if (it == cb + len || *it != col) return -3;   // pattern does not contain the entry
                        vals[row_ptr[row] + (it - cb)] += wk * acc;
                    }
                f[row] += (w[p] * phi[i]) * body[a];
            }
        }
    }
    if (n_singular) *n_singular = nsing;
    return 0;
}

int orc_assemble(const double* nodes, const double* pts, const double* w, const int32_t* support,
                 int64_t M, int k, double E, double nu, double alpha_c, double d_c, double q,
                 const double* body, int64_t node_lo, int64_t node_hi, const int64_t* row_ptr,
                 const int64_t* col_idx, double* vals, double* f, int64_t* n_singular) {
    return assemble_impl(nodes, pts, w, nullptr, support, M, k, E, nu, alpha_c, d_c, q, body, node_lo, node_hi, row_ptr, col_idx,
                         vals, f, n_singular);
}

// R8b: strata with one Poisson ratio -- per-point modulus E_q = E * escale[q]
int orc_assemble_strata(const double* nodes, const double* pts, const double* w, const double* escale, const int32_t* support,
                        int64_t M, int k, double E, double nu, double alpha_c, double d_c, double q,
                        const double* body, int64_t node_lo, int64_t node_hi, const int64_t* row_ptr,
                        const int64_t* col_idx, double* vals, double* f, int64_t* n_singular) {
    return assemble_impl(nodes, pts, w, escale, support, M, k, E, nu, alpha_c, d_c, q, body, node_lo, node_hi, row_ptr, col_idx,
                         vals, f, n_singular);
}

// R9: point loads (face traction): f_{3I+c} += (w * phi_I) * t_c at given points with their
// own supports; f is NOT zeroed (adds to the body-force vector).
int orc_point_loads(const double* nodes, const double* pts, const double* w, const double* t,
                    const int32_t* support, int64_t M, int k, double alpha_c, double d_c, double q,
                    double* f) {
    ShapeParams SP;
    shape_setup(alpha_c, d_c, q, SP);
    std::vector<double> phi(k), dphi(3 * (size_t)k), work;
    for (int64_t p = 0; p < M; ++p) {
        const int32_t* s = support + (size_t)p * k;
        if (shape_point(nodes, s, k, pts + 3 * p, SP, phi.data(), dphi.data(), work)) continue;
        for (int i = 0; i < k; ++i)
            for (int a = 0; a < 3; ++a) f[3 * (int64_t)s[i] + a] += (w[p] * phi[i]) * t[3 * p + a];
    }
    return 0;
}

// R10: penalty method.  alpha_used = alpha * max_d K_dd if relative (max over
// all 3N diagonals BEFORE any penalty), K_dd += alpha_used, f_d += alpha_used * ubar_d for each
// constrained DOF d = 3*node + c with mask bit c set (mask NULL = all three).
int orc_penalty(const int64_t* bc_nodes, const uint8_t* bc_mask, const double* ubar, int64_t m,
                double alpha, int relative, int64_t N, const int64_t* row_ptr, const int64_t* col_idx,
                double* vals, double* f, double* alpha_used) {
    auto diag_slot = [&](int64_t d) -> int64_t {
        const int64_t* cb = col_idx + row_ptr[d];
        const int64_t len = row_ptr[d + 1] - row_ptr[d];
        const int64_t* it = std::lower_bound(cb, cb + len, d);
        if (it == cb + len || *it != d) return -1;
        return row_ptr[d] + (it - cb);
    };
    double a = alpha;
    if (relative) {
        double mx = 0.0;
        for (int64_t d = 0; d < 3 * N; ++d) {
            int64_t s = diag_slot(d);
            if (s >= 0) mx = std::max(mx, vals[s]);
        }
        a = alpha * mx;
    }
    if (alpha_used) *alpha_used = a;
    for (int64_t i = 0; i < m; ++i) {
        if (bc_nodes[i] < 0 || bc_nodes[i] >= N) return -4;
        for (int c = 0; c < 3; ++c) {
            if (bc_mask && !((bc_mask[i] >> c) & 1)) continue;
            int64_t d = 3 * bc_nodes[i] + c;
            int64_t s = diag_slot(d);
            if (s < 0) return -4;
            vals[s] += a;
            f[d] += a * ubar[3 * i + c];
        }
    }
    return 0;
}

// Pin for orc_assemble (and the definition-level bar of the CUDA path): K and f from the
// DEFINITION end to end, with none of the operation-level machinery (no pow_qm1, no local
// coordinates, no structured LDL^T, no closed form): shape functions and gradients from
// orc_shape_dense_ref (plain G in global coordinates, powl, partial-pivoting LU in long double),
// the literal B (6 x 3k) and D, w * B^T D B and w * phi * b summed over the points in long double,
// rounded to double once at the end.  Same row restriction and CSR arguments as orc_assemble.
// (BASELINE.json north_star: "form B (6x3k) and w*B^T*D*B, and reduce the result into a global
// CSR matrix"; R8.)  Singular points are not detected here (use on regular clouds).
int orc_assemble_dense_ref(const double* nodes, const double* pts, const double* w, const int32_t* support,
                           int64_t M, int k, double E, double nu, double alpha_c, double d_c, double q,
                           const double* body, int64_t node_lo, int64_t node_hi, const int64_t* row_ptr,
                           const int64_t* col_idx, double* vals, double* f) {
    typedef long double ld;
    const ld lam = (ld)E * (ld)nu / (((ld)1 + (ld)nu) * ((ld)1 - 2 * (ld)nu));
    const ld mu = (ld)E / (2 * ((ld)1 + (ld)nu));
    ld D[6][6] = {};
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) D[i][j] = lam;
        D[i][i] = lam + 2 * mu;
        D[3 + i][3 + i] = mu;
    }
    const int64_t nrows = 3 * (node_hi - node_lo);
    std::vector<ld> V((size_t)row_ptr[nrows], (ld)0), F((size_t)nrows, (ld)0);
    const int nc = 3 * k;
    std::vector<double> phi(k), dphi(3 * (size_t)k);
    std::vector<ld> B(6 * (size_t)nc), DB(6 * (size_t)nc);
    for (int64_t p = 0; p < M; ++p) {
        const int32_t* s = support + (size_t)p * k;
        bool touches = false;
        for (int i = 0; i < k; ++i) touches |= (s[i] >= node_lo && s[i] < node_hi);
        if (!touches) continue;
        orc_shape_dense_ref(nodes, pts + 3 * p, s, 1, k, alpha_c, d_c, q, phi.data(), dphi.data());
        std::fill(B.begin(), B.end(), (ld)0);
        for (int i = 0; i < k; ++i) {
            const ld gx = dphi[i], gy = dphi[k + i], gz = dphi[2 * k + i];
            B[0 * nc + 3 * i + 0] = gx;                                   // eps_xx
            B[1 * nc + 3 * i + 1] = gy;                                   // eps_yy
            B[2 * nc + 3 * i + 2] = gz;                                   // eps_zz
            B[3 * nc + 3 * i + 0] = gy; B[3 * nc + 3 * i + 1] = gx;       // gamma_xy
            B[4 * nc + 3 * i + 1] = gz; B[4 * nc + 3 * i + 2] = gy;       // gamma_yz
            B[5 * nc + 3 * i + 0] = gz; B[5 * nc + 3 * i + 2] = gx;       // gamma_zx
        }
        for (int r = 0; r < 6; ++r)
            for (int c = 0; c < nc; ++c) {
                ld acc = 0;
                for (int t = 0; t < 6; ++t) acc += D[r][t] * B[t * nc + c];
                DB[r * nc + c] = acc;
            }
        for (int i = 0; i < k; ++i) {
            const int64_t I = s[i];
            if (I < node_lo || I >= node_hi) continue;
            for (int a = 0; a < 3; ++a) {
                const int64_t row = 3 * (I - node_lo) + a;
                const int64_t* cb = col_idx + row_ptr[row];
                const int64_t len = row_ptr[row + 1] - row_ptr[row];
                for (int j = 0; j < k; ++j)
                    for (int b = 0; b < 3; ++b) {
                        ld acc = 0;
                        for (int t = 0; t < 6; ++t) acc += B[t * nc + 3 * i + a] * DB[t * nc + 3 * j + b];
                        const int64_t col = 3 * (int64_t)s[j] + b;
                        const int64_t* it = std::lower_bound(cb, cb + len, col);
                        if (it == cb + len || *it != col) return -3;
                        V[(size_t)(row_ptr[row] + (it - cb))] += (ld)w[p] * acc;
                    }
                F[(size_t)row] += (ld)w[p] * (ld)phi[i] * (ld)body[a];
            }
        }
    }
    for (size_t e = 0; e < V.size(); ++e) vals[e] = (double)V[e];
    for (size_t e = 0; e < F.size(); ++e) f[e] = (double)F[e];
    return 0;
}


}  // extern "C"
