// Driver for the sanitizer run of the oracle (TEST INFRASTRUCTURE): compiled
// together with rpim_oracle.cpp under -fsanitize=address,undefined by tests/test_oracle_sanitize.py
// and run on a small jittered block.  It exercises every exported function once; the test fails on
// any sanitizer report.  The inputs are built here (no arithmetic of the method: a jittered grid,
// cell-centre points) so that the program needs nothing but the oracle.
#include <cstdint>
#include <cstdio>
#include <vector>

extern "C" {
double orc_pow_qm1(double t, double q);
int orc_knn(const double*, int64_t, const double*, int64_t, int, int, int32_t*);
int orc_pattern_count(const int32_t*, int64_t, int, int64_t, int64_t*);
int orc_pattern_fill(const int32_t*, int64_t, int, int64_t, const int64_t*, int64_t*);
int orc_shape(const double*, const double*, const int32_t*, int64_t, int, double, double, double, double*, double*, uint8_t*);
int orc_shape_dense_ref(const double*, const double*, const int32_t*, int64_t, int, double, double, double, double*, double*);
int orc_assemble(const double*, const double*, const double*, const int32_t*, int64_t, int, double, double, double, double, double,
                 const double*, int64_t, int64_t, const int64_t*, const int64_t*, double*, double*, int64_t*);
int orc_assemble_dense_ref(const double*, const double*, const double*, const int32_t*, int64_t, int, double, double, double, double,
                           double, const double*, int64_t, int64_t, const int64_t*, const int64_t*, double*, double*);
int orc_point_loads(const double*, const double*, const double*, const double*, const int32_t*, int64_t, int, double, double, double, double*);
int orc_penalty(const int64_t*, const uint8_t*, const double*, int64_t, double, int, int64_t, const int64_t*, const int64_t*, double*, double*, double*);
}

int main() {
    const int nx = 6, ny = 5, nz = 5, k = 20;
    const int64_t N = nx * ny * nz;
    std::vector<double> nodes(3 * N);
    uint64_t st = 12345;
    auto rnd = [&]() { st = st * 6364136223846793005ull + 1442695040888963407ull; return (double)(st >> 11) / 9007199254740992.0 - 0.5; };
    for (int z = 0; z < nz; ++z)
        for (int y = 0; y < ny; ++y)
            for (int x = 0; x < nx; ++x) {
                const int64_t i = x + nx * (y + (int64_t)ny * z);
                nodes[3 * i] = x + 0.5 * rnd(); nodes[3 * i + 1] = y + 0.5 * rnd(); nodes[3 * i + 2] = z + 0.5 * rnd();
            }
    std::vector<double> pts, w;
    for (int z = 0; z < nz - 1; ++z)
        for (int y = 0; y < ny - 1; ++y)
            for (int x = 0; x < nx - 1; ++x) { pts.push_back(x + 0.5); pts.push_back(y + 0.5); pts.push_back(z + 0.5); w.push_back(1.0); }
    const int64_t M = (int64_t)w.size();
    std::vector<int32_t> sb(M * k), sg(M * k);
    if (orc_knn(nodes.data(), N, pts.data(), M, k, 0, sb.data()) || orc_knn(nodes.data(), N, pts.data(), M, k, 1, sg.data())) return 2;
    if (sb != sg) return 3;
    std::vector<int64_t> rp(3 * N + 1);
    orc_pattern_count(sg.data(), M, k, N, rp.data());
    std::vector<int64_t> ci(rp[3 * N]);
    if (orc_pattern_fill(sg.data(), M, k, N, rp.data(), ci.data())) return 4;
    std::vector<double> phi(M * k), dphi(M * 3 * k), phir(M * k), dphir(M * 3 * k);
    std::vector<uint8_t> sing(M);
    orc_shape(nodes.data(), pts.data(), sg.data(), M, k, 4.0, 1.0, 1.03, phi.data(), dphi.data(), sing.data());
    orc_shape_dense_ref(nodes.data(), pts.data(), sg.data(), M, k, 4.0, 1.0, 1.03, phir.data(), dphir.data());
    const double body[3] = {0.0, 0.0, -1.0};
    std::vector<double> vals(ci.size()), f(3 * N), valsr(ci.size()), fr(3 * N);
    int64_t ns = 0;
    if (orc_assemble(nodes.data(), pts.data(), w.data(), sg.data(), M, k, 1e9, 0.3, 4.0, 1.0, 1.03, body, 0, N, rp.data(), ci.data(),
                     vals.data(), f.data(), &ns)) return 5;
    if (orc_assemble_dense_ref(nodes.data(), pts.data(), w.data(), sg.data(), M, k, 1e9, 0.3, 4.0, 1.0, 1.03, body, 0, N, rp.data(),
                               ci.data(), valsr.data(), fr.data())) return 6;
    // a row slab as the full-size tests use it
    {
        const int64_t lo = 40, hi = 70;
        std::vector<int64_t> rps(3 * (hi - lo) + 1);
        for (size_t i = 0; i < rps.size(); ++i) rps[i] = rp[3 * lo + i] - rp[3 * lo];
        std::vector<double> v(rps.back()), ff(3 * (hi - lo));
        if (orc_assemble(nodes.data(), pts.data(), w.data(), sg.data(), M, k, 1e9, 0.3, 4.0, 1.0, 1.03, body, lo, hi, rps.data(),
                         ci.data() + rp[3 * lo], v.data(), ff.data(), &ns)) return 7;
    }
    const double t[3] = {0.0, 0.0, -1e3};
    orc_point_loads(nodes.data(), pts.data(), w.data(), t, sg.data(), 1, k, 4.0, 1.0, 1.03, f.data());
    std::vector<int64_t> bc = {0, 1, 2, N - 1};
    std::vector<uint8_t> mask = {7, 1, 2, 4};
    std::vector<double> ub(3 * bc.size(), 0.001);
    double used = 0.0;
    if (orc_penalty(bc.data(), mask.data(), ub.data(), (int64_t)bc.size(), 1e8, 1, N, rp.data(), ci.data(), vals.data(), f.data(), &used)) return 8;
    std::printf("sanitize ok nnz=%lld pow=%.17g alpha=%.6e\n", (long long)ci.size(), orc_pow_qm1(17.0, 1.03), used);
    return 0;
}
