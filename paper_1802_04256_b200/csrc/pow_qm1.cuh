// Reproducible power t^(q-1) on the device (R5): tables staged in shared memory,
// Horner coefficients read from the kernel-parameter constant bank.
#pragma once
#include "common.cuh"

struct PowSmem {
    double invc[32];
    double E[32];
    double F[128];
};

__device__ __forceinline__ void pow_smem_fill(PowSmem& T, const PowTables& src) {
    for (int i = threadIdx.x; i < 32; i += blockDim.x) { T.invc[i] = src.invc[i]; T.E[i] = src.E[i]; }
    for (int i = threadIdx.x; i < 128; i += blockDim.x) T.F[i] = src.F[i];
}

// b = the ten binomial-series coefficients (b[0] = 1)
__device__ __forceinline__ double pow_qm1(double t, const PowSmem& T, const double* __restrict__ b) {
    const long long bits = __double_as_longlong(t);
    const int e = (int)((unsigned long long)bits >> 52) - 1023;   // sign bit set -> e >= 1025
    if (e < -64 || e > 63) return __longlong_as_double(0x7ff8000000000000LL);
    const int i = (int)((bits >> 47) & 31);
    const double m = __longlong_as_double((bits & 0x000FFFFFFFFFFFFFLL) | 0x3FF0000000000000LL);
    const double r = fma(m, T.invc[i], -1.0);
    double p = b[9];
#pragma unroll
    for (int j = 8; j >= 0; --j) p = fma(p, r, b[j]);
    return (T.F[e + 64] * T.E[i]) * p;
}
