// Steps a5 + a6 (R8): w * B^T D B blocks and their deterministic reduction into the
// CSR values, body-force load; step a5b (R9) point loads; step a7 (R10) penalty BCs.
//
// Reduction design: ROW OWNER.  Block row I (node I) is owned by one group of warps; it walks the
// node's incidence list (points q whose support contains I, ascending q) and accumulates, for
// every column J of supp(q), S_IJ += (w g_I) (x) g_J.  Every CSR entry is therefore summed in
// ascending q by exactly one thread: no floating-point atomics, bitwise run-to-run reproducible,
// and K is written to HBM exactly once (never read).  The isotropic closed form
// K_IJ = lambda S + mu S^T + mu tr(S) I is applied once per block at write-out.
//
// reduce_rows_kernel (rows of up to 1024 block columns): the accumulators live in REGISTERS.
// Lane l of chunk c owns column slot 32 c + l of the row.  One resident wave of CTAs; every group
// of warps draws its next row from a ticket counter, so the rows in flight form one contiguous
// stripe.  For a batch of incident points one thread bulk-copies (cp.async.bulk + mbarrier) the
// points' staged [phi gx gy gz][k] rows into a double-buffered staging area, and every lane learns
// whether the point hits its slot and at which support position:
//   MASKED   from the slot masks precomputed with the pattern (pattern.cu): bit test, then
//            position = set bits before the chunk + popc(bits below the lane);
//   !MASKED  (masks over budget, e.g. config 5) from an open-addressing table column -> slot built
//            per row in shared memory and a byte table pos[point][slot] filled with one probe per
//            support node.
// A hit lane gathers that node's gradient (three doubles) from the staging area and does nine
// fused multiply-adds.
// accumulate_generic_kernel: fallback for longer rows, accumulators in shared memory.
#include "bulk_copy.cuh"
#include "common.cuh"

namespace {

constexpr unsigned FULLMASK = 0xffffffffu;

template <int NWARP>
__device__ __forceinline__ void group_sync(int rg) {
    if constexpr (NWARP == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(rg + 1), "r"(NWARP * 32) : "memory");
}

constexpr int ilog2_ce(int v) { return v <= 1 ? 0 : 1 + ilog2_ce(v >> 1); }

constexpr int RED_NB = 32;   // incident points per batch

// MASKED = false: slot lookup on the fly (hash table + byte table).  MASKED = true: the slot masks
// precomputed by rpim_stage_slot_masks (pattern.cu) are used instead.
template <int NWARP, int CPW, bool MASKED>
struct alignas(16) RedSmem {
    static constexpr int NW = NWARP * CPW;                 // 32-slot chunks of the row
    static constexpr int NS = 32 * NW;                     // column slots
    static constexpr int HLOG = ilog2_ce(4 * NS - 1);
    static constexpr int HSZ = 1 << HLOG;                  // open-addressing table: 2..4 x the row length
    unsigned long long hent[MASKED ? 2 : HSZ];             // (column node id << 32) | slot, ~0 = empty
    unsigned char pos[MASKED ? 1 : RED_NB][NS];            // position of slot's node in the support of point b, 0xFF = absent
    unsigned long long mp[MASKED ? RED_NB : 1][NW];        // (support positions before chunk c << 32) | slot mask of chunk c
    double a[RED_NB][4];                // w * grad phi_I at point b (+ pad)
    const double* qbase[RED_NB];        // staged shape functions of point b
    unsigned cmask[RED_NB];             // chunks of the row hit by point b
    unsigned long long full[2];         // mbarriers of the two staging buffers
    double fpart[NWARP];
    long long next_row[2];              // row handed to this group (two slots: written one row ahead of its last reader)
};

// Dynamic shared memory of one row group: RedSmem followed by the double-buffered gradient
// staging area G[2][nbg][k][4] (bulk-copied straight from the staged shape functions).
__host__ __device__ inline size_t red_group_bytes(size_t head, int k, int nbg) {
    return head + (size_t)2 * nbg * k * 4 * sizeof(double);
}

// NWARP warps own one block row, each CPW chunks of 32 column slots (chunk c = cc * NWARP + wg);
// a CTA holds ROWS such groups working on consecutive rows.
template <int NWARP, int CPW, int ROWS, bool MASKED>
__global__ void __launch_bounds__(NWARP * ROWS * 32)
reduce_rows_kernel(int64_t N, int k, int nbg, const int64_t* __restrict__ inc_ptr, const int32_t* __restrict__ inc_q,
                   const uint8_t* __restrict__ inc_j, const int32_t* __restrict__ support,
                   const double* __restrict__ stage, const double* __restrict__ qw, const double* __restrict__ escale,
                   const int64_t* __restrict__ brow_ptr, const int32_t* __restrict__ bcol,
                   const int64_t* __restrict__ mask_ptr, const unsigned* __restrict__ masks, int mask_stride,
                   unsigned long long* __restrict__ ticket, double lambda, double mu, double bx, double by, double bz, double* __restrict__ vals, double* __restrict__ f) {
    using S = RedSmem<NWARP, CPW, MASKED>;
    constexpr int NS = S::NS, HSZ = S::HSZ, GT = NWARP * 32;
    constexpr int HSHIFT = 32 - S::HLOG;
    extern __shared__ __align__(16) unsigned char red_smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rg = warp / NWARP, wg = warp % NWARP, tg = wg * 32 + lane;
    unsigned char* gbase = red_smem_raw + (size_t)rg * red_group_bytes(sizeof(S), k, nbg);
    S& sm = *reinterpret_cast<S*>(gbase);
    double* G = reinterpret_cast<double*>(gbase + sizeof(S));
    const int gstride = nbg * k * 4;            // doubles per staging buffer
    const unsigned pbytes = (unsigned)k * 32u;  // bytes of one point's staged row
    const int npass = (k + 31) >> 5;
    const unsigned lbit = 1u << lane, lt = lbit - 1u;
    if (tg == 0) { mbar_init(&sm.full[0], 1); mbar_init(&sm.full[1], 1); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    unsigned ph0 = 0, ph1 = 0;   // parity of the next completion of each staging buffer
    __syncthreads();

    // rows are handed out in ascending order from a global ticket: the resident groups always work on
    // one contiguous stripe of rows (their staged gradients are shared through L2) and stay balanced
    // (the ticket of the next row is drawn while the current row is processed: its latency is hidden)
    long long drawn = (tg == 0) ? (long long)atomicAdd(ticket, 1ull) : 0;
    for (unsigned it = 0;; ++it) {
        if (tg == 0) sm.next_row[it & 1] = drawn;
        group_sync<NWARP>(rg);   // ticket visible; the previous row's shared data is dead
        const int64_t I = sm.next_row[it & 1];
        if (I >= N) break;
        if (tg == 0) drawn = (long long)atomicAdd(ticket, 1ull);
        const int64_t o = brow_ptr[I];
        const int L = (int)(brow_ptr[I + 1] - o);
        if constexpr (!MASKED) {
            for (int s = tg; s < HSZ; s += GT) sm.hent[s] = ~0ull;
            group_sync<NWARP>(rg);
            for (int s = tg; s < L; s += GT) {
                const unsigned J = (unsigned)bcol[o + s];
                unsigned h = (J * 2654435761u) >> HSHIFT;
                const unsigned long long ent = ((unsigned long long)J << 32) | (unsigned)s;
                while (atomicCAS(&sm.hent[h], ~0ull, ent) != ~0ull) h = (h + 1) & (HSZ - 1);
            }
        }
        const int NWc = (L + 31) >> 5;   // mask words per incident point of this row
        const int mstep = mask_stride > 0 ? mask_stride : NWc;   // words from one incident point to the next
        const unsigned* mrow = !MASKED ? nullptr : (mask_stride > 0 ? masks + inc_ptr[I] * mask_stride : masks + mask_ptr[I]);
        double acc[CPW][9];
#pragma unroll
        for (int cc = 0; cc < CPW; ++cc)
#pragma unroll
            for (int e = 0; e < 9; ++e) acc[cc][e] = 0.0;
        double fsum = 0.0;
        const int64_t pa = inc_ptr[I], pb = inc_ptr[I + 1];
        for (int64_t p0 = pa; p0 < pb; p0 += RED_NB) {
            const int nb = (int)min((int64_t)RED_NB, pb - p0);
            const int nsub = (nb + nbg - 1) / nbg;
            group_sync<NWARP>(rg);   // previous batch fully consumed (pos, a, staging buffers); hash table complete
            // ---- phase 1a: per-point scalars (thread b of the group) and a clean position table
            if (tg < nb) {
                const int64_t p = p0 + tg;
                const int q = inc_q[p];
                const int i = inc_j[p];
                const double w = qw[q];
                const double* base = stage + (int64_t)q * k * 4;
                fsum += w * base[i];   // staged layout [q][phi, d/dx, d/dy, d/dz][k]
                const double wk = escale ? w * escale[q] : w;   // R8b: the stiffness weight carries the point's modulus scale
                sm.a[tg][0] = wk * base[k + i]; sm.a[tg][1] = wk * base[2 * k + i]; sm.a[tg][2] = wk * base[3 * k + i];
                sm.qbase[tg] = base;
                if constexpr (MASKED) {
                    const unsigned* mw = mrow + (p - pa) * mstep;
                    unsigned pre = 0;
                    for (int w = 0; w < NWc; ++w) {
                        const unsigned word = mw[w];
                        sm.mp[tg][w] = ((unsigned long long)pre << 32) | word;
                        pre += __popc(word);
                    }
                    for (int w = NWc; w < S::NW; ++w) sm.mp[tg][w] = 0ull;
                }
            }
            if constexpr (!MASKED) {
                uint4* pz = reinterpret_cast<uint4*>(&sm.pos[0][0]);
                const uint4 ff = make_uint4(0xffffffffu, 0xffffffffu, 0xffffffffu, 0xffffffffu);
                for (int e = tg; e < nb * (NS / 16); e += GT) pz[e] = ff;
            }
            group_sync<NWARP>(rg);   // qbase visible, table clean
            // gradient rows of sub-batch sb -> staging buffer sb & 1 (bulk copies issued by one thread)
            auto issue = [&](int sb) {
                const int b0 = sb * nbg, cnt = min(nbg, nb - b0);
                unsigned long long* bar = &sm.full[sb & 1];
                mbar_expect_tx(bar, (unsigned)cnt * pbytes);
                double* dstb = G + (sb & 1) * gstride;
                for (int bb = 0; bb < cnt; ++bb) bulk_g2s(dstb + bb * k * 4, sm.qbase[b0 + bb], pbytes, bar);
            };
            if (tg == 0) { issue(0); if (nsub > 1) issue(1); }
            // ---- phase 1b: positions of this warp's points b = wg, wg + NWARP, ... (overlaps the copies)
            if constexpr (!MASKED) {
                // support nodes of the next point are fetched while the current one is looked up
                // (k <= RPIM_MAX_K = 124: at most four passes of 32 lanes)
                auto fetch = [&](int b, int (&J)[4]) {
                    const int32_t* sp = support + (sm.qbase[min(b, nb - 1)] - stage) / 4;   // = support + q * k
#pragma unroll
                    for (int ps = 0; ps < 4; ++ps) {
                        const int j = ps * 32 + lane;
                        J[ps] = (b < nb && j < k) ? sp[j] : -1;
                    }
                };
                int Jc[4], Jn[4];
                fetch(wg, Jc);
                for (int b = wg; b < nb; b += NWARP) {
                    fetch(b + NWARP, Jn);
                    unsigned cm = 0;
#pragma unroll
                    for (int ps = 0; ps < 4; ++ps) {
                        if (ps >= npass) break;
                        unsigned wbit = 0;
                        if (Jc[ps] >= 0) {
                            const unsigned J = (unsigned)Jc[ps];
                            unsigned h = (J * 2654435761u) >> HSHIFT;
                            unsigned long long ent = sm.hent[h];
                            while ((unsigned)(ent >> 32) != J) { h = (h + 1) & (HSZ - 1); ent = sm.hent[h]; }
                            const unsigned slot = (unsigned)ent;
                            sm.pos[b][slot] = (unsigned char)(ps * 32 + lane);
                            wbit = 1u << (slot >> 5);
                        }
                        cm |= __reduce_or_sync(FULLMASK, wbit);
                    }
                    if (lane == 0) sm.cmask[b] = cm;
#pragma unroll
                    for (int ps = 0; ps < 4; ++ps) Jc[ps] = Jn[ps];
                }
            }
            // ---- phase 2: every lane accumulates its slots over the points, sub-batch by sub-batch
            for (int sb = 0; sb < nsub; ++sb) {
                group_sync<NWARP>(rg);   // positions visible (sb = 0); buffer (sb + 1) & 1 fully consumed (sb > 0)
                if (sb > 0 && sb + 1 < nsub && tg == 0) issue(sb + 1);
                if (sb & 1) { mbar_wait(&sm.full[1], ph1); ph1 ^= 1u; }
                else { mbar_wait(&sm.full[0], ph0); ph0 ^= 1u; }
                const int b0 = sb * nbg, cnt = min(nbg, nb - b0);
                const double* Gb = G + (sb & 1) * gstride;
                for (int bb = 0; bb < cnt; ++bb) {
                    const int b = b0 + bb;
                    const double ax = sm.a[b][0], ay = sm.a[b][1], az = sm.a[b][2];
                    const double* base = Gb + bb * k * 4;
                    if constexpr (MASKED) {
                        // all chunk words first (independent loads), then the hits; an empty chunk
                        // (word = 0, also every chunk beyond the row's length) is skipped by the whole warp
                        unsigned long long mpv[CPW];
#pragma unroll
                        for (int cc = 0; cc < CPW; ++cc) mpv[cc] = sm.mp[b][cc * NWARP + wg];
#pragma unroll
                        for (int cc = 0; cc < CPW; ++cc) {
                            const unsigned word = (unsigned)mpv[cc];
                            if (word & lbit) {
                                const unsigned j = (unsigned)(mpv[cc] >> 32) + __popc(word & lt);
                                const double gx = base[k + j], gy = base[2 * k + j], gz = base[3 * k + j];
                                acc[cc][0] = fma(ax, gx, acc[cc][0]); acc[cc][1] = fma(ax, gy, acc[cc][1]); acc[cc][2] = fma(ax, gz, acc[cc][2]);
                                acc[cc][3] = fma(ay, gx, acc[cc][3]); acc[cc][4] = fma(ay, gy, acc[cc][4]); acc[cc][5] = fma(ay, gz, acc[cc][5]);
                                acc[cc][6] = fma(az, gx, acc[cc][6]); acc[cc][7] = fma(az, gy, acc[cc][7]); acc[cc][8] = fma(az, gz, acc[cc][8]);
                            }
                        }
                    } else {
                        const unsigned cm = sm.cmask[b];
                        const unsigned char* prow = &sm.pos[b][lane];
#pragma unroll
                        for (int cc = 0; cc < CPW; ++cc) {
                            const int c = cc * NWARP + wg;
                            if (!((cm >> c) & 1u)) continue;
                            const unsigned j = prow[32 * c];
                            if (j != 0xFFu) {
                                const double gx = base[k + j], gy = base[2 * k + j], gz = base[3 * k + j];
                                acc[cc][0] = fma(ax, gx, acc[cc][0]); acc[cc][1] = fma(ax, gy, acc[cc][1]); acc[cc][2] = fma(ax, gz, acc[cc][2]);
                                acc[cc][3] = fma(ay, gx, acc[cc][3]); acc[cc][4] = fma(ay, gy, acc[cc][4]); acc[cc][5] = fma(ay, gz, acc[cc][5]);
                                acc[cc][6] = fma(az, gx, acc[cc][6]); acc[cc][7] = fma(az, gy, acc[cc][7]); acc[cc][8] = fma(az, gz, acc[cc][8]);
                            }
                        }
                    }
                }
            }
        }
        // ---- K_IJ = lambda S + mu S^T + mu tr(S) I, three scalar rows per block row
#pragma unroll
        for (int cc = 0; cc < CPW; ++cc) {
            const int s = 32 * (cc * NWARP + wg) + lane;
            if (s < L) {
                const double* a = acc[cc];
                const double mtr = mu * ((a[0] + a[4]) + a[8]);
#pragma unroll
                for (int r = 0; r < 3; ++r) {
                    double* dst = vals + 9 * o + (int64_t)r * 3 * L + 3 * s;
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        double v = fma(lambda, a[3 * r + c], mu * a[3 * c + r]);
                        if (r == c) v += mtr;
                        dst[c] = v;
                    }
                }
            }
        }
        // ---- body-force load: partial sums of the warps in a fixed order
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) fsum += __shfl_xor_sync(FULLMASK, fsum, d);
        if constexpr (NWARP > 1) {
            if (lane == 0) sm.fpart[wg] = fsum;
            group_sync<NWARP>(rg);
            fsum = 0.0;
#pragma unroll
            for (int w = 0; w < NWARP; ++w) fsum += sm.fpart[w];
        }
        if (wg == 0 && lane == 0) { f[3 * I] = fsum * bx; f[3 * I + 1] = fsum * by; f[3 * I + 2] = fsum * bz; }
    }
}

__global__ void __launch_bounds__(256)
accumulate_generic_kernel(int64_t N, int k, int Lcap, const int64_t* __restrict__ inc_ptr,
                          const int32_t* __restrict__ inc_q, const uint8_t* __restrict__ inc_j,
                          const int32_t* __restrict__ support, const double* __restrict__ stage,
                          const double* __restrict__ qw, const double* __restrict__ escale, const int64_t* __restrict__ brow_ptr,
                          const int32_t* __restrict__ bcol, double lambda, double mu, double bx, double by,
                          double bz, double* __restrict__ vals, double* __restrict__ f) {
    extern __shared__ double smem_d[];
    const int nwarps = blockDim.x >> 5;
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* acc = smem_d + (size_t)wid * ((size_t)Lcap * 9 + (Lcap + 1) / 2);
    int* cols = (int*)(acc + (size_t)Lcap * 9);

    for (int64_t I = (int64_t)blockIdx.x * nwarps + wid; I < N; I += (int64_t)gridDim.x * nwarps) {
        const int64_t o = brow_ptr[I];
        const int L = (int)(brow_ptr[I + 1] - o);
        for (int s = lane; s < L; s += 32) cols[s] = bcol[o + s];
        for (int s = lane; s < 9 * L; s += 32) acc[s] = 0.0;
        __syncwarp();
        double fI = 0.0;
        const int64_t pa = inc_ptr[I], pb = inc_ptr[I + 1];
        for (int64_t p = pa; p < pb; ++p) {
            const int64_t q = inc_q[p];
            const int i = inc_j[p];
            const double w = qw[q];
            const double* st = stage + q * 4 * (int64_t)k;
            const double wk = escale ? w * escale[q] : w;
            const double wgx = wk * st[k + i], wgy = wk * st[2 * k + i], wgz = wk * st[3 * k + i];
            fI += w * st[i];
            const int32_t* sp = support + q * k;
            for (int j = lane; j < k; j += 32) {
                const int J = sp[j];
                const double gx = st[k + j], gy = st[2 * k + j], gz = st[3 * k + j];
                int lo = 0, hi = L - 1;   // J is always present in the row
                while (lo < hi) {
                    const int mid = (lo + hi) >> 1;
                    if (cols[mid] < J) lo = mid + 1; else hi = mid;
                }
                double* a = acc + 9 * lo;
                a[0] = fma(wgx, gx, a[0]); a[1] = fma(wgx, gy, a[1]); a[2] = fma(wgx, gz, a[2]);
                a[3] = fma(wgy, gx, a[3]); a[4] = fma(wgy, gy, a[4]); a[5] = fma(wgy, gz, a[5]);
                a[6] = fma(wgz, gx, a[6]); a[7] = fma(wgz, gy, a[7]); a[8] = fma(wgz, gz, a[8]);
            }
            __syncwarp();
        }
        // K_IJ = lambda S + mu S^T + mu tr(S) I, written row by row (each scalar row is contiguous)
        for (int s = lane; s < L; s += 32) {
            const double* a = acc + 9 * s;
            const double mtr = mu * ((a[0] + a[4]) + a[8]);
#pragma unroll
            for (int r = 0; r < 3; ++r) {
                double* dst = vals + 9 * o + (int64_t)r * 3 * L + 3 * s;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    double v = fma(lambda, a[3 * r + c], mu * a[3 * c + r]);
                    if (r == c) v += mtr;
                    dst[c] = v;
                }
            }
        }
        if (lane == 0) { f[3 * I] = fI * bx; f[3 * I + 1] = fI * by; f[3 * I + 2] = fI * bz; }
        __syncwarp();
    }
}

// one warp, points in order: f_{3J+c} += (w phi_J) t_c  (deterministic; M is small: face points)
__global__ void point_loads_kernel(const int32_t* __restrict__ support, const double* __restrict__ stage,
                                   const double* __restrict__ w, const double* __restrict__ t, int64_t M, int k,
                                   double* __restrict__ f) {
    const int lane = threadIdx.x;
    for (int64_t p = 0; p < M; ++p) {
        const double* st = stage + p * 4 * (int64_t)k;
        const double wp = w[p], tx = t[3 * p], ty = t[3 * p + 1], tz = t[3 * p + 2];
        for (int j = lane; j < k; j += 32) {
            const int64_t J = support[p * k + j];
            const double wphi = wp * st[j];
            f[3 * J] += wphi * tx;
            f[3 * J + 1] += wphi * ty;
            f[3 * J + 2] += wphi * tz;
        }
        __syncwarp();
        __threadfence_block();
    }
}

// ------------------------------------------------------------------ penalty
__global__ void diag_max_partial_kernel(int64_t N, const int64_t* __restrict__ brow_ptr,
                                        const int* __restrict__ bdiag, const double* __restrict__ vals,
                                        double* __restrict__ part) {
    double m = 0.0;
    for (int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; I < N; I += (int64_t)gridDim.x * blockDim.x) {
        const int64_t o = brow_ptr[I];
        const int64_t L = brow_ptr[I + 1] - o;
        if (L == 0) continue;
        const int64_t d = bdiag[I];
#pragma unroll
        for (int a = 0; a < 3; ++a) m = fmax(m, vals[9 * o + a * 3 * L + 3 * d + a]);
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, d));
    __shared__ double s[32];
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x < 32) {
        m = (threadIdx.x < (blockDim.x >> 5)) ? s[threadIdx.x] : 0.0;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, d));
        if (threadIdx.x == 0) part[blockIdx.x] = m;
    }
}

__global__ void diag_max_final_kernel(double* part, int nparts, double alpha, int relative) {
    double m = 0.0;
    for (int b = threadIdx.x; b < nparts; b += 32) m = fmax(m, part[b]);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, d));
    __syncwarp();
    if (threadIdx.x == 0) part[0] = relative ? alpha * m : alpha;
}

// validity of the boundary list, before anything is applied: ids in range, with a matrix row, each listed once
// (seen = one bit per node, zeroed by the caller)
__global__ void penalty_check_kernel(int64_t N, const int64_t* __restrict__ bc_nodes, int64_t m,
                                     const int64_t* __restrict__ brow_ptr, unsigned* __restrict__ seen,
                                     long long* __restrict__ flags) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    const int64_t I = bc_nodes[i];
    bool bad = I < 0 || I >= N || brow_ptr[I + 1] == brow_ptr[I];
    if (!bad) bad = (atomicOr(&seen[I >> 5], 1u << (I & 31)) >> (I & 31)) & 1u;
    if (bad) atomicAdd((unsigned long long*)&flags[FLAG_BC_BAD], 1ull);
}

__global__ void penalty_apply_kernel(int64_t N, const int64_t* __restrict__ bc_nodes,
                                     const uint8_t* __restrict__ bc_mask, const double* __restrict__ ubar, int64_t m,
                                     const double* __restrict__ alpha_used, const int64_t* __restrict__ brow_ptr,
                                     const int* __restrict__ bdiag, double* __restrict__ vals, double* __restrict__ f,
                                     long long* __restrict__ flags) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    const int64_t I = bc_nodes[i];
    if (I < 0 || I >= N || brow_ptr[I + 1] == brow_ptr[I]) {
        atomicAdd((unsigned long long*)&flags[FLAG_BC_BAD], 1ull);
        return;
    }
    const double a = alpha_used[0];
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

static int accumulate_generic(rpim_ctx* ctx, const double* d_qw, double lambda, double mu, const double body[3],
                          double* d_vals, double* d_f) {
    const int Lcap = std::max(ctx->max_blen, 1);
    const size_t per_warp = ((size_t)Lcap * 9 + (Lcap + 1) / 2) * sizeof(double);
    int warps = 8;
    while (warps > 1 && per_warp * warps > 200 * 1024) --warps;
    if (per_warp * warps > 220 * 1024) RPIM_FAIL(ctx, RPIM_ERR_CAPACITY, "block row of %d columns does not fit on chip", Lcap);
    const size_t smem = per_warp * warps;
    CUDA_TRY(ctx, cudaFuncSetAttribute(accumulate_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int per_sm = (int)std::max<size_t>(1, (220 * 1024) / (smem + 1024));
    int64_t blocks = (ctx->N + warps - 1) / warps;
    blocks = std::min<int64_t>(blocks, 148LL * per_sm * 8);
    accumulate_generic_kernel<<<(unsigned)blocks, warps * 32, smem, ctx->stream>>>(
        ctx->N, ctx->k, Lcap, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_inc_j, ctx->d_support, ctx->d_stage, d_qw, ctx->d_escale,
        ctx->d_brow_ptr, ctx->d_bcol, lambda, mu, body[0], body[1], body[2], d_vals, d_f);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}

namespace {
template <int NWARP, int CPW, int ROWS, bool MASKED>
int launch_reduce_rows_m(rpim_ctx* ctx, const double* d_qw, double lambda, double mu, const double body[3],
                         double* d_vals, double* d_f) {
    auto kern = reduce_rows_kernel<NWARP, CPW, ROWS, MASKED>;
    // gradient staging: two buffers of nbg points each per row group.  Larger sub-batches mean fewer
    // group barriers; take the largest nbg (<= 8) that does not cost a resident CTA
    CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    int nbg = 2, per_sm = 1;
    size_t smem = red_group_bytes(sizeof(RedSmem<NWARP, CPW, MASKED>), ctx->k, nbg) * ROWS;
    if (smem > 227 * 1024) RPIM_FAIL(ctx, RPIM_ERR_CAPACITY, "k = %d does not fit the staging area of the reduction", ctx->k);
    CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NWARP * ROWS * 32, smem));
    if (per_sm < 1) per_sm = 1;
    for (int cand = 8; cand > 2; --cand) {
        const size_t sc = red_group_bytes(sizeof(RedSmem<NWARP, CPW, MASKED>), ctx->k, cand) * ROWS;
        int occ = 0;
        if (sc <= 227 * 1024 &&
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, NWARP * ROWS * 32, sc) == cudaSuccess && occ >= per_sm) {
            nbg = cand;
            smem = sc;
            break;
        }
    }
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->device);
    int64_t blocks = (ctx->N + ROWS - 1) / ROWS;
    // persistent: exactly one resident wave; its row groups draw rows from a ticket counter
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_flags + FLAG_ROW_TICKET, 0, sizeof(long long), ctx->stream));
    blocks = std::min<int64_t>(blocks, (int64_t)sms * per_sm);
    kern<<<(unsigned)blocks, NWARP * ROWS * 32, smem, ctx->stream>>>(
        ctx->N, ctx->k, nbg, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_inc_j, ctx->d_support, ctx->d_stage, d_qw, ctx->d_escale,
        ctx->d_brow_ptr, ctx->d_bcol, ctx->d_mask_ptr, ctx->d_masks, ctx->mask_stride,
        (unsigned long long*)(ctx->d_flags + FLAG_ROW_TICKET), lambda, mu, body[0], body[1], body[2], d_vals, d_f);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}
// precomputed slot masks when the pattern stage could afford them (pattern.cu), else on-the-fly lookup
template <int NWARP, int CPW, int ROWS>
int launch_reduce_rows(rpim_ctx* ctx, const double* d_qw, double lambda, double mu, const double body[3],
                       double* d_vals, double* d_f) {
    return ctx->have_masks ? launch_reduce_rows_m<NWARP, CPW, ROWS, true>(ctx, d_qw, lambda, mu, body, d_vals, d_f)
                           : launch_reduce_rows_m<NWARP, CPW, ROWS, false>(ctx, d_qw, lambda, mu, body, d_vals, d_f);
}
}  // namespace

int rpim_stage_accumulate(rpim_ctx* ctx, const double* d_qw, double lambda, double mu, const double body[3],
                          double* d_vals, double* d_f) {
    const int Lmax = std::max(ctx->max_blen, 1);
    if (ctx->reduce_mode == 3) return accumulate_generic(ctx, d_qw, lambda, mu, body, d_vals, d_f);
    static_assert(sizeof(RedSmem<1, 4, false>) % 16 == 0 && sizeof(RedSmem<8, 4, true>) % 16 == 0 && sizeof(RedSmem<2, 3, true>) % 16 == 0, "group stride keeps 16-byte alignment");
    if (Lmax <= 128) return launch_reduce_rows<1, 4, 8>(ctx, d_qw, lambda, mu, body, d_vals, d_f);
    if (Lmax <= 192) return launch_reduce_rows<2, 3, 4>(ctx, d_qw, lambda, mu, body, d_vals, d_f);
    if (Lmax <= 256) return launch_reduce_rows<2, 4, 4>(ctx, d_qw, lambda, mu, body, d_vals, d_f);
    if (Lmax <= 384) return launch_reduce_rows<4, 3, 2>(ctx, d_qw, lambda, mu, body, d_vals, d_f);
    if (Lmax <= 512) return launch_reduce_rows<4, 4, 2>(ctx, d_qw, lambda, mu, body, d_vals, d_f);
    if (Lmax <= 768) return launch_reduce_rows<8, 3, 1>(ctx, d_qw, lambda, mu, body, d_vals, d_f);
    if (Lmax <= 1024) return launch_reduce_rows<8, 4, 1>(ctx, d_qw, lambda, mu, body, d_vals, d_f);
    return accumulate_generic(ctx, d_qw, lambda, mu, body, d_vals, d_f);
}

int rpim_stage_point_loads(rpim_ctx* ctx, const int32_t* d_support, const double* d_stage, const double* d_w,
                           const double* d_t, int64_t M, double* d_f) {
    if (M == 0) return RPIM_OK;
    point_loads_kernel<<<1, 32, 0, ctx->stream>>>(d_support, d_stage, d_w, d_t, M, ctx->k, d_f);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}

int rpim_stage_penalty(rpim_ctx* ctx, const int64_t* d_bc_nodes, const uint8_t* d_bc_mask, const double* d_u_bar,
                       int64_t m, double alpha, int relative, double* d_vals, double* d_f, double* out_alpha) {
    cudaStream_t st = ctx->stream;
    const int nparts = 592;
    diag_max_partial_kernel<<<nparts, 256, 0, st>>>(ctx->N, ctx->d_brow_ptr, ctx->d_bdiag, d_vals, ctx->d_scratch);
    KERNEL_CHECK(ctx);
    diag_max_final_kernel<<<1, 32, 0, st>>>(ctx->d_scratch, nparts, alpha, relative);
    KERNEL_CHECK(ctx);
    double a = 0.0;
    long long bad = 0;
    if (m > 0) {
        // the list is validated first: nothing is applied unless every id is in range, has a row and is unique
        unsigned* d_seen = nullptr;
        const int64_t words = (ctx->N + 31) / 32;
        int rc = ws_alloc(ctx, &d_seen, words);
        if (rc) return rc;
        cudaError_t e = cudaMemsetAsync(d_seen, 0, (size_t)words * sizeof(unsigned), st);
        if (e == cudaSuccess) {
            penalty_check_kernel<<<(unsigned)((m + 127) / 128), 128, 0, st>>>(ctx->N, d_bc_nodes, m, ctx->d_brow_ptr, d_seen,
                                                                              ctx->d_flags);
            ctx->launches++;
            e = cudaGetLastError();
        }
        ws_free(ctx, &d_seen);   // parked: reuse is ordered by the stream
        if (e != cudaSuccess) RPIM_FAIL(ctx, RPIM_ERR_CUDA, "boundary list check failed: %s", cudaGetErrorString(e));
    }
    CUDA_TRY(ctx, cudaMemcpyAsync(&a, ctx->d_scratch, sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaMemcpyAsync(&bad, ctx->d_flags + FLAG_BC_BAD, sizeof(long long), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    if (out_alpha) *out_alpha = a;
    if (bad) {
        CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_flags + FLAG_BC_BAD, 0, sizeof(long long), st));
        RPIM_FAIL(ctx, RPIM_ERR_BC_NODE_INVALID,
                  "%lld boundary node ids are out of range, listed more than once or have no matrix row; nothing applied", bad);
    }
    if (m > 0) {
        penalty_apply_kernel<<<(unsigned)((m + 127) / 128), 128, 0, st>>>(ctx->N, d_bc_nodes, d_bc_mask, d_u_bar, m,
                                                                          ctx->d_scratch, ctx->d_brow_ptr,
                                                                          ctx->d_bdiag, d_vals, d_f, ctx->d_flags);
        KERNEL_CHECK(ctx);
    }
    return RPIM_OK;
}
