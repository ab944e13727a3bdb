// Steps a5 + a6 (R8), PANEL form: w * B^T D B blocks reduced deterministically into the CSR
// values, for quadrature points that come in groups with overlapping supports (several Gauss points per
// background cell, or neighbouring cells).  Integer preprocessing: groups.cu.
//
// K is symmetric block-wise (K_JI = K_IJ^T, R8: one support per point), so only the UPPER blocks
// (column node J >= row node I) are accumulated; mirror_lower_kernel then fills the lower blocks with the
// transposes.  Half the arithmetic, half the on-chip accumulators (twice the rows per tile).
//
// A CTA owns a TILE of T = R RP consecutive block rows at a time (tiles strided over a persistent grid).
// The accumulators S_IJ of their upper blocks (nine doubles per block column) live in SHARED memory, next to
// each row's upper column list and a 16-bit open-addressing table column node -> slot.  The point groups
// incident to the tile arrive through a ring of NSTAGE shared-memory stages filled by a PRODUCER warp with
// TWO requests per group (mbarrier completion): the gradient rows of the group's eight consecutive points as
// one 2-D tensor copy (TMA: box 8 points x 3 k doubles of the [point][4 k] staged array) or, when that does
// not buy ring depth or 24 k bytes is no 16-byte multiple, their whole staged rows as one plain bulk copy;
// and the group's record (its sorted union of supports U_g, the map (union entry, point) -> support position,
// the quadrature weights) as one plain bulk copy.  The copy engine has a per-request cost: few large
// requests, not one per point.  Row group rp (R = 1: one block row; R = 2: a pair that shares the gradient
// loads) has CW consumer warps; the chunks of 32 union entries from the one that holds the rows' own nodes
// upwards (U_g is ascending: everything below is a lower block) are dealt to them round-robin.  In a chunk a
// lane owns one union entry and sums (w grad phi_I) (x) grad phi_{U_g[u]} over the group's points IN REGISTERS
// (dense: |U_g| is 1.3 .. 1.6 k), then adds its nine sums per row to the row's accumulator of that column:
// one table probe and one read-modify-write per (row, group, column) instead of per (row, point, column).
// The CW warps of a row group meet at a named barrier between their read-modify-write phases of consecutive
// groups; nothing else synchronises in the steady state, and the producer runs ahead across tile
// boundaries.  Every CSR entry is summed in a fixed order (points ascending inside a group, groups
// ascending) by one lane: no floating-point atomics, bitwise run-to-run reproducible and independent of the
// launch shape; every entry of K is written once, with the isotropic closed form
// K_IJ = lambda S + mu S^T + mu tr(S) I applied at write-out.
// The body-force load f_I = b sum_q w phi_I(q) is a separate row-owner pass over the incidence lists.
#include <cuda.h>

#include "bulk_copy.cuh"
#include "common.cuh"

namespace {

constexpr int GB = RPIM_GROUP_POINTS;
constexpr unsigned FULLMASK = 0xffffffffu;

__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// predicated shared-memory load: 0.0 when `on` is false (no branch, no access)
__device__ __forceinline__ double lds_f64_if(unsigned addr, bool on) {
    double v = 0.0;
    asm("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %2, 0;\n\t@q ld.shared.f64 %0, [%1];\n\t}" : "+d"(v) : "r"(addr), "r"((int)on));
    return v;
}
__device__ __forceinline__ void named_bar(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

struct PanelArgs {
    int64_t N, Nq, ntiles;
    int k, C, hlog, nstage;
    const int64_t* brow_ptr;
    const int32_t* bcol;
    const int* bdiag;
    const double* stage;
    const unsigned char* gmeta;
    const int64_t* tile_ptr;
    const unsigned* tdesc;
    double lambda, mu;
    double* vals;
    PanelSmem L;
    int grad_only;               // 1: the staged rows travel through `tmap` (gradient rows only), 0: plain bulk copy of whole rows
    alignas(64) CUtensorMap tmap;   // staged array as [point][4 k] doubles, box = 8 points x 3 k doubles
};

// 2-D tensor copy (TMA) global -> shared, completion on an mbarrier
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, unsigned long long* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(smem_u32(dst)), "l"(reinterpret_cast<unsigned long long>(map)), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}

// quadrature weights of every group into the group's record (once per rpim_assemble: the weights are its input)
// (times the point's modulus scale of DESIGN.md R8b when there is one: the record's weights only feed the stiffness)
__global__ void panel_weights_kernel(int64_t Nq, int64_t G, unsigned meta_bytes, unsigned off_w, const double* __restrict__ qw,
                                     const double* __restrict__ escale, unsigned char* __restrict__ gmeta) {
    const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= G * GB) return;
    double w = 0.0;
    if (q < Nq) w = escale ? qw[q] * escale[q] : qw[q];
    reinterpret_cast<double*>(gmeta + (q / GB) * meta_bytes + off_w)[q % GB] = w;
}

// R = block rows per consumer warp (2: a row pair shares the gradient loads; 1: twice the warps), RP = row groups
template <int CW, int RP, int R>
__global__ void __launch_bounds__((RP * CW + 1) * 32, 1)
reduce_panels_kernel(const __grid_constant__ PanelArgs A) {
    constexpr int T = R * RP, NCW = RP * CW, NCT = NCW * 32, DW = 1 + T / 2;
    constexpr int AWS = 6 * GB;   // doubles of one warp's a-vectors: [p][ax0 ay0 az0 ax1 ay1 az1]
    extern __shared__ __align__(128) unsigned char panel_smem[];
    const PanelSmem& L = A.L;
    double* acc = reinterpret_cast<double*>(panel_smem + L.off_acc);                    // [T][LS][9]
    int* bcol_s = reinterpret_cast<int*>(panel_smem + L.off_bcol);                      // [T][LS]
    unsigned short* hash_s = reinterpret_cast<unsigned short*>(panel_smem + L.off_hash);   // [T][HSZ]
    double* aw_s = reinterpret_cast<double*>(panel_smem + L.off_aw);                    // [NCW][AWS]
    unsigned char* stages = panel_smem + L.off_stage;
    unsigned long long* full = reinterpret_cast<unsigned long long*>(panel_smem + L.off_bar);
    unsigned long long* empty = full + A.nstage;
    long long* rowo_s = reinterpret_cast<long long*>(panel_smem + L.off_rowo);          // [T] first block of the row
    int* rowL_s = reinterpret_cast<int*>(panel_smem + L.off_rowo + 8 * T);              // [T] block columns of the row
    int* rowd_s = rowL_s + T;                                                           // [T] slot of the diagonal block

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int k = A.k, C = A.C, LS = L.LS, HSZ = 1 << A.hlog, hshift = 32 - A.hlog, nstage = A.nstage;
    // stage: [the group's staged rows: GB x 4 x k doubles][group record: jinv, union ids, weights][desc: 8 words]
    const unsigned gcap = 32u * C, meta = gcap * 12u + GB * 8u;
    const unsigned prow8 = (unsigned)(A.grad_only ? 3 : 4) * (unsigned)k * 8u;   // bytes of a point's rows inside a stage
    const unsigned goff8 = A.grad_only ? 0u : (unsigned)k * 8u;                    // its d/dx row starts here
    const unsigned gbytes = GB * prow8, off_desc = gbytes + meta, stage_bytes = L.stage_bytes;
    const unsigned k8 = (unsigned)k * 8u;

    if (tid == 0) {
        for (int s = 0; s < nstage; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NCW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NCW) {
        // ------------------------------------------------------------------ producer warp
        int s = 0;
        unsigned par = 1u;
        for (int64_t tile = blockIdx.x; tile < A.ntiles; tile += gridDim.x) {
            const int64_t t0 = A.tile_ptr[tile];
            const int ng = (int)(A.tile_ptr[tile + 1] - t0);
            for (int it0 = 0; it0 < ng; it0 += 32) {
                const int cnt = min(32, ng - it0);
                unsigned dsc[DW];
#pragma unroll
                for (int w = 0; w < DW; ++w) dsc[w] = (lane < cnt) ? A.tdesc[(t0 + it0 + lane) * DW + w] : 0u;
                for (int i = 0; i < cnt; ++i) {
                    unsigned mine = 0;   // lane w < DW takes word w of descriptor i
#pragma unroll
                    for (int w = 0; w < DW; ++w) {
                        const unsigned v = __shfl_sync(FULLMASK, dsc[w], i);
                        if (lane == w) mine = v;
                    }
                    const int64_t g = __shfl_sync(FULLMASK, mine, 0);
                    unsigned char* st = stages + (unsigned)s * stage_bytes;
                    mbar_wait(&empty[s], par);
                    if (lane < DW) reinterpret_cast<unsigned*>(st + off_desc)[lane] = mine;
                    __syncwarp();
                    if (lane == 0) {
                        mbar_expect_tx(&full[s], gbytes + meta);
                        if (A.grad_only) tma_load_2d(st, &A.tmap, k, (int)(g * GB), &full[s]);
                        else bulk_g2s(st, A.stage + g * (GB * 4) * k, gbytes, &full[s]);
                        bulk_g2s(st + gbytes, A.gmeta + g * meta, meta, &full[s]);
                    }
                    if (++s == nstage) { s = 0; par ^= 1u; }
                }
            }
        }
        return;
    }

    // ---------------------------------------------------------------------- consumer warps
    const int rp = warp / CW, w = warp % CW;
    const int r0 = R * rp, r1 = r0 + (R - 1);   // (R = 1: the second row is the first; its half of the code is compiled out)
    double* aw = aw_s + warp * AWS;
    double* acc0 = acc + (size_t)r0 * 9 * LS;
    double* acc1 = acc + (size_t)r1 * 9 * LS;
    const unsigned short* hash0 = hash_s + (size_t)r0 * HSZ;
    const unsigned short* hash1 = hash_s + (size_t)r1 * HSZ;
    const int* bcol0 = bcol_s + (size_t)r0 * LS;
    const int* bcol1 = bcol_s + (size_t)r1 * LS;
    int s = 0;
    unsigned par = 0u;

    for (int64_t tile = blockIdx.x; tile < A.ntiles; tile += gridDim.x) {
        named_bar(1, NCT);   // the previous tile's write-out has read its accumulators
        if (tid < T) {
            const int64_t I = tile * T + tid;
            int64_t o = 0;
            int Lr = 0, d = 0;
            if (I < A.N) { o = A.brow_ptr[I]; Lr = (int)(A.brow_ptr[I + 1] - o); d = Lr ? A.bdiag[I] : 0; }
            rowo_s[tid] = o;
            rowL_s[tid] = Lr;
            rowd_s[tid] = d;
        }
        {
            double2* z = reinterpret_cast<double2*>(acc);
            const double2 zz = make_double2(0.0, 0.0);
            for (int i = tid; i < T * 9 * LS / 2; i += NCT) z[i] = zz;
            unsigned* hz = reinterpret_cast<unsigned*>(hash_s);
            for (int i = tid; i < T * HSZ / 2; i += NCT) hz[i] = 0xFFFFFFFFu;
        }
        named_bar(1, NCT);
        // upper column lists (from the diagonal on) and tables: the CW warps of a row pair fill the pair's two rows
#pragma unroll
        for (int rr = 0; rr < R; ++rr) {
            const int r = r0 + rr;
            const int64_t o_r = rowo_s[r] + rowd_s[r];
            const int Lu = rowL_s[r] - rowd_s[r];
            unsigned short* hw = hash_s + (size_t)r * HSZ;
            int* bc = bcol_s + (size_t)r * LS;
            for (int sl = w * 32 + lane; sl < Lu; sl += CW * 32) {
                const unsigned J = (unsigned)A.bcol[o_r + sl];
                bc[sl] = (int)J;
                unsigned h = (J * 2654435761u) >> hshift;
                while (atomicCAS(&hw[h], (unsigned short)0xFFFFu, (unsigned short)sl) != (unsigned short)0xFFFFu) h = (h + 1) & (HSZ - 1);
            }
        }
        named_bar(1, NCT);
        const int I0 = (int)(tile * T) + r0, I1 = I0 + 1;
        const int ng = (int)(A.tile_ptr[tile + 1] - A.tile_ptr[tile]);
        for (int it = 0; it < ng; ++it) {
            const unsigned char* st = stages + (unsigned)s * stage_bytes;
            mbar_wait(&full[s], par);
            // descriptor word 1 + r / 2 holds rows r (low half, r even) and r + 1 (high half)
            unsigned dw = reinterpret_cast<const unsigned*>(st + off_desc)[1 + (r0 >> 1)];
            if (R == 1 && (r0 & 1)) dw >>= 16;
            const unsigned u0 = dw & 0xFFu, m0 = (dw >> 8) & 0xFFu, u1 = (R == 2) ? (dw >> 16) & 0xFFu : 0u, m1 = (R == 2) ? dw >> 24 : 0u;
            const unsigned mm = m0 | m1;
            if (mm != 0u) {
                const unsigned long long* jinv = reinterpret_cast<const unsigned long long*>(st + gbytes);
                const int* un = reinterpret_cast<const int*>(st + gbytes + gcap * 8u);
                // w * grad phi_I of the two rows' nodes at the group's points: lane p + 8 rr (zero when the
                // point does not hold the row's node)
                if (lane < R * GB) {
                    const int p = lane & (GB - 1), rr = lane >> 3;
                    const unsigned ur = rr ? u1 : u0, mr = rr ? m1 : m0;
                    double ax = 0.0, ay = 0.0, az = 0.0;
                    if ((mr >> p) & 1u) {
                        const unsigned j = (unsigned)(jinv[ur] >> (8 * p)) & 0xFFu;
                        const double wq = reinterpret_cast<const double*>(st + gbytes + gcap * 12u)[p];
                        const double* gp = reinterpret_cast<const double*>(st + (unsigned)p * prow8 + goff8) + j;
                        ax = wq * gp[0]; ay = wq * gp[k]; az = wq * gp[2 * k];
                    }
                    double* dst = aw + p * 6 + rr * 3;
                    dst[0] = ax; dst[1] = ay; dst[2] = az;
                }
                __syncwarp();
                // U_g ascends: the upper blocks start in the chunk that holds the rows' own nodes
                const int Ilow = m0 ? I0 : I1;
                bool met = false;
                for (int cc = (int)((m0 ? u0 : u1) >> 5) + w; cc < C; cc += CW) {
                    const int u = 32 * cc + lane;
                    const int J = un[u];
                    if (__ballot_sync(FULLMASK, J >= Ilow) == 0u) break;   // (padding: -1)
                    const unsigned long long jv = jinv[u];
                    const unsigned jlo = (unsigned)jv, jhi = (unsigned)(jv >> 32);
                    const unsigned st_u32 = smem_u32(st);
                    double s0[9], s1[9];
#pragma unroll
                    for (int p = 0; p < GB; ++p) {
                        const unsigned jb = ((p < 4 ? jlo : jhi) >> (8 * (p & 3))) & 0xFFu;
                        // a union entry the point does not hold (0xFF) contributes zeros: predicated loads
                        const bool have = jb != 0xFFu;
                        const unsigned gq = st_u32 + ((unsigned)p * prow8 + goff8) + jb * 8u;
                        const double gx = lds_f64_if(gq, have), gy = lds_f64_if(gq + k8, have), gz = lds_f64_if(gq + 2 * k8, have);
                        const double2 a01 = *reinterpret_cast<const double2*>(aw + p * 6);       // ax0 ay0
                        const double2 a23 = *reinterpret_cast<const double2*>(aw + p * 6 + 2);   // az0 ax1
                        double2 a45 = make_double2(0.0, 0.0);
                        if constexpr (R == 2) a45 = *reinterpret_cast<const double2*>(aw + p * 6 + 4);   // ay1 az1
                        if (p == 0) {
                            s0[0] = a01.x * gx; s0[1] = a01.x * gy; s0[2] = a01.x * gz;
                            s0[3] = a01.y * gx; s0[4] = a01.y * gy; s0[5] = a01.y * gz;
                            s0[6] = a23.x * gx; s0[7] = a23.x * gy; s0[8] = a23.x * gz;
                            if constexpr (R == 2) {
                                s1[0] = a23.y * gx; s1[1] = a23.y * gy; s1[2] = a23.y * gz;
                                s1[3] = a45.x * gx; s1[4] = a45.x * gy; s1[5] = a45.x * gz;
                                s1[6] = a45.y * gx; s1[7] = a45.y * gy; s1[8] = a45.y * gz;
                            }
                        } else {
                            s0[0] = fma(a01.x, gx, s0[0]); s0[1] = fma(a01.x, gy, s0[1]); s0[2] = fma(a01.x, gz, s0[2]);
                            s0[3] = fma(a01.y, gx, s0[3]); s0[4] = fma(a01.y, gy, s0[4]); s0[5] = fma(a01.y, gz, s0[5]);
                            s0[6] = fma(a23.x, gx, s0[6]); s0[7] = fma(a23.x, gy, s0[7]); s0[8] = fma(a23.x, gz, s0[8]);
                            if constexpr (R == 2) {
                                s1[0] = fma(a23.y, gx, s1[0]); s1[1] = fma(a23.y, gy, s1[1]); s1[2] = fma(a23.y, gz, s1[2]);
                                s1[3] = fma(a45.x, gx, s1[3]); s1[4] = fma(a45.x, gy, s1[4]); s1[5] = fma(a45.x, gz, s1[5]);
                                s1[6] = fma(a45.y, gx, s1[6]); s1[7] = fma(a45.y, gy, s1[7]); s1[8] = fma(a45.y, gz, s1[8]);
                            }
                        }
                    }
                    // column slots: the entry (I, U_g[u]) exists iff some point holds both nodes; a pair without
                    // an entry has only zero sums and is skipped
                    int slot0 = -1, slot1 = -1;
                    const unsigned h00 = ((unsigned)J * 2654435761u) >> hshift;
                    if (m0 && J >= I0) {
                        unsigned h = h00;
                        while (true) {
                            const unsigned sl = hash0[h];
                            if (sl == 0xFFFFu) break;
                            if (bcol0[sl] == J) { slot0 = (int)sl; break; }
                            h = (h + 1) & (HSZ - 1);
                        }
                    }
                    if (R == 2 && m1 && J >= I1) {
                        unsigned h = h00;
                        while (true) {
                            const unsigned sl = hash1[h];
                            if (sl == 0xFFFFu) break;
                            if (bcol1[sl] == J) { slot1 = (int)sl; break; }
                            h = (h + 1) & (HSZ - 1);
                        }
                    }
                    // read-modify-write phases of consecutive groups are separated for the CW warps of the row pair
                    if (CW > 1 && !met) { named_bar(2 + rp, CW * 32); met = true; }
                    if (slot0 >= 0) {
                        double* a = acc0 + slot0 * 9;
#pragma unroll
                        for (int e = 0; e < 9; ++e) a[e] += s0[e];
                    }
                    if (R == 2 && slot1 >= 0) {
                        double* a = acc1 + slot1 * 9;
#pragma unroll
                        for (int e = 0; e < 9; ++e) a[e] += s1[e];
                    }
                }
                if (CW > 1 && !met) named_bar(2 + rp, CW * 32);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);   // the stage (and this warp's a-vectors) are no longer read
            if (++s == nstage) { s = 0; par ^= 1u; }
        }
        named_bar(1, NCT);   // every contribution is in the accumulators
        // ---- upper blocks K_IJ = lambda S + mu S^T + mu tr(S) I: per block row three contiguous pieces
        for (int r = 0; r < T; ++r) {
            const int Lr = rowL_s[r];
            if (Lr == 0) continue;
            const int d = rowd_s[r];
            const double* ar = acc + (size_t)r * 9 * LS;
            double* dst = A.vals + 9 * rowo_s[r] + 3 * d;
            const int L3 = 3 * Lr, U3 = 3 * (Lr - d);
#pragma unroll
            for (int row = 0; row < 3; ++row) {
                for (int col = tid; col < U3; col += NCT) {
                    const int sl = (int)(((unsigned)col * 43691u) >> 17);   // col / 3 for col < 2^15 (columns <= 3 * 1024)
                    const int cc = col - 3 * sl;
                    const double* a = ar + sl * 9;
                    double v = fma(A.lambda, a[3 * row + cc], A.mu * a[3 * cc + row]);
                    if (row == cc) v += A.mu * ((a[0] + a[4]) + a[8]);
                    __stcs(dst + (size_t)row * L3 + col, v);   // streaming: K is not read again by this kernel, the groups' staged rows are
                }
            }
        }
    }
}

// Lower blocks: K_IJ = K_JI^T for J < I.  One warp per block row; a lane takes a lower slot, finds the slot of I
// in row J by bisection of that row's ascending column list and copies the transposed block.
__global__ void __launch_bounds__(256)
mirror_lower_kernel(int64_t N, const int64_t* __restrict__ brow_ptr, const int32_t* __restrict__ bcol,
                    const int* __restrict__ bdiag, double* __restrict__ vals) {
    const int lane = threadIdx.x & 31;
    const int64_t I = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (I >= N) return;
    const int64_t o = brow_ptr[I];
    const int L = (int)(brow_ptr[I + 1] - o);
    if (L == 0) return;
    const int d = bdiag[I];
    for (int s = lane; s < d; s += 32) {
        const int64_t J = bcol[o + s];
        const int64_t oj = brow_ptr[J];
        const int Lj = (int)(brow_ptr[J + 1] - oj);
        int lo = bdiag[J] + 1, hi = Lj - 1;   // I > J sits right of row J's diagonal
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (bcol[oj + mid] < (int)I) lo = mid + 1; else hi = mid;
        }
        const double* src = vals + 9 * oj + 3 * lo;
        double* dst = vals + 9 * o + 3 * s;
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c) dst[(size_t)r * 3 * L + c] = src[(size_t)c * 3 * Lj + r];
    }
}

// f_I = b * sum over the incident points (ascending) of w phi_I: one warp per block row, lane-strided
// partial sums combined in a fixed order (bitwise reproducible)
__global__ void __launch_bounds__(256)
load_rows_kernel(int64_t N, int k, const int64_t* __restrict__ inc_ptr, const int32_t* __restrict__ inc_q,
                 const uint8_t* __restrict__ inc_j, const double* __restrict__ stage, const double* __restrict__ qw,
                 double bx, double by, double bz, double* __restrict__ f) {
    const int lane = threadIdx.x & 31;
    const int64_t I = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (I >= N) return;
    const int64_t pa = inc_ptr[I], pb = inc_ptr[I + 1];
    double sum = 0.0;
    for (int64_t p = pa + lane; p < pb; p += 32) {
        const int64_t q = inc_q[p];
        sum += qw[q] * stage[q * 4 * k + inc_j[p]];
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) sum += __shfl_xor_sync(FULLMASK, sum, d);
    if (lane == 0) { f[3 * I] = sum * bx; f[3 * I + 1] = sum * by; f[3 * I + 2] = sum * bz; }
}

template <int CW, int RP, int R>
int launch_panels(rpim_ctx* ctx, PanelArgs& A) {
    auto kern = reduce_panels_kernel<CW, RP, R>;
    const size_t smem = A.L.total;
    CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 1, sms = 148;
    CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, (RP * CW + 1) * 32, smem));
    if (per_sm < 1) RPIM_FAIL(ctx, RPIM_ERR_CAPACITY, "panel reduction does not fit on chip (rows of %d upper block columns)", ctx->max_ulen);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->device);
    const int64_t blocks = std::min<int64_t>(A.ntiles, (int64_t)sms * per_sm);
    kern<<<(unsigned)blocks, (RP * CW + 1) * 32, smem, ctx->stream>>>(A);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}

}  // namespace

int rpim_stage_accumulate_panels(rpim_ctx* ctx, const double* d_qw, double lambda, double mu, const double body[3],
                                 double* d_vals, double* d_f) {
    PanelArgs A;
    A.N = ctx->N; A.Nq = ctx->Nq; A.ntiles = ctx->ntiles;
    A.k = ctx->k; A.C = ctx->tg_C;
    A.L = rpim_panel_smem(ctx->tg_C, ctx->tg_CW, ctx->tg_R, ctx->tg_T, ctx->k, std::max(ctx->max_ulen, 1), ctx->tg_nstage, ctx->tg_grad_only);
    A.hlog = A.L.hlog; A.nstage = ctx->tg_nstage;
    A.brow_ptr = ctx->d_brow_ptr; A.bcol = ctx->d_bcol; A.bdiag = ctx->d_bdiag; A.stage = ctx->d_stage;
    A.gmeta = ctx->d_gmeta;
    A.tile_ptr = ctx->d_tile_ptr; A.tdesc = ctx->d_tdesc;
    A.lambda = lambda; A.mu = mu; A.vals = d_vals;
    const int64_t G = (ctx->Nq + GB - 1) / GB;
    A.grad_only = 0;
    memset(&A.tmap, 0, sizeof(A.tmap));
    if (ctx->tg_grad_only) {
        // the staged array as a 2-D tensor [8 G points][4 k doubles]; a box is 8 points x the 3 k gradient doubles
        typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                      const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                      CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
            qres != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            RPIM_FAIL(ctx, RPIM_ERR_CUDA, "cuTensorMapEncodeTiled is not available from this driver");
        }
        const cuuint64_t dims[2] = {(cuuint64_t)(4 * ctx->k), (cuuint64_t)(G * GB)};
        const cuuint64_t strides[1] = {(cuuint64_t)(4 * ctx->k) * 8u};
        const cuuint32_t box[2] = {(cuuint32_t)(3 * ctx->k), (cuuint32_t)GB};
        const cuuint32_t estr[2] = {1u, 1u};
        const CUresult cr = ((encode_fn)fn)(&A.tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)ctx->d_stage, dims, strides, box, estr,
                                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (cr != CUDA_SUCCESS) RPIM_FAIL(ctx, RPIM_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d)", (int)cr);
        A.grad_only = 1;
    }
    const unsigned meta = rpim_panel_meta_bytes(ctx->tg_C);
    panel_weights_kernel<<<(unsigned)((G * GB + 255) / 256), 256, 0, ctx->stream>>>(ctx->Nq, G, meta, 32u * ctx->tg_C * 12u, d_qw, ctx->d_escale, ctx->d_gmeta);
    KERNEL_CHECK(ctx);
    const int wpb = 8;
    load_rows_kernel<<<(unsigned)((ctx->N + wpb - 1) / wpb), wpb * 32, 0, ctx->stream>>>(
        ctx->N, ctx->k, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_inc_j, ctx->d_stage, d_qw, body[0], body[1], body[2], d_f);
    KERNEL_CHECK(ctx);
    const int CW = ctx->tg_CW, R = ctx->tg_R, RP = ctx->tg_T / R;
    int rc = RPIM_ERR_STATE;
#define RPIM_PANELS_CASE(CC, RR) if (R == 2 && CW == CC && RP == RR) rc = launch_panels<CC, RR, 2>(ctx, A)
    RPIM_PANELS_CASE(1, 1); RPIM_PANELS_CASE(1, 2); RPIM_PANELS_CASE(1, 3); RPIM_PANELS_CASE(1, 4);
    RPIM_PANELS_CASE(2, 1); RPIM_PANELS_CASE(2, 2); RPIM_PANELS_CASE(2, 3); RPIM_PANELS_CASE(2, 4);
    RPIM_PANELS_CASE(3, 1); RPIM_PANELS_CASE(3, 2); RPIM_PANELS_CASE(3, 3); RPIM_PANELS_CASE(3, 4);
    RPIM_PANELS_CASE(4, 1); RPIM_PANELS_CASE(4, 2); RPIM_PANELS_CASE(4, 3); RPIM_PANELS_CASE(4, 4);
#undef RPIM_PANELS_CASE
#define RPIM_PANELS_CASE1(CC, RR) if (R == 1 && CW == CC && RP == RR) rc = launch_panels<CC, RR, 1>(ctx, A)
    RPIM_PANELS_CASE1(1, 2); RPIM_PANELS_CASE1(1, 4); RPIM_PANELS_CASE1(1, 6); RPIM_PANELS_CASE1(1, 8);
    RPIM_PANELS_CASE1(2, 2); RPIM_PANELS_CASE1(2, 4); RPIM_PANELS_CASE1(2, 6); RPIM_PANELS_CASE1(2, 8);
    RPIM_PANELS_CASE1(3, 2); RPIM_PANELS_CASE1(3, 4); RPIM_PANELS_CASE1(3, 6); RPIM_PANELS_CASE1(3, 8);
#undef RPIM_PANELS_CASE1
    if (rc == RPIM_ERR_STATE) RPIM_FAIL(ctx, RPIM_ERR_STATE, "no panel reduction kernel for CW = %d, R = %d, T = %d", CW, R, ctx->tg_T);
    if (rc) return rc;
    mirror_lower_kernel<<<(unsigned)((ctx->N + wpb - 1) / wpb), wpb * 32, 0, ctx->stream>>>(ctx->N, ctx->d_brow_ptr, ctx->d_bcol,
                                                                                              ctx->d_bdiag, d_vals);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}
