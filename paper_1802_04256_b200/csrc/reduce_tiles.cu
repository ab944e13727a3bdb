// Steps a5 + a6 (R8), TILED form: w * B^T D B blocks reduced deterministically into the CSR
// values when the quadrature points come in groups with nearly coincident supports (several Gauss
// points per background cell).  Integer preprocessing: groups.cu.
//
// A CTA owns a TILE of T consecutive block rows.  Their accumulators S_IJ (9 doubles per column) live in
// SHARED memory, with one open-addressing table (column node -> slot) per row.  The CTA walks the point
// groups incident to any of its rows in ascending order (tile descriptors).  For a group the staged
// shape functions of its 8 points are scattered once into a dense PANEL indexed by the position u in
// the group's sorted union of supports U_g, shared by the T rows (a byte per union entry says which of
// the 8 points hold it; entries a point lacks are never read).  Warp (r, c) owns row r and union
// positions 32 c .. 32 c + 31: every lane accumulates sum_p (w g_I) (x) g_{U_g[u]} over the group's
// points IN REGISTERS (dense: |U_g| ~ 1.3 k), then adds the nine sums to the row's shared accumulator of
// that column: one table probe and
// one read-modify-write per (row, group, column) instead of per contribution.  Every CSR entry is summed
// in a fixed order (points ascending inside a group, groups ascending) by one lane: no floating-point
// atomics, bitwise run-to-run reproducible; K is written once with the isotropic closed form applied at
// write-out.  Panels are double-buffered (one CTA barrier per group); the next group's data travel
// global -> registers while the current group is computed.
#include "common.cuh"

namespace {

constexpr int GB = RPIM_GROUP_POINTS;
constexpr int TD_CAP = RPIM_TILE_DESC_CAP;
constexpr int PD = 4;          // L2 prefetch distance in groups
constexpr unsigned FULLMASK = 0xffffffffu;

struct TileArgs {
    int64_t N, Nq, ntiles;
    int k, Lcap, hlog;
    unsigned kmagic;   // ceil(2^20 / k): e / k = (e * kmagic) >> 20 for e < 1024
    const int64_t* brow_ptr;
    const int32_t* bcol;
    const double* stage;
    const double* qw;
    const int32_t* gu_nodes;
    const uint8_t* gpos;
    const uint8_t* gu_mask;
    const int64_t* tile_ptr;
    const unsigned* tdesc;
    unsigned long long* ticket;
    double lambda, mu, bx, by, bz;
    double* vals;
    double* f;
};

template <int C, int T>
__global__ void __launch_bounds__(T * C * 32, 1)
reduce_tiles_kernel(const TileArgs A) {
    constexpr int GCAP = 32 * C, NT = T * C * 32, DW = 1 + (T + 1) / 2, ITEMS = (GB + T - 1) / T;
    constexpr int PANEL = GB * 3 * GCAP;   // doubles per panel: [point][gx, gy, gz][u]
    extern __shared__ __align__(16) unsigned char tiles_smem[];
    const int HSZ = 1 << A.hlog, hshift = 32 - A.hlog;
    double* acc = reinterpret_cast<double*>(tiles_smem);                               // [T][Lcap * 9]
    unsigned long long* hent = reinterpret_cast<unsigned long long*>(acc + (size_t)T * A.Lcap * 9);   // [T][HSZ]
    double* panel0 = reinterpret_cast<double*>(hent + (size_t)T * HSZ);               // [2][PANEL]
    double* aw_s = panel0 + 2 * PANEL;                                                // [T * C][GB][4] w * grad phi_I
    double* w_s = aw_s + T * C * GB * 4;                                              // [2][GB] quadrature weights
    double* fphi_s = w_s + 2 * GB;                                                    // [2][T][GB] phi_I of point pl at row r's node
    long long* slot_s = reinterpret_cast<long long*>(fphi_s + 2 * T * GB);            // [2] tile handed to the CTA
    long long* rowo_s = slot_s + 2;                                                   // [8] first block of row r
    int* rowL_s = reinterpret_cast<int*>(rowo_s + 8);                                 // [8] block columns of row r
    int* un_s = rowL_s + 8;                                                           // [2][GCAP] union node ids (-1 pad)
    unsigned* um_s = reinterpret_cast<unsigned*>(un_s + 2 * GCAP);                    // [2][GCAP / 4] union masks (bytes)
    unsigned* desc_s = um_s + 2 * (GCAP / 4);                                         // [TD_CAP + PD][DW]

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int r = warp / C, c = warp % C;
    const int k = A.k;
    double* acc_r = acc + (size_t)r * A.Lcap * 9;
    const unsigned long long* hent_r = hent + (size_t)r * HSZ;
    double* aw = aw_s + warp * GB * 4;

    // prefetch registers: the next group's staged rows (one 32-byte sector per (point, support node)),
    // their positions in the union, the union ids and the weights
    double2 pv01[ITEMS], pv23[ITEMS];
    int ppos[ITEMS];
    int pun = -1;
    unsigned pum = 0u;
    double pw = 0.0;
    auto prefetch = [&](int g) {
        const int64_t q0 = (int64_t)g * GB;
        const int nb = (int)min((int64_t)GB, A.Nq - q0);
        const int nitem = nb * k;
        const double2* src = reinterpret_cast<const double2*>(A.stage + q0 * k * 4) + 2 * tid;
        const uint8_t* gp = A.gpos + q0 * k + tid;
#pragma unroll
        for (int it = 0; it < ITEMS; ++it) {
            ppos[it] = -1;
            if (tid + it * NT < nitem) {
                pv01[it] = src[2 * it * NT];
                pv23[it] = src[2 * it * NT + 1];
                ppos[it] = gp[it * NT];   // position in the union; the point's panel offset is added at scatter time
            }
        }
        if (tid < GCAP) pun = A.gu_nodes[(int64_t)g * GCAP + tid];
        if (tid < GCAP / 4) pum = reinterpret_cast<const unsigned*>(A.gu_mask + (int64_t)g * GCAP)[tid];
        if (tid < GB) pw = (tid < nb) ? A.qw[q0 + tid] : 0.0;
    };

    unsigned gi = 0;   // groups processed by this CTA so far: panel buffer = gi & 1
    long long drawn = (tid == 0) ? (long long)atomicAdd(A.ticket, 1ull) : 0;
    for (unsigned itile = 0;; ++itile) {
        if (tid == 0) slot_s[itile & 1] = drawn;
        __syncthreads();   // ticket visible; the previous tile's write-out has read its accumulators
        const int64_t tile = slot_s[itile & 1];
        if (tile >= A.ntiles) break;
        if (tid == 0) drawn = (long long)atomicAdd(A.ticket, 1ull);
        if (tid < T) {
            const int64_t I = tile * T + tid;
            int64_t o = 0;
            int L = 0;
            if (I < A.N) { o = A.brow_ptr[I]; L = (int)(A.brow_ptr[I + 1] - o); }
            rowo_s[tid] = o;
            rowL_s[tid] = L;
        }
        for (int i = tid; i < T * A.Lcap * 9; i += NT) acc[i] = 0.0;
        for (int i = tid; i < T * HSZ; i += NT) hent[i] = ~0ull;
        const int64_t t0 = A.tile_ptr[tile];
        const int ng = (int)(A.tile_ptr[tile + 1] - t0);
        {   // first window of tile descriptors
            const int cnt = min(ng, TD_CAP + PD) * DW;
            const unsigned* src = A.tdesc + t0 * DW;
            for (int i = tid; i < cnt; i += NT) desc_s[i] = src[i];
        }
        __syncthreads();
        if (ng > 0) prefetch((int)desc_s[0]);
        {
            const int64_t o_r = rowo_s[r];
            const int L_r = rowL_s[r];
            unsigned long long* hw = hent + (size_t)r * HSZ;
            for (int s = c * 32 + lane; s < L_r; s += C * 32) {
                const unsigned J = (unsigned)A.bcol[o_r + s];
                unsigned h = (J * 2654435761u) >> hshift;
                const unsigned long long ent = ((unsigned long long)J << 32) | (unsigned)s;
                while (atomicCAS(&hw[h], ~0ull, ent) != ~0ull) h = (h + 1) & (HSZ - 1);
            }
        }
        double fsum = 0.0;   // lanes 0..7 of warp (r, 0): sum of w * phi_I over the points pl = lane of all groups
        int chunk0 = 0;
        for (int it = 0; it < ng; ++it, ++gi) {
            if (it == chunk0 + TD_CAP) {
                // next window [it, it + TD_CAP] (once per TD_CAP groups): wait until every warp has read
                // its part of the old window; the new one is visible after the group's barrier below
                __syncthreads();
                chunk0 = it;
                const int cnt = min(ng - it, TD_CAP + PD) * DW;
                const unsigned* src = A.tdesc + (t0 + it) * DW;
                for (int i = tid; i < cnt; i += NT) desc_s[i] = src[i];
                __syncthreads();
            }
            const int b = gi & 1;
            double* panel = panel0 + b * PANEL;
            // ---- the group's data, registers -> shared memory: gradients into the panel, phi only where a
            //      row of the tile needs it (the entry of the row's own node in a point that holds it)
            const unsigned d1 = desc_s[(it - chunk0) * DW + 1], d2 = (DW > 2) ? desc_s[(it - chunk0) * DW + 2] : 0u;
#pragma unroll
            for (int j = 0; j < ITEMS; ++j) {
                if (ppos[j] >= 0) {
                    const int pl = (int)(((unsigned)(tid + j * NT) * A.kmagic) >> 20);
                    double* dst = panel + pl * 3 * GCAP + ppos[j];
                    dst[0] = pv01[j].y;
                    dst[GCAP] = pv23[j].x;
                    dst[2 * GCAP] = pv23[j].y;
#pragma unroll
                    for (int rr = 0; rr < T; ++rr) {
                        const unsigned h16 = ((rr < 2 ? d1 : d2) >> ((rr & 1) * 16)) & 0xFFFFu;
                        if ((h16 & 0xFFu) == (unsigned)ppos[j] && ((h16 >> (8 + pl)) & 1u))
                            fphi_s[(b * T + rr) * GB + pl] = pv01[j].x;
                    }
                }
            }
            if (tid < GCAP) un_s[b * GCAP + tid] = pun;
            if (tid < GCAP / 4) um_s[b * (GCAP / 4) + tid] = pum;
            if (tid < GB) w_s[b * GB + tid] = pw;
            __syncthreads();   // the only CTA barrier of the group: buffer b complete, buffer b ^ 1 free
            // ---- the next group's data start travelling (registers); the group PD ahead is pulled into L2
            if (tid == NT - 1 && it + PD < ng && it + PD - chunk0 <= TD_CAP + PD - 1) {
                const int64_t q0 = (int64_t)desc_s[(it + PD - chunk0) * DW] * GB;
                const unsigned bytes = (unsigned)min((int64_t)GB, A.Nq - q0) * (unsigned)k * 32u;
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(A.stage + q0 * k * 4), "r"(bytes) : "memory");
            }
            if (it + 1 < ng) prefetch((int)desc_s[(it + 1 - chunk0) * DW]);
            // ---- warp (r, c): contributions of the group to row r, union positions 32 c + lane
            const unsigned dr = (desc_s[(it - chunk0) * DW + 1 + (r >> 1)] >> ((r & 1) * 16)) & 0xFFFFu;
            const unsigned u_r = dr & 0xFFu, m_r = dr >> 8;
            if (m_r == 0u) continue;
            // points (of those incident to the row) that hold this lane's union entry
            const unsigned um = reinterpret_cast<const unsigned char*>(um_s + b * (GCAP / 4))[c * 32 + lane] & m_r;
            if (c > 0 && __ballot_sync(FULLMASK, um != 0u) == 0u) continue;   // nothing for this chunk (c = 0 keeps f)
            if (lane < GB) {
                double ax = 0.0, ay = 0.0, az = 0.0;
                if ((m_r >> lane) & 1u) {
                    const double wq = w_s[b * GB + lane];
                    const double* pp = panel + lane * 3 * GCAP + u_r;
                    ax = wq * pp[0];
                    ay = wq * pp[GCAP];
                    az = wq * pp[2 * GCAP];
                    if (c == 0) fsum += wq * fphi_s[(b * T + r) * GB + lane];
                }
                aw[lane * 4] = ax; aw[lane * 4 + 1] = ay; aw[lane * 4 + 2] = az;
            }
            int slot = -1;
            if (um) {
                const unsigned J = (unsigned)un_s[b * GCAP + c * 32 + lane];
                unsigned h = (J * 2654435761u) >> hshift;
                while (true) {
                    const unsigned long long ent = hent_r[h];
                    if ((unsigned)(ent >> 32) == J) { slot = (int)(unsigned)ent; break; }
                    if (ent == ~0ull) break;
                    h = (h + 1) & (HSZ - 1);
                }
            }
            __syncwarp();
            double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0, s4 = 0.0, s5 = 0.0, s6 = 0.0, s7 = 0.0, s8 = 0.0;
            const double* pg = panel + c * 32 + lane;
#pragma unroll
            for (int pl = 0; pl < GB; ++pl) {
                if (!((m_r >> pl) & 1u)) continue;
                const double2 axy = *reinterpret_cast<const double2*>(aw + pl * 4);
                const double az = aw[pl * 4 + 2];
                if (!((um >> pl) & 1u)) continue;
                const double gx = pg[pl * 3 * GCAP], gy = pg[pl * 3 * GCAP + GCAP], gz = pg[pl * 3 * GCAP + 2 * GCAP];
                s0 = fma(axy.x, gx, s0); s1 = fma(axy.x, gy, s1); s2 = fma(axy.x, gz, s2);
                s3 = fma(axy.y, gx, s3); s4 = fma(axy.y, gy, s4); s5 = fma(axy.y, gz, s5);
                s6 = fma(az, gx, s6); s7 = fma(az, gy, s7); s8 = fma(az, gz, s8);
            }
            if (slot >= 0) {
                double* a = acc_r + slot * 9;
                a[0] += s0; a[1] += s1; a[2] += s2; a[3] += s3; a[4] += s4;
                a[5] += s5; a[6] += s6; a[7] += s7; a[8] += s8;
            }
            __syncwarp();   // aw is rewritten in the next iteration
        }
        __syncthreads();    // all contributions are in the accumulators
        // ---- body-force load: the eight per-point partial sums of a row in a fixed order
        if (c == 0) {
            fsum += __shfl_xor_sync(FULLMASK, fsum, 4);
            fsum += __shfl_xor_sync(FULLMASK, fsum, 2);
            fsum += __shfl_xor_sync(FULLMASK, fsum, 1);
            const int64_t I = tile * T + r;
            if (lane == 0 && I < A.N) {
                A.f[3 * I] = fsum * A.bx;
                A.f[3 * I + 1] = fsum * A.by;
                A.f[3 * I + 2] = fsum * A.bz;
            }
        }
        // ---- K_IJ = lambda S + mu S^T + mu tr(S) I, three scalar rows of 3 L entries per block row
        for (int rr = 0; rr < T; ++rr) {
            const int L = rowL_s[rr];
            if (L == 0) continue;
            const double* ar = acc + (size_t)rr * A.Lcap * 9;
            double* dst = A.vals + 9 * rowo_s[rr];
            const int L3 = 3 * L;
            for (int i = tid; i < 3 * L3; i += NT) {
                const int row = i / L3, col = i - row * L3;
                const int s = col / 3, cc = col - 3 * s;
                const double* a = ar + s * 9;
                double v = fma(A.lambda, a[3 * row + cc], A.mu * a[3 * cc + row]);
                if (row == cc) v += A.mu * ((a[0] + a[4]) + a[8]);
                dst[i] = v;
            }
        }
    }
}

template <int C, int T>
int launch_tiles(rpim_ctx* ctx, const TileArgs& A) {
    auto kern = reduce_tiles_kernel<C, T>;
    const size_t smem = rpim_tiles_smem_bytes(C, T, A.Lcap);
    CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 1, sms = 148;
    CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, T * C * 32, smem));
    if (per_sm < 1) RPIM_FAIL(ctx, RPIM_ERR_CAPACITY, "tiled reduction does not fit on chip (rows of %d block columns)", A.Lcap);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->device);
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_flags + FLAG_ROW_TICKET, 0, sizeof(long long), ctx->stream));
    const int64_t blocks = std::min<int64_t>(A.ntiles, (int64_t)sms * per_sm);
    kern<<<(unsigned)blocks, T * C * 32, smem, ctx->stream>>>(A);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}

}  // namespace

int rpim_stage_accumulate_tiles(rpim_ctx* ctx, const double* d_qw, double lambda, double mu, const double body[3],
                                double* d_vals, double* d_f) {
    TileArgs A;
    A.N = ctx->N; A.Nq = ctx->Nq; A.ntiles = ctx->ntiles;
    A.k = ctx->k; A.Lcap = std::max(ctx->max_blen, 1); A.hlog = rpim_tiles_hlog(A.Lcap);
    A.kmagic = ((1u << 20) + (unsigned)ctx->k - 1u) / (unsigned)ctx->k;
    A.brow_ptr = ctx->d_brow_ptr; A.bcol = ctx->d_bcol; A.stage = ctx->d_stage; A.qw = d_qw;
    A.gu_nodes = ctx->d_gu_nodes; A.gpos = ctx->d_gpos; A.gu_mask = ctx->d_gu_mask;
    A.tile_ptr = ctx->d_tile_ptr; A.tdesc = ctx->d_tdesc;
    A.ticket = (unsigned long long*)(ctx->d_flags + FLAG_ROW_TICKET);
    A.lambda = lambda; A.mu = mu; A.bx = body[0]; A.by = body[1]; A.bz = body[2];
    A.vals = d_vals; A.f = d_f;
    const int C = ctx->tg_C, T = ctx->tg_T;
#define RPIM_TILES_CASE(CC, TT) if (C == CC && T == TT) return launch_tiles<CC, TT>(ctx, A)
    RPIM_TILES_CASE(2, 4); RPIM_TILES_CASE(3, 4); RPIM_TILES_CASE(4, 4); RPIM_TILES_CASE(6, 4);
    RPIM_TILES_CASE(2, 2); RPIM_TILES_CASE(3, 2); RPIM_TILES_CASE(4, 2); RPIM_TILES_CASE(6, 2);
#undef RPIM_TILES_CASE
    RPIM_FAIL(ctx, RPIM_ERR_STATE, "no tiled reduction kernel for C = %d, T = %d", C, T);
}
