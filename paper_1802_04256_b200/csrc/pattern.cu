// Step a2 (R2): node -> point incidence lists, block-CSR pattern (union of
// supp x supp), scalar CSR emission.  Integer work only; every list is sorted, so the
// result does not depend on the order in which threads happen to run.
#include <cstdlib>

#include "common.cuh"

namespace {

// ------------------------------------------------------------------ incidence (transpose of the support table)
__global__ void inc_count_kernel(const int32_t* __restrict__ support, int64_t total, int* __restrict__ count) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x)
        atomicAdd(&count[support[e]], 1);
}

__global__ void inc_fill_kernel(const int32_t* __restrict__ support, int64_t total, int k,
                                const int64_t* __restrict__ inc_ptr, int* __restrict__ cursor,
                                int32_t* __restrict__ inc_q, uint8_t* __restrict__ inc_j) {
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
        int node = support[e];
        int p = atomicAdd(&cursor[node], 1);
        int64_t dst = inc_ptr[node] + p;
        inc_q[dst] = (int32_t)(e / k);
        inc_j[dst] = (uint8_t)(e % k);
    }
}

constexpr int INC_CAP = 4096;   // longest incidence list sorted on chip
constexpr int INC_WARPS = 4;
constexpr int INC_FAST_CAP = 128;   // lists up to this length take the high-occupancy launch
constexpr int INC_FAST_WARPS = 8;
constexpr int INC_MID_CAP = 1024;   // lists up to this length: 8 KB of shared memory per warp

// one warp per node: sort its list ascending by point id (the position byte rides along).
// Three tiers by list length, each with the shared memory (and so the occupancy) its capacity needs:
// up to INC_FAST_CAP, up to INC_MID_CAP, up to INC_CAP.  A tier raises FLAG_OUT when it meets a list
// that is too long for it; the next tier returns at once unless its FLAG_IN was raised.
template <int CAP, int LO, int WARPS, int FLAG_IN, int FLAG_OUT>
__global__ void __launch_bounds__(WARPS * 32)
inc_sort_kernel(int64_t N, const int64_t* __restrict__ inc_ptr, int32_t* __restrict__ inc_q,
                uint8_t* __restrict__ inc_j, long long* __restrict__ flags) {
    extern __shared__ unsigned char smem_raw[];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned long long* key = (unsigned long long*)smem_raw + (size_t)wid * CAP;
    if (FLAG_IN >= 0 && flags[FLAG_IN] == 0) return;   // the previous tier met no list beyond its capacity
    for (int64_t I = (int64_t)blockIdx.x * WARPS + wid; I < N; I += (int64_t)gridDim.x * WARPS) {
        const int64_t a = inc_ptr[I];
        const int len = (int)(inc_ptr[I + 1] - a);
        if (len <= 1 || len <= LO) continue;
        if (len > CAP) {
            if (FLAG_OUT < 0 && lane == 0) atomicAdd((unsigned long long*)&flags[FLAG_INC_CAP], 1ull);
            if (FLAG_OUT >= 0 && lane == 0) flags[FLAG_OUT] = 1;
            continue;
        }
        const int np = next_pow2(len);
        for (int i = lane; i < np; i += 32)
            key[i] = (i < len) ? (((unsigned long long)(unsigned)inc_q[a + i] << 8) | inc_j[a + i])
                               : 0xFFFFFFFFFFFFFFFFull;
        __syncwarp();
        warp_bitonic_u64(key, np);
        for (int i = lane; i < len; i += 32) {
            inc_q[a + i] = (int32_t)(key[i] >> 8);
            inc_j[a + i] = (uint8_t)(key[i] & 0xFF);
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------ block rows: union of the supports of incident points
// Block row I = sorted union of supp(q) over the points q incident to node I.  A warp owns a row.
// Fast path: brow_bitmap_kernel below (two-level bitmap, one pass, rows parked in a fixed-stride
// pool).  Rows that do not fit it go to an overflow list and take the general two-pass path
// (count, scan, fill) with an open-addressing table in shared memory and a bitonic sort.
constexpr int PAT_HASH = 4096;          // general path: open-addressing table per warp (power of two)
constexpr int PAT_MAXROW = 2048;        // longest block row handled
constexpr int PAT_WARPS = 4;

template <int HASH>
__device__ __forceinline__ unsigned pat_hash(int key) {
    return (((unsigned)key * 2654435761u) >> 16) & (HASH - 1);
}

// Number of distinct columns of block row I (same value in all lanes), leaving them in `table`
// (HASH entries, -1 = empty); LIMIT + 1 when the row has more than LIMIT columns.  The total is
// checked after every point, a point adds at most RPIM_MAX_K keys, so the table never holds more
// than LIMIT + RPIM_MAX_K < HASH keys and probing always terminates.
template <int HASH, int LIMIT>
__device__ __forceinline__ int row_union(int* table, int64_t I, const int64_t* __restrict__ inc_ptr,
                                         const int32_t* __restrict__ inc_q, const int32_t* __restrict__ support,
                                         int k) {
    static_assert(LIMIT + RPIM_MAX_K < HASH, "table too small");
    const int lane = lane_id();
    for (int i = lane; i < HASH; i += 32) table[i] = -1;
    __syncwarp();
    int total = 0;
    const int64_t a = inc_ptr[I], b = inc_ptr[I + 1];
    for (int64_t p0 = a; p0 < b; p0 += 32) {
        const int64_t pl = p0 + lane;
        const int qmine = (pl < b) ? inc_q[pl] : 0;
        const int np = (int)min((int64_t)32, b - p0);
        for (int pp = 0; pp < np; ++pp) {
            const int q = __shfl_sync(0xffffffffu, qmine, pp);
            const int32_t* s = support + (int64_t)q * k;
            int fresh = 0;
            for (int j = lane; j < k; j += 32) {
                const int key = s[j];
                unsigned h = pat_hash<HASH>(key);
                while (true) {
                    const int old = atomicCAS(&table[h], -1, key);
                    if (old == -1) { ++fresh; break; }
                    if (old == key) break;
                    h = (h + 1) & (HASH - 1);
                }
            }
            total += __reduce_add_sync(0xffffffffu, fresh);
            if (total > LIMIT) return LIMIT + 1;
        }
    }
    __syncwarp();
    return total;
}

// compact the table into `list`, pad to a power of two and sort ascending; returns nothing
template <int HASH>
__device__ __forceinline__ void table_to_sorted_list(const int* table, int* list, int L) {
    const int lane = lane_id();
    int base = 0;
    for (int i0 = 0; i0 < HASH; i0 += 32) {
        const int v = table[i0 + lane];
        const unsigned m = __ballot_sync(0xffffffffu, v >= 0);
        if (v >= 0) list[base + __popc(m & ((1u << lane) - 1))] = v;
        base += __popc(m);
    }
    const int np = next_pow2(L);
    for (int i = L + lane; i < np; i += 32) list[i] = 0x7FFFFFFF;
    __syncwarp();
    warp_bitonic_i32(list, np);
}

// Fast path (brow_bitmap_kernel): the union of a row as a TWO-LEVEL BITMAP over the window of node
// ids its supports span -- no hashing, no probing, no sort.  Level 1 has one bit per block of 32
// consecutive ids (which blocks are touched), level 2 one 32-bit word per TOUCHED block, stored
// compactly in block order (rank = set level-1 bits below).  Three sweeps over the (incident point,
// support node) pairs: mark blocks, mark ids, and -- once prefix popcounts are known -- turn every
// support node into its column slot (set bits below it), which gives the slot masks of the
// reduction (step a6) in the same pass.  The sorted row is the set bits in order.  With a
// spatially coherent numbering the window is a few z-planes of ids; rows whose window, number of
// touched blocks or length does not fit go to the overflow list and take the general path.
constexpr int B1W = 320;      // level-1 words per warp: windows of up to 320 * 32 * 32 = 327,680 node ids
constexpr int B2CAP = 512;    // touched 32-id blocks per row
constexpr int BM_WARPS = 8;
constexpr int BM_PER_WARP = B1W + B1W / 2 + B2CAP + B2CAP / 2 + 32;   // 32-bit words of shared memory

template <int PSTRIDE>
__global__ void __launch_bounds__(BM_WARPS * 32)
brow_bitmap_kernel(int64_t N, const int64_t* __restrict__ inc_ptr, const int32_t* __restrict__ inc_q,
                   const int32_t* __restrict__ support, int k, int* __restrict__ blen, int32_t* __restrict__ pool,
                   int* __restrict__ bdiag, int32_t* __restrict__ ovf_rows, unsigned* __restrict__ masks,
                   long long* __restrict__ flags) {
    constexpr int NWS = PSTRIDE / 32;   // mask words per (row, incident point)
    constexpr int NPASS = PSTRIDE / 256; // passes of 32 lanes over a support (8 k <= PSTRIDE)
    constexpr unsigned FULLW = 0xffffffffu;
    extern __shared__ unsigned bm_smem[];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned* ws = bm_smem + (size_t)wid * BM_PER_WARP;
    unsigned* l2 = ws;                                                                // [B2CAP] ids of a touched block
    unsigned* l1 = ws + B2CAP;                                                    // [B1W] touched blocks
    unsigned short* p1 = reinterpret_cast<unsigned short*>(l1 + B1W);                 // [B1W] touched blocks before word
    unsigned short* p2 = reinterpret_cast<unsigned short*>(l1 + B1W + B1W / 2);       // [B2CAP] columns before block
    unsigned* mw = l1 + B1W + B1W / 2 + B2CAP / 2;                                    // [32] mask words of one point
    for (int64_t I = (int64_t)blockIdx.x * BM_WARPS + wid; I < N; I += (int64_t)gridDim.x * BM_WARPS) {
        const int64_t pa = inc_ptr[I], pb = inc_ptr[I + 1];
        const int np = (int)(pb - pa);
        if (np == 0) {
            if (lane == 0) blen[I] = 0;
            continue;
        }
        // window of node ids: supports are ascending, so first and last entries bound each of them
        int lo = 0x7FFFFFFF, hi = -1;
        for (int p = lane; p < np; p += 32) {
            const int32_t* sp = support + (int64_t)inc_q[pa + p] * k;
            lo = min(lo, sp[0]);
            hi = max(hi, sp[k - 1]);
        }
        lo = __reduce_min_sync(FULLW, lo);
        hi = __reduce_max_sync(FULLW, hi);
        const int base = lo & ~31;
        const int nblk = ((hi - base) >> 5) + 1;
        const int n1 = (nblk + 31) >> 5;
        bool ovf = n1 > B1W;
        int L = 0, nb2 = 0;
        // sweep over the (incident point, support node) pairs: lane j of pass ps holds node sp[32 ps + j]
        auto sweep = [&](auto&& body_point_begin, auto&& body, auto&& body_point_end) {
            // software pipeline: the point id two points ahead, the support nodes one point ahead
            // (PSTRIDE = 256 serves k <= 32: one pass of 32 lanes; PSTRIDE = 512 serves k <= 64: two)
            auto fetch = [&](int q, bool valid, int (&J)[NPASS]) {
#pragma unroll
                for (int ps = 0; ps < NPASS; ++ps) {
                    const int j = ps * 32 + lane;
                    J[ps] = (valid && j < k) ? support[(int64_t)q * k + j] : -1;
                }
            };
            int q_n = (np > 1) ? inc_q[pa + 1] : 0;
            int J_c[NPASS], J_n[NPASS];
            fetch(inc_q[pa], true, J_c);
            for (int t = 0; t < np; ++t) {
                const int q_nn = (t + 2 < np) ? inc_q[pa + t + 2] : 0;
                fetch(q_n, t + 1 < np, J_n);
                body_point_begin(t);
#pragma unroll
                for (int ps = 0; ps < NPASS; ++ps)
                    if (J_c[ps] >= 0) body(J_c[ps]);
                body_point_end(t);
                q_n = q_nn;
#pragma unroll
                for (int ps = 0; ps < NPASS; ++ps) J_c[ps] = J_n[ps];
            }
        };
        auto nop = [](int) {};
        // exclusive prefix of a per-lane count over the warp; returns (prefix, total)
        auto warp_excl = [&](int cnt, int& total) {
            int incl = cnt;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int up = __shfl_up_sync(FULLW, incl, d);
                if (lane >= d) incl += up;
            }
            total = __shfl_sync(FULLW, incl, 31);
            return incl - cnt;
        };
        if (!ovf) {
            __syncwarp();
            for (int w = lane; w < n1; w += 32) l1[w] = 0u;
            __syncwarp();
            // ---- sweep A: touched blocks
            auto markA = [&](int J) {
                const int b = (J - base) >> 5;
                atomicOr(&l1[b >> 5], 1u << (b & 31));
            };
            sweep(nop, markA, nop);
            __syncwarp();
            const int C1 = (n1 + 31) >> 5;   // level-1 words per lane: lane owns [lane C1, lane C1 + C1)
            {
                int cnt = 0;
                for (int i = 0; i < C1; ++i) {
                    const int w = lane * C1 + i;
                    if (w < n1) cnt += __popc(l1[w]);
                }
                int pre = warp_excl(cnt, nb2);
                for (int i = 0; i < C1; ++i) {
                    const int w = lane * C1 + i;
                    if (w < n1) { p1[w] = (unsigned short)pre; pre += __popc(l1[w]); }
                }
            }
            ovf = nb2 > B2CAP;
            if (!ovf) {
                for (int r = lane; r < nb2; r += 32) l2[r] = 0u;
                __syncwarp();
                // ---- sweep B: ids inside the touched blocks
                auto markB = [&](int J) {
                    const int d = J - base, b = d >> 5;
                    const int r = p1[b >> 5] + __popc(l1[b >> 5] & ((1u << (b & 31)) - 1u));
                    atomicOr(&l2[r], 1u << (d & 31));
                };
                sweep(nop, markB, nop);
                __syncwarp();
                const int C2 = (nb2 + 31) >> 5;
                {
                    int cnt = 0;
                    for (int i = 0; i < C2; ++i) {
                        const int r = lane * C2 + i;
                        if (r < nb2) cnt += __popc(l2[r]);
                    }
                    int pre = warp_excl(cnt, L);
                    for (int i = 0; i < C2; ++i) {
                        const int r = lane * C2 + i;
                        if (r < nb2) { p2[r] = (unsigned short)pre; pre += __popc(l2[r]); }
                    }
                }
                ovf = L > PSTRIDE;
            }
        }
        if (ovf) {
            if (lane == 0) {
                blen[I] = 0;
                const unsigned long long slot = atomicAdd((unsigned long long*)&flags[FLAG_OVF_ROWS], 1ull);
                ovf_rows[slot] = (int32_t)I;
            }
            __syncwarp();
            continue;
        }
        __syncwarp();   // p1, p2 complete
        // ---- the sorted row: set bits in order (lane owns a run of level-1 words)
        {
            const int C1 = (n1 + 31) >> 5;
            int32_t* dst = pool + I * PSTRIDE;
            for (int i = 0; i < C1; ++i) {
                const int w = lane * C1 + i;
                if (w >= n1) break;
                unsigned bits = l1[w];
                int r = p1[w];
                while (bits) {
                    const int blk = 32 * w + __ffs(bits) - 1;
                    bits &= bits - 1;
                    unsigned ids = l2[r];
                    int pre = p2[r];
                    while (ids) {
                        const int key = base + 32 * blk + __ffs(ids) - 1;
                        ids &= ids - 1;
                        dst[pre] = key;
                        if (key == (int)I) bdiag[I] = pre;
                        ++pre;
                    }
                    ++r;
                }
            }
        }
        if (lane == 0) blen[I] = L;
        if (!masks) continue;
        // ---- sweep C: slot masks, bit (slot of node J) for every support node J of every incident point
        {
            unsigned* mdst = masks + pa * NWS;
            sweep([&](int) {
                if (lane < NWS) mw[lane] = 0u;
                __syncwarp();
            }, [&](int J) {
                const int d = J - base, b = d >> 5;
                const int r = p1[b >> 5] + __popc(l1[b >> 5] & ((1u << (b & 31)) - 1u));
                const int slot = p2[r] + __popc(l2[r] & ((1u << (d & 31)) - 1u));
                atomicOr(&mw[slot >> 5], 1u << (slot & 31));
            }, [&](int t) {
                __syncwarp();
                if (lane < NWS) mdst[(int64_t)t * NWS + lane] = mw[lane];
                __syncwarp();
            });
        }
    }
}

// Block rows THROUGH THE POINT GROUPS (panel reduction's preprocessing, groups.cu), ONE sweep: the row's incident
// groups (runs of q / 8 in its ascending incidence list) are visited once; a node J of a group's sorted union U_g
// is a column of the row iff one of the group's points holds both J and the row's node (a byte-mask test).  The
// columns go into a small open-addressing table block of 32 ids -> 32-bit word of members; the touched blocks
// (~ a hundred) are then compacted, sorted and expanded in order.  No window, no second sweep: the two-level
// bitmap of brow_bitmap_kernel needs the touched blocks before it can place the ids.
constexpr int BG_HB = 512;      // table entries per warp (touched blocks of a row: ~ L / 4)
constexpr int BG_GCAP = 256;    // (group, point mask) pairs of a row
constexpr int BG_WARPS = 8;
constexpr int BG_PER_WARP = 2 * BG_HB + 2 * BG_GCAP;   // 32-bit words per warp (keys and words double as the 64-bit sort buffer)

template <int PSTRIDE>
__global__ void __launch_bounds__(BG_WARPS * 32)
brow_groups_kernel(int64_t N, const int64_t* __restrict__ inc_ptr, const int32_t* __restrict__ inc_q, int* __restrict__ blen,
                   int32_t* __restrict__ pool, int* __restrict__ bdiag, int32_t* __restrict__ ovf_rows,
                   const unsigned char* __restrict__ gmeta, int gC, long long* __restrict__ flags) {
    constexpr unsigned FULLW = 0xffffffffu;
    extern __shared__ __align__(16) unsigned bg_smem[];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned* ws = bg_smem + (size_t)wid * BG_PER_WARP;
    unsigned long long* kw = reinterpret_cast<unsigned long long*>(ws);   // [BG_HB] (block id << 32) | member word; ~0 = empty
    int* gl = reinterpret_cast<int*>(ws + 2 * BG_HB);                      // [BG_GCAP] groups incident to the row
    unsigned* gm = reinterpret_cast<unsigned*>(gl + BG_GCAP);              // [BG_GCAP] their points that hold the row's node
    const unsigned gcap = 32u * (unsigned)gC, gmeta_bytes = gcap * 12u + RPIM_GROUP_POINTS * 8u;
    const unsigned lt = (1u << lane) - 1u;
    for (int64_t I = (int64_t)blockIdx.x * BG_WARPS + wid; I < N; I += (int64_t)gridDim.x * BG_WARPS) {
        const int64_t pa = inc_ptr[I], pb = inc_ptr[I + 1];
        const int np = (int)(pb - pa);
        if (np == 0) {
            if (lane == 0) blen[I] = 0;
            continue;
        }
        __syncwarp();
        for (int i = lane; i < BG_HB; i += 32) kw[i] = ~0ull;
        // (group, point mask) pairs of the row; a run cut by a 32-entry boundary gives two pairs (harmless for a union)
        int ngl = 0;
        for (int t0 = 0; t0 < np; t0 += 32) {
            const int t = t0 + lane;
            const int q = t < np ? inc_q[pa + t] : -1;
            const int g = q >= 0 ? q / RPIM_GROUP_POINTS : -1;
            const unsigned bit = q >= 0 ? 1u << (q % RPIM_GROUP_POINTS) : 0u;
            const int gp = __shfl_up_sync(FULLW, g, 1);
            const bool head = q >= 0 && (lane == 0 || g != gp);
            unsigned m = bit;
#pragma unroll
            for (int d = 1; d < RPIM_GROUP_POINTS; ++d) {
                const int gd = __shfl_down_sync(FULLW, g, d);
                const unsigned bd = __shfl_down_sync(FULLW, bit, d);
                if (lane + d < 32 && gd == g) m |= bd;
            }
            const unsigned heads = __ballot_sync(FULLW, head);
            const int pos = ngl + __popc(heads & lt);
            if (head && pos < BG_GCAP) { gl[pos] = g; gm[pos] = m; }
            ngl += __popc(heads);
        }
        bool ovf = ngl > BG_GCAP;
        __syncwarp();
        if (!ovf) {
            // ---- the sweep: lane u of pass ps holds union entry 32 ps + u of the group
            auto fetch = [&](int i, int (&J)[4], unsigned (&pm)[4]) {
                const unsigned char* rec = gmeta + (int64_t)gl[i] * gmeta_bytes;
#pragma unroll
                for (int ps = 0; ps < 4; ++ps) {
                    J[ps] = -1;
                    pm[ps] = 0u;
                    if (ps < gC) {
                        const int u = 32 * ps + lane;
                        J[ps] = reinterpret_cast<const int*>(rec + gcap * 8u)[u];
                        const uint2 jv = reinterpret_cast<const uint2*>(rec)[u];
                        const unsigned a = __vcmpne4(jv.x, 0xFFFFFFFFu) & 0x01010101u, b = __vcmpne4(jv.y, 0xFFFFFFFFu) & 0x01010101u;
                        pm[ps] = ((a * 0x01020408u) >> 24) | (((b * 0x01020408u) >> 24) << 4);
                    }
                }
            };
            int J_c[4], J_n[4];
            unsigned pm_c[4], pm_n[4];
            bool full = false;
            fetch(0, J_c, pm_c);
            for (int i = 0; i < ngl; ++i) {
                if (i + 1 < ngl) fetch(i + 1, J_n, pm_n);
                const unsigned m = gm[i];
#pragma unroll
                for (int ps = 0; ps < 4; ++ps) {
                    if (J_c[ps] >= 0 && (pm_c[ps] & m)) {
                        const unsigned blk = (unsigned)J_c[ps] >> 5;
                        const unsigned long long bitw = 1ull << (J_c[ps] & 31);
                        unsigned h = (blk * 2654435761u) >> (32 - 9);   // BG_HB = 2^9
                        int probes = 0;
                        while (true) {
                            const unsigned long long cur = kw[h];
                            if ((unsigned)(cur >> 32) == blk) { atomicOr(&kw[h], bitw); break; }
                            if (cur == ~0ull) {
                                // claim the entry with an empty member word, then set the bit (another lane may have claimed it for
                                // the same or another block in between: look again)
                                atomicCAS(&kw[h], ~0ull, (unsigned long long)blk << 32);
                                continue;
                            }
                            h = (h + 1) & (BG_HB - 1);
                            if (++probes >= BG_HB) { full = true; break; }
                        }
                    }
                }
#pragma unroll
                for (int ps = 0; ps < 4; ++ps) { J_c[ps] = J_n[ps]; pm_c[ps] = pm_n[ps]; }
            }
            ovf = __any_sync(FULLW, full);
        }
        __syncwarp();
        int nb = 0, L = 0;
        if (!ovf) {
            // ---- compact the touched blocks to the front (reads of a 32-entry slice complete before its writes), count columns
            for (int i0 = 0; i0 < BG_HB; i0 += 32) {
                const unsigned long long v = kw[i0 + lane];
                const bool used = v != ~0ull;
                const unsigned mk = __ballot_sync(FULLW, used);
                __syncwarp();
                if (used) kw[nb + __popc(mk & lt)] = v;
                nb += __popc(mk);
                L += __popc((unsigned)v & (used ? 0xffffffffu : 0u));
                __syncwarp();
            }
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) L += __shfl_xor_sync(FULLW, L, d);
            ovf = L > PSTRIDE;
        }
        if (ovf) {
            if (lane == 0) {
                blen[I] = 0;
                const unsigned long long slot = atomicAdd((unsigned long long*)&flags[FLAG_OVF_ROWS], 1ull);
                ovf_rows[slot] = (int32_t)I;
            }
            __syncwarp();
            continue;
        }
        // ---- sort the blocks by id (the key is the high half), then expand the member words in order
        const int npow = next_pow2(nb);
        for (int i = nb + lane; i < npow; i += 32) kw[i] = ~0ull;
        __syncwarp();
        warp_bitonic_u64(kw, npow);
        int32_t* dst = pool + I * PSTRIDE;
        int base = 0;
        for (int i0 = 0; i0 < nb; i0 += 32) {
            const int i = i0 + lane;
            const unsigned long long v = i < nb ? kw[i] : 0ull;
            unsigned ids = i < nb ? (unsigned)v : 0u;
            const int cnt = __popc(ids);
            int incl = cnt;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int up = __shfl_up_sync(FULLW, incl, d);
                if (lane >= d) incl += up;
            }
            int pre = base + incl - cnt;
            const int blk32 = (int)(unsigned)(v >> 32) << 5;
            while (ids) {
                const int key = blk32 + __ffs(ids) - 1;
                ids &= ids - 1;
                dst[pre] = key;
                if (key == (int)I) bdiag[I] = pre;
                ++pre;
            }
            base += __shfl_sync(FULLW, incl, 31);
        }
        if (lane == 0) blen[I] = L;
    }
}

// rows parked in the pool -> their place in the block-CSR column array (overflow rows have a
// negative pool marker: their length was set by the count pass, the fill pass writes them)
template <int PSTRIDE>
__global__ void __launch_bounds__(256)
brow_copy_kernel(int64_t N, const int64_t* __restrict__ brow_ptr, const int32_t* __restrict__ pool,
                 const uint8_t* __restrict__ is_ovf, int32_t* __restrict__ bcol) {
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int64_t I = (int64_t)blockIdx.x * 8 + wid; I < N; I += (int64_t)gridDim.x * 8) {
        if (is_ovf[I]) continue;
        const int64_t o = brow_ptr[I];
        const int L = (int)(brow_ptr[I + 1] - o);
        const int32_t* src = pool + I * PSTRIDE;
        for (int i = lane; i < L; i += 32) bcol[o + i] = src[i];
    }
}

__global__ void mark_rows_kernel(const int32_t* __restrict__ rows, const long long* __restrict__ nrows,
                                 uint8_t* __restrict__ mark) {
    const long long n = *nrows;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        mark[rows[i]] = 1;
}

// General path over a row list (rows == nullptr: all N rows).
__global__ void __launch_bounds__(PAT_WARPS * 32)
brow_count_kernel(int64_t N, const int32_t* __restrict__ rows, const long long* __restrict__ nrows,
                  const int64_t* __restrict__ inc_ptr, const int32_t* __restrict__ inc_q,
                  const int32_t* __restrict__ support, int k, int* __restrict__ blen, long long* __restrict__ flags) {
    extern __shared__ int pat_smem[];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int* table = pat_smem + (size_t)wid * PAT_HASH;
    const int64_t n = rows ? (int64_t)*nrows : N;
    for (int64_t r = (int64_t)blockIdx.x * PAT_WARPS + wid; r < n; r += (int64_t)gridDim.x * PAT_WARPS) {
        const int64_t I = rows ? rows[r] : r;
        const int L = row_union<PAT_HASH, PAT_MAXROW>(table, I, inc_ptr, inc_q, support, k);
        if (L > PAT_MAXROW && lane == 0) atomicAdd((unsigned long long*)&flags[FLAG_PAT_CAP], 1ull);
        if (lane == 0) blen[I] = min(L, PAT_MAXROW);
        __syncwarp();
    }
}

__global__ void __launch_bounds__(PAT_WARPS * 32)
brow_fill_kernel(int64_t N, const int32_t* __restrict__ rows, const long long* __restrict__ nrows,
                 const int64_t* __restrict__ inc_ptr, const int32_t* __restrict__ inc_q,
                 const int32_t* __restrict__ support, int k, const int64_t* __restrict__ brow_ptr,
                 int32_t* __restrict__ bcol, int* __restrict__ bdiag) {
    extern __shared__ int pat_smem[];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int* table = pat_smem + (size_t)wid * PAT_HASH;
    int* list = pat_smem + (size_t)PAT_WARPS * PAT_HASH + (size_t)wid * PAT_MAXROW;
    const int64_t n = rows ? (int64_t)*nrows : N;
    for (int64_t r = (int64_t)blockIdx.x * PAT_WARPS + wid; r < n; r += (int64_t)gridDim.x * PAT_WARPS) {
        const int64_t I = rows ? rows[r] : r;
        const int L = row_union<PAT_HASH, PAT_MAXROW>(table, I, inc_ptr, inc_q, support, k);
        if (L > PAT_MAXROW) continue;   // reported by the count pass
        table_to_sorted_list<PAT_HASH>(table, list, L);
        const int64_t o = brow_ptr[I];
        for (int i = lane; i < L; i += 32) {
            const int c = list[i];
            bcol[o + i] = c;
            if (c == (int)I) bdiag[I] = i;
        }
        __syncwarp();
    }
}

__global__ void max_i32_kernel(const int* __restrict__ v, int64_t n, int* __restrict__ out) {
    int m = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        m = max(m, v[i]);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, d));
    if ((threadIdx.x & 31) == 0) atomicMax(out, m);
}

// ------------------------------------------------------------------ scalar CSR emission (3x3 expansion)
template <typename IdxT>
__global__ void emit_rowptr_kernel(int64_t N, const int64_t* __restrict__ brow_ptr, IdxT* __restrict__ row_ptr) {
    int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (I > N) return;
    if (I == N) { row_ptr[3 * N] = (IdxT)(9 * brow_ptr[N]); return; }
    const int64_t o = brow_ptr[I], L = brow_ptr[I + 1] - o;
#pragma unroll
    for (int a = 0; a < 3; ++a) row_ptr[3 * I + a] = (IdxT)(9 * o + a * 3 * L);
}

template <typename IdxT>
__global__ void __launch_bounds__(256)
emit_colidx_kernel(int64_t N, const int64_t* __restrict__ brow_ptr, const int32_t* __restrict__ bcol,
                   IdxT* __restrict__ col_idx) {
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int64_t I = (int64_t)blockIdx.x * 8 + wid; I < N; I += (int64_t)gridDim.x * 8) {
        const int64_t o = brow_ptr[I];
        const int L = (int)(brow_ptr[I + 1] - o);
        for (int a = 0; a < 3; ++a) {
            IdxT* dst = col_idx + 9 * o + (int64_t)a * 3 * L;
            for (int i = lane; i < 3 * L; i += 32) dst[i] = (IdxT)(3 * (int64_t)bcol[o + i / 3] + i % 3);
        }
    }
}

}  // namespace

int rpim_stage_incidence(rpim_ctx* ctx) {
    cudaStream_t st = ctx->stream;
    const int64_t N = ctx->N, total = ctx->Nq * ctx->k;
    int rc;
    if ((rc = ws_alloc(ctx, &ctx->d_inc_count, N))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_inc_ptr, N + 1))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_inc_q, total))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_inc_j, total))) return rc;
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_inc_count, 0, N * sizeof(int), st));
    const unsigned nb = (unsigned)std::min<int64_t>((total + 255) / 256, 148 * 32);
    inc_count_kernel<<<nb, 256, 0, st>>>(ctx->d_support, total, ctx->d_inc_count);
    KERNEL_CHECK(ctx);
    if ((rc = rpim_scan_i32_to_i64(ctx, ctx->d_inc_count, ctx->d_inc_ptr, N))) return rc;
    // longest list (for capacity checks and launch sizing later)
    int* d_max = (int*)ctx->d_scratch;
    CUDA_TRY(ctx, cudaMemsetAsync(d_max, 0, sizeof(int), st));
    max_i32_kernel<<<(unsigned)std::min<int64_t>((N + 255) / 256, 1024), 256, 0, st>>>(ctx->d_inc_count, N, d_max);
    KERNEL_CHECK(ctx);
    CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_inc_count, 0, N * sizeof(int), st));
    inc_fill_kernel<<<nb, 256, 0, st>>>(ctx->d_support, total, ctx->k, ctx->d_inc_ptr, ctx->d_inc_count,
                                        ctx->d_inc_q, ctx->d_inc_j);
    KERNEL_CHECK(ctx);
    {
        auto fast = inc_sort_kernel<INC_FAST_CAP, 0, INC_FAST_WARPS, -1, FLAG_INC_LONG>;
        const size_t smem_f = (size_t)INC_FAST_WARPS * INC_FAST_CAP * sizeof(unsigned long long);
        fast<<<(unsigned)std::min<int64_t>((N + INC_FAST_WARPS - 1) / INC_FAST_WARPS, 148 * 64), INC_FAST_WARPS * 32,
               smem_f, st>>>(N, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_inc_j, ctx->d_flags);
        KERNEL_CHECK(ctx);
        auto mid = inc_sort_kernel<INC_MID_CAP, INC_FAST_CAP, INC_WARPS, FLAG_INC_LONG, FLAG_INC_LONG2>;
        const size_t smem_m = (size_t)INC_WARPS * INC_MID_CAP * sizeof(unsigned long long);
        mid<<<(unsigned)std::min<int64_t>((N + INC_WARPS - 1) / INC_WARPS, 148 * 16), INC_WARPS * 32, smem_m, st>>>(
            N, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_inc_j, ctx->d_flags);
        KERNEL_CHECK(ctx);
        auto slow = inc_sort_kernel<INC_CAP, INC_MID_CAP, INC_WARPS, FLAG_INC_LONG2, -1>;
        const size_t smem = (size_t)INC_WARPS * INC_CAP * sizeof(unsigned long long);
        CUDA_TRY(ctx, cudaFuncSetAttribute(slow, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        slow<<<(unsigned)std::min<int64_t>((N + INC_WARPS - 1) / INC_WARPS, 148), INC_WARPS * 32, smem, st>>>(
            N, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_inc_j, ctx->d_flags);
        KERNEL_CHECK(ctx);
    }
    CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->max_inc, d_max, sizeof(int), cudaMemcpyDeviceToHost, st));
    return RPIM_OK;
}

namespace {
template <int PSTRIDE>
int launch_brow_bitmap(rpim_ctx* ctx, int32_t* d_pool, int32_t* d_ovf_rows, unsigned* d_masks) {
    const int64_t N = ctx->N;
    auto kern = brow_bitmap_kernel<PSTRIDE>;
    const size_t smem = (size_t)BM_WARPS * BM_PER_WARP * sizeof(unsigned);
    CUDA_TRY(ctx, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const unsigned nb = (unsigned)std::min<int64_t>((N + BM_WARPS - 1) / BM_WARPS, 148 * 16);
    // (point groups exist: the row unions go through theirs, in one sweep; they never coexist with the slot masks)
    const int gC = (ctx->tg_C > 0 && ctx->d_gmeta && !d_masks) ? ctx->tg_C : 0;
    if (gC > 0) {
        auto kg = brow_groups_kernel<PSTRIDE>;
        const size_t smg = (size_t)BG_WARPS * BG_PER_WARP * sizeof(unsigned);
        CUDA_TRY(ctx, cudaFuncSetAttribute(kg, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smg));
        const unsigned nbg = (unsigned)std::min<int64_t>((N + BG_WARPS - 1) / BG_WARPS, 148 * 16);
        kg<<<nbg, BG_WARPS * 32, smg, ctx->stream>>>(N, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_blen, d_pool, ctx->d_bdiag, d_ovf_rows,
                                                      ctx->d_gmeta, gC, ctx->d_flags);
        KERNEL_CHECK(ctx);
        return RPIM_OK;
    }
    kern<<<nb, BM_WARPS * 32, smem, ctx->stream>>>(N, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_support, ctx->k, ctx->d_blen,
                                                   d_pool, ctx->d_bdiag, d_ovf_rows, d_masks, ctx->d_flags);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}
template <int PSTRIDE>
int launch_brow_copy(rpim_ctx* ctx, const int32_t* d_pool, const uint8_t* d_is_ovf) {
    const int64_t N = ctx->N;
    brow_copy_kernel<PSTRIDE><<<(unsigned)std::min<int64_t>((N + 7) / 8, 148 * 32), 256, 0, ctx->stream>>>(
        N, ctx->d_brow_ptr, d_pool, d_is_ovf, ctx->d_bcol);
    KERNEL_CHECK(ctx);
    return RPIM_OK;
}
}  // namespace

int rpim_stage_block_pattern(rpim_ctx* ctx) {
    cudaStream_t st = ctx->stream;
    const int64_t N = ctx->N;
    int rc;
    if ((rc = ws_alloc(ctx, &ctx->d_blen, N))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_brow_ptr, N + 1))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_bdiag, N))) return rc;
    // Fast path when the expected row length (about 5..8 supports' worth of columns) fits the
    // pool stride; pstride = 0 selects the general two-pass path for every row.
    const int pstride = (8 * ctx->k <= 256) ? 256 : (8 * ctx->k <= 512) ? 512 : 0;
    int masks_stride = 0;
    int32_t *d_pool = nullptr, *d_ovf_rows = nullptr;
    uint8_t* d_is_ovf = nullptr;
    auto drop_tmp = [&]() { ws_free(ctx, &d_pool); ws_free(ctx, &d_ovf_rows); ws_free(ctx, &d_is_ovf); };
    const long long* d_novf = ctx->d_flags + FLAG_OVF_ROWS;
    const unsigned nb = (unsigned)std::min<int64_t>((N + PAT_WARPS - 1) / PAT_WARPS, 148 * 16);
    const unsigned nb_ovf = 148 * 2;   // the overflow list is normally empty: a small fixed grid
    const size_t smem_cnt = (size_t)PAT_WARPS * PAT_HASH * sizeof(int);
    const size_t smem_fill = smem_cnt + (size_t)PAT_WARPS * PAT_MAXROW * sizeof(int);
    CUDA_TRY(ctx, cudaFuncSetAttribute(brow_count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cnt));
    CUDA_TRY(ctx, cudaFuncSetAttribute(brow_fill_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_fill));
    if (pstride) {
        if ((rc = ws_alloc(ctx, &d_pool, N * pstride)) || (rc = ws_alloc(ctx, &d_ovf_rows, N)) ||
            (rc = ws_alloc(ctx, &d_is_ovf, N))) { drop_tmp(); return rc; }
        CUDA_TRY(ctx, cudaMemsetAsync(ctx->d_flags + FLAG_OVF_ROWS, 0, sizeof(long long), st));
        CUDA_TRY(ctx, cudaMemsetAsync(d_is_ovf, 0, (size_t)N, st));
        // slot masks of the reduction ride along (fixed stride of pstride / 32 words per incident
        // point); they are an accelerator: skipped when they would take more than a quarter of the
        // free device memory
        unsigned* d_masks = nullptr;
        {
            const int64_t words = ctx->Nq * (int64_t)ctx->k * (pstride / 32);
            const int64_t bytes = words * (int64_t)sizeof(unsigned);
            bool reuse = false;   // a block we already own does not count against the budget
            for (auto& b : ctx->ws_cache) reuse = reuse || (b.second >= bytes && b.second <= 2 * bytes + 4096);
            if (ctx->d_masks) {
                auto it = ctx->ws_sizes.find((void*)ctx->d_masks);
                reuse = reuse || (it != ctx->ws_sizes.end() && it->second >= bytes && it->second <= 2 * bytes + 4096);
            }
            size_t free_b = 0, total_b = 0;
            if (!reuse && ctx->tg_C == 0) CUDA_TRY(ctx, cudaMemGetInfo(&free_b, &total_b));   // a driver call: only when it matters
            if (ctx->tg_C > 0) {
                // the panel reduction (reduce_panels.cu) needs no slot masks
            } else if (reuse || (uint64_t)bytes <= free_b / 4) {
                if (ws_alloc(ctx, &ctx->d_masks, words) == RPIM_OK) d_masks = ctx->d_masks;
                else ctx->err.clear();
            }
        }
        rc = (pstride == 256) ? launch_brow_bitmap<256>(ctx, d_pool, d_ovf_rows, d_masks)
                              : launch_brow_bitmap<512>(ctx, d_pool, d_ovf_rows, d_masks);
        masks_stride = d_masks ? pstride / 32 : 0;
        if (rc) { drop_tmp(); return rc; }
        mark_rows_kernel<<<64, 256, 0, st>>>(d_ovf_rows, d_novf, d_is_ovf);
        KERNEL_CHECK(ctx);
        brow_count_kernel<<<nb_ovf, PAT_WARPS * 32, smem_cnt, st>>>(N, d_ovf_rows, d_novf, ctx->d_inc_ptr, ctx->d_inc_q,
                                                                     ctx->d_support, ctx->k, ctx->d_blen, ctx->d_flags);
        KERNEL_CHECK(ctx);
    } else {
        brow_count_kernel<<<nb, PAT_WARPS * 32, smem_cnt, st>>>(N, nullptr, nullptr, ctx->d_inc_ptr, ctx->d_inc_q,
                                                                 ctx->d_support, ctx->k, ctx->d_blen, ctx->d_flags);
        KERNEL_CHECK(ctx);
    }
    if ((rc = rpim_scan_i32_to_i64(ctx, ctx->d_blen, ctx->d_brow_ptr, N))) { drop_tmp(); return rc; }
    int* d_max = (int*)ctx->d_scratch;
    CUDA_TRY(ctx, cudaMemsetAsync(d_max, 0, sizeof(int), st));
    max_i32_kernel<<<(unsigned)std::min<int64_t>((N + 255) / 256, 1024), 256, 0, st>>>(ctx->d_blen, N, d_max);
    KERNEL_CHECK(ctx);
    long long h_flags[NUM_FLAGS];
    CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->nnzb, ctx->d_brow_ptr + N, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaMemcpyAsync(&ctx->max_blen, d_max, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaMemcpyAsync(h_flags, ctx->d_flags, sizeof(h_flags), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    if (h_flags[FLAG_KNN_CAP]) {
        drop_tmp();
        RPIM_FAIL(ctx, RPIM_ERR_CAPACITY, "kNN: %lld points found fewer than k nodes (k > N?)",
                  h_flags[FLAG_KNN_CAP]);
    }
    if (h_flags[FLAG_INC_CAP]) {
        drop_tmp();
        RPIM_FAIL(ctx, RPIM_ERR_CAPACITY, "incidence: %lld nodes belong to more than %d supports", h_flags[FLAG_INC_CAP],
                  INC_CAP);
    }
    if (h_flags[FLAG_PAT_CAP]) {
        drop_tmp();
        RPIM_FAIL(ctx, RPIM_ERR_CAPACITY, "pattern: %lld block rows are longer than %d", h_flags[FLAG_PAT_CAP],
                  PAT_MAXROW);
    }
    // the ride-along masks are complete only if no row took the general path
    ctx->have_masks = masks_stride > 0 && h_flags[FLAG_OVF_ROWS] == 0;
    ctx->mask_stride = ctx->have_masks ? masks_stride : 0;
    if ((rc = ws_alloc(ctx, &ctx->d_bcol, ctx->nnzb))) { drop_tmp(); return rc; }
    if (pstride) {
        rc = (pstride == 256) ? launch_brow_copy<256>(ctx, d_pool, d_is_ovf) : launch_brow_copy<512>(ctx, d_pool, d_is_ovf);
        if (rc) { drop_tmp(); return rc; }
        if (h_flags[FLAG_OVF_ROWS] > 0) {
            brow_fill_kernel<<<nb_ovf, PAT_WARPS * 32, smem_fill, st>>>(N, d_ovf_rows, d_novf, ctx->d_inc_ptr,
                                                                        ctx->d_inc_q, ctx->d_support, ctx->k,
                                                                        ctx->d_brow_ptr, ctx->d_bcol, ctx->d_bdiag);
            KERNEL_CHECK(ctx);
        }
        drop_tmp();   // parked in the workspace cache: reused in stream order, no synchronisation needed
    } else {
        brow_fill_kernel<<<nb, PAT_WARPS * 32, smem_fill, st>>>(N, nullptr, nullptr, ctx->d_inc_ptr, ctx->d_inc_q,
                                                                ctx->d_support, ctx->k, ctx->d_brow_ptr, ctx->d_bcol,
                                                                ctx->d_bdiag);
        KERNEL_CHECK(ctx);
    }
    return RPIM_OK;
}

// ------------------------------------------------------------------ precomputed slot maps of the reduction (step a6)
// For incident point p of block row I: ceil(L_I / 32) words, bit s set iff column slot s of the row
// is a support node of the point.  With the supports and the rows both ascending, the position of
// slot s's node in the support is the number of set bits below s, so the masks are all the
// reduction needs to route gradients to CSR slots (accumulate.cu, MASKED kernels).
namespace {
__global__ void mask_count_kernel(int64_t N, const int64_t* __restrict__ inc_ptr, const int64_t* __restrict__ brow_ptr,
                                  int* __restrict__ count) {
    const int64_t I = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (I >= N) return;
    const int64_t len = inc_ptr[I + 1] - inc_ptr[I];
    const int64_t nw = (brow_ptr[I + 1] - brow_ptr[I] + 31) >> 5;
    count[I] = (int)(len * nw);
}

template <int HLOG, int WARPS>
__global__ void __launch_bounds__(WARPS * 32)
slot_mask_kernel(int64_t N, int k, const int64_t* __restrict__ inc_ptr, const int32_t* __restrict__ inc_q,
                 const int32_t* __restrict__ support, const int64_t* __restrict__ brow_ptr,
                 const int32_t* __restrict__ bcol, const int64_t* __restrict__ mask_ptr, unsigned* __restrict__ masks) {
    constexpr int HSZ = 1 << HLOG;
    __shared__ unsigned long long hent_s[WARPS][HSZ];
    __shared__ unsigned words_s[WARPS][32];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned long long* hent = hent_s[wid];
    unsigned* words = words_s[wid];
    const int npass = (k + 31) >> 5;
    for (int64_t I = (int64_t)blockIdx.x * WARPS + wid; I < N; I += (int64_t)gridDim.x * WARPS) {
        const int64_t o = brow_ptr[I];
        const int L = (int)(brow_ptr[I + 1] - o);
        const int NWc = (L + 31) >> 5;
        const int64_t pa = inc_ptr[I], pb = inc_ptr[I + 1];
        if (pa == pb) continue;
        __syncwarp();
        for (int s = lane; s < HSZ; s += 32) hent[s] = ~0ull;
        __syncwarp();
        for (int s = lane; s < L; s += 32) {
            const unsigned J = (unsigned)bcol[o + s];
            unsigned h = (J * 2654435761u) >> (32 - HLOG);
            const unsigned long long ent = ((unsigned long long)J << 32) | (unsigned)s;
            while (atomicCAS(&hent[h], ~0ull, ent) != ~0ull) h = (h + 1) & (HSZ - 1);
        }
        __syncwarp();
        unsigned* dst = masks + mask_ptr[I];
        const int64_t nitems = (pb - pa) * npass;
        auto loadJ = [&](int64_t item) {
            const int64_t t = item / npass;
            const int j = (int)(item - t * npass) * 32 + lane;
            return (j < k) ? support[(int64_t)inc_q[pa + t] * k + j] : -1;
        };
        int Jnext = loadJ(0);
        for (int64_t item = 0; item < nitems; ++item) {
            const int J = Jnext;
            if (item + 1 < nitems) Jnext = loadJ(item + 1);
            const int64_t t = item / npass;
            const int ps = (int)(item - t * npass);
            if (ps == 0) {
                if (lane < NWc) words[lane] = 0u;
                __syncwarp();
            }
            if (J >= 0) {
                unsigned h = ((unsigned)J * 2654435761u) >> (32 - HLOG);
                unsigned long long ent = hent[h];
                while ((unsigned)(ent >> 32) != (unsigned)J) { h = (h + 1) & (HSZ - 1); ent = hent[h]; }
                const unsigned slot = (unsigned)ent;
                atomicOr(&words[slot >> 5], 1u << (slot & 31));
            }
            if (ps == npass - 1) {
                __syncwarp();
                if (lane < NWc) dst[t * NWc + lane] = words[lane];
                __syncwarp();
            }
        }
    }
}
}  // namespace

int rpim_stage_slot_masks(rpim_ctx* ctx) {
    cudaStream_t st = ctx->stream;
    const int64_t N = ctx->N;
    if (ctx->have_masks) return RPIM_OK;   // built together with the block rows (fixed stride)
    ctx->mask_stride = 0;
    if (ctx->max_blen > 1024 || ctx->max_blen < 1) return RPIM_OK;   // such rows take the generic reduction
    int rc;
    int* d_cnt = nullptr;
    if ((rc = ws_alloc(ctx, &d_cnt, N))) return rc;
    if ((rc = ws_alloc(ctx, &ctx->d_mask_ptr, N + 1))) { ws_free(ctx, &d_cnt); return rc; }
    mask_count_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(N, ctx->d_inc_ptr, ctx->d_brow_ptr, d_cnt);
    KERNEL_CHECK(ctx);
    rc = rpim_scan_i32_to_i64(ctx, d_cnt, ctx->d_mask_ptr, N);
    ws_free(ctx, &d_cnt);
    if (rc) return rc;
    int64_t nwords = 0;
    CUDA_TRY(ctx, cudaMemcpyAsync(&nwords, ctx->d_mask_ptr + N, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    // budget: the maps are an accelerator, not a requirement -- skip them when they would take
    // more than a quarter of the free device memory (config 5: ~55 GB) or the allocation fails
    size_t free_b = 0, total_b = 0;
    CUDA_TRY(ctx, cudaMemGetInfo(&free_b, &total_b));
    const int64_t bytes = nwords * (int64_t)sizeof(unsigned);
    bool reuse = false;   // a parked block of the right size does not count against the budget
    for (auto& b : ctx->ws_cache) reuse = reuse || (b.second >= bytes && b.second <= 2 * bytes + 4096);
    if (ctx->d_masks) { auto it = ctx->ws_sizes.find((void*)ctx->d_masks); reuse = reuse || (it != ctx->ws_sizes.end() && it->second >= bytes && it->second <= 2 * bytes + 4096); }
    if (!reuse && (uint64_t)bytes > free_b / 4) { ws_free(ctx, &ctx->d_masks); return RPIM_OK; }
    if (ws_alloc(ctx, &ctx->d_masks, nwords) != RPIM_OK) { ctx->err.clear(); return RPIM_OK; }
    const int Lmax = ctx->max_blen;
    constexpr int W = 8;
    const unsigned nb = (unsigned)std::min<int64_t>((N + W - 1) / W, 148 * 32);
    if (Lmax <= 256)
        slot_mask_kernel<9, W><<<nb, W * 32, 0, st>>>(N, ctx->k, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_support,
                                                      ctx->d_brow_ptr, ctx->d_bcol, ctx->d_mask_ptr, ctx->d_masks);
    else if (Lmax <= 512)
        slot_mask_kernel<10, 4><<<(unsigned)std::min<int64_t>((N + 3) / 4, 148 * 32), 128, 0, st>>>(
            N, ctx->k, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_support, ctx->d_brow_ptr, ctx->d_bcol, ctx->d_mask_ptr,
            ctx->d_masks);
    else
        slot_mask_kernel<11, 2><<<(unsigned)std::min<int64_t>((N + 1) / 2, 148 * 32), 64, 0, st>>>(
            N, ctx->k, ctx->d_inc_ptr, ctx->d_inc_q, ctx->d_support, ctx->d_brow_ptr, ctx->d_bcol, ctx->d_mask_ptr,
            ctx->d_masks);
    KERNEL_CHECK(ctx);
    ctx->have_masks = true;
    return RPIM_OK;
}

int rpim_stage_emit_pattern(rpim_ctx* ctx, void* d_row_ptr, void* d_col_idx) {
    cudaStream_t st = ctx->stream;
    const int64_t N = ctx->N;
    const unsigned nbr = (unsigned)((N + 1 + 255) / 256);
    const unsigned nbc = (unsigned)std::min<int64_t>((N + 7) / 8, 148 * 32);
    if (ctx->index_bits == RPIM_INDEX_MIXED) {   // 64-bit row offsets, 32-bit column ids (3 N < 2^31 always holds)
        if (d_row_ptr) { emit_rowptr_kernel<int64_t><<<nbr, 256, 0, st>>>(N, ctx->d_brow_ptr, (int64_t*)d_row_ptr); KERNEL_CHECK(ctx); }
        if (d_col_idx) { emit_colidx_kernel<int32_t><<<nbc, 256, 0, st>>>(N, ctx->d_brow_ptr, ctx->d_bcol, (int32_t*)d_col_idx); KERNEL_CHECK(ctx); }
    } else if (ctx->index_bits == 32) {
        if (d_row_ptr) { emit_rowptr_kernel<int32_t><<<nbr, 256, 0, st>>>(N, ctx->d_brow_ptr, (int32_t*)d_row_ptr); KERNEL_CHECK(ctx); }
        if (d_col_idx) { emit_colidx_kernel<int32_t><<<nbc, 256, 0, st>>>(N, ctx->d_brow_ptr, ctx->d_bcol, (int32_t*)d_col_idx); KERNEL_CHECK(ctx); }
    } else {
        if (d_row_ptr) { emit_rowptr_kernel<int64_t><<<nbr, 256, 0, st>>>(N, ctx->d_brow_ptr, (int64_t*)d_row_ptr); KERNEL_CHECK(ctx); }
        if (d_col_idx) { emit_colidx_kernel<int64_t><<<nbc, 256, 0, st>>>(N, ctx->d_brow_ptr, ctx->d_bcol, (int64_t*)d_col_idx); KERNEL_CHECK(ctx); }
    }
    return RPIM_OK;
}
