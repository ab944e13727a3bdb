/*
 * rpim.h -- C ABI of librpim: B200-native (sm_100a) RPIM global stiffness assembly with
 * penalty enforcement of displacement boundary conditions (GeoMFree3D, arXiv 1802.04256).
 *
 * The calls follow the paper's stage split ("assemble the global stiffness
 * matrix ... enforce the boundary conditions ... solve") and the names BASELINE.json
 * north_star fixes: rpim_build_pattern, rpim_assemble, rpim_apply_penalty.  The exact
 * arithmetic of every step is the set of readings R1..R12 in DESIGN.md section 2.
 *
 * Conventions
 *   - "d_" arguments are DEVICE pointers (caller-owned, e.g. torch tensors); "h_" and
 *     "out_" arguments and small by-value arrays are HOST pointers.
 *   - All coordinate / value arrays are fp64, row-major, densely packed.
 *   - DOF id = 3*node + component.  CSR rows are strictly ascending, every structural 3x3
 *     block stores all nine entries, the diagonal is always present (R2).
 *   - Every call returns 0 (RPIM_OK) or a negative rpim_status; rpim_last_error() gives a
 *     text for the last failure on that context.  No call aborts, throws or prints.
 *   - Work is enqueued on the stream given to rpim_create.  Calls that return host scalars
 *     (out_*) synchronise that stream before returning; the others are asynchronous.
 *   - The context owns only its internal workspace (cell grid, supports, incidence lists,
 *     block pattern, staged shape functions); it is freed by rpim_destroy.  The node and
 *     point arrays passed to rpim_build_pattern must stay valid and unchanged until the
 *     last rpim_assemble / rpim_add_point_loads that uses the pattern has completed.
 *   - There is no CPU fallback anywhere: without a CUDA device rpim_create fails.
 */
#ifndef RPIM_H
#define RPIM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rpim_ctx rpim_ctx;

typedef enum rpim_status {
    RPIM_OK = 0,
    RPIM_ERR_INVALID_ARG = -1,     /* null pointer, k < 4, k > N, k > RPIM_MAX_K, bad index_bits, ... */
    RPIM_ERR_ALLOC = -2,           /* device or host allocation failed */
    RPIM_ERR_CUDA = -3,            /* a CUDA runtime call or kernel failed */
    RPIM_ERR_STATE = -4,           /* call order violated (e.g. assemble before build_pattern) */
    RPIM_ERR_BC_NODE_INVALID = -5, /* boundary node id out of range, listed twice, or without a matrix row */
    RPIM_ERR_INDEX_OVERFLOW = -6,  /* 32-bit indices forced but nnz >= 2^31 */
    RPIM_ERR_CAPACITY = -7,        /* an on-chip work buffer would overflow (a node in more than 4096 supports, a block row
                                      of more than 2048 columns, k > N); the support search itself has no capacity limit */
    RPIM_ERR_BREAKDOWN = -8,       /* rpim_solve_pcg: p^T K p <= 0 or not finite (K is not positive definite) */
    RPIM_ERR_SINGULAR_POINT = -9   /* rpim_add_point_loads: a load point has a singular moment matrix */
} rpim_status;

#define RPIM_MAX_K 124  /* moment systems up to 128 x 128 */

/* index_bits value for CSR arrays of mixed width: row_ptr int64_t (offsets up to nnz), col_idx int32_t (DOF ids
 * below 3 N < 2^31, which rpim_build_pattern guarantees).  Where nnz > 2^31 - 1 forces 64-bit offsets this halves
 * col_idx: 31 GB less HBM and 31 GB less to copy at the `stress` configuration.  Never
 * chosen automatically: index_bits = 0 keeps BASELINE.json's rule (both arrays 64-bit iff nnz > 2^31 - 1). */
#define RPIM_INDEX_MIXED 6432

/* Create a context on CUDA device `device`; all work goes to `cuda_stream` (a cudaStream_t,
 * may be NULL for the default stream).  Fails with RPIM_ERR_CUDA when no device exists. */
int rpim_create(rpim_ctx** out_ctx, int device, void* cuda_stream);
int rpim_destroy(rpim_ctx* ctx);
const char* rpim_last_error(const rpim_ctx* ctx);

/* Bytes of device workspace currently owned by the context. */
int64_t rpim_workspace_bytes(const rpim_ctx* ctx);

/* Which kernel reduces the element matrices into the CSR values (step a6; all are deterministic and give
 * results within rounding of each other):
 *   0 = automatic (default): the panel kernel when the quadrature points come in groups of 8 consecutive
 *       points that share most of their supports (mean size of a group's union of supports <= 2 k and no
 *       union above 128 nodes: several Gauss points per background cell), else the row-owner kernel;
 *   1 = row-owner kernel (accumulators in registers, one lane per column slot);
 *   2 = panel kernel whenever its preprocessing fits (no union above 128 nodes);
 *   3 = the long-row kernel that rows of more than 1024 block columns take automatically (accumulators in
 *       shared memory, binary search of the column; for tests).
 * The panel kernel accumulates the upper blocks (column node >= row node) and fills the lower ones with the
 * transposes (K is symmetric block-wise, R8), so its K is bitwise symmetric.
 * Takes effect at the next rpim_build_pattern.  rpim_reduction_used: 1 or 2 for the current pattern
 * (0 before rpim_build_pattern).  rpim_reduction_params (host array of 10 ints; a report for benchmarks):
 * [0] kernel as rpim_reduction_used, [1] chunks of 32 entries per group union, [2] block rows per tile,
 * [3] consumer warps per row group, [4] ring stages, [5] most upper block columns of a row, [6] longest block
 * row, [7] 100 x mean size of a group's union of supports (0 when no statistics were taken), [8] block rows per
 * consumer warp group, [9] 1 when the groups' staged rows travel as a 2-D tensor copy of the gradient rows only. */
int rpim_set_reduction(rpim_ctx* ctx, int mode);
int rpim_reduction_used(const rpim_ctx* ctx);
int rpim_reduction_params(const rpim_ctx* ctx, int out[10]);

/* Tuning / test knob: force parts of the panel kernel's launch shape instead of the automatic choice (every
 * argument: 0 = automatic).  The result does not depend on it -- the order of summation per matrix entry is the
 * same for every shape -- only the speed does.  The library reads no environment variable.
 *   rows_per_tile    2, 4, 6 or 8 block rows per CTA tile (ignored when a row has more than 1024 upper columns)
 *   warps_per_group  1..4 consumer warps per row group (at most 3 with one row per group)
 *   rows_per_group   1 or 2 block rows per consumer warp group
 *   ring_stages      2..8 stages of the group ring
 *   staging          1 = gradient rows by a 2-D tensor copy (needs an even k <= 84), 2 = whole staged rows by a plain bulk copy
 *   tile_desc        1 = tile descriptors by one warp per tile, 2 = by one thread per tile
 * A shape that does not fit the shared memory falls back to the row-owner kernel (rpim_reduction_used tells).
 * Out-of-range values give RPIM_ERR_INVALID_ARG and change nothing.  Takes effect at the next
 * rpim_build_pattern / rpim_update_nodes; rpim_reduction_params reports the shape in use. */
int rpim_set_panel_shape(rpim_ctx* ctx, int rows_per_tile, int warps_per_group, int rows_per_group, int ring_stages,
                         int staging, int tile_desc);

/* Stage 0 (R1, R2; hot-path steps a1, a2): exact k-nearest-neighbour supports on a
 * uniform cell grid and the CSR pattern of the 3N x 3N stiffness matrix.
 *   d_nodes  N x 3 field-node coordinates        d_qpts  Nq x 3 quadrature points
 *   k        support size (4 <= k <= min(N, RPIM_MAX_K))
 *   index_bits  0 = auto (64 iff nnz > 2^31 - 1), 32 or 64: width of row_ptr AND col_idx;
 *               RPIM_INDEX_MIXED: row_ptr 64-bit, col_idx 32-bit
 *   out_nnz, out_index_bits  host scalars (number of stored scalar entries; chosen width: 32, 64 or RPIM_INDEX_MIXED)
 * Synchronises the stream. */
int rpim_build_pattern(rpim_ctx* ctx, const double* d_nodes, int64_t N, const double* d_qpts,
                       int64_t Nq, int k, int index_bits, int64_t* out_nnz, int* out_index_bits);

/* Moving nodes (the paper's motivation is large deformation): the
 * same N nodes at new coordinates d_nodes (and, if d_qpts is not NULL, the same Nq points at new coordinates).
 * The cell grid is updated incrementally (when no node left its cell only the cell-ordered coordinates are
 * refreshed, otherwise it is rebuilt), the supports are searched again and compared with the old table on the
 * device.  If no support changed the incidence lists, the CSR pattern and the reduction's slot maps are KEPT
 * (row_ptr / col_idx obtained earlier stay valid); otherwise they are rebuilt.  The result is in every case
 * identical, bit for bit, to a fresh rpim_build_pattern on the moved cloud with the same index width.
 *   out_changed_points   host: number of points whose support changed      (may be NULL)
 *   out_pattern_rebuilt  host: 1 if the pattern was rebuilt, 0 if kept     (may be NULL)
 *   out_nnz              host: stored scalar entries of the current pattern (may be NULL)
 * The new arrays replace the old ones in the lifetime rule above.  rpim_assemble must be called again
 * before anything that uses shape functions.  Synchronises the stream. */
int rpim_update_nodes(rpim_ctx* ctx, const double* d_nodes, const double* d_qpts, int64_t* out_changed_points,
                      int* out_pattern_rebuilt, int64_t* out_nnz);

/* Write the pattern built by rpim_build_pattern.
 *   d_row_ptr  3N+1 entries, d_col_idx  nnz entries, both int32_t or int64_t per index_bits (RPIM_INDEX_MIXED:
 *              d_row_ptr int64_t, d_col_idx int32_t; the same widths hold for h_row_ptr / h_col_idx of rpim_host_assemble)
 *   d_support  Nq x k int32 node ids, ascending per point; may be NULL
 * Any of the three may be NULL to skip it.  Asynchronous. */
int rpim_get_pattern(rpim_ctx* ctx, void* d_row_ptr, void* d_col_idx, int32_t* d_support);

/* Stage 1 (R3-R8; steps a3-a6): per quadrature point build and factor the
 * (k+4)x(k+4) moment matrix, solve for the shape functions and their derivatives, form
 * w * B^T D B and reduce it deterministically (fixed order, no floating-point atomics) into
 * the CSR values; body-force load f_{3I+c} = sum_q w phi_I b_c.
 *   d_qw    Nq quadrature weights           E, nu   isotropic elastic constants
 *   alpha_c, d_c, q   multiquadric R(r) = (r^2 + (alpha_c*d_c)^2)^q
 *   body    host array of 3 (force per unit volume)
 *   d_vals  nnz fp64 values (overwritten)   d_f  3N fp64 (overwritten)
 *   out_singular  host scalar: number of points whose moment matrix was singular (they
 *                 contribute nothing); may be NULL, in which case the call is asynchronous.
 * Singular points are REPORTED, not an error: the return value stays RPIM_OK (there is no
 * RPIM_ERR_SINGULAR_MOMENT; SURVEY.md section 8(b) proposed one), the caller decides from the count. */
int rpim_assemble(rpim_ctx* ctx, const double* d_qw, double E, double nu, double alpha_c,
                  double d_c, double q, const double body[3], double* d_vals, double* d_f,
                  int64_t* out_singular);

/* Strata with one Poisson ratio (R8b, part): a per-point modulus scale,
 * E_q = E * d_escale[q] for the stiffness contribution of quadrature point q in every later rpim_assemble (and the
 * stresses of rpim_recover_stress); the loads are not scaled.
 *   d_escale  Nq fp64 (DEVICE, caller-owned: must stay valid until replaced), or NULL to switch it off
 * Cleared by rpim_build_pattern (a new point set). */
int rpim_set_modulus_scale(rpim_ctx* ctx, const double* d_escale);

/* Step a5b (R9): f_{3I+c} += w * phi_I(x) * t_c at M given points (face Gauss
 * points of a traction boundary) using the shape parameters of the last rpim_assemble.
 *   d_pts M x 3, d_w M, d_t M x 3, d_f 3N (updated in place).  Synchronises the stream.
 * A load point whose support gives a singular moment matrix (e.g. k coplanar nodes on a face) would drop its
 * traction silently: the call then returns RPIM_ERR_SINGULAR_POINT (the other points' loads are in d_f). */
int rpim_add_point_loads(rpim_ctx* ctx, const double* d_pts, const double* d_w, const double* d_t,
                         int64_t M, double* d_f);

/* Stage 2 (R10; step a7): penalty method, in place.
 *   d_bc_nodes  m node ids, each at most once; an id that is out of range, listed twice or without a matrix
 *               row gives RPIM_ERR_BC_NODE_INVALID and NOTHING is applied (K and f unchanged)
 *   d_bc_mask   m bytes, bit c = constrain DOF c (NULL = all)
 *   d_u_bar     m x 3 prescribed displacements
 *   alpha, alpha_is_relative   alpha_used = alpha * max_d K_dd (before penalty) if relative
 *   out_alpha_used  host scalar, may be NULL
 * Synchronises the stream once (alpha and the validity of the list are read back); the penalty kernel
 * itself is enqueued after that and is asynchronous. */
int rpim_apply_penalty(rpim_ctx* ctx, const int64_t* d_bc_nodes, const uint8_t* d_bc_mask,
                       const double* d_u_bar, int64_t m, double alpha, int alpha_is_relative,
                       double* d_vals, double* d_f, double* out_alpha_used);

/* Stage 2 without any device allocation: same arguments, same checks and bitwise the same K, f and alpha_used as
 * rpim_apply_penalty, for callers that cannot let the library reach cudaMalloc at this point of their program:
 *   - a solver that has already handed (nearly) all of the GPU's memory to its own pool -- at the `stress`
 *     configuration K, col_idx and the staged shape functions take 174 of 180 GB, and a late cudaMalloc can fail;
 *   - a time-stepping or serving loop that runs other streams on the same device: cudaMalloc and cudaFree
 *     synchronise the whole device and would stall them;
 *   - several solver instances sharing one GPU under a device-memory budget that has to be accounted for byte by
 *     byte: what this call uses is fixed and known when the library is built.
 * rpim_apply_penalty takes its scratch memory (partial maxima of the diagonal, one bit per node for the
 * duplicate check, a counter) from the context's workspace and so may allocate; this call keeps the same scratch
 * in a fixed array inside the library image (about 0.5 MiB, held by every GPU that loads librpim until the
 * process exits) and calls no cudaMalloc, cudaFree or allocating library routine.
 *   Limit: at most RPIM_STATIC_PENALTY_MAX_NODES nodes in the context's pattern (rpim_apply_penalty_static_max_nodes
 *     returns the same number); a larger problem is refused with RPIM_ERR_CAPACITY and nothing is touched.  The
 *     length m of the boundary list is not limited.
 *   First call on a device: looks up the array's device address (once per device, with that device current) and
 *     may make the CUDA runtime load the library's kernels; make that first call during start-up, before any
 *     stream capture begins.
 *   Sharing: all contexts on a device use the one array, and it keeps the previous call's contents (the call
 *     clears what it needs to find at zero).  Two calls that overlap on the GPU -- different contexts or streams
 *     of one device -- race on it and give wrong results: serialise them.  Calls on different devices are
 *     independent.
 * Synchronises the stream once, like rpim_apply_penalty. */
#define RPIM_STATIC_PENALTY_MAX_NODES 4194304
int rpim_apply_penalty_static(rpim_ctx* ctx, const int64_t* d_bc_nodes, const uint8_t* d_bc_mask,
                              const double* d_u_bar, int64_t m, double alpha, int alpha_is_relative,
                              double* d_vals, double* d_f, double* out_alpha_used);
int64_t rpim_apply_penalty_static_max_nodes(void);

/* Stage 3 ("solve the system ... then the stresses").
 *
 * rpim_matvec: y = K x with K in the layout rpim_assemble / rpim_apply_penalty leave in d_vals (the
 * pattern is the context's).  d_x, d_y: 3N fp64.  Asynchronous.
 *
 * rpim_solve_pcg: conjugate gradients with block-Jacobi preconditioning (inverse of the 3x3 diagonal block of every
 * node) on the penalised K,
 * which is symmetric positive definite (R10).  d_u holds the initial guess on entry and
 * the solution on exit (3N).  Stops when the residual recurrence reaches rel_tol * ||f||_2 (looked at every
 * 25 iterations) or after max_iter iterations; out_iters (host, may be NULL) and out_rel_resid (host, may
 * be NULL) report what was reached, out_rel_resid being the TRUE ||f - K u||_2 / ||f||_2 of the returned
 * iterate, recomputed with one more product -- not converging is not an error.  If p^T K p <= 0 or is not
 * finite (K is not positive definite: singular points, unconstrained components) the iteration stops at
 * the next look and RPIM_ERR_BREAKDOWN is returned, outputs filled.  f = 0 returns u = 0; a load vector that is
 * not finite (NaN, Inf) also returns RPIM_ERR_BREAKDOWN, with d_u untouched.  All reductions
 * have a fixed order: the iterates are bitwise reproducible.  Synchronises the stream.
 *
 * rpim_recover_stress: sigma = D B u at every quadrature point of the last rpim_assemble (its staged
 * shape-function gradients), Voigt order xx yy zz xy yz zx, d_sigma Nq x 6 fp64.  Asynchronous. */
int rpim_matvec(rpim_ctx* ctx, const double* d_vals, const double* d_x, double* d_y);
int rpim_solve_pcg(rpim_ctx* ctx, const double* d_vals, const double* d_f, double* d_u, double rel_tol,
                   int max_iter, int* out_iters, double* out_rel_resid);
int rpim_recover_stress(rpim_ctx* ctx, const double* d_u, double E, double nu, double* d_sigma);

/* Test / inspection accessor: shape functions staged by the last rpim_assemble.
 *   d_phi Nq x k, d_dphi Nq x 3 x k (d/dx, d/dy, d/dz), d_singular Nq bytes; any may be NULL. */
int rpim_get_shape(rpim_ctx* ctx, double* d_phi, double* d_dphi, uint8_t* d_singular);

/* End-to-end variants with HOST buffers (pageable or pinned): copy inputs to the device,
 * run the same kernels, copy results back, all on the context's stream, then synchronise.
 * rpim_host_pattern builds the pattern and reports nnz so the caller can size the outputs of
 * rpim_host_assemble, which runs get_pattern + assemble + apply_penalty and returns the CSR
 * arrays, values and load vector.  bc arrays may be NULL with m = 0. */
int rpim_host_pattern(rpim_ctx* ctx, const double* h_nodes, int64_t N, const double* h_qpts,
                      int64_t Nq, int k, int index_bits, int64_t* out_nnz, int* out_index_bits);
int rpim_host_assemble(rpim_ctx* ctx, const double* h_qw, double E, double nu, double alpha_c,
                       double d_c, double q, const double body[3], const int64_t* h_bc_nodes,
                       const uint8_t* h_bc_mask, const double* h_u_bar, int64_t m, double alpha,
                       int alpha_is_relative, void* h_row_ptr, void* h_col_idx, double* h_vals,
                       double* h_f, int64_t* out_singular, double* out_alpha_used);

/* Per-phase device times (ms, CUDA events) of the last rpim_build_pattern / rpim_assemble:
 * [0] grid+kNN  [1] incidence  [2] block pattern  [3] shape functions  [4] reduction into CSR.
 * Host array of 5.  Synchronises. */
int rpim_last_phase_ms(rpim_ctx* ctx, float out_ms[5]);

/* Sum of the per-phase device times (ms, same five phases) over all rpim_build_pattern /
 * rpim_assemble calls since the last reset, measured with CUDA events recorded on the context's
 * stream around the kernels; out_calls = {build_pattern calls, assemble calls} (may be NULL).
 * Synchronises.  reset != 0 clears the totals afterwards. */
int rpim_phase_totals(rpim_ctx* ctx, double out_ms[5], int64_t out_calls[2], int reset);

/* Measurement aid for the roofline denominator: sustained FP64 fused multiply-add
 * rate of the device, eight independent chains per thread on every SM, no memory traffic; best of three
 * launches after a warm-up.  out_tflops (host, fma = 2 flops), out_ms (host, may be NULL) = duration of the
 * best launch.  Synchronises the stream. */
int rpim_probe_fp64(rpim_ctx* ctx, double* out_tflops, double* out_ms);

/* The same measurement for the FP64 tensor-core instruction sm_100a has (warp-level mma.sync m8n8k4; tcgen05 has no
 * FP64 kind): eight independent accumulator chains per warp, 2 x 8 x 8 x 4 flops per instruction.  It answers SURVEY.md
 * section 8(d) "measure DMMA against DFMA" for the B^T D B contraction; DESIGN.md section 5 has the outcome. */
int rpim_probe_fp64_dmma(rpim_ctx* ctx, double* out_tflops, double* out_ms);

/* Number of kernels this library has launched on the context since creation. */
int64_t rpim_launch_count(const rpim_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* RPIM_H */
