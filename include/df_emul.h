/* df_emul.h -- C-ABI boundary of libdfemul.so (NVIDIA B200, sm_100a only).
 *
 * The density-fitting (DF) Coulomb/exchange build of an SCF iteration with the
 * two exchange contractions run as FP64 GEMMs emulated by INT8 tensor-core
 * products (arXiv 2601.08077; citations are lines of the paper text PAPER.md).
 *
 *   rho_q  = sum_ij B^q_ij D_ij                PAPER.md:45   (Eq. 3)   FP64
 *   J_ij   = sum_q  B^q_ij rho_q               PAPER.md:47   (Eq. 4)   FP64
 *   X^q_ia = sum_j  B^q_ij C_ja                PAPER.md:49-51 (Eq. 5; blocked Eq. 12)  emulated
 *   K_ij   = sum_q sum_a X^q_ia X^q_ja         PAPER.md:53   (Eq. 6; blocked Eq. 13) emulated
 *
 * Emulation ("fixed point ... Ozaki scheme", s = ceil((m_emu+1)/8)
 * INT8 splits; s(s+1)/2 INT8 GEMMs).  Every detail the paper leaves
 * open is fixed in DESIGN.md section 2 (readings R1..R13).
 *
 * Conventions for EVERY entry point
 *  - All data pointers are DEVICE pointers to contiguous row-major arrays unless
 *    the argument is documented as "host".  The caller owns every buffer; the
 *    library only reads inputs, only writes outputs and its workspace, and keeps
 *    no reference to caller memory after the call's work has run.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the default stream).
 *    Work is enqueued on it; no entry point synchronises with the host unless it
 *    says so.  Results are valid once the stream has reached the end of the call.
 *  - Scratch memory comes from a caller-supplied workspace.  A CONTEXT (df_context_create) binds one
 *    workspace on one device together with its policy mode, debug knobs and cached tensor maps; one
 *    context serves one stream at a time, and several contexts (each with its own workspace) may run
 *    concurrently on several streams.  The entry points without a context argument use a process-wide
 *    default context whose workspace is registered with df_set_workspace().  A call made while another
 *    device is current than the one the workspace was registered on returns DF_ERR_DEVICE.
 *  - Return value: DF_OK (0) or a negative DF_ERR_* code.  No exceptions, no
 *    printing.  Data-dependent faults (Inf/NaN, out-of-range magnitudes) do not
 *    fail the call: they set bits in a device status word, see df_last_status().
 *  - There is no CPU fallback: on a machine without an sm_100 device every
 *    compute entry point returns DF_ERR_DEVICE.
 */
#ifndef DF_EMUL_H_
#define DF_EMUL_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DF_OK             0
#define DF_ERR_NULL      -1  /* a required pointer is NULL                    */
#define DF_ERR_DIM       -2  /* a dimension is <= 0 or too large              */
#define DF_ERR_TOL       -3  /* tol <= 0 or NaN, or slice count not in 1..8   */
#define DF_ERR_WORKSPACE -4  /* no workspace registered, or it is too small   */
#define DF_ERR_DEVICE    -5  /* no CUDA device of compute capability 10.x     */
#define DF_ERR_CUDA      -6  /* a CUDA runtime / driver call failed           */
#define DF_ERR_ALIGN     -7  /* a pointer is not 16-byte aligned              */
#define DF_ERR_TOO_LARGE -8  /* df_emul_gemm_static: the problem needs more scratch than the built-in array holds */

#define DF_MODE_NOMINAL 0    /* tol -> s exactly as Table 1 */
#define DF_MODE_GUARDED 1    /* one extra byte of margin (R7); default   */

#define DF_STATUS_NONFINITE 1 /* an Inf/NaN was seen in an emulated operand   */
#define DF_STATUS_RANGE     2 /* a row/column maximum outside [2^-450, 2^450] */

/* ---- policy (host only, no device needed) ------------------------------- */

/* Slice count s in 1..8 for a target relative Frobenius error `tol`
 * (PAPER.md:130 s = ceil((m_emu+1)/8); R7).  mode = DF_MODE_*.
 * Returns DF_ERR_TOL for tol <= 0 or NaN. */
int df_slices_for_tol(double tol, int mode);

/* Number of INT8 slice-pair products for s slices: s(s+1)/2. */
int df_num_int8_gemms(int s);

/* Largest contraction length accumulated in INT32 before a flush to FP64:
 * 32*floor(131071/(32 s))  (R4). */
int df_kflush(int s);

/* Select the tol -> s mapping used by df_emul_gemm / df_jk_build (default context). */
int df_set_policy_mode(int mode);

/* ---- workspace ---------------------------------------------------------- */

/* Bytes of workspace df_emul_gemm needs for these sizes (s slices). */
int64_t df_emul_gemm_workspace_bytes(int64_t m, int64_t n, int64_t k, int s);

/* Minimum bytes of workspace df_jk_build needs (s slices, naux processed in
 * blocks of 512, BASELINE.json config 4).  A larger workspace lets the library
 * batch several 512-blocks per launch. */
int64_t df_jk_workspace_bytes(int64_t nao, int64_t naux, int64_t nocc, int s);

/* Bytes needed to batch `nblocks` 512-q blocks per launch (nblocks >= ceil(naux/512)
 * = the whole auxiliary range in one super-block). */
int64_t df_jk_workspace_bytes_blocks(int64_t nao, int64_t naux, int64_t nocc, int s, int64_t nblocks);

/* Register a device buffer (256-byte aligned, on the current device) as the workspace of the
 * default context.  The library never frees it.  Passing NULL/0 unregisters it. */
int df_set_workspace(void* ptr, int64_t bytes);

/* ---- contexts: one workspace per concurrent stream ---------- */

typedef struct df_context df_context;

/* Creates a context on the CURRENT device with `workspace` (device memory, 256-byte aligned, `bytes`
 * long, owned by the caller and never freed by the library) and the default policy mode.  *ctx (host)
 * receives the handle.  DF_ERR_DEVICE without an sm_100 device. */
int df_context_create(void* workspace, int64_t bytes, df_context** ctx);
/* Frees the handle (not the workspace).  The caller synchronises its stream first. */
int df_context_destroy(df_context* ctx);
int df_context_set_policy_mode(df_context* ctx, int mode);
/* The knobs of df_debug_set_gemm_flags, for this context. */
int df_context_set_debug_flags(df_context* ctx, int flags);
/* The entry points below with a context in front; same arguments, same results (bit for bit). */
int df_context_emul_gemm(df_context* ctx, const double* A, const double* B, double* C,
                         int64_t m, int64_t n, int64_t k, double tol, void* stream);
int df_context_emul_gemm_slices(df_context* ctx, const double* A, const double* B, double* C,
                                int64_t m, int64_t n, int64_t k, int s, void* stream);
int df_context_jk_build(df_context* ctx, const double* B_packed, int64_t nao, int64_t naux,
                        const double* C_occ, int64_t nocc, const double* D,
                        double tol, double* J, double* K, void* stream);
int df_context_jk_build_slices(df_context* ctx, const double* B_packed, int64_t nao, int64_t naux,
                               const double* C_occ, int64_t nocc, const double* D,
                               int s, double* J, double* K, void* stream);
int df_context_jk_plan_create(df_context* ctx, const double* B_packed, int64_t nao, int64_t naux, int smax,
                              void* plan, int64_t plan_bytes, void* stream);
int df_context_jk_build_planned(df_context* ctx, const void* plan, int smax, const double* B_packed,
                                int64_t nao, int64_t naux, const double* C_occ, int64_t nocc,
                                const double* D, double tol, double* J, double* K, void* stream);
int df_context_jk_build_planned_slices(df_context* ctx, const void* plan, int smax, const double* B_packed,
                                       int64_t nao, int64_t naux, const double* C_occ, int64_t nocc,
                                       const double* D, int s, double* J, double* K, void* stream);
int df_context_last_status(df_context* ctx, void* stream, int* status);
int df_context_screen_stats(df_context* ctx, void* stream, int64_t* active, int64_t* total);

/* ---- the two mandated entry points (default context) --------------------- */

/* C = A . B emulated with s = df_slices_for_tol(tol) INT8 slices.
 * A: m x k, B: k x n, C: m x n, all FP64 row-major, device.  C is overwritten.
 * ||C_emul - A.B||_F / ||A.B||_F <= tol is the contract (guarded mode). */
int df_emul_gemm(const double* A, const double* B, double* C,
                 int64_t m, int64_t n, int64_t k, double tol, void* stream);

/* One DF J/K build.
 * B_packed: npair x naux FP64, npair = nao(nao+1)/2, q fastest, row
 *           p = i(i+1)/2 + j holds B^q_ij for i >= j   (BASELINE.json config 0).
 * C_occ: nao x nocc.  D: nao x nao, read as symmetric (0.5 (D + D^T)).
 * J, K: nao x nao outputs, both triangles written, exactly symmetric.
 * J is plain FP64; K = sum_q X^q X^q^T (no occupation factor,
 * PAPER.md:53) is emulated with s = df_slices_for_tol(tol) in both GEMMs.
 * Every reduction has a fixed order: the same inputs and s give the same bits
 * on every call, whatever the workspace size. */
int df_jk_build(const double* B_packed, int64_t nao, int64_t naux,
                const double* C_occ, int64_t nocc, const double* D,
                double tol, double* J, double* K, void* stream);

/* ---- df_emul_gemm without a workspace: for callers that cannot allocate device memory ---- */

/* df_emul_gemm (same arguments, same bits in C, tol -> s by the default context's policy mode) that needs
 * NO workspace and allocates no device memory: no cudaMalloc / cudaFree / cudaMallocAsync, here or in
 * anything it calls.  Every other compute entry point takes its scratch from a workspace the caller
 * allocated; this one is for the callers that cannot allocate --
 *   - an SCF driver that committed all of HBM (B, the plan, its own pool) at start-up,
 *   - a callback invoked while its stream is being captured, where cudaMalloc is forbidden,
 *   - a host thread next to other contexts' running builds, which cudaMalloc would stall
 *     (it synchronises the whole device).
 * The caller still owns and passes A, B and C (device, FP64, row-major, as for df_emul_gemm).
 *
 * The scratch (digit planes, scale indices, column maxima, status words) is a fixed array of
 * df_emul_gemm_static_scratch_bytes() = 64 MiB inside the library's device image.  Every GPU on which
 * the library is used holds that array until the process exits, called or not.
 *   LIMIT   the problem must satisfy df_emul_gemm_workspace_bytes(m, n, k, s) <= 64 MiB, about
 *           s (m + n) round_up(k, 32) bytes: 2048^3 up to s = 7, 1024 x 1024 x 3000 at s = 8.  Beyond it the
 *           call returns DF_ERR_TOO_LARGE before touching the GPU; C is not written.
 *   SHARED  all calls on one device use the same array.  Calls on ONE stream are ordered and safe.  Two
 *           calls that may overlap on the GPU (two streams, two host threads) race on it and give
 *           garbage: serialise them, or give the second caller a context with a workspace.  The array
 *           keeps the previous call's contents; the call clears, in stream order, the one part that must
 *           start at zero (the column maxima) and overwrites the rest, so a call never sees another's data.
 *   SET-UP  the FIRST call on each device looks the array's address up on that device (with the device
 *           current), clears its status words with a synchronous cudaMemset and creates a small host-side
 *           tensor-map cache.  Make that first call outside any stream capture.
 *   STATUS  DF_STATUS_* bits this entry point raises are kept in the array and not reported by
 *           df_last_status(); validate the operands yourself if Inf/NaN can occur.
 * Returns DF_ERR_TOO_LARGE as above, otherwise what df_emul_gemm returns. */
int df_emul_gemm_static(const double* A, const double* B, double* C,
                        int64_t m, int64_t n, int64_t k, double tol, void* stream);
/* The size of that array in bytes (host only, no device needed). */
int64_t df_emul_gemm_static_scratch_bytes(void);

/* ---- plan: B split once for a whole SCF --- */

/* B is computed once and is constant over the SCF; its row scales
 * and INT8 digit planes do not depend on C_occ, D or tol, and the planes have the
 * prefix property (R3: a build with s slices reads the first s of smax
 * planes).  A plan is a caller-owned device buffer (256-byte aligned) of
 * df_jk_plan_bytes() bytes holding them: naux x nao x (8 + round_up(nao,128) x smax)
 * bytes plus the tile maxima of the screening mask (4 bytes per 32 x 32 tile pair and q),
 * 37 GB at config 3 with smax = 6.  df_jk_plan_create() fills it (row maxima
 * + unpack + split of all q, the H2 row of SURVEY.md section 8(a)); of the registered
 * workspace it uses the status words and, when it is large enough (4 bytes per 256 rows
 * (q, i) and 32 K blocks behind the first 256 bytes), room for the screening mask at smax
 * slices.  DF_ERR_WORKSPACE if plan_bytes is too small. */
int64_t df_jk_plan_bytes(int64_t nao, int64_t naux, int smax);
int df_jk_plan_create(const double* B_packed, int64_t nao, int64_t naux, int smax,
                      void* plan, int64_t plan_bytes, void* stream);

/* Workspace of a planned build (no GEMM(5) operand planes in it), nblocks as in
 * df_jk_workspace_bytes_blocks. */
int64_t df_jk_planned_workspace_bytes(int64_t nao, int64_t naux, int64_t nocc, int s, int64_t nblocks);

/* df_jk_build with GEMM(5)'s left operand read from `plan` (created from the same
 * B_packed, nao, naux with `smax` planes; the library cannot check that).  B_packed
 * is still read for rho and J (plain FP64).  Bit-identical to
 * df_jk_build.  DF_ERR_TOL if the slice count exceeds smax.  Status bits that B
 * causes (Inf/NaN, range) are raised by df_jk_plan_create, not again per build. */
int df_jk_build_planned(const void* plan, int smax, const double* B_packed, int64_t nao, int64_t naux,
                        const double* C_occ, int64_t nocc, const double* D,
                        double tol, double* J, double* K, void* stream);
int df_jk_build_planned_slices(const void* plan, int smax, const double* B_packed, int64_t nao, int64_t naux,
                               const double* C_occ, int64_t nocc, const double* D,
                               int s, double* J, double* K, void* stream);

/* Same two calls with a forced slice count s in 1..8 (config 1's sweep). */
int df_emul_gemm_slices(const double* A, const double* B, double* C,
                        int64_t m, int64_t n, int64_t k, int s, void* stream);
int df_jk_build_slices(const double* B_packed, int64_t nao, int64_t naux,
                       const double* C_occ, int64_t nocc, const double* D,
                       int s, double* J, double* K, void* stream);

/* Copies the device status word (OR of DF_STATUS_* bits since the last call of
 * this function) to *status (host) and clears it.  SYNCHRONISES `stream`. */
int df_last_status(void* stream, int* status);

/* Screening ("N_scr <= N_bf^2", PAPER.md:164 grouped GEMM).
 * Every J/K build judges, from the row scales and the maxima of 32 x 32 tiles its first pass over B
 * leaves, which (256 rows (q, i), 128 columns j) blocks of GEMM(5)'s left operand hold no non-zero digit
 * at the build's slice count (every |B^q_ij| below 2^(e_qi - 8 s - 1)); those blocks are neither written by
 * the unpack pass nor loaded or multiplied by GEMM(5).  Only exact zeros are skipped: J and K are the
 * dense results bit for bit.  *active / *total (host) receive the number of active and of all such
 * blocks summed over the builds (and plan creations) since the last call; the counters are cleared.
 * SYNCHRONISES `stream`.  N_scr / N_bf^2 of the paper's FLOP model ~ active / total. */
int df_screen_stats(void* stream, int64_t* active, int64_t* total);

/* ---- debug exports (tests only; not on the timed path) ------------------ */

/* Row split (R2, steps 1-3): X is rows x cols FP64.  Writes
 * e[rows] (int32 scale index) and planes[t][row][pitch] (int8, t = 0..s-1 is
 * digit d_{t+1}); pitch = df_plane_pitch(cols); bytes past `cols` are zero. */
int df_debug_split_rows(const double* X, int64_t rows, int64_t cols, int s,
                        int32_t* e, int8_t* planes, void* stream);

/* Column split of a k x n matrix: scale per column; planes[t][col][pitch]
 * hold the TRANSPOSED digits (contraction index fastest), pitch = df_plane_pitch(k). */
int df_debug_split_cols(const double* X, int64_t k, int64_t n, int s,
                        int32_t* e, int8_t* planes, void* stream);

/* Row pitch in bytes of a digit plane with `cols` contraction elements. */
int64_t df_plane_pitch(int64_t cols);

/* INT32 weight sums of one flush chunk, straight from TMEM:
 * P[w-2][i][j] = sum_{t+u=w} sum_{kk in chunk} DA_t[i,kk] DB_u[j,kk], w = 2..s+1,
 * chunk = [chunk*df_kflush(s), min(k, (chunk+1)*df_kflush(s))).
 * DA: [s][m][pitch] int8, DB: [s][n][pitch] int8 (pitch = df_plane_pitch(k)).
 * P: [s][m][n] int32.  With s = 1 this is one slice-pair product P^(1,1).
 * bk selects the shared-memory swizzle / K-block width in bytes (32, 64, 128;
 * 0 = the library's choice). */
int df_debug_weight_sums(const int8_t* DA, const int8_t* DB,
                         int64_t m, int64_t n, int64_t k, int s, int chunk,
                         int bk, int32_t* P, void* stream);

/* df_jk_build_slices that also exports GEMM(5)'s FP64 output
 * X[q][i][a_pad] (a_pad = 16*ceil(nocc/16), padded columns are zero) and the
 * GEMM(6) scale indices e6[g][i] of every q-group g (R5).  X_out /
 * e6_out may be NULL.  *ngroups_out (host) receives the number of groups. */
int df_debug_jk_build(const double* B_packed, int64_t nao, int64_t naux,
                      const double* C_occ, int64_t nocc, const double* D,
                      int s, double* J, double* K,
                      double* X_out, int32_t* e6_out, int* ngroups_out, void* stream);

/* Knobs for timing experiments and for forcing the alternative code paths in tests; 0 = the
 * library's own choices.  Results stay correct except with bits 0, 1, 4, 5.
 *   bit 0      GEMM issues no MMAs (operand feed only)        bit 1  GEMM issues no TMA loads
 *   bit 2      GEMM(5) keeps one N tile of a_pad columns      bit 3  multi-pass tiles keep the FP64
 *                                                                    running sum in global memory
 *   bit 4 / 5  unpack kernel writes nothing / reads nothing   bit 6  GEMM(5) N halves without the
 *                                                                    cluster-pair multicast
 *   bits 8-15  force the K-block width in bytes (32, 64, 128) bits 16-19 MMA probe: operand tiles
 *   bit 20     no cta_group::2 pair tiles                            walked (2 bits), swizzle (2 bits)
 *   bit 22     GEMM(5) N halves on multicast CTA pairs, never on MMA pairs
 *   bit 23     GEMM epilogue moves FP64 through the staged 16-byte path, never 256-bit accesses
 *   bit 24     df_emul_gemm keeps 128-column tiles at s <= 3 (default: 256 columns at s <= 2, 160 at s = 3)
 *   bit 25     no screening: every K block of GEMM(5) is written, loaded and multiplied (plain builds and
 *              plan creation; a planned build always screens, its plan may hold the active blocks only) */
int df_debug_set_gemm_flags(int flags);

/* Number of GPU kernels this library has launched in this process. */
int64_t df_launch_count(void);

/* Per-kernel-class device timing for the roofline report (bench.py); process-wide: while it is on,
 * the brackets of all contexts and host threads land in the same per-class sums (the records are
 * guarded by a mutex; enable / read it from one thread).  While
 * enabled, every entry point brackets each kernel class it launches with a pair
 * of CUDA events on the caller's stream.  df_profile_read() SYNCHRONISES on the
 * recorded events, returns the summed milliseconds and the number of brackets
 * per class since the last read in ms_by_class[df_profile_num_classes()] /
 * count_by_class[...] (host arrays), and clears the records. */
int df_profile_enable(int on);
int df_profile_num_classes(void);
const char* df_profile_class_name(int cls);
int df_profile_read(float* ms_by_class, int* count_by_class);

/* Back-to-back tcgen05.mma.kind::i8 issue-rate probe (operands resident in
 * shared memory, no loads): runs `iters` MMAs of shape 128 x n_mma x 32 per CTA
 * on every SM.  Returns the launch's device time in milliseconds in *ms (host);
 * INT8 op/s = 2*128*n_mma*32*iters*grid / time.  Synchronises.  n_mma may carry
 * a number of issuing warps w (1..4, 2*w*N <= 512) in bits 16+: N | w << 16, each
 * issuing `iters` MMAs into its own accumulators (measured: more issuers do not
 * raise the rate; an MMA of M = 128 takes max(~50, N/2 + 3) cycles).  Bit 24 set
 * (N % 32 == 0, grid >= 2): the same on SM pairs, cta_group::2 MMAs of M = 256. */
int df_debug_mma_peak(int n_mma, int iters, int grid, float* ms, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* DF_EMUL_H_ */
