// internal.h -- host-side launch interfaces between the translation units of libdfemul.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dfe {

constexpr int kMaxSlices = 8;
constexpr int kTileM = 128;

inline int64_t round_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }
inline int64_t plane_pitch(int64_t cols) { return round_up(cols, 32); }
inline int kflush_for(int s) { return 32 * (131071 / (32 * s)); }

void count_launch(int n = 1);

// q-groups of GEMM(6) (R5): q is cut into blocks of 512, every block into runs of
// QG = floor(KFLUSH(s) / nocc) consecutive q (one group's |g| nocc contraction elements fit one INT32
// chunk).  In planes6 a q owns a_pad = pad16(nocc) columns (the padding columns are zero digits) and
// every group starts at a multiple of 32 columns -- the K extent of one MMA -- with zero bytes
// between the end of a group and the start of the next, so no MMA ever straddles two groups.
constexpr int kQBlock = 512;  // BASELINE.json config 4: "naux blocks of 512"
struct GroupGeom {
  int QG, gpb, a_pad;
  int wfull;   // padded column width of a full group
  int wblock;  // padded column width of a full 512-q block
};
inline GroupGeom group_geom(int s, int nocc) {
  GroupGeom g;
  g.a_pad = (int)round_up(nocc, 16);
  g.QG = kflush_for(s) / nocc;
  if (g.QG < 1) g.QG = 1;
  if (g.QG > kQBlock) g.QG = kQBlock;
  g.gpb = (kQBlock + g.QG - 1) / g.QG;
  g.wfull = (int)round_up((int64_t)g.QG * g.a_pad, 32);
  g.wblock = (g.gpb - 1) * g.wfull + (int)round_up((int64_t)(kQBlock - (g.gpb - 1) * g.QG) * g.a_pad, 32);
  return g;
}
// number of groups of nq consecutive q (a super-block starts at a multiple of 512)
inline int group_count(const GroupGeom& g, int nq) {
  return (nq / kQBlock) * g.gpb + ((nq % kQBlock) + g.QG - 1) / g.QG;
}
// first q of group gi; first planes6 column of group gi (gi == ng: the end)
__host__ __device__ inline int group_q0(const GroupGeom& g, int gi) { return (gi / g.gpb) * 512 + (gi % g.gpb) * g.QG; }
__host__ __device__ inline int group_col(const GroupGeom& g, int gi, int nq, int ng) {
  if (gi < ng) return (gi / g.gpb) * g.wblock + (gi % g.gpb) * g.wfull;
  const int last = ng - 1;
  const int q0 = (last / g.gpb) * 512 + (last % g.gpb) * g.QG;
  const int w = (nq - q0) * g.a_pad;
  return (last / g.gpb) * g.wblock + (last % g.gpb) * g.wfull + (w + 31) / 32 * 32;
}

// What a launch needs beyond its problem; owned by a context (api.cu), one per concurrent stream.
struct TmapCache;  // gemm_i8.cu: tensor maps of the GEMM operands, keyed by (pointer, shape, box)
TmapCache* tmap_cache_create();
void tmap_cache_destroy(TmapCache* c);
struct LaunchEnv {
  int num_sms = 0;
  int flags = 0;               // df_debug_set_gemm_flags / df_context_set_debug_flags bits
  TmapCache* tmaps = nullptr;  // may be null: every launch encodes its maps
};

// ---- tmap.cu ---------------------------------------------------------------
// cuTensorMapEncodeTiled through the runtime's driver entry point (libcuda is not linked).
// dtype: 0 = UINT8, 1 = FLOAT64; swizzle: 0 (none), 32, 64, 128 bytes.  dims/box: rank entries,
// strides: rank - 1 entries in bytes (dimension 0 is contiguous).  map: a CUtensorMap (128 bytes).
bool encode_tensor_map(void* map, int dtype, int rank, const void* base, const uint64_t* dims,
                       const uint64_t* strides, const uint32_t* box, int swizzle);

// ---- split.cu -------------------------------------------------------------
// rows x cols FP64 (leading dimension ld) -> e[rows], planes[t][rows][pitch].
// num_sms: LaunchEnv::num_sms of the calling context (0: the launcher asks the runtime).
cudaError_t launch_split_rows(const double* X, int64_t rows, int64_t cols, int64_t ld, int s, int32_t* e,
                              int8_t* planes, int64_t pitch, int64_t plane_stride, int* status,
                              cudaStream_t st, int num_sms = 0);
// k x n FP64 row-major -> e[n] (scratch cmax[n] uint32), planes[t][n][pitch] transposed.
cudaError_t launch_split_cols(const double* X, int64_t k, int64_t n, int s, uint32_t* cmax, int32_t* e,
                              int8_t* planes, int64_t pitch, int64_t plane_stride, int* status,
                              cudaStream_t st);

// ---- gemm_i8.cu -----------------------------------------------------------
enum EpiMode { kEpiC = 0, kEpiX = 1, kEpiInt32 = 2 };

struct GemmProblem {
  // operands: digit planes [plane][rows][pitch] int8, contraction index fastest
  const int8_t* A;
  const int8_t* B;
  int64_t a_rows, b_rows;        // rows of the A planes (output rows), of the B planes (output cols)
  int64_t k;                     // contraction extent (tensor-map K dimension)
  int64_t a_pitch, b_pitch;      // bytes per row
  int64_t a_plane_stride, b_plane_stride;  // bytes between planes
  int s;                         // slices
  int n_tile;                    // output columns per CTA tile (multiple of 16, <= 256)
  int bk;                        // K-block bytes = swizzle span: 32, 64, 128 (0 = auto)
  // z items (q-groups): item z contracts K range [zk[z], zk[z+1]) (device int array of nz+1; every
  // entry a multiple of 32, the K extent of one MMA, and every item ONE flush chunk: at most
  // kflush(s) of its contraction elements are not zero padding), or the whole [0, k) when
  // zk == nullptr (then nz must be 1), cut into flush chunks of kflush(s) contraction elements.
  int nz;
  const int* zk;
  const int32_t* eA;  // scale indices, eA[z * ea_stride + row]
  const int32_t* eB;
  int64_t ea_stride, eb_stride;
  int pair;           // 1: 256-row tiles on CTA pairs with cta_group::2 MMAs (n_tile 128, FP64 C output)
  int cluster_n;      // 2: CTA pairs over the two N tiles share the A operand by TMA multicast
  int lower_only;     // 1: skip tiles strictly above the block diagonal (GEMM(6))
  int mode;           // EpiMode
  // kEpiC: C[z * c_stride + row * ldc + col] (FP64)
  double* C;
  int64_t ldc, c_stride;
  // kEpiX: row r = (q, i) = (r / nao, r % nao); X[r * ldx + col] (ldx = a_pad); running max of the
  // upper word of |X| per (group of q, i): xmax[qgroup[q] * nao + i]
  int nao;
  int x_cols;       // columns of X per q (a_pad); the N tiles of GEMM(5) cut this range
  int acc_stride;   // TMEM columns between weight accumulators (0 = n_tile rounded up to 32)
  int64_t ldx;
  const int* qgroup;
  uint32_t* xmax;
  // screening (kEpiX; may be null): kmask[(row / 256) * kmask_words + J / 32] bit J % 32 = the K block
  // of columns 128 J .. 128 J + 127 of the 256-row block is active; inactive blocks are neither
  // loaded nor multiplied (their planes need not exist)
  const uint32_t* kmask;
  int kmask_words;
  // kEpiInt32: P[(w - 2) * a_rows * b_rows + row * b_rows + col] of flush chunk `dbg_chunk`
  int32_t* P;
  int dbg_chunk;
};

cudaError_t launch_gemm_i8(const GemmProblem& g, const LaunchEnv& env, cudaStream_t st);
void set_peak_tiles(int n);  // probe walks n distinct operand tiles (1 = the same tile every MMA)
cudaError_t launch_mma_peak(int n_mma, int iters, int grid, float* ms, cudaStream_t st);

// ---- jk.cu ----------------------------------------------------------------
// pass A over packed B: rho[q] (through rho_part[jk_rho_part_rows(nao)][naux], every element of
// which is written, summed in a fixed order) and emax[i * naux + q] = upper word of max_j |B^q_ij|
// (atomicMax, must be zeroed).  rho == nullptr: the maxima alone (df_jk_plan_create); emax == nullptr:
// rho alone, lower tiles only (planned builds).
int64_t jk_rho_part_rows(int nao);
// tilemax (may be null; only with emax): [jk_rho_part_rows(nao)][naux], upper word of the maximum of
// every 32 x 32 tile pair and q (every element written) -- the input of the screening mask
cudaError_t launch_jk_pass_a(const double* Bp, int nao, int naux, const double* D, double* rho_part, double* rho,
                             uint32_t* emax, uint32_t* tilemax, cudaStream_t st);
// screening mask of the 256-row blocks of the flattened rows (q - q0, i), q in [q0, q0 + nq):
// mask[block][screen_mask_words(nao)], bit J = K block of columns 128 J .. may hold a non-zero digit at s
// slices; stats[0] / stats[1] += active / all (block, K block) pairs
inline int screen_mask_words(int64_t nao) { return (int)(((nao + 127) / 128 + 31) / 32); }
cudaError_t launch_jk_screen_mask(const uint32_t* emax, const uint32_t* tilemax, int nao, int naux, int q0, int nq,
                                  int s, uint32_t* mask, unsigned long long* stats, cudaStream_t st);
// J_packed[p] = sum_q B[p, q] rho[q]
cudaError_t launch_jk_j_gemv(const double* Bp, int64_t npair, int naux, const double* rho, double* Jp,
                             cudaStream_t st);
// unpack + split q in [q0, q1): planes5[t][(q - q0) * nao + i][pitch], e5[(q - q0) * nao + i]
// dbg (timing experiments): bit 0 = the kernel writes nothing, bit 1 = reads nothing
// kmask (may be null): screening mask of [q0, q1); planes of inactive (256-row block, K block) pairs are
// not written (and, where Eq. 4 does not ride on the block, not read)
cudaError_t launch_jk_unpack_split(const double* Bp, int nao, int naux, int q0, int q1, const uint32_t* emax,
                                   int s, int32_t* e5, int8_t* planes5, int64_t pitch, int64_t plane_stride,
                                   int* status, const double* rho, double* jpart, int dbg, const uint32_t* kmask,
                                   int mask_words, cudaStream_t st);
// jpart (may be null): [chunk of 32 q, counted from q0][npair] partials of Eq. 4; J_p = their sum in order
cudaError_t launch_jk_j_reduce(const double* jpart, int nchunks, int64_t npair, double* Jp, cudaStream_t st);
// X[(q, i)][a_pad] -> planes6[t][i][qcol[q] + a] (pitch6), e6[g][i] from xmax; qgroup[q] = group of q,
// qcol[q] = its first column, gcol[g] = first column of group g (gcol[ng] = the end; multiples of 32).
// The gap between the last q of a group and the next group is filled with zero bytes; bytes past
// gcol[ng] in a row are never read (TMA extent).
cudaError_t launch_jk_split_x(const double* X, int nao, int nq, int a_pad, int s, int ng, const int* qgroup,
                              const int* qcol, const int* gcol, const uint32_t* xmax, int32_t* e6,
                              int8_t* planes6, int64_t pitch6, int64_t plane_stride6, int* status,
                              cudaStream_t st);
// K (+)= sum_g Kpart[g] over lower block-triangle tiles (tile = 128), mirrored.
cudaError_t launch_jk_k_reduce(const double* Kpart, int ng, int nao, int accumulate, double* K,
                               cudaStream_t st);
cudaError_t launch_jk_j_unpack(const double* Jp, int nao, double* J, cudaStream_t st);

}  // namespace dfe
