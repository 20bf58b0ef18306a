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

// ---- split.cu -------------------------------------------------------------
// rows x cols FP64 (leading dimension ld) -> e[rows], planes[t][rows][pitch].
cudaError_t launch_split_rows(const double* X, int64_t rows, int64_t cols, int64_t ld, int s, int32_t* e,
                              int8_t* planes, int64_t pitch, int64_t plane_stride, int* status,
                              cudaStream_t st);
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
  // z items (q-groups): item z contracts K range [zk[z], zk[z+1]) (device int array of nz+1), or
  // the whole [0, k) when zk == nullptr (then nz must be 1).  Each z item is cut into flush
  // chunks of kflush(s) contraction elements.
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
  // kEpiInt32: P[(w - 2) * a_rows * b_rows + row * b_rows + col] of flush chunk `dbg_chunk`
  int32_t* P;
  int dbg_chunk;
};

cudaError_t launch_gemm_i8(const GemmProblem& g, cudaStream_t st);
void set_gemm_debug_flags(int flags);
void set_peak_tiles(int n);  // probe walks n distinct operand tiles (1 = the same tile every MMA)
cudaError_t launch_mma_peak(int n_mma, int iters, int grid, float* ms, cudaStream_t st);

void set_jk_debug_flags(int flags);  // timing experiments: bit 0 = unpack writes nothing, bit 1 = reads nothing
// ---- jk.cu ----------------------------------------------------------------
// pass A over packed B: rho[q] (through rho_part[jk_rho_part_rows(nao)][naux], every element of
// which is written, summed in a fixed order) and emax[i * naux + q] = upper word of max_j |B^q_ij|
// (atomicMax, must be zeroed).  rho == nullptr: the maxima alone (df_jk_plan_create); emax == nullptr:
// rho alone, lower tiles only (planned builds).
int64_t jk_rho_part_rows(int nao);
cudaError_t launch_jk_pass_a(const double* Bp, int nao, int naux, const double* D, double* rho_part, double* rho,
                             uint32_t* emax, cudaStream_t st);
// J_packed[p] = sum_q B[p, q] rho[q]
cudaError_t launch_jk_j_gemv(const double* Bp, int64_t npair, int naux, const double* rho, double* Jp,
                             cudaStream_t st);
// unpack + split q in [q0, q1): planes5[t][(q - q0) * nao + i][pitch], e5[(q - q0) * nao + i]
cudaError_t launch_jk_unpack_split(const double* Bp, int nao, int naux, int q0, int q1, const uint32_t* emax,
                                   int s, int32_t* e5, int8_t* planes5, int64_t pitch, int64_t plane_stride,
                                   int* status, const double* rho, double* jpart, cudaStream_t st);
// jpart (may be null): [chunk of 32 q, counted from q0][npair] partials of Eq. 4; J_p = their sum in order
cudaError_t launch_jk_j_reduce(const double* jpart, int nchunks, int64_t npair, double* Jp, cudaStream_t st);
// X[(q, i)][a_pad] -> planes6[t][i][q * a_pad + a] (pitch6), e6[g][i] from xmax; qgroup[q] = group of q.
// planes6 bytes past nq * a_pad in a row are never read (TMA extent).
cudaError_t launch_jk_split_x(const double* X, int nao, int nq, int a_pad, int s, int ng, const int* qgroup,
                              const uint32_t* xmax, int32_t* e6, int8_t* planes6, int64_t pitch6,
                              int64_t plane_stride6, int* status, cudaStream_t st);
// K (+)= sum_g Kpart[g] over lower block-triangle tiles (tile = 128), mirrored.
cudaError_t launch_jk_k_reduce(const double* Kpart, int ng, int nao, int accumulate, double* K,
                               cudaStream_t st);
cudaError_t launch_jk_j_unpack(const double* Jp, int nao, double* J, cudaStream_t st);

}  // namespace dfe
