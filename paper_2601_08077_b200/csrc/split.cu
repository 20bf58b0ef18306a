// split.cu -- FP64 -> scale index + balanced INT8 digit planes (rows H1, H2 of SURVEY.md 8(a)).
// HBM-bound passes: 8 B read + s B written per element (rows), the row re-read for the digit
// pass hits L2 because the same block has just streamed it for the maximum.
//
// Definition (R2; PAPER.md:130 is silent on the internals):
//   e   = scale index of max_k |x| (common.cuh: scale_index_from_hi)
//   Q   = rint(x 2^(63-e))  (int64, round to nearest even)
//   d_t = balanced base-256 digits of Q, t = 1..8; plane t-1 holds d_t
#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"
#include "internal.h"

namespace dfe {

__device__ __forceinline__ uint32_t warp_max_u32(uint32_t v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// Insert byte `b` (0..255) at byte position `pos` (0..3) of `word`.
__device__ __forceinline__ uint32_t put_byte(uint32_t word, uint32_t b, int pos) {
  return word | (b << (8 * pos));
}

// One block per row: pass 1 = max of the upper words of |x|, pass 2 = digits.
// Each thread converts runs of 16 consecutive elements and writes 16 B per plane.
template <int S>
__global__ void __launch_bounds__(256) split_rows_kernel(const double* __restrict__ X, long long rows,
                                                         long long cols, long long ld, int32_t* __restrict__ e,
                                                         int8_t* __restrict__ planes, long long pitch,
                                                         long long plane_stride, int* __restrict__ status) {
  const long long row = blockIdx.x;
  const double* x = X + row * ld;
  __shared__ uint32_t wmax[8];
  __shared__ int e_sh;

  uint32_t hm = 0;
  for (long long c = threadIdx.x; c < cols; c += blockDim.x) hm = max(hm, abs_hi_word(__ldg(x + c)));
  hm = warp_max_u32(hm);
  if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = hm;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t m = 0;
    for (int i = 0; i < (int)(blockDim.x >> 5); ++i) m = max(m, wmax[i]);
    const int ee = scale_index_from_hi(m);
    e_sh = ee;
    e[row] = ee;
    const int stt = status_from_hi(m);
    if (stt) atomicOr(status, stt);
  }
  __syncthreads();
  const double scale = pow2_double(63 - e_sh);

  const long long nrun = pitch / 16;
  for (long long run = threadIdx.x; run < nrun; run += blockDim.x) {
    const long long c0 = run * 16;
    uint32_t w[S][4];
#pragma unroll
    for (int t = 0; t < S; ++t)
#pragma unroll
      for (int j = 0; j < 4; ++j) w[t][j] = 0;
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const long long c = c0 + j;
      const double v = (c < cols) ? __ldg(x + c) : 0.0;
      const uint64_t dg = balanced_digits(v, scale);
#pragma unroll
      for (int t = 0; t < S; ++t) w[t][j >> 2] = put_byte(w[t][j >> 2], digit_byte(dg, t), j & 3);
    }
#pragma unroll
    for (int t = 0; t < S; ++t) {
      uint4 o = make_uint4(w[t][0], w[t][1], w[t][2], w[t][3]);
      *reinterpret_cast<uint4*>(planes + t * plane_stride + row * pitch + c0) = o;
    }
  }
}

// Column maxima of a k x n row-major matrix: thread per column, grid.y over row chunks.
__global__ void __launch_bounds__(256) col_max_kernel(const double* __restrict__ X, long long k, long long n,
                                                      int rows_per_block, uint32_t* __restrict__ cmax) {
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n) return;
  const long long r0 = (long long)blockIdx.y * rows_per_block;
  const long long r1 = min(k, r0 + rows_per_block);
  uint32_t hm = 0;
  for (long long r = r0; r < r1; ++r) hm = max(hm, abs_hi_word(__ldg(X + r * n + c)));
  atomicMax(&cmax[c], hm);
}

__global__ void col_scale_kernel(const uint32_t* __restrict__ cmax, long long n, int32_t* __restrict__ e,
                                 int* __restrict__ status) {
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n) return;
  const uint32_t m = cmax[c];
  e[c] = scale_index_from_hi(m);
  const int stt = status_from_hi(m);
  if (stt) atomicOr(status, stt);
}

// Transposing split of a k x n matrix: lane <-> column (coalesced 256 B reads along n), each
// thread converts 32 consecutive k of its column and writes 32 B per plane to
// planes[t][col][k0 .. k0+31].  Block = 32 columns x 8 k-runs.
template <int S>
__global__ void __launch_bounds__(256) split_cols_kernel(const double* __restrict__ X, long long k, long long n,
                                                         const int32_t* __restrict__ e,
                                                         int8_t* __restrict__ planes, long long pitch,
                                                         long long plane_stride) {
  const long long c = (long long)blockIdx.x * 32 + (threadIdx.x & 31);
  const long long k0 = ((long long)blockIdx.y * 8 + (threadIdx.x >> 5)) * 32;
  if (c >= n || k0 >= pitch) return;
  const double scale = pow2_double(63 - e[c]);
  uint32_t w[S][8];
#pragma unroll
  for (int t = 0; t < S; ++t)
#pragma unroll
    for (int j = 0; j < 8; ++j) w[t][j] = 0;
#pragma unroll
  for (int j = 0; j < 32; ++j) {
    const long long r = k0 + j;
    const double v = (r < k) ? __ldg(X + r * n + c) : 0.0;
    const uint64_t dg = balanced_digits(v, scale);
#pragma unroll
    for (int t = 0; t < S; ++t) w[t][j >> 2] = put_byte(w[t][j >> 2], digit_byte(dg, t), j & 3);
  }
#pragma unroll
  for (int t = 0; t < S; ++t) {
    uint4* dst = reinterpret_cast<uint4*>(planes + t * plane_stride + c * pitch + k0);
    dst[0] = make_uint4(w[t][0], w[t][1], w[t][2], w[t][3]);
    dst[1] = make_uint4(w[t][4], w[t][5], w[t][6], w[t][7]);
  }
}

#define DFE_DISPATCH_S(S_, CALL)      \
  switch (S_) {                       \
    case 1: { constexpr int SS = 1; CALL; } break; \
    case 2: { constexpr int SS = 2; CALL; } break; \
    case 3: { constexpr int SS = 3; CALL; } break; \
    case 4: { constexpr int SS = 4; CALL; } break; \
    case 5: { constexpr int SS = 5; CALL; } break; \
    case 6: { constexpr int SS = 6; CALL; } break; \
    case 7: { constexpr int SS = 7; CALL; } break; \
    default: { constexpr int SS = 8; CALL; } break; \
  }

cudaError_t launch_split_rows(const double* X, int64_t rows, int64_t cols, int64_t ld, int s, int32_t* e,
                              int8_t* planes, int64_t pitch, int64_t plane_stride, int* status,
                              cudaStream_t st) {
  if (rows <= 0) return cudaSuccess;
  DFE_DISPATCH_S(s, (split_rows_kernel<SS><<<(unsigned)rows, 256, 0, st>>>(X, rows, cols, ld, e, planes, pitch,
                                                                         plane_stride, status)));
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_split_cols(const double* X, int64_t k, int64_t n, int s, uint32_t* cmax, int32_t* e,
                              int8_t* planes, int64_t pitch, int64_t plane_stride, int* status,
                              cudaStream_t st) {
  cudaError_t err = cudaMemsetAsync(cmax, 0, sizeof(uint32_t) * n, st);
  if (err != cudaSuccess) return err;
  const int rows_per_block = 64;
  dim3 g1((unsigned)((n + 255) / 256), (unsigned)((k + rows_per_block - 1) / rows_per_block));
  col_max_kernel<<<g1, 256, 0, st>>>(X, k, n, rows_per_block, cmax);
  col_scale_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(cmax, n, e, status);
  dim3 g2((unsigned)((n + 31) / 32), (unsigned)((pitch / 32 + 7) / 8));
  DFE_DISPATCH_S(s, (split_cols_kernel<SS><<<g2, 256, 0, st>>>(X, k, n, e, planes, pitch, plane_stride)));
  count_launch(3);
  return cudaGetLastError();
}

}  // namespace dfe
