// split.cu -- FP64 -> scale index + balanced INT8 digit planes (rows H1, H2 of SURVEY.md 8(a)).
// HBM-bound passes: 8 B read + s B written per element.  Rows: a block streams its row twice (the
// maximum, then the digits; the second read hits L2) with 256-bit loads, stages the digit bytes in
// shared memory and writes whole 1 KB runs per plane.  Columns (the transposing split): column
// maxima in one pass over the matrix, then 128-row x 32-column tiles: lane = column (256-byte runs
// per load instruction), 16 bytes per plane and thread into a staging tile, whole 128-byte lines of
// planes[t][column][k ..] out.  The scalar kernels below them serve operands whose rows are not
// 32-byte aligned.
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

// Column maxima of a k x n row-major matrix: thread per column, grid.x over row chunks (odd n).
__global__ void __launch_bounds__(256) col_max_kernel(const double* __restrict__ X, long long k, long long n,
                                                      int rows_per_block, uint32_t* __restrict__ cmax) {
  const long long c = (long long)blockIdx.y * blockDim.x + threadIdx.x;
  if (c >= n) return;
  const long long r0 = (long long)blockIdx.x * rows_per_block;
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

// ---------------------------------------------------------------------------
// Vectorised row split: ld % 4 == 0 and a 32-byte aligned base.  One block per row.
// ---------------------------------------------------------------------------
// NT threads per block (256, or 512 for long rows: more loads in flight per resident row).  The launcher
// limits the resident blocks per SM (through the dynamic shared memory it asks for) so that the rows in
// flight stay well inside L2 and the digit pass finds its row there: at 16384 columns eight blocks
// per SM hold 151 MB of rows and the second pass read all of them from HBM again (ncu: 4.1 GB for 2.1).
template <int S, int NT>
__global__ void __launch_bounds__(NT) split_rows_v4_kernel(const double* __restrict__ X, long long cols, long long ld,
                                                           int32_t* __restrict__ e, int8_t* __restrict__ planes,
                                                           long long pitch, long long plane_stride,
                                                           int* __restrict__ status) {
  constexpr int kChunk = 4 * NT;  // elements per block iteration
  const long long row = blockIdx.x;
  const double* x = X + row * ld;
  __shared__ uint32_t wmax[NT / 32];
  __shared__ int e_sh;
  __shared__ __align__(16) uint32_t stage[2][S][NT];  // [buffer][plane][thread]: 4 digit bytes per thread
  const int tid = threadIdx.x;
  const long long nvec = cols >> 2;  // whole 4-element vectors
  uint32_t hm = 0;
  {
    long long v = tid;
    for (; v + 3 * NT < nvec; v += 4 * NT) {  // four 256-bit loads in flight per thread
      double a[16];
#pragma unroll
      for (int u = 0; u < 4; ++u) ldg_nc_v4f64(x + 4 * (v + NT * u), a[4 * u], a[4 * u + 1], a[4 * u + 2], a[4 * u + 3]);
#pragma unroll
      for (int j = 0; j < 16; ++j) hm = max(hm, abs_hi_word(a[j]));
    }
    for (; v < nvec; v += NT) {
      double a0, a1, a2, a3;
      ldg_nc_v4f64(x + 4 * v, a0, a1, a2, a3);
      hm = max(max(hm, abs_hi_word(a0)), max(abs_hi_word(a1), max(abs_hi_word(a2), abs_hi_word(a3))));
    }
    for (long long c = 4 * nvec + tid; c < cols; c += NT) hm = max(hm, abs_hi_word(__ldg(x + c)));
  }
  hm = warp_max_u32(hm);
  if ((tid & 31) == 0) wmax[tid >> 5] = hm;
  __syncthreads();
  if (tid == 0) {
    uint32_t m = 0;
    for (int i = 0; i < NT / 32; ++i) m = max(m, wmax[i]);
    const int ee = scale_index_from_hi(m);
    e_sh = ee;
    e[row] = ee;
    const int stt = status_from_hi(m);
    if (stt) atomicOr(status, stt);
  }
  __syncthreads();
  const double scale = pow2_double(63 - e_sh);
  int8_t* const prow = planes + row * pitch;
  int buf = 0;
  for (long long c0 = 0; c0 < pitch; c0 += kChunk, buf ^= 1) {
    const long long c = c0 + 4 * tid;
    double a[4] = {0.0, 0.0, 0.0, 0.0};
    if (c + 3 < cols) {
      ldg_nc_v4f64(x + c, a[0], a[1], a[2], a[3]);
    } else {
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (c + j < cols) a[j] = __ldg(x + c + j);
    }
    uint32_t hi[4], lo[4], ph[4], pl[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const uint64_t dg = balanced_digits(a[j], scale);
      hi[j] = (uint32_t)(dg >> 32);
      lo[j] = (uint32_t)dg;
    }
    transpose4x4_bytes(hi, ph);
    if (S > 4) transpose4x4_bytes(lo, pl);
#pragma unroll
    for (int t = 0; t < S; ++t) stage[buf][t][tid] = (t < 4) ? ph[3 - t] : pl[7 - t];
    __syncthreads();  // one barrier per chunk: buffer buf ^ 1 was last read before this barrier
    // S planes x 4 NT bytes: NT / 4 sixteen-byte vectors per plane, whole runs per plane
    for (int idx = tid; idx < S * (NT / 4); idx += NT) {
      const int t = idx / (NT / 4), v = idx % (NT / 4);
      const long long col = c0 + 16 * v;
      if (col < pitch)
        *reinterpret_cast<uint4*>(prow + t * plane_stride + col) = *reinterpret_cast<const uint4*>(&stage[buf][t][4 * v]);
    }
  }
}

// Column maxima, two columns per thread (16-byte loads), rows in chunks over grid.x.
__global__ void __launch_bounds__(256) col_max_v2_kernel(const double* __restrict__ X, long long k, long long n,
                                                         int rows_per_block, uint32_t* __restrict__ cmax) {
  const long long c = ((long long)blockIdx.y * blockDim.x + threadIdx.x) * 2;
  if (c >= n) return;
  const long long r0 = (long long)blockIdx.x * rows_per_block;
  const long long r1 = min(k, r0 + rows_per_block);
  uint32_t h0 = 0, h1 = 0;
  long long r = r0;
  for (; r + 8 <= r1; r += 8) {  // eight loads in flight
    double2 v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = __ldg(reinterpret_cast<const double2*>(X + (r + u) * n + c));
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      h0 = max(h0, abs_hi_word(v[u].x));
      h1 = max(h1, abs_hi_word(v[u].y));
    }
  }
  for (; r < r1; ++r) {
    const double2 v = __ldg(reinterpret_cast<const double2*>(X + r * n + c));
    h0 = max(h0, abs_hi_word(v.x));
    h1 = max(h1, abs_hi_word(v.y));
  }
  atomicMax(&cmax[c], h0);
  atomicMax(&cmax[c + 1], h1);
}

// Transposing split in 128-row x 32-column tiles: lane = column, warp = 16-row group.  A thread loads
// its 16 values (a warp instruction reads one 256-byte run of a row), converts them with its column's
// scale and writes 16 bytes per plane into the staging tile [plane][column][128 + 16]; after the
// barrier 8 lanes copy each 128-byte line planes[t][column][k0 .. k0 + 127] out.
constexpr int kColPitch = 144;
template <int S>
__global__ void __launch_bounds__(256) split_cols_tile_kernel(const double* __restrict__ X, long long k, long long n,
                                                              const int32_t* __restrict__ e,
                                                              int8_t* __restrict__ planes, long long pitch,
                                                              long long plane_stride) {
  __shared__ __align__(16) uint8_t tile[S * 32 * kColPitch];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long c0 = (long long)blockIdx.y * 32;
  const long long k0 = (long long)blockIdx.x * 128;
  const long long c = c0 + lane;
  const bool c_ok = c < n;
  const double scale = pow2_double(63 - (c_ok ? e[c] : 0));
  const long long r0 = k0 + warp * 16;
  double x[16];
#pragma unroll
  for (int j = 0; j < 16; ++j) x[j] = (c_ok && r0 + j < k) ? __ldg(X + (r0 + j) * n + c) : 0.0;
#pragma unroll
  for (int g4 = 0; g4 < 4; ++g4) {
    uint32_t hi[4], lo[4], ph[4], pl[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const uint64_t dg = balanced_digits(x[4 * g4 + j], scale);
      hi[j] = (uint32_t)(dg >> 32);
      lo[j] = (uint32_t)dg;
    }
    transpose4x4_bytes(hi, ph);
    if (S > 4) transpose4x4_bytes(lo, pl);
#pragma unroll
    for (int t = 0; t < S; ++t)
      *reinterpret_cast<uint32_t*>(tile + (t * 32 + lane) * kColPitch + warp * 16 + g4 * 4) = (t < 4) ? ph[3 - t] : pl[7 - t];
  }
  __syncthreads();
  for (int idx = warp * 4 + (lane >> 3); idx < S * 32; idx += 32) {
    const int t = idx >> 5, cc = idx & 31;
    const long long kk = k0 + (lane & 7) * 16;
    if (c0 + cc < n && kk < pitch)
      *reinterpret_cast<uint4*>(planes + t * plane_stride + (c0 + cc) * pitch + kk) =
          *reinterpret_cast<const uint4*>(tile + (t * 32 + cc) * kColPitch + (lane & 7) * 16);
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
                              cudaStream_t st, int num_sms) {
  if (rows <= 0) return cudaSuccess;
  if (ld % 4 == 0 && ((uintptr_t)X & 31) == 0 && pitch % 16 == 0 && plane_stride % 16 == 0 &&
      ((uintptr_t)planes & 15) == 0) {
    // resident rows stay inside ~48 MB of L2: blocks per SM = 48 MB / (SMs x row bytes), 1..8, enforced by the
    // dynamic shared memory each block asks for (it is not used); long rows take 512-thread blocks
    if (num_sms <= 0) {  // callers without a context (a context passes the count of its device)
      int dev = 0;
      num_sms = 148;
      cudaGetDevice(&dev);
      cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
    }
    const bool wide = cols >= 8192;
    long long per_sm = (48ll << 20) / ((long long)num_sms * cols * 8);
    per_sm = per_sm < 1 ? 1 : (per_sm > (wide ? 4 : 8) ? (wide ? 4 : 8) : per_sm);
    const int used = (wide ? 2 * s * 2048 : 2 * s * 1024) + 1024;
    const int pad = per_sm >= 8 ? 0 : (int)((200 * 1024) / per_sm) - used;
    // The attribute belongs to the kernel instantiation, not to a context or stream: it is always set to
    // the largest request any call can make (one block per SM), the same value from every host thread,
    // and only the launch's own dynamic size varies -- two contexts with different `cols` cannot make
    // each other's launch fail.
    const int max_pad = 200 * 1024 - used;
    cudaError_t err = cudaSuccess;
    if (wide) {
      DFE_DISPATCH_S(s, (err = cudaFuncSetAttribute(split_rows_v4_kernel<SS, 512>,
                                                    cudaFuncAttributeMaxDynamicSharedMemorySize, max_pad),
                         split_rows_v4_kernel<SS, 512><<<(unsigned)rows, 512, pad > 0 ? pad : 0, st>>>(
                             X, cols, ld, e, planes, pitch, plane_stride, status)));
    } else {
      DFE_DISPATCH_S(s, (err = cudaFuncSetAttribute(split_rows_v4_kernel<SS, 256>,
                                                    cudaFuncAttributeMaxDynamicSharedMemorySize, max_pad),
                         split_rows_v4_kernel<SS, 256><<<(unsigned)rows, 256, pad > 0 ? pad : 0, st>>>(
                             X, cols, ld, e, planes, pitch, plane_stride, status)));
    }
    if (err != cudaSuccess) return err;
    count_launch();
    return cudaGetLastError();
  }
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
  // row chunks ride on grid.x (2^31 - 1 blocks), column blocks on grid.y: k up to the 2^30 the entry points
  // accept and n up to 2^31 stay inside the grid limits
  const int rows_per_block = 128;
  const unsigned kchunks = (unsigned)((k + rows_per_block - 1) / rows_per_block);
  if ((n + 31) / 32 > 65535) return cudaErrorInvalidValue;
  if (n % 2 == 0 && ((uintptr_t)X & 15) == 0) {
    dim3 g1(kchunks, (unsigned)((n / 2 + 255) / 256));
    col_max_v2_kernel<<<g1, 256, 0, st>>>(X, k, n, rows_per_block, cmax);
  } else {
    dim3 g1(kchunks, (unsigned)((n + 255) / 256));
    col_max_kernel<<<g1, 256, 0, st>>>(X, k, n, rows_per_block, cmax);
  }
  col_scale_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(cmax, n, e, status);
  if (pitch % 16 != 0 || plane_stride % 16 != 0 || ((uintptr_t)planes & 15) != 0) return cudaErrorInvalidValue;
  dim3 g2((unsigned)((pitch + 127) / 128), (unsigned)((n + 31) / 32));
  DFE_DISPATCH_S(s, (split_cols_tile_kernel<SS><<<g2, 256, 0, st>>>(X, k, n, e, planes, pitch, plane_stride)));
  count_launch(3);
  return cudaGetLastError();
}

}  // namespace dfe
