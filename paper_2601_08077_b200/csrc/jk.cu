// jk.cu -- the HBM-bound passes of df_jk_build around the two emulated GEMMs
// (rows H1, H2, H5, H6, H7 of SURVEY.md section 8(a)).
//
//   jk_pass_a        rho_q = sum_ij B^q_ij D_ij (Eq. 3) fused with the row maxima
//                    max_j |B^q_ij| that GEMM(5)'s left-operand scales need (R5)
//   jk_j_gemv        J_p = sum_q B[p,q] rho_q   (Eq. 4), plain FP64; a plain
//                    build takes the chunk partials from the unpack pass instead (jk_j_reduce)
//   jk_unpack_split  packed-symmetric B -> dense rows (q,i) x j as INT8 digit planes
//                    ("symmetrise block to dense", fused with the split)
//   jk_split_x       X (GEMM(5) output) -> digit planes with one scale per (i, q-group)
//   jk_k_reduce      K = sum_g K_g in increasing-q order (Eq. 13), mirrored
//
// Geometry of the passes over packed B (q fastest): a block owns a 32 x 32 tile (rows R, columns
// C) of the UNPACKED nao x nao matrix and 32 consecutive q; lane <-> q so every load is a 256-byte
// run of one packed row p(max(R,C), min(R,C)).  Pass A reads every lower tile once and serves the
// mirrored tile from the same registers; the unpack pass runs tile (a,b) and its mirror (b,a) back
// to back (adjacent block indices), so the second read of the same packed rows is an L2 hit.
#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"
#include "internal.h"

namespace dfe {

// (tile pair index, flip) -> (row tile TR, column tile TC) of the full square; returns false for
// the unused mirror of a diagonal tile.  Pair idx = a(a+1)/2 + b, a >= b.
__device__ __forceinline__ bool tile_of_block(unsigned idx, int flip, int& TR, int& TC, bool& lower) {
  int a = (int)((sqrtf(8.0f * (float)idx + 1.0f) - 1.0f) * 0.5f);
  while ((unsigned)(a + 1) * (unsigned)(a + 2) / 2 <= idx) ++a;
  while ((unsigned)a * (unsigned)(a + 1) / 2 > idx) --a;
  const int b = (int)(idx - (unsigned)a * (unsigned)(a + 1) / 2);
  if (flip && a == b) return false;
  TR = flip ? b : a;
  TC = flip ? a : b;
  lower = !flip;
  return true;
}

// 16 consecutive elements (R, Cs .. Cs+15) of the unpacked matrix for one q (bqb = byte address of
// Bp + q, naux8 = bytes per packed row).  KIND 0: every C < R (consecutive packed rows); KIND 1:
// every C > R (the mirror: packed rows p(C, R), stride growing by one row per column); KIND 2: mixed
// (diagonal blocks).  FULL: all 16 columns are < nao; otherwise the column is clamped to nao - 1
// (a valid address) and the value replaced by zero.  Row indices are unsigned 32-bit and the byte
// offset one 32 x 32 -> 64 multiply-add, 2-3 instructions per element (signed 64-bit index
// arithmetic cost 5-10 and made the passes issue bound).
template <int KIND, bool FULL>
__device__ __forceinline__ void load_row16(double (&x)[16], const char* __restrict__ bqb, unsigned naux8, int R,
                                           int Cs, int nao) {
  const unsigned uR = (unsigned)R;
#pragma unroll
  for (int cc = 0; cc < 16; ++cc) {
    const unsigned c = FULL ? (unsigned)(Cs + cc) : (unsigned)min(Cs + cc, nao - 1);
    unsigned row;
    if (KIND == 0) row = uR * (uR + 1) / 2 + c;
    else if (KIND == 1) row = c * (c + 1) / 2 + uR;
    else row = (c <= uR) ? uR * (uR + 1) / 2 + c : c * (c + 1) / 2 + uR;
    x[cc] = __ldg(reinterpret_cast<const double*>(bqb + (unsigned long long)row * naux8));
  }
  if (!FULL) {
#pragma unroll
    for (int cc = 0; cc < 16; ++cc) x[cc] = (Cs + cc < nao) ? x[cc] : 0.0;
  }
}

__device__ __forceinline__ long long packed_row(int R, int C) {
  const long long hi = max(R, C), lo = min(R, C);
  return hi * (hi + 1) / 2 + lo;
}

// RHO: the rho partials; EMAX: the row maxima of the UNPACKED matrix.  One block per lower tile
// (TR >= TC) and q chunk reads its packed rows ONCE: an element B[p(R,C)][q] of an off-diagonal
// tile belongs to row R (maximum over C, kept per thread) and, mirrored, to row C (maximum over R:
// 16 running maxima per thread and column half, merged over the eight warps by shared-memory
// atomicMax, then one global atomicMax per (C, q)).  The first version ran a second "mirror" block
// per tile that re-read the same 256 KB through L2: 13 % of those reads missed (26.1 GB of DRAM
// reads for 23.1 GB of B).  A plan (df_jk_plan_create) runs EMAX alone once, a planned build RHO alone.
template <bool RHO, bool EMAX>
__global__ void __launch_bounds__(256, EMAX ? 4 : 5) jk_pass_a_kernel(const double* __restrict__ Bp, int nao, int naux,
                                                        const double* __restrict__ D,
                                                        double* __restrict__ rho_part,
                                                        uint32_t* __restrict__ emax,
                                                        uint32_t* __restrict__ tilemax) {
  int TR, TC;
  bool lower;
  tile_of_block(blockIdx.y, 0, TR, TC, lower);
  const bool offdiag = TR != TC;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int q = (int)blockIdx.x * 32 + lane;
  const bool q_ok = q < naux;
  __shared__ double rho_sh[8][32];
  __shared__ double dw_sh[32][33];  // weighted density of this tile: (i == j ? 1 : 2) * 0.5 (D_ij + D_ji), 0 above the diagonal
  __shared__ uint32_t cmax_sh[32][32];  // [column of the tile][q]: max over the tile's rows
  __shared__ uint32_t tmax_sh[32];      // [q]: max over the whole 32 x 32 tile (screening)
  if (EMAX && offdiag) {
    for (int idx = threadIdx.x; idx < 1024; idx += 256) cmax_sh[idx >> 5][idx & 31] = 0u;
  }
  if (EMAX && threadIdx.x < 32) tmax_sh[threadIdx.x] = 0u;
  if (RHO) {
    for (int idx = threadIdx.x; idx < 1024; idx += 256) {
      const int rl = idx >> 5, cl = idx & 31;
      const int R = TR * 32 + rl, C = TC * 32 + cl;
      double v = 0.0;
      if (R < nao && C <= R) {
        const double d = 0.5 * (__ldg(D + (long long)R * nao + C) + __ldg(D + (long long)C * nao + R));
        v = (R == C) ? d : 2.0 * d;
      }
      dw_sh[rl][cl] = v;
    }
  }
  if (RHO || EMAX) __syncthreads();
  double rsum = 0.0;
  uint32_t hm[4] = {0u, 0u, 0u, 0u};
  const char* bq = reinterpret_cast<const char*>(Bp + (q_ok ? q : 0));
  const unsigned naux8 = (unsigned)naux * 8u;
  const int kind = offdiag ? 0 : 2;  // block-uniform: every C < R, or a diagonal tile (mixed)
  const bool full = TC * 32 + 32 <= nao;
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    uint32_t cm[16];
#pragma unroll
    for (int cc = 0; cc < 16; ++cc) cm[cc] = 0u;
    const int Cs = TC * 32 + half * 16;
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) {
      const int rl = warp + 8 * rr;
      const int R = TR * 32 + rl;
      if (R >= nao) continue;  // warp-uniform
      // 16 loads in flight per thread before the first use (HBM-latency bound otherwise)
      double x[16];
      if (!q_ok) {
#pragma unroll
        for (int cc = 0; cc < 16; ++cc) x[cc] = 0.0;
      } else if (full) {
        if (kind == 0) load_row16<0, true>(x, bq, naux8, R, Cs, nao);
        else load_row16<2, true>(x, bq, naux8, R, Cs, nao);
      } else {
        load_row16<2, false>(x, bq, naux8, R, Cs, nao);  // only the last diagonal tile is ragged
      }
#pragma unroll
      for (int cc = 0; cc < 16; ++cc) {
        if (EMAX) {
          const uint32_t a = abs_hi_word(x[cc]);
          hm[rr] = max(hm[rr], a);
          cm[cc] = max(cm[cc], a);
        }
        if (RHO) rsum = fma(dw_sh[rl][half * 16 + cc], x[cc], rsum);
      }
    }
    if (EMAX && offdiag) {
#pragma unroll
      for (int cc = 0; cc < 16; ++cc) atomicMax(&cmax_sh[half * 16 + cc][lane], cm[cc]);
    }
  }
  if (EMAX && q_ok) {
#pragma unroll
    for (int rr = 0; rr < 4; ++rr) {
      const int R = TR * 32 + warp + 8 * rr;
      if (R < nao) atomicMax(&emax[(long long)R * naux + q], hm[rr]);
    }
  }
  if (EMAX && tilemax) atomicMax(&tmax_sh[lane], max(max(hm[0], hm[1]), max(hm[2], hm[3])));
  if (RHO) rho_sh[warp][lane] = rsum;
  if (RHO || (EMAX && offdiag)) __syncthreads();
  if (EMAX && offdiag && q_ok) {
    for (int cl = warp; cl < 32; cl += 8)  // TC < TR: every column of the tile is < nao
      atomicMax(&emax[(long long)(TC * 32 + cl) * naux + q], cmax_sh[cl][lane]);
  }
  if (EMAX && tilemax) {
    if (!RHO && !offdiag) __syncthreads();  // the other variants have passed a barrier since the atomics
    if (warp == 1 && q_ok) tilemax[(long long)blockIdx.y * naux + q] = tmax_sh[lane];
  }
  if (RHO) {
    if (warp == 0 && q_ok) {
      double t = 0.0;
#pragma unroll
      for (int w = 0; w < 8; ++w) t += rho_sh[w][lane];
      rho_part[(long long)blockIdx.y * naux + q] = t;  // one block per (tile pair, q chunk)
    }
  }
}

// rho[q] = sum over tile pairs of rho_part[pair][q] in a fixed order (eight contiguous runs of
// pairs, one per warp, then the eight run sums in order): bitwise reproducible, unlike atomics.
__global__ void __launch_bounds__(256) jk_rho_reduce_kernel(const double* __restrict__ rho_part, int npairs,
                                                            int naux, double* __restrict__ rho) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int q = blockIdx.x * 32 + lane;
  __shared__ double part[8][32];
  const int per = (npairs + 7) / 8;
  const int y0 = warp * per, y1 = min(npairs, y0 + per);
  double t = 0.0;
  if (q < naux) {
    int y = y0;
    for (; y + 8 <= y1; y += 8) {
      double v[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) v[u] = __ldg(rho_part + (long long)(y + u) * naux + q);
#pragma unroll
      for (int u = 0; u < 8; ++u) t += v[u];
    }
    for (; y < y1; ++y) t += __ldg(rho_part + (long long)y * naux + q);
  }
  part[warp][lane] = t;
  __syncthreads();
  if (warp == 0 && q < naux) {
    double r = 0.0;
#pragma unroll
    for (int w = 0; w < 8; ++w) r += part[w][lane];
    rho[q] = r;
  }
}

// J (Eq. 4) is summed the same way on both routes, so that a planned build and a plain build
// give the same bits: J_p = sum over the 32-q chunks c, in increasing c, of the chunk's partial
// sum_{q in c} B[p,q] rho_q, and the partial is the butterfly over the 32 lanes (lane = q within the
// chunk; partners at distance 16, 8, 4, 2, 1; products rounded before the additions).
//
// tree4: four such butterflies at once.  Lane q holds y0..y3 = its terms of four packed rows; after
// the first two levels a lane carries only one of the four sums (rows are handed over instead of
// duplicated: 6 shuffles and 6 additions instead of 20), and every lane returns the complete sum
// of row v = 2 * (lane bit 4) + (lane bit 3).  Additions commute bit for bit, so each row's result
// equals the plain butterfly's.
__device__ __forceinline__ double shfl_xor_f64(double v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }
__device__ __forceinline__ double tree4(double y0, double y1, double y2, double y3, int lane) {
  const bool b4 = (lane & 16) != 0, b3 = (lane & 8) != 0;
  double k0 = b4 ? y2 : y0, k1 = b4 ? y3 : y1;
  const double s0 = b4 ? y0 : y2, s1 = b4 ? y1 : y3;
  k0 += shfl_xor_f64(s0, 16);
  k1 += shfl_xor_f64(s1, 16);
  double k = b3 ? k1 : k0;
  const double sd = b3 ? k0 : k1;
  k += shfl_xor_f64(sd, 8);
  k += shfl_xor_f64(k, 4);
  k += shfl_xor_f64(k, 2);
  k += shfl_xor_f64(k, 1);
  return k;
}

// tree16: the same for sixteen rows (x[i] = this lane's element of row i, rq = its rho): 16 shuffles and
// additions for sixteen butterflies; lane 2 i (and 2 i + 1) returns the complete sum of row i.
__device__ __forceinline__ double tree16(const double (&x)[16], double rq, int lane) {
  const bool b4 = (lane & 16) != 0, b3 = (lane & 8) != 0, b2 = (lane & 4) != 0, b1 = (lane & 2) != 0;
  double k8[8], k4[4], k2[2];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const double lo = x[i] * rq, hi = x[8 + i] * rq;
    k8[i] = (b4 ? hi : lo) + shfl_xor_f64(b4 ? lo : hi, 16);
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) k4[i] = (b3 ? k8[4 + i] : k8[i]) + shfl_xor_f64(b3 ? k8[i] : k8[4 + i], 8);
#pragma unroll
  for (int i = 0; i < 2; ++i) k2[i] = (b2 ? k4[2 + i] : k4[i]) + shfl_xor_f64(b2 ? k4[i] : k4[2 + i], 4);
  double k = (b1 ? k2[1] : k2[0]) + shfl_xor_f64(b1 ? k2[0] : k2[1], 2);
  k += shfl_xor_f64(k, 1);
  return k;
}

// Planned builds (no unpack pass to ride on): a warp owns four consecutive packed rows and walks
// the chunks; sixteen loads of B per lane are in flight.
__global__ void __launch_bounds__(256) jk_j_gemv_kernel(const double* __restrict__ Bp, long long npair, int naux,
                                                        const double* __restrict__ rho, double* __restrict__ Jp) {
  const int lane = threadIdx.x & 31;
  const long long p0 = ((long long)blockIdx.x * 8 + (threadIdx.x >> 5)) * 4;
  if (p0 >= npair) return;
  const double* b[4];
#pragma unroll
  for (int r = 0; r < 4; ++r) b[r] = Bp + (p0 + r < npair ? p0 + r : npair - 1) * naux;
  const int nchunks = (naux + 31) >> 5;
  double acc = 0.0;
  int c = 0;
  for (; c + 4 <= nchunks; c += 4) {
    double x[4][4], rq[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int q = (c + u) * 32 + lane;
      const bool ok = q < naux;
      rq[u] = ok ? __ldg(rho + q) : 0.0;
#pragma unroll
      for (int r = 0; r < 4; ++r) x[u][r] = ok ? __ldg(b[r] + q) : 0.0;
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) acc += tree4(x[u][0] * rq[u], x[u][1] * rq[u], x[u][2] * rq[u], x[u][3] * rq[u], lane);
  }
  for (; c < nchunks; ++c) {
    const int q = c * 32 + lane;
    const bool ok = q < naux;
    const double rq = ok ? __ldg(rho + q) : 0.0;
    double x[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) x[r] = ok ? __ldg(b[r] + q) : 0.0;
    acc += tree4(x[0] * rq, x[1] * rq, x[2] * rq, x[3] * rq, lane);
  }
  const int v = ((lane >> 4) & 1) * 2 + ((lane >> 3) & 1);
  if ((lane & 7) == 0 && p0 + v < npair) Jp[p0 + v] = acc;
}

// Plain builds: the unpack pass leaves one partial per (chunk, packed row) in jpart; J_p is their
// sum in increasing chunk order.
__global__ void __launch_bounds__(256) jk_j_reduce_kernel(const double* __restrict__ jpart, int nchunks,
                                                          long long npair, double* __restrict__ Jp) {
  const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= npair) return;
  double acc = 0.0;
  int c = 0;
  for (; c + 8 <= nchunks; c += 8) {
    double v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = __ldg(jpart + (long long)(c + u) * npair + p);
#pragma unroll
    for (int u = 0; u < 8; ++u) acc += v[u];
  }
  for (; c < nchunks; ++c) acc += __ldg(jpart + (long long)c * npair + p);
  Jp[p] = acc;
}

// Unpack + split.  Output planes[t][(q, R)][C] want C-contiguous 128-byte lines, the input wants
// q-contiguous runs; the block transposes through shared memory so that both are whole lines.
// A block owns kUnpackRows consecutive output rows R of one 128 x 128 tile, 32 consecutive q and
// the tile's 128 columns: lane = q, warp = 16-column group.  Per row a thread loads its 16 values
// (a warp instruction reads one 256-byte run of a packed row), converts them with the scale of
// (q, R), and writes 16 bytes per plane into the staging tile [plane][q][128 + 16 pad]; after one
// barrier (the tile is double buffered) the warps copy it out, 8 lanes per 128-byte line of
// (plane, q, R).  Blocks are ordered [q chunk][128 x 128 super-tile pair (A >= B)][sub]: the first
// half of the subs are the row groups of the (A, B) block (rows in A, columns in B), the second
// half those of the mirrored (B, A) block; both read the same 128 x 128 packed rows of this q
// chunk (4 MB) back to back, so the second read is an L2 hit.  The q chunk is the slowest index:
// all lines written in a stretch of time then fall into the 32 q x nao rows of one chunk (49 MB
// per plane), which the L2 write-back turns into longer DRAM bursts than with the tile pair
// slowest (10.7 -> 10.1 ms at s = 4, 15.4 -> 14.3 ms at s = 6; groups of 2, 4, 8 chunks lie between).  Two rows per block keep the number
// of tiles in flight, and with it the L2 working set, small (8 rows: 11.2 / 16.9 ms at s = 4 / 6
// against 10.5 / 14.3 ms).  Four resident blocks per SM up to s = 4, three above (measured both ways).
constexpr int kUnpackRows = 2;
// Row r stages through buffer r & 1 and is protected by ONE barrier per processed row; a row that the
// screening mask skips (`continue` below) skips its barrier too.  With two rows every buffer is used
// once per block, so that is safe; with three or more, row r + 2 could overwrite buffer r & 1 while
// other warps still copy row r out of it.  Drive the buffer parity and the barrier by a count of the
// processed rows before raising this.
static_assert(kUnpackRows <= 2, "jk_unpack_split_kernel: skipped rows skip the barrier that guards the double buffer");
constexpr int kUnpackPitch = 144;  // staging row: 128 bytes + 16 (conflict-free 16-byte stores by 8 lanes)
template <int S>
__global__ void __launch_bounds__(256, S <= 4 ? 4 : 3) jk_unpack_split_kernel(const double* __restrict__ Bp, int nao, int naux,
                                                              int q0, int q1, const uint32_t* __restrict__ emax,
                                                              int32_t* __restrict__ e5, int8_t* __restrict__ planes,
                                                              long long pitch, long long plane_stride,
                                                              int* __restrict__ status, int dbg,
                                                              const double* __restrict__ rho,
                                                              double* __restrict__ jpart, long long npair,
                                                              const uint32_t* __restrict__ kmask, int mask_words) {
  extern __shared__ __align__(16) uint8_t ubuf[];  // [2][S][32][kUnpackPitch]
  constexpr int kSubs = 128 / kUnpackRows;
  int A, B;
  bool lower;
  const int sub = (int)(blockIdx.x % (2 * kSubs));
  const int chunk = (int)blockIdx.y;
  const unsigned tpair = blockIdx.x / (2 * kSubs);
  if (!tile_of_block(tpair, sub / kSubs, A, B, lower)) return;  // (A, B) = (row block, column block)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int qg = q0 + chunk * 32 + lane;
  const bool q_ok = qg < q1;
  const int q = q_ok ? qg : q1 - 1;  // a valid address; the lane's results are dropped
  const int Cs = B * 128 + warp * 16;
  const char* bq = reinterpret_cast<const char*>(Bp + q);
  const unsigned naux8 = (unsigned)naux * 8u;
  // block-uniform shape of the tile: rows in block A, columns in block B
  const int kind = (A > B) ? 0 : (A < B) ? 1 : 2;
  const bool full = B * 128 + 128 <= nao;
  const int nq_blk = min(32, q1 - (q0 + chunk * 32));
  // Eq. 4 rides on the lower blocks: they hold every packed element of this q chunk exactly once
  const bool do_j = jpart != nullptr && lower;
  const double rq = (do_j && q_ok) ? __ldg(rho + qg) : 0.0;
  double* const jp_chunk = do_j ? jpart + (long long)chunk * npair : nullptr;
#pragma unroll 1
  for (int r = 0; r < kUnpackRows; ++r) {
    const int R = A * 128 + (sub % kSubs) * kUnpackRows + r;
    if (R >= nao) break;  // block-uniform
    // screening: bit B of the mask of the 256-row block of (q, R) -- lane = q in every warp, so the
    // ballot is the same in all warps and the branches below are block-uniform
    const uint32_t hm = emax[(long long)R * naux + q];
    const int e = scale_index_from_hi(hm);
    if (lower && B == 0 && warp == 0 && q_ok) {  // the row's scale index is written whether or not its block is active
      e5[(long long)(qg - q0) * nao + R] = e;
      const int stt = status_from_hi(hm);
      if (stt) atomicOr(status, stt);
    }
    uint32_t act = 0xffffffffu;
    if (kmask) {
      const long long mb = ((long long)(q - q0) * nao + R) >> 8;
      act = __ballot_sync(0xffffffffu, q_ok && ((kmask[mb * mask_words + (B >> 5)] >> (B & 31)) & 1u));
      if (act == 0u && !do_j) continue;  // nothing to write, nothing to sum: the row is not even read
    }
    const double scale = pow2_double(63 - e);
    double x[16];
    if (dbg & 2) {
#pragma unroll
      for (int cc = 0; cc < 16; ++cc) x[cc] = 0.0;
    } else if (full) {
      if (kind == 0) load_row16<0, true>(x, bq, naux8, R, Cs, nao);
      else if (kind == 1) load_row16<1, true>(x, bq, naux8, R, Cs, nao);
      else load_row16<2, true>(x, bq, naux8, R, Cs, nao);
    } else {
      if (kind == 1) load_row16<1, false>(x, bq, naux8, R, Cs, nao);
      else load_row16<2, false>(x, bq, naux8, R, Cs, nao);  // kind 0 has B < A: always full
    }
    if (do_j) {
      // partial of J_p over this chunk's 32 q for the 16 packed rows p(R, Cs .. Cs + 15): lane 2 i
      // ends up with the sum of column i (tree16), the even lanes store 128 contiguous bytes
      const double k = tree16(x, rq, lane);
      const int C = Cs + (lane >> 1);
      if ((lane & 1) == 0 && C <= R)  // C <= R < nao; a diagonal tile holds the rest as mirrors
        jp_chunk[(long long)R * (R + 1) / 2 + C] = k;
      if (act == 0u) continue;  // Eq. 4 needs every element, the planes only the active blocks
    }
    uint32_t w[S][4];
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
      for (int t = 0; t < S; ++t) w[t][g4] = (t < 4) ? ph[3 - t] : pl[7 - t];
    }
    uint8_t* const buf = ubuf + (size_t)(r & 1) * (S * 32 * kUnpackPitch);
#pragma unroll
    for (int t = 0; t < S; ++t)
      *reinterpret_cast<uint4*>(buf + (t * 32 + lane) * kUnpackPitch + warp * 16) =
          make_uint4(w[t][0], w[t][1], w[t][2], w[t][3]);
    __syncthreads();  // one barrier per row: buffer (r + 1) & 1 was last read before this barrier
    if (dbg & 1) continue;
    const long long row0 = ((long long)chunk * 32 * nao + R) * pitch + B * 128 + (lane & 7) * 16;
    for (int idx = warp * 4 + (lane >> 3); idx < S * 32; idx += 32) {
      const int t = idx >> 5, qq = idx & 31;
      if (qq < nq_blk && ((act >> qq) & 1u))
        *reinterpret_cast<uint4*>(planes + t * plane_stride + row0 + (long long)qq * nao * pitch) =
            *reinterpret_cast<const uint4*>(buf + (t * 32 + qq) * kUnpackPitch + (lane & 7) * 16);
    }
  }
}

// ---------------------------------------------------------------------------
// Screening (PAPER.md:120 N_scr <= N_bf^2, "grouped
// GEMM"): which 128-column K blocks of GEMM(5)'s left operand hold a non-zero digit at s slices.
// An element of row (q, i) has its first s balanced digits all zero when |x| < 2^(e_qi - 8 s - 1)
// (then |Q| <= 2^(62 - 8 s) < 0.498 * 2^(64 - 8 s), the largest magnitude whose top s digits vanish).
// mask[mb] bit J = 0 says that in the 256 flattened rows (q, i) of block mb every element of columns
// 128 J .. 128 J + 127 is below its row's threshold -- judged conservatively from the maxima of the
// 32 x 32 tiles pass A left in tilemax.  The unpack pass writes no planes for such a block and GEMM(5)
// neither loads it nor issues its MMAs: skipping exact zeros, the result is the dense one bit for bit.
// A block with no active K block at all (zero rows) keeps bit 0, so its accumulators are written.
// stats[0] / stats[1] += active / all (block, K block) pairs.
// ---------------------------------------------------------------------------
__global__ void __launch_bounds__(256) jk_screen_mask_kernel(const uint32_t* __restrict__ emax,
                                                             const uint32_t* __restrict__ tilemax, int nao, int naux,
                                                             int q0, int nq, int s, int nJ, int words,
                                                             uint32_t* __restrict__ mask,
                                                             unsigned long long* __restrict__ stats) {
  __shared__ uint32_t m_sh[4];
  if (threadIdx.x < 4) m_sh[threadIdx.x] = 0u;
  __syncthreads();
  const long long row = (long long)blockIdx.x * 256 + threadIdx.x;
  uint32_t m[4] = {0u, 0u, 0u, 0u};
  if (row < (long long)nq * nao) {
    const int ql = (int)(row / nao), i = (int)(row - (long long)ql * nao), q = q0 + ql;
    const int e = scale_index_from_hi(__ldg(emax + (long long)i * naux + q));
    const int eb = 1023 + e - 8 * s - 1;                       // biased exponent of the threshold
    const uint32_t thr = eb > 0 ? (uint32_t)eb << 20 : 0u;      // below the normal range: everything counts
    const unsigned ti = (unsigned)i >> 5;
    const int T32 = (nao + 31) >> 5;
    for (int tj = 0; tj < T32; ++tj) {
      const unsigned hi = max(ti, (unsigned)tj), lo = min(ti, (unsigned)tj);
      const uint32_t tm = __ldg(tilemax + (long long)(hi * (hi + 1) / 2 + lo) * naux + q);
      if (tm >= thr && tm != 0u) m[tj >> 7] |= 1u << ((tj >> 2) & 31);
    }
  }
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    const uint32_t r = __reduce_or_sync(0xffffffffu, m[w]);
    if ((threadIdx.x & 31) == 0 && r) atomicOr(&m_sh[w], r);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t any = 0u;
    for (int w = 0; w < words; ++w) any |= m_sh[w];
    if (!any) m_sh[0] = 1u;
    int act = 0;
    for (int w = 0; w < words; ++w) {
      mask[(long long)blockIdx.x * words + w] = m_sh[w];
      act += __popc(m_sh[w]);
    }
    atomicAdd(&stats[0], (unsigned long long)act);
    atomicAdd(&stats[1], (unsigned long long)nJ);
  }
}

// e6[g][i] from the running maxima GEMM(5)'s epilogue left in xmax[g][i].
__global__ void jk_x_scale_kernel(const uint32_t* __restrict__ xmax, long long n, int32_t* __restrict__ e6,
                                  int* __restrict__ status) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  const uint32_t m = xmax[t];
  e6[t] = scale_index_from_hi(m);
  const int stt = status_from_hi(m);
  if (stt) atomicOr(status, stt);
}

// X[(q, i)][a_pad] (GEMM(5)'s output, one contiguous 128-row block per tile) -> planes6[t][i][qcol[q] + a]
// with the scale of (i, group of q).  A block owns one i and 32 consecutive q: it reads 32 runs of
// a_pad doubles and writes one contiguous run of 32 * a_pad bytes per plane (with a 16-byte gap of
// zeros where a group ends off a multiple of 32 columns: every group of GEMM(6) starts on the K extent
// of an MMA); a thread converts 16 consecutive columns.
template <int S>
__global__ void __launch_bounds__(256) jk_split_x_kernel(const double* __restrict__ X, int nao, int nq, int a_pad,
                                                         const int* __restrict__ qgroup,
                                                         const int* __restrict__ qcol,
                                                         const int* __restrict__ gcol,
                                                         const int32_t* __restrict__ e6,
                                                         int8_t* __restrict__ planes, long long pitch,
                                                         long long plane_stride) {
  const int i = blockIdx.y;
  const int runs_per_q = a_pad >> 4;
  const int units = 32 * runs_per_q;
  for (int u = threadIdx.x; u < units; u += blockDim.x) {
    const int ql = u / runs_per_q, run = u - ql * runs_per_q;
    const int q = blockIdx.x * 32 + ql;
    if (q >= nq) break;
    const int g = qgroup[q];
    const double scale = pow2_double(63 - e6[(long long)g * nao + i]);
    const double2* src = reinterpret_cast<const double2*>(X + ((long long)q * nao + i) * a_pad + run * 16);
    double2 v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = __ldg(src + j);
    uint32_t w[S][4];
#pragma unroll
    for (int g4 = 0; g4 < 4; ++g4) {
      uint32_t hi[4], lo[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const double x = (j & 1) ? v[2 * g4 + (j >> 1)].y : v[2 * g4 + (j >> 1)].x;
        const uint64_t dg = balanced_digits(x, scale);
        hi[j] = (uint32_t)(dg >> 32);
        lo[j] = (uint32_t)dg;
      }
#pragma unroll
      for (int t = 0; t < S; ++t)
        w[t][g4] = (t < 4) ? pack4_digit(hi[0], hi[1], hi[2], hi[3], 3 - t) : pack4_digit(lo[0], lo[1], lo[2], lo[3], 7 - t);
    }
    const long long col = qcol[q];
    int8_t* const dst = planes + (long long)i * pitch + col + run * 16;
#pragma unroll
    for (int t = 0; t < S; ++t)
      *reinterpret_cast<uint4*>(dst + t * plane_stride) = make_uint4(w[t][0], w[t][1], w[t][2], w[t][3]);
    // the last q of a group whose end is not a multiple of 32 columns: zero digits up to the next group
    if (run == runs_per_q - 1 && col + a_pad < gcol[g + 1] && (q + 1 == nq || qgroup[q + 1] != g)) {
#pragma unroll
      for (int t = 0; t < S; ++t)
        *reinterpret_cast<uint4*>(dst + t * plane_stride + 16) = make_uint4(0u, 0u, 0u, 0u);
    }
  }
}

// K[i][j] (+)= sum_g Kpart[g][i][j] for column tile <= row tile (tile = 128), mirrored to [j][i].
__global__ void __launch_bounds__(256) jk_k_reduce_kernel(const double* __restrict__ Kpart, int ng, int nao,
                                                          int accumulate, double* __restrict__ K) {
  const int i = blockIdx.y;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= nao || (j / kTileM) > (i / kTileM)) return;
  const long long nn = (long long)nao * nao;
  const long long ij = (long long)i * nao + j;
  double acc = accumulate ? K[ij] : 0.0;
  for (int g = 0; g < ng; ++g) acc += Kpart[g * nn + ij];
  K[ij] = acc;
  if ((j / kTileM) < (i / kTileM)) K[(long long)j * nao + i] = acc;
}

__global__ void __launch_bounds__(256) jk_j_unpack_kernel(const double* __restrict__ Jp, int nao,
                                                          double* __restrict__ J) {
  const int i = blockIdx.y;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= nao) return;
  J[(long long)i * nao + j] = Jp[packed_row(i, j)];
}

// ---------------------------------------------------------------------------
static unsigned tile_pairs(int nao) {
  const unsigned T = (unsigned)((nao + 31) / 32);
  return T * (T + 1) / 2;
}

int64_t jk_rho_part_rows(int nao) { return tile_pairs(nao); }

cudaError_t launch_jk_pass_a(const double* Bp, int nao, int naux, const double* D, double* rho_part, double* rho,
                             uint32_t* emax, uint32_t* tilemax, cudaStream_t st) {
  const unsigned qchunks = (unsigned)((naux + 31) / 32);
  if (emax && rho) {
    jk_pass_a_kernel<true, true><<<dim3(qchunks, tile_pairs(nao)), 256, 0, st>>>(Bp, nao, naux, D, rho_part, emax, tilemax);
  } else if (rho) {
    jk_pass_a_kernel<true, false><<<dim3(qchunks, tile_pairs(nao)), 256, 0, st>>>(Bp, nao, naux, D, rho_part, emax, nullptr);
  } else {
    jk_pass_a_kernel<false, true><<<dim3(qchunks, tile_pairs(nao)), 256, 0, st>>>(Bp, nao, naux, D, rho_part, emax, tilemax);
  }
  count_launch();
  if (rho) {
    jk_rho_reduce_kernel<<<qchunks, 256, 0, st>>>(rho_part, (int)tile_pairs(nao), naux, rho);
    count_launch();
  }
  return cudaGetLastError();
}

cudaError_t launch_jk_j_gemv(const double* Bp, int64_t npair, int naux, const double* rho, double* Jp,
                             cudaStream_t st) {
  jk_j_gemv_kernel<<<(unsigned)((npair + 31) / 32), 256, 0, st>>>(Bp, npair, naux, rho, Jp);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_jk_j_reduce(const double* jpart, int nchunks, int64_t npair, double* Jp, cudaStream_t st) {
  jk_j_reduce_kernel<<<(unsigned)((npair + 255) / 256), 256, 0, st>>>(jpart, nchunks, npair, Jp);
  count_launch();
  return cudaGetLastError();
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

template <int S>
static cudaError_t unpack_split_s(dim3 grid, int smem, cudaStream_t st, const double* Bp, int nao, int naux, int q0,
                                  int q1, const uint32_t* emax, int32_t* e5, int8_t* planes5, int64_t pitch,
                                  int64_t plane_stride, int* status, const double* rho, double* jpart,
                                  long long npair, int dbg, const uint32_t* kmask, int mask_words) {
  // set on every launch (s >= 6 stages more than 48 KB): the attribute is per device
  cudaError_t err = cudaFuncSetAttribute(jk_unpack_split_kernel<S>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         2 * S * 32 * kUnpackPitch);
  if (err != cudaSuccess) return err;
  jk_unpack_split_kernel<S><<<grid, 256, smem, st>>>(Bp, nao, naux, q0, q1, emax, e5, planes5, pitch, plane_stride,
                                                     status, dbg, rho, jpart, npair, kmask, mask_words);
  return cudaSuccess;
}

cudaError_t launch_jk_unpack_split(const double* Bp, int nao, int naux, int q0, int q1, const uint32_t* emax,
                                   int s, int32_t* e5, int8_t* planes5, int64_t pitch, int64_t plane_stride,
                                   int* status, const double* rho, double* jpart, int dbg, const uint32_t* kmask,
                                   int mask_words, cudaStream_t st) {
  const unsigned T128 = (unsigned)((nao + 127) / 128);
  if (pitch % 128 != 0 || pitch < 128 * (int64_t)T128) return cudaErrorInvalidValue;
  dim3 grid((unsigned)(2 * (128 / kUnpackRows)) * (T128 * (T128 + 1) / 2), (unsigned)((q1 - q0 + 31) / 32));
  const int smem = 2 * s * 32 * kUnpackPitch;
  cudaError_t err = cudaSuccess;
  DFE_DISPATCH_S(s, (err = unpack_split_s<SS>(grid, smem, st, Bp, nao, naux, q0, q1, emax, e5, planes5, pitch,
                                              plane_stride, status, rho, jpart, (long long)nao * (nao + 1) / 2, dbg, kmask,
                                              mask_words)));
  if (err != cudaSuccess) return err;
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_jk_screen_mask(const uint32_t* emax, const uint32_t* tilemax, int nao, int naux, int q0, int nq,
                                  int s, uint32_t* mask, unsigned long long* stats, cudaStream_t st) {
  const int nJ = (nao + 127) / 128, words = (nJ + 31) / 32;
  if (words > 4) return cudaErrorInvalidValue;
  const long long nblk = ((long long)nq * nao + 255) / 256;
  jk_screen_mask_kernel<<<(unsigned)nblk, 256, 0, st>>>(emax, tilemax, nao, naux, q0, nq, s, nJ, words, mask, stats);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_jk_split_x(const double* X, int nao, int nq, int a_pad, int s, int ng, const int* qgroup,
                              const int* qcol, const int* gcol, const uint32_t* xmax, int32_t* e6,
                              int8_t* planes6, int64_t pitch6, int64_t plane_stride6, int* status,
                              cudaStream_t st) {
  const long long n = (long long)ng * nao;
  jk_x_scale_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(xmax, n, e6, status);
  dim3 grid((unsigned)((nq + 31) / 32), (unsigned)nao);
  DFE_DISPATCH_S(s, (jk_split_x_kernel<SS><<<grid, 256, 0, st>>>(X, nao, nq, a_pad, qgroup, qcol, gcol, e6, planes6,
                                                                 pitch6, plane_stride6)));
  count_launch(2);
  return cudaGetLastError();
}

cudaError_t launch_jk_k_reduce(const double* Kpart, int ng, int nao, int accumulate, double* K, cudaStream_t st) {
  dim3 grid((unsigned)((nao + 255) / 256), (unsigned)nao);
  jk_k_reduce_kernel<<<grid, 256, 0, st>>>(Kpart, ng, nao, accumulate, K);
  count_launch();
  return cudaGetLastError();
}

cudaError_t launch_jk_j_unpack(const double* Jp, int nao, double* J, cudaStream_t st) {
  dim3 grid((unsigned)((nao + 255) / 256), (unsigned)nao);
  jk_j_unpack_kernel<<<grid, 256, 0, st>>>(Jp, nao, J);
  count_launch();
  return cudaGetLastError();
}

}  // namespace dfe
