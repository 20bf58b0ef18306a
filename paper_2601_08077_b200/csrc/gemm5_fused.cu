// gemm5_fused.cu -- GEMM(5) X = B . C_occ (Eq. 5; blocked Eq. 12) with
// the unpack + split of packed B (rows H1/H2 of SURVEY.md 8(a)) fused into the
// operand producer: the dense INT8 planes of B never exist in HBM.
//
// Rows of the left operand are ordered (i, q): a tile = one i and 128 consecutive q, so the
// element (i, j, q) = B_packed[p(max(i,j), min(i,j))][q] is read as 1 KB runs of 64 packed rows per
// K block (j) -- coalesced along q -- and X comes out as X[i][q][a], the layout GEMM(6) contracts.
//
// A cluster of two CTAs owns one tile: CTA r computes the N half r (80 of a_pad = 160 columns, so
// that all s <= 6 weight accumulators fit its TMEM: s * 80 <= 512 columns).  The FP64 operand is
// staged once per cluster: CTA r copies the q range [64r, 64r+64) of every packed row (1-D bulk
// copies, 16 rows per ring unit) and MULTICASTS it to both CTAs, so B crosses L2 once; each CTA then
// converts all 128 rows into its own shared memory (strided DSMEM stores measured 10x too slow).
// Roles per CTA: warp 0 staging, warp 1 MMA, warp 2 TMA of the C_occ planes, warps 3..6 epilogue,
// warps 7..14 converters (FP64 -> balanced INT8 digits -> swizzled K-major smem tiles).  Barriers:
//   fp_full[unit]  (tx bytes from both CTAs' multicasts)   fp_empty[unit] (4 local + 4 peer warps)
//   full[stage]    (count 257: 256 converter threads + the TMA expect_tx arrive)
//   empty[stage]   (count 1: tcgen05.commit)
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"
#include "internal.h"

namespace dfe {

constexpr int kF5Threads = 480;
constexpr int kF5MaxUnits = 8;       // staging ring units of 16 packed rows x 128 q (16 KB)
constexpr int kF5UnitRows = 16;
constexpr bool kF5Mcast = false;
constexpr bool kF5Exp = false;  // timing experiment only: one 2-D TMA box per unit (wrong rows for j > i)     // stage through multicast (B crosses L2 once per cluster) or per CTA
constexpr int kF5UnitBytes = kF5UnitRows * 128 * 8;
constexpr int kF5BK = 64;            // K block bytes = swizzle span
constexpr int kF5MaxStages = 6;

struct Gemm5FusedParams {
  CUtensorMap mapB2;                 // packed B as [npair][naux] FP64, box (128 q, 16 rows)
  CUtensorMap mapC;                  // C_occ planes [t][a_pad][pitch], box (64, n_half, 1)
  const double* Bp;                  // packed B
  const uint32_t* emax;              // [nao][naux] upper word of max_j |B^q_ij|
  const int32_t* eC;                 // column scales of C_occ
  double* X;                         // [i][nq][a_pad]
  const int* qgroup;                 // [nq] local q-group id
  uint32_t* xmax;                    // [group][nao]
  int* status;
  int nao, naux, qs0, nq, a_pad, n_half, s;
  int tiles_q, num_stages, num_units;
  uint32_t stage_stride;
  long long total_tiles;
  int npairs;
  uint2 pairs[kMaxSlices * (kMaxSlices + 1) / 2];
};

struct PackedWalk {  // packed row of (i, j) for j = j0, j0+1, ...
  long long p;
  int i, j;
  __device__ __forceinline__ PackedWalk(int i_, int j0) : i(i_), j(j0) {
    const long long hi = max(i_, j0), lo = min(i_, j0);
    p = hi * (hi + 1) / 2 + lo;
  }
  __device__ __forceinline__ void next() {
    p += (j < i) ? 1 : (j + 1);
    ++j;
  }
};

template <int S>
__global__ void __launch_bounds__(kF5Threads, 1) gemm5_fused_kernel(const __grid_constant__ Gemm5FusedParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t full_bar[kF5MaxStages];
  __shared__ __align__(8) uint64_t empty_bar[kF5MaxStages];
  __shared__ __align__(8) uint64_t tmem_full_bar;
  __shared__ __align__(8) uint64_t tmem_empty_bar;
  __shared__ __align__(8) uint64_t fp_full[kF5MaxUnits];
  __shared__ __align__(8) uint64_t fp_empty[kF5MaxUnits];
  __shared__ uint32_t tmem_slot;
  __shared__ __align__(16) double epi_stage[4][32][10];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t crank = cluster_ctarank();
  const int St = p.num_stages;
  const int nkb = (p.nao + kF5BK - 1) / kF5BK;
  constexpr uint32_t kAPlane = kTileM * kF5BK;            // 8 KB
  const uint32_t b_plane = (uint32_t)p.n_half * kF5BK;
  const uint32_t b_off = (uint32_t)S * kAPlane;

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&p.mapC);
    for (int i = 0; i < St; ++i) {
      mbar_init(&full_bar[i], 257);
      mbar_init(&empty_bar[i], 1);
    }
    for (int i = 0; i < p.num_units; ++i) {
      mbar_init(&fp_full[i], 1);
      mbar_init(&fp_empty[i], kF5Mcast ? 8 : 4);
    }
    mbar_init(&tmem_full_bar, 1);
    mbar_init(&tmem_empty_bar, 128);
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(&tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = tmem_slot;
  const long long first_tile = blockIdx.x >> 1, tile_step = gridDim.x >> 1;
  uint8_t* fp_ring = smem + (size_t)St * p.stage_stride;  // num_units x 16 KB: [32 packed rows][64 q] doubles
  const int NU = p.num_units;

  if (warp == 0) {
    // ================= FP64 staging: q range [64r, 64r+64) of every packed row, to both CTAs =================
    {  // the whole warp: lane 0 handles the barriers, lanes 0..15 each copy one packed row of the unit
      uint32_t ui = 0;
      const int units_per_tile = 4 * nkb;
      for (long long tile = first_tile; tile < p.total_tiles; tile += tile_step) {
        const int i = (int)(tile / p.tiles_q);
        const int qt0 = (int)(tile - (long long)i * p.tiles_q) * kTileM;
        const int nv_all = max(0, min(128, p.nq - qt0));               // valid q of the tile
        const int nv_mine = max(0, min(64, p.nq - qt0 - (int)crank * 64));  // of this CTA's 64
        const double* bq = p.Bp + p.qs0 + qt0 + (int)crank * 64;
        for (int u = 0; u < units_per_tile; ++u, ++ui) {
          const uint32_t slot = ui % NU, ph = (ui / NU) & 1u;
          const int j0 = u * kF5UnitRows;
          const int nrows = max(0, min(kF5UnitRows, p.nao - j0));
          if (lane == 0) {
            mbar_wait(&fp_empty[slot], ph ^ 1u);
            mbar_expect_tx(&fp_full[slot], kF5Exp ? (nrows > 0 ? (uint32_t)kF5UnitBytes : 0u) : (uint32_t)(nrows * nv_all * 8));
          }
          __syncwarp();
          if (lane < nrows) {
            const int j = j0 + lane;
            const long long hi = max(i, j), lo = min(i, j);
            const long long prow = hi * (hi + 1) / 2 + lo;
            double* dst = reinterpret_cast<double*>(fp_ring + (size_t)slot * kF5UnitBytes) + lane * 128;
            if (kF5Mcast) {
              if (nv_mine > 0)
                bulk_load_1d_mcast(dst + (int)crank * 64, bq + prow * p.naux, (uint32_t)(nv_mine * 8), &fp_full[slot],
                                   (uint16_t)3);
            } else if (nv_all > 0 && !kF5Exp) {
              bulk_load_1d(dst, bq - (int)crank * 64 + prow * p.naux, (uint32_t)(nv_all * 8), &fp_full[slot]);
            } else if (kF5Exp && lane == 0) {  // TIMING EXPERIMENT: one 2-D box, wrong rows for j > i
              tma_load_2d(dst, &p.mapB2, &fp_full[slot], p.qs0 + qt0, (int)prow);
            }
          }
        }
      }
    }
  } else if (warp == 2) {
    // ================= TMA producer: C_occ planes of this CTA's N half =================
    if (lane == 0) {
      uint32_t it = 0;
      for (long long tile = first_tile; tile < p.total_tiles; tile += tile_step) {
        for (int kb = 0; kb < nkb; ++kb, ++it) {
          const uint32_t stage = it % St, ph = (it / St) & 1u;
          mbar_wait(&empty_bar[stage], ph ^ 1u);
          uint8_t* st = smem + (size_t)stage * p.stage_stride;
          mbar_expect_tx(&full_bar[stage], (uint32_t)S * b_plane);
          for (int u = 0; u < S; ++u)
            tma_load_3d(st + b_off + u * b_plane, &p.mapC, &full_bar[stage], kb * kF5BK, (int)crank * p.n_half, u);
        }
      }
    }
  } else if (warp == 1) {
    // ================= MMA issuer =================
    const uint32_t idesc = make_idesc_i8(kTileM, p.n_half);
    const uint64_t desc_proto = make_smem_desc(0, kF5BK);
    const uint32_t desc_hi = (uint32_t)(desc_proto >> 32), desc_lo0 = (uint32_t)desc_proto;
    const uint32_t smem_base16 = (smem_u32(smem) & 0x3FFFFu) >> 4, stage16 = p.stage_stride >> 4;
    uint32_t it = 0, iter = 0;
    for (long long tile = first_tile; tile < p.total_tiles; tile += tile_step, ++iter) {
      if (iter > 0) {
        mbar_wait(&tmem_empty_bar, (iter - 1) & 1u);
        tc_fence_after();
      }
      for (int kb = 0; kb < nkb; ++kb, ++it) {
        const uint32_t stage = it % St, ph = (it / St) & 1u;
        mbar_wait(&full_bar[stage], ph);
        tc_fence_after();
        const uint32_t lo_base = desc_lo0 | (smem_base16 + stage * stage16);
        const int nkk = (min(kF5BK, p.nao - kb * kF5BK) + 31) / 32;
        if (elect_one()) {
          for (int kk = 0; kk < nkk; ++kk) {
            const uint32_t lo = lo_base + 2u * kk;
            const uint32_t later = (kb | kk) ? 1u : 0u;
#pragma unroll 2
            for (int i = 0; i < p.npairs; ++i) {
              const uint2 e = p.pairs[i];
              const uint64_t adesc = ((uint64_t)desc_hi << 32) | (lo + (e.x & 0xFFFFu));
              const uint64_t bdesc = ((uint64_t)desc_hi << 32) | (lo + (e.x >> 16));
              mma_i8_ss(tmem_base + (e.y & 0xFFFFu), adesc, bdesc, idesc, later | (e.y >> 16));
            }
          }
          mma_commit(&empty_bar[stage]);
        }
        __syncwarp();
      }
      if (elect_one()) mma_commit(&tmem_full_bar);
      __syncwarp();
    }
  } else if (warp >= 7) {
    // ================= converters: staged FP64 B -> digit planes in shared memory =================
    const int ct = threadIdx.x - 224;  // 0..255
    const int row = ct & 127;          // row of the A tile = q within the tile
    const int jh = ct >> 7;            // which 32 of the K block's 64 j
    const uint32_t peer = crank ^ 1u;
    // swizzled (SW64) offset of this thread's two 16-byte chunks inside a plane tile
    const uint32_t sw = (uint32_t)((row >> 1) & 3);
    const uint32_t off0 = (uint32_t)row * 64u + (((uint32_t)(2 * jh) ^ sw) << 4);
    const uint32_t off1 = (uint32_t)row * 64u + (((uint32_t)(2 * jh + 1) ^ sw) << 4);
    uint32_t it = 0;
    long long k_wfp = 0, k_conv = 0, k_wst = 0, k_store = 0;
    for (long long tile = first_tile; tile < p.total_tiles; tile += tile_step) {
      const int i = (int)(tile / p.tiles_q);
      const int ql = (int)(tile - (long long)i * p.tiles_q) * kTileM + row;
      const bool q_ok = ql < p.nq;
      double scale = 0.0;
      if (q_ok) {
        const uint32_t hm = p.emax[(long long)i * p.naux + p.qs0 + ql];
        scale = pow2_double(63 - scale_index_from_hi(hm));
        if (jh == 0 && crank == 0) {
          const int stt = status_from_hi(hm);
          if (stt) atomicOr(p.status, stt);
        }
      }
      for (int kb = 0; kb < nkb; ++kb, ++it) {
        const uint32_t stage = it % St, ph = (it / St) & 1u;
        const int j0 = kb * kF5BK + jh * 32;
        const long long c0 = clock64();
        double x[32];
#pragma unroll
        for (int h = 0; h < 2; ++h) {  // this thread's 32 j come from staging units 4 kb + 2 jh + {0, 1}
          const uint32_t ui = 4u * it + 2u * (uint32_t)jh + (uint32_t)h;
          const uint32_t slot = ui % NU, uph = (ui / NU) & 1u;
          const double* src = reinterpret_cast<const double*>(fp_ring + (size_t)slot * kF5UnitBytes) + row;
          mbar_wait(&fp_full[slot], uph);
#pragma unroll
          for (int jj = 0; jj < 16; ++jj) x[16 * h + jj] = (q_ok && j0 + 16 * h + jj < p.nao) ? src[jj * 128] : 0.0;
          __syncwarp();
          if (lane == 0) {  // the unit may be overwritten (by either CTA's multicast) once all 8 warps are done
            const uint32_t eb = smem_u32(&fp_empty[slot]);
            mbar_arrive_cluster(eb);
            if (kF5Mcast) mbar_arrive_cluster(mapa_shared(eb, peer));
          }
        }
        const long long c1 = clock64();
        uint32_t w[S][8];
#pragma unroll
        for (int g4 = 0; g4 < 8; ++g4) {
          uint32_t hi[4], lo[4];
#pragma unroll
          for (int k4 = 0; k4 < 4; ++k4) {
            const uint64_t dg = balanced_digits(x[4 * g4 + k4], scale);
            hi[k4] = (uint32_t)(dg >> 32);
            lo[k4] = (uint32_t)dg;
          }
#pragma unroll
          for (int t = 0; t < S; ++t)
            w[t][g4] = (t < 4) ? pack4_digit(hi[0], hi[1], hi[2], hi[3], 3 - t)
                               : pack4_digit(lo[0], lo[1], lo[2], lo[3], 7 - t);
        }
        const long long c2 = clock64();
        mbar_wait(&empty_bar[stage], ph ^ 1u);
        const long long c3 = clock64();
        uint8_t* stp = smem + (size_t)stage * p.stage_stride;
#pragma unroll
        for (int t = 0; t < S; ++t) {
          *reinterpret_cast<uint4*>(stp + t * kAPlane + off0) = make_uint4(w[t][0], w[t][1], w[t][2], w[t][3]);
          *reinterpret_cast<uint4*>(stp + t * kAPlane + off1) = make_uint4(w[t][4], w[t][5], w[t][6], w[t][7]);
        }
        fence_proxy_async();
        mbar_arrive(&full_bar[stage]);
        const long long c4 = clock64();
        k_wfp += c1 - c0; k_conv += c2 - c1; k_wst += c3 - c2; k_store += c4 - c3;
      }
    }
    if (blockIdx.x == 0 && ct == 0) {
      long long* d = (long long*)(p.status + 16);
      d[0] = k_wfp; d[1] = k_conv; d[2] = k_wst; d[3] = k_store;
    }
  } else {
    // ================= epilogue (warps 3..6): TMEM -> FP64 recombination -> X =================
    const int quarter = warp & 3;
    const int row_local = quarter * 32 + lane;
    const uint32_t t_lane = tmem_base + ((uint32_t)(quarter * 32) << 16);
    const int cpair = (lane & 3) * 2;
    double(*stg)[10] = epi_stage[warp - 3];
    const int col_base = (int)crank * p.n_half;
    uint32_t iter = 0;
    for (long long tile = first_tile; tile < p.total_tiles; tile += tile_step, ++iter) {
      const int i = (int)(tile / p.tiles_q);
      const int ql0 = (int)(tile - (long long)i * p.tiles_q) * kTileM;
      const int ql = ql0 + row_local;
      const bool row_ok = ql < p.nq;
      const int eA = row_ok ? scale_index_from_hi(p.emax[(long long)i * p.naux + p.qs0 + ql]) : 0;
      double* srow[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int qr = ql0 + quarter * 32 + (lane >> 2) + 8 * j;
        srow[j] = (qr < p.nq) ? p.X + ((long long)i * p.nq + qr) * p.a_pad + col_base : nullptr;
      }
      uint32_t hi_max = 0;
      mbar_wait(&tmem_full_bar, iter & 1u);
      tc_fence_after();
      for (int c = 0; c < p.n_half; c += 16) {
        double acc[16];
        int eBv[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          eBv[j] = p.eC[col_base + c + j];
          acc[j] = 0.0;
        }
#pragma unroll
        for (int t = 0; t < S; ++t) {  // w = S + 1 - t: smallest weight first (R6)
          uint32_t v[16];
          tmem_ld16(t_lane + (uint32_t)(t * p.n_half + c), v);
          tmem_ld_wait();
          const int eb = eA + 2 - 8 * (S + 1 - t);
#pragma unroll
          for (int j = 0; j < 16; ++j) acc[j] = fma((double)(int32_t)v[j], pow2_double(eb + eBv[j]), acc[j]);
        }
        if (row_ok) {
#pragma unroll
          for (int j = 0; j < 16; ++j) hi_max = max(hi_max, abs_hi_word(acc[j]));
        }
#pragma unroll
        for (int h = 0; h < 2; ++h) {
#pragma unroll
          for (int k2 = 0; k2 < 4; ++k2)
            *reinterpret_cast<double2*>(&stg[lane][2 * k2]) = make_double2(acc[8 * h + 2 * k2], acc[8 * h + 2 * k2 + 1]);
          __syncwarp();
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const double2 v2 = *reinterpret_cast<const double2*>(&stg[(lane >> 2) + 8 * j][cpair]);
            if (srow[j]) *reinterpret_cast<double2*>(srow[j] + c + 8 * h + cpair) = v2;
          }
          __syncwarp();
        }
      }
      tc_fence_before();
      mbar_arrive(&tmem_empty_bar);
      if (row_ok) atomicMax(&p.xmax[(long long)p.qgroup[ql] * p.nao + i], hi_max);
    }
  }

  tc_fence_before();
  __syncthreads();
  cluster_sync_all();  // no CTA leaves while its peer may still write into it
  if (warp == 1) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

// ---------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn5)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

bool gemm5_fused_supported(int nao, int a_pad, int s) {
  // two N halves of a multiple of 16 columns, all s accumulators of a half in 512 TMEM columns,
  // at least two pipeline stages in shared memory
  if (a_pad % 32 != 0 || s < 1 || s > kMaxSlices) return false;
  const int n_half = a_pad / 2;
  if (s * n_half > 512) return false;
  const int64_t stride = round_up((int64_t)s * (kTileM + n_half) * kF5BK, 1024);
  return (232448 - 12288 - 2048 - 3 * kF5UnitBytes) / stride >= 2 && nao >= 1;
}

cudaError_t launch_gemm5_fused(const Gemm5FusedProblem& g, cudaStream_t st) {
  static EncodeTiledFn5 encode = nullptr;
  if (!encode) {
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess)
      return cudaErrorInvalidValue;
    encode = (EncodeTiledFn5)ptr;
  }
  Gemm5FusedParams p;
  const int s = g.s, n_half = g.a_pad / 2;
  {
    cuuint64_t dims[3] = {(cuuint64_t)g.nao, (cuuint64_t)g.a_pad, (cuuint64_t)s};
    cuuint64_t strides[2] = {(cuuint64_t)g.c_pitch, (cuuint64_t)g.c_plane_stride};
    cuuint32_t box[3] = {(cuuint32_t)kF5BK, (cuuint32_t)n_half, 1u};
    cuuint32_t estr[3] = {1u, 1u, 1u};
    if (encode(&p.mapC, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, (void*)g.planesC, dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  {
    const long long npair = (long long)g.nao * (g.nao + 1) / 2;
    cuuint64_t dims[2] = {(cuuint64_t)g.naux, (cuuint64_t)npair};
    cuuint64_t strides[1] = {(cuuint64_t)g.naux * 8};
    cuuint32_t box[2] = {128u, (cuuint32_t)kF5UnitRows};
    cuuint32_t estr[2] = {1u, 1u};
    if (encode(&p.mapB2, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void*)g.Bp, dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cudaErrorInvalidValue;
  }
  p.Bp = g.Bp;
  p.emax = g.emax;
  p.eC = g.eC;
  p.X = g.X;
  p.qgroup = g.qgroup;
  p.xmax = g.xmax;
  p.status = g.status;
  p.nao = g.nao;
  p.naux = g.naux;
  p.qs0 = g.qs0;
  p.nq = g.nq;
  p.a_pad = g.a_pad;
  p.n_half = n_half;
  p.s = s;
  p.tiles_q = (g.nq + kTileM - 1) / kTileM;
  p.total_tiles = (long long)g.nao * p.tiles_q;
  p.stage_stride = (uint32_t)round_up((int64_t)s * (kTileM + n_half) * kF5BK, 1024);
  // shared memory: MMA stages first, the rest (at least 3 units) is the FP64 staging ring
  const int64_t budget = 232448 - 12288 - 2048;
  p.num_stages = (int)((budget - 4 * kF5UnitBytes) / p.stage_stride);
  if (p.num_stages < 2) p.num_stages = 2;
  if (p.num_stages > 3) p.num_stages = 3;
  p.num_units = (int)((budget - (int64_t)p.num_stages * p.stage_stride) / kF5UnitBytes);
  if (p.num_units > kF5MaxUnits) p.num_units = kF5MaxUnits;
  if (p.num_units < 3) return cudaErrorInvalidValue;
  {  // slice pairs, round-robin over the weights (consecutive MMAs hit different accumulators)
    const uint32_t a_plane = kTileM * kF5BK, b_plane = (uint32_t)n_half * kF5BK, b_off = (uint32_t)s * a_plane;
    int np = 0, next_t[kMaxSlices + 2];
    for (int w = 2; w <= s + 1; ++w) next_t[w] = 1;
    for (bool any = true; any;) {
      any = false;
      for (int w = s + 1; w >= 2; --w) {
        const int t = next_t[w], t_hi = (w - 1) < s ? (w - 1) : s;
        if (t > t_hi) continue;
        any = true;
        next_t[w] = t + 1;
        p.pairs[np].x = (((uint32_t)(t - 1) * a_plane) >> 4) | (((b_off + (uint32_t)(w - t - 1) * b_plane) >> 4) << 16);
        p.pairs[np].y = (uint32_t)((s + 1 - w) * n_half) | ((t > 1 ? 1u : 0u) << 16);
        ++np;
      }
    }
    p.npairs = np;
  }
  static int num_sms = 0;
  if (!num_sms) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
  }
  long long nclusters = num_sms / 2;
  if (nclusters > p.total_tiles) nclusters = p.total_tiles;
  const size_t smem = (size_t)p.num_stages * p.stage_stride + (size_t)p.num_units * kF5UnitBytes + 1024;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(2 * nclusters), 1, 1);
  cfg.blockDim = dim3(kF5Threads, 1, 1);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  cudaError_t err;
#define DFE_F5(SV)                                                                                          \
  case SV:                                                                                                  \
    err = cudaFuncSetAttribute(gemm5_fused_kernel<SV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
    if (err != cudaSuccess) return err;                                                                     \
    err = cudaLaunchKernelEx(&cfg, gemm5_fused_kernel<SV>, p);                                              \
    break;
  switch (s) {
    DFE_F5(1) DFE_F5(2) DFE_F5(3) DFE_F5(4) DFE_F5(5) DFE_F5(6) DFE_F5(7) DFE_F5(8)
    default: return cudaErrorInvalidValue;
  }
#undef DFE_F5
  if (err != cudaSuccess) return err;
  count_launch();
  return cudaGetLastError();
}

}  // namespace dfe
