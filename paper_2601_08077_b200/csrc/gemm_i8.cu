// gemm_i8.cu -- the INT8 slice-pair GEMM with fused FP64 recombination (rows H3, H4, H7 of
// SURVEY.md section 8(a)); hand-written tcgen05.mma.kind::i8 for sm_100a.
//
// What one CTA computes (R3, R4, R6):
//   for one 128 x n_tile output tile and one z item (a q-group, or the whole contraction),
//   for each flush chunk of the contraction (<= kflush(s) elements, increasing k),
//     for each pass (a run of at most W = 512 / n_tile weights, largest w first),
//       P^(w) = sum_{t+u=w} D^A_t . D^B_u^T        -- INT32 accumulators in TMEM, one per weight
//       out  += 2^(eA_i + eB_j + 2 - 8 w) P^(w)    -- w descending, ONE running FP64 sum
//
// Structure: warp 0 = TMA producer (one lane), warp 1 = TMEM allocator + MMA issuer (one lane),
// warps 2..9 = epilogue (TMEM lane quarter = warp % 4, two warps per quarter).  All s digit planes
// of a K block sit in shared memory together, so 2 s plane tiles feed up to s(s+1)/2 MMAs (SURVEY
// section 7, hard part 4).  Operands are K-major INT8 planes; the K-block width BK equals the
// TMA/UMMA swizzle span (32, 64 or 128 bytes): the widest one that still leaves two stages.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "common.cuh"
#include "internal.h"

namespace dfe {

constexpr int kMaxStages = 8;
#ifndef DFE_EPI_PER_QUARTER
#define DFE_EPI_PER_QUARTER 2
#endif
constexpr int kEpiPerQuarter = DFE_EPI_PER_QUARTER;  // epilogue warps per TMEM lane quarter
constexpr int kEpiWarps = 4 * kEpiPerQuarter;
constexpr int kGemmThreads = 64 + 32 * kEpiWarps;  // warp 0 TMA, warp 1 MMA, warps 2.. epilogue
// 227 KB minus the static shared memory (barriers, epilogue staging, column scales)
constexpr int kSmemLimit = 232448 - (kEpiWarps * 1280 + 2048 + 512);

struct GemmKernelParams {
  CUtensorMap mapA;
  CUtensorMap mapB;
  CUtensorMap mapBh;  // B planes with a 64-row box (cta_group::2 pair: each CTA holds half of the N rows)
  CUtensorMap mapA2;  // A planes with a 64-row box (cluster pair: each CTA loads and multicasts half a tile)
  int s, n_tile, acc_stride, weights_per_pass;
  // pass structure: weights_per_pass weights in pass 0; tp = 1 ("TMEM partial"): the FP64 running
  // sum stays in TMEM between passes (low words in accumulator slot 0, high words in slot 1) and
  // later passes use slots 2.. (weights_later each); tp = 0: every pass takes weights_per_pass and
  // the running sum is read-modify-written in global memory
  int tp, weights_later, npass;
  int tiles_m, tiles_n, group_m, tiles_per_z, pair;
  long long total_work;
  int num_stages;
  uint32_t stage_stride;
  long long a_rows, b_rows;
  int k;  // contraction extent
  int kflush;
  const int* zk;
  const int32_t* eA;
  const int32_t* eB;
  long long ea_stride, eb_stride;
  int lower_only, mode;
  double* C;
  long long ldc, c_stride;
  int nao, x_cols;
  long long ldx;
  const int* qgroup;
  uint32_t* xmax;
  const uint32_t* kmask;  // screening: active 128-column K blocks per 256-row block (null: all)
  int kmask_words;
  int32_t* P;
  int dbg_chunk;
  // flattened slice-pair list: x = A plane offset>>4 within a stage, y = B plane offset>>4,
  // z = accumulator column, w = accumulate-from-the-start flag (one 16-byte constant load and four
  // uniform adds per MMA: the packed 8-byte form cost 12 uniform instructions per MMA, which at
  // N = 80 is the MMA's own duration); pass ps owns [pass_start[ps], pass_start[ps+1])
  uint4 pairs[kMaxSlices * (kMaxSlices + 1) / 2];
  int pass_start[kMaxSlices + 1];
  int dbg_flags;  // bit 0: no MMAs (operand feed only); bit 1: no TMA loads (MMA issue only); bit 2: no 256-bit epilogue accesses
};

// weights of pass `ps`: w_hi down to w_lo; weight w accumulates in TMEM slot slot0 + (w_hi - w)
__device__ __forceinline__ void pass_weights(const GemmKernelParams& p, int ps, int& w_hi, int& w_lo, int& slot0) {
  const int W = p.weights_per_pass;
  if (!p.tp || ps == 0) {
    w_hi = p.s + 1 - ps * W;
    w_lo = max(2, w_hi - W + 1);
    slot0 = 0;
  } else {
    w_hi = p.s + 1 - W - (ps - 1) * p.weights_later;
    w_lo = max(2, w_hi - p.weights_later + 1);
    slot0 = 2;
  }
}

// Screening (GEMM(5), internal.h GemmProblem::kmask): the K blocks of a tile that are loaded and
// multiplied.  Bit J of the mask covers the contraction range [128 J, 128 J + 128), i.e. 128 / BK
// consecutive K blocks.  Producer and MMA issuer walk the same sequence of active blocks.
template <int BK>
struct KBlocks {
  uint32_t m[4];
  __device__ __forceinline__ void load(const GemmKernelParams& p, int tm) {
    if (p.kmask) {
      const uint32_t* src = p.kmask + (long long)(tm >> 1) * p.kmask_words;
#pragma unroll
      for (int w = 0; w < 4; ++w) m[w] = w < p.kmask_words ? src[w] : 0u;
    } else {
#pragma unroll
      for (int w = 0; w < 4; ++w) m[w] = 0xffffffffu;
    }
  }
  __device__ __forceinline__ bool active(int kb) const {
    const int J = (kb * BK) >> 7, wi = J >> 5;
    const uint32_t w = wi == 0 ? m[0] : wi == 1 ? m[1] : wi == 2 ? m[2] : m[3];  // no dynamic register indexing
    return (w >> (J & 31)) & 1u;
  }
  __device__ __forceinline__ int count(int nkb) const {
    int n = 0;
    for (int kb = 0; kb < nkb; ++kb) n += active(kb) ? 1 : 0;
    return n;
  }
};

// One unit of work of the persistent kernel: an output tile of one z item.
struct WorkItem {
  int tm, tn, z, zk0, zk1, chunk_lo, chunk_hi;
};

// Work index -> tile.  z is the slowest index; inside a z item tiles are rasterised in bands of
// group_m tile rows (operand reuse in L2), or -- lower_only -- over the pairs tm >= tn.
__device__ __forceinline__ WorkItem decode_work(const GemmKernelParams& p, long long wi) {
  WorkItem w;
  w.z = (int)(wi / p.tiles_per_z);
  const int lin = (int)(wi - (long long)w.z * p.tiles_per_z);
  if (p.lower_only && p.pair) {
    // pairs of M tiles (256 rows) against N tiles of 128: tn <= 2 tm2 + 1; a(a+1) items precede row a
    int a = (int)((sqrtf(4.0f * (float)lin + 1.0f) - 1.0f) * 0.5f);
    while ((a + 1) * (a + 2) <= lin) ++a;
    while (a * (a + 1) > lin) --a;
    w.tm = a;
    w.tn = lin - a * (a + 1);
  } else if (p.lower_only) {
    int a = (int)((sqrtf(8.0f * (float)lin + 1.0f) - 1.0f) * 0.5f);
    while ((a + 1) * (a + 2) / 2 <= lin) ++a;
    while (a * (a + 1) / 2 > lin) --a;
    w.tm = a;
    w.tn = lin - a * (a + 1) / 2;
  } else {
    const int per_band = p.group_m * p.tiles_n;
    const int band = lin / per_band;
    const int first_m = band * p.group_m;
    const int gm = min(p.group_m, p.tiles_m - first_m);
    const int r = lin - band * per_band;
    w.tm = first_m + r % gm;
    w.tn = r / gm;
  }
  w.zk0 = p.zk ? p.zk[w.z] : 0;
  w.zk1 = p.zk ? p.zk[w.z + 1] : p.k;
  w.chunk_lo = 0;
  w.chunk_hi = max(1, (w.zk1 - w.zk0 + p.kflush - 1) / p.kflush);
  if (p.mode == kEpiInt32) {
    w.chunk_lo = p.dbg_chunk;
    w.chunk_hi = p.dbg_chunk + 1;
  }
  return w;
}

#define DFE_WORK_LOOP                                                                  \
  for (long long wi = (CL == 1) ? (long long)blockIdx.x                                \
                      : (CL == 2) ? (long long)(blockIdx.x & ~1u) + crank              \
                                  : (long long)(blockIdx.x >> 1);                      \
       wi < p.total_work; wi += (CL == 4) ? (gridDim.x >> 1) : gridDim.x) {            \
    const WorkItem wk = decode_work(p, wi);                                            \
    if (CL == 4 && wk.tn >= p.tiles_n) continue; /* ragged last pair row, lower_only */ \
    const int tm = (CL == 4) ? 2 * wk.tm + (int)crank : wk.tm;                         \
    const int tn = wk.tn, z = wk.z, zk0 = wk.zk0, zk1 = wk.zk1;                        \
    const int chunk_lo = wk.chunk_lo, chunk_hi = wk.chunk_hi;                          \
    (void)tm; (void)tn; (void)z; (void)zk0; (void)zk1;

// Persistent: grid = min(work items, SMs); every role walks the same work sequence, the pipeline
// counters run on across tiles, so the producer prefetches the next tile during the epilogue.
template <int BK, int CL>
__global__ void __launch_bounds__(kGemmThreads, 1) gemm_i8_kernel(const __grid_constant__ GemmKernelParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t full_bar[kMaxStages];
  __shared__ __align__(8) uint64_t empty_bar[kMaxStages];
  __shared__ __align__(8) uint64_t tmem_full_bar;
  __shared__ __align__(8) uint64_t tmem_empty_bar;
  __shared__ uint32_t tmem_slot;
  __shared__ __align__(16) double epi_stage[kEpiWarps][16][10];  // per epilogue warp: 16 rows x 8 cols, 80 B pitch
  __shared__ int eb_sh[2][256];  // scale indices of the tile's columns (double buffered over tiles)

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int s = p.s;
  const int npass = p.npass;
  const int S = p.num_stages;
  // CL == 2: a cluster of two CTAs owns the two N tiles of one M tile (work items 2c, 2c+1); each
  // loads half of every A plane tile and multicasts it to both, so the A operand crosses L2 once.
  // CL == 4: the pair runs cta_group::2 MMAs of M = 256: CTA r owns rows 128 r .. 128 r + 127 of the
  // 256-row tile and holds N rows 64 r .. 64 r + 63 of every B plane tile; CTA 0 issues.
  const uint32_t crank = (CL != 1) ? cluster_ctarank() : 0u;
  (void)crank;

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&p.mapA);
    prefetch_tensormap(&p.mapB);
    for (int i = 0; i < S; ++i) {
      mbar_init(&full_bar[i], 1);
      mbar_init(&empty_bar[i], CL == 2 ? 2 : 1);
    }
    mbar_init(&tmem_full_bar, 1);
    mbar_init(&tmem_empty_bar, CL == 4 ? 2 * kEpiWarps : kGemmThreads - 64);  // pair: one arrival per epilogue warp of both CTAs
    fence_barrier_init();
  }
  if (warp == 1) {
    if (CL == 4) tmem_alloc_pair(&tmem_slot, 512);
    else tmem_alloc(&tmem_slot, 512);
  }
  tc_fence_before();
  __syncthreads();
  if (CL != 1) cluster_sync_all();  // the peer's barriers are initialised before anything arrives on them
  tc_fence_after();
  const uint32_t tmem_base = tmem_slot;

  const uint32_t a_plane_bytes = kTileM * BK;
  const uint32_t b_plane_bytes = (uint32_t)(CL == 4 ? p.n_tile / 2 : p.n_tile) * BK;
  const uint32_t b_off = (uint32_t)s * a_plane_bytes;

  if (warp == 0) {
    // ================= TMA producer =================
    if (lane == 0) {
      uint32_t it = 0;
      DFE_WORK_LOOP
      KBlocks<BK> kbl;
      kbl.load(p, tm);
      for (int ch = chunk_lo; ch < chunk_hi; ++ch) {
        const int kc0 = zk0 + ch * p.kflush;
        const int kc1 = min(zk1, kc0 + p.kflush);
        const int nkb = (kc1 - kc0 + BK - 1) / BK;
        const int nact = p.kmask ? kbl.count(nkb) : nkb;  // active K blocks (screening)
        for (int ps = 0; ps < npass; ++ps) {
          int w_hi, w_lo, slot0;
          pass_weights(p, ps, w_hi, w_lo, slot0);
          const int P = min(s, w_hi - 1);
          // a pass that needs P < s planes packs kp = s / P consecutive K blocks into one stage
          // (K block j of plane t in plane slot j P + t): fewer, fuller stages -- the one-plane
          // pass of a two-pass tile was waiting 1230 cycles per K block for 4 MMAs
          const int kp = s / P;
          int kb = 0;
          for (int left = nact; left > 0; ++it) {
            const uint32_t stage = it % S;
            const uint32_t ph = (it / S) & 1u;
            const int nj = min(kp, left);  // K blocks in this stage
            left -= nj;
            mbar_wait(&empty_bar[stage], ph ^ 1u);
            if (p.dbg_flags & 2) {
              if (CL != 4 || crank == 0) mbar_arrive(&full_bar[stage]);
              continue;
            }
            uint8_t* st = smem + (size_t)stage * p.stage_stride;
            const uint32_t tx = (uint32_t)(nj * P) * (a_plane_bytes + b_plane_bytes);
            if (CL == 4) {
              // both CTAs' loads count on the LEADER's full barrier, which expects the bytes of both
              const uint32_t lead_bar = mapa_shared(smem_u32(&full_bar[stage]), 0u);
              if (crank == 0) mbar_expect_tx(&full_bar[stage], 2u * tx);
              for (int j = 0; j < nj; ++j, ++kb) {
                while (!kbl.active(kb)) ++kb;
                const int kpos = kc0 + kb * BK;
                for (int t = 0; t < P; ++t)
                  tma_load_3d_pair(st + (j * P + t) * a_plane_bytes, &p.mapA, lead_bar, kpos, tm * kTileM, t);
                for (int u = 0; u < P; ++u)
                  tma_load_3d_pair(st + b_off + (j * P + u) * b_plane_bytes, &p.mapBh, lead_bar, kpos,
                                   tn * p.n_tile + (int)crank * (p.n_tile / 2), u);
              }
              continue;
            }
            mbar_expect_tx(&full_bar[stage], tx);
            for (int j = 0; j < nj; ++j, ++kb) {
              while (!kbl.active(kb)) ++kb;
              const int kpos = kc0 + kb * BK;
              if (CL == 2) {
                for (int t = 0; t < P; ++t)
                  tma_load_3d_mcast(st + (j * P + t) * a_plane_bytes + crank * (64 * BK), &p.mapA2, &full_bar[stage],
                                    kpos, tm * kTileM + (int)crank * 64, t, (uint16_t)3);
              } else {
                for (int t = 0; t < P; ++t)
                  tma_load_3d(st + (j * P + t) * a_plane_bytes, &p.mapA, &full_bar[stage], kpos, tm * kTileM, t);
              }
              for (int u = 0; u < P; ++u)
                tma_load_3d(st + b_off + (j * P + u) * b_plane_bytes, &p.mapB, &full_bar[stage], kpos,
                            tn * p.n_tile, u);
            }
          }
        }
      }
      }  // work loop
    }
  } else if (warp == 1) {
    // ================= MMA issuer =================
    // The whole warp runs this loop with warp-uniform control flow and one elected lane issues,
    // so descriptors live in uniform registers.  The (w, t, u) nest is flattened on the host into
    // p.pairs (constant bank): per MMA the loop adds two 16-bit offsets to the descriptor address
    // field -- far fewer issue cycles than the MMA's own 64+ cycles.
    const uint32_t idesc = make_idesc_i8(CL == 4 ? 2 * kTileM : kTileM, p.n_tile);
    const uint64_t desc_proto = make_smem_desc(0, BK);
    const uint32_t desc_hi = (uint32_t)(desc_proto >> 32);
    const uint32_t desc_lo0 = (uint32_t)desc_proto;  // LBO field, address 0
    const uint32_t smem_base16 = (smem_u32(smem) & 0x3FFFFu) >> 4;
    const uint32_t stage16 = p.stage_stride >> 4;
    uint32_t it = 0, iter = 0;
    if (CL != 4 || crank == 0) {  // pair mode: only the leader CTA issues (and waits)
    DFE_WORK_LOOP
    KBlocks<BK> kbl;
    kbl.load(p, tm);
    for (int ch = chunk_lo; ch < chunk_hi; ++ch) {
      const int kc0 = zk0 + ch * p.kflush;
      const int kc1 = min(zk1, kc0 + p.kflush);
      const int nkb = (kc1 - kc0 + BK - 1) / BK;
      const int nact = p.kmask ? kbl.count(nkb) : nkb;  // active K blocks (screening)
      for (int ps = 0; ps < npass; ++ps, ++iter) {
        const int pr0 = p.pass_start[ps], pr1 = p.pass_start[ps + 1];
        if (iter > 0) {
          mbar_wait(&tmem_empty_bar, (iter - 1) & 1u);
          tc_fence_after();
        }
        int w_hi_p, w_lo_p, slot0_p;
        pass_weights(p, ps, w_hi_p, w_lo_p, slot0_p);
        const int P = min(s, w_hi_p - 1);
        const int kp = s / P;  // K blocks per stage (see the producer)
        const uint32_t a_sub16 = (uint32_t)P * (a_plane_bytes >> 4), b_sub16 = (uint32_t)P * (b_plane_bytes >> 4);
        int kb = 0;
        uint32_t started = 0u;  // the accumulators of this pass hold a product already
        for (int left = nact; left > 0; ++it) {
          const uint32_t stage = it % S;
          const uint32_t ph = (it / S) & 1u;
          const int nj = min(kp, left);
          left -= nj;
          mbar_wait(&full_bar[stage], ph);
          tc_fence_after();
          if (p.dbg_flags & 1) {
            if (lane == 0) {
              if (CL == 4 || CL == 2) {
                mbar_arrive_cluster(mapa_shared(smem_u32(&empty_bar[stage]), 0u));
                mbar_arrive_cluster(mapa_shared(smem_u32(&empty_bar[stage]), 1u));
              } else {
                mbar_arrive(&empty_bar[stage]);
              }
            }
            continue;
          }
          const uint32_t lo_base = desc_lo0 | (smem_base16 + stage * stage16);
          // every lane walks the active blocks of this stage (kb stays warp-uniform); the elected lane issues
          int kb_end = kb;
          for (int j = 0; j < nj; ++j, ++kb_end)
            while (!kbl.active(kb_end)) ++kb_end;
          if (elect_one()) {
            int kbe = kb;
            for (int j = 0; j < nj; ++j, ++kbe) {
              while (!kbl.active(kbe)) ++kbe;
              const int kpos = kc0 + kbe * BK;
              const int nkk = (min(BK, kc1 - kpos) + 31) / 32;
              const uint32_t aj = (uint32_t)j * a_sub16, bj = (uint32_t)j * b_sub16;
              for (int kk = 0; kk < nkk; ++kk) {
                const uint32_t lo = lo_base + 2u * kk;  // +32 bytes per K step, in 16-byte units
                const uint32_t later = started;
                started = 1u;
#pragma unroll 4
                for (int i = pr0; i < pr1; ++i) {
                  const uint4 e = p.pairs[i];
                  const uint64_t adesc = ((uint64_t)desc_hi << 32) | (lo + e.x + aj);
                  const uint64_t bdesc = ((uint64_t)desc_hi << 32) | (lo + e.y + bj);
                  if (CL == 4) mma_i8_ss_pair(tmem_base + e.z, adesc, bdesc, idesc, later | e.w);
                  else mma_i8_ss(tmem_base + e.z, adesc, bdesc, idesc, later | e.w);
                }
              }
            }
            // frees the smem stage once these MMAs have read it (in both CTAs of a pair: the peer
            // multicasts into this stage too)
            if (CL == 4) mma_commit_pair(&empty_bar[stage], (uint16_t)3);
            else if (CL == 2) mma_commit_mcast(&empty_bar[stage], (uint16_t)3);
            else mma_commit(&empty_bar[stage]);
          }
          started = 1u;  // warp-uniform copies of the elected lane's state
          kb = kb_end;
          __syncwarp();
        }
        if (elect_one()) {  // accumulators of this pass are complete (in both CTAs of a pair)
          if (CL == 4) mma_commit_pair(&tmem_full_bar, (uint16_t)3);
          else mma_commit(&tmem_full_bar);
        }
        __syncwarp();
      }
    }
    }  // work loop
    }
  } else {
    // ================= epilogue: TMEM -> FP64 recombination -> global =================
    const int quarter = warp & 3;
    uint32_t iter = 0, tile_no = 0;
    DFE_WORK_LOOP
    // the column scale indices of this tile, staged once by the 256 epilogue threads (they were 16
    // global loads at the head of every 16-column chunk, on the epilogue's critical path)
    int* const ebs = eb_sh[tile_no & 1u];
    ++tile_no;
    {
      const int et = (warp - 2) * 32 + lane;
      const long long col = (long long)tn * p.n_tile + et;
      if (et < 256)
        ebs[et] = (p.mode != kEpiInt32 && et < p.n_tile && col < p.b_rows) ? p.eB[z * p.eb_stride + col] : 0;
      asm volatile("bar.sync 1, %0;" ::"n"(32 * kEpiWarps) : "memory");  // epilogue warps only; buffer tile_no & 1 is free again
    }                                                  // once every warp has passed the next tile's barrier
    const int row_local = quarter * 32 + lane;
    const long long row = (long long)tm * kTileM + row_local;
    const bool row_ok = row < p.a_rows;
    const int eA = (row_ok && p.mode != kEpiInt32) ? p.eA[z * p.ea_stride + row] : 0;
    const uint32_t t_lane = tmem_base + ((uint32_t)(quarter * 32) << 16);
    const int col0 = tn * p.n_tile;

    double* out = nullptr;
    if (p.mode == kEpiC) {
      out = p.C + z * p.c_stride + row * p.ldc;
    } else if (p.mode == kEpiX) {
      out = p.C + row * p.ldx;  // X[(q, i)][a_pad]: the tile is one contiguous block
    }
    // two epilogue warps per lane quarter: warps 2..5 take the even 16-column blocks, 6..9 the odd
    const int chalf = (warp - 2) >> 2;
    // coalesced phase: lane moves columns cpair, cpair+1 (of an 8-column half block) of rows
    // (lane >> 2) + 8 j, j = 0..3: one store instruction covers 8 rows x 64 bytes
    const int cpair = (lane & 3) * 2;
    double(*stg)[10] = epi_stage[warp - 2];
    double* srow[4];
    const long long ld_out = (p.mode == kEpiX) ? p.ldx : p.ldc;
    const bool vec_ok = p.mode != kEpiInt32 && ((ld_out | p.c_stride | (long long)col0) & 1) == 0 &&
                        ((uintptr_t)p.C & 15) == 0;
    // whole 32-byte sectors per lane (256-bit accesses): the thread's own row, no transposition
    const bool v4_ok = vec_ok && ((ld_out | p.c_stride | (long long)col0) & 3) == 0 && ((uintptr_t)p.C & 31) == 0 &&
                       !(p.dbg_flags & 4);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const long long rr = (long long)tm * kTileM + quarter * 32 + (lane >> 2) + 8 * j;
      srow[j] = nullptr;
      if (rr < p.a_rows) {
        if (p.mode == kEpiC) {
          srow[j] = p.C + z * p.c_stride + rr * p.ldc;
        } else if (p.mode == kEpiX) {
          srow[j] = p.C + rr * p.ldx;
        }
      }
    }
    uint32_t hi_max = 0;
    for (int ch = chunk_lo; ch < chunk_hi; ++ch) {
      for (int ps = 0; ps < npass; ++ps, ++iter) {
        int w_hi, w_lo, slot0;
        pass_weights(p, ps, w_hi, w_lo, slot0);
        const bool first = (ch == chunk_lo) && (ps == 0);
        const bool last = (ch == chunk_hi - 1) && (ps == npass - 1);
        mbar_wait(&tmem_full_bar, iter & 1u);
        tc_fence_after();
        for (int c = chalf * 16; c < p.n_tile; c += 16 * kEpiPerQuarter) {
          uint32_t v[16];
          if (p.mode == kEpiInt32) {
            for (int w = w_hi; w >= w_lo; --w) {
              tmem_ld16(t_lane + (uint32_t)((slot0 + w_hi - w) * p.acc_stride + c), v);
              tmem_ld_wait();
              if (row_ok) {
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                  const long long col = col0 + c + j;
                  if (col < p.b_rows) p.P[((long long)(w - 2) * p.a_rows + row) * p.b_rows + col] = (int32_t)v[j];
                }
              }
            }
            continue;
          }
          double acc[16];
          int eBv[16];
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            eBv[j] = row_ok ? ebs[c + j] : 0;
            acc[j] = 0.0;
          }
          if (!first && p.tp) {
            // running sum of the earlier passes: low words in slot 0, high words in slot 1
            uint32_t plo[16];
            tmem_ld16(t_lane + (uint32_t)c, plo);
            tmem_ld16(t_lane + (uint32_t)(p.acc_stride + c), v);
            tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 16; ++j) acc[j] = __hiloint2double((int)v[j], (int)plo[j]);
          } else if (!first) {
            // running sum of the earlier passes/chunks: one 32-byte sector per lane and load, or
            // coalesced 16-byte loads (4 lanes cover 64 bytes of a row), transposed through shared
            // memory to "lane = row"
            if (v4_ok) {
              if (row_ok) {
#pragma unroll
                for (int k4 = 0; k4 < 4; ++k4) {
                  const long long colv = col0 + c + 4 * k4;
                  if (colv + 3 < p.b_rows) {
                    ld_global_v4f64(out + colv, acc[4 * k4], acc[4 * k4 + 1], acc[4 * k4 + 2], acc[4 * k4 + 3]);
                  } else {
#pragma unroll
                    for (int j = 0; j < 4; ++j)
                      if (colv + j < p.b_rows) acc[4 * k4 + j] = out[colv + j];
                  }
                }
              }
            } else if (vec_ok) {
#pragma unroll
              for (int h = 0; h < 2; ++h) {
                const long long colv = col0 + c + 8 * h + cpair;
#pragma unroll
                for (int r = 0; r < 2; ++r) {  // 16 rows per round (the staging tile holds 16)
#pragma unroll
                  for (int jj = 0; jj < 2; ++jj) {
                    const int j = 2 * r + jj;
                    double2 v2 = make_double2(0.0, 0.0);
                    if (srow[j] && colv + 1 < p.b_rows) v2 = *reinterpret_cast<const double2*>(srow[j] + colv);
                    else if (srow[j] && colv < p.b_rows) v2.x = srow[j][colv];
                    *reinterpret_cast<double2*>(&stg[(lane >> 2) + 8 * jj][cpair]) = v2;
                  }
                  __syncwarp();
                  if ((lane >> 4) == r) {
#pragma unroll
                    for (int k2 = 0; k2 < 4; ++k2) {
                      const double2 v2 = *reinterpret_cast<const double2*>(&stg[lane & 15][2 * k2]);
                      acc[8 * h + 2 * k2] = v2.x;
                      acc[8 * h + 2 * k2 + 1] = v2.y;
                    }
                  }
                  __syncwarp();
                }
              }
            } else {
#pragma unroll
              for (int j = 0; j < 16; ++j) {
                const long long col = col0 + c + j;
                if (row_ok && col < p.b_rows) acc[j] = out[col];
              }
            }
          }
          if (first) {
            // Nothing accumulated yet: sum_w 2^(eb_w) P_w, w descending, in Horner form
            // t = P_whi; t = fma(t, 2^-8, P_w); acc = t 2^(eb_wlo).  The scale factors are exact
            // powers of two, so every rounding is the rounding of the running sum of R6 scaled by one:
            // the same bits with one multiply-add per term and one scale per element.
            for (int w = w_hi; w >= w_lo; --w) {
              tmem_ld16(t_lane + (uint32_t)((slot0 + w_hi - w) * p.acc_stride + c), v);
              tmem_ld_wait();
              if (w == w_hi) {
#pragma unroll
                for (int j = 0; j < 16; ++j) acc[j] = (double)(int32_t)v[j];
              } else {
#pragma unroll
                for (int j = 0; j < 16; ++j) acc[j] = fma(acc[j], 0x1p-8, (double)(int32_t)v[j]);
              }
            }
            const int eb = eA + 2 - 8 * w_lo;
#pragma unroll
            for (int j = 0; j < 16; ++j) acc[j] *= pow2_double(eb + eBv[j]);
          } else {
            for (int w = w_hi; w >= w_lo; --w) {
              tmem_ld16(t_lane + (uint32_t)((slot0 + w_hi - w) * p.acc_stride + c), v);
              tmem_ld_wait();
              const int eb = eA + 2 - 8 * w;
#pragma unroll
              for (int j = 0; j < 16; ++j)
                acc[j] = fma((double)(int32_t)v[j], pow2_double(eb + eBv[j]), acc[j]);
            }
          }
          if (last && row_ok) {
#pragma unroll
            for (int j = 0; j < 16; ++j)
              if (col0 + c + j < p.b_rows) hi_max = max(hi_max, abs_hi_word(acc[j]));
          }
          if (p.tp && !last) {
            // park the running sum in TMEM (the columns this block of slots 0 and 1 just gave up)
            uint32_t plo[16];
#pragma unroll
            for (int j = 0; j < 16; ++j) {
              plo[j] = (uint32_t)__double2loint(acc[j]);
              v[j] = (uint32_t)__double2hiint(acc[j]);
            }
            tmem_st16(t_lane + (uint32_t)c, plo);
            tmem_st16(t_lane + (uint32_t)(p.acc_stride + c), v);
          } else if (v4_ok) {
            if (row_ok) {
#pragma unroll
              for (int k4 = 0; k4 < 4; ++k4) {
                const long long colv = col0 + c + 4 * k4;
                if (colv + 3 < p.b_rows) {
                  st_global_v4f64(out + colv, acc[4 * k4], acc[4 * k4 + 1], acc[4 * k4 + 2], acc[4 * k4 + 3]);
                } else {
#pragma unroll
                  for (int j = 0; j < 4; ++j)
                    if (colv + j < p.b_rows) out[colv + j] = acc[4 * k4 + j];
                }
              }
            }
          } else if (vec_ok) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              const long long colv = col0 + c + 8 * h + cpair;
#pragma unroll
              for (int r = 0; r < 2; ++r) {  // 16 rows per round
                if ((lane >> 4) == r) {
#pragma unroll
                  for (int k2 = 0; k2 < 4; ++k2)
                    *reinterpret_cast<double2*>(&stg[lane & 15][2 * k2]) =
                        make_double2(acc[8 * h + 2 * k2], acc[8 * h + 2 * k2 + 1]);
                }
                __syncwarp();
#pragma unroll
                for (int jj = 0; jj < 2; ++jj) {
                  const int j = 2 * r + jj;
                  const double2 v2 = *reinterpret_cast<const double2*>(&stg[(lane >> 2) + 8 * jj][cpair]);
                  if (srow[j] && colv + 1 < p.b_rows) *reinterpret_cast<double2*>(srow[j] + colv) = v2;
                  else if (srow[j] && colv < p.b_rows) srow[j][colv] = v2.x;
                }
                __syncwarp();
              }
            }
          } else {
#pragma unroll
            for (int j = 0; j < 16; ++j) {
              const long long col = col0 + c + j;
              if (row_ok && col < p.b_rows) out[col] = acc[j];
            }
          }
        }
        if (p.tp && !last) tmem_st_wait();
        tc_fence_before();
        if (CL == 4) {  // one arrival per warp on the leader's barrier
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster_relaxed(mapa_shared(smem_u32(&tmem_empty_bar), 0u));
        } else {
          mbar_arrive_relaxed(&tmem_empty_bar);
        }
      }
    }
    if (p.mode == kEpiX && row_ok) {
      const long long q = row / p.nao;
      const long long i = row - q * p.nao;
      atomicMax(&p.xmax[(long long)p.qgroup[q] * p.nao + i], hi_max);
    }
    }  // work loop
  }

  tc_fence_before();
  __syncthreads();
  if (CL != 1) cluster_sync_all();  // no CTA leaves while its peer may still write to it
  if (warp == 1) {
    tc_fence_after();
    if (CL == 4) tmem_dealloc_pair(tmem_base, 512);
    else tmem_dealloc(tmem_base, 512);
  }
}

// ---------------------------------------------------------------------------
// tcgen05.mma.kind::i8 issue-rate probe: operands resident in shared memory, no loads.
// MEASURED_PEAKS.json has no INT8 figure; this gives the roofline denominator.
// ---------------------------------------------------------------------------
static int g_peak_tiles = 1, g_peak_swz = 32;
void set_peak_tiles(int n) {
  g_peak_tiles = (n & 3) + 1;                                   // 1..4 distinct operand tiles
  g_peak_swz = ((n >> 2) & 3) == 1 ? 64 : ((n >> 2) & 3) == 2 ? 128 : 32;  // swizzle span of the tiles
}

__global__ void __launch_bounds__(128, 1) mma_peak_kernel(int n_mma, int iters, int ntiles, int swz) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t done_bar;
  __shared__ uint32_t tmem_slot;
  const int warp = threadIdx.x >> 5;
  // ntiles A tiles of 128 rows x 32 B (SW32, 4 KB each) and ntiles B tiles of 256 rows x 32 B,
  // zero-filled; ntiles > 1 walks different tiles so that no operand can be reused from the
  // previous MMA (shared-memory operand bandwidth shows).
  for (int i = threadIdx.x; i < ntiles * (128 + 256) * swz / 4; i += blockDim.x) ((uint32_t*)smem)[i] = 0;
  if (threadIdx.x == 0) {
    mbar_init(&done_bar, (n_mma >> 16) ? (n_mma >> 16) : 1);
    fence_barrier_init();
  }
  fence_proxy_async();
  if (warp == 0) tmem_alloc(&tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_slot;
  // n_mma = N | (number of issuing warps << 16) (0 = one).  Issuer w accumulates into its own two
  // TMEM slots; all issuers commit to done_bar.
  const int nissue = (n_mma >> 16) ? (n_mma >> 16) : 1;
  n_mma &= 0xFFFF;
  if (warp < nissue) {
    const uint32_t idesc = make_idesc_i8(128, n_mma);
    const uint64_t proto = make_smem_desc(0, swz);
    const uint32_t a_t16 = 128u * swz / 16u, b_t16 = 256u * swz / 16u, nk = swz / 32;
    const uint32_t hi = (uint32_t)(proto >> 32), lo0 = (uint32_t)proto;
    const uint32_t a16 = (smem_u32(smem) & 0x3FFFFu) >> 4, b16 = a16 + (uint32_t)ntiles * a_t16;
    const uint32_t slot = tmem_base + (uint32_t)(warp * (512 / nissue));
    const uint32_t half = (uint32_t)(256 / nissue);
    if (elect_one()) {
      int ta = 0, tb = 0;
      uint32_t kk2 = 0;
      for (int i = 0; i < iters; ++i) {
        const uint64_t adesc = ((uint64_t)hi << 32) | (lo0 | (a16 + (uint32_t)ta * a_t16 + kk2));
        const uint64_t bdesc = ((uint64_t)hi << 32) | (lo0 | (b16 + (uint32_t)tb * b_t16 + kk2));
        mma_i8_ss(slot + (uint32_t)(i & 1) * half, adesc, bdesc, idesc, i > 1);
        kk2 += 2u;  // K step inside the swizzle row, 16-byte units
        if (kk2 == 2u * nk) kk2 = 0;
        if (++ta == ntiles) { ta = 0; if (++tb == ntiles) tb = 0; }
      }
      mma_commit(&done_bar);
    }
    __syncwarp();
  }
  if (warp == 0) mbar_wait(&done_bar, 0);
  tc_fence_before();
  __syncthreads();
  if (warp == 0) {
    tc_fence_after();
    tmem_dealloc(tmem_base, 512);
  }
}

// The same probe on SM pairs: cta_group::2 MMAs of M = 256 (128 rows per CTA), N = n_mma with half
// of the B rows in each CTA's shared memory; the leader CTA issues and commits to both CTAs.
__global__ void __launch_bounds__(128, 1) mma_peak_pair_kernel(int n_mma, int iters, int ntiles, int swz) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t done_bar;
  __shared__ uint32_t tmem_slot;
  const int warp = threadIdx.x >> 5;
  const uint32_t crank = cluster_ctarank();
  for (int i = threadIdx.x; i < ntiles * (128 + 128) * swz / 4; i += blockDim.x) ((uint32_t*)smem)[i] = 0;
  if (threadIdx.x == 0) {
    mbar_init(&done_bar, 1);
    fence_barrier_init();
  }
  fence_proxy_async();
  if (warp == 0) tmem_alloc_pair(&tmem_slot, 512);
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = tmem_slot;
  if (warp == 0) {
    if (crank == 0) {
      const uint32_t idesc = make_idesc_i8(256, n_mma);
      const uint64_t proto = make_smem_desc(0, swz);
      const uint32_t a_t16 = 128u * swz / 16u, b_t16 = 128u * swz / 16u, nk = swz / 32;
      const uint32_t hi = (uint32_t)(proto >> 32), lo0 = (uint32_t)proto;
      const uint32_t a16 = (smem_u32(smem) & 0x3FFFFu) >> 4, b16 = a16 + (uint32_t)ntiles * a_t16;
      const uint32_t half = (uint32_t)(n_mma <= 256 ? 256 : 0);
      if (elect_one()) {
        int ta = 0, tb = 0;
        uint32_t kk2 = 0;
        for (int i = 0; i < iters; ++i) {
          const uint64_t adesc = ((uint64_t)hi << 32) | (lo0 | (a16 + (uint32_t)ta * a_t16 + kk2));
          const uint64_t bdesc = ((uint64_t)hi << 32) | (lo0 | (b16 + (uint32_t)tb * b_t16 + kk2));
          mma_i8_ss_pair(tmem_base + (uint32_t)(i & 1) * half, adesc, bdesc, idesc, i > 1);
          kk2 += 2u;
          if (kk2 == 2u * nk) kk2 = 0;
          if (++ta == ntiles) { ta = 0; if (++tb == ntiles) tb = 0; }
        }
        mma_commit_pair(&done_bar, (uint16_t)3);
      }
      __syncwarp();
    }
    mbar_wait(&done_bar, 0);
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == 0) {
    tc_fence_after();
    tmem_dealloc_pair(tmem_base, 512);
  }
}

static cudaError_t launch_pair_probe(int n_mma, int iters, int grid, int ntiles, int swz, int smem_bytes,
                                     cudaStream_t st) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(grid & ~1), 1, 1);
  cfg.blockDim = dim3(128, 1, 1);
  cfg.dynamicSmemBytes = (size_t)smem_bytes;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, mma_peak_pair_kernel, n_mma, iters, ntiles, swz);
}

cudaError_t launch_mma_peak(int n_mma, int iters, int grid, float* ms, cudaStream_t st) {
  if (n_mma & (1 << 24)) {  // bit 24: the cta_group::2 pair probe
    n_mma &= 0xFFFF;
    const int ntiles = g_peak_tiles, swz = g_peak_swz;
    const int smem_bytes = ntiles * 256 * swz + 2048;
    cudaError_t err = cudaFuncSetAttribute(mma_peak_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
    if (err != cudaSuccess) return err;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    err = launch_pair_probe(n_mma, 64, grid, ntiles, swz, smem_bytes, st);  // warm-up
    cudaEventRecord(e0, st);
    if (err == cudaSuccess) err = launch_pair_probe(n_mma, iters, grid, ntiles, swz, smem_bytes, st);
    cudaEventRecord(e1, st);
    count_launch(2);
    if (err == cudaSuccess) err = cudaEventSynchronize(e1);
    if (err == cudaSuccess) err = cudaEventElapsedTime(ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (err != cudaSuccess) return err;
    return cudaGetLastError();
  }
  const int ntiles = g_peak_tiles;
  const int swz = g_peak_swz;
  const int smem_bytes = ntiles * (128 + 256) * swz + 2048;
  cudaError_t err = cudaFuncSetAttribute(mma_peak_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
  if (err != cudaSuccess) return err;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  mma_peak_kernel<<<grid, 128, smem_bytes, st>>>(n_mma, 64, ntiles, swz);  // warm-up
  cudaEventRecord(e0, st);
  mma_peak_kernel<<<grid, 128, smem_bytes, st>>>(n_mma, iters, ntiles, swz);
  cudaEventRecord(e1, st);
  count_launch(2);
  err = cudaEventSynchronize(e1);
  if (err == cudaSuccess) err = cudaEventElapsedTime(ms, e0, e1);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (err != cudaSuccess) return err;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------
// host side: tensor maps and launch
// ---------------------------------------------------------------------------
// planes [plane][rows][pitch] int8 -> 3-D map (k, rows, plane), box (bk, box_rows, 1)
static bool make_plane_map(CUtensorMap* map, const int8_t* base, int64_t k, int64_t rows, int planes,
                           int64_t pitch, int64_t plane_stride, int bk, int box_rows) {
  const uint64_t dims[3] = {(uint64_t)k, (uint64_t)rows, (uint64_t)planes};
  const uint64_t strides[2] = {(uint64_t)pitch, (uint64_t)plane_stride};
  const uint32_t box[3] = {(uint32_t)bk, (uint32_t)box_rows, 1u};
  return encode_tensor_map(map, 0, 3, base, dims, strides, box, bk);
}

static uint32_t stage_stride_for(int s, int n_tile, int bk) {
  return (uint32_t)round_up((int64_t)s * (kTileM + n_tile) * bk, 1024);  // n_tile / 2 passed in pair mode
}

// Tensor maps of the GEMM operands, cached per context: a map depends only on the pointer, the shape
// and the box, and a build of a small problem spends more host time encoding its maps (four driver
// calls per GEMM launch) than launching the kernel.
struct TmapKey {
  const void* base;
  int64_t k, rows, pitch, plane_stride;
  int planes, bk, box_rows;
  bool operator==(const TmapKey& o) const {
    return base == o.base && k == o.k && rows == o.rows && pitch == o.pitch && plane_stride == o.plane_stride &&
           planes == o.planes && bk == o.bk && box_rows == o.box_rows;
  }
};
struct TmapCache {
  static constexpr int kSlots = 48;
  TmapKey keys[kSlots];
  CUtensorMap maps[kSlots];
  int used = 0, next = 0;
};
TmapCache* tmap_cache_create() { return new TmapCache(); }
void tmap_cache_destroy(TmapCache* c) { delete c; }

static bool cached_plane_map(TmapCache* cache, CUtensorMap* map, const int8_t* base, int64_t k, int64_t rows, int planes,
                             int64_t pitch, int64_t plane_stride, int bk, int box_rows) {
  if (!cache) return make_plane_map(map, base, k, rows, planes, pitch, plane_stride, bk, box_rows);
  const TmapKey key = {base, k, rows, pitch, plane_stride, planes, bk, box_rows};
  for (int i = 0; i < cache->used; ++i)
    if (cache->keys[i] == key) {
      *map = cache->maps[i];
      return true;
    }
  if (!make_plane_map(map, base, k, rows, planes, pitch, plane_stride, bk, box_rows)) return false;
  const int slot = cache->used < TmapCache::kSlots ? cache->used++ : (cache->next++ % TmapCache::kSlots);
  cache->keys[slot] = key;
  cache->maps[slot] = *map;
  return true;
}

cudaError_t launch_gemm_i8(const GemmProblem& g, const LaunchEnv& env, cudaStream_t st) {
  GemmKernelParams p;
  const int s = g.s;
  // debug knobs (include/df_emul.h, df_debug_set_gemm_flags)
  const int flags = env.flags;
  const int dbg_kernel = (flags & 3) | (((flags >> 23) & 1) << 2);  // bit 23: staged 16-byte epilogue accesses, no 256-bit ones
  const bool no_pair = (flags >> 20) & 1;                           // bit 20: no cta_group::2 pair tiles
  const bool no_tp = (flags >> 3) & 1;  // bit 3: multi-pass through global read-modify-write instead of TMEM
  const int fbk = (flags >> 8) & 0xFF;  // bits 8..15: force the K-block width (32, 64, 128; 0 = auto)
  const int force_bk = (fbk == 32 || fbk == 64 || fbk == 128) ? fbk : 0;
  // cta_group::2 pair: 256-row tiles on an SM pair, each CTA holds half of the B tile's N rows --
  // the MMA then reads 6 KB instead of 8 KB of shared memory per 128 x 128 x 32 step
  const bool pair = g.pair && g.n_tile % 16 == 0 && g.mode != kEpiInt32 && g.a_rows > kTileM &&
                    (!g.lower_only || g.n_tile == 128) && !no_pair;
  const int nb = pair ? g.n_tile / 2 : g.n_tile;  // B rows per CTA and stage
  int bk = g.bk;
  if (bk == 0) bk = force_bk;
  if (bk == 0) {
    // widest swizzle span that still gives two stages (measured: 128-byte K blocks with two stages
    // beat 64-byte blocks with four: full 128-byte lines per TMA row and half the barrier traffic)
    auto stages = [&](int cand) { return (kSmemLimit - 1024) / (int)stage_stride_for(s, nb, cand); };
    if (stages(128) >= 2) bk = 128;
    else if (stages(64) >= 2) bk = 64;
    else bk = 32;
  }
  // a forced K-block width that leaves no room for even one stage is narrowed
  while (bk > 32 && (kSmemLimit - 1024) / (int)stage_stride_for(s, nb, bk) < 1) bk /= 2;
  p.stage_stride = stage_stride_for(s, nb, bk);
  p.num_stages = (int)((kSmemLimit - 1024) / p.stage_stride);
  if (p.num_stages > kMaxStages) p.num_stages = kMaxStages;
  if (p.num_stages < 1) return cudaErrorInvalidValue;
  if (!cached_plane_map(env.tmaps, &p.mapA, g.A, g.k, g.a_rows, s, g.a_pitch, g.a_plane_stride, bk, kTileM) ||
      !cached_plane_map(env.tmaps, &p.mapB, g.B, g.k, g.b_rows, s, g.b_pitch, g.b_plane_stride, bk, g.n_tile))
    return cudaErrorInvalidValue;
  p.s = s;
  p.n_tile = g.n_tile;
  p.acc_stride = g.acc_stride > 0 ? g.acc_stride : (int)round_up(g.n_tile, 32);
  {
    const int W0 = 512 / p.acc_stride;  // accumulator slots in TMEM
    const bool one_chunk = g.zk != nullptr || g.k <= kflush_for(s);  // q-groups fit one chunk by construction
    p.tp = 0;
    p.weights_later = 0;
    if (s <= W0) {
      p.weights_per_pass = s;
      p.npass = 1;
    } else if (W0 >= 3 && one_chunk && g.mode != kEpiInt32 && !no_tp &&
               1 + (s - W0 + W0 - 3) / (W0 - 2) <= (s + W0 - 1) / W0) {
      // park the running sum in TMEM when that costs no extra pass over the contraction
      p.tp = 1;
      p.weights_per_pass = W0;
      p.weights_later = W0 - 2;
      p.npass = 1 + (s - W0 + p.weights_later - 1) / p.weights_later;
    } else {
      p.weights_per_pass = W0;
      p.npass = (s + W0 - 1) / W0;
    }
  }
  {
    const int npass = p.npass;
    const uint32_t a_plane = (uint32_t)kTileM * bk, b_plane = (uint32_t)nb * bk, b_off = (uint32_t)s * a_plane;
    int np = 0;
    for (int ps = 0; ps < npass; ++ps) {
      p.pass_start[ps] = np;
      int w_hi, w_lo, slot0 = 0;
      if (!p.tp || ps == 0) {
        w_hi = s + 1 - ps * p.weights_per_pass;
        w_lo = w_hi - p.weights_per_pass + 1;
      } else {
        w_hi = s + 1 - p.weights_per_pass - (ps - 1) * p.weights_later;
        w_lo = w_hi - p.weights_later + 1;
        slot0 = 2;
      }
      if (w_lo < 2) w_lo = 2;
      // round-robin over the weights of the pass, so that consecutive MMAs target different TMEM
      // accumulators (back-to-back MMAs into one accumulator wait on each other)
      int next_t[kMaxSlices + 2];
      for (int w = w_lo; w <= w_hi; ++w) next_t[w] = (w - s) > 1 ? (w - s) : 1;
      for (bool any = true; any;) {
        any = false;
        for (int w = w_hi; w >= w_lo; --w) {
          const int t_lo = (w - s) > 1 ? (w - s) : 1, t_hi = (w - 1) < s ? (w - 1) : s;
          const int t = next_t[w];
          if (t > t_hi) continue;
          any = true;
          next_t[w] = t + 1;
          const uint32_t ao = ((uint32_t)(t - 1) * a_plane) >> 4, bo = (b_off + (uint32_t)(w - t - 1) * b_plane) >> 4;
          p.pairs[np].x = ao;
          p.pairs[np].y = bo;
          p.pairs[np].z = (uint32_t)((slot0 + w_hi - w) * p.acc_stride);
          p.pairs[np].w = t > t_lo ? 1u : 0u;
          ++np;
        }
      }
    }
    p.pass_start[npass] = np;
  }
  p.tiles_m = (int)((g.a_rows + kTileM - 1) / kTileM);
  p.tiles_n = (int)((g.b_rows + g.n_tile - 1) / g.n_tile);
  p.group_m = 16;
  p.a_rows = g.a_rows;
  p.b_rows = g.b_rows;
  p.k = (int)g.k;
  // a z item (q-group of GEMM(6)) is one flush chunk by construction: its contraction holds at most
  // kflush(s) elements that are not zero padding (R5), whatever its padded extent
  p.kflush = g.zk ? (1 << 30) : kflush_for(s);
  p.zk = g.zk;
  p.eA = g.eA;
  p.eB = g.eB;
  p.ea_stride = g.ea_stride;
  p.eb_stride = g.eb_stride;
  p.lower_only = g.lower_only;
  p.mode = g.mode;
  p.C = g.C;
  p.ldc = g.ldc;
  p.c_stride = g.c_stride;
  p.nao = g.nao;
  p.x_cols = g.x_cols;
  p.ldx = g.ldx;
  p.qgroup = g.qgroup;
  p.xmax = g.xmax;
  p.kmask = g.mode == kEpiX ? g.kmask : nullptr;
  p.kmask_words = g.kmask_words;
  p.P = g.P;
  p.dbg_chunk = g.dbg_chunk;
  p.dbg_flags = dbg_kernel;

  p.pair = pair ? 1 : 0;
  const int tiles_m2 = (p.tiles_m + 1) / 2;  // 256-row tiles of the pair mode
  p.tiles_per_z = pair ? (g.lower_only ? tiles_m2 * (tiles_m2 + 1) : tiles_m2 * p.tiles_n)
                       : (g.lower_only ? p.tiles_m * (p.tiles_m + 1) / 2 : p.tiles_m * p.tiles_n);
  if (pair) {
    p.tiles_m = tiles_m2;  // decode_work rasterises pair rows; the kernel maps them back to 2 tm2 + rank
    if (!cached_plane_map(env.tmaps, &p.mapBh, g.B, g.k, g.b_rows, s, g.b_pitch, g.b_plane_stride, bk, g.n_tile / 2))
      return cudaErrorInvalidValue;
  }
  p.total_work = (long long)p.tiles_per_z * g.nz;
  int num_sms = env.num_sms;
  if (num_sms <= 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
  }
  const size_t smem = (size_t)p.num_stages * p.stage_stride + 1024;
  // cluster pair: the two N tiles of an M tile share the A operand through TMA multicast
  const int cl = pair ? 4
                 : (g.cluster_n == 2 && p.tiles_n == 2 && !g.lower_only && num_sms >= 2) ? 2 : 1;
  if (cl == 2) {
    p.group_m = 1;  // work items 2c, 2c+1 = (tm = c, tn = 0 / 1)
    if (!cached_plane_map(env.tmaps, &p.mapA2, g.A, g.k, g.a_rows, s, g.a_pitch, g.a_plane_stride, bk, 64)) return cudaErrorInvalidValue;
  }
  // persistent when tiles are short (the per-CTA set-up of ~4 us would show); long-K tiles are left
  // to the hardware scheduler, which balances them better than a static round-robin
  const long long k_item = g.zk ? g.k / (g.nz > 0 ? g.nz : 1) : g.k;
  const bool persistent = cl == 2 || k_item <= 8192;
  long long nblocks = cl == 4 ? 2 * p.total_work : p.total_work;  // pair mode: one work item per cluster
  if (persistent && nblocks > num_sms) nblocks = num_sms;
  if (cl != 1) nblocks = (nblocks + 1) / 2 * 2;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)nblocks, 1, 1);
  cfg.blockDim = dim3(kGemmThreads, 1, 1);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = cl == 1 ? 1 : 2;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  cudaError_t err;
#define DFE_LAUNCH(BKV, CLV)                                                                                    \
  err = cudaFuncSetAttribute(gemm_i8_kernel<BKV, CLV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
  if (err != cudaSuccess) return err;                                                                           \
  err = cudaLaunchKernelEx(&cfg, gemm_i8_kernel<BKV, CLV>, p);                                                  \
  if (err != cudaSuccess) return err;
  if (cl == 4) {
    if (bk == 128) { DFE_LAUNCH(128, 4) } else if (bk == 64) { DFE_LAUNCH(64, 4) } else { DFE_LAUNCH(32, 4) }
  } else if (cl == 2) {
    if (bk == 128) { DFE_LAUNCH(128, 2) } else if (bk == 64) { DFE_LAUNCH(64, 2) } else { DFE_LAUNCH(32, 2) }
  } else {
    if (bk == 128) { DFE_LAUNCH(128, 1) } else if (bk == 64) { DFE_LAUNCH(64, 1) } else { DFE_LAUNCH(32, 1) }
  }
#undef DFE_LAUNCH
  count_launch();
  return cudaGetLastError();
}

}  // namespace dfe
