// api.cu -- the C-ABI of libdfemul.so (include/df_emul.h): policy, workspace carving and the
// launch sequences of df_emul_gemm and df_jk_build.  Host logic only; every step of the path
// runs in the kernels of split.cu, gemm_i8.cu and jk.cu.  No cuBLAS, no CPU fallback.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <atomic>
#include <mutex>
#include <vector>

#include "../../include/df_emul.h"
#include "internal.h"

namespace dfe {

static std::atomic<long long> g_launches{0};
void count_launch(int n) { g_launches += n; }

}  // namespace dfe

// A context: one workspace, one device, its policy mode, debug knobs and tensor-map cache.  One
// context serves one stream at a time; two contexts (two workspaces) may run concurrently.  The entry
// points without a context argument use the process-wide default context (df_set_workspace).
struct df_context {
  void* ws = nullptr;
  int64_t ws_bytes = 0;
  int device = -1;  // the device the workspace was registered on
  int mode = DF_MODE_GUARDED;
  dfe::LaunchEnv env;
  // knobs decoded from env.flags (include/df_emul.h, df_debug_set_gemm_flags)
  bool g5_split_n() const { return !(env.flags & 4); }            // bit 2: GEMM(5) keeps one N tile
  bool g5_cluster() const { return !(env.flags & 64); }           // bit 6: N halves without the multicast pair
  bool wide_n() const { return !((env.flags >> 24) & 1); }        // bit 24: df_emul_gemm never takes wide tiles
  bool g5_pair_halves() const { return !((env.flags >> 22) & 1); }  // bit 22: N halves never on MMA pairs
  int jk_dbg() const { return (env.flags >> 4) & 3; }             // bits 4, 5: unpack kernel without stores / loads
  bool screening() const { return !((env.flags >> 25) & 1); }     // bit 25: no screening of zero K blocks
};

namespace dfe {

static df_context g_default;

// ---- optional per-kernel-class CUDA-event timing (df_profile_*; bench.py's roofline) ----
enum ProfClass { kPSplit = 0, kPPassA, kPJGemv, kPUnpack, kPGemm5, kPSplitX, kPGemm6, kPReduce, kPGemm, kPScreen, kPNum };
static const char* const kProfNames[kPNum] = {"split",   "jk_pass_a", "jk_j_gemv", "jk_unpack_split", "gemm5_i8",
                                              "jk_split_x", "gemm6_i8",  "jk_k_reduce", "emul_gemm_i8", "jk_screen_mask"};
struct ProfRec {
  int cls;
  cudaEvent_t e0, e1;
};
static std::atomic<bool> g_prof_on{false};
static std::mutex g_prof_mu;                // guards the two vectors: contexts may run on several host threads
static std::vector<ProfRec> g_prof_recs;    // records of the current profiling window
static std::vector<cudaEvent_t> g_prof_pool;  // recycled events
static cudaEvent_t prof_event() {
  cudaEvent_t e;
  std::lock_guard<std::mutex> lock(g_prof_mu);
  if (!g_prof_pool.empty()) {
    e = g_prof_pool.back();
    g_prof_pool.pop_back();
  } else {
    cudaEventCreate(&e);
  }
  return e;
}
struct ProfScope {
  cudaStream_t st;
  bool on;
  ProfRec r;
  ProfScope(int cls, cudaStream_t s) : st(s), on(g_prof_on) {
    if (on) {
      r.cls = cls;
      r.e0 = prof_event();
      r.e1 = prof_event();
      cudaEventRecord(r.e0, st);
    }
  }
  ~ProfScope() {
    if (on) {
      cudaEventRecord(r.e1, st);
      std::lock_guard<std::mutex> lock(g_prof_mu);
      g_prof_recs.push_back(r);
    }
  }
};

// The current device when it is of compute capability 10.x, else -1.
static int current_sm100_device(int* num_sms = nullptr) {
  int dev = 0, major = 0;
  if (cudaGetDevice(&dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
    cudaGetLastError();
    return -1;
  }
  if (major != 10) return -1;
  if (num_sms) cudaDeviceGetAttribute(num_sms, cudaDevAttrMultiProcessorCount, dev);
  return dev;
}

// DF_OK when the context has a workspace and the current device is the one it was registered on.
static int context_ready(const df_context& c) {
  const int dev = current_sm100_device();
  if (dev < 0) return DF_ERR_DEVICE;
  if (!c.ws) return DF_ERR_WORKSPACE;
  if (dev != c.device) return DF_ERR_DEVICE;
  return DF_OK;
}

static int context_set_workspace(df_context& c, void* ptr, int64_t bytes) {
  if (!ptr || bytes <= 0) {
    c.ws = nullptr;
    c.ws_bytes = 0;
    c.device = -1;
    return DF_OK;
  }
  if (((uintptr_t)ptr & 255) != 0) return DF_ERR_ALIGN;
  if (bytes < 256) return DF_ERR_WORKSPACE;
  int num_sms = 0;
  const int dev = current_sm100_device(&num_sms);
  if (dev < 0) return DF_ERR_DEVICE;
  if (cudaMemset(ptr, 0, 256) != cudaSuccess) return DF_ERR_CUDA;  // the status word
  c.ws = ptr;
  c.ws_bytes = bytes;
  c.device = dev;
  c.env.num_sms = num_sms;
  if (!c.env.tmaps) c.env.tmaps = tmap_cache_create();
  return DF_OK;
}

static int slices_for_tol(double tol, int mode) {
  if (!(tol > 0.0) || isnan(tol)) return DF_ERR_TOL;
  const double lg = log2(1.0 / tol);
  int s;
  if (mode == DF_MODE_NOMINAL) {
    // m_emu = ceil(log2(1/tol) - 0.05); s = ceil((m_emu + 1) / 8)   (Table 1)
    long long m_emu = (long long)ceil(lg - 0.05);
    if (m_emu < 0) m_emu = 0;
    s = (int)((m_emu + 1 + 7) / 8);
  } else {
    // one extra byte of margin (R7)
    s = (int)ceil((lg + 7.0) / 8.0);
  }
  if (s < 1) s = 1;
  if (s > kMaxSlices) s = kMaxSlices;
  return s;
}

// bump allocator over the registered workspace, 256-byte granularity
struct Carver {
  char* base;
  int64_t off = 0;
  explicit Carver(void* b) : base((char*)b) {}
  template <typename T>
  T* take(int64_t count) {
    T* p = (T*)(base ? base + off : nullptr);
    off += round_up(count * (int64_t)sizeof(T), 256);
    return p;
  }
};

static inline int pad16(int64_t n) { return (int)round_up(n, 16); }

// ---------------------------------------------------------------------------
// df_emul_gemm
// ---------------------------------------------------------------------------
struct GemmWs {
  int* status;
  int32_t *eA, *eB;
  uint32_t* cmax;
  int8_t *pa, *pb;
  int64_t pitch, bytes;
};

static GemmWs carve_gemm(void* base, int64_t m, int64_t n, int64_t k, int s) {
  Carver c(base);
  GemmWs w;
  w.status = c.take<int>(64);
  w.eA = c.take<int32_t>(m);
  w.eB = c.take<int32_t>(n);
  w.cmax = c.take<uint32_t>(n);
  w.pitch = plane_pitch(k);
  w.pa = c.take<int8_t>((int64_t)s * m * w.pitch);
  w.pb = c.take<int8_t>((int64_t)s * n * w.pitch);
  w.bytes = c.off;
  return w;
}

static int emul_gemm_impl(df_context& c, const double* A, const double* B, double* C, int64_t m, int64_t n,
                          int64_t k, int s, cudaStream_t st) {
  if (!A || !B || !C) return DF_ERR_NULL;
  // n: the column split puts 32-column blocks on grid.y (65535)
  if (m <= 0 || n <= 0 || k <= 0 || k > (1ll << 30) || m >= (1ll << 31) || n > 65535ll * 32) return DF_ERR_DIM;
  if (s < 1 || s > kMaxSlices) return DF_ERR_TOL;
  if (const int rc = context_ready(c)) return rc;
  GemmWs w = carve_gemm(c.ws, m, n, k, s);
  if (w.bytes > c.ws_bytes) return DF_ERR_WORKSPACE;

  {
    ProfScope ps(kPSplit, st);
    if (launch_split_rows(A, m, k, k, s, w.eA, w.pa, w.pitch, m * w.pitch, w.status, st, c.env.num_sms) != cudaSuccess)
      return DF_ERR_CUDA;
    if (launch_split_cols(B, k, n, s, w.cmax, w.eB, w.pb, w.pitch, n * w.pitch, w.status, st) != cudaSuccess)
      return DF_ERR_CUDA;
  }

  GemmProblem g = {};
  g.A = w.pa;
  g.B = w.pb;
  g.a_rows = m;
  g.b_rows = n;
  g.k = k;
  g.a_pitch = g.b_pitch = w.pitch;
  g.a_plane_stride = m * w.pitch;
  g.b_plane_stride = n * w.pitch;
  g.s = s;
  // 256-column tiles when all s accumulators still fit TMEM (s <= 2): one or three MMAs per K step
  // are fed by 2 s plane tiles, so the operand feed, not the tensor pipe, bounds s = 1, 2
  g.n_tile = n > 128 ? ((s <= 2 && n >= 256 && c.wide_n()) ? 256 : (s == 3 && n >= 160 && c.wide_n()) ? 160 : 128) : pad16(n);
  g.bk = 0;
  g.nz = 1;
  g.zk = nullptr;
  g.eA = w.eA;
  g.eB = w.eB;
  g.mode = kEpiC;
  g.pair = 1;
  g.C = C;
  g.ldc = n;
  {
    ProfScope ps(kPGemm, st);
    if (launch_gemm_i8(g, c.env, st) != cudaSuccess) return DF_ERR_CUDA;
  }
  return DF_OK;
}

// ---------------------------------------------------------------------------
// df_jk_build
// ---------------------------------------------------------------------------
struct JkWs {
  int* status;
  double *rho, *rho_part;
  uint32_t* emax5;
  uint32_t* tilemax;  // [32 x 32 tile pair][naux]: the tile maxima pass A leaves for the screening mask
  uint32_t* kmask;    // [256-row block of the super-block][mask words]: active K blocks of GEMM(5)
  double* Jp;
  double* jpart;  // [ceil(naux / 32)][npair] chunk partials of Eq. 4 (plain builds)
  uint32_t* cmaxC;
  int32_t* eC;
  int8_t* pc;
  int32_t* e5;
  int8_t* p5;
  double* X;
  int *qgroup, *qcol, *gcol;
  uint32_t* xmax;
  int32_t* e6;
  int8_t* p6;
  double* Kpart;
  int64_t pitchj, pitch6, bytes;
  int a_pad, ngmax;
  GroupGeom gg;
};

// Plan buffer (df_jk_plan_create): everything about B that does not change over an SCF.
//   [emax5: nao x naux u32][tilemax: tile pairs x naux u32][e5: (q, i) i32][planes: smax x (q, i) x pitch int8]
// The digit planes have the prefix property (R3): a build with s <= smax slices reads
// the first s planes.
struct PlanLayout {
  int64_t pitch, rows, emax_off, tilemax_off, e5_off, planes_off, plane_stride, bytes;
};
static PlanLayout plan_layout(int64_t nao, int64_t naux, int smax) {
  PlanLayout L;
  L.pitch = round_up(nao, 128);
  L.rows = naux * nao;
  L.emax_off = 0;
  L.tilemax_off = round_up(L.rows * 4, 256);
  L.e5_off = L.tilemax_off + round_up(jk_rho_part_rows((int)nao) * naux * 4, 256);
  L.planes_off = L.e5_off + round_up(L.rows * 4, 256);
  L.plane_stride = L.rows * L.pitch;
  L.bytes = L.planes_off + smax * L.plane_stride;
  return L;
}

// QS = q per super-block (a multiple of 512, or naux when naux < 512); planned: GEMM(5)'s left
// operand comes from a plan, no emax5 / e5 / planes5 in the workspace
static JkWs carve_jk(void* base, int64_t nao, int64_t naux, int64_t nocc, int s, int64_t QS, bool planned = false) {
  Carver c(base);
  JkWs w;
  w.gg = group_geom(s, (int)nocc);
  w.a_pad = w.gg.a_pad;
  w.ngmax = group_count(w.gg, (int)QS);
  // rows of whole 128-byte lines: the unpack pass writes full lines (1.2 % of a build at config 3)
  w.pitchj = round_up(nao, 128);
  // every q-group starts at a multiple of 32 columns: at most 16 zero columns after each group
  w.pitch6 = plane_pitch(QS * w.a_pad + 16 * (int64_t)w.ngmax);
  w.status = c.take<int>(64);
  w.rho = c.take<double>(naux);
  w.rho_part = c.take<double>(jk_rho_part_rows((int)nao) * naux);
  w.emax5 = planned ? nullptr : c.take<uint32_t>(nao * naux);
  w.tilemax = planned ? nullptr : c.take<uint32_t>(jk_rho_part_rows((int)nao) * naux);
  w.kmask = c.take<uint32_t>(((QS * nao + 255) / 256) * screen_mask_words(nao));
  w.Jp = c.take<double>(nao * (nao + 1) / 2);
  w.jpart = planned ? nullptr : c.take<double>(((naux + 31) / 32) * (nao * (nao + 1) / 2));
  w.cmaxC = c.take<uint32_t>(w.a_pad);
  w.eC = c.take<int32_t>(w.a_pad);
  w.pc = c.take<int8_t>((int64_t)s * w.a_pad * w.pitchj);
  w.e5 = planned ? nullptr : c.take<int32_t>(QS * nao);
  w.p5 = planned ? nullptr : c.take<int8_t>((int64_t)s * QS * nao * w.pitchj);
  w.X = c.take<double>(nao * QS * w.a_pad);
  w.qgroup = c.take<int>(QS);
  w.qcol = c.take<int>(QS);
  w.gcol = c.take<int>(w.ngmax + 1);
  w.xmax = c.take<uint32_t>((int64_t)w.ngmax * nao);
  w.e6 = c.take<int32_t>((int64_t)w.ngmax * nao);
  w.p6 = c.take<int8_t>((int64_t)s * nao * w.pitch6);
  w.Kpart = c.take<double>((int64_t)w.ngmax * nao * nao);
  w.bytes = c.off;
  return w;
}

// q-group tables of one super-block of nq consecutive q (R5, internal.h GroupGeom):
// qgroup[ql] = local group id, qcol[ql] = first planes6 column of q, gcol[g] = first column
// (= contraction offset of GEMM(6)) of group g, a multiple of 32; gcol[ng] = the end.
__global__ void jk_group_tables_kernel(int nq, GroupGeom gg, int ng, int* qgroup, int* qcol, int* gcol) {
  for (int ql = threadIdx.x; ql < nq; ql += blockDim.x) {
    const int g = (ql / kQBlock) * gg.gpb + (ql % kQBlock) / gg.QG;
    qgroup[ql] = g;
    qcol[ql] = group_col(gg, g, nq, ng) + (ql - group_q0(gg, g)) * gg.a_pad;
  }
  for (int g = threadIdx.x; g <= ng; g += blockDim.x) gcol[g] = group_col(gg, g, nq, ng);
}

// plan != nullptr (with its slice count smax): a planned build, GEMM(5) reads the plan's planes.
static int jk_impl(df_context& c, const double* Bp, int64_t nao, int64_t naux, const double* Cocc, int64_t nocc,
                   const double* D, int s, double* J, double* K, double* X_out, int32_t* e6_out, int* ngroups_out,
                   cudaStream_t st, const void* plan = nullptr, int smax = 0) {
  if (!Bp || !Cocc || !D || !J || !K) return DF_ERR_NULL;
  const bool planned = plan != nullptr;
  if (planned && (smax < 1 || smax > kMaxSlices || s > smax)) return DF_ERR_TOL;
  if (planned && ((uintptr_t)plan & 255) != 0) return DF_ERR_ALIGN;
  if (nao <= 0 || naux <= 0 || nocc <= 0 || nocc > 256 || nao > 11552 || naux > (1 << 20)) return DF_ERR_DIM;
  if (s < 1 || s > kMaxSlices) return DF_ERR_TOL;
  if (const int rc = context_ready(c)) return rc;
  // largest super-block (multiple of 512 q, capped so that GEMM(6)'s contraction offsets and the
  // row count of GEMM(5) stay in int32) that fits the workspace
  int64_t QS = 0;
  {
    const int64_t nblk = (naux + kQBlock - 1) / kQBlock;
    for (int64_t nb = nblk; nb >= 1; --nb) {
      const int64_t qs = (nb == nblk) ? naux : nb * kQBlock;
      if (qs * pad16(nocc) >= (1ll << 30) || qs * nao >= (1ll << 31) - 256) continue;
      if (carve_jk(nullptr, nao, naux, nocc, s, qs, planned).bytes <= c.ws_bytes) {
        QS = qs;
        break;
      }
    }
  }
  if (QS == 0) return DF_ERR_WORKSPACE;
  JkWs w = carve_jk(c.ws, nao, naux, nocc, s, QS, planned);
  const PlanLayout PL = plan_layout(nao, naux, planned ? smax : 1);
  const char* const plan_b = static_cast<const char*>(plan);
  const int64_t npair = nao * (nao + 1) / 2;

#define DFE_CK(x) \
  if ((x) != cudaSuccess) return DF_ERR_CUDA;

  // ---- J: rho (Eq. 3) fused with GEMM(5)'s row maxima, then J (Eq. 4) ----
  if (!planned) DFE_CK(cudaMemsetAsync(w.emax5, 0, sizeof(uint32_t) * nao * naux, st));
  {
    ProfScope ps(kPPassA, st);
    DFE_CK(launch_jk_pass_a(Bp, (int)nao, (int)naux, D, w.rho_part, w.rho, w.emax5,
                            c.screening() ? w.tilemax : nullptr, st));
  }
  if (planned) {
    ProfScope ps(kPJGemv, st);
    DFE_CK(launch_jk_j_gemv(Bp, npair, (int)naux, w.rho, w.Jp, st));
    DFE_CK(launch_jk_j_unpack(w.Jp, (int)nao, J, st));
  }  // a plain build sums Eq. 4 inside the unpack pass (chunk partials) and reduces them after it

  // ---- right operand of GEMM(5): C_occ columns -> K-major planes, a_pad rows (padding rows 0) ----
  DFE_CK(cudaMemsetAsync(w.eC, 0, sizeof(int32_t) * w.a_pad, st));
  DFE_CK(cudaMemsetAsync(w.pc, 0, (size_t)s * w.a_pad * w.pitchj, st));
  {
    ProfScope ps(kPSplit, st);
    DFE_CK(launch_split_cols(Cocc, nao, nocc, s, w.cmaxC, w.eC, w.pc, w.pitchj, (int64_t)w.a_pad * w.pitchj,
                             w.status, st));
  }

  int gtotal = 0;
  for (int64_t qs0 = 0; qs0 < naux; qs0 += QS) {
    const int64_t qs1 = qs0 + QS < naux ? qs0 + QS : naux;
    const int nq = (int)(qs1 - qs0);
    const int ng = group_count(w.gg, nq);
    // contraction extent of GEMM(6): the padded columns of all groups (every group boundary is a
    // multiple of 32, the K extent of one MMA: an MMA never straddles two groups)
    const int64_t ncol = group_col(w.gg, ng, nq, ng);
    const int64_t pitch6 = plane_pitch(ncol);
    if (ncol % 32 != 0 || pitch6 > w.pitch6) return DF_ERR_DIM;

    jk_group_tables_kernel<<<1, 256, 0, st>>>(nq, w.gg, ng, w.qgroup, w.qcol, w.gcol);
    count_launch();
    DFE_CK(cudaGetLastError());
    DFE_CK(cudaMemsetAsync(w.xmax, 0, sizeof(uint32_t) * ng * nao, st));

    // screening: the K blocks of GEMM(5)'s left operand that hold a
    // non-zero digit at s slices; the unpack pass writes and GEMM(5) reads only those
    // (a planned build always screens: its plan may hold planes for the active blocks only)
    const uint32_t* kmask = nullptr;
    if (planned || c.screening()) {
      const uint32_t* em = planned ? reinterpret_cast<const uint32_t*>(plan_b + PL.emax_off) : w.emax5;
      const uint32_t* tmx = planned ? reinterpret_cast<const uint32_t*>(plan_b + PL.tilemax_off) : w.tilemax;
      {
        ProfScope ps(kPScreen, st);
        DFE_CK(launch_jk_screen_mask(em, tmx, (int)nao, (int)naux, (int)qs0, nq, s, w.kmask,
                                     reinterpret_cast<unsigned long long*>(w.status + 8), st));
      }
      kmask = w.kmask;
    }

    // H2: unpack + split packed B -> planes5 rows (q, i), contraction j (a plan holds them already)
    if (!planned) {
      ProfScope ps(kPUnpack, st);
      DFE_CK(launch_jk_unpack_split(Bp, (int)nao, (int)naux, (int)qs0, (int)qs1, w.emax5, s, w.e5, w.p5,
                                    w.pitchj, (int64_t)nq * nao * w.pitchj, w.status, w.rho,
                                    w.jpart + (qs0 / 32) * npair, c.jk_dbg(), kmask, screen_mask_words(nao), st));
    }
    if (!planned && qs1 == naux) {
      ProfScope ps(kPJGemv, st);
      DFE_CK(launch_jk_j_reduce(w.jpart, (int)((naux + 31) / 32), npair, w.Jp, st));
      DFE_CK(launch_jk_j_unpack(w.Jp, (int)nao, J, st));
    }
    // GEMM(5): X[i][q][a] = sum_j B^q_ij C_ja   (Eq. 5 / Eq. 12)
    GemmProblem g5 = {};
    g5.A = planned ? reinterpret_cast<const int8_t*>(plan_b + PL.planes_off) + qs0 * nao * PL.pitch : w.p5;
    g5.B = w.pc;
    g5.a_rows = (int64_t)nq * nao;
    g5.b_rows = w.a_pad;
    g5.k = nao;
    g5.a_pitch = g5.b_pitch = w.pitchj;
    g5.a_plane_stride = planned ? PL.plane_stride : (int64_t)nq * nao * w.pitchj;
    g5.b_plane_stride = (int64_t)w.a_pad * w.pitchj;
    g5.s = s;
    // N tile: the whole a_pad when all s weight accumulators fit TMEM (s * a_pad <= 512 columns), else
    // two halves on a CTA pair that shares the A operand by multicast (measured at nocc = 150:
    // 12.6 / 15.9 / 20.5 ms at s = 4 / 5 / 6 against 13.8 / 19.8 / 26.8 ms for one 160-column tile
    // in two or more passes -- N = 160 MMAs are shared-memory-bandwidth bound)
    g5.n_tile = w.a_pad;
    {
      const int W0 = 512 / (int)round_up(w.a_pad, 32);
      if (s == W0 + 1 && W0 >= 3 && w.a_pad % 32 == 0 && c.g5_split_n()) {
        // one more weight than TMEM slots: the whole a_pad on cta_group::2 pairs, second pass (one
        // weight) with the running sum parked in TMEM -- 9.3-10.5 ms at nocc = 150, s = 4, against
        // 10.8-11.5 ms for two single-pass halves on MMA pairs (A streamed twice)
        g5.pair = 1;
      } else if ((int64_t)s * round_up(w.a_pad, 32) > 512 && w.a_pad % 32 == 0 && c.g5_split_n()) {
        g5.n_tile = w.a_pad / 2;
        // one pass per half (all s accumulators in TMEM): the halves run as 256-row tiles on MMA pairs
        // (an MMA costs at least ~50 cycles per 128 rows whatever N, and a pair instruction covers
        // 256) -- 13.6 / 17.6 ms against 14.6 / 21.9 ms at s = 5 / 6 for the multicast pair below;
        // with several passes (s >= 7 at nocc = 150) the two are equal
        if (c.g5_pair_halves() && (int64_t)s * g5.n_tile <= 512) g5.pair = 1;
      }
    }
    g5.acc_stride = (g5.n_tile % 32) ? g5.n_tile : 0;
    g5.x_cols = w.a_pad;
    g5.cluster_n = (c.g5_cluster() && g5.n_tile * 2 == w.a_pad && !g5.pair) ? 2 : 1;
    g5.nz = 1;
    g5.eA = planned ? reinterpret_cast<const int32_t*>(plan_b + PL.e5_off) + qs0 * nao : w.e5;
    g5.eB = w.eC;
    g5.mode = kEpiX;
    g5.C = w.X;
    g5.nao = (int)nao;
    g5.ldx = w.a_pad;
    g5.qgroup = w.qgroup;
    g5.xmax = w.xmax;
    g5.kmask = kmask;
    g5.kmask_words = screen_mask_words(nao);
      {
      ProfScope ps(kPGemm5, st);
      DFE_CK(launch_gemm_i8(g5, c.env, st));
    }
    if (X_out)
      DFE_CK(cudaMemcpyAsync(X_out + qs0 * nao * w.a_pad, w.X, sizeof(double) * nq * nao * w.a_pad,
                             cudaMemcpyDeviceToDevice, st));

    // X -> planes6 with one scale per (i, group)
    {
      ProfScope ps(kPSplitX, st);
      DFE_CK(launch_jk_split_x(w.X, (int)nao, nq, w.a_pad, s, ng, w.qgroup, w.qcol, w.gcol, w.xmax, w.e6, w.p6,
                               pitch6, (int64_t)nao * pitch6, w.status, st));
    }
    if (e6_out)
      DFE_CK(cudaMemcpyAsync(e6_out + (int64_t)gtotal * nao, w.e6, sizeof(int32_t) * ng * nao,
                             cudaMemcpyDeviceToDevice, st));

    // GEMM(6): K_g = X_g X_g^T per group (Eq. 6 / Eq. 13), lower block triangle only
    GemmProblem g6 = {};
    g6.A = w.p6;
    g6.B = w.p6;
    g6.a_rows = g6.b_rows = nao;
    g6.k = ncol;
    g6.a_pitch = g6.b_pitch = pitch6;
    g6.a_plane_stride = g6.b_plane_stride = (int64_t)nao * pitch6;
    g6.s = s;
    g6.n_tile = 128;
    g6.nz = ng;
    g6.zk = w.gcol;
    g6.eA = w.e6;
    g6.eB = w.e6;
    g6.ea_stride = g6.eb_stride = nao;
    g6.lower_only = 1;
    g6.pair = 1;
    g6.mode = kEpiC;
    g6.C = w.Kpart;
    g6.ldc = nao;
    g6.c_stride = nao * nao;
    {
      ProfScope ps(kPGemm6, st);
      DFE_CK(launch_gemm_i8(g6, c.env, st));
    }
    // H7: K += sum_g K_g in increasing-q order, mirrored to the upper triangle
    {
      ProfScope ps(kPReduce, st);
      DFE_CK(launch_jk_k_reduce(w.Kpart, ng, (int)nao, qs0 > 0 ? 1 : 0, K, st));
    }
    gtotal += ng;
  }
  if (ngroups_out) *ngroups_out = gtotal;
#undef DFE_CK
  return DF_OK;
}

// ---------------------------------------------------------------------------
// df_emul_gemm_static: df_emul_gemm for callers that have no device memory to give as a workspace
// ---------------------------------------------------------------------------
// Every other compute entry point carves its scratch (digit planes, scale indices, column maxima, status
// words) from a workspace the CALLER allocated.  Some callers cannot allocate: an SCF driver that handed
// all of HBM to B and its plan at start-up and has nothing left to give; a callback that runs while its
// stream is being captured, where cudaMalloc is not allowed; a host thread that shares the device with
// other contexts' builds, which a cudaMalloc would stall (it synchronises the whole device).  For them
// the scratch of this one entry point is the array below, part of the library's device image: every GPU
// that loads libdfemul holds these 64 MiB from the first use of the library until the process exits,
// whether or not df_emul_gemm_static is ever called.
constexpr int64_t kStaticScratchBytes = 64ll << 20;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

// In host code `g_static_scratch` is only a handle for the runtime's symbol calls, NOT a device address
// (a kernel handed it would fault, or quietly use host memory where the GPU can reach it); and the
// array has a different address on every device.  static_context() asks the runtime for the address
// with the target device current and keeps it, with the tensor-map cache and SM count of that device,
// in a context of its own.
constexpr int kMaxStaticDevices = 64;
static df_context g_static_ctx[kMaxStaticDevices];
static std::mutex g_static_mu;

// The context of the CURRENT device whose workspace is that device's copy of g_static_scratch.  Its
// first call on a device sets the context up: cudaGetSymbolAddress, a synchronous cudaMemset of the
// status words, a small host-side allocation (the tensor-map cache).  No device memory is allocated.
static int static_context(df_context** out) {
  const int dev = current_sm100_device();
  if (dev < 0 || dev >= kMaxStaticDevices) return DF_ERR_DEVICE;
  std::lock_guard<std::mutex> lock(g_static_mu);
  df_context& c = g_static_ctx[dev];
  if (!c.ws) {
    void* ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, g_static_scratch) != cudaSuccess || !ptr) {
      cudaGetLastError();
      return DF_ERR_CUDA;
    }
    if (const int rc = context_set_workspace(c, ptr, kStaticScratchBytes)) return rc;
  }
  *out = &c;
  return DF_OK;
}

}  // namespace dfe

// ===========================================================================
// extern "C" boundary
// ===========================================================================
using namespace dfe;

extern "C" {

int64_t df_emul_gemm_static_scratch_bytes(void) { return kStaticScratchBytes; }

int df_emul_gemm_static(const double* A, const double* B, double* C, int64_t m, int64_t n, int64_t k, double tol,
                        void* stream) {
  if (!A || !B || !C) return DF_ERR_NULL;
  if (m <= 0 || n <= 0 || k <= 0 || k > (1ll << 30) || m >= (1ll << 31) || n > 65535ll * 32) return DF_ERR_DIM;
  const int s = slices_for_tol(tol, g_default.mode);
  if (s < 0) return s;
  // the size check comes before any CUDA call: a problem that does not fit is refused, never truncated
  if (carve_gemm(nullptr, m, n, k, s).bytes > kStaticScratchBytes) return DF_ERR_TOO_LARGE;
  df_context* c = nullptr;
  if (const int rc = static_context(&c)) return rc;
  c->mode = g_default.mode;
  // Nothing in the array has to start at zero except what the launch sequence clears itself, in stream
  // order: the column maxima (cudaMemsetAsync inside launch_split_cols); planes, scale indices and the
  // padding bytes of every plane row are rewritten in full by the split kernels of this call.
  return emul_gemm_impl(*c, A, B, C, m, n, k, s, (cudaStream_t)stream);
}

int df_slices_for_tol(double tol, int mode) {
  if (mode != DF_MODE_NOMINAL && mode != DF_MODE_GUARDED) return DF_ERR_TOL;
  return slices_for_tol(tol, mode);
}

int df_num_int8_gemms(int s) { return (s < 1 || s > kMaxSlices) ? DF_ERR_TOL : s * (s + 1) / 2; }

int df_kflush(int s) { return (s < 1 || s > kMaxSlices) ? DF_ERR_TOL : kflush_for(s); }

int64_t df_plane_pitch(int64_t cols) { return cols <= 0 ? DF_ERR_DIM : plane_pitch(cols); }

int64_t df_emul_gemm_workspace_bytes(int64_t m, int64_t n, int64_t k, int s) {
  if (m <= 0 || n <= 0 || k <= 0) return DF_ERR_DIM;
  if (s < 1 || s > kMaxSlices) return DF_ERR_TOL;
  return carve_gemm(nullptr, m, n, k, s).bytes;
}

int64_t df_jk_workspace_bytes(int64_t nao, int64_t naux, int64_t nocc, int s) {
  if (nao <= 0 || naux <= 0 || nocc <= 0 || nocc > 256) return DF_ERR_DIM;
  if (s < 1 || s > kMaxSlices) return DF_ERR_TOL;
  const int64_t qs = naux < kQBlock ? naux : kQBlock;
  return carve_jk(nullptr, nao, naux, nocc, s, qs).bytes;
}

int64_t df_jk_workspace_bytes_blocks(int64_t nao, int64_t naux, int64_t nocc, int s, int64_t nblocks) {
  if (nao <= 0 || naux <= 0 || nocc <= 0 || nocc > 256 || nblocks < 1) return DF_ERR_DIM;
  if (s < 1 || s > kMaxSlices) return DF_ERR_TOL;
  int64_t qs = nblocks * kQBlock;
  if (qs > naux) qs = naux;
  return carve_jk(nullptr, nao, naux, nocc, s, qs).bytes;
}

int64_t df_jk_planned_workspace_bytes(int64_t nao, int64_t naux, int64_t nocc, int s, int64_t nblocks) {
  if (nao <= 0 || naux <= 0 || nocc <= 0 || nocc > 256 || nblocks < 1) return DF_ERR_DIM;
  if (s < 1 || s > kMaxSlices) return DF_ERR_TOL;
  int64_t qs = nblocks * kQBlock;
  if (qs > naux) qs = naux;
  return carve_jk(nullptr, nao, naux, nocc, s, qs, true).bytes;
}

int64_t df_jk_plan_bytes(int64_t nao, int64_t naux, int smax) {
  if (nao <= 0 || naux <= 0 || nao > 11552 || naux > (1 << 20)) return DF_ERR_DIM;
  if (smax < 1 || smax > kMaxSlices) return DF_ERR_TOL;
  return plan_layout(nao, naux, smax).bytes;
}

// ---- contexts -------------------------------------------------------------------------------

int df_context_create(void* workspace, int64_t bytes, df_context** ctx) {
  if (!ctx || !workspace) return DF_ERR_NULL;
  df_context* c = new df_context();
  const int rc = context_set_workspace(*c, workspace, bytes);
  if (rc != DF_OK) {
    delete c;
    return rc;
  }
  *ctx = c;
  return DF_OK;
}

int df_context_destroy(df_context* ctx) {
  if (!ctx) return DF_ERR_NULL;
  if (ctx == &g_default) return DF_ERR_NULL;
  tmap_cache_destroy(ctx->env.tmaps);
  delete ctx;
  return DF_OK;
}

int df_context_set_policy_mode(df_context* ctx, int mode) {
  if (!ctx) return DF_ERR_NULL;
  if (mode != DF_MODE_NOMINAL && mode != DF_MODE_GUARDED) return DF_ERR_TOL;
  ctx->mode = mode;
  return DF_OK;
}

int df_context_set_debug_flags(df_context* ctx, int flags) {
  if (!ctx) return DF_ERR_NULL;
  ctx->env.flags = flags;
  return DF_OK;
}

int df_context_emul_gemm(df_context* ctx, const double* A, const double* B, double* C, int64_t m, int64_t n,
                         int64_t k, double tol, void* stream) {
  if (!ctx) return DF_ERR_NULL;
  const int s = slices_for_tol(tol, ctx->mode);
  if (s < 0) return s;
  return emul_gemm_impl(*ctx, A, B, C, m, n, k, s, (cudaStream_t)stream);
}

int df_context_emul_gemm_slices(df_context* ctx, const double* A, const double* B, double* C, int64_t m, int64_t n,
                                int64_t k, int s, void* stream) {
  if (!ctx) return DF_ERR_NULL;
  return emul_gemm_impl(*ctx, A, B, C, m, n, k, s, (cudaStream_t)stream);
}

int df_context_jk_build(df_context* ctx, const double* B_packed, int64_t nao, int64_t naux, const double* C_occ,
                        int64_t nocc, const double* D, double tol, double* J, double* K, void* stream) {
  if (!ctx) return DF_ERR_NULL;
  const int s = slices_for_tol(tol, ctx->mode);
  if (s < 0) return s;
  return jk_impl(*ctx, B_packed, nao, naux, C_occ, nocc, D, s, J, K, nullptr, nullptr, nullptr, (cudaStream_t)stream);
}

int df_context_jk_build_slices(df_context* ctx, const double* B_packed, int64_t nao, int64_t naux,
                               const double* C_occ, int64_t nocc, const double* D, int s, double* J, double* K,
                               void* stream) {
  if (!ctx) return DF_ERR_NULL;
  return jk_impl(*ctx, B_packed, nao, naux, C_occ, nocc, D, s, J, K, nullptr, nullptr, nullptr, (cudaStream_t)stream);
}

int df_context_jk_plan_create(df_context* ctx, const double* B_packed, int64_t nao, int64_t naux, int smax,
                              void* plan, int64_t plan_bytes, void* stream) {
  if (!ctx || !B_packed || !plan) return DF_ERR_NULL;
  if (nao <= 0 || naux <= 0 || nao > 11552 || naux > (1 << 20)) return DF_ERR_DIM;
  if (smax < 1 || smax > kMaxSlices) return DF_ERR_TOL;
  if (((uintptr_t)plan & 255) != 0) return DF_ERR_ALIGN;
  if (const int rc = context_ready(*ctx)) return rc;  // the workspace holds the status word
  const PlanLayout L = plan_layout(nao, naux, smax);
  if (plan_bytes < L.bytes) return DF_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  char* pb = static_cast<char*>(plan);
  uint32_t* emax = reinterpret_cast<uint32_t*>(pb + L.emax_off);
  uint32_t* tilemax = reinterpret_cast<uint32_t*>(pb + L.tilemax_off);
  if (cudaMemsetAsync(emax, 0, sizeof(uint32_t) * L.rows, st) != cudaSuccess) return DF_ERR_CUDA;
  {
    ProfScope ps(kPPassA, st);
    if (launch_jk_pass_a(B_packed, (int)nao, (int)naux, nullptr, nullptr, nullptr, emax, tilemax, st) != cudaSuccess)
      return DF_ERR_CUDA;
  }
  // the planes are written for the K blocks that are active at smax slices: every build with s <= smax
  // reads a subset of them (its threshold 2^(e - 8 s - 1) is the larger one).  The mask of all q needs
  // ceil(naux nao / 256) words per 32 K blocks of workspace behind the status words; without that room
  // (or with screening off) every block is written.
  const uint32_t* kmask = nullptr;
  {
    const int words = screen_mask_words(nao);
    const int64_t need = 256 + round_up(((naux * nao + 255) / 256) * words * 4, 256);
    if (ctx->screening() && ctx->ws_bytes >= need) {
      uint32_t* km = reinterpret_cast<uint32_t*>(static_cast<char*>(ctx->ws) + 256);
      if (launch_jk_screen_mask(emax, tilemax, (int)nao, (int)naux, 0, (int)naux, smax, km,
                                reinterpret_cast<unsigned long long*>(static_cast<int*>(ctx->ws) + 8), st) != cudaSuccess)
        return DF_ERR_CUDA;
      kmask = km;
    }
  }
  {
    ProfScope ps(kPUnpack, st);
    if (launch_jk_unpack_split(B_packed, (int)nao, (int)naux, 0, (int)naux, emax, smax,
                               reinterpret_cast<int32_t*>(pb + L.e5_off),
                               reinterpret_cast<int8_t*>(pb + L.planes_off), L.pitch, L.plane_stride,
                               (int*)ctx->ws, nullptr, nullptr, ctx->jk_dbg(), kmask, screen_mask_words(nao), st) !=
        cudaSuccess)
      return DF_ERR_CUDA;
  }
  return DF_OK;
}

int df_context_jk_build_planned(df_context* ctx, const void* plan, int smax, const double* B_packed, int64_t nao,
                                int64_t naux, const double* C_occ, int64_t nocc, const double* D, double tol,
                                double* J, double* K, void* stream) {
  if (!ctx || !plan) return DF_ERR_NULL;
  const int s = slices_for_tol(tol, ctx->mode);
  if (s < 0) return s;
  return jk_impl(*ctx, B_packed, nao, naux, C_occ, nocc, D, s, J, K, nullptr, nullptr, nullptr,
                 (cudaStream_t)stream, plan, smax);
}

int df_context_jk_build_planned_slices(df_context* ctx, const void* plan, int smax, const double* B_packed,
                                       int64_t nao, int64_t naux, const double* C_occ, int64_t nocc,
                                       const double* D, int s, double* J, double* K, void* stream) {
  if (!ctx || !plan) return DF_ERR_NULL;
  return jk_impl(*ctx, B_packed, nao, naux, C_occ, nocc, D, s, J, K, nullptr, nullptr, nullptr,
                 (cudaStream_t)stream, plan, smax);
}

int df_context_last_status(df_context* ctx, void* stream, int* status) {
  if (!ctx || !status) return DF_ERR_NULL;
  if (!ctx->ws) return DF_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  if (cudaMemcpyAsync(status, ctx->ws, sizeof(int), cudaMemcpyDeviceToHost, st) != cudaSuccess) return DF_ERR_CUDA;
  if (cudaMemsetAsync(ctx->ws, 0, sizeof(int), st) != cudaSuccess) return DF_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return DF_ERR_CUDA;
  return DF_OK;
}

int df_context_screen_stats(df_context* ctx, void* stream, int64_t* active, int64_t* total) {
  if (!ctx || !active || !total) return DF_ERR_NULL;
  if (!ctx->ws) return DF_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  unsigned long long v[2] = {0ull, 0ull};
  char* src = static_cast<char*>(ctx->ws) + 32;
  if (cudaMemcpyAsync(v, src, sizeof(v), cudaMemcpyDeviceToHost, st) != cudaSuccess) return DF_ERR_CUDA;
  if (cudaMemsetAsync(src, 0, sizeof(v), st) != cudaSuccess) return DF_ERR_CUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess) return DF_ERR_CUDA;
  *active = (int64_t)v[0];
  *total = (int64_t)v[1];
  return DF_OK;
}

// ---- the same calls on the process-wide default context ------------------------------------

int df_set_policy_mode(int mode) { return df_context_set_policy_mode(&g_default, mode); }

int df_set_workspace(void* ptr, int64_t bytes) { return context_set_workspace(g_default, ptr, bytes); }

int df_emul_gemm(const double* A, const double* B, double* C, int64_t m, int64_t n, int64_t k, double tol,
                 void* stream) {
  return df_context_emul_gemm(&g_default, A, B, C, m, n, k, tol, stream);
}

int df_emul_gemm_slices(const double* A, const double* B, double* C, int64_t m, int64_t n, int64_t k, int s,
                        void* stream) {
  return df_context_emul_gemm_slices(&g_default, A, B, C, m, n, k, s, stream);
}

int df_jk_build(const double* B_packed, int64_t nao, int64_t naux, const double* C_occ, int64_t nocc,
                const double* D, double tol, double* J, double* K, void* stream) {
  return df_context_jk_build(&g_default, B_packed, nao, naux, C_occ, nocc, D, tol, J, K, stream);
}

int df_jk_build_slices(const double* B_packed, int64_t nao, int64_t naux, const double* C_occ, int64_t nocc,
                       const double* D, int s, double* J, double* K, void* stream) {
  return df_context_jk_build_slices(&g_default, B_packed, nao, naux, C_occ, nocc, D, s, J, K, stream);
}

int df_jk_plan_create(const double* B_packed, int64_t nao, int64_t naux, int smax, void* plan, int64_t plan_bytes,
                      void* stream) {
  return df_context_jk_plan_create(&g_default, B_packed, nao, naux, smax, plan, plan_bytes, stream);
}

int df_jk_build_planned(const void* plan, int smax, const double* B_packed, int64_t nao, int64_t naux,
                        const double* C_occ, int64_t nocc, const double* D, double tol, double* J, double* K,
                        void* stream) {
  return df_context_jk_build_planned(&g_default, plan, smax, B_packed, nao, naux, C_occ, nocc, D, tol, J, K, stream);
}

int df_jk_build_planned_slices(const void* plan, int smax, const double* B_packed, int64_t nao, int64_t naux,
                               const double* C_occ, int64_t nocc, const double* D, int s, double* J, double* K,
                               void* stream) {
  return df_context_jk_build_planned_slices(&g_default, plan, smax, B_packed, nao, naux, C_occ, nocc, D, s, J, K,
                                            stream);
}

int df_last_status(void* stream, int* status) { return df_context_last_status(&g_default, stream, status); }

int df_screen_stats(void* stream, int64_t* active, int64_t* total) {
  return df_context_screen_stats(&g_default, stream, active, total);
}

// ---- debug exports (default context) --------------------------------------------------------

int df_debug_jk_build(const double* B_packed, int64_t nao, int64_t naux, const double* C_occ, int64_t nocc,
                      const double* D, int s, double* J, double* K, double* X_out, int32_t* e6_out,
                      int* ngroups_out, void* stream) {
  return jk_impl(g_default, B_packed, nao, naux, C_occ, nocc, D, s, J, K, X_out, e6_out, ngroups_out,
                 (cudaStream_t)stream);
}

int df_debug_split_rows(const double* X, int64_t rows, int64_t cols, int s, int32_t* e, int8_t* planes,
                        void* stream) {
  if (!X || !e || !planes) return DF_ERR_NULL;
  if (rows <= 0 || cols <= 0 || rows >= (1ll << 31)) return DF_ERR_DIM;
  if (s < 1 || s > kMaxSlices) return DF_ERR_TOL;
  if (const int rc = context_ready(g_default)) return rc;
  const int64_t pitch = plane_pitch(cols);
  if (launch_split_rows(X, rows, cols, cols, s, e, planes, pitch, rows * pitch, (int*)g_default.ws,
                        (cudaStream_t)stream, g_default.env.num_sms) != cudaSuccess)
    return DF_ERR_CUDA;
  return DF_OK;
}

int df_debug_split_cols(const double* X, int64_t k, int64_t n, int s, int32_t* e, int8_t* planes, void* stream) {
  if (!X || !e || !planes) return DF_ERR_NULL;
  if (k <= 0 || n <= 0 || k > (1ll << 30) || n > 65535ll * 32) return DF_ERR_DIM;
  if (s < 1 || s > kMaxSlices) return DF_ERR_TOL;
  if (const int rc = context_ready(g_default)) return rc;
  if (g_default.ws_bytes < 256 + round_up(4 * n, 256)) return DF_ERR_WORKSPACE;
  const int64_t pitch = plane_pitch(k);
  uint32_t* cmax = (uint32_t*)((char*)g_default.ws + 256);
  if (launch_split_cols(X, k, n, s, cmax, e, planes, pitch, n * pitch, (int*)g_default.ws, (cudaStream_t)stream) !=
      cudaSuccess)
    return DF_ERR_CUDA;
  return DF_OK;
}

int df_debug_weight_sums(const int8_t* DA, const int8_t* DB, int64_t m, int64_t n, int64_t k, int s, int chunk,
                         int bk, int32_t* P, void* stream) {
  if (!DA || !DB || !P) return DF_ERR_NULL;
  if (m <= 0 || n <= 0 || k <= 0 || k > (1ll << 30)) return DF_ERR_DIM;
  if (s < 1 || s > kMaxSlices) return DF_ERR_TOL;
  if (bk != 0 && bk != 32 && bk != 64 && bk != 128) return DF_ERR_DIM;
  if (chunk < 0 || (int64_t)chunk * kflush_for(s) >= k) return DF_ERR_DIM;
  if (current_sm100_device() < 0) return DF_ERR_DEVICE;
  const int64_t pitch = plane_pitch(k);
  GemmProblem g = {};
  g.A = DA;
  g.B = DB;
  g.a_rows = m;
  g.b_rows = n;
  g.k = k;
  g.a_pitch = g.b_pitch = pitch;
  g.a_plane_stride = m * pitch;
  g.b_plane_stride = n * pitch;
  g.s = s;
  g.n_tile = n > 128 ? 128 : pad16(n);
  g.bk = bk;
  g.nz = 1;
  g.mode = kEpiInt32;
  g.P = P;
  g.dbg_chunk = chunk;
  LaunchEnv env;  // no cache, the SM count of the current device
  env.flags = g_default.env.flags;
  if (launch_gemm_i8(g, env, (cudaStream_t)stream) != cudaSuccess) return DF_ERR_CUDA;
  return DF_OK;
}

int df_debug_set_gemm_flags(int flags) {
  g_default.env.flags = flags;
  set_peak_tiles((flags >> 16) & 15);  // bits 16-19: MMA probe operand tiles / swizzle
  return DF_OK;
}

int64_t df_launch_count(void) { return (int64_t)g_launches.load(); }

int df_profile_enable(int on) {
  g_prof_on = on != 0;
  return DF_OK;
}

int df_profile_num_classes(void) { return kPNum; }

const char* df_profile_class_name(int cls) { return (cls < 0 || cls >= kPNum) ? "" : kProfNames[cls]; }

int df_profile_read(float* ms_by_class, int* count_by_class) {
  if (!ms_by_class || !count_by_class) return DF_ERR_NULL;
  for (int i = 0; i < kPNum; ++i) {
    ms_by_class[i] = 0.f;
    count_by_class[i] = 0;
  }
  int rc = DF_OK;
  std::lock_guard<std::mutex> lock(g_prof_mu);
  for (ProfRec& r : g_prof_recs) {
    float ms = 0.f;
    if (cudaEventSynchronize(r.e1) != cudaSuccess || cudaEventElapsedTime(&ms, r.e0, r.e1) != cudaSuccess)
      rc = DF_ERR_CUDA;
    ms_by_class[r.cls] += ms;
    count_by_class[r.cls] += 1;
    g_prof_pool.push_back(r.e0);
    g_prof_pool.push_back(r.e1);
  }
  g_prof_recs.clear();
  return rc;
}

int df_debug_mma_peak(int n_mma, int iters, int grid, float* ms, void* stream) {
  if (!ms) return DF_ERR_NULL;
  // N | issuing warps << 16 (0 = one) | pair probe << 24 (cta_group::2, M = 256, one issuer)
  const int n = n_mma & 0xFFFF, nissue = (n_mma >> 16) & 0xFF, pairp = (n_mma >> 24) & 1;
  if (n < 16 || n > 256 || (n % 16) != 0 || iters < 2 || grid < 1) return DF_ERR_DIM;
  if (nissue < 0 || nissue > 4 || 2 * (nissue ? nissue : 1) * n > 512) return DF_ERR_DIM;
  if (pairp && (nissue != 0 || grid < 2 || (n % 32) != 0)) return DF_ERR_DIM;
  if (current_sm100_device() < 0) return DF_ERR_DEVICE;
  if (launch_mma_peak(n_mma, iters, grid, ms, (cudaStream_t)stream) != cudaSuccess) return DF_ERR_CUDA;
  return DF_OK;
}

}  // extern "C"
