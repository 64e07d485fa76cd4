// msas_api.cu — the C ABI of libmsas (include/msas.h): plan construction, argument validation and kernel launches.
// Every step of the pass runs in the CUDA kernels of this directory; there is no CPU path.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/msas.h"
#include "k_score_simple.cuh"
#include "k_score_tc.cuh"
#include "k_entropy.cuh"
#include "k_segment.cuh"
#include "k_heads.cuh"
#include "k_compress.cuh"

using namespace msas;

static thread_local int g_last_cuda = 0;
#define CK(x)                                             \
  do {                                                    \
    cudaError_t e_ = (x);                                 \
    if (e_ != cudaSuccess) { g_last_cuda = (int)e_; (void)cudaGetLastError(); return MAS_ERR_CUDA; } \
  } while (0)

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Layout {
  size_t segs, tiles, req, tc_sched, tc_sched_x, tc_sched_u, tc_sched_xu, tc_segrank, tc_segrank_u, frames, tables_end;   // uploaded tables (contiguous from 0)
  size_t qinv, s, gamma, rel, mas, mask, segout, nkept, keptoff, counter, tc_xflag, tc_xchg, heads_part, gridw, heads_cq, merge_part, merge_cnt, total;
};

struct mas_plan {
  int32_t n_segs = 0, n_requests = 0, d = 0, dtype = 0;
  int64_t N = 0, nQ = 0, kept_cap = 0;
  int32_t n_tiles = 0;
  int32_t max_L = 0;
  int64_t n_frames = 0;       // sum of T over the segments
  int32_t max_patches = 0;    // largest P
  bool tc_inline_qnorm = true; // query norms in the score kernel's prologue (cooperative launch) vs a launch of their own
  int32_t seg_cluster = 1;    // CTAs per segment in the segment kernel (from the longest segment)
  int32_t seg_threads = 1024; // threads per CTA of the segment kernel
  DevParams prm{};
  Layout lay{};
  char* ws = nullptr;
  void* pinned = nullptr;
  size_t pinned_bytes = 0;
  int sm_count = 148;
  TcSchedule tc{};            // tcgen05 fast-path schedule (tc.enabled == false -> generic kernels)
  TcSchedule tcu{}, tcxu{};   // tc / tcx without K-split (no CTA waits for another one): used once a cooperative launch was refused
  TcSchedule tcx{};           // the schedule of the calls that append 64 B rows (mas_forward_lsh / mas_forward_heads; needs every L <= 64)
  mutable TcMapCache tc_maps; // tensor maps of the last few (X, Q, R) pointer sets (a plan is used by one host thread at a time)
  mutable bool tc_coop_ok = true;   // false once a cooperative launch was refused on this device: query norms get a launch of their own
  mutable std::vector<cudaEvent_t> prof_ev;   // profiling ring: 4 events per slot
  mutable int64_t prof_calls = 0;
  int32_t prof_slots = 0;
  template <class T> T* at(size_t off) const { return reinterpret_cast<T*>(ws + off); }
};

// ------------------------------------------------------------------------------------------------ host helpers
extern "C" int mas_version(void) { return MAS_VERSION; }
extern "C" int mas_last_cuda_error(void) { return g_last_cuda; }
extern "C" const char* mas_status_string(int st) {
  switch (st) {
    case MAS_OK: return "ok";
    case MAS_ERR_INVALID_ARG: return "invalid argument";
    case MAS_ERR_UNSUPPORTED: return "unsupported shape, dtype or alignment";
    case MAS_ERR_WORKSPACE: return "workspace too small";
    case MAS_ERR_CUDA: return "CUDA error (see mas_last_cuda_error)";
    default: return "unknown status";
  }
}
extern "C" void mas_params_default(mas_params* p) {
  if (!p) return;
  p->lambda_spatial = 0.6f; p->lambda_temp = 0.4f; p->tau_s = 0.3f; p->kappa = 10.0f;
  p->spatial_gain = 1.0f; p->spatial_bias = 0.0f; p->rel_gain = 1.0f; p->rel_bias = 0.0f;
  p->cut = 0.5f; p->select_mode = MAS_SELECT_TOPK;
}
extern "C" int32_t mas_keep_count(int64_t n, double ratio) {
  if (n <= 0) return 0;
  int64_t k = (int64_t)std::ceil(ratio * (double)n - 1e-9);
  if (k < 1) k = 1;
  if (k > n) k = n;
  return (int32_t)k;
}

// ------------------------------------------------------------------------------------------------ validation + layout
// Rows per tile of the generic (one CTA per tile) score kernels: 128, halved while the batch would not give every SM
// of a B200 about two tiles (a single 576-token image becomes 36 tiles of 16 rows instead of 5 of 128).
static int generic_tile_rows(int64_t n_total) {
  int rows = kTileRows;
  while (rows > 16 && n_total / rows < 296) rows >>= 1;
  return rows;
}

static int validate(const mas_segment* segs, int32_t n_segs, const int64_t* q_off, int32_t n_req, int32_t d, int32_t dtype,
                    const mas_params* prm, int64_t* N_out, int64_t* nQ_out, int32_t* n_tiles_out, int32_t* maxL_out) {
  if (!segs || !q_off || n_segs <= 0 || n_req <= 0) return MAS_ERR_INVALID_ARG;
  if (dtype != MAS_F32 && dtype != MAS_BF16) return MAS_ERR_INVALID_ARG;
  if (d < 8 || d > 65536) return MAS_ERR_UNSUPPORTED;
  if (dtype == MAS_BF16 ? (d % 8 != 0) : (d % 4 != 0)) return MAS_ERR_UNSUPPORTED;
  if (q_off[0] != 0) return MAS_ERR_INVALID_ARG;
  int32_t maxL = 0;
  for (int32_t r = 0; r < n_req; ++r) {
    const int64_t L = q_off[r + 1] - q_off[r];
    if (L < 0) return MAS_ERR_INVALID_ARG;
    if (L < 1 || L > MAS_MAX_QUERY_TOKENS) return MAS_ERR_UNSUPPORTED;
    if (L > maxL) maxL = (int32_t)L;
  }
  if (q_off[n_req] > (int64_t)0x7fffffff) return MAS_ERR_UNSUPPORTED;
  int64_t row = 0, tiles = 0;
  int32_t prev_req = -1;
  for (int32_t k = 0; k < n_segs; ++k) {
    const mas_segment& s = segs[k];
    if (s.n_frames < 1 || s.n_patches < 1) return MAS_ERR_INVALID_ARG;
    if (s.request < 0 || s.request >= n_req || s.request < prev_req) return MAS_ERR_INVALID_ARG;
    if (s.row0 != row) return MAS_ERR_INVALID_ARG;
    const int64_t n = (int64_t)s.n_frames * s.n_patches;
    if (n > (int64_t)0x7fffffff) return MAS_ERR_UNSUPPORTED;
    if (prm && prm->select_mode == MAS_SELECT_TOPK && (s.keep_k < 1 || s.keep_k > n)) return MAS_ERR_INVALID_ARG;
    prev_req = s.request;
    row += n;
  }
  {
    const int tr = generic_tile_rows(row);
    for (int32_t k = 0; k < n_segs; ++k) { const int64_t n = (int64_t)segs[k].n_frames * segs[k].n_patches; tiles += (n + tr - 1) / tr; }
  }
  if (row > (int64_t)0x7fffffff - kTileRows) return MAS_ERR_UNSUPPORTED;   // kept_idx is int32
  if (prm) {
    if (prm->select_mode != MAS_SELECT_TOPK && prm->select_mode != MAS_SELECT_THRESHOLD && prm->select_mode != MAS_SELECT_ADAPTIVE) return MAS_ERR_INVALID_ARG;
    if (!(prm->lambda_spatial >= 0.f) || !(prm->lambda_temp >= 0.f) || !(prm->lambda_spatial + prm->lambda_temp <= 1.0f + 1e-6f))
      return MAS_ERR_INVALID_ARG;
  }
  *N_out = row; *nQ_out = q_off[n_req]; *n_tiles_out = (int32_t)tiles; *maxL_out = maxL;
  return MAS_OK;
}

static Layout make_layout(int32_t n_segs, int32_t n_req, int64_t N, int64_t nQ, int32_t n_tiles, size_t tc_bytes, size_t tc_parts_max,
                          int64_t n_frames, int d) {
  Layout l{};
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes, 256); return at; };
  l.segs = take(sizeof(DevSeg) * n_segs);
  l.tiles = take(sizeof(DevTile) * n_tiles);
  l.req = take(sizeof(int32_t) * (n_req + 1));
  l.tc_sched = take(tc_bytes);
  l.tc_sched_x = take(tc_bytes);   // the schedule of the calls that add 64 B rows (NEXT-1, NEXT-2)
  l.tc_sched_u = take(tc_bytes);   // the same two schedules without K-split, for devices that refuse the cooperative launch
  l.tc_sched_xu = take(tc_bytes);
  l.tc_segrank_u = take(sizeof(int32_t) * (n_segs + 1));
  l.tc_segrank = take(sizeof(int32_t) * (n_segs + 1));   // first partial slot of every segment (TcTile::part0), NEXT-2
  l.frames = take(sizeof(DevFrame) * (size_t)n_frames);   // NEXT-3: first row and patch count of every frame
  l.tables_end = o;
  l.qinv = take(sizeof(float) * nQ);
  l.s = take(sizeof(float) * N);
  l.gamma = take(sizeof(float) * N);
  l.rel = take(sizeof(float) * N);
  l.mas = take(sizeof(float) * N);
  l.mask = take(N);
  l.segout = take(sizeof(mas_segment_out) * n_segs);
  l.nkept = take(sizeof(int32_t) * n_segs);
  l.keptoff = take(sizeof(int64_t) * (n_segs + 1));
  l.counter = take(256);
  l.tc_xflag = take(sizeof(unsigned int) * kTcMaxCtas);   // K-split: one flag and one exchange slot per CTA of the score kernel
  l.tc_xchg = take(tc_xchg_bytes());
  l.heads_part = take(sizeof(float) * kHeadRows * std::max((size_t)n_tiles, tc_parts_max));   // NEXT-2 scratch: per-tile / per-block column sums
  l.merge_part = take(sizeof(float) * std::max<size_t>(1024 * (size_t)kMergeCtas, 2 * (size_t)kTcMaxCtas * (size_t)d));   // NEXT-3 scratch: partial sums of the merged tokens
  l.merge_cnt = take(sizeof(int32_t) * (size_t)kMergeCtas);
  l.gridw = take(sizeof(int32_t) * n_segs);   // NEXT-3 scratch: the caller's grid widths
  l.heads_cq = take(sizeof(float) * kHeadRows * kHeadSlabs * (size_t)n_req);
  l.total = o;
  return l;
}

static int64_t count_frames(const mas_segment* segs, int32_t n_segs) {
  int64_t f = 0;
  for (int32_t k = 0; k < n_segs; ++k) f += segs[k].n_frames;
  return f;
}

extern "C" int mas_plan_workspace_bytes(const mas_segment* h_segs, int32_t n_segs, const int64_t* h_q_off, int32_t n_requests,
                                        int32_t d, int32_t dtype, size_t* out_bytes) {
  if (!out_bytes) return MAS_ERR_INVALID_ARG;
  int64_t N, nQ; int32_t nt, maxL;
  int st = validate(h_segs, n_segs, h_q_off, n_requests, d, dtype, nullptr, &N, &nQ, &nt, &maxL);
  if (st != MAS_OK) return st;
  *out_bytes = make_layout(n_segs, n_requests, N, nQ, nt, tc_schedule_bytes(h_segs, n_segs), tc_max_parts(h_segs, n_segs), count_frames(h_segs, n_segs), d).total;
  return MAS_OK;
}

// The opt-in to large dynamic shared memory applies to the device that is current when it is made: once per device.
static std::mutex g_attr_mu;
static bool g_attr_done[64] = {};
static cudaError_t set_kernel_attrs(int dev) {
  std::lock_guard<std::mutex> lk(g_attr_mu);
  if (dev >= 0 && dev < 64 && g_attr_done[dev]) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(k_score_mma<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, score_mma_smem_bytes(0));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_score_mma<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, score_mma_smem_bytes(1));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_lsh_sig<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, score_mma_smem_bytes(0));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_lsh_sig<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, score_mma_smem_bytes(1));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_heads_proj<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, score_mma_smem_bytes(0));
  if (e == cudaSuccess) e = cudaFuncSetAttribute(k_heads_proj<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, score_mma_smem_bytes(1));
  if (e == cudaSuccess) e = tc_set_kernel_attrs();
  {
    typedef void (*merge_fn)(const DevFrame*, int, const char*, const uint8_t*, float*, int32_t*, float*, int32_t*, int, long long, long long, int);
    const merge_fn mk[6] = {k_merge_tma<0, 1>, k_merge_tma<0, 2>, k_merge_tma<0, 4>, k_merge_tma<1, 1>, k_merge_tma<1, 2>, k_merge_tma<1, 4>};
    for (merge_fn k : mk)
      if (e == cudaSuccess) e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, kMergeTmaSmem + 1024);
  }
  if (e == cudaSuccess && dev >= 0 && dev < 64) g_attr_done[dev] = true;
  return e;
}

extern "C" int mas_plan_create(mas_plan** out, const mas_segment* h_segs, int32_t n_segs, const int64_t* h_q_off,
                               int32_t n_requests, int32_t d, int32_t dtype, const mas_params* params,
                               void* d_workspace, size_t workspace_bytes, mas_stream_t stream_) {
  if (!out || !params || !d_workspace) return MAS_ERR_INVALID_ARG;
  *out = nullptr;
  cudaStream_t stream = (cudaStream_t)stream_;
  int64_t N, nQ; int32_t nt, maxL;
  int st = validate(h_segs, n_segs, h_q_off, n_requests, d, dtype, params, &N, &nQ, &nt, &maxL);
  if (st != MAS_OK) return st;
  if ((reinterpret_cast<uintptr_t>(d_workspace) & 255u) != 0) return MAS_ERR_UNSUPPORTED;
  const size_t tc_bytes = tc_schedule_bytes(h_segs, n_segs);
  Layout lay = make_layout(n_segs, n_requests, N, nQ, nt, tc_bytes, tc_max_parts(h_segs, n_segs), count_frames(h_segs, n_segs), d);
  if (workspace_bytes < lay.total) return MAS_ERR_WORKSPACE;

  mas_plan* p = new (std::nothrow) mas_plan();
  if (!p) return MAS_ERR_INVALID_ARG;
  p->n_segs = n_segs; p->n_requests = n_requests; p->d = d; p->dtype = dtype;
  p->N = N; p->nQ = nQ; p->n_tiles = nt; p->max_L = maxL; p->lay = lay; p->ws = static_cast<char*>(d_workspace);
  p->prm.lambda_spatial = params->lambda_spatial; p->prm.lambda_temp = params->lambda_temp; p->prm.tau_s = params->tau_s;
  p->prm.kappa = params->kappa; p->prm.spatial_gain = params->spatial_gain; p->prm.spatial_bias = params->spatial_bias;
  p->prm.rel_gain = params->rel_gain; p->prm.rel_bias = params->rel_bias; p->prm.cut = params->cut;
  p->prm.select_mode = params->select_mode;

  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, dev);
  if (e == cudaSuccess) { p->pinned_bytes = lay.tables_end + 256; e = cudaHostAlloc(&p->pinned, p->pinned_bytes, cudaHostAllocDefault); }
  if (e == cudaSuccess) e = set_kernel_attrs(dev);
  if (e != cudaSuccess) { g_last_cuda = (int)e; (void)cudaGetLastError(); if (p->pinned) cudaFreeHost(p->pinned); delete p; return MAS_ERR_CUDA; }

  char* h = static_cast<char*>(p->pinned);
  std::memset(h, 0, p->pinned_bytes);
  DevSeg* hs = reinterpret_cast<DevSeg*>(h + lay.segs);
  DevTile* ht = reinterpret_cast<DevTile*>(h + lay.tiles);
  int32_t* hr = reinterpret_cast<int32_t*>(h + lay.req);
  int64_t kept = 0;
  int32_t ti = 0;
  for (int32_t r = 0; r <= n_requests; ++r) hr[r] = n_segs;
  const int tile_rows = generic_tile_rows(N);
  for (int32_t k = 0; k < n_segs; ++k) {
    const mas_segment& s = h_segs[k];
    DevSeg& ds = hs[k];
    ds.row0 = s.row0;
    ds.kept_off_static = kept;
    ds.n_rows = s.n_frames * s.n_patches;
    ds.n_patches = s.n_patches;
    ds.n_frames = s.n_frames;
    ds.request = s.request;
    ds.q0 = (int32_t)h_q_off[s.request];
    ds.L = (int32_t)(h_q_off[s.request + 1] - h_q_off[s.request]);
    ds.keep_k = params->select_mode == MAS_SELECT_TOPK ? s.keep_k : ds.n_rows;
    ds.tile0 = ti;
    kept += params->select_mode == MAS_SELECT_TOPK ? s.keep_k : 0;
    if (hr[s.request] > k) hr[s.request] = k;
    for (int32_t r0 = 0; r0 < ds.n_rows; r0 += tile_rows) {
      ht[ti].row_start = (int32_t)(s.row0 + r0);
      ht[ti].n_rows = ds.n_rows - r0 < tile_rows ? ds.n_rows - r0 : tile_rows;
      ht[ti].seg = k;
      ++ti;
    }
  }
  {
    DevFrame* hf = reinterpret_cast<DevFrame*>(h + lay.frames);
    int64_t f = 0;
    for (int32_t k = 0; k < n_segs; ++k)
      for (int32_t t = 0; t < h_segs[k].n_frames; ++t, ++f) {
        hf[f].row0 = h_segs[k].row0 + (int64_t)t * h_segs[k].n_patches;
        hf[f].n_patches = h_segs[k].n_patches;
        hf[f].seg = k;
      }
    p->n_frames = f;
    for (int32_t k = 0; k < n_segs; ++k) p->max_patches = std::max(p->max_patches, h_segs[k].n_patches);
  }
  for (int32_t r = n_requests - 1; r >= 0; --r)   // requests without segments get an empty range
    if (hr[r] > hr[r + 1]) hr[r] = hr[r + 1];
  p->kept_cap = params->select_mode == MAS_SELECT_TOPK ? kept : N;
  {   // segment kernel: about 2 tokens per thread on the longest segment, 1..8 CTAs per cluster (power of two)
    int64_t longest = 0;
    for (int32_t k = 0; k < n_segs; ++k) longest = std::max<int64_t>(longest, (int64_t)h_segs[k].n_frames * h_segs[k].n_patches);
    int c = 1;
    while (c < 8 && (int64_t)c * 2 * kSegThreads < longest) c *= 2;
    p->seg_cluster = c;
    const int64_t slice = (longest + c - 1) / c;     // tokens per CTA: up to 4 stay in registers per thread
    p->seg_threads = slice <= 1024 ? 256 : slice <= 2048 ? 512 : kSegThreads;
  }
  tc_build_schedule(p->tc, h_segs, n_segs, h_q_off, d, dtype, p->sm_count, h + lay.tc_sched, p->ws + lay.tc_sched);
  tc_build_schedule(p->tcx, h_segs, n_segs, h_q_off, d, dtype, p->sm_count, h + lay.tc_sched_x, p->ws + lay.tc_sched_x, true);
  tc_build_schedule(p->tcu, h_segs, n_segs, h_q_off, d, dtype, p->sm_count, h + lay.tc_sched_u, p->ws + lay.tc_sched_u, false, false);
  tc_build_schedule(p->tcxu, h_segs, n_segs, h_q_off, d, dtype, p->sm_count, h + lay.tc_sched_xu, p->ws + lay.tc_sched_xu, true, false);
  // per-segment range of partial slots (one per block of every tile that writes results; a segment's slots are contiguous)
  auto seg_ranks = [&](const TcSchedule& sc, size_t sched_off, size_t rank_off) {
    if (!sc.enabled) return;
    const TcTile* tt = reinterpret_cast<const TcTile*>(h + sched_off);
    int32_t* sr = reinterpret_cast<int32_t*>(h + rank_off);
    std::vector<int32_t> cnt(n_segs + 1, 0);
    for (int i = 0; i < sc.n_tiles; ++i)
      cnt[tt[i].seg + 1] += tt[i].n_blocks - (tt[i].k1 < d / 64 ? 1 : 0);   // a dumped first block writes no results
    sr[0] = 0;
    for (int32_t k = 0; k < n_segs; ++k) sr[k + 1] = sr[k] + cnt[k + 1];
  };
  seg_ranks(p->tcx, lay.tc_sched_x, lay.tc_segrank);
  seg_ranks(p->tcxu, lay.tc_sched_xu, lay.tc_segrank_u);

  // plan creation is set-up, not the hot path: it returns when the tables are on the device, so that the plan may be used on
  // any stream afterwards without further ordering (the entry points themselves never synchronise)
  e = cudaMemcpyAsync(p->ws, p->pinned, lay.tables_end, cudaMemcpyHostToDevice, stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(p->ws + lay.counter, 0, 256, stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(p->ws + lay.tc_xflag, 0, sizeof(unsigned int) * kTcMaxCtas, stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
  if (e != cudaSuccess) { g_last_cuda = (int)e; (void)cudaGetLastError(); cudaFreeHost(p->pinned); delete p; return MAS_ERR_CUDA; }
  *out = p;
  return MAS_OK;
}

extern "C" int mas_plan_enable_profiling(mas_plan* p, int32_t max_calls) {
  if (!p || max_calls < 0) return MAS_ERR_INVALID_ARG;
  for (cudaEvent_t e : p->prof_ev) cudaEventDestroy(e);
  p->prof_ev.clear();
  p->prof_slots = 0;
  p->prof_calls = 0;
  for (int32_t i = 0; i < max_calls * 4; ++i) {
    cudaEvent_t e;
    CK(cudaEventCreate(&e));
    p->prof_ev.push_back(e);
  }
  p->prof_slots = max_calls;
  return MAS_OK;
}
extern "C" int mas_plan_stage_times(const mas_plan* p, int32_t call, float* ms) {
  if (!p || !ms || p->prof_slots <= 0 || call < 0 || call >= p->prof_calls) return MAS_ERR_INVALID_ARG;
  const cudaEvent_t* e = &p->prof_ev[(size_t)(call % p->prof_slots) * 4];
  for (int i = 0; i < 3; ++i) CK(cudaEventElapsedTime(&ms[i], e[i], e[i + 1]));
  return MAS_OK;
}

extern "C" int mas_plan_destroy(mas_plan* p) {
  if (!p) return MAS_OK;
  for (cudaEvent_t e : p->prof_ev) cudaEventDestroy(e);
  if (p->pinned) cudaFreeHost(p->pinned);
  delete p;
  return MAS_OK;
}
extern "C" int mas_plan_set_inline_query_norms(mas_plan* p, int32_t on) {
  if (!p) return MAS_ERR_INVALID_ARG;
  p->tc_inline_qnorm = on != 0;
  return MAS_OK;
}
extern "C" int64_t mas_plan_n_tokens(const mas_plan* p) { return p ? p->N : -1; }
extern "C" int64_t mas_plan_n_queries(const mas_plan* p) { return p ? p->nQ : -1; }
extern "C" int64_t mas_plan_n_frames(const mas_plan* p) { return p ? p->n_frames : -1; }
extern "C" int64_t mas_plan_kept_capacity(const mas_plan* p) { return p ? p->kept_cap : -1; }

extern "C" int32_t mas_score_schedule(const mas_segment* h_segs, int32_t n_segs, const int64_t* h_q_off, int32_t n_requests,
                                      int32_t d, int32_t dtype, int32_t sm_count, int32_t* out_tiles, int32_t cap_tiles) {
  int64_t N, nQ; int32_t nt, maxL;
  const int st = validate(h_segs, n_segs, h_q_off, n_requests, d, dtype, nullptr, &N, &nQ, &nt, &maxL);
  if (st != MAS_OK) return -st;
  if (cap_tiles < 0 || (cap_tiles > 0 && !out_tiles)) return -MAS_ERR_INVALID_ARG;
  std::vector<char> buf(tc_schedule_bytes(h_segs, n_segs));
  TcSchedule sc;
  tc_build_schedule(sc, h_segs, n_segs, h_q_off, d, dtype, sm_count, buf.data(), buf.data());
  if (!sc.enabled) return 0;
  const TcTile* t = reinterpret_cast<const TcTile*>(buf.data());
  const int32_t* off = reinterpret_cast<const int32_t*>(buf.data() + (size_t)sc.n_tiles * sizeof(TcTile));
  for (int c = 0; c < sc.n_ctas; ++c)
    for (int i = off[c]; i < off[c + 1] && i < cap_tiles; ++i) {
      int32_t* o = out_tiles + (size_t)i * 16;
      o[0] = c; o[1] = t[i].row0; o[2] = t[i].n_rows; o[3] = t[i].n_blocks; o[4] = t[i].stride; o[5] = t[i].mode; o[6] = t[i].prev;
      o[7] = t[i].halo; o[8] = t[i].q_row0; o[9] = t[i].L; o[10] = t[i].seg; o[11] = t[i].part0;
      o[12] = t[i].k0; o[13] = t[i].k1; o[14] = t[i].n_wait; o[15] = t[i].peer;
    }
  return sc.n_tiles;
}

// ------------------------------------------------------------------------------------------------ launches
static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static int launch_qprep(const mas_plan* p, const void* Q, cudaStream_t st, bool pdl = false) {
  const unsigned grid = (unsigned)((p->nQ + 7) / 8);
  if (p->dtype == MAS_BF16) CK(launch_k(k_qprep<1>, dim3(grid), dim3(256), 0, st, pdl, Q, p->at<float>(p->lay.qinv), p->nQ, p->d));
  else CK(launch_k(k_qprep<0>, dim3(grid), dim3(256), 0, st, pdl, Q, p->at<float>(p->lay.qinv), p->nQ, p->d));
  return MAS_OK;
}

static ScoreArgs score_args(const mas_plan* p, const void* X, const void* Q, float* s, float* gamma, float* rel, float* S_opt) {
  ScoreArgs a;
  a.X = X; a.Q = Q; a.qinv = p->at<float>(p->lay.qinv);
  a.segs = p->at<DevSeg>(p->lay.segs); a.tiles = p->at<DevTile>(p->lay.tiles);
  a.s = s; a.gamma = gamma; a.rel = rel; a.S_opt = S_opt; a.sig = nullptr; a.d = p->d;
  a.heads_part = nullptr; a.heads_m = nullptr; a.heads_bias = 0.f; a.heads_tau = 0.f;
  return a;
}

static int launch_rowstats(const mas_plan* p, const void* X, float* s, float* gamma, cudaStream_t st) {
  ScoreArgs a = score_args(p, X, nullptr, s, gamma, nullptr, nullptr);
  if (p->dtype == MAS_BF16) k_rowstats<1><<<p->n_tiles, 256, 0, st>>>(a);
  else k_rowstats<0><<<p->n_tiles, 256, 0, st>>>(a);
  CK(cudaGetLastError());
  return MAS_OK;
}

static int launch_score_mma(const mas_plan* p, const void* X, const void* Q, float* s, float* gamma, float* rel, float* S_opt, cudaStream_t st) {
  ScoreArgs a = score_args(p, X, Q, s, gamma, rel, S_opt);
  if (p->dtype == MAS_BF16) k_score_mma<1><<<p->n_tiles, 256, score_mma_smem_bytes(1), st>>>(a);
  else k_score_mma<0><<<p->n_tiles, 256, score_mma_smem_bytes(0), st>>>(a);
  CK(cudaGetLastError());
  return MAS_OK;
}

// a0-a3 on the tcgen05 path.  The query norms ride the score kernel's prologue (one cooperative launch) unless the plan asks for,
// or the device forces, a launch of their own (k_qprep, then the plain score launch chained behind it).
static const TcSchedule& score_schedule_of(const mas_plan* p, bool rider) {
  // K-split tiles make CTAs wait for one another: only where the launch can be cooperative (all CTAs co-resident)
  return p->tc_coop_ok ? (rider ? p->tcx : p->tc) : (rider ? p->tcxu : p->tcu);
}
static int launch_score_tc(const mas_plan* p, bool rider, const void* X, const void* Q, float* s, float* dnorm, float* rel,
                           const void* Rm, unsigned long long* sig, const TcHeads* hf, cudaStream_t st, bool pdl) {
  unsigned long long* qr = p->at<unsigned long long>(p->lay.counter) + 8;
  float* qinv = p->at<float>(p->lay.qinv);
  float* xchg = p->at<float>(p->lay.tc_xchg);
  unsigned int* xflag = p->at<unsigned int>(p->lay.tc_xflag);
  if (p->tc_inline_qnorm && p->tc_coop_ok) {
    const cudaError_t e = tc_launch_score(score_schedule_of(p, rider), p->tc_maps, X, Q, qinv, s, dnorm, rel, qr, xchg, xflag, p->N, p->nQ, p->d, true,
                                          Rm, sig, hf, st);
    if (e == cudaSuccess) return MAS_OK;
    if (e != cudaErrorCooperativeLaunchTooLarge && e != cudaErrorNotSupported) { g_last_cuda = (int)e; (void)cudaGetLastError(); return MAS_ERR_CUDA; }
    (void)cudaGetLastError();     // not all CTAs can be co-resident here (e.g. an MPS partition): remembered for the plan's lifetime
    p->tc_coop_ok = false;
  }
  const bool chain = pdl && !(p->tc_inline_qnorm && !p->tc_coop_ok);
  int rc = launch_qprep(p, Q, st, chain);
  if (rc != MAS_OK) return rc;
  CK(tc_launch_score(score_schedule_of(p, rider), p->tc_maps, X, Q, qinv, s, dnorm, rel, qr, xchg, xflag, p->N, p->nQ, p->d, false, Rm, sig, hf, st, chain));
  return MAS_OK;
}

static SegArgs seg_args(const mas_plan* p, const float* s, float* gamma, const float* rel, float* m_spatial, float* mas_tok,
                        mas_segment_out* seg_out, uint8_t* keep_mask, int32_t* kept_idx, int64_t* kept_off, int64_t cap_rows,
                        bool gamma_raw = false) {
  SegArgs a;
  a.segs = p->at<DevSeg>(p->lay.segs); a.req_seg_off = p->at<int32_t>(p->lay.req);
  a.n_segs = p->n_segs; a.n_requests = p->n_requests; a.prm = p->prm;
  a.s = s; a.gamma = gamma; a.rel = rel; a.m_spatial = m_spatial; a.mas_tok = mas_tok; a.seg_out = seg_out;
  a.keep_mask = keep_mask; a.kept_idx = kept_idx; a.kept_off = kept_off; a.cap_rows = cap_rows;
  a.seg_nkept = p->at<int32_t>(p->lay.nkept);
  a.done_counter = p->at<unsigned int>(p->lay.counter);
  a.gamma_raw = gamma_raw ? 1 : 0;
  a.sqrt_d = sqrtf((float)p->d);
  return a;
}

static int launch_gather(const mas_plan* p, const void* X, const int32_t* kept_idx, const int64_t* kept_off, void* Y, int64_t cap_rows,
                         cudaStream_t st, bool pdl = false) {
  if (Y && cap_rows > 0) {
    const int64_t rows = cap_rows < p->kept_cap ? cap_rows : p->kept_cap;
    int64_t grid = (rows + 7) / 8;
    const int64_t gmax = (int64_t)p->sm_count * 16;
    if (grid > gmax) grid = gmax;
    if (grid < 1) grid = 1;
    const int esz = p->dtype == MAS_BF16 ? 2 : 4;
    CK(launch_k(k_gather, dim3((unsigned)grid), dim3(256), 0, st, pdl, static_cast<const char*>(X), static_cast<char*>(Y), kept_idx,
                kept_off + p->n_segs, cap_rows, p->d * esz));
  }
  return MAS_OK;
}

static int launch_select_tail(const mas_plan* p, const void* X, const uint8_t* mask, int32_t* kept_idx, const int64_t* kept_off,
                              void* Y, int64_t cap_rows, cudaStream_t st) {
  if (p->prm.select_mode != MAS_SELECT_TOPK && kept_idx) {
    k_compact_idx<<<p->n_segs, kSegThreads, 0, st>>>(p->at<DevSeg>(p->lay.segs), mask, kept_off, kept_idx, cap_rows);
    CK(cudaGetLastError());
  }
  return launch_gather(p, X, kept_idx, kept_off, Y, cap_rows, st);
}

extern "C" int32_t mas_plan_forward_launches(const mas_plan* p) {
  if (!p) return -1;
  // [qprep, generic path only] + score + segment (+ index compaction in threshold mode) + gather
  // adaptive mode: fuse and select are two launches (MAS_s needs every segment of the request before any keep count exists)
  return (p->tc.enabled && p->tc_inline_qnorm ? 3 : 4) + (p->prm.select_mode == MAS_SELECT_THRESHOLD ? 1 : 0) +
         (p->prm.select_mode == MAS_SELECT_ADAPTIVE ? 2 : 0);
}

// ------------------------------------------------------------------------------------------------ staged entry points
extern "C" int mas_spatial(const mas_plan* p, const void* X, float* s, float* m_spatial, mas_stream_t stream) {
  if (!p || !X || (!s && !m_spatial)) return MAS_ERR_INVALID_ARG;
  if (!aligned16(X)) return MAS_ERR_UNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  float* sb = s ? s : p->at<float>(p->lay.s);
  int rc = launch_rowstats(p, X, sb, nullptr, st);
  if (rc != MAS_OK) return rc;
  if (m_spatial) {
    k_spatial_finish<<<p->n_segs, kSegThreads, 0, st>>>(p->at<DevSeg>(p->lay.segs), p->prm, sb, m_spatial);
    CK(cudaGetLastError());
  }
  return MAS_OK;
}

extern "C" int mas_temporal(const mas_plan* p, const void* X, float* gamma, mas_stream_t stream) {
  if (!p || !X || !gamma) return MAS_ERR_INVALID_ARG;
  if (!aligned16(X)) return MAS_ERR_UNSUPPORTED;
  return launch_rowstats(p, X, nullptr, gamma, (cudaStream_t)stream);
}

extern "C" int mas_temporal_lsh(const mas_plan* p, const void* X, const void* Rm, uint64_t* sig, float* gamma_lsh, mas_stream_t stream) {
  if (!p || !X || !Rm || !sig) return MAS_ERR_INVALID_ARG;
  if (!aligned16(X) || !aligned16(Rm)) return MAS_ERR_UNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  ScoreArgs a = score_args(p, X, Rm, nullptr, nullptr, nullptr, nullptr);
  a.sig = reinterpret_cast<unsigned long long*>(sig);
  if (p->dtype == MAS_BF16) k_lsh_sig<1><<<p->n_tiles, 256, score_mma_smem_bytes(1), st>>>(a);
  else k_lsh_sig<0><<<p->n_tiles, 256, score_mma_smem_bytes(0), st>>>(a);
  CK(cudaGetLastError());
  if (gamma_lsh) {
    k_lsh_gamma<<<p->n_tiles, 128, 0, st>>>(p->at<DevSeg>(p->lay.segs), p->at<DevTile>(p->lay.tiles), a.sig, gamma_lsh);
    CK(cudaGetLastError());
  }
  return MAS_OK;
}

extern "C" int mas_crossmodal(const mas_plan* p, const void* X, const void* Q, float* rel, float* S_opt, mas_stream_t stream) {
  if (!p || !X || !Q || (!rel && !S_opt)) return MAS_ERR_INVALID_ARG;
  if (!aligned16(X) || !aligned16(Q)) return MAS_ERR_UNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  // without the similarity matrix this is the score sweep with two of its three outputs left in the plan's workspace: the tcgen05
  // kernel (bf16, d % 64 == 0) instead of the generic mma.sync one
  if (!S_opt && p->tc.enabled)
    return launch_score_tc(p, false, X, Q, p->at<float>(p->lay.s), p->at<float>(p->lay.gamma), rel, nullptr, nullptr, nullptr, st, false);
  int rc = launch_qprep(p, Q, st);
  if (rc != MAS_OK) return rc;
  return launch_score_mma(p, X, Q, nullptr, nullptr, rel ? rel : p->at<float>(p->lay.rel), S_opt, st);
}

// a0-a3 in one pass (the score stage of mas_forward on its own): s, gamma, rel
extern "C" int mas_score(const mas_plan* p, const void* X, const void* Q, float* s, float* gamma, float* rel, mas_stream_t stream) {
  if (!p || !X || !Q || !s || !rel) return MAS_ERR_INVALID_ARG;
  if (!aligned16(X) || !aligned16(Q)) return MAS_ERR_UNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  int rc;
  if (p->tc.enabled) {
    float* gb = gamma ? gamma : p->at<float>(p->lay.gamma);
    if ((rc = launch_score_tc(p, false, X, Q, s, gb, rel, nullptr, nullptr, nullptr, st, false)) != MAS_OK) return rc;
    if (gamma) {
      k_gamma_finish<<<p->n_tiles, 256, 0, st>>>(p->at<DevSeg>(p->lay.segs), p->at<DevTile>(p->lay.tiles), s, gamma, sqrtf((float)p->d));
      CK(cudaGetLastError());
    }
    return MAS_OK;
  }
  if ((rc = launch_qprep(p, Q, st)) != MAS_OK) return rc;
  return launch_score_mma(p, X, Q, s, gamma, rel, nullptr, st);
}

extern "C" int mas_fuse(const mas_plan* p, const float* s, const float* gamma, const float* rel, float* m_spatial, float* mas_tok,
                        mas_segment_out* seg_out, mas_stream_t stream) {
  if (!p || !s || !gamma || !rel || !mas_tok) return MAS_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  SegArgs a = seg_args(p, s, const_cast<float*>(gamma), rel, m_spatial, mas_tok, seg_out ? seg_out : p->at<mas_segment_out>(p->lay.segout),
                       nullptr, nullptr, nullptr, 0);
  CK(launch_kc(k_segment<true, false>, dim3((unsigned)(p->n_segs * p->seg_cluster)), dim3((unsigned)p->seg_threads), p->seg_cluster, st, false, a));
  return MAS_OK;
}

extern "C" int mas_select_compact(const mas_plan* p, const void* X, const float* mas_tok, uint8_t* keep_mask, int32_t* kept_idx,
                                  int64_t* kept_off, void* Y, int64_t cap_rows, mas_segment_out* seg_out, mas_stream_t stream) {
  if (!p || !mas_tok || cap_rows < 0) return MAS_ERR_INVALID_ARG;
  if (p->prm.select_mode == MAS_SELECT_ADAPTIVE && !seg_out) return MAS_ERR_INVALID_ARG;
  if (Y && (!X || !kept_idx)) return MAS_ERR_INVALID_ARG;
  if (Y && !aligned16(X)) return MAS_ERR_UNSUPPORTED;
  if (Y && !aligned16(Y)) return MAS_ERR_UNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  uint8_t* mask = keep_mask ? keep_mask : p->at<uint8_t>(p->lay.mask);
  int64_t* koff = kept_off ? kept_off : p->at<int64_t>(p->lay.keptoff);
  SegArgs a = seg_args(p, nullptr, nullptr, nullptr, nullptr, const_cast<float*>(mas_tok), seg_out, mask, kept_idx, koff, cap_rows);
  CK(launch_kc(k_segment<false, true>, dim3((unsigned)(p->n_segs * p->seg_cluster)), dim3((unsigned)p->seg_threads), p->seg_cluster, st, false, a));
  return launch_select_tail(p, X, mask, kept_idx, koff, Y, cap_rows, st);
}

// NEXT-3: pooling, merged token, residual coding (k_compress.cuh)
extern "C" int mas_spatial_pool(const mas_plan* p, const int32_t* h_grid_w, int32_t k, const float* s, float* s_pooled, mas_stream_t stream) {
  if (!p || !h_grid_w || !s || !s_pooled || s == s_pooled || k < 1 || k > 31) return MAS_ERR_INVALID_ARG;
  const DevSeg* hs = reinterpret_cast<const DevSeg*>(static_cast<const char*>(p->pinned) + p->lay.segs);
  for (int32_t q = 0; q < p->n_segs; ++q)
    if (h_grid_w[q] < 1 || hs[q].n_patches % h_grid_w[q] != 0) return MAS_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  // the caller's array is read during this call only, whatever memory it lives in: a copy from PAGEABLE memory is staged by the
  // runtime before cudaMemcpyAsync returns (a pinned source would be read when the copy executes)
  const std::vector<int32_t> gw(h_grid_w, h_grid_w + p->n_segs);
  CK(cudaMemcpyAsync(p->at<int32_t>(p->lay.gridw), gw.data(), sizeof(int32_t) * p->n_segs, cudaMemcpyHostToDevice, st));
  k_spatial_pool<<<p->n_tiles, 256, 0, st>>>(p->at<DevSeg>(p->lay.segs), p->at<DevTile>(p->lay.tiles), p->at<int32_t>(p->lay.gridw), k, s, s_pooled);
  CK(cudaGetLastError());
  return MAS_OK;
}

extern "C" int mas_merge_dropped(const mas_plan* p, const void* X, const uint8_t* keep_mask, float* Ymerge, int32_t* n_dropped,
                                 mas_stream_t stream) {
  if (!p || !X || !keep_mask || !Ymerge || !n_dropped) return MAS_ERR_INVALID_ARG;
  if (!aligned16(X)) return MAS_ERR_UNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  {   // rows of at most 16 KB: through the TMA unit (k_merge_tma), persistent CTAs over equal runs of rows
    const size_t row_bytes = (size_t)p->d * (p->dtype == MAS_BF16 ? 2 : 4);
    const int n_slots = (int)std::min<size_t>(32, kMergeTmaSmem / row_bytes);
    if (row_bytes % 16 == 0 && row_bytes / 16 <= (size_t)kMergeTmaWarps * 32 * kMergeTmaVPL && n_slots >= 4 && p->n_frames < 2147483647ll) {
      const int n_max = std::min(p->sm_count, kTcMaxCtas);
      const long long R = std::max<long long>(64, (p->N + n_max - 1) / n_max);
      const unsigned grid = (unsigned)((p->N + R - 1) / R);
      const size_t smem = 128 + 512 + (size_t)n_slots * row_bytes;
      float* part = p->at<float>(p->lay.merge_part);
      int32_t* cnt = p->at<int32_t>(p->lay.merge_cnt);
      const DevFrame* fr = p->at<DevFrame>(p->lay.frames);
      const int vpw = (int)((row_bytes / 16 + kMergeTmaWarps - 1) / kMergeTmaWarps), vpl = vpw <= 32 ? 1 : vpw <= 64 ? 2 : 4;
      const dim3 blk(32 * (kMergeTmaWarps + 1));
#define MSAS_MERGE_TMA(DT, VPL) \
  k_merge_tma<DT, VPL><<<grid, blk, smem, st>>>(fr, (int)p->n_frames, static_cast<const char*>(X), keep_mask, Ymerge, n_dropped, part, cnt, p->d, (long long)p->N, R, n_slots)
      if (p->dtype == MAS_BF16) { if (vpl == 1) MSAS_MERGE_TMA(1, 1); else if (vpl == 2) MSAS_MERGE_TMA(1, 2); else MSAS_MERGE_TMA(1, 4); }
      else { if (vpl == 1) MSAS_MERGE_TMA(0, 1); else if (vpl == 2) MSAS_MERGE_TMA(0, 2); else MSAS_MERGE_TMA(0, 4); }
#undef MSAS_MERGE_TMA
      CK(cudaGetLastError());
      k_merge_tma_finish<<<(unsigned)p->n_frames, 256, 0, st>>>(fr, part, cnt, Ymerge, n_dropped, p->d, R);
      CK(cudaGetLastError());
      return MAS_OK;
    }
  }
  const int slab = 32 * kMergeVPL * (p->dtype == MAS_BF16 ? 8 : 4);
  const int64_t slabs = (p->d + slab - 1) / slab;
  if (slabs > 65535) return MAS_ERR_UNSUPPORTED;
  // few frames (a batch of images): split each frame's rows over several CTAs, partial sums added in split order afterwards;
  // the scratch holds kMergeCtas slabs at most
  int64_t rs = (kMergeCtas + p->n_frames * slabs - 1) / (p->n_frames * slabs);
  rs = std::max<int64_t>(1, std::min<int64_t>(rs, std::min<int64_t>(16, (p->max_patches + 63) / 64)));
  while (rs > 1 && p->n_frames * slabs * rs > kMergeCtas) --rs;
  const dim3 grid((unsigned)p->n_frames, (unsigned)slabs, (unsigned)rs);
  float* part = p->at<float>(p->lay.merge_part);
  int32_t* cnt = p->at<int32_t>(p->lay.merge_cnt);
  if (p->dtype == MAS_BF16) k_merge_dropped<1><<<grid, 32 * kMergeWarps, 0, st>>>(p->at<DevFrame>(p->lay.frames), X, keep_mask, Ymerge, n_dropped, part, cnt, p->d);
  else k_merge_dropped<0><<<grid, 32 * kMergeWarps, 0, st>>>(p->at<DevFrame>(p->lay.frames), X, keep_mask, Ymerge, n_dropped, part, cnt, p->d);
  CK(cudaGetLastError());
  if (rs > 1) {
    k_merge_finish<<<dim3((unsigned)p->n_frames, (unsigned)slabs), 256, 0, st>>>(part, cnt, Ymerge, n_dropped, (int)rs, slab, p->d);
    CK(cudaGetLastError());
  }
  return MAS_OK;
}

extern "C" int mas_gather_residual(const mas_plan* p, const void* X, const int32_t* kept_idx, const int64_t* kept_off, void* Y,
                                   int64_t cap_rows, mas_stream_t stream) {
  if (!p || !X || !kept_idx || !kept_off || !Y || cap_rows < 0) return MAS_ERR_INVALID_ARG;
  if (!aligned16(X) || !aligned16(Y)) return MAS_ERR_UNSUPPORTED;
  if (cap_rows == 0) return MAS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t rows = cap_rows < p->kept_cap ? cap_rows : p->kept_cap;
  int64_t grid = (rows + 7) / 8;
  const int64_t gmax = (int64_t)p->sm_count * 16;
  grid = grid > gmax ? gmax : grid < 1 ? 1 : grid;
  if (p->dtype == MAS_BF16)
    k_gather_residual<1><<<(unsigned)grid, 256, 0, st>>>(p->at<DevSeg>(p->lay.segs), p->n_segs, static_cast<const char*>(X),
                                                         static_cast<char*>(Y), kept_idx, kept_off + p->n_segs, cap_rows, p->d);
  else
    k_gather_residual<0><<<(unsigned)grid, 256, 0, st>>>(p->at<DevSeg>(p->lay.segs), p->n_segs, static_cast<const char*>(X),
                                                         static_cast<char*>(Y), kept_idx, kept_off + p->n_segs, cap_rows, p->d);
  CK(cudaGetLastError());
  return MAS_OK;
}

// NEXT-2: learned heads (k_heads.cuh)
static int heads_check(const mas_plan* p, const void* X, const void* Q, const float* gamma, bool gamma_follows, const mas_heads* hd) {
  if (!p || !X || !Q || !hd) return MAS_ERR_INVALID_ARG;
  if (!hd->W || !hd->Wp || !hd->b1 || !hd->w2 || hd->hidden < 1 || hd->hidden >= kHeadRows) return MAS_ERR_INVALID_ARG;
  if (!aligned16(X) || !aligned16(Q) || !aligned16(hd->W) || !aligned16(hd->Wp) || p->d > 65536) return MAS_ERR_UNSUPPORTED;
  if (!gamma && !gamma_follows) {
    const DevSeg* hs = reinterpret_cast<const DevSeg*>(static_cast<const char*>(p->pinned) + p->lay.segs);
    for (int32_t k = 0; k < p->n_segs; ++k)
      if (hs[k].n_frames > 1) return MAS_ERR_INVALID_ARG;
  }
  return MAS_OK;
}
// p-half of the first layer, then per segment: partial sums -> hidden layer -> alpha; last CTA: softmax, Eq. 7
static int heads_q(const mas_plan* p, const void* Q, const mas_heads* hd, cudaStream_t st) {
  float* cq = p->at<float>(p->lay.heads_cq);
  const size_t qs = 0;
  const dim3 qgrid((unsigned)p->n_requests, kHeadSlabs);
  if (p->dtype == MAS_BF16) k_heads_q<1><<<qgrid, 256, qs, st>>>(Q, hd->Wp, p->at<int32_t>(p->lay.req), p->at<DevSeg>(p->lay.segs), cq, p->d);
  else k_heads_q<0><<<qgrid, 256, qs, st>>>(Q, hd->Wp, p->at<int32_t>(p->lay.req), p->at<DevSeg>(p->lay.segs), cq, p->d);
  CK(cudaGetLastError());
  return MAS_OK;
}
static int heads_finish(const mas_plan* p, const float* gamma, const mas_heads* hd, bool tc_slots, mas_segment_out* seg_out, cudaStream_t st,
                        bool pdl = false) {
  float* cq = p->at<float>(p->lay.heads_cq);
  HeadsArgs h;
  h.segs = p->at<DevSeg>(p->lay.segs); h.req_seg_off = p->at<int32_t>(p->lay.req);
  h.n_segs = p->n_segs; h.n_requests = p->n_requests; h.tile_rows = generic_tile_rows(p->N); h.hidden = hd->hidden;
  h.prm = p->prm; h.part = p->at<float>(p->lay.heads_part); h.slot_rank = tc_slots ? p->at<int32_t>(p->tc_coop_ok ? p->lay.tc_segrank : p->lay.tc_segrank_u) : nullptr;
  h.cq = cq; h.gamma = gamma; h.b1 = hd->b1; h.w2 = hd->w2; h.b2 = hd->b2;
  h.seg_out = seg_out; h.done_counter = p->at<unsigned int>(p->lay.counter);
  CK(launch_k(k_heads_finish, dim3((unsigned)p->n_segs), dim3(p->seg_cluster * p->seg_threads > 1024 ? 1024u : 256u), 0, st, pdl, h));
  return MAS_OK;
}

extern "C" int mas_learned_heads(const mas_plan* p, const void* X, const void* Q, const float* gamma, const mas_heads* hd, float* m_spatial,
                                 mas_segment_out* seg_out, mas_stream_t stream) {
  if (!m_spatial || !seg_out) return MAS_ERR_INVALID_ARG;
  int rc = heads_check(p, X, Q, gamma, false, hd);
  if (rc != MAS_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  if (p->tc.enabled && p->max_L <= 64) {
    // bf16, d % 64 == 0, every L <= 64: the weight rows ride the tcgen05 score kernel's MMA as 64 more B rows, exactly as in
    // mas_forward_heads; its own three outputs go to plan scratch (not to the gamma workspace: the caller's `gamma` may be that)
    TcHeads hf{p->at<float>(p->lay.heads_part), m_spatial, hd->b_spatial, p->prm.tau_s};
    if ((rc = heads_q(p, Q, hd, st)) != MAS_OK) return rc;
    if ((rc = launch_score_tc(p, true, X, Q, p->at<float>(p->lay.s), p->at<float>(p->lay.mas), p->at<float>(p->lay.rel), hd->W, nullptr, &hf, st,
                              false)) != MAS_OK)
      return rc;
    return heads_finish(p, gamma, hd, true, seg_out, st);
  }
  ScoreArgs a = score_args(p, X, hd->W, nullptr, nullptr, nullptr, nullptr);
  a.heads_part = p->at<float>(p->lay.heads_part); a.heads_m = m_spatial; a.heads_bias = hd->b_spatial; a.heads_tau = p->prm.tau_s;
  if (p->dtype == MAS_BF16) k_heads_proj<1><<<p->n_tiles, 256, score_mma_smem_bytes(1), st>>>(a);
  else k_heads_proj<0><<<p->n_tiles, 256, score_mma_smem_bytes(0), st>>>(a);
  CK(cudaGetLastError());
  if ((rc = heads_q(p, Q, hd, st)) != MAS_OK) return rc;
  return heads_finish(p, gamma, hd, false, seg_out, st);
}

// ------------------------------------------------------------------------------------------------ fused entry point
static int forward_impl(const mas_plan* p, const void* X, const void* Q, float* m_spatial, float* gamma, float* rel, float* mas_tok,
                        mas_segment_out* seg_out, uint8_t* keep_mask, int32_t* kept_idx, int64_t* kept_off, void* Y, int64_t cap_rows,
                        const void* Rm, unsigned long long* sig, const TcHeads* hf, mas_stream_t stream) {
  if (!p || !X || !Q || cap_rows < 0) return MAS_ERR_INVALID_ARG;
  if (Y && !kept_idx) return MAS_ERR_INVALID_ARG;
  if (!aligned16(X) || !aligned16(Q) || (Y && !aligned16(Y))) return MAS_ERR_UNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  float* sb = p->at<float>(p->lay.s);
  float* gb = gamma ? gamma : p->at<float>(p->lay.gamma);
  float* rb = rel ? rel : p->at<float>(p->lay.rel);
  float* mb = mas_tok ? mas_tok : p->at<float>(p->lay.mas);
  mas_segment_out* so = seg_out ? seg_out : p->at<mas_segment_out>(p->lay.segout);
  uint8_t* mask = keep_mask ? keep_mask : p->at<uint8_t>(p->lay.mask);
  int64_t* koff = kept_off ? kept_off : p->at<int64_t>(p->lay.keptoff);

  const cudaEvent_t* pev = p->prof_slots > 0 ? &p->prof_ev[(size_t)(p->prof_calls++ % p->prof_slots) * 4] : nullptr;
  if (pev) CK(cudaEventRecord(pev[0], st));
  int rc;
  const bool pdl = pev == nullptr;   // stage events between the kernels would serialise them anyway
  if (p->tc.enabled) {
    // a0-a3 in one launch: TMA + tcgen05, query norms in its prologue; gb receives sqrt(D), finished into gamma by the segment kernel
    if ((rc = launch_score_tc(p, Rm != nullptr || hf != nullptr, X, Q, sb, gb, rb, Rm, sig, hf, st, pdl)) != MAS_OK) return rc;
  } else {
    if ((rc = launch_qprep(p, Q, st)) != MAS_OK) return rc;
    if ((rc = launch_score_mma(p, X, Q, sb, gb, rb, nullptr, st)) != MAS_OK) return rc;
  }
  SegArgs a = seg_args(p, sb, gb, rb, m_spatial, mb, so, mask, kept_idx, koff, cap_rows, p->tc.enabled);
  if (pev) CK(cudaEventRecord(pev[1], st));
  const dim3 sgrid((unsigned)(p->n_segs * p->seg_cluster)), sblock((unsigned)p->seg_threads);
  if (p->prm.select_mode == MAS_SELECT_ADAPTIVE) {   // keep counts come from MAS_s, which the LAST cluster of the fuse launch writes
    CK(launch_kc(k_segment<true, false>, sgrid, sblock, p->seg_cluster, st, pdl, a));
    a.gamma_raw = 0;
    CK(launch_kc(k_segment<false, true>, sgrid, sblock, p->seg_cluster, st, pdl, a));
  } else {
    CK(launch_kc(k_segment<true, true>, sgrid, sblock, p->seg_cluster, st, pdl, a));
  }
  if (p->prm.select_mode != MAS_SELECT_TOPK && kept_idx) {
    CK(launch_k(k_compact_idx, dim3((unsigned)p->n_segs), dim3(kSegThreads), 0, st, pdl, (const DevSeg*)p->at<DevSeg>(p->lay.segs),
                (const uint8_t*)mask, (const int64_t*)koff, kept_idx, cap_rows));
  }
  if (pev) CK(cudaEventRecord(pev[2], st));
  rc = launch_gather(p, X, kept_idx, koff, Y, cap_rows, st, pdl);
  if (pev) CK(cudaEventRecord(pev[3], st));
  return rc;
}

extern "C" int mas_forward(const mas_plan* p, const void* X, const void* Q, float* m_spatial, float* gamma, float* rel, float* mas_tok,
                           mas_segment_out* seg_out, uint8_t* keep_mask, int32_t* kept_idx, int64_t* kept_off, void* Y, int64_t cap_rows,
                           mas_stream_t stream) {
  return forward_impl(p, X, Q, m_spatial, gamma, rel, mas_tok, seg_out, keep_mask, kept_idx, kept_off, Y, cap_rows, nullptr, nullptr, nullptr, stream);
}

extern "C" int mas_forward_heads(const mas_plan* p, const void* X, const void* Q, const mas_heads* hd, float* heads_m_spatial,
                                 mas_segment_out* heads_seg_out, const mas_outputs* o, mas_stream_t stream) {
  if (!heads_m_spatial || !heads_seg_out || !o) return MAS_ERR_INVALID_ARG;
  int rc = heads_check(p, X, Q, nullptr, true, hd);
  if (rc != MAS_OK) return rc;
  const float* gam = o->gamma ? o->gamma : p->at<float>(p->lay.gamma);   // finished by the segment kernel of this same call
  // the weight rows ride the score kernel's MMA as 64 more B rows when the accumulator has room for them (L <= 64 everywhere)
  if (p->tc.enabled && p->max_L <= 64) {
    TcHeads hf{p->at<float>(p->lay.heads_part), heads_m_spatial, hd->b_spatial, p->prm.tau_s};
    if ((rc = heads_q(p, Q, hd, (cudaStream_t)stream)) != MAS_OK) return rc;   // independent of X: ahead of the PDL-chained kernels
    rc = forward_impl(p, X, Q, o->m_spatial, o->gamma, o->rel, o->mas_tok, o->seg_out, o->keep_mask, o->kept_idx, o->kept_off, o->Y,
                      o->cap_rows, hd->W, nullptr, &hf, stream);
    if (rc != MAS_OK) return rc;
    return heads_finish(p, gam, hd, true, heads_seg_out, (cudaStream_t)stream, p->prof_slots == 0);
  }
  rc = forward_impl(p, X, Q, o->m_spatial, o->gamma, o->rel, o->mas_tok, o->seg_out, o->keep_mask, o->kept_idx, o->kept_off, o->Y,
                    o->cap_rows, nullptr, nullptr, nullptr, stream);
  if (rc != MAS_OK) return rc;
  return mas_learned_heads(p, X, Q, gam, hd, heads_m_spatial, heads_seg_out, stream);
}

extern "C" int mas_forward_lsh(const mas_plan* p, const void* X, const void* Q, const void* Rm, uint64_t* sig, float* gamma_lsh,
                               const mas_outputs* o, mas_stream_t stream) {
  if (!p || !Rm || !sig || !o) return MAS_ERR_INVALID_ARG;
  if (!aligned16(Rm)) return MAS_ERR_UNSUPPORTED;
  // the hash rows ride the score kernel's MMA as 64 more B rows when the accumulator has room for them (L <= 64 everywhere)
  const bool fused = p->tc.enabled && p->max_L <= 64;
  int rc = forward_impl(p, X, Q, o->m_spatial, o->gamma, o->rel, o->mas_tok, o->seg_out, o->keep_mask, o->kept_idx, o->kept_off, o->Y,
                        o->cap_rows, fused ? Rm : nullptr, fused ? reinterpret_cast<unsigned long long*>(sig) : nullptr, nullptr, stream);
  if (rc != MAS_OK) return rc;
  if (!fused) return mas_temporal_lsh(p, X, Rm, sig, gamma_lsh, stream);
  if (gamma_lsh) {
    k_lsh_gamma<<<p->n_tiles, 128, 0, (cudaStream_t)stream>>>(p->at<DevSeg>(p->lay.segs), p->at<DevTile>(p->lay.tiles),
                                                              reinterpret_cast<const unsigned long long*>(sig), gamma_lsh);
    CK(cudaGetLastError());
  }
  return MAS_OK;
}

// ------------------------------------------------------------------------------------------------ NEXT-4: draft-confidence entropy
static int entropy_geometry(int64_t n_rows, int64_t V, int* splits, int64_t* chunk) {
  int dev = 0, sm = 148;
  if (cudaGetDevice(&dev) == cudaSuccess) (void)cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev);
  (void)cudaGetLastError();
  *splits = entropy_splits(n_rows, V, sm);
  *chunk = ((V + *splits - 1) / *splits + 7) / 8 * 8;
  *splits = (int)((V + *chunk - 1) / *chunk);
  return MAS_OK;
}
extern "C" int mas_draft_entropy_workspace_bytes(int64_t n_rows, int64_t V, size_t* out_bytes) {
  if (!out_bytes || n_rows < 1 || V < 1) return MAS_ERR_INVALID_ARG;
  *out_bytes = (size_t)n_rows * 256 * sizeof(EntTriple);   // upper bound: 256 splits per row
  return MAS_OK;
}
extern "C" int mas_draft_entropy(const void* logits, int64_t n_rows, int64_t V, int64_t row_stride, int32_t dtype, float theta_conf,
                                 float* H, uint8_t* speculate, void* d_workspace, size_t workspace_bytes, mas_stream_t stream) {
  if (!logits || n_rows < 1 || V < 1 || row_stride < V || (!H && !speculate) || !d_workspace) return MAS_ERR_INVALID_ARG;
  if (dtype != MAS_F32 && dtype != MAS_BF16) return MAS_ERR_INVALID_ARG;
  const int esz = dtype == MAS_BF16 ? 2 : 4;
  if (!aligned16(logits) || (row_stride * esz) % 16 != 0 || n_rows > 65535) return MAS_ERR_UNSUPPORTED;
  int splits; int64_t chunk;
  entropy_geometry(n_rows, V, &splits, &chunk);
  if (workspace_bytes < (size_t)n_rows * splits * sizeof(EntTriple)) return MAS_ERR_WORKSPACE;
  cudaStream_t st = (cudaStream_t)stream;
  EntTriple* part = static_cast<EntTriple*>(d_workspace);
  const dim3 grid((unsigned)splits, (unsigned)n_rows);
  if (dtype == MAS_BF16) k_entropy_partial<1><<<grid, 256, 0, st>>>(logits, V, row_stride, chunk, part);
  else k_entropy_partial<0><<<grid, 256, 0, st>>>(logits, V, row_stride, chunk, part);
  CK(cudaGetLastError());
  CK(launch_k(k_entropy_finish, dim3((unsigned)((n_rows + 3) / 4)), dim3(128), 0, st, true, (const EntTriple*)part, splits, n_rows, theta_conf,
              H, speculate));
  return MAS_OK;
}

// The same with the partial sums in a static device array: the call allocates nothing (include/msas.h).  In host code the array's
// name is only a host-side stand-in: the kernels get its device address, looked up once per device with that device current.
static __device__ __align__(256) EntTriple g_ent_static[MAS_DRAFT_ENTROPY_STATIC_MAX_PARTIALS];

static int ent_static_address(EntTriple** out) {
  constexpr int kMaxDev = 64;
  static std::mutex mu;
  static EntTriple* addr[kMaxDev] = {};
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDev) return MAS_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lk(mu);
  if (!addr[dev]) {
    void* ptr = nullptr;
    CK(cudaGetSymbolAddress(&ptr, g_ent_static));
    addr[dev] = static_cast<EntTriple*>(ptr);
  }
  *out = addr[dev];
  return MAS_OK;
}

extern "C" int mas_draft_entropy_static(const void* logits, int64_t n_rows, int64_t V, int64_t row_stride, int32_t dtype, float theta_conf,
                                        float* H, uint8_t* speculate, mas_stream_t stream) {
  if (!logits || n_rows < 1 || V < 1 || row_stride < V || (!H && !speculate)) return MAS_ERR_INVALID_ARG;
  if (dtype != MAS_F32 && dtype != MAS_BF16) return MAS_ERR_INVALID_ARG;
  const int esz = dtype == MAS_BF16 ? 2 : 4;
  if (!aligned16(logits) || (row_stride * esz) % 16 != 0 || n_rows > 65535) return MAS_ERR_UNSUPPORTED;
  int splits; int64_t chunk;
  entropy_geometry(n_rows, V, &splits, &chunk);
  if (n_rows * (int64_t)splits > (int64_t)MAS_DRAFT_ENTROPY_STATIC_MAX_PARTIALS) return MAS_ERR_WORKSPACE;   // beyond the static array
  EntTriple* part = nullptr;
  const int rc = ent_static_address(&part);
  if (rc != MAS_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const dim3 grid((unsigned)splits, (unsigned)n_rows);
  if (dtype == MAS_BF16) k_entropy_partial<1><<<grid, 256, 0, st>>>(logits, V, row_stride, chunk, part);
  else k_entropy_partial<0><<<grid, 256, 0, st>>>(logits, V, row_stride, chunk, part);
  CK(cudaGetLastError());
  CK(launch_k(k_entropy_finish, dim3((unsigned)((n_rows + 3) / 4)), dim3(128), 0, st, true, (const EntTriple*)part, splits, n_rows, theta_conf,
              H, speculate));
  return MAS_OK;
}

// ------------------------------------------------------------------------------------------------ host-buffer convenience
static int forward_host_impl(const mas_plan* p, const void* h_X, const void* h_Q, void* d_X, void* d_Q, const mas_outputs* d_out,
                             const mas_outputs* h_out, mas_stream_t stream, bool final_sync) {
  if (!p || !h_X || !h_Q || !d_X || !d_Q || !d_out) return MAS_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t esz = p->dtype == MAS_BF16 ? 2 : 4;
  CK(cudaMemcpyAsync(d_X, h_X, (size_t)p->N * p->d * esz, cudaMemcpyHostToDevice, st));
  CK(cudaMemcpyAsync(d_Q, h_Q, (size_t)p->nQ * p->d * esz, cudaMemcpyHostToDevice, st));
  int64_t* koff = d_out->kept_off ? d_out->kept_off : p->at<int64_t>(p->lay.keptoff);
  int rc = mas_forward(p, d_X, d_Q, d_out->m_spatial, d_out->gamma, d_out->rel, d_out->mas_tok, d_out->seg_out, d_out->keep_mask,
                       d_out->kept_idx, koff, d_out->Y, d_out->cap_rows, stream);
  if (rc != MAS_OK) return rc;
  if (h_out) {
    const size_t N = (size_t)p->N;
    auto back = [&](void* h, const void* d, size_t bytes) -> cudaError_t {
      if (!h) return cudaSuccess;
      if (!d) return cudaErrorInvalidValue;
      return cudaMemcpyAsync(h, d, bytes, cudaMemcpyDeviceToHost, st);
    };
    CK(back(h_out->m_spatial, d_out->m_spatial, N * 4));
    CK(back(h_out->gamma, d_out->gamma, N * 4));
    CK(back(h_out->rel, d_out->rel, N * 4));
    CK(back(h_out->mas_tok, d_out->mas_tok, N * 4));
    CK(back(h_out->seg_out, d_out->seg_out, sizeof(mas_segment_out) * p->n_segs));
    CK(back(h_out->keep_mask, d_out->keep_mask, N));
    CK(back(h_out->kept_off, koff, sizeof(int64_t) * (p->n_segs + 1)));
    if (h_out->kept_idx || h_out->Y) {
      int64_t* total_h = reinterpret_cast<int64_t*>(static_cast<char*>(p->pinned) + p->lay.tables_end);
      int64_t total = p->kept_cap;
      if (p->prm.select_mode != MAS_SELECT_TOPK) {   // the kept count is data dependent: read it before sizing the copies
        CK(cudaMemcpyAsync(total_h, koff + p->n_segs, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        total = *total_h;
      }
      if (total > d_out->cap_rows) total = d_out->cap_rows;
      if (total > h_out->cap_rows) total = h_out->cap_rows;
      if (total > 0) {
        CK(back(h_out->kept_idx, d_out->kept_idx, sizeof(int32_t) * (size_t)total));
        CK(back(h_out->Y, d_out->Y, (size_t)total * p->d * esz));
      }
    }
  }
  if (final_sync) CK(cudaStreamSynchronize(st));
  return MAS_OK;
}
extern "C" int mas_forward_host(const mas_plan* p, const void* h_X, const void* h_Q, void* d_X, void* d_Q, const mas_outputs* d_out,
                                const mas_outputs* h_out, mas_stream_t stream) {
  return forward_host_impl(p, h_X, h_Q, d_X, d_Q, d_out, h_out, stream, true);
}
extern "C" int mas_forward_host_async(const mas_plan* p, const void* h_X, const void* h_Q, void* d_X, void* d_Q, const mas_outputs* d_out,
                                      const mas_outputs* h_out, mas_stream_t stream) {
  return forward_host_impl(p, h_X, h_Q, d_X, d_Q, d_out, h_out, stream, false);
}
