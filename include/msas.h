/*
 * msas.h — C ABI of libmsas: the Modality Activation Sparsity (MAS) pass of MSAO
 * (arxiv/paper_2604_02945, §4.1 "Lightweight Heterogeneous Modality-Aware via Fine-Grained Sparsity",
 * PAPER.md:81-124, Eq. 3-7), B200 / sm_100a.
 *
 * What the pass computes (normative definitions: SPEC.md S0-S5):
 *   spatial     per-token RMS activation, per-segment standardise, sigmoid  -> M_spatial, rho_spatial  (Eq. 3-4)
 *   temporal    per-patch relative L2 change against the previous frame     -> gamma, gamma_avg       (Eq. 5,   PAPER.md:100-105)
 *   crossmodal  max-over-query cosine relevance (X·Q^T on tensor cores)      -> rel, alpha, beta       (Eq. 6,   PAPER.md:107-116)
 *   fuse        per-token and per-modality MAS                               -> mas_tok, MAS_m         (Eq. 7,   PAPER.md:118-124)
 *   select      top-k (ties -> lower index) or threshold, stream compaction  -> keep_mask, kept_idx, Y
 *
 * Conventions
 *   - Plain C ABI. Every call returns an int status (MAS_OK = 0). No exceptions, no printing, no global mutable state
 *     (the last CUDA error code is kept per thread).
 *   - Pointers named h_* are HOST pointers, read during the call. All other data pointers are DEVICE pointers.
 *   - The caller owns every buffer. The library never allocates or frees device memory. Device entry points never
 *     synchronise: all work is enqueued on the caller's stream (`mas_stream_t` is a `cudaStream_t`) and outputs are
 *     valid once the caller has synchronised that stream. Only `mas_forward_host` blocks (documented there).
 *   - Inputs are never modified. Inputs must be finite; NaN/Inf give unspecified scores but no out-of-bounds access.
 *   - X is [N, d] row-major (bf16 or fp32), row stride d, base pointer 16-byte aligned, rows of all segments packed in
 *     segment order. Q is [sum L_r, d] row-major, same dtype, 16-byte aligned; request r owns rows q_off[r]..q_off[r+1].
 *   - Limits: d % 8 == 0 (bf16) or d % 4 == 0 (fp32), 8 <= d <= 65536; 1 <= L_r <= MAS_MAX_QUERY_TOKENS; T, P >= 1.
 *     Anything else returns MAS_ERR_UNSUPPORTED (never a silent fallback; there is no CPU path).
 */
#ifndef MSAS_H_
#define MSAS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MAS_VERSION 100              /* 0.1.0 */
#define MAS_MAX_QUERY_TOKENS 128     /* per request */

enum { MAS_OK = 0, MAS_ERR_INVALID_ARG = 1, MAS_ERR_UNSUPPORTED = 2, MAS_ERR_WORKSPACE = 3, MAS_ERR_CUDA = 4 };

typedef enum { MAS_F32 = 0, MAS_BF16 = 1 } mas_dtype;
typedef enum { MAS_MOD_IMAGE = 1, MAS_MOD_VIDEO = 2, MAS_MOD_AUDIO = 3 } mas_modality;   /* text is the query, never a segment */
/* MAS_SELECT_ADAPTIVE (NEXT-3, "beta_m >= 1 - MAS_m"): top-k with keep_k = clamp(ceil((1 - MAS_s) N_s - 1e-9), 1, N_s)
 * taken on the device from the segment score of the fuse step (double arithmetic on the fp32 MAS_s); keep_k in the table is ignored. */
typedef enum { MAS_SELECT_TOPK = 0, MAS_SELECT_THRESHOLD = 1, MAS_SELECT_ADAPTIVE = 2 } mas_select_mode;

typedef void* mas_stream_t;          /* a cudaStream_t (0 = the legacy default stream) */

/* One per (request, modality). Segments of one request are contiguous and in request order; segments tile X
 * in order without gaps: row0[0] = 0, row0[s+1] = row0[s] + n_frames[s]*n_patches[s].  (SPEC.md "Data model") */
typedef struct {
  int32_t request;          /* 0..R-1, non-decreasing */
  int32_t modality;         /* mas_modality, informational: n_frames > 1 decides temporal applicability (G11) */
  int64_t row0;             /* first row in X */
  int32_t n_frames;         /* T >= 1 */
  int32_t n_patches;        /* P >= 1, N_s = T*P */
  int32_t keep_k;           /* top-k mode: 1..N_s (see mas_keep_count); ignored in threshold mode */
  int32_t reserved_;        /* must be 0 */
} mas_segment;              /* 32 bytes */

typedef struct {
  float lambda_spatial;     /* 0.6 */
  float lambda_temp;        /* 0.4   PAPER.md:255 ; both >= 0, lambda_spatial + lambda_temp <= 1 */
  float tau_s;              /* 0.3   PAPER.md:255, Eq. 4 */
  float kappa;              /* 10.0  softmax temperature on the mean cosine (SPEC G20) */
  float spatial_gain;       /* 1     the 1x1 conv on the one-channel statistic (SPEC G2) */
  float spatial_bias;       /* 0 */
  float rel_gain;           /* 1 */
  float rel_bias;           /* 0 */
  float cut;                /* 0.5   threshold mode: keep iff MAS_i <= cut (SPEC G17) */
  int32_t select_mode;      /* mas_select_mode */
} mas_params;               /* 40 bytes */

/* Per-segment result (device). 36 bytes. */
typedef struct {
  float rho_spatial;        /* Eq. 4 */
  float gamma_avg;          /* S2: mean frame change over t = 1..T-1 (0 if T = 1) */
  float alpha_mean;         /* S3: mean_i max_j cos */
  float beta;               /* softmax over the request's segments */
  float mas;                /* Eq. 7 (redundancy reading G8) */
  float mean_s, std_s;      /* standardisation statistics of s (diagnostic) */
  int32_t n_tokens;
  int32_t n_kept;
} mas_segment_out;

/* Output bundle used by mas_forward_host; any member may be NULL (that output is skipped). */
typedef struct {
  float* m_spatial;         /* [N] */
  float* gamma;             /* [N] */
  float* rel;               /* [N] */
  float* mas_tok;           /* [N] */
  mas_segment_out* seg_out; /* [n_segs] */
  uint8_t* keep_mask;       /* [N] */
  int32_t* kept_idx;        /* [cap_rows] */
  int64_t* kept_off;        /* [n_segs+1] */
  void* Y;                  /* [cap_rows, d] */
  int64_t cap_rows;
} mas_outputs;

typedef struct mas_plan mas_plan;    /* opaque host object */

/* ---- host helpers (no GPU needed) ---- */
int         mas_version(void);
int         mas_last_cuda_error(void);                   /* cudaError_t of the last MAS_ERR_CUDA on this thread */
const char* mas_status_string(int status);
void        mas_params_default(mas_params* p);           /* the values in the comments above, MAS_SELECT_TOPK */
int32_t     mas_keep_count(int64_t n, double ratio);     /* SPEC S5/G16: min(n, max(1, ceil(ratio*n - 1e-9))) */

/* ---- plan: validates the tables, lays out the device workspace, builds the tile schedule ----
 * h_segs[n_segs], h_q_off[n_requests+1] are host arrays read during the call only.
 * mas_plan_workspace_bytes: bytes of device workspace the plan needs (256-byte aligned base expected).
 * mas_plan_create: copies the tables into d_workspace on `stream` (from a pinned staging area owned by the plan), waits
 * for that copy (plan creation is set-up: it is the one call besides mas_forward_host that synchronises) and returns a
 * host object, which may then be used on any stream; the workspace must stay alive and untouched until mas_plan_destroy.
 * One plan may be used by one stream and one host thread at a time (the workspace holds per-call scratch, the plan
 * caches the tensor maps of the last few (X, Q) pointer sets).  The kernels' shared-memory opt-in is made once per device,
 * at the first plan created on it.
 * Errors: INVALID_ARG (NULL, negative sizes, tables not tiling / not ordered, keep_k out of range in top-k mode,
 * bad params), UNSUPPORTED (limits above), WORKSPACE (too small), CUDA. */
int mas_plan_workspace_bytes(const mas_segment* h_segs, int32_t n_segs, const int64_t* h_q_off, int32_t n_requests,
                             int32_t d, int32_t dtype, size_t* out_bytes);
int mas_plan_create(mas_plan** out, const mas_segment* h_segs, int32_t n_segs, const int64_t* h_q_off,
                    int32_t n_requests, int32_t d, int32_t dtype, const mas_params* params,
                    void* d_workspace, size_t workspace_bytes, mas_stream_t stream);
int mas_plan_destroy(mas_plan* plan);                    /* frees the host object and its pinned staging only */

/* plan queries (host) */
int64_t mas_plan_n_tokens(const mas_plan* plan);         /* N */
int64_t mas_plan_n_queries(const mas_plan* plan);        /* sum L_r */
int64_t mas_plan_kept_capacity(const mas_plan* plan);    /* top-k: sum keep_k ; threshold, adaptive: N (worst case) */
int32_t mas_plan_forward_launches(const mas_plan* plan); /* number of kernels one mas_forward enqueues */

/* Profiling aid (bench.py's roofline leg).  After mas_plan_enable_profiling(plan, max_calls > 0) every mas_forward
 * records CUDA events on the caller's stream at its stage boundaries (score | segment+select | gather) into a ring of
 * max_calls slots; max_calls = 0 switches it off again.  mas_plan_stage_times reads the slot of call number `call`
 * (counted from the enable, modulo the ring) once the caller has synchronised the stream: ms[0..2] = stage durations.
 * The events are host-side driver objects owned by the plan; no device memory is allocated. */
int mas_plan_enable_profiling(mas_plan* plan, int32_t max_calls);
int mas_plan_stage_times(const mas_plan* plan, int32_t call, float* ms /*[3]*/);

/* ---- staged entry points (device pointers; each usable alone; outputs fp32 unless noted) ---- */

/* S1 (Eq. 3-4): s_i = RMS of row i; m_spatial = sigmoid of the per-segment standardised s. Either output may be NULL. */
int mas_spatial(const mas_plan* plan, const void* X, float* s /*[N]*/, float* m_spatial /*[N]*/, mas_stream_t stream);

/* S2 (Eq. 5 exact form): gamma[N]; 0 for T = 1 segments, 1 on keyframe rows. */
int mas_temporal(const mas_plan* plan, const void* X, float* gamma /*[N]*/, mas_stream_t stream);

/* a0-a3 in ONE pass over X (the score stage of mas_forward on its own): s[N] (S1's RMS), gamma[N] (S2; may be NULL: skipped) and
 * rel[N] (S3).  On the bf16 / d % 64 == 0 fast path this is the TMA + tcgen05 score kernel (plus one elementwise launch that
 * finishes gamma when it is asked for); otherwise the generic tile kernels.  Outputs as mas_spatial / mas_temporal /
 * mas_crossmodal give them (within summation order). */
int mas_score(const mas_plan* plan, const void* X, const void* Q, float* s /*[N]*/, float* gamma /*[N] or NULL*/, float* rel /*[N]*/,
              mas_stream_t stream);

/* S3 (Eq. 6 training-free): rel[N] = max_j cos(x_i, q_j). S_opt (may be NULL) receives the raw dot products
 * S_ij, row-major [N, MAS_MAX_QUERY_TOKENS] with columns >= L_r left untouched (tests only). */
int mas_crossmodal(const mas_plan* plan, const void* X, const void* Q, float* rel /*[N]*/, float* S_opt, mas_stream_t stream);

/* S1 stats + S3 stats + S4 (Eq. 7): per-token m_spatial, mas_tok; per-segment record (n_kept left 0). */
int mas_fuse(const mas_plan* plan, const float* s, const float* gamma, const float* rel,
             float* m_spatial /*[N] or NULL*/, float* mas_tok /*[N]*/, mas_segment_out* seg_out /*[n_segs]*/, mas_stream_t stream);

/* S5: selection on mas_tok, index compaction, row gather. Y may be NULL (indices only). cap_rows >= sum keep_k
 * (top-k) or any value >= 0 (threshold, adaptive): nothing is written past cap_rows and kept_off[n_segs] still holds the
 * true total so the caller detects overflow. seg_out (may be NULL): only n_kept is written. Adaptive mode READS
 * seg_out[k].mas (as mas_fuse left it) to size each segment's keep count: seg_out NULL is INVALID_ARG there. */
int mas_select_compact(const mas_plan* plan, const void* X, const float* mas_tok,
                       uint8_t* keep_mask /*[N]*/, int32_t* kept_idx /*[cap_rows]*/, int64_t* kept_off /*[n_segs+1]*/,
                       void* Y /*[cap_rows, d] or NULL*/, int64_t cap_rows, mas_segment_out* seg_out, mas_stream_t stream);

/* NEXT-1: the LITERAL temporal probe of Eq. 5: K = MAS_LSH_K sign-random-projection
 * hashes h_k(x) = [r_k . x >= 0] from the caller's matrix Rm[MAS_LSH_K, d] (device, same dtype and row stride as X,
 * 16-byte aligned; any seeded Gaussian matrix), sim = (1/K) sum_k 1[h_k(f_t) = h_k(f_{t-1})], gamma = 1 - sim.
 * sig[N] (device, required): bit k of sig[i] = h_k(x_i) -- the paper's "temporal similarity cache", 8 B per token.
 * gamma_lsh[N] (device, may be NULL): popcount(sig_t xor sig_{t-1}) / K per patch; keyframe 1; T = 1 segments 0.
 * The exact form mas_temporal computes is what this estimates (E[gamma_lsh] = angle / pi). */
#define MAS_LSH_K 64
int mas_temporal_lsh(const mas_plan* plan, const void* X, const void* Rm, uint64_t* sig /*[N]*/, float* gamma_lsh /*[N] or NULL*/,
                     mas_stream_t stream);

/* ---- fused entry point: one streaming score pass over X (a1+a2+a3), one segment kernel (a4+a5), one gather (a6).
 * Same outputs as the staged calls; any output may be NULL except kept_idx/kept_off when Y is requested. */
int mas_forward(const mas_plan* plan, const void* X, const void* Q,
                float* m_spatial, float* gamma, float* rel, float* mas_tok, mas_segment_out* seg_out,
                uint8_t* keep_mask, int32_t* kept_idx, int64_t* kept_off, void* Y, int64_t cap_rows, mas_stream_t stream);

/* mas_forward plus the literal LSH probe of NEXT-1 in the same pass: on the bf16 fast path with every L_r <= 64 the hash
 * rows Rm ride the score kernel's tensor-core contraction as 64 more B rows (no second sweep over X); otherwise the
 * call is mas_forward followed by mas_temporal_lsh.  `out`: device pointers as for mas_forward (any may be NULL as
 * there); sig[N] required, gamma_lsh[N] may be NULL. */
int mas_forward_lsh(const mas_plan* plan, const void* X, const void* Q, const void* Rm, uint64_t* sig /*[N]*/,
                    float* gamma_lsh /*[N] or NULL*/, const mas_outputs* out, mas_stream_t stream);

/* NEXT-2: the paper's LEARNED heads with caller-supplied weights (the trained ones are unpublished), giving the
 * per-modality descriptors of PAPER.md:118-124 as printed:
 *   Eq. 3   m_spatial_i = sigmoid(w_sp . x_i + b_spatial)            (1x1 convolution C -> 1 per patch)
 *   Eq. 4      rho_s = |{i : m_spatial_i < tau_s}| / N_s
 *   Eq. 6 alpha_s = w2 . relu(W1z z_s + W1p p_r + b1) + b2,  z_s = mean of the segment's rows of X,
 *                            p_r = mean of the request's rows of Q (one hidden ReLU layer of `hidden` units: reading N2)
 *   PAPER.md:116             beta_s = softmax of alpha over the request's segments (no temperature)
 *   Eq. 7 (reading G8)       MAS_s = 1 - beta_s (1 - lambda_sp rho_s - [T > 1] lambda_t (1 - gamma_avg_s))
 * W[MAS_HEADS_ROWS, d]: row 0 = w_sp, rows 1..hidden = W1z; Wp[MAS_HEADS_ROWS, d]: rows 1..hidden = W1p; b1, w2[MAS_HEADS_ROWS]:
 * entries 1..hidden.  Other rows / entries are ignored but must be readable and finite.  W and Wp: device, dtype and row
 * stride of X, 16-byte aligned; b1, w2: device fp32.  The struct itself is host memory, read during the call.
 * gamma[N]: the temporal probe's output (mas_temporal / mas_forward); NULL allowed iff no segment has T > 1.
 * Outputs: m_spatial[N] and seg_out[n_segs] (rho_spatial, gamma_avg, alpha_mean = alpha_s, beta, mas, n_tokens; mean_s, std_s,
 * n_kept = 0).  X is read once (one tile kernel with W as the B operand of its MMA); three launches.
 * Errors: INVALID_ARG (NULL, hidden outside 1..63, gamma NULL with a temporal segment), UNSUPPORTED (alignment). */
#define MAS_HEADS_ROWS 64
typedef struct {
  const void* W;
  const void* Wp;
  const float* b1;
  const float* w2;
  float b_spatial;
  float b2;
  int32_t hidden;
  int32_t reserved_;
} mas_heads;
int mas_learned_heads(const mas_plan* plan, const void* X, const void* Q, const float* gamma /*[N] or NULL*/, const mas_heads* heads,
                      float* m_spatial /*[N]*/, mas_segment_out* seg_out /*[n_segs]*/, mas_stream_t stream);
/* mas_forward plus the learned heads in the same pass: on the bf16 fast path with every L_r <= 64 the weight rows W ride the
 * score kernel's tensor-core contraction as 64 more B rows (no second sweep over X); otherwise the call is mas_forward followed
 * by mas_learned_heads.  `out` as for mas_forward_lsh; the learned descriptors go to heads_m_spatial[N] / heads_seg_out[n_segs]
 * (their gamma_avg is the one of this pass); the training-free outputs in `out` are unchanged by the presence of the heads. */
int mas_forward_heads(const mas_plan* plan, const void* X, const void* Q, const mas_heads* heads, float* heads_m_spatial /*[N]*/,
                      mas_segment_out* heads_seg_out /*[n_segs]*/, const mas_outputs* out, mas_stream_t stream);

/* NEXT-3, the rest of PAPER.md:98 / 105 ("coarsely compressed", "represented using only the residual difference").
 * All pointers device unless said otherwise.
 *
 * mas_spatial_pool: Eq. 3's AvgPool as a k x k window mean (1 <= k <= 31) of the per-token scalar map s[N] (mas_spatial's output)
 * on the H x W patch grid of every frame, W = h_grid_w[segment] (HOST array [n_segs], read during the call), H = P / W; the window
 * of cell (i, j) spans rows i-(k-1)/2 .. i+k/2 and the same columns, and the mean runs over the cells inside the grid.  The
 * pooled map goes to s_pooled[N] (must not alias s) and can be fed to mas_fuse in place of s.  INVALID_ARG if W < 1 or P % W != 0.
 *
 * mas_merge_dropped: one mean token per frame from the rows the selection dropped (keep_mask = 0).  Frames are numbered segment
 * by segment (mas_plan_n_frames of them): Ymerge[f, :] fp32 = mean of frame f's dropped rows (zeros if none), n_dropped[f] their
 * number.  Reads every dropped row once.
 *
 * mas_gather_residual: like the gather step of mas_select_compact (kept_idx / kept_off as produced there), but a kept token of
 * frame t >= 1 of a temporal segment is written as x_t - x_{t-1} (same patch, previous frame; bf16: the exact difference rounded
 * to nearest even), everything else as a copy.  Y[cap_rows, d] has the dtype of X; nothing is written past cap_rows. */
int64_t mas_plan_n_frames(const mas_plan* plan);         /* sum of n_frames over the segments */
int mas_spatial_pool(const mas_plan* plan, const int32_t* h_grid_w /*host [n_segs]*/, int32_t k, const float* s /*[N]*/,
                     float* s_pooled /*[N]*/, mas_stream_t stream);
int mas_merge_dropped(const mas_plan* plan, const void* X, const uint8_t* keep_mask /*[N]*/, float* Ymerge /*[n_frames, d]*/,
                      int32_t* n_dropped /*[n_frames]*/, mas_stream_t stream);
int mas_gather_residual(const mas_plan* plan, const void* X, const int32_t* kept_idx, const int64_t* kept_off /*[n_segs+1]*/,
                        void* Y /*[cap_rows, d]*/, int64_t cap_rows, mas_stream_t stream);

/* NEXT-4: the draft-confidence entropy of Eq. 9 and the speculate rule of Eq. 10, the
 * consumer-side step next to the MAS pass.  logits[n_rows, V] (device, fp32 or bf16, row stride `row_stride` elements,
 * base and stride 16-byte aligned, n_rows <= 65535): per row p = softmax(l), H = -sum_v p_v ln p_v,
 * speculate = [H <= theta_conf].  H[n_rows] fp32 and speculate[n_rows] u8 (device; either may be NULL).  Needs
 * mas_draft_entropy_workspace_bytes of device workspace; no plan.  Every logit is read once. */
int mas_draft_entropy_workspace_bytes(int64_t n_rows, int64_t V, size_t* out_bytes);
int mas_draft_entropy(const void* logits, int64_t n_rows, int64_t V, int64_t row_stride, int32_t dtype, float theta_conf,
                      float* H, uint8_t* speculate, void* d_workspace, size_t workspace_bytes, mas_stream_t stream);

/* The same for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): no workspace argument, and the call allocates nothing -- no cudaMalloc / cudaFree, no allocating library
 * routine.  The per-row partial sums (one {max, sum, sum of l e^l} triple per slice of a row) live in a static device array of
 * MAS_DRAFT_ENTROPY_STATIC_MAX_PARTIALS triples (12 bytes each: 192 KiB) that every GPU which loads the library holds until the
 * process exits.  Arguments, results and arithmetic are those of mas_draft_entropy (bit-identical H and speculate).
 * Returns MAS_ERR_WORKSPACE when n_rows x (slices per row, at most ceil(V / 8192) and about 4 x SM count / n_rows) exceeds
 * MAS_DRAFT_ENTROPY_STATIC_MAX_PARTIALS -- nothing is launched then (a row has one slice from 4 x SM count rows on: any
 * n_rows <= 16384 fits).  Every call on a device
 * shares the one array, which keeps the last call's contents (every triple a call reads it has written first, so nothing needs
 * clearing): calls that overlap on the GPU -- two streams, or two threads -- race; order them on one stream or with events.
 * The array's device address is looked up once per device (cudaGetSymbolAddress, the device current) on the first call there. */
#define MAS_DRAFT_ENTROPY_STATIC_MAX_PARTIALS 16384
int mas_draft_entropy_static(const void* logits, int64_t n_rows, int64_t V, int64_t row_stride, int32_t dtype, float theta_conf,
                             float* H, uint8_t* speculate, mas_stream_t stream);

/* ---- end-to-end convenience: HOST inputs -> HOST outputs.
 * Copies h_X -> d_X and h_Q -> d_Q (cudaMemcpyAsync; pinned host memory recommended), runs mas_forward into d_out,
 * copies every non-NULL member of h_out back (Y/kept_idx: only the rows actually kept) and SYNCHRONISES the stream
 * before returning. d_out members needed by the requested h_out members must be non-NULL. */
int mas_forward_host(const mas_plan* plan, const void* h_X, const void* h_Q, void* d_X, void* d_Q,
                     const mas_outputs* d_out, const mas_outputs* h_out, mas_stream_t stream);
/* The same without the final synchronisation: everything is enqueued on `stream` and the host outputs are valid once the caller
 * has synchronised it (in threshold / adaptive mode the call still waits once, for the kept count, before it sizes the last two
 * copies).  Two plans on two streams, called alternately, overlap one step's device-to-host copies with the next step's
 * host-to-device copies (PCIe is full duplex): bench.py's `e2e` leg does exactly that.  Host buffers must be pinned for the
 * copies to be asynchronous and must stay untouched until the stream has been synchronised. */
int mas_forward_host_async(const mas_plan* plan, const void* h_X, const void* h_Q, void* d_X, void* d_Q,
                     const mas_outputs* d_out, const mas_outputs* h_out, mas_stream_t stream);

/* The fused bf16 fast path computes the query norms (row a0) in the prologue of its score kernel, which needs every
 * CTA of that kernel resident at once (cooperative launch).  Where that is impossible (e.g. a partitioned GPU) the
 * library falls back by itself to a separate query-norm launch; `on = 0` forces that fallback (tests, diagnosis),
 * `on = 1` (default) restores the single-launch form.  Results are identical either way. */
int mas_plan_set_inline_query_norms(mas_plan* plan, int32_t on);

/* ---- introspection (host only, no CUDA call): the tile schedule mas_plan_create would build for the tcgen05 score
 * kernel on a device with `sm_count` SMs ("persistent CTAs over a host-built tile table; a tile
 * never straddles a segment").  A tile is up to 10 row blocks (one TMEM accumulator slot each: 512 columns / pad16 of the
 * longest query block) of one segment that share the request's query rows and are swept K-chunk by K-chunk.  Writes up to `cap_tiles` records of 16 int32 each, in per-CTA order:
 *   {cta, row0, n_rows, n_blocks, stride, mode, prev, halo, q_row0, L, seg, part0, k0, k1, n_wait, peer}
 *   k0, k1: K-SPLIT.  CTAs may share a row block along K so that every CTA carries the same cost: the tile's LAST block is swept
 *          over the 64-column K-chunks [k0, d / 64) only and its FIRST block over [0, k1) only (a one-block tile: [k0, k1)); the
 *          blocks in between, and every block of an unsplit tile (k0 = 0, k1 = d / 64), over all of K.  The part of a block
 *          that ends at chunk d / 64 owns it and writes its results (it is the last thing its CTA does): n_wait = number of
 *          other parts of the tile's last block, peer = CTA of the first of them (the CTAs that follow, each STARTING with its
 *          part, in descending K, and handing its partial sums over through the exchange slot of its CTA early in its sweep);
 *          n_wait = 0 and peer = -1 for every other tile;
 *   mode 0 (single-frame segment): the tile scores rows [row0, row0 + n_rows) in blocks of `stride` <= 128 rows (a multiple of 8);
 *   mode 1 (frames of P >= 64 rows): block b scores rows [row0 + b * stride, + n_rows), stride = prev = P, i.e. the same
 *          n_rows <= 128 patch rows in n_blocks consecutive frames; halo = 1 if the frame before block 0 is read as well;
 *   mode 2 (frames of P < 64 rows): the tile loads rows [row0, row0 + n_rows) in overlapping 128-row windows (block b = rows
 *          [row0 + b * stride, + 128), stride = 128 - P, prev = P; it scores its rows from P on, block 0 from `halo` in {0, P} on).
 * Returns the number of tiles the schedule has (which may exceed cap_tiles), 0 if the shape does not take the fast path
 * (fp32, d % 64 != 0), or a negative status (-MAS_ERR_*) for invalid descriptors.  Used by the CPU tests to check
 * coverage and balance. */
int32_t mas_score_schedule(const mas_segment* h_segs, int32_t n_segs, const int64_t* h_q_off, int32_t n_requests,
                           int32_t d, int32_t dtype, int32_t sm_count, int32_t* out_tiles, int32_t cap_tiles);

#ifdef __cplusplus
}
#endif
#endif /* MSAS_H_ */
