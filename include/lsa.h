/* lsa.h - C ABI of liblsa: the decode hot path of Lookahead Sparse Attention (LSA),
 * arxiv/paper_2606_09079 "FlashMemory-DeepSeek-V4", hand-written CUDA for sm_100a (B200).
 *
 * Citations: `P:n` = PAPER.md line n; `BJ` = BASELINE.json north_star/configs; `R#` = the
 * numbered readings in DESIGN.md.  Every step S0..S8 of DESIGN.md runs in CUDA kernels of this
 * library; there is no CPU fallback.  No torch / C++ types cross this boundary.
 *
 * The path (BJ north_star):
 *   every tau decode steps (S0) the Memory Indexer maps the hidden state h to a query embedding
 *   (S1), scores it against one embedding per CSA chunk (S2), a per-sequence top-k picks the
 *   chunks (S3), chunks missing from HBM are given pages of a shared paged hot pool (S4) and
 *   copied from the pinned-host cold pool on a side stream (S5); the new page table becomes
 *   visible `recall_lag` steps later (S6); every step split-K decode attention runs over
 *   all HCA entries (+) the selected resident chunks (+) the window ring (S7) and a combine
 *   kernel merges the splits (S8).
 *
 * Conventions
 *   - All functions return LSA_OK (0) or a negative lsa_status; lsa_last_error gives text.
 *   - "DEVICE" pointers are CUDA device memory of the current device, "PINNED HOST" is page-locked
 *     host memory (cudaHostAlloc / cudaHostRegister, e.g. torch pin_memory), "HOST" is any host
 *     memory.  Every buffer is CALLER-OWNED and must outlive the context; the library owns only
 *     the opaque context (page tables, LRU state, split-K scratch, events).
 *   - dtype is LSA_F32 or LSA_BF16 for q, K, V, W_q, h, chunk embeddings and out; scores, lse
 *     and all accumulation are fp32.
 *   - Row-major, innermost dimension contiguous, no padding, 16-byte aligned base pointers.
 *   - The five path calls only ENQUEUE work on the caller's two streams and return; they never
 *     block the host.  lsa_sync / lsa_get_* / lsa_step_host block.
 *   - Stream order is the caller's contract for its own buffers: q, k_new, v_new and out are read / written
 *     on stream_compute, h and sel_idx on stream_fetch; whatever produces them must be ordered before the
 *     call on that stream (lsa_step_host does this itself for its staging copies).
 *   - Not thread-safe per context.
 */
#ifndef LSA_H_
#define LSA_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LSA_VERSION 4

typedef struct lsa_ctx lsa_ctx; /* opaque */

enum lsa_status {
  LSA_OK = 0,
  LSA_ERR_INVALID_ARG = -1,    /* bad shape / null pointer / non-pinned cold pool / k > pages ... */
  LSA_ERR_CUDA = -2,           /* a CUDA runtime call failed (text in lsa_last_error)             */
  LSA_ERR_POOL_EXHAUSTED = -3, /* S4 found no unpinned page (cannot happen if hot_pages >= 2*sum k): reported by lsa_sync / */
                               /* lsa_get_stats; the pass that failed changed no table, residency or counter, but the   */
                               /* host's step bookkeeping has moved on - destroy the context                              */
  LSA_ERR_OOM = -4,
  LSA_ERR_STATE = -5,          /* call sequence not allowed (e.g. destroyed ctx)                  */
  LSA_ERR_UNSUPPORTED = -6     /* shape has no compiled kernel */
};

enum lsa_dtype { LSA_F32 = 0, LSA_BF16 = 1 };
enum lsa_attn_impl { LSA_ATTN_AUTO = 0, LSA_ATTN_SIMT = 1, LSA_ATTN_TCGEN05 = 2 };
/* S8 (merge of the split-K partials, tcgen05 path): AUTO = KERNEL = a separate combine kernel chained to the
 * attention kernel by programmatic dependent launch.  FUSED (B <= 4 only, else ignored) merges inside the
 * attention kernel behind a grid-wide arrival counter: one launch per step; measured slower than KERNEL on
 * B200, kept as a tested alternative. */
enum lsa_merge_mode { LSA_MERGE_AUTO = 0, LSA_MERGE_KERNEL = 1, LSA_MERGE_FUSED = 2 };

/* Cold-pool page format (NEXT-4 "FP8 KV pages", the host-link half; R34-R36).  NATIVE: a cold page is the hot
 * page image (dtype).  FP8_E4M3 (dtype must be LSA_BF16): a cold page is [2][C][D] e4m3 codes (1 byte each: sign, 4
 * exponent bits with bias 7, 3 mantissa bits, no infinities, S.1111.111 = NaN which must not occur) and the sequence has
 * one fp32 scale per block in lsa_seq_desc.cold_scale.  S5 dequantises while it copies: hot element = bf16_rne(fp32(code)
 * * scale) - exact when the scale is a power of two - so a recall moves HALF the bytes over the host link and everything
 * behind it (hot pool, S7) is unchanged.  lsa_export_chunks quantises: per block e = exponent of the largest magnitude - 7,
 * scale = 2^e, code = e4m3 round-to-nearest-even of x * 2^-e (all-zero block: scale 1); it writes codes and scales. */
enum lsa_cold_format { LSA_COLD_NATIVE = 0, LSA_COLD_FP8_E4M3 = 1 };

/* Shape and resources of one LSA layer shared by B sequences (BJ configs). */
typedef struct lsa_config {
  uint32_t struct_size;  /* = sizeof(lsa_config), ABI check                                     */
  int32_t dtype;         /* lsa_dtype                                                           */
  int32_t B;             /* sequences                                                           */
  int32_t H;             /* query heads, all sharing ONE K and ONE V head (MQA; R19)       */
  int32_t D;             /* K/V/q head dim                                                      */
  int32_t C;             /* compressed entries per CSA chunk = rows per page                    */
  int32_t W;             /* window ring capacity in raw tokens ("last 8K tokens"; R6)      */
  int32_t Dh;            /* indexer hidden size d                                        */
  int32_t E;             /* query / chunk embedding dim (BJ)                                    */
  int32_t k;             /* chunks selected per sequence = K_max (R2)                    */
  int32_t tau;           /* trigger interval (tau = 64)                                   */
  int32_t recall_lag;    /* 0: new table visible at the trigger step; 1: at t+1 (R9);     */
                         /* 2..tau-1: at t+lag - a longer fetch hides behind more steps          */
  float sm_scale;        /* softmax scale; 0 -> 1/sqrt(D) (R18)                                 */
  int64_t hot_pages;     /* P: pages in the hot pool; must be >= 2 * sum_b min(k, n_chunks_b)   */
  void* hot_pool;        /* DEVICE [P][2][C][D]: page = K block [C][D] then V block [C][D]      */
  const void* W_q;       /* DEVICE [E][Dh] query-tower weight (P:61-65 collapsed; R1)           */
  void* stream_compute;  /* cudaStream_t: S6-S8 (and S1-S5 when recall_lag == 0 waits on them)  */
  void* stream_fetch;    /* cudaStream_t: side band for S1-S5 ("async side band")         */
  int32_t attn_impl;     /* lsa_attn_impl; AUTO picks tcgen05 for bf16,H=64,D=512,C=128          */
  int32_t step_overlap;  /* 0 (default): q / k_new / v_new may be produced by the work enqueued on stream_compute  */
                         /* just before the call.  1: the caller guarantees they do NOT depend on the previous  */
                         /* lsa_step's output (independent layers / requests): B <= 4 steps then run underneath  */
                         /* the previous step's S8 instead of after it              */
  int32_t max_ctas;      /* 0 -> one split-K wave sized from the SM count                       */
  int32_t merge_mode;    /* lsa_merge_mode: where S8 runs (tcgen05 path)                        */
  int32_t cold_format;   /* lsa_cold_format: how a page is stored in the cold pool (host link)  */
  int32_t reserved0;
} lsa_config;

/* One sequence (CPU cold mirror + always-resident tiers).  n_chunks = ceil(n_csa/C);
 * the last chunk may be partial: rows >= n_csa - c*C of it are never attended (R22). */
typedef struct lsa_seq_desc {
  const void* cold_csa;  /* PINNED HOST [n_chunks][2][C][D]: chunk c = one page image (dtype; or  */
                         /* e4m3 codes, 1 byte each, with lsa_config.cold_format = FP8_E4M3)    */
  int64_t n_csa;         /* valid compressed (CSA) entries                                      */
  const void* chunk_emb; /* DEVICE [n_chunks][E], rows L2-normalised by the producer (R3)        */
  const void* hca_k;     /* DEVICE [n_hca][D] heavily-compressed (128:1) keys, always resident   */
  const void* hca_v;     /* DEVICE [n_hca][D]                                                   */
  int64_t n_hca;
  void* win_k;           /* DEVICE ring [W][D] raw-token window keys                            */
  void* win_v;           /* DEVICE ring [W][D]                                                  */
  int32_t w_len;         /* filled ring rows [0, w_len) are attended                            */
  int32_t w_head;        /* next ring slot to be written by lsa_step(k_new, v_new)              */
  int64_t step0;         /* initial decode-step counter (staggered triggers, R26)               */
  /* NEXT-4 growth (lsa_append_compressed); 0 = the compressed history of this sequence is static.  When cap_csa > 0:
   * cold_csa and chunk_emb hold ceil(cap_csa / C) chunks / rows (cold_csa writable), hca_k / hca_v hold cap_hca rows
   * (writable; the library zeroes rows [n_hca, cap_hca) at init), cap_csa >= n_csa, cap_hca >= n_hca.  Either every
   * sequence of a context grows or none does. */
  int64_t cap_csa;
  int64_t cap_hca;
  /* LSA_COLD_FP8_E4M3 only: DEVICE [n_chunks][2] fp32, (K scale, V scale) of every cold page; positive, finite.  Read by S5,
   * written by lsa_export_chunks.  NULL otherwise. */
  void* cold_scale;
} lsa_seq_desc;

typedef struct lsa_stats {
  uint64_t triggers;      /* per-sequence trigger events processed by S4                         */
  uint64_t hits;          /* selected chunks already resident                                   */
  uint64_t misses;        /* selected chunks fetched from the cold pool                          */
  uint64_t evictions;     /* pages whose previous owner was evicted                              */
  uint64_t bytes_fetched; /* misses * page_bytes                                                */
  uint64_t steps;         /* lsa_step calls                                                     */
  uint64_t attn_launches; /* kernels launched by S7+S8                                          */
  uint64_t index_launches;/* kernels launched by S1-S5                                          */
  int32_t pool_error;     /* nonzero if S4 ever ran out of pages                                 */
  int32_t attn_impl;      /* implementation actually in use (lsa_attn_impl)                      */
  int32_t attn_ctas;      /* CTAs of the last S7 launch                                          */
  int32_t reserved;
  uint64_t csa_appended;  /* CSA entries handed over by lsa_append_compressed (all sequences)    */
  uint64_t hca_appended;  /* HCA entries handed over                                            */
  uint64_t chunks_exported;/* chunks completed by an append and mirrored to the cold pool         */
} lsa_stats;

/* Create a context.  All pages start FREE, every chunk starts in the cold pool, the attended
 * page table of every sequence is empty (BJ cfg 1 "all chunks start in the host cold pool"; R10).
 * Errors: INVALID_ARG for null pointers, B/H/D/C/k/tau < 1, D % 8 != 0, hot_pages too small,
 * non-pinned cold_csa; UNSUPPORTED if no kernel is compiled for (dtype,H,D). */
int lsa_init_pools(const lsa_config* cfg, const lsa_seq_desc* seqs /* HOST [B] */, lsa_ctx** out);

/* S1-S3 for n sequences: q_hat = normalize(W_q h_i), score_c = q_hat . Emb[c]
 * (P:71-75), first min(k, n_chunks) chunk ids by (score desc, chunk idx asc) (R2, R14).
 *   h         DEVICE [n][Dh], row i belongs to sequence seq_ids[i]
 *   seq_ids   HOST   [n], strictly ascending
 *   sel_idx   DEVICE [n][k] int32 out, score order, unused slots -1
 *   sel_score DEVICE [n][k] fp32 out (may be NULL), unused slots -inf
 * Pure: mutates no pool state.  Runs on stream_fetch. */
int lsa_index_select(lsa_ctx* ctx, const void* h, const int32_t* seq_ids, int32_t n,
                     int32_t* sel_idx, float* sel_score);

/* S4-S5 for n sequences (ascending seq_ids): residency diff against the hot pool, page
 * allocation (never-used pages lowest index first, else LRU by (last_used, page), never a page
 * of any current or staged table; R11-R12), copy of every missing chunk cold -> hot on
 * stream_fetch, and staging of the next page table in ascending chunk id (R13).  The
 * staged table becomes current at the first lsa_step / lsa_decode_attention whose per-sequence
 * step counter is >= (counter at this call) + recall_lag, or at lsa_commit_tables.
 *   sel_idx DEVICE [n][k] int32 (-1 = unused slot), e.g. from lsa_index_select. */
int lsa_fetch_chunks(lsa_ctx* ctx, const int32_t* seq_ids, int32_t n, const int32_t* sel_idx);

/* Make every staged page table current now (stream_compute waits for its fetch). */
int lsa_commit_tables(lsa_ctx* ctx);

/* S6-S8 for all B sequences on stream_compute: (swap due tables, then) per head
 * softmax(sm_scale q K^T) V over HCA rows (+) rows [0, valid(c)) of every page of the current
 * table (+) window rows [0, w_len)  - one softmax over the union (R5).
 *   q   DEVICE [B][H][D]   out DEVICE [B][H][D] (dtype)   lse DEVICE [B][H] fp32 or NULL.
 * A sequence with no keys gets out = 0, lse = -inf.  Does not advance step counters. */
int lsa_decode_attention(lsa_ctx* ctx, const void* q, void* out, float* lse);

/* One decode step for all sequences:
 *  (a) staged tables that are due become current;  (b) sequences with step_b % tau == 0 run
 *  S1-S5 on stream_fetch with h;  (c) recall_lag == 0: their tables become current;
 *  (d) k_new/v_new (DEVICE [B][D], or both NULL) are written to ring slot w_head, so the new
 *  token attends to itself;  (e) attention + combine -> out;  (f) step_b += 1.
 *   h DEVICE [B][Dh] (row b = sequence b; only read at trigger steps; may be NULL otherwise). */
int lsa_step(lsa_ctx* ctx, const void* q, const void* h, const void* k_new, const void* v_new,
             void* out);

/* lsa_step with the fixed-shape part replayed from a CUDA graph ("CUDA-graph-compatible recall": the captured
 * graph holds only fixed-shape GPU work, Level-1 scoring and copying run out-of-graph in the side band).  On a step
 * without a trigger and without a table swap, the launches of (a)/(d)/(e) - S6, the window append, attention and
 * combine - are one captured graph, replayed as long as q, k_new, v_new, out and the split geometry stay the same
 * (the state they read - window fill, ring head, tables - lives in device records, so the same graph serves every
 * such step); any other step, or a context with profiling / fused merge enabled, runs exactly as lsa_step and
 * the graph is re-captured when the key changes.  Results are identical to lsa_step. */
int lsa_step_graph(lsa_ctx* ctx, const void* q, const void* h, const void* k_new, const void* v_new,
                   void* out);
/* captures / replays so far (HOST pointers, either may be NULL) */
int lsa_graph_stats(lsa_ctx* ctx, uint64_t* captures, uint64_t* replays);

/* lsa_step with HOST buffers.  Pinned + mapped inputs (e.g. torch pin_memory) are pulled over the host link by
 * one small kernel and a pinned `out` is written in place by S8; pageable buffers go through one packed
 * host->device copy and one device->host copy.  h is only read at trigger steps.  Blocks until the result
 * has landed.  Used for end-to-end timing.  Pinned buffers are recognised once per address (the device alias is
 * cached): a buffer passed here must stay registered, at that address, while the context lives. */
int lsa_step_host(lsa_ctx* ctx, const void* q, const void* h, const void* k_new,
                  const void* v_new, void* out);

/* lsa_step_host without the wait: the step is enqueued (inputs pulled from the pinned host buffers, result written to the
 * pinned `out` in place) and *ticket identifies it; lsa_host_wait(ctx, ticket) returns once that step's `out` has landed
 * (a completion word in pinned memory, written by the step's last CTA, is read - no stream synchronisation).  Steps
 * complete in order.  Up to 8 steps may be in flight: q, k_new, v_new, h and out of a step must stay untouched until its
 * ticket has been waited for.  Needs lsa_config.step_overlap = 1, B <= 4 on the tcgen05 path and pinned + mapped buffers;
 * otherwise the call completes synchronously and returns ticket 0 (which lsa_host_wait accepts). */
int lsa_step_host_async(lsa_ctx* ctx, const void* q, const void* h, const void* k_new, const void* v_new, void* out,
                        uint64_t* ticket);
int lsa_host_wait(lsa_ctx* ctx, uint64_t ticket);

/* ---- paper-exact Level-1 Memory Indexer (Eq.(1)-(5), l.142 Eq.(13))) --------
 * An alternative to lsa_index_select with the scorer the paper states: per indexer layer
 *   c = h W^DQ (1), q = c W^IUQ split into n_h heads of c_I (2), w = h W^w (3),
 *   I_s = sigmoid(sum_h w_h ReLU(q_h . K_s)) for every compressed entry s (4),
 * an entry is recalled if I_s >= threshold in ANY layer (5, 13); recall is page granular (l.185): chunk
 * c = entries [c*C, (c+1)*C) is selected iff one of its entries is, with score = max I over its entries and
 * layers, and if more than k (= K_max) chunks qualify the k best by (score desc, chunk id asc) are kept.
 * All weights are stored TRANSPOSED, [out][in] row-major, bf16.  Supported: dtype bf16, C = 128, c_I = 128,
 * n_h = 64 (else LSA_ERR_UNSUPPORTED); d_c % 8 == 0; 1..4 layers. */
typedef struct lsa_l1_layer {
  const void* W_dq;      /* DEVICE [d_c][Dh]          = (W^DQ)^T                                         */
  const void* W_iuq;     /* DEVICE [n_h*c_I][d_c]     = (W^IUQ)^T, head h = rows [h*c_I, (h+1)*c_I)      */
  const void* W_w;       /* DEVICE [n_h][Dh]          = (W^w)^T                                          */
} lsa_l1_layer;

typedef struct lsa_l1_config {
  uint32_t struct_size;  /* = sizeof(lsa_l1_config)                                                      */
  int32_t n_layers;      /* indexer layers whose sets are OR-ed (the paper uses 3: layers 10, 12, 20)    */
  int32_t d_c;           /* low-rank query dim (paper: r = 2048, l.153)                                  */
  int32_t c_I;           /* index-key dim per head                                                       */
  int32_t n_h;           /* indexer heads                                                                */
  float threshold;       /* 0 -> 0.5 (l.77); must be in (0, 1)                                           */
  lsa_l1_layer layers[4];
} lsa_l1_config;

/* index_k: HOST array of B * n_layers DEVICE pointers; index_k[b * n_layers + l] = compressed indexer keys
 * K^IComp of sequence b for layer l, [n_csa_b][c_I] bf16, caller-owned, must outlive the context (the
 * index-K of the Memory-Indexer layers stays on the GPU).  May be called once per context. */
int lsa_l1_init(lsa_ctx* ctx, const lsa_l1_config* cfg, const void* const* index_k);

/* Eq.(1)-(5), (13) for n sequences on stream_fetch; same argument conventions and output format as
 * lsa_index_select (sel_idx DEVICE [n][k], valid ids first in (score desc, id asc) order, then -1;
 * sel_score DEVICE [n][k] = I of the chunk, -inf padding, may be NULL), so the result feeds lsa_fetch_chunks. */
int lsa_l1_select(lsa_ctx* ctx, const void* h, const int32_t* seq_ids, int32_t n, int32_t* sel_idx, float* sel_score);

/* Which indexer lsa_step runs at trigger steps: BASELINE.json's dual encoder (S1-S3, default) or the
 * paper-exact Level-1 indexer (needs lsa_l1_init). */
enum lsa_indexer { LSA_INDEXER_DUAL_ENCODER = 0, LSA_INDEXER_LEVEL1 = 1 };
int lsa_set_indexer(lsa_ctx* ctx, int32_t indexer);

/* ---- Level 2: the native Lightning Indexer inside the resident set (Eq.(6), l.187) ----
 * Every decode step i, per sequence: Score_native(i, s) = sum_h w_{i,h} ReLU(q_{i,h} . K_s^IComp) - Eq.(4) without
 * the sigmoid (l.75) - for the entries s of C_t^MemComp = the valid rows of the pages of the CURRENT page table;
 * the first min(k2, |C_t^MemComp|) entries by (score descending, entry id s = chunk*C + row ascending) form
 * C_i^CoreComp, and core attention runs over HCA (+) C_i^CoreComp (+) window (l.85; HCA per BJ north_star).
 * Supported: dtype bf16, C = 128, c_I = 128, n_h = 64, tcgen05 attention path, 1 <= k2 <= 4096 (else
 * LSA_ERR_UNSUPPORTED / INVALID_ARG). */
typedef struct lsa_l2_config {
  uint32_t struct_size;  /* = sizeof(lsa_l2_config)                                                      */
  int32_t c_I;           /* index-key dim per head                                                       */
  int32_t n_h;           /* indexer heads                                                                */
  int32_t k2;            /* Top-k entries kept per sequence and step (Eq.(6))                            */
} lsa_l2_config;

/* index_k: HOST array of B DEVICE pointers; index_k[b] = this layer's compressed indexer keys of sequence b,
 * [n_csa_b][c_I] bf16, caller-owned, must outlive the context.  May be called once per context. */
int lsa_l2_init(lsa_ctx* ctx, const lsa_l2_config* cfg, const void* const* index_k);

/* Eq.(6) for all B sequences on stream_compute: staged tables that are due become current first (S6), then the
 * entries of the current tables are scored and the Top-k2 marked.  The selection applies to the NEXT
 * lsa_decode_attention call only (one-shot), which then attends HCA (+) the marked rows (+) window; an lsa_step
 * in between discards it (a step may change the tables: use lsa_step_l2).
 *   q_idx DEVICE [B][n_h][c_I] bf16   w_idx DEVICE [B][n_h] fp32 (both read on stream_compute)
 *   sel_entries DEVICE [B][k2] int32 or NULL: entry ids in (score desc, id asc) order, then -1
 *   sel_score   DEVICE [B][k2] fp32  or NULL: their native scores, -inf padding */
int lsa_l2_select(lsa_ctx* ctx, const void* q_idx, const float* w_idx, int32_t* sel_entries, float* sel_score);

/* Blocking read-back of the row mask the last lsa_l2_select / lsa_step_l2 wrote for sequence seq:
 * words HOST [k][4] uint32, bit r of word [j][r / 32] = row r of the j-th page of the current table is selected. */
int lsa_l2_get_mask(lsa_ctx* ctx, int32_t seq, uint32_t* words);

/* lsa_step with Level 2 between (d) and (e): the step's attention runs over HCA (+) the Top-k2 entries of the
 * current tables (+) window.  Other arguments and the step order as lsa_step. */
int lsa_step_l2(lsa_ctx* ctx, const void* q, const void* h, const void* k_new, const void* v_new,
                const void* q_idx, const float* w_idx, void* out);

/* S1-S3 (as lsa_index_select: P:61-65, P:71-79 in BASELINE's dual-encoder form, R1-R3, R14-R16) for callers that may
 * not allocate: code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  No context; the scratch
 * between the three kernels (z, the scores, the per-sequence records) is a file-scope device array of the library
 * (~641 KiB, held by every GPU that loads the library until exit) and the call allocates nothing - no cudaMalloc /
 * cudaFree, no memcpy: it only enqueues four kernels on `stream` (a cudaStream_t of the CURRENT device).
 *   dtype lsa_dtype; W_q DEVICE [E][Dh]; h DEVICE [n][Dh]; chunk_emb HOST [n] of DEVICE pointers [n_chunks[i]][E];
 *   n_chunks HOST [n]; sel_idx DEVICE [n][k] int32 (unused slots -1); sel_score DEVICE [n][k] fp32 or NULL.
 * Limits (the array's size): n <= 8, E <= 4096 (multiple of 8), n_chunks[i] <= 16384, k <= 1024, Dh % 8 == 0; anything
 * beyond is LSA_ERR_INVALID_ARG (text: lsa_last_error(NULL)) and nothing is enqueued.
 * The array is shared by every call on the device and keeps the last call's contents; nothing in it needs to start at
 * zero.  Calls that OVERLAP on the GPU (different streams without an ordering between them) race on it: keep calls on one
 * stream or order them with events.  Results are identical to lsa_index_select on the same inputs. */
int lsa_index_select_static(int32_t dtype, const void* W_q, const void* h, const void* const* chunk_emb,
                            const int32_t* n_chunks, int32_t n, int32_t E, int32_t Dh, int32_t k, int32_t* sel_idx,
                            float* sel_score, void* stream);

/* NEXT-4 (first half; P:179, P:199 VRAM -> DRAM): KV export into the cold pool.  Copies n_chunks page images
 * src DEVICE [n_chunks][2][C][D] (dtype) into chunks [first_chunk, first_chunk + n_chunks) of sequence seq's pinned-host
 * cold pool (which must be writable), by a device kernel over the mapped pool on stream_fetch - ordered before every
 * later trigger's fetch.  Meant for admission, before the chunks are first selected: a chunk that is already resident
 * keeps its old hot copy until it is evicted.  Enqueues and returns; bit-exact. */
int lsa_export_chunks(lsa_ctx* ctx, int32_t seq, int32_t first_chunk, int32_t n_chunks, const void* src);

/* NEXT-4 (second half; "all actively decoded tokens' CSA chunks" are an always-resident tier; P:179 VRAM -> DRAM;
 * DESIGN.md R29-R33): hand over already-compressed entries of the tokens decoded since the last call - at most one CSA
 * entry and one HCA entry per listed sequence - BEFORE the lsa_step that first attends them.  The compressors themselves
 * belong to the model; the library takes their output, as it takes k_new / v_new.
 *   seq_ids HOST [n] strictly ascending; csa_k / csa_v DEVICE [n][D] (both or neither); hca_k / hca_v DEVICE [n][D] (both
 *   or neither); emb_rows DEVICE [n][E]: row i is read only if sequence seq_ids[i]'s CSA entry completes a chunk (it is
 *   that chunk's embedding, L2-normalised by the producer) - may be NULL when no listed sequence completes one.
 * Effect per sequence, in stream order on stream_compute: the HCA entry becomes row n_hca of hca_k / hca_v (n_hca += 1);
 * the CSA entry becomes row n_csa % C of the TAIL chunk n_csa / C, which lives in a reserved page of the hot pool (the last
 * 2 B pages: page hot_pages - 2 B + 2 b + (chunk % 2); the LRU manages the pages before them) and is attended with its valid
 * rows through an entry at the end of the page table (n_csa += 1).  When the entry completes the chunk: emb row -> chunk_emb,
 * the page image is exported to the cold pool (stream_fetch), the chunk becomes a candidate of the indexer from the next
 * trigger on, and it stays attended through the table until a table becomes current whose trigger saw it as a candidate;
 * from then on it is attended iff recalled.  Two of the k table slots are the tier's: at most k - 2 chunks are recalled.
 * Only the dual-encoder indexer supports growth (Level 1 / Level 2 contexts: LSA_ERR_UNSUPPORTED).
 * Errors: INVALID_ARG (ids, null pairs, capacity exceeded, missing emb_rows at a completion), STATE (the context was not
 * created with cap_csa > 0; or a third chunk would enter the tier before the oldest one left it - needs the table of a
 * trigger that saw it, i.e. chunks must not complete faster than every tau + recall_lag steps).  Enqueues and returns. */
int lsa_append_compressed(lsa_ctx* ctx, const int32_t* seq_ids, int32_t n, const void* csa_k, const void* csa_v,
                          const void* hca_k, const void* hca_v, const void* emb_rows);

/* Replace the embedding table pointer of one sequence (DEVICE [n_chunks][E]). */
int lsa_set_chunk_emb(lsa_ctx* ctx, int32_t seq, const void* chunk_emb);

/* Blocking read-back of a page table.  which: 0 = current, 1 = staged.  chunk_idx/page HOST [k].
 * *n = entries (0 if none / nothing staged).  Entries are in ascending chunk id. */
int lsa_get_page_table(lsa_ctx* ctx, int32_t seq, int32_t which, int32_t* chunk_idx,
                       int32_t* page, int32_t* n);

/* Blocking: page_of[seq][0..n_chunks) -> HOST int32 (-1 = cold). */
int lsa_get_residency(lsa_ctx* ctx, int32_t seq, int32_t* page_of);

int lsa_get_stats(lsa_ctx* ctx, lsa_stats* out); /* blocking */

/* Per-phase device timing with CUDA events recorded on the launching stream (off by default;
 * each enabled launch costs two event records).  capacity = event pairs kept per phase; 0 disables.
 * lsa_profile_read blocks, returns the summed milliseconds and launch counts per phase since the
 * last read and rearms.  Phases: */
enum lsa_phase { LSA_PH_PRESTEP = 0, LSA_PH_ATTENTION = 1, LSA_PH_COMBINE = 2, LSA_PH_INDEX = 3,
                 LSA_PH_RESIDENCY = 4, LSA_PH_FETCH = 5,
                 LSA_PH_ATTENTION_DEV = 6, /* tcgen05 attention kernel's own working time by %globaltimer: first CTA
                                              past its launch dependency -> last CTA done (no event in the way) */
                 LSA_PH_COUNT = 7 };
int lsa_profile_enable(lsa_ctx* ctx, int32_t capacity);
int lsa_profile_read(lsa_ctx* ctx, double* ms_sum /* HOST [LSA_PH_COUNT] */, int64_t* count /* HOST [LSA_PH_COUNT] */);

/* Per-CTA timeline of the small-batch attention launches (B <= 4 with lsa_config.step_overlap; DESIGN.md 7.3 explains what
 * it showed: the step time of that path is the CTAs' summed residence / SM count, not bytes / bandwidth).
 * lsa_timeline_enable(ctx, 1) allocates, once, a device ring of LSA_TL_LAUNCHES launch records and makes every small-batch
 * launch of the context stamp %globaltimer (nanoseconds) at the points below, one row per CTA, into record (launch number mod
 * LSA_TL_LAUNCHES); (ctx, 0) stops the stamping (the ring is kept).  Off, the launches run a kernel without any of it.
 * lsa_timeline_read blocks on both streams, copies the ring to HOST dst[LSA_TL_LAUNCHES][LSA_TL_CTAS][LSA_TL_EVENTS]
 * (uint64; rows of CTAs a launch did not have, and records never written, are 0) and stores the number of launches
 * stamped so far in *n_launches (may be NULL).  Launches of more than LSA_TL_CTAS CTAs are not stamped.
 * Errors: LSA_ERR_STATE (null ctx), LSA_ERR_INVALID_ARG (null dst), LSA_ERR_OOM, LSA_ERR_CUDA. */
#define LSA_TL_LAUNCHES 16
#define LSA_TL_CTAS 160
#define LSA_TL_EVENTS 12
enum lsa_tl_event {
  LSA_TL_ENTRY = 0,        /* the CTA's barriers are initialised, its roles start                                      */
  LSA_TL_SETUP = 1,        /* warp 0 has the piece boundaries, the table entries and the counters of its range         */
  LSA_TL_FIRST_S = 2,      /* Q and the first K sub-tile have landed, the first S^T = K Q^T has been issued             */
  LSA_TL_LAST_PV = 3,      /* the last O^T += V^T P^T has been issued (every K / V row of the piece has landed)         */
  LSA_TL_EPILOGUE = 4,     /* the partial (O^T, l, m) of the last piece has been stored                                 */
  LSA_TL_ARRIVED = 5,      /* the CTA has published its partials and taken its arrival number                          */
  LSA_TL_ALL_ARRIVED = 6,  /* mergers only (0 for a CTA that left): every CTA of the launch has arrived                 */
  LSA_TL_MERGED = 7,       /* mergers only: this CTA's share of `out` has been written                                  */
  LSA_TL_EXIT = 8,         /* the CTA returns                                                                          */
  LSA_TL_SMID = 9,         /* %smid, not a time                                                                        */
  LSA_TL_NCTAS = 10,       /* CTAs of the launch, not a time                                                           */
  LSA_TL_SEQ = 11          /* number of the launch among the context's stamped launches, not a time                    */
};
int lsa_timeline_enable(lsa_ctx* ctx, int32_t on);
int lsa_timeline_read(lsa_ctx* ctx, uint64_t* dst /* HOST */, uint64_t* n_launches /* HOST, may be NULL */);
int lsa_get_step(lsa_ctx* ctx, int32_t seq, int64_t* step);
int lsa_sync(lsa_ctx* ctx);                      /* waits for both streams, reports device errors */
const char* lsa_last_error(lsa_ctx* ctx);        /* ctx may be NULL: last init error             */
void lsa_destroy(lsa_ctx* ctx);
int lsa_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LSA_H_ */
