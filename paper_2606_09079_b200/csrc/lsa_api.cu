// lsa_api.cu - the C ABI of liblsa (include/lsa.h): host-side orchestration only.
// Every step of the path runs in the kernels of lsa_index.cu / lsa_residency.cu /
// lsa_attn_simt.cu / lsa_attn_tc.cu; this file validates arguments, keeps deterministic host
// mirrors of the per-sequence counters (so no call ever waits for the device), orders the two
// streams with events and launches.  Step order: DESIGN.md "Step order".
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include "../../include/lsa.h"
#include "lsa_attn_tc.h"
#include "lsa_kernels.h"
#include "lsa_l1.h"
#include "lsa_l2.h"

using namespace lsa;

static thread_local std::string g_init_error;

struct lsa_ctx {
  lsa_config cfg{};
  int B = 0, k = 0;
  float sm_scale = 0.f;
  long long page_bytes = 0;
  long long cold_page_bytes = 0;       // = page_bytes, or half of it with FP8 cold pages (lsa_config.cold_format)
  int elem = 0;
  cudaStream_t sc = nullptr, sf = nullptr;
  cudaEvent_t ev_fetch = nullptr, ev_compute = nullptr;
  int n_sms = 0;
  // device state
  SeqDev* d_seqs = nullptr;
  PoolDev pool{};
  std::vector<void*> owned;          // cudaMalloc'ed blocks to free
  std::vector<SeqDev> seq_host;      // immutable fields (host copy)
  int total_chunks = 0, n_chunks_max = 0;
  // host mirrors (deterministic: advanced by the same rules the kernels apply)
  std::vector<long long> step, visible_at;
  std::vector<char> pending;
  std::vector<int> k_eff;
  // mirrors the small-batch attention path passes by value (lsa_attn_tc_small.cuh): attended table buffer, entries per
  // buffer (-1: only the device knows, the selection was given on the device), ring head, appends so far
  std::vector<int> cur_buf, w_head;
  std::vector<int> n_tbl[2];
  std::vector<unsigned int> app_count;
  bool no_small = false;               // lsa_step_graph: the captured launch must read the device records
  bool serialize_next = false;         // something the next attention launch reads was enqueued on another stream
  bool inputs_from_prev_kernel = false;// lsa_step_host: q / k_new / v_new come from the gather kernel just enqueued
  unsigned int* host_flag = nullptr;   // lsa_step_host: pinned completion word (host address / device alias below)
  unsigned int* host_flag_dev = nullptr;
  unsigned int host_flag_seq = 0;
  bool host_flag_armed = false;        // the launch just enqueued will write host_flag_seq to the flag
  bool next_alone = false;             // the caller will block on the step being enqueued
  int qtower_tc = 1;                   // S1 on tensor cores when 8..16 sequences fire together
  unsigned int* gather_ctr = nullptr;  // DEVICE: finished blocks of the gather kernels of lsa_step_host_async
  unsigned int gather_total = 0;       // as enqueued
  bool inputs_by_counter = false;      // the next attention launch waits for gather_total instead of for the stream
  // index scratch
  float* d_z = nullptr;
  float* d_scores = nullptr;
  int32_t* d_sel = nullptr;
  // attention
  int attn_impl = LSA_ATTN_SIMT;
  AttnGeom geom{};
  float* part_o = nullptr;
  float* part_ml = nullptr;
  int fetch_ctas = 0;
  TcPlan* tc = nullptr;
  L1Plan* l1 = nullptr;               // paper-exact Level-1 indexer (lsa_l1_init)
  float l1_threshold = 0.5f;
  L2Plan* l2 = nullptr;               // Level 2 (lsa_l2_init)
  bool l2_armed = false;              // a Level-2 selection waits for the next attention launch
  // lsa_step_graph: the captured non-trigger step and the key it is valid for
  cudaGraphExec_t sg_exec = nullptr;
  const void *sg_q = nullptr, *sg_kn = nullptr, *sg_vn = nullptr, *sg_out = nullptr;
  long long sg_tiles = -1;
  unsigned long long sg_launches = 0, sg_captures = 0, sg_replays = 0;
  int indexer = 0;                     // lsa_indexer used by lsa_step at trigger steps
  // host-buffer staging (lsa_step_host)
  void *st_q = nullptr, *st_out = nullptr, *st_pin = nullptr;
  unsigned long long st_calls = 0;                  // lsa_step_host calls so far: image st_calls % kStRing is next
  uint64_t st_ticket[8] = {0, 0, 0, 0, 0, 0, 0, 0}; // ticket of the step that used each image last (0: none / complete)
  const void* out_host_cached = nullptr;
  std::vector<std::pair<const void*, void*>> alias_cache;   // host pointer -> device alias (or null)
  void* out_dev_alias = nullptr;
  // optional per-phase event timing
  int prof_cap = 0;
  std::vector<cudaEvent_t> prof_ev[LSA_PH_COUNT];   // 2*cap events per phase
  int prof_n[LSA_PH_COUNT] = {0, 0, 0, 0, 0, 0, 0};
  unsigned long long* d_tl = nullptr;               // lsa_timeline_enable: [LSA_TL_LAUNCHES][LSA_TL_CTAS][LSA_TL_EVENTS]
  bool tl_on = false;
  unsigned long long tl_seq = 0;                    // launches stamped so far
  unsigned long long* d_ktime = nullptr;            // [prof_cap][2] attention-kernel globaltimer stamps
  int ktime_cap = 0;
  // bookkeeping
  unsigned long long n_steps = 0, attn_launches = 0, index_launches = 0;
  // NEXT-4 growth (lsa_append_compressed; DESIGN R29-R33)
  bool growth = false;
  int k_sel = 0;                       // recalled chunks per table at most: k, or k - 2 when the context grows
  int P_lru = 0;                       // pages the LRU manages: hot_pages, or hot_pages - 2 B
  std::vector<long long> cap_csa;
  std::vector<int> ncand_cur, ncand_nxt;   // candidates seen by the trigger of the current / the staged table (host mirror)
  cudaEvent_t ev_roll = nullptr;       // fetch-stream position a roll (chunk completed / new tail) must wait for
  unsigned long long csa_appended = 0, hca_appended = 0, chunks_exported = 0;
  std::vector<unsigned int> grow_count;    // lsa_append_compressed calls per sequence (mirror of SeqDev::grow_epoch as enqueued)
  bool grow_wait_next = false;         // an append kernel was enqueued beside the previous attention launch
  int last_attn_ctas = 0;
  std::string err;
};

#define LSA_FAIL(ctx, code, ...)                          \
  do {                                                    \
    char _b[512];                                         \
    snprintf(_b, sizeof(_b), __VA_ARGS__);                \
    if (ctx) (ctx)->err = _b; else g_init_error = _b;     \
    return (code);                                        \
  } while (0)

#define LSA_CUDA(ctx, expr)                                                                   \
  do {                                                                                        \
    cudaError_t _e = (expr);                                                                  \
    if (_e != cudaSuccess)                                                                    \
      LSA_FAIL(ctx, LSA_ERR_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
  } while (0)

// Records a start event now and an end event at scope exit on `st` when profiling is enabled.
struct ProfScope {
  lsa_ctx* c; int ph; cudaStream_t st; bool on;
  ProfScope(lsa_ctx* c_, int ph_, cudaStream_t st_) : c(c_), ph(ph_), st(st_), on(false) {
    if (c->prof_cap > 0 && c->prof_n[ph] < c->prof_cap) {
      on = true;
      cudaEventRecord(c->prof_ev[ph][2 * c->prof_n[ph]], st);
    }
  }
  ~ProfScope() {
    if (on) {
      cudaEventRecord(c->prof_ev[ph][2 * c->prof_n[ph] + 1], st);
      c->prof_n[ph] += 1;
    }
  }
};

template <typename T>
static int dev_alloc(lsa_ctx* c, T** p, size_t n, bool zero = true) {
  void* q = nullptr;
  size_t bytes = std::max<size_t>(n, 1) * sizeof(T);
  cudaError_t e = cudaMalloc(&q, bytes);
  if (e != cudaSuccess) LSA_FAIL(c, LSA_ERR_OOM, "cudaMalloc(%zu) failed: %s", bytes, cudaGetErrorString(e));
  if (zero) {
    e = cudaMemset(q, 0, bytes);
    if (e != cudaSuccess) LSA_FAIL(c, LSA_ERR_CUDA, "cudaMemset failed: %s", cudaGetErrorString(e));
  }
  c->owned.push_back(q);
  *p = reinterpret_cast<T*>(q);
  return LSA_OK;
}

extern "C" int lsa_version(void) { return LSA_VERSION; }

extern "C" const char* lsa_last_error(lsa_ctx* ctx) { return ctx ? ctx->err.c_str() : g_init_error.c_str(); }

extern "C" void lsa_destroy(lsa_ctx* ctx) {
  if (!ctx) return;
  if (ctx->sc) cudaStreamSynchronize(ctx->sc);
  if (ctx->sf) cudaStreamSynchronize(ctx->sf);
  if (ctx->tc) tc_destroy(ctx->tc);
  if (ctx->l1) l1_destroy(ctx->l1);
  if (ctx->l2) l2_destroy(ctx->l2);
  if (ctx->sg_exec) cudaGraphExecDestroy(ctx->sg_exec);
  if (ctx->st_pin) cudaFreeHost(ctx->st_pin);
  if (ctx->host_flag) cudaFreeHost(ctx->host_flag);
  for (void* p : ctx->owned) cudaFree(p);
  if (ctx->ev_fetch) cudaEventDestroy(ctx->ev_fetch);
  if (ctx->ev_compute) cudaEventDestroy(ctx->ev_compute);
  if (ctx->ev_roll) cudaEventDestroy(ctx->ev_roll);
  for (auto& v : ctx->prof_ev)
    for (cudaEvent_t e : v) cudaEventDestroy(e);
  delete ctx;
}

static int init_impl(lsa_ctx* c, const lsa_config* cfg, const lsa_seq_desc* seqs) {
  c->cfg = *cfg;
  const int B = cfg->B, H = cfg->H, D = cfg->D, C = cfg->C, k = cfg->k;
  c->B = B;
  c->k = k;
  c->elem = cfg->dtype == LSA_F32 ? 4 : 2;
  c->page_bytes = 2ll * C * D * c->elem;
  const bool fp8_cold = cfg->cold_format == LSA_COLD_FP8_E4M3;
  c->cold_page_bytes = fp8_cold ? 2ll * C * D : c->page_bytes;
  if (fp8_cold && (cfg->dtype != LSA_BF16 || (C * (long long)D) % 16))
    LSA_FAIL(c, LSA_ERR_UNSUPPORTED, "FP8 cold pages need dtype = LSA_BF16 and C * D a multiple of 16");
  c->sm_scale = cfg->sm_scale > 0.f ? cfg->sm_scale : 1.0f / std::sqrt((float)D);
  c->sc = (cudaStream_t)cfg->stream_compute;
  c->sf = (cudaStream_t)cfg->stream_fetch;
  int dev = 0;
  LSA_CUDA(c, cudaGetDevice(&dev));
  LSA_CUDA(c, cudaDeviceGetAttribute(&c->n_sms, cudaDevAttrMultiProcessorCount, dev));
  LSA_CUDA(c, cudaEventCreateWithFlags(&c->ev_fetch, cudaEventDisableTiming));
  LSA_CUDA(c, cudaEventCreateWithFlags(&c->ev_compute, cudaEventDisableTiming));

  c->seq_host.resize(B);
  c->step.resize(B);
  c->visible_at.assign(B, 0);
  c->pending.assign(B, 0);
  c->k_eff.resize(B);
  c->cur_buf.assign(B, 0);
  c->w_head.assign(B, 0);
  c->n_tbl[0].assign(B, 0);
  c->n_tbl[1].assign(B, 0);
  c->app_count.assign(B, 0u);
  c->growth = seqs[0].cap_csa > 0;
  c->k_sel = c->growth ? k - 2 : k;
  c->P_lru = (int)cfg->hot_pages - (c->growth ? 2 * B : 0);
  c->cap_csa.assign(B, 0);
  c->ncand_cur.assign(B, 0);
  c->ncand_nxt.assign(B, 0);
  c->grow_count.assign(B, 0u);
  if (c->growth && k < 3) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "a growing context needs k >= 3 (two table slots belong to the decode tier)");
  if (c->growth) LSA_CUDA(c, cudaEventCreateWithFlags(&c->ev_roll, cudaEventDisableTiming));
  long long sum_k = 0, total_keys_max = 0, n_keys_max = 0;
  for (int b = 0; b < B; ++b) {
    const lsa_seq_desc& s = seqs[b];
    if (fp8_cold && s.n_csa > 0 && !s.cold_scale) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq %d: cold_scale is NULL with FP8 cold pages", b);
    if (fp8_cold && s.cap_csa > 0)
      LSA_FAIL(c, LSA_ERR_UNSUPPORTED, "a growing compressed history (cap_csa) with FP8 cold pages is not built");
    if ((s.cap_csa > 0) != c->growth) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq %d: either every sequence grows (cap_csa > 0) or none", b);
    if (c->growth && (s.cap_csa < s.n_csa || s.cap_hca < s.n_hca || s.cap_hca > (1ll << 30)))
      LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq %d: cap_csa / cap_hca below n_csa / n_hca", b);
    if (s.n_csa < 0 || s.n_hca < 0 || s.w_len < 0 || s.w_len > cfg->W || s.w_head < 0 || s.w_head >= std::max(cfg->W, 1))
      LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq %d: bad n_csa/n_hca/w_len/w_head", b);
    // candidates of the indexer: every chunk (a partial last one included, R22); for a growing sequence the FULL chunks
    // only - the partial one is the tail of the decode tier (R30).  cap_chunks: what the caller's arrays can hold.
    const long long cap_chunks = c->growth ? (s.cap_csa + C - 1) / C : (s.n_csa + C - 1) / C;
    const long long n_chunks = c->growth ? s.n_csa / C : cap_chunks;
    c->cap_csa[b] = c->growth ? s.cap_csa : s.n_csa;
    if (cap_chunks > 0 && (!s.cold_csa || !s.chunk_emb)) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq %d: null cold_csa/chunk_emb", b);
    if (s.n_hca > 0 && (!s.hca_k || !s.hca_v)) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq %d: null hca_k/hca_v", b);
    if (cfg->W > 0 && (!s.win_k || !s.win_v)) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq %d: null win_k/win_v", b);
    SeqDev d{};
    if (cap_chunks > 0) {
      cudaPointerAttributes at{};
      cudaError_t e = cudaPointerGetAttributes(&at, s.cold_csa);
      if (e != cudaSuccess || at.type != cudaMemoryTypeHost || !at.devicePointer) {
        cudaGetLastError();
        LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq %d: cold_csa must be pinned (page-locked, mapped) host memory", b);
      }
      d.cold = at.devicePointer;
    }
    d.emb = s.chunk_emb;
    d.cold_scale = fp8_cold ? static_cast<const float*>(s.cold_scale) : nullptr;
    d.hca_k = s.hca_k;
    d.hca_v = s.hca_v;
    d.win_k = s.win_k;
    d.win_v = s.win_v;
    d.n_csa = s.n_csa;
    d.n_chunks = (int)n_chunks;
    d.n_hca = (int)s.n_hca;
    d.cap_hca = c->growth ? (int)s.cap_hca : (int)s.n_hca;
    d.tier_page0 = c->growth ? c->P_lru + 2 * b : -1;
    d.k_eff = (int)std::min<long long>(c->k_sel, n_chunks);
    d.page_of_off = c->total_chunks;
    d.w_len = s.w_len;
    d.w_head = s.w_head;
    c->ncand_cur[b] = c->ncand_nxt[b] = (int)n_chunks;
    c->total_chunks += (int)cap_chunks;
    c->n_chunks_max = std::max(c->n_chunks_max, (int)cap_chunks);
    c->seq_host[b] = d;
    c->step[b] = s.step0;
    c->k_eff[b] = d.k_eff;
    c->w_head[b] = s.w_head;
    sum_k += std::min<long long>(c->k_sel, cap_chunks);
    const long long nk = d.cap_hca + (long long)(c->growth ? k : d.k_eff) * C + cfg->W;
    total_keys_max += nk;
    n_keys_max = std::max(n_keys_max, nk);
  }
  if (c->P_lru < 2 * sum_k)
    LSA_FAIL(c, LSA_ERR_INVALID_ARG, "hot_pages=%lld%s < 2*sum_b min(k,n_chunks_b)=%lld (current + staged tables are pinned)",
             (long long)c->P_lru, c->growth ? " (after the 2 B pages of the decode tier)" : "", 2 * sum_k);
  if (cfg->hot_pages > (1ll << kPageBits)) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "hot_pages > 2^%d", kPageBits);

  // ---- device state ----
  const int P = (int)cfg->hot_pages;
  int rc;
  if ((rc = dev_alloc(c, &c->d_seqs, B))) return rc;
  LSA_CUDA(c, cudaMemcpy(c->d_seqs, c->seq_host.data(), sizeof(SeqDev) * B, cudaMemcpyHostToDevice));
  if ((rc = dev_alloc(c, &c->pool.page_of, c->total_chunks, false))) return rc;
  LSA_CUDA(c, cudaMemset(c->pool.page_of, 0xff, sizeof(int) * std::max(c->total_chunks, 1)));
  if ((rc = dev_alloc(c, &c->pool.owner_seq, P, false))) return rc;
  LSA_CUDA(c, cudaMemset(c->pool.owner_seq, 0xff, sizeof(int) * P));
  if ((rc = dev_alloc(c, &c->pool.owner_chunk, P))) return rc;
  if ((rc = dev_alloc(c, &c->pool.last_used, P))) return rc;
  if ((rc = dev_alloc(c, &c->pool.pin_mark, P))) return rc;
  if ((rc = dev_alloc(c, &c->pool.tbl_chunk, (size_t)B * 2 * k))) return rc;
  if ((rc = dev_alloc(c, &c->pool.tbl_page, (size_t)B * 2 * k))) return rc;
  if ((rc = dev_alloc(c, &c->pool.fetch_src, (size_t)B * k))) return rc;
  if ((rc = dev_alloc(c, &c->pool.fetch_page, (size_t)B * k))) return rc;
  if (fp8_cold && (rc = dev_alloc(c, &c->pool.fetch_scale, (size_t)B * k))) return rc;
  if ((rc = dev_alloc(c, &c->pool.counters, 8))) return rc;
  if ((rc = dev_alloc(c, &c->pool.epoch, 1))) return rc;
  if (c->growth) {
    // decode tier (DESIGN R30, R32): HCA rows not in use yet must be finite (the tensor-core path multiplies them by
    // P = 0); a partial last chunk of the prompt is the first tail chunk - its rows are copied from the cold pool into the
    // sequence's reserved page and listed in the (otherwise empty) attended table
    for (int b = 0; b < B; ++b) {
      SeqDev& d = c->seq_host[b];
      if (d.cap_hca > d.n_hca) {
        const size_t off = (size_t)d.n_hca * D * c->elem, nb = (size_t)(d.cap_hca - d.n_hca) * D * c->elem;
        LSA_CUDA(c, cudaMemset((char*)const_cast<void*>(d.hca_k) + off, 0, nb));
        LSA_CUDA(c, cudaMemset((char*)const_cast<void*>(d.hca_v) + off, 0, nb));
      }
      if (d.n_csa % C) {
        const int ch = (int)(d.n_csa / C), page = d.tier_page0 + (ch & 1);
        LSA_CUDA(c, cudaMemcpy((char*)cfg->hot_pool + (long long)page * c->page_bytes,
                               (const char*)seqs[b].cold_csa + (long long)ch * c->page_bytes, (size_t)c->page_bytes, cudaMemcpyHostToDevice));
        LSA_CUDA(c, cudaMemcpy(c->pool.tbl_chunk + (size_t)b * 2 * k, &ch, sizeof(int), cudaMemcpyHostToDevice));
        LSA_CUDA(c, cudaMemcpy(c->pool.tbl_page + (size_t)b * 2 * k, &page, sizeof(int), cudaMemcpyHostToDevice));
        d.n_tbl[0] = 1;
        c->n_tbl[0][b] = 1;
      }
    }
    LSA_CUDA(c, cudaMemcpy(c->d_seqs, c->seq_host.data(), sizeof(SeqDev) * B, cudaMemcpyHostToDevice));
  }
  // ---- index scratch ----
  if ((rc = dev_alloc(c, &c->d_z, (size_t)std::max(B, 16 * std::max(1, cfg->Dh / 512)) * cfg->E))) return rc;   // or [Dh/512][16][E] partials
  if ((rc = dev_alloc(c, &c->d_scores, (size_t)B * std::max(c->n_chunks_max, 1)))) return rc;
  if ((rc = dev_alloc(c, &c->d_sel, (size_t)B * k))) return rc;

  // ---- attention implementation + split geometry ----
  int impl = cfg->attn_impl;
  const bool tc_ok = tc_supported(cfg->dtype, H, D, C);
  if (impl == LSA_ATTN_AUTO) impl = tc_ok ? LSA_ATTN_TCGEN05 : LSA_ATTN_SIMT;
  if (impl == LSA_ATTN_TCGEN05 && !tc_ok)
    LSA_FAIL(c, LSA_ERR_UNSUPPORTED, "tcgen05 attention needs bf16, H=64, D=512, C=128 (got dtype=%d H=%d D=%d C=%d)", cfg->dtype, H, D, C);
  if (impl == LSA_ATTN_SIMT && !simt_supported(cfg->dtype, H, D))
    LSA_FAIL(c, LSA_ERR_UNSUPPORTED, "no SIMT attention kernel compiled for H=%d D=%d", H, D);
  c->attn_impl = impl;
  if (impl == LSA_ATTN_SIMT) {
    int occ = 0;
    LSA_CUDA(c, simt_max_ctas_per_sm(cfg->dtype, H, D, k, &occ));
    if (occ < 1) LSA_FAIL(c, LSA_ERR_UNSUPPORTED, "SIMT attention kernel does not fit on an SM for H=%d D=%d", H, D);
    const int target = cfg->max_ctas > 0 ? cfg->max_ctas : c->n_sms * occ;
    const int tile = simt_tile_keys();
    long long kpc = (total_keys_max + target - 1) / std::max(target, 1);
    kpc = std::max<long long>(tile, (kpc + tile - 1) / tile * tile);
    c->geom.keys_per_cta = (int)kpc;
    c->geom.s_max = (int)std::max<long long>(1, (n_keys_max + kpc - 1) / kpc);
    if ((rc = dev_alloc(c, &c->part_o, (size_t)B * c->geom.s_max * H * D, false))) return rc;
    if ((rc = dev_alloc(c, &c->part_ml, (size_t)B * c->geom.s_max * H * 2, false))) return rc;
  } else {
    std::vector<long long> nk(B);
    for (int b = 0; b < B; ++b) nk[b] = c->seq_host[b].cap_hca + (long long)(c->growth ? k : c->k_eff[b]) * C + cfg->W;
    TcInit ti{};
    ti.B = B; ti.k = k; ti.W = cfg->W; ti.P = P; ti.n_sms = c->n_sms; ti.max_ctas = cfg->max_ctas;
    ti.fuse_combine = cfg->merge_mode == LSA_MERGE_FUSED ? 1 : 0;
    ti.hot_pool = cfg->hot_pool; ti.seq_host = c->seq_host.data(); ti.d_seqs = c->d_seqs; ti.pool = c->pool;
    ti.sm_scale = c->sm_scale; ti.stream = c->sc;
    std::string msg;
    int trc = tc_create(ti, &c->tc, &msg);
    if (trc != 0) LSA_FAIL(c, trc, "tcgen05 attention init failed: %s", msg.c_str());
  }
  c->fetch_ctas = std::max(8, std::min(64, c->n_sms / 2));
  LSA_CUDA(c, cudaDeviceSynchronize());
  return LSA_OK;
}

extern "C" int lsa_init_pools(const lsa_config* cfg, const lsa_seq_desc* seqs, lsa_ctx** out) {
  if (!cfg || !seqs || !out) LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "null argument");
  *out = nullptr;
  if (cfg->struct_size != sizeof(lsa_config))
    LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "lsa_config.struct_size=%u, library expects %zu", cfg->struct_size, sizeof(lsa_config));
  if (cfg->dtype != LSA_F32 && cfg->dtype != LSA_BF16) LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "bad dtype %d", cfg->dtype);
  if (cfg->B < 1 || cfg->B > 1024 || cfg->H < 1 || cfg->D < 1 || cfg->C < 1 || cfg->W < 0 || cfg->Dh < 1 || cfg->E < 1)
    LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "B (1..1024), H, D, C, Dh, E must be >= 1 and W >= 0");
  if (cfg->k < 1 || cfg->k > kMaxK) LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "k must be in [1, %d]", kMaxK);
  if (cfg->tau < 1) LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "tau must be >= 1");
  // one staged table per sequence: it must have become current before the next trigger stages another
  if (cfg->recall_lag < 0 || (cfg->recall_lag > 1 && cfg->recall_lag >= cfg->tau))
    LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "recall_lag must be 0, 1, or at most tau - 1");
  if (cfg->D % 8 || cfg->Dh % 8 || cfg->E % 8) LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "D, Dh, E must be multiples of 8 (16-byte vector loads)");
  if (!cfg->hot_pool || !cfg->W_q) LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "null hot_pool / W_q");
  if (cfg->hot_pages < 1) LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "hot_pages must be >= 1");
  if (cfg->merge_mode < LSA_MERGE_AUTO || cfg->merge_mode > LSA_MERGE_FUSED)
    LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "bad merge_mode");
  if (cfg->cold_format != LSA_COLD_NATIVE && cfg->cold_format != LSA_COLD_FP8_E4M3)
    LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "bad cold_format");
  if (cfg->step_overlap != 0 && cfg->step_overlap != 1)
    LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_INVALID_ARG, "step_overlap must be 0 or 1");
  lsa_ctx* c = new (std::nothrow) lsa_ctx();
  if (!c) LSA_FAIL((lsa_ctx*)nullptr, LSA_ERR_OOM, "out of host memory");
  int rc = init_impl(c, cfg, seqs);
  if (rc != LSA_OK) {
    g_init_error = c->err;
    lsa_destroy(c);
    return rc;
  }
  *out = c;
  return LSA_OK;
}

// ---- S1-S3 ------------------------------------------------------------------------------------
// rows[i] = row of `h` holding the hidden state of sequence ids[i]
static int index_select_impl(lsa_ctx* c, const void* h, const int* ids, const int* rows, int n, int32_t* sel_idx,
                             float* sel_score) {
  const lsa_config& cfg = c->cfg;
  for (int off = 0; off < n;) {
    // 8..16 sequences firing together with consecutive rows of h: the projection is a GEMM on tensor cores
    int m = std::min(kFireMax, n - off);
    const int m_tc = std::min(16, n - off);
    const bool tc = c->qtower_tc != 0 && qtower_tc_usable(cfg.dtype, cfg.E, cfg.Dh, m_tc, rows + off);
    if (tc) m = m_tc;
    FireList fire{}, hrows{};
    fire.n = hrows.n = m;
    for (int i = 0; i < m; ++i) { fire.ids[i] = ids[off + i]; hrows.ids[i] = rows[off + i]; }
    ProfScope prof(c, LSA_PH_INDEX, c->sf);
    if (tc) {
      LSA_CUDA(c, launch_qtower_tc(cfg.W_q, h, rows[off], m, c->d_z, cfg.E, cfg.Dh, c->sf));
      LSA_CUDA(c, launch_scores(cfg.dtype, c->d_seqs, fire, c->d_z, c->d_scores, cfg.E, std::max(c->n_chunks_max, 1), c->sf,
                                qtower_tc_splits(cfg.Dh)));
    } else {
      LSA_CUDA(c, launch_qtower(cfg.dtype, cfg.W_q, h, hrows, c->d_z, cfg.E, cfg.Dh, c->sf));
      LSA_CUDA(c, launch_scores(cfg.dtype, c->d_seqs, fire, c->d_z, c->d_scores, cfg.E, std::max(c->n_chunks_max, 1), c->sf));
    }
    LSA_CUDA(c, launch_topk(c->d_seqs, fire, c->d_scores, std::max(c->n_chunks_max, 1), c->k,
                            sel_idx + (size_t)off * c->k, sel_score ? sel_score + (size_t)off * c->k : nullptr, c->sf));
    c->index_launches += 3;
    off += m;
  }
  return LSA_OK;
}

static int check_ids(lsa_ctx* c, const int32_t* seq_ids, int n) {
  if (!seq_ids || n < 1 || n > c->B) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq_ids null or n out of range");
  for (int i = 0; i < n; ++i) {
    if (seq_ids[i] < 0 || seq_ids[i] >= c->B) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq id %d out of range", seq_ids[i]);
    if (i && seq_ids[i] <= seq_ids[i - 1]) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq_ids must be strictly ascending");
  }
  return LSA_OK;
}

extern "C" int lsa_index_select(lsa_ctx* ctx, const void* h, const int32_t* seq_ids, int32_t n, int32_t* sel_idx,
                                float* sel_score) {
  if (!ctx) return LSA_ERR_STATE;
  if (!h || !sel_idx) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "null h / sel_idx");
  int rc = check_ids(ctx, seq_ids, n);
  if (rc) return rc;
  std::vector<int> rows(n);
  for (int i = 0; i < n; ++i) rows[i] = i;
  return index_select_impl(ctx, h, seq_ids, rows.data(), n, sel_idx, sel_score);
}

// S1-S3 without a context and without any allocation (scratch = a file-scope device array in lsa_index.cu)
extern "C" int lsa_index_select_static(int32_t dtype, const void* W_q, const void* h, const void* const* chunk_emb,
                                       const int32_t* n_chunks, int32_t n, int32_t E, int32_t Dh, int32_t k, int32_t* sel_idx,
                                       float* sel_score, void* stream) {
  char msg[256] = "";
  const int rc = index_select_static(dtype, W_q, h, chunk_emb, n_chunks, n, E, Dh, k, sel_idx, sel_score, (cudaStream_t)stream, msg, sizeof(msg));
  if (rc != 0) g_init_error = msg;                 // read with lsa_last_error(NULL)
  return rc == 0 ? LSA_OK : (rc == -1 ? LSA_ERR_INVALID_ARG : LSA_ERR_CUDA);
}

// ---- paper-exact Level-1 indexer (NEXT-1) ---------------------------------------------------------
extern "C" int lsa_l1_init(lsa_ctx* ctx, const lsa_l1_config* cfg, const void* const* index_k) {
  if (!ctx) return LSA_ERR_STATE;
  lsa_ctx* c = ctx;
  if (!cfg || !index_k) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "null argument");
  if (cfg->struct_size != sizeof(lsa_l1_config)) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "lsa_l1_config.struct_size mismatch");
  if (c->l1) LSA_FAIL(c, LSA_ERR_STATE, "lsa_l1_init was already called on this context");
  if (cfg->n_layers < 1 || cfg->n_layers > 4 || cfg->d_c < 8 || cfg->d_c % 8) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "n_layers must be 1..4, d_c a multiple of 8");
  const float thr = cfg->threshold == 0.f ? 0.5f : cfg->threshold;
  if (!(thr > 0.f && thr < 1.f)) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "threshold must be in (0, 1)");
  if (!l1_supported(c->cfg.dtype, c->cfg.C, cfg->c_I, cfg->n_h))
    LSA_FAIL(c, LSA_ERR_UNSUPPORTED, "Level-1 indexer needs bf16, C=128, c_I=128, n_h=64 (got dtype=%d C=%d c_I=%d n_h=%d)", c->cfg.dtype, c->cfg.C,
             cfg->c_I, cfg->n_h);
  L1Init in{};
  in.B = c->B; in.n_layers = cfg->n_layers; in.Dh = c->cfg.Dh; in.d_c = cfg->d_c; in.n_chunks_max = c->n_chunks_max; in.n_sms = c->n_sms;
  for (int l = 0; l < cfg->n_layers; ++l) {
    if (!cfg->layers[l].W_dq || !cfg->layers[l].W_iuq || !cfg->layers[l].W_w) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "null weight pointer in layer %d", l);
    in.layers[l].W_dq = cfg->layers[l].W_dq; in.layers[l].W_iuq = cfg->layers[l].W_iuq; in.layers[l].W_w = cfg->layers[l].W_w;
  }
  in.index_k = index_k;
  in.seq_host = c->seq_host.data();
  std::string msg;
  const int rc = l1_create(in, &c->l1, &msg);
  if (rc != 0) LSA_FAIL(c, rc, "Level-1 indexer init failed: %s", msg.c_str());
  c->l1_threshold = thr;
  return LSA_OK;
}

static int l1_select_impl(lsa_ctx* ctx, const void* h, const int* ids, const int* rows, int n, int32_t* sel_idx, float* sel_score) {
  std::string msg;
  int launches = 0;
  ProfScope prof(ctx, LSA_PH_INDEX, ctx->sf);
  const int rc = l1_select(ctx->l1, ctx->d_seqs, h, ids, rows, n, ctx->k, ctx->l1_threshold, sel_idx, sel_score, ctx->sf, &launches, &msg);
  ctx->index_launches += launches;
  if (rc != 0) LSA_FAIL(ctx, rc == -1 ? LSA_ERR_INVALID_ARG : LSA_ERR_CUDA, "Level-1 indexer: %s", msg.c_str());
  return LSA_OK;
}

extern "C" int lsa_l1_select(lsa_ctx* ctx, const void* h, const int32_t* seq_ids, int32_t n, int32_t* sel_idx, float* sel_score) {
  if (!ctx) return LSA_ERR_STATE;
  if (!ctx->l1) LSA_FAIL(ctx, LSA_ERR_STATE, "lsa_l1_init has not been called");
  if (!h || !sel_idx) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "null h / sel_idx");
  int rc = check_ids(ctx, seq_ids, n);
  if (rc) return rc;
  std::vector<int> rows(n);
  for (int i = 0; i < n; ++i) rows[i] = i;
  return l1_select_impl(ctx, h, seq_ids, rows.data(), n, sel_idx, sel_score);
}

extern "C" int lsa_set_indexer(lsa_ctx* ctx, int32_t indexer) {
  if (!ctx) return LSA_ERR_STATE;
  if (indexer != LSA_INDEXER_DUAL_ENCODER && indexer != LSA_INDEXER_LEVEL1) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "bad indexer");
  if (indexer == LSA_INDEXER_LEVEL1 && !ctx->l1) LSA_FAIL(ctx, LSA_ERR_STATE, "lsa_l1_init has not been called");
  ctx->indexer = indexer;
  return LSA_OK;
}

// ---- S4-S5 ------------------------------------------------------------------------------------
// sel_is_topk: the selection is S3's own output, i.e. exactly k_eff valid ids per sequence (the host then knows the
// size of the staged table without asking the device)
static int fetch_impl(lsa_ctx* c, const int* ids, int n, const int32_t* sel_idx, bool sel_is_topk = false) {
  const lsa_config& cfg = c->cfg;
  // the side band must see the tables as of "now" on the compute stream, and may not evict pages
  // an earlier attention launch is still reading
  LSA_CUDA(c, cudaEventRecord(c->ev_compute, c->sc));
  LSA_CUDA(c, cudaStreamWaitEvent(c->sf, c->ev_compute, 0));
  for (int off = 0; off < n; off += kFireMax) {
    const int m = std::min(kFireMax, n - off);
    FireList fire{};
    fire.n = m;
    for (int i = 0; i < m; ++i) fire.ids[i] = ids[off + i];
    {
      ProfScope prof(c, LSA_PH_RESIDENCY, c->sf);
      // (the residency pass only uses the page size on the COLD side: source offsets and the byte counter)
      LSA_CUDA(c, launch_residency(c->d_seqs, c->pool, fire, sel_idx + (size_t)off * c->k, c->B, c->k, c->P_lru,
                                   c->cold_page_bytes, c->sf, c->k_sel, c->growth ? cfg.C : 0));
    }
    {
      ProfScope prof(c, LSA_PH_FETCH, c->sf);
      LSA_CUDA(c, launch_fetch(c->pool, cfg.hot_pool, c->page_bytes, c->fetch_ctas, c->sf, c->cold_page_bytes));
    }
    c->index_launches += 2;
  }
  LSA_CUDA(c, cudaEventRecord(c->ev_fetch, c->sf));
  for (int i = 0; i < n; ++i) {
    c->pending[ids[i]] = 1;
    c->visible_at[ids[i]] = c->step[ids[i]] + cfg.recall_lag;
    const int b = ids[i];
    // entries of the staged table: the recalled chunks, then the tail chunk of a growing sequence if it holds rows
    const int tail = (c->growth && c->seq_host[b].n_csa % cfg.C) ? 1 : 0;
    c->n_tbl[1 - c->cur_buf[b]][b] = sel_is_topk ? c->k_eff[b] + tail : -1;
    c->ncand_nxt[b] = c->seq_host[b].n_chunks;
  }
  return LSA_OK;
}

extern "C" int lsa_fetch_chunks(lsa_ctx* ctx, const int32_t* seq_ids, int32_t n, const int32_t* sel_idx) {
  if (!ctx) return LSA_ERR_STATE;
  if (!sel_idx) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "null sel_idx");
  int rc = check_ids(ctx, seq_ids, n);
  if (rc) return rc;
  return fetch_impl(ctx, seq_ids, n, sel_idx);
}

// ---- S6 -----------------------------------------------------------------------------------------
// Swap every staged table that is due (or all of them if force) and optionally append k_new/v_new.
// Which staged tables are due (or all of them if force)?  Clears their host-side pending flags.
static bool due_mask(lsa_ctx* c, bool force, uint32_t words[32]) {
  bool any = false;
  for (int i = 0; i < 32; ++i) words[i] = 0;
  for (int b = 0; b < c->B; ++b) {
    if (c->pending[b] && (force || c->step[b] >= c->visible_at[b])) {
      words[b >> 5] |= 1u << (b & 31);
      c->pending[b] = 0;
      c->cur_buf[b] ^= 1;                         // the device flips its record under the same condition
      c->ncand_cur[b] = c->ncand_nxt[b];
      any = true;
    }
  }
  return any;
}

static void mirror_append(lsa_ctx* c) {            // host mirror of the ring (the kernels apply the same rule)
  for (int b = 0; b < c->B; ++b) {
    c->seq_host[b].w_len = std::min(c->cfg.W, c->seq_host[b].w_len + 1);
    c->w_head[b] = c->w_head[b] + 1 == c->cfg.W ? 0 : c->w_head[b] + 1;
    c->app_count[b] += 1u;
  }
}

// Swap every staged table that is due (or all of them if force) and optionally append k_new/v_new.
static int prestep_impl(lsa_ctx* c, bool force, const void* k_new, const void* v_new) {
  uint32_t words[32];
  const bool any = due_mask(c, force, words);
  if (!any && !k_new) return LSA_OK;
  if (any) LSA_CUDA(c, cudaStreamWaitEvent(c->sc, c->ev_fetch, 0));
  ProfScope prof(c, LSA_PH_PRESTEP, c->sc);
  LSA_CUDA(c, launch_prestep(c->cfg.dtype, c->d_seqs, c->B, c->cfg.D, c->cfg.W, any ? words : nullptr, 32, k_new, v_new, c->sc));
  c->serialize_next = true;        // the next attention launch reads what this kernel writes: no early start
  c->attn_launches += 1;
  if (k_new) mirror_append(c);
  return LSA_OK;
}

extern "C" int lsa_commit_tables(lsa_ctx* ctx) {
  if (!ctx) return LSA_ERR_STATE;
  return prestep_impl(ctx, true, nullptr, nullptr);
}

// ---- S7-S8 --------------------------------------------------------------------------------------
static int attention_impl(lsa_ctx* c, const void* q, void* out, float* lse, const TcPrestep* pre = nullptr) {
  const lsa_config& cfg = c->cfg;
  if (c->attn_impl == LSA_ATTN_SIMT) {
    {
      ProfScope prof(c, LSA_PH_ATTENTION, c->sc);
      LSA_CUDA(c, launch_attn_simt(cfg.dtype, cfg.H, cfg.D, cfg.C, c->k, c->d_seqs, c->pool, cfg.hot_pool, q, c->sm_scale,
                                   c->geom, c->B, c->part_o, c->part_ml, c->sc));
    }
    {
      ProfScope prof(c, LSA_PH_COMBINE, c->sc);
      LSA_CUDA(c, launch_combine(cfg.dtype, cfg.H, cfg.D, cfg.C, c->d_seqs, c->geom, c->B, c->part_o, c->part_ml, out, lse, c->sc));
    }
    c->attn_launches += 2;
    c->last_attn_ctas = c->geom.s_max * c->B;
  } else {
    int launches = 0, ctas = 0;
    std::string msg;
    // profiling: attention = start .. mid, combine = mid .. end (the events between the two kernels cost the
    // programmatic overlap of that pair, so phase times are upper bounds of what an unprofiled step sees)
    const bool prof = c->prof_cap > 0 && c->prof_n[LSA_PH_ATTENTION] < c->prof_cap && c->prof_n[LSA_PH_COMBINE] < c->prof_cap;
    const int ia = c->prof_n[LSA_PH_ATTENTION], ic = c->prof_n[LSA_PH_COMBINE];
    if (prof) cudaEventRecord(c->prof_ev[LSA_PH_ATTENTION][2 * ia], c->sc);
    long long tiles = 0;                          // host mirror: HCA + selected pages + window, in 128-key tiles
    for (int b = 0; b < c->B; ++b)
      tiles += (c->seq_host[b].n_hca + 127) / 128 + c->k_eff[b] + (c->growth ? 2 : 0) + (c->seq_host[b].w_len + 127) / 128;
    int rc;
    if (c->cfg.step_overlap && tc_small_supported(c->tc) && !c->l2_armed && !c->no_small) {
      // small batches whose steps do not depend on one another (lsa_config.step_overlap): one launch per step that
      // gets the host's mirrors by value, does not wait for its predecessor and merges its own partials.  The
      // mirrors already hold the state AFTER this step's swap and append (due_mask / mirror_append ran).
      TcSmallStep stp{};
      const bool app = pre && pre->k_new;
      for (int b = 0; b < c->B; ++b) {
        TcSmallSeq& q_ = stp.seq[b];
        q_.cur = c->cur_buf[b];
        q_.n_cur = c->n_tbl[q_.cur][b];
        q_.w_len = c->seq_host[b].w_len;
        q_.app_slot = app ? (c->w_head[b] == 0 ? c->cfg.W - 1 : c->w_head[b] - 1) : -1;
        q_.app_count = app ? c->app_count[b] - 1u : c->app_count[b];
        q_.grow_count = c->grow_count[b];
      }
      stp.grow_wait = c->grow_wait_next ? 1 : 0;
      c->grow_wait_next = false;
      stp.swap = pre ? pre->swap[0] : 0u;
      stp.k_new = app ? pre->k_new : nullptr;
      stp.v_new = app ? pre->v_new : nullptr;
      stp.serialize = (!pre || stp.swap || c->serialize_next) ? 1 : 0;
      stp.wait_inputs = (c->cfg.step_overlap && !c->inputs_from_prev_kernel) ? 0 : 1;
      if (c->inputs_by_counter) { stp.wait_inputs = 0; stp.in_ctr = c->gather_ctr; stp.in_need = c->gather_total; }
      c->inputs_by_counter = false;
      stp.alone = c->next_alone ? 1 : 0;
      c->serialize_next = false;
      c->inputs_from_prev_kernel = false;
      c->next_alone = false;
      if (c->tl_on) {                               // lsa_timeline_enable: this launch's record of the ring
        stp.tl = c->d_tl + (size_t)(c->tl_seq % LSA_TL_LAUNCHES) * LSA_TL_CTAS * LSA_TL_EVENTS;
        stp.tl_seq = (unsigned int)c->tl_seq;
        c->tl_seq += 1;
      }
      if (c->host_flag_dev) {                       // lsa_step_host spins on the flag instead of synchronising the stream
        stp.host_flag = c->host_flag_dev;
        stp.host_flag_val = ++c->host_flag_seq;
        c->host_flag_armed = true;
      }
      rc = tc_attention_small(c->tc, q, out, lse, stp, c->sc, &launches, &ctas, &msg,
                              prof ? c->prof_ev[LSA_PH_ATTENTION][2 * ia + 1] : nullptr,
                              prof ? c->prof_ev[LSA_PH_COMBINE][2 * ic] : nullptr,
                              prof && c->d_ktime ? c->d_ktime + 2 * ia : nullptr);
    } else {
      tc_set_l2_mask(c->tc, c->l2_armed ? l2_mask(c->l2) : nullptr);      // one-shot: the selection of this step
      c->l2_armed = false;
      rc = tc_attention(c->tc, q, out, lse, tiles, pre, c->sc, &launches, &ctas, &msg,
                        prof ? c->prof_ev[LSA_PH_ATTENTION][2 * ia + 1] : nullptr,
                        prof ? c->prof_ev[LSA_PH_COMBINE][2 * ic] : nullptr,
                        prof && c->d_ktime ? c->d_ktime + 2 * ia : nullptr);
    }
    if (prof) {
      cudaEventRecord(c->prof_ev[LSA_PH_COMBINE][2 * ic + 1], c->sc);
      c->prof_n[LSA_PH_ATTENTION] += 1;
      c->prof_n[LSA_PH_COMBINE] += 1;
    }
    if (rc != 0) LSA_FAIL(c, rc, "tcgen05 attention: %s", msg.c_str());
    c->attn_launches += launches;
    c->last_attn_ctas = ctas;
  }
  return LSA_OK;
}

extern "C" int lsa_decode_attention(lsa_ctx* ctx, const void* q, void* out, float* lse) {
  if (!ctx) return LSA_ERR_STATE;
  if (!q || !out) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "null q / out");
  if (ctx->attn_impl == LSA_ATTN_TCGEN05) {        // S6 is folded into the attention launch
    TcPrestep pre{};
    uint32_t words[32];
    if (due_mask(ctx, false, words)) {
      LSA_CUDA(ctx, cudaStreamWaitEvent(ctx->sc, ctx->ev_fetch, 0));
      for (int i = 0; i < 8; ++i) pre.swap[i] = words[i];
    }
    return attention_impl(ctx, q, out, lse, &pre);
  }
  int rc = prestep_impl(ctx, false, nullptr, nullptr);
  if (rc) return rc;
  return attention_impl(ctx, q, out, lse);
}

static int l2_select_impl(lsa_ctx* c, const void* q_idx, const float* w_idx, int32_t* sel_entries, float* sel_score,
                          const unsigned* folded_swap = nullptr);

static int step_impl(lsa_ctx* ctx, const void* q, const void* h, const void* k_new, const void* v_new, void* out,
                     const void* q_idx, const float* w_idx) {
  lsa_ctx* c = ctx;
  if (!q || !out) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "null q / out");
  if ((k_new == nullptr) != (v_new == nullptr)) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "k_new and v_new must both be given or both NULL");
  if (k_new && c->cfg.W < 1) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "k_new given but W == 0");
  if (!q_idx) c->l2_armed = false;        // a selection left by lsa_l2_select belongs to lsa_decode_attention, not to a step
  int ids[1024];
  int n_fire = 0;
  for (int b = 0; b < c->B; ++b)
    if (c->step[b] % c->cfg.tau == 0) ids[n_fire++] = b;           // S0
  if (n_fire && !h) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "h is NULL at a trigger step");
  int rc;
  if (n_fire == 0 && c->attn_impl == LSA_ATTN_TCGEN05) {
    // no trigger this step: (a) and (d) ride on the attention launch itself (one kernel less per step).  On a
    // trigger step the residency pass must see the swapped tables, so they stay a kernel of their own.
    TcPrestep pre{};
    uint32_t words[32];
    if (due_mask(c, false, words)) {
      LSA_CUDA(c, cudaStreamWaitEvent(c->sc, c->ev_fetch, 0));
      for (int i = 0; i < 8; ++i) pre.swap[i] = words[i];
    }
    // Level 2 scores the tables as this launch will see them (the swap rides on the attention launch)
    if (q_idx && (rc = l2_select_impl(c, q_idx, w_idx, nullptr, nullptr, pre.swap))) return rc;
    pre.k_new = k_new; pre.v_new = v_new;
    if (k_new) mirror_append(c);
    if ((rc = attention_impl(c, q, out, nullptr, &pre))) return rc;
    for (int b = 0; b < c->B; ++b) c->step[b] += 1;
    c->n_steps += 1;
    return LSA_OK;
  }
  if (n_fire && c->attn_impl == LSA_ATTN_TCGEN05 && c->cfg.step_overlap && tc_small_supported(c->tc) && !q_idx && !c->no_small &&
      c->cfg.recall_lag >= 1) {
    // Independent steps (lsa_config.step_overlap), trigger step: with recall_lag >= 1 no table swap can be due now (the
    // table staged by the previous trigger became current lag < tau steps after it), so the side band reads the records
    // as the PREVIOUS step left them and nothing on the compute stream has to wait: the attention launch stays in the
    // overlapped chain, the window append rides on it as on any other step.
    bool due = false;
    for (int b = 0; b < c->B; ++b) due |= c->pending[b] && c->step[b] >= c->visible_at[b];
    if (!due) {
      if (c->indexer == LSA_INDEXER_LEVEL1 ? (rc = l1_select_impl(c, h, ids, ids, n_fire, c->d_sel, nullptr))
                                           : (rc = index_select_impl(c, h, ids, ids, n_fire, c->d_sel, nullptr)))
        return rc;
      if ((rc = fetch_impl(c, ids, n_fire, c->d_sel, c->indexer != LSA_INDEXER_LEVEL1))) return rc;
      TcPrestep pre{};
      pre.k_new = k_new; pre.v_new = v_new;
      if (k_new) mirror_append(c);
      if ((rc = attention_impl(c, q, out, nullptr, &pre))) return rc;
      for (int b = 0; b < c->B; ++b) c->step[b] += 1;
      c->n_steps += 1;
      return LSA_OK;
    }
  }
  if ((rc = prestep_impl(c, false, k_new, v_new))) return rc;       // (a) + (d)
  if (n_fire) {                                                     // (b)
    if (c->indexer == LSA_INDEXER_LEVEL1 ? (rc = l1_select_impl(c, h, ids, ids, n_fire, c->d_sel, nullptr))
                                         : (rc = index_select_impl(c, h, ids, ids, n_fire, c->d_sel, nullptr)))
      return rc;
    if ((rc = fetch_impl(c, ids, n_fire, c->d_sel, c->indexer != LSA_INDEXER_LEVEL1))) return rc;
    if (c->cfg.recall_lag == 0 && (rc = prestep_impl(c, false, nullptr, nullptr))) return rc;   // (c)
  }
  if (q_idx && (rc = l2_select_impl(c, q_idx, w_idx, nullptr, nullptr))) return rc;   // Level 2 sees the tables attention will
  if ((rc = attention_impl(c, q, out, nullptr))) return rc;         // (e)
  for (int b = 0; b < c->B; ++b) c->step[b] += 1;                   // (f)
  c->n_steps += 1;
  return LSA_OK;
}

extern "C" int lsa_step(lsa_ctx* ctx, const void* q, const void* h, const void* k_new, const void* v_new, void* out) {
  if (!ctx) return LSA_ERR_STATE;
  return step_impl(ctx, q, h, k_new, v_new, out, nullptr, nullptr);
}

// ---- NEXT-3: the non-trigger step as a CUDA graph ------------------------------------------------------------
extern "C" int lsa_step_graph(lsa_ctx* ctx, const void* q, const void* h, const void* k_new, const void* v_new, void* out) {
  if (!ctx) return LSA_ERR_STATE;
  lsa_ctx* c = ctx;
  if (!q || !out) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "null q / out");
  if ((k_new == nullptr) != (v_new == nullptr)) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "k_new and v_new must both be given or both NULL");
  bool plain = c->growth || c->attn_impl != LSA_ATTN_TCGEN05 || c->prof_cap > 0 || c->cfg.merge_mode == LSA_MERGE_FUSED || (k_new && c->cfg.W < 1);
  for (int b = 0; b < c->B && !plain; ++b)
    plain = (c->step[b] % c->cfg.tau == 0) || (c->pending[b] && c->step[b] >= c->visible_at[b]);   // trigger, or a swap is due
  c->no_small = true;             // the captured launch reads the device records: this context stays on the general kernels
  if (plain) return step_impl(c, q, h, k_new, v_new, out, nullptr, nullptr);
  c->l2_armed = false;
  if (k_new) mirror_append(c);
  long long tiles = 0;                              // same host mirror attention_impl sizes the grid from
  for (int b = 0; b < c->B; ++b) tiles += (c->seq_host[b].n_hca + 127) / 128 + c->k_eff[b] + (c->seq_host[b].w_len + 127) / 128;
  if (!c->sg_exec || q != c->sg_q || k_new != c->sg_kn || v_new != c->sg_vn || out != c->sg_out || tiles != c->sg_tiles) {
    if (c->sg_exec) { cudaGraphExecDestroy(c->sg_exec); c->sg_exec = nullptr; }
    const unsigned long long before = c->attn_launches;
    LSA_CUDA(c, cudaStreamBeginCapture(c->sc, cudaStreamCaptureModeThreadLocal));
    TcPrestep pre{};
    pre.k_new = k_new; pre.v_new = v_new;
    const int rc = attention_impl(c, q, out, nullptr, &pre);
    cudaGraph_t g = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->sc, &g);
    c->sg_launches = c->attn_launches - before;
    c->attn_launches = before;                      // nothing ran during the capture
    if (rc) { if (g) cudaGraphDestroy(g); return rc; }
    if (e != cudaSuccess || !g) LSA_FAIL(c, LSA_ERR_CUDA, "stream capture of the step failed: %s", cudaGetErrorString(e));
    const cudaError_t ei = cudaGraphInstantiate(&c->sg_exec, g, 0);
    cudaGraphDestroy(g);
    if (ei != cudaSuccess) { c->sg_exec = nullptr; LSA_FAIL(c, LSA_ERR_CUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(ei)); }
    c->sg_q = q; c->sg_kn = k_new; c->sg_vn = v_new; c->sg_out = out; c->sg_tiles = tiles;
    c->sg_captures += 1;
  } else {
    c->sg_replays += 1;
  }
  LSA_CUDA(c, cudaGraphLaunch(c->sg_exec, c->sc));
  c->attn_launches += c->sg_launches;
  for (int b = 0; b < c->B; ++b) c->step[b] += 1;
  c->n_steps += 1;
  return LSA_OK;
}

extern "C" int lsa_graph_stats(lsa_ctx* ctx, uint64_t* captures, uint64_t* replays) {
  if (!ctx) return LSA_ERR_STATE;
  if (captures) *captures = ctx->sg_captures;
  if (replays) *replays = ctx->sg_replays;
  return LSA_OK;
}

// ---- Level 2 (NEXT-2) ---------------------------------------------------------------------------------------
extern "C" int lsa_l2_init(lsa_ctx* ctx, const lsa_l2_config* cfg, const void* const* index_k) {
  if (!ctx) return LSA_ERR_STATE;
  lsa_ctx* c = ctx;
  if (!cfg || !index_k) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "null argument");
  if (cfg->struct_size != sizeof(lsa_l2_config)) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "lsa_l2_config.struct_size mismatch");
  if (c->l2) LSA_FAIL(c, LSA_ERR_STATE, "lsa_l2_init was already called on this context");
  if (cfg->k2 < 1 || cfg->k2 > kSortCap) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "k2 must be in 1..%d", kSortCap);
  if (c->attn_impl != LSA_ATTN_TCGEN05 || !l2_supported(c->cfg.dtype, c->cfg.C, cfg->c_I, cfg->n_h))
    LSA_FAIL(c, LSA_ERR_UNSUPPORTED, "Level 2 needs the tcgen05 attention path, bf16, C=128, c_I=128, n_h=64 (got dtype=%d C=%d c_I=%d n_h=%d)",
             c->cfg.dtype, c->cfg.C, cfg->c_I, cfg->n_h);
  L2Init in{};
  in.B = c->B; in.k = c->k; in.k2 = cfg->k2; in.n_sms = c->n_sms;
  in.index_k = index_k; in.seq_host = c->seq_host.data(); in.tbl_chunk = c->pool.tbl_chunk;
  std::string msg;
  const int rc = l2_create(in, &c->l2, &msg);
  if (rc != 0) LSA_FAIL(c, rc == -1 ? LSA_ERR_INVALID_ARG : LSA_ERR_CUDA, "Level 2 init failed: %s", msg.c_str());
  return LSA_OK;
}

static int l2_select_impl(lsa_ctx* c, const void* q_idx, const float* w_idx, int32_t* sel_entries, float* sel_score,
                          const unsigned* folded_swap) {
  if (!c->l2) LSA_FAIL(c, LSA_ERR_STATE, "lsa_l2_init has not been called");
  if (!q_idx || !w_idx) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "null q_idx / w_idx");
  int rc = folded_swap ? 0 : prestep_impl(c, false, nullptr, nullptr);   // the tables the next attention launch will read
  if (rc) return rc;
  std::string msg;
  int launches = 0;
  rc = l2_select(c->l2, c->d_seqs, q_idx, w_idx, sel_entries, sel_score, folded_swap, c->sc, &launches, &msg);
  c->attn_launches += launches;
  if (rc != 0) LSA_FAIL(c, LSA_ERR_CUDA, "Level 2: %s", msg.c_str());
  c->l2_armed = true;
  return LSA_OK;
}

extern "C" int lsa_l2_select(lsa_ctx* ctx, const void* q_idx, const float* w_idx, int32_t* sel_entries, float* sel_score) {
  if (!ctx) return LSA_ERR_STATE;
  return l2_select_impl(ctx, q_idx, w_idx, sel_entries, sel_score);
}

extern "C" int lsa_l2_get_mask(lsa_ctx* ctx, int32_t seq, uint32_t* words) {
  if (!ctx) return LSA_ERR_STATE;
  if (!ctx->l2) LSA_FAIL(ctx, LSA_ERR_STATE, "lsa_l2_init has not been called");
  if (seq < 0 || seq >= ctx->B || !words) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "bad seq / null words");
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sc));
  LSA_CUDA(ctx, cudaMemcpy(words, l2_mask(ctx->l2) + (size_t)seq * ctx->k * 4, (size_t)ctx->k * 4 * sizeof(uint32_t), cudaMemcpyDeviceToHost));
  return LSA_OK;
}

extern "C" int lsa_step_l2(lsa_ctx* ctx, const void* q, const void* h, const void* k_new, const void* v_new, const void* q_idx,
                           const float* w_idx, void* out) {
  if (!ctx) return LSA_ERR_STATE;
  if (!ctx->l2) LSA_FAIL(ctx, LSA_ERR_STATE, "lsa_l2_init has not been called");
  if (!q_idx || !w_idx) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "null q_idx / w_idx");
  return step_impl(ctx, q, h, k_new, v_new, out, q_idx, w_idx);
}

// lsa_step_host: one launch pulls the step's inputs out of pinned, mapped host buffers (16-byte loads over the
// host link) into the device staging area - no CPU-side packing, no copy-engine operation in the chain.
struct HostGather {
  const uint4* src[4];
  uint4* dst[4];
  unsigned n16[4];     // 16-byte units per part (0 = absent)
  unsigned int* ctr;   // or null: every block adds 1 (release) once its share is written - the attention launch that runs
                       // beside it waits for the total instead of for the grid
};
__global__ void __launch_bounds__(256) host_gather_kernel(HostGather g) {
  // the attention launch that follows may start its K/V stream now; it waits for this grid before it reads q / k_new
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x, nthr = gridDim.x * blockDim.x;
#pragma unroll
  for (int p = 0; p < 4; ++p)
    for (unsigned i = tid; i < g.n16[p]; i += nthr) g.dst[p][i] = g.src[p][i];
  if (g.ctr) {
    asm volatile("fence.proxy.async;" ::: "memory");      // the image is read by TMA (async proxy)
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(g.ctr) : "memory");
  }
}

// device alias of a pinned + mapped host pointer, or null (cached: the attribute query costs about a microsecond)
static void* host_alias(lsa_ctx* c, const void* p) {
  if (!p) return nullptr;
  for (const auto& e : c->alias_cache) if (e.first == p) return e.second;
  cudaPointerAttributes at{};
  void* d = nullptr;
  if (cudaPointerGetAttributes(&at, p) == cudaSuccess && at.type == cudaMemoryTypeHost && at.devicePointer) d = at.devicePointer;
  else cudaGetLastError();
  if (c->alias_cache.size() >= 256) c->alias_cache.clear();
  c->alias_cache.emplace_back(p, d);
  return d;
}

constexpr int kStRing = 8;            // staging images in rotation: lsa_step_host_async calls in flight at most

static int host_wait_impl(lsa_ctx* c, uint64_t ticket) {
  if (ticket == 0 || !c->host_flag) { LSA_CUDA(c, cudaStreamSynchronize(c->sc)); return LSA_OK; }
  volatile unsigned int* f = c->host_flag;
  const unsigned int want = (unsigned int)ticket;
  for (long long spin = 0; (int)(*f - want) < 0; ++spin) {
    if (spin > 20000000ll) { LSA_CUDA(c, cudaStreamSynchronize(c->sc)); break; }     // bounded: fall back to the stream
#if defined(__x86_64__)
    __builtin_ia32_pause();
#endif
  }
  return LSA_OK;
}

// ticket: null = block until the result has landed; else the step is only enqueued and *ticket identifies it
static int step_host_impl(lsa_ctx* c, const void* q, const void* h, const void* k_new, const void* v_new, void* out, uint64_t* ticket) {
  if (!q || !out) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "null q / out");
  if ((k_new == nullptr) != (v_new == nullptr)) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "k_new and v_new must both be given or both NULL");
  const lsa_config& cfg = c->cfg;
  auto up = [](size_t n) { return (n + 255) / 256 * 256; };
  const size_t qb = (size_t)c->B * cfg.H * cfg.D * c->elem, hb = (size_t)c->B * cfg.Dh * c->elem,
               nb = (size_t)c->B * cfg.D * c->elem;
  // one packed image [q | k_new | v_new | h] per step; kStRing of them in rotation, so that the image of a step still
  // in flight is not overwritten by the next ones
  const size_t o_kn = up(qb), o_vn = o_kn + up(nb), o_h = o_vn + up(nb), in_bytes = o_h + up(hb);
  if (!c->st_q) {
    int rc;
    unsigned char* p = nullptr;
    if ((rc = dev_alloc(c, &p, kStRing * in_bytes + up(qb)))) return rc;
    c->st_q = p; c->st_out = p + kStRing * in_bytes;
    LSA_CUDA(c, cudaHostAlloc(&c->st_pin, in_bytes, cudaHostAllocDefault));
    if (c->cfg.step_overlap && c->attn_impl == LSA_ATTN_TCGEN05 && tc_small_supported(c->tc)) {
      void* f = nullptr;
      LSA_CUDA(c, cudaHostAlloc(&f, 64, cudaHostAllocMapped));
      memset(f, 0, 64);
      c->host_flag = static_cast<unsigned int*>(f);
      void* fd = nullptr;
      LSA_CUDA(c, cudaHostGetDevicePointer(&fd, f, 0));
      c->host_flag_dev = static_cast<unsigned int*>(fd);
      if ((rc = dev_alloc(c, &c->gather_ctr, 1))) return rc;
    }
  }
  const int slot = (int)(c->st_calls % kStRing);
  if (c->st_ticket[slot]) {                       // the step that used this image last has completed (normally long ago)
    int rc = host_wait_impl(c, c->st_ticket[slot]);
    if (rc) return rc;
    c->st_ticket[slot] = 0;
  }
  c->st_calls += 1;
  unsigned char* img = static_cast<unsigned char*>(c->st_q) + (size_t)slot * in_bytes;
  void *st_q = img, *st_kn = img + o_kn, *st_vn = img + o_vn, *st_h = img + o_h;
  bool fire = false;
  for (int b = 0; b < c->B; ++b) fire |= (c->step[b] % cfg.tau == 0);
  if (fire && !h) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "h is NULL at a trigger step");
  void* aq = host_alias(c, q);
  void* akn = k_new ? host_alias(c, k_new) : nullptr;
  void* avn = v_new ? host_alias(c, v_new) : nullptr;
  void* ah = fire ? host_alias(c, h) : nullptr;
  bool gathered = false;
  if (aq && (!k_new || (akn && avn)) && (!fire || ah) && qb % 16 == 0 && nb % 16 == 0 && hb % 16 == 0) {
    HostGather g{};
    g.src[0] = (const uint4*)aq; g.dst[0] = (uint4*)st_q; g.n16[0] = (unsigned)(qb / 16);
    if (k_new) {
      g.src[1] = (const uint4*)akn; g.dst[1] = (uint4*)st_kn; g.n16[1] = (unsigned)(nb / 16);
      g.src[2] = (const uint4*)avn; g.dst[2] = (uint4*)st_vn; g.n16[2] = (unsigned)(nb / 16);
    }
    if (fire) { g.src[3] = (const uint4*)ah; g.dst[3] = (uint4*)st_h; g.n16[3] = (unsigned)(hb / 16); }
    const unsigned total = g.n16[0] + g.n16[1] + g.n16[2] + g.n16[3];
    const dim3 grid(std::max(1u, std::min(64u, (total + 255u) / 256u)));
    // it reads host buffers and writes an image no step in flight uses: with the overlapped path it need not wait for
    // the previous step either (programmatic launch, no griddepcontrol.wait inside)
    if (c->host_flag_dev && ticket && !fire) {
      // asynchronous step: the gather runs beside the previous step (programmatic launch, no wait inside) and the
      // attention launch waits for ITS blocks only - a grid dependency would wait for the previous step as well
      g.ctr = c->gather_ctr;
      c->gather_total += grid.x;
      c->inputs_by_counter = true;
      LSA_CUDA(c, launch_pdl(host_gather_kernel, grid, dim3(256), 0, c->sc, g));
    } else if (c->host_flag_dev) LSA_CUDA(c, launch_pdl(host_gather_kernel, grid, dim3(256), 0, c->sc, g));
    else {
      host_gather_kernel<<<grid, 256, 0, c->sc>>>(g);
      LSA_CUDA(c, cudaGetLastError());
    }
    c->inputs_from_prev_kernel = true;
    gathered = true;
  } else {                         // pageable inputs: pack into the pinned staging image, one host-to-device copy
    LSA_CUDA(c, cudaStreamSynchronize(c->sc));                        // the one pinned image is reused every call
    unsigned char* pin = static_cast<unsigned char*>(c->st_pin);
    memcpy(pin, q, qb);
    size_t upto = qb;
    if (k_new) { memcpy(pin + o_kn, k_new, nb); memcpy(pin + o_vn, v_new, nb); upto = o_vn + nb; }
    if (fire) { memcpy(pin + o_h, h, hb); upto = o_h + hb; }          // h is only read at trigger steps
    LSA_CUDA(c, cudaMemcpyAsync(st_q, pin, upto, cudaMemcpyHostToDevice, c->sc));
    c->serialize_next = true;
  }
  if (fire) {                      // the indexer reads the staged h on the fetch stream: order it behind the copy
    LSA_CUDA(c, cudaEventRecord(c->ev_compute, c->sc));
    LSA_CUDA(c, cudaStreamWaitEvent(c->sf, c->ev_compute, 0));
  }
  // result: if `out` is pinned and mapped, S8 writes it in place over the host link (no device-to-host copy
  // operation in the chain); otherwise through a device buffer and one copy
  if (out != c->out_host_cached) {
    c->out_dev_alias = host_alias(c, out);
    c->out_host_cached = out;
  }
  void* out_dev = c->out_dev_alias ? c->out_dev_alias : c->st_out;
  c->host_flag_armed = false;
  c->next_alone = ticket == nullptr;
  int rc = lsa_step(c, st_q, fire ? st_h : nullptr, k_new ? st_kn : nullptr, k_new ? st_vn : nullptr, out_dev);
  c->next_alone = false;
  if (rc) return rc;
  const bool flagged = c->host_flag_armed && c->out_dev_alias && gathered;
  c->host_flag_armed = false;
  if (!flagged) {                  // no completion word on this path: finish synchronously (a ticket of 0 is always complete)
    if (!c->out_dev_alias) LSA_CUDA(c, cudaMemcpyAsync(out, c->st_out, qb, cudaMemcpyDeviceToHost, c->sc));
    LSA_CUDA(c, cudaStreamSynchronize(c->sc));
    if (ticket) *ticket = 0;
    return LSA_OK;
  }
  // the launch's last CTA writes the step's sequence number to a pinned word once `out` (pinned, written in place) is
  // complete: the host reads that word instead of synchronising the stream
  c->st_ticket[slot] = c->host_flag_seq;
  if (ticket) { *ticket = c->host_flag_seq; return LSA_OK; }
  return host_wait_impl(c, c->host_flag_seq);
}

extern "C" int lsa_step_host(lsa_ctx* ctx, const void* q, const void* h, const void* k_new, const void* v_new, void* out) {
  if (!ctx) return LSA_ERR_STATE;
  return step_host_impl(ctx, q, h, k_new, v_new, out, nullptr);
}

extern "C" int lsa_step_host_async(lsa_ctx* ctx, const void* q, const void* h, const void* k_new, const void* v_new, void* out,
                                   uint64_t* ticket) {
  if (!ctx) return LSA_ERR_STATE;
  if (!ticket) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "null ticket");
  return step_host_impl(ctx, q, h, k_new, v_new, out, ticket);
}

extern "C" int lsa_host_wait(lsa_ctx* ctx, uint64_t ticket) {
  if (!ctx) return LSA_ERR_STATE;
  return host_wait_impl(ctx, ticket);
}

// ---- NEXT-4 (first half): KV export into the cold pool -------------------------------------------------------
extern "C" int lsa_export_chunks(lsa_ctx* ctx, int32_t seq, int32_t first_chunk, int32_t n_chunks, const void* src) {
  if (!ctx) return LSA_ERR_STATE;
  lsa_ctx* c = ctx;
  if (seq < 0 || seq >= c->B) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "bad seq");
  if (first_chunk < 0 || n_chunks < 0 || (long long)first_chunk + n_chunks > c->seq_host[seq].n_chunks)
    LSA_FAIL(c, LSA_ERR_INVALID_ARG, "chunks [%d, %d) outside the sequence's %d chunks", first_chunk, first_chunk + n_chunks, c->seq_host[seq].n_chunks);
  if (n_chunks == 0) return LSA_OK;
  if (!src) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "null src");
  if (c->cold_page_bytes != c->page_bytes) {       // FP8 cold pages: quantise; one block per (page, K | V block)
    void* dst8 = const_cast<unsigned char*>(reinterpret_cast<const unsigned char*>(c->seq_host[seq].cold)) + (long long)first_chunk * c->cold_page_bytes;
    float* sc = const_cast<float*>(c->seq_host[seq].cold_scale) + 2ll * first_chunk;
    LSA_CUDA(c, launch_export_fp8(src, dst8, sc, 2ll * n_chunks, (long long)c->cfg.C * c->cfg.D, c->sf));
    c->index_launches += 1;
    return LSA_OK;
  }
  const long long bytes = (long long)n_chunks * c->page_bytes;
  void* dst = const_cast<unsigned char*>(reinterpret_cast<const unsigned char*>(c->seq_host[seq].cold)) + (long long)first_chunk * c->page_bytes;
  const int ctas = (int)std::max<long long>(1, std::min<long long>(c->fetch_ctas > 0 ? c->fetch_ctas : 64, (bytes + 16383) / 16384));
  LSA_CUDA(c, launch_export(src, dst, bytes, ctas, c->sf));
  c->index_launches += 1;
  return LSA_OK;
}

// ---- NEXT-4 (second half): decoded tokens' compressed entries ---------------------------------------------------
extern "C" int lsa_append_compressed(lsa_ctx* ctx, const int32_t* seq_ids, int32_t n, const void* csa_k, const void* csa_v,
                                     const void* hca_k, const void* hca_v, const void* emb_rows) {
  if (!ctx) return LSA_ERR_STATE;
  lsa_ctx* c = ctx;
  if (!c->growth) LSA_FAIL(c, LSA_ERR_STATE, "the context was created without growth capacity (lsa_seq_desc.cap_csa)");
  if (c->l1 || c->l2) LSA_FAIL(c, LSA_ERR_UNSUPPORTED, "growth is only built for the dual-encoder indexer (no Level-1 / Level-2 index keys are appended)");
  if ((csa_k == nullptr) != (csa_v == nullptr) || (hca_k == nullptr) != (hca_v == nullptr))
    LSA_FAIL(c, LSA_ERR_INVALID_ARG, "csa_k / csa_v and hca_k / hca_v must be given in pairs");
  int rc = check_ids(c, seq_ids, n);
  if (rc) return rc;
  if (!csa_k && !hca_k) return LSA_OK;
  const int C = c->cfg.C;
  bool roll = false, any_done = false;
  for (int i = 0; i < n; ++i) {                     // validate everything before anything is enqueued
    const int b = seq_ids[i];
    const SeqDev& s = c->seq_host[b];
    if (hca_k && s.n_hca >= s.cap_hca) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq %d: HCA capacity %d exceeded", b, s.cap_hca);
    if (!csa_k) continue;
    if (s.n_csa >= c->cap_csa[b]) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq %d: CSA capacity %lld exceeded", b, c->cap_csa[b]);
    const int ch = (int)(s.n_csa / C), r = (int)(s.n_csa % C);
    if (r == 0) {
      // chunks [ncand_cur, ch) are still attended through the tier: a third one would need the reserved page of the oldest
      if (ch - c->ncand_cur[b] >= 2)
        LSA_FAIL(c, LSA_ERR_STATE, "seq %d: chunk %d would be the third chunk of the decode tier (chunks complete faster than tables turn over)", b, ch);
      if (c->n_tbl[c->cur_buf[b]][b] < 0 || (c->pending[b] && c->n_tbl[1 - c->cur_buf[b]][b] < 0))
        LSA_FAIL(c, LSA_ERR_UNSUPPORTED, "seq %d: growth needs tables staged from the library's own top-k (lsa_step), not from lsa_fetch_chunks", b);
      roll = true;
    }
    if (r == C - 1) {
      if (!emb_rows) LSA_FAIL(c, LSA_ERR_INVALID_ARG, "seq %d: the entry completes chunk %d, emb_rows is required", b, ch);
      roll = any_done = true;
    }
  }
  if (roll) {
    // a completed chunk / a new tail changes what the side band reads (candidates, the staged table): let the side band
    // and earlier exports finish first.  Rare: twice per C entries.
    LSA_CUDA(c, cudaEventRecord(c->ev_roll, c->sf));
    LSA_CUDA(c, cudaStreamWaitEvent(c->sc, c->ev_roll, 0));
  }
  // Independent steps on the small-batch path: an append that only writes rows (no table entry, no new candidate) runs
  // BESIDE the previous attention launch - nothing in flight reads those rows unmasked - and the next launch waits for
  // SeqDev::grow_epoch instead of for the stream.  Everything else is stream-ordered (the next launch does not start early).
  const bool beside = !roll && c->cfg.step_overlap && c->attn_impl == LSA_ATTN_TCGEN05 && tc_small_supported(c->tc) && !c->no_small &&
                      !c->serialize_next && c->prof_cap == 0;
  for (int off = 0; off < n; off += kFireMax) {
    AppendList list{};
    list.n = std::min(kFireMax, n - off);
    for (int i = 0; i < list.n; ++i) {
      const int b = seq_ids[off + i];
      list.ids[i] = b;
      list.n_csa[i] = c->seq_host[b].n_csa;
      list.n_hca[i] = c->seq_host[b].n_hca;
      list.epoch[i] = ++c->grow_count[b];
    }
    LSA_CUDA(c, launch_append_compressed(c->cfg.dtype, c->d_seqs, c->pool, c->cfg.hot_pool, list, off, csa_k, csa_v, hca_k, hca_v, emb_rows,
                                         c->cfg.D, c->cfg.E, C, c->k, c->k_sel, c->page_bytes, c->sc, beside));
    c->attn_launches += 1;
  }
  if (beside) c->grow_wait_next = true;
  else c->serialize_next = true;                     // the next attention launch reads what these kernels wrote
  if (any_done) {
    LSA_CUDA(c, cudaEventRecord(c->ev_compute, c->sc));
    LSA_CUDA(c, cudaStreamWaitEvent(c->sf, c->ev_compute, 0));
  }
  for (int i = 0; i < n; ++i) {                     // host mirrors + export of completed chunks (P:179 direction)
    const int b = seq_ids[i];
    SeqDev& s = c->seq_host[b];
    if (hca_k) { s.n_hca += 1; c->hca_appended += 1; }
    if (!csa_k) continue;
    const int ch = (int)(s.n_csa / C), r = (int)(s.n_csa % C);
    if (r == 0) {
      c->n_tbl[c->cur_buf[b]][b] += 1;
      if (c->pending[b]) c->n_tbl[1 - c->cur_buf[b]][b] += 1;
    }
    s.n_csa += 1;
    c->csa_appended += 1;
    if (r == C - 1) {
      s.n_chunks = ch + 1;
      s.k_eff = std::min(c->k_sel, ch + 1);
      c->k_eff[b] = s.k_eff;
      const unsigned char* src = static_cast<const unsigned char*>(c->cfg.hot_pool) + (long long)(s.tier_page0 + (ch & 1)) * c->page_bytes;
      void* dst = const_cast<unsigned char*>(reinterpret_cast<const unsigned char*>(s.cold)) + (long long)ch * c->page_bytes;
      const int ctas = (int)std::max<long long>(1, std::min<long long>(c->fetch_ctas, (c->page_bytes + 16383) / 16384));
      LSA_CUDA(c, launch_export(src, dst, c->page_bytes, ctas, c->sf));
      c->index_launches += 1;
      c->chunks_exported += 1;
    }
  }
  return LSA_OK;
}

// ---- support --------------------------------------------------------------------------------------
extern "C" int lsa_set_chunk_emb(lsa_ctx* ctx, int32_t seq, const void* chunk_emb) {
  if (!ctx) return LSA_ERR_STATE;
  if (seq < 0 || seq >= ctx->B || !chunk_emb) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "bad seq / null chunk_emb");
  ctx->seq_host[seq].emb = chunk_emb;
  // ordered after every index launch already enqueued on the side band
  LSA_CUDA(ctx, cudaMemcpyAsync(reinterpret_cast<char*>(ctx->d_seqs + seq) + offsetof(SeqDev, emb), &ctx->seq_host[seq].emb,
                                sizeof(void*), cudaMemcpyHostToDevice, ctx->sf));
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sf));
  return LSA_OK;
}

extern "C" int lsa_sync(lsa_ctx* ctx) {
  if (!ctx) return LSA_ERR_STATE;
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sf));
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sc));
  unsigned long long err = 0;
  LSA_CUDA(ctx, cudaMemcpy(&err, ctx->pool.counters + C_ERROR, sizeof(err), cudaMemcpyDeviceToHost));
  if (err) LSA_FAIL(ctx, LSA_ERR_POOL_EXHAUSTED, "hot pool exhausted during a residency pass");
  return LSA_OK;
}

extern "C" int lsa_get_page_table(lsa_ctx* ctx, int32_t seq, int32_t which, int32_t* chunk_idx, int32_t* page, int32_t* n) {
  if (!ctx) return LSA_ERR_STATE;
  if (seq < 0 || seq >= ctx->B || (which != 0 && which != 1) || !chunk_idx || !page || !n)
    LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "bad argument");
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sf));
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sc));
  SeqDev d{};
  LSA_CUDA(ctx, cudaMemcpy(&d, ctx->d_seqs + seq, sizeof(SeqDev), cudaMemcpyDeviceToHost));
  int buf = which == 0 ? d.cur_buf : 1 - d.cur_buf;
  int cnt = (which == 1 && !d.pending) ? 0 : d.n_tbl[buf];
  *n = cnt;
  if (cnt > 0) {
    LSA_CUDA(ctx, cudaMemcpy(chunk_idx, ctx->pool.tbl_chunk + ((size_t)seq * 2 + buf) * ctx->k, sizeof(int) * cnt, cudaMemcpyDeviceToHost));
    LSA_CUDA(ctx, cudaMemcpy(page, ctx->pool.tbl_page + ((size_t)seq * 2 + buf) * ctx->k, sizeof(int) * cnt, cudaMemcpyDeviceToHost));
  }
  return LSA_OK;
}

extern "C" int lsa_get_residency(lsa_ctx* ctx, int32_t seq, int32_t* page_of) {
  if (!ctx) return LSA_ERR_STATE;
  if (seq < 0 || seq >= ctx->B || !page_of) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "bad argument");
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sf));
  const SeqDev& d = ctx->seq_host[seq];
  if (d.n_chunks > 0)
    LSA_CUDA(ctx, cudaMemcpy(page_of, ctx->pool.page_of + d.page_of_off, sizeof(int) * d.n_chunks, cudaMemcpyDeviceToHost));
  return LSA_OK;
}

extern "C" int lsa_get_stats(lsa_ctx* ctx, lsa_stats* out) {
  if (!ctx) return LSA_ERR_STATE;
  if (!out) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "null out");
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sf));
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sc));
  unsigned long long cnt[8];
  LSA_CUDA(ctx, cudaMemcpy(cnt, ctx->pool.counters, sizeof(cnt), cudaMemcpyDeviceToHost));
  memset(out, 0, sizeof(*out));
  out->triggers = cnt[C_TRIGGERS];
  out->hits = cnt[C_HITS];
  out->misses = cnt[C_MISSES];
  out->evictions = cnt[C_EVICTIONS];
  out->bytes_fetched = cnt[C_BYTES];
  out->pool_error = (int)cnt[C_ERROR];
  out->steps = ctx->n_steps;
  out->attn_launches = ctx->attn_launches;
  out->index_launches = ctx->index_launches;
  out->attn_impl = ctx->attn_impl;
  out->attn_ctas = ctx->last_attn_ctas;
  out->csa_appended = ctx->csa_appended;
  out->hca_appended = ctx->hca_appended;
  out->chunks_exported = ctx->chunks_exported;
  return LSA_OK;
}

extern "C" int lsa_get_step(lsa_ctx* ctx, int32_t seq, int64_t* step) {
  if (!ctx) return LSA_ERR_STATE;
  if (seq < 0 || seq >= ctx->B || !step) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "bad argument");
  *step = ctx->step[seq];
  return LSA_OK;
}

extern "C" int lsa_timeline_enable(lsa_ctx* ctx, int32_t on) {
  if (!ctx) return LSA_ERR_STATE;
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sc));
  if (on && !ctx->d_tl) {
    int rc = dev_alloc(ctx, &ctx->d_tl, (size_t)LSA_TL_LAUNCHES * LSA_TL_CTAS * LSA_TL_EVENTS);   // zeroed
    if (rc) return rc;
  }
  ctx->tl_on = on != 0;
  return LSA_OK;
}

extern "C" int lsa_timeline_read(lsa_ctx* ctx, uint64_t* dst, uint64_t* n_launches) {
  if (!ctx) return LSA_ERR_STATE;
  if (!dst) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "null dst");
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sf));
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sc));
  const size_t bytes = (size_t)LSA_TL_LAUNCHES * LSA_TL_CTAS * LSA_TL_EVENTS * sizeof(uint64_t);
  if (ctx->d_tl) LSA_CUDA(ctx, cudaMemcpy(dst, ctx->d_tl, bytes, cudaMemcpyDeviceToHost));
  else memset(dst, 0, bytes);
  if (n_launches) *n_launches = ctx->tl_seq;
  return LSA_OK;
}

extern "C" int lsa_profile_enable(lsa_ctx* ctx, int32_t capacity) {
  if (!ctx) return LSA_ERR_STATE;
  if (capacity < 0 || capacity > (1 << 20)) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "capacity out of range");
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sf));
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sc));
  for (int ph = 0; ph < LSA_PH_ATTENTION_DEV; ++ph) {
    while ((int)ctx->prof_ev[ph].size() < 2 * capacity) {
      cudaEvent_t e;
      LSA_CUDA(ctx, cudaEventCreate(&e));
      ctx->prof_ev[ph].push_back(e);
    }
    ctx->prof_n[ph] = 0;
  }
  if (capacity > ctx->ktime_cap) {
    int rc = dev_alloc(ctx, &ctx->d_ktime, (size_t)2 * capacity, false);
    if (rc) return rc;
    ctx->ktime_cap = capacity;
  }
  if (capacity > 0) {
    std::vector<unsigned long long> init((size_t)2 * capacity);
    for (int i = 0; i < capacity; ++i) { init[2 * i] = ~0ull; init[2 * i + 1] = 0ull; }
    LSA_CUDA(ctx, cudaMemcpy(ctx->d_ktime, init.data(), init.size() * sizeof(unsigned long long), cudaMemcpyHostToDevice));
  }
  ctx->prof_cap = capacity;
  return LSA_OK;
}

extern "C" int lsa_profile_read(lsa_ctx* ctx, double* ms_sum, int64_t* count) {
  if (!ctx) return LSA_ERR_STATE;
  if (!ms_sum || !count) LSA_FAIL(ctx, LSA_ERR_INVALID_ARG, "null output");
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sf));
  LSA_CUDA(ctx, cudaStreamSynchronize(ctx->sc));
  {                                                 // device-clock working time of the tcgen05 attention kernel
    const int n = ctx->d_ktime ? std::min(ctx->prof_n[LSA_PH_ATTENTION], ctx->ktime_cap) : 0;
    std::vector<unsigned long long> kt((size_t)2 * std::max(n, 1));
    if (n > 0) LSA_CUDA(ctx, cudaMemcpy(kt.data(), ctx->d_ktime, (size_t)2 * n * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
    double sum = 0;
    int cnt = 0;
    for (int i = 0; i < n; ++i)
      if (kt[2 * i] != ~0ull && kt[2 * i + 1] > kt[2 * i]) { sum += (double)(kt[2 * i + 1] - kt[2 * i]) * 1e-6; ++cnt; }
    ms_sum[LSA_PH_ATTENTION_DEV] = sum;
    count[LSA_PH_ATTENTION_DEV] = cnt;
    if (n > 0) {
      for (int i = 0; i < n; ++i) { kt[2 * i] = ~0ull; kt[2 * i + 1] = 0ull; }
      LSA_CUDA(ctx, cudaMemcpy(ctx->d_ktime, kt.data(), (size_t)2 * n * sizeof(unsigned long long), cudaMemcpyHostToDevice));
    }
  }
  for (int ph = 0; ph < LSA_PH_ATTENTION_DEV; ++ph) {
    double sum = 0;
    for (int i = 0; i < ctx->prof_n[ph]; ++i) {
      float ms = 0.f;
      LSA_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->prof_ev[ph][2 * i], ctx->prof_ev[ph][2 * i + 1]));
      sum += ms;
    }
    ms_sum[ph] = sum;
    count[ph] = ctx->prof_n[ph];
    ctx->prof_n[ph] = 0;
  }
  return LSA_OK;
}
