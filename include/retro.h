/* retro.h — C ABI of the B200-native (sm_100a) RetroAttention decode hot path.
 *
 * One decode step of retrospective sparse attention (arxiv 2508.09001, Alg. 1):
 *   S1 retro_update_page_bounds  page digests Kmin/Kmax
 *   S2 retro_select_pages        Eq. 1 page score + top-k + Alg. 2 mask
 *   S3 retro_sparse_attend       one fused GQA pass, current + w past queries (Eq. 2/6/7)
 *   S4 retro_merge_output_cache  LSE merge into the output cache              (Eq. 8-9; 83-85)
 *
 * Conventions (every function):
 *   - Returns RETRO_OK (0) or a negative RETRO_ERR_* code; retro_error_string() names it.
 *   - Unless a parameter is marked HOST, every pointer is a DEVICE pointer OWNED BY THE CALLER.  The library
 *     never allocates, frees or retains device memory, never synchronises and never copies to the host; all
 *     work is enqueued on `stream` (a cudaStream_t passed as void*, NULL = default stream) and is CUDA-graph
 *     capturable: every step-varying quantity (seq_lens, q_pos, budgets, cache_pos) lives in device memory
 *     and grids are sized from the descriptor's upper bounds only.
 *     (One documented exception: retro_debug_status in the RETRO_DEBUG_CHECKS build synchronises `stream` and
 *     reads two counters back.)
 *   - Host-side state kept by the library (per process, one mutex, safe to call from several threads): the last
 *     CUDA error, per-device facts (SM count, shared-memory limit), per-(device, kernel) shared-memory grants and
 *     resident-cluster capacities, and a 64-entry cache of TMA tensor-map descriptors keyed by the K/V pool
 *     addresses and shapes.  Nothing else survives a call.
 *   - Device pointers must be 16-byte aligned.  Validation is host-side only (null / shape / alignment); the debug
 *     build (libretro_dbg.so) adds device-side checks of every index the kernels consume.
 *   - `w` = desc->window counts PAST queries (the paper's window counts the current one: w_paper = w + 1);
 *     w = 0 is plain Quest sparse attention and needs no mask / cache buffers.
 *   - t_b = seq_lens[b] - 1 is the position of sequence b's current token.  "Decode step" and "position of the
 *     current token" are the same number, so the retrospective mask A stores positions.
 *
 * Layouts (row-major, innermost last; T = desc->dtype element, P = page_size, d = head_dim):
 *   k_pages, v_pages [num_phys_pages][h_k][P][d] T   each (page, KV head) tile is contiguous (4 KB for bf16 d128).
 *                                                   Slots at positions >= seq_len are never used: they may hold
 *                                                   anything (unwritten memory, NaN, Inf).  bf16 path: VALID V values
 *                                                   must satisfy |v| <= 65504 - the normalised partial of a KV split
 *                                                   (a convex combination of V rows) is handed to the split combine
 *                                                   as fp16; larger magnitudes overflow to Inf there.
 *   block_table      [B][max_pages_per_seq] int32   logical page j of sequence b -> physical page
 *   seq_lens         [B] int32                      tokens valid in sequence b, current token included
 *   bounds           [B][h_k][max_pages_per_seq][2][d] T   [..][0][:] = Kmax, [..][1][:] = Kmin
 *   last_loaded (A)  [B][h_k][max_pages_per_seq] int32     last position whose step loaded the page, -1 = never
 *   sel_pages        [B][h_k][max_sel_pages] int32  selected LOGICAL pages, ascending, -1 beyond sel_count
 *   sel_prev  (M)    [B][h_k][max_sel_pages] int32  A[page] before this step's update, -1 beyond sel_count
 *   sel_count        [B][h_k] int32
 *   q_cur            [B][h_q][d] T                  the current query (drives selection)
 *   q_win            [B][w+1][h_q][d] T             window rows in ANY order
 *   q_pos            [B][w+1] int32                 position of each row, -1 = empty row; the row whose position
 *                                                   is seq_lens[b]-1 is the current query; rows outside
 *                                                   [t-w, t] are treated as empty
 *   part_o           [B][w+1][h_q][d] float         normalised partial output of each row over its unseen pages
 *   part_lse         [B][w+1][h_q] float            natural-log sum-exp of the same; empty set -> o = 0, lse = -inf
 *   cache_o          [B][w][h_q][d] float           output cache ring, slot = position mod w; bf16 instead of float
 *                                                   with desc->cache_dtype == RETRO_BF16 (needs dtype RETRO_BF16):
 *                                                   the paper's footprint, 16-bit O + fp32 LSE (Eq. 12,
 *                                                   PAPER.md:502-507); merges run in fp32, the STORED row is rounded
 *   cache_lse        [B][w][h_q] float
 *   cache_pos        [B][w] int32                   position held by each slot, -1 = empty
 *   out              [B][w+1][h_q][d] T             merged outputs, row r belongs to q_pos[b][r]; empty rows = 0
 *   out_lse          [B][w+1][h_q] float            optional (may be NULL)
 */
#ifndef RETRO_H_
#define RETRO_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RETRO_OK 0
#define RETRO_ERR_ARG (-1)         /* null pointer, non-positive dim, h_q % h_k != 0, misaligned pointer      */
#define RETRO_ERR_UNSUPPORTED (-2) /* (dtype, head_dim, page_size) not instantiated, or a size limit exceeded */
#define RETRO_ERR_WORKSPACE (-3)   /* workspace smaller than retro_workspace_bytes()                          */
#define RETRO_ERR_CUDA (-4)        /* launch / runtime error; retro_last_cuda_error() returns the cudaError_t */

#define RETRO_F32 0
#define RETRO_BF16 1
#define RETRO_GROUP_SUM 0 /* Eq. 1 scores of a KV head's q heads are summed (default; reading Q2) */
#define RETRO_GROUP_MAX 1

/* Supported instantiations: {RETRO_F32, head_dim 64, page_size 16}, {RETRO_BF16, head_dim 128, page_size 16}.
 * Limits: window <= 32, group (h_q / h_k) <= 8, max_pages_per_seq <= 16384, batch <= 65535 (<= 64 for the
 * window-advance helpers). */
typedef struct retro_desc {
  int32_t batch;             /* B                                                              */
  int32_t num_q_heads;       /* h_q                                                            */
  int32_t num_kv_heads;      /* h_k, divides h_q                                               */
  int32_t head_dim;          /* d                                                              */
  int32_t page_size;         /* P tokens per page                                              */
  int32_t max_pages_per_seq; /* row stride of block_table / bounds / last_loaded               */
  int32_t max_sel_pages;     /* k_max: row stride of sel_pages / sel_prev, upper bound on k    */
  int32_t num_phys_pages;    /* pages in the K/V pools                                         */
  int32_t window;            /* w = number of PAST queries; 0 = plain Quest                    */
  int32_t dtype;             /* RETRO_F32 | RETRO_BF16: q, K, V, bounds, out                   */
  int32_t group_reduce;      /* RETRO_GROUP_SUM | RETRO_GROUP_MAX                              */
  int32_t force_last_page;   /* 1: newest page always selected and counted in k (reading Q3)   */
  float sm_scale;            /* softmax scale, 1/sqrt(head_dim)                  */
  int32_t cache_dtype;       /* RETRO_F32 (0, default) | RETRO_BF16: element type of cache_o   */
} retro_desc_t;

/* Bytes of scratch the S2/S3 entry points need for this descriptor (page scores, split-KV partials,
 * arrival counters).  HOST pointers.  The workspace must be passed to retro_workspace_init() once after
 * allocation; the library leaves it consistent after every call. */
int retro_workspace_bytes(const retro_desc_t* desc /*HOST*/, size_t* bytes /*HOST out*/);
int retro_workspace_init(const retro_desc_t* desc /*HOST*/, void* workspace, size_t ws_bytes, void* stream);

const char* retro_error_string(int code);
int retro_last_cuda_error(void);
int retro_version(void);

/* S1.  For every sequence b, recompute the digests of the logical pages that overlap positions
 * [pos_begin[b], seq_lens[b]): per channel, max and min of K over the page's VALID tokens (l < seq_len).
 * At most `max_touched_pages` pages per sequence are updated, starting at page pos_begin[b] / P (HOST int:
 * 1 for a decode step with pos_begin = seq_len - 1; max_pages_per_seq for a rebuild after prefill).
 * pos_begin == NULL means pos_begin[b] = seq_lens[b] - 1 (only the newest token's page).
 * Bit-exact: min/max of T values is a T value. */
int retro_update_page_bounds(const retro_desc_t* desc, const void* k_pages, const int32_t* block_table,
                             const int32_t* seq_lens, const int32_t* pos_begin /*[B]*/,
                             int32_t max_touched_pages /*HOST*/, void* bounds, void* stream);

/* S2 (Eq. 1; top-k PAPER.md:42, 248; Alg. 2).  Per (b, KV head):
 * score_j = reduce over the head's q heads g of sum_c max(q_gc * Kmin_jc, q_gc * Kmax_jc).  The ranking is the one
 * of the fp64 scores: the digest stream is scored in fp32 next to a proven bound on the fp32 error, and the pages the
 * bound cannot decide are re-scored in fp64 and ranked exactly (reading Q7);
 * k = min(budget_pages[b], #pages, max_sel_pages); k == #pages selects every page, else the newest page (if
 * force_last_page) plus the best of the others ordered by (score desc, index asc); emitted ascending.
 * Then M_i = A[page_i] -> sel_prev and A[page_i] = seq_lens[b] - 1.  last_loaded may be NULL iff window == 0
 * (sel_prev is then filled with -1).  scores_out (optional, [B][h_k][max_pages_per_seq] double, -inf for pages
 * that do not exist) exposes the fp64 scores for tests. */
int retro_select_pages(const retro_desc_t* desc, const void* q_cur, const void* bounds, const int32_t* seq_lens,
                       const int32_t* budget_pages /*[B]*/, int32_t* last_loaded, int32_t* sel_pages,
                       int32_t* sel_prev, int32_t* sel_count, double* scores_out, void* workspace,
                       size_t ws_bytes, void* stream);

/* S3 (Eq. 2 / 6 / 7; Alg. 1 line 6).  For every non-empty window row r at position p and
 * every q head: softmax(q K^T * sm_scale) V over the tokens l of the selected pages j with sel_prev_j < p (page
 * not yet seen by that query), l <= p and l < seq_len.  The current row (p = t) sees all of S_t (O_org); a past
 * row sees only its unseen pages (O_sup).  Each selected page is read from HBM once and serves every row of the
 * GQA group x (w+1) block.  fp32 accumulation and softmax.  A pure function of its inputs. */
int retro_sparse_attend(const retro_desc_t* desc, const void* q_win, const int32_t* q_pos, const void* k_pages,
                        const void* v_pages, const int32_t* block_table, const int32_t* seq_lens,
                        const int32_t* sel_pages, const int32_t* sel_prev, const int32_t* sel_count,
                        float* part_o, float* part_lse, void* workspace, size_t ws_bytes, void* stream);

/* S4 (Eq. 8-9 with alpha = e^lse; push / update / pop; Alg. 1 lines 7-8).
 * Past row at position p (t-w <= p < t): (o, lse) = merge(cache[p mod w] if cache_pos == p, part); emitted to
 * `out`; written back to its slot unless p = t-w (popped after its last merge).  Current row: out = part, pushed
 * into slot t mod w.  window == 0: out = part, cache_* may be NULL. */
int retro_merge_output_cache(const retro_desc_t* desc, const float* part_o, const float* part_lse,
                             const int32_t* q_pos, const int32_t* seq_lens, void* cache_o, float* cache_lse,
                             int32_t* cache_pos, void* out, float* out_lse, void* stream);

/* AppendKV (Alg. 1 line 3).  Writes k_new / v_new [B][h_k][d] T into position seq_lens[b] - 1 of
 * each sequence (seq_lens already counts the new token).  Capacity: a sequence holds at most
 * max_pages_per_seq * page_size tokens; positions beyond that are never written (every kernel clamps its page count
 * to max_pages_per_seq), and the window-advance helpers below leave the length of a full sequence unchanged (it is
 * not advanced: check seq_lens before appending to it - retro_decode_step_host skips the append itself). */
int retro_append_kv(const retro_desc_t* desc, const void* k_new, const void* v_new, const int32_t* block_table,
                    const int32_t* seq_lens, void* k_pages, void* v_pages, void* stream);

/* One layer's persistent device state, for the whole-step entry points below. */
typedef struct retro_layer_state {
  void* k_pages;
  void* v_pages;
  int32_t* block_table;
  int32_t* seq_lens;
  int32_t* budget_pages; /* [B] */
  void* bounds;
  int32_t* last_loaded;
  int32_t* sel_pages;
  int32_t* sel_prev;
  int32_t* sel_count;
  float* part_o;
  float* part_lse;
  void* cache_o;         /* float or bf16, see cache_dtype */
  float* cache_lse;
  int32_t* cache_pos;
  void* workspace;
  size_t workspace_bytes;
} retro_layer_state_t;

/* S1..S4 of Alg. 1 back to back on `stream` for one layer (digest refresh of the newest page, select, attend,
 * merge).  seq_lens already counts the current token.  Same results as the four calls above. */
int retro_decode_step(const retro_desc_t* desc, const retro_layer_state_t* st /*HOST struct of device ptrs*/,
                      const void* q_win, const int32_t* q_pos, const void* q_cur, void* out, float* out_lse,
                      void* stream);

/* Measurement helpers.  retro_decode_step_part enqueues ONE of the step's kernels exactly as retro_decode_step
 * does: part 0 = S1 + S2 (select kernel, newest page's digest rebuilt in line), part 1 = S3 + S4 (attend kernel
 * with the split combine and the cache merge in its epilogue; S3 then S4 as two launches where the fusion does not
 * apply: fp32, or more than 128 query rows per KV head).  retro_launches_per_step: kernels retro_decode_step
 * enqueues for this descriptor (2 or 3). */
int retro_decode_step_part(const retro_desc_t* desc, const retro_layer_state_t* st, const void* q_win,
                           const int32_t* q_pos, const void* q_cur, void* out, float* out_lse, int32_t part /*HOST*/,
                           void* stream);
int retro_launches_per_step(const retro_desc_t* desc /*HOST*/, int32_t* launches /*HOST out*/);

/* Debug build.  Compiled with -DRETRO_DEBUG_CHECKS (paper_2508_09001_b200/lib/libretro_dbg.so) the kernels validate
 * the caller-supplied indices on the device - sel_pages entries against the sequence's page count, block_table entries
 * against num_phys_pages, sel_count, seq_lens, budget_pages, q_pos - count the violations in the workspace, and
 * neutralise the offending entry (an invalid page is treated as already seen by every row) instead of reading out
 * of bounds.  retro_debug_status reports enabled (0 in the release build, where the counts read 0 and nothing is
 * synchronised), the violations since retro_workspace_init and the code of the last one (1 sel_pages, 2 block_table,
 * 3 q_pos, 4 seq_lens, 5 budget_pages, 6 sel_count).  enabled / violations / last_code: HOST out.  In the debug build
 * this call SYNCHRONISES `stream` (the one exception to the conventions above). */
int retro_debug_status(const retro_desc_t* desc, const void* workspace, size_t ws_bytes, int32_t* enabled /*HOST*/,
                       uint32_t* violations /*HOST*/, uint32_t* last_code /*HOST*/, void* stream);

/* End-to-end step with HOST buffers (pinned for async copies): ONE host->device copy of this step's packed
 * inputs host_qkv_new = [q_new [B][h_q][d] | k_new [B][h_k][d] | v_new [B][h_k][d]] (T), one launch that advances
 * seq_lens and the query window ring and appends the token to the KV pool, retro_decode_step, and ONE device->host
 * copy of out [B][w+1][h_q][d].  Five stream operations, CUDA-graph capturable (the host addresses are baked into a
 * captured graph: refill the same pinned buffers before every replay).  dev_io holds caller-owned device staging
 * buffers; batch <= 64. */
typedef struct retro_step_io {
  void* qkv_new;    /* device [q_new | k_new | v_new] T, packed as above */
  void* q_win;      /* device [B][w+1][h_q][d] T ring                   */
  int32_t* q_pos;   /* device [B][w+1]                                  */
  void* out;        /* device [B][w+1][h_q][d] T                        */
} retro_step_io_t;
int retro_decode_step_host(const retro_desc_t* desc, const retro_layer_state_t* st, const retro_step_io_t* dev_io,
                           const void* host_qkv_new /*HOST*/, void* host_out /*HOST*/, void* stream);

/* The same for n_layers layers of one decode step with ONE copy in and ONE copy out: host_qkv_new
 * [n_layers][q | k | v], host_out [n_layers][B][w+1][h_q][d].  states / dev_ios: HOST arrays of n_layers records;
 * the records' qkv_new (and out) device buffers must be consecutive slices of one device buffer
 * (dev_ios[l].qkv_new == dev_ios[0].qkv_new + l * token bytes; likewise out), else RETRO_ERR_ARG. */
int retro_decode_steps_host(const retro_desc_t* desc, const retro_layer_state_t* states /*HOST*/,
                            const retro_step_io_t* dev_ios /*HOST*/, int32_t n_layers /*HOST*/,
                            const void* host_qkv_new /*HOST*/, void* host_out /*HOST*/, void* stream);

/* NEXT-1: UpdateKV of Alg. 1 line 2 (Sec. 2.4): overwrite the K
 * and V rows of up to n_upd past tokens per sequence with the caller's re-embedded K^, V^.
 * positions [B][n_upd] int32 (-1 or >= seq_len: skipped), k_hat / v_hat [B][n_upd][h_k][d] T, all DEVICE.
 * The digests of the touched pages become stale: follow with
 * retro_update_page_bounds(pos_begin = oldest overwritten position, max_touched_pages = ceil(w / P) + 1). */
int retro_update_kv(const retro_desc_t* desc, const void* k_hat, const void* v_hat, const int32_t* positions,
                    int32_t n_upd /*HOST*/, const int32_t* block_table, const int32_t* seq_lens, void* k_pages,
                    void* v_pages, void* stream);

/* NEXT-2.  Relative budget policy on the device (budget = 0.15 x context length,
 * at least 256 tokens, re-evaluated every step): budget_pages[b] = max(1, max(min_tokens,
 * seq_lens[b] * ratio_permille / 1000) / page_size), integer arithmetic.  seq_lens, budget_pages: DEVICE [B]. */
int retro_budget_policy(const retro_desc_t* desc, const int32_t* seq_lens, int32_t ratio_permille /*HOST*/,
                        int32_t min_tokens /*HOST*/, int32_t* budget_pages, void* stream);

/* NEXT-2: Alg. 2 on its own, for a page set S_t chosen by another selector (the method is
 * selector-agnostic): for every page p of sel_pages[b][h][0..sel_count): sel_prev <- A[p];
 * A[p] <- t (t = seq_lens[b] - 1); entries past sel_count get -1.  Pages of one (b, h) list must be distinct.
 * Follow with retro_sparse_attend and retro_merge_output_cache.  All pointers DEVICE. */
int retro_build_mask(const retro_desc_t* desc, const int32_t* sel_pages, const int32_t* sel_count,
                     const int32_t* seq_lens, int32_t* last_loaded, int32_t* sel_prev, void* stream);

/* NEXT-4: per-step diagnostics of the retrospective rows, computed from the outputs of
 * retro_select_pages / retro_sparse_attend / retro_merge_output_cache of the SAME step (call it after the merge):
 *   supp_pages[b][h][r] = number of this step's selected pages that window row r reads (sel_prev_j < q_pos[b][r]
 *       and first token of the page <= q_pos[b][r]); for the current row this is the pages it can see.  Summed
 *       over the steps a query stays in the window it is that query's EFFECTIVE KV budget in pages.
 *   supp_mass[b][r][g] = exp(part_lse - out_lse): the share of the row's merged softmax mass contributed by this
 *       step's pages (supplementary attention); 1 for the current row, 0 for an empty partial.
 * Rows with q_pos = -1 (or outside [t - w, t]) give 0.  supp_pages [B][h_k][w+1] int32, supp_mass [B][w+1][h_q]
 * f32, all DEVICE.  Not part of retro_decode_step; one small launch. */
int retro_step_diagnostics(const retro_desc_t* desc, const int32_t* sel_pages, const int32_t* sel_prev,
                           const int32_t* sel_count, const int32_t* q_pos, const int32_t* seq_lens,
                           const float* part_lse, const float* out_lse, int32_t* supp_pages, float* supp_mass,
                           void* stream);

/* Window-ring bookkeeping used by the two calls above and by the synthetic benchmark: seq_lens[b] += 1;
 * row (new position mod (w+1)) of q_win <- q_new[b], q_pos <- new position.  q_new [B][h_q][d] T.
 * If step_counter != NULL, q_new is taken as q_pool[(*step_counter) % pool_steps] ([pool][B][h_q][d]) and the
 * counter is incremented (lets a captured CUDA graph replay successive steps of a pre-generated query stream). */
int retro_window_advance(const retro_desc_t* desc, const void* q_new_or_pool, int32_t* step_counter,
                         int32_t pool_steps /*HOST*/, int32_t* seq_lens, void* q_win, int32_t* q_pos,
                         void* q_cur_out /*optional [B][h_q][d]*/, void* stream);

/* The same bookkeeping for n_layers independent layers in ONE launch (one CTA per layer).  Used by the synthetic
 * benchmark, where every layer's pre-generated query stream advances at the start of a step - the stand-in for
 * the QKV projections that feed this path in a model.  `table` is a DEVICE array of n_layers records of DEVICE
 * pointers; every layer uses `desc`'s shapes and a query pool of pool_steps steps. */
typedef struct retro_advance_rec {
  const void* q_pool;     /* [pool_steps][B][h_q][d] T */
  int32_t* step_counter;  /* [1]                       */
  int32_t* seq_lens;      /* [B]                       */
  void* q_win;            /* [B][w+1][h_q][d] T        */
  int32_t* q_pos;         /* [B][w+1]                  */
  void* q_cur_out;        /* [B][h_q][d] T, may be NULL */
} retro_advance_rec_t;
int retro_window_advance_layers(const retro_desc_t* desc, const retro_advance_rec_t* table /*DEVICE*/,
                                int32_t n_layers, int32_t pool_steps /*HOST*/, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* RETRO_H_ */
