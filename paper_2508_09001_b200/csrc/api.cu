// C ABI of libretro (include/retro.h): host-side validation, workspace layout, entry points.
#include <atomic>

#include "common.cuh"

// -DRETRO_NVTX (lib/libretro_nvtx.so): every entry point that enqueues work is an NVTX range named after itself, so a
// timeline tool shows the host side of a step (validation, launch calls) next to the kernels.  Header-only NVTX 3:
// nothing is linked and the calls are no-ops until a tool attaches.  The release build compiles the macro away.
#ifdef RETRO_NVTX
#include <nvtx3/nvToolsExt.h>
namespace {
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
  NvtxRange(const NvtxRange&) = delete;
  NvtxRange& operator=(const NvtxRange&) = delete;
};
}  // namespace
#define RETRO_RANGE(name) NvtxRange nvtx_range__(name)
#else
#define RETRO_RANGE(name) do {} while (0)
#endif

namespace retro {

static std::atomic<int> g_last_cuda_error{0};
void set_cuda_error(cudaError_t e) { g_last_cuda_error.store((int)e); }
std::mutex& host_mutex() {
  static std::mutex m;
  return m;
}

DeviceInfo device_info() {
  constexpr int kMaxDev = 64;
  static DeviceInfo table[kMaxDev];
  static bool known[kMaxDev];
  DeviceInfo fallback{-1, 148, 232448};   // B200; used when no device is present (CPU-only symbol / header tests)
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0) {
    (void)cudaGetLastError();
    return fallback;
  }
  std::lock_guard<std::mutex> lock(host_mutex());
  if (dev < kMaxDev && known[dev]) return table[dev];
  DeviceInfo di{dev, 148, 232448};
  int v = 0;
  if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) di.sm_count = v;
  if (cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) == cudaSuccess && v > 0)
    di.max_smem_optin = v;
  if (dev < kMaxDev) { table[dev] = di; known[dev] = true; }
  return di;
}

int ensure_dynamic_smem(const void* kern, size_t smem_bytes, bool max_carveout) {
  if (smem_bytes <= 48 * 1024 && !max_carveout) return RETRO_OK;
  struct Entry { int dev; const void* kern; size_t granted; };
  constexpr int kEntries = 256;
  static Entry tab[kEntries];
  static int n_used = 0;
  int dev = 0;
  RETRO_CUDA_TRY(cudaGetDevice(&dev));
  std::lock_guard<std::mutex> lock(host_mutex());
  Entry* e = nullptr;
  for (int i = 0; i < n_used && e == nullptr; ++i)
    if (tab[i].dev == dev && tab[i].kern == kern) e = &tab[i];
  if (e != nullptr && e->granted >= smem_bytes) return RETRO_OK;
  RETRO_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes));
  if (max_carveout)
    RETRO_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout,
                                        cudaSharedmemCarveoutMaxShared));
  if (e == nullptr && n_used < kEntries) e = &tab[n_used++];   // table full: the attribute is simply set again
  if (e != nullptr) { e->dev = dev; e->kern = kern; e->granted = smem_bytes; }
  return RETRO_OK;
}

int max_active_clusters(const void* kern, int block_threads, size_t smem_bytes, int cluster_x) {
  struct Entry { int dev; const void* kern; size_t smem; int cluster; int max_active; };
  constexpr int kEntries = 512;
  static Entry tab[kEntries];
  static int n_used = 0;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return 0; }
  {
    std::lock_guard<std::mutex> lock(host_mutex());
    for (int i = 0; i < n_used; ++i)
      if (tab[i].dev == dev && tab[i].kern == kern && tab[i].smem == smem_bytes && tab[i].cluster == cluster_x)
        return tab[i].max_active;
  }
  int max_active = 0;
  bool ok = ensure_dynamic_smem(kern, smem_bytes) == RETRO_OK;   // (only ever raises the kernel's limit)
  if (ok && cluster_x > 8)
    ok = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess;
  if (ok) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cluster_x, 1, 1);
    cfg.blockDim = dim3(block_threads);
    cfg.dynamicSmemBytes = smem_bytes;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cluster_x;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    ok = cudaOccupancyMaxActiveClusters(&max_active, kern, &cfg) == cudaSuccess;
  }
  if (!ok) { (void)cudaGetLastError(); max_active = 0; }
  std::lock_guard<std::mutex> lock(host_mutex());
  if (n_used < kEntries) tab[n_used++] = Entry{dev, kern, smem_bytes, cluster_x, max_active};
  return max_active;
}

int validate_desc(const retro_desc_t* d) {
  if (d == nullptr) return RETRO_ERR_ARG;
  if (d->batch <= 0 || d->num_q_heads <= 0 || d->num_kv_heads <= 0 || d->head_dim <= 0 || d->page_size <= 0 ||
      d->max_pages_per_seq <= 0 || d->max_sel_pages < 1 || d->num_phys_pages <= 0 || d->window < 0)
    return RETRO_ERR_ARG;
  if (d->num_q_heads % d->num_kv_heads != 0) return RETRO_ERR_ARG;
  if (d->group_reduce != RETRO_GROUP_SUM && d->group_reduce != RETRO_GROUP_MAX) return RETRO_ERR_ARG;
  if (d->cache_dtype != RETRO_F32 && d->cache_dtype != RETRO_BF16) return RETRO_ERR_ARG;
  if (d->cache_dtype == RETRO_BF16 && d->dtype != RETRO_BF16) return RETRO_ERR_UNSUPPORTED;
  if (!(d->sm_scale > 0.f)) return RETRO_ERR_ARG;
  const bool f32 = d->dtype == RETRO_F32 && d->head_dim == 64 && d->page_size == 16;
  const bool bf16 = d->dtype == RETRO_BF16 && d->head_dim == 128 && d->page_size == 16;
  if (!f32 && !bf16) return RETRO_ERR_UNSUPPORTED;
  if (d->window > kMaxWindow || d->num_q_heads / d->num_kv_heads > kMaxGroup ||
      d->max_pages_per_seq > kMaxPagesPerSeq || d->batch > 65535)
    return RETRO_ERR_UNSUPPORTED;
  return RETRO_OK;
}

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

WorkspaceLayout workspace_layout(const retro_desc_t* d) {
  WorkspaceLayout wl;
  const int units = d->batch * d->num_kv_heads;
  wl.rows = (d->window + 1) * (d->num_q_heads / d->num_kv_heads);
  // split-KV.  Scalar path: units * nsplit covers the SMs about twice, at least 2 pages per split.  The
  // tensor-core path (bf16) consumes pages in blocks of 8; the splits of a (unit, row group) are the CTAs of one
  // thread-block cluster (<= 8) that combine their partials through distributed shared memory, and the grid
  // (units x row groups x splits) is at most ONE wave of resident CTAs (one CTA per SM).  More than 128 query
  // rows are handled as row groups of whole window ranks (G rows each).
  const bool umma = d->dtype == RETRO_BF16;
  const int sm_count = device_info().sm_count;
  const int G = d->num_q_heads / d->num_kv_heads, R = d->window + 1;
  wl.nrg = umma ? ceil_div(wl.rows, 128) : 1;
  wl.rg_ranks = ceil_div(R, wl.nrg);
  while (umma && wl.rg_ranks * G > 128) { ++wl.nrg; wl.rg_ranks = ceil_div(R, wl.nrg); }
  int nsplit = umma ? sm_count / (units * wl.nrg) : ceil_div(2 * sm_count, units);
  if (umma) {
    // the largest split count whose clusters (one per unit and row group) are all resident at once: the device
    // keeps fewer CTAs resident in large clusters (B200, one CTA per SM: 74 x 2, 33 x 4, 22 x 6, 15 x 8)
    if (nsplit > 8) nsplit = 8;
    const int nch = ceil_div(wl.rg_ranks * G, 16);
    while (nsplit > 1 && umma_max_active_clusters(nch, nsplit) < units * wl.nrg) --nsplit;
  }
  const int min_pages = umma ? 8 : 2;
  const int max_split = d->max_sel_pages >= min_pages ? d->max_sel_pages / min_pages : 1;
  if (nsplit > max_split) nsplit = max_split;
  if (nsplit < 1) nsplit = 1;
  wl.pages_per_split = ceil_div(d->max_sel_pages, nsplit);
  if (umma) wl.pages_per_split = ceil_div(wl.pages_per_split, 8) * 8;
  // the page list of a split lives in shared memory (<= 2048 pages x 8 splits = the 16 384-page limit); the
  // scalar path's list is capped the same way and takes more splits instead
  if (wl.pages_per_split > 2048) wl.pages_per_split = 2048;
  wl.nsplit = ceil_div(d->max_sel_pages, wl.pages_per_split);
  if (umma && wl.nsplit > 8) wl.nsplit = 8;   // (unreachable within the limits of validate_desc)
  size_t off = 0;
  wl.scores_off = off;
  off = align_up(off + (size_t)units * d->max_pages_per_seq * sizeof(double), 256);
  wl.amb_idx_off = off;
  off = align_up(off + (size_t)units * d->max_pages_per_seq * sizeof(int32_t), 256);
  wl.split_o_off = off;
  off = align_up(off + (size_t)units * wl.nsplit * wl.rows * d->head_dim * sizeof(float), 256);
  wl.split_lse_off = off;
  off = align_up(off + (size_t)units * wl.nsplit * wl.rows * sizeof(float), 256);
  wl.debug_off = off;     // (zeroed by retro_workspace_init together with the counters after it)
  off = align_up(off + 2 * sizeof(unsigned int), 256);
  wl.counters_off = off;
  off = align_up(off + (size_t)4 * units * sizeof(unsigned int), 256);
  wl.slot_counters_off = off;   // (zeroed by retro_workspace_init together with the counters before it)
  off = align_up(off + (size_t)d->batch * (d->window + 1) * sizeof(unsigned int), 256);
  wl.total = off;
  return wl;
}

}  // namespace retro

using namespace retro;

#define RETRO_CHECK_DESC(d)              \
  do {                                   \
    const int rc__ = validate_desc(d);   \
    if (rc__ != RETRO_OK) return rc__;   \
  } while (0)
#define RETRO_CHECK_PTR(p) \
  if ((p) == nullptr || !aligned16(p)) return RETRO_ERR_ARG

extern "C" {

int retro_version(void) { return 100; }

const char* retro_error_string(int code) {
  switch (code) {
    case RETRO_OK: return "ok";
    case RETRO_ERR_ARG: return "invalid argument (null / misaligned pointer or bad dimension)";
    case RETRO_ERR_UNSUPPORTED: return "unsupported (dtype, head_dim, page_size) combination or size limit";
    case RETRO_ERR_WORKSPACE: return "workspace too small";
    case RETRO_ERR_CUDA: return "CUDA error (see retro_last_cuda_error)";
    default: return "unknown error code";
  }
}

int retro_last_cuda_error(void) { return g_last_cuda_error.load(); }

int retro_workspace_bytes(const retro_desc_t* desc, size_t* bytes) {
  RETRO_CHECK_DESC(desc);
  if (bytes == nullptr) return RETRO_ERR_ARG;
  *bytes = workspace_layout(desc).total;
  return RETRO_OK;
}

int retro_workspace_init(const retro_desc_t* desc, void* workspace, size_t ws_bytes, void* stream) {
  RETRO_RANGE("retro_workspace_init");
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(workspace);
  const WorkspaceLayout wl = workspace_layout(desc);
  if (ws_bytes < wl.total) return RETRO_ERR_WORKSPACE;
  RETRO_CUDA_TRY(cudaMemsetAsync(static_cast<char*>(workspace) + wl.debug_off, 0, wl.total - wl.debug_off,
                                 (cudaStream_t)stream));
  return RETRO_OK;
}

int retro_update_page_bounds(const retro_desc_t* desc, const void* k_pages, const int32_t* block_table,
                             const int32_t* seq_lens, const int32_t* pos_begin, int32_t max_touched_pages,
                             void* bounds, void* stream) {
  RETRO_RANGE("retro_update_page_bounds");
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(k_pages); RETRO_CHECK_PTR(block_table); RETRO_CHECK_PTR(seq_lens); RETRO_CHECK_PTR(bounds);
  if (pos_begin != nullptr && !aligned16(pos_begin)) return RETRO_ERR_ARG;
  if (max_touched_pages < 1) return RETRO_ERR_ARG;
  return launch_update_page_bounds(desc, k_pages, block_table, seq_lens, pos_begin, max_touched_pages, bounds,
                                   (cudaStream_t)stream);
}

int retro_select_pages(const retro_desc_t* desc, const void* q_cur, const void* bounds, const int32_t* seq_lens,
                       const int32_t* budget_pages, int32_t* last_loaded, int32_t* sel_pages, int32_t* sel_prev,
                       int32_t* sel_count, double* scores_out, void* workspace, size_t ws_bytes, void* stream) {
  RETRO_RANGE("retro_select_pages");
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(q_cur); RETRO_CHECK_PTR(bounds); RETRO_CHECK_PTR(seq_lens); RETRO_CHECK_PTR(budget_pages);
  RETRO_CHECK_PTR(sel_pages); RETRO_CHECK_PTR(sel_prev); RETRO_CHECK_PTR(sel_count); RETRO_CHECK_PTR(workspace);
  if (last_loaded == nullptr && desc->window != 0) return RETRO_ERR_ARG;
  if (last_loaded != nullptr && !aligned16(last_loaded)) return RETRO_ERR_ARG;
  if (scores_out != nullptr && !aligned16(scores_out)) return RETRO_ERR_ARG;
  const WorkspaceLayout wl = workspace_layout(desc);
  if (ws_bytes < wl.total) return RETRO_ERR_WORKSPACE;
  return launch_select_pages(desc, wl, q_cur, bounds, seq_lens, budget_pages, last_loaded, sel_pages, sel_prev,
                             sel_count, scores_out, workspace, (cudaStream_t)stream);
}

int retro_sparse_attend(const retro_desc_t* desc, const void* q_win, const int32_t* q_pos, const void* k_pages,
                        const void* v_pages, const int32_t* block_table, const int32_t* seq_lens,
                        const int32_t* sel_pages, const int32_t* sel_prev, const int32_t* sel_count, float* part_o,
                        float* part_lse, void* workspace, size_t ws_bytes, void* stream) {
  RETRO_RANGE("retro_sparse_attend");
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(q_win); RETRO_CHECK_PTR(q_pos); RETRO_CHECK_PTR(k_pages); RETRO_CHECK_PTR(v_pages);
  RETRO_CHECK_PTR(block_table); RETRO_CHECK_PTR(seq_lens); RETRO_CHECK_PTR(sel_pages); RETRO_CHECK_PTR(sel_prev);
  RETRO_CHECK_PTR(sel_count); RETRO_CHECK_PTR(part_o); RETRO_CHECK_PTR(part_lse); RETRO_CHECK_PTR(workspace);
  const WorkspaceLayout wl = workspace_layout(desc);
  if (ws_bytes < wl.total) return RETRO_ERR_WORKSPACE;
  return launch_sparse_attend(desc, wl, q_win, q_pos, k_pages, v_pages, block_table, seq_lens, sel_pages, sel_prev,
                              sel_count, part_o, part_lse, workspace, (cudaStream_t)stream);
}

int retro_merge_output_cache(const retro_desc_t* desc, const float* part_o, const float* part_lse,
                             const int32_t* q_pos, const int32_t* seq_lens, void* cache_o, float* cache_lse,
                             int32_t* cache_pos, void* out, float* out_lse, void* stream) {
  RETRO_RANGE("retro_merge_output_cache");
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(part_o); RETRO_CHECK_PTR(part_lse); RETRO_CHECK_PTR(q_pos); RETRO_CHECK_PTR(seq_lens);
  RETRO_CHECK_PTR(out);
  if (desc->window > 0) { RETRO_CHECK_PTR(cache_o); RETRO_CHECK_PTR(cache_lse); RETRO_CHECK_PTR(cache_pos); }
  if (out_lse != nullptr && !aligned16(out_lse)) return RETRO_ERR_ARG;
  return launch_merge_output_cache(desc, part_o, part_lse, q_pos, seq_lens, cache_o, cache_lse, cache_pos, out,
                                   out_lse, (cudaStream_t)stream);
}

int retro_append_kv(const retro_desc_t* desc, const void* k_new, const void* v_new, const int32_t* block_table,
                    const int32_t* seq_lens, void* k_pages, void* v_pages, void* stream) {
  RETRO_RANGE("retro_append_kv");
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(k_new); RETRO_CHECK_PTR(v_new); RETRO_CHECK_PTR(block_table); RETRO_CHECK_PTR(seq_lens);
  RETRO_CHECK_PTR(k_pages); RETRO_CHECK_PTR(v_pages);
  return launch_append_kv(desc, k_new, v_new, block_table, seq_lens, k_pages, v_pages, (cudaStream_t)stream);
}

int retro_window_advance(const retro_desc_t* desc, const void* q_new_or_pool, int32_t* step_counter,
                         int32_t pool_steps, int32_t* seq_lens, void* q_win, int32_t* q_pos, void* q_cur_out,
                         void* stream) {
  RETRO_RANGE("retro_window_advance");
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(q_new_or_pool); RETRO_CHECK_PTR(seq_lens); RETRO_CHECK_PTR(q_win); RETRO_CHECK_PTR(q_pos);
  if (step_counter != nullptr && pool_steps < 1) return RETRO_ERR_ARG;
  if (q_cur_out != nullptr && !aligned16(q_cur_out)) return RETRO_ERR_ARG;
  return launch_window_advance(desc, q_new_or_pool, step_counter, pool_steps, seq_lens, q_win, q_pos, q_cur_out,
                               (cudaStream_t)stream);
}

int retro_budget_policy(const retro_desc_t* desc, const int32_t* seq_lens, int32_t ratio_permille, int32_t min_tokens,
                        int32_t* budget_pages, void* stream) {
  RETRO_RANGE("retro_budget_policy");
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(seq_lens); RETRO_CHECK_PTR(budget_pages);
  if (ratio_permille < 0 || min_tokens < 0) return RETRO_ERR_ARG;
  return launch_budget_policy(desc, seq_lens, ratio_permille, min_tokens, budget_pages, (cudaStream_t)stream);
}

int retro_build_mask(const retro_desc_t* desc, const int32_t* sel_pages, const int32_t* sel_count,
                     const int32_t* seq_lens, int32_t* last_loaded, int32_t* sel_prev, void* stream) {
  RETRO_RANGE("retro_build_mask");
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(sel_pages); RETRO_CHECK_PTR(sel_count); RETRO_CHECK_PTR(seq_lens); RETRO_CHECK_PTR(last_loaded);
  RETRO_CHECK_PTR(sel_prev);
  return launch_build_mask(desc, sel_pages, sel_count, seq_lens, last_loaded, sel_prev, (cudaStream_t)stream);
}

int retro_step_diagnostics(const retro_desc_t* desc, const int32_t* sel_pages, const int32_t* sel_prev,
                           const int32_t* sel_count, const int32_t* q_pos, const int32_t* seq_lens,
                           const float* part_lse, const float* out_lse, int32_t* supp_pages, float* supp_mass,
                           void* stream) {
  RETRO_RANGE("retro_step_diagnostics");
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(sel_pages); RETRO_CHECK_PTR(sel_prev); RETRO_CHECK_PTR(sel_count); RETRO_CHECK_PTR(q_pos);
  RETRO_CHECK_PTR(seq_lens); RETRO_CHECK_PTR(part_lse); RETRO_CHECK_PTR(out_lse); RETRO_CHECK_PTR(supp_pages);
  RETRO_CHECK_PTR(supp_mass);
  if (desc->num_q_heads / desc->num_kv_heads > 32) return RETRO_ERR_UNSUPPORTED;
  return launch_step_diagnostics(desc, sel_pages, sel_prev, sel_count, q_pos, seq_lens, part_lse, out_lse,
                                 supp_pages, supp_mass, (cudaStream_t)stream);
}

int retro_update_kv(const retro_desc_t* desc, const void* k_hat, const void* v_hat, const int32_t* positions,
                    int32_t n_upd, const int32_t* block_table, const int32_t* seq_lens, void* k_pages, void* v_pages,
                    void* stream) {
  RETRO_RANGE("retro_update_kv");
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(k_hat); RETRO_CHECK_PTR(v_hat); RETRO_CHECK_PTR(positions); RETRO_CHECK_PTR(block_table);
  RETRO_CHECK_PTR(seq_lens); RETRO_CHECK_PTR(k_pages); RETRO_CHECK_PTR(v_pages);
  if (n_upd < 1) return RETRO_ERR_ARG;
  return launch_update_kv(desc, k_hat, v_hat, positions, n_upd, block_table, seq_lens, k_pages, v_pages,
                          (cudaStream_t)stream);
}

int retro_window_advance_layers(const retro_desc_t* desc, const retro_advance_rec_t* table, int32_t n_layers,
                                int32_t pool_steps, void* stream) {
  RETRO_RANGE("retro_window_advance_layers");
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(table);
  if (n_layers < 1 || pool_steps < 1) return RETRO_ERR_ARG;
  return launch_window_advance_layers(desc, table, n_layers, pool_steps, (cudaStream_t)stream);
}

static int check_state(const retro_desc_t* desc, const retro_layer_state_t* st) {
  if (st == nullptr) return RETRO_ERR_ARG;
  RETRO_CHECK_PTR(st->k_pages); RETRO_CHECK_PTR(st->v_pages); RETRO_CHECK_PTR(st->block_table);
  RETRO_CHECK_PTR(st->seq_lens); RETRO_CHECK_PTR(st->budget_pages); RETRO_CHECK_PTR(st->bounds);
  RETRO_CHECK_PTR(st->sel_pages); RETRO_CHECK_PTR(st->sel_prev); RETRO_CHECK_PTR(st->sel_count);
  RETRO_CHECK_PTR(st->part_o); RETRO_CHECK_PTR(st->part_lse); RETRO_CHECK_PTR(st->workspace);
  if (desc->window > 0) {
    RETRO_CHECK_PTR(st->last_loaded); RETRO_CHECK_PTR(st->cache_o); RETRO_CHECK_PTR(st->cache_lse);
    RETRO_CHECK_PTR(st->cache_pos);
  }
  return RETRO_OK;
}

// parts: bit 0 = S1 + S2 (the select kernel, newest digest rebuilt in line), bit 1 = S3 + S4
static int decode_step_parts(const retro_desc_t* desc, const retro_layer_state_t* st, const void* q_win,
                             const int32_t* q_pos, const void* q_cur, void* out, float* out_lse, int parts,
                             void* stream) {
  RETRO_CHECK_DESC(desc);
  int rc = check_state(desc, st);
  if (rc != RETRO_OK) return rc;
  RETRO_CHECK_PTR(q_win); RETRO_CHECK_PTR(q_pos); RETRO_CHECK_PTR(q_cur); RETRO_CHECK_PTR(out);
  const WorkspaceLayout wl = workspace_layout(desc);
  if (st->workspace_bytes < wl.total) return RETRO_ERR_WORKSPACE;
  cudaStream_t s = (cudaStream_t)stream;
  if (parts & 1) {
    // S1 + S2: the digest of the newest token's page is rebuilt inside the select kernel (by the warp that scores
    // that page) and written back, so the step needs no separate digest launch.
    rc = launch_select_pages(desc, wl, q_cur, st->bounds, st->seq_lens, st->budget_pages, st->last_loaded,
                             st->sel_pages, st->sel_prev, st->sel_count, nullptr, st->workspace, s, st->k_pages,
                             st->block_table);
    if (rc != RETRO_OK) return rc;
  }
  if (!(parts & 2)) return RETRO_OK;
  // S3 (+ S4): on the tensor-core path with one row group the attend kernel also merges the output cache (the
  // splits of a unit are one cluster: split combine and Eq. 8-9 in its epilogue, TWO launches per layer-step)
  if (attend_can_fuse_merge(desc, wl)) {
    const FusedMerge fm{st->cache_o, st->cache_lse, st->cache_pos, out, out_lse};
    return launch_sparse_attend(desc, wl, q_win, q_pos, st->k_pages, st->v_pages, st->block_table, st->seq_lens,
                                st->sel_pages, st->sel_prev, st->sel_count, st->part_o, st->part_lse, st->workspace, s,
                                &fm);
  }
  rc = launch_sparse_attend(desc, wl, q_win, q_pos, st->k_pages, st->v_pages, st->block_table, st->seq_lens,
                            st->sel_pages, st->sel_prev, st->sel_count, st->part_o, st->part_lse, st->workspace, s);
  if (rc != RETRO_OK) return rc;
  return launch_merge_output_cache(desc, st->part_o, st->part_lse, q_pos, st->seq_lens, st->cache_o, st->cache_lse,
                                   st->cache_pos, out, out_lse, s);
}

int retro_decode_step(const retro_desc_t* desc, const retro_layer_state_t* st, const void* q_win,
                      const int32_t* q_pos, const void* q_cur, void* out, float* out_lse, void* stream) {
  RETRO_RANGE("retro_decode_step");
  return decode_step_parts(desc, st, q_win, q_pos, q_cur, out, out_lse, 3, stream);
}

int retro_decode_step_part(const retro_desc_t* desc, const retro_layer_state_t* st, const void* q_win,
                           const int32_t* q_pos, const void* q_cur, void* out, float* out_lse, int32_t part,
                           void* stream) {
  RETRO_RANGE("retro_decode_step_part");
  if (part != 0 && part != 1) return RETRO_ERR_ARG;
  return decode_step_parts(desc, st, q_win, q_pos, q_cur, out, out_lse, 1 << part, stream);
}

int retro_debug_status(const retro_desc_t* desc, const void* workspace, size_t ws_bytes, int32_t* enabled,
                       uint32_t* violations, uint32_t* last_code, void* stream) {
  RETRO_CHECK_DESC(desc);
  RETRO_CHECK_PTR(workspace);
  if (enabled == nullptr || violations == nullptr || last_code == nullptr) return RETRO_ERR_ARG;
  const WorkspaceLayout wl = workspace_layout(desc);
  if (ws_bytes < wl.total) return RETRO_ERR_WORKSPACE;
  *violations = 0; *last_code = 0;
#ifdef RETRO_DEBUG_CHECKS
  *enabled = 1;
  unsigned int host[2] = {0, 0};
  RETRO_CUDA_TRY(cudaMemcpyAsync(host, static_cast<const char*>(workspace) + wl.debug_off, sizeof(host),
                                 cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  RETRO_CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream));
  *violations = host[0]; *last_code = host[1];
#else
  *enabled = 0;
  (void)stream;
#endif
  return RETRO_OK;
}

int retro_launches_per_step(const retro_desc_t* desc, int32_t* launches) {
  RETRO_CHECK_DESC(desc);
  if (launches == nullptr) return RETRO_ERR_ARG;
  *launches = attend_can_fuse_merge(desc, workspace_layout(desc)) ? 2 : 3;
  return RETRO_OK;
}

int retro_decode_step_host(const retro_desc_t* desc, const retro_layer_state_t* st, const retro_step_io_t* io,
                           const void* host_qkv_new, void* host_out, void* stream) {
  RETRO_RANGE("retro_decode_step_host");
  RETRO_CHECK_DESC(desc);
  int rc = check_state(desc, st);
  if (rc != RETRO_OK) return rc;
  if (io == nullptr || host_qkv_new == nullptr || host_out == nullptr) return RETRO_ERR_ARG;
  RETRO_CHECK_PTR(io->qkv_new); RETRO_CHECK_PTR(io->q_win); RETRO_CHECK_PTR(io->q_pos); RETRO_CHECK_PTR(io->out);
  cudaStream_t s = (cudaStream_t)stream;
  const size_t esz = desc->dtype == RETRO_BF16 ? 2 : 4;
  const size_t q_bytes = (size_t)desc->batch * desc->num_q_heads * desc->head_dim * esz;
  const size_t kv_bytes = (size_t)desc->batch * desc->num_kv_heads * desc->head_dim * esz;
  // ONE host->device copy (the packed token), one launch for the window ring + AppendKV, the step's two (three)
  // kernels, ONE device->host copy: five stream operations, all CUDA-graph capturable
  RETRO_CUDA_TRY(cudaMemcpyAsync(io->qkv_new, host_qkv_new, q_bytes + 2 * kv_bytes, cudaMemcpyHostToDevice, s));
  rc = launch_ingest_token(desc, io->qkv_new, st->block_table, st->seq_lens, io->q_win, io->q_pos, st->k_pages,
                           st->v_pages, s);
  if (rc != RETRO_OK) return rc;
  rc = retro_decode_step(desc, st, io->q_win, io->q_pos, io->qkv_new, io->out, nullptr, stream);
  if (rc != RETRO_OK) return rc;
  RETRO_CUDA_TRY(cudaMemcpyAsync(host_out, io->out, q_bytes * (desc->window + 1), cudaMemcpyDeviceToHost, s));
  return RETRO_OK;
}

int retro_decode_steps_host(const retro_desc_t* desc, const retro_layer_state_t* states, const retro_step_io_t* ios,
                            int32_t n_layers, const void* host_qkv_new, void* host_out, void* stream) {
  RETRO_RANGE("retro_decode_steps_host");
  RETRO_CHECK_DESC(desc);
  if (states == nullptr || ios == nullptr || n_layers < 1 || host_qkv_new == nullptr || host_out == nullptr)
    return RETRO_ERR_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  const size_t esz = desc->dtype == RETRO_BF16 ? 2 : 4;
  const size_t q_bytes = (size_t)desc->batch * desc->num_q_heads * desc->head_dim * esz;
  const size_t kv_bytes = (size_t)desc->batch * desc->num_kv_heads * desc->head_dim * esz;
  const size_t tok_bytes = q_bytes + 2 * kv_bytes, out_bytes = q_bytes * (desc->window + 1);
  for (int l = 0; l < n_layers; ++l) {
    int rc = check_state(desc, &states[l]);
    if (rc != RETRO_OK) return rc;
    RETRO_CHECK_PTR(ios[l].qkv_new); RETRO_CHECK_PTR(ios[l].q_win); RETRO_CHECK_PTR(ios[l].q_pos); RETRO_CHECK_PTR(ios[l].out);
    // the layers' staging buffers are slices of ONE device buffer each, so that one copy serves them all
    if (static_cast<char*>(ios[l].qkv_new) != static_cast<char*>(ios[0].qkv_new) + l * tok_bytes ||
        static_cast<char*>(ios[l].out) != static_cast<char*>(ios[0].out) + l * out_bytes)
      return RETRO_ERR_ARG;
  }
  RETRO_CUDA_TRY(cudaMemcpyAsync(ios[0].qkv_new, host_qkv_new, tok_bytes * n_layers, cudaMemcpyHostToDevice, s));
  for (int l = 0; l < n_layers; ++l) {
    int rc = launch_ingest_token(desc, ios[l].qkv_new, states[l].block_table, states[l].seq_lens, ios[l].q_win,
                                 ios[l].q_pos, states[l].k_pages, states[l].v_pages, s);
    if (rc != RETRO_OK) return rc;
    rc = retro_decode_step(desc, &states[l], ios[l].q_win, ios[l].q_pos, ios[l].qkv_new, ios[l].out, nullptr, stream);
    if (rc != RETRO_OK) return rc;
  }
  RETRO_CUDA_TRY(cudaMemcpyAsync(host_out, ios[0].out, out_bytes * n_layers, cudaMemcpyDeviceToHost, s));
  return RETRO_OK;
}

}  // extern "C"
