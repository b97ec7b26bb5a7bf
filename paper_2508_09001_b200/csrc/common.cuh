// Internal helpers of libretro (sm_100a).  Not part of the C ABI; see include/retro.h.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdlib.h>

#include <mutex>

#include "../../include/retro.h"

namespace retro {

constexpr int kWarp = 32;
constexpr int kMaxWindow = 32;
constexpr int kMaxGroup = 8;
constexpr int kMaxPagesPerSeq = 16384;   // top-k: 256 threads x 64-bit ownership masks; 128 KB of keys

// ---- error plumbing ---------------------------------------------------------------------------
void set_cuda_error(cudaError_t e);
#define RETRO_CUDA_TRY(expr)                      \
  do {                                            \
    cudaError_t e__ = (expr);                     \
    if (e__ != cudaSuccess) {                     \
      ::retro::set_cuda_error(e__);               \
      return RETRO_ERR_CUDA;                      \
    }                                             \
  } while (0)
#define RETRO_LAUNCH_CHECK() RETRO_CUDA_TRY(cudaGetLastError())

// Host-side launcher state (tensor-map cache, per-device facts, raised shared-memory limits) is guarded by one
// mutex, so the entry points may be called from several host threads; apart from that and the last CUDA error
// there is no global state.
std::mutex& host_mutex();   // api.cu

// Facts about the CURRENT device, queried once per device (api.cu).  Without a device (header / symbol tests on a
// CPU-only box) the B200 values are assumed.
struct DeviceInfo {
  int device;          // ordinal, -1 = no device
  int sm_count;        // multiProcessorCount
  int max_smem_optin;  // bytes of dynamic shared memory a CTA may opt in to
};
DeviceInfo device_info();
// cudaFuncAttributeMaxDynamicSharedMemorySize is per device: remembers per (device, kernel) what was granted.
int ensure_dynamic_smem(const void* kern, size_t smem_bytes, bool max_carveout = false);   // RETRO_OK / RETRO_ERR_CUDA
// How many clusters of cluster_x CTAs of this kernel (with this much dynamic shared memory) can be resident at once
// on the current device (cudaOccupancyMaxActiveClusters; 0 = not launchable).  Sizes above 8 opt the kernel in to
// non-portable cluster sizes.  Cached per (device, kernel, shared memory, cluster size).
int max_active_clusters(const void* kern, int block_threads, size_t smem_bytes, int cluster_x);
// tensor-core attend kernel with NT = 16 * nch padded rows: resident clusters of `cluster_x` splits (attend_umma.cu)
int umma_max_active_clusters(int nch, int cluster_x);

inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

int validate_desc(const retro_desc_t* d);  // RETRO_OK / RETRO_ERR_ARG / RETRO_ERR_UNSUPPORTED

// ---- workspace layout (host + device agree through this struct) --------------------------------
struct WorkspaceLayout {
  size_t scores_off;    // uint64 [B][h_k][max_pages]: fp64 keys of the select kernel's exact refinement
  size_t amb_idx_off;   // int32  [B][h_k][max_pages]: the pages those keys belong to
  size_t split_o_off;   // float  [B][h_k][nsplit][rows][d]
  size_t split_lse_off; // float  [B][h_k][nsplit][rows]
  size_t slot_counters_off;  // uint32 [B][w+1]: arrivals per (sequence, cache slot) of the combine + merge kernel
  size_t debug_off;     // uint32 [2]: violations counted by a -DRETRO_DEBUG_CHECKS build, code of the last one
  size_t counters_off;  // uint32 [4][B][h_k]: score-chunk counters first, then split arrival counters per row group
  size_t total;
  int nsplit;           // split-KV factor of the attend kernel
  int pages_per_split;
  int rows;             // G * (w+1)
  int nrg, rg_ranks;    // query-row groups of the tensor-core attend path (one group unless rows > 128): window
                        // ranks per group
};
WorkspaceLayout workspace_layout(const retro_desc_t* d);

// S4 operands for the attend kernel that also merges the output cache (retro_decode_step)
struct FusedMerge {
  void* cache_o; float* cache_lse; int32_t* cache_pos; void* out; float* out_lse;
};

// ---- kernel launchers (one per stage; defined in the matching .cu) ------------------------------
int launch_update_page_bounds(const retro_desc_t* d, const void* k_pages, const int32_t* block_table,
                              const int32_t* seq_lens, const int32_t* pos_begin, int max_touched, void* bounds,
                              cudaStream_t s);
int launch_select_pages(const retro_desc_t* d, const WorkspaceLayout& wl, const void* q_cur, const void* bounds,
                        const int32_t* seq_lens, const int32_t* budget_pages, int32_t* last_loaded,
                        int32_t* sel_pages, int32_t* sel_prev, int32_t* sel_count, double* scores_out,
                        void* workspace, cudaStream_t s, const void* k_pages_refresh = nullptr,
                        const int32_t* block_table = nullptr);   // k_pages_refresh: S1 of the newest page in line
int launch_sparse_attend(const retro_desc_t* d, const WorkspaceLayout& wl, const void* q_win, const int32_t* q_pos,
                         const void* k_pages, const void* v_pages, const int32_t* block_table,
                         const int32_t* seq_lens, const int32_t* sel_pages, const int32_t* sel_prev,
                         const int32_t* sel_count, float* part_o, float* part_lse, void* workspace, cudaStream_t s,
                         const FusedMerge* fused = nullptr);   // non-null (tensor-core path, one row group): S4 in the same kernel
bool attend_can_fuse_merge(const retro_desc_t* d, const WorkspaceLayout& wl);
int launch_merge_output_cache(const retro_desc_t* d, const float* part_o, const float* part_lse,
                              const int32_t* q_pos, const int32_t* seq_lens, void* cache_o, float* cache_lse,
                              int32_t* cache_pos, void* out, float* out_lse, cudaStream_t s);
int launch_append_kv(const retro_desc_t* d, const void* k_new, const void* v_new, const int32_t* block_table,
                     const int32_t* seq_lens, void* k_pages, void* v_pages, cudaStream_t s);
int launch_budget_policy(const retro_desc_t* d, const int32_t* seq_lens, int ratio_permille, int min_tokens,
                         int32_t* budget_pages, cudaStream_t s);
int launch_build_mask(const retro_desc_t* d, const int32_t* sel_pages, const int32_t* sel_count,
                      const int32_t* seq_lens, int32_t* last_loaded, int32_t* sel_prev, cudaStream_t s);
int launch_step_diagnostics(const retro_desc_t* d, const int32_t* sel_pages, const int32_t* sel_prev,
                            const int32_t* sel_count, const int32_t* q_pos, const int32_t* seq_lens,
                            const float* part_lse, const float* out_lse, int32_t* supp_pages, float* supp_mass,
                            cudaStream_t s);
int launch_update_kv(const retro_desc_t* d, const void* k_hat, const void* v_hat, const int32_t* positions, int n_upd,
                     const int32_t* block_table, const int32_t* seq_lens, void* k_pages, void* v_pages,
                     cudaStream_t s);
int launch_ingest_token(const retro_desc_t* d, const void* qkv_new, const int32_t* block_table, int32_t* seq_lens,
                        void* q_win, int32_t* q_pos, void* k_pages, void* v_pages, cudaStream_t s);
int launch_window_advance_layers(const retro_desc_t* d, const retro_advance_rec_t* table, int n_layers,
                                 int pool_steps, cudaStream_t s);
int launch_window_advance(const retro_desc_t* d, const void* q_new_or_pool, int32_t* step_counter, int pool_steps,
                          int32_t* seq_lens, void* q_win, int32_t* q_pos, void* q_cur_out, cudaStream_t s);

// Codes a -DRETRO_DEBUG_CHECKS build records next to its violation count (retro_debug_status)
enum : unsigned int {
  kDbgSelPage = 1,      // sel_pages entry outside [0, #pages of the sequence)
  kDbgPhysPage = 2,     // block_table entry outside [0, num_phys_pages)
  kDbgQPos = 3,         // q_pos entry above the current position
  kDbgSeqLen = 4,       // seq_lens entry outside [0, max_pages_per_seq * page_size]
  kDbgBudget = 5,       // negative budget_pages entry
  kDbgSelCount = 6,     // sel_count entry outside [0, max_sel_pages]
};

#ifdef __CUDACC__
#ifdef RETRO_DEBUG_CHECKS
#define RETRO_DBG_ONLY(...) __VA_ARGS__
__device__ __forceinline__ void dbg_violation(unsigned int* dbg, unsigned int code) {
  atomicAdd(dbg, 1u);
  dbg[1] = code;
}
#else
#define RETRO_DBG_ONLY(...)
#endif
// ---- programmatic dependent launch ---------------------------------------------------------------
// Every libretro kernel is launched with the programmatic-stream-serialization attribute, waits for the
// COMPLETION of its predecessor (pdl_wait) before it touches global memory and then lets its own dependent
// start launching (pdl_trigger).  The next kernel's launch latency, CTA scheduling and shared-memory / TMEM
// set-up overlap the current kernel (also inside a captured CUDA graph); the data dependence is unchanged and at
// most two kernels are resident at a time (triggering before the wait let the whole chain pile up on the SMs).
// Compiling with -DRETRO_NO_PDL leaves the attribute out (griddepcontrol.* are then no-ops).
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// cluster_x > 1: thread-block cluster of cluster_x CTAs along grid x (gridDim.x must be a multiple of it).
template <typename... KArgs, typename... Args>
inline cudaError_t launch_cluster_kernel(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s,
                                         int cluster_x, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute attr[2];
  int n = 0;
#ifndef RETRO_NO_PDL
  attr[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[n].val.programmaticStreamSerializationAllowed = 1;
  ++n;
#endif
  if (cluster_x > 1) {
    attr[n].id = cudaLaunchAttributeClusterDimension;
    attr[n].val.clusterDim.x = (unsigned)cluster_x;
    attr[n].val.clusterDim.y = 1;
    attr[n].val.clusterDim.z = 1;
    ++n;
  }
  cfg.attrs = attr;
  cfg.numAttrs = n;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}
template <typename... KArgs, typename... Args>
inline cudaError_t launch_kernel(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s,
                                 Args... args) {
  return launch_cluster_kernel(kern, grid, block, smem, s, 1, args...);
}

// ---- thread-block clusters: rank, barrier, distributed shared memory --------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t cluster_nctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
  return r;
}
// release / acquire at cluster scope: shared-memory writes (local and remote) before the arrive are visible to
// every CTA of the cluster after its wait.  Executed by ALL threads of every CTA of the cluster.
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
// the same barrier without memory ordering: "every CTA has got this far" (e.g. before a CTA whose shared memory the
// others read may exit)
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait_end() { asm volatile("barrier.cluster.wait.aligned;" ::: "memory"); }
// address of `local_smem_addr` (shared::cta window) in CTA `rank`'s shared memory (shared::cluster window)
__device__ __forceinline__ uint32_t dsmem_addr(uint32_t local_smem_addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_smem_addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void dsmem_st_u32(uint32_t addr, uint32_t v) {
  asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void dsmem_st_f32(uint32_t addr, float v) {
  asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void dsmem_st_v4(uint32_t addr, float4 v) {
  asm volatile("st.shared::cluster.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w)
               : "memory");
}
__device__ __forceinline__ float4 dsmem_ld_v4(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared::cluster.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr)
               : "memory");
  return v;
}
__device__ __forceinline__ uint2 dsmem_ld_v2(uint32_t addr) {
  uint2 v;
  asm volatile("ld.shared::cluster.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ float dsmem_ld_f32(uint32_t addr) {
  float v;
  asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void dsmem_red_min_u32(uint32_t addr, uint32_t v) {
  asm volatile("red.relaxed.cluster.shared::cluster.min.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void dsmem_red_max_u32(uint32_t addr, uint32_t v) {
  asm volatile("red.relaxed.cluster.shared::cluster.max.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

// ---- device helpers ---------------------------------------------------------------------------
template <typename T> struct Elem;
template <> struct Elem<float> {
  static constexpr int kPer16B = 4;
  __device__ static __forceinline__ float to_f32(float x) { return x; }
  __device__ static __forceinline__ float from_f32(float x) { return x; }
};
template <> struct Elem<__nv_bfloat16> {
  static constexpr int kPer16B = 8;
  __device__ static __forceinline__ float to_f32(__nv_bfloat16 x) { return __bfloat162float(x); }
  __device__ static __forceinline__ __nv_bfloat16 from_f32(float x) { return __float2bfloat16_rn(x); }
};

__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

// mbarrier + 1-D bulk async copy (TMA unit, SASS UBLKCP): whole KV page tiles global -> shared.
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {
  }
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(smem_dst)),
               "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// 128-bit read-only streaming load that does not allocate in L1 (digests are read once per step).
__device__ __forceinline__ uint4 ldg_stream(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

// Arrival ticket with release + acquire in one L2 operation.  Used as  bar.sync ; thread 0: ticket ; bar.sync :
// the CTA's earlier writes are released (cumulativity through the barrier), the last arriver's later reads of
// other CTAs' data (ld.cg) are acquired.
__device__ __forceinline__ unsigned int ticket_acq_rel(unsigned int* p) {
  unsigned int old;
  asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(old) : "l"(p) : "memory");
  return old;
}

__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
#endif  // __CUDACC__

}  // namespace retro
