// Shared by the two S3 kernels (scalar-ALU and tcgen05): parameters and the split-KV combine.
#pragma once
#include "common.cuh"

namespace retro {

constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;

struct AttendParams {
  const void* q_win; const int32_t* q_pos; const void* k_pages; const void* v_pages;
  const int32_t* block_table; const int32_t* seq_lens; const int32_t* sel_pages; const int32_t* sel_prev;
  const int32_t* sel_count; float* part_o; float* part_lse; float* split_o; float* split_lse;
  unsigned int* counters;
  int B, h_q, h_k, max_pages, k_max, window, nsplit, pages_per_split;
  int nrg, rg_ranks;  // query-row groups of the tensor-core path (rows > 128): the CTAs of group rg own the window
                      // ranks (t - position) [rg * rg_ranks, (rg + 1) * rg_ranks), i.e. rg_ranks * G query rows
  float scale_log2;   // sm_scale * log2(e)
  // tensor-core path inside retro_decode_step (fused = 1, nrg == 1): S4 runs in the same kernel
  int fused;
  void* cache_o; int cache_bf16;     // output cache rows: float, or bf16 (Eq. 12's 16-bit O) when cache_bf16
  float* cache_lse; int32_t* cache_pos; void* out; float* out_lse; unsigned int* seq_counters;
  unsigned int* dbg; int num_phys;   // -DRETRO_DEBUG_CHECKS: violation counter in the workspace, pool size
};

#ifdef __CUDACC__
// Called by every thread of the CTA after it wrote its split partial (normalised o, base-2 lse) to the
// workspace.  The last CTA of the (b, KV head) unit to arrive merges the nsplit partials (Eq. 8 applied to
// splits: weights 2^(lse_s - max)) into part_o / part_lse (natural-log lse).  D = 128 or 64; one warp per row.
// Rows [row_begin, row_end) of the unit are combined; `counter` is the arrival counter of that row group.
template <int D>
__device__ __forceinline__ void combine_splits_last_cta(const AttendParams& p, size_t unit, int b, int h, int rows,
                                                        int G, int R, unsigned int* s_ticket, int row_begin,
                                                        int row_end, unsigned int* counter) {
  constexpr int kCh = D / 32;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
  // Release: every thread's partial stores happen-before the barrier; thread 0's acq_rel ticket is cumulative.
  __syncthreads();
  if (tid == 0) *s_ticket = ticket_acq_rel(counter);
  __syncthreads();
  if (*s_ticket != (unsigned)(p.nsplit - 1)) return;
  if (tid == 0) *counter = 0;   // leave the workspace consistent for the next call
  for (int rho = row_begin + warp; rho < row_end; rho += nwarps) {
    const float* lse_s = p.split_lse + unit * p.nsplit * rows + rho;
    const float* o_s = p.split_o + (unit * p.nsplit * rows + rho) * D + lane * kCh;
    const size_t o_stride = (size_t)rows * D;
    // the partial loads do not depend on the weights: the first 8 go out together with the lse loads
    float4 v4[8];
    float v1[8][kCh];
    auto load8 = [&](int s_first) {
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const float* src = o_s + (size_t)min(s_first + u, p.nsplit - 1) * o_stride;
        if constexpr (kCh == 4) {
          v4[u] = __ldcg(reinterpret_cast<const float4*>(src));
        } else {
#pragma unroll
          for (int c = 0; c < kCh; ++c) v1[u][c] = __ldcg(src + c);
        }
      }
    };
    load8(0);
    float mx = -INFINITY;
    for (int s = lane; s < p.nsplit; s += 32) mx = fmaxf(mx, __ldcg(lse_s + (size_t)s * rows));
    mx = warp_max(mx);
    float o[kCh];
#pragma unroll
    for (int c = 0; c < kCh; ++c) o[c] = 0.f;
    float wsum = 0.f;
    if (mx > -INFINITY) {
      for (int s0 = 0; s0 < p.nsplit; s0 += 32) {
        const int sl = s0 + lane;
        const float ls = sl < p.nsplit ? __ldcg(lse_s + (size_t)sl * rows) : -INFINITY;
        const float wl_ = exp2f(ls - mx);                 // lane s holds the weight of split s0 + s; 0 if empty
        const int cnt = min(32, p.nsplit - s0);
        for (int s1 = 0; s1 < cnt; s1 += 8) {
          if (s0 + s1 > 0) load8(s0 + s1);
#pragma unroll
          for (int u = 0; u < 8; ++u) {
            float wgt = __shfl_sync(0xffffffffu, wl_, (s1 + u) & 31);
            if (s1 + u >= cnt) wgt = 0.f;
            if (wgt > 0.f) {                              // an empty split's o is unspecified: never multiply it
              wsum += wgt;
              if constexpr (kCh == 4) {
                o[0] = fmaf(wgt, v4[u].x, o[0]); o[1] = fmaf(wgt, v4[u].y, o[1]);
                o[2] = fmaf(wgt, v4[u].z, o[2]); o[3] = fmaf(wgt, v4[u].w, o[3]);
              } else {
#pragma unroll
                for (int c = 0; c < kCh; ++c) o[c] = fmaf(wgt, v1[u][c], o[c]);
              }
            }
          }
        }
      }
    }
    const float inv = wsum > 0.f ? 1.f / wsum : 0.f;
    const int r = rho / G, g = rho % G;
    float* dst = p.part_o + (((size_t)b * R + r) * p.h_q + h * G + g) * D + lane * kCh;
#pragma unroll
    for (int c = 0; c < kCh; ++c) dst[c] = o[c] * inv;
    if (lane == 0)
      p.part_lse[((size_t)b * R + r) * p.h_q + h * G + g] = wsum > 0.f ? (mx + log2f(wsum)) * kLn2 : -INFINITY;
  }
}
#endif

int launch_attend_umma(const retro_desc_t* d, const AttendParams& prm, cudaStream_t s);   // attend_umma.cu

}  // namespace retro
