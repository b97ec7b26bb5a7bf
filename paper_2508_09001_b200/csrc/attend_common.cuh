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
  float scale_log2;   // sm_scale * log2(e)
};

#ifdef __CUDACC__
#ifndef RETRO_COMBINE_STAMP
#define RETRO_COMBINE_STAMP(i) do { } while (0)
#endif
// Called by every thread of the CTA after it wrote its split partial (normalised o, base-2 lse) to the
// workspace.  The last CTA of the (b, KV head) unit to arrive merges the nsplit partials (Eq. 8 applied to
// splits: weights 2^(lse_s - max)) into part_o / part_lse (natural-log lse).  D = 128 or 64; one warp per row.
template <int D>
__device__ __forceinline__ void combine_splits_last_cta(const AttendParams& p, size_t unit, int b, int h, int rows,
                                                        int G, int R, unsigned int* s_ticket) {
  constexpr int kCh = D / 32;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
  __threadfence();
  RETRO_COMBINE_STAMP(24);
  __syncthreads();
  if (tid == 0) *s_ticket = atomicAdd(&p.counters[unit], 1u);
  __syncthreads();
  RETRO_COMBINE_STAMP(25);
  if (*s_ticket != (unsigned)(p.nsplit - 1)) return;
  if (tid == 0) p.counters[unit] = 0;   // leave the workspace consistent for the next call
  __threadfence();
  for (int rho = warp; rho < rows; rho += nwarps) {
    const float* lse_s = p.split_lse + unit * p.nsplit * rows + rho;
    float mx = -INFINITY;
    for (int s = lane; s < p.nsplit; s += 32) mx = fmaxf(mx, __ldcg(lse_s + (size_t)s * rows));
    mx = warp_max(mx);
    float o[kCh];
#pragma unroll
    for (int c = 0; c < kCh; ++c) o[c] = 0.f;
    float wsum = 0.f;
    if (mx > -INFINITY) {
      for (int s = 0; s < p.nsplit; ++s) {
        const float ls = __ldcg(lse_s + (size_t)s * rows);
        if (ls == -INFINITY) continue;
        const float wgt = exp2f(ls - mx);
        wsum += wgt;
        const float* src = p.split_o + ((unit * p.nsplit + s) * rows + rho) * D + lane * kCh;
        if constexpr (kCh == 4) {
          const float4 v = __ldcg(reinterpret_cast<const float4*>(src));
          o[0] = fmaf(wgt, v.x, o[0]); o[1] = fmaf(wgt, v.y, o[1]);
          o[2] = fmaf(wgt, v.z, o[2]); o[3] = fmaf(wgt, v.w, o[3]);
        } else {
#pragma unroll
          for (int c = 0; c < kCh; ++c) o[c] = fmaf(wgt, __ldcg(src + c), o[c]);
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
