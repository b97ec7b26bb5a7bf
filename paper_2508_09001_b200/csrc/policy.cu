// NEXT-2: the relative budget policy evaluated on the device (budget = 0.15 x
// context length, at least 256 tokens, re-evaluated as decoding continues) and Alg. 2 on its own for a page set
// chosen by another selector (the method is selector-agnostic).
// Both are a handful of integers per (sequence, KV head): one small launch each, latency-bound.
#include "common.cuh"

namespace retro {

__global__ void budget_policy_kernel(const int32_t* __restrict__ seq_lens, int32_t* __restrict__ budget_pages, int B,
                                     int P, int ratio_permille, int min_tokens) {
  pdl_wait();
  pdl_trigger();
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  const long long scaled = (long long)seq_lens[b] * ratio_permille / 1000;   // integer on both sides of the parity
  const int tokens = max(min_tokens, (int)scaled);
  budget_pages[b] = max(1, tokens / P);
}

// one CTA per (KV head, sequence): M.append(A[p]); A[p] <- t for every page of the given S_t (pages are distinct)
__global__ void build_mask_kernel(const int32_t* __restrict__ sel_pages, const int32_t* __restrict__ sel_count,
                                  const int32_t* __restrict__ seq_lens, int32_t* __restrict__ last_loaded,
                                  int32_t* __restrict__ sel_prev, int h_k, int max_pages, int k_max) {
  pdl_wait();
  pdl_trigger();
  const int h = blockIdx.x, b = blockIdx.y;
  const size_t row = (size_t)b * h_k + h;
  const int t = seq_lens[b] - 1;
  const int count = min(sel_count[row], k_max);
  for (int i = threadIdx.x; i < k_max; i += blockDim.x) {
    int prev = -1;
    if (i < count) {
      const int p = sel_pages[row * k_max + i];
      if (p >= 0 && p < max_pages) {
        prev = last_loaded[row * max_pages + p];
        last_loaded[row * max_pages + p] = t;
      }
    }
    sel_prev[row * k_max + i] = prev;
  }
}

// NEXT-4 diagnostics.  Per step and window row: how many of the step's selected pages the row
// may read (the pages that ENLARGE its effective KV budget) and which share of the row's merged
// softmax mass they carry (supplementary attention).  One CTA per (KV head, sequence).
__global__ void step_diagnostics_kernel(const int32_t* __restrict__ sel_pages, const int32_t* __restrict__ sel_prev,
                                        const int32_t* __restrict__ sel_count, const int32_t* __restrict__ q_pos,
                                        const int32_t* __restrict__ seq_lens, const float* __restrict__ part_lse,
                                        const float* __restrict__ out_lse, int32_t* __restrict__ supp_pages,
                                        float* __restrict__ supp_mass, int h_q, int h_k, int k_max, int R, int P) {
  pdl_wait();
  pdl_trigger();
  const int h = blockIdx.x, b = blockIdx.y, G = h_q / h_k;
  const size_t unit = (size_t)b * h_k + h;
  const int t = seq_lens[b] - 1;
  const int count = min(sel_count[unit], k_max);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
  for (int r = warp; r < R; r += nwarp) {           // one warp per window row
    int pos = q_pos[b * R + r];
    if (pos > t || pos < t - (R - 1)) pos = -1;
    int n = 0;
    if (pos >= 0)
      for (int i = lane; i < count; i += 32) {
        const int j = sel_pages[unit * k_max + i];
        n += (sel_prev[unit * k_max + i] < pos && (long long)j * P <= pos) ? 1 : 0;   // same rule as the attend kernel
      }
    n = __reduce_add_sync(0xffffffffu, n);
    if (lane == 0) supp_pages[unit * R + r] = n;
    if (lane < G) {
      const size_t o = ((size_t)b * R + r) * h_q + h * G + lane;
      const float pl = part_lse[o];
      supp_mass[o] = (pos >= 0 && pl > -INFINITY) ? __expf(pl - out_lse[o]) : 0.f;
    }
  }
}

int launch_step_diagnostics(const retro_desc_t* d, const int32_t* sel_pages, const int32_t* sel_prev,
                            const int32_t* sel_count, const int32_t* q_pos, const int32_t* seq_lens,
                            const float* part_lse, const float* out_lse, int32_t* supp_pages, float* supp_mass,
                            cudaStream_t s) {
  RETRO_CUDA_TRY(launch_kernel(step_diagnostics_kernel, dim3(d->num_kv_heads, d->batch), dim3(256), 0, s, sel_pages,
                               sel_prev, sel_count, q_pos, seq_lens, part_lse, out_lse, supp_pages, supp_mass,
                               d->num_q_heads, d->num_kv_heads, d->max_sel_pages, d->window + 1, d->page_size));
  return RETRO_OK;
}

int launch_budget_policy(const retro_desc_t* d, const int32_t* seq_lens, int ratio_permille, int min_tokens,
                         int32_t* budget_pages, cudaStream_t s) {
  RETRO_CUDA_TRY(launch_kernel(budget_policy_kernel, dim3(ceil_div(d->batch, 128)), dim3(128), 0, s, seq_lens,
                               budget_pages, d->batch, d->page_size, ratio_permille, min_tokens));
  return RETRO_OK;
}

int launch_build_mask(const retro_desc_t* d, const int32_t* sel_pages, const int32_t* sel_count,
                      const int32_t* seq_lens, int32_t* last_loaded, int32_t* sel_prev, cudaStream_t s) {
  RETRO_CUDA_TRY(launch_kernel(build_mask_kernel, dim3(d->num_kv_heads, d->batch), dim3(256), 0, s, sel_pages,
                               sel_count, seq_lens, last_loaded, sel_prev, d->num_kv_heads, d->max_pages_per_seq,
                               d->max_sel_pages));
  return RETRO_OK;
}

}  // namespace retro
