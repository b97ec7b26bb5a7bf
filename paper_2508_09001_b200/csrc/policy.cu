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
