// S1  page-bound maintenance: per-channel max / min of K over each page's valid tokens.
// Also AppendKV (Alg. 1 line 3) and the window-ring bookkeeping kernel.
//
// HBM-bound, comparisons only.  One warp per (sequence, KV head, touched page): a (page, head) K tile is
// P*d*esize contiguous bytes; the warp streams it with 128-bit loads (a row of 256 B = 16 lanes), reduces
// across the two half-warps with one shuffle and writes the [Kmax;Kmin] record (512 B) with 128-bit stores.
#include "common.cuh"
#include "digest.cuh"

namespace retro {

// Row of D elements = kRowBytes; 16 lanes cover 256 B.  Instantiated for rows of exactly 256 B
// ({f32, d64} and {bf16, d128}): two rows per warp pass.
template <typename T, int D, int P>
__global__ void __launch_bounds__(128) page_bounds_kernel(const T* __restrict__ k_pages,
                                                          const int32_t* __restrict__ block_table,
                                                          const int32_t* __restrict__ seq_lens,
                                                          const int32_t* __restrict__ pos_begin, T* __restrict__ bounds,
                                                          int B, int h_k, int max_pages, int max_touched) {
  static_assert(D * sizeof(T) == 256, "one K row must be 256 bytes");
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  const int total = B * h_k * max_touched;
  pdl_wait();
  pdl_trigger();
  if (warp >= total) return;
  const int jj = warp % max_touched;
  const int h = (warp / max_touched) % h_k;
  const int b = warp / (max_touched * h_k);
  const int L = seq_lens[b];
  if (L <= 0) return;
  int pb = pos_begin != nullptr ? pos_begin[b] : L - 1;   // NULL: only the newest token's page
  pb = pb < 0 ? 0 : pb;
  const int j = pb / P + jj;
  if (j > (L - 1) / P || j >= max_pages) return;
  const int n_valid = min(P, L - j * P);
  const int phys = block_table[(size_t)b * max_pages + j];
  const uint4* tile = reinterpret_cast<const uint4*>(k_pages + ((size_t)phys * h_k + h) * P * D);
  const uint4 mine = warp_page_digest<T, P>(tile, n_valid, lane);
  uint4* rec = reinterpret_cast<uint4*>(bounds + (((size_t)b * h_k + h) * max_pages + j) * 2 * D);
  rec[lane] = mine;   // lanes 0..15 -> Kmax (256 B), lanes 16..31 -> Kmin (256 B)
}

int launch_update_page_bounds(const retro_desc_t* d, const void* k_pages, const int32_t* block_table,
                              const int32_t* seq_lens, const int32_t* pos_begin, int max_touched, void* bounds,
                              cudaStream_t s) {
  if (max_touched > d->max_pages_per_seq) max_touched = d->max_pages_per_seq;
  const long long warps = (long long)d->batch * d->num_kv_heads * max_touched;
  const int block = 128;
  const unsigned grid = (unsigned)((warps * 32 + block - 1) / block);
  if (d->dtype == RETRO_BF16) {
    RETRO_CUDA_TRY(launch_kernel(page_bounds_kernel<__nv_bfloat16, 128, 16>, dim3(grid), dim3(block), 0, s,
        (const __nv_bfloat16*)k_pages, block_table, seq_lens, pos_begin, (__nv_bfloat16*)bounds, d->batch,
        d->num_kv_heads, d->max_pages_per_seq, max_touched));
  } else {
    RETRO_CUDA_TRY(launch_kernel(page_bounds_kernel<float, 64, 16>, dim3(grid), dim3(block), 0, s, (const float*)k_pages,
                                 block_table, seq_lens, pos_begin, (float*)bounds, d->batch, d->num_kv_heads,
                                 d->max_pages_per_seq, max_touched));
  }
  return RETRO_OK;
}

// ---- AppendKV (Alg. 1 line 3): one token's K and V rows (256 B each) into the pool ----------------
template <typename T, int D, int P>
__global__ void append_kv_kernel(const T* __restrict__ k_new, const T* __restrict__ v_new,
                                 const int32_t* __restrict__ block_table, const int32_t* __restrict__ seq_lens,
                                 T* __restrict__ k_pages, T* __restrict__ v_pages, int B, int h_k, int max_pages) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;   // one 16 B chunk each: [B][h_k][2][16]
  pdl_wait();
  pdl_trigger();
  if (idx >= B * h_k * 32) return;
  const int col = idx & 15, kv = (idx >> 4) & 1, h = (idx >> 5) % h_k, b = idx / (32 * h_k);
  const int pos = seq_lens[b] - 1;
  if (pos < 0 || pos / P >= max_pages) return;   // a sequence never outgrows its block-table row
  const int phys = block_table[(size_t)b * max_pages + pos / P];
  const T* src = (kv ? v_new : k_new) + ((size_t)b * h_k + h) * D;
  T* dst = (kv ? v_pages : k_pages) + (((size_t)phys * h_k + h) * P + pos % P) * D;
  reinterpret_cast<uint4*>(dst)[col] = reinterpret_cast<const uint4*>(src)[col];
}

int launch_append_kv(const retro_desc_t* d, const void* k_new, const void* v_new, const int32_t* block_table,
                     const int32_t* seq_lens, void* k_pages, void* v_pages, cudaStream_t s) {
  const int n = d->batch * d->num_kv_heads * 32;
  const int block = 128, grid = ceil_div(n, block);
  if (d->dtype == RETRO_BF16) {
    RETRO_CUDA_TRY(launch_kernel(append_kv_kernel<__nv_bfloat16, 128, 16>, dim3(grid), dim3(block), 0, s,
        (const __nv_bfloat16*)k_new, (const __nv_bfloat16*)v_new, block_table, seq_lens, (__nv_bfloat16*)k_pages,
        (__nv_bfloat16*)v_pages, d->batch, d->num_kv_heads, d->max_pages_per_seq));
  } else {
    RETRO_CUDA_TRY(launch_kernel(append_kv_kernel<float, 64, 16>, dim3(grid), dim3(block), 0, s, (const float*)k_new,
                                 (const float*)v_new, block_table, seq_lens, (float*)k_pages, (float*)v_pages,
                                 d->batch, d->num_kv_heads, d->max_pages_per_seq));
  }
  return RETRO_OK;
}

// ---- UpdateKV (Alg. 1 line 2; Sec. 2.4): overwrite the rows of past tokens with K^, V^ ----------
template <typename T, int D, int P>
__global__ void update_kv_kernel(const T* __restrict__ k_hat, const T* __restrict__ v_hat,
                                 const int32_t* __restrict__ positions, const int32_t* __restrict__ block_table,
                                 const int32_t* __restrict__ seq_lens, T* __restrict__ k_pages,
                                 T* __restrict__ v_pages, int B, int n_upd, int h_k, int max_pages) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;   // one 16 B chunk each: [B][n_upd][h_k][2][16]
  pdl_wait();
  pdl_trigger();
  if (idx >= B * n_upd * h_k * 32) return;
  const int col = idx & 15, kv = (idx >> 4) & 1, h = (idx >> 5) % h_k;
  const int u = (idx / (32 * h_k)) % n_upd, b = idx / (32 * h_k * n_upd);
  const int pos = positions[b * n_upd + u];
  if (pos < 0 || pos >= seq_lens[b] || pos / P >= max_pages) return;
  const int phys = block_table[(size_t)b * max_pages + pos / P];
  const T* src = (kv ? v_hat : k_hat) + (((size_t)b * n_upd + u) * h_k + h) * D;
  T* dst = (kv ? v_pages : k_pages) + (((size_t)phys * h_k + h) * P + pos % P) * D;
  reinterpret_cast<uint4*>(dst)[col] = reinterpret_cast<const uint4*>(src)[col];
}

int launch_update_kv(const retro_desc_t* d, const void* k_hat, const void* v_hat, const int32_t* positions, int n_upd,
                     const int32_t* block_table, const int32_t* seq_lens, void* k_pages, void* v_pages,
                     cudaStream_t s) {
  const int n = d->batch * n_upd * d->num_kv_heads * 32;
  const int block = 128, grid = ceil_div(n, block);
  if (d->dtype == RETRO_BF16) {
    RETRO_CUDA_TRY(launch_kernel(update_kv_kernel<__nv_bfloat16, 128, 16>, dim3(grid), dim3(block), 0, s,
                                 (const __nv_bfloat16*)k_hat, (const __nv_bfloat16*)v_hat, positions, block_table,
                                 seq_lens, (__nv_bfloat16*)k_pages, (__nv_bfloat16*)v_pages, d->batch, n_upd,
                                 d->num_kv_heads, d->max_pages_per_seq));
  } else {
    RETRO_CUDA_TRY(launch_kernel(update_kv_kernel<float, 64, 16>, dim3(grid), dim3(block), 0, s, (const float*)k_hat,
                                 (const float*)v_hat, positions, block_table, seq_lens, (float*)k_pages,
                                 (float*)v_pages, d->batch, n_upd, d->num_kv_heads, d->max_pages_per_seq));
  }
  return RETRO_OK;
}

// ---- window ring bookkeeping: seq_lens++, q_win[slot] <- q_new, q_pos[slot] <- new position -----------
// Single CTA (the payload is B*h_q*256 bytes).  All threads read the step counter before thread 0 bumps it.
// A sequence whose block-table row is full (seq_len == capacity) is NOT advanced: nothing is written for it.
__device__ __forceinline__ void window_advance_cta(const uint4* __restrict__ q_src, int32_t* step_counter,
                                                   int pool_steps, int32_t* seq_lens, uint4* q_win, int32_t* q_pos,
                                                   uint4* q_cur_out, int B, int h_q, int rows, int capacity) {
  __shared__ int s_pos[64];
  const int row_chunks = h_q * 16;   // uint4 per [h_q][d] block (a q row is 256 B)
  size_t src_off = 0;
  if (step_counter != nullptr) src_off = (size_t)(*step_counter % pool_steps) * B * row_chunks;
  for (int b = threadIdx.x; b < B; b += blockDim.x) {
    const int pos = seq_lens[b];     // position of the token being appended
    if (b < 64) s_pos[b] = pos;
  }
  __syncthreads();
  for (int i = threadIdx.x; i < B * row_chunks; i += blockDim.x) {
    const int b = i / row_chunks, c = i % row_chunks;
    const int pos = s_pos[b];
    const uint4 v = q_src[src_off + i];
    if (pos < capacity) q_win[((size_t)b * rows + pos % rows) * row_chunks + c] = v;
    if (q_cur_out != nullptr) q_cur_out[i] = v;
  }
  __syncthreads();
  for (int b = threadIdx.x; b < B; b += blockDim.x) {
    const int pos = s_pos[b];
    if (pos < capacity) {
      q_pos[b * rows + pos % rows] = pos;
      seq_lens[b] = pos + 1;
    }
  }
  if (threadIdx.x == 0 && step_counter != nullptr) *step_counter += 1;
}

__global__ void __launch_bounds__(1024) window_advance_kernel(const uint4* __restrict__ q_src, int32_t* step_counter,
                                                               int pool_steps, int32_t* seq_lens, uint4* q_win,
                                                               int32_t* q_pos, uint4* q_cur_out, int B, int h_q,
                                                               int rows, int capacity) {
  pdl_wait();
  pdl_trigger();
  window_advance_cta(q_src, step_counter, pool_steps, seq_lens, q_win, q_pos, q_cur_out, B, h_q, rows, capacity);
}

// one CTA per layer record
__global__ void __launch_bounds__(1024) window_advance_layers_kernel(const retro_advance_rec_t* __restrict__ table,
                                                                      int pool_steps, int B, int h_q, int rows,
                                                                      int capacity) {
  pdl_wait();
  pdl_trigger();
  const retro_advance_rec_t rec = table[blockIdx.x];
  window_advance_cta((const uint4*)rec.q_pool, rec.step_counter, pool_steps, rec.seq_lens, (uint4*)rec.q_win,
                     rec.q_pos, (uint4*)rec.q_cur_out, B, h_q, rows, capacity);
}

// ---- host-buffer step: window advance + AppendKV of the packed new token [q | k | v] in one launch ----------------
template <typename T, int D, int P>
__global__ void __launch_bounds__(1024) ingest_token_kernel(const uint4* __restrict__ qkv_new, int32_t* seq_lens,
                                                            uint4* q_win, int32_t* q_pos,
                                                            const int32_t* __restrict__ block_table, T* k_pages,
                                                            T* v_pages, int B, int h_q, int h_k, int rows,
                                                            int max_pages) {
  __shared__ int s_full[64];
  pdl_wait();
  pdl_trigger();
  for (int b = threadIdx.x; b < B; b += blockDim.x) s_full[b] = seq_lens[b] >= max_pages * P;
  __syncthreads();
  window_advance_cta(qkv_new, nullptr, 1, seq_lens, q_win, q_pos, nullptr, B, h_q, rows, max_pages * P);
  __syncthreads();               // seq_lens[b] now counts the new token (unless the sequence is full: no append)
  const uint4* k_new = qkv_new + (size_t)B * h_q * 16;
  const uint4* v_new = k_new + (size_t)B * h_k * 16;
  for (int idx = threadIdx.x; idx < B * h_k * 32; idx += blockDim.x) {   // one 16 B chunk each: [B][h_k][2][16]
    const int col = idx & 15, kv = (idx >> 4) & 1, h = (idx >> 5) % h_k, b = idx / (32 * h_k);
    const int pos = seq_lens[b] - 1;
    if (pos < 0 || pos / P >= max_pages || s_full[b]) continue;
    const int phys = block_table[(size_t)b * max_pages + pos / P];
    T* dst = (kv ? v_pages : k_pages) + (((size_t)phys * h_k + h) * P + pos % P) * D;
    reinterpret_cast<uint4*>(dst)[col] = (kv ? v_new : k_new)[((size_t)b * h_k + h) * 16 + col];
  }
}

int launch_ingest_token(const retro_desc_t* d, const void* qkv_new, const int32_t* block_table, int32_t* seq_lens,
                        void* q_win, int32_t* q_pos, void* k_pages, void* v_pages, cudaStream_t s) {
  if (d->batch > 64) return RETRO_ERR_UNSUPPORTED;
  if (d->dtype == RETRO_BF16)
    RETRO_CUDA_TRY(launch_kernel(ingest_token_kernel<__nv_bfloat16, 128, 16>, dim3(1), dim3(1024), 0, s,
                                 (const uint4*)qkv_new, seq_lens, (uint4*)q_win, q_pos, block_table,
                                 (__nv_bfloat16*)k_pages, (__nv_bfloat16*)v_pages, d->batch, d->num_q_heads,
                                 d->num_kv_heads, d->window + 1, d->max_pages_per_seq));
  else
    RETRO_CUDA_TRY(launch_kernel(ingest_token_kernel<float, 64, 16>, dim3(1), dim3(1024), 0, s, (const uint4*)qkv_new,
                                 seq_lens, (uint4*)q_win, q_pos, block_table, (float*)k_pages, (float*)v_pages,
                                 d->batch, d->num_q_heads, d->num_kv_heads, d->window + 1, d->max_pages_per_seq));
  return RETRO_OK;
}

int launch_window_advance(const retro_desc_t* d, const void* q_new_or_pool, int32_t* step_counter, int pool_steps,
                          int32_t* seq_lens, void* q_win, int32_t* q_pos, void* q_cur_out, cudaStream_t s) {
  if (d->batch > 64) return RETRO_ERR_UNSUPPORTED;
  RETRO_CUDA_TRY(launch_kernel(window_advance_kernel, dim3(1), dim3(1024), 0, s, (const uint4*)q_new_or_pool,
                               step_counter, pool_steps, seq_lens, (uint4*)q_win, q_pos, (uint4*)q_cur_out, d->batch,
                               d->num_q_heads, d->window + 1, d->max_pages_per_seq * d->page_size));
  return RETRO_OK;
}

int launch_window_advance_layers(const retro_desc_t* d, const retro_advance_rec_t* table, int n_layers,
                                 int pool_steps, cudaStream_t s) {
  if (d->batch > 64) return RETRO_ERR_UNSUPPORTED;
  RETRO_CUDA_TRY(launch_kernel(window_advance_layers_kernel, dim3(n_layers), dim3(1024), 0, s, table, pool_steps,
                               d->batch, d->num_q_heads, d->window + 1, d->max_pages_per_seq * d->page_size));
  return RETRO_OK;
}

}  // namespace retro
