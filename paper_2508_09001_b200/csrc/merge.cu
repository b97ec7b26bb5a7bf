// S4  output-cache merge (Eq. 8-9 with alpha = e^lse) and the cache ring
// (push / update / pop; Alg. 1 lines 7-8).
//
// One CTA per (sequence, cache slot): the slot's reader (the past row whose position maps to it) and its writer
// (that row's merged value, or the current row when the slot is t mod w) are handled by the same CTA, so the
// pop of position t-w and the push of position t never race.  One extra CTA per sequence writes the empty rows.
// HBM-trivial: 2*w*h_q*(d+1) floats per sequence; 128-bit accesses.
#include "common.cuh"

namespace retro {

template <typename T> struct OutVec;   // 4 consecutive outputs of type T from a float4
template <> struct OutVec<float> {
  __device__ static __forceinline__ void store(float* dst, float4 v) { *reinterpret_cast<float4*>(dst) = v; }
};
template <> struct OutVec<__nv_bfloat16> {
  __device__ static __forceinline__ void store(__nv_bfloat16* dst, float4 v) {
    __nv_bfloat162 a = __floats2bfloat162_rn(v.x, v.y), c = __floats2bfloat162_rn(v.z, v.w);
    uint2 u;
    u.x = *reinterpret_cast<uint32_t*>(&a);
    u.y = *reinterpret_cast<uint32_t*>(&c);
    *reinterpret_cast<uint2*>(dst) = u;
  }
};

template <typename C> struct CacheVec;   // 4 consecutive cache values as a float4
template <> struct CacheVec<float> {
  __device__ static __forceinline__ float4 load(const float* p) { return *reinterpret_cast<const float4*>(p); }
  __device__ static __forceinline__ void store(float* p, float4 v) { *reinterpret_cast<float4*>(p) = v; }
};
template <> struct CacheVec<__nv_bfloat16> {
  __device__ static __forceinline__ float4 load(const __nv_bfloat16* p) {
    const uint2 u = *reinterpret_cast<const uint2*>(p);
    return make_float4(bf16_lo(u.x), bf16_hi(u.x), bf16_lo(u.y), bf16_hi(u.y));
  }
  __device__ static __forceinline__ void store(__nv_bfloat16* p, float4 v) { OutVec<__nv_bfloat16>::store(p, v); }
};

template <typename T, typename C>
__global__ void __launch_bounds__(256) merge_cache_kernel(const float* __restrict__ part_o,
                                                          const float* __restrict__ part_lse,
                                                          const int32_t* __restrict__ q_pos,
                                                          const int32_t* __restrict__ seq_lens, C* cache_o,
                                                          float* cache_lse, int32_t* cache_pos, T* __restrict__ out,
                                                          float* __restrict__ out_lse, int h_q, int D, int w) {
  const int b = blockIdx.y, x = blockIdx.x;
  pdl_wait();
  pdl_trigger();
  const int R = w + 1;
  const int t = seq_lens[b] - 1;
  const int vec_per_row = D / 4;
  const int n_vec = h_q * vec_per_row;
  __shared__ int s_past_row, s_cur_row, s_cached, s_ppast;

  if (x == w) {   // empty rows -> zeros / -inf
    for (int r = 0; r < R; ++r) {
      const int p = q_pos[b * R + r];
      if (p >= 0 && p <= t && p >= t - w) continue;
      for (int i = threadIdx.x; i < n_vec; i += blockDim.x)
        OutVec<T>::store(out + ((size_t)b * R + r) * h_q * D + (size_t)i * 4, make_float4(0.f, 0.f, 0.f, 0.f));
      if (out_lse != nullptr)
        for (int i = threadIdx.x; i < h_q; i += blockDim.x) out_lse[((size_t)b * R + r) * h_q + i] = -INFINITY;
    }
    if (w == 0) {   // plain Quest: out = part of the current row, no cache
      for (int r = 0; r < R; ++r) {
        if (q_pos[b * R + r] != t) continue;
        for (int i = threadIdx.x; i < n_vec; i += blockDim.x) {
          const size_t o = ((size_t)b * R + r) * h_q * D + (size_t)i * 4;
          OutVec<T>::store(out + o, *reinterpret_cast<const float4*>(part_o + o));
        }
        if (out_lse != nullptr)
          for (int i = threadIdx.x; i < h_q; i += blockDim.x)
            out_lse[((size_t)b * R + r) * h_q + i] = part_lse[((size_t)b * R + r) * h_q + i];
      }
    }
    return;
  }

  // slot x: the past position p in [t-w, t-1] with p mod w == x, and (if x == t mod w) the current row.
  // A slot has exactly one writer per step: if the current row lands here, the past row of this slot is the
  // evicted one (position t-w).  Latency-bound, so: one round trip for the roles, one for ALL the operands
  // (issued unconditionally where the address is valid), then the stores.
  const int slot = x;
  if (threadIdx.x == 0) { s_past_row = -1; s_cur_row = -1; s_cached = 0; s_ppast = -1; }
  __syncthreads();
  if (threadIdx.x < R) {
    const int r = threadIdx.x;
    const int p = q_pos[b * R + r];
    const int cp = cache_pos[b * w + slot];          // unconditional: rides the same round trip as q_pos
    if (p >= 0 && p <= t && p >= t - w) {
      if (p == t) { if (t % w == slot) s_cur_row = r; }
      else if (p % w == slot) { s_past_row = r; s_ppast = p; s_cached = (cp == p) ? 1 : 0; }
    }
  }
  __syncthreads();
  const int past = s_past_row, cur = s_cur_row;
  const bool cached = s_cached != 0;
  const int p_past = s_ppast;
  const bool evict = past >= 0 && p_past == t - w;   // popped after its last merge
  C* c_o = cache_o + ((size_t)b * w + slot) * h_q * D;
  float* c_l = cache_lse + ((size_t)b * w + slot) * h_q;
  const float* po = part_o + ((size_t)b * R + (past >= 0 ? past : 0)) * h_q * D;
  const float* pl = part_lse + ((size_t)b * R + (past >= 0 ? past : 0)) * h_q;
  const float* qo = part_o + ((size_t)b * R + (cur >= 0 ? cur : 0)) * h_q * D;
  const float* ql = part_lse + ((size_t)b * R + (cur >= 0 ? cur : 0)) * h_q;
  for (int i0 = 0; i0 < n_vec; i0 += 4 * blockDim.x) {
    float4 vp[4], vc[4], vq[4];
    float lp[4], lc[4], lq[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {             // every load of the pass is in flight before the first use
      const int i = i0 + u * blockDim.x + threadIdx.x;
      if (i < n_vec) {
        const int hh = i / vec_per_row;
        if (past >= 0) { vp[u] = *reinterpret_cast<const float4*>(po + (size_t)i * 4); lp[u] = pl[hh]; }
        if (past >= 0 && cached) { vc[u] = CacheVec<C>::load(c_o + (size_t)i * 4); lc[u] = c_l[hh]; }
        if (cur >= 0) { vq[u] = *reinterpret_cast<const float4*>(qo + (size_t)i * 4); lq[u] = ql[hh]; }
      }
    }
    if (!cached) {
#pragma unroll
      for (int u = 0; u < 4; ++u) lc[u] = -INFINITY;
    }
    __syncthreads();   // c_l / c_o of this pass are in registers before anybody rewrites them
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = i0 + u * blockDim.x + threadIdx.x;
      if (i >= n_vec) continue;
      const int hh = i / vec_per_row;
      const bool head_lane = (i % vec_per_row) == 0;
      if (past >= 0) {
        T* oo = out + ((size_t)b * R + past) * h_q * D;
        float4 res;
        float lse;
        if (lc[u] == -INFINITY) { res = vp[u]; lse = lp[u]; }
        else if (lp[u] == -INFINITY) { res = vc[u]; lse = lc[u]; }
        else {
          const float mx = fmaxf(lc[u], lp[u]);
          const float wc = __expf(lc[u] - mx), wp = __expf(lp[u] - mx);
          const float inv = 1.f / (wc + wp);
          res.x = (wc * vc[u].x + wp * vp[u].x) * inv; res.y = (wc * vc[u].y + wp * vp[u].y) * inv;
          res.z = (wc * vc[u].z + wp * vp[u].z) * inv; res.w = (wc * vc[u].w + wp * vp[u].w) * inv;
          lse = mx + __logf(wc + wp);
        }
        OutVec<T>::store(oo + (size_t)i * 4, res);
        if (!evict) CacheVec<C>::store(c_o + (size_t)i * 4, res);
        if (head_lane) {
          if (out_lse != nullptr) out_lse[((size_t)b * R + past) * h_q + hh] = lse;
          if (!evict) c_l[hh] = lse;
        }
      }
      if (cur >= 0) {   // push O_org of the current query (the popped row is already in registers)
        T* oo = out + ((size_t)b * R + cur) * h_q * D;
        OutVec<T>::store(oo + (size_t)i * 4, vq[u]);
        CacheVec<C>::store(c_o + (size_t)i * 4, vq[u]);
        if (head_lane) {
          if (out_lse != nullptr) out_lse[((size_t)b * R + cur) * h_q + hh] = lq[u];
          c_l[hh] = lq[u];
        }
      }
    }
  }
  if (threadIdx.x == 0) {
    if (cur >= 0) cache_pos[b * w + slot] = t;
    else if (past >= 0 && !evict) cache_pos[b * w + slot] = p_past;
  }
}

int launch_merge_output_cache(const retro_desc_t* d, const float* part_o, const float* part_lse,
                              const int32_t* q_pos, const int32_t* seq_lens, void* cache_o, float* cache_lse,
                              int32_t* cache_pos, void* out, float* out_lse, cudaStream_t s) {
  dim3 grid(d->window + 1, d->batch);
  if (d->dtype == RETRO_BF16 && d->cache_dtype == RETRO_BF16)
    RETRO_CUDA_TRY(launch_kernel(merge_cache_kernel<__nv_bfloat16, __nv_bfloat16>, grid, dim3(256), 0, s, part_o,
                                 part_lse, q_pos, seq_lens, (__nv_bfloat16*)cache_o, cache_lse, cache_pos,
                                 (__nv_bfloat16*)out, out_lse, d->num_q_heads, d->head_dim, d->window));
  else if (d->dtype == RETRO_BF16)
    RETRO_CUDA_TRY(launch_kernel(merge_cache_kernel<__nv_bfloat16, float>, grid, dim3(256), 0, s, part_o, part_lse,
                                 q_pos, seq_lens, (float*)cache_o, cache_lse, cache_pos, (__nv_bfloat16*)out, out_lse,
                                 d->num_q_heads, d->head_dim, d->window));
  else
    RETRO_CUDA_TRY(launch_kernel(merge_cache_kernel<float, float>, grid, dim3(256), 0, s, part_o, part_lse, q_pos,
                                 seq_lens, (float*)cache_o, cache_lse, cache_pos, (float*)out, out_lse,
                                 d->num_q_heads, d->head_dim, d->window));
  return RETRO_OK;
}

}  // namespace retro
