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

template <typename T>
__global__ void __launch_bounds__(256) merge_cache_kernel(const float* __restrict__ part_o,
                                                          const float* __restrict__ part_lse,
                                                          const int32_t* __restrict__ q_pos,
                                                          const int32_t* __restrict__ seq_lens, float* cache_o,
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
  float* c_o = cache_o + ((size_t)b * w + slot) * h_q * D;
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
        if (past >= 0 && cached) { vc[u] = *reinterpret_cast<const float4*>(c_o + (size_t)i * 4); lc[u] = c_l[hh]; }
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
        if (!evict) *reinterpret_cast<float4*>(c_o + (size_t)i * 4) = res;
        if (head_lane) {
          if (out_lse != nullptr) out_lse[((size_t)b * R + past) * h_q + hh] = lse;
          if (!evict) c_l[hh] = lse;
        }
      }
      if (cur >= 0) {   // push O_org of the current query (the popped row is already in registers)
        T* oo = out + ((size_t)b * R + cur) * h_q * D;
        OutVec<T>::store(oo + (size_t)i * 4, vq[u]);
        *reinterpret_cast<float4*>(c_o + (size_t)i * 4) = vq[u];
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

// ---- split combine + S4 in one launch (retro_decode_step, bf16 tensor-core path with nsplit > 1) ----------------
// The attend kernel then ends after writing its split partials (no in-kernel ticket / combine); this kernel merges
// the nsplit partials of a row (Eq. 8 applied to splits, base-2 lse) and the cached (o, lse) in one pass: the
// split partials and the cache operands ride the same round trip.  One CTA per (cache slot | empties, KV head,
// sequence); warp g handles q head h*G+g: first the slot's past row (reads the cache), then the current row if it
// lands in this slot (writes it), so the pop of position t-w and the push of position t are ordered by the warp.
// cache_pos is shared by the KV heads: the last CTA of a (sequence, slot) to finish reading rewrites it.
__global__ void __launch_bounds__(256) combine_merge_kernel(
    const float* __restrict__ split_o, const float* __restrict__ split_lse, int nsplit, int rows,
    float* __restrict__ part_o, float* __restrict__ part_lse, const int32_t* __restrict__ q_pos,
    const int32_t* __restrict__ seq_lens, float* cache_o, float* cache_lse, int32_t* cache_pos,
    __nv_bfloat16* __restrict__ out, float* __restrict__ out_lse, unsigned int* slot_counters, int h_q, int h_k,
    int w) {
  constexpr int D = 128;
  constexpr float kLn2f = 0.6931471805599453f;
  const int x = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  pdl_wait();
  pdl_trigger();
  const int R = w + 1, G = h_q / h_k;
  const int t = seq_lens[b] - 1;
  const size_t unit = (size_t)b * h_k + h;
  __shared__ int s_past_row, s_cur_row, s_ppast, s_cpos;
  __shared__ unsigned int s_tk;
  if (threadIdx.x == 0) { s_past_row = -1; s_cur_row = -1; s_ppast = -1; s_cpos = -2; }
  __syncthreads();
  const bool empties = (x == w);              // the extra CTA: rows without a valid position -> zeros / -inf
  if (threadIdx.x < R) {
    const int r = threadIdx.x;
    const int p = q_pos[b * R + r];
    const int cp = (w > 0 && !empties) ? cache_pos[b * w + x] : -2;
    if (p >= 0 && p <= t && p >= t - w) {
      if (p == t) { if (w == 0 || (!empties && t % w == x)) s_cur_row = r; }
      else if (!empties && p % w == x) { s_past_row = r; s_ppast = p; s_cpos = cp; }
    }
  }
  __syncthreads();
  if (empties && w > 0) {
    for (int r = 0; r < R; ++r) {
      const int p = q_pos[b * R + r];
      if (p >= 0 && p <= t && p >= t - w) continue;
      for (int i = threadIdx.x; i < G * 32; i += blockDim.x) {
        const size_t o = (((size_t)b * R + r) * h_q + h * G + i / 32) * D + (i % 32) * 4;
        OutVec<__nv_bfloat16>::store(out + o, make_float4(0.f, 0.f, 0.f, 0.f));
        *reinterpret_cast<float4*>(part_o + o) = make_float4(0.f, 0.f, 0.f, 0.f);
      }
      for (int i = threadIdx.x; i < G; i += blockDim.x) {
        const size_t o = ((size_t)b * R + r) * h_q + h * G + i;
        part_lse[o] = -INFINITY;
        if (out_lse != nullptr) out_lse[o] = -INFINITY;
      }
    }
    return;
  }
  const int past = s_past_row, cur = s_cur_row, p_past = s_ppast;
  const bool cached = past >= 0 && s_cpos == p_past;
  const bool evict = past >= 0 && p_past == t - w;
  // Work items: (past row | current row) x q head of the group.  With G <= 4 the eight warps take one item each
  // (both rows in parallel); otherwise warp g takes both rows of head g.  Phase 1 loads, combines, merges and
  // writes `out`; the cache is rewritten in phase 2, after a barrier: the slot popped by the row at t-w is the
  // slot the current row is pushed into.
  const bool one_item = 2 * G <= 8;
  float4 res_k[2];
  float lse_k[2];
  bool wr_k[2] = {false, false};
  int hq_k[2] = {0, 0};
#pragma unroll
  for (int kind = 0; kind < 2; ++kind) {
    const bool active = one_item ? (warp >= kind * G && warp < (kind + 1) * G) : (warp < G);
    const int g = one_item ? warp - kind * G : warp;
    const int r = kind == 0 ? past : cur;
    if (!active || r < 0) continue;
    const int hq = h * G + g;
    hq_k[kind] = hq;
    const size_t ce = w > 0 ? ((size_t)b * w + x) * h_q + hq : 0;
    // every operand of the item goes out before the first use: split partials (first 8), their lse, the cache
    const int rho = r * G + g;
    const float* ls = split_lse + unit * nsplit * rows + rho;
    const float* os = split_o + (unit * nsplit * rows + rho) * D + lane * 4;
    const size_t stride = (size_t)rows * D;
    float4 v[8];
    auto load8 = [&](int s_first) {
#pragma unroll
      for (int u = 0; u < 8; ++u)
        v[u] = __ldcg(reinterpret_cast<const float4*>(os + (size_t)min(s_first + u, nsplit - 1) * stride));
    };
    load8(0);
    float lc = -INFINITY;
    float4 vc = make_float4(0.f, 0.f, 0.f, 0.f);
    if (kind == 0 && cached) {
      lc = cache_lse[ce];
      vc = *reinterpret_cast<const float4*>(cache_o + ce * D + lane * 4);
    }
    float mx = -INFINITY;
    for (int s = lane; s < nsplit; s += 32) mx = fmaxf(mx, __ldcg(ls + (size_t)s * rows));
    mx = warp_max(mx);
    float o[4] = {0.f, 0.f, 0.f, 0.f};
    float wsum = 0.f;
    if (mx > -INFINITY) {
      for (int s0 = 0; s0 < nsplit; s0 += 32) {
        const int sl = s0 + lane;
        const float l_mine = sl < nsplit ? __ldcg(ls + (size_t)sl * rows) : -INFINITY;
        const float w_mine = exp2f(l_mine - mx);           // lane s holds the weight of split s0 + s; 0 if empty
        const int cnt = min(32, nsplit - s0);
        for (int s1 = 0; s1 < cnt; s1 += 8) {
          if (s0 + s1 > 0) load8(s0 + s1);
#pragma unroll
          for (int u = 0; u < 8; ++u) {
            float wg = __shfl_sync(0xffffffffu, w_mine, (s1 + u) & 31);
            if (s1 + u >= cnt) wg = 0.f;
            if (wg > 0.f) {                                // an empty split's o is unspecified: never multiply it
              wsum += wg;
              o[0] = fmaf(wg, v[u].x, o[0]); o[1] = fmaf(wg, v[u].y, o[1]);
              o[2] = fmaf(wg, v[u].z, o[2]); o[3] = fmaf(wg, v[u].w, o[3]);
            }
          }
        }
      }
    }
    const float inv = wsum > 0.f ? 1.f / wsum : 0.f;
    o[0] *= inv; o[1] *= inv; o[2] *= inv; o[3] *= inv;
    const float lp = wsum > 0.f ? (mx + log2f(wsum)) * kLn2f : -INFINITY;
    const size_t e = ((size_t)b * R + r) * h_q + hq;
    *reinterpret_cast<float4*>(part_o + e * D + lane * 4) = make_float4(o[0], o[1], o[2], o[3]);
    if (lane == 0) part_lse[e] = lp;
    float4 res;
    float lse;
    if (lc == -INFINITY) { res = make_float4(o[0], o[1], o[2], o[3]); lse = lp; }
    else if (lp == -INFINITY) { res = vc; lse = lc; }
    else {
      const float m2 = fmaxf(lc, lp);
      const float wc = __expf(lc - m2), wp = __expf(lp - m2);
      const float iv = 1.f / (wc + wp);
      res.x = (wc * vc.x + wp * o[0]) * iv; res.y = (wc * vc.y + wp * o[1]) * iv;
      res.z = (wc * vc.z + wp * o[2]) * iv; res.w = (wc * vc.w + wp * o[3]) * iv;
      lse = m2 + __logf(wc + wp);
    }
    OutVec<__nv_bfloat16>::store(out + e * D + lane * 4, res);
    if (lane == 0 && out_lse != nullptr) out_lse[e] = lse;
    res_k[kind] = res;
    lse_k[kind] = lse;
    wr_k[kind] = w > 0 && (kind == 0 ? !evict : true);
  }
  __syncthreads();                        // every cache read of this (slot, KV head) is done
#pragma unroll
  for (int kind = 0; kind < 2; ++kind) {
    if (wr_k[kind]) {
      const size_t ce = ((size_t)b * w + x) * h_q + hq_k[kind];
      *reinterpret_cast<float4*>(cache_o + ce * D + lane * 4) = res_k[kind];
      if (lane == 0) cache_lse[ce] = lse_k[kind];
    }
  }
  if (w > 0) {
    // every KV head of (b, slot) has read cache_pos before the last one rewrites it
    __syncthreads();
    if (threadIdx.x == 0) s_tk = ticket_acq_rel(&slot_counters[b * (w + 1) + x]);
    __syncthreads();
    if (s_tk == (unsigned)(h_k - 1) && threadIdx.x == 0) {
      slot_counters[b * (w + 1) + x] = 0;
      if (cur >= 0) cache_pos[b * w + x] = t;
      else if (past >= 0 && !evict) cache_pos[b * w + x] = p_past;
    }
  }
}

int launch_combine_merge(const retro_desc_t* d, const float* split_o, const float* split_lse, int nsplit, int rows,
                         float* part_o, float* part_lse, const int32_t* q_pos, const int32_t* seq_lens, float* cache_o,
                         float* cache_lse, int32_t* cache_pos, void* out, float* out_lse, unsigned int* slot_counters,
                         cudaStream_t s) {
  RETRO_CUDA_TRY(launch_kernel(combine_merge_kernel, dim3(d->window + 1, d->num_kv_heads, d->batch), dim3(256), 0, s,
                               split_o, split_lse, nsplit, rows, part_o, part_lse, q_pos, seq_lens, cache_o, cache_lse,
                               cache_pos, (__nv_bfloat16*)out, out_lse, slot_counters, d->num_q_heads,
                               d->num_kv_heads, d->window));
  return RETRO_OK;
}

int launch_merge_output_cache(const retro_desc_t* d, const float* part_o, const float* part_lse,
                              const int32_t* q_pos, const int32_t* seq_lens, float* cache_o, float* cache_lse,
                              int32_t* cache_pos, void* out, float* out_lse, cudaStream_t s) {
  dim3 grid(d->window + 1, d->batch);
  if (d->dtype == RETRO_BF16)
    RETRO_CUDA_TRY(launch_kernel(merge_cache_kernel<__nv_bfloat16>, grid, dim3(256), 0, s, part_o, part_lse, q_pos,
                                 seq_lens, cache_o, cache_lse, cache_pos, (__nv_bfloat16*)out, out_lse,
                                 d->num_q_heads, d->head_dim, d->window));
  else
    RETRO_CUDA_TRY(launch_kernel(merge_cache_kernel<float>, grid, dim3(256), 0, s, part_o, part_lse, q_pos, seq_lens,
                                 cache_o, cache_lse, cache_pos, (float*)out, out_lse, d->num_q_heads, d->head_dim,
                                 d->window));
  return RETRO_OK;
}

}  // namespace retro
