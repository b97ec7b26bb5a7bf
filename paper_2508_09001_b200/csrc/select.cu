// S2  Quest page score (Eq. 1) + top-k under the budget + Alg. 2 mask build
// (PAPER.md:551-571).
//
// Score: HBM stream over the digests (512 B per (page, KV head)).  With q+ = max(q,0), q- = min(q,0) and
// Kmax >= Kmin, max(q*Kmin, q*Kmax) = q+*Kmax + q-*Kmin exactly, so the group-SUMMED score is one 2d-long dot
// product [sum_g q+ ; sum_g q-] . [Kmax ; Kmin] per page.  A digest record is exactly 32 lanes x 16 B: one
// coalesced 128-bit load per lane per page.  Accumulation is fp64 (products of bf16/fp32 inputs are exact in
// fp64), so ranking ties against the fp64 oracle only arise within ~1e-12 relative.
//
// Top-k: one CTA per (b, KV head).  Order-preserving 64-bit keys of the fp64 scores live in shared memory;
// a range-adaptive radix select (2048 buckets over [min,max] of the live range, 11 bits per pass, early exit
// when the threshold bucket is taken whole) finds the k-th key, then an in-order two-scan compaction emits
// ascending page indices with ties resolved to the lower index, and the same pass does Alg. 2's
// M.append(A[p]); A[p] <- t.
#include "common.cuh"

namespace retro {

constexpr int kScoreWarps = 8;
constexpr int kPagesPerWarp = 8;
constexpr int kPagesPerCta = kScoreWarps * kPagesPerWarp;

template <typename T> struct Rec;   // how a lane turns its 16 B of a digest record into floats
template <> struct Rec<__nv_bfloat16> {
  static constexpr int kVals = 8;
  __device__ static __forceinline__ void unpack(uint4 v, float* f) {
    f[0] = bf16_lo(v.x); f[1] = bf16_hi(v.x); f[2] = bf16_lo(v.y); f[3] = bf16_hi(v.y);
    f[4] = bf16_lo(v.z); f[5] = bf16_hi(v.z); f[6] = bf16_lo(v.w); f[7] = bf16_hi(v.w);
  }
};
template <> struct Rec<float> {
  static constexpr int kVals = 4;
  __device__ static __forceinline__ void unpack(uint4 v, float* f) {
    f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y); f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
  }
};

// record = [Kmax (D) ; Kmin (D)] = 2*D*sizeof(T) = 512 B: lane l holds elements [l*kVals, (l+1)*kVals) of the
// concatenated vector, i.e. lanes 0..15 see Kmax channels, lanes 16..31 see Kmin channels.
template <typename T, int D>
__global__ void __launch_bounds__(kScoreWarps * 32) page_score_kernel(
    const T* __restrict__ q_cur, const T* __restrict__ bounds, const int32_t* __restrict__ seq_lens,
    double* __restrict__ scores, double* __restrict__ scores_out, int h_q, int h_k, int max_pages, int P,
    int group_reduce) {
  static_assert(2 * D * sizeof(T) == 512, "digest record must be 512 bytes");
  constexpr int kVals = Rec<T>::kVals;
  __shared__ double s_q[kMaxGroup][2 * D];   // per q head: [q+ ; q-] (GROUP_MAX) ; row 0 = group sum (GROUP_SUM)
  const int b = blockIdx.z, h = blockIdx.y;
  const int G = h_q / h_k;
  const int n_pages = (seq_lens[b] + P - 1) / P;
  const int page0 = blockIdx.x * kPagesPerCta;
  const size_t row = ((size_t)b * h_k + h) * max_pages;
  if (page0 >= n_pages) {
    if (scores_out != nullptr)
      for (int j = page0 + threadIdx.x; j < min(page0 + kPagesPerCta, max_pages); j += blockDim.x)
        scores_out[row + j] = -INFINITY;
    return;
  }
  // q+ / q- in fp64 (exact), summed over the group for GROUP_SUM
  for (int i = threadIdx.x; i < 2 * D; i += blockDim.x) {
    const int c = i % D;
    const bool neg = i >= D;
    double acc = 0.0;
    for (int g = 0; g < G; ++g) {
      const double qv = (double)Elem<T>::to_f32(q_cur[((size_t)b * h_q + h * G + g) * D + c]);
      const double part = neg ? fmin(qv, 0.0) : fmax(qv, 0.0);
      if (group_reduce == RETRO_GROUP_SUM) acc += part; else s_q[g][i] = part;
    }
    if (group_reduce == RETRO_GROUP_SUM) s_q[0][i] = acc;
  }
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int jbase = page0 + warp * kPagesPerWarp;
  const uint4* rec = reinterpret_cast<const uint4*>(bounds + (row + jbase) * 2 * D) + lane;
  uint4 raw[kPagesPerWarp];
#pragma unroll
  for (int i = 0; i < kPagesPerWarp; ++i)
    if (jbase + i < n_pages) raw[i] = ldg_stream(rec + i * 32);
  double acc[kPagesPerWarp];
  if (group_reduce == RETRO_GROUP_SUM) {
    double qreg[kVals];
#pragma unroll
    for (int c = 0; c < kVals; ++c) qreg[c] = s_q[0][lane * kVals + c];
#pragma unroll
    for (int i = 0; i < kPagesPerWarp; ++i) {
      acc[i] = 0.0;
      if (jbase + i < n_pages) {
        float f[kVals];
        Rec<T>::unpack(raw[i], f);
#pragma unroll
        for (int c = 0; c < kVals; ++c) acc[i] = fma(qreg[c], (double)f[c], acc[i]);
      }
    }
#pragma unroll
    for (int i = 0; i < kPagesPerWarp; ++i) acc[i] = warp_sum(acc[i]);
  } else {
#pragma unroll
    for (int i = 0; i < kPagesPerWarp; ++i) {
      acc[i] = -INFINITY;
      if (jbase + i < n_pages) {
        float f[kVals];
        Rec<T>::unpack(raw[i], f);
        for (int g = 0; g < G; ++g) {
          double a = 0.0;
#pragma unroll
          for (int c = 0; c < kVals; ++c) a = fma(s_q[g][lane * kVals + c], (double)f[c], a);
          a = warp_sum(a);
          acc[i] = fmax(acc[i], a);
        }
      }
    }
  }
  if (lane == 0) {
#pragma unroll
    for (int i = 0; i < kPagesPerWarp; ++i) {
      const int j = jbase + i;
      if (j < max_pages) {
        const double v = j < n_pages ? acc[i] : -INFINITY;
        if (j < n_pages) scores[row + j] = v;
        if (scores_out != nullptr) scores_out[row + j] = v;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// top-k + mask
// ------------------------------------------------------------------------------------------------
constexpr int kTopkThreads = 1024;
constexpr int kBuckets = 2048;

__device__ __forceinline__ uint64_t order_key(double s) {
  const uint64_t u = (uint64_t)__double_as_longlong(s);
  return (u >> 63) ? ~u : (u | 0x8000000000000000ull);   // larger score <=> larger key
}

// exclusive block scan of one int per thread (1024 threads); returns exclusive prefix, *total = block sum
__device__ __forceinline__ int block_excl_scan(int v, int* s_warp /*[33]*/, int* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int n = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += n;
  }
  __syncthreads();   // protect s_warp reuse
  if (lane == 31) s_warp[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int w = s_warp[lane];
    int winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int n = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += n;
    }
    s_warp[lane] = winc - w;
    if (lane == 31) s_warp[32] = winc;
  }
  __syncthreads();
  *total = s_warp[32];
  return s_warp[warp] + inc - v;
}

__global__ void __launch_bounds__(kTopkThreads) topk_mask_kernel(
    const double* __restrict__ scores, const int32_t* __restrict__ seq_lens, const int32_t* __restrict__ budget_pages,
    int32_t* __restrict__ last_loaded, int32_t* __restrict__ sel_pages, int32_t* __restrict__ sel_prev,
    int32_t* __restrict__ sel_count, int h_k, int max_pages, int k_max, int P, int force_last) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  uint64_t* keys = reinterpret_cast<uint64_t*>(smem_raw);   // [max_pages]
  __shared__ int s_hist[kBuckets];
  __shared__ int s_warp[33];
  __shared__ uint64_t s_red[2][32];
  __shared__ uint64_t s_lo, s_width;
  __shared__ int s_need, s_done;

  const int b = blockIdx.y, h = blockIdx.x;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int L = seq_lens[b];
  const int t = L - 1;
  const int n_pages = L > 0 ? (L + P - 1) / P : 0;
  int k = min(min(budget_pages[b], n_pages), k_max);
  k = max(k, 0);
  const size_t row = ((size_t)b * h_k + h);
  int32_t* out_pages = sel_pages + row * k_max;
  int32_t* out_prev = sel_prev + row * k_max;
  int32_t* A = last_loaded != nullptr ? last_loaded + row * max_pages : nullptr;

  // candidates 0..m-1 compete for k_sel places; the newest page is appended last when forced
  const bool forced = force_last && k > 0 && k < n_pages;
  const int m = forced ? n_pages - 1 : n_pages;
  const int k_sel = forced ? k - 1 : k;

  uint64_t thr_lo = 0, thr_hi_excl_width = 0;   // band [thr_lo, thr_lo + width) ; keys above are all taken
  int need_in_band = 0;
  bool take_all = (k_sel >= m);

  if (!take_all && k_sel > 0) {
    uint64_t kmin = ~0ull, kmax = 0ull;
    for (int i = tid; i < m; i += kTopkThreads) {
      const uint64_t key = order_key(scores[row * max_pages + i]);
      keys[i] = key;
      kmin = key < kmin ? key : kmin;
      kmax = key > kmax ? key : kmax;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const uint64_t a = __shfl_xor_sync(0xffffffffu, kmin, o), c = __shfl_xor_sync(0xffffffffu, kmax, o);
      kmin = a < kmin ? a : kmin;
      kmax = c > kmax ? c : kmax;
    }
    if (lane == 0) { s_red[0][warp] = kmin; s_red[1][warp] = kmax; }
    __syncthreads();
    if (warp == 0) {
      kmin = s_red[0][lane]; kmax = s_red[1][lane];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        const uint64_t a = __shfl_xor_sync(0xffffffffu, kmin, o), c = __shfl_xor_sync(0xffffffffu, kmax, o);
        kmin = a < kmin ? a : kmin;
        kmax = c > kmax ? c : kmax;
      }
      if (lane == 0) { s_lo = kmin; s_width = kmax - kmin; s_need = k_sel; s_done = 0; }
    }
    __syncthreads();
    // range-adaptive radix select: live range [lo, lo + range], `need` keys still to take from it
    for (int pass = 0; pass < 8; ++pass) {
      const uint64_t lo = s_lo, range = s_width;
      const int need = s_need;
      const int nbits = range == 0 ? 0 : 64 - __clzll((long long)range);
      const int shift = nbits > 11 ? nbits - 11 : 0;
      for (int i = tid; i < kBuckets; i += kTopkThreads) s_hist[i] = 0;
      __syncthreads();
      for (int i = tid; i < m; i += kTopkThreads) {
        const uint64_t off = keys[i] - lo;
        if (off <= range) atomicAdd(&s_hist[(int)(off >> shift)], 1);
      }
      __syncthreads();
      // thread i owns buckets (2047-2i) and (2046-2i): scanning threads in order walks buckets downward
      const int b_hi = kBuckets - 1 - 2 * tid, b_lo = b_hi - 1;
      const int c_hi = s_hist[b_hi], c_lo = s_hist[b_lo];
      int total;
      const int before = block_excl_scan(c_hi + c_lo, s_warp, &total);   // keys in strictly higher buckets
      int hit = -1, above = 0, cnt = 0;
      if (before < need && need <= before + c_hi) { hit = b_hi; above = before; cnt = c_hi; }
      else if (before + c_hi < need && need <= before + c_hi + c_lo) { hit = b_lo; above = before + c_hi; cnt = c_lo; }
      if (hit >= 0) {
        const uint64_t new_lo = lo + ((uint64_t)hit << shift);
        const uint64_t width_m1 = shift == 0 ? 0 : ((1ull << shift) - 1);
        const uint64_t new_range = (range - ((uint64_t)hit << shift)) < width_m1 ? (range - ((uint64_t)hit << shift)) : width_m1;
        s_lo = new_lo;
        s_width = new_range;
        s_need = need - above;
        s_done = (cnt == need - above || shift == 0) ? 1 : 0;
      }
      __syncthreads();
      if (s_done) break;
    }
    thr_lo = s_lo;
    thr_hi_excl_width = s_width;   // band = [thr_lo, thr_lo + width] inclusive
    need_in_band = s_need;
  }

  // in-order compaction: thread owns a contiguous chunk of candidate indices
  const int per = (m + kTopkThreads - 1) / kTopkThreads;
  const int i0 = min(tid * per, m), i1 = min(i0 + per, m);
  int band_cnt = 0;
  if (!take_all && k_sel > 0)
    for (int i = i0; i < i1; ++i) {
      const uint64_t off = keys[i] - thr_lo;
      band_cnt += (off <= thr_hi_excl_width) ? 1 : 0;
    }
  int tot_band;
  int band_rank = block_excl_scan(band_cnt, s_warp, &tot_band);
  int sel_cnt = 0;
  uint32_t mybits_lo = 0;   // chunk sizes are tiny (<= 24): one bit per element
  if (k_sel > 0)
    for (int i = i0; i < i1; ++i) {
      bool take;
      if (take_all) take = true;
      else {
        const uint64_t key = keys[i];
        const uint64_t off = key - thr_lo;
        if (off <= thr_hi_excl_width) { take = band_rank < need_in_band; ++band_rank; }
        else take = key > thr_lo;   // above the band (off wrapped => key < thr_lo => not taken)
      }
      if (take) { mybits_lo |= 1u << (i - i0); ++sel_cnt; }
    }
  int tot_sel;
  int pos = block_excl_scan(sel_cnt, s_warp, &tot_sel);
  for (int i = i0; i < i1; ++i)
    if (mybits_lo & (1u << (i - i0))) {
      if (pos < k_max) {
        out_pages[pos] = i;
        int prev = -1;
        if (A != nullptr) { prev = A[i]; A[i] = t; }
        out_prev[pos] = prev;
      }
      ++pos;
    }
  int count = min(tot_sel, k_max);
  if (forced && tid == 0 && count < k_max) {
    const int p = n_pages - 1;
    out_pages[count] = p;
    int prev = -1;
    if (A != nullptr) { prev = A[p]; A[p] = t; }
    out_prev[count] = prev;
  }
  if (forced) count = min(count + 1, k_max);
  for (int i = count + tid; i < k_max; i += kTopkThreads) { out_pages[i] = -1; out_prev[i] = -1; }
  if (tid == 0) sel_count[row] = count;
}

int launch_select_pages(const retro_desc_t* d, const WorkspaceLayout& wl, const void* q_cur, const void* bounds,
                        const int32_t* seq_lens, const int32_t* budget_pages, int32_t* last_loaded,
                        int32_t* sel_pages, int32_t* sel_prev, int32_t* sel_count, double* scores_out,
                        void* workspace, cudaStream_t s) {
  double* scores = reinterpret_cast<double*>(static_cast<char*>(workspace) + wl.scores_off);
  dim3 grid(ceil_div(d->max_pages_per_seq, kPagesPerCta), d->num_kv_heads, d->batch);
  if (d->dtype == RETRO_BF16) {
    page_score_kernel<__nv_bfloat16, 128><<<grid, kScoreWarps * 32, 0, s>>>(
        (const __nv_bfloat16*)q_cur, (const __nv_bfloat16*)bounds, seq_lens, scores, scores_out, d->num_q_heads,
        d->num_kv_heads, d->max_pages_per_seq, d->page_size, d->group_reduce);
  } else {
    page_score_kernel<float, 64><<<grid, kScoreWarps * 32, 0, s>>>(
        (const float*)q_cur, (const float*)bounds, seq_lens, scores, scores_out, d->num_q_heads, d->num_kv_heads,
        d->max_pages_per_seq, d->page_size, d->group_reduce);
  }
  RETRO_LAUNCH_CHECK();
  const size_t smem = (size_t)d->max_pages_per_seq * sizeof(uint64_t);
  static bool attr_set = false;
  if (!attr_set) {
    RETRO_CUDA_TRY(cudaFuncSetAttribute(topk_mask_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
    attr_set = true;
  }
  topk_mask_kernel<<<dim3(d->num_kv_heads, d->batch), kTopkThreads, smem, s>>>(
      scores, seq_lens, budget_pages, last_loaded, sel_pages, sel_prev, sel_count, d->num_kv_heads,
      d->max_pages_per_seq, d->max_sel_pages, d->page_size, d->force_last_page);
  RETRO_LAUNCH_CHECK();
  return RETRO_OK;
}

}  // namespace retro
