// S2  Quest page score (Eq. 1) + top-k under the budget + Alg. 2 mask build
// (PAPER.md:551-571).
//
// Score: HBM stream over the digests (512 B per (page, KV head)).  With q+ = max(q,0), q- = min(q,0) and
// Kmax >= Kmin, max(q*Kmin, q*Kmax) = q+*Kmax + q-*Kmin exactly, so the group-SUMMED score is one 2d-long dot
// product [sum_g q+ ; sum_g q-] . [Kmax ; Kmin] per page.  A digest record is exactly 32 lanes x 16 B: one
// coalesced 128-bit load per lane per page.  Accumulation is fp64 (products of bf16/fp32 inputs are exact in
// fp64), so ranking ties against the fp64 oracle only arise within ~1e-12 relative.
//
// Score and top-k run in ONE kernel: every CTA scores 64 pages of one (b, KV head) unit; the last CTA of the unit
// to finish (arrival counter in the workspace) selects.  Order-preserving 64-bit keys of the fp64 scores live in shared memory;
// a range-adaptive radix select (2048 buckets over [min,max] of the live range, 11 bits per pass, early exit
// when the threshold bucket is taken whole) finds the k-th key, then an in-order two-scan compaction emits
// ascending page indices with ties resolved to the lower index, and the same pass does Alg. 2's
// M.append(A[p]); A[p] <- t.
#include "common.cuh"
#include "digest.cuh"

namespace retro {


constexpr int kScoreWarps = 8;
constexpr int kPagesPerWarp = 8;
constexpr int kPagesPerCta = kScoreWarps * kPagesPerWarp;
constexpr int kStages = 2;                       // digest batches in flight per CTA
constexpr int kStageBytes = kPagesPerCta * 512;  // 32 KB

template <typename T> struct Rec;   // how a lane turns its 16 B of a digest record into fp64 values
template <> struct Rec<__nv_bfloat16> {
  static constexpr int kVals = 8;
  __device__ static __forceinline__ void unpack(uint4 v, double* f) {
    f[0] = (double)bf16_lo(v.x); f[1] = (double)bf16_hi(v.x); f[2] = (double)bf16_lo(v.y); f[3] = (double)bf16_hi(v.y);
    f[4] = (double)bf16_lo(v.z); f[5] = (double)bf16_hi(v.z); f[6] = (double)bf16_lo(v.w); f[7] = (double)bf16_hi(v.w);
  }
};
template <> struct Rec<float> {
  static constexpr int kVals = 4;
  __device__ static __forceinline__ void unpack(uint4 v, double* f) {
    f[0] = (double)__uint_as_float(v.x); f[1] = (double)__uint_as_float(v.y);
    f[2] = (double)__uint_as_float(v.z); f[3] = (double)__uint_as_float(v.w);
  }
};

// record = [Kmax (D) ; Kmin (D)] = 2*D*sizeof(T) = 512 B: lane l holds elements [l*kVals, (l+1)*kVals) of the
// concatenated vector, i.e. lanes 0..15 see Kmax channels, lanes 16..31 see Kmin channels.
// ------------------------------------------------------------------------------------------------
// top-k + mask
// ------------------------------------------------------------------------------------------------
constexpr int kBuckets = 2048;

__device__ __forceinline__ uint64_t order_key(double s) {
  const uint64_t u = (uint64_t)__double_as_longlong(s);
  return (u >> 63) ? ~u : (u | 0x8000000000000000ull);   // larger score <=> larger key
}

// exclusive block scan of one int per thread (NT threads, NT / 32 <= 32 warps); returns the exclusive prefix,
// *total = block sum.  One barrier per call: the warp totals alternate between two buffers (`phase` counts the
// calls), so a buffer is rewritten only after every thread has passed the barrier of the call in between.
template <int NT>
__device__ __forceinline__ int block_excl_scan(int v, int* s_warp /*[2][32]*/, int* total, int& phase) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int n = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += n;
  }
  int* buf = s_warp + (phase & 1) * 32;
  ++phase;
  if (lane == 31) buf[warp] = inc;
  __syncthreads();
  int before = 0, sum = 0;
#pragma unroll
  for (int w = 0; w < NT / 32; ++w) {
    const int tw = buf[w];
    before += w < warp ? tw : 0;
    sum += tw;
  }
  *total = sum;
  return before + inc - v;
}

// Executed by all NT threads of one CTA for unit (b, h); scores are read through L2 (written by other CTAs).
template <int NT>
__device__ __forceinline__ void topk_mask_block(
    uint64_t* keys /*shared [max_pages]*/, const double* scores, int L /*seq_lens[b]*/, int budget /*budget_pages[b]*/,
    int32_t* __restrict__ last_loaded, int32_t* __restrict__ sel_pages,
    int32_t* __restrict__ sel_prev, int32_t* __restrict__ sel_count, int b, int h, int h_k, int max_pages, int k_max,
    int P, int force_last) {
  constexpr int kTopkThreads = NT;
  __shared__ int s_hist[kBuckets];
  __shared__ int s_warp[64];
  int scan_phase = 0;
  __shared__ uint64_t s_red[2][32];
  __shared__ uint64_t s_lo, s_width;
  __shared__ int s_need, s_done;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int t = L - 1;
  const int n_pages = L > 0 ? (L + P - 1) / P : 0;
  int k = min(min(budget, n_pages), k_max);
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
#pragma unroll 4
    for (int i = tid; i < m; i += kTopkThreads) {
      const uint64_t key = order_key(__ldcg(scores + row * max_pages + i));
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
      kmin = lane < NT / 32 ? s_red[0][lane] : ~0ull;
      kmax = lane < NT / 32 ? s_red[1][lane] : 0ull;
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
      for (int i0 = tid; i0 < m; i0 += 8 * kTopkThreads) {   // loads first: they cannot be hoisted over the atomics
        uint64_t kk[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) kk[u] = keys[min(i0 + u * kTopkThreads, m - 1)];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          const uint64_t off = kk[u] - lo;
          if (i0 + u * kTopkThreads < m && off <= range) atomicAdd(&s_hist[(int)(off >> shift)], 1);
        }
      }
      __syncthreads();
      // thread i owns kBuckets / NT consecutive buckets, highest first: scanning threads in order walks buckets
      // downward
      constexpr int kPer = kBuckets / NT;
      int cbk[kPer], csum = 0;
#pragma unroll
      for (int u = 0; u < kPer; ++u) { cbk[u] = s_hist[kBuckets - 1 - (tid * kPer + u)]; csum += cbk[u]; }
      int total;
      int run = block_excl_scan<NT>(csum, s_warp, &total, scan_phase);   // keys in strictly higher buckets
      int hit = -1, above = 0, cnt = 0;
#pragma unroll
      for (int u = 0; u < kPer; ++u) {
        if (run < need && need <= run + cbk[u]) { hit = kBuckets - 1 - (tid * kPer + u); above = run; cnt = cbk[u]; }
        run += cbk[u];
      }
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
  // one packed scan: low 16 bits = candidates above the band (always taken), high bits = candidates inside it
  // (the first need_in_band of them, in index order, are taken); counts are <= kMaxPagesPerSeq < 2^15
  int above_cnt = 0, band_cnt = 0;
  uint64_t above_bits = 0, band_bits = 0;   // one bit per owned candidate: chunks are <= kMaxPagesPerSeq / NT = 64
  if (k_sel > 0)
    for (int i = i0; i < i1; ++i) {
      if (take_all) { above_bits |= 1ull << (i - i0); ++above_cnt; continue; }
      const uint64_t key = keys[i];
      const uint64_t off = key - thr_lo;
      if (off <= thr_hi_excl_width) { band_bits |= 1ull << (i - i0); ++band_cnt; }
      else if (key > thr_lo) { above_bits |= 1ull << (i - i0); ++above_cnt; }   // off wrapped <=> key < thr_lo
    }
  int tot_packed;
  const int before = block_excl_scan<NT>(above_cnt | (band_cnt << 16), s_warp, &tot_packed, scan_phase);   // (ends all reads of keys[])
  int above_rank = before & 0xffff, band_rank = before >> 16;
  const int tot_sel = (tot_packed & 0xffff) + min(tot_packed >> 16, need_in_band);
  int32_t* sel_s = reinterpret_cast<int32_t*>(keys);           // selected pages, ascending; reuses the key storage
  for (int i = i0; i < i1; ++i) {
    const uint64_t bit = 1ull << (i - i0);
    bool take = false;
    if (above_bits & bit) { take = true; }
    else if (band_bits & bit) { take = band_rank < need_in_band; }
    if (take) {
      const int pos = above_rank + min(band_rank, need_in_band);
      if (pos < k_max) sel_s[pos] = i;
    }
    if (above_bits & bit) ++above_rank;
    if (band_bits & bit) ++band_rank;
  }
  int count = min(tot_sel, k_max);
  if (forced && tid == 0 && count < k_max) sel_s[count] = n_pages - 1;
  if (forced) count = min(count + 1, k_max);
  __syncthreads();
  // Alg. 2: M.append(A[p]); A[p] <- t.  One selected page per thread, so the A gathers overlap.
  for (int i = tid; i < count; i += kTopkThreads) {
    const int j = sel_s[i];
    int prev = -1;
    if (A != nullptr) { prev = A[j]; A[j] = t; }
    out_pages[i] = j;
    out_prev[i] = prev;
  }
  for (int i = count + tid; i < k_max; i += kTopkThreads) { out_pages[i] = -1; out_prev[i] = -1; }
  if (tid == 0) sel_count[row] = count;
}

template <typename T, int D, bool kGroupMax>
__global__ void __launch_bounds__(kScoreWarps * 32, 3) select_pages_kernel(
    const T* __restrict__ q_cur, const T* bounds, const int32_t* __restrict__ seq_lens,
    const int32_t* __restrict__ budget_pages, int32_t* __restrict__ last_loaded, int32_t* __restrict__ sel_pages,
    int32_t* __restrict__ sel_prev, int32_t* __restrict__ sel_count, double* scores, double* __restrict__ scores_out,
    unsigned int* counters, int h_q, int h_k, int max_pages, int k_max, int P, int group_reduce, int force_last,
    int pages_per_cta /*multiple of kPagesPerCta*/,
    // S1 in line (retro_decode_step): the warp that owns the newest page recomputes its digest from the K tile,
    // patches the staged record and writes it back to `bounds`.  k_pages == NULL: digests are up to date.
    const T* __restrict__ k_pages, const int32_t* __restrict__ block_table, T* bounds_out) {
  static_assert(2 * D * sizeof(T) == 512, "digest record must be 512 bytes");
  constexpr int kVals = Rec<T>::kVals;
  // digest rings [warp][kStages][8 records x 512 B]; the unit's last CTA reuses the space for the top-k keys
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ double s_q[kGroupMax ? kMaxGroup : 1][2 * D];   // per q head: [q+ ; q-] (GROUP_MAX) ; row 0 = group sum (GROUP_SUM)
  __shared__ unsigned int s_ticket;
  pdl_wait();
  pdl_trigger();
  const int b = blockIdx.z, h = blockIdx.y;
  const int G = h_q / h_k;
  // the group's query values go out together with the length: the first round trip covers both (blockDim = 2 D)
  T q_raw[kMaxGroup];
  {
    const int c = threadIdx.x % D;
#pragma unroll
    for (int g = 0; g < kMaxGroup; ++g)
      if (g < G) q_raw[g] = q_cur[((size_t)b * h_q + h * G + g) * D + c];
  }
  const int budget_b = budget_pages[b];       // only the unit's last CTA needs it: fetched with the first round trip
  const int seq_len_b = seq_lens[b];
  const int n_pages = (seq_len_b + P - 1) / P;
  const int cta_page0 = blockIdx.x * pages_per_cta;
  const size_t row = ((size_t)b * h_k + h) * max_pages;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (scores_out != nullptr)   // test output: pages past the end read -inf
    for (int j = max(cta_page0, n_pages) + threadIdx.x; j < min(cta_page0 + pages_per_cta, max_pages); j += blockDim.x)
      scores_out[row + j] = -INFINITY;
  if (cta_page0 < n_pages) {
  // The digest stream does not depend on q: it starts before q is staged.  Every warp streams its own pages
  // (8 records = 4 KB per batch, lane l copies the 16 B it will read) with cp.async (LDGSTS, 16 B per lane) into a
  // warp-private ring of kStages buffers: bytes in flight are bounded by shared memory, not registers, and the
  // pipeline needs no CTA-wide barrier (cp.async.wait_group + __syncwarp per batch).
  const int page_end = min(cta_page0 + pages_per_cta, n_pages);
  const int nbatch = (page_end - cta_page0 + kPagesPerCta - 1) / kPagesPerCta;
  unsigned char* wring = smem_raw + (size_t)warp * kStages * (kPagesPerWarp * 512);
  auto issue_batch = [&](int it) {   // all lanes; always one commit group, possibly empty
    if (it < nbatch) {
      const int jb = cta_page0 + it * kPagesPerCta + warp * kPagesPerWarp;
      const uint32_t dst = smem_u32(wring + (size_t)(it % kStages) * (kPagesPerWarp * 512)) + lane * 16;
      const unsigned char* src = reinterpret_cast<const unsigned char*>(bounds + (row + jb) * 2 * D) + lane * 16;
#pragma unroll
      for (int i = 0; i < kPagesPerWarp; ++i)
        if (jb + i < n_pages)
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + i * 512), "l"(src + (size_t)i * 512)
                       : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
#pragma unroll
  for (int it = 0; it < kStages - 1; ++it) issue_batch(it);
  // S1 in line: the warp that will reduce the newest page (j_last) rebuilds its digest while the first batches fly
  const int j_last = n_pages - 1;
  const bool own_last = k_pages != nullptr && j_last >= cta_page0 && j_last < page_end &&
                        ((j_last - cta_page0) % kPagesPerCta) / kPagesPerWarp == warp;   // warp-uniform
  uint4 fresh = make_uint4(0, 0, 0, 0);
  if (own_last) {
    const int phys = block_table[(size_t)b * max_pages + j_last];
    const uint4* tile = reinterpret_cast<const uint4*>(k_pages + ((size_t)phys * h_k + h) * P * D);
    fresh = warp_page_digest<T, 16>(tile, seq_lens[b] - j_last * P, lane);
    reinterpret_cast<uint4*>(bounds_out + (row + j_last) * 2 * D)[lane] = fresh;
  }
  // q+ / q- in fp64 (exact), summed over the group for GROUP_SUM
  static_assert(kScoreWarps * 32 == 2 * D || kScoreWarps * 32 == 4 * D, "one thread per element of [q+ ; q-]");
  if (threadIdx.x < 2 * D) {
    const int i = threadIdx.x;
    const bool neg = i >= D;
    double acc = 0.0;
#pragma unroll
    for (int g = 0; g < kMaxGroup; ++g) {
      if (g < G) {
        const double qv = (double)Elem<T>::to_f32(q_raw[g]);
        const double part = neg ? fmin(qv, 0.0) : fmax(qv, 0.0);
        if (!kGroupMax) acc += part; else s_q[g][i] = part;
      }
    }
    if (!kGroupMax) s_q[0][i] = acc;
  }
  __syncthreads();
  double qreg[kVals];
#pragma unroll
  for (int c = 0; c < kVals; ++c) qreg[c] = s_q[0][lane * kVals + c];
  auto reduce_store = [&](unsigned char* wstage /*this warp's 8 records*/, int page0) {
    const int jbase = page0 + warp * kPagesPerWarp;
    const uint4* rec = reinterpret_cast<const uint4*>(wstage) + lane;
    if (own_last && j_last >= jbase && j_last < jbase + kPagesPerWarp)   // patch the staged (stale) record
      reinterpret_cast<uint4*>(wstage)[(j_last - jbase) * 32 + lane] = fresh;   // (each lane reads back its own 16 B)
    double acc[kPagesPerWarp];
    if constexpr (!kGroupMax) {
#pragma unroll
      for (int i = 0; i < kPagesPerWarp; ++i) {   // records past the last page hold stale bytes: their sums are
        double f[kVals];                            // computed branch-free and never stored
        Rec<T>::unpack(rec[i * 32], f);
        acc[i] = 0.0;
#pragma unroll
        for (int c = 0; c < kVals; ++c) acc[i] = fma(qreg[c], f[c], acc[i]);
      }
      // 8 sums over 32 lanes: three halving levels (4 + 2 + 1 exchanges) then two butterfly levels; the lanes
      // with (lane & 3) == 0 end up with page jbase + (lane >> 2)
      static_assert(kPagesPerWarp == 8, "halving reduction is written for 8 pages per warp");
      {
        const bool up = lane & 16;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const double send = up ? acc[i] : acc[i + 4], keep = up ? acc[i + 4] : acc[i];
          acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
        }
      }
      {
        const bool up = lane & 8;
#pragma unroll
        for (int i = 0; i < 2; ++i) {
          const double send = up ? acc[i] : acc[i + 2], keep = up ? acc[i + 2] : acc[i];
          acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
        }
      }
      double v;
      {
        const bool up = lane & 4;
        const double send = up ? acc[0] : acc[1], keep = up ? acc[1] : acc[0];
        v = keep + __shfl_xor_sync(0xffffffffu, send, 4);
      }
      v += __shfl_xor_sync(0xffffffffu, v, 2);
      v += __shfl_xor_sync(0xffffffffu, v, 1);
      const int j = jbase + (lane >> 2);
      if ((lane & 3) == 0 && j < n_pages) {
        scores[row + j] = v;
        if (scores_out != nullptr) scores_out[row + j] = v;
      }
    } else {
#pragma unroll
      for (int i = 0; i < kPagesPerWarp; ++i) {
        acc[i] = -INFINITY;
        if (jbase + i < n_pages) {
          double f[kVals];
          Rec<T>::unpack(rec[i * 32], f);
          for (int g = 0; g < G; ++g) {
            double a = 0.0;
#pragma unroll
            for (int c = 0; c < kVals; ++c) a = fma(s_q[g][lane * kVals + c], f[c], a);
            a = warp_sum(a);
            acc[i] = fmax(acc[i], a);
          }
        }
      }
      if (lane == 0) {
#pragma unroll
        for (int i = 0; i < kPagesPerWarp; ++i) {
          const int j = jbase + i;
          if (j < n_pages) {
            scores[row + j] = acc[i];
            if (scores_out != nullptr) scores_out[row + j] = acc[i];
          }
        }
      }
    }
  };
  for (int it = 0; it < nbatch; ++it) {
    issue_batch(it + kStages - 1);                     // refills the buffer reduced in the previous iteration
    asm volatile("cp.async.wait_group %0;" ::"n"(kStages - 1) : "memory");
    __syncwarp();
    reduce_store(wring + (size_t)(it % kStages) * (kPagesPerWarp * 512), cta_page0 + it * kPagesPerCta);
    __syncwarp();
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  }   // cta_page0 < n_pages
  // ---- the last CTA of the unit to get here selects (release: barrier, then one cumulative fence) ----
  const size_t unit = (size_t)b * h_k + h;
  __syncthreads();
  if (threadIdx.x == 0) s_ticket = ticket_acq_rel(&counters[unit]);
  __syncthreads();
  if (s_ticket != gridDim.x - 1) return;
  if (threadIdx.x == 0) counters[unit] = 0;   // leave the workspace consistent for the next call
  topk_mask_block<kScoreWarps * 32>(reinterpret_cast<uint64_t*>(smem_raw), scores, seq_len_b, budget_b,
                                    last_loaded, sel_pages, sel_prev, sel_count, b, h, h_k, max_pages, k_max, P,
                                    force_last);
}


int launch_select_pages(const retro_desc_t* d, const WorkspaceLayout& wl, const void* q_cur, const void* bounds,
                        const int32_t* seq_lens, const int32_t* budget_pages, int32_t* last_loaded,
                        int32_t* sel_pages, int32_t* sel_prev, int32_t* sel_count, double* scores_out,
                        void* workspace, cudaStream_t s, const void* k_pages_refresh, const int32_t* block_table) {
  char* ws = static_cast<char*>(workspace);
  double* scores = reinterpret_cast<double*>(ws + wl.scores_off);
  unsigned int* counters = reinterpret_cast<unsigned int*>(ws + wl.counters_off);   // [units] score-chunk arrivals
  // at most ONE wave of CTAs (three are resident per SM), each streaming whole batches of 64 pages: the per-CTA
  // costs (q staging, arrival ticket) amortise over several batches, and no unit waits for a second wave before
  // its last CTA can select
  const int units = d->batch * d->num_kv_heads;
  // a small digest set (latency-bound launch, e.g. 9 MB on C2) takes one CTA per SM: fewer, fatter CTAs and fewer
  // arrival tickets; a large one (bandwidth-bound) fills the three resident CTAs per SM
  const size_t digest_bytes = (size_t)units * d->max_pages_per_seq * 512;
  int nchunk = ((digest_bytes >= ((size_t)32 << 20) ? 3 : 1) * 148) / units;
  if (nchunk < 1) nchunk = 1;
  const int max_chunks = ceil_div(d->max_pages_per_seq, kPagesPerCta);
  if (nchunk > max_chunks) nchunk = max_chunks;
  const int pages_per_cta = ceil_div(ceil_div(d->max_pages_per_seq, nchunk), kPagesPerCta) * kPagesPerCta;
  dim3 grid(ceil_div(d->max_pages_per_seq, pages_per_cta), d->num_kv_heads, d->batch);
  const size_t keys_bytes = (size_t)d->max_pages_per_seq * sizeof(uint64_t);
  const size_t smem = keys_bytes > (size_t)kStages * kStageBytes ? keys_bytes : (size_t)kStages * kStageBytes;
  auto launch = [&](auto kern, auto* qp, auto* bp) -> int {
    auto* bw = bp;   // the same digest array, writable for the in-line S1 refresh
    // raise the dynamic shared-memory limit once per kernel instantiation (not a stream operation)
    std::lock_guard<std::mutex> lock(host_mutex());
    static const void* raised[8];
    static size_t raised_to[8];
    int slot = -1;
    for (int i = 0; i < 8 && slot < 0; ++i)
      if (raised[i] == (const void*)kern || raised[i] == nullptr) slot = i;
    if (slot < 0) slot = 0;
    if (raised[slot] != (const void*)kern || raised_to[slot] < smem) {
      RETRO_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      raised[slot] = (const void*)kern;
      raised_to[slot] = smem;
    }
    RETRO_CUDA_TRY(launch_kernel(kern, grid, dim3(kScoreWarps * 32), smem, s, qp, bp, seq_lens, budget_pages,
                                 last_loaded, sel_pages, sel_prev, sel_count, scores, scores_out, counters,
                                 d->num_q_heads, d->num_kv_heads, d->max_pages_per_seq, d->max_sel_pages,
                                 d->page_size, d->group_reduce, d->force_last_page, pages_per_cta,
                                 (decltype(qp))k_pages_refresh, block_table, const_cast<decltype(bw)>(bw)));
    return RETRO_OK;
  };
  const bool gmax = d->group_reduce == RETRO_GROUP_MAX;
  if (d->dtype == RETRO_BF16) {
    const auto* qp = (const __nv_bfloat16*)q_cur;
    const auto* bp = (const __nv_bfloat16*)bounds;
    return gmax ? launch(select_pages_kernel<__nv_bfloat16, 128, true>, qp, bp)
                : launch(select_pages_kernel<__nv_bfloat16, 128, false>, qp, bp);
  }
  const auto* qp = (const float*)q_cur;
  const auto* bp = (const float*)bounds;
  return gmax ? launch(select_pages_kernel<float, 64, true>, qp, bp)
              : launch(select_pages_kernel<float, 64, false>, qp, bp);
}

}  // namespace retro
