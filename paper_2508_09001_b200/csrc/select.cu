// S2  Quest page score (Eq. 1) + top-k under the budget + Alg. 2 mask build
// (PAPER.md:551-571).  One kernel, one thread-block CLUSTER per (sequence, KV head) unit.
//
// Score: HBM stream over the digests (512 B per (page, KV head)).  With q+ = max(q,0), q- = min(q,0) and
// Kmax >= Kmin, max(q*Kmin, q*Kmax) = q+*Kmax + q-*Kmin exactly, so the group-SUMMED score is one 2d-long dot
// product [sum_g q+ ; sum_g q-] . [Kmax ; Kmin] per page.  A digest record is exactly 32 lanes x 16 B: one
// coalesced 128-bit load per lane per page.
//
// Exact ranking at fp32 speed.  The stream is scored in fp32 (the fp32 -> fp64 conversions of an fp64 stream
// saturate the conversion pipe long before HBM) together with a rigorous bound on the fp32 error: with
// A_j = sum_c |q_c| |K_jc| (accumulated next to the score), |s32_j - s_j| <= eps_j = 2^-20 A_j (13 roundings on
// the summation path + the rounding of q, each <= 2^-24 A_j, with slack for the rounding of A_j itself).  The
// top-k runs on order-preserving 32-bit keys of s32.  Let T be the smallest selected and U the largest rejected
// fp32 score and eps = max_j eps_j: if T - U > 2 eps the selected SET is the exact fp64 one.  Otherwise only
// the pages with s32 in [T - 2 eps, U + 2 eps] are undecided: they are re-scored in fp64 (products of bf16 / fp32
// inputs are exact in fp64) and ranked exactly, ties to the lower page index; pages above the interval are
// selected for certain, pages below it rejected for certain.  The result is the fp64 oracle's set up to ties
// within ~1e-12 relative, as with the fp64 stream it replaces.
//
// Cluster: the CTAs of a unit each stream a slice of its pages and push the 32-bit keys straight into the LEADER
// CTA's shared memory (distributed shared memory), together with min / max key and max eps (remote atomics);
// one cluster barrier later the leader selects out of its own shared memory: no global score array, no
// arrival ticket, no reload.  Top-k: range-adaptive radix select (2048 buckets over [min,max] of the live range,
// 11 bits per pass, early exit when the threshold bucket is taken whole), then an in-order compaction emits
// ascending page indices with ties resolved to the lower index, and the same pass does Alg. 2's
// M.append(A[p]); A[p] <- t.
#include "common.cuh"
#include "digest.cuh"

namespace retro {

constexpr int kScoreWarps = 8;
constexpr int kSelThreads = kScoreWarps * 32;
constexpr int kPagesPerWarp = 8;                                  // records per warp batch (4 KB)
constexpr int kSelStages = 2;                                     // warp batches in flight per warp
constexpr int kWarpStageBytes = kPagesPerWarp * 512;              // 4 KB
constexpr int kRingBytes = kScoreWarps * kSelStages * kWarpStageBytes;   // 64 KB
constexpr int kBuckets = 2048;
constexpr int kMaxSelCluster = 16;

template <typename T> struct Rec;   // how a lane turns its 16 B of a digest record into numbers
template <> struct Rec<__nv_bfloat16> {
  static constexpr int kVals = 8;
  __device__ static __forceinline__ void unpack32(uint4 v, float* f) {
    f[0] = bf16_lo(v.x); f[1] = bf16_hi(v.x); f[2] = bf16_lo(v.y); f[3] = bf16_hi(v.y);
    f[4] = bf16_lo(v.z); f[5] = bf16_hi(v.z); f[6] = bf16_lo(v.w); f[7] = bf16_hi(v.w);
  }
  __device__ static __forceinline__ void unpack64(uint4 v, double* f) {
    f[0] = (double)bf16_lo(v.x); f[1] = (double)bf16_hi(v.x); f[2] = (double)bf16_lo(v.y); f[3] = (double)bf16_hi(v.y);
    f[4] = (double)bf16_lo(v.z); f[5] = (double)bf16_hi(v.z); f[6] = (double)bf16_lo(v.w); f[7] = (double)bf16_hi(v.w);
  }
};
template <> struct Rec<float> {
  static constexpr int kVals = 4;
  __device__ static __forceinline__ void unpack32(uint4 v, float* f) {
    f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y); f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
  }
  __device__ static __forceinline__ void unpack64(uint4 v, double* f) {
    f[0] = (double)__uint_as_float(v.x); f[1] = (double)__uint_as_float(v.y);
    f[2] = (double)__uint_as_float(v.z); f[3] = (double)__uint_as_float(v.w);
  }
};

// record = [Kmax (D) ; Kmin (D)] = 2*D*sizeof(T) = 512 B: lane l holds elements [l*kVals, (l+1)*kVals) of the
// concatenated vector, i.e. lanes 0..15 see Kmax channels, lanes 16..31 see Kmin channels.

// order-preserving integer images (larger score <=> larger key; -0.0 and +0.0 share one key)
__device__ __forceinline__ uint32_t order_key(float s) {
  const uint32_t u = __float_as_uint(s + 0.0f);
  return (u >> 31) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float key_score(uint32_t k) {
  return __uint_as_float((k >> 31) ? (k & 0x7fffffffu) : ~k);
}
__device__ __forceinline__ uint64_t order_key(double s) {
  const uint64_t u = (uint64_t)__double_as_longlong(s + 0.0);
  return (u >> 63) ? ~u : (u | 0x8000000000000000ull);
}
__device__ __forceinline__ int key_bits(uint32_t range) { return range == 0 ? 0 : 32 - __clz((int)range); }
__device__ __forceinline__ int key_bits(uint64_t range) { return range == 0 ? 0 : 64 - __clzll((long long)range); }

// 8 per-lane partial sums (one per page of the warp batch) over 32 lanes: three halving levels (4 + 2 + 1
// exchanges), then two butterfly levels; every lane ends with the total of page (lane >> 2).
template <typename V>
__device__ __forceinline__ V halving_reduce8(V (&acc)[8], int lane) {
  {
    const bool up = lane & 16;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const V send = up ? acc[i] : acc[i + 4], keep = up ? acc[i + 4] : acc[i];
      acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
  }
  {
    const bool up = lane & 8;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const V send = up ? acc[i] : acc[i + 2], keep = up ? acc[i + 2] : acc[i];
      acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
  }
  V v;
  {
    const bool up = lane & 4;
    const V send = up ? acc[0] : acc[1], keep = up ? acc[1] : acc[0];
    v = keep + __shfl_xor_sync(0xffffffffu, send, 4);
  }
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  return v;
}

// Exact fp64 score of one page from the 16 B of its record this lane holds; every lane returns the score.
template <typename T, int D, bool kGroupMax>
__device__ __forceinline__ double score64_rec(uint4 v, const double (*s_q)[2 * D], int G, int lane) {
  constexpr int kVals = Rec<T>::kVals;
  double f[kVals];
  Rec<T>::unpack64(v, f);
  if constexpr (!kGroupMax) {
    double a = 0.0;
#pragma unroll
    for (int c = 0; c < kVals; ++c) a = fma(s_q[0][lane * kVals + c], f[c], a);
    return warp_sum(a);
  } else {
    double best = -INFINITY;
    for (int g = 0; g < G; ++g) {
      double a = 0.0;
#pragma unroll
      for (int c = 0; c < kVals; ++c) a = fma(s_q[g][lane * kVals + c], f[c], a);
      best = fmax(best, warp_sum(a));
    }
    return best;
  }
}

// ------------------------------------------------------------------------------------------------
// top-k building blocks (one CTA of NT threads)
// ------------------------------------------------------------------------------------------------
struct TopkShared {
  int hist[kBuckets];                         // radix histogram
  unsigned int mask[kMaxPagesPerSeq / 32];    // "selected" bit per page (exact refinement only)
  int warp[64];                               // block scan, two alternating buffers
  unsigned long long red[2][32];
  unsigned long long lo, width;
  int need, done;
  unsigned int below;                         // largest key under the threshold band
};

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

// keys above lo + width are all taken; `need` of the keys in [lo, lo + width], in index order
template <typename Key> struct Band { Key lo, width; int need; };

// Range-adaptive radix select of the k_sel largest of keys[0..m) (0 < k_sel < m); [lo0, lo0 + range0] contains
// every key.  Ends with a band that is either taken whole or a single key value.  sh.hist must be zero on entry.
template <typename Key, int NT>
__device__ __forceinline__ Band<Key> radix_select(const Key* keys, int m, int k_sel, Key lo0, Key range0,
                                                  TopkShared& sh, int& scan_phase) {
  const int tid = threadIdx.x;
  if (tid == 0) { sh.lo = lo0; sh.width = range0; sh.need = k_sel; sh.done = 0; }
  __syncthreads();
  for (int pass = 0; pass < 8; ++pass) {
    const Key lo = (Key)sh.lo, range = (Key)sh.width;
    const int need = sh.need;
    const int nbits = key_bits(range);
    const int shift = nbits > 11 ? nbits - 11 : 0;
    if (pass > 0) {
      for (int i = tid; i < kBuckets; i += NT) sh.hist[i] = 0;
      __syncthreads();
    }
    for (int i0 = tid; i0 < m; i0 += 8 * NT) {     // loads first: they cannot be hoisted over the atomics
      Key kk[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) kk[u] = keys[min(i0 + u * NT, m - 1)];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const Key off = kk[u] - lo;
        if (i0 + u * NT < m && off <= range) atomicAdd(&sh.hist[(int)(off >> shift)], 1);
      }
    }
    __syncthreads();
    // thread i owns kBuckets / NT consecutive buckets, highest first: scanning threads in order walks buckets
    // downward
    constexpr int kPer = kBuckets / NT;
    int cbk[kPer], csum = 0;
#pragma unroll
    for (int u = 0; u < kPer; ++u) { cbk[u] = sh.hist[kBuckets - 1 - (tid * kPer + u)]; csum += cbk[u]; }
    int total;
    int run = block_excl_scan<NT>(csum, sh.warp, &total, scan_phase);   // keys in strictly higher buckets
    int hit = -1, above = 0, cnt = 0;
#pragma unroll
    for (int u = 0; u < kPer; ++u) {
      if (run < need && need <= run + cbk[u]) { hit = kBuckets - 1 - (tid * kPer + u); above = run; cnt = cbk[u]; }
      run += cbk[u];
    }
    if (hit >= 0) {
      const Key base = (Key)hit << shift;
      const Key width_m1 = shift == 0 ? (Key)0 : (Key)((((Key)1) << shift) - 1);
      sh.lo = lo + base;
      sh.width = (Key)(range - base) < width_m1 ? (Key)(range - base) : width_m1;
      sh.need = need - above;
      sh.done = (cnt == need - above || shift == 0) ? 1 : 0;
    }
    __syncthreads();
    if (sh.done) break;
  }
  Band<Key> b;
  b.lo = (Key)sh.lo; b.width = (Key)sh.width; b.need = sh.need;
  return b;
}

// In-order compaction of the selected candidates (thread owns a contiguous chunk of <= 64 indices): emit(pos, i)
// for the pos-th selected index i, ascending.  Returns the number selected; *band_pop = candidates inside the
// band.  With kTrackBelow the largest key under the band is folded into sh.below (zeroed by the caller).
template <typename Key, int NT, bool kTrackBelow, typename Emit>
__device__ __forceinline__ int compact_selected(const Key* keys, int m, bool take_all, bool take_none, Band<Key> band,
                                                TopkShared& sh, int& scan_phase, int* band_pop, Emit emit) {
  const int tid = threadIdx.x;
  const int per = (m + NT - 1) / NT;
  const int i0 = min(tid * per, m), i1 = min(i0 + per, m);
  // one packed scan: low 16 bits = candidates above the band (always taken), high bits = candidates inside it
  // (the first band.need of them, in index order, are taken); counts are <= kMaxPagesPerSeq < 2^15
  int above_cnt = 0, band_cnt = 0;
  uint64_t above_bits = 0, band_bits = 0;   // one bit per owned candidate: chunks are <= kMaxPagesPerSeq / NT = 64
  [[maybe_unused]] Key below = 0;
  if (!take_none)
    for (int i = i0; i < i1; ++i) {
      if (take_all) { above_bits |= 1ull << (i - i0); ++above_cnt; continue; }
      const Key key = keys[i];
      const Key off = key - band.lo;
      if (off <= band.width) { band_bits |= 1ull << (i - i0); ++band_cnt; }
      else if (key > band.lo) { above_bits |= 1ull << (i - i0); ++above_cnt; }   // off wrapped <=> key < band.lo
      else if (kTrackBelow) below = key > below ? key : below;
    }
  if constexpr (kTrackBelow) {
    const unsigned int wmax = __reduce_max_sync(0xffffffffu, (unsigned int)below);
    if ((tid & 31) == 0 && wmax > 0) atomicMax(&sh.below, wmax);
  }
  int tot_packed;
  const int before = block_excl_scan<NT>(above_cnt | (band_cnt << 16), sh.warp, &tot_packed, scan_phase);
  int above_rank = before & 0xffff, band_rank = before >> 16;
  const int need = take_all ? 0 : band.need;
  for (int i = i0; i < i1; ++i) {
    const uint64_t bit = 1ull << (i - i0);
    bool take = false;
    if (above_bits & bit) { take = true; }
    else if (band_bits & bit) { take = band_rank < need; }
    if (take) emit(above_rank + min(band_rank, need), i);
    if (above_bits & bit) ++above_rank;
    if (band_bits & bit) ++band_rank;
  }
  *band_pop = tot_packed >> 16;
  return (tot_packed & 0xffff) + min(tot_packed >> 16, need);
}

struct SelectParams {
  const void* q_cur; const void* bounds; const int32_t* seq_lens; const int32_t* budget_pages;
  int32_t* last_loaded; int32_t* sel_pages; int32_t* sel_prev; int32_t* sel_count;
  double* scores_out;            // optional fp64 scores (tests)
  unsigned long long* amb_keys;  // workspace [units][max_pages]: fp64 keys of the undecided pages (exact refinement)
  int32_t* amb_idx;              // workspace [units][max_pages]
  unsigned int* dbg;             // -DRETRO_DEBUG_CHECKS: violation counter in the workspace
  int h_q, h_k, max_pages, k_max, P, force_last, pages_per_cta;
  int prefetch_a;                // the leader stages the unit's row of A in shared memory
  // S1 in line (retro_decode_step): the warp that owns the newest page recomputes its digest from the K tile,
  // patches the staged record and writes it back to `bounds`.  k_pages == NULL: digests are up to date.
  const void* k_pages; const int32_t* block_table; void* bounds_out;
};

template <typename T, int D, bool kGroupMax, bool kEmit64>
__global__ void __launch_bounds__(kSelThreads, 2) select_pages_kernel(const SelectParams p) {
  static_assert(2 * D * sizeof(T) == 512, "digest record must be 512 bytes");
  constexpr int kVals = Rec<T>::kVals;
  constexpr int NT = kSelThreads;
  // [ring: warp-private digest stages, 64 KB][keys: uint32 per page; the LEADER's copy holds the whole unit]
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ double s_q[kGroupMax ? kMaxGroup : 1][2 * D];   // per q head: [q+ ; q-] (GROUP_MAX) ; row 0 = group sum
  __shared__ TopkShared sh;
  __shared__ unsigned int s_kmin, s_kmax, s_epsbits;          // the leader's copies are written by the whole cluster
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t rank = cluster_ctarank();
  uint32_t* keys = reinterpret_cast<uint32_t*>(smem_raw + kRingBytes);
  int32_t* s_A = reinterpret_cast<int32_t*>(smem_raw + kRingBytes + (((size_t)p.max_pages * 4 + 15) & ~(size_t)15));
  if (tid == 0) { s_kmin = 0xffffffffu; s_kmax = 0u; s_epsbits = 0u; sh.below = 0u; }
  for (int i = tid; i < kBuckets; i += NT) sh.hist[i] = 0;
  cluster_arrive();            // (#0) the leader's accumulators are initialised before anybody adds to them
  pdl_wait();
  pdl_trigger();
  // Alg. 2 reads A[p] of the selected pages: the leader prefetches the unit's row of A (it does not depend on
  // anything this kernel computes), so the selection tail has no global round trip left
  if (p.last_loaded != nullptr && p.prefetch_a && rank == 0) {
    const int32_t* a_src = p.last_loaded + ((size_t)blockIdx.z * p.h_k + blockIdx.y) * p.max_pages;
#pragma unroll 1
    for (int i = tid; i < p.max_pages; i += NT)
      asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(s_A + i)), "l"(a_src + i) : "memory");
  }
  asm volatile("cp.async.commit_group;" ::: "memory");
  const T* q_cur = reinterpret_cast<const T*>(p.q_cur);
  const T* bounds = reinterpret_cast<const T*>(p.bounds);
  const int b = blockIdx.z, h = blockIdx.y;
  const int G = p.h_q / p.h_k;
  // the group's query values go out together with the length: the first round trip covers both (blockDim = 2 D)
  T q_raw[kMaxGroup];
  {
    const int c = tid % D;
#pragma unroll
    for (int g = 0; g < kMaxGroup; ++g)
      if (g < G) q_raw[g] = q_cur[((size_t)b * p.h_q + h * G + g) * D + c];
  }
  int budget_b = p.budget_pages[b];           // only the leader needs it: fetched with the first round trip
  int seq_len_b = p.seq_lens[b];
  RETRO_DBG_ONLY(if (seq_len_b < 0 || seq_len_b > p.max_pages * p.P) { if (tid == 0 && rank == 0) dbg_violation(p.dbg, kDbgSeqLen); seq_len_b = 0; })
  RETRO_DBG_ONLY(if (budget_b < 0) { if (tid == 0 && rank == 0) dbg_violation(p.dbg, kDbgBudget); budget_b = 0; })
  const int n_pages = min((seq_len_b + p.P - 1) / p.P, p.max_pages);   // a sequence never outgrows its block-table row
  const int cta_page0 = (int)rank * p.pages_per_cta;
  const int page_end = min(cta_page0 + p.pages_per_cta, n_pages);
  const size_t row = ((size_t)b * p.h_k + h) * p.max_pages;
  if constexpr (kEmit64) {   // test output: pages past the end read -inf
    for (int j = max(cta_page0, n_pages) + tid; j < min(cta_page0 + p.pages_per_cta, p.max_pages); j += NT)
      p.scores_out[row + j] = -INFINITY;
  }
  // The digest stream does not depend on q: it starts before q is staged.  Every warp streams its own pages
  // (8 records = 4 KB per batch, lane l copies the 16 B it will read) with cp.async (LDGSTS, 16 B per lane) into a
  // warp-private ring of kSelStages buffers: bytes in flight are bounded by shared memory, not registers, and the
  // pipeline needs no CTA-wide barrier (cp.async.wait_group + __syncwarp per batch).
  constexpr int kCtaBatch = kScoreWarps * kPagesPerWarp;
  const int nbatch = page_end > cta_page0 ? (page_end - cta_page0 + kCtaBatch - 1) / kCtaBatch : 0;
  unsigned char* wring = smem_raw + (size_t)warp * kSelStages * kWarpStageBytes;
  auto batch_page0 = [&](int it) { return cta_page0 + (it * kScoreWarps + warp) * kPagesPerWarp; };
  auto issue_batch = [&](int it) {   // all lanes; always one commit group, possibly empty
    if (it < nbatch) {
      const int jb = batch_page0(it);
      const uint32_t dst = smem_u32(wring + (size_t)(it % kSelStages) * kWarpStageBytes) + lane * 16;
      const unsigned char* src = reinterpret_cast<const unsigned char*>(bounds + (row + jb) * 2 * D) + lane * 16;
#pragma unroll
      for (int i = 0; i < kPagesPerWarp; ++i)
        if (jb + i < page_end)
          asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + i * 512), "l"(src + (size_t)i * 512)
                       : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
#pragma unroll
  for (int it = 0; it < kSelStages - 1; ++it) issue_batch(it);
  // q+ / q- in fp64 (exact), summed over the group for GROUP_SUM
  static_assert(NT == 2 * D || NT == 4 * D, "one thread per element of [q+ ; q-]");
  if (tid < 2 * D) {
    const bool neg = tid >= D;
    double acc = 0.0;
#pragma unroll
    for (int g = 0; g < kMaxGroup; ++g) {
      if (g < G) {
        const double qv = (double)Elem<T>::to_f32(q_raw[g]);
        const double part = neg ? fmin(qv, 0.0) : fmax(qv, 0.0);
        if (!kGroupMax) acc += part; else s_q[g][tid] = part;
      }
    }
    if (!kGroupMax) s_q[0][tid] = acc;
  }
  __syncthreads();
  // S1 in line: the warp that will reduce the newest page (j_last) rebuilds its digest while its batches fly (after
  // the barrier above: its two dependent round trips must not hold up the other warps of the CTA)
  const int j_last = n_pages - 1;
  const bool own_last = p.k_pages != nullptr && j_last >= cta_page0 && j_last < page_end &&
                        ((j_last - cta_page0) / kPagesPerWarp) % kScoreWarps == warp;   // warp-uniform
  uint4 fresh = make_uint4(0, 0, 0, 0);
  if (own_last) {
    const int phys = p.block_table[(size_t)b * p.max_pages + j_last];
    const uint4* tile = reinterpret_cast<const uint4*>(reinterpret_cast<const T*>(p.k_pages) +
                                                       ((size_t)phys * p.h_k + h) * p.P * D);
    fresh = warp_page_digest<T, 16>(tile, min(seq_len_b - j_last * p.P, p.P), lane);
    reinterpret_cast<uint4*>(reinterpret_cast<T*>(p.bounds_out) + (row + j_last) * 2 * D)[lane] = fresh;
  }
  cluster_wait();              // (#0)
  const uint32_t keys_leader = dsmem_addr(smem_u32(keys), 0);
  float qreg[kVals], qabs[kVals];   // fp32 image of [sum q+ ; sum q-] (one rounding, inside eps) and its magnitude
#pragma unroll
  for (int c = 0; c < kVals; ++c) { qreg[c] = (float)s_q[0][lane * kVals + c]; qabs[c] = fabsf(qreg[c]); }
  uint32_t my_kmin = 0xffffffffu, my_kmax = 0u;
  float my_eps = 0.f;
  for (int it = 0; it < nbatch; ++it) {
    issue_batch(it + kSelStages - 1);                  // refills the buffer reduced in the previous iteration
    asm volatile("cp.async.wait_group %0;" ::"n"(kSelStages - 1) : "memory");
    __syncwarp();
    unsigned char* wstage = wring + (size_t)(it % kSelStages) * kWarpStageBytes;
    const int jbase = batch_page0(it);
    const uint4* rec = reinterpret_cast<const uint4*>(wstage) + lane;
    if (own_last && j_last >= jbase && j_last < jbase + kPagesPerWarp)        // patch the staged (stale) record
      reinterpret_cast<uint4*>(wstage)[(j_last - jbase) * 32 + lane] = fresh;   // (each lane reads back its own 16 B)
    float s32, e32;
    if constexpr (!kGroupMax) {
      float acc[kPagesPerWarp], aab[kPagesPerWarp];
#pragma unroll
      for (int i = 0; i < kPagesPerWarp; ++i) {   // records past the last page hold stale bytes: their sums are
        float f[kVals];                             // computed branch-free and never stored
        Rec<T>::unpack32(rec[i * 32], f);
        acc[i] = 0.f; aab[i] = 0.f;
#pragma unroll
        for (int c = 0; c < kVals; ++c) {
          acc[i] = fmaf(qreg[c], f[c], acc[i]);
          aab[i] = fmaf(qabs[c], fabsf(f[c]), aab[i]);
        }
      }
      static_assert(kPagesPerWarp == 8, "halving reduction is written for 8 pages per warp");
      s32 = halving_reduce8(acc, lane);
      e32 = halving_reduce8(aab, lane) * 9.5463e-7f;   // 2^-20 (1 + 2^-10)
      if constexpr (kEmit64) {
#pragma unroll 1
        for (int i = 0; i < kPagesPerWarp; ++i) {
          if (jbase + i >= page_end) break;
          const double s64 = score64_rec<T, D, kGroupMax>(rec[i * 32], s_q, G, lane);
          if (lane == 0) p.scores_out[row + jbase + i] = s64;
        }
      }
    } else {
      // GROUP_MAX: the maximum over the group's q heads is taken on exact fp64 scores; the 32-bit key is their
      // rounding (eps = one fp32 rounding), so the exact refinement sees the same values
      double mine = 0.0;
#pragma unroll 1
      for (int i = 0; i < kPagesPerWarp; ++i) {
        if (jbase + i >= page_end) break;
        const double s64 = score64_rec<T, D, kGroupMax>(rec[i * 32], s_q, G, lane);
        if (kEmit64 && lane == 0) p.scores_out[row + jbase + i] = s64;
        if ((lane >> 2) == i) mine = s64;
      }
      s32 = (float)mine;
      e32 = fabsf(s32) * 1.2e-7f + 1e-37f;
    }
    const int j = jbase + (lane >> 2);
    if ((lane & 3) == 0 && j < page_end) {
      const uint32_t key = order_key(s32);
      dsmem_st_u32(keys_leader + (uint32_t)j * 4u, key);
      my_kmin = min(my_kmin, key);
      my_kmax = max(my_kmax, key);
      my_eps = fmaxf(my_eps, e32);
    }
    __syncwarp();
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  if (nbatch > 0) {
    my_kmin = __reduce_min_sync(0xffffffffu, my_kmin);
    my_kmax = __reduce_max_sync(0xffffffffu, my_kmax);
    const uint32_t eb = __reduce_max_sync(0xffffffffu, __float_as_uint(my_eps));   // eps >= 0: bit order = value order
    if (lane == 0 && my_kmin <= my_kmax) {
      dsmem_red_min_u32(dsmem_addr(smem_u32(&s_kmin), 0), my_kmin);
      dsmem_red_max_u32(dsmem_addr(smem_u32(&s_kmax), 0), my_kmax);
      dsmem_red_max_u32(dsmem_addr(smem_u32(&s_epsbits), 0), eb);
    }
  }
  cluster_arrive();            // (#1) every key of the unit is in the leader's shared memory
  cluster_wait();
  if (rank != 0) return;

  // ---- the leader selects ------------------------------------------------------------------------------------
  const int t = seq_len_b - 1;
  int k = min(min(budget_b, n_pages), p.k_max);
  k = max(k, 0);
  const size_t unit = (size_t)b * p.h_k + h;
  int32_t* out_pages = p.sel_pages + unit * p.k_max;
  int32_t* out_prev = p.sel_prev + unit * p.k_max;
  int32_t* A = p.last_loaded != nullptr ? p.last_loaded + unit * p.max_pages : nullptr;
  // candidates 0..m-1 compete for k_sel places; the newest page is appended last when forced
  const bool forced = p.force_last && k > 0 && k < n_pages;
  const int m = forced ? n_pages - 1 : n_pages;
  const int k_sel = forced ? k - 1 : k;
  const bool take_all = k_sel >= m, take_none = k_sel <= 0;
  int scan_phase = 0;
  int32_t* sel_s = reinterpret_cast<int32_t*>(smem_raw);   // selected pages, ascending (the ring is idle now)
  Band<uint32_t> band{0u, 0u, 0};
  if (!take_all && !take_none)
    band = radix_select<uint32_t, NT>(keys, m, k_sel, s_kmin, s_kmax - s_kmin, sh, scan_phase);
  int band_pop = 0;
  int tot_sel = compact_selected<uint32_t, NT, true>(keys, m, take_all, take_none, band, sh, scan_phase, &band_pop,
                                                    [&](int pos, int i) { if (pos < p.k_max) sel_s[pos] = i; });
  if (!take_all && !take_none) {
    __syncthreads();                                   // sh.below complete
    // T = smallest selected fp32 score (>= the band's lower end); U = largest rejected one: the band's own value
    // when the band is a single tied value that was not taken whole, else the largest key under the band
    const double eps = (double)__uint_as_float(s_epsbits);
    const double sT = (double)key_score(band.lo);
    const bool band_split = band.need < band_pop;
    const bool has_rejected = band_split || sh.below != 0u;
    const double sU = band_split ? (double)key_score(band.lo + band.width) : (double)key_score(sh.below);
    if (has_rejected && !(sT - sU > 2.0 * eps)) {
      // ---- exact refinement (rare): re-score the undecided pages in fp64, rank them exactly ----
      const double lo_s = sT - 2.0 * eps, hi_s = sU + 2.0 * eps;   // undecided: lo_s <= s32 <= hi_s; above: selected
      for (int i = tid; i < kMaxPagesPerSeq / 32; i += NT) sh.mask[i] = 0u;
      __syncthreads();
      uint64_t* keys64 = reinterpret_cast<uint64_t*>(p.amb_keys) + unit * p.max_pages;
      int32_t* amb_idx = p.amb_idx + unit * p.max_pages;
      const int per = (m + NT - 1) / NT;
      const int i0 = min(tid * per, m), i1 = min(i0 + per, m);
      int n_amb = 0, n_sure = 0;
      uint64_t amb_bits = 0;
      for (int i = i0; i < i1; ++i) {
        const double s = (double)key_score(keys[i]);
        if (s > hi_s) { atomicOr(&sh.mask[i >> 5], 1u << (i & 31)); ++n_sure; }
        else if (s >= lo_s) { amb_bits |= 1ull << (i - i0); ++n_amb; }
      }
      int tot_packed;
      int pos = block_excl_scan<NT>(n_amb | (n_sure << 16), sh.warp, &tot_packed, scan_phase) & 0xffff;
      for (int i = i0; i < i1; ++i)
        if (amb_bits & (1ull << (i - i0))) amb_idx[pos++] = i;
      const int ma = tot_packed & 0xffff, need2 = k_sel - (tot_packed >> 16);
      __syncthreads();
      for (int a = warp; a < ma; a += NT / 32) {       // one warp per undecided page
        const int j = amb_idx[a];
        const uint4 v = __ldcg(reinterpret_cast<const uint4*>(bounds + (row + j) * 2 * D) + lane);
        const double s64 = score64_rec<T, D, kGroupMax>(v, s_q, G, lane);
        if (lane == 0) keys64[a] = order_key(s64);
      }
      for (int i = tid; i < kBuckets; i += NT) sh.hist[i] = 0;
      __syncthreads();
      const bool all2 = need2 >= ma, none2 = need2 <= 0;
      Band<uint64_t> band2{0ull, 0ull, 0};
      if (!all2 && !none2) {
        uint64_t kmin = ~0ull, kmax = 0ull;
        for (int i = tid; i < ma; i += NT) {
          const uint64_t key = keys64[i];
          kmin = key < kmin ? key : kmin;
          kmax = key > kmax ? key : kmax;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          const uint64_t a = __shfl_xor_sync(0xffffffffu, kmin, o), c = __shfl_xor_sync(0xffffffffu, kmax, o);
          kmin = a < kmin ? a : kmin;
          kmax = c > kmax ? c : kmax;
        }
        if (lane == 0) { sh.red[0][warp] = kmin; sh.red[1][warp] = kmax; }
        __syncthreads();
        kmin = ~0ull; kmax = 0ull;
        for (int w = 0; w < NT / 32; ++w) {
          kmin = sh.red[0][w] < kmin ? sh.red[0][w] : kmin;
          kmax = sh.red[1][w] > kmax ? sh.red[1][w] : kmax;
        }
        band2 = radix_select<uint64_t, NT>(keys64, ma, need2, kmin, kmax - kmin, sh, scan_phase);
      }
      int pop2;
      (void)compact_selected<uint64_t, NT, false>(keys64, ma, all2, none2, band2, sh, scan_phase, &pop2,
                                                  [&](int, int a) {
                                                    const int j = amb_idx[a];
                                                    atomicOr(&sh.mask[j >> 5], 1u << (j & 31));
                                                  });
      __syncthreads();
      // final in-order compaction over the mask
      int c = 0;
      for (int i = i0; i < i1; ++i) c += (sh.mask[i >> 5] >> (i & 31)) & 1u;
      int tot;
      int at = block_excl_scan<NT>(c, sh.warp, &tot, scan_phase);
      for (int i = i0; i < i1; ++i)
        if ((sh.mask[i >> 5] >> (i & 31)) & 1u) { if (at < p.k_max) sel_s[at] = i; ++at; }
      tot_sel = tot;
    }
  }
  int count = min(tot_sel, p.k_max);
  if (forced && tid == 0 && count < p.k_max) sel_s[count] = n_pages - 1;
  if (forced) count = min(count + 1, p.k_max);
  __syncthreads();
  // Alg. 2: M.append(A[p]); A[p] <- t.  One selected page per thread, so the A gathers overlap.
  for (int i = tid; i < count; i += NT) {
    const int j = sel_s[i];
    int prev = -1;
    if (A != nullptr) { prev = p.prefetch_a ? s_A[j] : A[j]; A[j] = t; }
    out_pages[i] = j;
    out_prev[i] = prev;
  }
  for (int i = count + tid; i < p.k_max; i += NT) { out_pages[i] = -1; out_prev[i] = -1; }
  if (tid == 0) p.sel_count[unit] = count;
}

int launch_select_pages(const retro_desc_t* d, const WorkspaceLayout& wl, const void* q_cur, const void* bounds,
                        const int32_t* seq_lens, const int32_t* budget_pages, int32_t* last_loaded,
                        int32_t* sel_pages, int32_t* sel_prev, int32_t* sel_count, double* scores_out,
                        void* workspace, cudaStream_t s, const void* k_pages_refresh, const int32_t* block_table) {
  char* ws = static_cast<char*>(workspace);
  SelectParams prm;
  prm.q_cur = q_cur; prm.bounds = bounds; prm.seq_lens = seq_lens; prm.budget_pages = budget_pages;
  prm.last_loaded = last_loaded; prm.sel_pages = sel_pages; prm.sel_prev = sel_prev; prm.sel_count = sel_count;
  prm.scores_out = scores_out;
  prm.amb_keys = reinterpret_cast<unsigned long long*>(ws + wl.scores_off);
  prm.amb_idx = reinterpret_cast<int32_t*>(ws + wl.amb_idx_off);
  prm.h_q = d->num_q_heads; prm.h_k = d->num_kv_heads; prm.max_pages = d->max_pages_per_seq;
  prm.k_max = d->max_sel_pages; prm.P = d->page_size; prm.force_last = d->force_last_page;
  prm.pages_per_cta = 0;
  prm.prefetch_a = 0;
  prm.dbg = reinterpret_cast<unsigned int*>(ws + wl.debug_off);
  prm.k_pages = k_pages_refresh; prm.block_table = block_table; prm.bounds_out = const_cast<void*>(bounds);
  const DeviceInfo di = device_info();
  const int units = d->batch * d->num_kv_heads;
  const size_t keys_bytes = ((size_t)d->max_pages_per_seq * 4 + 15) & ~(size_t)15;
  auto launch = [&](auto kern) -> int {
    // How many CTAs (= cluster size) stream one unit, and whether the leader prefetches the unit's row of A.  A
    // plan's cost = pages the busiest SM streams + a fixed latency (worth ~350 pages) per wave of resident clusters
    // (cudaOccupancyMaxActiveClusters knows how many clusters of that size and shared-memory footprint the device
    // keeps resident: e.g. 15 of size 8 at one CTA per SM on a B200); within 2 % the plan with more CTAs wins (more
    // bytes in flight), then the one that prefetches.
    int best_n = 1, best_pref = 0;
    double best_cost = 1e30;
    const int max_chunks = ceil_div(d->max_pages_per_seq, kPagesPerWarp);
    for (int pref = 0; pref <= (last_loaded != nullptr ? 1 : 0); ++pref)
      for (int n = 1; n <= kMaxSelCluster; ++n) {
        if ((n > 8 && n != 16) || n > max_chunks) continue;
        const size_t smem = (size_t)kRingBytes + keys_bytes * (1 + pref);
        const int cap = max_active_clusters((const void*)kern, kSelThreads, smem, n);
        if (cap <= 0) continue;
        const int ppc = ceil_div(ceil_div(d->max_pages_per_seq, n), kPagesPerWarp) * kPagesPerWarp;
        const double cost = (double)ceil_div(units * n, di.sm_count) * ppc + 350.0 * ceil_div(units, cap);
        if (cost <= best_cost * 1.02) { best_n = n; best_pref = pref; best_cost = cost < best_cost ? cost : best_cost; }
      }
    const size_t smem = (size_t)kRingBytes + keys_bytes * (1 + best_pref);
    const int rc = ensure_dynamic_smem((const void*)kern, smem);
    if (rc != RETRO_OK) return rc;
    prm.prefetch_a = best_pref;
    prm.pages_per_cta = ceil_div(ceil_div(d->max_pages_per_seq, best_n), kPagesPerWarp) * kPagesPerWarp;
    RETRO_CUDA_TRY(launch_cluster_kernel(kern, dim3(best_n, d->num_kv_heads, d->batch), dim3(kSelThreads), smem, s,
                                         best_n, prm));
    return RETRO_OK;
  };
  const bool gmax = d->group_reduce == RETRO_GROUP_MAX;
  const bool emit = scores_out != nullptr;
  if (d->dtype == RETRO_BF16) {
    if (gmax) return emit ? launch(select_pages_kernel<__nv_bfloat16, 128, true, true>)
                          : launch(select_pages_kernel<__nv_bfloat16, 128, true, false>);
    return emit ? launch(select_pages_kernel<__nv_bfloat16, 128, false, true>)
                : launch(select_pages_kernel<__nv_bfloat16, 128, false, false>);
  }
  if (gmax) return emit ? launch(select_pages_kernel<float, 64, true, true>)
                        : launch(select_pages_kernel<float, 64, true, false>);
  return emit ? launch(select_pages_kernel<float, 64, false, true>)
              : launch(select_pages_kernel<float, 64, false, false>);
}

}  // namespace retro
