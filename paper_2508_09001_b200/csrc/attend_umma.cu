// S3 on the 5th-generation tensor cores (bf16, d = 128, P = 16): the GQA group x (w+1) query block against
// the selected pages is a dense contraction (Eq. 2 / 6 / 7; arithmetic intensity ~ rows
// flop per KV byte), far above what the fp32 ALUs sustain at HBM rate once rows > ~8.
//
// Per block of 8 pages (128 keys), two tensor-core passes; keys sit on the 128 TMEM lanes of S, query rows on N,
// so no tensor-core or softmax work is spent on row padding and every softmax thread owns one key:
//   S^T = K Q^T     A = K block [128 keys x 128 ch] (K-major, TMA SW128), B = Q [NT rows x 128 ch], N = NT
//                   -> TMEM S [lane = key][column = row]
//   O^T += V^T P^T  A = V block (MN-major, M = 128 channels), B = [P_hi | P_lo] [128 keys x 2 NT] (MN-major),
//                   N = 2 NT -> TMEM O [lane = channel][column = row (hi) | NT + row (lo)]; O = O_hi + O_lo.
// Measured on B200 (probe: one tcgen05.mma costs ~42 + N/2 cycles with A from shared memory, M = 64 or 128):
// the fixed part is the A fetch, so the P hi / lo halves share one MMA (stacked on N) instead of two.
// P = 2^(s*scale - m_ref[row]) with the retrospective mask (page j is visible to the row at position p iff
// sel_prev_j < p; token l iff l <= p) goes to shared memory as bf16 hi + bf16 lo: a single bf16 P (2^-9) leaves
// |err| ~ 2^-9 |v| on the x8 outlier channels of V, outside the 2e-2 tolerance, and the hardware rejects a bf16
// A with an fp16 B operand.  Row sums L are accumulated in registers by the softmax threads (one key each) and
// reduced once per CTA.  m_ref is a per-row reference in shared memory; it is raised (and O, L rescaled) only
// when some logit exceeds it by more than 64 (log2 units: bf16 and fp32 share the exponent range, so P up to
// 2^64 costs no precision), so the common block needs no reduction.
//
// One CTA per (split, row group, KV head, sequence), 640 threads, warp-specialised; the splits of a (unit, row
// group) are the CTAs of one thread-block cluster (<= 8):
//   warp 0, 1   TMA producers, one for K and one for V (separate rings of 32 KB slots = 8 pages = 128 keys, so a
//               K block never queues behind the longer-lived V block): every selected (page, head) tile arrives
//               as two 64-channel boxes with the 128-byte swizzle (cp.async.bulk.tensor.2d + mbarrier).
//   warp 2      MMA issuer (converged warp, elect.sync: the operands stay in uniform registers), owns the TMEM
//               allocation; tcgen05.commit signals mbarriers.
//   warp 3      S4 service (fused step only; also keeps the softmax warps aligned to the TMEM lane quadrants):
//               prefetches this CTA's output-cache operands into shared memory, snapshots cache_pos, takes the
//               cross-head arrival ticket whose last holder rewrites cache_pos.
//   warps 4..19 softmax: TMEM lane quadrant = warp % 4 (32 keys), column group = (warp - 4) / 4 (a quarter of the rows).
// Every page is read from HBM once and serves all rows.  Epilogue: every split stages its normalised partial (fp16
// tile + base-2 lse) in its own shared memory, one cluster barrier, then each CTA merges a share of the
// (cache slot, q head) items, reading the other splits' rows through distributed shared memory (Eq. 8 over the
// splits), and - inside retro_decode_step - merges with the cached (o, lse) and writes out / cache (S4, Eq. 8-9).
// In the fused step everything that does not depend on this step's selection runs before griddepcontrol.wait.
#include <cuda.h>
#include <cuda_fp16.h>

#include <cstdlib>

#include "attend_common.cuh"

namespace retro {

constexpr int kUmmaThreads = 640;
constexpr int kSoftmaxThreads = 512;
constexpr int kPB = 8;                        // pages per KV block (128 keys)
constexpr int kTileHalfBytes = 16 * 128;      // one (page, head, 64-channel half) box: 16 rows x 128 B
constexpr int kHalfStride = kPB * kTileHalfBytes;   // 16 KB: [half][page][16][128 B]
constexpr int kSlotBytes = 2 * kHalfStride;   // 32 KB: one K block or one V block
constexpr int kTmemCols = 512;
constexpr int kUmmaSmemBudget = 232448 - 1024 - 4096;   // dynamic shared memory the launcher plans with (one CTA per SM)
constexpr int kMaxNT = 128;                   // rows padded to 16; larger row blocks take the scalar path
constexpr float kRescaleThreshold = 64.f;     // log2 units: P <= 2^64, sums stay far below the fp32 / bf16 range
constexpr float kMrefInit = -1.0e30f;         // finite "row not started" reference: -inf - kMrefInit stays -inf

// ---- PTX wrappers -------------------------------------------------------------------------------
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(smem_u32(smem_dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(smem_u32(bar))
      : "memory");
}
// One lane of a converged warp; code under it is single-threaded, so tensor-map / descriptor operands need no
// per-lane "waterfall" loop (a plain lane == 0 test costs ~90 cycles per tcgen05.mma or TMA instruction).
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                          uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// P is handed to the tensor core as a bf16 hi + bf16 lo pair (two MMAs per K step, 16 mantissa bits): a single
// bf16 P (2^-9) leaves |err| ~ 2^-9 * |v| on the x8 outlier channels of V, outside the 2e-2 tolerance.
__device__ __forceinline__ void split_bf16x2(float e0, float e1, uint32_t& hi, uint32_t& lo) {
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(hi) : "f"(e1), "f"(e0));
  const float r0 = e0 - __uint_as_float(hi << 16), r1 = e1 - __uint_as_float(hi & 0xffff0000u);
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(lo) : "f"(r1), "f"(r0));
}
// Shared-memory matrix descriptors (cute::UMMA::SmemDescriptor bit layout), 128B swizzle, version 1.
// K-major operand (rows of 128 B = 64 bf16 along K; 8-row groups SBO = 1024 B apart).
__device__ __forceinline__ uint64_t desc_kmajor_sw128(uint32_t saddr) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) |
         ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
// MN-major operand (64 MN-elements = 128 B contiguous; the next 64 are LBO away; 8-deep K groups SBO apart).
__device__ __forceinline__ uint64_t desc_mnmajor_sw128(uint32_t saddr, uint32_t lbo_bytes) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(1024 >> 4) << 32) |
         ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
// Instruction descriptor (cute::UMMA::InstrDescriptor): D = f32, A = B = bf16, M = 128, N = n.
__device__ __forceinline__ uint32_t idesc_bf16_ab(int n, bool a_mn_major, bool b_mn_major) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((a_mn_major ? 1u : 0u) << 15) |
         ((b_mn_major ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}
__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float lg2_approx(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ void tmem_ld4(uint32_t taddr, uint32_t* r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
               : "r"(taddr)
               : "memory");
}
__device__ __forceinline__ void tmem_st4(uint32_t taddr, const uint32_t* r) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};"
               ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3])
               : "memory");
}
__device__ __forceinline__ void store_bf16x4(__nv_bfloat16* dst, float4 v) {
  __nv_bfloat162 a = __floats2bfloat162_rn(v.x, v.y), c = __floats2bfloat162_rn(v.z, v.w);
  uint2 u;
  u.x = *reinterpret_cast<uint32_t*>(&a);
  u.y = *reinterpret_cast<uint32_t*>(&c);
  *reinterpret_cast<uint2*>(dst) = u;
}
__device__ __forceinline__ void softmax_bar() { asm volatile("bar.sync 1, 512;" ::: "memory"); }
// order-preserving float <-> int image (signed compare), so a column max is one REDUX + one shared atomicMax
__device__ __forceinline__ int f2o(float f) {
  const int i = __float_as_int(f);
  return i >= 0 ? i : i ^ 0x7fffffff;
}
__device__ __forceinline__ float o2f(int i) { return __int_as_float(i >= 0 ? i : i ^ 0x7fffffff); }
constexpr int kOrdNegInf = (int)0x807fffff;   // f2o(-inf)

// Dynamic shared memory map (1024 B aligned).  NT = padded rows, NS = ring slots, NP = P buffers.
constexpr int kPreItems = 16;                 // output-cache operands a CTA prefetches for its merge items
constexpr int kPreStride = 132;               // floats per prefetched item: o[128], lse, padding (16 B multiple)
struct UmmaLayout {
  int q, p, ring, list, pre, bt, total;
  int p_buf_bytes, p_hl_bytes;
};
__host__ __device__ inline UmmaLayout umma_layout(int NT, int NS, int NP, int pages_per_split, int bt_pages) {
  UmmaLayout L;
  const int natom = (2 * NT + 63) / 64;
  L.q = 0;                                   // [half][NT rows][128 B]
  L.p = L.q + 2 * NT * 128;                  // [buf][atom][128 keys][128 B = 64 columns]; columns = hi rows | lo rows
  L.p_hl_bytes = 0;
  L.p_buf_bytes = natom * 16384;
  L.ring = L.p + NP * L.p_buf_bytes;
  L.list = L.ring + NS * kSlotBytes;         // int32 [3][pages_per_split]
  L.pre = (L.list + 3 * pages_per_split * 4 + 15) & ~15;   // prefetched cache operands [kPreItems][128 o + lse + pad]
  L.bt = L.pre + kPreItems * kPreStride * 4;           // int32 [bt_pages] block-table row of the sequence
  L.total = L.bt + bt_pages * 4;
  return L;
}


struct UmmaCfg {
  int NK, NV;     // K and V ring slots (32 KB each)
  int NP;         // P buffers (1 or 2)
  int NSB;        // S buffers in TMEM (1 or 2)
  int tmem_cols;  // power of two >= (NSB + 2) * NT
  int bt_pages;   // block-table entries staged in shared memory (0: looked up in global memory)
};

// NCH = NT / 16; every softmax thread owns one key and NC = 4 * NCH of the padded rows (four column groups).
template <int NCH>
__global__ void __launch_bounds__(kUmmaThreads, 1)
attend_umma_kernel(const AttendParams p, const UmmaCfg cfg, const __grid_constant__ CUtensorMap tmap_k,
                   const __grid_constant__ CUtensorMap tmap_v) {
  constexpr int NT = 16 * NCH;
  constexpr int NC = 4 * NCH;
  extern __shared__ __align__(1024) unsigned char smem[];
  __shared__ __align__(8) uint64_t bars[24];
  __shared__ uint32_t tmem_ptr_s;
  __shared__ int s_flag[3];
  __shared__ int s_fix[2];                       // (block, page slot) of the newest page if its tail is unwritten, else -1
  __shared__ int s_rowr[kMaxWindow + 1];         // window rank (t - position) -> row of q_win / out, -1 = none
  __shared__ int s_posr[kMaxWindow + 1];         // q_pos of every row of q_win
  __shared__ int s_cpos[kMaxWindow + 1];         // cache_pos of the sequence as this kernel found it
  __shared__ __align__(16) float s_lse2[NT];     // base-2 log-sum-exp of this split's partial (cluster combine)
  __shared__ __align__(16) int s_colpos[NT];     // position of the row, -1 = none
  __shared__ __align__(16) float s_mref[NT];     // running reference (log2 units)
  __shared__ __align__(16) int s_colmax[NT];     // ordered-int block max (slow path)
  __shared__ __align__(16) float s_alpha[NT];
  __shared__ __align__(16) float s_L[NT];        // row sums (epilogue)
  const int pps = p.pages_per_split;
  const UmmaLayout lay = umma_layout(NT, cfg.NK + cfg.NV, cfg.NP, pps, cfg.bt_pages);
  uint64_t* k_full = bars;               // [NK <= 3]
  uint64_t* k_empty = bars + 3;          // [NK <= 3]
  uint64_t* v_full = bars + 6;           // [NV <= 3]
  uint64_t* v_empty = bars + 9;          // [NV <= 3]
  uint64_t* s_full = bars + 12;          // [2]
  uint64_t* p_ready = bars + 14;         // [2]
  uint64_t* o_full = bars + 16;          // [2] PV of block blk retired -> o_full[blk & 1], phase blk >> 1 (the
                                         // softmax warps run up to two blocks ahead: one barrier would alias)
  int32_t* s_list = reinterpret_cast<int32_t*>(smem + lay.list);       // [3][pps] logical, prev, physical

  const int split = blockIdx.x % p.nsplit, rg = blockIdx.x / p.nsplit, h = blockIdx.y, b = blockIdx.z;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int G = p.h_q / p.h_k, R = p.window + 1;
  // Query rows are laid out by window RANK (t - position: 0 = the current query, 1 = the newest past query, ...):
  // local row = (rank - rk0) * G + q head of the group.  This CTA's row group owns the ranks [rk0, rk0 + nrk).
  const int rk0 = rg * p.rg_ranks;
  const int nrk = min(p.rg_ranks, R - rk0);
  const int rows_cta = nrk * G;
  const size_t unit = (size_t)b * p.h_k + h;

  // ---- prologue.  Barriers and TMEM do not depend on the previous kernel: set them up before waiting for it.
  if (tid == 0) {
    for (int i = 0; i < 12; ++i) mbar_init(&bars[i], 1);
    mbar_init(&s_full[0], 1); mbar_init(&s_full[1], 1);
    mbar_init(&p_ready[0], kSoftmaxThreads / 32); mbar_init(&p_ready[1], kSoftmaxThreads / 32);
    mbar_init(&o_full[0], 1); mbar_init(&o_full[1], 1);
    fence_mbar_init();
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_ptr_s)),
                 "r"(cfg.tmem_cols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid <= kMaxWindow) s_rowr[tid] = -1;
  __syncthreads();
  // Inside retro_decode_step (fused) the kernel that precedes this one is the select kernel of the same step, and
  // it releases its dependents only after its own dependency wait: everything older than it is complete when this
  // CTA starts.  Only the selection (sel_*) needs the wait; the query window, positions, lengths, block table and
  // output cache do not, so that part of the prologue - and the idle warp's S4 service - overlap the select kernel.
  // Stand-alone (retro_sparse_attend) nothing is known about the predecessor: wait first.
  if (!p.fused) { pdl_wait(); pdl_trigger(); }
  const int L = p.seq_lens[b];
  // One row group: the unit's R * G rows (<= NT).  Several row groups (R * G > 128): every CTA fetches all of them
  // and keeps its own ranks (the rank of a row is only known once q_pos and the length are back).
  constexpr int kQIter = ((NCH >= 5 ? 3 : 1) * NT * 16 + kUmmaThreads - 1) / kUmmaThreads;
  uint4 q_regs[kQIter];
  int q_rpos[kQIter];
  {
    const uint4* src = reinterpret_cast<const uint4*>(p.q_win);
    const int n_chunks = R * G * 16;                           // rows of the window x 16 chunks of 16 B
#pragma unroll
    for (int it = 0; it < kQIter; ++it) {
      const int i = tid + it * kUmmaThreads;
      q_regs[it] = make_uint4(0, 0, 0, 0);
      q_rpos[it] = -1;
      if (i < n_chunks) {
        const int rho = i >> 4, c = i & 15;
        const int r = rho / G, g = rho - r * G;
        q_regs[it] = __ldg(src + (((size_t)b * R + r) * p.h_q + h * G + g) * 16 + c);
        q_rpos[it] = __ldg(p.q_pos + b * R + r);
      }
    }
  }
  int my_pos_raw = -1;
  if (tid < R) my_pos_raw = __ldg(p.q_pos + b * R + tid);
  // the sequence's block-table row goes to shared memory when it is small enough (cfg.bt_pages > 0): the logical ->
  // physical lookup of the selected pages then costs no global round trip after the wait
  int32_t* s_bt = reinterpret_cast<int32_t*>(smem + lay.bt);
  for (int i = tid; i < cfg.bt_pages; i += kUmmaThreads)
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(s_bt + i)),
                 "l"(p.block_table + (size_t)b * p.max_pages + i) : "memory");
  asm volatile("cp.async.commit_group;" ::: "memory");
  const int t = L - 1;
  // rows of the padded tile that no window row fills must read as zeros for the tensor core
  for (int i = tid; i < NT * 16; i += kUmmaThreads)
    *reinterpret_cast<uint4*>(smem + lay.q + (i & 1) * (NT * 128) + (i >> 1) * 16) = make_uint4(0, 0, 0, 0);
  if (tid < R) {
    s_posr[tid] = my_pos_raw;
    const int rank = t - my_pos_raw;
    if (my_pos_raw >= 0 && rank >= rk0 && rank < rk0 + nrk) s_rowr[rank - rk0] = tid;
  }
  if (tid < 3) s_flag[tid] = 0;
  if (tid == 0) s_fix[0] = -1;
  __syncthreads();
#pragma unroll
  for (int it = 0; it < kQIter; ++it) {
    const int i = tid + it * kUmmaThreads;
    const int rank = t - q_rpos[it];
    if (q_rpos[it] >= 0 && rank >= rk0 && rank < rk0 + nrk) {
      const int g = (i >> 4) % G, c = i & 15;
      const int rho = (rank - rk0) * G + g;
      const int half = c >> 3, ch = c & 7;
      *reinterpret_cast<uint4*>(smem + lay.q + half * (NT * 128) + rho * 128 + ((ch ^ (rho & 7)) << 4)) = q_regs[it];
    }
  }
  for (int c = tid; c < NT; c += kUmmaThreads) {
    int pos = -1;
    if (c < rows_cta && s_rowr[c / G] >= 0) pos = t - (rk0 + c / G);
    s_colpos[c] = pos;
    s_lse2[c] = -INFINITY;
    s_mref[c] = kMrefInit;
    s_colmax[c] = kOrdNegInf;
    s_alpha[c] = 1.f;
    s_L[c] = 0.f;
  }
  if (p.fused) {
    __syncthreads();             // s_posr / s_rowr are complete
    if (warp == 3 && p.window > 0) {
    // ---- the idle warp serves S4 while the others attend: (a) the cache operands of this CTA's merge items are
    // prefetched into shared memory, (b) cache_pos is snapshotted, (c) the CTA reports that it has read cache_pos;
    // the LAST CTA of the sequence to report rewrites it (the new values depend on q_pos and t only: Push slot
    // t mod w <- t, Update keeps the slot of a merged past row, Pop: position t - w is overwritten by the push).
    const int w = p.window;
    float* pre = reinterpret_cast<float*>(smem + lay.pre);
#pragma unroll 1
    for (int k = 0; k < kPreItems; ++k) {
      const int it = split + p.nsplit * k;
      if (it >= w * G) break;
      const int x = it / G, g = it - x * G;
      const size_t ce = ((size_t)b * w + x) * p.h_q + h * G + g;
      if (!p.cache_bf16)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(pre + k * kPreStride + lane * 4)),
                     "l"(static_cast<const float*>(p.cache_o) + ce * 128 + lane * 4) : "memory");
      else if (lane < 16)                          // a bf16 row is 256 B
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(pre + k * kPreStride + lane * 4)),
                     "l"(static_cast<const __nv_bfloat16*>(p.cache_o) + ce * 128 + lane * 8) : "memory");
      if (lane == 0)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(pre + k * kPreStride + 128)),
                     "l"(p.cache_lse + ce) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    if (lane < w) s_cpos[lane] = p.cache_pos[b * w + lane];
    __syncwarp();
    unsigned int tk = 0;
    if (lane == 0) tk = ticket_acq_rel(&p.seq_counters[b]);
    tk = __shfl_sync(0xffffffffu, tk, 0);
    if (tk == (unsigned)(p.h_k * p.nsplit - 1)) {
      if (lane == 0) p.seq_counters[b] = 0;              // leave the workspace consistent for the next call
      for (int r = lane; r < R; r += 32) {
        const int pos = s_posr[r];
        if (pos == t) p.cache_pos[b * w + t % w] = t;
        else if (pos > t - w && pos < t && pos >= 0) p.cache_pos[b * w + pos % w] = pos;
      }
    }
      }
    pdl_wait();
    pdl_trigger();
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
  __syncthreads();               // block-table row (and the S4 prefetch) landed
  int count = p.sel_count[unit];
  RETRO_DBG_ONLY(if (count < 0 || count > p.k_max) { if (tid == 0) dbg_violation(p.dbg, kDbgSelCount); count = 0; })
  RETRO_DBG_ONLY(if (L < 0 || L > p.max_pages * 16) { if (tid == 0) dbg_violation(p.dbg, kDbgSeqLen); count = 0; })
  RETRO_DBG_ONLY(if (tid < R && my_pos_raw > L - 1) dbg_violation(p.dbg, kDbgQPos);)
  const int beg0 = min(split * pps, count);
  for (int i = tid; i < pps; i += kUmmaThreads) {
    const int idx = split * pps + i;
    int j = 0, prev = 0;
    if (idx < p.k_max) {
      j = p.sel_pages[unit * p.k_max + idx];
      prev = p.sel_prev[unit * p.k_max + idx];
    }
    RETRO_DBG_ONLY(if (idx < count && (j < 0 || j >= min((L + 15) / 16, p.max_pages))) { dbg_violation(p.dbg, kDbgSelPage); j = 0; prev = 0x7fffffff; })
    int phys = 0;
    if (idx < count) phys = j < cfg.bt_pages ? s_bt[j] : p.block_table[(size_t)b * p.max_pages + j];
    RETRO_DBG_ONLY(if (phys < 0 || phys >= p.num_phys) { dbg_violation(p.dbg, kDbgPhysPage); phys = 0; prev = 0x7fffffff; })
    s_list[i] = j;
    s_list[pps + i] = prev;
    s_list[2 * pps + i] = phys;
    // slots of the newest page past the sequence's last token are unwritten memory (possibly NaN / Inf): P is 0
    // there, but 0 x NaN would poison the PV product, so those V rows are zeroed in shared memory (below)
    if (idx < count && j == (L - 1) / 16 && (L & 15) != 0) { s_fix[0] = (idx - beg0) / kPB; s_fix[1] = (idx - beg0) % kPB; }
  }
  const int beg = min(split * pps, count);
  const int end = min(beg + pps, count);
  const int n_my = end - beg;
  const int nblk = (n_my + kPB - 1) / kPB;
  const int colS = 0, colO = cfg.NSB * NT;
  fence_proxy_async();          // Q written through the generic proxy, read by the tensor core
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_ptr_s;

  if (nblk > 0) {
    if (warp < 2) {
      // ===== TMA producers: warp 0 streams the K blocks, warp 1 the V blocks, each through its own ring =====
      const int NR = warp == 0 ? cfg.NK : cfg.NV;
      uint64_t* full = warp == 0 ? k_full : v_full;
      uint64_t* empty = warp == 0 ? k_empty : v_empty;
      const CUtensorMap* map = warp == 0 ? &tmap_k : &tmap_v;
      unsigned char* ring = smem + lay.ring + (warp == 0 ? 0 : cfg.NK * kSlotBytes);
      for (int blk = 0; blk < nblk; ++blk) {
        const int slot = blk % NR, n = blk / NR;
        const int np = min(kPB, n_my - blk * kPB);
        unsigned char* dst = ring + slot * kSlotBytes;
        if (n > 0) mbar_wait(&empty[slot], (n - 1) & 1);
        if (elect_one()) {
          mbar_expect_tx(&full[slot], np * 2 * kTileHalfBytes);
          for (int pg = 0; pg < np; ++pg) {
            const int row0 = (s_list[2 * pps + blk * kPB + pg] * p.h_k + h) * 16;
            tma_load_2d(dst + pg * kTileHalfBytes, map, 0, row0, &full[slot]);
            tma_load_2d(dst + kHalfStride + pg * kTileHalfBytes, map, 64, row0, &full[slot]);
          }
        }
        __syncwarp();
      }
    } else if (warp == 2) {
      // ===== MMA issuer: the whole warp walks the loop (waits), one elected lane issues =====
      const uint32_t q_addr = smem_u32(smem + lay.q);
      const uint32_t idesc_s = idesc_bf16_ab(NT, false, false);
      const uint32_t idesc_o = idesc_bf16_ab(2 * NT, true, true);
      auto issue_s = [&](int blk) {
        const int slot = blk % cfg.NK, n = blk / cfg.NK;
        mbar_wait(&k_full[slot], n & 1);
        tc_fence_after();
        if (elect_one()) {
          const uint32_t k_addr = smem_u32(smem + lay.ring + slot * kSlotBytes);
          const uint32_t d_tmem = tmem_base + colS + (blk % cfg.NSB) * NT;
#pragma unroll
          for (int ks = 0; ks < 8; ++ks) {    // K = 128 channels = 8 steps of 16; 4 steps per 64-channel half
            const uint32_t koff = (ks >> 2) * kHalfStride + (ks & 3) * 32;
            const uint32_t qoff = (ks >> 2) * (NT * 128) + (ks & 3) * 32;
            umma_bf16(d_tmem, desc_kmajor_sw128(k_addr + koff), desc_kmajor_sw128(q_addr + qoff), idesc_s, ks > 0);
          }
          tc_commit(&k_empty[slot]);
          tc_commit(&s_full[blk % cfg.NSB]);
        }
        __syncwarp();
      };
      if (cfg.NSB == 2) issue_s(0);
      for (int blk = 0; blk < nblk; ++blk) {
        if (cfg.NSB == 2) {
          if (blk + 1 < nblk) issue_s(blk + 1);
        } else if (blk == 0) {
          issue_s(0);
        }
        const int slot = blk % cfg.NV, n = blk / cfg.NV;
        const int np = min(kPB, n_my - blk * kPB);
        mbar_wait(&p_ready[blk % cfg.NP], (blk / cfg.NP) & 1);
        if (cfg.NSB == 1 && blk + 1 < nblk) issue_s(blk + 1);   // S is free once P(blk) is written
        mbar_wait(&v_full[slot], n & 1);
        tc_fence_after();
        if (elect_one()) {
          const uint32_t v_addr = smem_u32(smem + lay.ring + (cfg.NK + slot) * kSlotBytes);
          const uint32_t p_addr = smem_u32(smem + lay.p + (blk % cfg.NP) * lay.p_buf_bytes);
          for (int ks = 0; ks < np; ++ks) {   // K = 16 keys (one page) per step
            const uint64_t vdesc = desc_mnmajor_sw128(v_addr + ks * kTileHalfBytes, kHalfStride);
            const uint64_t pdesc = desc_mnmajor_sw128(p_addr + ks * 2048, 16384);
            umma_bf16(tmem_base + colO, vdesc, pdesc, idesc_o, (blk > 0 || ks > 0) ? 1u : 0u);
          }
          tc_commit(&v_empty[slot]);
          tc_commit(&o_full[blk & 1]);
        }
        __syncwarp();
      }
    } else if (warp >= 4) {
      // ===== softmax warps: thread <-> TMEM lane <-> key of the block; NC = NT / 4 columns (rows) each =====
      const int sw = warp - 4;                            // 0..15
      const int quadrant = warp & 3;                      // TMEM lanes a warp may touch: 32*(warp%4)..+31
      const int cg = sw >> 2;                             // column group
      const int key = quadrant * 32 + lane;
      const int cbeg = cg * NC;
      const int st = tid - 128;                           // 0..511
      const uint32_t lane_addr = tmem_base + ((uint32_t)(quadrant * 32) << 16);
      float l_acc[NC];                                    // this key-thread's share of the row sums
#pragma unroll
      for (int j = 0; j < NC; ++j) l_acc[j] = 0.f;
      for (int blk = 0; blk < nblk; ++blk) {
        const int np = min(kPB, n_my - blk * kPB);
        // key visible to the row at position pos  <=>  sel_prev < pos and token position <= pos  <=>  pos > thr
        int thr = 0x7fffffff;
        if ((key >> 4) < np) {
          const int j = s_list[blk * kPB + (key >> 4)], prev = s_list[pps + blk * kPB + (key >> 4)];
          thr = max(prev, j * 16 + (key & 15) - 1);
        }
        if (st == 0) s_flag[(blk + 1) % 3] = 0;
        mbar_wait(&s_full[blk % cfg.NSB], (blk / cfg.NSB) & 1);
        tc_fence_after();
        const uint32_t s_addr = lane_addr + colS + (blk % cfg.NSB) * NT + cbeg;
        // d = s * scale - m_ref (log2 units), -inf where masked; the common block needs nothing else
        float d[NC];
        float tmax = -INFINITY;
        {
          uint32_t raw[NC];
#pragma unroll
          for (int i = 0; i < NCH; ++i) tmem_ld4(s_addr + 4 * i, raw + 4 * i);
          tmem_wait_ld();
#pragma unroll
          for (int i = 0; i < NCH; ++i) {
            const int4 ps = *reinterpret_cast<const int4*>(s_colpos + cbeg + 4 * i);
            const float4 mr = *reinterpret_cast<const float4*>(s_mref + cbeg + 4 * i);
            const int pv[4] = {ps.x, ps.y, ps.z, ps.w};
            const float mv[4] = {mr.x, mr.y, mr.z, mr.w};
#pragma unroll
            for (int u = 0; u < 4; ++u) {
              const float v = fmaf(__uint_as_float(raw[4 * i + u]), p.scale_log2, -mv[u]);
              d[4 * i + u] = pv[u] > thr ? v : -INFINITY;
              tmax = fmaxf(tmax, d[4 * i + u]);
            }
          }
        }
        if (__any_sync(0xffffffffu, tmax > kRescaleThreshold) && lane == 0) s_flag[blk % 3] = 1;
        softmax_bar();
        if (s_flag[blk % 3] != 0) {
          // ---- slow path: exact column max of this block, raise m_ref, rescale O and L ----
          float xs[NC];
          {
            uint32_t raw[NC];
#pragma unroll
            for (int i = 0; i < NCH; ++i) tmem_ld4(s_addr + 4 * i, raw + 4 * i);
            tmem_wait_ld();
#pragma unroll
            for (int j = 0; j < NC; ++j)
              xs[j] = s_colpos[cbeg + j] > thr ? __uint_as_float(raw[j]) * p.scale_log2 : -INFINITY;
          }
#pragma unroll
          for (int j = 0; j < NC; ++j) {
            const int r = __reduce_max_sync(0xffffffffu, f2o(xs[j]));
            if (lane == 0) atomicMax(&s_colmax[cbeg + j], r);
          }
          softmax_bar();
          if (st < NT) {
            const float bm = o2f(s_colmax[st]), old = s_mref[st];
            const float nw = fmaxf(old, bm);
            s_alpha[st] = ex2_approx(old - nw);             // old = kMrefInit (row not started): 0, O and L are 0
            s_mref[st] = nw;
            s_colmax[st] = kOrdNegInf;
          }
          softmax_bar();
#pragma unroll
          for (int j = 0; j < NC; ++j) {
            l_acc[j] *= s_alpha[cbeg + j];
            d[j] = xs[j] - s_mref[cbeg + j];
          }
          if (blk > 0) {
            mbar_wait(&o_full[(blk - 1) & 1], ((blk - 1) >> 1) & 1);   // PV(blk-1) retired: O is ours
            tc_fence_after();
#pragma unroll
            for (int i = 0; i < NCH; ++i) {                  // this thread's columns of O_hi and O_lo
              const float4 al4 = *reinterpret_cast<const float4*>(s_alpha + cbeg + 4 * i);
              const float al[4] = {al4.x, al4.y, al4.z, al4.w};
              uint32_t oh[4], ol[4];
              tmem_ld4(lane_addr + colO + cbeg + 4 * i, oh);
              tmem_ld4(lane_addr + colO + NT + cbeg + 4 * i, ol);
              tmem_wait_ld();
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                oh[u] = __float_as_uint(__uint_as_float(oh[u]) * al[u]);
                ol[u] = __float_as_uint(__uint_as_float(ol[u]) * al[u]);
              }
              tmem_st4(lane_addr + colO + cbeg + 4 * i, oh);
              tmem_st4(lane_addr + colO + NT + cbeg + 4 * i, ol);
            }
            tmem_wait_st();
          }
        }
        if (cfg.NP == 1 && blk > 0) mbar_wait(&o_full[(blk - 1) & 1], ((blk - 1) >> 1) & 1);   // PV(blk-1) has read P
        // ---- P = 2^d as bf16 hi + lo into the MN-major SW128 operand (8-byte stores: NC is a multiple of 4) ----
        unsigned char* p_row = smem + lay.p + (blk % cfg.NP) * lay.p_buf_bytes + key * 128;
#pragma unroll
        for (int i = 0; i < NCH; ++i) {
          float e[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            e[u] = ex2_approx(d[4 * i + u]);
            l_acc[4 * i + u] += e[u];
          }
          const int c_hi = cbeg + 4 * i, c_lo = NT + c_hi;
          uint2 hi, lo;
          split_bf16x2(e[0], e[1], hi.x, lo.x);
          split_bf16x2(e[2], e[3], hi.y, lo.y);
          *reinterpret_cast<uint2*>(p_row + (c_hi >> 6) * 16384 + ((((c_hi & 63) >> 3) ^ (key & 7)) << 4) +
                                    ((c_hi & 4) << 1)) = hi;
          *reinterpret_cast<uint2*>(p_row + (c_lo >> 6) * 16384 + ((((c_lo & 63) >> 3) ^ (key & 7)) << 4) +
                                    ((c_lo & 4) << 1)) = lo;
        }
        if (blk == s_fix[0] && sw == 0) {
          // the unwritten tail rows of the newest page's V tile (both 64-channel halves) are zeroed before this
          // block's PV product can start (it needs every softmax warp's arrival below).  The V slot of block blk
          // cannot be refilled before that product, so its barrier is in phase blk / NV or one later: the parity
          // wait cannot alias with another fill of the slot.
          const int slot = blk % cfg.NV, pg = s_fix[1], nv = L & 15;
          mbar_wait(&v_full[slot], (blk / cfg.NV) & 1);
          unsigned char* vt = smem + lay.ring + (cfg.NK + slot) * kSlotBytes + pg * kTileHalfBytes;
          for (int i = lane; i < (16 - nv) * 8; i += 32) {           // 16-byte chunks of rows nv..15 (128 B per row and half)
            *reinterpret_cast<uint4*>(vt + nv * 128 + i * 16) = make_uint4(0, 0, 0, 0);
            *reinterpret_cast<uint4*>(vt + kHalfStride + nv * 128 + i * 16) = make_uint4(0, 0, 0, 0);
          }
        }
        fence_proxy_async();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&p_ready[blk % cfg.NP]);   // one arrival per warp (512 would serialise)
      }
      // ---- epilogue: L per row, O = (O_hi + O_lo) / L through a shared-memory stage, coalesced stores ----
      {
        // sum over the 32 keys of the warp: two halving levels, then a 3-level butterfly on NCH values
        const bool up16 = lane & 16, up8 = lane & 8;
#pragma unroll
        for (int i = 0; i < 2 * NCH; ++i) {
          const float send = up16 ? l_acc[i] : l_acc[i + 2 * NCH], keep = up16 ? l_acc[i + 2 * NCH] : l_acc[i];
          l_acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
        }
#pragma unroll
        for (int i = 0; i < NCH; ++i) {
          const float send = up8 ? l_acc[i] : l_acc[i + NCH], keep = up8 ? l_acc[i + NCH] : l_acc[i];
          float v = keep + __shfl_xor_sync(0xffffffffu, send, 8);
          v += __shfl_xor_sync(0xffffffffu, v, 4);
          v += __shfl_xor_sync(0xffffffffu, v, 2);
          v += __shfl_xor_sync(0xffffffffu, v, 1);
          if ((lane & 7) == 0) atomicAdd(&s_L[cbeg + ((lane >> 3) & 3) * NCH + i], v);
        }
      }
      mbar_wait(&o_full[(nblk - 1) & 1], ((nblk - 1) >> 1) & 1);
      tc_fence_after();
      softmax_bar();                                       // s_L complete
      // thread = channel `key`; its NC rows: O = (O_hi + O_lo) / L into the staging tile [row][128 channels] (the
      // K / V ring is idle: every tensor-core read of it has retired), base-2 lse next to it.  The tile is fp16
      // (|o| <= max |v|, 11 significant bits: far inside the bf16 tolerance): distributed shared memory serves
      // ~19 B/clk per SM, and the combine below is bound by exactly that.
      __half* stage = reinterpret_cast<__half*>(smem + lay.ring);
#pragma unroll
      for (int i = 0; i < NCH; ++i) {
        if (cbeg + 4 * i < rows_cta) {                      // warp-uniform
          uint32_t oh[4], ol[4];
          tmem_ld4(lane_addr + colO + cbeg + 4 * i, oh);
          tmem_ld4(lane_addr + colO + NT + cbeg + 4 * i, ol);
          tmem_wait_ld();
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int c = cbeg + 4 * i + u;
            if (c < rows_cta) {
              const float l = s_L[c];
              const float inv = rcp_approx(l);
              stage[c * 128 + key] = __float2half_rn(l > 0.f ? (__uint_as_float(oh[u]) + __uint_as_float(ol[u])) * inv : 0.f);
              if (key == 0) s_lse2[c] = l > 0.f ? s_mref[c] + lg2_approx(l) : -INFINITY;
            }
          }
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(cfg.tmem_cols));
  }
  // ---- split combine (+ S4 when fused) over the cluster: the splits of a (unit, row group) are the CTAs of one
  // cluster; every CTA merges a share of the rows, reading the other splits' partials out of their shared memory.
  // This tail runs every instruction once (latency-bound): ONE loop, one combine site, no unrolling.
  cluster_arrive();
  cluster_wait();
  {
    const uint32_t stage_a = smem_u32(smem + lay.ring) + lane * 8, lse_a = smem_u32(s_lse2);
    const float* pre = reinterpret_cast<const float*>(smem + lay.pre);
    const int nsplit = p.nsplit, w = p.window, nwarps = kUmmaThreads / 32;
    const bool fused = p.fused != 0;
    // Work items.  Stand-alone S3: item = local row.  Fused S3 + S4: item = (cache slot x, q head g) with two
    // sub-steps, the slot's past row (position = x mod w; merged with the cache, Eq. 8-9) and then the current row if
    // it lands in this slot (pushed): the pop of position t - w and the push of position t are ordered by the warp.
    const int nslot = w > 0 ? w : 1;
    const int n_items = fused ? nslot * G : rows_cta;
#pragma unroll 1
    for (int k = warp; split + nsplit * k < n_items; k += nwarps) {
      const int it = split + nsplit * k;
      const int x = it / G, g = it - x * G;
#pragma unroll 1
      for (int sub = 0; sub < (fused ? 2 : 1); ++sub) {
        int rank, mode;                                  // mode 0: plain partial, 1: merge with the cache, 2: push
        if (!fused) { rank = x; mode = 0; }
        else if (sub == 0) {
          if (w == 0) continue;
          const int p_past = t - 1 - (((t - 1 - x) % w + w) % w);     // the position in [t-w, t-1] with p mod w == x
          if (p_past < 0) continue;
          rank = t - p_past; mode = 1;
        } else {
          if (w > 0 && t % w != x) continue;
          rank = 0; mode = 2;
        }
        const int r = s_rowr[rank];
        if (r < 0) continue;
        const int c = rank * G + g;
        // Eq. 8 applied to the splits of local row c (weights 2^(lse_s - max)).  An empty split's tile is
        // unspecified: it is never multiplied.
        uint2 v[8];                                      // 4 halves per lane; all remote loads in flight before the first use
#pragma unroll
        for (int s2 = 0; s2 < 8; ++s2)
          if (s2 < nsplit) v[s2] = dsmem_ld_v2(dsmem_addr(stage_a + c * 256, s2));
        float l_mine = -INFINITY;
        if (lane < nsplit) l_mine = dsmem_ld_f32(dsmem_addr(lse_a + c * 4, lane));
        const float mx = warp_max(l_mine);
        const float w_mine = mx > -INFINITY ? ex2_approx(l_mine - mx) : 0.f;
        float wsum = 0.f;
        float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int s2 = 0; s2 < 8; ++s2) {
          const float wg = __shfl_sync(0xffffffffu, w_mine, s2);
          if (s2 < nsplit && wg > 0.f) {
            wsum += wg;
            const float2 f01 = __half22float2(*reinterpret_cast<const __half2*>(&v[s2].x));
            const float2 f23 = __half22float2(*reinterpret_cast<const __half2*>(&v[s2].y));
            o.x = fmaf(wg, f01.x, o.x); o.y = fmaf(wg, f01.y, o.y);
            o.z = fmaf(wg, f23.x, o.z); o.w = fmaf(wg, f23.y, o.w);
          }
        }
        const float inv = wsum > 0.f ? rcp_approx(wsum) : 0.f;
        o.x *= inv; o.y *= inv; o.z *= inv; o.w *= inv;
        float lse = wsum > 0.f ? (mx + lg2_approx(wsum)) * kLn2 : -INFINITY;
        const size_t e = ((size_t)b * R + r) * p.h_q + h * G + g;
        *reinterpret_cast<float4*>(p.part_o + e * 128 + lane * 4) = o;
        if (lane == 0) p.part_lse[e] = lse;
        if (mode == 0) continue;
        const size_t ce = ((size_t)b * nslot + x) * p.h_q + h * G + g;
        bool write_back = w > 0;
        if (mode == 1) {
          if (s_cpos[x] == t - rank) {                   // something is cached for this position
            float lc;
            float4 vc;
            if (k < kPreItems) lc = pre[k * kPreStride + 128];
            else lc = p.cache_lse[ce];
            if (!p.cache_bf16) {
              vc = k < kPreItems ? *reinterpret_cast<const float4*>(pre + k * kPreStride + lane * 4)
                                 : *reinterpret_cast<const float4*>(static_cast<const float*>(p.cache_o) + ce * 128 + lane * 4);
            } else {                                     // 16-bit cache rows (Eq. 12): 4 bf16 per lane
              const uint2 u = k < kPreItems
                  ? *reinterpret_cast<const uint2*>(reinterpret_cast<const unsigned char*>(pre + k * kPreStride) + lane * 8)
                  : *reinterpret_cast<const uint2*>(static_cast<const __nv_bfloat16*>(p.cache_o) + ce * 128 + lane * 4);
              vc = make_float4(bf16_lo(u.x), bf16_hi(u.x), bf16_lo(u.y), bf16_hi(u.y));
            }
            if (lc > -INFINITY) {
              if (lse == -INFINITY) { o = vc; lse = lc; }
              else {
                const float m2 = fmaxf(lc, lse);
                const float wc = ex2_approx((lc - m2) * kLog2e), wp = ex2_approx((lse - m2) * kLog2e);
                const float iv = rcp_approx(wc + wp);
                o.x = (wc * vc.x + wp * o.x) * iv; o.y = (wc * vc.y + wp * o.y) * iv;
                o.z = (wc * vc.z + wp * o.z) * iv; o.w = (wc * vc.w + wp * o.w) * iv;
                lse = m2 + lg2_approx(wc + wp) * kLn2;
              }
            }
          }
          write_back = rank != w;                        // the row at position t - w is popped after its last merge
        }
        store_bf16x4(reinterpret_cast<__nv_bfloat16*>(p.out) + e * 128 + lane * 4, o);
        if (lane == 0 && p.out_lse != nullptr) p.out_lse[e] = lse;
        if (write_back) {
          if (!p.cache_bf16) *reinterpret_cast<float4*>(static_cast<float*>(p.cache_o) + ce * 128 + lane * 4) = o;
          else store_bf16x4(static_cast<__nv_bfloat16*>(p.cache_o) + ce * 128 + lane * 4, o);
          if (lane == 0) p.cache_lse[ce] = lse;
        }
      }
    }
    // rows of q_win without a position inside the window: zeros / -inf (one CTA of the unit's first row group)
    if (split == 0 && rg == 0) {
#pragma unroll 1
      for (int it = warp; it < R * G; it += nwarps) {
        const int r = it / G, g = it - r * G;
        const int pos = s_posr[r];
        if (pos >= 0 && pos <= t && pos >= t - w) continue;
        const size_t e = ((size_t)b * R + r) * p.h_q + h * G + g;
        *reinterpret_cast<float4*>(p.part_o + e * 128 + lane * 4) = make_float4(0.f, 0.f, 0.f, 0.f);
        if (lane == 0) p.part_lse[e] = -INFINITY;
        if (fused) {
          store_bf16x4(reinterpret_cast<__nv_bfloat16*>(p.out) + e * 128 + lane * 4, make_float4(0.f, 0.f, 0.f, 0.f));
          if (lane == 0 && p.out_lse != nullptr) p.out_lse[e] = -INFINITY;
        }
      }
    }
  }
  cluster_arrive_relaxed();    // nobody leaves while its partial may still be read (no data is handed over: no fence)
  cluster_wait_end();
}

// ---- host: tensor maps over the K / V pools viewed as [(phys * h_k + head) * 16 rows][128 channels] ----
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess) f = nullptr;
    return reinterpret_cast<EncodeTiledFn>(f);
  }();
  return fn;
}

static int make_pool_map(CUtensorMap* map, const void* pool, const retro_desc_t* d) {
  EncodeTiledFn fn = encode_fn();
  if (fn == nullptr) return RETRO_ERR_CUDA;
  const cuuint64_t dims[2] = {128, (cuuint64_t)d->num_phys_pages * d->num_kv_heads * 16};
  const cuuint64_t strides[1] = {256};
  const cuuint32_t box[2] = {64, 16};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(pool), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    set_cuda_error(cudaErrorInvalidValue);
    return RETRO_ERR_CUDA;
  }
  return RETRO_OK;
}

template <int NCH>
static int launch_nch(const retro_desc_t* d, const AttendParams& prm, const UmmaCfg& cfg, size_t smem,
                      const CUtensorMap& mk, const CUtensorMap& mv, cudaStream_t s) {
  auto kern = attend_umma_kernel<NCH>;
  const int rc = ensure_dynamic_smem((const void*)kern, smem, /*max_carveout=*/true);
  if (rc != RETRO_OK) return rc;
  // the splits of a (unit, row group) form one cluster (<= 8 CTAs: portable)
  RETRO_CUDA_TRY(launch_cluster_kernel(kern, dim3(prm.nsplit * prm.nrg, d->num_kv_heads, d->batch), dim3(kUmmaThreads),
                                       smem, s, prm.nsplit, prm, cfg, mk, mv));
  RETRO_LAUNCH_CHECK();
  return RETRO_OK;
}

// Resident clusters of `cluster_x` CTAs of attend_umma_kernel<nch> at the largest shared-memory footprint the
// launcher plans with.  Without a device (symbol / header tests on a CPU-only box): the B200's measured table.
int umma_max_active_clusters(int nch, int cluster_x) {
  const void* kern = nullptr;
  switch (nch) {
    case 1: kern = (const void*)attend_umma_kernel<1>; break;
    case 2: kern = (const void*)attend_umma_kernel<2>; break;
    case 3: kern = (const void*)attend_umma_kernel<3>; break;
    case 4: kern = (const void*)attend_umma_kernel<4>; break;
    case 5: kern = (const void*)attend_umma_kernel<5>; break;
    case 6: kern = (const void*)attend_umma_kernel<6>; break;
    case 7: kern = (const void*)attend_umma_kernel<7>; break;
    case 8: kern = (const void*)attend_umma_kernel<8>; break;
    default: return 0;
  }
  if (device_info().device < 0) {
    static const int b200[9] = {0, 148, 74, 45, 33, 26, 22, 15, 15};
    return cluster_x >= 1 && cluster_x <= 8 ? b200[cluster_x] : 0;
  }
  return max_active_clusters(kern, kUmmaThreads, (size_t)kUmmaSmemBudget, cluster_x);
}

int launch_attend_umma(const retro_desc_t* d, const AttendParams& prm, cudaStream_t s) {
  // the encode is pure host work (~1 us); cache the maps per (pool pair, shape).  The cache holds tensor-map
  // DESCRIPTORS of the caller's pools (addresses, never dereferenced on the host): see retro.h "global state".
  CUtensorMap map_k, map_v;
  {
  std::lock_guard<std::mutex> lock(host_mutex());
  struct Cached { const void* k; const void* v; int phys, hk; CUtensorMap mk, mv; };
  constexpr int kCache = 64;
  static Cached cache[kCache];
  static int n_cached = 0;
  Cached* hit = nullptr;
  for (int i = 0; i < n_cached; ++i)
    if (cache[i].k == prm.k_pages && cache[i].v == prm.v_pages && cache[i].phys == d->num_phys_pages &&
        cache[i].hk == d->num_kv_heads) { hit = &cache[i]; break; }
  if (hit == nullptr) {
    Cached c;
    c.k = prm.k_pages; c.v = prm.v_pages; c.phys = d->num_phys_pages; c.hk = d->num_kv_heads;
    int rc = make_pool_map(&c.mk, prm.k_pages, d);
    if (rc != RETRO_OK) return rc;
    rc = make_pool_map(&c.mv, prm.v_pages, d);
    if (rc != RETRO_OK) return rc;
    static int next = 0;
    const int slot = n_cached < kCache ? n_cached++ : (next++ % kCache);
    cache[slot] = c;
    hit = &cache[slot];
  }
  map_k = hit->mk;
  map_v = hit->mv;
  }
  const int nch = ceil_div(prm.rg_ranks * (d->num_q_heads / d->num_kv_heads), 16), NT = 16 * nch;
  if (prm.nsplit > 8) return RETRO_ERR_UNSUPPORTED;
  if (NT > kMaxNT) return RETRO_ERR_UNSUPPORTED;
  // Shared-memory plan (one CTA per SM: 232448 B less the reserved KB and ~5 KB of static shared memory).  Prefer
  // two P buffers; the ring takes what is left (>= 2 slots: K and V of one block in flight per CTA).
  UmmaCfg cfg;
  cfg.NSB = 2;
  cfg.bt_pages = d->max_pages_per_seq <= 4096 ? d->max_pages_per_seq : 0;   // <= 16 KB of shared memory
  int slots = 0;
  auto plan = [&](int budget) {
    cfg.NP = 2;
    slots = (budget - umma_layout(NT, 0, cfg.NP, prm.pages_per_split, cfg.bt_pages).total) / kSlotBytes;
    if (slots < 4) {
      cfg.NP = 1;
      slots = (budget - umma_layout(NT, 0, cfg.NP, prm.pages_per_split, cfg.bt_pages).total) / kSlotBytes;
    }
  };
  plan(kUmmaSmemBudget);
  if (slots < 2) return RETRO_ERR_UNSUPPORTED;
  if (slots > 6) slots = 6;
  cfg.NK = slots / 2;             // a V block lives longer (it waits for the softmax of its own block)
  cfg.NV = slots - cfg.NK;
  int cols = 32;
  while (cols < (cfg.NSB + 2) * NT) cols <<= 1;
  if (cols > kTmemCols) return RETRO_ERR_UNSUPPORTED;
  cfg.tmem_cols = cols;
  const size_t smem = (size_t)umma_layout(NT, cfg.NK + cfg.NV, cfg.NP, prm.pages_per_split, cfg.bt_pages).total;
  switch (nch) {
    case 1: return launch_nch<1>(d, prm, cfg, smem, map_k, map_v, s);
    case 2: return launch_nch<2>(d, prm, cfg, smem, map_k, map_v, s);
    case 3: return launch_nch<3>(d, prm, cfg, smem, map_k, map_v, s);
    case 4: return launch_nch<4>(d, prm, cfg, smem, map_k, map_v, s);
    case 5: return launch_nch<5>(d, prm, cfg, smem, map_k, map_v, s);
    case 6: return launch_nch<6>(d, prm, cfg, smem, map_k, map_v, s);
    case 7: return launch_nch<7>(d, prm, cfg, smem, map_k, map_v, s);
    case 8: return launch_nch<8>(d, prm, cfg, smem, map_k, map_v, s);
  }
  return RETRO_ERR_UNSUPPORTED;
}

}  // namespace retro
