// S3 on the 5th-generation tensor cores (bf16, d = 128, P = 16): the GQA group x (w+1) query block against
// the selected pages is a dense [rows x 128] x [128 x keys] contraction followed by [rows x keys] x [keys x 128]
// (Eq. 2 / 6 / 7; arithmetic intensity ~ rows flop/B), far above what
// the fp32 ALUs sustain at HBM rate once rows > ~8.
//
// One CTA per (split, KV head, sequence), 192 threads, warp-specialised:
//   warp 0      TMA producer: each selected (page, head) K tile and V tile arrives as two 64-column boxes with
//               the 128-byte swizzle (cp.async.bulk.tensor.2d + mbarrier), 8 pages = 128 keys per KV block,
//               double-buffered (2 x 64 KB in flight per SM).
//   warp 1      MMA issuer (one elected thread): S = Q K^T  -> TMEM (M = 128 rows, N = 16 * pages, K = 128) and
//               O += P V -> TMEM (M = 128, N = 128, K = 16 * pages) with tcgen05.mma.kind::f16; completion is
//               signalled to the other warps with tcgen05.commit on mbarriers.  Owns the TMEM allocation.
//   warps 2..5  softmax: thread <-> TMEM lane <-> query row.  Reads its S row with tcgen05.ld, applies the
//               retrospective mask (page j active for row at position p iff sel_prev_j < p; token l iff l <= p),
//               keeps (m, l) in registers, overwrites S in place with P (bf16 hi + lo, the TMEM A operand
//               of the PV MMA), rescales O in TMEM only when the running max moved by more than 2^8.
// S is double-buffered in TMEM so QK^T of block i+1 overlaps the softmax of block i.
// Every page is read from HBM once and serves all rows.  Split partials are combined by the last CTA of the unit.
#include <cuda.h>

#include "attend_common.cuh"

namespace retro {

constexpr int kUmmaThreads = 192;
constexpr int kPB = 8;                    // pages per KV block
constexpr int kKvStages = 2;
constexpr int kTileHalfBytes = 16 * 128;  // one (page, head, 64-column half) box: 16 rows x 128 B
constexpr int kHalfStride = kPB * kTileHalfBytes;          // 16 KB: [half][page][16][128 B]
constexpr int kStageBytes = 2 * kHalfStride;               // 32 KB of K (or V) per stage
constexpr int kQBytes = 2 * 128 * 128;                     // [half][128 rows][128 B] = 32 KB
constexpr int kTmemCols = 512;
constexpr int kColS = 0, kColO = 256;                      // S0: 0..127, S1: 128..255, O: 256..383
constexpr float kRescaleThreshold = 8.f;                   // log2 units

// ---- PTX wrappers -------------------------------------------------------------------------------
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(smem_u32(smem_dst)), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(smem_u32(bar))
      : "memory");
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
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,"
      "%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
      "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,"
      "%30,%31,%32};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
        "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]),
        "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]),
        "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
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
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* r) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]),
        "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}
// A operand from TMEM (lanes = rows, one 32-bit column = two consecutive K elements), B from shared memory.
__device__ __forceinline__ void umma_bf16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc,
                                             uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
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
// Instruction descriptor (cute::UMMA::InstrDescriptor): D = f32, A = B = bf16, M = 128.
__device__ __forceinline__ uint32_t idesc_bf16(int n, bool b_mn_major) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn_major ? 1u : 0u) << 16) | ((uint32_t)(n >> 3) << 17) |
         ((uint32_t)(128 >> 4) << 24);
}

struct UmmaSmem {   // offsets into dynamic shared memory (base aligned to 1024 B)
  static constexpr int q = 0;
  static constexpr int k = q + kQBytes;
  static constexpr int v = k + kKvStages * kStageBytes;
  static constexpr int bars = v + kKvStages * kStageBytes;   // 16 mbarriers
  static constexpr int tmem_ptr = bars + 16 * 8;
  static constexpr int list = tmem_ptr + 16;                  // int32 [3][pages_per_split]
};

__global__ void __launch_bounds__(kUmmaThreads, 1)
attend_umma_kernel(const AttendParams p, const __grid_constant__ CUtensorMap tmap_k,
                   const __grid_constant__ CUtensorMap tmap_v) {
  extern __shared__ unsigned char smem_raw[];
  unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + UmmaSmem::bars);
  uint64_t* k_full = bars;          // [2]
  uint64_t* v_full = bars + 2;      // [2]
  uint64_t* k_empty = bars + 4;     // [2]
  uint64_t* v_empty = bars + 6;     // [2]
  uint64_t* s_full = bars + 8;      // [2]
  uint64_t* p_ready = bars + 10;    // [2] one per S buffer: a fast warp may run one block ahead of a slow one
  uint64_t* o_full = bars + 12;
  uint64_t* o_done = bars + 13;     // last PV retired (a parity wait on o_full could alias two phases back)
  uint32_t* tmem_ptr_s = reinterpret_cast<uint32_t*>(smem + UmmaSmem::tmem_ptr);
  int32_t* s_list = reinterpret_cast<int32_t*>(smem + UmmaSmem::list);
  __shared__ unsigned int s_ticket;

  const int split = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int G = p.h_q / p.h_k, R = p.window + 1, rows = R * G;
  const int L = p.seq_lens[b];
  const int t = L - 1;
  const size_t unit = (size_t)b * p.h_k + h;
  const int count = p.sel_count[unit];
  const int beg = min(split * p.pages_per_split, count);
  const int end = min(beg + p.pages_per_split, count);
  const int n_my = end - beg;
  const int nblk = (n_my + kPB - 1) / kPB;
  const int pps = p.pages_per_split;

  if (nblk > 0) {
    // ---- prologue: page list, Q (swizzled K-major operand), zeroed P, barriers, TMEM ----------------------
    for (int i = tid; i < n_my; i += kUmmaThreads) {
      const int j = p.sel_pages[unit * p.k_max + beg + i];
      s_list[i] = j;
      s_list[pps + i] = p.sel_prev[unit * p.k_max + beg + i];
      s_list[2 * pps + i] = p.block_table[(size_t)b * p.max_pages + j];
    }
    {
      const uint4* src = reinterpret_cast<const uint4*>(p.q_win);
      for (int i = tid; i < 128 * 16; i += kUmmaThreads) {      // 128 rows x 16 chunks of 16 B
        const int rho = i >> 4, c = i & 15;
        uint4 v = make_uint4(0, 0, 0, 0);
        if (rho < rows) {
          const int r = rho / G, g = rho % G;
          v = __ldg(src + (((size_t)b * R + r) * p.h_q + h * G + g) * 16 + c);
        }
        const int half = c >> 3, ch = c & 7;
        *reinterpret_cast<uint4*>(smem + UmmaSmem::q + half * 16384 + rho * 128 + ((ch ^ (rho & 7)) << 4)) = v;
      }
    }
    if (tid == 0) {
      for (int i = 0; i < 8; ++i) mbar_init(&bars[i], 1);
      mbar_init(&s_full[0], 1); mbar_init(&s_full[1], 1);
      mbar_init(&p_ready[0], 128); mbar_init(&p_ready[1], 128);
      mbar_init(o_full, 1);
      mbar_init(o_done, 1);
      fence_mbar_init();
    }
    if (warp == 1) {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_ptr_s)),
                   "n"(kTmemCols));
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    fence_proxy_async();          // Q / P written through the generic proxy, read by the tensor core (async proxy)
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_ptr_s;

    if (warp == 0) {
      // ===== TMA producer =====
      if (lane == 0) {
        for (int blk = 0; blk < nblk; ++blk) {
          const int s = blk % kKvStages, n = blk / kKvStages;
          const int np = min(kPB, n_my - blk * kPB);
          unsigned char* kdst = smem + UmmaSmem::k + s * kStageBytes;
          unsigned char* vdst = smem + UmmaSmem::v + s * kStageBytes;
          if (n > 0) mbar_wait(&k_empty[s], (n - 1) & 1);
          mbar_expect_tx(&k_full[s], np * 2 * kTileHalfBytes);
          for (int pg = 0; pg < np; ++pg) {
            const int row0 = (s_list[2 * pps + blk * kPB + pg] * p.h_k + h) * 16;
            tma_load_2d(kdst + pg * kTileHalfBytes, &tmap_k, 0, row0, &k_full[s]);
            tma_load_2d(kdst + kHalfStride + pg * kTileHalfBytes, &tmap_k, 64, row0, &k_full[s]);
          }
          if (n > 0) mbar_wait(&v_empty[s], (n - 1) & 1);
          mbar_expect_tx(&v_full[s], np * 2 * kTileHalfBytes);
          for (int pg = 0; pg < np; ++pg) {
            const int row0 = (s_list[2 * pps + blk * kPB + pg] * p.h_k + h) * 16;
            tma_load_2d(vdst + pg * kTileHalfBytes, &tmap_v, 0, row0, &v_full[s]);
            tma_load_2d(vdst + kHalfStride + pg * kTileHalfBytes, &tmap_v, 64, row0, &v_full[s]);
          }
        }
      }
    } else if (warp == 1) {
      // ===== MMA issuer =====
      if (lane == 0) {
        const uint32_t q_addr = smem_u32(smem + UmmaSmem::q);
        auto issue_s = [&](int blk) {
          const int s = blk % kKvStages, n = blk / kKvStages;
          const int np = min(kPB, n_my - blk * kPB);
          mbar_wait(&k_full[s], n & 1);
          tc_fence_after();
          const uint32_t k_addr = smem_u32(smem + UmmaSmem::k + s * kStageBytes);
          const uint32_t idesc = idesc_bf16(16 * np, false);
          const uint32_t d_tmem = tmem_base + kColS + (blk & 1) * 128;
#pragma unroll
          for (int ks = 0; ks < 8; ++ks) {    // K = 128 channels = 8 steps of 16; 4 steps per 64-column half
            const uint32_t off = (ks >> 2) * 16384 + (ks & 3) * 32;
            umma_bf16(d_tmem, desc_kmajor_sw128(q_addr + off), desc_kmajor_sw128(k_addr + off), idesc, ks > 0);
          }
          tc_commit(&k_empty[s]);
          tc_commit(&s_full[blk & 1]);
        };
        issue_s(0);
        for (int blk = 0; blk < nblk; ++blk) {
          if (blk + 1 < nblk) issue_s(blk + 1);
          const int s = blk % kKvStages, n = blk / kKvStages;
          const int np = min(kPB, n_my - blk * kPB);
          mbar_wait(&p_ready[blk & 1], (blk >> 1) & 1);
          mbar_wait(&v_full[s], n & 1);
          tc_fence_after();
          const uint32_t v_addr = smem_u32(smem + UmmaSmem::v + s * kStageBytes);
          const uint32_t idesc = idesc_bf16(128, true);
          const uint32_t p_tmem = tmem_base + kColS + (blk & 1) * 128;   // P overwrote S in place: [hi 64 | lo 64]
          for (int ks = 0; ks < np; ++ks) {   // K = 16 keys (one page) per step = 8 TMEM columns of A
            const uint64_t vdesc = desc_mnmajor_sw128(v_addr + ks * kTileHalfBytes, kHalfStride);
            umma_bf16_ts(tmem_base + kColO, p_tmem + 8 * ks, vdesc, idesc, (blk > 0 || ks > 0));
            umma_bf16_ts(tmem_base + kColO, p_tmem + 64 + 8 * ks, vdesc, idesc, 1u);
          }
          tc_commit(&v_empty[s]);
          tc_commit(o_full);
          if (blk == nblk - 1) tc_commit(o_done);
        }
      }
    } else {
      // ===== softmax warps: thread <-> TMEM lane <-> query row =====
      const int quarter = warp & 3;                       // TMEM lanes a warp may touch: 32*(warp%4)..+31
      const int rho = quarter * 32 + lane;
      const uint32_t lane_addr = tmem_base + ((uint32_t)(quarter * 32) << 16);
      int pos = -1;
      if (rho < rows) {
        pos = p.q_pos[b * R + rho / G];
        if (pos > t || pos < t - p.window) pos = -1;
      }
      const bool real = pos >= 0;
      float m_ref = -INFINITY, l_run = 0.f;               // running max (log2 units) used as exponent reference
      for (int blk = 0; blk < nblk; ++blk) {
        const int np = min(kPB, n_my - blk * kPB);
        // valid-token count of each page of the block for this row (0 = page masked for this query)
        uint32_t nv_lo = 0, nv_hi = 0;                    // 8 x 5 bits packed: pages 0..5 in lo, 6..7 in hi
        if (real) {
          for (int pg = 0; pg < np; ++pg) {
            const int j = s_list[blk * kPB + pg], prev = s_list[pps + blk * kPB + pg];
            int nv = (prev < pos) ? min(pos - j * 16 + 1, 16) : 0;
            nv = max(nv, 0);
            if (pg < 6) nv_lo |= (uint32_t)nv << (5 * pg); else nv_hi |= (uint32_t)nv << (5 * (pg - 6));
          }
        }
        auto nvalid = [&](int pg) -> int {
          return pg < 6 ? (int)((nv_lo >> (5 * pg)) & 31u) : (int)((nv_hi >> (5 * (pg - 6))) & 31u);
        };
        mbar_wait(&s_full[blk & 1], (blk >> 1) & 1);
        tc_fence_after();
        const uint32_t s_addr = lane_addr + kColS + (blk & 1) * 128;
        // pass 1: row max over the unmasked columns
        float mx = -INFINITY;
#pragma unroll
        for (int c4 = 0; c4 < 4; ++c4) {
          if (c4 * 2 < np) {                               // warp-uniform
            uint32_t sv[32];
            tmem_ld32(s_addr + c4 * 32, sv);
            tmem_wait_ld();
            const int nv0 = nvalid(c4 * 2), nv1 = nvalid(c4 * 2 + 1);
#pragma unroll
            for (int c = 0; c < 16; ++c) {
              if (c < nv0) mx = fmaxf(mx, __uint_as_float(sv[c]));
              if (c < nv1) mx = fmaxf(mx, __uint_as_float(sv[16 + c]));
            }
          }
        }
        mx *= p.scale_log2;                                // scale > 0: max commutes with the scaling; -inf stays
        // O is rescaled only when some row of the warp moved its max by more than 2^kRescaleThreshold; otherwise
        // the stale reference keeps P <= 2^8 and the final 1/l normalisation absorbs it.  While m_ref = -inf the
        // row's P has been all zeros, so its O row is exactly 0 and needs no rescale.
        const bool need = real && m_ref > -INFINITY && mx > m_ref + kRescaleThreshold;
        if (__any_sync(0xffffffffu, need)) {
          mbar_wait(o_full, (blk - 1) & 1);                // PV(blk-1) retired: O is ours (need implies blk > 0)
          tc_fence_after();
          float alpha = 1.f;
          if (need) {
            alpha = ex2_approx(m_ref - mx);
            m_ref = mx;
            l_run *= alpha;
          }
#pragma unroll
          for (int c4 = 0; c4 < 4; ++c4) {
            uint32_t ov[32];
            tmem_ld32(lane_addr + kColO + c4 * 32, ov);
            tmem_wait_ld();
#pragma unroll
            for (int c = 0; c < 32; ++c) ov[c] = __float_as_uint(__uint_as_float(ov[c]) * alpha);
            tmem_st32(lane_addr + kColO + c4 * 32, ov);
          }
          tmem_wait_st();
        }
        if (real && m_ref == -INFINITY && mx > -INFINITY) m_ref = mx;   // first visible keys of this row
        // pass 2: P = 2^(s*scale - m_ref) as bf16 hi + lo, written over S in place: hi of chunk c4 lands in
        // columns [16 c4, 16 c4 + 16) (already read), lo is held back until every S chunk has been read.
        const float m_use = (m_ref == -INFINITY) ? 0.f : m_ref;
        float lsum = 0.f;
        uint32_t plo[4][16];
#pragma unroll
        for (int c4 = 0; c4 < 4; ++c4) {
          if (c4 * 2 < np) {
            uint32_t sv[32];
            tmem_ld32(s_addr + c4 * 32, sv);
            tmem_wait_ld();
            const int nv0 = nvalid(c4 * 2), nv1 = nvalid(c4 * 2 + 1);   // 0 for padding / empty rows
            uint32_t phi[16];
#pragma unroll
            for (int c = 0; c < 32; c += 2) {
              const int nv = c < 16 ? nv0 : nv1;
              const int tk = c & 15;
              float e0 = 0.f, e1 = 0.f;
              if (tk < nv) e0 = ex2_approx(fmaf(__uint_as_float(sv[c]), p.scale_log2, -m_use));
              if (tk + 1 < nv) e1 = ex2_approx(fmaf(__uint_as_float(sv[c + 1]), p.scale_log2, -m_use));
              lsum += e0 + e1;
              split_bf16x2(e0, e1, phi[c >> 1], plo[c4][c >> 1]);
            }
            tmem_st16(s_addr + c4 * 16, phi);
          }
        }
#pragma unroll
        for (int c4 = 0; c4 < 4; ++c4)
          if (c4 * 2 < np) tmem_st16(s_addr + 64 + c4 * 16, plo[c4]);
        tmem_wait_st();
        l_run += lsum;
        tc_fence_before();
        mbar_arrive(&p_ready[blk & 1]);
      }
      // ---- epilogue: O / l and the base-2 lse of this split ----
      mbar_wait(o_done, 0);
      tc_fence_after();
      const float inv = l_run > 0.f ? 1.f / l_run : 0.f;
      const float lse2 = l_run > 0.f ? m_ref + log2f(l_run) : -INFINITY;
      float* dst;
      if (p.nsplit > 1) {
        dst = p.split_o + ((unit * p.nsplit + split) * rows + rho) * 128;
        if (rho < rows) p.split_lse[(unit * p.nsplit + split) * rows + rho] = lse2;
      } else {
        const int r = rho / G, g = rho % G;
        dst = p.part_o + (((size_t)b * R + r) * p.h_q + h * G + g) * 128;
        if (rho < rows) p.part_lse[((size_t)b * R + r) * p.h_q + h * G + g] = lse2 * kLn2;
      }
      if (quarter * 32 < rows) {                           // warp-uniform: this warp owns at least one real row
#pragma unroll
        for (int c4 = 0; c4 < 4; ++c4) {
          uint32_t ov[32];
          tmem_ld32(lane_addr + kColO + c4 * 32, ov);
          tmem_wait_ld();
          if (rho < rows) {
#pragma unroll
            for (int c = 0; c < 32; c += 4)
              *reinterpret_cast<float4*>(dst + c4 * 32 + c) =
                  make_float4(__uint_as_float(ov[c]) * inv, __uint_as_float(ov[c + 1]) * inv,
                              __uint_as_float(ov[c + 2]) * inv, __uint_as_float(ov[c + 3]) * inv);
          }
        }
      }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
      tc_fence_after();
      asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols));
    }
  } else {
    // no page for this split: empty partial for every row
    for (int rho = tid; rho < rows; rho += kUmmaThreads) {
      if (p.nsplit > 1) {
        p.split_lse[(unit * p.nsplit + split) * rows + rho] = -INFINITY;
      } else {
        const int r = rho / G, g = rho % G;
        float* dst = p.part_o + (((size_t)b * R + r) * p.h_q + h * G + g) * 128;
        for (int c = 0; c < 128; ++c) dst[c] = 0.f;
        p.part_lse[((size_t)b * R + r) * p.h_q + h * G + g] = -INFINITY;
      }
    }
  }
  if (p.nsplit == 1) return;
  combine_splits_last_cta<128>(p, unit, b, h, rows, G, R, &s_ticket);
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

int launch_attend_umma(const retro_desc_t* d, const AttendParams& prm, cudaStream_t s) {
  // the encode is pure host work (~1 us); cache the last pair of maps (one layer stack reuses its pools)
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
  const size_t smem = 1024 + UmmaSmem::list + (size_t)3 * prm.pages_per_split * sizeof(int32_t);
  static size_t smem_allowed = 0;
  if (smem > smem_allowed) {
    RETRO_CUDA_TRY(cudaFuncSetAttribute(attend_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    smem_allowed = smem;
  }
  attend_umma_kernel<<<dim3(prm.nsplit, d->num_kv_heads, d->batch), kUmmaThreads, smem, s>>>(prm, hit->mk, hit->mv);
  RETRO_LAUNCH_CHECK();
  return RETRO_OK;
}

}  // namespace retro
