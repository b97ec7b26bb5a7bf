// S3  fused multi-query sparse attention (Eq. 2 / 6 / 7; Alg. 1 line 6).
//
// Grid (split, KV head, sequence).  A CTA walks its share of the selected-page list once; every (page, head)
// K tile and V tile (P*d*esize contiguous bytes, 4 KB) is staged into shared memory by the TMA unit
// (cp.async.bulk + mbarrier, kStages deep) and serves EVERY query row of the GQA group x (w+1) block.
// Rows are spread round-robin over the CTA's warps; a lane owns d/32 channels, so logits are finished with a
// transposed warp-shuffle reduction (16 tokens in 16 shuffles) and the softmax state (m, l) never leaves
// registers.  Row at position p attends page j iff sel_prev_j < p, token l iff l <= p and l < seq_len.
// Split partials (normalised o, base-2 lse) go to the workspace; the last CTA to finish a (b, head) unit
// combines them (LSE merge, Eq. 8 applied to splits) into part_o / part_lse.
//
// This is the scalar-ALU path: exact fp32 products (C1's 1e-4 tolerance rules out TF32) and small row blocks.
#include "attend_common.cuh"

namespace retro {

constexpr int kAttWarps = 8;
constexpr int kStages = 4;

template <typename T, int D> struct LaneSlice;   // a lane's D/32 channels of one row
template <> struct LaneSlice<__nv_bfloat16, 128> {
  static constexpr int kCh = 4;
  using Raw = uint2;
  __device__ static __forceinline__ void unpack(Raw r, float* f) {
    f[0] = bf16_lo(r.x); f[1] = bf16_hi(r.x); f[2] = bf16_lo(r.y); f[3] = bf16_hi(r.y);
  }
};
template <> struct LaneSlice<float, 64> {
  static constexpr int kCh = 2;
  using Raw = float2;
  __device__ static __forceinline__ void unpack(Raw r, float* f) { f[0] = r.x; f[1] = r.y; }
};

// Reduce 16 per-lane partial sums across the warp so that lane L ends with the total of token (L >> 1).
__device__ __forceinline__ float transpose_reduce16(float (&v)[16], int lane) {
  float a[8];
  {
    const bool up = lane & 16;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const float mine = up ? v[i + 8] : v[i], theirs = up ? v[i] : v[i + 8];
      a[i] = mine + __shfl_xor_sync(0xffffffffu, theirs, 16);
    }
  }
  float c[4];
  {
    const bool up = lane & 8;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const float mine = up ? a[i + 4] : a[i], theirs = up ? a[i] : a[i + 4];
      c[i] = mine + __shfl_xor_sync(0xffffffffu, theirs, 8);
    }
  }
  float e[2];
  {
    const bool up = lane & 4;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const float mine = up ? c[i + 2] : c[i], theirs = up ? c[i] : c[i + 2];
      e[i] = mine + __shfl_xor_sync(0xffffffffu, theirs, 4);
    }
  }
  const bool up = lane & 2;
  const float mine = up ? e[1] : e[0], theirs = up ? e[0] : e[1];
  float r = mine + __shfl_xor_sync(0xffffffffu, theirs, 2);
  r += __shfl_xor_sync(0xffffffffu, r, 1);
  return r;
}

template <typename T, int D, int RPW>
__global__ void __launch_bounds__(kAttWarps * 32) attend_simt_kernel(const AttendParams p) {
  constexpr int P = 16;
  constexpr int kCh = LaneSlice<T, D>::kCh;
  using Raw = typename LaneSlice<T, D>::Raw;
  constexpr int kTileBytes = P * D * sizeof(T);
  extern __shared__ __align__(128) unsigned char smem[];
  // [kStages][2][tile] | q rows [rows][D] T | page list (logical prev phys) | mbarriers
  T* s_kv = reinterpret_cast<T*>(smem);
  const int G = p.h_q / p.h_k;
  const int R = p.window + 1;
  const int rows = R * G;
  T* s_q = reinterpret_cast<T*>(smem + (size_t)kStages * 2 * kTileBytes);
  int32_t* s_list = reinterpret_cast<int32_t*>(s_q + (size_t)rows * D);   // [3][pages_per_split]
  uint64_t* s_bar = reinterpret_cast<uint64_t*>(
      (reinterpret_cast<uintptr_t>(s_list + 3 * p.pages_per_split) + 7) & ~uintptr_t(7));

  const int split = blockIdx.x, h = blockIdx.y, b = blockIdx.z;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  pdl_wait();
  pdl_trigger();
  const int L = p.seq_lens[b];
  const int t = L - 1;
  const size_t unit = (size_t)b * p.h_k + h;
  int count = p.sel_count[unit];
  RETRO_DBG_ONLY(if (count < 0 || count > p.k_max) { if (tid == 0) dbg_violation(p.dbg, kDbgSelCount); count = 0; })
  RETRO_DBG_ONLY(if (L < 0 || L > p.max_pages * P) { if (tid == 0) dbg_violation(p.dbg, kDbgSeqLen); count = 0; })
  const int beg = min(split * p.pages_per_split, count);
  const int end = min(beg + p.pages_per_split, count);
  const int n_my = end - beg;

  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&s_bar[s], 1);
    fence_mbar_init();
  }
  for (int i = tid; i < n_my; i += blockDim.x) {
    int j = p.sel_pages[unit * p.k_max + beg + i];
    int prev = p.sel_prev[unit * p.k_max + beg + i];
    RETRO_DBG_ONLY(if (j < 0 || j >= min((L + P - 1) / P, p.max_pages)) { dbg_violation(p.dbg, kDbgSelPage); j = 0; prev = 0x7fffffff; })
    int phys = p.block_table[(size_t)b * p.max_pages + j];
    RETRO_DBG_ONLY(if (phys < 0 || phys >= p.num_phys) { dbg_violation(p.dbg, kDbgPhysPage); phys = 0; prev = 0x7fffffff; })
    s_list[i] = j;
    s_list[p.pages_per_split + i] = prev;
    s_list[2 * p.pages_per_split + i] = phys;
  }
  // q rows of this KV head: row rho = r*G + g  <-  q_win[b][r][h*G+g][:]
  {
    constexpr int kChunks = D * sizeof(T) / 16;
    const uint4* src = reinterpret_cast<const uint4*>(p.q_win);
    uint4* dst = reinterpret_cast<uint4*>(s_q);
    for (int i = tid; i < rows * kChunks; i += blockDim.x) {
      const int rho = i / kChunks, c = i % kChunks;
      const int r = rho / G, g = rho % G;
      dst[i] = src[(((size_t)b * R + r) * p.h_q + h * G + g) * kChunks + c];
    }
  }
  __syncthreads();

  const T* kbase = reinterpret_cast<const T*>(p.k_pages);
  const T* vbase = reinterpret_cast<const T*>(p.v_pages);
  auto issue = [&](int i) {   // thread 0 only
    const int s = i % kStages;
    const size_t off = ((size_t)s_list[2 * p.pages_per_split + i] * p.h_k + h) * P * D;
    mbar_expect_tx(&s_bar[s], 2 * kTileBytes);
    bulk_g2s(s_kv + (size_t)s * 2 * P * D, kbase + off, kTileBytes, &s_bar[s]);
    bulk_g2s(s_kv + (size_t)s * 2 * P * D + P * D, vbase + off, kTileBytes, &s_bar[s]);
  };
  if (tid == 0)
    for (int i = 0; i < min(kStages, n_my); ++i) issue(i);

  // per-row state of this warp's rows: rho = warp + kAttWarps * i
  float m_run[RPW], l_run[RPW], acc[RPW][kCh];
  int row_pos[RPW];
#pragma unroll
  for (int i = 0; i < RPW; ++i) {
    m_run[i] = -INFINITY; l_run[i] = 0.f;
#pragma unroll
    for (int c = 0; c < kCh; ++c) acc[i][c] = 0.f;
    const int rho = warp + kAttWarps * i;
    int pos = -1;
    if (rho < rows) {
      pos = p.q_pos[b * R + rho / G];
      if (pos > t || pos < t - p.window) pos = -1;
    }
    row_pos[i] = pos;
  }

  for (int it = 0; it < n_my; ++it) {
    const int s = it % kStages;
    mbar_wait(&s_bar[s], (it / kStages) & 1);
    const int j = s_list[it], prev = s_list[p.pages_per_split + it];
    const T* kt = s_kv + (size_t)s * 2 * P * D;
    const T* vt = kt + P * D;
    Raw kraw[P], vraw[P];
#pragma unroll
    for (int l = 0; l < P; ++l) {
      kraw[l] = *reinterpret_cast<const Raw*>(kt + l * D + lane * kCh);
      vraw[l] = *reinterpret_cast<const Raw*>(vt + l * D + lane * kCh);
      // slots past the sequence's last token are unwritten memory: their weight is 0, and 0 x NaN must not happen
      if (j * P + l >= L) vraw[l] = Raw{};
    }
#pragma unroll
    for (int i = 0; i < RPW; ++i) {
      const int pos = row_pos[i];
      if (pos < 0 || !(prev < pos)) continue;                  // empty row, or page already seen by this query
      const int n_valid = min(min(pos, t) - j * P + 1, P);     // tokens l <= pos and l < seq_len
      if (n_valid <= 0) continue;
      const int rho = warp + kAttWarps * i;
      float qf[kCh];
      LaneSlice<T, D>::unpack(*reinterpret_cast<const Raw*>(s_q + (size_t)rho * D + lane * kCh), qf);
      float part[P];
#pragma unroll
      for (int l = 0; l < P; ++l) {
        float kf[kCh];
        LaneSlice<T, D>::unpack(kraw[l], kf);
        float d = 0.f;
#pragma unroll
        for (int c = 0; c < kCh; ++c) d = fmaf(qf[c], kf[c], d);
        part[l] = d;
      }
      float sc = transpose_reduce16(part, lane) * p.scale_log2;   // lane holds token (lane >> 1)
      const int tok = lane >> 1;
      if (tok >= n_valid) sc = -INFINITY;
      float mx = sc;
#pragma unroll
      for (int o = 16; o > 1; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
      const float m_new = fmaxf(m_run[i], mx);                     // finite: token 0 of the page is valid
      const float alpha = exp2f(m_run[i] - m_new);
      const float pw = exp2f(sc - m_new);
      m_run[i] = m_new;
      l_run[i] = l_run[i] * alpha + ((lane & 1) ? 0.f : pw);
#pragma unroll
      for (int c = 0; c < kCh; ++c) acc[i][c] *= alpha;
#pragma unroll
      for (int l = 0; l < P; ++l) {
        const float pl = __shfl_sync(0xffffffffu, pw, 2 * l);
        float vf[kCh];
        LaneSlice<T, D>::unpack(vraw[l], vf);
#pragma unroll
        for (int c = 0; c < kCh; ++c) acc[i][c] = fmaf(pl, vf[c], acc[i][c]);
      }
    }
    __syncthreads();                                             // every warp is done with stage s
    if (tid == 0 && it + kStages < n_my) issue(it + kStages);
  }

  // write this split's partial (normalised o, base-2 lse)
  float* so = p.nsplit > 1 ? p.split_o : nullptr;
#pragma unroll
  for (int i = 0; i < RPW; ++i) {
    const int rho = warp + kAttWarps * i;
    if (rho >= rows) continue;
    const float l_tot = warp_sum(l_run[i]);
    const float inv = l_tot > 0.f ? 1.f / l_tot : 0.f;
    const float lse2 = l_tot > 0.f ? m_run[i] + log2f(l_tot) : -INFINITY;
    if (so != nullptr) {
      float* dst = so + ((unit * p.nsplit + split) * rows + rho) * D + lane * kCh;
#pragma unroll
      for (int c = 0; c < kCh; ++c) dst[c] = acc[i][c] * inv;
      if (lane == 0) p.split_lse[(unit * p.nsplit + split) * rows + rho] = lse2;
    } else {
      const int r = rho / G, g = rho % G;
      float* dst = p.part_o + (((size_t)b * R + r) * p.h_q + h * G + g) * D + lane * kCh;
#pragma unroll
      for (int c = 0; c < kCh; ++c) dst[c] = acc[i][c] * inv;
      if (lane == 0) p.part_lse[((size_t)b * R + r) * p.h_q + h * G + g] = lse2 * kLn2;
    }
  }
  if (p.nsplit == 1) return;

  __shared__ unsigned int s_ticket;
  combine_splits_last_cta<D>(p, unit, b, h, rows, G, R, &s_ticket, 0, rows, &p.counters[unit]);
}

template <typename T, int D, int RPW>
static int launch_simt(const retro_desc_t* d, const AttendParams& prm, cudaStream_t s) {
  const int rows = (d->window + 1) * (d->num_q_heads / d->num_kv_heads);
  const size_t smem = (size_t)kStages * 2 * 16 * D * sizeof(T) + (size_t)rows * D * sizeof(T) +
                      (size_t)3 * prm.pages_per_split * sizeof(int32_t) + 8 + kStages * sizeof(uint64_t);
  auto kern = attend_simt_kernel<T, D, RPW>;
  if (smem > (size_t)device_info().max_smem_optin) return RETRO_ERR_UNSUPPORTED;
  const int rc = ensure_dynamic_smem((const void*)kern, smem);
  if (rc != RETRO_OK) return rc;
  RETRO_CUDA_TRY(launch_kernel(kern, dim3(prm.nsplit, d->num_kv_heads, d->batch), dim3(kAttWarps * 32), smem, s, prm));
  RETRO_LAUNCH_CHECK();
  return RETRO_OK;
}

template <typename T, int D>
static int dispatch_rpw(const retro_desc_t* d, const AttendParams& prm, cudaStream_t s) {
  const int rows = (d->window + 1) * (d->num_q_heads / d->num_kv_heads);
  const int rpw = ceil_div(rows, kAttWarps);
  if (rpw <= 1) return launch_simt<T, D, 1>(d, prm, s);
  if (rpw <= 2) return launch_simt<T, D, 2>(d, prm, s);
  if (rpw <= 5) return launch_simt<T, D, 5>(d, prm, s);
  if (rpw <= 9) return launch_simt<T, D, 9>(d, prm, s);
  if (rpw <= 17) return launch_simt<T, D, 17>(d, prm, s);
  if (rpw <= 33) return launch_simt<T, D, 33>(d, prm, s);
  return RETRO_ERR_UNSUPPORTED;
}

bool attend_can_fuse_merge(const retro_desc_t* d, const WorkspaceLayout& wl) {
  return d->dtype == RETRO_BF16 && wl.nrg == 1;
}

int launch_sparse_attend(const retro_desc_t* d, const WorkspaceLayout& wl, const void* q_win, const int32_t* q_pos,
                         const void* k_pages, const void* v_pages, const int32_t* block_table,
                         const int32_t* seq_lens, const int32_t* sel_pages, const int32_t* sel_prev,
                         const int32_t* sel_count, float* part_o, float* part_lse, void* workspace, cudaStream_t s,
                         const FusedMerge* fused) {
  AttendParams prm;
  char* ws = static_cast<char*>(workspace);
  prm.q_win = q_win; prm.q_pos = q_pos; prm.k_pages = k_pages; prm.v_pages = v_pages;
  prm.block_table = block_table; prm.seq_lens = seq_lens; prm.sel_pages = sel_pages; prm.sel_prev = sel_prev;
  prm.sel_count = sel_count; prm.part_o = part_o; prm.part_lse = part_lse;
  prm.split_o = reinterpret_cast<float*>(ws + wl.split_o_off);
  prm.split_lse = reinterpret_cast<float*>(ws + wl.split_lse_off);
  prm.counters = reinterpret_cast<unsigned int*>(ws + wl.counters_off) + d->batch * d->num_kv_heads;   // [units]
  prm.B = d->batch; prm.h_q = d->num_q_heads; prm.h_k = d->num_kv_heads; prm.max_pages = d->max_pages_per_seq;
  prm.k_max = d->max_sel_pages; prm.window = d->window; prm.nsplit = wl.nsplit;
  prm.pages_per_split = wl.pages_per_split;
  prm.scale_log2 = d->sm_scale * kLog2e;
  prm.nrg = wl.nrg;
  prm.rg_ranks = wl.rg_ranks;
  prm.fused = 0;
  prm.cache_bf16 = 0;
  prm.cache_o = nullptr; prm.cache_lse = nullptr; prm.cache_pos = nullptr; prm.out = nullptr; prm.out_lse = nullptr;
  prm.seq_counters = reinterpret_cast<unsigned int*>(ws + wl.slot_counters_off);   // [B]
  prm.dbg = reinterpret_cast<unsigned int*>(ws + wl.debug_off);
  prm.num_phys = d->num_phys_pages;
  if (d->dtype == RETRO_BF16) {
    // bf16: the rows x keys block is a dense contraction -> tcgen05 tensor cores (attend_umma.cu; more than 128
    // rows run as row groups)
    if (fused != nullptr) {
      if (!attend_can_fuse_merge(d, wl)) return RETRO_ERR_UNSUPPORTED;
      prm.fused = 1;
      prm.cache_o = fused->cache_o; prm.cache_lse = fused->cache_lse; prm.cache_pos = fused->cache_pos;
      prm.cache_bf16 = d->cache_dtype == RETRO_BF16;
      prm.out = fused->out; prm.out_lse = fused->out_lse;
    }
    return launch_attend_umma(d, prm, s);
  }
  if (fused != nullptr) return RETRO_ERR_UNSUPPORTED;
  return dispatch_rpw<float, 64>(d, prm, s);
}

}  // namespace retro
