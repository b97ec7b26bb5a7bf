// Per-warp digest of one (page, KV head) K tile: shared by the S1 kernel (bounds.cu) and by the
// select kernel's in-line refresh of the newest page (select.cu, retro_decode_step).
#pragma once
#include "common.cuh"

namespace retro {

template <typename T> struct Vec16;
template <> struct Vec16<float> {
  __device__ static __forceinline__ uint4 vmax(uint4 a, uint4 b) {
    uint4 r;
    r.x = __float_as_uint(fmaxf(__uint_as_float(a.x), __uint_as_float(b.x)));
    r.y = __float_as_uint(fmaxf(__uint_as_float(a.y), __uint_as_float(b.y)));
    r.z = __float_as_uint(fmaxf(__uint_as_float(a.z), __uint_as_float(b.z)));
    r.w = __float_as_uint(fmaxf(__uint_as_float(a.w), __uint_as_float(b.w)));
    return r;
  }
  __device__ static __forceinline__ uint4 vmin(uint4 a, uint4 b) {
    uint4 r;
    r.x = __float_as_uint(fminf(__uint_as_float(a.x), __uint_as_float(b.x)));
    r.y = __float_as_uint(fminf(__uint_as_float(a.y), __uint_as_float(b.y)));
    r.z = __float_as_uint(fminf(__uint_as_float(a.z), __uint_as_float(b.z)));
    r.w = __float_as_uint(fminf(__uint_as_float(a.w), __uint_as_float(b.w)));
    return r;
  }
};
template <> struct Vec16<__nv_bfloat16> {
  __device__ static __forceinline__ uint32_t max2(uint32_t a, uint32_t b) {
    __nv_bfloat162 r = __hmax2(*reinterpret_cast<__nv_bfloat162*>(&a), *reinterpret_cast<__nv_bfloat162*>(&b));
    return *reinterpret_cast<uint32_t*>(&r);
  }
  __device__ static __forceinline__ uint32_t min2(uint32_t a, uint32_t b) {
    __nv_bfloat162 r = __hmin2(*reinterpret_cast<__nv_bfloat162*>(&a), *reinterpret_cast<__nv_bfloat162*>(&b));
    return *reinterpret_cast<uint32_t*>(&r);
  }
  __device__ static __forceinline__ uint4 vmax(uint4 a, uint4 b) {
    return make_uint4(max2(a.x, b.x), max2(a.y, b.y), max2(a.z, b.z), max2(a.w, b.w));
  }
  __device__ static __forceinline__ uint4 vmin(uint4 a, uint4 b) {
    return make_uint4(min2(a.x, b.x), min2(a.y, b.y), min2(a.z, b.z), min2(a.w, b.w));
  }
};

__device__ __forceinline__ uint4 shfl_xor_u4(uint4 v, int m) {
  v.x = __shfl_xor_sync(0xffffffffu, v.x, m);
  v.y = __shfl_xor_sync(0xffffffffu, v.y, m);
  v.z = __shfl_xor_sync(0xffffffffu, v.z, m);
  v.w = __shfl_xor_sync(0xffffffffu, v.w, m);
  return v;
}

// A K row is 256 B = 16 lanes x 16 B ({f32, d64} and {bf16, d128}); the two half-warps take alternate rows.
// Returns the 16 B of the [Kmax ; Kmin] record that `lane` owns (lanes 0..15: Kmax, 16..31: Kmin), over the first
// n_valid (>= 1) rows of the tile.
template <typename T, int P>
__device__ __forceinline__ uint4 warp_page_digest(const uint4* tile, int n_valid, int lane) {
  const int sub = lane >> 4;   // which of the two rows of a pass
  const int col = lane & 15;   // 16-byte column within the row
  uint4 vmax = make_uint4(0, 0, 0, 0), vmin = make_uint4(0, 0, 0, 0);
  bool have = false;
#pragma unroll
  for (int r0 = 0; r0 < P; r0 += 2) {
    const int row = r0 + sub;
    if (row < n_valid) {
      const uint4 v = __ldg(tile + row * 16 + col);
      if (!have) {
        vmax = v; vmin = v; have = true;
      } else {
        vmax = Vec16<T>::vmax(vmax, v);
        vmin = Vec16<T>::vmin(vmin, v);
      }
    }
  }
  // combine the two half-warps; the odd half may be empty when n_valid == 1
  uint4 omax = shfl_xor_u4(vmax, 16), omin = shfl_xor_u4(vmin, 16);
  const bool ohave = __shfl_xor_sync(0xffffffffu, (int)have, 16) != 0;
  if (have && ohave) {
    vmax = Vec16<T>::vmax(vmax, omax);
    vmin = Vec16<T>::vmin(vmin, omin);
  } else if (!have) {
    vmax = omax; vmin = omin;
  }
  return sub == 0 ? vmax : vmin;
}

}  // namespace retro
