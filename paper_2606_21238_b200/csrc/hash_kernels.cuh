// K1 — chained block hashing (H1-H6).  All arithmetic is u64 mod 2^64.
//   g_i   = sum_k fold((w_k + (k+1) M) C1),  w_k = t[2k] | t[2k+1] << 32,  fold(e) = e ^ (e >> 32)
//   s_i   = s_{i-1} K + g_i,  s_{-1} = S0      (affine => a segmented scan over the blocks of a request)
//   key_i = mix(s_i), values 0 and 1 bumped by 2
// The constants below are typed in from the definition; the oracle has its own copy (no shared header).
#pragma once
#include "arc_device.cuh"

namespace arc {

constexpr unsigned long long H_M = 0x9E3779B97F4A7C15ull;
constexpr unsigned long long H_C1 = 0xBF58476D1CE4E5B9ull;
constexpr unsigned long long H_C2 = 0x94D049BB133111EBull;
constexpr unsigned long long H_K = 0xD1342543DE82EF95ull;
constexpr unsigned long long H_S0 = 0x243F6A8885A308D3ull;

__host__ __device__ constexpr unsigned long long kpow(unsigned n) {
  unsigned long long r = 1, b = H_K;
  while (n) { if (n & 1) r *= b; b *= b; n >>= 1; }
  return r;
}

__device__ __forceinline__ unsigned long long hash_word(uint32_t lo, uint32_t hi, unsigned k) {
  unsigned long long w = (unsigned long long)lo | ((unsigned long long)hi << 32);
  unsigned long long e = (w + (unsigned long long)(k + 1) * H_M) * H_C1;
  return e ^ (e >> 32);
}

__device__ __forceinline__ unsigned long long finalize_key(unsigned long long z) {
  z ^= z >> 30; z *= H_C1;
  z ^= z >> 27; z *= H_C2;
  z ^= z >> 31;
  return z < 2 ? z + 2 : z;
}

__device__ __forceinline__ unsigned long long shfl_up64(unsigned long long v, int d) {
  return __shfl_up_sync(0xFFFFFFFFu, v, d);
}

// Inclusive warp scan of the affine chain: on return lane l holds sum_{j<=l} K^(l-j) g_j.
__device__ __forceinline__ unsigned long long warp_chain_scan(unsigned long long g, int lane) {
  unsigned long long s = g, up;
  up = shfl_up64(s, 1);  if (lane >= 1)  s += kpow(1) * up;
  up = shfl_up64(s, 2);  if (lane >= 2)  s += kpow(2) * up;
  up = shfl_up64(s, 4);  if (lane >= 4)  s += kpow(4) * up;
  up = shfl_up64(s, 8);  if (lane >= 8)  s += kpow(8) * up;
  up = shfl_up64(s, 16); if (lane >= 16) s += kpow(16) * up;
  return s;
}

// K^(lane+1) without a table: square-and-multiply over the 6 bits of lane+1.
__device__ __forceinline__ unsigned long long kpow_lane(int e) {
  unsigned long long r = 1;
  if (e & 1) r *= kpow(1);
  if (e & 2) r *= kpow(2);
  if (e & 4) r *= kpow(4);
  if (e & 8) r *= kpow(8);
  if (e & 16) r *= kpow(16);
  if (e & 32) r *= kpow(32);
  return r;
}

// v1 kernel: one warp per request, 32 blocks per round, lane l hashes block base+l.
// ACCESS_ORDER = true writes keys at blk_off[r] + (nb-1-i) (the order K3 consumes, R2) plus the
// request-start flags; false writes natural order (arc_hash_blocks).
template <bool ACCESS_ORDER>
__global__ void __launch_bounds__(256) hash_warp_per_request_kernel(const int32_t* __restrict__ tokens,
                                                                   const int64_t* __restrict__ offsets,
                                                                   const int64_t* __restrict__ blk_off, uint32_t n_req,
                                                                   unsigned long long* __restrict__ keys,
                                                                   uint8_t* __restrict__ acc_start) {
  const int lane = threadIdx.x & 31;
  const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const uint32_t n_warps = (gridDim.x * blockDim.x) >> 5;
  for (uint32_t r = warp; r < n_req; r += n_warps) {
    const int64_t o = blk_off[r];
    const int64_t nb = blk_off[r + 1] - o;
    const uint32_t* t0 = reinterpret_cast<const uint32_t*>(tokens) + offsets[r];
    const bool aligned = (reinterpret_cast<uintptr_t>(t0) & 15) == 0;
    unsigned long long carry = H_S0;
    for (int64_t base = 0; base < nb; base += 32) {
      const int64_t i = base + lane;
      unsigned long long g = 0;
      if (i < nb) {
        const uint32_t* t = t0 + i * 16;
        if (aligned) {
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            uint4 v = __ldg(reinterpret_cast<const uint4*>(t) + q);
            g += hash_word(v.x, v.y, 2 * q) + hash_word(v.z, v.w, 2 * q + 1);
          }
        } else {
#pragma unroll
          for (int k = 0; k < 8; ++k) g += hash_word(__ldg(t + 2 * k), __ldg(t + 2 * k + 1), k);
        }
      }
      const unsigned long long s = warp_chain_scan(g, lane) + kpow_lane(lane + 1) * carry;
      if (i < nb) {
        const int64_t dst = ACCESS_ORDER ? (o + (nb - 1 - i)) : (o + i);
        keys[dst] = finalize_key(s);
        if (ACCESS_ORDER) acc_start[dst] = (i == nb - 1) ? 1 : 0;
      }
      carry = __shfl_sync(0xFFFFFFFFu, s, 31);
    }
  }
}

}  // namespace arc
