// K1 for callers that may not allocate (arc_hash_blocks_static): the segmented hashing of hash_kernels.cuh (requests cut
// into K1_SEG-block segments scanned from a zero carry, then put together: H4 is affine) with ALL its scratch in one
// fixed-size block of device memory that the library holds as a file-scope __device__ array (libarc.cu), keys in natural
// order.  Differences from hash_segments_kernel / hash_fixup_kernel: segments are dealt to the warps statically (no ticket:
// nothing in the scratch has to be zero when a call starts), the block offsets the second kernel needs are parked in the
// scratch by the first, new prompts only (every chain starts at S0).
#pragma once
#include "hash_kernels.cuh"

namespace arc {

constexpr uint32_t K1_STATIC_MAX_REQ = K1_INLINE_SMALL;     // the offsets travel as a 4 KB kernel argument
constexpr uint32_t K1_STATIC_MAX_SEGS = 4096;               // n_req x segments of the longest request, at most
constexpr uint32_t K1_STATIC_MAX_SEG_PER_REQ = 1024;        // kpow_segT takes exponents below 2^11

struct K1StaticScratch {
  long long blk_off[K1_STATIC_MAX_REQ + 3];                 // [n_req + 1] block offsets of the call in flight
  unsigned long long seg_end[K1_STATIC_MAX_SEGS];           // seg_end[r * max_seg + s]: local end state of segment s of request r
};

// keys[] gets the LOCAL states of every block in natural order (blk_off[r] + i); warp w takes segments w, w + n_warps, ...
__global__ void __launch_bounds__(256, 3) hash_segments_static_kernel(const int32_t* __restrict__ tokens, uint32_t n_req, uint32_t max_seg,
                                                                      unsigned long long* __restrict__ keys, K1StaticScratch* __restrict__ sc,
                                                                      const __grid_constant__ OffsetsArgT<K1_STATIC_MAX_REQ> arg) {
  extern __shared__ __align__(128) unsigned char k1_smem[];
  const int lane = threadIdx.x & 31;
  const long long* offsets = arg.v;
  const long long* blk_off = arg.v + (n_req + 1);
  if (blockIdx.x == 0)
    for (uint32_t i = threadIdx.x; i <= n_req; i += blockDim.x) sc->blk_off[i] = blk_off[i];
  const uint32_t* tok = reinterpret_cast<const uint32_t*>(tokens);
  const int64_t lo = offsets[0], hi = offsets[n_req];
  const LaneConsts LC = lane_consts(lane);
  WarpPipe W = pipe_init(k1_smem, threadIdx.x >> 5, lane);
  const int base_mis = (int)((reinterpret_cast<uintptr_t>(tok) >> 2) & 3);
  const uint32_t total = max_seg * n_req;
  const uint32_t warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
  for (uint32_t t = warp0; t < total; t += n_warps) {
    const uint32_t r = t % n_req, sg = t / n_req;
    const int64_t o = blk_off[r], nb = blk_off[r + 1] - o;
    const int64_t b0 = (int64_t)sg * K1_SEG;
    if (b0 >= nb) continue;
    const int64_t nbs = min((int64_t)K1_SEG, nb - b0);
    unsigned long long* out = keys + (o + b0 + lane);
    const unsigned long long end = hash_run(W, tok, base_mis, lo, hi, offsets[r] + 16 * b0, (uint32_t)nbs, 0ull, lane, LC,
      [&](uint32_t rb, int cnt, unsigned long long st) {
        if (lane < cnt) out[rb] = st;
      });
    if (lane == 0) sc->seg_end[(size_t)r * max_seg + sg] = end;
  }
}

// One warp per segment: the true state before it from the end states of the request's earlier segments, then keys.
__global__ void __launch_bounds__(256) hash_fixup_static_kernel(uint32_t n_req, uint32_t max_seg, unsigned long long* __restrict__ keys,
                                                                const K1StaticScratch* __restrict__ sc) {
  const int lane = threadIdx.x & 31;
  const uint32_t warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
  const unsigned long long kp = kpow_small(lane + 1);                 // K^(lane+1)
  const uint32_t total = n_req * max_seg;
  for (uint32_t w = warp0; w < total; w += n_warps) {
    const uint32_t r = w % n_req, sg = w / n_req;
    const int64_t o = sc->blk_off[r], nb = sc->blk_off[r + 1] - o;
    const int64_t b0 = (int64_t)sg * K1_SEG;
    if (b0 >= nb) continue;
    unsigned long long part = 0;
    for (uint32_t jb = 0; jb < sg; jb += 32) {
      const uint32_t jj = jb + (uint32_t)lane;
      if (jj < sg) part += kpow_seg(sg - 1 - jj) * sc->seg_end[(size_t)r * max_seg + jj];
    }
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) part += shfl_xor64(part, d);
    const unsigned long long carry = kpow_seg(sg) * H_S0 + part;      // the state before this segment's first block
    const int len = (int)min((int64_t)K1_SEG, nb - b0);
    unsigned long long kr = kp;                                        // K^(32 it + lane + 1)
#pragma unroll
    for (int it = 0; it < K1_SEG / 32; ++it) {
      const int i = 32 * it + lane;
      if (i < len) {
        const int64_t at = o + b0 + i;
        keys[at] = finalize_key(keys[at] + kr * carry);
      }
      kr *= kpow(32);
    }
  }
}

}  // namespace arc
