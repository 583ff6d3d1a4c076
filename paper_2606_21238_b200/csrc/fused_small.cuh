// The one-launch path for SMALL steps (the paper's own regime is batch size 1 with one request of a few
// hundred blocks per step): K1, K2, K3 and K4 as four phases of ONE kernel run by ONE CTA of 256 threads,
// __syncthreads between the phases instead of kernel boundaries.  Nothing is computed differently: the phases are the
// bodies of the stand-alone kernels (hash_run, probe_range, the one-warp / the wide machine, finalize_body), so every
// result is the same bit for bit; what goes away is five launches and their dependency gaps (about 2.5 us each), which
// is most of a step of a few hundred accesses.
//   phase 1a  every request is cut into segments of FUSED_SEG = 64 blocks; warp w hashes segments w, w + 8, ... from a
//             zero carry through its bulk-copy stage ring (local states to keys_acc, end states to seg_end);
//   phase 1b  one warp per segment rebuilds the true state before it (H4 is affine) and turns the states into keys;
//   phase 2   the 256 threads probe / reserve (K2);   phase 3  the ARC machine;   phase 4  finalize (K4).
// The offsets come as the kernel argument (at most K1_INLINE_SMALL requests); CTA-wide scratch lives in shared memory.
#pragma once
#include "directory_kernels.cuh"
#include "hash_kernels.cuh"
#include "machine_wide.cuh"

namespace arc {

constexpr int FUSED_SEG_LOG2 = 6, FUSED_SEG = 1 << FUSED_SEG_LOG2;
constexpr uint32_t FUSED_MAX_ACCESS = 4096;                       // N of a step the kernel takes at most (64 + 253 segments at most)
constexpr uint32_t FUSED_MAX_ITEMS = FUSED_MAX_ACCESS / FUSED_SEG + K1_INLINE_SMALL + 1;

struct FusedShared {
  WideShared wide;
  uint4 vic[5][32];                                               // the one-warp machine's victims
  uint32_t seg_off[K1_INLINE_SMALL + 2];                          // exclusive scan of the segments per request
  unsigned long long seg_end[FUSED_MAX_ITEMS];                    // local end state of every segment
};

// machine: 2 = one warp, 3 = wide.  LRU / HOLD as in the wide machine: every variant carries only its own code.
template <bool LRU, bool HOLD>
__global__ void __launch_bounds__(2 * WIDE_W, 1) arc_fused_small_kernel(const __grid_constant__ StepParams P, const unsigned long long* __restrict__ chain_in,
                                                                      unsigned long long* __restrict__ chain_out, int64_t* __restrict__ offsets_g,
                                                                      int64_t* __restrict__ blk_off_g, int machine,
                                                                      const __grid_constant__ OffsetsArgT<K1_INLINE_SMALL> arg) {
  extern __shared__ __align__(128) unsigned char k1_smem[];
  __shared__ FusedShared F;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t n_req = P.n_req;
  const long long* offsets = arg.v;
  const long long* blk_off = arg.v + (n_req + 1);
  for (uint32_t i = tid; i <= n_req; i += blockDim.x) { offsets_g[i] = arg.v[i]; blk_off_g[i] = arg.v[n_req + 1 + i]; }   // for K3 / K4 and the caller
  if (warp == 0) {                                                 // segments per request, exclusive scan (n_req <= 253: 8 rounds of 32)
    uint32_t run = 0;
    for (uint32_t base = 0; base <= n_req; base += 32) {
      const uint32_t r = base + (uint32_t)lane;
      const uint32_t ns = (r < n_req) ? (uint32_t)((blk_off[r + 1] - blk_off[r] + FUSED_SEG - 1) >> FUSED_SEG_LOG2) : 0u;
      uint32_t incl = ns;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) { const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, incl, d); if (lane >= d) incl += v; }
      if (r <= n_req) F.seg_off[r] = run + incl - ns;
      run += __shfl_sync(0xFFFFFFFFu, incl, 31);
    }
  }
  __syncthreads();
  const uint32_t n_items = F.seg_off[n_req];
  auto item_request = [&](uint32_t it) {                           // request r with seg_off[r] <= it < seg_off[r + 1]
    uint32_t lo = 0, hi = n_req;
    while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (F.seg_off[mid] <= it) lo = mid; else hi = mid; }
    return lo;
  };
  // ---- phase 1a: local scans of the segments
  {
    const uint32_t* tok = reinterpret_cast<const uint32_t*>(P.tokens);
    const int64_t lo = offsets[0], hi = offsets[n_req];
    const LaneConsts LC = lane_consts(lane);
    WarpPipe W = pipe_init(k1_smem, warp, lane);
    const int base_mis = (int)((reinterpret_cast<uintptr_t>(tok) >> 2) & 3);
    for (uint32_t it = (uint32_t)warp; it < n_items; it += K1_WARPS) {
      const uint32_t r = item_request(it), sg = it - F.seg_off[r];
      const int64_t o = blk_off[r], nb = blk_off[r + 1] - o;
      const int64_t b0 = (int64_t)sg * FUSED_SEG;
      const uint32_t nbs = (uint32_t)min((int64_t)FUSED_SEG, nb - b0);
      unsigned long long* out = P.keys_acc + (o + nb - 1 - b0 - lane);
      const unsigned long long end = hash_run(W, tok, base_mis, lo, hi, offsets[r] + 16 * b0, nbs, 0ull, lane, LC,
        [&](uint32_t rb, int cnt, unsigned long long st) { if (lane < cnt) *(out - rb) = st; });
      if (lane == 0) F.seg_end[it] = end;
    }
  }
  __syncthreads();
  // ---- phase 1b: true carries, keys, chain states
  {
    const unsigned long long kp = kpow_small(lane + 1);             // K^(lane+1)
    for (uint32_t it = (uint32_t)warp; it < n_items; it += K1_WARPS) {
      const uint32_t r = item_request(it), first = F.seg_off[r], sg = it - first;
      const int64_t o = blk_off[r], nb = blk_off[r + 1] - o;
      const int64_t b0 = (int64_t)sg * FUSED_SEG;
      const unsigned long long c0 = chain_in ? chain_in[r] : H_S0;
      unsigned long long part = 0;
      for (uint32_t jb = 0; jb < sg; jb += 32) {
        const uint32_t jj = jb + (uint32_t)lane;
        if (jj < sg) part += kpow_segT<FUSED_SEG_LOG2>(sg - 1 - jj) * F.seg_end[first + jj];
      }
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) part += shfl_xor64(part, d);
      const unsigned long long carry = kpow_segT<FUSED_SEG_LOG2>(sg) * c0 + part;   // the state before this segment's first block
      const int len = (int)min((int64_t)FUSED_SEG, nb - b0);
      unsigned long long kr = kp, last = 0;
#pragma unroll
      for (int q = 0; q < FUSED_SEG / 32; ++q) {
        const int i = 32 * q + lane;
        if (i < len) {
          unsigned long long* at = P.keys_acc + (o + (nb - 1 - (b0 + i)));
          const unsigned long long st = __ldcg(at) + kr * carry;
          *at = finalize_key(st);
          if (i == len - 1) last = st;
        }
        kr *= kpow(32);
      }
      if (b0 + len == nb) {                                          // the request's last segment: its end state goes out
        last = shfl64(last, (len - 1) & 31);
        if (lane == 0) chain_out[r] = last;
      }
    }
    for (uint32_t r = tid; r < n_req; r += blockDim.x)               // a request without a full block keeps the state it came with
      if (blk_off[r + 1] == blk_off[r]) chain_out[r] = chain_in ? chain_in[r] : H_S0;
  }
  __syncthreads();
  // ---- phase 2: K2
  probe_range(P, (uint32_t)tid, blockDim.x);
  __syncthreads();
  if (P.pin_scope != 0) {                                            // the window machines' windows span requests there (nat_index_body)
    nat_index_body(P, (uint32_t)warp, blockDim.x >> 5, (uint32_t)lane);
    __syncthreads();
  }
  // ---- phase 3: K3
  if (machine == 2) { if (warp == 0) batched_machine_run(P, F.vic); }
  else wide_machine_run<LRU, HOLD, false>(P, F.wide);
  __syncthreads();
  // ---- phase 4: K4
  finalize_body(P);
}

}  // namespace arc
