// K1 — chained block hashing (H1-H6).  All arithmetic is u64 mod 2^64.
//   g_i   = sum_k fold((w_k + (k+1) M) C1),  w_k = t[2k] | t[2k+1] << 32,  fold(e) = e ^ (e >> 32)
//   s_i   = s_{i-1} K + g_i,  s_{-1} = S0      (affine => a segmented scan over the blocks of a request)
//   key_i = mix(s_i), values 0 and 1 bumped by 2
// The constants below are typed in from the definition; the oracle has its own copy (no shared header).
//
// Kernel shape.  HBM-bound: 64 B read + 8 B written per block.  One warp owns one request
// at a time; requests are handed out through an atomic ticket, longest length class first, so long and
// short requests balance.  A warp walks its request in rounds of 32 blocks = 2 KB of tokens:
//   * loads: the round's tokens are fetched as 128-bit vectors from the 16-byte-ALIGNED cover of the
//     round, lane l taking vector 32*it + l (it = 0..3): every load instruction is one fully coalesced
//     512-byte access whatever the request's alignment; the next round's vectors are issued before the
//     current round is hashed (register double buffer), streaming through L1/L2 (ld.global.cs);
//   * a request that starts s tokens past a 16-byte boundary is realigned in registers with s shuffles;
//   * lane l then holds 4 tokens = words 2q, 2q+1 (q = l % 4) of block 8*it + l/4; the four partial sums
//     of a block are combined with a transpose-reduce (6 shuffles for the four iterations together),
//     one more shuffle puts block i in lane i, and a 5-step warp scan with the constants K^(2^d)
//     evaluates the affine chain; the carry into the next round is lane 31's state.
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

// fold((w + salt) C1) with w = lo | hi << 32; salt = (k+1) M is passed in
__device__ __forceinline__ unsigned long long hash_word(uint32_t lo, uint32_t hi, unsigned long long salt) {
  const unsigned long long w = (unsigned long long)lo | ((unsigned long long)hi << 32);
  const unsigned long long e = (w + salt) * H_C1;
  return e ^ (e >> 32);
}

__device__ __forceinline__ unsigned long long finalize_key(unsigned long long z) {
  z ^= z >> 30; z *= H_C1;
  z ^= z >> 27; z *= H_C2;
  z ^= z >> 31;
  return z < 2 ? z + 2 : z;
}

__device__ __forceinline__ unsigned long long shfl64(unsigned long long v, int src) { return __shfl_sync(0xFFFFFFFFu, v, src); }
__device__ __forceinline__ unsigned long long shfl_xor64(unsigned long long v, int m) { return __shfl_xor_sync(0xFFFFFFFFu, v, m); }
__device__ __forceinline__ unsigned long long shfl_up64(unsigned long long v, int d) { return __shfl_up_sync(0xFFFFFFFFu, v, d); }

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

// K^e for e in 1..32, without a table: square-and-multiply over the 6 bits of e.
__device__ __forceinline__ unsigned long long kpow_small(int e) {
  unsigned long long r = 1;
  if (e & 1) r *= kpow(1);
  if (e & 2) r *= kpow(2);
  if (e & 4) r *= kpow(4);
  if (e & 8) r *= kpow(8);
  if (e & 16) r *= kpow(16);
  if (e & 32) r *= kpow(32);
  return r;
}

// The tokens of one round as this lane sees them: vector 32*it + lane of the round's aligned cover (it = 0..3),
// and vector 128 (x) in lane 0 only (needed when the request is misaligned and the round is full).
struct RoundVecs {
  uint4 v[4];
  uint4 x;
};

// 128-bit streaming load of tokens [g0, g0 + 4) (absolute token indices, tok + g0 is 16-byte aligned); words outside
// the valid range [lo, hi) of the caller's buffer are not touched and read as 0.  Only rounds at the very edge of the
// caller's buffer come here.
__device__ __noinline__ uint4 ld_tokens4_guarded(const uint32_t* __restrict__ tok, int64_t g0, int64_t lo, int64_t hi) {
  uint4 r = make_uint4(0, 0, 0, 0);
  if (g0 + 0 >= lo && g0 + 0 < hi) r.x = __ldcs(tok + g0 + 0);
  if (g0 + 1 >= lo && g0 + 1 < hi) r.y = __ldcs(tok + g0 + 1);
  if (g0 + 2 >= lo && g0 + 2 < hi) r.z = __ldcs(tok + g0 + 2);
  if (g0 + 3 >= lo && g0 + 3 < hi) r.w = __ldcs(tok + g0 + 3);
  return r;
}

// va = absolute token index of the aligned cover's first word for this round; n_vec = vectors the round needs (0..129).
__device__ __forceinline__ RoundVecs load_round(const uint32_t* __restrict__ tok, int64_t va, int n_vec, int lane, int64_t lo, int64_t hi) {
  RoundVecs R;
  if (va >= lo && va + 4 * (int64_t)n_vec <= hi) {            // the whole cover is inside the caller's buffer (warp-uniform)
    const uint4* p = reinterpret_cast<const uint4*>(tok + va) + lane;
#pragma unroll
    for (int it = 0; it < 4; ++it) R.v[it] = (it * 32 + lane < n_vec) ? __ldcs(p + it * 32) : make_uint4(0, 0, 0, 0);
    R.x = (lane == 0 && n_vec > 128) ? __ldcs(p + 128) : make_uint4(0, 0, 0, 0);
  } else {
#pragma unroll
    for (int it = 0; it < 4; ++it) {
      const int e = it * 32 + lane;
      R.v[it] = (e < n_vec) ? ld_tokens4_guarded(tok, va + 4 * (int64_t)e, lo, hi) : make_uint4(0, 0, 0, 0);
    }
    R.x = (lane == 0 && n_vec > 128) ? ld_tokens4_guarded(tok, va + 512, lo, hi) : make_uint4(0, 0, 0, 0);
  }
  return R;
}

// word c (0..2) of the vector that FOLLOWS this lane's vector `cur` in the round: lane l+1's cur, and for lane 31
// lane 0's `nxt` (the same lane-0 register of the next iteration / the 129th vector).
__device__ __forceinline__ uint32_t next_word(uint32_t cur, uint32_t nxt, int lane) {
  return __shfl_sync(0xFFFFFFFFu, lane == 0 ? nxt : cur, (lane + 1) & 31);
}

struct LaneConsts {
  unsigned long long salt0, salt1;   // (k+1) M C1 for this lane's two words k = 2q, 2q+1 (the salt is folded into the multiply-add)
  unsigned long long kp;             // K^(lane+1)
  int owner;                         // after the transpose-reduce, block i of the round sits in lane `owner` of lane i
};

// Local chain states of one round: lane i returns sum_{j<=i} K^(i-j) g_j over the round's blocks (no carry-in);
// lanes >= cnt contribute g = 0.  s = request misalignment in tokens.
__device__ __forceinline__ unsigned long long round_local_scan(const RoundVecs& cur, int s, int cnt, int lane, const LaneConsts& LC) {
  unsigned long long part[4];
#pragma unroll
  for (int it = 0; it < 4; ++it) {
    const uint4 v = cur.v[it];
    const uint4 w = (it < 3) ? cur.v[it + 1] : cur.x;     // lane 0's copy is what lane 31 needs
    uint32_t a, b, c2, d;
    if (s == 0) { a = v.x; b = v.y; c2 = v.z; d = v.w; }
    else if (s == 1) { a = v.y; b = v.z; c2 = v.w; d = next_word(v.x, w.x, lane); }
    else if (s == 2) { a = v.z; b = v.w; c2 = next_word(v.x, w.x, lane); d = next_word(v.y, w.y, lane); }
    else { a = v.w; b = next_word(v.x, w.x, lane); c2 = next_word(v.y, w.y, lane); d = next_word(v.z, w.z, lane); }
    // fold((w + (k+1) M) C1) = fold(w C1 + (k+1) M C1)
    const unsigned long long e0 = ((unsigned long long)a | ((unsigned long long)b << 32)) * H_C1 + LC.salt0;
    const unsigned long long e1 = ((unsigned long long)c2 | ((unsigned long long)d << 32)) * H_C1 + LC.salt1;
    part[it] = (e0 ^ (e0 >> 32)) + (e1 ^ (e1 >> 32));
  }
  // transpose-reduce over the 4 lanes of a block: afterwards lane l holds g of block (l/4) + 8*(l%4)
  const bool b0 = lane & 1, b1 = lane & 2;
  const unsigned long long r0 = shfl_xor64(b0 ? part[0] : part[1], 1), r1 = shfl_xor64(b0 ? part[2] : part[3], 1);
  const unsigned long long pa = (b0 ? part[1] : part[0]) + r0, pb = (b0 ? part[3] : part[2]) + r1;
  const unsigned long long g_own = (b1 ? pb : pa) + shfl_xor64(b1 ? pa : pb, 2);
  unsigned long long g = shfl64(g_own, LC.owner);      // lane i <- block i
  if (lane >= cnt) g = 0;
  return warp_chain_scan(g, lane);
}

// Length classes for the ticket passes: requests of at least K1_CLASS_MIN[c] blocks are started in pass c, so the
// longest chains start first and the short requests fill the tail of the launch (longest-processing-time-first).
constexpr int K1_PASSES = 4;
__device__ __forceinline__ int k1_class(int64_t nb) { return nb >= 1024 ? 0 : nb >= 384 ? 1 : nb >= 128 ? 2 : 3; }

// ACCESS_ORDER = true writes keys at blk_off[r] + (nb-1-i) (the order K3 consumes, R2); false writes natural
// order (arc_hash_blocks).  ticket: device counter, 0 at launch, reset by the caller's stream work; it runs over
// K1_PASSES * n_req values: ticket t is request t % n_req in pass t / n_req.
// CHAIN = true reads each request's initial H4 state from chain_in (NULL = S0) and writes its final state to chain_out
// (arc_step / arc_step_resume); false is the stateless arc_hash_blocks, which pays nothing for it.
template <bool ACCESS_ORDER, bool CHAIN>
__global__ void __launch_bounds__(256, 4) hash_blocks_kernel(const int32_t* __restrict__ tokens, const int64_t* __restrict__ offsets,
                                                         const int64_t* __restrict__ blk_off, uint32_t n_req,
                                                         unsigned long long* __restrict__ keys, uint32_t* __restrict__ ticket, uint32_t batch,
                                                         const unsigned long long* __restrict__ chain_in,
                                                         unsigned long long* __restrict__ chain_out) {
  const int lane = threadIdx.x & 31;
  const uint32_t* tok = reinterpret_cast<const uint32_t*>(tokens);
  const int64_t lo = offsets[0], hi = offsets[n_req];
  LaneConsts LC;
  const int q = lane & 3;
  LC.salt0 = (unsigned long long)(2 * q + 1) * H_M * H_C1;
  LC.salt1 = (unsigned long long)(2 * q + 2) * H_M * H_C1;
  LC.kp = kpow_small(lane + 1);
  LC.owner = 4 * (lane & 7) + (lane >> 3);
  const int base_mis = (int)((reinterpret_cast<uintptr_t>(tok) >> 2) & 3);   // tokens of the buffer start past a 16-byte boundary
  const unsigned long long total = (unsigned long long)K1_PASSES * n_req;

  for (;;) {
    // `batch` (<= 32) tickets per atomic: lane l < batch examines ticket t0 + l, the warp then hashes the ones that belong to the pass
    uint32_t t0 = 0;
    if (lane == 0) t0 = atomicAdd(ticket, batch);
    t0 = __shfl_sync(0xFFFFFFFFu, t0, 0);
    if (t0 >= total) break;
    const unsigned long long t = (unsigned long long)t0 + lane;
    bool mine = false;
    uint32_t my_r = 0;
    if (t < total && (uint32_t)lane < batch) {
      my_r = (uint32_t)(t % n_req);
      const int64_t nb = blk_off[my_r + 1] - blk_off[my_r];
      mine = nb > 0 && k1_class(nb) == (int)(t / n_req);
      // a request without a full block keeps the state it came with (written once, in the last pass)
      if (CHAIN && nb == 0 && t / n_req == K1_PASSES - 1) chain_out[my_r] = chain_in ? chain_in[my_r] : H_S0;
    }
    uint32_t todo = __ballot_sync(0xFFFFFFFFu, mine);
    while (todo) {
      const int src = __ffs(todo) - 1;
      todo &= todo - 1;
      const uint32_t r = __shfl_sync(0xFFFFFFFFu, my_r, src);
      const int64_t o = blk_off[r], nb = blk_off[r + 1] - o;
      const int64_t ts = offsets[r];
      const int s = (int)((base_mis + ts) & 3);          // tokens of the request's start past a 16-byte boundary (same for every round)
      unsigned long long carry = (CHAIN && chain_in) ? chain_in[r] : H_S0;     // the H4 state before block 0 (a prompt: S0)
      const int64_t va = ts - s;                         // absolute token index of the aligned cover of round 0
      // two register buffers ping-pong (no copies): the loads of round i+1 are in flight while round i is hashed
      auto n_vec = [&](int64_t rb) { return (int)((16 * min((int64_t)32, nb - rb) + s + 3) >> 2); };
      auto finish = [&](const RoundVecs& cur, int64_t rb) {
        const int cnt = (int)min((int64_t)32, nb - rb);
        const unsigned long long st = round_local_scan(cur, s, cnt, lane, LC) + LC.kp * carry;
        if (lane < cnt) {
          const int64_t i = rb + lane;
          keys[ACCESS_ORDER ? (o + (nb - 1 - i)) : (o + i)] = finalize_key(st);
          if (CHAIN && i == nb - 1) chain_out[r] = st;           // the state a continuation of this sequence starts from
        }
        carry = shfl64(st, 31);
      };
      RoundVecs A = load_round(tok, va, n_vec(0), lane, lo, hi), B;
      for (int64_t rb = 0;;) {
        if (rb + 32 < nb) B = load_round(tok, va + 16 * (rb + 32), n_vec(rb + 32), lane, lo, hi);
        finish(A, rb);
        rb += 32;
        if (rb >= nb) break;
        if (rb + 32 < nb) A = load_round(tok, va + 16 * (rb + 32), n_vec(rb + 32), lane, lo, hi);
        finish(B, rb);
        rb += 32;
        if (rb >= nb) break;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------------
// In-step hashing of steps with FEW requests: one warp per request leaves the step waiting for its longest request (a
// 1,000-block document is 32 dependent rounds).  H4 is affine, so a request is cut into segments of K1_SEG blocks that are
// scanned independently from a zero carry (hash_segments_kernel: one warp per segment, the same loads and scans as
// above) and put together afterwards (hash_fixup_kernel): with c_s the true state before segment s and E_s the local end
// state of the segment, c_{s+1} = E_s + K^len_s c_s, and block i of the segment has state local_i + K^(i+1) c_s.
// Steps with up to K1_INLINE_REQ requests hand their offsets and block offsets to the device as a kernel argument: a launch
// costs a few microseconds less than the copy engine's round trip, and the step's first kernel waits for them.
constexpr uint32_t K1_INLINE_REQ = 253;
struct OffsetsArg { long long v[2 * (K1_INLINE_REQ + 1)]; };       // offsets[n_req + 1] then blk_off[n_req + 1]: 4,064 bytes
__global__ void __launch_bounds__(256) store_offsets_kernel(const __grid_constant__ OffsetsArg a, uint32_t n_req, int64_t* offsets, int64_t* blk_off) {
  for (uint32_t i = threadIdx.x; i <= n_req; i += blockDim.x) { offsets[i] = a.v[i]; blk_off[i] = a.v[n_req + 1 + i]; }
}

constexpr int K1_SEG = 128;

// states[] gets the LOCAL states, in access order (index blk_off[r] + nb - 1 - i); seg_end[r * max_seg + s] = E_s.
// ARG = true: the offsets come as the kernel argument `arg` (steps of up to K1_INLINE_REQ requests) and CTA 0 also stores
// them to offsets_g / blk_off_g for the kernels that follow; false: they are read from those arrays.
template <bool ARG>
__global__ void __launch_bounds__(256, 4) hash_segments_kernel(const int32_t* __restrict__ tokens, int64_t* __restrict__ offsets_g,
                                                               int64_t* __restrict__ blk_off_g, uint32_t n_req, uint32_t max_seg,
                                                               unsigned long long* __restrict__ states,
                                                               unsigned long long* __restrict__ seg_end, uint32_t* __restrict__ ticket,
                                                               const __grid_constant__ OffsetsArg arg) {
  const int lane = threadIdx.x & 31;
  const long long* offsets = ARG ? arg.v : reinterpret_cast<const long long*>(offsets_g);
  const long long* blk_off = ARG ? arg.v + (n_req + 1) : reinterpret_cast<const long long*>(blk_off_g);
  if (ARG && blockIdx.x == 0)
    for (uint32_t i = threadIdx.x; i <= n_req; i += blockDim.x) { offsets_g[i] = arg.v[i]; blk_off_g[i] = arg.v[n_req + 1 + i]; }
  const uint32_t* tok = reinterpret_cast<const uint32_t*>(tokens);
  const int64_t lo = offsets[0], hi = offsets[n_req];
  LaneConsts LC;
  const int q = lane & 3;
  LC.salt0 = (unsigned long long)(2 * q + 1) * H_M * H_C1;
  LC.salt1 = (unsigned long long)(2 * q + 2) * H_M * H_C1;
  LC.kp = kpow_small(lane + 1);
  LC.owner = 4 * (lane & 7) + (lane >> 3);
  const int base_mis = (int)((reinterpret_cast<uintptr_t>(tok) >> 2) & 3);
  const unsigned long long total = (unsigned long long)max_seg * n_req;
  for (;;) {
    uint32_t t0 = 0;
    if (lane == 0) t0 = atomicAdd(ticket, 1u);                      // one segment per ticket: segments are equal pieces of work
    t0 = __shfl_sync(0xFFFFFFFFu, t0, 0);
    if (t0 >= total) break;
    const uint32_t r = t0 % n_req, sg = t0 / n_req;                 // ticket t = segment t / n_req of request t % n_req
    if ((int64_t)sg * K1_SEG >= blk_off[r + 1] - blk_off[r]) continue;
    {
      const int64_t o = blk_off[r], nb = blk_off[r + 1] - o;
      const int64_t b0 = (int64_t)sg * K1_SEG, nbs = min((int64_t)K1_SEG, nb - b0);
      const int64_t ts = offsets[r] + 16 * b0;
      const int s = (int)((base_mis + ts) & 3);
      const int64_t va = ts - s;
      unsigned long long carry = 0;
      auto n_vec = [&](int64_t rb) { return (int)((16 * min((int64_t)32, nbs - rb) + s + 3) >> 2); };
      auto finish = [&](const RoundVecs& cur, int64_t rb) {
        const int cnt = (int)min((int64_t)32, nbs - rb);
        const unsigned long long st = round_local_scan(cur, s, cnt, lane, LC) + LC.kp * carry;
        if (lane < cnt) {
          const int64_t i = b0 + rb + lane;
          states[o + (nb - 1 - i)] = st;
          if (rb + lane == nbs - 1) seg_end[(size_t)r * max_seg + sg] = st;
        }
        carry = shfl64(st, 31);
      };
      RoundVecs A = load_round(tok, va, n_vec(0), lane, lo, hi), B;
      for (int64_t rb = 0;;) {
        if (rb + 32 < nbs) B = load_round(tok, va + 16 * (rb + 32), n_vec(rb + 32), lane, lo, hi);
        finish(A, rb);
        rb += 32;
        if (rb >= nbs) break;
        if (rb + 32 < nbs) A = load_round(tok, va + 16 * (rb + 32), n_vec(rb + 32), lane, lo, hi);
        finish(B, rb);
        rb += 32;
        if (rb >= nbs) break;
      }
    }
  }
}

// K^(128 m): square-and-multiply over the bits of m (m < 2^11)
__device__ __forceinline__ unsigned long long kpow_seg(uint32_t m) {
  unsigned long long r = 1;
#pragma unroll
  for (int b = 0; b < 11; ++b) {
    unsigned long long f = 1;                       // K^(128 2^b) as a compile-time constant
    switch (b) {
      case 0: f = kpow(128u); break;       case 1: f = kpow(256u); break;      case 2: f = kpow(512u); break;
      case 3: f = kpow(1024u); break;      case 4: f = kpow(2048u); break;     case 5: f = kpow(4096u); break;
      case 6: f = kpow(8192u); break;      case 7: f = kpow(16384u); break;    case 8: f = kpow(32768u); break;
      case 9: f = kpow(65536u); break;     default: f = kpow(131072u); break;
    }
    if (m & (1u << b)) r *= f;
  }
  return r;
}

// One warp per segment (warp w: segment w / n_req of request w % n_req).  All segments before the warp's own are full,
// so the true state before segment s is c_s = K^(128 s) c_0 + sum_{j<s} K^(128 (s-1-j)) E_j: one term per lane and a
// warp sum; then the segment's local states become keys.  The warp of a request's last segment also writes chain_out.
__global__ void __launch_bounds__(256) hash_fixup_kernel(const int64_t* __restrict__ blk_off, uint32_t n_req, uint32_t max_seg,
                                                         unsigned long long* __restrict__ keys, const unsigned long long* __restrict__ seg_end,
                                                         const unsigned long long* __restrict__ chain_in, unsigned long long* __restrict__ chain_out) {
  const int lane = threadIdx.x & 31;
  const uint32_t warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
  const unsigned long long kp = kpow_small(lane + 1);                 // K^(lane+1)
  const uint32_t total = n_req * max_seg;
  for (uint32_t w = warp0; w < total; w += n_warps) {
    const uint32_t r = w % n_req, sg = w / n_req;
    const int64_t o = blk_off[r], nb = blk_off[r + 1] - o;
    const int64_t b0 = (int64_t)sg * K1_SEG;
    const unsigned long long c0 = chain_in ? chain_in[r] : H_S0;
    if (nb == 0) { if (sg == 0 && lane == 0 && chain_out) chain_out[r] = c0; continue; }
    if (b0 >= nb) continue;
    unsigned long long part = 0;
    for (uint32_t jb = 0; jb < sg; jb += 32) {
      const uint32_t jj = jb + (uint32_t)lane;
      if (jj < sg) part += kpow_seg(sg - 1 - jj) * seg_end[(size_t)r * max_seg + jj];
    }
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) part += shfl_xor64(part, d);
    const unsigned long long carry = kpow_seg(sg) * c0 + part;        // the state before this segment's first block
    const int len = (int)min((int64_t)K1_SEG, nb - b0);
    unsigned long long kr = kp;                                        // K^(32 it + lane + 1)
    unsigned long long last = 0;
#pragma unroll
    for (int it = 0; it < K1_SEG / 32; ++it) {
      const int i = 32 * it + lane;
      if (i < len) {
        const int64_t at = o + (nb - 1 - (b0 + i));
        const unsigned long long st = keys[at] + kr * carry;
        keys[at] = finalize_key(st);
        if (i == len - 1) last = st;
      }
      kr *= kpow(32);
    }
    if (b0 + len == nb && chain_out) {                                 // the request's last segment: its end state goes out
      const int src = (len - 1) & 31;
      last = shfl64(last, src);
      if (lane == 0) chain_out[r] = last;
    }
  }
}

// the last thing on the stream after a hashing launch: the ticket returns to 0 for the next launch
__global__ void reset_ticket_kernel(uint32_t* ticket) { *ticket = 0; }

__global__ void fill_u64_kernel(unsigned long long* p, uint32_t n, unsigned long long v) {
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) p[i] = v;
}

}  // namespace arc
