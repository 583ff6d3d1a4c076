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

// Inclusive warp scan of the affine chain: on return lane l holds sum_{j<=l} K^(l-j) g_j.  sc[d] = K^(2^d) for the lanes
// that take part in step d (lane >= 2^d) and 0 for the others: multiply-adds only, no branch, no select.
struct ScanConsts { unsigned long long c[5]; };
__device__ __forceinline__ ScanConsts scan_consts(int lane) {
  ScanConsts S;
  S.c[0] = lane >= 1 ? kpow(1) : 0ull; S.c[1] = lane >= 2 ? kpow(2) : 0ull; S.c[2] = lane >= 4 ? kpow(4) : 0ull;
  S.c[3] = lane >= 8 ? kpow(8) : 0ull; S.c[4] = lane >= 16 ? kpow(16) : 0ull;
  return S;
}
__device__ __forceinline__ unsigned long long warp_chain_scan(unsigned long long g, const ScanConsts& S) {
  unsigned long long s = g;
  s += S.c[0] * shfl_up64(s, 1);
  s += S.c[1] * shfl_up64(s, 2);
  s += S.c[2] * shfl_up64(s, 4);
  s += S.c[3] * shfl_up64(s, 8);
  s += S.c[4] * shfl_up64(s, 16);
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

// ---------------------------------------------------------------------------------------------------------------------
// Token staging: every warp owns a ring of K1_STAGES shared-memory stages, each holding the 16-byte-aligned cover of one
// round (32 blocks = 2 KB, plus one vector when the request is misaligned).  Lane 0 fills a stage with ONE bulk
// asynchronous copy (cp.async.bulk global -> shared, the 1-D form of TMA; SASS UBLKCP) that signals the stage's mbarrier
// with the byte count; the warp waits on the barrier's phase and hashes from shared memory.  K1_STAGES - 1 rounds are in
// flight while one is hashed, with no load instruction, no address arithmetic and no register buffer in the hashing
// loop.  The copies carry an L2 evict-first policy (the tokens are read once).
constexpr int K1_STAGES = 4;
constexpr int K1_STAGE_BYTES = 2080;                    // 129 vectors of 16 B, rounded up to a multiple of 32
constexpr int K1_WARPS = 8;
constexpr int K1_SMEM_BYTES = K1_WARPS * K1_STAGES * K1_STAGE_BYTES + K1_WARPS * K1_STAGES * 8;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile("{\n\t.reg .pred p;\n\tK1_WAIT:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@!p bra K1_WAIT;\n\t}"
               ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, unsigned long long policy) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(policy) : "memory");
}

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

// Per-warp pipeline state (registers; identical in every lane).
struct WarpPipe {
  uint32_t stage0;      // shared address of this warp's first stage
  uint32_t bar0;        // shared address of this warp's first mbarrier
  uint32_t parity;      // bit k: the phase stage k's barrier completes next
  unsigned long long policy;
};

__device__ __forceinline__ WarpPipe pipe_init(unsigned char* smem, int warp, int lane) {
  WarpPipe W;
  W.stage0 = smem_u32(smem) + (uint32_t)(warp * K1_STAGES * K1_STAGE_BYTES);
  W.bar0 = smem_u32(smem) + (uint32_t)(K1_WARPS * K1_STAGES * K1_STAGE_BYTES + warp * K1_STAGES * 8);
  W.parity = 0;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(W.policy));
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < K1_STAGES; ++k) mbar_init(W.bar0 + 8u * k, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncwarp();
  return W;
}

// Starts the fill of stage k with the n_vec vectors from absolute token index va (tok + va is 16-byte aligned).
__device__ __forceinline__ void pipe_issue(WarpPipe& W, int k, const uint32_t* __restrict__ tok, int64_t va, int n_vec, int lane,
                                           int64_t lo, int64_t hi) {
  const uint32_t dst = W.stage0 + (uint32_t)(k * K1_STAGE_BYTES);
  if (va >= lo && va + 4 * (int64_t)n_vec <= hi) {          // the whole cover is inside the caller's buffer (warp-uniform)
    if (lane == 0) {
      mbar_expect_tx(W.bar0 + 8u * k, 16u * (uint32_t)n_vec);
      bulk_g2s(dst, tok + va, 16u * (uint32_t)n_vec, W.bar0 + 8u * k, W.policy);
    }
  } else {                                                   // an edge of the buffer: words outside it are never touched
    for (int e = lane; e < n_vec; e += 32) {
      const uint4 v = ld_tokens4_guarded(tok, va + 4 * (int64_t)e, lo, hi);
      asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(dst + 16u * e), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
    }
    __syncwarp();
    if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(W.bar0 + 8u * k) : "memory");   // the phase completes as a copy's would
  }
}
__device__ __forceinline__ void pipe_wait(WarpPipe& W, int k) {
  mbar_wait(W.bar0 + 8u * k, (W.parity >> k) & 1u);
  W.parity ^= 1u << k;
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
  return v;
}

struct LaneConsts {
  unsigned long long salt0, salt1;   // (k+1) M C1 for this lane's two words k = 2q, 2q+1 (the salt is folded into the multiply-add)
  unsigned long long kp;             // K^(lane+1)
  int owner;                         // after the transpose-reduce, block i of the round sits in lane `owner` of lane i
  ScanConsts sc;
};
__device__ __forceinline__ LaneConsts lane_consts(int lane) {
  LaneConsts LC;
  const int q = lane & 3;
  LC.salt0 = (unsigned long long)(2 * q + 1) * H_M * H_C1;
  LC.salt1 = (unsigned long long)(2 * q + 2) * H_M * H_C1;
  LC.kp = kpow_small(lane + 1);
  LC.owner = 4 * (lane & 7) + (lane >> 3);
  LC.sc = scan_consts(lane);
  return LC;
}

// Local chain states of one round held in the stage at shared address `st`: lane i returns sum_{j<=i} K^(i-j) g_j over
// the round's blocks (no carry-in); lanes >= cnt contribute g = 0.  s = request misalignment in tokens.  Lane l reads
// vector 32 it + l (conflict-free) and, for a misaligned request, the vector after it: no shuffle realigns anything.
template <int S>
__device__ __forceinline__ unsigned long long round_local_scan(uint32_t st, int cnt, int lane, const LaneConsts& LC) {
  unsigned long long part[4];
#pragma unroll
  for (int it = 0; it < 4; ++it) {
    const uint32_t at = st + 16u * (uint32_t)(it * 32 + lane);
    const uint4 v = lds128(at);
    uint32_t a = v.x, b = v.y, c2 = v.z, d = v.w;
    if (S != 0) {
      const uint4 w = lds128(at + 16u);
      if (S == 1) { a = v.y; b = v.z; c2 = v.w; d = w.x; }
      else if (S == 2) { a = v.z; b = v.w; c2 = w.x; d = w.y; }
      else { a = v.w; b = w.x; c2 = w.y; d = w.z; }
    }
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
  return warp_chain_scan(g, LC.sc);
}

// One run of nbs consecutive blocks starting at absolute token index ts (a request, or a segment of one), hashed by one
// warp through its stage ring.  emit(rb, cnt, st): lane l < cnt holds the chain state st of block rb + l of the run.
// Returns the state after the run's last block.  Everything inside the round loop is 32-bit (nbs < 2^28).
template <int S, typename Emit>
__device__ __forceinline__ unsigned long long hash_run_s(WarpPipe& W, const uint32_t* __restrict__ tok, int64_t lo, int64_t hi,
                                                         int64_t ts, uint32_t nbs, unsigned long long carry, int lane, const LaneConsts& LC,
                                                         Emit emit) {
  constexpr int s = S;                               // tokens of the run's start past a 16-byte boundary (same for every round)
  const int64_t va = ts - s;                         // absolute token index of the aligned cover of round 0
  const uint32_t rounds = (nbs + 31u) >> 5;
  const uint32_t vec_full = (uint32_t)(512 + s + 3) >> 2, vec_last = (16u * (nbs - 32u * (rounds - 1)) + (uint32_t)s + 3u) >> 2;
  // only the first and the last round of a run can reach outside the caller's buffer (the cover's few words before / after)
  const bool head_in = va >= lo, tail_in = va + 512 * (int64_t)(rounds - 1) + 4 * (int64_t)vec_last <= hi;
  const uint32_t* src = tok + va;                    // 16-byte aligned
  auto issue = [&](uint32_t r, int k) {
    const uint32_t nv = (r + 1 == rounds) ? vec_last : vec_full;
    if ((r != 0 || head_in) && (r + 1 != rounds || tail_in)) {
      if (lane == 0) {
        mbar_expect_tx(W.bar0 + 8u * k, 16u * nv);
        bulk_g2s(W.stage0 + (uint32_t)(k * K1_STAGE_BYTES), src + 512u * (size_t)r, 16u * nv, W.bar0 + 8u * k, W.policy);
      }
    } else {
      pipe_issue(W, k, tok, va + 512 * (int64_t)r, (int)nv, lane, lo, hi);
    }
  };
  uint32_t issued = 0;
  for (; issued < rounds && issued < (uint32_t)(K1_STAGES - 1); ++issued) issue(issued, (int)issued);
  int k = 0, kn = K1_STAGES - 1;                     // stage of the round being hashed / of the next round to issue
  for (uint32_t r = 0; r < rounds; ++r) {
    if (issued < rounds) {                           // the stage hashed last round is free: every lane has its words in registers
      issue(issued, kn);
      ++issued;
      kn = (kn + 1 == K1_STAGES) ? 0 : kn + 1;
    }
    pipe_wait(W, k);
    const int cnt = (int)min(32u, nbs - 32u * r);
    const unsigned long long st = round_local_scan<S>(W.stage0 + (uint32_t)(k * K1_STAGE_BYTES), cnt, lane, LC) + LC.kp * carry;
    emit(32u * r, cnt, st);
    carry = shfl64(st, cnt - 1);
    __syncwarp();                                    // all lanes are done with stage k before it is filled again
    k = (k + 1 == K1_STAGES) ? 0 : k + 1;
  }
  return carry;
}

// The misalignment is a property of the run: four copies of the round loop, none of them with a select or a branch on it.
template <typename Emit>
__device__ __forceinline__ unsigned long long hash_run(WarpPipe& W, const uint32_t* __restrict__ tok, int base_mis, int64_t lo, int64_t hi,
                                                       int64_t ts, uint32_t nbs, unsigned long long carry, int lane, const LaneConsts& LC,
                                                       Emit emit) {
  switch ((int)((base_mis + ts) & 3)) {
    case 0: return hash_run_s<0>(W, tok, lo, hi, ts, nbs, carry, lane, LC, emit);
    case 1: return hash_run_s<1>(W, tok, lo, hi, ts, nbs, carry, lane, LC, emit);
    case 2: return hash_run_s<2>(W, tok, lo, hi, ts, nbs, carry, lane, LC, emit);
    default: return hash_run_s<3>(W, tok, lo, hi, ts, nbs, carry, lane, LC, emit);
  }
}

// Length classes for the ticket passes: requests of at least K1_CLASS_MIN[c] blocks are started in pass c, so the
// longest chains start first and the short requests fill the tail of the launch (longest-processing-time-first).
constexpr int K1_PASSES = 4;
__device__ __forceinline__ int k1_class(int64_t nb) { return nb >= 1024 ? 0 : nb >= 384 ? 1 : nb >= 128 ? 2 : 3; }

// The last warp of a launch to leave puts the work ticket back to 0 (ticket[0] = ticket, ticket[1] = warps that left):
// no reset kernel, and the ticket of a handle or of a caller's scratch is always 0 between launches.
__device__ __forceinline__ void k1_leave(uint32_t* ticket, int lane) {
  if (lane == 0) {
    __threadfence();
    const uint32_t n_warps = (gridDim.x * blockDim.x) >> 5;
    if (atomicAdd(ticket + 1, 1u) == n_warps - 1) { ticket[1] = 0; __threadfence(); ticket[0] = 0; }
  }
}

// ACCESS_ORDER = true writes keys at blk_off[r] + (nb-1-i) (the order K3 consumes, R2); false writes natural
// order (arc_hash_blocks).  ticket: two device words, 0 at launch (see k1_leave); it runs over K1_PASSES * n_req values:
// ticket t is request t % n_req in pass t / n_req.
// CHAIN = true reads each request's initial H4 state from chain_in (NULL = S0) and writes its final state to chain_out
// (arc_step / arc_step_resume); false is the stateless arc_hash_blocks, which pays nothing for it.
// ACAP > 0: the offsets come as the kernel argument `arg` (steps of up to ACAP requests: a launch costs less than the copy
// engine's round trip, and the step's first kernel waits for nothing) and CTA 0 also stores them to offsets_g / blk_off_g
// for the kernels that follow; ACAP = 0: they are read from those arrays.  Two argument sizes are built: 253 requests
// (4 KB, the classic parameter limit) and 1,999 requests (32 KB, the large-parameter limit of CUDA 12.1+ on sm_70+).
constexpr uint32_t K1_INLINE_SMALL = 253, K1_INLINE_LARGE = 1999;
template <int CAP> struct OffsetsArgT { long long v[2 * (CAP + 1)]; };   // offsets[n_req + 1] then blk_off[n_req + 1]
constexpr uint32_t K1_TICKET_BATCH = 2;

template <bool ACCESS_ORDER, bool CHAIN, int ACAP>
__global__ void __launch_bounds__(256, 3) hash_blocks_kernel(const int32_t* __restrict__ tokens, int64_t* __restrict__ offsets_g,
                                                         int64_t* __restrict__ blk_off_g, uint32_t n_req,
                                                         unsigned long long* __restrict__ keys, uint32_t* __restrict__ ticket,
                                                         const unsigned long long* __restrict__ chain_in,
                                                         unsigned long long* __restrict__ chain_out,
                                                         const __grid_constant__ OffsetsArgT<ACAP> arg) {
  extern __shared__ __align__(128) unsigned char k1_smem[];
  const int lane = threadIdx.x & 31;
  constexpr bool ARG = ACAP > 0;
  const long long* offsets = ARG ? arg.v : reinterpret_cast<const long long*>(offsets_g);
  const long long* blk_off = ARG ? arg.v + (n_req + 1) : reinterpret_cast<const long long*>(blk_off_g);
  if (ARG && blockIdx.x == 0)
    for (uint32_t i = threadIdx.x; i <= n_req; i += blockDim.x) { offsets_g[i] = arg.v[i]; blk_off_g[i] = arg.v[n_req + 1 + i]; }
  const uint32_t* tok = reinterpret_cast<const uint32_t*>(tokens);
  const int64_t lo = offsets[0], hi = offsets[n_req];
  const LaneConsts LC = lane_consts(lane);
  WarpPipe W = pipe_init(k1_smem, threadIdx.x >> 5, lane);
  const int base_mis = (int)((reinterpret_cast<uintptr_t>(tok) >> 2) & 3);   // tokens of the buffer start past a 16-byte boundary
  const unsigned long long total = (unsigned long long)K1_PASSES * n_req;

  for (;;) {
    // K1_TICKET_BATCH tickets per atomic: lane l < batch examines ticket t0 + l, the warp then hashes the ones that belong to the pass
    uint32_t t0 = 0;
    if (lane == 0) t0 = atomicAdd(ticket, K1_TICKET_BATCH);
    t0 = __shfl_sync(0xFFFFFFFFu, t0, 0);
    if (t0 >= total) break;
    const unsigned long long t = (unsigned long long)t0 + lane;
    bool mine = false;
    uint32_t my_r = 0;
    if (t < total && (uint32_t)lane < K1_TICKET_BATCH) {
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
      const unsigned long long c0 = (CHAIN && chain_in) ? chain_in[r] : H_S0;     // the H4 state before block 0 (a prompt: S0)
      unsigned long long* out = keys + (ACCESS_ORDER ? (o + nb - 1 - lane) : (o + lane));    // this lane's key of round 0
      const unsigned long long end = hash_run(W, tok, base_mis, lo, hi, offsets[r], (uint32_t)nb, c0, lane, LC,
        [&](uint32_t rb, int cnt, unsigned long long st) {
          if (lane < cnt) { if (ACCESS_ORDER) *(out - rb) = finalize_key(st); else out[rb] = finalize_key(st); }
        });
      if (CHAIN && lane == 0) chain_out[r] = end;                                 // the state a continuation of this sequence starts from
    }
  }
  k1_leave(ticket, lane);
}

// ---------------------------------------------------------------------------------------------------------------------
// The stateless bulk form (arc_hash_blocks): the host, which validates the offsets anyway, hands the kernel a WORK LIST -
// one item per request with at least one full block, longest length class first (the same longest-processing-time-first
// order the ticket passes above produce, without the tickets that find nothing) - and a warp always knows its NEXT
// item: the ticket for the item after next is requested, and the next item is loaded, while the current one is hashed,
// so neither the atomic nor the metadata load is ever waited for.  Keys in natural order, no chain states.
struct __align__(16) HashItem { long long tok_off; long long key_off; uint32_t n_blocks; uint32_t reserved[3]; };   // 32 bytes = arc_hash_item (arc.h)

__global__ void __launch_bounds__(256, 3) hash_items_kernel(const int32_t* __restrict__ tokens, const HashItem* __restrict__ items, uint32_t n_items,
                                                            int64_t lo, int64_t hi, unsigned long long* __restrict__ keys, uint32_t* __restrict__ ticket) {
  extern __shared__ __align__(128) unsigned char k1_smem[];
  const int lane = threadIdx.x & 31;
  const uint32_t* tok = reinterpret_cast<const uint32_t*>(tokens);
  const LaneConsts LC = lane_consts(lane);
  WarpPipe W = pipe_init(k1_smem, threadIdx.x >> 5, lane);
  const int base_mis = (int)((reinterpret_cast<uintptr_t>(tok) >> 2) & 3);
  uint32_t t_req = 0;                                   // lane 0: the ticket last requested
  if (lane == 0) t_req = atomicAdd(ticket, 1u);
  uint32_t t = __shfl_sync(0xFFFFFFFFu, t_req, 0);
  if (t < n_items) {
    const uint4* ip = reinterpret_cast<const uint4*>(items + t);     // 32-byte items: two aligned 16-byte loads
    uint4 a = __ldg(ip);
    uint4 b = __ldg(ip + 1);
    if (lane == 0) t_req = atomicAdd(ticket, 1u);
    for (;;) {
      const long long tok_off = (long long)((unsigned long long)a.x | ((unsigned long long)a.y << 32));
      const long long key_off = (long long)((unsigned long long)a.z | ((unsigned long long)a.w << 32));
      const uint32_t nb = b.x;
      // the item after this one: its ticket was requested an item ago; its words are on their way while this one is hashed
      const uint32_t tn = __shfl_sync(0xFFFFFFFFu, t_req, 0);
      uint4 na = make_uint4(0, 0, 0, 0), nbv = make_uint4(0, 0, 0, 0);
      if (tn < n_items) {
        const uint4* np = reinterpret_cast<const uint4*>(items + tn);
        na = __ldg(np);
        nbv = __ldg(np + 1);
        if (lane == 0) t_req = atomicAdd(ticket, 1u);
      }
      unsigned long long* out = keys + (key_off + lane);
      hash_run(W, tok, base_mis, lo, hi, tok_off, nb, H_S0, lane, LC,
        [&](uint32_t rb, int cnt, unsigned long long st) { if (lane < cnt) out[rb] = finalize_key(st); });
      if (tn >= n_items) break;
      a = na; b = nbv;
    }
  }
  k1_leave(ticket, lane);
}

// ---------------------------------------------------------------------------------------------------------------------
// In-step hashing of steps with FEW requests: one warp per request leaves the step waiting for its longest request (a
// 1,000-block document is 32 dependent rounds).  H4 is affine, so a request is cut into segments of K1_SEG blocks that are
// scanned independently from a zero carry (hash_segments_kernel: one warp per segment, the same staging and scans as
// above) and put together afterwards (hash_fixup_kernel): with c_s the true state before segment s and E_s the local end
// state of the segment, c_{s+1} = E_s + K^len_s c_s, and block i of the segment has state local_i + K^(i+1) c_s.
constexpr int K1_SEG = 128;

// states[] gets the LOCAL states, in access order (index blk_off[r] + nb - 1 - i); seg_end[r * max_seg + s] = E_s.
template <int ACAP>
__global__ void __launch_bounds__(256, 3) hash_segments_kernel(const int32_t* __restrict__ tokens, int64_t* __restrict__ offsets_g,
                                                               int64_t* __restrict__ blk_off_g, uint32_t n_req, uint32_t max_seg,
                                                               unsigned long long* __restrict__ states,
                                                               unsigned long long* __restrict__ seg_end, uint32_t* __restrict__ ticket,
                                                               const __grid_constant__ OffsetsArgT<ACAP> arg) {
  extern __shared__ __align__(128) unsigned char k1_smem[];
  const int lane = threadIdx.x & 31;
  constexpr bool ARG = ACAP > 0;
  const long long* offsets = ARG ? arg.v : reinterpret_cast<const long long*>(offsets_g);
  const long long* blk_off = ARG ? arg.v + (n_req + 1) : reinterpret_cast<const long long*>(blk_off_g);
  if (ARG && blockIdx.x == 0)
    for (uint32_t i = threadIdx.x; i <= n_req; i += blockDim.x) { offsets_g[i] = arg.v[i]; blk_off_g[i] = arg.v[n_req + 1 + i]; }
  const uint32_t* tok = reinterpret_cast<const uint32_t*>(tokens);
  const int64_t lo = offsets[0], hi = offsets[n_req];
  const LaneConsts LC = lane_consts(lane);
  WarpPipe W = pipe_init(k1_smem, threadIdx.x >> 5, lane);
  const int base_mis = (int)((reinterpret_cast<uintptr_t>(tok) >> 2) & 3);
  const unsigned long long total = (unsigned long long)max_seg * n_req;
  for (;;) {
    uint32_t t0 = 0;
    if (lane == 0) t0 = atomicAdd(ticket, 1u);                      // one segment per ticket: segments are equal pieces of work
    t0 = __shfl_sync(0xFFFFFFFFu, t0, 0);
    if (t0 >= total) break;
    const uint32_t r = t0 % n_req, sg = t0 / n_req;                 // ticket t = segment t / n_req of request t % n_req
    const int64_t o = blk_off[r], nb = blk_off[r + 1] - o;
    const int64_t b0 = (int64_t)sg * K1_SEG;
    if (b0 >= nb) continue;
    const int64_t nbs = min((int64_t)K1_SEG, nb - b0);
    unsigned long long* out = states + (o + nb - 1 - b0 - lane);
    const unsigned long long end = hash_run(W, tok, base_mis, lo, hi, offsets[r] + 16 * b0, (uint32_t)nbs, 0ull, lane, LC,
      [&](uint32_t rb, int cnt, unsigned long long st) {
        if (lane < cnt) *(out - rb) = st;
      });
    if (lane == 0) seg_end[(size_t)r * max_seg + sg] = end;
  }
  k1_leave(ticket, lane);
}

// K^(2^LOG2 m): square-and-multiply over the bits of m (m < 2^11); the factors K^(2^(LOG2 + b)) are compile-time constants
template <int LOG2>
__device__ __forceinline__ unsigned long long kpow_segT(uint32_t m) {
  unsigned long long r = 1;
#pragma unroll
  for (int b = 0; b < 11; ++b) {
    const unsigned long long f = kpow(1u << (LOG2 + b));
    if (m & (1u << b)) r *= f;
  }
  return r;
}
__device__ __forceinline__ unsigned long long kpow_seg(uint32_t m) { return kpow_segT<7>(m); }   // segments of K1_SEG = 128 blocks

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

// Prefix-affinity routing: destination shard of every request = (key of its FIRST block >> 33) mod
// world, 0 for a request without a full block.  One thread per request: 16 tokens, H3, one step of H4 from S0, H5.
__global__ void __launch_bounds__(256) route_first_block_kernel(const int32_t* __restrict__ tokens, const int64_t* __restrict__ offsets, uint32_t n_req,
                                                                uint32_t world, int32_t* __restrict__ dst) {
  const uint32_t* tok = reinterpret_cast<const uint32_t*>(tokens);
  for (uint32_t r = blockIdx.x * blockDim.x + threadIdx.x; r < n_req; r += gridDim.x * blockDim.x) {
    const int64_t a = offsets[r], len = offsets[r + 1] - a;
    int32_t d = 0;
    if (len >= 16) {
      unsigned long long g = 0;
#pragma unroll
      for (int k = 0; k < 8; ++k) g += hash_word(__ldg(tok + a + 2 * k), __ldg(tok + a + 2 * k + 1), (unsigned long long)(k + 1) * H_M);
      const unsigned long long key = finalize_key(H_S0 * H_K + g);
      d = (int32_t)((key >> 33) % world);
    }
    dst[r] = d;
  }
}

__global__ void fill_u64_kernel(unsigned long long* p, uint32_t n, unsigned long long v) {
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) p[i] = v;
}

}  // namespace arc
