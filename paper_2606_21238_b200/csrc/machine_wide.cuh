// K3, wide form: one CTA consumes the step's accesses in the fixed order R2, a window of up to 128 accesses at a time.
// Two forms of one source (template parameter PIPE): the plain form (8 warps: owners 0..3, scanners 4..7; every owner warp
// rolls the counters of its window itself; also the third phase of the one-launch kernel) and the pipelined form (12
// warps: four ROLLER warps work out the recurrence and every access's plan one window ahead of the owners, see
// wide_roller; named barriers instead of __syncthreads).
// Same equivalence argument as machine_batched.cuh; what changes is who does what:
//   * thread g = 32 w + lane owns access g of the window: it fetches the node record, checks the window's cut
//     conditions for its access, and applies its access;
//   * the counter recurrence (wide_roll: 32 accesses at a time, phases inlined) is run redundantly and identically by all four
//     warps on the class masks exchanged through shared memory, so no decision is ever broadcast;
//   * warp w scans the LRU end of list w + 1 (T1, T2, B1, B2): 128 self-validating ring entries per round;
//   * latencies (node fetch, ring fetch, barriers) are paid once per 128 accesses instead of once per 32.
// The same node twice in a window is possible only through a 64-bit key collision inside one request (windows never
// cross a request boundary).  It is found exactly and for free: every owner stamps its node with the window's number by
// an atomic EXCHANGE (node_stamp[]; normally one window ahead, together with the speculative record load, so the
// latency is hidden); two threads of one window that own the same node exchange the same number, and whichever comes
// second in the atomic's order reads it back.  Only then (next to never) does the window compare its node ids pairwise
// and cut itself before the second occurrence, as the 32-wide machine does with __match_any_sync.
#pragma once
#include "machine_batched.cuh"

namespace arc {

constexpr int WIDE_WARPS = 4;
constexpr int WIDE_W = 32 * WIDE_WARPS;      // accesses per window
constexpr int WIDE_IDS = 512;                // node-id staging ring: the current window, the next one and what is in flight

__device__ __forceinline__ void cp_async_u32(uint32_t* smem_dst, const uint32_t* gmem_src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Named barriers of the pipelined form (PIPE): the owners and scanners meet on barrier 1 (256 threads) where the plain form
// uses __syncthreads; the roller warps are handed their work on barrier 2 and hand it back on barrier 3 (128 owners +
// 128 roller threads: one side arrives, the other waits).
__device__ __forceinline__ void bar_sync_n(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive_n(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
constexpr int BAR_CTA = 1, BAR_REQ = 2, BAR_DONE = 3;
constexpr int ROLL_PARTIES = 2 * 32 * WIDE_WARPS;          // the owners and as many roller threads
template <bool PIPE>
__device__ __forceinline__ void cta_sync() {
  if (PIPE) bar_sync_n(BAR_CTA, 2 * WIDE_W); else __syncthreads();
}
template <bool PIPE>
__device__ __forceinline__ bool cta_or(bool pred) {
  if (!PIPE) return __syncthreads_or(pred) != 0;
  uint32_t r;
  asm volatile("{\n\t.reg .pred p, q;\n\tsetp.ne.u32 q, %1, 0;\n\tbar.red.or.pred p, 1, 256, q;\n\tselp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(r) : "r"((uint32_t)pred) : "memory");
  return r != 0;
}
static_assert(2 * WIDE_W == 256, "the reducing barrier above spells the thread count out");

// What the owners hand the roller warp (one request outstanding at a time) and what comes back (two buffers, by the
// request's parity: the scanners and owners of a window read one while the next request's result goes into the other).
struct RollReq {
  uint32_t m[4][WIDE_WARPS];                 // class masks m0, m1, m2, me per chunk
  int32_t st[8];                             // t1, t2, b1, b2, p, next_fresh, elig1, elig2 before the window
  int32_t k;
  uint32_t quit;
};
struct RollRes {
  uint4 plan[WIDE_W];                        // what each access does, as ranks inside the window (WidePlan, packed)
  int32_t st[8];                             // the same eight after the window
  uint32_t need[5];                          // victims / drops the window takes per list
  uint32_t pt1, g1, nh, ev;                  // pushes to T1 and to B1, allocations, evictions of the window
  uint32_t err, phases;
  uint32_t all_hit, badnode, h1, e1d, e2d;   // the window is hits only; a FREE node is among its nodes; if hits only: hits in T1,
                                             // hits on entries of T1 / T2 that were still evictable
};

struct WideShared {
  uint32_t m[4][WIDE_WARPS];                 // m0, m1, m2, me per chunk
  uint32_t reload[WIDE_WARPS];               // PIPE: owners that could not use their speculative record
  uint32_t ctl_prov, ctl_par;                // PIPE: a result rolled ahead for this window exists, and its buffer
  RollReq req;
  RollRes res[2];
  uint32_t bad[WIDE_WARPS];
  uint32_t twin[WIDE_WARPS], twinc[WIDE_WARPS];   // accesses that repeat an earlier node of the window; threads whose stamp exchange says "maybe"
  uint32_t twin_k;                           // the window's size after a twin cut (written between the two twin barriers only)
  uint32_t found[5], more[5], need[5];       // scanners: live entries found so far, whether the list has more to scan; owners: victims needed
  uint32_t ctl_done, ctl_k, ctl_head[5], ctl_limit[5]; // published by thread 0 before a window's first barrier, read by the scanner warps
  uint32_t red[WIDE_WARPS][5];               // per-warp class counts, summed by thread 0 at the end
  uint32_t ids[WIDE_IDS];                    // node ids of the upcoming accesses: access a sits in ids[a % WIDE_IDS] (filled by cp.async)
  uint4 vic[5][WIDE_W];                      // per list: entries found from the LRU end {node, block, -, position}
  SerialCtx ctx;                             // the machine state after a by-the-book access done by warp 0
};

// Rank of a thread's access inside a window-wide mask (four 32-bit chunks): the set bits below it.  lm[] is per thread
// and fixed for the kernel: all ones for the chunks below its own, the bits below its lane for its own chunk, zero above;
// me[] has the thread's own bit in its own chunk.  No selects on the (run-time) warp index.
__device__ __forceinline__ uint32_t wide_rank(const uint32_t (&mask)[WIDE_WARPS], const uint32_t (&lm)[WIDE_WARPS]) {
  uint32_t r = 0;
#pragma unroll
  for (int u = 0; u < WIDE_WARPS; ++u) r += (uint32_t)__popc(mask[u] & lm[u]);
  return r;
}
__device__ __forceinline__ bool wide_has(const uint32_t (&mask)[WIDE_WARPS], const uint32_t (&me)[WIDE_WARPS]) {
  uint32_t r = 0;
#pragma unroll
  for (int u = 0; u < WIDE_WARPS; ++u) r |= mask[u] & me[u];
  return r != 0;
}
__device__ __forceinline__ uint32_t wide_count(const uint32_t (&mask)[WIDE_WARPS]) {
  uint32_t r = 0;
#pragma unroll
  for (int u = 0; u < WIDE_WARPS; ++u) r += (uint32_t)__popc(mask[u]);
  return r;
}

// window numbers: 31 bits, never 0 (0 = never stamped)
__device__ __forceinline__ uint32_t wide_next_seq(uint32_t s) { s = (s + 1u) & 0x7FFFFFFFu; return s ? s : 1u; }

// What a thread keeps of the decisions of a roll: not the masks of all four chunks (the chunk loop is not unrolled, so
// they would be reached by chains of predicated moves: 250 of the 720 instructions a roller warp spent per window) but,
// for each of the six decision masks, exactly what its plan and the window's counts need - the mask of ITS chunk, the
// bits set in the chunks below it, the bits set in the whole window - accumulated chunk by chunk while the roll goes on.
enum : int { F_S0 = 0,                       // evicts T1's LRU entry (with or without a ghost)
             F_S2,                           // evicts T2's LRU entry (it becomes a ghost of B2)
             F_G1,                           // its T1 victim becomes a ghost of B1
             F_D1, F_D2,                     // drops the LRU ghost of B1 / B2
             F_FM,                           // takes a fresh block id
             F_COUNT };
struct WideDecisions {
  uint32_t mine[F_COUNT], below[F_COUNT], total[F_COUNT];
  int32_t my_p;
  Roll R;                                    // state after the window
};
// chunk u's decision masks join the accumulators of a thread whose access is in chunk `warp`
__device__ __forceinline__ void wide_acc(WideDecisions& D, int u, int warp, uint32_t s0, uint32_t s1, uint32_t d1, uint32_t d2, uint32_t fm) {
  const uint32_t f[F_COUNT] = {s0, s1 & ~s0, s0 & ~s1, d1, d2, fm};
#pragma unroll
  for (int i = 0; i < F_COUNT; ++i) {
    const uint32_t pc = (uint32_t)__popc(f[i]);
    D.total[i] += pc;
    if (u < warp) D.below[i] += pc;
    if (u == warp) D.mine[i] = f[i];
  }
}

// The recurrence over the first k accesses of the window, chunk by chunk (every warp computes the same thing).
// Sm: the class masks m0, m1, m2, me per chunk (shared memory); warp = the chunk this thread's access is in.
template <bool lru>
__device__ __forceinline__ void wide_roll(WideDecisions& D, const Roll& R0, int32_t c, const uint32_t (*Sm)[WIDE_WARPS], int k,
                                          int warp, int lane) {
  D.R = R0;
  D.my_p = R0.p;
  {
    // The commonest whole window of a cache in steady state: every access a miss, case 4A (t1 + b1 = c) with T1 above its
    // target and enough evictable entries for all of them: each miss drops B1's LRU ghost and evicts T1's LRU entry, no
    // counter moves (phase_miss's first case, for the window instead of chunk by chunk).
    uint32_t any = 0;
#pragma unroll
    for (int u = 0; u < WIDE_WARPS; ++u) any |= (Sm[0][u] | Sm[1][u] | Sm[2][u]) & bits_from(0, min(32, max(0, k - 32 * u)));
    Roll& R = D.R;
    if (!lru && any == 0 && R.t1 + R.t2 == c && R.t1 + R.b1 == c && R.t1 < c && R.t1 > R.p && R.e1 >= k) {
      // every access evicts from T1 into B1 and drops B1's LRU ghost
      const uint32_t mine = bits_from(0, min(32, max(0, k - 32 * warp))), below = (uint32_t)min(k, 32 * warp);
#pragma unroll
      for (int i = 0; i < F_COUNT; ++i) {
        const bool on = (i == F_S0 || i == F_G1 || i == F_D1);
        D.mine[i] = on ? mine : 0u; D.below[i] = on ? below : 0u; D.total[i] = on ? (uint32_t)k : 0u;
      }
      R.e1 -= k;
      R.phases++;
      return;
    }
  }
  // ONE copy of the chunk body, looped over (not unrolled): the body with its inlined phases is the largest piece of code of
  // the kernel, and four copies each run once per window are four times the instruction-cache footprint of one copy run
  // four times.
#pragma unroll
  for (int i = 0; i < F_COUNT; ++i) D.mine[i] = D.below[i] = D.total[i] = 0;
#pragma unroll 1
  for (int u = 0; u < WIDE_WARPS; ++u) {
    const int ku = min(32, max(0, k - 32 * u));
    if (ku > 0) {
      const uint32_t km = bits_from(0, ku);
      const uint32_t m0 = Sm[0][u] & km, m1 = Sm[1][u] & km, m2 = Sm[2][u] & km, me = Sm[3][u] & km;
      Roll& R = D.R;
      const uint32_t hits = lru ? (m0 & ~m1 & ~m2) : ((m0 ^ m1) & ~m2);
      const uint32_t absent = ~(m0 | m1 | m2) & km, gb1 = m0 & m1 & ~m2, gb2 = m2 & ~m0 & ~m1;
      if (hits == km) {
        // the chunk is all hits: T1 entries move to T2 (ARC); evictable entries stop being so
        if (!lru) { const int32_t h1 = __popc(m0); R.t1 -= h1; R.t2 += h1; R.e2 -= __popc(me & m1); }
        R.e1 -= __popc(me & m0);
        R.s0 = R.s1 = R.d1 = R.d2 = R.fm = 0; R.my_p = R.p;
      } else {
        // anything else: run after run, the phases inlined here (no call, no copy of the roll state); a chunk that is one
        // run of misses or of ghost hits skips the run detection
        R.s0 = R.s1 = R.d1 = R.d2 = R.fm = 0; R.my_p = R.p;
        const bool pure = absent == km || (!lru && (gb1 == km || gb2 == km));
        const uint32_t li_pure = (absent == km) ? L_ABSENT : ((gb1 == km) ? L_B1 : L_B2);
        const int my = (u == warp) ? lane : 64;
        for (int i = 0; i < ku;) {
          R.phases++;
          uint32_t li = li_pure;
          int m = ku - i;
          if (!pure) {
            li = ((m0 >> i) & 1u) | (((m1 >> i) & 1u) << 1) | (((m2 >> i) & 1u) << 2);
            // the run of accesses with this same list code (ARC: hits in T1 and in T2 form one run)
            const bool hit_run = !lru && (li == L_T1 || li == L_T2);
            const uint32_t same = (hit_run ? hits : (((li & 1u) ? m0 : ~m0) & ((li & 2u) ? m1 : ~m1) & ((li & 4u) ? m2 : ~m2))) & km;
            const uint32_t brk = ~(same >> i);
            m = brk ? (__ffs(brk) - 1) : 32;
          }
          int n;
          if (li == L_T1 || (!lru && li == L_T2)) {             // hits: T1 entries move to T2 (ARC); evictable entries stop being so
            n = m;
            const uint32_t run = bits_from(i, n);
            if (!lru) { const int32_t h1 = __popc(m0 & run); R.t1 -= h1; R.t2 += h1; R.e2 -= __popc(me & m1 & run); }
            R.e1 -= __popc(me & m0 & run);
          } else if (li == L_ABSENT || lru) {
            n = lru ? phase_lru_miss(R, c, i, m) : phase_miss(R, c, i, m);
          } else {
            n = phase_ghost(R, c, li, i, m, my);
          }
          i += n;
        }
      }
      if (hits != km) wide_acc(D, u, warp, D.R.s0, D.R.s1, D.R.d1, D.R.d2, D.R.fm);   // (a chunk of hits decides nothing)
      if (u == warp) D.my_p = D.R.my_p;
    }
  }
}

// What one access of a general window does, as ranks inside the window: everything the decision masks say about it.
struct WidePlan {
  uint32_t src;                              // eviction source: 0 none, 1 T1 -> B1, 2 T2 -> B2, 3 T1 without a ghost
  bool d1, d2, fm;                           // drops the LRU ghost of B1 / B2; takes a fresh block id
  uint32_t vic_rank;                         // its victim is the vic_rank-th live entry from the LRU end of T1 (src 1, 3) / T2 (src 2)
  uint32_t gpush_rank;                       // ... and becomes the gpush_rank-th ghost the window appends to B1 (src 1) / B2 (src 2)
  uint32_t drop_rank, fresh_rank;            // the ghost it drops; the fresh id it takes
  uint32_t push_rank;                        // its own node is the push_rank-th the window appends to T1 (ABSENT; LRU: all) / T2
  uint32_t alloc_rank, evict_rank;           // positions in the step's alloc_ids / evict_ids, counted from the window's first
  int32_t p;                                 // p after the access
};
struct WideCounts { uint32_t need[5]; uint32_t pt1, g1, nh, ev; };

__device__ __forceinline__ uint4 plan_pack(const WidePlan& A) {
  return make_uint4(A.src | ((uint32_t)A.d1 << 2) | ((uint32_t)A.d2 << 3) | ((uint32_t)A.fm << 4) | (A.vic_rank << 8) | (A.gpush_rank << 16) | (A.drop_rank << 24),
                    A.push_rank | (A.alloc_rank << 8) | (A.evict_rank << 16) | (A.fresh_rank << 24), (uint32_t)A.p, 0u);
}
__device__ __forceinline__ WidePlan plan_unpack(const uint4 v) {
  WidePlan A;
  A.src = v.x & 3u; A.d1 = (v.x >> 2) & 1u; A.d2 = (v.x >> 3) & 1u; A.fm = (v.x >> 4) & 1u;
  A.vic_rank = (v.x >> 8) & 0xFFu; A.gpush_rank = (v.x >> 16) & 0xFFu; A.drop_rank = v.x >> 24;
  A.push_rank = v.y & 0xFFu; A.alloc_rank = (v.y >> 8) & 0xFFu; A.evict_rank = (v.y >> 16) & 0xFFu; A.fresh_rank = v.y >> 24;
  A.p = (int32_t)v.z;
  return A;
}

// The plan of this thread's access and the window's counts from what the roll over k accesses accumulated (D).  Sm: the
// class masks the roll used; lm / me: the thread's rank masks (wide_rank / wide_has); g: its index in the window.  Ranks in
// the decision masks come from the accumulators; the pushes to T1 and to T2 partition the window, so do hits and
// allocations, and an eviction comes either from T1 or from T2: two ranks are counted in the class masks, the rest follows.
template <bool lru>
__device__ __forceinline__ void wide_make_plan(WidePlan& A, WideCounts& N, const WideDecisions& D, const uint32_t (*Sm)[WIDE_WARPS], int k,
                                               uint32_t g, const uint32_t (&lm)[WIDE_WARPS], const uint32_t (&me)[WIDE_WARPS]) {
  uint32_t PT1[WIDE_WARPS], HIT[WIDE_WARPS];
#pragma unroll
  for (int u = 0; u < WIDE_WARPS; ++u) {
    const uint32_t km = bits_from(0, min(32, max(0, k - 32 * u)));
    const uint32_t m0 = Sm[0][u], m1 = Sm[1][u], m2 = Sm[2][u];
    PT1[u] = lru ? km : (~(m0 | m1 | m2) & km);                        // ABSENT nodes enter T1 (LRU: everything)
    HIT[u] = (lru ? (m0 & ~m1 & ~m2) : ((m0 ^ m1) & ~m2)) & km;
  }
  const uint32_t bit = 1u << (g & 31u), lt = bit - 1u;
  uint32_t rk[F_COUNT];
  bool on[F_COUNT];
#pragma unroll
  for (int i = 0; i < F_COUNT; ++i) { on[i] = (D.mine[i] & bit) != 0; rk[i] = D.below[i] + (uint32_t)__popc(D.mine[i] & lt); }
  A.src = on[F_S2] ? 2u : (on[F_S0] ? (on[F_G1] ? 1u : 3u) : 0u);
  A.d1 = on[F_D1]; A.d2 = on[F_D2]; A.fm = on[F_FM];
  A.vic_rank = on[F_S2] ? rk[F_S2] : rk[F_S0];
  A.gpush_rank = on[F_G1] ? rk[F_G1] : rk[F_S2];
  A.drop_rank = on[F_D1] ? rk[F_D1] : rk[F_D2];
  A.fresh_rank = rk[F_FM];
  const uint32_t r_pt1 = wide_rank(PT1, lm);
  A.push_rank = wide_has(PT1, me) ? r_pt1 : g - r_pt1;
  A.alloc_rank = g - wide_rank(HIT, lm);
  A.evict_rank = rk[F_S0] + rk[F_S2];
  A.p = D.my_p;
  N.need[0] = 0; N.need[L_T1] = D.total[F_S0]; N.need[L_T2] = D.total[F_S2]; N.need[L_B1] = D.total[F_D1]; N.need[L_B2] = D.total[F_D2];
  N.pt1 = wide_count(PT1); N.g1 = D.total[F_G1]; N.nh = (uint32_t)k - wide_count(HIT); N.ev = D.total[F_S0] + D.total[F_S2];
}

// One scan round of a scanner warp: 128 ring entries from q0 (a multiple of 4), 4 per lane; live entries are appended
// to vic[] in LRU order.  Returns the number of live entries found in the round.
struct ScanRegs { uint4 e0, e1; };
// the loads of one round (positions q0 + 4 lane .. + 3); issued a round ahead so that their latency overlaps the previous
// round's bookkeeping.  Positions past the limit are loaded too (the ring is a power-of-two buffer) and ignored.
__device__ __forceinline__ ScanRegs wide_scan_load(const RingEnt* ring, uint32_t ring_mask, uint32_t q0, int lane) {
  const uint32_t qA = q0 + 4u * (uint32_t)lane;
  ScanRegs r;
  r.e0 = __ldcg(reinterpret_cast<const uint4*>(ring + (qA & ring_mask)));
  r.e1 = __ldcg(reinterpret_cast<const uint4*>(ring + ((qA + 2u) & ring_mask)));
  return r;
}
__device__ __forceinline__ uint32_t wide_scan_round(const ScanRegs& regs, uint32_t q0, uint32_t head, uint32_t limit,
                                                    uint32_t found, uint4* vic, int lane, uint32_t lt) {
  const uint32_t FULL = 0xFFFFFFFFu;
  const uint32_t qA = q0 + 4u * (uint32_t)lane;
  const uint4 e0 = regs.e0, e1 = regs.e1;
  // live = inside [head, limit) and not a tombstone
  const bool l0 = (int32_t)(qA - head) >= 0 && (int32_t)(limit - qA) > 0 && e0.x != RING_TOMB;
  const bool l1 = (int32_t)(qA + 1u - head) >= 0 && (int32_t)(limit - qA - 1u) > 0 && e0.z != RING_TOMB;
  const bool l2 = (int32_t)(qA + 2u - head) >= 0 && (int32_t)(limit - qA - 2u) > 0 && e1.x != RING_TOMB;
  const bool l3 = (int32_t)(qA + 3u - head) >= 0 && (int32_t)(limit - qA - 3u) > 0 && e1.z != RING_TOMB;
  const uint32_t c0 = __ballot_sync(FULL, l0), c1 = __ballot_sync(FULL, l1), c2 = __ballot_sync(FULL, l2), c3 = __ballot_sync(FULL, l3);
  uint32_t rk = found + (uint32_t)(__popc(c0 & lt) + __popc(c1 & lt) + __popc(c2 & lt) + __popc(c3 & lt));
  if (l0) { if (rk < (uint32_t)WIDE_W) vic[rk] = make_uint4(e0.x, e0.y, 0u, qA); ++rk; }
  if (l1) { if (rk < (uint32_t)WIDE_W) vic[rk] = make_uint4(e0.z, e0.w, 0u, qA + 1u); ++rk; }
  if (l2) { if (rk < (uint32_t)WIDE_W) vic[rk] = make_uint4(e1.x, e1.y, 0u, qA + 2u); ++rk; }
  if (l3) { if (rk < (uint32_t)WIDE_W) vic[rk] = make_uint4(e1.z, e1.w, 0u, qA + 3u); ++rk; }
  return (uint32_t)(__popc(c0) + __popc(c1) + __popc(c2) + __popc(c3));
}

// Scanner warp for list L (warps 4..7 of the CTA): follows the owners' barrier sequence window by window.  The first
// 128 entries from the list head are scanned while the owners fetch node records and roll the counters forward; more
// rounds follow only if the window turns out to need more victims than that.
template <bool LRU, bool PIPE>
__device__ __forceinline__ void wide_scanner(const StepParams& P, WideShared& S, uint32_t L, int lane) {
  const uint32_t lt = (1u << lane) - 1u;
  const RingEnt* ring = P.ring[L];
  unsigned long long rounds = 0;
  for (;;) {
    cta_sync<PIPE>();                                  // (S0) the window's control block is published
    if (S.ctl_done) break;
    const uint32_t head = S.ctl_head[L], limit = S.ctl_limit[L];
    uint32_t q0 = head & ~3u, found = 0;
    int want = (int)S.ctl_k;
    ScanRegs cur = wide_scan_load(ring, P.ring_mask, q0, lane);   // in flight while the owners fetch; used after B1
    // The LRU end of a list is the part of its ring that was written longest ago: in a cache larger than L2 it is in DRAM by
    // now, and a scan that waits for it holds up the whole window.  Each lane asks for one 128-byte line of the 512 entries
    // AFTER this window's first round to be brought into L2 (the next windows' first rounds); a line that is there costs nothing.
    if (PIPE) asm volatile("prefetch.global.L2 [%0];" ::"l"(ring + (((q0 & ~15u) + (uint32_t)WIDE_W + 16u * (uint32_t)lane) & P.ring_mask)));
    cta_sync<PIPE>();                                  // (B1) the scanners never hold this barrier up
    if (S.twinc[0] | S.twinc[1] | S.twinc[2] | S.twinc[3]) { cta_sync<PIPE>(); cta_sync<PIPE>(); want = (int)S.twin_k; }
    // while the owners roll (not in an all-hit window, which needs no victim): up to 3 rounds, until as many live entries
    // are known as the window has accesses, so that the owners rarely wait for a scan after the roll
    bool all_hit = true;
#pragma unroll
    for (int u = 0; u < WIDE_WARPS; ++u) {
      const uint32_t km = bits_from(0, min(32, max(0, want - 32 * u)));
      const uint32_t m0 = S.m[0][u], m1 = S.m[1][u], m2 = S.m[2][u];
      const uint32_t hit = LRU ? (m0 & ~m1 & ~m2) : ((m0 ^ m1) & ~m2);
      all_hit = all_hit && ((hit & km) == km);
    }
    if (all_hit) continue;                             // the owners apply an all-hit window without any further barrier
    // PIPE: the window's decisions were rolled ahead and stand (the owners judge that the same way): what the window takes
    // from this list is known now, and the owners are waiting for nothing else
    const bool known = PIPE && S.ctl_prov && !(S.reload[0] | S.reload[1] | S.reload[2] | S.reload[3]) && want == (int)S.ctl_k;
    if (known) {
      const uint32_t need = S.res[S.ctl_par & 1u].need[L];
      while (found < need && (int32_t)(limit - q0) > 0) {
        const ScanRegs nxt = wide_scan_load(ring, P.ring_mask, q0 + (uint32_t)WIDE_W, lane);
        found += wide_scan_round(cur, q0, head, limit, found, S.vic[L], lane, lt); q0 += (uint32_t)WIDE_W; ++rounds;
        cur = nxt;
      }
    } else {
      for (int it = 0; it < 4 && (int)found < want && (int32_t)(limit - q0) > 0; ++it) {
        const ScanRegs nxt = wide_scan_load(ring, P.ring_mask, q0 + (uint32_t)WIDE_W, lane);
        found += wide_scan_round(cur, q0, head, limit, found, S.vic[L], lane, lt); q0 += (uint32_t)WIDE_W; ++rounds;
        cur = nxt;
      }
    }
    __syncwarp();
    if (lane == 0) { S.found[L] = found; S.more[L] = (int32_t)(limit - q0) > 0; }
    cta_sync<PIPE>();                                  // (B2) the owners have published what the window needs, the scanners what they have
    bool extra = false;                                // some list must be scanned further: CTA-uniform, computed by everybody
#pragma unroll
    for (int X = 1; X <= 4; ++X) extra = extra || (S.found[X] < S.need[X] && S.more[X]);
    if (extra) {
      const uint32_t need = S.need[L];
      while (found < need && (int32_t)(limit - q0) > 0) {
        cur = wide_scan_load(ring, P.ring_mask, q0, lane);
        found += wide_scan_round(cur, q0, head, limit, found, S.vic[L], lane, lt); q0 += (uint32_t)WIDE_W; ++rounds;
      }
      cta_sync<PIPE>();                                // (B2x) everybody has read the first report
      __syncwarp();
      if (lane == 0) S.found[L] = found;
      cta_sync<PIPE>();                                // (B2') victims of all four lists are in shared memory
    }
    if (cta_or<PIPE>(false)) {                         // (B3) some access cannot be applied with the window
      cta_sync<PIPE>();                                // (B3x) the owners' reports are in shared memory
      bool serial = false;
#pragma unroll
      for (int u = WIDE_WARPS - 1; u >= 0; --u) if (S.bad[u]) serial = (32 * u + __ffs(S.bad[u]) - 1) == 0;
      if (serial) cta_sync<PIPE>();                    // the by-the-book access of warp 0
    }
  }
  if (lane == 0 && rounds) atomicAdd(&P.state->dbg[DBG_SCAN_ROUNDS], rounds);
}

// PIPE: the roller warps (warps 8..11).  The counter recurrence is the one strictly serial piece of a window and depends on
// nothing but the class masks and eight counters, so it runs here, a window AHEAD of the owners: while they check and
// apply window w, these warps roll window w + 1 from the masks of its speculative records and the counters after w, and
// turn the decisions into one plan per access (WidePlan: what the access evicts, drops and pushes, as ranks) plus the
// window's counts, so that the owners' part of a window is loads, checks and stores only.  The owners take the result if
// every speculative record stood and w was applied whole; otherwise they ask again with what they then know.  The four
// warps roll redundantly, like the owner warps of the plain form (no decision is ever broadcast); thread g plans access
// g.  They keep no state of their own: every request carries the counters it starts from.
template <bool LRU>
__device__ __forceinline__ void wide_roller(const StepParams& P, WideShared& S, int g) {
  const int lane = g & 31, w = g >> 5;
  const uint32_t FULL = 0xFFFFFFFFu, lt = (1u << lane) - 1u;
  uint32_t lm[WIDE_WARPS], me[WIDE_WARPS];
#pragma unroll
  for (int u = 0; u < WIDE_WARPS; ++u) { lm[u] = (u < w) ? FULL : ((u == w) ? lt : 0u); me[u] = (u == w) ? (1u << lane) : 0u; }
  const int32_t c = P.capacity;
  const bool dbl = (P.policy == POLICY_DBL);
  for (uint32_t i = 0;; ++i) {
    bar_sync_n(BAR_REQ, ROLL_PARTIES);                 // a request is in S.req
    if (S.req.quit) break;
    Roll R0;
    R0.t1 = S.req.st[0]; R0.t2 = S.req.st[1]; R0.b1 = S.req.st[2]; R0.b2 = S.req.st[3]; R0.p = S.req.st[4]; R0.nf = S.req.st[5];
    R0.e1 = S.req.st[6]; R0.e2 = S.req.st[7];
    R0.s0 = R0.s1 = R0.d1 = R0.d2 = R0.fm = 0; R0.my_p = R0.p; R0.err = 0; R0.calls = 0; R0.phases = 0; R0.dbl = dbl;
    const int k = S.req.k;
    RollRes& Q = S.res[i & 1u];
    {
      // A window of hits only (half of all windows of a warm cache) on a short path of its own: T1 entries move to T2,
      // evictable entries stop being so, nothing else.
      bool all_hit = true;
      int32_t h1 = 0, e1d = 0, e2d = 0;
      uint32_t badnode = 0;
#pragma unroll
      for (int u = 0; u < WIDE_WARPS; ++u) {
        const uint32_t km = bits_from(0, min(32, max(0, k - 32 * u)));
        const uint32_t m0 = S.req.m[0][u] & km, m1 = S.req.m[1][u] & km, m2 = S.req.m[2][u] & km, mev = S.req.m[3][u] & km;
        all_hit = all_hit && ((LRU ? (m0 & ~m1 & ~m2) : ((m0 ^ m1) & ~m2)) == km);
        h1 += __popc(m0); e1d += __popc(mev & m0); e2d += __popc(mev & m1);
        badnode |= m2 & m0;
      }
      // the owners of a window whose roll-ahead stands take these instead of reading the class masks themselves
      if (g == 0) { Q.all_hit = all_hit ? 1u : 0u; Q.badnode = badnode; Q.h1 = (uint32_t)h1; Q.e1d = (uint32_t)e1d; Q.e2d = (uint32_t)e2d; }
      if (all_hit) {
        // (the plan is still written: a window cut back to its leading hits after a conflict is applied by the general path)
        WidePlan A;
        A.src = 0; A.d1 = A.d2 = A.fm = false; A.vic_rank = A.gpush_rank = A.drop_rank = A.fresh_rank = A.alloc_rank = A.evict_rank = 0;
        A.push_rank = (uint32_t)g;                       // every access pushes its node to T2 (LRU: T1), in access order
        A.p = R0.p;
        Q.plan[g] = plan_pack(A);
        if (g == 0) {
          Q.st[0] = R0.t1 - (LRU ? 0 : h1); Q.st[1] = R0.t2 + (LRU ? 0 : h1); Q.st[2] = R0.b1; Q.st[3] = R0.b2; Q.st[4] = R0.p; Q.st[5] = R0.nf;
          Q.st[6] = R0.e1 - e1d; Q.st[7] = R0.e2 - (LRU ? 0 : e2d);
#pragma unroll
          for (int L = 0; L <= 4; ++L) Q.need[L] = 0;
          Q.pt1 = LRU ? (uint32_t)k : 0u; Q.g1 = 0; Q.nh = 0; Q.ev = 0; Q.err = 0; Q.phases = 0;
        }
        __threadfence_block();
        __syncwarp();
        bar_arrive_n(BAR_DONE, ROLL_PARTIES);
        continue;
      }
    }
    WideDecisions D;
    wide_roll<LRU>(D, R0, c, S.req.m, k, w, lane);
    WidePlan A;
    WideCounts N;
    wide_make_plan<LRU>(A, N, D, S.req.m, k, (uint32_t)g, lm, me);
    Q.plan[g] = plan_pack(A);
    if (g == 0) {
      Q.st[0] = D.R.t1; Q.st[1] = D.R.t2; Q.st[2] = D.R.b1; Q.st[3] = D.R.b2; Q.st[4] = D.R.p; Q.st[5] = D.R.nf; Q.st[6] = D.R.e1; Q.st[7] = D.R.e2;
#pragma unroll
      for (int L = 0; L <= 4; ++L) Q.need[L] = N.need[L];
      Q.pt1 = N.pt1; Q.g1 = N.g1; Q.nh = N.nh; Q.ev = N.ev;
      Q.err = D.R.err; Q.phases = D.R.phases;
    }
    __threadfence_block();
    __syncwarp();
    bar_arrive_n(BAR_DONE, ROLL_PARTIES);              // the result is in S.res[i & 1]
  }
}

// The machine itself, run by the first 2 * WIDE_W threads of a CTA (all of them must call it; it ends with every thread
// past the last barrier).  S: the CTA's WideShared.  Also the third phase of the one-launch small-step kernel.
// The policy (LRU or the two-list ARC / DBL) and the held pin scope are template parameters: the kernel is one CTA whose
// instruction fetch nothing hides (ncu: one fetch stall per issued instruction, 20 % instruction-cache misses), so every
// variant carries only its own code.
template <bool LRU, bool HOLD, bool PIPE>
__device__ __forceinline__ void wide_machine_run(const StepParams& P, WideShared& S) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t FULL = 0xFFFFFFFFu, lt = (1u << lane) - 1u;
  uint32_t lm[WIDE_WARPS], me[WIDE_WARPS];   // see wide_rank / wide_has
#pragma unroll
  for (int u = 0; u < WIDE_WARPS; ++u) { lm[u] = (u < warp) ? FULL : ((u == warp) ? lt : 0u); me[u] = (u == warp) ? (1u << lane) : 0u; }
  constexpr bool lru = LRU;
  constexpr bool hold = HOLD;                // held scope: see machine_batched.cuh
  const int32_t c = P.capacity;
  const int64_t N = (int64_t)P.n_access;
  if (P.state->error == DEV_ERR_NODE_POOL) return;       // K2 could not give every key a node: the step is void (sticky error; CTA-uniform)
  if (PIPE && warp >= 2 * WIDE_WARPS) { wide_roller<LRU>(P, S, tid - 2 * WIDE_W); return; }   // warps 8..11 roll the counters a window ahead
  SerialCtx C;            // identical in every thread
  ctx_load(C, P);
  uint32_t dbg[DBG_COUNT];                    // per-step sums fit 32 bits (a step is a few 10^7 cycles); clock() is the low word of the SM clock
#pragma unroll
  for (int i = 0; i < DBG_COUNT; ++i) dbg[i] = 0;
  const uint32_t t_begin = (uint32_t)clock();
#ifdef ARC_PROBES
  uint32_t tp_ = t_begin;
#endif
  if (warp >= WIDE_WARPS) {                                 // warps 4..7 scan the LRU ends of T1, T2, B1, B2
    wide_scanner<LRU, PIPE>(P, S, (uint32_t)(warp - WIDE_WARPS) + 1u, lane);
    return;
  }

  // Node ids travel ahead of the windows through a shared-memory ring filled with cp.async: at the start of a window the
  // ids of that window AND of the one after it are already there (they were requested at least one window earlier),
  // wherever a cut made the window start.
  uint32_t ids_loaded = 0;                               // ids [0, ids_loaded) have been requested; a multiple of WIDE_W
  auto ids_request = [&](int64_t upto) {
    while ((int64_t)ids_loaded < upto && (int64_t)ids_loaded < N) {
      const uint32_t a = ids_loaded + (uint32_t)tid;
      if ((int64_t)a < N) cp_async_u32(&S.ids[a & (WIDE_IDS - 1)], P.node_acc + a);
      ids_loaded += (uint32_t)WIDE_W;
    }
    cp_async_commit();
  };
  ids_request(2 * WIDE_W);
  int64_t spec_base = -1;                                // the access index the speculative record below belongs to, minus tid
  // ... and so is the node RECORD, speculatively: it is loaded while the current window rolls (after B1, when everything
  // the previous window wrote is visible) and is exact unless the current window itself changes that node, which happens
  // in two ways only: the window also accesses the node, or it takes the node as a victim / dropped ghost (the node's
  // ring position lies in a range the window consumes).  Either way the record is then loaded again at the start of the
  // next window, as it is after a cut window.  Every node of a window carries the window's number in node_stamp[] BEFORE
  // the window's first barrier; the speculative load, issued AFTER it, exchanges the stamp for the NEXT window's number
  // and gets the old one back: equal to the current window's number = this window accesses the node too (only a window
  // of another request can); equal to the next window's number = another thread of the next window owns the same node
  // (a twin candidate, see the top of the file).  A window that does not start where the previous one was due to end
  // (after a cut) stamps its nodes itself, synchronously, with a number no earlier exchange used.
  Node spec;
  spec.list = L_FREE; spec.pos = 0; spec.block = -1; spec.slot = 0;
  bool spec_ok = false;
  uint32_t win_seq = P.state->win_seq;                     // numbers the windows across steps; 31 bits, never 0
  uint32_t spec_mark = 0;                                  // what node_stamp of the speculated node held before this thread's exchange
  uint32_t my_cls[5] = {0, 0, 0, 0, 0};                  // accesses of general windows this thread applied, by class

  // PIPE: the roller warp's mailbox.  At most one request is outstanding; request number i answers into S.res[i & 1].
  uint32_t req_no = 0;
  bool have_prov = false;                                  // a request for the NEXT window (rolled ahead) is outstanding
  uint32_t prov_par = 0;                                   // ... and the buffer its result goes to
  // every owner thread calls these (warp-uniform control flow); tid 0 has written the request's scalars
  auto roll_send = [&]() -> uint32_t {
    __threadfence_block();
    bar_arrive_n(BAR_REQ, ROLL_PARTIES);
    return (req_no++) & 1u;
  };
  auto roll_wait = [&]() { bar_sync_n(BAR_DONE, ROLL_PARTIES); };
  auto roll_state = [&](int32_t t1, int32_t t2, int32_t b1, int32_t b2, int32_t p, int32_t nf, int32_t e1, int32_t e2, int kk) {
    if (tid == 0) {
      S.req.st[0] = t1; S.req.st[1] = t2; S.req.st[2] = b1; S.req.st[3] = b2; S.req.st[4] = p; S.req.st[5] = nf; S.req.st[6] = e1; S.req.st[7] = e2;
      S.req.k = kk; S.req.quit = 0;
    }
  };

  // Held pins: nothing restarts at a request boundary (the evictable counts carry over, every ring entry is a possible
  // victim), so the whole step is ONE run of accesses and a window may span requests: 24 one-block decode
  // appends are one window, not 24.  Only the natural-order index of an access then depends on its request: it comes
  // from nat_acc[] (nat_index_kernel / the one-launch kernel).  A node that two requests of a window share is a repeated node
  // like any other: the window is cut before its second occurrence.
  constexpr bool merged = HOLD;            // (a compile-time fact on purpose: as a run-time flag for the step-wide scope too it cost
                                           // the default scope 12 - 19 % - seven more registers and a different schedule of the whole loop)
  const uint32_t* nat_acc = reinterpret_cast<const uint32_t*>(P.keys_acc);   // the keys are K2's input only: their buffer is free now
  const uint32_t n_groups = merged ? 1u : P.n_req;
  int64_t my_off = 0, my_off1 = 0, my_off2 = 0;
  for (uint32_t r = 0; r < n_groups; ++r) {
    if (!merged && (r & 31u) == 0) {      // block offsets of the next 32 requests, one per lane (every warp keeps its own copy)
      const uint32_t rr = min(r + (uint32_t)lane, P.n_req - 1);
      my_off = P.blk_off[rr]; my_off1 = P.blk_off[rr + 1]; my_off2 = P.blk_off[min(rr + 2, P.n_req)];
    }
    const int64_t o = merged ? 0 : __shfl_sync(FULL, my_off, r & 31), nb = merged ? N : __shfl_sync(FULL, my_off1, r & 31) - o;
    if (!hold && (r == 0 || P.pin_scope == 0)) begin_request(C);   // step-wide scope: the pins of earlier requests of the step stay
    int64_t j = 0;
    while (j < nb) {
      const int kmax = (int)min((int64_t)WIDE_W, nb - j);
      int k = kmax;
      const int64_t a0 = o + j;
      const bool act0 = tid < k;
      // size of the window after this one if this one is not cut (an upper bound where the next request is empty)
      int next_k = WIDE_W;
      bool next_exact = false, next_new_req = false;       // the size is exact; that window is the first of a request
      if (j + kmax < nb) { next_k = (int)min((int64_t)WIDE_W, nb - j - kmax); next_exact = true; }
      else if (!merged && r + 1u < P.n_req) {
        const int64_t nb1 = __shfl_sync(FULL, my_off2, r & 31) - __shfl_sync(FULL, my_off1, r & 31);
        if (nb1 > 0) { next_k = (int)min((int64_t)WIDE_W, nb1); next_exact = true; next_new_req = true; }
      }
      if (tid == 0) {
        S.ctl_done = 0; S.ctl_k = (uint32_t)kmax;
        if (PIPE) { S.ctl_prov = have_prov ? 1u : 0u; S.ctl_par = prov_par; }
#pragma unroll
        for (int L = 1; L <= 4; ++L) { S.ctl_head[L] = C.head[L]; S.ctl_limit[L] = (L <= 2) ? C.bound[L] : C.tail[L]; }
      }
      cp_async_wait_all();                                           // ids requested in earlier windows have landed
      PROBE(0);                                                      // window top: loop, control block, ids landed
      cta_sync<PIPE>();                                              // (S0) the previous window's writes are visible; the scanners start
      PROBE(1);                                                      // S0 wait
      const uint32_t tw0 = (uint32_t)clock();
      const uint32_t n = act0 ? S.ids[(uint32_t)(a0 + tid) & (WIDE_IDS - 1)] : NODE_NONE;
      Node rec;
      rec.list = L_FREE; rec.pos = 0; rec.block = -1; rec.slot = 0;
      const bool aligned = (spec_base == a0);                        // the window starts where the previous one was due to end:
      const uint32_t prev_seq = win_seq;                             // its nodes were stamped with its number a window ago
      win_seq = wide_next_seq(win_seq);
      if (!aligned) win_seq = wide_next_seq(win_seq);                // a number no exchange has used yet
      bool twin_c = false;                                           // the stamp says another thread of this window may own the same node
      bool reloaded = act0;                                          // this owner could not use a speculative record
      if (act0) {
        if (aligned) {
          // The exchange returned the stamp's last value only.  This window's number there means another exchange for
          // this window came first (a twin, or a thread that stamped a position beyond the window because next_k was an
          // upper bound) and took away what the stamp said before: the record cannot be trusted either.
          twin_c = (spec_mark == win_seq);
          if (spec_mark == prev_seq || twin_c) spec_ok = false;      // the previous window accessed the speculated node too
          if (spec_ok) { rec = spec; reloaded = false; } else rec = ld_node(P.nodes + n);
        } else {
          const uint32_t old = atomicExch(P.node_stamp + n, win_seq);   // seen by the exchanges after B1
          rec = ld_node(P.nodes + n);
          twin_c = (old == win_seq);
        }
      }
      // the id this thread will own if the next window starts where this one is due to end
      const uint32_t pre_n = (a0 + kmax + tid < N) ? S.ids[(uint32_t)(a0 + kmax + tid) & (WIDE_IDS - 1)] : NODE_NONE;
      // The next window's record, speculatively, and its stamp (see above).  An aligned window's own stamps were written a
      // window ago, so nothing of this window touches node_stamp before its first barrier and the exchange can go out right
      // here, a whole fetch phase earlier: the round trip is then over when the next window starts even after an all-hit
      // window.  (A window that stamps its nodes itself, above, sends it after the barrier instead.)
      auto issue_spec = [&]() {
        spec_ok = false;
        spec_base = a0 + kmax;
        if (pre_n != NODE_NONE && tid < next_k) {                      // next_k >= the next window's size: every owner of it is covered
          spec = ld_node(P.nodes + pre_n);
          spec_mark = atomicExch(P.node_stamp + pre_n, wide_next_seq(win_seq));   // looked at when the next window starts, not now
          spec_ok = true;
        }
      };
      PROBE(2);                                                      // ids, record (speculative or loaded)
      if (aligned) issue_spec();
      PROBE(12);
      ids_request(a0 + kmax + 2 * WIDE_W);
      PROBE(13);
      const uint32_t lst = rec.list & NODE_LIST_MASK;
      const bool held = (rec.list & NODE_HELD) != 0;                 // held scope: in no ring, rec.pos = its holds
      {
        const uint32_t b0 = __ballot_sync(FULL, lst & 1u), b1 = __ballot_sync(FULL, lst & 2u), b2 = __ballot_sync(FULL, lst & 4u);
        // hits on entries that were still evictable by this request (below bound): they stop being so
        const uint32_t be = __ballot_sync(FULL, !held && ((lst == L_T1 && (int32_t)(C.bound[L_T1] - rec.pos) > 0) ||
                                                              (lst == L_T2 && (int32_t)(C.bound[L_T2] - rec.pos) > 0)));
        const uint32_t bt = __ballot_sync(FULL, twin_c);
        const uint32_t br = PIPE ? __ballot_sync(FULL, reloaded) : 0u;
        if (lane == 0) { S.m[0][warp] = b0; S.m[1][warp] = b1; S.m[2][warp] = b2; S.m[3][warp] = be; S.twinc[warp] = bt; if (PIPE) S.reload[warp] = br; }
      }
      // PIPE: the result rolled ahead for this window is taken out of the mailbox before the barrier, so that the scanners
      // may read it after the barrier; whether it stands is known after the barrier (to everybody, from shared memory)
      const bool got_prov = PIPE && have_prov;
      const uint32_t got_par = prov_par;
      PROBE(3);                                                      // spec issue, ids request, ballots
      if (got_prov) { roll_wait(); have_prov = false; }
      PROBE(4);                                                      // wait for the roller
      cta_sync<PIPE>();                                              // (B1) class masks and twin candidates are complete
      PROBE(5);                                                      // B1 wait
      // (1) the same node twice in the window: cut before the second occurrence
      if (S.twinc[0] | S.twinc[1] | S.twinc[2] | S.twinc[3]) {       // CTA-uniform, next to never taken
        bool later = false;                                          // an earlier access of the window has this thread's node
        if (act0) for (int i = 0; i < tid; ++i) later = later || (S.ids[(uint32_t)(a0 + i) & (WIDE_IDS - 1)] == n);
        const uint32_t tb = __ballot_sync(FULL, later);
        if (lane == 0) S.twin[warp] = tb;
        cta_sync<PIPE>();
        int first = k;
#pragma unroll
        for (int u = WIDE_WARPS - 1; u >= 0; --u) if (S.twin[u]) first = 32 * u + __ffs(S.twin[u]) - 1;
        if (first < k) { k = first; dbg[DBG_CUT_TWIN]++; }
        if (tid == 0) S.twin_k = (uint32_t)k;                        // the scanners judge "all hits" on the same accesses
        cta_sync<PIPE>();
      }
      const bool prov_valid = got_prov && !(S.reload[0] | S.reload[1] | S.reload[2] | S.reload[3]) && k == kmax;
      // PIPE: the request for the window after this one, from the masks of its speculative records and the counters this
      // window leaves (t1 .. e2), on the assumption that this window is applied whole.  bn1 / bn2: where the victim scans of
      // that window stop (its request's pin bound: the tails after this window if it starts a request).
      auto roll_ahead = [&](int32_t t1, int32_t t2, int32_t b1, int32_t b2, int32_t p, int32_t nf, int32_t e1, int32_t e2,
                            uint32_t tail1_after, uint32_t tail2_after) {
        const bool fresh = next_new_req && !hold && P.pin_scope == 0;   // begin_request before that window
        const uint32_t bn1 = fresh ? tail1_after : C.bound[L_T1], bn2 = fresh ? tail2_after : C.bound[L_T2];
        const uint32_t ls = spec_ok ? (spec.list & NODE_LIST_MASK) : 0u;
        const bool hd = spec_ok && (spec.list & NODE_HELD) != 0;
        const uint32_t b0 = __ballot_sync(FULL, ls & 1u), b1m = __ballot_sync(FULL, ls & 2u), b2m = __ballot_sync(FULL, ls & 4u);
        const uint32_t be = __ballot_sync(FULL, !hd && ((ls == L_T1 && (int32_t)(bn1 - spec.pos) > 0) || (ls == L_T2 && (int32_t)(bn2 - spec.pos) > 0)));
        if (lane == 0) { S.req.m[0][warp] = b0; S.req.m[1][warp] = b1m; S.req.m[2][warp] = b2m; S.req.m[3][warp] = be; }
        roll_state(t1, t2, b1, b2, p, nf, fresh ? t1 : e1, fresh ? t2 : e2, next_k);
        prov_par = roll_send();
        have_prov = true;
      };
      if (!aligned) issue_spec();                                    // a node this window accesses too is not trusted (its stamp says so)
      // hits only?  and if so: hits in T1, hits on entries of T1 / T2 that were still evictable.  From the rollers when their
      // roll-ahead of this window stands (they read the same masks), else from the class masks in shared memory.
      bool all_hit = true;
      uint32_t badnode = 0, t1hits = 0, e1d = 0, e2d = 0;
      if (prov_valid) {
        const RollRes& Q = S.res[got_par & 1u];
        all_hit = Q.all_hit != 0; badnode = Q.badnode; t1hits = Q.h1; e1d = Q.e1d; e2d = Q.e2d;
      } else {
#pragma unroll
        for (int u = 0; u < WIDE_WARPS; ++u) {
          const uint32_t km = bits_from(0, min(32, max(0, k - 32 * u)));
          const uint32_t m0 = S.m[0][u] & km, m1 = S.m[1][u] & km, m2 = S.m[2][u] & km, mev = S.m[3][u] & km;
          all_hit = all_hit && ((lru ? (m0 & ~m1 & ~m2) : ((m0 ^ m1) & ~m2)) == km);
          badnode |= m2 & m0;
          t1hits += (uint32_t)__popc(m0); e1d += (uint32_t)__popc(mev & m0); e2d += (uint32_t)__popc(mev & m1);
        }
      }
      if (badnode) C.err = DEV_ERR_BAD_NODE;                         // a FREE node reached K3
      const uint32_t tw1 = (uint32_t)clock();
      dbg[DBG_CYC_FETCH] += tw1 - tw0;
      PROBE(6);                                                      // twin check, masks

      if (all_hit) {
        // ---- every access of the window is a hit: no counter other than t1/t2 moves, nothing is evicted
        const uint32_t q = (lru ? C.tail[L_T1] : C.tail[L_T2]) + (uint32_t)tid;
        if (lru) { C.tail[L_T1] += hold ? 0u : (uint32_t)k; C.stat[ST_HIT_T1] += (uint32_t)k; }
        else { C.tail[L_T2] += hold ? 0u : (uint32_t)k; C.t1 -= (int32_t)t1hits; C.t2 += (int32_t)t1hits; C.stat[ST_HIT_T1] += t1hits; C.stat[ST_HIT_T2] += (uint32_t)k - t1hits; }
        C.elig1 -= (int32_t)e1d; C.elig2 -= (int32_t)e2d;
        C.stat[ST_ACCESSES] += (uint32_t)k;
        if (PIPE) {                                  // the counters after the window are known: the next one goes to the roller
          dbg[prov_valid ? DBG_PROV_OK : DBG_PROV_MISS]++;   // first, so that it rolls while this one is stored
          if (next_exact && k == kmax && a0 + kmax < N)
            roll_ahead(C.t1, C.t2, C.b1, C.b2, C.p, C.next_fresh, C.elig1, C.elig2, C.tail[L_T1], C.tail[L_T2]);
        }
        if (tid < k) {
          if (!held) ring_tomb(P, lst, rec.pos);
          if (hold) {
            st_node(P.nodes + n, (lru ? L_T1 : L_T2) | NODE_HELD, held ? rec.pos + 1u : 1u, rec.block, rec.slot);
            P.node_of_block[rec.block] = n;
          } else {
            __stcg((lru ? P.ring[L_T1] : P.ring[L_T2]) + (q & P.ring_mask), ring_ent(n, rec.block));
            st_node(P.nodes + n, lru ? L_T1 : L_T2, q, rec.block, rec.slot);
          }
          const int64_t out = merged ? (int64_t)__ldcg(nat_acc + a0 + tid) : o + (nb - 1 - (j + tid));
          P.cls[out] = (uint8_t)lst;                               // L_T1 == CLS_HIT_T1, L_T2 == CLS_HIT_T2
          P.block_id[out] = rec.block;
          P.evicted_id[out] = -1;
          P.p_after[out] = C.p;
          P.dropped[a0 + tid] = NODE_NONE;
        }
        if (tid < 5) S.need[tid] = 0;
        if (lane == 0) S.bad[warp] = 0;
        PROBE(7);                                                    // all-hit window: roll ahead + stores
        j += k;
        dbg[DBG_WIN_HIT]++; dbg[DBG_ACC_HIT_WIN] += (unsigned)k;
        dbg[DBG_CYC_APPLY] += (uint32_t)clock() - tw1;
        continue;
      }

      // ---- general window: the decisions (rolled ahead by the roller warps, or here by every owner warp), scans, checks, apply
      WidePlan A;                                                    // what this thread's access does
      WideCounts NC;                                                 // what the window takes and appends
      int32_t RS[8];                                                 // t1, t2, b1, b2, p, next_fresh, elig1, elig2 after the window
      uint32_t r_err = 0, r_phases = 0;
      // PIPE: what the roller warps worked out (ahead of time, or now on request) comes out of their result buffer
      auto roll_take = [&](uint32_t par) {
        const RollRes& Q = S.res[par & 1u];
        A = plan_unpack(Q.plan[tid]);
#pragma unroll
        for (int i = 0; i < 8; ++i) RS[i] = Q.st[i];
#pragma unroll
        for (int L = 0; L <= 4; ++L) NC.need[L] = Q.need[L];
        NC.pt1 = Q.pt1; NC.g1 = Q.g1; NC.nh = Q.nh; NC.ev = Q.ev;
        r_err = Q.err; r_phases = Q.phases;
      };
      auto roll_now = [&](int kk) {                                  // this window's first kk accesses, from the state in C
        if (PIPE) {
          if (tid < 4 * WIDE_WARPS) (&S.req.m[0][0])[tid] = (&S.m[0][0])[tid];
          roll_state(C.t1, C.t2, C.b1, C.b2, C.p, C.next_fresh, C.elig1, C.elig2, kk);
          const uint32_t par = roll_send();
          roll_wait();
          roll_take(par);
        } else {                                                     // the plain form: every owner warp rolls, every thread plans
          WideDecisions D;
          wide_roll<LRU>(D, roll_init(C), c, S.m, kk, warp, lane);
          wide_make_plan<LRU>(A, NC, D, S.m, kk, (uint32_t)tid, lm, me);
          RS[0] = D.R.t1; RS[1] = D.R.t2; RS[2] = D.R.b1; RS[3] = D.R.b2; RS[4] = D.R.p; RS[5] = D.R.nf; RS[6] = D.R.e1; RS[7] = D.R.e2;
          r_err = D.R.err; r_phases = D.R.phases;
        }
      };
      if (PIPE) {
        dbg[prov_valid ? DBG_PROV_OK : DBG_PROV_MISS]++;
        if (prov_valid) roll_take(got_par); else roll_now(k);
        if (next_exact && k == kmax && a0 + kmax < N)
          roll_ahead(RS[0], RS[1], RS[2], RS[3], RS[4], RS[5], RS[6], RS[7],
                     C.tail[L_T1] + (hold ? 0u : NC.pt1), C.tail[L_T2] + (hold ? 0u : (uint32_t)k - NC.pt1));
      } else {
        roll_now(k);
      }
      const uint32_t tw2 = (uint32_t)clock();
      dbg[DBG_CYC_ROLL] += tw2 - tw1;
      PROBE(8);                                                      // decisions taken, next window sent ahead
      if (tid == 0) { S.need[L_T1] = NC.need[L_T1]; S.need[L_T2] = NC.need[L_T2]; S.need[L_B1] = NC.need[L_B1]; S.need[L_B2] = NC.need[L_B2]; }
      cta_sync<PIPE>();                                              // (B2) the scanners learn what the window needs, the owners what they have
      PROBE(9);                                                      // need published, B2 wait
      uint32_t found[5], endpos[5];
      bool extra = false;                                            // CTA-uniform: some list must be scanned further
#pragma unroll
      for (int L = 1; L <= 4; ++L) { found[L] = S.found[L]; extra = extra || (found[L] < NC.need[L] && S.more[L]); }
      if (extra) {
        cta_sync<PIPE>();                                            // (B2x) everybody has read the first report
        cta_sync<PIPE>();                                            // (B2') victims of all four lists are in shared memory
#pragma unroll
        for (int L = 1; L <= 4; ++L) found[L] = S.found[L];
      }
#pragma unroll
      for (int L = 1; L <= 4; ++L) {
        const uint32_t limit = (L <= 2) ? C.bound[L] : C.tail[L];
        endpos[L] = NC.need[L] ? ((found[L] >= NC.need[L]) ? S.vic[L][NC.need[L] - 1].w + 1u : limit) : C.head[L];
      }
      // (2) an accessed node whose ring entry lies inside a consumed range, or a victim / drop that does not exist
      bool act = tid < k;
      bool bad = false;
      if (act) {
#pragma unroll
        for (int L = 1; L <= 4; ++L)
          if (lst == (uint32_t)L && !held && NC.need[L] && (rec.pos - C.head[L]) < (endpos[L] - C.head[L])) bad = true;
        // a victim / drop can be missing only from a list that has fewer live entries than the window wants (uniform)
        if (found[L_T1] < NC.need[L_T1] || found[L_T2] < NC.need[L_T2] || found[L_B1] < NC.need[L_B1] || found[L_B2] < NC.need[L_B2]) {
          if ((A.src & 1u) && A.vic_rank >= found[L_T1]) bad = true;
          if (A.src == 2 && A.vic_rank >= found[L_T2]) bad = true;
          if (A.d1 && A.drop_rank >= found[L_B1]) bad = true;
          if (A.d2 && A.drop_rank >= found[L_B2]) bad = true;
        }
      }
      int first_bad = -1;
      if (cta_or<PIPE>(bad)) {                                       // (B3) next to always: nobody is bad, nothing to exchange
        const uint32_t bb = __ballot_sync(FULL, bad);
        if (lane == 0) S.bad[warp] = bb;
        cta_sync<PIPE>();                                            // (B3x)
#pragma unroll
        for (int u = WIDE_WARPS - 1; u >= 0; --u) if (S.bad[u]) first_bad = 32 * u + __ffs(S.bad[u]) - 1;
      }
      const uint32_t tw3 = (uint32_t)clock();
      dbg[DBG_CYC_SCAN] += tw3 - tw2;
      PROBE(10);                                                     // checks, B3
      if (first_bad >= 0) {
        k = first_bad;
        dbg[DBG_CUT_CONFLICT]++;
        if (PIPE && have_prov) { roll_wait(); have_prov = false; }   // the window after this one was rolled ahead for nothing
        if (k == 0) {
          // the by-the-book routine, by warp 0 alone; the new machine state reaches the other warps through shared memory
          if (warp == 0) {
            SerialCtx T = C;                           // the callee is not inlined: keep C itself in registers
            serial_access(T, P, a0, merged ? (int64_t)__ldcg(nat_acc + a0) : o + (nb - 1 - j));
            __syncwarp();
            if (lane == 0) S.ctx = T;
          }
          cta_sync<PIPE>();
          C = S.ctx;
          j += 1;
          spec_ok = false;                             // the by-the-book access may have changed any node
          dbg[DBG_WIN_SERIAL]++;
          dbg[DBG_CYC_SERIAL] += (uint32_t)clock() - tw3;
          continue;
        }
        roll_now(k);                                   // the decisions, plans and counts of the first k accesses alone
#pragma unroll
        for (int L = 1; L <= 4; ++L) endpos[L] = NC.need[L] ? S.vic[L][NC.need[L] - 1].w + 1u : C.head[L];
        act = tid < k;
      }
      if (r_err) C.err = r_err;
      dbg[DBG_ROLL_PHASES] += r_phases;

      // ---- apply (threads < k): the plan says what, the scans say which entries, C says where the lists end
      if (act) {
        const bool is_hit = lru ? (lst == L_T1) : (lst == L_T1 || lst == L_T2);
        const bool toT1 = lru || lst == L_ABSENT;                   // ABSENT nodes enter T1 (LRU: everything), the rest T2
        int32_t blk = rec.block, ev = -1;
        uint32_t dropped = NODE_NONE;
        if (A.src) {
          const uint4 v = (A.src == 2) ? S.vic[L_T2][A.vic_rank] : S.vic[L_T1][A.vic_rank];
          blk = ev = (int32_t)v.y;
          if (A.src == 3) {                         // leaves no ghost: the key leaves the directory in K4
            st_node_keep_slot(P.nodes + v.x, L_ABSENT, 0, -1);
            dropped = v.x;
          } else {
            const uint32_t q = ((A.src == 1) ? C.tail[L_B1] : C.tail[L_B2]) + A.gpush_rank;
            __stcg(((A.src == 1) ? P.ring[L_B1] : P.ring[L_B2]) + (q & P.ring_mask), ring_ent(v.x, -1));
            st_node_keep_slot(P.nodes + v.x, (A.src == 1) ? L_B1 : L_B2, q, -1);
          }
        } else if (A.fm) {
          blk = C.next_fresh + (int32_t)A.fresh_rank;
        }
        if (A.d1 || A.d2) {
          const uint4 d = A.d1 ? S.vic[L_B1][A.drop_rank] : S.vic[L_B2][A.drop_rank];
          st_node_keep_slot(P.nodes + d.x, L_ABSENT, 0, -1);
          dropped = d.x;
        }
        const uint32_t q = (toT1 ? C.tail[L_T1] : C.tail[L_T2]) + A.push_rank;
        if (lst >= L_T1 && lst <= L_B2 && !held) ring_tomb(P, lst, rec.pos);     // the node leaves its old position
        if (hold) {
          st_node(P.nodes + n, (toT1 ? L_T1 : L_T2) | NODE_HELD, held ? rec.pos + 1u : 1u, blk, rec.slot);
          P.node_of_block[blk] = n;
        } else {
          __stcg((toT1 ? P.ring[L_T1] : P.ring[L_T2]) + (q & P.ring_mask), ring_ent(n, blk));
          st_node(P.nodes + n, toT1 ? L_T1 : L_T2, q, blk, rec.slot);
        }
        const int64_t out = merged ? (int64_t)__ldcg(nat_acc + a0 + tid) : o + (nb - 1 - (j + tid));
        P.cls[out] = (uint8_t)lst;                    // ABSENT -> MISS(0), T1 -> 1, T2 -> 2, B1 -> 3, B2 -> 4
        P.block_id[out] = blk;
        P.evicted_id[out] = ev;
        P.p_after[out] = A.p;
        P.dropped[a0 + tid] = dropped;
        if (!is_hit) P.alloc_ids[C.n_alloc + A.alloc_rank] = blk;
        if (ev >= 0) P.evict_ids[C.n_evict + A.evict_rank] = ev;
      }
      // class counts: every thread counts its own access, the warps add them up at the end of the kernel
      if (act) {
        my_cls[0] += (lst == L_ABSENT); my_cls[1] += (lst == L_T1); my_cls[2] += (lst == L_T2) && !lru;
        my_cls[3] += (lst == L_B1); my_cls[4] += (lst == L_B2);
      }
      // uniform state (every thread computes the same)
      C.stat[ST_ACCESSES] += (uint32_t)k;
      C.stat[ST_EVICT_T1] += NC.need[L_T1];
      C.stat[ST_EVICT_T2] += NC.need[L_T2];
      C.stat[ST_DROP_B1] += NC.need[L_B1];
      C.stat[ST_DROP_B2] += NC.need[L_B2];
      C.stat[ST_FRESH] += (uint32_t)(RS[5] - C.next_fresh);
      C.n_alloc += NC.nh;
      C.n_evict += NC.ev;
      if (spec_ok) {                                 // did this window take the speculated node as a victim or drop it?
#pragma unroll
        for (int L = 1; L <= 4; ++L)
          if (spec.list == (uint32_t)L && NC.need[L] && (spec.pos - C.head[L]) < (endpos[L] - C.head[L])) spec_ok = false;
      }
#pragma unroll
      for (int L = 1; L <= 4; ++L) C.head[L] = endpos[L];
      if (!hold) { C.tail[L_T1] += NC.pt1; C.tail[L_T2] += (uint32_t)k - NC.pt1; }
      C.tail[L_B1] += NC.g1;
      C.tail[L_B2] += NC.need[L_T2];
      C.t1 = RS[0]; C.t2 = RS[1]; C.b1 = RS[2]; C.b2 = RS[3]; C.p = RS[4]; C.next_fresh = RS[5];
      C.elig1 = RS[6]; C.elig2 = RS[7];
      j += k;
      dbg[DBG_WIN_GENERAL]++; dbg[DBG_ACC_GENERAL_WIN] += (unsigned)k;
      dbg[DBG_CYC_APPLY] += (uint32_t)clock() - tw3;
      PROBE(11);                                                     // apply of a general window
    }
  }
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    const uint32_t t = __reduce_add_sync(FULL, my_cls[i]);
    if (lane == 0) S.red[warp][i] = t;
  }
  if (tid == 0) S.ctl_done = 1;
  cta_sync<PIPE>();                                                  // the scanners leave; the last window's writes are done
  if (PIPE) {                                                        // so does the roller warp
    if (have_prov) roll_wait();
    if (tid == 0) S.req.quit = 1;
    roll_send();
  }
  if (tid == 0) {
#pragma unroll
    for (int w = 0; w < WIDE_WARPS; ++w) {
      C.stat[ST_MISS] += S.red[w][0]; C.stat[ST_HIT_T1] += S.red[w][1]; C.stat[ST_HIT_T2] += S.red[w][2];
      C.stat[ST_GHOST_B1] += S.red[w][3]; C.stat[ST_GHOST_B2] += S.red[w][4];
    }
  }
  dbg[DBG_CYC_TOTAL] = (uint32_t)clock() - t_begin;
  if (tid == 0) {
    P.state->win_seq = win_seq;
    ctx_store(C, P);
#pragma unroll
    for (int i = 0; i < DBG_COUNT; ++i) P.state->dbg[i] += dbg[i];
  }
}

// PIPE: 8 warps as above plus the four roller warps (384 threads); plain: 8 warps, every owner warp rolls for itself.
template <bool LRU, bool HOLD, bool PIPE>
__global__ void __launch_bounds__(2 * WIDE_W + (PIPE ? WIDE_W : 0)) arc_machine_wide_kernel(const __grid_constant__ StepParams P) {
  __shared__ WideShared S;
  wide_machine_run<LRU, HOLD, PIPE>(P, S);
}

template <bool PIPE>
inline void launch_machine_wide(const StepParams& P, cudaStream_t s) {
  const bool lru = P.policy == POLICY_LRU, hold = P.pin_scope == 2;
  constexpr int T = 2 * WIDE_W + (PIPE ? WIDE_W : 0);
  if (lru) { if (hold) arc_machine_wide_kernel<true, true, PIPE><<<1, T, 0, s>>>(P); else arc_machine_wide_kernel<true, false, PIPE><<<1, T, 0, s>>>(P); }
  else { if (hold) arc_machine_wide_kernel<false, true, PIPE><<<1, T, 0, s>>>(P); else arc_machine_wide_kernel<false, false, PIPE><<<1, T, 0, s>>>(P); }
}

}  // namespace arc
