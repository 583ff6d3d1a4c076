// K3, batched form: one warp consumes the step's accesses in the fixed order R2, a *window* of up to 32
// accesses at a time, and produces exactly what the serial walk (machine_serial.cuh) produces.
//
// Why a window can be applied at once:
//  * K2 has already given every access its node id, so the 32 node records are fetched in parallel
//    (one L2 round trip instead of 32 dependent ones); the node ids of the following window are
//    prefetched, and the first 32 ring entries of every list head (the possible victims) travel in the
//    same two round trips.
//  * An access's class is decided by its node's list.  Inside a window the only ways an earlier access
//    can change a later access's class are (1) both touch the same node (the window is cut before the
//    second occurrence), (2) the earlier access evicts / drops the later one's node.  (2) needs the
//    later node's ring position to lie inside the range of ring positions the window's victim scans
//    consume; that is checked, and the window is cut before the first such access.
//  * Given the classes, the counters t1,t2,b1,b2,p and with them every REPLACE decision (R5-R7) follow
//    from a scalar recurrence that every lane rolls forward in registers (no memory access).  The pin
//    fallback of R7 is part of the recurrence: elig1 / elig2 count the entries of T1 / T2 that the
//    current request may still evict.  Runs of equal classes whose decisions are provably identical
//    (hits; misses at the fixed points of the recurrence) are rolled in O(1).
//  * The j-th eviction from list L takes the j-th live entry from L's LRU end: a 32-wide scan of the
//    lazy-FIFO ring with ballot/popc ranks; entries pushed by the current request sit at positions
//    >= bound[L] and are therefore never reached (pins, R4).
//  * If a ghost list cannot supply a drop from the entries it held before the window, the window is cut
//    before that access and the access is done by the by-the-book single-access routine.
// Windows never cross a request boundary (the pin scope changes there).
#pragma once
#include "machine_serial.cuh"

namespace arc {

struct Roll {
  int32_t t1, t2, b1, b2, p, nf, e1, e2;
  uint32_t s0, s1;     // eviction source of access i, bit-sliced: 0 none, 1 T1 -> B1, 2 T2 -> B2, 3 T1 without a ghost
  uint32_t d1, d2;     // access i drops the LRU ghost of B1 / B2
  uint32_t fm;         // access i takes a fresh block id
  int32_t my_p;        // p after this lane's access
  uint32_t err;
  uint32_t calls, phases;   // diagnostics
  bool dbl;                 // DBL policy: p never moves
};

__device__ __forceinline__ uint32_t bits_from(int i, int n) { return ((n >= 32) ? 0xFFFFFFFFu : ((1u << n) - 1u)) << i; }

// R7 with pins: the preferred list if it still has an entry this request may evict, else the other one.
__device__ __forceinline__ void roll_replace(Roll& R, bool inb2, int i) {
  const bool prefer1 = R.t1 >= 1 && (R.t1 > R.p || (inb2 && R.t1 == R.p));
  const bool from1 = prefer1 ? (R.e1 > 0) : !(R.e2 > 0);
  if (from1) { R.s0 |= 1u << i; R.t1--; R.b1++; R.e1--; if (R.e1 < 0) R.err = DEV_ERR_NO_VICTIM; }
  else { R.s1 |= 1u << i; R.t2--; R.b2++; R.e2--; }
}

// The counter recurrence of R5-R7 / R10 over the first k accesses of the window.  (m0, m1, m2) = the node lists,
// bit-sliced; me = the access is a hit on an entry that was still evictable (below bound).  Uniform across lanes.
__device__ __forceinline__ Roll roll_init(const SerialCtx& C) {
  Roll R;
  R.t1 = C.t1; R.t2 = C.t2; R.b1 = C.b1; R.b2 = C.b2; R.p = C.p; R.nf = C.next_fresh; R.e1 = C.elig1; R.e2 = C.elig2;
  R.s0 = R.s1 = R.d1 = R.d2 = R.fm = 0; R.my_p = C.p; R.err = 0; R.calls = 0; R.phases = 0; R.dbl = C.dbl;
  return R;
}

// One phase of a run of m ghost hits starting at window position i (ARC).  Returns the number of accesses it covers.
__device__ __forceinline__ int phase_ghost(Roll& R, int32_t c, uint32_t li, int i, int m, int lane) {
  int n = 1;
  if (R.dbl) {
    // DBL: p is frozen.  B1: REPLACE prefers T1 while t1 > p; B2: while t1 >= max(p, 1).  Victims from T1 shrink t1 by one
    // per step (regime a), victims from T2 change nothing that REPLACE looks at (regime b).
    const bool inb2 = (li == L_B2);
    const bool pref1 = inb2 ? (R.t1 >= 1 && R.t1 >= R.p) : (R.t1 > R.p);
    const bool ra = pref1 && R.e1 > 0, rb = !pref1 && R.e2 > 0;
    if (ra || rb) {
      n = ra ? min(min(m, R.e1), inb2 ? (R.t1 - max(R.p, 1) + 1) : (R.t1 - R.p)) : min(m, R.e2);
      const uint32_t run = bits_from(i, n);
      R.s0 |= ra ? run : 0u; R.s1 |= ra ? 0u : run;
      R.e1 -= ra ? n : 0; R.e2 -= ra ? 0 : n;
      R.t1 -= ra ? n : 0; R.t2 += ra ? n : 0;
      const int32_t db1 = (!inb2 && !ra) ? -n : ((inb2 && ra) ? n : 0);   // B1+T2: b1 -= n, b2 += n; B2+T1: b1 += n, b2 -= n
      R.b1 += db1; R.b2 -= db1;
    } else {
      roll_replace(R, inb2, i);
      if (inb2) R.b2--; else R.b1--;
      R.t2++;
    }
    return n;
  }
  // Ghost hit (R5 cases 2, 3).  A run of ghost hits in the same list is rolled in O(1) for as long as (1) delta, the step
  // of p, keeps its value d and (2) the victim keeps coming from the same list.  The regime and its length are computed
  // with selects (one warp has no other warp to hide a branch behind); anything else is one by-the-book step.
  //   bx = the list that was hit, by = the other ghost list.  d = max(1, by / bx) (R6).
  //   victims from T1 while hitting B2, or from T2 while hitting B1, move one entry from bx's side to by's side per step:
  //   bx -= 1, by += 1, and d stays the same for the steps j with (by + j) < (d + 1)(bx - j); the other two combinations
  //   leave b1, b2 and with them d alone.
  //   R7's fallback is part of the regimes: a list with nothing left to evict (e = 0) stays that way, so once the
  //   preferred list is exhausted the victims come from the other one whatever the preference does.
  const bool inb2 = (li == L_B2);
  const int32_t bx = inb2 ? R.b2 : R.b1, by = inb2 ? R.b1 : R.b2;
  const int32_t p0 = R.p;
  int32_t d = 1, n_delta;
  if (by < 2 * bx) {
    n_delta = (2 * bx - by + 2) / 3;
  } else {
    d = by / max(bx, 1);
    n_delta = (bx - (by - d * bx) + d + 1) / (d + 2);             // ((d + 1) bx - by + d + 1) / (d + 2), without the overflow
  }
  // the preference of REPLACE at the run's first step, and for how many steps it keeps it
  //   B1: p rises by d, T1 is preferred at step j iff t1_j > p + (j + 1) d
  //   B2: p falls by d, T1 is preferred at step j iff t1_j >= 1 and t1_j >= p - (j + 1) d
  const bool pref1 = inb2 ? (R.t1 >= 1 && R.t1 >= R.p - d) : (R.t1 > R.p + d);
  const bool from1 = pref1 ? (R.e1 > 0) : !(R.e2 > 0);              // R7 with its fallback, first step
  const bool ok = from1 ? (R.e1 > 0) : (R.e2 > 0);
  int32_t keep;                                                     // steps for which the victim's list cannot change
  if (from1) {
    // victims from T1: t1 falls by one per step.  Forced (T2 exhausted): no limit from the preference.
    // B1: preferred while t1 - j > p + (j + 1) d, i.e. (t1 - p) / (d + 1) steps; B2: the preference only gets stronger.
    keep = (R.e2 > 0 && !inb2) ? ((d == 1) ? (R.t1 - R.p) / 2 : (R.t1 - R.p) / (d + 1)) : R.e1;
    keep = min(keep, R.e1);
    if (inb2) keep = min(keep, n_delta);                            // B2 + T1: b2 -= 1, b1 += 1
  } else {
    // victims from T2: t1 stays.  Forced (T1 exhausted): no limit.  B1: p only rises, T1 stays unpreferred.
    // B2: unpreferred while t1 < p - (j + 1) d, i.e. (p - t1 - 1) / d steps (t1 = 0: for ever).
    keep = (R.e1 > 0 && inb2 && R.t1 >= 1) ? ((d == 1) ? (R.p - R.t1 - 1) : (R.p - R.t1 - 1) / d) : R.e2;
    keep = min(keep, R.e2);
    if (!inb2) keep = min(keep, n_delta);                           // B1 + T2: b1 -= 1, b2 += 1
  }
  if (ok && keep >= 1) {
    n = min(m, keep);
    const uint32_t run = bits_from(i, n);
    R.s0 |= from1 ? run : 0u; R.s1 |= from1 ? 0u : run;
    R.e1 -= from1 ? n : 0; R.e2 -= from1 ? 0 : n;
    R.t1 -= from1 ? n : 0; R.t2 += from1 ? n : 0;
    // ghost list sizes: B1+T1 none; B1+T2: b1 -= n, b2 += n; B2+T1: b1 += n, b2 -= n; B2+T2: none
    const int32_t db1 = (!inb2 && !from1) ? -n : ((inb2 && from1) ? n : 0);
    R.b1 += db1; R.b2 -= db1;
    const long long dd = d;                                         // n d can exceed 32 bits when one ghost list is tiny
    R.p = inb2 ? (int32_t)max(0ll, p0 - n * dd) : (int32_t)min((long long)c, p0 + n * dd);
    if (lane >= i) { const int32_t t = min(lane - i + 1, n); R.my_p = inb2 ? (int32_t)max(0ll, p0 - t * dd) : (int32_t)min((long long)c, p0 + t * dd); }
  } else {
    R.p = inb2 ? max(0, R.p - d) : min(c, R.p + d);
    roll_replace(R, inb2, i);
    if (inb2) R.b2--; else R.b1--;
    R.t2++;
    if (lane >= i) R.my_p = R.p;
  }
  return n;
}

// One phase of a run of m misses starting at window position i (ARC).  Returns the number of accesses it covers.
__device__ __forceinline__ int phase_miss(Roll& R, int32_t c, int i, int m) {
  // the steady state first, on its own short path: full cache, case 4A, T1 above its target, enough evictable entries
  // for the whole run: drop B1's LRU ghost, evict T1's LRU entry, no counter moves
  if (R.t1 + R.t2 == c && R.t1 + R.b1 == c && R.t1 < c && R.t1 > R.p && R.e1 >= m) {
    const uint32_t run = bits_from(i, m);
    R.s0 |= run; R.d1 |= run; R.e1 -= m;
    return m;
  }
  int n = 1;
  // Miss (R5 case 4), same idea.  fill: the cache is not full yet (b1 = b2 = 0, I7).  r1: REPLACE takes T1's LRU
  // entry (t1 stays); r2: REPLACE takes T2's LRU entry and T1 grows by one per miss.  REPLACE prefers T1 while t1 > p;
  // R7's fallback is part of the regimes: a list with nothing left to evict stays that way, so with T2 exhausted the
  // victims come from T1 whatever the preference (r1), with T1 exhausted from T2 (r2).
  // In case 4A (t1 + b1 = c) B1's LRU ghost is dropped; in case 4B B2's LRU ghost is dropped while b1 + b2 = c.
  const bool fill = R.t1 + R.t2 < c;
  const int32_t gapA = c - R.t1 - R.b1, gapS = c - R.b1 - R.b2;
  const bool isA = gapA == 0, isS = gapS == 0;
  const bool pref1 = R.t1 > R.p;
  const bool r1 = !fill && R.t1 < c && R.e1 > 0 && (pref1 || R.e2 <= 0);
  const bool r2 = !fill && R.t1 < c && R.e2 > 0 && (!pref1 || R.e1 <= 0);
  const int32_t lim_gap = isA ? m : (isS ? gapA : min(gapA, gapS));     // steps until the case changes
  const int32_t nf = min(m, c - R.t1 - R.t2);
  const int32_t n1 = min(min(m, R.e1), lim_gap);
  // r2 by preference lasts until t1 passes p; r2 because T1 is exhausted has no such end
  const int32_t n2 = min(min(min(m, R.e2), lim_gap), min((!pref1 && R.e1 > 0) ? (R.p - R.t1 + 1) : m, c - R.t1));
  if (fill || r1 || r2) {
    n = fill ? nf : (r1 ? n1 : n2);
    const uint32_t run = bits_from(i, n);
    R.fm |= fill ? run : 0u;
    R.s0 |= r1 ? run : 0u; R.s1 |= r2 ? run : 0u;
    R.d1 |= (!fill && isA) ? run : 0u; R.d2 |= (!fill && !isA && isS) ? run : 0u;
    R.nf += fill ? n : 0;
    R.e1 -= r1 ? n : 0; R.e2 -= r2 ? n : 0;
    R.t1 += (fill || r2) ? n : 0; R.t2 -= r2 ? n : 0;
    // r1: 4A nothing, 4B b1 += n and (b1 + b2 = c) b2 -= n.   r2: 4A b1 -= n, b2 += n; 4B (b1 + b2 < c) b2 += n
    R.b1 += (r1 && !isA) ? n : ((r2 && isA) ? -n : 0);
    R.b2 += (r1 && !isA && isS) ? -n : ((r2 && (isA || !isS)) ? n : 0);
  } else {                                // pin fallback, or T1 holding everything: one by-the-book step
    if (isA) {
      if (R.t1 < c) { R.d1 |= 1u << i; R.b1--; roll_replace(R, false, i); }
      else { R.s0 |= 1u << i; R.s1 |= 1u << i; R.t1--; R.e1--; if (R.e1 < 0) R.err = DEV_ERR_NO_VICTIM; }
    } else {
      if (isS) { R.d2 |= 1u << i; R.b2--; }
      roll_replace(R, false, i);          // t1 + t2 + b1 + b2 >= c here because the cache is full
    }
    R.t1++;
  }
  return n;
}

// One phase of a run of m misses in LRU mode (R10).
__device__ __forceinline__ int phase_lru_miss(Roll& R, int32_t c, int i, int m) {
  int n;
  if (R.t1 < c) {                           // cold fill
    n = min(m, c - R.t1); R.fm |= bits_from(i, n); R.t1 += n; R.nf += n;
  } else {                                  // full: every miss evicts T1's LRU entry, no ghost
    n = max(1, min(m, R.e1));
    R.s0 |= bits_from(i, n); R.s1 |= bits_from(i, n); R.e1 -= n;
    if (R.e1 < 0) R.err = DEV_ERR_NO_VICTIM;
  }
  return n;
}

// Rolls k (<= 32) accesses from the state in R; the decision masks of these accesses replace those in R.  lane = this
// thread's index among the k accesses (my_p is captured for it), or >= 32 when the thread owns none of them.
// Deliberately NOT inlined: K3 runs one CTA, so instruction fetch is never hidden by other warps and the kernel has to
// stay inside the instruction cache; this is the one large routine and it is called up to eight times per window.
__device__ __noinline__ void roll_chunk(Roll& Rio, int32_t c, bool lru, uint32_t m0, uint32_t m1, uint32_t m2,
                                        uint32_t me, int k, int lane) {
  Roll R = Rio;
  R.s0 = R.s1 = R.d1 = R.d2 = R.fm = 0; R.my_p = R.p;
  R.calls++;
  const uint32_t km = bits_from(0, k);
  int i = 0;
  while (i < k) {
    R.phases++;
    const uint32_t li = ((m0 >> i) & 1u) | (((m1 >> i) & 1u) << 1) | (((m2 >> i) & 1u) << 2);
    // length of the run of accesses with this same list code (ARC: hits in T1 and in T2 form one run)
    const bool arc_hit = !lru && (li == L_T1 || li == L_T2);
    const uint32_t same = (arc_hit ? ((m0 ^ m1) & ~m2) : (((li & 1u) ? m0 : ~m0) & ((li & 2u) ? m1 : ~m1) & ((li & 4u) ? m2 : ~m2))) & km;
    const uint32_t brk = ~(same >> i);
    const int m = brk ? (__ffs(brk) - 1) : 32;
    int n;
    if (lru) {
      if (li == L_T1) { n = m; R.e1 -= __popc(me & bits_from(i, n)); }      // hits: only the evictable count moves
      else n = phase_lru_miss(R, c, i, m);
    } else if (arc_hit) {                     // hits: T1 entries move to T2; evictable entries stop being so
      n = m;
      const uint32_t run = bits_from(i, n);
      const int32_t h1 = __popc(m0 & run);
      R.t1 -= h1; R.t2 += h1; R.e1 -= __popc(me & m0 & run); R.e2 -= __popc(me & m1 & run);
    } else if (li == L_B1 || li == L_B2) {
      n = phase_ghost(R, c, li, i, m, lane);
    } else {
      n = phase_miss(R, c, i, m);
    }
    i += n;
  }
  Rio = R;
}

__device__ __forceinline__ Roll roll_forward(const SerialCtx& C, int32_t c, bool lru, uint32_t m0, uint32_t m1, uint32_t m2,
                                             uint32_t me, int k, int lane) {
  Roll T = roll_init(C);
  roll_chunk(T, c, lru, m0, m1, m2, me, k, lane);
  Roll R = T;
  return R;
}

// The machine itself, run by ONE warp (s_vic: shared memory of that warp, per list the first entries found from the LRU
// end {node, block, slot, position}).  Also the third phase of the one-launch small-step kernel when requests are short.
__device__ __forceinline__ void batched_machine_run(const StepParams& P, uint4 (*s_vic)[32]) {
  const int lane = threadIdx.x & 31;
  const uint32_t FULL = 0xFFFFFFFFu, lt = (1u << lane) - 1u;
  const bool lru = (P.policy == POLICY_LRU);
  const bool hold = (P.pin_scope == 2);
  const int32_t c = P.capacity;
  const int64_t N = (int64_t)P.n_access;
  if (P.state->error == DEV_ERR_NODE_POOL) return;       // K2 could not give every key a node: the step is void (sticky error)
  SerialCtx C;            // identical in every lane
  ctx_load(C, P);
  unsigned long long dbg[DBG_COUNT];
#pragma unroll
  for (int i = 0; i < DBG_COUNT; ++i) dbg[i] = 0;
  const long long t_begin = clock64();

  // node ids are prefetched one window ahead: pre_n = node_acc[pre_base + lane]
  int64_t pre_base = 0;
  uint32_t pre_n = (lane < N) ? P.node_acc[lane] : NODE_NONE;

  // step-wide and held pins: nothing restarts at a request boundary, so the step is one run of accesses and a window may
  // span requests (16 one-block decode appends are one window); the natural-order index of an access then comes from
  // nat_acc[] (see machine_wide.cuh)
  const bool merged = P.pin_scope != 0;
  const uint32_t* nat_acc = reinterpret_cast<const uint32_t*>(P.keys_acc);
  const uint32_t n_groups = merged ? 1u : P.n_req;
  int64_t my_off = 0, my_off1 = 0;
  for (uint32_t r = 0; r < n_groups; ++r) {
    if (!merged && (r & 31u) == 0) {      // block offsets of the next 32 requests, one per lane
      const uint32_t rr = min(r + (uint32_t)lane, P.n_req - 1);
      my_off = P.blk_off[rr]; my_off1 = P.blk_off[rr + 1];
    }
    const int64_t o = merged ? 0 : __shfl_sync(FULL, my_off, r & 31), nb = merged ? N : __shfl_sync(FULL, my_off1, r & 31) - o;
    // step-wide scope: the pins of earlier requests of the step stay.  Held scope (2): accessed nodes leave the rings and
    // come back through arc_release, so every ring entry is a possible victim (bound = tail), no tail of T1 / T2 moves
    // during a step, and elig1 / elig2 (the unheld entries) carry over from step to step in DevState.
    if (!hold && (r == 0 || P.pin_scope == 0)) begin_request(C);
    int64_t j = 0;
    while (j < nb) {
      const int kmax = (int)min((int64_t)32, nb - j);
      int k = kmax;
      const int64_t a0 = o + j;
      const bool act0 = lane < k;
      const long long tw0 = clock64();
      uint32_t n = pre_n;
      if (pre_base != a0) n = (a0 + lane < N) ? P.node_acc[a0 + lane] : NODE_NONE;   // the last window was cut short
      Node rec;
      rec.list = L_FREE; rec.pos = 0; rec.block = -1; rec.slot = 0;
      if (act0) rec = ld_node(P.nodes + n);
      // the first 64 ring entries from every list head travel with the node records (used only by general windows):
      // lane l holds positions qa + 2l and qa + 2l + 1 of each list, qa = head rounded down to even (16-byte aligned load)
      uint32_t limit[5];
      uint4 ent[5];
#pragma unroll
      for (int L = 1; L <= 4; ++L) {
        limit[L] = (L <= 2) ? C.bound[L] : C.tail[L];
        const uint32_t qA = (C.head[L] & ~1u) + 2u * (uint32_t)lane;
        ent[L] = __ldcg(reinterpret_cast<const uint4*>(P.ring[L] + (qA & P.ring_mask)));
      }
      pre_base = a0 + kmax;
      pre_n = (pre_base + lane < N) ? P.node_acc[pre_base + lane] : NODE_NONE;
      // (1) the same node twice: cut before the second occurrence (lane 0 never has an earlier twin)
      const uint32_t twins = __match_any_sync(FULL, act0 ? n : (0xF0000000u | (uint32_t)lane));
      const uint32_t dupm = __ballot_sync(FULL, act0 && (twins & lt));
      if (dupm) { k = __ffs(dupm) - 1; dbg[DBG_CUT_TWIN]++; }
      uint32_t km = bits_from(0, k);
      const uint32_t lst = rec.list & NODE_LIST_MASK;
      const bool held = (rec.list & NODE_HELD) != 0;            // held scope: in no ring, rec.pos = its holds
      const uint32_t m0 = __ballot_sync(FULL, lst & 1u), m1 = __ballot_sync(FULL, lst & 2u), m2 = __ballot_sync(FULL, lst & 4u);
      if (m2 & m0 & km) C.err = DEV_ERR_BAD_NODE;                 // a FREE node reached K3
      const uint32_t hitm = lru ? (m0 & ~m1 & ~m2) : ((m0 ^ m1) & ~m2);   // list T1 (LRU) / T1 or T2 (ARC)
      // hits on entries that were still evictable by this request (below bound): they stop being so
      const uint32_t me = __ballot_sync(FULL, !held && ((lst == L_T1 && (int32_t)(C.bound[L_T1] - rec.pos) > 0) ||
                                                            (lst == L_T2 && (int32_t)(C.bound[L_T2] - rec.pos) > 0)));
      const long long tw1 = clock64();
      dbg[DBG_CYC_FETCH] += (unsigned long long)(tw1 - tw0);

      if ((hitm & km) == km) {
        // ---- every access of the window is a hit: no counter other than t1/t2 moves, nothing is evicted
        const uint32_t t1hits = lru ? 0u : (uint32_t)__popc(m0 & km);
        const uint32_t Lp = lru ? L_T1 : L_T2;
        if (lane < k) {
          const uint32_t q = (lru ? C.tail[L_T1] : C.tail[L_T2]) + (uint32_t)lane;
          if (!held) ring_tomb(P, lst, rec.pos);
          if (hold) {
            st_node(P.nodes + n, Lp | NODE_HELD, held ? rec.pos + 1u : 1u, rec.block, rec.slot);
            P.node_of_block[rec.block] = n;
          } else {
            __stcg((lru ? P.ring[L_T1] : P.ring[L_T2]) + (q & P.ring_mask), ring_ent(n, rec.block));
            st_node(P.nodes + n, Lp, q, rec.block, rec.slot);
          }
          const int64_t out = merged ? (int64_t)__ldcg(nat_acc + a0 + lane) : o + (nb - 1 - (j + lane));
          P.cls[out] = (uint8_t)lst;                               // L_T1 == CLS_HIT_T1, L_T2 == CLS_HIT_T2
          P.block_id[out] = rec.block;
          P.evicted_id[out] = -1;
          P.p_after[out] = C.p;
          P.dropped[a0 + lane] = NODE_NONE;
        }
        if (!hold) { if (lru) C.tail[L_T1] += (uint32_t)k; else C.tail[L_T2] += (uint32_t)k; }
        C.t1 -= (int32_t)t1hits; C.t2 += (int32_t)t1hits;
        C.elig1 -= __popc(me & m0 & km);
        C.elig2 -= __popc(me & m1 & km);
        C.stat[ST_ACCESSES] += (uint32_t)k;
        C.stat[ST_HIT_T1] += lru ? (uint32_t)k : t1hits;
        C.stat[ST_HIT_T2] += lru ? 0u : (uint32_t)k - t1hits;
        j += k;
        __syncwarp();
        dbg[DBG_WIN_HIT]++; dbg[DBG_ACC_HIT_WIN] += (unsigned)k;
        dbg[DBG_CYC_APPLY] += (unsigned long long)(clock64() - tw1);
        continue;
      }

      // ---- general window: roll the counters forward, fetch the victims, check, apply
      Roll R = roll_forward(C, c, lru, m0, m1, m2, me, k, lane);
      const long long tw2 = clock64();
      dbg[DBG_CYC_ROLL] += (unsigned long long)(tw2 - tw1);
      uint32_t need[5], found[5], q0[5], endpos[5];
      need[0] = 0; need[L_T1] = __popc(R.s0); need[L_T2] = __popc(R.s1 & ~R.s0); need[L_B1] = __popc(R.d1); need[L_B2] = __popc(R.d2);
#pragma unroll
      for (int L = 1; L <= 4; ++L) { found[L] = 0; q0[L] = C.head[L] & ~1u; }
      bool first = true;
      for (;;) {
        bool want[5];
        bool any = false;
#pragma unroll
        for (int L = 1; L <= 4; ++L) {
          want[L] = found[L] < need[L] && (int32_t)(limit[L] - q0[L]) > 0;
          any |= want[L];
          if (!first && want[L])               // later rounds: the next 64 ring entries
            ent[L] = __ldcg(reinterpret_cast<const uint4*>(P.ring[L] + ((q0[L] + 2u * (uint32_t)lane) & P.ring_mask)));
        }
        if (!any) break;
        dbg[DBG_SCAN_ROUNDS]++;
#pragma unroll
        for (int L = 1; L <= 4; ++L) {
          if (!want[L]) continue;                                   // warp-uniform
          const uint32_t qA = q0[L] + 2u * (uint32_t)lane, qB = qA + 1u;
          // live = inside [head, limit) and not a tombstone (entries leave a ring only by head consumption or a tombstone)
          const bool liveA = (int32_t)(qA - C.head[L]) >= 0 && (int32_t)(limit[L] - qA) > 0 && ent[L].x != RING_TOMB;
          const bool liveB = (int32_t)(qB - C.head[L]) >= 0 && (int32_t)(limit[L] - qB) > 0 && ent[L].z != RING_TOMB;
          const uint32_t balA = __ballot_sync(FULL, liveA), balB = __ballot_sync(FULL, liveB);
          const uint32_t rankA = found[L] + (uint32_t)__popc(balA & lt) + (uint32_t)__popc(balB & lt);
          const uint32_t rankB = rankA + (liveA ? 1u : 0u);
          if (liveA && rankA < 32u) s_vic[L][rankA] = make_uint4(ent[L].x, ent[L].y, 0u, qA);
          if (liveB && rankB < 32u) s_vic[L][rankB] = make_uint4(ent[L].z, ent[L].w, 0u, qB);
          found[L] += (uint32_t)__popc(balA) + (uint32_t)__popc(balB);
          q0[L] += 64u;
        }
        first = false;
      }
      __syncwarp();
#pragma unroll
      for (int L = 1; L <= 4; ++L) {
        endpos[L] = C.head[L];
        if (need[L]) endpos[L] = (found[L] >= need[L]) ? s_vic[L][need[L] - 1].w + 1u : limit[L];
      }
      // (2) an accessed node whose ring entry lies inside a consumed range, or a victim that does not exist
      bool act = lane < k;
      uint32_t my_src = ((R.s0 >> lane) & 1u) | (((R.s1 >> lane) & 1u) << 1);
      uint32_t srcT1m = R.s0, srcT2m = R.s1 & ~R.s0;
      bool bad = false;
      if (act) {
#pragma unroll
        for (int L = 1; L <= 4; ++L)
          if (lst == (uint32_t)L && !held && need[L] && (rec.pos - C.head[L]) < (endpos[L] - C.head[L])) bad = true;
        if ((my_src & 1u) && (uint32_t)__popc(srcT1m & lt) >= found[L_T1]) bad = true;
        if (my_src == 2 && (uint32_t)__popc(srcT2m & lt) >= found[L_T2]) bad = true;
        if (((R.d1 >> lane) & 1u) && (uint32_t)__popc(R.d1 & lt) >= found[L_B1]) bad = true;
        if (((R.d2 >> lane) & 1u) && (uint32_t)__popc(R.d2 & lt) >= found[L_B2]) bad = true;
      }
      const uint32_t badm = __ballot_sync(FULL, bad);
      const long long tw3 = clock64();
      dbg[DBG_CYC_SCAN] += (unsigned long long)(tw3 - tw2);
      if (badm) {
        k = __ffs(badm) - 1;
        dbg[DBG_CUT_CONFLICT]++;
        if (k == 0) {                       // the by-the-book routine, run identically by every lane
          SerialCtx T = C;                           // the callee is not inlined: keep C itself in registers
          serial_access(T, P, a0, merged ? (int64_t)__ldcg(nat_acc + a0) : o + (nb - 1 - j));
          C = T;
          j += 1;
          __syncwarp();
          dbg[DBG_WIN_SERIAL]++;
          dbg[DBG_CYC_SERIAL] += (unsigned long long)(clock64() - tw3);
          continue;
        }
        km = bits_from(0, k);
        R = roll_forward(C, c, lru, m0, m1, m2, me, k, lane);
        act = lane < k;
        my_src = ((R.s0 >> lane) & 1u) | (((R.s1 >> lane) & 1u) << 1);
        srcT1m = R.s0; srcT2m = R.s1 & ~R.s0;
        need[L_T1] = __popc(R.s0); need[L_T2] = __popc(srcT2m); need[L_B1] = __popc(R.d1); need[L_B2] = __popc(R.d2);
#pragma unroll
        for (int L = 1; L <= 4; ++L) endpos[L] = need[L] ? s_vic[L][need[L] - 1].w + 1u : C.head[L];
      }
      if (R.err) C.err = R.err;
      dbg[DBG_ROLL_CALLS] += R.calls; dbg[DBG_ROLL_PHASES] += R.phases;

      // ---- apply (lanes < k); ranks come from the decision masks
      const uint32_t ghost1m = R.s0 & ~R.s1;                                          // pushes to B1, in access order
      const uint32_t src3m = R.s0 & R.s1;
      const uint32_t pushT1m = lru ? km : (~(m0 | m1 | m2) & km);                     // ABSENT nodes enter T1 (LRU: everything)
      const uint32_t pushT2m = km & ~pushT1m;
      const uint32_t nonhitm = km & ~hitm;
      const uint32_t evictm = srcT1m | srcT2m;
      if (act) {
        const bool is_hit = (hitm >> lane) & 1u;
        const bool my_d1 = (R.d1 >> lane) & 1u, my_d2 = (R.d2 >> lane) & 1u;
        int32_t blk = rec.block, ev = -1;
        uint32_t dropped = NODE_NONE;
        if (my_src) {
          const uint4 v = (my_src == 2) ? s_vic[L_T2][__popc(srcT2m & lt)] : s_vic[L_T1][__popc(srcT1m & lt)];
          blk = ev = (int32_t)v.y;
          if (my_src == 3) {                        // leaves no ghost: the key leaves the directory in K4
            st_node_keep_slot(P.nodes + v.x, L_ABSENT, 0, -1);
            dropped = v.x;
          } else {
            const uint32_t G = (my_src == 1) ? L_B1 : L_B2;
            const uint32_t q = (my_src == 1) ? C.tail[L_B1] + (uint32_t)__popc(ghost1m & lt) : C.tail[L_B2] + (uint32_t)__popc(srcT2m & lt);
            __stcg(((my_src == 1) ? P.ring[L_B1] : P.ring[L_B2]) + (q & P.ring_mask), ring_ent(v.x, -1));
            st_node_keep_slot(P.nodes + v.x, G, q, -1);
          }
        } else if ((R.fm >> lane) & 1u) {
          blk = C.next_fresh + __popc(R.fm & lt);
        }
        if (my_d1 || my_d2) {
          const uint4 d = my_d1 ? s_vic[L_B1][__popc(R.d1 & lt)] : s_vic[L_B2][__popc(R.d2 & lt)];
          st_node_keep_slot(P.nodes + d.x, L_ABSENT, 0, -1);
          dropped = d.x;
        }
        const bool toT1 = (pushT1m >> lane) & 1u;
        const uint32_t Lp = toT1 ? L_T1 : L_T2;
        const uint32_t q = (toT1 ? C.tail[L_T1] : C.tail[L_T2]) + (uint32_t)__popc((toT1 ? pushT1m : pushT2m) & lt);
        if (lst >= L_T1 && lst <= L_B2 && !held) ring_tomb(P, lst, rec.pos);     // the node leaves its old position
        if (hold) {
          st_node(P.nodes + n, Lp | NODE_HELD, held ? rec.pos + 1u : 1u, blk, rec.slot);
          P.node_of_block[blk] = n;
        } else {
          __stcg((toT1 ? P.ring[L_T1] : P.ring[L_T2]) + (q & P.ring_mask), ring_ent(n, blk));
          st_node(P.nodes + n, Lp, q, blk, rec.slot);
        }
        const int64_t out = merged ? (int64_t)__ldcg(nat_acc + a0 + lane) : o + (nb - 1 - (j + lane));
        P.cls[out] = (uint8_t)lst;                    // ABSENT -> MISS(0), T1 -> 1, T2 -> 2, B1 -> 3, B2 -> 4
        P.block_id[out] = blk;
        P.evicted_id[out] = ev;
        P.p_after[out] = R.my_p;
        P.dropped[a0 + lane] = dropped;
        if (!is_hit) P.alloc_ids[C.n_alloc + (uint32_t)__popc(nonhitm & lt)] = blk;
        if (ev >= 0) P.evict_ids[C.n_evict + (uint32_t)__popc(evictm & lt)] = ev;
      }
      // uniform state
      C.stat[ST_ACCESSES] += (uint32_t)k;
      C.stat[ST_HIT_T1] += __popc(hitm & km & m0);
      C.stat[ST_HIT_T2] += lru ? 0u : (uint32_t)__popc(hitm & km & m1);
      C.stat[ST_GHOST_B1] += __popc(m0 & m1 & ~m2 & km);
      C.stat[ST_GHOST_B2] += __popc(m2 & ~m0 & ~m1 & km);
      C.stat[ST_MISS] += __popc(~(m0 | m1 | m2) & km);
      C.stat[ST_EVICT_T1] += need[L_T1];
      C.stat[ST_EVICT_T2] += need[L_T2];
      C.stat[ST_DROP_B1] += need[L_B1];
      C.stat[ST_DROP_B2] += need[L_B2];
      C.stat[ST_FRESH] += (uint32_t)(R.nf - C.next_fresh);
      C.n_alloc += __popc(nonhitm);
      C.n_evict += __popc(evictm);
#pragma unroll
      for (int L = 1; L <= 4; ++L) C.head[L] = endpos[L];
      if (!hold) { C.tail[L_T1] += __popc(pushT1m); C.tail[L_T2] += __popc(pushT2m); }
      C.tail[L_B1] += __popc(ghost1m);
      C.tail[L_B2] += need[L_T2];
      (void)src3m;
      C.t1 = R.t1; C.t2 = R.t2; C.b1 = R.b1; C.b2 = R.b2; C.p = R.p; C.next_fresh = R.nf;
      C.elig1 = R.e1; C.elig2 = R.e2;
      j += k;
      __syncwarp();
      dbg[DBG_WIN_GENERAL]++; dbg[DBG_ACC_GENERAL_WIN] += (unsigned)k;
      dbg[DBG_CYC_APPLY] += (unsigned long long)(clock64() - tw3);
    }
  }
  dbg[DBG_CYC_TOTAL] = (unsigned long long)(clock64() - t_begin);
  if (lane == 0) {
    ctx_store(C, P);
#pragma unroll
    for (int i = 0; i < DBG_COUNT; ++i) P.state->dbg[i] += dbg[i];
  }
}

__global__ void __launch_bounds__(32) arc_machine_batched_kernel(const __grid_constant__ StepParams P) {
  __shared__ uint4 s_vic[5][32];
  batched_machine_run(P, s_vic);
}

inline void launch_machine_batched(const StepParams& P, cudaStream_t s) { arc_machine_batched_kernel<<<1, 32, 0, s>>>(P); }

}  // namespace arc
