// K3, batched form: one warp consumes the step's accesses in the fixed order R2, a *window* of up to 32
// accesses at a time, and produces exactly what the serial walk (machine_serial.cuh) produces.
//
// Why a window can be applied at once:
//  * K2 has already given every access its node id, so the 32 node records are fetched in parallel
//    (one L2 round trip instead of 32 dependent ones).
//  * An access's class is decided by its node's list.  Inside a window the only ways an earlier access
//    can change a later access's class are (1) both touch the same node (the window is cut before the
//    second occurrence), (2) the earlier access evicts / drops the later one's node.  (2) needs the
//    later node's ring position to lie inside the range of ring positions the window's victim scans
//    consume; that is checked, and the window is cut before the first such access.
//  * Given the classes, the counters t1,t2,b1,b2,p and with them every REPLACE decision (R5-R7) follow
//    from a scalar recurrence that every lane rolls forward in registers (no memory access).
//  * The j-th eviction from list L takes the j-th live entry from L's LRU end: a 32-wide scan of the
//    lazy-FIFO ring with ballot/popc ranks; entries pushed by the current request sit at positions
//    >= bound[L] and are therefore never reached (pins, R4).
//  * If a list cannot supply the victims the recurrence assumed (the pin fallback of R7), the window is cut
//    before that access and the access is done by the by-the-book single-access routine.
// Windows never cross a request boundary (the pin scope changes there).
#pragma once
#include "machine_serial.cuh"

namespace arc {

struct Roll {
  int32_t t1, t2, b1, b2, p, nf;
  uint32_t my_src;    // 0 none / fresh id, 1 T1 -> B1, 2 T2 -> B2, 3 T1 without a ghost
  uint32_t my_drop;   // 0, L_B1, L_B2
  int32_t my_p, my_fresh;
};

// The counter recurrence of R5-R7 / R10 over the first k accesses of the window whose node lists are given
// bit-sliced in (m0, m1, m2).  Every lane runs it identically; lane i keeps the decisions of access i.
__device__ __forceinline__ Roll roll_forward(const SerialCtx& C, int32_t c, bool lru, uint32_t m0, uint32_t m1, uint32_t m2,
                                             int k, int lane) {
  Roll R;
  R.t1 = C.t1; R.t2 = C.t2; R.b1 = C.b1; R.b2 = C.b2; R.p = C.p; R.nf = C.next_fresh;
  R.my_src = 0; R.my_drop = 0; R.my_p = C.p; R.my_fresh = -1;
  for (int i = 0; i < k; ++i) {
    const uint32_t li = ((m0 >> i) & 1u) | (((m1 >> i) & 1u) << 1) | (((m2 >> i) & 1u) << 2);
    uint32_t src = 0, drop = 0;
    int32_t fresh = -1;
    if (lru) {
      if (li != L_T1) {
        if (R.t1 < c) { fresh = R.nf++; R.t1++; } else src = 3;
      }
    } else if (li == L_T1) {
      R.t1--; R.t2++;
    } else if (li == L_T2) {
    } else if (li == L_B1 || li == L_B2) {
      const bool inb2 = (li == L_B2);
      int32_t delta = inb2 ? (R.b1 / max(R.b2, 1)) : (R.b2 / max(R.b1, 1));
      delta = max(delta, 1);
      R.p = inb2 ? max(0, R.p - delta) : min(c, R.p + delta);
      const bool from_t1 = R.t1 >= 1 && (R.t1 > R.p || (inb2 && R.t1 == R.p));
      if (from_t1) { src = 1; R.t1--; R.b1++; } else { src = 2; R.t2--; R.b2++; }
      if (inb2) R.b2--; else R.b1--;
      R.t2++;
    } else {
      bool repl = false;
      if (R.t1 + R.b1 == c) {
        if (R.t1 < c) { drop = L_B1; R.b1--; repl = true; } else { src = 3; R.t1--; }
      } else {
        const int32_t tot = R.t1 + R.t2 + R.b1 + R.b2;
        if (tot >= c) { if (tot == 2 * c) { drop = L_B2; R.b2--; } repl = true; }
        else fresh = R.nf++;
      }
      if (repl) {
        if (R.t1 >= 1 && R.t1 > R.p) { src = 1; R.t1--; R.b1++; } else { src = 2; R.t2--; R.b2++; }
      }
      R.t1++;
    }
    if (i == lane) { R.my_src = src; R.my_drop = drop; R.my_p = R.p; R.my_fresh = fresh; }
  }
  return R;
}

__global__ void __launch_bounds__(32) arc_machine_batched_kernel(StepParams P) {
  __shared__ uint4 s_vic[5][32];    // per list: the first entries found from the LRU end {node, block, slot, position}
  const int lane = threadIdx.x;
  const uint32_t FULL = 0xFFFFFFFFu, lt = (1u << lane) - 1u;
  const bool lru = (P.policy == POLICY_LRU);
  const int32_t c = P.capacity;
  SerialCtx C;            // identical in every lane
  ctx_load(C, P);

  int64_t my_off = 0, my_off1 = 0;
  for (uint32_t r = 0; r < P.n_req; ++r) {
    if ((r & 31u) == 0) {      // block offsets of the next 32 requests, one per lane
      const uint32_t rr = min(r + (uint32_t)lane, P.n_req - 1);
      my_off = P.blk_off[rr]; my_off1 = P.blk_off[rr + 1];
    }
    const int64_t o = __shfl_sync(FULL, my_off, r & 31), nb = __shfl_sync(FULL, my_off1, r & 31) - o;
    C.bound[L_T1] = C.tail[L_T1];
    C.bound[L_T2] = C.tail[L_T2];
    int64_t j = 0;
    while (j < nb) {
      int k = (int)min((int64_t)32, nb - j);
      const int64_t a0 = o + j;
      const bool act0 = lane < k;
      const uint32_t n = act0 ? P.node_acc[a0 + lane] : NODE_NONE;
      Node rec;
      rec.list = L_FREE; rec.pos = 0; rec.block = -1; rec.slot = 0;
      if (act0) rec = ld_node(P.nodes + n);
      // (1) the same node twice: cut before the second occurrence (lane 0 never has an earlier twin)
      const uint32_t twins = __match_any_sync(FULL, act0 ? n : (0xF0000000u | (uint32_t)lane));
      const uint32_t dupm = __ballot_sync(FULL, act0 && (twins & lt));
      if (dupm) k = __ffs(dupm) - 1;
      uint32_t km = (k == 32) ? FULL : ((1u << k) - 1u);
      const uint32_t lst = rec.list;
      const uint32_t m0 = __ballot_sync(FULL, lst & 1u), m1 = __ballot_sync(FULL, lst & 2u), m2 = __ballot_sync(FULL, lst & 4u);
      if (m2 & m0 & km) C.err = DEV_ERR_BAD_NODE;                 // a FREE node reached K3
      const uint32_t hitm = lru ? (m0 & ~m1 & ~m2) : ((m0 ^ m1) & ~m2);   // list T1 (LRU) / T1 or T2 (ARC)

      if ((hitm & km) == km) {
        // ---- every access of the window is a hit: no counter other than t1/t2 moves, nothing is evicted
        const uint32_t t1hits = lru ? 0u : (uint32_t)__popc(m0 & km);
        const uint32_t Lp = lru ? L_T1 : L_T2;
        if (lane < k) {
          const uint32_t q = (lru ? C.tail[L_T1] : C.tail[L_T2]) + (uint32_t)lane;
          (lru ? P.ring[L_T1] : P.ring[L_T2])[q & P.ring_mask] = n;
          st_node(P.nodes + n, Lp, q, rec.block, rec.slot);
          const int64_t out = o + (nb - 1 - (j + lane));
          P.cls[out] = (uint8_t)lst;                               // L_T1 == CLS_HIT_T1, L_T2 == CLS_HIT_T2
          P.block_id[out] = rec.block;
          P.evicted_id[out] = -1;
          P.p_after[out] = C.p;
          P.dropped[a0 + lane] = NODE_NONE;
        }
        if (lru) C.tail[L_T1] += (uint32_t)k; else C.tail[L_T2] += (uint32_t)k;
        C.t1 -= (int32_t)t1hits; C.t2 += (int32_t)t1hits;
        C.stat[ST_ACCESSES] += (uint32_t)k;
        C.stat[ST_HIT_T1] += lru ? (uint32_t)k : t1hits;
        C.stat[ST_HIT_T2] += lru ? 0u : (uint32_t)k - t1hits;
        j += k;
        __syncwarp();
        continue;
      }

      // ---- general window: roll the counters forward, fetch the victims, check, apply
      Roll R = roll_forward(C, c, lru, m0, m1, m2, k, lane);
      bool act = lane < k;
      uint32_t srcT1m = __ballot_sync(FULL, act && (R.my_src == 1 || R.my_src == 3));
      uint32_t srcT2m = __ballot_sync(FULL, act && R.my_src == 2);
      uint32_t drop1m = __ballot_sync(FULL, act && R.my_drop == L_B1);
      uint32_t drop2m = __ballot_sync(FULL, act && R.my_drop == L_B2);
      uint32_t need[5], found[5], q0[5], limit[5], endpos[5];
      need[0] = 0; need[L_T1] = __popc(srcT1m); need[L_T2] = __popc(srcT2m); need[L_B1] = __popc(drop1m); need[L_B2] = __popc(drop2m);
#pragma unroll
      for (int L = 1; L <= 4; ++L) { found[L] = 0; q0[L] = C.head[L]; limit[L] = (L <= 2) ? C.bound[L] : C.tail[L]; }
      for (;;) {
        bool want[5], valid[5];
        uint32_t ent[5];
        Node vr[5];
        bool any = false;
#pragma unroll
        for (int L = 1; L <= 4; ++L) {
          want[L] = found[L] < need[L] && q0[L] != limit[L];
          any |= want[L];
          const uint32_t q = q0[L] + (uint32_t)lane;
          valid[L] = want[L] && (int32_t)(limit[L] - q) > 0;
          ent[L] = valid[L] ? __ldcg(P.ring[L] + (q & P.ring_mask)) : 0u;
        }
        if (!any) break;
#pragma unroll
        for (int L = 1; L <= 4; ++L) {
          vr[L].list = L_FREE; vr[L].pos = 0; vr[L].block = -1; vr[L].slot = 0;
          if (valid[L]) vr[L] = ld_node(P.nodes + ent[L]);
        }
#pragma unroll
        for (int L = 1; L <= 4; ++L) {
          if (!want[L]) continue;                                   // warp-uniform
          const uint32_t q = q0[L] + (uint32_t)lane;
          const bool live = valid[L] && vr[L].list == (uint32_t)L && vr[L].pos == q;
          const uint32_t bal = __ballot_sync(FULL, live);
          const uint32_t rank = found[L] + (uint32_t)__popc(bal & lt);
          if (live && rank < 32u) s_vic[L][rank] = make_uint4(ent[L], (uint32_t)vr[L].block, vr[L].slot, q);
          found[L] += (uint32_t)__popc(bal);
          q0[L] = ((int32_t)(limit[L] - (q0[L] + 32u)) > 0) ? q0[L] + 32u : limit[L];
        }
      }
      __syncwarp();
#pragma unroll
      for (int L = 1; L <= 4; ++L) {
        endpos[L] = C.head[L];
        if (need[L]) endpos[L] = (found[L] >= need[L]) ? s_vic[L][need[L] - 1].w + 1u : limit[L];
      }
      // (2) an accessed node whose ring entry lies inside a consumed range, or a victim that does not exist
      bool bad = false;
      if (act) {
#pragma unroll
        for (int L = 1; L <= 4; ++L)
          if (lst == (uint32_t)L && need[L] && (rec.pos - C.head[L]) < (endpos[L] - C.head[L])) bad = true;
        if ((R.my_src == 1 || R.my_src == 3) && (uint32_t)__popc(srcT1m & lt) >= found[L_T1]) bad = true;
        if (R.my_src == 2 && (uint32_t)__popc(srcT2m & lt) >= found[L_T2]) bad = true;
        if (R.my_drop == L_B1 && (uint32_t)__popc(drop1m & lt) >= found[L_B1]) bad = true;
        if (R.my_drop == L_B2 && (uint32_t)__popc(drop2m & lt) >= found[L_B2]) bad = true;
      }
      const uint32_t badm = __ballot_sync(FULL, bad);
      if (badm) {
        k = __ffs(badm) - 1;
        if (k == 0) {                       // the by-the-book routine, run identically by every lane
          serial_access(C, P, a0, o + (nb - 1 - j));
          j += 1;
          __syncwarp();
          continue;
        }
        km = (1u << k) - 1u;
        R = roll_forward(C, c, lru, m0, m1, m2, k, lane);
        act = lane < k;
        srcT1m = __ballot_sync(FULL, act && (R.my_src == 1 || R.my_src == 3));
        srcT2m = __ballot_sync(FULL, act && R.my_src == 2);
        drop1m = __ballot_sync(FULL, act && R.my_drop == L_B1);
        drop2m = __ballot_sync(FULL, act && R.my_drop == L_B2);
        need[L_T1] = __popc(srcT1m); need[L_T2] = __popc(srcT2m); need[L_B1] = __popc(drop1m); need[L_B2] = __popc(drop2m);
#pragma unroll
        for (int L = 1; L <= 4; ++L) endpos[L] = need[L] ? s_vic[L][need[L] - 1].w + 1u : C.head[L];
      }

      // ---- apply (lanes < k); ranks come from the ballots
      const uint32_t ghost1m = __ballot_sync(FULL, act && R.my_src == 1);            // pushes to B1, in access order
      const uint32_t pushT1m = lru ? km : (~(m0 | m1 | m2) & km);                     // ABSENT nodes enter T1 (LRU: everything)
      const uint32_t pushT2m = km & ~pushT1m;
      const uint32_t nonhitm = km & ~hitm;
      const uint32_t evictm = srcT1m | srcT2m;
      if (act) {
        const bool is_hit = (hitm >> lane) & 1u;
        int32_t blk = rec.block, ev = -1;
        uint32_t dropped = NODE_NONE;
        if (R.my_src) {
          const uint32_t Ls = (R.my_src == 2) ? L_T2 : L_T1;
          const uint4 v = s_vic[Ls][__popc(((R.my_src == 2) ? srcT2m : srcT1m) & lt)];
          blk = ev = (int32_t)v.y;
          if (R.my_src == 3) {                      // leaves no ghost: the key leaves the directory in K4
            st_node(P.nodes + v.x, L_ABSENT, 0, -1, v.z);
            dropped = v.x;
          } else {
            const uint32_t G = (R.my_src == 1) ? L_B1 : L_B2;
            const uint32_t q = ((R.my_src == 1) ? C.tail[L_B1] : C.tail[L_B2]) + (uint32_t)__popc(((R.my_src == 1) ? ghost1m : srcT2m) & lt);
            ((R.my_src == 1) ? P.ring[L_B1] : P.ring[L_B2])[q & P.ring_mask] = v.x;
            st_node(P.nodes + v.x, G, q, -1, v.z);
          }
        } else if (!is_hit) {
          blk = R.my_fresh;
        }
        if (R.my_drop) {
          const uint4 d = s_vic[R.my_drop][__popc(((R.my_drop == L_B1) ? drop1m : drop2m) & lt)];
          st_node(P.nodes + d.x, L_ABSENT, 0, -1, d.z);
          dropped = d.x;
        }
        const bool toT1 = (pushT1m >> lane) & 1u;
        const uint32_t Lp = toT1 ? L_T1 : L_T2;
        const uint32_t q = (toT1 ? C.tail[L_T1] : C.tail[L_T2]) + (uint32_t)__popc((toT1 ? pushT1m : pushT2m) & lt);
        (toT1 ? P.ring[L_T1] : P.ring[L_T2])[q & P.ring_mask] = n;
        st_node(P.nodes + n, Lp, q, blk, rec.slot);
        const int64_t out = o + (nb - 1 - (j + lane));
        P.cls[out] = (uint8_t)lst;                    // ABSENT -> MISS(0), T1 -> 1, T2 -> 2, B1 -> 3, B2 -> 4
        P.block_id[out] = blk;
        P.evicted_id[out] = ev;
        P.p_after[out] = R.my_p;
        P.dropped[a0 + lane] = dropped;
        if (!is_hit) P.alloc_ids[C.n_alloc + (uint32_t)__popc(nonhitm & lt)] = blk;
        if (ev >= 0) P.evict_ids[C.n_evict + (uint32_t)__popc(evictm & lt)] = ev;
      }
      // uniform state
      const uint32_t n3 = __popc(__ballot_sync(FULL, act && R.my_src == 3));
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
      C.tail[L_T1] += __popc(pushT1m);
      C.tail[L_T2] += __popc(pushT2m);
      C.tail[L_B1] += need[L_T1] - n3;
      C.tail[L_B2] += need[L_T2];
      C.t1 = R.t1; C.t2 = R.t2; C.b1 = R.b1; C.b2 = R.b2; C.p = R.p; C.next_fresh = R.nf;
      j += k;
      __syncwarp();
    }
  }
  if (lane == 0) ctx_store(C, P);
}

inline void launch_machine_batched(const StepParams& P, cudaStream_t s) { arc_machine_batched_kernel<<<1, 32, 0, s>>>(P); }

}  // namespace arc
