// K3, serial form: one thread walks the step's accesses in the fixed order R2 and applies R5-R8 (ARC)
// or R10 (LRU) on the ring-list directory.  This is the on-device correctness reference
// (arc_set_machine(h, 1)); the batched machine in machine_batched.cuh must produce identical results.
#pragma once
#include "arc_device.cuh"

namespace arc {

struct SerialCtx {
  uint32_t head[5], tail[5];   // only ever indexed with compile-time constants, so they live in registers
  uint32_t bound[5];     // victim scans stop here: tail of T1/T2 when the request began (R4), current tail for B1/B2
  int32_t t1, t2, b1, b2, p, next_fresh;
  int32_t elig1, elig2;  // live entries of T1 / T2 below bound[] = victims still available to the current request (R4, R7)
  uint32_t stat[ST_COUNT];   // per-step deltas (a step has < 2^31 accesses)
  uint32_t err;
  uint32_t n_alloc, n_evict;
  bool dbl;              // DBL policy: p is frozen at capacity / 2
};

template <uint32_t L>
__device__ __forceinline__ void ring_push(SerialCtx& C, const StepParams& P, uint32_t n, int32_t block, uint32_t slot) {
  const uint32_t q = C.tail[L]++;
  __stcg(P.ring[L] + (q & P.ring_mask), ring_ent(n, block));
  st_node(P.nodes + n, L, q, block, slot);
}

// The accessed node takes its place in list L: at the MRU end of the ring, or (pin scope 2) outside every ring with one
// more hold; holds_before = the holds it had (0 if it was not held).
template <uint32_t L>
__device__ __forceinline__ void place_accessed(SerialCtx& C, const StepParams& P, uint32_t n, int32_t block, uint32_t slot, uint32_t holds_before) {
  if (P.pin_scope == 2) {
    st_node(P.nodes + n, L | NODE_HELD, holds_before + 1u, block, slot);
    P.node_of_block[block] = n;
  } else {
    ring_push<L>(C, P, n, block, slot);
  }
}

// first live entry of list L in [head, bound); advances head past everything it skipped.  NODE_NONE if none.
template <uint32_t L>
__device__ __forceinline__ uint32_t ring_pop_lru(SerialCtx& C, const StepParams& P, uint32_t bound, Node* rec_out) {
  uint32_t q = C.head[L];
  while (q != bound) {
    const uint32_t n = ent_node(__ldcg(P.ring[L] + (q & P.ring_mask)));
    if (n != RING_TOMB) {
      const Node r = ld_node(P.nodes + n);
      if (r.list == L && r.pos == q) { C.head[L] = q + 1; *rec_out = r; return n; }
    }
    ++q;
  }
  C.head[L] = bound;
  return NODE_NONE;
}

// R7.  Returns the freed block id; the victim becomes a ghost at the MRU end of B1 / B2.
__device__ __forceinline__ int32_t replace_serial(SerialCtx& C, const StepParams& P, bool in_b2) {
  const bool prefer_t1 = C.t1 >= 1 && (C.t1 > C.p || (in_b2 && C.t1 == C.p));
  for (int attempt = 0; attempt < 2; ++attempt) {
    const bool from_t1 = (attempt == 0) ? prefer_t1 : !prefer_t1;
    Node r;
    if (from_t1) {
      const uint32_t v = ring_pop_lru<L_T1>(C, P, C.bound[L_T1], &r);
      if (v == NODE_NONE) continue;
      ring_push<L_B1>(C, P, v, -1, r.slot);
      C.t1--; C.b1++; C.elig1--; C.stat[ST_EVICT_T1]++;
    } else {
      const uint32_t v = ring_pop_lru<L_T2>(C, P, C.bound[L_T2], &r);
      if (v == NODE_NONE) continue;
      ring_push<L_B2>(C, P, v, -1, r.slot);
      C.t2--; C.b2++; C.elig2--; C.stat[ST_EVICT_T2]++;
    }
    return r.block;
  }
  C.err = DEV_ERR_NO_VICTIM;
  return -1;
}

// evict the first unpinned entry of T1 without leaving a ghost (case 4A-else, LRU mode); node -> ABSENT
__device__ __forceinline__ int32_t evict_t1_no_ghost_serial(SerialCtx& C, const StepParams& P, uint32_t* dropped) {
  Node r;
  const uint32_t v = ring_pop_lru<L_T1>(C, P, C.bound[L_T1], &r);
  if (v == NODE_NONE) { C.err = DEV_ERR_NO_VICTIM; return -1; }
  st_node(P.nodes + v, L_ABSENT, 0, -1, r.slot);
  *dropped = v;
  C.t1--; C.elig1--; C.stat[ST_EVICT_T1]++;
  return r.block;
}

template <uint32_t L>
__device__ __forceinline__ void drop_ghost_serial(SerialCtx& C, const StepParams& P, uint32_t* dropped) {
  Node r;
  const uint32_t d = ring_pop_lru<L>(C, P, C.tail[L], &r);
  if (d == NODE_NONE) { C.err = DEV_ERR_BAD_NODE; return; }
  st_node(P.nodes + d, L_ABSENT, 0, -1, r.slot);
  *dropped = d;
  if (L == L_B1) { C.b1--; C.stat[ST_DROP_B1]++; } else { C.b2--; C.stat[ST_DROP_B2]++; }
}

// Loads / stores the scalar machine state kept in DevState.
__device__ __forceinline__ void ctx_load(SerialCtx& C, const StepParams& P) {
  const DevState* S = P.state;
#pragma unroll
  for (int L = 1; L <= 4; ++L) { C.head[L] = S->head[L]; C.tail[L] = S->tail[L]; C.bound[L] = S->tail[L]; }
  C.t1 = S->t1; C.t2 = S->t2; C.b1 = S->b1; C.b2 = S->b2; C.p = S->p; C.next_fresh = S->next_fresh;
  C.elig1 = C.t1; C.elig2 = C.t2;
  if (P.pin_scope == 2) { C.elig1 = S->u1; C.elig2 = S->u2; }   // held scope: the unheld entries, whatever step held the others
  C.dbl = (P.policy == POLICY_DBL);
#pragma unroll
  for (int i = 0; i < ST_COUNT; ++i) C.stat[i] = 0;
  C.err = 0;
  C.n_alloc = 0; C.n_evict = 0;
}
__device__ __forceinline__ void ctx_store(const SerialCtx& C, const StepParams& P) {
  DevState* S = P.state;
#pragma unroll
  for (int L = 1; L <= 4; ++L) { S->head[L] = C.head[L]; S->tail[L] = C.tail[L]; }
  S->t1 = C.t1; S->t2 = C.t2; S->b1 = C.b1; S->b2 = C.b2; S->p = C.p; S->next_fresh = C.next_fresh;
  S->counts[0] = C.n_alloc; S->counts[1] = C.n_evict;
  S->u1 = C.elig1; S->u2 = C.elig2;
#pragma unroll
  for (int i = 0; i < ST_COUNT; ++i) S->stat[i] += C.stat[i];
  if (C.err) S->error = C.err;
}

// Entries pushed from here on belong to the new request: pinned (R4); everything already in T1 / T2 is a possible victim.
__device__ __forceinline__ void begin_request(SerialCtx& C) {
  C.bound[L_T1] = C.tail[L_T1];
  C.bound[L_T2] = C.tail[L_T2];
  C.elig1 = C.t1; C.elig2 = C.t2;
}

// The node leaves ring position (list, pos) by a hit or a ghost hit: its old entry becomes a tombstone.
__device__ __forceinline__ void ring_tomb(const StepParams& P, uint32_t list, uint32_t pos) {
  RingEnt* r = (list == L_T1) ? P.ring[L_T1] : (list == L_T2) ? P.ring[L_T2] : (list == L_B1) ? P.ring[L_B1] : P.ring[L_B2];
  __stcg(r + (pos & P.ring_mask), ring_ent(RING_TOMB, -1));
}

// One access (R5 for ARC, R10 for LRU) against the live state: access index a (access order), output index out
// (natural order).  C.bound[T1/T2] must hold the tails recorded when the access's request began (R4).
__device__ __noinline__ void serial_access(SerialCtx& C, const StepParams& P, int64_t a, int64_t out) {
  const int32_t c = P.capacity;
  const uint32_t n = P.node_acc[a];
  Node rec = ld_node(P.nodes + n);
  const bool held = (rec.list & NODE_HELD) != 0;             // pin scope 2 only: resident, in no ring, rec.pos = holds
  const uint32_t holds = held ? rec.pos : 0u;
  rec.list &= NODE_LIST_MASK;
  int cls;
  int32_t blk = rec.block, ev = -1;
  uint32_t dropped = NODE_NONE;
  C.stat[ST_ACCESSES]++;
  if (rec.list >= L_T1 && rec.list <= L_B2 && !held) ring_tomb(P, rec.list, rec.pos);   // every class but MISS moves the node
  if (P.policy == POLICY_LRU) {             // R10
    if (rec.list == L_T1) {
      cls = CLS_HIT_T1; C.stat[ST_HIT_T1]++;
      if (!held && (int32_t)(C.bound[L_T1] - rec.pos) > 0) C.elig1--;
      place_accessed<L_T1>(C, P, n, blk, rec.slot, holds);
    } else {
      cls = CLS_MISS; C.stat[ST_MISS]++;
      if (C.t1 < c) { blk = C.next_fresh++; C.stat[ST_FRESH]++; }
      else blk = ev = evict_t1_no_ghost_serial(C, P, &dropped);
      place_accessed<L_T1>(C, P, n, blk, rec.slot, 0);
      C.t1++;
    }
  } else if (rec.list == L_T1 || rec.list == L_T2) {      // R5 case 1
    if (rec.list == L_T1) {
      cls = CLS_HIT_T1; C.stat[ST_HIT_T1]++; C.t1--; C.t2++;
      if (!held && (int32_t)(C.bound[L_T1] - rec.pos) > 0) C.elig1--;
    } else {
      cls = CLS_HIT_T2; C.stat[ST_HIT_T2]++;
      if (!held && (int32_t)(C.bound[L_T2] - rec.pos) > 0) C.elig2--;
    }
    place_accessed<L_T2>(C, P, n, blk, rec.slot, holds);
  } else if (rec.list == L_B1) {                          // case 2
    cls = CLS_GHOST_B1; C.stat[ST_GHOST_B1]++;
    int32_t delta = C.b2 / C.b1; if (delta < 1) delta = 1;
    if (P.policy != POLICY_DBL) C.p = min(c, C.p + delta);      // DBL: no adaptation
    blk = ev = replace_serial(C, P, false);
    C.b1--; C.t2++;
    place_accessed<L_T2>(C, P, n, blk, rec.slot, 0);
  } else if (rec.list == L_B2) {                          // case 3
    cls = CLS_GHOST_B2; C.stat[ST_GHOST_B2]++;
    int32_t delta = C.b1 / C.b2; if (delta < 1) delta = 1;
    if (P.policy != POLICY_DBL) C.p = max(0, C.p - delta);
    blk = ev = replace_serial(C, P, true);
    C.b2--; C.t2++;
    place_accessed<L_T2>(C, P, n, blk, rec.slot, 0);
  } else {                                                // case 4 (ABSENT)
    cls = CLS_MISS; C.stat[ST_MISS]++;
    if (rec.list != L_ABSENT) C.err = DEV_ERR_BAD_NODE;
    if (C.t1 + C.b1 == c) {                               // (A)
      if (C.t1 < c) { drop_ghost_serial<L_B1>(C, P, &dropped); blk = ev = replace_serial(C, P, false); }
      else blk = ev = evict_t1_no_ghost_serial(C, P, &dropped);
    } else {                                              // (B)
      const int32_t tot = C.t1 + C.t2 + C.b1 + C.b2;
      if (tot >= c) {
        if (tot == 2 * c) drop_ghost_serial<L_B2>(C, P, &dropped);
        blk = ev = replace_serial(C, P, false);
      } else { blk = C.next_fresh++; C.stat[ST_FRESH]++; }
    }
    place_accessed<L_T1>(C, P, n, blk, rec.slot, 0);
    C.t1++;
  }
  P.cls[out] = (uint8_t)cls;
  P.block_id[out] = blk;
  P.evicted_id[out] = ev;
  P.p_after[out] = C.p;
  P.dropped[a] = dropped;
  if (cls != CLS_HIT_T1 && cls != CLS_HIT_T2) P.alloc_ids[C.n_alloc++] = blk;
  if (ev >= 0) P.evict_ids[C.n_evict++] = ev;
}

__global__ void arc_machine_serial_kernel(const __grid_constant__ StepParams P) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  if (P.state->error == DEV_ERR_NODE_POOL) return;       // K2 could not give every key a node: the step is void (sticky error)
  SerialCtx C;
  ctx_load(C, P);
  for (uint32_t r = 0; r < P.n_req; ++r) {
    const int64_t o = P.blk_off[r], nb = P.blk_off[r + 1] - o;
    // step-wide scope: the pins of earlier requests of the step stay; held scope: nothing enters T1 / T2's rings during a
    // step, every ring entry is a possible victim (bound = tail, set by ctx_load) and elig1/2 carry over from DevState
    if (P.pin_scope != 2 && (r == 0 || P.pin_scope == 0)) begin_request(C);
    for (int64_t j = 0; j < nb; ++j) {                                               // tail block first (R2)
      const long long t0 = clock64();
      serial_access(C, P, o + j, o + (nb - 1 - j));
      const unsigned long long dt = (unsigned long long)(clock64() - t0);
      const int bin = dt < 64 ? 0 : min(15, 64 - __clzll(dt) - 6);                  // the K3 per-access latency histogram
      P.state->lat_hist[P.cls[o + (nb - 1 - j)]][bin] += 1;
    }
  }
  ctx_store(C, P);
}

}  // namespace arc
