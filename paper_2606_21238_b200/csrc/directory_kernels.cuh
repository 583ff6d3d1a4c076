// K2 (batched directory probe + reserve), K4 (finalize), and the maintenance kernels of the
// device-resident directory (table rebuild, ring compaction, init, debug dump).
#pragma once
#include <cooperative_groups.h>

#include "arc_device.cuh"

namespace arc {
namespace cg = cooperative_groups;

__device__ __forceinline__ Slot ld_slot(const Slot* p) {
  uint4 v = __ldcg(reinterpret_cast<const uint4*>(p));   // L2: other CTAs CAS into this line during K2
  Slot s;
  s.key = (unsigned long long)v.x | ((unsigned long long)v.y << 32);
  s.node = v.z; s.pad = v.w;
  return s;
}

// ---------------------------------------------------------------------------------------------------
// K2: for every key of the step find its node; if the key is not in the table, insert it and reserve a
// node in state ABSENT, so that every access carries a node index into K3 and duplicates inside the
// step share one node.  Warp-cooperative: a tile of 8 lanes probes one 128 B bucket
// (8 slots x 16 B) per iteration with one coalesced load; the probe sequence is linear over buckets and
// ends at the first bucket that still has a never-used (EMPTY) slot.  Inserts claim the lowest EMPTY
// slot of that bucket with a 64-bit CAS on the key; a failed CAS re-reads the bucket, so two tiles
// inserting the same key can never both succeed.  Tombstones are not reused;
// rebuild_table clears them.
__global__ void __launch_bounds__(256) probe_reserve_kernel(StepParams P) {
  cg::thread_block_tile<8> tile = cg::tiled_partition<8>(cg::this_thread_block());
  const uint32_t sub = tile.thread_rank();
  const uint32_t tiles = (gridDim.x * blockDim.x) >> 3;
  for (uint32_t a = (blockIdx.x * blockDim.x + threadIdx.x) >> 3; a < P.n_access; a += tiles) {
    unsigned long long key = P.keys_acc[a] & P.key_and;
    if (key < 2) key += 2;                       // 0 and 1 stay reserved under the test mask too
    uint32_t bucket = (uint32_t)key & P.bucket_mask;
    uint32_t result = NODE_NONE;
    for (;;) {
      const uint32_t idx = bucket * BUCKET_SLOTS + sub;
      const Slot s = ld_slot(P.table + idx);
      const uint32_t match = tile.ballot(s.key == key);
      if (match) {
        const int src = __ffs(match) - 1;
        const uint32_t node = tile.shfl(s.node, src);
        result = (node == SLOT_NODE_PENDING) ? (SLOT_FLAG | (bucket * BUCKET_SLOTS + src)) : node - 1;
        break;
      }
      const uint32_t empty = tile.ballot(s.key == KEY_EMPTY);
      if (!empty) { bucket = (bucket + 1) & P.bucket_mask; continue; }
      const int src = __ffs(empty) - 1;
      uint32_t got = NODE_NONE;
      if ((int)sub == src) {
        const unsigned long long old = atomicCAS(&P.table[idx].key, KEY_EMPTY, key);
        if (old == KEY_EMPTY) {            // we own the slot: take a node and publish it
          const uint32_t top = atomicSub(&P.state->free_top, 1u);
          if (top == 0 || top > 0x7FFFFFFFu) {
            atomicExch(&P.state->error, DEV_ERR_NODE_POOL);
            got = 0;
          } else {
            got = P.free_stack[top - 1];
            st_node(P.nodes + got, L_ABSENT, 0, -1, idx);
            P.node_key[got] = key;
          }
          __stcg(&P.table[idx].node, got + 1);
        }
      }
      got = tile.shfl(got, src);
      if (got != NODE_NONE) { result = got; break; }
      // lost the race for that slot: look at the bucket again (the winner may hold our key)
    }
    if (sub == 0) P.node_acc[a] = result;
  }
}

// After K2: entries that raced with the winner of their key carry a slot index; the winner's node id is
// visible now (kernel boundary).
// Also K2's twin check: every access stamps its node with (step, request); finding one's own stamp already there means
// the request reaches that node twice - possible only through a 64-bit key collision inside one request (or the test
// hook that forces equal keys).  K3's wide machine pays for exact twin detection only in steps that carry the flag.
__global__ void __launch_bounds__(256) resolve_nodes_kernel(StepParams P) {
  for (uint32_t a = blockIdx.x * blockDim.x + threadIdx.x; a < P.n_access; a += gridDim.x * blockDim.x) {
    uint32_t v = P.node_acc[a];
    if (v != NODE_NONE && (v & SLOT_FLAG)) { v = __ldcg(&P.table[v & ~SLOT_FLAG].node) - 1; P.node_acc[a] = v; }
    if (P.n_req == 0 || v == NODE_NONE) continue;          // arc_debug_probe: no requests
    uint32_t lo = 0, hi = P.n_req;                          // request r with blk_off[r] <= a < blk_off[r+1]
    while (hi - lo > 1) {
      const uint32_t mid = (lo + hi) >> 1;
      if (P.blk_off[mid] <= (int64_t)a) lo = mid; else hi = mid;
    }
    const uint32_t tag = P.step_tag | lo;
    if (atomicExch(&P.node_stamp[v], tag) == tag) P.state->step_twins = 1;
  }
}

// ---------------------------------------------------------------------------------------------------
// K4: (1) keys whose node ended the step ABSENT (dropped ghosts, evictions that leave no ghost) leave
// the table and their nodes return to the free stack; (2) prefix_len[r] = B x leading hit blocks (R9).
__global__ void __launch_bounds__(256) finalize_kernel(StepParams P) {
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nthr = gridDim.x * blockDim.x;
  for (uint32_t a = tid; a < P.n_access; a += nthr) {
    const uint32_t d = P.dropped[a];
    if (d == NODE_NONE) continue;
    if (atomicCAS(&P.nodes[d].list, L_ABSENT, L_FREE) == L_ABSENT) {   // still absent, and only once
      const uint32_t slot = P.nodes[d].slot;
      P.table[slot].node = SLOT_NODE_PENDING;
      P.table[slot].key = KEY_TOMB;
      const uint32_t top = atomicAdd(&P.state->free_top, 1u);
      P.free_stack[top] = d;
      atomicAdd(&P.state->tombs, 1u);
    }
  }
  // one warp per request: scan the classes from block 0 upward, 32 at a time
  const uint32_t lane = threadIdx.x & 31, warp = tid >> 5, n_warps = nthr >> 5;
  unsigned long long tokens_hit = 0;
  for (uint32_t r = warp; r < P.n_req; r += n_warps) {
    const int64_t o = P.blk_off[r], nb = P.blk_off[r + 1] - o;
    int64_t lead = nb;
    for (int64_t base = 0; base < nb && lead == nb; base += 128) {      // 128 classes per round trip: four independent loads per lane
      int c[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) { const int64_t i = base + 32 * q + lane; c[q] = (i < nb) ? P.cls[o + i] : CLS_MISS; }
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const uint32_t nonhit = __ballot_sync(0xFFFFFFFFu, !(c[q] == CLS_HIT_T1 || c[q] == CLS_HIT_T2));
        if (nonhit && lead == nb) lead = base + 32 * q + (__ffs(nonhit) - 1);
      }
    }
    if (lead > nb) lead = nb;
    if (lane == 0) { P.prefix_len[r] = (int32_t)(lead * P.block_size); tokens_hit += (unsigned long long)lead * P.block_size; }
  }
  if (lane == 0 && tokens_hit) atomicAdd(&P.state->stat[ST_PREFIX_TOKENS], tokens_hit);
  if (tid == 0) {
    P.state->k1_ticket = 0; P.state->step_twins = 0;                   // K1 of the next step starts from request 0
    P.counts_out[0] = P.state->counts[0]; P.counts_out[1] = P.state->counts[1];
  }
}

// ---------------------------------------------------------------------------------------------------
// Maintenance

__global__ void init_state_kernel(DevState* st, Node* nodes, uint32_t* free_stack, uint32_t node_cap, int32_t p0) {
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  for (uint32_t i = tid; i < node_cap; i += gridDim.x * blockDim.x) {
    st_node(nodes + i, L_FREE, 0, -1, 0);
    free_stack[i] = node_cap - 1 - i;   // node 0 is handed out first
  }
  if (tid == 0) {
    DevState z;
    memset(&z, 0, sizeof(z));
    z.free_top = node_cap;
    z.p = p0;                           // 0, or capacity / 2 for the DBL policy
    *st = z;
  }
}

// Growth of the node pool: ids [old_cap, new_cap) become free; they go *under* the existing stack
// content so that already-free ids keep their order.
__global__ void extend_free_stack_kernel(DevState* st, Node* nodes, const uint32_t* old_stack, uint32_t* new_stack,
                                         uint32_t old_cap, uint32_t new_cap) {
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nthr = gridDim.x * blockDim.x;
  const uint32_t extra = new_cap - old_cap, top = st->free_top;
  for (uint32_t i = tid; i < extra; i += nthr) {
    new_stack[i] = new_cap - 1 - i;
    st_node(nodes + old_cap + i, L_FREE, 0, -1, 0);
  }
  for (uint32_t i = tid; i < top; i += nthr) new_stack[extra + i] = old_stack[i];
}
__global__ void bump_free_top_kernel(DevState* st, uint32_t extra) { st->free_top += extra; }

// Re-inserts every live key into a cleared table (drops tombstones, or moves to a bigger table).
__global__ void __launch_bounds__(256) rebuild_table_kernel(DevState* st, Node* nodes, const unsigned long long* node_key,
                                                           uint32_t node_cap, Slot* table, uint32_t bucket_mask) {
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
  if (tid == 0) st->tombs = 0;
  for (uint32_t n = tid; n < node_cap; n += gridDim.x * blockDim.x) {
    const uint32_t list = nodes[n].list;
    if (list == L_FREE) continue;
    const unsigned long long key = node_key[n];
    uint32_t idx = ((uint32_t)key & bucket_mask) * BUCKET_SLOTS;
    const uint32_t slot_mask = (bucket_mask + 1) * BUCKET_SLOTS - 1;
    for (;;) {   // live keys are distinct: plain claim of the first EMPTY slot in probe order
      if (atomicCAS(&table[idx].key, KEY_EMPTY, key) == KEY_EMPTY) break;
      idx = (idx + 1) & slot_mask;
    }
    table[idx].node = n + 1;
    nodes[n].slot = idx;
  }
}

// Ring compaction, two kernels.  The live entries of list L move, in order, to fresh positions
// [old_tail, old_tail + live) of the *other* buffer: new positions never overlap old ones, so a stale
// entry can never be mistaken for a live one while CTAs run concurrently.
// blockIdx.y selects the list (L0 + blockIdx.y): all four lists are compacted by ONE pair of launches when the step-time
// upkeep asks for it (their host-side bounds grow together, so they are due together).
constexpr int CMP_THREADS = 1024;
struct RingPtrs { const RingEnt* src[5]; RingEnt* dst[5]; };
__global__ void __launch_bounds__(CMP_THREADS) ring_count_kernel(DevState* st, const Node* nodes, const RingPtrs rp,
                                                                uint32_t ring_mask, uint32_t L0, uint32_t* block_counts_all) {
  const uint32_t L = L0 + blockIdx.y;
  const RingEnt* ring = rp.src[L];
  uint32_t* block_counts = block_counts_all + (size_t)blockIdx.y * gridDim.x;
  const uint32_t head = st->head[L], tail = st->tail[L];
  const uint32_t window = tail - head;
  const uint32_t off = blockIdx.x * CMP_THREADS + threadIdx.x;
  bool live = false;
  if (off < window) {
    const uint32_t q = head + off;
    const uint32_t n = ent_node(ring[q & ring_mask]);
    if (n != RING_TOMB) {
      const Node r = ld_node(nodes + n);
      live = (r.list == L && r.pos == q);
    }
  }
  const int cnt = __syncthreads_count(live);
  if (threadIdx.x == 0) {
    block_counts[blockIdx.x] = cnt;
    if (blockIdx.x == 0) { st->cmp_head[L] = head; st->cmp_tail[L] = tail; }
  }
}
__global__ void __launch_bounds__(CMP_THREADS) ring_scatter_kernel(DevState* st, Node* nodes, const RingPtrs rp,
                                                                  uint32_t ring_mask, uint32_t dst_mask,
                                                                  uint32_t L0, const uint32_t* block_counts_all) {
  __shared__ uint32_t s_warp[32];
  __shared__ uint32_t s_base, s_total;
  const uint32_t L = L0 + blockIdx.y;
  const RingEnt* ring = rp.src[L];
  RingEnt* ring_dst = rp.dst[L];
  const uint32_t* block_counts = block_counts_all + (size_t)blockIdx.y * gridDim.x;
  const uint32_t head = st->cmp_head[L], tail = st->cmp_tail[L];
  const uint32_t window = tail - head;
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  // exclusive prefix of block_counts up to this block (and the grand total in block 0)
  uint32_t mine = 0, all = 0;
  for (uint32_t b = threadIdx.x; b < gridDim.x; b += CMP_THREADS) {
    const uint32_t v = block_counts[b];
    if (b < blockIdx.x) mine += v;
    all += v;
  }
  for (int d = 16; d; d >>= 1) { mine += __shfl_xor_sync(0xFFFFFFFFu, mine, d); all += __shfl_xor_sync(0xFFFFFFFFu, all, d); }
  if (lane == 0) s_warp[warp] = mine;
  __syncthreads();
  if (warp == 0) {
    uint32_t v = s_warp[lane];
    for (int d = 16; d; d >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, d);
    if (lane == 0) s_base = v;
  }
  __syncthreads();
  if (lane == 0) s_warp[warp] = all;
  __syncthreads();
  if (warp == 0) {
    uint32_t v = s_warp[lane];
    for (int d = 16; d; d >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, d);
    if (lane == 0) s_total = v;
  }
  __syncthreads();
  const uint32_t off = blockIdx.x * CMP_THREADS + threadIdx.x;
  bool live = false;
  uint32_t n = 0;
  int32_t blk = -1;
  if (off < window) {
    const uint32_t q = head + off;
    n = ent_node(ring[q & ring_mask]);
    if (n != RING_TOMB) {
      const Node r = ld_node(nodes + n);
      live = (r.list == L && r.pos == q);
      blk = r.block;
    }
  }
  const uint32_t bal = __ballot_sync(0xFFFFFFFFu, live);
  __syncthreads();
  if (lane == 0) s_warp[warp] = __popc(bal);
  __syncthreads();
  uint32_t before = 0;
  for (uint32_t w = 0; w < warp; ++w) before += s_warp[w];
  if (live) {
    const uint32_t q_new = tail + s_base + before + __popc(bal & ((1u << lane) - 1));
    ring_dst[q_new & dst_mask] = ring_ent(n, blk);
    nodes[n].pos = q_new;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) { st->head[L] = tail; st->tail[L] = tail + s_total; }
}

// Debug: write list L (LRU -> MRU) as keys and block ids.  Single CTA, sequential chunks.
__global__ void __launch_bounds__(CMP_THREADS) dump_list_kernel(const DevState* st, const Node* nodes,
                                                               const unsigned long long* node_key, const RingEnt* ring,
                                                               uint32_t ring_mask, uint32_t L, unsigned long long* keys_out,
                                                               int32_t* blocks_out, unsigned long long cap,
                                                               unsigned long long* n_out) {
  __shared__ uint32_t s_warp[32];
  __shared__ uint32_t s_done;
  const uint32_t head = st->head[L], tail = st->tail[L], window = tail - head;
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_done = 0;
  __syncthreads();
  for (uint32_t base = 0; base < window; base += CMP_THREADS) {
    const uint32_t off = base + threadIdx.x;
    bool live = false;
    uint32_t n = 0;
    Node r;
    r.block = -1;
    if (off < window) {
      n = ent_node(ring[(head + off) & ring_mask]);
      if (n != RING_TOMB) {
        r = ld_node(nodes + n);
        live = (r.list == L && r.pos == head + off);
      }
    }
    const uint32_t bal = __ballot_sync(0xFFFFFFFFu, live);
    if (lane == 0) s_warp[warp] = __popc(bal);
    __syncthreads();
    uint32_t before = s_done;
    for (uint32_t w = 0; w < warp; ++w) before += s_warp[w];
    if (live) {
      const unsigned long long k = before + __popc(bal & ((1u << lane) - 1));
      if (k < cap) {
        if (keys_out) keys_out[k] = node_key[n];
        if (blocks_out) blocks_out[k] = r.block;
      }
    }
    __syncthreads();
    if (threadIdx.x == 0) { uint32_t t = 0; for (int w = 0; w < 32; ++w) t += s_warp[w]; s_done += t; }
    __syncthreads();
  }
  if (threadIdx.x == 0) *n_out = s_done;
}

// ---------------------------------------------------------------------------------------------------------------------
// arc_release (pin scope 2): one hold back per listed block id, in the order given; a block whose last
// hold goes re-enters its list (T1 or T2) at the MRU end.  One CTA of 1024 threads, everything data-parallel:
//   pass 1  every id must name a resident held block; rel_cnt[id] counts how often it is listed, rel_last[id] keeps the
//           index (+1) of its last occurrence;
//   pass 2  no id is listed more often than it is held.  If either check fails nothing changes and the handle gets the
//           sticky error DEV_ERR_BAD_RELEASE;
//   pass 3  walking the ids in order, a block's count reaches zero exactly at its LAST occurrence and only if
//           rel_cnt == holds, so the occurrences that re-enter a ring are known up front; their ring positions are the
//           tail plus a CTA-wide exclusive scan of those flags, 1024 ids per round, per list;
//   pass 4  the scratch is zeroed again (rel_cnt / rel_last are all zero between calls).
constexpr int REL_THREADS = 1024;
__global__ void __launch_bounds__(REL_THREADS) release_kernel(const __grid_constant__ StepParams P, const int32_t* ids, uint32_t n,
                                                              uint32_t* rel_cnt, uint32_t* rel_last) {
  __shared__ uint32_t s_bad;
  __shared__ uint32_t s_w1[32], s_w2[32];
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5, FULL = 0xFFFFFFFFu, lt = (1u << lane) - 1u;
  DevState* S = P.state;
  if (tid == 0) s_bad = 0;
  __syncthreads();
  for (uint32_t i = tid; i < n; i += REL_THREADS) {
    const int32_t id = ids[i];
    bool ok = id >= 0 && id < P.capacity;
    if (ok) {
      const uint32_t nd = P.node_of_block[id];
      ok = nd != NODE_NONE;
      if (ok) { const Node r = ld_node(P.nodes + nd); ok = (r.list & NODE_HELD) && r.block == id; }
    }
    if (ok) { atomicAdd(&rel_cnt[id], 1u); atomicMax(&rel_last[id], i + 1u); } else s_bad = 1;
  }
  __syncthreads();
  if (!s_bad) {
    for (uint32_t i = tid; i < n; i += REL_THREADS) {
      const int32_t id = ids[i];
      if (__ldcg(&rel_cnt[id]) > ld_node(P.nodes + P.node_of_block[id]).pos) s_bad = 1;
    }
  }
  __syncthreads();
  const bool bad = s_bad != 0;
  if (!bad) {
    uint32_t tail1 = S->tail[L_T1], tail2 = S->tail[L_T2];      // every thread carries the same running tails
    for (uint32_t base = 0; base < n; base += REL_THREADS) {
      const uint32_t i = base + tid;
      bool last = false, zero = false;
      uint32_t nd = 0, L = 0, left = 0;
      Node r;
      r.list = 0; r.pos = 0; r.block = -1; r.slot = 0;
      if (i < n) {
        const int32_t id = ids[i];
        last = __ldcg(&rel_last[id]) == i + 1u;
        if (last) {
          nd = P.node_of_block[id];
          r = ld_node(P.nodes + nd);
          left = r.pos - __ldcg(&rel_cnt[id]);
          zero = left == 0;
          L = r.list & NODE_LIST_MASK;
        }
      }
      const uint32_t z1 = __ballot_sync(FULL, zero && L == L_T1), z2 = __ballot_sync(FULL, zero && L == L_T2);
      if (lane == 0) { s_w1[warp] = (uint32_t)__popc(z1); s_w2[warp] = (uint32_t)__popc(z2); }
      __syncthreads();
      uint32_t before1 = 0, before2 = 0, tot1 = 0, tot2 = 0;
      {
        const uint32_t a1 = s_w1[lane], a2 = s_w2[lane];              // REL_THREADS / 32 = 32 warps: one per lane
        uint32_t p1 = a1, p2 = a2;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
          const uint32_t x1 = __shfl_up_sync(FULL, p1, d), x2 = __shfl_up_sync(FULL, p2, d);
          if ((int)lane >= d) { p1 += x1; p2 += x2; }
        }
        before1 = __shfl_sync(FULL, p1 - a1, warp); before2 = __shfl_sync(FULL, p2 - a2, warp);
        tot1 = __shfl_sync(FULL, p1, 31); tot2 = __shfl_sync(FULL, p2, 31);
      }
      if (zero) {
        const uint32_t q = (L == L_T1) ? tail1 + before1 + (uint32_t)__popc(z1 & lt) : tail2 + before2 + (uint32_t)__popc(z2 & lt);
        __stcg(((L == L_T1) ? P.ring[L_T1] : P.ring[L_T2]) + (q & P.ring_mask), ring_ent(nd, r.block));
        st_node(P.nodes + nd, L, q, r.block, r.slot);
      } else if (last) {
        st_node(P.nodes + nd, r.list, left, r.block, r.slot);
      }
      tail1 += tot1; tail2 += tot2;
      __syncthreads();
    }
    if (tid == 0) {
      S->u1 += (int32_t)(tail1 - S->tail[L_T1]); S->u2 += (int32_t)(tail2 - S->tail[L_T2]);
      S->tail[L_T1] = tail1; S->tail[L_T2] = tail2;
    }
  }
  __syncthreads();
  for (uint32_t i = tid; i < n; i += REL_THREADS) {
    const int32_t id = ids[i];
    if (id >= 0 && id < P.capacity) { rel_cnt[id] = 0; rel_last[id] = 0; }
  }
  if (bad && tid == 0) S->error = DEV_ERR_BAD_RELEASE;
}

// entering pin scope 2 with nothing held: every resident entry is in a ring
__global__ void set_unheld_kernel(DevState* st) { st->u1 = st->t1; st->u2 = st->t2; }

}  // namespace arc
