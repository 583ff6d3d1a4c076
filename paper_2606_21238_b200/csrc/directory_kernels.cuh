// K2 (batched directory probe + reserve), K4 (finalize), and the maintenance kernels of the
// device-resident directory (table rebuild, ring compaction, init, debug dump).
#pragma once
#include <cooperative_groups.h>

#include "arc_device.cuh"

namespace arc {
namespace cg = cooperative_groups;

// ---------------------------------------------------------------------------------------------------
// K2: for every key of the step find its node; if the key is not in the table, insert it and reserve a
// node in state ABSENT, so that every access carries a node index into K3 and duplicates inside the
// step share one node.
//
// Layout: buckets of BUCKET_SLOTS = 2 slots x 16 B = ONE 32-byte sector, the unit HBM and L2 move.  One thread owns one
// key: it fetches the key's bucket with a single 256-bit load (LDG.256), compares both slots, and moves to the next
// bucket only when this one is full of other keys (linear over buckets; the probe ends at the first bucket that still
// has a never-used slot).  A probe therefore costs one sector = 32 B next to the 8 B of the key and the 4 B of the
// node id: 44 B per key against 28 B algorithmic.  Each thread keeps PROBE_ILP keys in flight.
//
// Insert-if-absent, in warp-synchronous phases, so that (1) the free stack's top - one address for the whole GPU - sees
// one atomic per warp and not one per insert, (2) exactly as many node ids are popped as keys are new, and (3) nobody
// ever waits for a thread that could be waiting for him:
//   A  every thread walks each of its keys' buckets until it finds the key or a bucket with a never-used slot;
//   C1 claims: 64-bit CAS EMPTY -> key on the slot.  The winner of a key is the one thread whose CAS put it there; a
//      thread that finds its key already there (CAS result, or a bucket read) is a waiter of that slot; a thread that
//      finds another key there walks on;
//   B  the warp pops one node id per winner with ONE atomicSub (shuffle scan of the counts);
//   C2 winners write the node record and publish the id in the slot (Slot::node = id + 1);  __syncwarp;
//   C3 waiters read the slot until the id is there.  The winner may sit in another warp; it never waits between its
//      claim and its publish (C2 comes before C3 in every warp), so the wait is bounded and cannot be circular.
// Tombstones are not reused; rebuild_table clears them.
constexpr int PROBE_ILP = 4;

struct Bucket { Slot s[BUCKET_SLOTS]; };
__device__ __forceinline__ Bucket ld_bucket(const Slot* p) {          // p is 32-byte aligned
  uint32_t r[8];
  asm volatile("ld.global.cg.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "l"(p) : "memory");
  Bucket b;
  b.s[0].key = (unsigned long long)r[0] | ((unsigned long long)r[1] << 32); b.s[0].node = r[2]; b.s[0].pad = r[3];
  b.s[1].key = (unsigned long long)r[4] | ((unsigned long long)r[5] << 32); b.s[1].node = r[6]; b.s[1].pad = r[7];
  return b;
}

// the same load under a predicate (no branch, the destination keeps its content): keeps the buckets of a round in registers
__device__ __forceinline__ void ld_bucket_if(Bucket& b, const Slot* p, bool take) {
  uint32_t r0 = (uint32_t)b.s[0].key, r1 = (uint32_t)(b.s[0].key >> 32), r2 = b.s[0].node, r3 = b.s[0].pad;
  uint32_t r4 = (uint32_t)b.s[1].key, r5 = (uint32_t)(b.s[1].key >> 32), r6 = b.s[1].node, r7 = b.s[1].pad;
  asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %9, 0;\n\t@q ld.global.cg.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n\t}"
               : "+r"(r0), "+r"(r1), "+r"(r2), "+r"(r3), "+r"(r4), "+r"(r5), "+r"(r6), "+r"(r7) : "l"(p), "r"((uint32_t)take) : "memory");
  b.s[0].key = (unsigned long long)r0 | ((unsigned long long)r1 << 32); b.s[0].node = r2; b.s[0].pad = r3;
  b.s[1].key = (unsigned long long)r4 | ((unsigned long long)r5 << 32); b.s[1].node = r6; b.s[1].pad = r7;
}

enum : uint32_t { PR_DONE = 0, PR_CLAIM = 1, PR_WAIT = 2, PR_WON = 3, PR_LOAD = 4 };

// Looks at bucket content c (bucket index bk) for `key`: found with its node -> PR_DONE (node set); found, node not yet
// published -> PR_WAIT (idx = the slot); a never-used slot -> PR_CLAIM (idx = that slot); else 0xFF: full of other keys.
__device__ __forceinline__ uint32_t probe_bucket(const Bucket& c, uint32_t bk, unsigned long long key, uint32_t& node, uint32_t& idx) {
#pragma unroll
  for (int e = 0; e < (int)BUCKET_SLOTS; ++e)
    if (c.s[e].key == key) {
      idx = bk * BUCKET_SLOTS + (uint32_t)e;
      if (c.s[e].node == SLOT_NODE_PENDING) return PR_WAIT;
      node = c.s[e].node - 1;
      return PR_DONE;
    }
#pragma unroll
  for (int e = 0; e < (int)BUCKET_SLOTS; ++e)
    if (c.s[e].key == KEY_EMPTY) { idx = bk * BUCKET_SLOTS + (uint32_t)e; return PR_CLAIM; }
  return 0xFFu;
}

// One pass of a warp over 32 x PROBE_ILP keys (key u of lane l is access first + u * stride).  Phases A and C1 run as
// ROUNDS over all of a thread's keys at once - every key that still needs a bucket gets its load issued, then every key
// that found a never-used slot gets its CAS issued - so that the dependent memory round trips a warp pays are those of
// its longest probe sequence, not the sum over its keys.
__device__ __forceinline__ void probe_warp_pass(const StepParams& P, uint32_t first, uint32_t stride, int lane) {
  const uint32_t FULL = 0xFFFFFFFFu;
  unsigned long long key[PROBE_ILP];
  uint32_t idx[PROBE_ILP], node[PROBE_ILP], st[PROBE_ILP];   // idx: bucket index while st = PR_LOAD, slot index otherwise
#pragma unroll
  for (int u = 0; u < PROBE_ILP; ++u) {
    const uint32_t a = first + u * stride;
    key[u] = (a < P.n_access) ? (__ldcg(P.keys_acc + a) & P.key_and) : 2ull;
    if (key[u] < 2) key[u] += 2;                       // 0 and 1 stay reserved under the test mask too
    idx[u] = (uint32_t)key[u] & P.bucket_mask;
    node[u] = NODE_NONE;
    st[u] = (a < P.n_access) ? PR_LOAD : PR_DONE;
  }
  uint32_t won = 0;
  Bucket b[PROBE_ILP];
#pragma unroll
  for (int u = 0; u < PROBE_ILP; ++u) { b[u].s[0].key = b[u].s[1].key = 0; b[u].s[0].node = b[u].s[1].node = b[u].s[0].pad = b[u].s[1].pad = 0; }
  for (;;) {
    // A: one bucket for every key that needs one
    bool busy = false;
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) {
      const bool take = st[u] == PR_LOAD;
      ld_bucket_if(b[u], P.table + (size_t)(take ? idx[u] : 0u) * BUCKET_SLOTS, take);
      busy = busy || take;
    }
    if (!busy) break;
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) {
      if (st[u] != PR_LOAD) continue;
      const uint32_t bk = idx[u];
      st[u] = probe_bucket(b[u], bk, key[u], node[u], idx[u]);
      if (st[u] == 0xFFu) { st[u] = PR_LOAD; idx[u] = (bk + 1) & P.bucket_mask; }   // full of other keys: the next bucket, next round
    }
    // C1: claims.  The winner of a key is the one thread whose CAS put it there.
    unsigned long long old[PROBE_ILP];
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) if (st[u] == PR_CLAIM) old[u] = atomicCAS(&P.table[idx[u]].key, KEY_EMPTY, key[u]);
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) {
      if (st[u] != PR_CLAIM) continue;
      if (old[u] == KEY_EMPTY) { st[u] = PR_WON; ++won; }
      else if (old[u] == key[u]) st[u] = PR_WAIT;
      else { st[u] = PR_LOAD; idx[u] /= BUCKET_SLOTS; }   // another key took the slot: look at the same bucket again
    }
  }
  // B: one pop for the warp
  uint32_t incl = won;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const uint32_t v = __shfl_up_sync(FULL, incl, d); if (lane >= d) incl += v; }
  const uint32_t total = __shfl_sync(FULL, incl, 31);
  if (total) {
    uint32_t top = 0;
    if (lane == 0) {
      top = atomicSub(&P.state->free_top, total);
      if (top < total || top > 0x7FFFFFFFu) {          // the pool cannot serve the warp: nothing is taken
        atomicAdd(&P.state->free_top, total);
        atomicExch(&P.state->error, DEV_ERR_NODE_POOL);
        top = 0;
      }
    }
    top = __shfl_sync(FULL, top, 0);
    uint32_t next = top - (incl - won);                // this thread's ids: free_stack[next - 1], free_stack[next - 2], ...
    // C2: winners publish.  On an exhausted pool (top == 0, sticky error, K3 will not run) the slot gets a value that
    // makes every waiter leave with NODE_NONE.
    uint32_t id[PROBE_ILP];
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) if (st[u] == PR_WON && top) id[u] = __ldcg(P.free_stack + (--next));
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) {
      if (st[u] != PR_WON) continue;
      uint32_t pub = NODE_NONE;
      if (top) {
        st_node(P.nodes + id[u], L_ABSENT, 0, -1, idx[u]);   // read by K3 only, after the kernel boundary
        P.node_key[id[u]] = key[u];
        node[u] = id[u];
        pub = id[u] + 1u;
      }
      __stcg(&P.table[idx[u]].node, pub);
    }
  }
  __syncwarp();
  // C3: waiters
#pragma unroll
  for (int u = 0; u < PROBE_ILP; ++u) {
    if (st[u] != PR_WAIT) continue;
    const volatile uint32_t* p = &P.table[idx[u]].node;
    uint32_t v;
    while ((v = *p) == SLOT_NODE_PENDING) {}
    node[u] = (v == NODE_NONE) ? NODE_NONE : v - 1u;   // NODE_NONE: the winner found the pool exhausted
  }
#pragma unroll
  for (int u = 0; u < PROBE_ILP; ++u) if (first + u * stride < P.n_access) P.node_acc[first + u * stride] = node[u];
}

// Warp gw of n_warps takes chunks gw, gw + n_warps, ... of 32 x PROBE_ILP consecutive accesses: key u of lane l is access
// chunk * 32 * PROBE_ILP + 32 u + l (every load of a warp is one coalesced 256-byte access).  The trip count is
// warp-uniform (the passes use warp collectives).
__device__ __forceinline__ void probe_range(const StepParams& P, uint32_t thread, uint32_t n_threads) {
  const int lane = (int)(thread & 31u);
  const uint32_t n_warps = n_threads >> 5;
  for (uint64_t chunk = thread >> 5; chunk * (32u * PROBE_ILP) < P.n_access; chunk += n_warps)
    probe_warp_pass(P, (uint32_t)(chunk * (32u * PROBE_ILP)) + (uint32_t)lane, 32u, lane);
}

__global__ void __launch_bounds__(256) probe_reserve_kernel(const __grid_constant__ StepParams P) {
  probe_range(P, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}

// The ceiling K2 is measured against (arc_debug_gather_sectors): the same grid, the same loads - an 8-byte key, the 32-byte
// sector it selects, a 4-byte result - and nothing else (no compare, no insert).  What this kernel reaches is what random
// 32-byte sector reads can reach on the machine.
__global__ void __launch_bounds__(256) gather32_kernel(const unsigned long long* __restrict__ keys, uint32_t n, const Slot* __restrict__ buf,
                                                       uint32_t sector_mask, uint32_t* __restrict__ out) {
  const uint32_t first = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x;
  for (uint32_t a0 = first; a0 < n; a0 += stride * PROBE_ILP) {
    Bucket b[PROBE_ILP];
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) {
      const uint32_t a = a0 + u * stride;
      const unsigned long long key = (a < n) ? __ldcg(keys + a) : 0ull;
      b[u] = ld_bucket(buf + (size_t)((uint32_t)key & sector_mask) * BUCKET_SLOTS);
    }
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) {
      const uint32_t a = a0 + u * stride;
      if (a < n) out[a] = (uint32_t)b[u].s[0].key ^ (uint32_t)(b[u].s[0].key >> 32) ^ b[u].s[0].node ^ b[u].s[0].pad ^
                          (uint32_t)b[u].s[1].key ^ (uint32_t)(b[u].s[1].key >> 32) ^ b[u].s[1].node ^ b[u].s[1].pad;
    }
  }
}

// Step-wide / held pins: the wide K3 machine lets a window span requests there and takes each access's natural-order index
// (blk_off[r] + i for the access at blk_off[r] + nb_r - 1 - i) from nat[]: one warp per request.  Launched after K2 into the
// buffer of the keys, which nothing reads after the probe.
__device__ __forceinline__ void nat_index_body(const StepParams& P, uint32_t warp, uint32_t n_warps, uint32_t lane) {
  uint32_t* nat = reinterpret_cast<uint32_t*>(P.keys_acc);
  for (uint32_t r = warp; r < P.n_req; r += n_warps) {
    const int64_t o = P.blk_off[r], nb = P.blk_off[r + 1] - o;
    for (int64_t i = lane; i < nb; i += 32) nat[o + (nb - 1 - i)] = (uint32_t)(o + i);
  }
}
__global__ void __launch_bounds__(256) nat_index_kernel(const __grid_constant__ StepParams P) {
  nat_index_body(P, (blockIdx.x * blockDim.x + threadIdx.x) >> 5, (gridDim.x * blockDim.x) >> 5, threadIdx.x & 31);
}

// ---------------------------------------------------------------------------------------------------
// K4: (1) keys whose node ended the step ABSENT (dropped ghosts, evictions that leave no ghost) leave
// the table and their nodes return to the free stack; (2) prefix_len[r] = B x leading hit blocks (R9).
__device__ __forceinline__ void finalize_body(const StepParams& P) {
  const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nthr = gridDim.x * blockDim.x;
  for (uint32_t a = tid; a < P.n_access; a += nthr) {
    const uint32_t d = P.dropped[a];
    if (d == NODE_NONE) continue;
    if (atomicCAS(&P.nodes[d].list, L_ABSENT, L_FREE) == L_ABSENT) {   // still absent, and only once
      // the key's slot: found by probing (the key is in the table: this thread is the one that takes it out; a probe
      // sequence never crosses a never-used slot)
      const unsigned long long key = P.node_key[d];
      const uint32_t slot_mask = (P.bucket_mask + 1u) * BUCKET_SLOTS - 1u;
      uint32_t slot = ((uint32_t)key & P.bucket_mask) * BUCKET_SLOTS;
      for (;;) {
        const unsigned long long k2 = __ldcg(&P.table[slot].key);
        if (k2 == key) break;
        if (k2 == KEY_EMPTY) { P.state->error = DEV_ERR_BAD_NODE; break; }
        slot = (slot + 1u) & slot_mask;
      }
      if (P.table[slot].key != key) continue;
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
    P.counts_out[0] = P.state->counts[0]; P.counts_out[1] = P.state->counts[1];
  }
}

__global__ void __launch_bounds__(256) finalize_kernel(const __grid_constant__ StepParams P) { finalize_body(P); }

// The host entry's results, written by the device straight into pinned, mapped HOST memory (arc_step_host_async): exactly
// the words that exist - n_alloc | n_evict | device error | prefix_len[n_req] | alloc_ids[n_alloc] | evict_ids[n_evict] - so no
// copy has to be sized from an upper bound and nothing crosses the bus twice.  The sticky device error (DEV_ERR_*: node
// pool, bad release, ...) travels with every result, so a scheduler that never calls arc_stats still learns of it.
__global__ void __launch_bounds__(256) pack_results_kernel(const DevState* __restrict__ st, const int32_t* __restrict__ prefix_len,
                                                           const int32_t* __restrict__ alloc_ids, const int32_t* __restrict__ evict_ids,
                                                           uint32_t n_req, int32_t* __restrict__ out) {
  const uint32_t n_alloc = st->counts[0], n_evict = st->counts[1];
  const uint32_t total = 3u + n_req + n_alloc + n_evict;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
    int32_t v;
    if (i < 3u) v = (int32_t)(i == 0 ? n_alloc : (i == 1 ? n_evict : st->error));
    else if (i < 3u + n_req) v = prefix_len[i - 3u];
    else if (i < 3u + n_req + n_alloc) v = alloc_ids[i - 3u - n_req];
    else v = evict_ids[i - 3u - n_req - n_alloc];
    out[i] = v;
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
