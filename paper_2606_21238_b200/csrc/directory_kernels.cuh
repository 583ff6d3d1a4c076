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
// Insert-if-absent: the lowest EMPTY slot of that bucket is claimed with ONE 128-bit compare-and-swap
// (atom.cas.b128, sm_90+) that writes key and node id together, so a slot is never seen half-published: there is no
// "claimed, node pending" state, no second pass and no spinning.  The node id is popped from the free stack before the
// CAS; a thread that loses the race (another thread took the slot - possibly for the same key, which the re-read of
// the bucket then finds) keeps the id for its next insert and hands a leftover to DevState::spare[], which K4 pushes
// back (pushes never run concurrently with pops).  Tombstones are not reused; rebuild_table clears them.
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
// {EMPTY, 0, 0} -> {key, node + 1, 0} in one atomic; true if this thread now owns the slot
__device__ __forceinline__ bool slot_claim(Slot* p, unsigned long long key, uint32_t node_plus_1) {
  unsigned long long ok, ov;
  asm volatile("{\n\t.reg .b128 c, n, o;\n\tmov.b128 c, {%2, %3};\n\tmov.b128 n, {%4, %5};\n\t"
               "atom.relaxed.gpu.global.cas.b128 o, [%6], c, n;\n\tmov.b128 {%0, %1}, o;\n\t}"
               : "=l"(ok), "=l"(ov) : "l"(0ull), "l"(0ull), "l"(key), "l"((unsigned long long)node_plus_1), "l"(p) : "memory");
  return ok == KEY_EMPTY && ov == 0ull;
}

// Finds or inserts `key`, starting with bucket content `b` already loaded for bucket index `bucket`.  `spare` is a node
// id this thread popped earlier and did not use (NODE_NONE if none).  Returns the node id, or NODE_NONE when the node
// pool is exhausted (sticky DEV_ERR_NODE_POOL: the step's results are void, K3 does not run).
__device__ __forceinline__ uint32_t probe_one(const StepParams& P, unsigned long long key, uint32_t bucket, Bucket b, uint32_t& spare) {
  for (;;) {
    if (b.s[0].key == key) return b.s[0].node - 1;
    if (b.s[1].key == key) return b.s[1].node - 1;
    const int e = (b.s[0].key == KEY_EMPTY) ? 0 : ((b.s[1].key == KEY_EMPTY) ? 1 : -1);
    if (e < 0) { bucket = (bucket + 1) & P.bucket_mask; b = ld_bucket(P.table + (size_t)bucket * BUCKET_SLOTS); continue; }
    if (spare == NODE_NONE) {
      const uint32_t top = atomicSub(&P.state->free_top, 1u);
      if (top == 0 || top > 0x7FFFFFFFu) {
        atomicAdd(&P.state->free_top, 1u);
        atomicExch(&P.state->error, DEV_ERR_NODE_POOL);
        return NODE_NONE;
      }
      spare = P.free_stack[top - 1];
    }
    const uint32_t idx = bucket * BUCKET_SLOTS + (uint32_t)e;
    st_node(P.nodes + spare, L_ABSENT, 0, -1, idx);        // read by K3 only, after the kernel boundary
    P.node_key[spare] = key;
    if (slot_claim(P.table + idx, key, spare + 1)) { const uint32_t got = spare; spare = NODE_NONE; return got; }
    b = ld_bucket(P.table + (size_t)bucket * BUCKET_SLOTS);   // lost the race for that slot: the winner may hold our key
  }
}

__device__ __forceinline__ void probe_range(const StepParams& P, uint32_t first, uint32_t stride) {
  uint32_t spare = NODE_NONE;
  for (uint32_t a0 = first; a0 < P.n_access; a0 += stride * PROBE_ILP) {
    unsigned long long key[PROBE_ILP];
    uint32_t bucket[PROBE_ILP];
    Bucket b[PROBE_ILP];
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) {
      const uint32_t a = a0 + u * stride;
      key[u] = (a < P.n_access) ? (__ldcg(P.keys_acc + a) & P.key_and) : 2ull;
      if (key[u] < 2) key[u] += 2;                   // 0 and 1 stay reserved under the test mask too
      bucket[u] = (uint32_t)key[u] & P.bucket_mask;
    }
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) b[u] = ld_bucket(P.table + (size_t)bucket[u] * BUCKET_SLOTS);
#pragma unroll
    for (int u = 0; u < PROBE_ILP; ++u) {
      const uint32_t a = a0 + u * stride;
      if (a < P.n_access) P.node_acc[a] = probe_one(P, key[u], bucket[u], b[u], spare);
    }
  }
  if (spare != NODE_NONE) P.spare[atomicAdd(&P.state->n_spare, 1u)] = spare;     // at most one per thread: P.spare has K2_MAX_THREADS entries
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

// Node ids that K2's threads popped and did not use go back on the free stack (no pop runs concurrently: K4, or the
// tail of arc_debug_probe).
__device__ __forceinline__ void return_spares(const StepParams& P, uint32_t tid, uint32_t nthr) {
  const uint32_t n = P.state->n_spare;
  for (uint32_t i = tid; i < n; i += nthr) {
    const uint32_t d = P.spare[i];
    st_node(P.nodes + d, L_FREE, 0, -1, 0);
    P.free_stack[atomicAdd(&P.state->free_top, 1u)] = d;
  }
}
__global__ void __launch_bounds__(256) return_spares_kernel(const __grid_constant__ StepParams P) {
  return_spares(P, threadIdx.x, blockDim.x);
  __syncthreads();
  if (threadIdx.x == 0) P.state->n_spare = 0;
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
    P.state->k1_ticket = 0;                                            // K1 of the next step starts from request 0
    P.counts_out[0] = P.state->counts[0]; P.counts_out[1] = P.state->counts[1];
  }
  if (blockIdx.x == 0 && P.state->n_spare) {                           // CTA-uniform (nobody writes n_spare during K4 but this CTA)
    return_spares(P, threadIdx.x, blockDim.x);
    __syncthreads();
    if (threadIdx.x == 0) P.state->n_spare = 0;
  }
}

__global__ void __launch_bounds__(256) finalize_kernel(const __grid_constant__ StepParams P) { finalize_body(P); }

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
