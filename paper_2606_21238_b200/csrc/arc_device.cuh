// Device-side types shared by the kernels of libarc_b200 (sm_100a).  Nothing here is shared with oracle/.
//
// Directory layout in HBM:
//   Node[node_cap]      16 B records {list, pos, block, slot}; node ids are stable for the life of a key
//   node_key[node_cap]  the 64-bit key of each node (only needed by rebuilds and debug dumps)
//   Slot[table_slots]   open-addressing table, 16 B slots {key, node + 1}, buckets of 2 slots = one 32 B sector
//   ring[L][ring_cap]   one lazy FIFO of 8 B entries {node id, block id} per list L in {T1, T2, B1, B2}: an entry at absolute
//                       position q is *live* iff nodes[id].list == L && nodes[id].pos == q.  Every list
//                       insertion is at the MRU end (tail++), every LRU-end removal scans from head and
//                       skips stale entries; a hit leaves its old entry behind as stale.  Entries pushed
//                       during the current request are exactly the pinned ones (R4), so the victim scan
//                       simply stops at the tail position recorded when the request began.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace arc {

constexpr uint32_t L_ABSENT = 0, L_T1 = 1, L_T2 = 2, L_B1 = 3, L_B2 = 4, L_FREE = 5;
constexpr unsigned long long KEY_EMPTY = 0ull, KEY_TOMB = 1ull;  // H5 keeps real keys >= 2
constexpr uint32_t SLOT_NODE_PENDING = 0;        // Slot::node holds node id + 1; 0 = EMPTY slot, tombstone, or (inside K2 only) a key
                                                 // whose winner has not published its node id yet
constexpr uint32_t NODE_NONE = 0xFFFFFFFFu;
constexpr uint32_t NODE_HELD = 0x100u;           // Node::list flag (pin scope 2): the node is resident, has holds and is in NO ring;
                                                 // Node::pos then carries the hold count instead of a ring position
constexpr uint32_t NODE_LIST_MASK = 0xFFu;
constexpr uint32_t BUCKET_SLOTS = 2;             // 2 x 16 B = one 32 B sector: what one probe reads

enum : int { CLS_MISS = 0, CLS_HIT_T1 = 1, CLS_HIT_T2 = 2, CLS_GHOST_B1 = 3, CLS_GHOST_B2 = 4 };
enum : int { POLICY_ARC = 0, POLICY_LRU = 1, POLICY_DBL = 2 };

// Ring entry: low word = node id (RING_TOMB once the node has left that position by a hit / ghost hit), high word = the
// block id the node held when it was pushed.  Inside [head, tail) an entry is live iff it is not a tombstone; the node
// record (list, pos) stays the authoritative copy, used by the maintenance kernels and the by-the-book routine.
typedef unsigned long long RingEnt;
constexpr uint32_t RING_TOMB = 0xFFFFFFFFu;
__host__ __device__ __forceinline__ RingEnt ring_ent(uint32_t node, int32_t block) { return (RingEnt)node | ((RingEnt)(uint32_t)block << 32); }
__host__ __device__ __forceinline__ uint32_t ent_node(RingEnt e) { return (uint32_t)e; }
__host__ __device__ __forceinline__ int32_t ent_block(RingEnt e) { return (int32_t)(uint32_t)(e >> 32); }

struct __align__(16) Node {
  uint32_t list;   // L_*
  uint32_t pos;    // absolute ring position of the live entry (mod 2^32)
  int32_t block;   // physical block id if resident, -1 otherwise
  uint32_t slot;   // index of this key's table slot when K2 or a rebuild wrote the record; not maintained by K3 (see st_node_keep_slot)
};

struct __align__(16) Slot {
  unsigned long long key;
  uint32_t node;
  uint32_t pad;
};

// indices into DevState::stat
enum : int { ST_HIT_T1 = 0, ST_HIT_T2, ST_GHOST_B1, ST_GHOST_B2, ST_MISS, ST_EVICT_T1, ST_EVICT_T2, ST_DROP_B1,
             ST_DROP_B2, ST_FRESH, ST_PREFIX_TOKENS, ST_ACCESSES, ST_COUNT };
enum : uint32_t { DEV_ERR_NONE = 0, DEV_ERR_NODE_POOL = 1, DEV_ERR_NO_VICTIM = 2, DEV_ERR_RING_OVERFLOW = 3,
                  DEV_ERR_BAD_NODE = 4, DEV_ERR_BAD_RELEASE = 5 };

struct DevState {
  uint32_t head[5], tail[5];      // per list (index L_T1..L_B2); wrapping 32-bit absolute positions
  int32_t t1, t2, b1, b2;         // live sizes
  int32_t p;                      // target size of T1 (R6: integer)
  int32_t next_fresh;             // R8
  uint32_t free_top;              // number of ids on the free stack
  uint32_t counts[2];             // n_alloc, n_evict of the current step
  uint32_t error;                 // DEV_ERR_*
  uint32_t tombs;                 // tombstones currently in the table
  uint32_t k1_ticket;             // K1 work ticket and, right behind it, the count of warps that have left the launch:
  uint32_t k1_done;               // both 0 between launches (the last warp out resets them, hash_kernels.cuh k1_leave)
  unsigned long long stat[ST_COUNT];
  // scratch for ring compaction (old window of the list being compacted)
  uint32_t cmp_head[5], cmp_tail[5];
  // K3 diagnostics, cumulative (arc_debug_counters): see DBG_* below
  unsigned long long dbg[32];
  // pin scope 2: entries of T1 / T2 without holds (= the entries in the rings = the possible victims), kept across steps
  int32_t u1, u2;
  uint32_t release_bad;           // scratch of release_kernel
  uint32_t win_seq;               // K3 wide machine: number of the last window (31 bits, never 0), see node_stamp
  // by-the-book machine only (arc_set_machine(h, 1)): per-access latency in SM cycles (clock64 around serial_access) by
  // class, 16 logarithmic bins: bin b holds the accesses that took [64 * 2^(b-1), 64 * 2^b) cycles, bin 0 fewer than 64
  uint32_t lat_hist[5][16];
};
enum : int { DBG_WIN_HIT = 0, DBG_WIN_GENERAL, DBG_WIN_SERIAL, DBG_CUT_TWIN, DBG_CUT_CONFLICT, DBG_SCAN_ROUNDS, DBG_ACC_HIT_WIN,
             DBG_ACC_GENERAL_WIN, DBG_CYC_FETCH, DBG_CYC_ROLL, DBG_CYC_SCAN, DBG_CYC_APPLY, DBG_CYC_SERIAL, DBG_CYC_TOTAL, DBG_ROLL_CALLS, DBG_ROLL_PHASES,
             DBG_PROV_OK, DBG_PROV_MISS,   // pipelined wide machine: windows whose roll-ahead stood / had to be rolled on request
#ifdef ARC_PROBES
             DBG_PROBE0, DBG_PROBE_END = DBG_PROBE0 + 13,   // ad-hoc cycle probes of a diagnostic build (-DARC_PROBES), see PROBE()
#endif
             DBG_COUNT };
#ifdef ARC_PROBES
#define PROBE(i) do { const uint32_t t_ = (uint32_t)clock(); dbg[DBG_PROBE0 + (i)] += t_ - tp_; tp_ = t_; } while (0)
#define PROBE_RESET() do { tp_ = (uint32_t)clock(); } while (0)
#else
#define PROBE(i) do { } while (0)
#define PROBE_RESET() do { } while (0)
#endif

// Everything a step's kernels need, passed by value.
struct StepParams {
  DevState* state;
  Node* nodes;
  unsigned long long* node_key;
  uint32_t* free_stack;
  Slot* table;
  uint32_t bucket_mask;           // (table_slots / 8) - 1
  RingEnt* ring[5];
  uint32_t ring_mask;
  // step inputs
  const int32_t* tokens;
  const int64_t* offsets;         // [n_req+1] token offsets
  const int64_t* blk_off;         // [n_req+1]
  uint32_t n_req;
  uint32_t n_access;
  // step scratch (access order: index blk_off[r] + (nb_r - 1 - i))
  unsigned long long* keys_acc;
  uint32_t* node_acc;
  uint32_t* dropped;              // node made ABSENT by access a, or NODE_NONE
  // outputs (natural order: blk_off[r] + i)
  int32_t* prefix_len;
  uint8_t* cls;
  int32_t* block_id;
  int32_t* evicted_id;
  int32_t* p_after;
  int32_t* alloc_ids;
  int32_t* evict_ids;
  int32_t capacity;
  int32_t policy;
  uint32_t block_size;
  int32_t pin_scope;              // 0: pins end with their request, 1: with the step, 2: held until arc_release
  uint32_t* node_of_block;        // pin scope 2: node id of the resident entry that owns each block id
  uint32_t* node_stamp;           // [node_cap] K3 wide machine: number of the last window that accessed the node (twin check, speculation)
  uint32_t* counts_out;           // [2] copy of DevState::counts next to prefix_len / alloc_ids / evict_ids (one D2H copy in arc_step_host)
  unsigned long long key_and;     // test hook (arc_debug_set_key_mask): keys are ANDed with this before the probe; all ones normally
};

__device__ __forceinline__ Node ld_node(const Node* p) {
  // nodes are read-write shared between kernels of one stream only; within K3 they are re-read after
  // other threads of the CTA wrote them, so go to L2 (ld.cg) rather than trusting L1.
  uint4 v = __ldcg(reinterpret_cast<const uint4*>(p));
  Node n;
  n.list = v.x; n.pos = v.y; n.block = (int32_t)v.z; n.slot = v.w;
  return n;
}
__device__ __forceinline__ void st_node(Node* p, uint32_t list, uint32_t pos, int32_t block, uint32_t slot) {
  __stcg(reinterpret_cast<uint4*>(p), make_uint4(list, pos, (uint32_t)block, slot));
}
// A record written for a node whose record was never read (a victim or a dropped ghost, known from its ring entry): ONE
// 16-byte store.  The slot word is not kept up by K3 any more - K4 finds the table slot of a key that leaves the directory
// by probing for it (finalize_body) - because the two narrower stores that left it alone cost K3 one more random sector
// per victim and per dropped ghost, and K3's apply is bound by the store sectors its one SM can issue.
__device__ __forceinline__ void st_node_keep_slot(Node* p, uint32_t list, uint32_t pos, int32_t block) {
  __stcg(reinterpret_cast<uint4*>(p), make_uint4(list, pos, (uint32_t)block, 0u));
}

}  // namespace arc
