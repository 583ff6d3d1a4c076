// libarc_b200 — host side of the C ABI declared in include/arc.h.
// Validates, sizes buffers from the host offsets, enqueues the kernels on the caller's stream and owns
// all device buffers.  No torch types, no CPU fallback: every step of the path runs in the kernels.
#include <algorithm>
#include <atomic>
#include <cstdarg>
#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/arc.h"
#include "arc_device.cuh"
#include "directory_kernels.cuh"
#include "hash_kernels.cuh"
#include "machine_batched.cuh"
#include "machine_serial.cuh"
#include "machine_wide.cuh"
#include "hash_static.cuh"
#include "fused_small.cuh"

using namespace arc;

namespace {

thread_local std::string g_create_error = "";
std::atomic<uint64_t> g_hash_launches{0};

constexpr int kStageSlots = 4;
constexpr int kHostSlots = 3;                     // steps the host entry keeps in flight (arc_step_host_async)
constexpr uint32_t kMaxReq = 1u << 20;
constexpr uint64_t kMaxCapacity = 1ull << 28;   // node ids carry two flag bits
constexpr uint32_t kSegEndCap = 1u << 16;       // n_req * segments-per-request the segmented K1 is used up to
constexpr uint32_t kFusedAutoMax = 1536;        // steps of up to this many accesses take the one-launch kernel by default
constexpr uint32_t kSegMaxReq = 512;            // with more requests than this one warp per request already fills the GPU

uint32_t pow2_at_least(uint64_t x) {
  uint64_t p = 64;
  while (p < x) p <<= 1;
  return (uint32_t)p;
}

template <typename T>
cudaError_t dalloc(T** p, size_t n) {
  *p = nullptr;
  return cudaMalloc((void**)p, std::max<size_t>(n, 1) * sizeof(T));
}
template <typename T>
void dfree(T*& p) {
  if (p) cudaFree(p);
  p = nullptr;
}

}  // namespace

struct arc_cache {
  int device = 0;
  uint64_t c = 0;
  uint32_t B = 16;
  int policy = 0;
  unsigned long long key_and = ~0ull;   // test hook
  int pin_scope = ARC_PIN_REQUEST;
  int machine = 0;            // 0 auto (wide, or one-warp when requests are short), 1 serial, 2 one-warp, 3 wide with the roller warp, 4 one launch, 5 wide without it
  // capacities
  uint64_t n_cap = 0;         // max full blocks per step the buffers are sized for
  uint32_t req_cap = 0;
  uint32_t node_cap = 0, table_slots = 0, ring_cap = 0;
  // directory
  DevState* d_state = nullptr;
  Node* d_nodes = nullptr;
  unsigned long long* d_node_key = nullptr;
  uint32_t* d_free_stack = nullptr;
  uint32_t* d_node_stamp = nullptr;   // [node_cap] K3 wide machine: window numbers (twin check, speculation)
  unsigned long long* d_seg_end = nullptr;   // [kSegEndCap] end states of K1's segments (steps with few, long requests)
  Slot* d_table = nullptr;
  RingEnt* d_ring[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
  RingEnt* d_ring_alt[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
  uint32_t* d_block_counts = nullptr;
  // per-step buffers
  int64_t* d_offsets = nullptr;   // [2 * (req_cap + 1)] : token offsets, then blk_off
  unsigned long long* d_keys = nullptr;
  uint32_t* d_node_acc = nullptr;
  uint32_t* d_dropped = nullptr;
  int32_t* d_result_pack = nullptr;   // prefix_len[req_cap] | counts[2] | alloc_ids[n_cap] | evict_ids[n_cap]: same layout as h_result
  int32_t* d_prefix_len = nullptr;    // = d_result_pack
  unsigned long long* d_chain_state = nullptr;   // [req_cap] H4 state after each request's last full block
  uint8_t* d_cls = nullptr;
  int32_t *d_block_id = nullptr, *d_evicted_id = nullptr, *d_p_after = nullptr, *d_alloc_ids = nullptr, *d_evict_ids = nullptr;
  void* d_machine_scratch = nullptr;
  // pin scope 2 (held): block id -> node id, per-block scratch of arc_release, holds outstanding (host-side, exact)
  uint32_t* d_node_of_block = nullptr;
  uint32_t* d_rel_cnt = nullptr;
  uint64_t hold_units = 0;
  // host staging
  int64_t* h_stage = nullptr;     // pinned, kStageSlots * 2 * (req_cap + 1)
  cudaEvent_t stage_done[kStageSlots] = {};
  int stage_next = 0;
  // arc_step_host
  // arc_step_host_async / _wait: kHostSlots steps in flight.  Per slot a device copy of the step's tokens (filled on the
  // handle's own copy stream) and a pinned, device-mapped host buffer that K4's pack kernel writes the results into.
  int32_t* d_tok[kHostSlots] = {};
  uint64_t tok_cap[kHostSlots] = {};
  int32_t* h_out[kHostSlots] = {};        // pinned + mapped: n_alloc | n_evict | error | prefix_len[n_req] | alloc_ids[n_alloc] | evict_ids[n_evict]
  cudaEvent_t ev_h2d[kHostSlots] = {}, ev_comp[kHostSlots] = {};
  uint32_t slot_ticket[kHostSlots] = {};  // 0 = free
  uint32_t slot_n_req[kHostSlots] = {};
  uint64_t slot_n_access[kHostSlots] = {}, slot_h2d[kHostSlots] = {};
  uint32_t next_ticket = 1;
  cudaStream_t copy_stream = nullptr;
  // host-side conservative bounds (no device read-back on the hot path)
  uint64_t slots_used_bound = 0;
  uint64_t window_bound[5] = {0, 0, 0, 0, 0};
  // host counters
  uint64_t steps = 0, requests = 0, tokens_seen = 0, tokens_hashed = 0;
  uint64_t launches = 0;
  cudaStream_t last_stream = nullptr;
  // profiling
  bool profiling = false;
  cudaEvent_t ev[7] = {};
  bool ev_valid = false;
  bool poisoned = false;      // a growth step failed half way (see ensure_capacity): every later call fails
  std::string err;
};

namespace {

int fail(arc_cache* h, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  if (h) h->err = buf; else g_create_error = buf;
  return code;
}

#define CUDA_TRY(h, expr)                                                                              \
  do {                                                                                                 \
    cudaError_t e_ = (expr);                                                                           \
    if (e_ != cudaSuccess) {                                                                           \
      int code_ = (e_ == cudaErrorMemoryAllocation) ? ARC_ERR_OOM : ARC_ERR_CUDA;                      \
      return fail(h, code_, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
    }                                                                                                  \
  } while (0)

StepParams make_params(arc_cache* h) {
  StepParams P;
  memset(&P, 0, sizeof(P));
  P.state = h->d_state; P.nodes = h->d_nodes; P.node_key = h->d_node_key; P.free_stack = h->d_free_stack;
  P.table = h->d_table; P.bucket_mask = h->table_slots / BUCKET_SLOTS - 1;
  for (int L = 1; L <= 4; ++L) P.ring[L] = h->d_ring[L];
  P.ring_mask = h->ring_cap - 1;
  P.offsets = h->d_offsets; P.blk_off = h->d_offsets + (h->req_cap + 1);
  P.keys_acc = h->d_keys; P.node_acc = h->d_node_acc; P.dropped = h->d_dropped;
  P.prefix_len = h->d_prefix_len; P.cls = h->d_cls; P.block_id = h->d_block_id; P.evicted_id = h->d_evicted_id;
  P.p_after = h->d_p_after; P.alloc_ids = h->d_alloc_ids; P.evict_ids = h->d_evict_ids;
  P.capacity = (int32_t)h->c; P.policy = h->policy; P.block_size = h->B; P.key_and = h->key_and; P.pin_scope = h->pin_scope;
  P.node_of_block = h->d_node_of_block;
  P.node_stamp = h->d_node_stamp;
  P.counts_out = reinterpret_cast<uint32_t*>(h->d_result_pack + h->req_cap);
  return P;
}

uint32_t grid_for(uint64_t work_items, uint32_t per_block, uint32_t max_blocks) {
  uint64_t b = (work_items + per_block - 1) / per_block;
  return (uint32_t)std::max<uint64_t>(1, std::min<uint64_t>(b, max_blocks));
}

int launch_rebuild(arc_cache* h, cudaStream_t s) {
  CUDA_TRY(h, cudaMemsetAsync(h->d_table, 0, (size_t)h->table_slots * sizeof(Slot), s));   // key 0 = EMPTY
  rebuild_table_kernel<<<grid_for(h->node_cap, 256, 148 * 8), 256, 0, s>>>(h->d_state, h->d_nodes, h->d_node_key, h->node_cap,
                                                                          h->d_table, h->table_slots / BUCKET_SLOTS - 1);
  h->launches += 1;
  CUDA_TRY(h, cudaGetLastError());
  h->slots_used_bound = std::min<uint64_t>(h->slots_used_bound, 2 * h->c);
  return ARC_OK;
}

// compacts lists L .. L + n_lists - 1 from d_ring[] (capacity src_cap) into d_ring_alt[] (capacity dst_cap) and swaps them:
// one pair of launches whatever n_lists is
int launch_compact(arc_cache* h, cudaStream_t s, int L, uint32_t src_cap, uint32_t dst_cap, int n_lists = 1) {
  const uint32_t blocks = std::max<uint32_t>(1, src_cap / CMP_THREADS);
  RingPtrs rp;
  for (int X = 0; X <= 4; ++X) { rp.src[X] = h->d_ring[X]; rp.dst[X] = h->d_ring_alt[X]; }
  const dim3 grid(blocks, (unsigned)n_lists);
  ring_count_kernel<<<grid, CMP_THREADS, 0, s>>>(h->d_state, h->d_nodes, rp, src_cap - 1, (uint32_t)L, h->d_block_counts);
  ring_scatter_kernel<<<grid, CMP_THREADS, 0, s>>>(h->d_state, h->d_nodes, rp, src_cap - 1, dst_cap - 1, (uint32_t)L, h->d_block_counts);
  h->launches += 2;
  CUDA_TRY(h, cudaGetLastError());
  for (int X = L; X < L + n_lists; ++X) {
    std::swap(h->d_ring[X], h->d_ring_alt[X]);
    h->window_bound[X] = std::min<uint64_t>(h->window_bound[X], h->c);
  }
  return ARC_OK;
}

// The buffers whose size follows the largest step seen (req_cap requests, n_cap full blocks).
struct StepBuffers {
  int64_t* d_offsets = nullptr;
  unsigned long long* d_keys = nullptr;
  uint32_t* d_node_acc = nullptr;
  uint32_t* d_dropped = nullptr;
  int32_t* d_result_pack = nullptr;
  unsigned long long* d_chain_state = nullptr;
  uint8_t* d_cls = nullptr;
  int32_t *d_block_id = nullptr, *d_evicted_id = nullptr, *d_p_after = nullptr;
  int64_t* h_stage = nullptr;
  int32_t* h_out[kHostSlots] = {};
};

void free_step_buffers(StepBuffers& b) {
  dfree(b.d_offsets); dfree(b.d_keys); dfree(b.d_node_acc); dfree(b.d_dropped); dfree(b.d_result_pack);
  dfree(b.d_chain_state); dfree(b.d_cls); dfree(b.d_block_id); dfree(b.d_evicted_id); dfree(b.d_p_after);
  if (b.h_stage) cudaFreeHost(b.h_stage);
  b.h_stage = nullptr;
  for (int k = 0; k < kHostSlots; ++k) { if (b.h_out[k]) cudaFreeHost(b.h_out[k]); b.h_out[k] = nullptr; }
}

int alloc_step_buffers(arc_cache* h, StepBuffers& b, uint32_t req_cap, uint64_t n_cap) {
  CUDA_TRY(h, dalloc(&b.d_offsets, 2 * ((size_t)req_cap + 1)));
  CUDA_TRY(h, dalloc(&b.d_keys, n_cap));
  CUDA_TRY(h, dalloc(&b.d_node_acc, n_cap));
  CUDA_TRY(h, dalloc(&b.d_dropped, n_cap));
  CUDA_TRY(h, dalloc(&b.d_result_pack, (size_t)req_cap + 2 + 2 * n_cap));
  CUDA_TRY(h, dalloc(&b.d_chain_state, req_cap));
  CUDA_TRY(h, dalloc(&b.d_cls, n_cap));
  CUDA_TRY(h, dalloc(&b.d_block_id, n_cap));
  CUDA_TRY(h, dalloc(&b.d_evicted_id, n_cap));
  CUDA_TRY(h, dalloc(&b.d_p_after, n_cap));
  CUDA_TRY(h, cudaMallocHost((void**)&b.h_stage, (size_t)kStageSlots * 2 * ((size_t)req_cap + 1) * sizeof(int64_t)));
  for (int k = 0; k < kHostSlots; ++k)
    CUDA_TRY(h, cudaHostAlloc((void**)&b.h_out[k], ((size_t)req_cap + 4 + 2 * n_cap) * sizeof(int32_t), cudaHostAllocMapped));
  return ARC_OK;
}

StepBuffers take_step_buffers(arc_cache* h) {
  StepBuffers b;
  b.d_offsets = h->d_offsets; b.d_keys = h->d_keys; b.d_node_acc = h->d_node_acc; b.d_dropped = h->d_dropped;
  b.d_result_pack = h->d_result_pack; b.d_chain_state = h->d_chain_state; b.d_cls = h->d_cls; b.d_block_id = h->d_block_id;
  b.d_evicted_id = h->d_evicted_id; b.d_p_after = h->d_p_after; b.h_stage = h->h_stage;
  for (int k = 0; k < kHostSlots; ++k) b.h_out[k] = h->h_out[k];
  return b;
}

void install_step_buffers(arc_cache* h, const StepBuffers& b, uint32_t req_cap, uint64_t n_cap) {
  h->d_offsets = b.d_offsets; h->d_keys = b.d_keys; h->d_node_acc = b.d_node_acc; h->d_dropped = b.d_dropped;
  h->d_result_pack = b.d_result_pack; h->d_chain_state = b.d_chain_state; h->d_cls = b.d_cls; h->d_block_id = b.d_block_id;
  h->d_evicted_id = b.d_evicted_id; h->d_p_after = b.d_p_after; h->h_stage = b.h_stage;
  for (int k = 0; k < kHostSlots; ++k) h->h_out[k] = b.h_out[k];
  h->d_prefix_len = b.d_result_pack;
  h->d_alloc_ids = b.d_result_pack ? b.d_result_pack + req_cap + 2 : nullptr;
  h->d_evict_ids = b.d_result_pack ? h->d_alloc_ids + n_cap : nullptr;
  h->req_cap = req_cap; h->n_cap = n_cap;
}

// Makes every buffer large enough for steps of (n_req, N).  Directory content is preserved.  Transactional towards the
// caller: every part (node pool, table, rings, step buffers) is grown into new memory and committed only when it is
// complete, and the sizes a step is checked against (req_cap, n_cap) are committed LAST, so a failure (out of memory,
// the 30-bit node index) leaves a handle that works as before and simply tries again on the next larger step.  The one
// failure that cannot be undone (a launch error while the rings move) poisons the handle: every later call fails.
int ensure_capacity(arc_cache* h, uint32_t n_req, uint64_t N, cudaStream_t s) {
  if (h->poisoned) return fail(h, ARC_ERR_CUDA, "the handle is unusable after an earlier CUDA failure during growth");
  if (n_req <= h->req_cap && N <= h->n_cap && h->d_state) return ARC_OK;
  const bool first = (h->d_state == nullptr);
  const uint32_t req_cap = std::max<uint32_t>(first ? 64 : h->req_cap, pow2_at_least(n_req));
  uint64_t n_cap = std::max<uint64_t>(first ? 4096 : h->n_cap, N);
  if (!first && N > h->n_cap) n_cap = std::max<uint64_t>(n_cap, h->n_cap * 2);
  const uint64_t node_cap64 = 2 * h->c + n_cap + 64;
  if (node_cap64 >= (1ull << 30)) return fail(h, ARC_ERR_UNSUPPORTED, "directory of %llu nodes exceeds the 30-bit node index", (unsigned long long)node_cap64);
  const uint32_t node_cap = (uint32_t)node_cap64;
  const uint32_t table_slots = pow2_at_least(2 * node_cap64);
  const uint32_t ring_cap = pow2_at_least(2 * (h->c + n_cap));
  if (!first) CUDA_TRY(h, cudaDeviceSynchronize());   // results of earlier steps die here (documented)

  if (first) {
    StepBuffers nb;
    int rc = alloc_step_buffers(h, nb, req_cap, n_cap);
    if (rc) { free_step_buffers(nb); return rc; }
    install_step_buffers(h, nb, req_cap, n_cap);     // arc_create destroys the handle if anything below fails
    CUDA_TRY(h, dalloc(&h->d_state, 1));
    CUDA_TRY(h, dalloc(&h->d_nodes, node_cap));
    CUDA_TRY(h, dalloc(&h->d_node_key, node_cap));
    CUDA_TRY(h, dalloc(&h->d_free_stack, node_cap));
    CUDA_TRY(h, dalloc(&h->d_node_stamp, node_cap));
    CUDA_TRY(h, cudaMemsetAsync(h->d_node_stamp, 0, (size_t)node_cap * sizeof(uint32_t), s));
    CUDA_TRY(h, dalloc(&h->d_table, table_slots));
    for (int L = 1; L <= 4; ++L) {
      CUDA_TRY(h, dalloc(&h->d_ring[L], ring_cap));
      CUDA_TRY(h, dalloc(&h->d_ring_alt[L], ring_cap));
    }
    CUDA_TRY(h, dalloc(&h->d_block_counts, 4 * (size_t)std::max<uint32_t>(1, ring_cap / CMP_THREADS)));
    h->node_cap = node_cap; h->table_slots = table_slots; h->ring_cap = ring_cap;
    CUDA_TRY(h, cudaMemsetAsync(h->d_table, 0, (size_t)table_slots * sizeof(Slot), s));
    init_state_kernel<<<grid_for(node_cap, 256, 148 * 8), 256, 0, s>>>(h->d_state, h->d_nodes, h->d_free_stack, node_cap, (h->policy == ARC_POLICY_DBL) ? (int32_t)(h->c / 2) : 0);
    h->launches += 1;
    CUDA_TRY(h, cudaGetLastError());
    h->slots_used_bound = 0;
    for (int L = 1; L <= 4; ++L) h->window_bound[L] = 0;
    return ARC_OK;
  }

  // (1) the new step buffers, kept aside until everything else has grown
  StepBuffers nb;
  int rc = alloc_step_buffers(h, nb, req_cap, n_cap);
  if (rc) { free_step_buffers(nb); return rc; }

  if (node_cap > h->node_cap) {       // (2) the node pool; ids are stable
    Node* nodes = nullptr; unsigned long long* keys = nullptr; uint32_t* stack = nullptr; uint32_t* stamp = nullptr;
    cudaError_t e = dalloc(&nodes, node_cap);
    if (e == cudaSuccess) e = dalloc(&keys, node_cap);
    if (e == cudaSuccess) e = dalloc(&stack, node_cap);
    if (e == cudaSuccess) e = dalloc(&stamp, node_cap);
    if (e != cudaSuccess) {
      dfree(nodes); dfree(keys); dfree(stack); dfree(stamp); free_step_buffers(nb);
      cudaGetLastError();
      return fail(h, ARC_ERR_OOM, "growing the node pool to %u nodes: %s", node_cap, cudaGetErrorString(e));
    }
    e = cudaMemcpyAsync(nodes, h->d_nodes, (size_t)h->node_cap * sizeof(Node), cudaMemcpyDeviceToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(keys, h->d_node_key, (size_t)h->node_cap * sizeof(unsigned long long), cudaMemcpyDeviceToDevice, s);
    if (e == cudaSuccess) e = cudaMemsetAsync(stamp, 0, (size_t)node_cap * sizeof(uint32_t), s);   // stamps only matter inside a step
    if (e == cudaSuccess) {
      // the new stack is built from the old one without touching it; DevState::free_top moves only when all of it worked
      extend_free_stack_kernel<<<grid_for(node_cap, 256, 148 * 8), 256, 0, s>>>(h->d_state, nodes, h->d_free_stack, stack, h->node_cap, node_cap);
      h->launches += 1;
      e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) {
      dfree(nodes); dfree(keys); dfree(stack); dfree(stamp); free_step_buffers(nb);
      return fail(h, ARC_ERR_CUDA, "growing the node pool: %s", cudaGetErrorString(e));
    }
    bump_free_top_kernel<<<1, 1, 0, s>>>(h->d_state, node_cap - h->node_cap);
    h->launches += 1;
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) {           // the old pool is still whole and still the handle's
      dfree(nodes); dfree(keys); dfree(stack); dfree(stamp); free_step_buffers(nb);
      return fail(h, ARC_ERR_CUDA, "growing the node pool: %s", cudaGetErrorString(e));
    }
    dfree(h->d_nodes); dfree(h->d_node_key); dfree(h->d_free_stack); dfree(h->d_node_stamp);
    h->d_nodes = nodes; h->d_node_key = keys; h->d_free_stack = stack; h->d_node_stamp = stamp; h->node_cap = node_cap;
  }
  if (table_slots > h->table_slots) {  // (3) the table: rebuilt from the node records into new memory
    Slot* table = nullptr;
    cudaError_t e = dalloc(&table, table_slots);
    if (e != cudaSuccess) {
      free_step_buffers(nb);
      cudaGetLastError();
      return fail(h, ARC_ERR_OOM, "growing the table to %u slots: %s", table_slots, cudaGetErrorString(e));
    }
    Slot* old = h->d_table; const uint32_t old_slots = h->table_slots;
    h->d_table = table; h->table_slots = table_slots;
    rc = launch_rebuild(h, s);          // writes the nodes' slot fields: from here on only the new table is valid
    if (rc == ARC_OK && cudaStreamSynchronize(s) != cudaSuccess) rc = fail(h, ARC_ERR_CUDA, "rebuilding the table failed");
    if (rc) { (void)old_slots; dfree(old); free_step_buffers(nb); h->poisoned = true; return rc; }
    dfree(old);
  }
  if (ring_cap > h->ring_cap) {        // (4) the four rings: all eight new buffers first, then one compaction moves the lists
    RingEnt* nr[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    RingEnt* na[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    uint32_t* counts = nullptr;
    cudaError_t e = dalloc(&counts, 4 * (size_t)std::max<uint32_t>(1, ring_cap / CMP_THREADS));
    for (int L = 1; L <= 4 && e == cudaSuccess; ++L) { e = dalloc(&nr[L], ring_cap); if (e == cudaSuccess) e = dalloc(&na[L], ring_cap); }
    if (e != cudaSuccess) {
      for (int L = 1; L <= 4; ++L) { dfree(nr[L]); dfree(na[L]); }
      dfree(counts); free_step_buffers(nb);
      cudaGetLastError();
      return fail(h, ARC_ERR_OOM, "growing the rings to %u entries: %s", ring_cap, cudaGetErrorString(e));
    }
    dfree(h->d_block_counts); h->d_block_counts = counts;
    for (int L = 1; L <= 4; ++L) { dfree(h->d_ring_alt[L]); h->d_ring_alt[L] = nr[L]; }
    rc = launch_compact(h, s, 1, h->ring_cap, ring_cap, 4);   // swaps: d_ring[] are the big ones now, d_ring_alt[] the old small ones
    if (rc == ARC_OK && cudaStreamSynchronize(s) != cudaSuccess) rc = fail(h, ARC_ERR_CUDA, "moving the rings failed");
    if (rc) { for (int L = 1; L <= 4; ++L) dfree(na[L]); free_step_buffers(nb); h->poisoned = true; return rc; }
    for (int L = 1; L <= 4; ++L) { dfree(h->d_ring_alt[L]); h->d_ring_alt[L] = na[L]; }
    h->ring_cap = ring_cap;
  }
  // (5) commit: the step buffers and, last of all, the sizes steps are checked against
  StepBuffers old = take_step_buffers(h);
  free_step_buffers(old);
  install_step_buffers(h, nb, req_cap, n_cap);
  return ARC_OK;
}

// Directory upkeep before a step of N accesses, decided from host-side upper bounds only.
int maintain(arc_cache* h, uint64_t N, cudaStream_t s) {
  // buckets are one 32-byte sector = 2 slots: beyond a load of about 0.45 (live keys + tombstones) the probe chains grow
  if (h->slots_used_bound + N > (uint64_t)(0.45 * h->table_slots)) {
    int rc = launch_rebuild(h, s);
    if (rc) return rc;
  }
  bool due = false;
  for (int L = 1; L <= 4; ++L) due = due || (h->window_bound[L] + N > h->ring_cap);
  if (due) {                             // the bounds grow together: all four lists in one pair of launches
    int rc = launch_compact(h, s, 1, h->ring_cap, h->ring_cap, 4);
    if (rc) return rc;
  }
  return ARC_OK;
}

int validate_offsets(arc_cache* h, const int64_t* off, uint32_t n_req, uint32_t B, uint64_t c, int64_t* blk_off_out, uint64_t* N_out) {
  if (off[0] < 0) return fail(h, ARC_ERR_INVALID_ARG, "h_offsets[0] < 0");
  uint64_t N = 0;
  for (uint32_t r = 0; r < n_req; ++r) {
    if (off[r + 1] < off[r]) return fail(h, ARC_ERR_INVALID_ARG, "h_offsets not monotone at request %u", r);
    const uint64_t nb = (B == 16) ? ((uint64_t)(off[r + 1] - off[r]) >> 4) : ((uint64_t)(off[r + 1] - off[r]) / B);
    if (c && nb > c) return fail(h, ARC_ERR_REQUEST_TOO_LARGE, "request %u has %llu blocks > capacity %llu", r, (unsigned long long)nb, (unsigned long long)c);
    if (blk_off_out) blk_off_out[r] = (int64_t)N;
    N += nb;
  }
  if (blk_off_out) blk_off_out[n_req] = (int64_t)N;
  if (N >= (1ull << 31)) return fail(h, ARC_ERR_INVALID_ARG, "step of %llu blocks is too large", (unsigned long long)N);
  *N_out = N;
  return ARC_OK;
}

// ---- K1 launches --------------------------------------------------------------------------------------------------
// The hashing kernels stage tokens in dynamic shared memory (K1_SMEM_BYTES per CTA, above the 48 KB default): the
// attribute is set once per process and device.
enum { K1_ARG_NONE = 0, K1_ARG_SMALL = 1, K1_ARG_LARGE = 2 };
struct K1HostArgs { OffsetsArgT<0> none; OffsetsArgT<K1_INLINE_SMALL> small; OffsetsArgT<K1_INLINE_LARGE> large; };

cudaError_t k1_configure() {
  static std::mutex mu;
  static bool done[64] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(mu);
  if (dev >= 0 && dev < 64 && done[dev]) return cudaSuccess;
#define K1_ATTR(f) if ((e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, K1_SMEM_BYTES)) != cudaSuccess) return e
  K1_ATTR((hash_blocks_kernel<false, false, 0>));
  K1_ATTR((hash_blocks_kernel<true, true, 0>));
  K1_ATTR((hash_blocks_kernel<true, true, (int)K1_INLINE_SMALL>));
  K1_ATTR((hash_blocks_kernel<true, true, (int)K1_INLINE_LARGE>));
  K1_ATTR((hash_segments_kernel<0>));
  K1_ATTR((hash_segments_kernel<(int)K1_INLINE_SMALL>));
  K1_ATTR((hash_segments_kernel<(int)K1_INLINE_LARGE>));
  K1_ATTR((arc_fused_small_kernel<false, false>));
  K1_ATTR((arc_fused_small_kernel<false, true>));
  K1_ATTR((arc_fused_small_kernel<true, false>));
  K1_ATTR((arc_fused_small_kernel<true, true>));
  K1_ATTR(hash_items_kernel);
#undef K1_ATTR
  if (dev >= 0 && dev < 64) done[dev] = true;
  return cudaSuccess;
}

int k1_arg_mode(uint32_t n_req) { return n_req <= K1_INLINE_SMALL ? K1_ARG_SMALL : (n_req <= K1_INLINE_LARGE ? K1_ARG_LARGE : K1_ARG_NONE); }

// offsets[n_req + 1] and blk_off[n_req + 1] side by side in the argument of the right size
void k1_fill_args(K1HostArgs& A, int mode, const int64_t* off, const int64_t* blk_off, uint32_t n_req) {
  long long* v = (mode == K1_ARG_SMALL) ? A.small.v : A.large.v;
  memcpy(v, off, ((size_t)n_req + 1) * sizeof(int64_t));
  memcpy(v + n_req + 1, blk_off, ((size_t)n_req + 1) * sizeof(int64_t));
}

// K1 grid: persistent warps that take requests through the ticket; enough CTAs to fill the 148 SMs three deep, never more
// warps than requests.  step = true: keys in access order, chain states in and out (arc_step); false: arc_hash_blocks.
void launch_hash_blocks(bool step, int mode, const K1HostArgs& A, const int32_t* d_tokens, int64_t* d_offsets, int64_t* d_blk_off,
                        uint32_t n_req, unsigned long long* d_keys, uint32_t* d_ticket, cudaStream_t s,
                        const unsigned long long* d_chain_in, unsigned long long* d_chain_out) {
  const uint32_t blocks = grid_for(n_req, K1_WARPS, 148 * 3);
  if (!step)
    hash_blocks_kernel<false, false, 0><<<blocks, 256, K1_SMEM_BYTES, s>>>(d_tokens, d_offsets, d_blk_off, n_req, d_keys, d_ticket, nullptr, nullptr, A.none);
  else if (mode == K1_ARG_SMALL)
    hash_blocks_kernel<true, true, (int)K1_INLINE_SMALL><<<blocks, 256, K1_SMEM_BYTES, s>>>(d_tokens, d_offsets, d_blk_off, n_req, d_keys, d_ticket, d_chain_in, d_chain_out, A.small);
  else if (mode == K1_ARG_LARGE)
    hash_blocks_kernel<true, true, (int)K1_INLINE_LARGE><<<blocks, 256, K1_SMEM_BYTES, s>>>(d_tokens, d_offsets, d_blk_off, n_req, d_keys, d_ticket, d_chain_in, d_chain_out, A.large);
  else
    hash_blocks_kernel<true, true, 0><<<blocks, 256, K1_SMEM_BYTES, s>>>(d_tokens, d_offsets, d_blk_off, n_req, d_keys, d_ticket, d_chain_in, d_chain_out, A.none);
}

void launch_hash_segments(int mode, const K1HostArgs& A, const int32_t* d_tokens, int64_t* d_offsets, int64_t* d_blk_off, uint32_t n_req,
                          uint32_t max_seg, unsigned long long* d_states, unsigned long long* d_seg_end, uint32_t* d_ticket, cudaStream_t s) {
  const uint32_t g = grid_for((uint64_t)n_req * max_seg, K1_WARPS, 148 * 3);
  if (mode == K1_ARG_SMALL)
    hash_segments_kernel<(int)K1_INLINE_SMALL><<<g, 256, K1_SMEM_BYTES, s>>>(d_tokens, d_offsets, d_blk_off, n_req, max_seg, d_states, d_seg_end, d_ticket, A.small);
  else if (mode == K1_ARG_LARGE)
    hash_segments_kernel<(int)K1_INLINE_LARGE><<<g, 256, K1_SMEM_BYTES, s>>>(d_tokens, d_offsets, d_blk_off, n_req, max_seg, d_states, d_seg_end, d_ticket, A.large);
  else
    hash_segments_kernel<0><<<g, 256, K1_SMEM_BYTES, s>>>(d_tokens, d_offsets, d_blk_off, n_req, max_seg, d_states, d_seg_end, d_ticket, A.none);
}

// host-side bookkeeping after a step's kernels are enqueued, and the result struct
int finish_step(arc_cache* h, const int64_t* h_offsets, uint32_t n_req, uint64_t N, cudaStream_t s, const StepParams& P, arc_step_result* out) {
  h->slots_used_bound += N;
  for (int L = 1; L <= 4; ++L) h->window_bound[L] += N;
  if (h->pin_scope == ARC_PIN_HELD) h->hold_units += N;
  h->steps += 1; h->requests += n_req;
  h->tokens_seen += (uint64_t)(h_offsets[n_req] - h_offsets[0]);
  h->tokens_hashed += N * h->B;
  h->last_stream = s;

  out->n_access = N;
  out->prefix_len = h->d_prefix_len; out->blk_off = P.blk_off; out->cls = h->d_cls; out->block_id = h->d_block_id;
  out->evicted_id = h->d_evicted_id; out->p_after = h->d_p_after; out->alloc_ids = h->d_alloc_ids;
  out->evict_ids = h->d_evict_ids;
  out->chain_state = reinterpret_cast<const uint64_t*>(h->d_chain_state);
  out->counts = reinterpret_cast<const uint32_t*>(reinterpret_cast<const char*>(h->d_state) + offsetof(DevState, counts));
  return ARC_OK;
}

}  // namespace

extern "C" {

int arc_create(uint64_t capacity_blocks, uint32_t block_size, int policy, arc_cache** out) {
  if (!out) return fail(nullptr, ARC_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (capacity_blocks == 0 || capacity_blocks > 0x7FFFFFFEull) return fail(nullptr, ARC_ERR_INVALID_ARG, "capacity_blocks out of range");
  if (policy != ARC_POLICY_ARC && policy != ARC_POLICY_LRU && policy != ARC_POLICY_DBL) return fail(nullptr, ARC_ERR_INVALID_ARG, "unknown policy %d", policy);
  if (block_size != 16) return fail(nullptr, ARC_ERR_UNSUPPORTED, "block_size %u: only 16 is built", block_size);
  if (capacity_blocks > kMaxCapacity) return fail(nullptr, ARC_ERR_UNSUPPORTED, "capacity_blocks > 2^28");
  arc_cache* h = new (std::nothrow) arc_cache();
  if (!h) return fail(nullptr, ARC_ERR_OOM, "host allocation failed");
  h->c = capacity_blocks; h->B = block_size; h->policy = policy;
  cudaError_t e = cudaGetDevice(&h->device);
  if (e != cudaSuccess) {
    int rc = fail(nullptr, ARC_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    delete h;
    return rc;
  }
  e = k1_configure();
  if (e != cudaSuccess) {
    int rc = fail(nullptr, ARC_ERR_CUDA, "K1 configuration: %s", cudaGetErrorString(e));
    delete h;
    return rc;
  }
  for (int i = 0; i < kStageSlots; ++i) cudaEventCreateWithFlags(&h->stage_done[i], cudaEventDisableTiming);
  for (int i = 0; i < 7; ++i) cudaEventCreate(&h->ev[i]);
  int rc = ensure_capacity(h, 64, std::max<uint64_t>(4096, std::min<uint64_t>(capacity_blocks, 1u << 20)), nullptr);
  if (rc == ARC_OK) {
    cudaError_t e2 = cudaStreamSynchronize(nullptr);
    if (e2 != cudaSuccess) rc = fail(h, ARC_ERR_CUDA, "init: %s", cudaGetErrorString(e2));
  }
  if (rc != ARC_OK) {
    g_create_error = h->err;
    arc_destroy(h);
    return rc;
  }
  *out = h;
  return ARC_OK;
}

int arc_reserve(arc_cache* h, uint32_t max_req, uint64_t max_blocks_per_step) {
  if (!h) return ARC_ERR_INVALID_ARG;
  if (max_req > kMaxReq) return fail(h, ARC_ERR_INVALID_ARG, "max_req > 2^20");
  return ensure_capacity(h, max_req, max_blocks_per_step, h->last_stream);
}

int arc_step(arc_cache* h, const int32_t* d_tokens, const int64_t* h_offsets, uint32_t n_req, void* cuda_stream, arc_step_result* out) {
  return arc_step_resume(h, d_tokens, h_offsets, nullptr, n_req, cuda_stream, out);
}

int arc_step_resume(arc_cache* h, const int32_t* d_tokens, const int64_t* h_offsets, const uint64_t* d_chain_in, uint32_t n_req,
                    void* cuda_stream, arc_step_result* out) {
  if (!h) return ARC_ERR_INVALID_ARG;
  if (!h_offsets || !out) return fail(h, ARC_ERR_INVALID_ARG, "NULL argument");
  if (n_req > kMaxReq) return fail(h, ARC_ERR_INVALID_ARG, "n_req > 2^20");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  // validation + block offsets on the host (a0), into a scratch vector first: no state change on error
  static thread_local std::vector<int64_t> blk_off;
  blk_off.resize((size_t)n_req + 1);
  uint64_t N = 0;
  int rc = validate_offsets(h, h_offsets, n_req, h->B, h->c, blk_off.data(), &N);
  if (rc) return rc;
  if (h->pin_scope == ARC_PIN_STEP && N > h->c)
    return fail(h, ARC_ERR_REQUEST_TOO_LARGE, "step-wide pins: the step holds %llu blocks > capacity %llu", (unsigned long long)N, (unsigned long long)h->c);
  if (h->pin_scope == ARC_PIN_HELD && h->hold_units + N > h->c)
    return fail(h, ARC_ERR_REQUEST_TOO_LARGE, "held pins: %llu holds outstanding + %llu blocks in the step > capacity %llu",
                (unsigned long long)h->hold_units, (unsigned long long)N, (unsigned long long)h->c);
  if (!d_tokens && h_offsets[n_req] > h_offsets[0]) return fail(h, ARC_ERR_INVALID_ARG, "d_tokens is NULL");

  rc = ensure_capacity(h, n_req, N, s);
  if (rc) return rc;
  if (h->profiling) cudaEventRecord(h->ev[0], s);
  rc = maintain(h, N, s);
  if (rc) return rc;
  if (h->profiling) cudaEventRecord(h->ev[1], s);

  // host -> device boundary #1: offsets and block offsets (<= 16 MB at n_req = 2^20, usually a few KB)
  uint64_t max_nb = 0;
  for (uint32_t r = 0; r < n_req; ++r) max_nb = std::max<uint64_t>(max_nb, (uint64_t)(blk_off[r + 1] - blk_off[r]));
  const uint32_t max_seg = (uint32_t)((max_nb + K1_SEG - 1) / K1_SEG);
  const bool segmented = N && n_req <= kSegMaxReq && max_seg >= 2 && max_seg <= 1024 && (uint64_t)n_req * max_seg <= kSegEndCap;
  static thread_local K1HostArgs k1_args;
  // small steps: K1-K4 as the phases of one kernel (fused_small.cuh); arc_set_machine(h, 4) asks for it whenever it fits
  const bool fused = N && n_req <= K1_INLINE_SMALL && N <= FUSED_MAX_ACCESS &&
                     (h->machine == 4 || (h->machine == 0 && N <= kFusedAutoMax));
  if (fused) {
    k1_fill_args(k1_args, K1_ARG_SMALL, h_offsets, blk_off.data(), n_req);
    StepParams P = make_params(h);
    P.tokens = d_tokens; P.n_req = n_req; P.n_access = (uint32_t)N;
    if (h->profiling) { cudaEventRecord(h->ev[2], s); cudaEventRecord(h->ev[3], s); }   // one kernel: its whole time is booked under the machine
    const unsigned long long* ci = reinterpret_cast<const unsigned long long*>(d_chain_in);
    int64_t* d_boff = h->d_offsets + (h->req_cap + 1);
    const int mach = (N < 48ull * n_req) ? 2 : 3;
    const bool lru = h->policy == ARC_POLICY_LRU, held = h->pin_scope == ARC_PIN_HELD;
#define FUSED_LAUNCH(L, H) arc_fused_small_kernel<L, H><<<1, 2 * WIDE_W, K1_SMEM_BYTES, s>>>(P, ci, h->d_chain_state, h->d_offsets, d_boff, mach, k1_args.small)
    if (lru) { if (held) FUSED_LAUNCH(true, true); else FUSED_LAUNCH(true, false); }
    else { if (held) FUSED_LAUNCH(false, true); else FUSED_LAUNCH(false, false); }
#undef FUSED_LAUNCH
    h->launches += 1;
    if (h->profiling) { cudaEventRecord(h->ev[4], s); cudaEventRecord(h->ev[5], s); h->ev_valid = true; }
    CUDA_TRY(h, cudaGetLastError());
    return finish_step(h, h_offsets, n_req, N, s, P, out);
  }
  const int arg_mode = N ? k1_arg_mode(n_req) : K1_ARG_NONE;   // small enough for a kernel argument: no copy-engine round trip, no staging
  if (arg_mode != K1_ARG_NONE) {
    k1_fill_args(k1_args, arg_mode, h_offsets, blk_off.data(), n_req);   // K1 takes the argument and stores the arrays for K3 / K4
  } else {
    const int slot = h->stage_next;
    h->stage_next = (slot + 1) % kStageSlots;
    CUDA_TRY(h, cudaEventSynchronize(h->stage_done[slot]));
    int64_t* stage = h->h_stage + (size_t)slot * 2 * ((size_t)h->req_cap + 1);
    memcpy(stage, h_offsets, ((size_t)n_req + 1) * sizeof(int64_t));
    memcpy(stage + (h->req_cap + 1), blk_off.data(), ((size_t)n_req + 1) * sizeof(int64_t));
    CUDA_TRY(h, cudaMemcpyAsync(h->d_offsets, stage, ((size_t)n_req + 1) * sizeof(int64_t), cudaMemcpyHostToDevice, s));
    CUDA_TRY(h, cudaMemcpyAsync(h->d_offsets + (h->req_cap + 1), stage + (h->req_cap + 1), ((size_t)n_req + 1) * sizeof(int64_t), cudaMemcpyHostToDevice, s));
    CUDA_TRY(h, cudaEventRecord(h->stage_done[slot], s));
  }

  StepParams P = make_params(h);
  P.tokens = d_tokens; P.n_req = n_req; P.n_access = (uint32_t)N;
  if (N) {
    if (segmented) {
      // K1, few long requests: segments hashed independently, then put together (hash_kernels.cuh)
      if (!h->d_seg_end) CUDA_TRY(h, dalloc(&h->d_seg_end, kSegEndCap));
      launch_hash_segments(arg_mode, k1_args, d_tokens, h->d_offsets, h->d_offsets + (h->req_cap + 1), n_req, max_seg, P.keys_acc, h->d_seg_end,
                           &h->d_state->k1_ticket, s);
      hash_fixup_kernel<<<grid_for((uint64_t)n_req * max_seg, 8, 148 * 4), 256, 0, s>>>(P.blk_off, n_req, max_seg, P.keys_acc, h->d_seg_end,
                                                                    reinterpret_cast<const unsigned long long*>(d_chain_in), h->d_chain_state);
      h->launches += 1;
    } else {
      launch_hash_blocks(true, arg_mode, k1_args, d_tokens, h->d_offsets, h->d_offsets + (h->req_cap + 1), n_req, P.keys_acc,   // K1
                         &h->d_state->k1_ticket, s, reinterpret_cast<const unsigned long long*>(d_chain_in), h->d_chain_state);
    }
    if (h->profiling) cudaEventRecord(h->ev[2], s);
    probe_reserve_kernel<<<grid_for(N, 256 * PROBE_ILP, 148 * 8), 256, 0, s>>>(P);                        // K2
    h->launches += 2;
    if (h->machine != 1 && h->pin_scope != ARC_PIN_REQUEST) {     // windows of the window machines span requests there: natural-order indices
      nat_index_kernel<<<grid_for((uint64_t)n_req * 32, 256, 148 * 4), 256, 0, s>>>(P);
      h->launches += 1;
    }
  } else {
    // no full block anywhere: every request keeps the state it came with
    if (n_req) {
      if (d_chain_in) CUDA_TRY(h, cudaMemcpyAsync(h->d_chain_state, d_chain_in, (size_t)n_req * sizeof(uint64_t), cudaMemcpyDeviceToDevice, s));
      else { fill_u64_kernel<<<grid_for(n_req, 256, 148), 256, 0, s>>>(h->d_chain_state, n_req, H_S0); h->launches += 1; }
    }
    if (h->profiling) cudaEventRecord(h->ev[2], s);
  }
  if (h->profiling) cudaEventRecord(h->ev[3], s);
  if (h->machine == 1) {
    arc_machine_serial_kernel<<<1, 32, 0, s>>>(P);                                                       // K3 (serial)
  } else if (h->machine == 2 || (h->machine == 0 && N < 48ull * n_req)) {
    // one warp, 32-wide windows: a window of the wide machine costs about twice as much, which only pays when requests
    // are long enough to fill it (windows never cross a request boundary)
    launch_machine_batched(P, s);
  } else if (h->machine == 5) {
    launch_machine_wide<false>(P, s);                                                                    // K3 (8 warps, 128-wide windows; every owner warp rolls)
  } else {
    launch_machine_wide<true>(P, s);                                                                     // K3 (the same with the roller warp a window ahead)
  }
  if (h->profiling) cudaEventRecord(h->ev[4], s);
  finalize_kernel<<<grid_for(std::max<uint64_t>(N, (uint64_t)n_req * 32), 256, 148 * 8), 256, 0, s>>>(P);  // K4
  h->launches += 2;
  if (h->profiling) { cudaEventRecord(h->ev[5], s); h->ev_valid = true; }
  CUDA_TRY(h, cudaGetLastError());

  return finish_step(h, h_offsets, n_req, N, s, P, out);
}

int arc_step_host_async(arc_cache* h, const int32_t* h_tokens, const int64_t* h_offsets, uint32_t n_req, void* cuda_stream, uint32_t* ticket_out) {
  if (!h) return ARC_ERR_INVALID_ARG;
  if (!h_offsets || !ticket_out) return fail(h, ARC_ERR_INVALID_ARG, "NULL argument");
  if (n_req > kMaxReq) return fail(h, ARC_ERR_INVALID_ARG, "n_req > 2^20");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  uint64_t N = 0;
  int rc = validate_offsets(h, h_offsets, n_req, h->B, h->c, nullptr, &N);
  if (rc) return rc;
  const int64_t first = h_offsets[0], total = h_offsets[n_req] - first;
  if (!h_tokens && total > 0) return fail(h, ARC_ERR_INVALID_ARG, "h_tokens is NULL");
  const int k = (int)(h->next_ticket % kHostSlots);
  if (h->slot_ticket[k]) return fail(h, ARC_ERR_INVALID_ARG, "%d steps are in flight: arc_step_host_wait(ticket %u) first", kHostSlots, h->slot_ticket[k]);
  // growth (rare) drops the mapped result buffers of the steps in flight: only with none in flight
  if (n_req > h->req_cap || N > h->n_cap) {
    for (int q = 0; q < kHostSlots; ++q)
      if (h->slot_ticket[q]) return fail(h, ARC_ERR_INVALID_ARG, "this step needs larger buffers: wait for the steps in flight first (or arc_reserve)");
    rc = ensure_capacity(h, n_req, N, s);
    if (rc) return rc;
  }
  if (!h->copy_stream) CUDA_TRY(h, cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
  if (!h->ev_h2d[k]) {
    CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_h2d[k], cudaEventDisableTiming));
    CUDA_TRY(h, cudaEventCreateWithFlags(&h->ev_comp[k], cudaEventDisableTiming));
  }
  if ((uint64_t)total > h->tok_cap[k]) {
    CUDA_TRY(h, cudaEventSynchronize(h->ev_comp[k]));           // the step that read this slot's tokens last has finished
    dfree(h->d_tok[k]);
    h->tok_cap[k] = std::max<uint64_t>((uint64_t)total, h->tok_cap[k] * 2);
    CUDA_TRY(h, dalloc(&h->d_tok[k], h->tok_cap[k]));
  }
  // tokens: on the handle's copy stream, as soon as the slot's previous step is through with them - while the steps
  // before this one are still computing on the caller's stream
  CUDA_TRY(h, cudaStreamWaitEvent(h->copy_stream, h->ev_comp[k], 0));
  if (total) CUDA_TRY(h, cudaMemcpyAsync(h->d_tok[k], h_tokens + first, (size_t)total * sizeof(int32_t), cudaMemcpyHostToDevice, h->copy_stream));
  CUDA_TRY(h, cudaEventRecord(h->ev_h2d[k], h->copy_stream));
  CUDA_TRY(h, cudaStreamWaitEvent(s, h->ev_h2d[k], 0));
  static thread_local std::vector<int64_t> rel;             // offsets relative to the staged copy
  rel.resize((size_t)n_req + 1);
  for (uint32_t r = 0; r <= n_req; ++r) rel[r] = h_offsets[r] - first;
  arc_step_result res;
  rc = arc_step(h, h->d_tok[k], rel.data(), n_req, cuda_stream, &res);
  if (rc) return rc;
  // results: packed by a kernel straight into pinned host memory (exactly the words that exist, no copy to size)
  int32_t* d_view = nullptr;
  CUDA_TRY(h, cudaHostGetDevicePointer((void**)&d_view, h->h_out[k], 0));
  pack_results_kernel<<<grid_for(N + n_req, 1024, 32), 256, 0, s>>>(h->d_state, h->d_prefix_len, h->d_alloc_ids, h->d_evict_ids, n_req, d_view);
  h->launches += 1;
  CUDA_TRY(h, cudaGetLastError());
  CUDA_TRY(h, cudaEventRecord(h->ev_comp[k], s));
  h->slot_ticket[k] = h->next_ticket; h->slot_n_req[k] = n_req; h->slot_n_access[k] = N;
  h->slot_h2d[k] = (uint64_t)total * sizeof(int32_t) + 2 * ((uint64_t)n_req + 1) * sizeof(int64_t);
  *ticket_out = h->next_ticket;
  h->next_ticket += 1;
  if (h->next_ticket == 0) h->next_ticket = 1;
  return ARC_OK;
}

int arc_step_host_wait(arc_cache* h, uint32_t ticket, arc_host_result* out) {
  if (!h) return ARC_ERR_INVALID_ARG;
  if (!out || !ticket) return fail(h, ARC_ERR_INVALID_ARG, "NULL argument");
  const int k = (int)(ticket % kHostSlots);
  if (h->slot_ticket[k] != ticket) return fail(h, ARC_ERR_INVALID_ARG, "ticket %u is not in flight", ticket);
  CUDA_TRY(h, cudaEventSynchronize(h->ev_comp[k]));
  const int32_t* hp = h->h_out[k];
  const uint32_t n_req = h->slot_n_req[k];
  out->n_access = h->slot_n_access[k];
  out->n_alloc = (uint32_t)hp[0]; out->n_evict = (uint32_t)hp[1];
  out->prefix_len = hp + 3; out->alloc_ids = hp + 3 + n_req; out->evict_ids = hp + 3 + n_req + out->n_alloc;
  out->h2d_bytes = h->slot_h2d[k];
  out->d2h_bytes = (3ull + n_req + out->n_alloc + out->n_evict) * sizeof(int32_t);
  h->slot_ticket[k] = 0;
  if (hp[2]) return fail(h, ARC_ERR_CUDA, "device-side directory error %u (1 node pool, 2 no victim, 3 ring overflow, 4 bad node, 5 bad release)", (unsigned)hp[2]);
  return ARC_OK;
}

int arc_step_host(arc_cache* h, const int32_t* h_tokens, const int64_t* h_offsets, uint32_t n_req, void* cuda_stream, arc_host_result* out) {
  if (!h) return ARC_ERR_INVALID_ARG;
  if (!out) return fail(h, ARC_ERR_INVALID_ARG, "NULL argument");
  uint32_t ticket = 0;
  int rc = arc_step_host_async(h, h_tokens, h_offsets, n_req, cuda_stream, &ticket);
  if (rc) return rc;
  return arc_step_host_wait(h, ticket, out);
}

int arc_stats(arc_cache* h, arc_stats_t* out) {
  if (!h) return ARC_ERR_INVALID_ARG;
  if (!out) return fail(h, ARC_ERR_INVALID_ARG, "out is NULL");
  CUDA_TRY(h, cudaStreamSynchronize(h->last_stream));
  DevState st;
  CUDA_TRY(h, cudaMemcpy(&st, h->d_state, sizeof(st), cudaMemcpyDeviceToHost));
  memset(out, 0, sizeof(*out));
  out->steps = h->steps; out->requests = h->requests; out->tokens_seen = h->tokens_seen; out->tokens_hashed = h->tokens_hashed;
  out->accesses = st.stat[ST_ACCESSES];
  out->hit_t1 = st.stat[ST_HIT_T1]; out->hit_t2 = st.stat[ST_HIT_T2]; out->ghost_b1 = st.stat[ST_GHOST_B1];
  out->ghost_b2 = st.stat[ST_GHOST_B2]; out->miss = st.stat[ST_MISS]; out->evict_t1 = st.stat[ST_EVICT_T1];
  out->evict_t2 = st.stat[ST_EVICT_T2]; out->drop_b1 = st.stat[ST_DROP_B1]; out->drop_b2 = st.stat[ST_DROP_B2];
  out->fresh_ids_used = st.stat[ST_FRESH]; out->prefix_hit_tokens = st.stat[ST_PREFIX_TOKENS];
  out->t1 = (uint64_t)st.t1; out->t2 = (uint64_t)st.t2; out->b1 = (uint64_t)st.b1; out->b2 = (uint64_t)st.b2; out->p = (uint64_t)st.p;
  out->capacity_blocks = h->c; out->block_size = h->B; out->policy = h->policy;
  // we are synchronised: tighten the host-side bounds with the true values
  h->slots_used_bound = (uint64_t)st.t1 + st.t2 + st.b1 + st.b2 + st.tombs;
  for (int L = 1; L <= 4; ++L) h->window_bound[L] = (uint32_t)(st.tail[L] - st.head[L]);
  if (st.error) return fail(h, ARC_ERR_CUDA, "device-side directory error %u (1 node pool, 2 no victim, 3 ring overflow, 4 bad node, 5 bad release)", st.error);
  return ARC_OK;
}

int arc_reset(arc_cache* h) {
  if (!h) return ARC_ERR_INVALID_ARG;
  cudaStream_t s = h->last_stream;
  CUDA_TRY(h, cudaMemsetAsync(h->d_table, 0, (size_t)h->table_slots * sizeof(Slot), s));
  init_state_kernel<<<grid_for(h->node_cap, 256, 148 * 8), 256, 0, s>>>(h->d_state, h->d_nodes, h->d_free_stack, h->node_cap, (h->policy == ARC_POLICY_DBL) ? (int32_t)(h->c / 2) : 0);
  CUDA_TRY(h, cudaGetLastError());
  CUDA_TRY(h, cudaStreamSynchronize(s));
  h->slots_used_bound = 0;
  for (int L = 1; L <= 4; ++L) h->window_bound[L] = 0;
  if (h->d_node_of_block) CUDA_TRY(h, cudaMemset(h->d_node_of_block, 0xFF, (size_t)h->c * sizeof(uint32_t)));
  CUDA_TRY(h, cudaMemset(h->d_node_stamp, 0, (size_t)h->node_cap * sizeof(uint32_t)));
  h->hold_units = 0;
  for (int k = 0; k < kHostSlots; ++k) h->slot_ticket[k] = 0;
  h->steps = h->requests = h->tokens_seen = h->tokens_hashed = 0;
  h->launches = 0;
  h->ev_valid = false;
  return ARC_OK;
}

void arc_destroy(arc_cache* h) {
  if (!h) return;
  cudaDeviceSynchronize();
  { StepBuffers b = take_step_buffers(h); free_step_buffers(b); }
  dfree(h->d_state); dfree(h->d_nodes); dfree(h->d_node_key); dfree(h->d_free_stack); dfree(h->d_table); dfree(h->d_node_stamp);
  for (int L = 1; L <= 4; ++L) { dfree(h->d_ring[L]); dfree(h->d_ring_alt[L]); }
  dfree(h->d_block_counts); for (int k = 0; k < kHostSlots; ++k) { dfree(h->d_tok[k]); if (h->ev_h2d[k]) cudaEventDestroy(h->ev_h2d[k]); if (h->ev_comp[k]) cudaEventDestroy(h->ev_comp[k]); }
  if (h->copy_stream) cudaStreamDestroy(h->copy_stream); dfree(h->d_machine_scratch);
  dfree(h->d_node_of_block); dfree(h->d_rel_cnt); dfree(h->d_seg_end);
  for (int i = 0; i < kStageSlots; ++i) if (h->stage_done[i]) cudaEventDestroy(h->stage_done[i]);
  for (int i = 0; i < 7; ++i) if (h->ev[i]) cudaEventDestroy(h->ev[i]);
  delete h;
}

const char* arc_last_error(const arc_cache* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

// Scratch of the stateless hashing entry: a small ring of slots, each with a pinned host buffer, a device buffer
// (ticket words, offsets, block offsets) and two events.  A call takes the next slot, fills it, copies it on the library's
// own copy stream (so the copy overlaps whatever the caller's stream is still doing) and makes the caller's stream wait
// for that copy; the slot is reused only after the kernel that read it has finished.  Calls on different streams or
// threads therefore never share scratch, and a call moves 16 + 16 (n_req + 1) bytes, not a fixed capacity.
namespace {
struct HashSlot {
  int64_t* h_buf = nullptr; int64_t* d_buf = nullptr; size_t cap = 0;     // cap in int64 entries
  cudaEvent_t copied = nullptr, done = nullptr;
};
struct HashScratch {
  std::mutex mu;
  HashSlot slot[8];
  int next = 0;
  cudaStream_t copy_stream = nullptr;
  int device = -1;
};
HashScratch g_hash;
}  // namespace

int arc_hash_blocks(const int32_t* d_tokens, const int64_t* h_offsets, uint32_t n_req, uint32_t block_size, uint64_t* d_keys_out, void* cuda_stream) {
  if (!h_offsets) return fail(nullptr, ARC_ERR_INVALID_ARG, "h_offsets is NULL");
  if (n_req > kMaxReq) return fail(nullptr, ARC_ERR_INVALID_ARG, "n_req > 2^20");
  if (block_size != 16) return fail(nullptr, ARC_ERR_UNSUPPORTED, "block_size %u: only 16 is built", block_size);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  cudaError_t e = k1_configure();
  if (e != cudaSuccess) return fail(nullptr, ARC_ERR_CUDA, "K1 configuration: %s", cudaGetErrorString(e));
  int dev = 0;
  cudaGetDevice(&dev);
  std::lock_guard<std::mutex> lock(g_hash.mu);
  if (g_hash.device != dev) {                      // first use, or the caller moved to another device: start again there
    if (g_hash.device >= 0) cudaDeviceSynchronize();
    for (HashSlot& k : g_hash.slot) {
      if (k.h_buf) cudaFreeHost(k.h_buf);
      if (k.d_buf) cudaFree(k.d_buf);
      if (k.copied) cudaEventDestroy(k.copied);
      if (k.done) cudaEventDestroy(k.done);
      k = HashSlot();
    }
    if (g_hash.copy_stream) cudaStreamDestroy(g_hash.copy_stream);
    g_hash.copy_stream = nullptr;
    if (cudaStreamCreateWithFlags(&g_hash.copy_stream, cudaStreamNonBlocking) != cudaSuccess) return fail(nullptr, ARC_ERR_CUDA, "copy stream");
    g_hash.device = dev;
  }
  HashSlot& k = g_hash.slot[g_hash.next];
  g_hash.next = (g_hash.next + 1) % 8;
  if (!k.copied) { cudaEventCreateWithFlags(&k.copied, cudaEventDisableTiming); cudaEventCreateWithFlags(&k.done, cudaEventDisableTiming); }
  // host staging: 16 bytes of ticket words, then one region of n_req items per length class (the classes' sizes are only
  // known after the pass); device: the ticket words, then the items, classes back to back.  Sizes in int64 entries.
  const size_t need = 2 + 4 * (size_t)K1_PASSES * n_req;
  cudaEventSynchronize(k.done);                                     // the kernel that read this slot last has finished
  if (need > k.cap) {
    if (k.h_buf) cudaFreeHost(k.h_buf);
    if (k.d_buf) cudaFree(k.d_buf);
    k.cap = std::max<size_t>(need, 4096);
    if (cudaMallocHost((void**)&k.h_buf, k.cap * sizeof(int64_t)) != cudaSuccess || cudaMalloc((void**)&k.d_buf, k.cap * sizeof(int64_t)) != cudaSuccess) {
      if (k.h_buf) cudaFreeHost(k.h_buf);
      k.h_buf = nullptr; k.d_buf = nullptr; k.cap = 0;
      cudaGetLastError();
      return fail(nullptr, ARC_ERR_OOM, "scratch allocation failed");
    }
  }
  // ONE pass over the offsets: validation, blocks per request (block_size is 16: a shift), and the work list - one
  // 32-byte item per request with a full block, written to the region of its length class (longest class first on the
  // device: the order the ticket passes of the in-step kernel produce, without the tickets that find nothing)
  if (h_offsets[0] < 0) return fail(nullptr, ARC_ERR_INVALID_ARG, "h_offsets[0] < 0");
  HashItem* region[K1_PASSES];
  for (int c = 0; c < K1_PASSES; ++c) region[c] = reinterpret_cast<HashItem*>(k.h_buf + 2) + (size_t)c * n_req;
  uint32_t cnt[K1_PASSES] = {};
  uint64_t N = 0;
  for (uint32_t r = 0; r < n_req; ++r) {
    const int64_t len = h_offsets[r + 1] - h_offsets[r];
    if (len < 0) return fail(nullptr, ARC_ERR_INVALID_ARG, "h_offsets not monotone at request %u", r);
    const uint64_t nb = (uint64_t)len >> 4;
    if (nb >= (1ull << 28)) return fail(nullptr, ARC_ERR_INVALID_ARG, "request %u is too large", r);
    const uint32_t c = (uint32_t)(nb < 1024) + (uint32_t)(nb < 384) + (uint32_t)(nb < 128);      // = k1_class
    HashItem& it = region[c][cnt[c]];
    it.tok_off = h_offsets[r]; it.key_off = (long long)N; it.n_blocks = (uint32_t)nb; it.reserved[0] = it.reserved[1] = it.reserved[2] = 0;
    cnt[c] += nb != 0;                                               // a request without a full block leaves no item
    N += nb;
  }
  if (N >= (1ull << 31)) return fail(nullptr, ARC_ERR_INVALID_ARG, "%llu blocks in one call is too large", (unsigned long long)N);
  if (!N) return ARC_OK;
  if (!d_tokens || !d_keys_out) return fail(nullptr, ARC_ERR_INVALID_ARG, "NULL device pointer");
  k.h_buf[0] = 0; k.h_buf[1] = 0;                                   // the ticket words travel with the items
  e = cudaMemcpyAsync(k.d_buf, k.h_buf, 2 * sizeof(int64_t), cudaMemcpyHostToDevice, g_hash.copy_stream);
  uint32_t n_items = 0;
  for (int c = 0; c < K1_PASSES && e == cudaSuccess; ++c) {
    if (cnt[c]) e = cudaMemcpyAsync(reinterpret_cast<HashItem*>(k.d_buf + 2) + n_items, region[c], (size_t)cnt[c] * sizeof(HashItem), cudaMemcpyHostToDevice, g_hash.copy_stream);
    n_items += cnt[c];
  }
  if (e == cudaSuccess) e = cudaEventRecord(k.copied, g_hash.copy_stream);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(s, k.copied, 0);
  if (e != cudaSuccess) return fail(nullptr, ARC_ERR_CUDA, "work list copy: %s", cudaGetErrorString(e));
  hash_items_kernel<<<grid_for(n_items, K1_WARPS, 148 * 3), 256, K1_SMEM_BYTES, s>>>(d_tokens, reinterpret_cast<const HashItem*>(k.d_buf + 2), n_items,
                                                                                  h_offsets[0], h_offsets[n_req], (unsigned long long*)d_keys_out,
                                                                                  reinterpret_cast<uint32_t*>(k.d_buf));
  g_hash_launches += 1;
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaEventRecord(k.done, s);
  if (e != cudaSuccess) return fail(nullptr, ARC_ERR_CUDA, "hash launch: %s", cudaGetErrorString(e));
  return ARC_OK;
}

int arc_route_requests(const int32_t* d_tokens, const int64_t* d_offsets, uint32_t n_req, uint32_t block_size, uint32_t world, int32_t* d_dst_out,
                       void* cuda_stream) {
  if (n_req > kMaxReq || world == 0) return fail(nullptr, ARC_ERR_INVALID_ARG, "n_req > 2^20 or world = 0");
  if (block_size != 16) return fail(nullptr, ARC_ERR_UNSUPPORTED, "block_size %u: only 16 is built", block_size);
  if (!n_req) return ARC_OK;
  if (!d_offsets || !d_dst_out) return fail(nullptr, ARC_ERR_INVALID_ARG, "NULL device pointer");
  route_first_block_kernel<<<grid_for(n_req, 256, 148 * 4), 256, 0, (cudaStream_t)cuda_stream>>>(d_tokens, d_offsets, n_req, world, d_dst_out);
  g_hash_launches += 1;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(nullptr, ARC_ERR_CUDA, "route launch: %s", cudaGetErrorString(e));
  return ARC_OK;
}

int arc_hash_blocks_device(const int32_t* d_tokens, const arc_hash_item* d_items, uint32_t n_items, int64_t tok_lo, int64_t tok_hi, uint32_t block_size,
                           uint64_t* d_keys_out, uint32_t* d_ticket, void* cuda_stream) {
  if (n_items > kMaxReq) return fail(nullptr, ARC_ERR_INVALID_ARG, "n_items > 2^20");
  if (block_size != 16) return fail(nullptr, ARC_ERR_UNSUPPORTED, "block_size %u: only 16 is built", block_size);
  if (!n_items) return ARC_OK;
  if (!d_tokens || !d_items || !d_keys_out || !d_ticket) return fail(nullptr, ARC_ERR_INVALID_ARG, "NULL device pointer");
  static_assert(sizeof(arc_hash_item) == sizeof(HashItem), "arc_hash_item is the kernel's HashItem");
  cudaError_t e = k1_configure();
  if (e != cudaSuccess) return fail(nullptr, ARC_ERR_CUDA, "K1 configuration: %s", cudaGetErrorString(e));
  hash_items_kernel<<<grid_for(n_items, K1_WARPS, 148 * 3), 256, K1_SMEM_BYTES, (cudaStream_t)cuda_stream>>>(
      d_tokens, reinterpret_cast<const HashItem*>(d_items), n_items, tok_lo, tok_hi, (unsigned long long*)d_keys_out, d_ticket);
  g_hash_launches += 1;
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(nullptr, ARC_ERR_CUDA, "hash launch: %s", cudaGetErrorString(e));
  return ARC_OK;
}

// ---- K1 without any allocation (arc_hash_blocks_static) -----------------------------------------------------------
// The scratch of the segmented hashing lives in the library image: one file-scope __device__ array per GPU that loads the
// library, held until the process exits.  In host code the array's NAME is only a stand-in for the symbol: the device
// address comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) unsigned char g_k1_static_scratch[sizeof(K1StaticScratch)];

namespace {
struct K1StaticSetup { std::mutex mu; K1StaticScratch* ptr[64] = {}; };
K1StaticSetup g_k1_static;

// the scratch's device address on the CURRENT device (set-up on first use: no allocation, two attribute / symbol queries)
cudaError_t k1_static_scratch(K1StaticScratch** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_k1_static.mu);
  if (!g_k1_static.ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_k1_static_scratch);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(hash_segments_static_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, K1_SMEM_BYTES);
    if (e != cudaSuccess) return e;
    g_k1_static.ptr[dev] = static_cast<K1StaticScratch*>(p);
  }
  *out = g_k1_static.ptr[dev];
  return cudaSuccess;
}
}  // namespace

int arc_hash_blocks_static(const int32_t* d_tokens, const int64_t* h_offsets, uint32_t n_req, uint32_t block_size, uint64_t* d_keys_out,
                           void* cuda_stream) {
  if (!h_offsets) return fail(nullptr, ARC_ERR_INVALID_ARG, "NULL argument");
  if (block_size != 16) return fail(nullptr, ARC_ERR_UNSUPPORTED, "block_size %u: only 16 is built", block_size);
  if (n_req > K1_STATIC_MAX_REQ)
    return fail(nullptr, ARC_ERR_REQUEST_TOO_LARGE, "arc_hash_blocks_static takes at most %u requests per call (got %u)", K1_STATIC_MAX_REQ, n_req);
  if (h_offsets[0] < 0) return fail(nullptr, ARC_ERR_INVALID_ARG, "h_offsets[0] < 0");
  static thread_local OffsetsArgT<K1_STATIC_MAX_REQ> arg;           // offsets[n_req + 1] then blk_off[n_req + 1]
  uint64_t N = 0, max_nb = 0;
  arg.v[n_req + 1] = 0;
  for (uint32_t r = 0; r < n_req; ++r) {
    const int64_t len = h_offsets[r + 1] - h_offsets[r];
    if (len < 0) return fail(nullptr, ARC_ERR_INVALID_ARG, "h_offsets not monotone at request %u", r);
    const uint64_t nb = (uint64_t)len >> 4;
    max_nb = std::max(max_nb, nb);
    N += nb;
    arg.v[n_req + 1 + r + 1] = (long long)N;
  }
  const uint64_t max_seg = (max_nb + K1_SEG - 1) / K1_SEG;
  if (max_seg > K1_STATIC_MAX_SEG_PER_REQ || (uint64_t)n_req * max_seg > K1_STATIC_MAX_SEGS)
    return fail(nullptr, ARC_ERR_REQUEST_TOO_LARGE,
                "arc_hash_blocks_static: %u requests x %llu segments of %d blocks (the longest request has %llu blocks) exceed the fixed scratch of %u segments",
                n_req, (unsigned long long)max_seg, K1_SEG, (unsigned long long)max_nb, K1_STATIC_MAX_SEGS);
  if (!N) return ARC_OK;
  if (!d_tokens || !d_keys_out) return fail(nullptr, ARC_ERR_INVALID_ARG, "NULL device pointer");
  memcpy(arg.v, h_offsets, ((size_t)n_req + 1) * sizeof(int64_t));
  K1StaticScratch* sc = nullptr;
  cudaError_t e = k1_static_scratch(&sc);
  if (e != cudaSuccess) return fail(nullptr, ARC_ERR_CUDA, "static scratch set-up: %s", cudaGetErrorString(e));
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const uint32_t total = n_req * (uint32_t)max_seg;
  hash_segments_static_kernel<<<grid_for(total, K1_WARPS, 148 * 3), 256, K1_SMEM_BYTES, s>>>(d_tokens, n_req, (uint32_t)max_seg,
                                                                                            (unsigned long long*)d_keys_out, sc, arg);
  hash_fixup_static_kernel<<<grid_for(total, 8, 148 * 4), 256, 0, s>>>(n_req, (uint32_t)max_seg, (unsigned long long*)d_keys_out, sc);
  g_hash_launches += 2;
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(nullptr, ARC_ERR_CUDA, "hash launch: %s", cudaGetErrorString(e));
  return ARC_OK;
}

int arc_set_profiling(arc_cache* h, int enabled) {
  if (!h) return ARC_ERR_INVALID_ARG;
  h->profiling = enabled != 0;
  h->ev_valid = false;
  return ARC_OK;
}

int arc_last_kernel_times(arc_cache* h, arc_kernel_times* out) {
  if (!h || !out) return ARC_ERR_INVALID_ARG;
  if (!h->ev_valid) return fail(h, ARC_ERR_INVALID_ARG, "no profiled step");
  CUDA_TRY(h, cudaEventSynchronize(h->ev[5]));
  cudaEventElapsedTime(&out->maint_ms, h->ev[0], h->ev[1]);
  cudaEventElapsedTime(&out->hash_ms, h->ev[1], h->ev[2]);
  cudaEventElapsedTime(&out->probe_ms, h->ev[2], h->ev[3]);
  cudaEventElapsedTime(&out->machine_ms, h->ev[3], h->ev[4]);
  cudaEventElapsedTime(&out->finalize_ms, h->ev[4], h->ev[5]);
  cudaEventElapsedTime(&out->total_ms, h->ev[0], h->ev[5]);
  return ARC_OK;
}

uint64_t arc_launch_count(const arc_cache* h) { return h ? h->launches : g_hash_launches.load(); }

int arc_set_machine(arc_cache* h, int which) {
  if (!h || which < 0 || which > 5) return ARC_ERR_INVALID_ARG;
  h->machine = which;
  return ARC_OK;
}

int arc_set_pin_scope(arc_cache* h, int scope) {
  if (!h) return ARC_ERR_INVALID_ARG;
  if (scope != ARC_PIN_REQUEST && scope != ARC_PIN_STEP && scope != ARC_PIN_HELD) return fail(h, ARC_ERR_INVALID_ARG, "unknown pin scope %d", scope);
  if (h->hold_units) return fail(h, ARC_ERR_INVALID_ARG, "%llu holds outstanding: release them before changing the pin scope", (unsigned long long)h->hold_units);
  if (scope == ARC_PIN_HELD && h->pin_scope != ARC_PIN_HELD) {
    if (!h->d_node_of_block) {
      CUDA_TRY(h, dalloc(&h->d_node_of_block, h->c));
      CUDA_TRY(h, dalloc(&h->d_rel_cnt, 2 * h->c));          // multiplicities, then last-occurrence indices
      CUDA_TRY(h, cudaMemset(h->d_node_of_block, 0xFF, (size_t)h->c * sizeof(uint32_t)));
      CUDA_TRY(h, cudaMemset(h->d_rel_cnt, 0, 2 * (size_t)h->c * sizeof(uint32_t)));
    }
    set_unheld_kernel<<<1, 1, 0, h->last_stream>>>(h->d_state);      // nothing is held: every resident entry is in a ring
    h->launches += 1;
    CUDA_TRY(h, cudaGetLastError());
  }
  h->pin_scope = scope;
  return ARC_OK;
}

int arc_release(arc_cache* h, const int32_t* d_block_ids, uint64_t n, void* cuda_stream) {
  if (!h) return ARC_ERR_INVALID_ARG;
  if (h->pin_scope != ARC_PIN_HELD) return fail(h, ARC_ERR_INVALID_ARG, "arc_release needs pin scope ARC_PIN_HELD");
  if (n && !d_block_ids) return fail(h, ARC_ERR_INVALID_ARG, "d_block_ids is NULL");
  if (n > h->hold_units) return fail(h, ARC_ERR_INVALID_ARG, "%llu ids released but only %llu holds are outstanding", (unsigned long long)n, (unsigned long long)h->hold_units);
  if (!n) return ARC_OK;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  int rc = maintain(h, n, s);            // room for up to n pushes at the MRU ends of T1 / T2
  if (rc) return rc;
  StepParams P = make_params(h);
  release_kernel<<<1, REL_THREADS, 0, s>>>(P, d_block_ids, (uint32_t)n, h->d_rel_cnt, h->d_rel_cnt + h->c);
  h->launches += 1;
  CUDA_TRY(h, cudaGetLastError());
  h->window_bound[L_T1] += n; h->window_bound[L_T2] += n;
  h->hold_units -= n;
  h->last_stream = s;
  return ARC_OK;
}

uint64_t arc_hold_units(const arc_cache* h) { return h ? h->hold_units : 0; }

int arc_debug_probe(arc_cache* h, const uint64_t* d_keys, uint64_t n, uint32_t* d_nodes_out, void* cuda_stream) {
  if (!h) return ARC_ERR_INVALID_ARG;
  if (n && (!d_keys || !d_nodes_out)) return fail(h, ARC_ERR_INVALID_ARG, "NULL device pointer");
  if (n >= (1ull << 31)) return fail(h, ARC_ERR_INVALID_ARG, "too many keys");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  int rc = ensure_capacity(h, 1, n, s);
  if (rc) return rc;
  // this entry creates no tombstones and every used slot belongs to a node: the pool size bounds the load (0.375 of the table)
  h->slots_used_bound = std::min<uint64_t>(h->slots_used_bound, h->node_cap);
  rc = maintain(h, std::min<uint64_t>(n, h->node_cap - h->slots_used_bound), s);
  if (rc) return rc;
  StepParams P = make_params(h);
  P.keys_acc = const_cast<unsigned long long*>(reinterpret_cast<const unsigned long long*>(d_keys));
  P.node_acc = d_nodes_out;
  P.n_access = (uint32_t)n; P.n_req = 0;
  if (n) {
    probe_reserve_kernel<<<grid_for(n, 256 * PROBE_ILP, 148 * 8), 256, 0, s>>>(P);
    h->launches += 1;
  }
  CUDA_TRY(h, cudaGetLastError());
  // every used slot belongs to a node and this entry creates no tombstones
  h->slots_used_bound = std::min<uint64_t>(h->slots_used_bound + n, h->node_cap);
  h->last_stream = s;
  return ARC_OK;
}

int arc_debug_gather_sectors(const uint64_t* d_keys, uint64_t n, const void* d_buf, uint64_t n_sectors, uint32_t* d_out, void* cuda_stream) {
  if (n && (!d_keys || !d_buf || !d_out)) return fail(nullptr, ARC_ERR_INVALID_ARG, "NULL device pointer");
  if (n >= (1ull << 31) || n_sectors == 0 || (n_sectors & (n_sectors - 1)) || n_sectors > (1ull << 32)) return fail(nullptr, ARC_ERR_INVALID_ARG, "n or n_sectors out of range");
  if (reinterpret_cast<uintptr_t>(d_buf) & 31) return fail(nullptr, ARC_ERR_INVALID_ARG, "d_buf must be 32-byte aligned");
  if (n) {
    gather32_kernel<<<grid_for(n, 256 * PROBE_ILP, 148 * 8), 256, 0, (cudaStream_t)cuda_stream>>>(
        reinterpret_cast<const unsigned long long*>(d_keys), (uint32_t)n, reinterpret_cast<const Slot*>(d_buf), (uint32_t)(n_sectors - 1), d_out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(nullptr, ARC_ERR_CUDA, "gather launch: %s", cudaGetErrorString(e));
  }
  return ARC_OK;
}

int arc_debug_set_key_mask(arc_cache* h, uint64_t mask) {
  if (!h) return ARC_ERR_INVALID_ARG;
  h->key_and = mask;
  return ARC_OK;
}

int arc_debug_counters(arc_cache* h, uint64_t* out, uint32_t n) {
  if (!h || !out) return ARC_ERR_INVALID_ARG;
  CUDA_TRY(h, cudaStreamSynchronize(h->last_stream));
  DevState st;
  CUDA_TRY(h, cudaMemcpy(&st, h->d_state, sizeof(st), cudaMemcpyDeviceToHost));
  for (uint32_t i = 0; i < n; ++i) out[i] = (i < (uint32_t)DBG_COUNT) ? st.dbg[i] : 0;
  return ARC_OK;
}

int arc_debug_latency_hist(arc_cache* h, uint32_t* out) {
  if (!h || !out) return ARC_ERR_INVALID_ARG;
  CUDA_TRY(h, cudaStreamSynchronize(h->last_stream));
  CUDA_TRY(h, cudaMemcpy(out, reinterpret_cast<const char*>(h->d_state) + offsetof(DevState, lat_hist), sizeof(uint32_t) * 5 * 16, cudaMemcpyDeviceToHost));
  return ARC_OK;
}

int arc_debug_list(arc_cache* h, int which, uint64_t* keys_out, int32_t* block_ids_out, uint64_t cap, uint64_t* n_out) {
  if (!h || which < 1 || which > 4 || !n_out) return ARC_ERR_INVALID_ARG;
  cudaStream_t s = h->last_stream;
  unsigned long long* d_keys = nullptr; int32_t* d_blocks = nullptr; unsigned long long* d_n = nullptr;
  CUDA_TRY(h, dalloc(&d_keys, cap));
  CUDA_TRY(h, dalloc(&d_blocks, cap));
  CUDA_TRY(h, dalloc(&d_n, 1));
  dump_list_kernel<<<1, CMP_THREADS, 0, s>>>(h->d_state, h->d_nodes, h->d_node_key, h->d_ring[which], h->ring_cap - 1, (uint32_t)which,
                                             d_keys, d_blocks, cap, d_n);
  CUDA_TRY(h, cudaStreamSynchronize(s));
  unsigned long long n = 0;
  CUDA_TRY(h, cudaMemcpy(&n, d_n, sizeof(n), cudaMemcpyDeviceToHost));
  const uint64_t m = std::min<uint64_t>(n, cap);
  if (keys_out && m) CUDA_TRY(h, cudaMemcpy(keys_out, d_keys, m * sizeof(uint64_t), cudaMemcpyDeviceToHost));
  if (block_ids_out && m) CUDA_TRY(h, cudaMemcpy(block_ids_out, d_blocks, m * sizeof(int32_t), cudaMemcpyDeviceToHost));
  cudaFree(d_keys); cudaFree(d_blocks); cudaFree(d_n);
  *n_out = n;
  return ARC_OK;
}

}  // extern "C"
