/* arc.h — C ABI of the B200-native prefix-KV-cache lookup + ARC block-replacement library.
 *
 * The method (PAPER.md = "Recency/Frequency Adaptive KV Caching for Large Language Model Serving",
 * arxiv/paper_2606_21238): the KV cache is cut into fixed-size KV blocks (e.g. 16 tokens);
 * prefixes shared between requests are reused at block level; the evictor keeps the
 * Adaptive Replacement Cache lists T1/T2 (blocks in memory) and B1/B2 (metadata of evicted blocks,
 * PAPER.md:47-48, :56-60), adapts the T1 target size p on ghost hits and is compared
 * with vLLM's LRU eviction.  The exact rules (hash H1-H6, semantics R1-R12) are in
 * DESIGN.md §3; they are restated from SURVEY.md §8(c).
 *
 * Everything behind this header runs in hand-written CUDA kernels for sm_100a; there is no CPU
 * fallback.  Signatures use plain pointers and sizes only.  Every pointer argument says HOST or DEVICE.
 *
 * Conventions
 *  - Every function returns ARC_OK (0) or a negative ARC_ERR_* code; nothing throws across the ABI.
 *  - Validation happens before any work is enqueued and leaves the handle unchanged.
 *  - A handle is not thread-safe; distinct handles are independent.  A handle is bound to the CUDA
 *    device that was current when it was created.
 *  - arc_step is asynchronous with respect to the host and ordered on `cuda_stream` (a cudaStream_t
 *    passed as void*, NULL = the legacy default stream).  All steps of one handle must be enqueued on
 *    streams that are ordered with respect to each other (normally: always the same stream).
 */
#ifndef ARC_B200_H
#define ARC_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct arc_cache arc_cache; /* opaque, owned by the library */

enum { ARC_POLICY_ARC = 0, ARC_POLICY_LRU = 1,
       ARC_POLICY_DBL = 2 /* ARC's lists and REPLACE with p frozen at capacity_blocks / 2: the paper's DBL ablation */ };
enum {
  ARC_OK = 0,
  ARC_ERR_INVALID_ARG = -1,       /* NULL pointer, capacity 0 or > 2^31-2, n_req > 2^20, offsets not monotone, bad policy */
  ARC_ERR_UNSUPPORTED = -2,       /* block_size other than 16; capacity beyond what the node index width allows (2^28) */
  ARC_ERR_REQUEST_TOO_LARGE = -3, /* some request has more full blocks than capacity_blocks (needed for the pin guarantee, R4) */
  ARC_ERR_OOM = -4,               /* device or pinned-host allocation failed */
  ARC_ERR_CUDA = -5               /* any other CUDA error; text in arc_last_error */
};
/* Scope of the pins (R4): a block accessed by a request is never a victim until ... */
enum { ARC_PIN_REQUEST = 0,   /* ... its request's last access (default)                                                  */
       ARC_PIN_STEP = 1,      /* ... the step's last access: everything a step touches stays resident for the whole step */
       ARC_PIN_HELD = 2 };    /* ... arc_release gives the access's hold back (one hold per access, across steps)           */
/* class of one block access, as decided against the live state at the moment of the access (R3, R5) */
enum { ARC_MISS = 0, ARC_HIT_T1 = 1, ARC_HIT_T2 = 2, ARC_GHOST_B1 = 3, ARC_GHOST_B2 = 4 };

/* Result of one arc_step.  The struct itself is HOST memory filled by the call; every pointer in it is
 * DEVICE memory owned by the library.  The arrays are written by the step's kernels, i.e. they are valid
 * in stream order after the call, and stay intact until the next arc_step / arc_reset / arc_destroy on
 * the same handle is enqueued.  Index of logical block i of request r is blk_off[r] + i. */
typedef struct {
  uint64_t n_access;         /* N = total number of full blocks in the step (known on the host)            */
  const int32_t *prefix_len; /* [n_req]    cached-prefix length in TOKENS (multiple of block_size), R9     */
  const int64_t *blk_off;    /* [n_req+1]  exclusive scan of full blocks per request                       */
  const uint8_t *cls;        /* [N]        ARC_MISS .. ARC_GHOST_B2                                        */
  const int32_t *block_id;   /* [N]        physical block now holding the logical block, in [0, capacity)  */
  const int32_t *evicted_id; /* [N]        block ID evicted by this access, or -1                          */
  const int32_t *p_after;    /* [N]        p (target size of T1) after this access; 0 in LRU, c/2 in DBL mode */
  const int32_t *alloc_ids;  /* [counts[0]] IDs handed to non-hit accesses, in ACCESS order (R2)           */
  const int32_t *evict_ids;  /* [counts[1]] IDs evicted, in ACCESS order                                   */
  const uint32_t *counts;    /* [2]        n_alloc, n_evict                                                */
  const uint64_t *chain_state; /* [n_req]  H4 state after each request's last full block: what arc_step_resume takes
                                *          to continue the sequence (the state the request came with if it had no full block) */
} arc_step_result;

/* Result of arc_step_host / arc_step_host_wait: every pointer is pinned HOST memory owned by the library, filled when the
 * call returns, valid until the third arc_step_host(_async) after this step's, arc_reset or arc_destroy. */
typedef struct {
  uint64_t n_access;
  uint32_t n_alloc, n_evict;
  const int32_t *prefix_len; /* [n_req] */
  const int32_t *alloc_ids;  /* [n_alloc] */
  const int32_t *evict_ids;  /* [n_evict] */
  uint64_t h2d_bytes, d2h_bytes; /* what the step moved over the bus: tokens + offsets in; the packed results out */
} arc_host_result;

/* Cumulative counters since create/reset plus the current list sizes (R12). */
typedef struct {
  uint64_t steps, requests, tokens_seen, tokens_hashed, accesses;
  uint64_t hit_t1, hit_t2, ghost_b1, ghost_b2, miss;
  uint64_t evict_t1, evict_t2, drop_b1, drop_b2, fresh_ids_used, prefix_hit_tokens;
  uint64_t t1, t2, b1, b2, p, capacity_blocks;
  uint32_t block_size;
  int32_t policy;
} arc_stats_t;

/* Device time of the kernels of the last profiled step, in milliseconds (see arc_set_profiling). */
typedef struct {
  float hash_ms;     /* K1 chained block hashing                               */
  float probe_ms;    /* K2 directory probe + reserve                            */
  float machine_ms;  /* K3 ARC state machine (incl. its request bookkeeping)    */
  float finalize_ms; /* K4 prefix lengths, directory cleanup                    */
  float maint_ms;    /* directory rebuild / list compaction done before the step */
  float total_ms;    /* first enqueue -> last kernel done                       */
} arc_kernel_times;

/* Create an empty cache of `capacity_blocks` KV blocks of `block_size` tokens (the cache
 * size is the experiment knob).  *out receives the handle (HOST pointer to an
 * opaque object).  Device memory for the directory is allocated here and grows when a larger step
 * arrives (see arc_reserve). */
int arc_create(uint64_t capacity_blocks, uint32_t block_size, int policy, arc_cache **out);

/* Optional: pre-size all step-dependent device buffers for steps of up to max_req requests and
 * max_blocks_per_step full blocks, so that no later arc_step reallocates. */
int arc_reserve(arc_cache *h, uint32_t max_req, uint64_t max_blocks_per_step);

/* One scheduler step (BASELINE.json north_star (a)-(d)): hashes every full block of every request
 * (H1-H6), probes the device-resident directory, classifies every block access against the live
 * state in the fixed order R2 (requests ascending; inside a request tail block first), applies the
 * ARC (R5-R8) or LRU (R10) transitions with per-request pins (R4), and reports per-request cached
 * prefix lengths and the allocated / evicted block IDs (R9).
 *   d_tokens  DEVICE int32, CSR by h_offsets; any 4-byte alignment; borrowed until the step's work on
 *             the stream is done.  Token IDs are reinterpreted as uint32, no range check (H1).
 *   h_offsets HOST int64[n_req+1], monotone non-decreasing, h_offsets[0] >= 0; request r is
 *             d_tokens[h_offsets[r] .. h_offsets[r+1]).  Copied before the call returns.
 *   out       HOST struct, filled with DEVICE pointers (see arc_step_result).
 * Errors: see the enum; on any error the handle is unchanged and nothing was enqueued. */
int arc_step(arc_cache *h, const int32_t *d_tokens, const int64_t *h_offsets, uint32_t n_req,
             void *cuda_stream, arc_step_result *out);

/* arc_step for requests that CONTINUE a sequence at a block boundary (a running request whose generated
 * tokens fill new blocks, or a prompt sent in chunks).  d_chain_in: DEVICE uint64[n_req], read in stream order; entry r
 * is the H4 state before request r's first block - the chain_state a previous step returned for the same sequence, or
 * the constant S0 = 0x243F6A8885A308D3 for a new prompt.  NULL = S0 for every request (= arc_step).  Request r's tokens
 * then start at that block boundary: the caller re-sends the tokens of a block that was not full last time.  The keys,
 * and with them every result, are those of the unsplit sequence.  May alias a previous result's chain_state only if that
 * result is from another handle (a step overwrites its handle's chain_state). */
int arc_step_resume(arc_cache *h, const int32_t *d_tokens, const int64_t *h_offsets, const uint64_t *d_chain_in,
                    uint32_t n_req, void *cuda_stream, arc_step_result *out);

/* The same step end to end from HOST memory, pipelined: arc_step_host_async enqueues
 *   - the copy of h_tokens (HOST int32; pinned memory makes the copy asynchronous) to a library-owned device buffer, on
 *     the handle's own copy stream, so that it overlaps the steps still computing on cuda_stream,
 *   - the step itself on cuda_stream (which waits for that copy),
 *   - a kernel that writes the results straight into pinned, device-mapped host memory: n_alloc | n_evict | device error
 *     | prefix_len[n_req] | alloc_ids[n_alloc] | evict_ids[n_evict], exactly 4 (3 + n_req + n_alloc + n_evict) bytes,
 * and returns a ticket (never 0).  arc_step_host_wait(ticket) blocks until that step is done and fills `out` with
 * pointers into the pinned buffer, valid until the third arc_step_host_async after this step's; it returns ARC_ERR_CUDA
 * (with `out` filled) when the handle carries a sticky device-side error (e.g. a bad arc_release), which therefore
 * reaches a caller that never asks for arc_stats.  Up to three steps may be
 * in flight; a fourth arc_step_host_async before the oldest was waited for fails with ARC_ERR_INVALID_ARG and changes
 * nothing.  h_tokens must stay valid and unchanged until its step has been waited for; h_offsets is copied before return.
 * A step that needs larger buffers than the handle has (see arc_reserve) is accepted only with no step in flight.
 * arc_step_host = arc_step_host_async + arc_step_host_wait. */
int arc_step_host_async(arc_cache *h, const int32_t *h_tokens, const int64_t *h_offsets, uint32_t n_req, void *cuda_stream,
                        uint32_t *ticket_out);
int arc_step_host_wait(arc_cache *h, uint32_t ticket, arc_host_result *out);
int arc_step_host(arc_cache *h, const int32_t *h_tokens, const int64_t *h_offsets, uint32_t n_req,
                  void *cuda_stream, arc_host_result *out);

/* Sets the pin scope for the following steps.  With ARC_PIN_STEP a step whose
 * requests hold more than capacity_blocks full blocks in total is refused with ARC_ERR_REQUEST_TOO_LARGE (nothing is
 * enqueued, the handle is unchanged): the admission rule that guarantees a victim always exists. */
/* With ARC_PIN_HELD every access adds one hold to its block; a block with holds is never a victim, in
 * this step or any later one, until arc_release has given all its holds back.  A step is refused with
 * ARC_ERR_REQUEST_TOO_LARGE when the holds outstanding plus its full blocks exceed capacity_blocks.  The scope can be
 * changed only while no hold is outstanding (else ARC_ERR_INVALID_ARG). */
int arc_set_pin_scope(arc_cache *h, int scope);

/* ARC_PIN_HELD only: gives back one hold for every block ID listed - normally a finished request's block_id output, in
 * any order; an ID may appear several times.  d_block_ids: DEVICE int32[n], read in stream order.  The IDs are processed
 * in the order given; a block whose last hold goes re-enters the list it belongs to (T1 or T2) at the MRU end at that
 * moment.  Asynchronous.  n greater than the holds outstanding -> ARC_ERR_INVALID_ARG, nothing enqueued.  An ID that is
 * not a resident held block, or is listed more often than it is held, is found on the device: the call then changes
 * nothing and the handle carries a sticky device error that the next arc_stats reports as ARC_ERR_CUDA. */
int arc_release(arc_cache *h, const int32_t *d_block_ids, uint64_t n, void *cuda_stream);

/* Holds outstanding (accesses made under ARC_PIN_HELD minus IDs released); host-side, exact, no synchronisation. */
uint64_t arc_hold_units(const arc_cache *h);

/* Synchronises the stream of the handle's last step and copies the counters.  out: HOST. */
int arc_stats(arc_cache *h, arc_stats_t *out);

/* Back to the empty state (lists, ghosts, p, block IDs, counters); buffers are kept. */
int arc_reset(arc_cache *h);

/* Frees everything.  NULL is a no-op. */
void arc_destroy(arc_cache *h);

/* Text of the last error on this handle (HOST, handle-owned, never NULL); h == NULL returns the text
 * of the last arc_create failure on this thread. */
const char *arc_last_error(const arc_cache *h);

/* Stateless K1: keys of every full block (H1-H6) in natural order, d_keys_out[blk_off[r] + i].
 *   d_tokens DEVICE, h_offsets HOST (as in arc_step), d_keys_out DEVICE uint64[N] with
 *   N = sum_r floor(len_r / block_size) (the caller computes it from the offsets).
 * Asynchronous on cuda_stream; thread-safe; calls on different streams may overlap (every call has scratch of its own:
 * the offsets go to the device through a library-owned copy stream, 16 (n_req + 1) + 16 bytes per call). */
int arc_hash_blocks(const int32_t *d_tokens, const int64_t *h_offsets, uint32_t n_req, uint32_t block_size,
                    uint64_t *d_keys_out, void *cuda_stream);

/* One entry of the work list of the bulk hashing kernel: a request (or any run of full blocks) of n_blocks blocks whose
 * tokens start at d_tokens[tok_off] and whose keys go to d_keys_out[key_off ..].  32 bytes. */
typedef struct { int64_t tok_off; int64_t key_off; uint32_t n_blocks; uint32_t reserved[3]; } arc_hash_item;

/* The bulk hashing kernel with its work list already on the device: the kernel-only figure of the K1 roofline run, and
 * for callers that build their batch on the device.  arc_hash_blocks builds exactly this list from the host offsets (one
 * item per request with a full block, longest first) and copies it.  d_items: DEVICE arc_hash_item[n_items]; warps take
 * the items in list order.  [tok_lo, tok_hi): the token indices of d_tokens the kernel may touch (the 16-byte-aligned
 * bulk copies read nothing outside it).  d_ticket: DEVICE, two uint32 words of caller-owned scratch that must be 0 at
 * launch; the kernel leaves them 0 again, so one scratch zeroed once serves every later call ON THE SAME STREAM (calls
 * that may run at the same time need scratch of their own).  Nothing is validated or copied; one kernel launch. */
int arc_hash_blocks_device(const int32_t *d_tokens, const arc_hash_item *d_items, uint32_t n_items, int64_t tok_lo, int64_t tok_hi,
                           uint32_t block_size, uint64_t *d_keys_out, uint32_t *d_ticket, void *cuda_stream);

/* arc_hash_blocks for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same arguments, same keys (natural order, every chain from S0), but the call and everything it
 * launches allocate NOTHING - no cudaMalloc / cudaFree / cudaMallocHost, no copy through a staging buffer.  The offsets
 * travel as a 4 KB kernel argument and the kernels' scratch is a fixed 34 KB (34,816-byte) __device__ array inside the library image
 * (every GPU that loads the library holds it until the process exits).  Limits, checked before anything is enqueued
 * (ARC_ERR_REQUEST_TOO_LARGE with the numbers in arc_last_error(NULL)): n_req <= 253, and n_req x ceil(longest request in
 * blocks / 128) <= 4,096 segments, no request longer than 1,024 segments (e.g. 64 requests of up to 8,192 blocks = 131,072
 * tokens each, or 4 of 131,072 blocks).  Two launches (requests cut into 128-block segments hashed from a zero carry, then put
 * together: H4 is affine), asynchronous on cuda_stream.  Every call on a device SHARES the one scratch array: calls whose
 * kernels may overlap on the GPU (different streams, several host threads) race and give wrong keys - keep them on one
 * stream or order them with events.  Nothing in the array has to be cleared: a call reads only words it has written. */
int arc_hash_blocks_static(const int32_t *d_tokens, const int64_t *h_offsets, uint32_t n_req, uint32_t block_size,
                           uint64_t *d_keys_out, void *cuda_stream);

/* Prefix-affinity routing for N per-GPU caches behind a router: writes to
 * d_dst_out[r] (DEVICE int32[n_req]) the shard of request r = (key of its first full block >> 33) mod world, 0 for a
 * request shorter than one block - requests that share a document or conversation prefix meet in the same cache.
 * d_tokens DEVICE, d_offsets DEVICE int64[n_req+1].  Stateless, one kernel, asynchronous on cuda_stream. */
int arc_route_requests(const int32_t *d_tokens, const int64_t *d_offsets, uint32_t n_req, uint32_t block_size, uint32_t world,
                       int32_t *d_dst_out, void *cuda_stream);

/* Diagnostics ------------------------------------------------------------------------------------ */

/* When enabled, arc_step records CUDA events between its kernels (on the step's stream); the times of
 * the last step are read with arc_last_kernel_times, which synchronises.  Off by default. */
int arc_set_profiling(arc_cache *h, int enabled);
int arc_last_kernel_times(arc_cache *h, arc_kernel_times *out);

/* Number of kernels the library launched for this handle since create/reset (arc_hash_blocks launches
 * are counted in a process-wide counter returned when h == NULL). */
uint64_t arc_launch_count(const arc_cache *h);

/* Selects the implementation of a step (all give identical results): 0 = automatic (default): steps of up to 1,024
 * accesses and 253 requests run as ONE kernel (K1-K4 as phases of a single CTA); larger steps run the
 * four kernels with the wide K3 machine, or the one-warp machine when requests average fewer than 48 blocks;
 * 1 = four kernels, K3 as a single-thread serial walk (the by-the-book routine on the device, much slower);
 * 2 = four kernels, one-warp machine with 32-access windows; 3 = four kernels, wide machine, pipelined form: one CTA of
 * 12 warps, 128-access windows - four owner warps (fetch, checks, apply), four scanner warps (victims from the LRU ends of
 * the four lists) and four roller warps that work out the counter recurrence and every access's plan one window AHEAD of
 * the owners; 4 = the one-launch kernel for every step it can take (up to 4,096 accesses and 253 requests), automatic
 * otherwise; 5 = the wide machine without the roller warps (8 warps, every owner warp rolls its window itself: round
 * 1's form, and the one-launch kernel's). */
int arc_set_machine(arc_cache *h, int which);

/* K2 alone, for the probe microbenchmark and its tests: looks every key of d_keys (DEVICE uint64[n], values >= 2) up in
 * the handle's directory, inserting unknown keys as placeholder nodes exactly as arc_step's probe does, and writes the
 * node index of key i to d_nodes_out[i] (DEVICE uint32[n]).  Asynchronous on cuda_stream.  The placeholders are never
 * cleaned up (no K4 runs), so use a handle that is destroyed afterwards.  Since round 2 the probe is one thread per key
 * reading one 32-byte bucket (two 16-byte slots) per probe, inserts publish key and node id with one 128-bit CAS. */
int arc_debug_probe(arc_cache *h, const uint64_t *d_keys, uint64_t n, uint32_t *d_nodes_out, void *cuda_stream);

/* Measurement aid: the random-sector ceiling K2 is compared with ("a measured random-sector ceiling").
 * For every d_keys[i] (DEVICE uint64[n]) reads the 32-byte sector number (low 32 bits of the key) & (n_sectors - 1) of
 * d_buf (DEVICE, 32-byte aligned, n_sectors * 32 bytes, n_sectors a power of two <= 2^32) with the load K2 uses and
 * writes the XOR of its eight words to d_out[i] (DEVICE uint32[n]).  Same grid and loads as K2, no compare, no insert.
 * Stateless; asynchronous on cuda_stream. */
int arc_debug_gather_sectors(const uint64_t *d_keys, uint64_t n, const void *d_buf, uint64_t n_sectors, uint32_t *d_out, void *cuda_stream);

/* Test hook: from the next step on every block key is ANDed with `mask` (results below 2 are bumped by 2) before the
 * directory probe, so that a test can force equal keys inside one request, which the 64-bit hash makes unobservable
 * otherwise (the "same node twice in a window" paths of K3).  ~0 restores normal operation.  Not for production use:
 * with a mask, different blocks share cache entries. */
int arc_debug_set_key_mask(arc_cache *h, uint64_t mask);

/* K3 diagnostics, cumulative since create/reset: out[0..n) (HOST) receives, in this order, the number of
 * all-hit windows, general windows, by-the-book single accesses, windows cut at a repeated node, windows cut at a
 * conflict, ring scan rounds, accesses applied in all-hit windows, accesses applied in general windows, then
 * SM cycles spent in: fetch, roll-forward, victim scan, apply, single accesses, the whole kernel; then the number of
 * calls of the roll-forward routine and of its phases; then (pipelined wide machine) the windows whose decisions had been
 * rolled ahead by the roller warps and stood, and the windows that had to be rolled on request.  Synchronises.  (In the
 * pipelined form "roll-forward" cycles are what the owners spend taking the rollers' result; the wait for it is booked
 * under fetch.) */
int arc_debug_counters(arc_cache *h, uint64_t *out, uint32_t n);

/* Per-access latency of the by-the-book K3 machine (arc_set_machine(h, 1)) by class, cumulative since create/reset:
 * out[cls * 16 + b] (HOST uint32[80], cls = ARC_MISS .. ARC_GHOST_B2) counts the accesses whose serial_access took
 * fewer than 64 SM cycles (b = 0) or [64 * 2^(b-1), 64 * 2^b) cycles (b = 1..15; clock64 on the SM).  The window machines
 * apply accesses in batches, so a per-access latency exists only here.  Synchronises. */
int arc_debug_latency_hist(arc_cache *h, uint32_t *out);

/* Copies one list (1 = T1, 2 = T2, 3 = B1, 4 = B2) in LRU -> MRU order to HOST arrays keys_out /
 * block_ids_out (either may be NULL), at most cap entries; *n_out receives the list length.
 * Synchronises.  For tests. */
int arc_debug_list(arc_cache *h, int which, uint64_t *keys_out, int32_t *block_ids_out, uint64_t cap, uint64_t *n_out);

#ifdef __cplusplus
}
#endif
#endif /* ARC_B200_H */
