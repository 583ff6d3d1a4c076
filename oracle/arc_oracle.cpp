// CPU oracle of the per-step prefix-KV lookup + ARC (or LRU) update.  TEST INFRASTRUCTURE ONLY.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may
// load this library.  It shares no source, header, constant table or helper with the CUDA path
// (paper_2606_21238_b200/csrc) and neither includes the other.
//
// One thread, requests in order, blocks tail-first, one by-the-book access each: the sequential
// *definition* that the GPU path must reproduce bit-exactly.  std::list + std::unordered_map, no
// blocking, no batching, no SIMD.
//
// Passages followed (PAPER.md = /root/reference/PAPER.md; R*/H* = DESIGN.md §3):
//   - lists: L1 = T1+B1 "accessed once", L2 = T2+B2 "accessed multiple times", promotion on a hit
//     (PAPER.md:47); T1/T2 "refer to KV blocks in memory", B1/B2 "store only the metadata"
//
//   - ghost hit flow: block in B2 is a miss, regenerated, put in T2, LRU block of T1 evicted; "the
//     combination of T1 and T2 is of fixed size"; B1 hits => invest in T1
//   - decisions at KV-block level, e.g. 16-token blocks; LRU = naive vLLM
//   - the case analysis is Megiddo & Modha's, restated as R5-R8
//   - everything the paper leaves open (hash, order of a request's blocks, pins, integer p, block IDs,
//     errors) is a reading listed in DESIGN.md §4.
// Pins of this file: hand traces A-E, invariants I1-I12, brute-force differential against
// oracle_bruteforce.py, LRU stack-distance closed form, ARC==LRU trace classes, step-partition
// invariance, hash vectors + closed forms (tests/test_oracle_*.py).  No function is "parity unpinned".
#include <chrono>
#include <cstdint>
#include <cstring>
#include <list>
#include <string>
#include <unordered_map>
#include <vector>

namespace {

// ---- H1-H6: the documented 64-bit chained block hash (all arithmetic mod 2^64) ------------------
const uint64_t HM = 0x9E3779B97F4A7C15ull;
const uint64_t HC1 = 0xBF58476D1CE4E5B9ull;
const uint64_t HC2 = 0x94D049BB133111EBull;
const uint64_t HK = 0xD1342543DE82EF95ull;
const uint64_t HS0 = 0x243F6A8885A308D3ull;

uint64_t mix(uint64_t z) {  // H5
  z ^= z >> 30; z *= HC1;
  z ^= z >> 27; z *= HC2;
  z ^= z >> 31;
  return z;
}

uint64_t content_hash(const int32_t* t, uint32_t B) {  // H2, H3
  uint64_t g = 0;
  for (uint32_t k = 0; k < B / 2; ++k) {
    uint64_t w = (uint64_t)(uint32_t)t[2 * k] | ((uint64_t)(uint32_t)t[2 * k + 1] << 32);  // H1
    uint64_t e = (w + (uint64_t)(k + 1) * HM) * HC1;
    g += e ^ (e >> 32);
  }
  return g;
}

uint64_t key_from_state(uint64_t s) {  // H5: 0 and 1 are reserved for table sentinels
  uint64_t key = mix(s);
  if (key < 2) key += 2;
  return key;
}

// keys of the full blocks of one request, block 0 first (H4, H5, H6).  s = the chain state before block 0: S0 for a
// prompt, or the state a previous call returned for the same sequence (a request that continues at a
// block boundary).  Returns the state after the last full block.
uint64_t request_keys(const int32_t* t, int64_t len, uint32_t B, uint64_t* out, uint64_t s = HS0) {
  for (int64_t i = 0; i < len / B; ++i) {
    s = s * HK + content_hash(t + i * B, B);
    if (out) out[i] = key_from_state(s);
  }
  return s;
}

enum { MISS = 0, HIT_T1 = 1, HIT_T2 = 2, GHOST_B1 = 3, GHOST_B2 = 4 };
enum { IN_T1 = 1, IN_T2 = 2, IN_B1 = 3, IN_B2 = 4 };
enum { POLICY_ARC = 0, POLICY_LRU = 1, POLICY_DBL = 2 };   // DBL = ARC's lists with p frozen at c/2
enum { OK = 0, ERR_INVALID_ARG = -1, ERR_UNSUPPORTED = -2, ERR_REQUEST_TOO_LARGE = -3, ERR_OOM = -4 };

typedef std::list<uint64_t> KeyList;  // front = LRU end, back = MRU end

struct Entry {
  int where;              // IN_T1 .. IN_B2
  KeyList::iterator it;   // position in that list
  int32_t block;          // block ID if resident, -1 for ghosts (I8)
  bool pinned;            // R4
  uint32_t holds;         // pin scope 2: accesses not yet released; > 0 = not evictable
};

}  // namespace

extern "C" {

struct oracle_stats_t {  // same fields and order as the C ABI's arc_stats_t
  uint64_t steps, requests, tokens_seen, tokens_hashed, accesses;
  uint64_t hit_t1, hit_t2, ghost_b1, ghost_b2, miss;
  uint64_t evict_t1, evict_t2, drop_b1, drop_b2, fresh_ids_used, prefix_hit_tokens;
  uint64_t t1, t2, b1, b2, p, capacity_blocks;
  uint32_t block_size;
  int32_t policy;
};

struct oracle_step_result {  // HOST pointers, owned by the handle, valid until the next step
  uint64_t n_access;
  const int32_t* prefix_len;   // [n_req]
  const int64_t* blk_off;      // [n_req+1]
  const uint8_t* cls;          // [n_access]  index blk_off[r]+i
  const int32_t* block_id;     // [n_access]
  const int32_t* evicted_id;   // [n_access]
  const int32_t* p_after;      // [n_access]
  const int32_t* alloc_ids;    // [n_alloc]  access order
  const int32_t* evict_ids;    // [n_evict]  access order
  uint32_t n_alloc, n_evict;
  const uint64_t* chain_state; // [n_req]    H4 state after each request's last full block (oracle_step / oracle_step_resume)
};

struct oracle_cache {
  uint64_t c;
  uint32_t B;
  int policy;
  int pin_scope;          // 0: pins end with their request (R4); 1: with the step (NEXT-3);
                          // 2: held until oracle_release (NEXT-3)
  uint64_t hold_units;    // scope 2: accesses made minus block IDs released = the sum of all hold counts
  std::vector<uint64_t> owner;   // scope 2: owner[block ID] = key of the resident entry that has it
  KeyList T1, T2, B1, B2;
  std::unordered_map<uint64_t, Entry> dir;
  uint64_t p;
  int32_t next_fresh;
  std::vector<uint64_t> pinned_keys;
  oracle_stats_t st;
  double hash_seconds, arc_seconds;
  // result storage
  std::vector<int32_t> prefix_len, block_id, evicted_id, p_after, alloc_ids, evict_ids;
  std::vector<int64_t> blk_off;
  std::vector<uint8_t> cls;
  std::vector<uint64_t> keys, chain_state;
};

}  // extern "C"

namespace {

KeyList& list_of(oracle_cache* h, int where) {
  switch (where) {
    case IN_T1: return h->T1;
    case IN_T2: return h->T2;
    case IN_B1: return h->B1;
    default: return h->B2;
  }
}

void put_mru(oracle_cache* h, uint64_t x, int where, int32_t block) {
  KeyList& l = list_of(h, where);
  l.push_back(x);
  Entry e;
  e.where = where;
  e.it = --l.end();
  e.block = block;
  e.pinned = false;
  e.holds = 0;
  h->dir[x] = e;
  if (block >= 0) { if (h->owner.size() <= (size_t)block) h->owner.resize((size_t)block + 1, 0); h->owner[block] = x; }
}

void remove_key(oracle_cache* h, uint64_t x) {
  Entry& e = h->dir.at(x);
  list_of(h, e.where).erase(e.it);
  h->dir.erase(x);
}

// first unpinned entry from the LRU end; returns false if none (R7)
bool first_unpinned(oracle_cache* h, KeyList& l, uint64_t* out) {
  for (KeyList::iterator it = l.begin(); it != l.end(); ++it)
    if (!h->dir.at(*it).pinned && h->dir.at(*it).holds == 0) { *out = *it; return true; }
  return false;
}

// R7.  Returns the freed block ID.
int32_t replace(oracle_cache* h, bool in_b2) {
  uint64_t t1 = h->T1.size();
  bool prefer_t1 = t1 >= 1 && (t1 > h->p || (in_b2 && t1 == h->p));
  for (int attempt = 0; attempt < 2; ++attempt) {
    bool from_t1 = (attempt == 0) ? prefer_t1 : !prefer_t1;
    uint64_t v;
    if (!first_unpinned(h, from_t1 ? h->T1 : h->T2, &v)) continue;
    int32_t block = h->dir.at(v).block;
    remove_key(h, v);
    put_mru(h, v, from_t1 ? IN_B1 : IN_B2, -1);  // the victim becomes a ghost and loses its ID
    if (from_t1) h->st.evict_t1++; else h->st.evict_t2++;
    return block;
  }
  return -2;  // unreachable while nb_r <= c holds (R4)
}

// evict the first unpinned entry of T1 without making it a ghost (case 4A-else and LRU mode)
int32_t evict_t1_no_ghost(oracle_cache* h) {
  uint64_t v;
  if (!first_unpinned(h, h->T1, &v)) return -2;
  int32_t block = h->dir.at(v).block;
  remove_key(h, v);
  h->st.evict_t1++;
  return block;
}

void pin(oracle_cache* h, uint64_t x) {
  Entry& e = h->dir.at(x);
  if (h->pin_scope == 2) { e.holds++; return; }     // held until released: one hold per access
  if (!e.pinned) { e.pinned = true; h->pinned_keys.push_back(x); }
}

// R5 (ARC) / R10 (LRU): one access.
void access(oracle_cache* h, uint64_t x, uint8_t* cls_out, int32_t* block_out, int32_t* evicted_out) {
  const uint64_t c = h->c;
  h->st.accesses++;
  int32_t evicted = -1;
  uint8_t cls;
  std::unordered_map<uint64_t, Entry>::iterator f = h->dir.find(x);

  if (h->policy == POLICY_LRU) {
    if (f != h->dir.end()) {  // hit: move to MRU
      cls = HIT_T1; h->st.hit_t1++;
      int32_t block = f->second.block; bool was_pinned = f->second.pinned; uint32_t holds = f->second.holds;
      remove_key(h, x); put_mru(h, x, IN_T1, block); h->dir.at(x).pinned = was_pinned; h->dir.at(x).holds = holds;
    } else {
      cls = MISS; h->st.miss++;
      int32_t v;
      if (h->T1.size() < c) { v = h->next_fresh++; h->st.fresh_ids_used++; }
      else { v = evicted = evict_t1_no_ghost(h); }
      put_mru(h, x, IN_T1, v);
    }
    pin(h, x);
    *cls_out = cls; *block_out = h->dir.at(x).block; *evicted_out = evicted;
    return;
  }

  const uint64_t t1 = h->T1.size(), t2 = h->T2.size(), b1 = h->B1.size(), b2 = h->B2.size();
  if (f != h->dir.end() && (f->second.where == IN_T1 || f->second.where == IN_T2)) {  // case 1
    if (f->second.where == IN_T1) { cls = HIT_T1; h->st.hit_t1++; } else { cls = HIT_T2; h->st.hit_t2++; }
    int32_t block = f->second.block; bool was_pinned = f->second.pinned; uint32_t holds = f->second.holds;
    remove_key(h, x); put_mru(h, x, IN_T2, block); h->dir.at(x).pinned = was_pinned; h->dir.at(x).holds = holds;
  } else if (f != h->dir.end() && f->second.where == IN_B1) {  // case 2
    cls = GHOST_B1; h->st.ghost_b1++;
    uint64_t delta = b2 / b1; if (delta < 1) delta = 1;          // R6: floor, at least 1
    if (h->policy != POLICY_DBL) h->p = (h->p + delta > c) ? c : h->p + delta;   // DBL: no adaptation
    int32_t v = evicted = replace(h, false);
    remove_key(h, x); put_mru(h, x, IN_T2, v);
  } else if (f != h->dir.end() && f->second.where == IN_B2) {  // case 3
    cls = GHOST_B2; h->st.ghost_b2++;
    uint64_t delta = b1 / b2; if (delta < 1) delta = 1;
    if (h->policy != POLICY_DBL) h->p = (h->p < delta) ? 0 : h->p - delta;
    int32_t v = evicted = replace(h, true);
    remove_key(h, x); put_mru(h, x, IN_T2, v);
  } else {  // case 4
    cls = MISS; h->st.miss++;
    int32_t v;
    if (t1 + b1 == c) {  // (A)
      if (t1 < c) {
        remove_key(h, h->B1.front()); h->st.drop_b1++;
        v = evicted = replace(h, false);
      } else {
        v = evicted = evict_t1_no_ghost(h);
      }
    } else {  // (B)
      uint64_t n = t1 + t2 + b1 + b2;
      if (n >= c) {
        if (n == 2 * c) { remove_key(h, h->B2.front()); h->st.drop_b2++; }
        v = evicted = replace(h, false);
      } else {
        v = h->next_fresh++; h->st.fresh_ids_used++;
      }
    }
    put_mru(h, x, IN_T1, v);
  }
  pin(h, x);
  *cls_out = cls; *block_out = h->dir.at(x).block; *evicted_out = evicted;
}

double now_s() {
  return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

// R2-R4, R9 over precomputed keys (block 0 first inside each request).
int step_keys(oracle_cache* h, const uint64_t* keys, const int64_t* blk_off, uint32_t n_req, oracle_step_result* out) {
  for (uint32_t r = 0; r < n_req; ++r)
    if ((uint64_t)(blk_off[r + 1] - blk_off[r]) > h->c) return ERR_REQUEST_TOO_LARGE;  // R11: before any change
  const int64_t N = blk_off[n_req];
  if (h->pin_scope == 1 && (uint64_t)N > h->c) return ERR_REQUEST_TOO_LARGE;   // step-wide pins: a step may pin at most c blocks
  if (h->pin_scope == 2 && h->hold_units + (uint64_t)N > h->c) return ERR_REQUEST_TOO_LARGE;   // holds outstanding + new <= c
  if (h->pin_scope == 2) h->hold_units += (uint64_t)N;
  h->prefix_len.assign(n_req, 0);
  h->blk_off.assign(blk_off, blk_off + n_req + 1);
  h->cls.assign(N, 0); h->block_id.assign(N, -1); h->evicted_id.assign(N, -1); h->p_after.assign(N, 0);
  h->alloc_ids.clear(); h->evict_ids.clear();
  for (uint32_t r = 0; r < n_req; ++r) {          // R2: requests ascending
    const int64_t o = blk_off[r], nb = blk_off[r + 1] - o;
    for (int64_t i = nb - 1; i >= 0; --i) {       // R2: tail first, block 0 last
      access(h, keys[o + i], &h->cls[o + i], &h->block_id[o + i], &h->evicted_id[o + i]);
      h->p_after[o + i] = (int32_t)h->p;
      if (h->cls[o + i] != HIT_T1 && h->cls[o + i] != HIT_T2) h->alloc_ids.push_back(h->block_id[o + i]);
      if (h->evicted_id[o + i] >= 0) h->evict_ids.push_back(h->evicted_id[o + i]);
    }
    if (h->pin_scope == 0) {
      for (size_t k = 0; k < h->pinned_keys.size(); ++k) {   // R4: pins drop when the request completes
        std::unordered_map<uint64_t, Entry>::iterator f = h->dir.find(h->pinned_keys[k]);
        if (f != h->dir.end()) f->second.pinned = false;
      }
      h->pinned_keys.clear();
    }
    int64_t lead = 0;                               // R9
    while (lead < nb && (h->cls[o + lead] == HIT_T1 || h->cls[o + lead] == HIT_T2)) ++lead;
    h->prefix_len[r] = (int32_t)(lead * h->B);
    h->st.prefix_hit_tokens += lead * h->B;
  }
  for (size_t k = 0; k < h->pinned_keys.size(); ++k) {     // step-wide scope: pins drop when the step completes
    std::unordered_map<uint64_t, Entry>::iterator f = h->dir.find(h->pinned_keys[k]);
    if (f != h->dir.end()) f->second.pinned = false;
  }
  h->pinned_keys.clear();
  h->st.steps++; h->st.requests += n_req;
  if (out) {
    out->n_access = (uint64_t)N;
    out->prefix_len = h->prefix_len.data(); out->blk_off = h->blk_off.data(); out->cls = h->cls.data();
    out->block_id = h->block_id.data(); out->evicted_id = h->evicted_id.data(); out->p_after = h->p_after.data();
    out->alloc_ids = h->alloc_ids.data(); out->evict_ids = h->evict_ids.data();
    out->n_alloc = (uint32_t)h->alloc_ids.size(); out->n_evict = (uint32_t)h->evict_ids.size();
    out->chain_state = h->chain_state.data();
  }
  return OK;
}

}  // namespace

extern "C" {

int oracle_create(uint64_t capacity_blocks, uint32_t block_size, int policy, oracle_cache** out) {
  if (!out) return ERR_INVALID_ARG;
  *out = 0;
  if (capacity_blocks == 0 || capacity_blocks > 0x7FFFFFFEull) return ERR_INVALID_ARG;
  if (policy != POLICY_ARC && policy != POLICY_LRU && policy != POLICY_DBL) return ERR_INVALID_ARG;
  if (block_size == 0 || (block_size & 1)) return ERR_UNSUPPORTED;   // the hash is defined for even B
  oracle_cache* h = new oracle_cache();
  h->c = capacity_blocks; h->B = block_size; h->policy = policy; h->next_fresh = 0; h->pin_scope = 0; h->hold_units = 0;
  h->p = (policy == POLICY_DBL) ? capacity_blocks / 2 : 0;   // DBL: the fixed 1:1 split
  std::memset(&h->st, 0, sizeof(h->st));
  h->hash_seconds = h->arc_seconds = 0.0;
  *out = h;
  return OK;
}

void oracle_destroy(oracle_cache* h) { delete h; }

// 0 = pins end with their request (R4, default); 1 = with the step (every block a step touches stays resident until the
// step's last access; a step of more than capacity blocks is refused).
// 2 = held: every access adds one hold to its block; a block with holds is never a victim; holds
// end only through oracle_release.  Scope 2 can be entered or left only while nothing is held.
int oracle_set_pin_scope(oracle_cache* h, int scope) {
  if (!h || (scope != 0 && scope != 1 && scope != 2)) return ERR_INVALID_ARG;
  if (h->hold_units != 0) return ERR_INVALID_ARG;
  h->pin_scope = scope;
  return OK;
}

// Scope 2: gives back one hold for every block ID listed (a request's block_id output, in any order; an ID may appear
// several times).  IDs are processed in the order given; a block whose hold count reaches zero moves to the MRU end of
// the list it is in (T1 or T2) at that moment - the position it had while held never matters, because held blocks are
// skipped by every victim choice.  All IDs are checked first: an ID that is not a resident block, or that is listed more
// often than it is held, makes the call fail with no change.
int oracle_release(oracle_cache* h, const int32_t* ids, uint64_t n) {
  if (!h || (!ids && n) || h->pin_scope != 2) return ERR_INVALID_ARG;
  std::unordered_map<int32_t, uint32_t> mult;
  for (uint64_t i = 0; i < n; ++i) {
    int32_t id = ids[i];
    if (id < 0 || (size_t)id >= h->owner.size()) return ERR_INVALID_ARG;
    std::unordered_map<uint64_t, Entry>::iterator f = h->dir.find(h->owner[id]);
    if (f == h->dir.end() || f->second.block != id) return ERR_INVALID_ARG;
    if (++mult[id] > f->second.holds) return ERR_INVALID_ARG;
  }
  for (uint64_t i = 0; i < n; ++i) {
    uint64_t x = h->owner[ids[i]];
    Entry& e = h->dir.at(x);
    if (--e.holds == 0) { int where = e.where; int32_t block = e.block; remove_key(h, x); put_mru(h, x, where, block); }
  }
  h->hold_units -= n;
  return OK;
}

uint64_t oracle_hold_units(oracle_cache* h) { return h->hold_units; }

// Stateless: keys of every full block, natural order (index blk_off[r]+i).  keys_out may be NULL to
// only fill blk_off_out ([n_req+1]).
int oracle_hash_blocks(const int32_t* tokens, const int64_t* offsets, uint32_t n_req, uint32_t block_size,
                       uint64_t* keys_out, int64_t* blk_off_out) {
  if (!offsets || (!tokens && n_req && offsets[n_req] > offsets[0])) return ERR_INVALID_ARG;
  if (block_size == 0 || (block_size & 1)) return ERR_UNSUPPORTED;
  if (offsets[0] < 0) return ERR_INVALID_ARG;
  for (uint32_t r = 0; r < n_req; ++r) if (offsets[r + 1] < offsets[r]) return ERR_INVALID_ARG;
  int64_t o = 0;
  for (uint32_t r = 0; r < n_req; ++r) {
    int64_t len = offsets[r + 1] - offsets[r];
    if (blk_off_out) blk_off_out[r] = o;
    if (keys_out) request_keys(tokens + offsets[r], len, block_size, keys_out + o);
    o += len / block_size;
  }
  if (blk_off_out) blk_off_out[n_req] = o;
  return OK;
}

int oracle_step_keys(oracle_cache* h, const uint64_t* keys, const int64_t* blk_off, uint32_t n_req, oracle_step_result* out) {
  if (!h || !blk_off || (!keys && blk_off[n_req] > 0)) return ERR_INVALID_ARG;
  double t0 = now_s();
  int rc = step_keys(h, keys, blk_off, n_req, out);
  h->arc_seconds += now_s() - t0;
  return rc;
}

// One step whose request r continues a sequence at a block boundary: chain_in[r] is the H4 state before its first block
// (S0 for a new prompt; chain_in == NULL means S0 for all).  Everything else is oracle_step.
int oracle_step_resume(oracle_cache* h, const int32_t* tokens, const int64_t* offsets, const uint64_t* chain_in, uint32_t n_req,
                       oracle_step_result* out) {
  if (!h || !offsets || n_req > (1u << 20)) return ERR_INVALID_ARG;
  if (offsets[0] < 0) return ERR_INVALID_ARG;
  for (uint32_t r = 0; r < n_req; ++r) if (offsets[r + 1] < offsets[r]) return ERR_INVALID_ARG;
  if (!tokens && offsets[n_req] > offsets[0]) return ERR_INVALID_ARG;
  double t0 = now_s();
  std::vector<int64_t> blk_off(n_req + 1);
  oracle_hash_blocks(tokens, offsets, n_req, h->B, 0, blk_off.data());
  for (uint32_t r = 0; r < n_req; ++r)
    if ((uint64_t)(blk_off[r + 1] - blk_off[r]) > h->c) return ERR_REQUEST_TOO_LARGE;   // before hashing: no state change
  if (h->pin_scope == 1 && (uint64_t)blk_off[n_req] > h->c) return ERR_REQUEST_TOO_LARGE;
  if (h->pin_scope == 2 && h->hold_units + (uint64_t)blk_off[n_req] > h->c) return ERR_REQUEST_TOO_LARGE;
  h->keys.resize(blk_off[n_req]);
  h->chain_state.resize(n_req);
  for (uint32_t r = 0; r < n_req; ++r)
    h->chain_state[r] = request_keys(tokens + offsets[r], offsets[r + 1] - offsets[r], h->B, h->keys.data() + blk_off[r],
                                     chain_in ? chain_in[r] : HS0);
  double t1 = now_s();
  int rc = step_keys(h, h->keys.data(), blk_off.data(), n_req, out);
  double t2 = now_s();
  h->hash_seconds += t1 - t0; h->arc_seconds += t2 - t1;
  if (rc == OK) {
    h->st.tokens_seen += (uint64_t)(offsets[n_req] - offsets[0]);
    h->st.tokens_hashed += (uint64_t)blk_off[n_req] * h->B;
  }
  return rc;
}

int oracle_step(oracle_cache* h, const int32_t* tokens, const int64_t* offsets, uint32_t n_req, oracle_step_result* out) {
  return oracle_step_resume(h, tokens, offsets, 0, n_req, out);
}

int oracle_stats(oracle_cache* h, oracle_stats_t* out) {
  if (!h || !out) return ERR_INVALID_ARG;
  *out = h->st;
  out->t1 = h->T1.size(); out->t2 = h->T2.size(); out->b1 = h->B1.size(); out->b2 = h->B2.size();
  out->p = h->p; out->capacity_blocks = h->c; out->block_size = h->B; out->policy = h->policy;
  return OK;
}

void oracle_timing(oracle_cache* h, double* hash_seconds, double* arc_seconds) {
  *hash_seconds = h->hash_seconds; *arc_seconds = h->arc_seconds;
}

// Introspection for the invariant tests: copies list `which` (1=T1, 2=T2, 3=B1, 4=B2) LRU -> MRU into
// keys_out / blocks_out (either may be NULL), at most cap entries; returns the list length.  Held entries (scope 2) are
// left out: their position means nothing until they are released.
uint64_t oracle_dump_list(oracle_cache* h, int which, uint64_t* keys_out, int32_t* blocks_out, uint64_t cap) {
  KeyList& l = list_of(h, which);
  uint64_t n = 0;
  for (KeyList::iterator it = l.begin(); it != l.end(); ++it) {
    if (h->dir.at(*it).holds > 0) continue;
    if (n < cap) {
      if (keys_out) keys_out[n] = *it;
      if (blocks_out) blocks_out[n] = h->dir.at(*it).block;
    }
    ++n;
  }
  return n;
}

int32_t oracle_next_fresh(oracle_cache* h) { return h->next_fresh; }

// Test hooks for the hash pins (H3 content hash of one block; H5 finaliser with the reserved-value rule).
uint64_t oracle_content_hash(const int32_t* block_tokens, uint32_t block_size) { return content_hash(block_tokens, block_size); }
uint64_t oracle_key_from_state(uint64_t s) { return key_from_state(s); }

}  // extern "C"
