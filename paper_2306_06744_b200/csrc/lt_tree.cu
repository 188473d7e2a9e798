// lt_tree.cu -- key codec (Alg. 1), uniform build, adaptation (Alg. 6) and the 2:1 balance
// ripple (Alg. 4 re-expressed) for sm_100a.  Product code.
//
// Every kernel here is a persistent grid (a multiple of the SM count) that reads the leaf
// count from device memory, so no launch depends on a host round trip.
#include <cooperative_groups.h>

#include "lt_internal.h"

namespace cg = cooperative_groups;

namespace lt {

constexpr int BT = 256;  // threads per block of the tree kernels
constexpr int kScanTiles = 4;  // tiles of BT leaves ordered by ONE block scan (16-bit packed counts)

enum { ACT_KEEP = 0, ACT_REFINE = 1, ACT_PARENT = 2, ACT_DROP = 3 };

// ------------------------------------------------------------------------ Alg. 1 (batch)
template <int DIM>
__global__ void k_encode(int maxl, const uint32_t* __restrict__ xyz, const int32_t* __restrict__ level,
                         int64_t n, uint64_t* __restrict__ keys) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    uint32_t x[3] = {xyz[3 * i], xyz[3 * i + 1], xyz[3 * i + 2]};
    int l = level[i];
    // steps 2-4: coordinates at the finest resolution with the low (maxl-l) bits cleared
    // are the level-l path digits followed by the zero padding
    uint32_t clr = l >= maxl ? 0xFFFFFFFFu : ~((1u << (maxl - l)) - 1u);
    for (int a = 0; a < 3; ++a) x[a] &= clr;
    keys[i] = make_key(interleave<DIM>(x), l);
  }
}

template <int DIM>
__global__ void k_decode(const uint64_t* __restrict__ keys, int64_t n, int32_t* __restrict__ level,
                         uint32_t* __restrict__ xyz) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    uint64_t k = keys[i];
    uint32_t x[3];
    deinterleave<DIM>(key_morton(k), x);
    if (level) level[i] = key_level(k);
    if (xyz) {
      xyz[3 * i] = x[0];
      xyz[3 * i + 1] = x[1];
      xyz[3 * i + 2] = x[2];
    }
  }
}

// (leaves of a tree: anchors in GLOBAL finest-cell units, the cube's offset in the brick added)
template <int DIM>
__global__ void k_decode_n(Geo g, const uint64_t* __restrict__ keys, const DevScalars* __restrict__ s,
                           int32_t* __restrict__ level, uint32_t* __restrict__ xyz) {
  const int64_t n = s->n;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    uint64_t k = keys[i];
    uint32_t x[3];
    deinterleave<DIM>(key_morton(k) & g.total, x);
    if (g.ntrees > 1) {
      int tree = (int)(key_morton(k) >> g.tshift);
#pragma unroll
      for (int a = 0; a < DIM; ++a) {
        x[a] += (uint32_t)(tree % g.nroot[a]) << g.maxl;
        tree /= g.nroot[a];
      }
    }
    if (level) level[i] = key_level(k);
    if (xyz) {
      xyz[3 * i] = x[0];
      xyz[3 * i + 1] = x[1];
      xyz[3 * i + 2] = x[2];
    }
  }
}

// ------------------------------------------------------------------------ uniform build
// Leaf i of the uniform level-`base` tree has raw ID i (Morton order), key =
// (i << dim*(maxl-base)) << 5 | base (Alg. 1 with the padding of step 4).  On a brick the cubes follow
// one another: leaf i of cube r is entry r * 2^(dim*base) + i, and the same formula places r above the
// path bits.
template <int DIM>
__global__ void k_build_uniform(Geo g, uint64_t* __restrict__ keys, int* __restrict__ first, DevScalars* s) {
  const int64_t nb = (int64_t)g.ntrees << (DIM * g.base);
  const int pad = DIM * (g.maxl - g.base);
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < nb; i += (int64_t)gridDim.x * blockDim.x) {
    keys[i] = make_key((uint64_t)i << pad, g.base);
    index_write<DIM>(g, first, (uint64_t)i << pad, g.base, (int)i);
    if (i == 0) {
      first[g.nbuckets] = (int)nb;
      s->n = (int)nb;
    }
  }
}

template <int DIM>
__global__ void k_build_index(Geo g, const uint64_t* __restrict__ keys, const DevScalars* __restrict__ s,
                              int* __restrict__ first) {
  const int64_t n = s->n;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const uint64_t k = keys[i];
    index_write<DIM>(g, first, key_morton(k), key_level(k), (int)i);
    if (i == 0) first[g.nbuckets] = (int)n;
  }
}

// volume sum + level >= base check (lt_build_from_keys completeness)
template <int DIM>
__global__ void k_check_tiling(Geo g, const uint64_t* __restrict__ keys, DevScalars* s) {
  __shared__ unsigned long long sm[33];
  const int64_t n = s->n;
  unsigned long long v = 0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    uint64_t k = keys[i];
    int l = key_level(k);
    if (l < g.base || l > g.maxl) {
      set_status(&s->status, LT_ERR_INCOMPLETE);
    } else {
      v += 1ull << (DIM * (g.maxl - l));
      // anchor must be aligned to the cell width
      if (key_morton(k) & ((1ull << (DIM * (g.maxl - l))) - 1)) set_status(&s->status, LT_ERR_INCOMPLETE);
    }
  }
  v = block_sum(v, sm);
  if (threadIdx.x == 0 && v) atomicAdd(&s->volume, v);
}

// ------------------------------------------------------------------------ Alg. 6
// What happens to leaf i (readings B-1..B-4):
//   a complete sibling group (2^dim consecutive entries) whose members all
//   carry a coarsen flag and sit above the base level is replaced by its parent (emitted
//   in place of child 0, the others are dropped); otherwise a refine flag below max_level
//   replaces the leaf by its 2^dim children; otherwise the leaf is kept.
template <int DIM>
__device__ __forceinline__ int adapt_action(const Geo& g, const uint64_t* __restrict__ keys,
                                            const int8_t* __restrict__ flags, int64_t i, int64_t n,
                                            uint64_t key, int8_t fl) {
  constexpr int NC = Dim<DIM>::NC;
  const int l = key_level(key);
  if (fl < 0 && l > g.base) {
    const uint64_t m = key_morton(key);
    const int sh = DIM * (g.maxl - l);
    const int cid = (int)((m >> sh) & (uint64_t)(NC - 1));
    const int64_t g0 = i - cid;
    if (g0 >= 0 && g0 + NC <= n) {
      const uint64_t pm = m & ~((uint64_t)(NC - 1) << sh);
      // first and last sibling present as leaves => the NC-2 entries between them are
      // exactly the other siblings (completeness)
      if (keys[g0] == make_key(pm, l) && keys[g0 + NC - 1] == make_key(pm | ((uint64_t)(NC - 1) << sh), l)) {
        bool all = true;
#pragma unroll
        for (int c = 0; c < NC; ++c) all = all && (flags[g0 + c] < 0);
        if (all) return cid == 0 ? ACT_PARENT : ACT_DROP;
      }
    }
  }
  if (fl > 0 && l < g.maxl) return ACT_REFINE;
  return ACT_KEEP;
}
template <int DIM>
__device__ __forceinline__ int adapt_action(const Geo& g, const uint64_t* __restrict__ keys,
                                            const int8_t* __restrict__ flags, int64_t i, int64_t n,
                                            uint64_t key) {
  return adapt_action<DIM>(g, keys, flags, i, n, key, flags[i]);
}

constexpr int kGroup = kScanTiles * BT;  // leaves a block orders with one scan

// Block scan of the packed per-thread counts of one group: field q (kFieldBits bits, q < kScanTiles) =
// leaves that element (q, thread) puts out (<= 2^dim * BT = 2048 per tile), top field = frontier entries
// the thread appends.  The lane that forms the block total reserves the group's frontier slots with ONE
// global atomic between the two barriers of the scan (*fbase = first slot): an atomic per warp and
// tile on the single counter word serialised in L2 (277 k atomics per lt_adapt of 8.9 M leaves, about
// 0.85 cycles each: most of that kernel's time).  `sm` holds 34 words.  Ends with a barrier.
constexpr int kFieldBits = 12, kFrShift = 48;
constexpr unsigned long long kFieldMask = (1ull << kFieldBits) - 1;
__device__ __forceinline__ unsigned long long block_scan_reserve(unsigned long long v, unsigned long long* sm,
                                                                 unsigned long long* total, int* counter,
                                                                 int* fbase) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const unsigned long long inc = warp_incl_scan(v);
  if (lane == 31) sm[w] = inc;
  __syncthreads();
  if (w == 0) {
    const unsigned long long s = lane < nw ? sm[lane] : 0ull;
    const unsigned long long si = warp_incl_scan(s);
    sm[lane] = si - s;
    if (lane == 31) {
      sm[32] = si;
      const int nfr = (int)(si >> kFrShift);
      sm[33] = (counter != nullptr && nfr > 0) ? (unsigned long long)atomicAdd(counter, nfr) : 0ull;
    }
  }
  __syncthreads();
  const unsigned long long res = sm[w] + inc - v;
  *total = sm[32];
  *fbase = (int)sm[33];
  __syncthreads();
  return res;
}

// pass 1: per-chunk output counts.  sums[b] = (kept << 32) | count_B   (see lt_adapt)
template <int DIM>
__global__ void __launch_bounds__(BT) k_adapt_count(Geo g, const uint64_t* __restrict__ keys,
                                                    const int8_t* __restrict__ flags, DevScalars* s,
                                                    unsigned long long* __restrict__ sums) {
  constexpr int NC = Dim<DIM>::NC;
  __shared__ unsigned long long sm[33];
  const int64_t n = s->n;
  // pass 2 overwrites s->n with the new count while its later blocks are still starting: they read the
  // count of the tree they work on from this snapshot
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    s->n_in = (int)n;
    s->nfront[0] = 0;  // pass 2 appends lt_balance's first frontier
  }
  int64_t lo, hi;
  block_chunk(n, gridDim.x, blockIdx.x, BT, &lo, &hi);
  unsigned long long acc = 0;
  for (int64_t i = lo + threadIdx.x; i < hi; i += BT) {
    int act = adapt_action<DIM>(g, keys, flags, i, n, keys[i]);
    unsigned long long c = act == ACT_REFINE ? NC : (act == ACT_DROP ? 0 : 1);
    unsigned long long kept = (act == ACT_KEEP || act == ACT_REFINE) ? 1 : 0;
    acc += c | (kept << 32);
  }
  acc = block_sum(acc, sm);
  if (threadIdx.x == 0) sums[blockIdx.x] = acc;
}

// pass 2 (path B, ordered expansion): children / parent are written in place of the
// source entries, which keeps the array sorted because a leaf's children occupy exactly
// its Morton interval (reading B-5).  Also rebuilds the bucket index.
template <int DIM>
__global__ void __launch_bounds__(BT) k_adapt_scatter(Geo g, const uint64_t* __restrict__ keys,
                                                      const int8_t* __restrict__ flags, DevScalars* s,
                                                      const unsigned long long* __restrict__ sums,
                                                      uint64_t* __restrict__ out, int* __restrict__ first_out,
                                                      int64_t cap, uint64_t* __restrict__ fkey,
                                                      uint8_t* __restrict__ ftag, int64_t fcap) {
  // fkey != nullptr: the tree entering lt_adapt was 2:1 balanced, so only the leaves created here
  // can be part of a violation; they are listed as the frontier of lt_balance's first sweep
  // (s->nfront[0] entries, any order): a refined leaf as a GROUP entry (its own key), a merged
  // parent as a SELF entry (its position)
  constexpr int NC = Dim<DIM>::NC;
  __shared__ unsigned long long sm[34];
  const int64_t n = s->n_in;  // (not s->n: block 0 of this kernel overwrites it, see k_adapt_count)
  int64_t lo, hi;
  block_chunk(n, gridDim.x, blockIdx.x, BT, &lo, &hi);
  unsigned long long before, total;
  chunk_offsets(sums, gridDim.x, blockIdx.x, sm, &before, &total);
  const int64_t n_out = (int64_t)(total & 0xffffffffull);
  if (n_out > cap) {
    if (threadIdx.x == 0 && blockIdx.x == 0) set_status(&s->status, LT_ERR_CAPACITY);
    return;
  }
  int64_t run = (int64_t)(before & 0xffffffffull);
  int* const fcounter = fkey != nullptr ? &s->nfront[0] : nullptr;
  // kScanTiles tiles of BT leaves share one block scan (counts packed in 12-bit fields)
  for (int64_t t0 = lo; t0 < hi; t0 += kGroup) {
    uint64_t keyq[kScanTiles];
    int actq[kScanTiles];
    unsigned long long packed = 0;
#pragma unroll
    for (int q = 0; q < kScanTiles; ++q) {
      const int64_t i = t0 + q * BT + threadIdx.x;
      actq[q] = ACT_DROP;
      keyq[q] = 0;
      if (i < hi) {
        keyq[q] = keys[i];
        actq[q] = adapt_action<DIM>(g, keys, flags, i, n, keyq[q]);
      }
      packed |= (unsigned long long)(actq[q] == ACT_REFINE ? NC : (actq[q] == ACT_DROP ? 0 : 1)) << (kFieldBits * q);
      // a refined leaf (GROUP entry) and a merged parent (SELF entry) go to lt_balance's first frontier
      if (fcounter != nullptr && (actq[q] == ACT_REFINE || actq[q] == ACT_PARENT)) packed += 1ull << kFrShift;
    }
    unsigned long long tile_total;
    int fbase;
    const unsigned long long ex = block_scan_reserve(packed, sm, &tile_total, fcounter, &fbase);
    int64_t fat = (int64_t)fbase + (int64_t)(ex >> kFrShift);
#pragma unroll
    for (int q = 0; q < kScanTiles; ++q) {
      const int act = actq[q];
      const uint64_t key = keyq[q];
      const int64_t pos = run + (int64_t)((ex >> (kFieldBits * q)) & kFieldMask);
      run += (int64_t)((tile_total >> (kFieldBits * q)) & kFieldMask);
      if (fcounter != nullptr && (act == ACT_REFINE || act == ACT_PARENT)) {
        // (kFrGroup = 2: its own key, kFrSelf = 3: its position; any order.  A list that does not fit
        // makes lt_balance sweep in full)
        if (fat < fcap) {
          fkey[fat] = act == ACT_REFINE ? key : (uint64_t)pos;
          ftag[fat] = act == ACT_REFINE ? 2 : 3;
        }
        ++fat;
      }
      if (act == ACT_DROP) continue;
      LT_DASSERT(pos >= 0 && pos + (act == ACT_REFINE ? NC : 1) <= n_out);
      const int l = key_level(key);
      const uint64_t m = key_morton(key);
      if (act == ACT_KEEP) {
        out[pos] = key;
        index_write<DIM>(g, first_out, m, l, (int)pos);
      } else if (act == ACT_PARENT) {
        out[pos] = make_key(m, l - 1);  // child 0 has the parent's anchor
        index_write<DIM>(g, first_out, m, l - 1, (int)pos);
      } else {
        const int sh = DIM * (g.maxl - l - 1);
#pragma unroll
        for (int k = 0; k < NC; ++k) {
          const uint64_t mc = m | ((uint64_t)k << sh);  // reading A-6
          out[pos + k] = make_key(mc, l + 1);
          index_write<DIM>(g, first_out, mc, l + 1, (int)(pos + k));
        }
      }
    }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    first_out[g.nbuckets] = (int)n_out;
    s->n = (int)n_out;
  }
}

// pass 2 (path A, as the paper does it): kept entries stay (a refined octant is removed
// later by the linearisation), children and parents are appended through
// an atomic cursor in no particular order; sort + linearise follow (Alg. 6 step 6).
template <int DIM>
__global__ void __launch_bounds__(BT) k_adapt_append(Geo g, const uint64_t* __restrict__ keys,
                                                     const int8_t* __restrict__ flags, DevScalars* s,
                                                     const unsigned long long* __restrict__ sums,
                                                     uint64_t* __restrict__ out, int64_t cap) {
  constexpr int NC = Dim<DIM>::NC;
  __shared__ unsigned long long sm[33];
  const int64_t n = s->n_in;  // (not s->n: block 0 of this kernel overwrites it, see k_adapt_count)
  unsigned long long before, total;
  chunk_offsets(sums, gridDim.x, blockIdx.x, sm, &before, &total);
  const int64_t n_kept = (int64_t)(total >> 32);
  if (n_kept + (int64_t)(total & 0xffffffffull) > cap) {
    if (threadIdx.x == 0 && blockIdx.x == 0) set_status(&s->status, LT_ERR_CAPACITY);
    return;
  }
  int64_t lo, hi;
  block_chunk(n, gridDim.x, blockIdx.x, BT, &lo, &hi);
  int64_t run = (int64_t)(before >> 32);
  for (int64_t t0 = lo; t0 < hi; t0 += BT) {
    const int64_t i = t0 + threadIdx.x;
    int act = ACT_DROP;
    uint64_t key = 0;
    if (i < hi) {
      key = keys[i];
      act = adapt_action<DIM>(g, keys, flags, i, n, key);
    }
    int kept = (act == ACT_KEEP || act == ACT_REFINE) ? 1 : 0;
    unsigned long long tile_total;
    unsigned long long ex = block_excl_scan<unsigned long long>((unsigned long long)kept, sm, &tile_total);
    int64_t pos = run + (int64_t)ex;
    run += (int64_t)tile_total;
    const int l = key_level(key);
    const uint64_t m = key_morton(key);
    if (kept) out[pos] = key;
    if (act == ACT_REFINE) {
      int64_t at = n_kept + atomicAdd(&s->aux, NC);
      const int sh = DIM * (g.maxl - l - 1);
      for (int k = 0; k < NC; ++k) out[at + k] = make_key(m | ((uint64_t)k << sh), l + 1);
    } else if (act == ACT_PARENT) {
      int64_t at = n_kept + atomicAdd(&s->aux, 1);
      out[at] = make_key(m, l - 1);
    }
  }
}

// ------------------------------------------------------------------------ 2:1 balance
// PAPER.md:130-161 (Alg. 4), face balance (reading C-1), Jacobi ripple (readings C-2,
// C-3): a sweep examines leaves against the tree as it stood at the start of the sweep;
// every face neighbour found >= 2 levels coarser is marked; marked leaves split once.
// All sweeps run inside this one cooperative kernel.
//
// After the first sweep only a FRONTIER is examined.  Its entries are keyed, so that they stay
// valid while the leaf array is rewritten by the splits:
//   GROUP  the key K (level l) of a leaf that was split (by lt_adapt or by the previous sweep): its
//          2^dim children are new leaves.  All exterior faces of the children lie on the 2*dim faces of
//          K and a child sees a neighbour >= 2 levels coarser exactly when the leaf across that face of
//          K is coarser than K, so ONE search per face of K (level < l: mark it) replaces the 2^(dim-1)
//          searches of the children on that face -- 6 searches per split leaf instead of 24 in 3-D.
//          If that leaf is even coarser than l - 1 it will still be too coarse after its split: the
//          entry is flagged and re-examined in the next sweep.
//   LEAF   the key of a single leaf that saw a neighbour >= 3 levels coarser in a full sweep.
//   SELF   (first sweep after lt_adapt only) the POSITION of a parent created by a coarsening: it is
//          too coarse iff a level-(l+1) cell of a neighbouring level-l cell is subdivided.
// DESIGN.md section 5 proves that frontier sweeps mark the same set as full sweeps.
struct BalanceArgs {
  Geo g;
  uint64_t* keys[2];
  int* first[2];
  uint8_t* mark;
  uint64_t* fkey[2];   // frontier ping-pong: entry keys (SELF: position) ...
  uint8_t* ftag[2];    // ... and tags: kFrLeaf / kFrGroup / kFrSelf | kFrAgain
  int64_t fcap;        // entries per frontier buffer
  int* cmarks[2];      // [G] leaves marked per chunk, counted when the mark is set (ping-pong per sweep)
  DevScalars* s;
  int64_t cap;
  int full_sweeps;
  int front0;  // 1: frontier 0 holds lt_adapt's list (s->nfront[0] entries) for sweep 1
  // neighbour directions of a LEAF examination (reading C-9): 2 bits per axis, 0 = no move,
  // 1 = move across the leaf's parent-EXTERIOR side on that axis, 2 = across the interior side
  int ndirs;
  uint8_t dirs[20];
  // neighbour directions of a GROUP examination: 2 bits per axis, 0 = no move, 1 = minus, 2 = plus
  int ngdirs;
  uint8_t gdirs[26];
  // Alg. 7 in the tail of the kernel (do_map): T_old -> the balanced tree
  int do_map, n_old;
  const uint64_t* keys_old;
  const int* first_old;
  int32_t* map_src;
  uint8_t* map_kind;
};

enum { kFrLeaf = 1, kFrGroup = 2, kFrSelf = 3, kFrAgain = 0x80 };

// mark leaf j for splitting; the first thread to set the mark counts it in j's chunk
__device__ __forceinline__ void mark_split(uint8_t* mark, int* cmarks, int per, int j) {
  const unsigned bit = 1u << (8 * (j & 3));
  const unsigned old = atomicOr((unsigned*)(mark + (j & ~3)), bit);
  if (!(old & bit)) atomicAdd(&cmarks[j / per], 1);
}

// The same-level cell reached from (m, l) by the absolute moves in `code` (2 bits per axis: 1 = minus,
// 2 = plus), chaining the one-axis step; false if it leaves a non-periodic domain.
template <int DIM>
__device__ __forceinline__ bool move_cell(const Geo& g, uint64_t m, int l, int code, uint64_t* out) {
  uint64_t mn = m;
#pragma unroll
  for (int a = 0; a < DIM; ++a) {
    const int c = (code >> (2 * a)) & 3;
    if (c) {
      uint64_t nx;
      if (!face_neighbour<DIM>(g, mn, l, 2 * a + (c - 1), &nx)) return false;
      mn = nx;
    }
  }
  *out = mn;
  return true;
}

// Face balance examines only the DIM faces of a leaf that are exterior to its parent: an
// interior face looks at a sibling's cell, which is tiled by leaves at least as fine as the
// leaf itself (the parent is subdivided), so it can never meet a coarser neighbour.  The
// exterior side on axis a is the minus side if bit a of the child id is 0, the plus side
// otherwise.  Strong balance (neighbours across edges, optionally corners) adds
// the directions that move on two / three axes; a direction whose moves are ALL interior lands
// inside the parent and is skipped for the same reason, so 3 + 9 (+ 7) directions per leaf are
// examined in 3-D.  Returns 0, 1 (the neighbour was marked) or 2 (marked, and it is >= 3 levels
// coarser: the leaf has to be examined again).
template <int DIM>
__device__ __forceinline__ int examine_leaf(const Geo& g, const uint64_t* __restrict__ keys,
                                            const int* __restrict__ first, uint8_t* mark, int* cmarks, int per,
                                            uint64_t key, int code) {
  const int l = key_level(key);
  if (l < g.base + 2) return 0;  // no leaf is coarser than the base level
  const uint64_t m = key_morton(key);
  const int cid = child_id<DIM>(g, m, l);
  int abs_code = 0;
#pragma unroll
  for (int a = 0; a < DIM; ++a) {
    const int c = (code >> (2 * a)) & 3;
    const int bit = (cid >> a) & 1;
    if (c) abs_code |= (1 + (c == 1 ? bit : (bit ^ 1))) << (2 * a);
  }
  uint64_t mn;
  if (!move_cell<DIM>(g, m, l, abs_code, &mn)) return 0;
  const int j = locate(g, keys, first, mn);
  const int lj = key_level(keys[j]);
  if (lj >= l - 1) return 0;
  LT_DASSERT(lj >= g.base);
  mark_split(mark, cmarks, per, j);
  return lj < l - 2 ? 2 : 1;
}

// GROUP entry: the children of K = (m, l) are leaves of level l + 1 (or finer); the leaf across K in
// direction `code` is too coarse for them iff its level is < l.
template <int DIM>
__device__ __forceinline__ int examine_group(const Geo& g, const uint64_t* __restrict__ keys,
                                             const int* __restrict__ first, uint8_t* mark, int* cmarks, int per,
                                             uint64_t key, int code) {
  const int l = key_level(key);
  if (l < g.base + 1) return 0;
  uint64_t mn;
  if (!move_cell<DIM>(g, key_morton(key), l, code, &mn)) return 0;
  const int j = locate(g, keys, first, mn);
  const int lj = key_level(keys[j]);
  if (lj >= l) return 0;
  mark_split(mark, cmarks, per, j);
  return lj < l - 1 ? 2 : 1;
}

// A parent created by lt_adapt (level l, position i) is too coarse iff, in one of the neighbour directions
// of the balance (`code`: 2 bits per axis, 1 = minus, 2 = plus; faces, and edges / corners for the strong
// balance), a level-(l+1) cell of the neighbouring level-l cell that touches the parent is itself
// subdivided (its leaves are >= 2 levels finer).  Those cells have, on every moved axis, the child bit of
// the side facing the parent and any bit on the other axes: 2^(dim - moves) searches.  Checked from the
// parent's side; marks the parent itself.
template <int DIM>
__device__ __forceinline__ void examine_self(const Geo& g, const uint64_t* __restrict__ keys,
                                             const int* __restrict__ first, uint8_t* mark, int* cmarks, int per,
                                             int i, int code) {
  const uint64_t key = keys[i];
  const int l = key_level(key);
  if (l + 2 > g.maxl) return;
  uint64_t mn;
  if (!move_cell<DIM>(g, key_morton(key), l, code, &mn)) return;
  int facing = 0, nfree = 0;
#pragma unroll
  for (int a = 0; a < DIM; ++a) {
    const int c = (code >> (2 * a)) & 3;
    if (c == 1) facing |= 1 << a;  // moved to the minus side: the neighbour's plus-side children touch
    nfree += c == 0;
  }
  bool hit = false;
#pragma unroll
  for (int sidx = 0; sidx < (1 << (DIM - 1)); ++sidx) {
    if (sidx >= (1 << nfree)) break;
    int c = facing, bit = 0;
#pragma unroll
    for (int b = 0; b < DIM; ++b) {
      if ((code >> (2 * b)) & 3) continue;
      c |= ((sidx >> bit) & 1) << b;
      ++bit;
    }
    const int j = locate(g, keys, first, mn | ((uint64_t)c << (DIM * (g.maxl - l - 1))));
    hit = hit || key_level(keys[j]) >= l + 2;
  }
  if (hit) mark_split(mark, cmarks, per, i);
}

// (whole warp) append the entries of the lanes with `pred` to a frontier; false if it is full
__device__ __forceinline__ bool frontier_push(bool pred, uint64_t key, int tag, uint64_t* fkey, uint8_t* ftag,
                                              int* counter, int64_t fcap) {
  const unsigned m = __ballot_sync(0xffffffffu, pred);
  if (m == 0) return true;
  const int lane = threadIdx.x & 31;
  int base = 0;
  if (lane == __ffs(m) - 1) base = atomicAdd(counter, __popc(m));
  base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
  const int64_t at = (int64_t)base + __popc(m & ((1u << lane) - 1));
  const bool fits = (int64_t)base + __popc(m) <= fcap;
  LT_DASSERT(base >= 0 && at >= 0);
  if (pred && fits) {
    fkey[at] = key;
    ftag[at] = (uint8_t)tag;
  }
  return fits;
}

// The split pass of one sweep for the chunk [lo, hi) of a block: marked leaves are replaced by their
// children (order-preserving), the bucket index is rebuilt and the next frontier is appended to.  Kept
// out of line so that its registers (kScanTiles keys and marks per thread) do not weigh on the search
// loops of the examination phases.  Returns false if the frontier buffer overflowed.
template <int DIM>
__device__ __noinline__ bool split_pass(const Geo& g, const uint64_t* __restrict__ keys, uint8_t* mark, int64_t lo,
                                        int64_t hi, int64_t run, uint64_t* __restrict__ out,
                                        int* __restrict__ first_out, bool emit, uint64_t* fk_out, uint8_t* ft_out,
                                        int* fcount, int64_t fcap, unsigned long long* sm, int64_t n_new) {
  constexpr int NC = Dim<DIM>::NC;
  bool fits = true;
  (void)n_new;
  // kScanTiles tiles of BT leaves share one block scan: the counts (<= NC * BT = 2^11 per tile) are
  // packed in 12-bit fields, the frontier entries of the group in the top field (block_scan_reserve).
  // Requesting the NEXT group's loads into registers before the barriers was tried: slower, 0.34 ->
  // 0.40-0.43 ms for the three splitting sweeps of config-5 cycle 3, because of the registers it takes;
  // so was a cp.async prefetch of the next group into shared memory, which takes no registers (0.52 ->
  // 0.54 ms, and 0.37 -> 0.38 ms in k_adapt_scatter): the pass does not wait for its loads.
  for (int64_t t0 = lo; t0 < hi; t0 += kGroup) {
    uint64_t key[kScanTiles];
    unsigned mk[kScanTiles];
    unsigned long long packed = 0;
#pragma unroll
    for (int q = 0; q < kScanTiles; ++q) {
      const int64_t i = t0 + q * BT + threadIdx.x;
      key[q] = 0;
      mk[q] = 0;
      if (i < hi) {
        key[q] = keys[i];
        mk[q] = mark[i];
      }
    }
#pragma unroll
    for (int q = 0; q < kScanTiles; ++q) {
      const int64_t i = t0 + q * BT + threadIdx.x;
      if (i < hi) {
        if (mk[q]) mark[i] = 0;
        packed |= (unsigned long long)((mk[q] & 1) ? NC : 1) << (kFieldBits * q);
        // a split leaf becomes a GROUP entry; an unsplit leaf that saw a neighbour >= 3 levels coarser
        // (full sweep) a LEAF entry
        if (emit && (mk[q] & 3)) packed += 1ull << kFrShift;
      }
    }
    unsigned long long tile_total;
    int fbase;
    const unsigned long long ex = block_scan_reserve(packed, sm, &tile_total, emit ? fcount : nullptr, &fbase);
    int64_t fat = (int64_t)fbase + (int64_t)(ex >> kFrShift);
    fits = fits && (int64_t)fbase + (int64_t)(tile_total >> kFrShift) <= fcap;
#pragma unroll
    for (int q = 0; q < kScanTiles; ++q) {
      const int64_t i = t0 + q * BT + threadIdx.x;
      const int64_t pos = run + (int64_t)((ex >> (kFieldBits * q)) & kFieldMask);
      run += (int64_t)((tile_total >> (kFieldBits * q)) & kFieldMask);
      if (i >= hi) continue;
      if (emit && (mk[q] & 3)) {
        LT_DASSERT(fat >= 0);
        if (fat < fcap) {
          fk_out[fat] = key[q];
          ft_out[fat] = (uint8_t)((mk[q] & 1) ? kFrGroup : kFrLeaf);
        }
        ++fat;
      }
      LT_DASSERT(pos >= 0 && pos + ((mk[q] & 1) ? NC : 1) <= n_new);
      const int l = key_level(key[q]);
      const uint64_t m = key_morton(key[q]);
      LT_DASSERT(!(mk[q] & 1) || l < g.maxl);  // a leaf at the finest level is never too coarse
      if (mk[q] & 1) {
        const int sh = DIM * (g.maxl - l - 1);
#pragma unroll
        for (int k = 0; k < NC; ++k) {
          const uint64_t mc = m | ((uint64_t)k << sh);
          out[pos + k] = make_key(mc, l + 1);
          index_write<DIM>(g, first_out, mc, l + 1, (int)(pos + k));
        }
      } else {
        out[pos] = key[q];
        index_write<DIM>(g, first_out, m, l, (int)pos);
      }
    }
  }
  return fits;
}

__device__ __forceinline__ unsigned long long global_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

template <int DIM>
__global__ void __launch_bounds__(BT, 4) k_balance(BalanceArgs a) {
  constexpr int NC = Dim<DIM>::NC;
  __shared__ unsigned long long sm[34];
  __shared__ uint8_t s_dirs[20], s_gdirs[26];
  cg::grid_group grid = cg::this_grid();
  const Geo g = a.g;
  if (threadIdx.x < 20) s_dirs[threadIdx.x] = a.dirs[threadIdx.x];
  if (threadIdx.x < 26) s_gdirs[threadIdx.x] = a.gdirs[threadIdx.x];
  __syncthreads();
  const int G = gridDim.x;
  const int64_t gtid = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  const int64_t gsize = (int64_t)G * blockDim.x;
  const int lane = threadIdx.x & 31;
  int64_t n = a.s->n;
  int par = 0, iters = 0, fpar = 0, sweep = 0;
  int64_t nfront = a.front0 ? (int64_t)a.s->nfront[0] : -1;  // -1: full sweep
  if (nfront > a.fcap) nfront = -1;                           // lt_adapt's list did not fit
  int64_t splits = 0;
  int err = 0;
  if (gtid == 0) a.s->map_bad = 0;  // (set again only by the Alg. 7 tail, many barriers later)
  // thread (0, 0) leaves every grid-wide barrier after all blocks have arrived, so its clock
  // readings bound the phases of the whole grid (lt_balance_phases)
  unsigned long long ns[4] = {0, 0, 0, 0}, t_prev = gtid == 0 ? global_ns() : 0;
  auto lap = [&](int phase) {
    if (gtid == 0) {
      const unsigned long long now = global_ns();
      ns[phase] += now - t_prev;
      t_prev = now;
    }
  };
  for (;; ++sweep) {
    const uint64_t* keys = a.keys[par];
    const int* first = a.first[par];
    int* cm = a.cmarks[sweep & 1];
    // chunk b of the leaf array = [b * per, (b + 1) * per) (block_chunk)
    int64_t per64 = (n + G - 1) / G;
    per64 = (per64 + BT - 1) / BT * BT;
    const int per = (int)(per64 > 0 ? per64 : BT);
    // the other halves of the ping-pong state are reset for the next sweep (nobody reads them now)
    if (threadIdx.x == 0) a.cmarks[(sweep + 1) & 1][blockIdx.x] = 0;
    if (gtid == 0) {
      a.s->nfront[fpar ^ 1] = 0;
      a.s->fr_overflow = 0;
    }
    // ---- sweep
    if (nfront < 0) {
      const int nd = a.ndirs;
      for (int64_t sidx = gtid; sidx < n * nd; sidx += gsize) {
        const int i = (int)(sidx / nd);
        const int r = examine_leaf<DIM>(g, keys, first, a.mark, cm, per, keys[i], s_dirs[sidx - (int64_t)i * nd]);
        if (r == 2) atomicOr((unsigned*)(a.mark + (i & ~3)), 2u << (8 * (i & 3)));
      }
    } else {
      const uint64_t* fk = a.fkey[fpar];
      uint8_t* ft = a.ftag[fpar];
      const int nd = a.ngdirs;  // >= ndirs and >= 2 * DIM
      for (int64_t sidx = gtid; sidx < nfront * nd; sidx += gsize) {
        const int64_t e = sidx / nd;
        const int d = (int)(sidx - e * nd);
        const int tag = ft[e] & 0x7f;
        const uint64_t key = fk[e];
        int r = 0;
        if (tag == kFrGroup) r = examine_group<DIM>(g, keys, first, a.mark, cm, per, key, s_gdirs[d]);
        else if (tag == kFrLeaf) r = d < a.ndirs ? examine_leaf<DIM>(g, keys, first, a.mark, cm, per, key, s_dirs[d]) : 0;
        else examine_self<DIM>(g, keys, first, a.mark, cm, per, (int)key, s_gdirs[d]);  // only in sweep 1
        if (r == 2) atomicOr((unsigned*)(ft + (e & ~3)), (unsigned)kFrAgain << (8 * (e & 3)));
      }
    }
    grid.sync();
    lap(0);
    // ---- leaves out per chunk = its length + (NC - 1) * its marks
    int64_t lo, hi;
    block_chunk(n, G, blockIdx.x, BT, &lo, &hi);
    unsigned long long mine = 0, all = 0;
    for (int i = threadIdx.x; i < G; i += BT) {
      int64_t l2, h2;
      block_chunk(n, G, i, BT, &l2, &h2);
      const unsigned long long c = (unsigned long long)(h2 - l2) + (unsigned long long)(NC - 1) * (unsigned)cm[i];
      all += c;
      if (i < (int)blockIdx.x) mine += c;
    }
    const int64_t before = (int64_t)block_sum(mine, sm);
    const int64_t n_new = (int64_t)block_sum(all, sm);
    lap(1);
    if (n_new == n) break;  // no leaf was marked: balanced
    if (n_new > a.cap) {
      err = LT_ERR_CAPACITY;
      break;
    }
    // ---- split marked leaves (order-preserving), rebuild the index, emit the next frontier
    uint64_t* out = a.keys[par ^ 1];
    int* first_out = a.first[par ^ 1];
    uint64_t* fk_out = a.fkey[fpar ^ 1];
    uint8_t* ft_out = a.ftag[fpar ^ 1];
    int* fcount = &a.s->nfront[fpar ^ 1];
    const bool emit = !a.full_sweeps;
    const int64_t run = before;
    bool fits = split_pass<DIM>(g, keys, a.mark, lo, hi, run, out, first_out, emit, fk_out, ft_out, fcount, a.fcap, sm, n_new);
    // entries flagged for another examination move on to the next frontier
    if (emit && nfront >= 0) {
      const uint64_t* fk = a.fkey[fpar];
      const uint8_t* ft = a.ftag[fpar];
      for (int64_t e0 = gtid - lane; e0 < nfront; e0 += gsize) {
        const int64_t e = e0 + lane;
        const int tag = e < nfront ? ft[e] : 0;
        fits = frontier_push((tag & kFrAgain) != 0, e < nfront ? fk[e] : 0, tag & 0x7f, fk_out, ft_out, fcount,
                             a.fcap) && fits;
      }
    }
    if (!fits) a.s->fr_overflow = 1;
    if (blockIdx.x == 0 && threadIdx.x == 0) first_out[g.nbuckets] = (int)n_new;
    splits += (n_new - n) / (NC - 1);
    n = n_new;
    par ^= 1;
    fpar ^= 1;
    ++iters;
    grid.sync();
    lap(2);
    // (a frontier that overflowed its buffer -- not reachable with fcap > cap * 8 / 7 -- falls back to a
    // full sweep, which needs no list)
    nfront = (a.full_sweeps || a.s->fr_overflow) ? -1 : (int64_t)a.s->nfront[fpar];
  }
  // ---- Alg. 7: T_old -> the balanced tree, in new-leaf order.  A new leaf more
  // than one level from T_old only raises map_bad here: lt_transfer then runs the checked k_map,
  // which reports LT_ERR_MAPPING where the header says it is reported.
  // The map is monotone (both arrays ascend), so the old leaves that a tile of consecutive new leaves
  // maps to are one contiguous range: its two ends are located by the bucketed search (all tiles of a
  // batch side by side), the range is copied to shared memory and every new leaf searches there -- one
  // dependent chain of global probes per TILE instead of one per leaf.  A range that does not fit (a
  // tile made of merged parents only can span 2^dim old leaves per new one) takes the per-leaf search.
  if (a.do_map && !err) {
    const uint64_t* keys = a.keys[par];
    bool bad = false;
    constexpr int kWin = 2 * kGroup;  // old keys per window
    __shared__ uint64_t win[kWin];
    __shared__ int s_b[BT + 1];
    int64_t lo, hi;
    block_chunk(n, G, blockIdx.x, BT, &lo, &hi);
    for (int64_t b0 = lo; b0 < hi; b0 += (int64_t)BT * kGroup) {
      const int64_t bh = b0 + (int64_t)BT * kGroup < hi ? b0 + (int64_t)BT * kGroup : hi;
      const int nt = (int)((bh - b0 + kGroup - 1) / kGroup);
      __syncthreads();  // (s_b and the window of the previous batch are no longer read)
      for (int k = threadIdx.x; k <= nt; k += BT) {
        const int64_t j = b0 + (int64_t)k * kGroup < bh ? b0 + (int64_t)k * kGroup : bh - 1;
        s_b[k] = locate(g, a.keys_old, a.first_old, key_morton(keys[j]));
      }
      __syncthreads();
      for (int k = 0; k < nt; ++k) {
        const int64_t t0 = b0 + (int64_t)k * kGroup;
        const int o0 = s_b[k];
        int w = s_b[k + 1] + NC - o0;  // (+ NC: the last sibling of a merged group is looked at)
        if (w > a.n_old - o0) w = a.n_old - o0;
        const bool in_smem = w <= kWin;
        if (in_smem)
          for (int x = threadIdx.x; x < w; x += BT) win[x] = a.keys_old[o0 + x];
        __syncthreads();
#pragma unroll
        for (int q = 0; q < kScanTiles; ++q) {
          const int64_t j = t0 + q * BT + threadIdx.x;
          if (j >= bh) continue;
          const uint64_t key = keys[j];
          int o, kd;
          if (!in_smem) {
            bad = !map_entry<DIM>(g, key, a.keys_old, a.first_old, a.n_old, &o, &kd) || bad;
          } else {
            // map_entry on the window: last old key with morton <= the new leaf's (Eq. 7)
            const int l = key_level(key);
            const uint64_t m = key_morton(key);
            const uint64_t bound = (m << kLevelBits) | kLevelMask;
            int a0 = 0, a1 = w;
            while (a1 - a0 > 1) {
              const int mid = (a0 + a1) >> 1;
              if (win[mid] <= bound) a0 = mid; else a1 = mid;
            }
            LT_DASSERT(win[a0] <= bound);
            const int lv = key_level(win[a0]);
            kd = 0;
            if (lv == l - 1) {
              kd = 1 | (child_id<DIM>(g, m, l) << 4);
            } else if (lv == l + 1) {
              const int sh = DIM * (g.maxl - l - 1);
              const uint64_t klast = make_key(m | ((uint64_t)(NC - 1) << sh), l + 1);
              if (a0 + NC - 1 >= w || win[a0 + NC - 1] != klast) bad = true;
              kd = 2;
            } else if (lv != l) {
              bad = true;
            }
            o = o0 + a0;
          }
          a.map_src[j] = o;
          a.map_kind[j] = (uint8_t)kd;
        }
        __syncthreads();
      }
    }
    if (bad) a.s->map_bad = 1;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    lap(3);  // (this block's share of the tail: the blocks run it side by side)
    for (int k = 0; k < 4; ++k) a.s->bal_ns[k] = ns[k];
    a.s->n = (int)n;
    a.s->iters = iters;
    a.s->parity = par;
    a.s->splits = (int)splits;
    if (err) set_status(&a.s->status, err);
  }
}

// ------------------------------------------------------------------------ launchers
int grid_for(const Tree* t, int blocks_per_sm) {
  int G = t->num_sms * blocks_per_sm;
  return G > kMaxGrid ? kMaxGrid : G;
}

#define LT_DISPATCH_DIM(t, expr2, expr3) \
  do {                                   \
    if ((t)->g.dim == 2) { expr2; } else { expr3; } \
  } while (0)

int launch_build_uniform(Tree* t) {
  int G = grid_for(t, 4);
  LT_DISPATCH_DIM(t, (k_build_uniform<2><<<G, BT, 0, t->stream>>>(t->g, t->keys[t->cur], t->first[t->cur], t->d_s)),
                  (k_build_uniform<3><<<G, BT, 0, t->stream>>>(t->g, t->keys[t->cur], t->first[t->cur], t->d_s)));
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

int launch_build_index(Tree* t, int buf) {
  int G = grid_for(t, 4);
  LT_DISPATCH_DIM(t, (k_build_index<2><<<G, BT, 0, t->stream>>>(t->g, t->keys[buf], t->d_s, t->first[buf])),
                  (k_build_index<3><<<G, BT, 0, t->stream>>>(t->g, t->keys[buf], t->d_s, t->first[buf])));
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

int launch_check_tiling(Tree* t) {
  int G = grid_for(t, 4);
  LT_DISPATCH_DIM(t, (k_check_tiling<2><<<G, BT, 0, t->stream>>>(t->g, t->keys[t->cur], t->d_s)),
                  (k_check_tiling<3><<<G, BT, 0, t->stream>>>(t->g, t->keys[t->cur], t->d_s)));
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

int launch_adapt_count(Tree* t, const int8_t* d_flags, int G) {
  LT_DISPATCH_DIM(t, (k_adapt_count<2><<<G, BT, 0, t->stream>>>(t->g, t->keys[t->cur], d_flags, t->d_s, t->d_sums)),
                  (k_adapt_count<3><<<G, BT, 0, t->stream>>>(t->g, t->keys[t->cur], d_flags, t->d_s, t->d_sums)));
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

int launch_adapt_scatter(Tree* t, const int8_t* d_flags, int G, int path_a, int emit_front) {
  uint64_t* fkey = (emit_front && !path_a) ? t->fkey[0] : nullptr;
  uint8_t* ftag = t->ftag[0];
  const int64_t fcap = t->fcap;
  if (path_a) {
    LT_DISPATCH_DIM(t,
                    (k_adapt_append<2><<<G, BT, 0, t->stream>>>(t->g, t->keys[t->cur], d_flags, t->d_s, t->d_sums,
                                                                t->keys[t->tmp], t->cap)),
                    (k_adapt_append<3><<<G, BT, 0, t->stream>>>(t->g, t->keys[t->cur], d_flags, t->d_s, t->d_sums,
                                                                t->keys[t->tmp], t->cap)));
  } else {
    LT_DISPATCH_DIM(t,
                    (k_adapt_scatter<2><<<G, BT, 0, t->stream>>>(t->g, t->keys[t->cur], d_flags, t->d_s, t->d_sums,
                                                                 t->keys[t->tmp], t->first[t->tmp], t->cap, fkey, ftag, fcap)),
                    (k_adapt_scatter<3><<<G, BT, 0, t->stream>>>(t->g, t->keys[t->cur], d_flags, t->d_s, t->d_sums,
                                                                 t->keys[t->tmp], t->first[t->tmp], t->cap, fkey, ftag, fcap)));
  }
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

int launch_balance(Tree* t, int64_t cap_told, int use_front) {
  BalanceArgs a;
  a.g = t->g;
  a.keys[0] = t->keys[t->cur];
  a.keys[1] = t->keys[t->tmp];
  a.first[0] = t->first[t->cur];
  a.first[1] = t->first[t->tmp];
  a.mark = t->mark;
  for (int b = 0; b < 2; ++b) {
    a.fkey[b] = t->fkey[b];
    a.ftag[b] = t->ftag[b];
    a.cmarks[b] = t->d_cmarks + b * kMaxGrid;
  }
  a.fcap = t->fcap;
  a.s = t->d_s;
  a.cap = cap_told;
  a.full_sweeps = t->opt_full_sweeps;
  a.front0 = use_front;
  // LEAF directions: per axis none / exterior / interior, at least one exterior move, at most
  // `conn` moves (conn 1: the dim exterior faces, in axis order); GROUP directions: every offset in
  // {-1, 0, +1}^dim with 1..conn non-zero entries (conn 1: the 2 * dim faces)
  const int conn = t->opt_balance_conn > 0 ? t->opt_balance_conn : 1;
  a.ndirs = 0;
  a.ngdirs = 0;
  for (int moves = 1; moves <= conn; ++moves)
    for (int code = 1; code < (1 << (2 * t->g.dim)); ++code) {
      int nz = 0, ext = 0, bad = 0;
      for (int ax = 0; ax < t->g.dim; ++ax) {
        const int c = (code >> (2 * ax)) & 3;
        if (c == 3) bad = 1;
        nz += c != 0;
        ext += c == 1;
      }
      if (bad || nz != moves) continue;
      if (ext >= 1) a.dirs[a.ndirs++] = (uint8_t)code;
      a.gdirs[a.ngdirs++] = (uint8_t)code;
    }
  a.do_map = t->have_old ? 1 : 0;
  a.n_old = (int)t->n_old;
  a.keys_old = t->keys[t->old];
  a.first_old = t->first[t->old];
  a.map_src = t->map_src;
  a.map_kind = t->map_kind;
  void* fn = t->g.dim == 2 ? (void*)k_balance<2> : (void*)k_balance<3>;
  static int occ[2] = {0, 0};
  int& per_sm = occ[t->g.dim - 2];
  if (per_sm == 0) LT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, BT, 0));
  if (per_sm < 1) return LT_ERR_CUDA;
  int G = t->num_sms * per_sm;
  if (G > kMaxGrid) G = kMaxGrid;
  // The marks-per-chunk counters of both sweep parities are zero on entry: zeroed when allocated, and a
  // kernel that ends without error leaves them zero (its last sweep marked nothing, the other half was
  // cleared at that sweep's start); lt_balance clears them before it retries after LT_ERR_CAPACITY.
  void* args[] = {&a};
  LT_CUDA(cudaLaunchCooperativeKernel(fn, dim3(G), dim3(BT), args, 0, t->stream));
  t->launches++;
  return LT_OK;
}

int launch_leaf_boxes(Tree* t, int32_t* d_level, uint32_t* d_xyz) {
  int G = grid_for(t, 8);
  LT_DISPATCH_DIM(t, (k_decode_n<2><<<G, BT, 0, t->stream>>>(t->g, t->keys[t->cur], t->d_s, d_level, d_xyz)),
                  (k_decode_n<3><<<G, BT, 0, t->stream>>>(t->g, t->keys[t->cur], t->d_s, d_level, d_xyz)));
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

static int grid_for_n(int64_t n) {
  int64_t G = (n + BT - 1) / BT;
  if (G < 1) G = 1;
  if (G > 148 * 16) G = 148 * 16;
  return (int)G;
}

int launch_encode(int dim, int maxl, const uint32_t* d_xyz, const int32_t* d_level, int64_t n, uint64_t* d_keys,
                  cudaStream_t s) {
  if (n == 0) return LT_OK;
  if (dim == 2) k_encode<2><<<grid_for_n(n), BT, 0, s>>>(maxl, d_xyz, d_level, n, d_keys);
  else k_encode<3><<<grid_for_n(n), BT, 0, s>>>(maxl, d_xyz, d_level, n, d_keys);
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

int launch_decode(int dim, int maxl, const uint64_t* d_keys, int64_t n, int32_t* d_level, uint32_t* d_xyz,
                  cudaStream_t s) {
  (void)maxl;
  if (n == 0) return LT_OK;
  if (dim == 2) k_decode<2><<<grid_for_n(n), BT, 0, s>>>(d_keys, n, d_level, d_xyz);
  else k_decode<3><<<grid_for_n(n), BT, 0, s>>>(d_keys, n, d_level, d_xyz);
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

}  // namespace lt
