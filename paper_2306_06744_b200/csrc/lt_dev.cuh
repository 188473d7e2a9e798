// lt_dev.cuh -- device-side helpers of liblt (key algebra, bucketed point location,
// block scans).  Product code: shares nothing with oracle/.
//
// Key format (include/lt.h; Alg. 1):  key = (morton << 5) | level,
// morton = bit-interleaved integer anchor in finest-cell units, x lowest.
// On a brick of root cubes (lt_build_brick; reading J-1) the index r of the cube sits above the
// dim * maxl path bits: morton = (r << dim * maxl) | in-cube morton, r = tx + nroot[0] * (ty + nroot[1] * tz).
// Every routine below works on this "global" morton code; a single cube has r = 0.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <stdint.h>

// -DLT_DEBUG (python -m paper_2306_06744_b200.build --debug -> liblt_debug.so): device-side checks of
// every located index, table write position, ticket and look-back word.  A failing check traps the
// kernel (the next synchronising call returns LT_ERR_CUDA and the assertion text goes to stderr).
// compute-sanitizer is not available on the GPU pool this library is developed on; this build and the
// small cases of tests/test_gpu_debug_build.py stand in for it.
#ifdef LT_DEBUG
#include <assert.h>
#define LT_DASSERT(cond) assert(cond)
#else
#define LT_DASSERT(cond) ((void)0)
#endif

namespace lt {

constexpr int kLevelBits = 5;
constexpr uint64_t kLevelMask = 31;

// Static description of a tree, passed by value to every kernel.
struct Geo {
  int dim, base, maxl;
  int ilevel;       // level of the bucket index (<= base + 1), see locate()
  int ishift;       // dim * (maxl - ilevel): morton >> ishift = bucket
  int nbuckets;     // 2^(dim*ilevel)
  int periodic;     // bit a set = axis a periodic
  uint64_t total;   // (1 << dim*maxl) - 1 : all in-cube morton bits
  int tshift;       // dim * maxl: the cube index sits above the path bits
  int ntrees;       // nroot[0] * nroot[1] * nroot[2] root cubes
  int nroot[3];     // the brick (1, 1, 1: a single cube)
  int keybits;      // bits of a key in use: dim * maxl + 5 + bits of the cube index
};

template <int DIM> struct Dim;
template <> struct Dim<2> {
  static constexpr int NC = 4, NF = 4;
  static constexpr uint64_t kAxis0 = 0x5555555555555555ull;  // bits 0,2,4,..
};
template <> struct Dim<3> {
  static constexpr int NC = 8, NF = 6;
  static constexpr uint64_t kAxis0 = 0x1249249249249249ull;  // bits 0,3,6,..
};

__host__ __device__ __forceinline__ int key_level(uint64_t k) { return (int)(k & kLevelMask); }
__host__ __device__ __forceinline__ uint64_t key_morton(uint64_t k) { return k >> kLevelBits; }
__host__ __device__ __forceinline__ uint64_t make_key(uint64_t m, int l) {
  return (m << kLevelBits) | (uint64_t)l;
}

// ---- bit interleave ("magic number approach") ---------------------------
__host__ __device__ __forceinline__ uint64_t dilate2(uint32_t v) {
  uint64_t x = v;
  x = (x | (x << 16)) & 0x0000FFFF0000FFFFull;
  x = (x | (x << 8)) & 0x00FF00FF00FF00FFull;
  x = (x | (x << 4)) & 0x0F0F0F0F0F0F0F0Full;
  x = (x | (x << 2)) & 0x3333333333333333ull;
  x = (x | (x << 1)) & 0x5555555555555555ull;
  return x;
}
__host__ __device__ __forceinline__ uint32_t compact2(uint64_t x) {
  x &= 0x5555555555555555ull;
  x = (x | (x >> 1)) & 0x3333333333333333ull;
  x = (x | (x >> 2)) & 0x0F0F0F0F0F0F0F0Full;
  x = (x | (x >> 4)) & 0x00FF00FF00FF00FFull;
  x = (x | (x >> 8)) & 0x0000FFFF0000FFFFull;
  x = (x | (x >> 16)) & 0x00000000FFFFFFFFull;
  return (uint32_t)x;
}
__host__ __device__ __forceinline__ uint64_t dilate3(uint32_t v) {
  uint64_t x = v & 0x1FFFFFu;
  x = (x | (x << 32)) & 0x001F00000000FFFFull;
  x = (x | (x << 16)) & 0x001F0000FF0000FFull;
  x = (x | (x << 8)) & 0x100F00F00F00F00Full;
  x = (x | (x << 4)) & 0x10C30C30C30C30C3ull;
  x = (x | (x << 2)) & 0x1249249249249249ull;
  return x;
}
__host__ __device__ __forceinline__ uint32_t compact3(uint64_t x) {
  x &= 0x1249249249249249ull;
  x = (x | (x >> 2)) & 0x10C30C30C30C30C3ull;
  x = (x | (x >> 4)) & 0x100F00F00F00F00Full;
  x = (x | (x >> 8)) & 0x001F0000FF0000FFull;
  x = (x | (x >> 16)) & 0x001F00000000FFFFull;
  x = (x | (x >> 32)) & 0x00000000001FFFFFull;
  return (uint32_t)x;
}
template <int DIM>
__host__ __device__ __forceinline__ uint64_t interleave(const uint32_t* x) {
  if (DIM == 2) return dilate2(x[0]) | (dilate2(x[1]) << 1);
  return dilate3(x[0]) | (dilate3(x[1]) << 1) | (dilate3(x[2]) << 2);
}
template <int DIM>
__host__ __device__ __forceinline__ void deinterleave(uint64_t m, uint32_t* x) {
  if (DIM == 2) {
    x[0] = compact2(m);
    x[1] = compact2(m >> 1);
    x[2] = 0;
  } else {
    x[0] = compact3(m);
    x[1] = compact3(m >> 1);
    x[2] = compact3(m >> 2);
  }
}

// child id of a leaf = digit (level-1) of its path = low DIM bits of the raw ID
// (PAPER.md:173); 0 for the root.
template <int DIM>
__device__ __forceinline__ int child_id(const Geo& g, uint64_t m, int l) {
  return (int)((m >> (DIM * (g.maxl - l))) & (uint64_t)(Dim<DIM>::NC - 1));
}

// a (level la) is a strict ancestor of b (level lb)
template <int DIM>
__device__ __forceinline__ bool is_ancestor(const Geo& g, uint64_t ka, uint64_t kb) {
  int la = key_level(ka), lb = key_level(kb);
  if (la >= lb) return false;
  int sh = DIM * (g.maxl - la);
  return (key_morton(ka) >> sh) == (key_morton(kb) >> sh);
}

// Same-level face neighbour of the cell (m, l) across local face f (0=-x 1=+x 2=-y ...),
// computed on the dilated integer: add / subtract the cell width on one axis with the
// carry rippling over the other axes' bit positions.  Inside a cube the coordinate wraps mod
// 2^maxl; a step over the cube's face moves to the adjacent cube of the brick, with the periodic
// wrap of the whole domain or, on a non-periodic axis, ends at the domain boundary
// (returns false).  The cube index bits of m are carried along.
template <int DIM>
__device__ __forceinline__ bool face_neighbour(const Geo& g, uint64_t m, int l, int f, uint64_t* mn) {
  const int a = f >> 1;
  const int sh = DIM * (g.maxl - l) + a;
  const uint64_t wbit = 1ull << sh;
  const uint64_t maskA = (Dim<DIM>::kAxis0 << a) & g.total;
  const uint64_t hiA = maskA & ~(wbit - 1);
  bool edge;
  uint64_t na;
  if (f & 1) {
    edge = (m & hiA) == hiA;
    na = ((m | ~maskA) + wbit) & maskA;
  } else {
    edge = (m & hiA) == 0;
    na = ((m & maskA) - wbit) & maskA;
  }
  *mn = (m & ~maskA) | na;
  if (!edge) return true;
  const bool per = (g.periodic >> a) & 1;
  if (g.nroot[a] == 1) return per;  // one cube along this axis: its own periodic image
  const int stride = a == 0 ? 1 : (a == 1 ? g.nroot[0] : g.nroot[0] * g.nroot[1]);
  const int tree = (int)(m >> g.tshift);
  const int ta = (tree / stride) % g.nroot[a];
  int tn = ta + ((f & 1) ? 1 : -1);
  if (tn < 0 || tn >= g.nroot[a]) {
    if (!per) return false;
    tn = tn < 0 ? g.nroot[a] - 1 : 0;
  }
  *mn = ((uint64_t)(tree + (tn - ta) * stride) << g.tshift) | (*mn & g.total);
  return true;
}

// Point location (the lower-bound search of PAPER.md:134-143, Eq. 7, in one form):
// index of the leaf whose cell contains the finest-level point with morton code `mn`,
// i.e. the last j with morton(keys[j]) <= mn.  `first` is the bucket index over the uniform
// level-`ilevel` grid: first[b] = index of the first leaf inside cell b, or, where a leaf is
// coarser than the grid, the index of that leaf in every cell it covers (the search range of
// such a cell is empty or holds only larger keys, and the leaf itself is returned).
__device__ __forceinline__ int locate(const Geo& g, const uint64_t* __restrict__ keys,
                                      const int* __restrict__ first, uint64_t mn) {
  const uint32_t b = (uint32_t)(mn >> g.ishift);
  LT_DASSERT(b < (uint32_t)g.nbuckets);
  int lo = first[b], hi = first[b + 1];
  LT_DASSERT(lo >= 0 && lo <= hi && hi <= first[g.nbuckets]);
  const uint64_t bound = (mn << kLevelBits) | kLevelMask;  // keys <= bound  <=>  morton <= mn
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (keys[mid] <= bound) lo = mid; else hi = mid;
  }
  // the located leaf starts at or before the point and ends after it (the leaves tile the domain)
  LT_DASSERT(lo < first[g.nbuckets] && keys[lo] <= bound);
  LT_DASSERT((mn >> (g.dim * (g.maxl - key_level(keys[lo])))) ==
             (key_morton(keys[lo]) >> (g.dim * (g.maxl - key_level(keys[lo])))));
  return lo;
}

// Record the leaf (m, l) stored at position `pos` in the bucket index (see locate()).
template <int DIM>
__device__ __forceinline__ void index_write(const Geo& g, int* __restrict__ first, uint64_t m, int l, int pos) {
  LT_DASSERT(pos >= 0 && (m >> g.ishift) < (uint64_t)g.nbuckets);
  if (l >= g.ilevel) {
    if ((m & ((1ull << g.ishift) - 1)) == 0) first[m >> g.ishift] = pos;
  } else {
    const int span = 1 << (DIM * (g.ilevel - l));
    const uint32_t b = (uint32_t)(m >> g.ishift);
    for (int c = 0; c < span; ++c) first[b + c] = pos;
  }
}

// ---- block-wide exclusive scan (blockDim.x multiple of 32, <= 1024) ------------------
template <typename T>
__device__ __forceinline__ T warp_incl_scan(T v) {
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    T o = __shfl_up_sync(0xffffffffu, v, d);
    if (lane >= d) v += o;
  }
  return v;
}
// returns the exclusive prefix of v within the block; *total = block sum.
// `sm` must hold 33 T's.  Ends with a barrier, so sm may be reused immediately.
template <typename T>
__device__ __forceinline__ T block_excl_scan(T v, T* sm, T* total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  T inc = warp_incl_scan(v);
  if (lane == 31) sm[w] = inc;
  __syncthreads();
  if (w == 0) {
    T s = lane < nw ? sm[lane] : T(0);
    T si = warp_incl_scan(s);
    sm[lane] = si - s;
    if (lane == 31) sm[32] = si;
  }
  __syncthreads();
  T res = sm[w] + inc - v;
  *total = sm[32];
  __syncthreads();
  return res;
}
template <typename T>
__device__ __forceinline__ T block_sum(T v, T* sm) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
  if (lane == 0) sm[w] = v;
  __syncthreads();
  T s = T(0);
  if (w == 0) {
    s = lane < nw ? sm[lane] : T(0);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    if (lane == 0) sm[32] = s;
  }
  __syncthreads();
  s = sm[32];
  __syncthreads();
  return s;
}

// Contiguous chunk of [0, n) owned by block b of G: multiples of `tile` items.
__device__ __forceinline__ void block_chunk(int64_t n, int G, int b, int tile, int64_t* lo, int64_t* hi) {
  int64_t per = (n + G - 1) / G;
  per = (per + tile - 1) / tile * tile;
  int64_t l = (int64_t)b * per, h = l + per;
  *lo = l < n ? l : n;
  *hi = h < n ? h : n;
}

// sum of sums[0..b) and of all G entries; every thread of the block gets both.
template <typename T>
__device__ __forceinline__ void chunk_offsets(const T* __restrict__ sums, int G, int b, T* sm, T* before, T* total) {
  T mine = T(0), all = T(0);
  for (int i = threadIdx.x; i < G; i += blockDim.x) {
    T s = sums[i];
    all += s;
    if (i < b) mine += s;
  }
  *before = block_sum(mine, sm);
  *total = block_sum(all, sm);
}

// sticky device status word: first error wins
__device__ __forceinline__ void set_status(int* status, int code) { atomicCAS(status, 0, code); }

// Alg. 7 for ONE new leaf: locate its anchor in T_old (lower bound, Eq. 7):
//   same ID                       -> copy   kind 0
//   old entry is its parent       -> refined-from   kind 1 | child_id << 4
//   old entry is its first child  -> fused-from      (reading E-6)   kind 2
// Returns false when the new leaf is more than one level from T_old (or the old sibling group is
// not complete): the caller decides where that error is reported.
template <int DIM>
__device__ __forceinline__ bool map_entry(const Geo& g, uint64_t key, const uint64_t* __restrict__ keys_old,
                                          const int* __restrict__ first_old, int n_old, int* src, int* kind) {
  constexpr int NC = Dim<DIM>::NC;
  const int l = key_level(key);
  const uint64_t m = key_morton(key);
  const int o = locate(g, keys_old, first_old, m);
  const int lo = key_level(keys_old[o]);
  bool ok = true;
  int kd = 0;
  if (lo == l) {
    kd = 0;
  } else if (lo == l - 1) {
    kd = 1 | (child_id<DIM>(g, m, l) << 4);
  } else if (lo == l + 1) {
    // complete group of leaves: last sibling present at o + NC - 1
    const int sh = DIM * (g.maxl - l - 1);
    const uint64_t klast = make_key(m | ((uint64_t)(NC - 1) << sh), l + 1);
    if (o + NC - 1 >= n_old || keys_old[o + NC - 1] != klast) ok = false;
    kd = 2;
  } else {
    ok = false;
  }
  *src = o;
  *kind = kd;
  return ok;
}

// ---- TMA (bulk asynchronous copy) plumbing: one lane arms an mbarrier with the byte count and issues
// cp.async.bulk global -> shared; the copy engine signals the barrier when the bytes have landed.  The copy
// does not go through the LSU / shared-memory data pipe that bounds these kernels.  Addresses and size
// must be multiples of 16 bytes.
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}


}  // namespace lt
