// lt_construct.cu -- tree construction from scattered points / octants (Alg. 2,
// PAPER.md:105-120) for liblt.  Product code: shares nothing with oracle/.
//
// The paper completes the sorted initial octants by splitting the largest common ancestor of
// two consecutive octants inside a thread block, keeping the children that lie between them
// in shared memory, de-duplicating with block-local and global atomic counters, appending
// to the global array and sorting + linearising again (Alg. 2 steps 2-6), repeating when
// shared memory overflows.  Here the same complete tree is written directly
// in Morton order with no atomics, no append and no second sort:
//
//   between two consecutive linearised octants P < Q the leaves of the coarsest complete
//   tree are, in ascending order, (i) for every level L from level(P) up to d+1 the later
//   siblings of P's level-L ancestor, (ii) the level-d cells strictly between the level-d
//   ancestors of P and Q, (iii) for every level L from d+1 down to level(Q) the earlier
//   siblings of Q's level-L ancestor, where d is the first level at which the two paths
//   differ.  D_min = base_level turns the levels above base into one "digit" with
//   2^(dim*base) values (the uniform base grid).  The domain ends are the gaps before the
//   first and after the last octant ("complete ... covers the entire domain").
//
// So a gap's size is a closed form of the two keys (k_complete_count), an exclusive scan
// places every segment "gap_i, octant_i", and an output-centric kernel (k_complete_fill:
// one thread per OUTPUT leaf, segment found by a shared-memory search of the scanned
// offsets of its tile) computes each leaf from its rank inside its gap.  Writes are fully
// coalesced and the work per thread is bounded by 2 * max_level regardless of gap size.
#include "lt_internal.h"

namespace lt {

constexpr int CT = 256;    // threads per block
constexpr int CTILE = 2048;  // output leaves per tile of k_complete_fill

// ---------------------------------------------------------------- points -> depth-Dmax keys
// Alg. 1 steps 1-2 / Alg. 2 step 1; reading G-1 of DESIGN.md:
// xi = floor((x - lo) / (hi - lo) * 2^Dmax) in fp64, in this order (IEEE division, the
// product by a power of two is exact, no FMA can form), clamped to [0, 2^Dmax - 1].
__device__ __forceinline__ uint32_t point_cell(double x, double lo, double hi, int maxl) {
  const double s = __ddiv_rn(__dsub_rn(x, lo), __dsub_rn(hi, lo));
  double v = floor(__dmul_rn(s, (double)(1ull << maxl)));
  const double top = (double)((1ull << maxl) - 1);
  if (!(v >= 0.0)) v = 0.0;
  if (v > top) v = top;
  return (uint32_t)v;
}

struct Box { double lo[3], hi[3]; };

template <int DIM>
__global__ void __launch_bounds__(CT) k_points_to_keys(int maxl, Box box, const double* __restrict__ xyz, int64_t n,
                                                       uint64_t* __restrict__ keys) {
  for (int64_t i = blockIdx.x * (int64_t)CT + threadIdx.x; i < n; i += (int64_t)gridDim.x * CT) {
    uint32_t c[3] = {0, 0, 0};
#pragma unroll
    for (int a = 0; a < DIM; ++a) c[a] = point_cell(xyz[i * DIM + a], box.lo[a], box.hi[a], maxl);
    keys[i] = make_key(interleave<DIM>(c), maxl);
  }
}

// ---------------------------------------------------------------- gap algebra
template <int DIM>
__device__ __forceinline__ int digit(const Geo& g, uint64_t m, int L) {
  return (int)((m >> (DIM * (g.maxl - L))) & (uint64_t)(Dim<DIM>::NC - 1));
}

// Description of the gap between consecutive linearised octants P (absent at the domain
// start) and Q (absent at the domain end).
template <int DIM>
struct Gap {
  uint64_t mp, mq;
  int lp, lq, d;        // d = first level at which the paths differ (>= base)
  int64_t topP, topQ;   // base-cell indices (-1 / 2^(dim*base) for the absent ends)
  bool hasP, hasQ;
};

template <int DIM>
__device__ __forceinline__ Gap<DIM> make_gap(const Geo& g, bool hasP, uint64_t kp, bool hasQ, uint64_t kq) {
  Gap<DIM> G;
  G.hasP = hasP;
  G.hasQ = hasQ;
  G.mp = hasP ? key_morton(kp) : 0;
  G.mq = hasQ ? key_morton(kq) : 0;
  G.lp = hasP ? key_level(kp) : g.base;
  G.lq = hasQ ? key_level(kq) : g.base;
  const int bsh = DIM * (g.maxl - g.base);
  G.topP = hasP ? (int64_t)(G.mp >> bsh) : -1;
  G.topQ = hasQ ? (int64_t)(G.mq >> bsh) : (int64_t)1 << (DIM * g.base);
  if (G.topP != G.topQ) {
    G.d = g.base;
  } else {
    const int hb = 63 - __clzll((long long)(G.mp ^ G.mq));
    G.d = g.maxl - hb / DIM;
  }
  return G;
}

template <int DIM>
__device__ __forceinline__ int64_t gap_middle(const Geo& g, const Gap<DIM>& G) {
  if (G.d == g.base) return G.topQ - G.topP - 1;
  return digit<DIM>(g, G.mq, G.d) - digit<DIM>(g, G.mp, G.d) - 1;
}

template <int DIM>
__device__ __forceinline__ int64_t gap_count(const Geo& g, const Gap<DIM>& G) {
  constexpr int NC = Dim<DIM>::NC;
  int64_t c = gap_middle<DIM>(g, G);
  if (G.hasP)
    for (int L = G.lp; L > G.d; --L) c += NC - 1 - digit<DIM>(g, G.mp, L);
  if (G.hasQ)
    for (int L = G.d + 1; L <= G.lq; ++L) c += digit<DIM>(g, G.mq, L);
  return c;
}

// the r-th leaf (ascending Morton order) of the gap
template <int DIM>
__device__ __forceinline__ uint64_t gap_key(const Geo& g, const Gap<DIM>& G, int64_t r) {
  constexpr int NC = Dim<DIM>::NC;
  if (G.hasP)
    for (int L = G.lp; L > G.d; --L) {  // later siblings of P's level-L ancestor, finest first
      const int dg = digit<DIM>(g, G.mp, L);
      const int c = NC - 1 - dg;
      if (r < c) {
        const int sh = DIM * (g.maxl - L);
        const uint64_t par = (G.mp >> (sh + DIM)) << (sh + DIM);
        return make_key(par | ((uint64_t)(dg + 1 + (int)r) << sh), L);
      }
      r -= c;
    }
  {
    const int64_t c = gap_middle<DIM>(g, G);
    if (r < c) {
      const int sh = DIM * (g.maxl - G.d);
      if (G.d == g.base) return make_key((uint64_t)(G.topP + 1 + r) << sh, g.base);
      const uint64_t par = (G.mp >> (sh + DIM)) << (sh + DIM);
      return make_key(par | ((uint64_t)(digit<DIM>(g, G.mp, G.d) + 1 + (int)r) << sh), G.d);
    }
    r -= c;
  }
  for (int L = G.d + 1; L <= G.lq; ++L) {  // earlier siblings of Q's level-L ancestor, coarsest first
    const int c = digit<DIM>(g, G.mq, L);
    if (r < c) {
      const int sh = DIM * (g.maxl - L);
      const uint64_t par = (G.mq >> (sh + DIM)) << (sh + DIM);
      return make_key(par | ((uint64_t)r << sh), L);
    }
    r -= c;
  }
  return ~0ull;  // unreachable for r < gap_count
}

// ---------------------------------------------------------------- segment sizes and offsets
// Segment i (0 <= i <= n) = the gap before octant i followed by octant i itself (segment n
// is the gap after the last octant).  Pass 1 writes each segment's exclusive offset inside
// its block's chunk and the chunk sum; pass 2 adds the chunk bases.
template <int DIM>
__device__ __forceinline__ int64_t segment_size(const Geo& g, const uint64_t* __restrict__ in, int64_t n, int64_t i,
                                                int* status) {
  const bool hasP = i > 0, hasQ = i < n;
  const uint64_t kp = hasP ? in[i - 1] : 0, kq = hasQ ? in[i] : 0;
  if (hasQ) {
    const int l = key_level(kq);
    if (l < g.base || l > g.maxl || (key_morton(kq) >> (DIM * g.maxl)) != 0 ||
        (key_morton(kq) & ((1ull << (DIM * (g.maxl - (l > g.maxl ? g.maxl : l)))) - 1)) != 0) {
      set_status(status, LT_ERR_ARG);
      return 1;
    }
  }
  const Gap<DIM> G = make_gap<DIM>(g, hasP, kp, hasQ, kq);
  return gap_count<DIM>(g, G) + (hasQ ? 1 : 0);
}

template <int DIM>
__global__ void __launch_bounds__(CT) k_complete_count(Geo g, const uint64_t* __restrict__ in, int64_t n,
                                                       uint32_t* __restrict__ offs,
                                                       unsigned long long* __restrict__ sums, DevScalars* s) {
  __shared__ unsigned long long sm[33];
  int64_t lo, hi;
  block_chunk(n + 1, gridDim.x, blockIdx.x, CT, &lo, &hi);
  unsigned long long run = 0;
  for (int64_t t0 = lo; t0 < hi; t0 += CT) {
    const int64_t i = t0 + threadIdx.x;
    const unsigned long long sz = i < hi ? (unsigned long long)segment_size<DIM>(g, in, n, i, &s->status) : 0ull;
    unsigned long long tot;
    const unsigned long long ex = block_excl_scan<unsigned long long>(sz, sm, &tot);
    if (i < hi) offs[i] = (uint32_t)(run + ex);  // < 2^31 once the host has checked the total
    run += tot;
  }
  if (threadIdx.x == 0) sums[blockIdx.x] = run;
}

__global__ void __launch_bounds__(CT) k_complete_offsets(int64_t n, uint32_t* __restrict__ offs,
                                                         const unsigned long long* __restrict__ sums,
                                                         unsigned long long* __restrict__ total_out) {
  __shared__ unsigned long long sm[33];
  unsigned long long before, total;
  chunk_offsets(sums, gridDim.x, blockIdx.x, sm, &before, &total);
  int64_t lo, hi;
  block_chunk(n + 1, gridDim.x, blockIdx.x, CT, &lo, &hi);
  if (total < (1ull << 31)) {
    for (int64_t i = lo + threadIdx.x; i < hi; i += CT) offs[i] += (uint32_t)before;
    if (blockIdx.x == 0 && threadIdx.x == 0) offs[n + 1] = (uint32_t)total;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) *total_out = total;
}

// ---------------------------------------------------------------- output-centric fill
// One thread per output leaf.  A tile of CTILE consecutive outputs touches at most
// CTILE + 1 segments: their scanned offsets are staged in shared memory and every thread
// finds its segment there (load-balanced search), then computes its leaf from its rank.
template <int DIM>
__global__ void __launch_bounds__(CT) k_complete_fill(Geo g, const uint64_t* __restrict__ in, int64_t n,
                                                      const uint32_t* __restrict__ offs, uint64_t* __restrict__ out,
                                                      DevScalars* s) {
  __shared__ uint32_t soff[CTILE + 4];
  __shared__ int64_t srange[2];
  const int64_t M = offs[n + 1];
  const int64_t ntiles = (M + CTILE - 1) / CTILE;
  for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const int64_t j0 = tile * CTILE, j1 = (j0 + CTILE < M) ? j0 + CTILE : M;
    if (threadIdx.x < 2) {  // last segment s with offs[s] <= j, for j = j0 and j = j1 - 1
      const uint32_t j = (uint32_t)(threadIdx.x == 0 ? j0 : j1 - 1);
      int64_t lo = 0, hi = n + 1;  // offs[0] = 0 <= j
      while (hi - lo > 1) {
        const int64_t mid = (lo + hi) >> 1;
        if (offs[mid] <= j) lo = mid; else hi = mid;
      }
      srange[threadIdx.x] = lo;
    }
    __syncthreads();
    const int64_t s_lo = srange[0];
    const int ns = (int)(srange[1] - s_lo) + 1;  // <= CTILE + 1
    for (int k = threadIdx.x; k <= ns; k += CT) soff[k] = offs[s_lo + k];
    __syncthreads();
    for (int64_t j = j0 + threadIdx.x; j < j1; j += CT) {
      int lo = 0, hi = ns;
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (soff[mid] <= (uint32_t)j) lo = mid; else hi = mid;
      }
      const int64_t seg = s_lo + lo;
      const int64_t r = j - soff[lo];
      const int64_t size = (int64_t)soff[lo + 1] - soff[lo];
      uint64_t key;
      if (seg < n && r == size - 1) {
        key = in[seg];
      } else {
        const bool hasP = seg > 0, hasQ = seg < n;
        const Gap<DIM> G = make_gap<DIM>(g, hasP, hasP ? in[seg - 1] : 0, hasQ, hasQ ? in[seg] : 0);
        key = gap_key<DIM>(g, G, r);
      }
      out[j] = key;
    }
    __syncthreads();
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) s->n = (int)M;
}

// ---------------------------------------------------------------- launchers
int launch_points_to_keys(int dim, int maxl, const double* domain, const double* d_xyz, int64_t n, uint64_t* d_keys,
                          int G, cudaStream_t s, int64_t* launches) {
  Box box;
  for (int a = 0; a < 3; ++a) {
    box.lo[a] = a < dim ? domain[a] : 0.0;
    box.hi[a] = a < dim ? domain[dim + a] : 1.0;
  }
  if (dim == 2) k_points_to_keys<2><<<G, CT, 0, s>>>(maxl, box, d_xyz, n, d_keys);
  else k_points_to_keys<3><<<G, CT, 0, s>>>(maxl, box, d_xyz, n, d_keys);
  *launches += 1;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

// sizes + offsets of the n + 1 segments of the linearised octants d_in[0..n); *total (host)
// = number of leaves of the completed tree.  d_offs holds n + 2 entries.  Synchronises.
int launch_complete_count(Tree* t, const uint64_t* d_in, int64_t n, uint32_t* d_offs, int64_t* total) {
  const int G = grid_for(t, 4);
  if (t->g.dim == 2) k_complete_count<2><<<G, CT, 0, t->stream>>>(t->g, d_in, n, d_offs, t->d_sums, t->d_s);
  else k_complete_count<3><<<G, CT, 0, t->stream>>>(t->g, d_in, n, d_offs, t->d_sums, t->d_s);
  k_complete_offsets<<<G, CT, 0, t->stream>>>(n, d_offs, t->d_sums, &t->d_s->volume);
  t->launches += 2;
  LT_CUDA(cudaGetLastError());
  LT_CUDA(cudaMemcpyAsync(t->h_s, t->d_s, sizeof(DevScalars), cudaMemcpyDeviceToHost, t->stream));
  t->host_syncs++;
  LT_CUDA(cudaStreamSynchronize(t->stream));
  *total = (int64_t)t->h_s->volume;
  return LT_OK;
}

int launch_complete_fill(Tree* t, const uint64_t* d_in, int64_t n, const uint32_t* d_offs, int64_t total) {
  int64_t tiles = (total + CTILE - 1) / CTILE;
  int G = grid_for(t, 4);
  if (tiles < G) G = tiles > 0 ? (int)tiles : 1;
  if (t->g.dim == 2) k_complete_fill<2><<<G, CT, 0, t->stream>>>(t->g, d_in, n, d_offs, t->keys[t->cur], t->d_s);
  else k_complete_fill<3><<<G, CT, 0, t->stream>>>(t->g, d_in, n, d_offs, t->keys[t->cur], t->d_s);
  t->launches += 1;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

}  // namespace lt
