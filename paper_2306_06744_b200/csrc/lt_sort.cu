// lt_sort.cu -- ascending LSD radix sort of uint64 Morton IDs and linearisation (Alg. 3,
// PAPER.md:122-128) for sm_100a.  Replaces the paper's thrust::sort / thrust::unique
// (PAPER.md:117, :126-128, :161, :223).  Product code.
//
// One-sweep design: one histogram kernel counts all digits of all passes; each pass is a
// single kernel in which a tile ranks its keys (warp match + per-warp digit counters in
// shared memory), publishes its per-digit counts and obtains the counts of all earlier
// tiles by decoupled look-back, then scatters.  Only bits [0, key_bits) are sorted.
#include "lt_internal.h"

namespace lt {

constexpr int ST = 256;                 // threads per sort block (= number of digit values)
constexpr int SITEMS = 16;              // keys per thread
constexpr int STILE = ST * SITEMS;      // keys per tile
constexpr unsigned FLAG_AGG = 1u << 30, FLAG_INC = 2u << 30, VAL_MASK = (1u << 30) - 1;

__global__ void __launch_bounds__(ST) k_sort_hist(const uint64_t* __restrict__ keys, int64_t n, int passes,
                                                  unsigned* __restrict__ hist) {
  __shared__ unsigned sh[8 * 256];
  for (int i = threadIdx.x; i < passes * 256; i += ST) sh[i] = 0;
  __syncthreads();
  for (int64_t i = blockIdx.x * (int64_t)ST + threadIdx.x; i < n; i += (int64_t)gridDim.x * ST) {
    uint64_t k = keys[i];
    for (int p = 0; p < passes; ++p) atomicAdd(&sh[p * 256 + (int)((k >> (8 * p)) & 255)], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < passes * 256; i += ST)
    if (sh[i]) atomicAdd(&hist[i], sh[i]);
}

// exclusive scan of each pass's 256 counters (one block per pass)
__global__ void __launch_bounds__(256) k_sort_scan_hist(unsigned* __restrict__ hist) {
  __shared__ unsigned sm[33];
  unsigned v = hist[blockIdx.x * 256 + threadIdx.x], tot;
  unsigned ex = block_excl_scan<unsigned>(v, sm, &tot);
  hist[blockIdx.x * 256 + threadIdx.x] = ex;
}

// status words are polled with GPU-scope relaxed loads (a volatile access is system scope and
// is not pipelined); the word carries its own payload, so no fence is needed
__device__ __forceinline__ unsigned ld_status(const volatile unsigned* p) {
  unsigned v;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_status(volatile unsigned* p, unsigned v) {
  asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

__global__ void __launch_bounds__(ST) k_sort_pass(const uint64_t* __restrict__ in, uint64_t* __restrict__ out,
                                                  int64_t n, int shift, const unsigned* __restrict__ base,
                                                  volatile unsigned* status, int* ticket) {
  __shared__ unsigned wcnt[(ST / 32) * 256];
  __shared__ unsigned gbase[256];
  __shared__ unsigned loff[256];
  __shared__ unsigned s_scan[33];
  __shared__ unsigned s_ntile;
  __shared__ uint64_t s_keys[STILE];
  __shared__ int s_tile;
  if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1);
  for (int i = threadIdx.x; i < (ST / 32) * 256; i += ST) wcnt[i] = 0;
  __syncthreads();
  const int tile = s_tile;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const unsigned lt_mask = (1u << lane) - 1;
  uint64_t key[SITEMS];
  unsigned rank[SITEMS];
  int dig[SITEMS];
  const int64_t t0 = (int64_t)tile * STILE + (int64_t)w * 32 * SITEMS + lane;
#pragma unroll
  for (int k = 0; k < SITEMS; ++k) {
    const int64_t idx = t0 + k * 32;
    const bool valid = idx < n;
    key[k] = valid ? in[idx] : 0;
    dig[k] = valid ? (int)((key[k] >> shift) & 255) : 256;
  }
  // stable rank of every key among the equal-digit keys of its warp (warp-striped order)
  // all match operations are issued before the (serial, shared-memory) counter updates: MATCH
  // has a long latency and the loop below would otherwise expose it SITEMS times
  // (peers by 9 ballots over the digit bits rather than MATCH.ANY, whose latency grows with the
  // number of distinct values in the warp -- about 28 of 32 for a random digit)
  unsigned peers[SITEMS];
#pragma unroll
  for (int k = 0; k < SITEMS; ++k) {
    unsigned pm = 0xffffffffu;
#pragma unroll
    for (int b = 0; b < 9; ++b) {
      const bool bit = (dig[k] >> b) & 1;
      const unsigned vote = __ballot_sync(0xffffffffu, bit);
      pm &= bit ? vote : ~vote;
    }
    peers[k] = pm;
  }
#pragma unroll
  for (int k = 0; k < SITEMS; ++k) {
    const unsigned before = __popc(peers[k] & lt_mask);
    unsigned pre = 0;
    if (dig[k] < 256) pre = wcnt[w * 256 + dig[k]];
    __syncwarp();
    if (dig[k] < 256 && before == 0) wcnt[w * 256 + dig[k]] = pre + __popc(peers[k]);
    __syncwarp();
    rank[k] = pre + before;
  }
  __syncthreads();
  {
    // thread d owns digit d: prefix over the warps, then decoupled look-back over tiles
    const int d = threadIdx.x;
    unsigned run = 0;
#pragma unroll
    for (int ww = 0; ww < ST / 32; ++ww) {
      unsigned c = wcnt[ww * 256 + d];
      wcnt[ww * 256 + d] = run;
      run += c;
    }
    unsigned excl = 0;
    if (tile == 0) {
      st_status(status + d, run | FLAG_INC);
    } else {
      st_status(status + (size_t)tile * 256 + d, run | FLAG_AGG);
      // look back over the earlier tiles, LB status words per round trip: in the first wave
      // every resident tile publishes its aggregate at about the same time, so the chain to
      // the nearest inclusive prefix can be hundreds of tiles long -- batching the (independent)
      // loads keeps it from being a chain of dependent L2 latencies
      constexpr int LB = 8;
      bool done = false;
      for (int t = tile - 1; t >= 0 && !done; t -= LB) {
        unsigned v[LB];
#pragma unroll
        for (int j = 0; j < LB; ++j) v[j] = t - j >= 0 ? ld_status(status + (size_t)(t - j) * 256 + d) : (2u << 30);
#pragma unroll
        for (int j = 0; j < LB; ++j) {
          if (done) break;
          while ((v[j] >> 30) == 0) v[j] = ld_status(status + (size_t)(t - j) * 256 + d);
          LT_DASSERT((v[j] >> 30) <= 2);  // look-back protocol: 0 not ready, 1 tile aggregate, 2 inclusive prefix
          excl += v[j] & VAL_MASK;
          if ((v[j] >> 30) == 2) done = true;
        }
      }
      st_status(status + (size_t)tile * 256 + d, ((excl + run) & VAL_MASK) | FLAG_INC);
    }
    // position of digit d's run inside the tile (exclusive scan of the tile histogram) and the
    // global address of the run's first key minus that position
    unsigned ntile;
    const unsigned tex = block_excl_scan<unsigned>(run, s_scan, &ntile);
    loff[d] = tex;
    gbase[d] = base[d] + excl - tex;
    if (d == 0) s_ntile = ntile;
  }
  __syncthreads();
  // reorder the tile by digit in shared memory, then write it out in tile order: consecutive
  // threads store consecutive addresses inside every digit run (instead of one scattered 8-byte
  // store per key, 25 sectors per request in the first version)
#pragma unroll
  for (int k = 0; k < SITEMS; ++k)
    if (dig[k] < 256) {
      LT_DASSERT(loff[dig[k]] + wcnt[w * 256 + dig[k]] + rank[k] < (unsigned)STILE);
      s_keys[loff[dig[k]] + wcnt[w * 256 + dig[k]] + rank[k]] = key[k];
    }
  __syncthreads();
  const int nt = (int)s_ntile;
#pragma unroll
  for (int k = 0; k < SITEMS; ++k) {
    const int i = k * ST + threadIdx.x;
    if (i < nt) {
      const uint64_t kk = s_keys[i];
      LT_DASSERT((int64_t)gbase[(int)((kk >> shift) & 255)] + i < n);
      out[(size_t)gbase[(int)((kk >> shift) & 255)] + i] = kk;
    }
  }
}

int sort_keys(uint64_t* d_keys, int64_t n, int key_bits, SortScratch* sc, cudaStream_t s, int64_t* launches) {
  if (n <= 1) return LT_OK;
  if (n >= (1ll << 30)) return LT_ERR_ARG;
  const int passes = (key_bits + 7) / 8;
  if (passes < 1 || passes > 8) return LT_ERR_ARG;
  const int64_t tiles = (n + STILE - 1) / STILE;
  if (sc->cap < n) {
    dev_free(sc->tmp, s);
    sc->tmp = nullptr;
    int rc = dev_alloc((void**)&sc->tmp, (size_t)n * sizeof(uint64_t), s);
    if (rc != LT_OK) return rc;
    sc->cap = n;
  }
  if (!sc->hist) {
    int rc = dev_alloc((void**)&sc->hist, (8 * 256 + 8) * sizeof(unsigned), s);
    if (rc != LT_OK) return rc;
  }
  if (sc->status_cap < tiles) {
    dev_free(sc->status, s);
    sc->status = nullptr;
    int rc = dev_alloc((void**)&sc->status, (size_t)tiles * 256 * sizeof(unsigned), s);
    if (rc != LT_OK) return rc;
    sc->status_cap = tiles;
  }
  int* tickets = (int*)(sc->hist + 8 * 256);
  LT_CUDA(cudaMemsetAsync(sc->hist, 0, (8 * 256 + 8) * sizeof(unsigned), s));
  int hg = (int)((n + ST * 16 - 1) / (ST * 16));
  if (hg > 148 * 8) hg = 148 * 8;
  k_sort_hist<<<hg, ST, 0, s>>>(d_keys, n, passes, sc->hist);
  k_sort_scan_hist<<<passes, 256, 0, s>>>(sc->hist);
  *launches += 2;
  uint64_t* src = d_keys;
  uint64_t* dst = sc->tmp;
  for (int p = 0; p < passes; ++p) {
    LT_CUDA(cudaMemsetAsync(sc->status, 0, (size_t)tiles * 256 * sizeof(unsigned), s));
    k_sort_pass<<<(int)tiles, ST, 0, s>>>(src, dst, n, 8 * p, sc->hist + p * 256, sc->status, tickets + p);
    *launches += 1;
    uint64_t* x = src;
    src = dst;
    dst = x;
  }
  LT_CUDA(cudaGetLastError());
  if (src != d_keys) LT_CUDA(cudaMemcpyAsync(d_keys, src, (size_t)n * sizeof(uint64_t), cudaMemcpyDeviceToDevice, s));
  return LT_OK;
}

// ------------------------------------------------------------------------ Alg. 3
// Sorted keys -> drop every key that equals or is an ancestor of its successor.  The
// paper does reverse / unique("overlapping") / reverse; on a sorted
// array the descendants of a key follow it contiguously, so "overlaps the next kept key"
// is the same as "overlaps the immediate successor".
template <int DIM>
__device__ __forceinline__ bool lin_keep(int maxl, const uint64_t* __restrict__ keys, int64_t i, int64_t n) {
  if (i + 1 >= n) return true;
  const uint64_t a = keys[i], b = keys[i + 1];
  if (a == b) return false;
  const int la = key_level(a), lb = key_level(b);
  if (la >= lb) return true;
  const int sh = DIM * (maxl - la);
  return (key_morton(a) >> sh) != (key_morton(b) >> sh);
}

template <int DIM>
__global__ void __launch_bounds__(256) k_lin_count(int maxl, const uint64_t* __restrict__ keys, int64_t n,
                                                   unsigned long long* __restrict__ sums) {
  __shared__ unsigned long long sm[33];
  int64_t lo, hi;
  block_chunk(n, gridDim.x, blockIdx.x, 256, &lo, &hi);
  unsigned long long acc = 0;
  for (int64_t i = lo + threadIdx.x; i < hi; i += 256) acc += lin_keep<DIM>(maxl, keys, i, n) ? 1 : 0;
  acc = block_sum(acc, sm);
  if (threadIdx.x == 0) sums[blockIdx.x] = acc;
}

template <int DIM>
__global__ void __launch_bounds__(256) k_lin_scatter(int maxl, const uint64_t* __restrict__ keys, int64_t n,
                                                     const unsigned long long* __restrict__ sums,
                                                     uint64_t* __restrict__ out, int* __restrict__ d_total) {
  __shared__ unsigned long long sm[33];
  unsigned long long before, total;
  chunk_offsets(sums, gridDim.x, blockIdx.x, sm, &before, &total);
  int64_t lo, hi;
  block_chunk(n, gridDim.x, blockIdx.x, 256, &lo, &hi);
  int64_t run = (int64_t)before;
  for (int64_t t0 = lo; t0 < hi; t0 += 256) {
    const int64_t i = t0 + threadIdx.x;
    const bool keep = i < hi && lin_keep<DIM>(maxl, keys, i, n);
    unsigned long long tot;
    unsigned long long ex = block_excl_scan<unsigned long long>(keep ? 1 : 0, sm, &tot);
    if (keep) out[run + (int64_t)ex] = keys[i];
    run += (int64_t)tot;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) *d_total = (int)total;
}

int linearise_keys(int dim, int maxl, const uint64_t* d_in, uint64_t* d_out, int64_t n, int64_t* n_out,
                   unsigned long long* d_sums, int* d_total, int* h_total, int G, cudaStream_t s,
                   int64_t* launches) {
  if (n == 0) {
    *n_out = 0;
    return LT_OK;
  }
  if (dim == 2) {
    k_lin_count<2><<<G, 256, 0, s>>>(maxl, d_in, n, d_sums);
    k_lin_scatter<2><<<G, 256, 0, s>>>(maxl, d_in, n, d_sums, d_out, d_total);
  } else {
    k_lin_count<3><<<G, 256, 0, s>>>(maxl, d_in, n, d_sums);
    k_lin_scatter<3><<<G, 256, 0, s>>>(maxl, d_in, n, d_sums, d_out, d_total);
  }
  *launches += 2;
  LT_CUDA(cudaGetLastError());
  LT_CUDA(cudaMemcpyAsync(h_total, d_total, sizeof(int), cudaMemcpyDeviceToHost, s));
  LT_CUDA(cudaStreamSynchronize(s));
  *n_out = *h_total;
  return LT_OK;
}

}  // namespace lt
