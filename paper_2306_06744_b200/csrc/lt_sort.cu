// lt_sort.cu -- ascending LSD radix sort of uint64 Morton IDs and linearisation (Alg. 3,
// PAPER.md:122-128) for sm_100a.  Replaces the paper's thrust::sort / thrust::unique
// (PAPER.md:117, :126-128, :161, :223).  Product code.
//
// One pass over an 8-bit digit = four launches, no inter-block waiting:
//   k_sort_tile_hist   per tile of 4096 keys: its 256 digit counts -> table[digit][tile]
//   k_scan_reduce / k_scan_apply   exclusive scan of the table in (digit, tile) order: entry (d, t)
//                      becomes the global position of the first key of tile t with digit d
//   k_sort_scatter     per tile: stable rank of every key among the tile's keys of its digit
//                      (peer masks by shared-memory atomicOr, per-warp digit counters), the tile
//                      reordered by digit in shared memory, coalesced write-out per digit run.
// Only bits [0, key_bits) are sorted.  (Rounds 1-2 used a one-sweep pass with decoupled look-back,
// in round 2 persistent with cp.async.bulk prefetch of the next tile: 0.84 ms per pass on 64 M keys
// whatever the loads did, because with ~300-450 resident blocks running in lock-step every tile
// looked back over most of the current wave -- about 18 status-word loads PER KEY.  Reading the keys
// a second time for the histogram costs 8 B per key and removes the serial dependency altogether.)
#include <cstddef>
#include <mutex>

#include "lt_internal.h"

namespace lt {

constexpr int ST = 256;                 // threads per sort block (= number of digit values)
constexpr int SITEMS = 16;              // keys per thread
constexpr int STILE = ST * SITEMS;      // keys per tile

// table[d * tiles + t] = number of keys of tile t whose digit is d
__global__ void __launch_bounds__(ST) k_sort_tile_hist(const uint64_t* __restrict__ in, int64_t n, int shift,
                                                       int tiles, unsigned* __restrict__ table) {
  __shared__ unsigned sh[(ST / 32) * 256];  // one histogram per warp: fewer same-address atomics
  const int w = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < (ST / 32) * 256; i += ST) sh[i] = 0;
  __syncthreads();
  const int t = blockIdx.x;
  const int64_t i0 = (int64_t)t * STILE;
  uint64_t k[SITEMS];
#pragma unroll
  for (int q = 0; q < SITEMS; ++q) {
    const int64_t i = i0 + q * ST + threadIdx.x;
    k[q] = i < n ? __ldg(in + i) : ~0ull;
  }
#pragma unroll
  for (int q = 0; q < SITEMS; ++q)
    if (i0 + q * ST + threadIdx.x < n) atomicAdd(&sh[w * 256 + (int)((k[q] >> shift) & 255)], 1u);
  __syncthreads();
  unsigned c = 0;
#pragma unroll
  for (int ww = 0; ww < ST / 32; ++ww) c += sh[ww * 256 + threadIdx.x];
  table[(size_t)threadIdx.x * tiles + t] = c;
}

// exclusive scan of a[0..L) in place, two kernels over G chunks (all partial sums < 2^30)
__global__ void __launch_bounds__(256) k_scan_reduce(const unsigned* __restrict__ a, int64_t L,
                                                     unsigned long long* __restrict__ sums) {
  __shared__ unsigned long long sm[33];
  int64_t lo, hi;
  block_chunk(L, gridDim.x, blockIdx.x, 1024, &lo, &hi);
  unsigned long long acc = 0;
  for (int64_t i = lo + threadIdx.x; i < hi; i += 256) acc += a[i];
  acc = block_sum(acc, sm);
  if (threadIdx.x == 0) sums[blockIdx.x] = acc;
}

__global__ void __launch_bounds__(256) k_scan_apply(unsigned* __restrict__ a, int64_t L,
                                                    const unsigned long long* __restrict__ sums) {
  __shared__ unsigned long long sm[33];
  __shared__ unsigned su[33];
  unsigned long long before, total;
  chunk_offsets(sums, gridDim.x, blockIdx.x, sm, &before, &total);
  int64_t lo, hi;
  block_chunk(L, gridDim.x, blockIdx.x, 1024, &lo, &hi);  // chunks are multiples of 1024: four per thread
  unsigned run = (unsigned)before;
  for (int64_t t0 = lo; t0 < hi; t0 += 1024) {
    const int64_t i = t0 + 4 * threadIdx.x;
    unsigned v[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) v[q] = i + q < hi ? a[i + q] : 0u;
    unsigned tot;
    unsigned ex = run + block_excl_scan<unsigned>(v[0] + v[1] + v[2] + v[3], su, &tot);
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      if (i + q < hi) a[i + q] = ex;
      ex += v[q];
    }
    run += tot;
  }
}

struct SortSmem {
  uint64_t out[STILE];             // the tile reordered by digit; before that: the peer masks
  unsigned wcnt[(ST / 32) * 256];  // per-warp digit counters
  unsigned gbase[256];
  unsigned scan[33];
};

// One tile of one pass.  Thread (w, lane) holds keys w * 512 + k * 32 + lane, k = 0..15 (warp-striped:
// coalesced loads, and ranks that follow the tile order).  Round k: every lane ORs its bit into the mask
// of its digit (match[k & 1][w][digit], shared memory); the mask read back is the set of lanes with that
// digit (what eight ballots over the digit bits delivered at three times the instruction count); every
// lane reads the warp's digit counter, then the lowest lane of each digit adds the number of its peers to
// the counter and clears the mask.  Rounds go in pairs, so that two chains of shared-memory round trips
// are in flight (the kernel stalls on those: ncu short-scoreboard).
template <bool FULL>
__device__ __forceinline__ void sort_scatter_tile(SortSmem& S, const uint64_t* __restrict__ in,
                                                  uint64_t* __restrict__ out, int cnt, int shift,
                                                  const unsigned* __restrict__ trow, int tiles) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const unsigned lt_mask = (1u << lane) - 1, bit = 1u << lane;
  const int i0 = w * 32 * SITEMS + lane;
  uint64_t key[SITEMS];
#pragma unroll
  for (int k = 0; k < SITEMS; ++k) key[k] = (FULL || i0 + k * 32 < cnt) ? __ldg(in + i0 + k * 32) : 0ull;
  unsigned* match = reinterpret_cast<unsigned*>(S.out);  // [2][ST / 32][256]
  {
    uint4* z = reinterpret_cast<uint4*>(S.out);  // (S.wcnt follows S.out: one run of 16 + 8 KB of zeros)
    static_assert(offsetof(SortSmem, wcnt) == sizeof(uint64_t) * STILE, "wcnt follows out");
    for (int i = threadIdx.x; i < (2 + 1) * (ST / 32) * 256 / 4; i += ST) {
      const int j = i < 2 * (ST / 32) * 256 / 4 ? i : i - 2 * (ST / 32) * 256 / 4 + (int)(sizeof(uint64_t) * STILE / 16);
      z[j] = make_uint4(0, 0, 0, 0);
    }
  }
  __syncthreads();
  volatile unsigned* mA = match + w * 256;             // masks of the even round of a pair
  volatile unsigned* mB = mA + (ST / 32) * 256;        // and of the odd round
  volatile unsigned* wc = S.wcnt + w * 256;
  unsigned rank[SITEMS / 2];  // two 16-bit ranks per word
#pragma unroll
  for (int k = 0; k < SITEMS; k += 2) {
    // two rounds at a time: two independent chains of shared-memory round trips per iteration
    const bool v0 = FULL || i0 + k * 32 < cnt, v1 = FULL || i0 + (k + 1) * 32 < cnt;
    const int d0 = (int)((key[k] >> shift) & 255), d1 = (int)((key[k + 1] >> shift) & 255);
    if (v0) atomicOr(const_cast<unsigned*>(mA) + d0, bit);
    if (v1) atomicOr(const_cast<unsigned*>(mB) + d1, bit);
    __syncwarp();
    const unsigned pm0 = v0 ? mA[d0] : 0u, pm1 = v1 ? mB[d1] : 0u;
    const unsigned x01 = v1 ? mA[d1] : 0u;  // the lanes whose even-round key has the digit of my odd-round key
    const unsigned c0 = wc[d0], c1 = wc[d1];
    __syncwarp();  // every lane has read its masks and counters
    if (v0 && (pm0 & lt_mask) == 0) {  // the lowest lane of a digit's peers: count them, clear the mask
      atomicAdd(const_cast<unsigned*>(wc) + d0, (unsigned)__popc(pm0));
      mA[d0] = 0;
    }
    if (v1 && (pm1 & lt_mask) == 0) {
      atomicAdd(const_cast<unsigned*>(wc) + d1, (unsigned)__popc(pm1));
      mB[d1] = 0;
    }
    __syncwarp();
    const unsigned r0 = c0 + __popc(pm0 & lt_mask);
    const unsigned r1 = c1 + __popc(x01) + __popc(pm1 & lt_mask);
    rank[k >> 1] = r0 | (r1 << 16);
  }
  __syncthreads();
  {
    // thread d owns digit d: prefix over the warps, prefix over the digits, global base of the digit run
    const int d = threadIdx.x;
    unsigned run = 0;
#pragma unroll
    unsigned c[ST / 32];
#pragma unroll
    for (int ww = 0; ww < ST / 32; ++ww) {
      c[ww] = S.wcnt[ww * 256 + d];
      run += c[ww];
    }
    const unsigned gpos = trow[(size_t)d * tiles];
    unsigned ntile;
    unsigned tex = block_excl_scan<unsigned>(run, S.scan, &ntile);
    LT_DASSERT((int)ntile == cnt);
    S.gbase[d] = gpos - tex;
    // wcnt[w][d] becomes the tile position of warp w's first key with digit d
#pragma unroll
    for (int ww = 0; ww < ST / 32; ++ww) {
      S.wcnt[ww * 256 + d] = tex;
      tex += c[ww];
    }
  }
  __syncthreads();
  // reorder the tile by digit in shared memory, then write it out in tile order: consecutive threads
  // store consecutive addresses inside every digit run
#pragma unroll
  for (int k = 0; k < SITEMS; ++k) {
    if (FULL || i0 + k * 32 < cnt) {
      const int dig = (int)((key[k] >> shift) & 255);
      const unsigned pos = S.wcnt[w * 256 + dig] + ((rank[k >> 1] >> (16 * (k & 1))) & 0xffffu);
      LT_DASSERT(pos < (unsigned)STILE);
      S.out[pos] = key[k];
    }
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < SITEMS; ++k) {
    const int i = k * ST + threadIdx.x;
    if (FULL || i < cnt) {
      const uint64_t kk = S.out[i];
      out[(size_t)S.gbase[(int)((kk >> shift) & 255)] + i] = kk;
    }
  }
}

__global__ void __launch_bounds__(ST, 3) k_sort_scatter(const uint64_t* __restrict__ in, uint64_t* __restrict__ out,
                                                        int64_t n, int shift, int tiles,
                                                        const unsigned* __restrict__ table) {
  __shared__ SortSmem S;
  const int tile = blockIdx.x;
  const int cnt = (int)min((int64_t)STILE, n - (int64_t)tile * STILE);
  if (cnt == STILE) sort_scatter_tile<true>(S, in + (size_t)tile * STILE, out, cnt, shift, table + tile, tiles);
  else sort_scatter_tile<false>(S, in + (size_t)tile * STILE, out, cnt, shift, table + tile, tiles);
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
  // sc->hist holds the G chunk sums of the table scan, sc->status the table itself: [256][tiles]
  unsigned long long* sums = (unsigned long long*)sc->hist;
  unsigned* table = sc->status;
  const int64_t L = tiles * 256;
  int num_sms = 148, dev = 0;
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
  int G = 4 * num_sms;
  if (G > 1024) G = 1024;  // (8 * 256 + 8) words of sc->hist = 1028 sums
  if ((int64_t)G * 1024 > L) G = (int)((L + 1023) / 1024);
  uint64_t* src = d_keys;
  uint64_t* dst = sc->tmp;
  for (int p = 0; p < passes; ++p) {
    k_sort_tile_hist<<<(int)tiles, ST, 0, s>>>(src, n, 8 * p, (int)tiles, table);
    k_scan_reduce<<<G, 256, 0, s>>>(table, L, sums);
    k_scan_apply<<<G, 256, 0, s>>>(table, L, sums);
    k_sort_scatter<<<(int)tiles, ST, 0, s>>>(src, dst, n, 8 * p, (int)tiles, table);
    *launches += 4;
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

// ------------------------------------------------------------------------ lt_sort_keys_static
// The radix sort with its scratch (ping-pong key buffer, chunk sums of the table scan, per-tile digit
// table) in a file-scope device array instead of cudaMalloc'd buffers, for callers that may not
// allocate (CUDA graph capture, serving loops).  Every GPU that loads the library holds the array
// until exit: 8 * 2^20 + 8448 + 2^18 bytes = 8.26 MiB for at most LT_SORT_STATIC_MAX_KEYS = 2^20 keys.
// In host code `g_sort_static` is a host-side stand-in, NOT a device address: the address the
// kernels get comes from cudaGetSymbolAddress, asked once per device with that device current.
constexpr int64_t kSortStaticMaxKeys = LT_SORT_STATIC_MAX_KEYS;
constexpr size_t kSortStaticTmpBytes = (size_t)kSortStaticMaxKeys * sizeof(uint64_t);
constexpr size_t kSortStaticHistBytes = ((8 * 256 + 8) * sizeof(unsigned) + 255) / 256 * 256;
constexpr size_t kSortStaticStatusBytes = (size_t)((kSortStaticMaxKeys + STILE - 1) / STILE) * 256 * sizeof(unsigned);
static __device__ __align__(256) unsigned char g_sort_static[kSortStaticTmpBytes + kSortStaticHistBytes +
                                                             kSortStaticStatusBytes];

// set-up, once per device: the array's device address
static int sort_static_base(unsigned char** base) {
  static std::mutex mu;
  static unsigned char* addr[64];
  int dev = -1;
  LT_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return LT_ERR_ARG;
  std::lock_guard<std::mutex> lk(mu);
  if (!addr[dev]) {
    unsigned char* ptr = nullptr;
    LT_CUDA(cudaGetSymbolAddress((void**)&ptr, g_sort_static));
    if (!ptr) return LT_ERR_CUDA;
    addr[dev] = ptr;
  }
  *base = addr[dev];
  return LT_OK;
}

}  // namespace lt

extern "C" int lt_sort_keys_static(int dim, int max_level, uint64_t* d_keys, int64_t n, void* cuda_stream) {
  using namespace lt;
  if ((dim != 2 && dim != 3) || n < 0 || (n > 0 && !d_keys)) return LT_ERR_ARG;
  if (dim * max_level + kLevelBits > 63 || max_level < 0) return LT_ERR_ARG;
  if (n > kSortStaticMaxKeys) return LT_ERR_CAPACITY;  // beyond the static scratch: use lt_sort_keys
  if (n <= 1) return LT_OK;
  unsigned char* base = nullptr;
  const int rc = sort_static_base(&base);
  if (rc != LT_OK) return rc;
  // sort_keys allocates only when a buffer is missing or too small: none is.  It clears what must
  // start at zero itself (every pass overwrites the whole digit table and the chunk sums before it reads them).
  SortScratch sc;
  sc.tmp = (uint64_t*)base;
  sc.cap = kSortStaticMaxKeys;
  sc.hist = (unsigned*)(base + kSortStaticTmpBytes);
  sc.status = (unsigned*)(base + kSortStaticTmpBytes + kSortStaticHistBytes);
  sc.status_cap = (kSortStaticMaxKeys + STILE - 1) / STILE;
  sc.counter = nullptr;
  int64_t launches = 0;
  return sort_keys(d_keys, n, dim * max_level + kLevelBits, &sc, (cudaStream_t)cuda_stream, &launches);
}
