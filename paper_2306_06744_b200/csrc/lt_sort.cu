// lt_sort.cu -- ascending LSD radix sort of uint64 Morton IDs and linearisation (Alg. 3,
// PAPER.md:122-128) for sm_100a.  Replaces the paper's thrust::sort / thrust::unique
// (PAPER.md:117, :126-128, :161, :223).  Product code.
//
// One-sweep design: one histogram kernel counts all digits of all passes; each pass is a
// single persistent kernel in which a block ranks a tile of 4096 keys (ballots over the digit bits +
// per-warp digit counters in shared memory), publishes its per-digit counts and obtains the counts
// of all earlier tiles by decoupled look-back, then scatters -- while the copy engine (cp.async.bulk +
// mbarrier) already brings in the block's next tile.  Only bits [0, key_bits) are sorted.
#include <mutex>

#include "lt_internal.h"

namespace lt {

constexpr int ST = 256;                 // threads per sort block (= number of digit values)
constexpr int SITEMS = 16;              // keys per thread (8: 4.2 -> 6.9 ms for 64 M keys, the per-tile look-back dominates)
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

// ---- TMA (bulk asynchronous copy) plumbing: one thread arms an mbarrier with the byte count of a tile and
// issues cp.async.bulk global -> shared; the copy engine signals the barrier when the bytes have landed.
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

struct SortSmem {
  alignas(128) uint64_t in[2][STILE];  // double-buffered input tiles (bulk-copy destinations)
  uint64_t out[STILE];                 // the tile reordered by digit
  unsigned wcnt[(ST / 32) * 256];
  unsigned gbase[256];
  unsigned loff[256];
  unsigned scan[33];
  unsigned ntile;
  int tile[2];
  alignas(8) uint64_t bar[2];
};

// One radix pass, PERSISTENT: a block takes tiles through a ticket and keeps TWO in flight -- while it ranks
// and scatters tile k out of one shared-memory buffer, the copy engine fills the other buffer with the tile
// of its next ticket (cp.async.bulk + mbarrier), so the DRAM latency of a tile load hides behind the
// ranking of the previous one.  Keys are re-read from shared memory where they are needed instead of
// being held in 16 x 2 registers per thread.  bulk == 0 (input not 16-byte aligned): the tile is loaded
// by the threads instead.
__global__ void __launch_bounds__(ST, 2) k_sort_pass(const uint64_t* __restrict__ in, uint64_t* __restrict__ out,
                                                  int64_t n, int shift, const unsigned* __restrict__ base,
                                                  volatile unsigned* status, int* ticket, int bulk) {
  extern __shared__ __align__(128) unsigned char sort_smem_raw[];
  SortSmem& S = *reinterpret_cast<SortSmem*>(sort_smem_raw);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const unsigned lt_mask = (1u << lane) - 1;
  const int ntiles = (int)((n + STILE - 1) / STILE);
  auto tile_count = [&](int t) { return (int)min((int64_t)STILE, n - (int64_t)t * STILE); };
  auto issue = [&](int buf, int t) {  // (one thread) request tile t into buffer buf
    const int cnt = tile_count(t);
    const uint32_t bytes = (uint32_t)(cnt * 8) & ~15u;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // earlier reads of the buffer are done
    mbar_arrive_expect_tx(&S.bar[buf], bytes);
    if (bytes) bulk_g2s(S.in[buf], in + (size_t)t * STILE, bytes, &S.bar[buf]);
  };
  if (threadIdx.x == 0) {
    mbar_init(&S.bar[0], 1);
    mbar_init(&S.bar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    const int t = atomicAdd(ticket, 1);
    S.tile[0] = t;
    if (bulk && t < ntiles) issue(0, t);
  }
  __syncthreads();
  for (int it = 0;; ++it) {
    const int b = it & 1;
    const int tile = S.tile[b];
    if (tile >= ntiles) break;
    const int cnt = tile_count(tile);
    if (threadIdx.x == 0) {  // the next ticket: its tile travels while this one is ranked
      const int t = atomicAdd(ticket, 1);
      S.tile[b ^ 1] = t;
      if (bulk && t < ntiles) issue(b ^ 1, t);
    }
    for (int i = threadIdx.x; i < (ST / 32) * 256; i += ST) S.wcnt[i] = 0;
    const uint64_t* sk = S.in[b];
    if (bulk) {
      while (!mbar_try_wait(&S.bar[b], (uint32_t)((it >> 1) & 1))) {
      }
      if ((cnt & 1) && threadIdx.x == 0) S.in[b][cnt - 1] = in[(size_t)tile * STILE + cnt - 1];  // odd tail key
    } else {
      for (int i = threadIdx.x; i < cnt; i += ST) S.in[b][i] = in[(size_t)tile * STILE + i];
    }
    __syncthreads();
    // stable rank of every key among the equal-digit keys of its warp (warp-striped order); peers by
    // ballots over the digit bits (MATCH.ANY's latency grows with the number of distinct values)
    unsigned rank[SITEMS];
    unsigned digs[SITEMS / 4];  // the 16 digits of this thread, one byte each
#pragma unroll
    for (int k = 0; k < SITEMS / 4; ++k) digs[k] = 0;
    const int i0 = w * 32 * SITEMS + lane;
    const bool full = cnt == STILE;
#pragma unroll
    for (int k = 0; k < SITEMS; ++k) {
      const int idx = i0 + k * 32;
      const bool valid = full || idx < cnt;
      const int dig = valid ? (int)((sk[idx] >> shift) & 255) : 0;
      digs[k >> 2] |= (unsigned)dig << (8 * (k & 3));
      unsigned pm = 0xffffffffu;
#pragma unroll
      for (int bb = 0; bb < 8; ++bb) {
        const bool bit = (dig >> bb) & 1;
        const unsigned vote = __ballot_sync(0xffffffffu, bit);
        pm &= bit ? vote : ~vote;
      }
      if (!full) {
        const unsigned vv = __ballot_sync(0xffffffffu, valid);
        pm &= valid ? vv : ~vv;
      }
      const unsigned before = __popc(pm & lt_mask);
      unsigned pre = 0;
      if (valid) pre = S.wcnt[w * 256 + dig];
      __syncwarp();
      if (valid && before == 0) S.wcnt[w * 256 + dig] = pre + __popc(pm);
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
        unsigned c = S.wcnt[ww * 256 + d];
        S.wcnt[ww * 256 + d] = run;
        run += c;
      }
      unsigned excl = 0;
      if (tile == 0) {
        st_status(status + d, run | FLAG_INC);
      } else {
        st_status(status + (size_t)tile * 256 + d, run | FLAG_AGG);
        // look back over the earlier tiles, LB status words per round trip (independent loads)
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
      unsigned ntile;
      const unsigned tex = block_excl_scan<unsigned>(run, S.scan, &ntile);
      S.loff[d] = tex;
      S.gbase[d] = base[d] + excl - tex;
      if (d == 0) S.ntile = ntile;
    }
    __syncthreads();
    // reorder the tile by digit in shared memory, then write it out in tile order: consecutive threads
    // store consecutive addresses inside every digit run
#pragma unroll
    for (int k = 0; k < SITEMS; ++k) {
      const int idx = i0 + k * 32;
      if (full || idx < cnt) {
        const int dig = (int)((digs[k >> 2] >> (8 * (k & 3))) & 255);
        const unsigned pos = S.loff[dig] + S.wcnt[w * 256 + dig] + rank[k];
        LT_DASSERT(pos < (unsigned)STILE);
        S.out[pos] = sk[idx];
      }
    }
    __syncthreads();
    LT_DASSERT((int)S.ntile == cnt);
#pragma unroll
    for (int k = 0; k < SITEMS; ++k) {
      const int i = k * ST + threadIdx.x;
      if (i < cnt) {
        const uint64_t kk = S.out[i];
        LT_DASSERT((int64_t)S.gbase[(int)((kk >> shift) & 255)] + i < n);
        out[(size_t)S.gbase[(int)((kk >> shift) & 255)] + i] = kk;
      }
    }
    __syncthreads();  // S.out, S.wcnt, S.in[b] and S.tile[b] are reused
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
  static int per_sm = 0;
  if (per_sm == 0) {
    LT_CUDA(cudaFuncSetAttribute(k_sort_pass, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem)));
    LT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_sort_pass, ST, sizeof(SortSmem)));
    if (per_sm < 1) per_sm = 1;
  }
  int num_sms = 148, dev = 0;
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev);
  const int G = (int)(tiles < (int64_t)num_sms * per_sm ? tiles : (int64_t)num_sms * per_sm);
  for (int p = 0; p < passes; ++p) {
    LT_CUDA(cudaMemsetAsync(sc->status, 0, (size_t)tiles * 256 * sizeof(unsigned), s));
    const int bulk = (((uintptr_t)src) & 15) == 0;  // cp.async.bulk needs 16-byte aligned addresses
    k_sort_pass<<<G, ST, sizeof(SortSmem), s>>>(src, dst, n, 8 * p, sc->hist + p * 256, sc->status, tickets + p, bulk);
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

// ------------------------------------------------------------------------ lt_sort_keys_static
// The radix sort with its scratch (ping-pong key buffer, digit histograms + tile tickets, look-back
// status words) in a file-scope device array instead of cudaMalloc'd buffers, for callers that may not
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

// set-up, once per device: the array's device address and the sort pass's shared-memory opt-in
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
    LT_CUDA(cudaFuncSetAttribute(k_sort_pass, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem)));
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
  // start at zero (histograms, tickets, the status words of every pass) on the stream itself.
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
