// lt_api.cu -- the C ABI of liblt (include/lt.h): argument checks, buffer management and
// the sequence of kernel launches behind each call.  Product code; no CPU fallback: every
// step of the path runs in the kernels of lt_tree.cu / lt_connect.cu / lt_transfer.cu /
// lt_sort.cu / lt_construct.cu.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <new>
#include <vector>

#include "lt_internal.h"

namespace lt {

thread_local int g_last_cuda_error = 0;

// Device memory comes from the device's default stream-ordered pool (cudaMallocAsync): a
// freed block is reused by the next allocation on the tree's stream without a driver call,
// so building a tree (two dozen buffers) costs microseconds of allocation once the pool is
// warm.  The pool keeps at most kPoolKeepBytes cached across synchronisation points.
constexpr unsigned long long kPoolKeepBytes = 8ull << 30;

static void pool_setup() {
  static thread_local int done_for = -1;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev == done_for) return;
  cudaMemPool_t pool;
  if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
    unsigned long long cur = 0;
    cudaMemPoolGetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &cur);
    if (cur < kPoolKeepBytes) {
      unsigned long long keep = kPoolKeepBytes;
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
  }
  cudaGetLastError();
  done_for = dev;
}

int dev_alloc(void** p, size_t bytes, cudaStream_t s) {
  *p = nullptr;
  if (bytes == 0) bytes = 16;
  pool_setup();
  LT_CUDA(cudaMallocAsync(p, bytes, s));
  return LT_OK;
}

void dev_free(void* p, cudaStream_t s) {
  if (p && cudaFreeAsync(p, s) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(p);
  }
}

static void free_dev(cudaStream_t s, void* p) { dev_free(p, s); }

// Pinned host mirrors (device scalars + chunk sums) are recycled through a small process-wide
// cache: cudaMallocHost / cudaFreeHost cost hundreds of microseconds each, which is most of the
// host time of building a tree from points.
constexpr size_t kMirrorBytes = 256 + (3 * kMaxGrid + 16) * sizeof(unsigned long long);
static std::mutex g_mirror_mu;
static std::vector<void*> g_mirror_free;

static void* mirror_get() {
  {
    std::lock_guard<std::mutex> lk(g_mirror_mu);
    if (!g_mirror_free.empty()) {
      void* p = g_mirror_free.back();
      g_mirror_free.pop_back();
      return p;
    }
  }
  void* p = nullptr;
  if (cudaMallocHost(&p, kMirrorBytes) != cudaSuccess) {
    cudaGetLastError();
    return nullptr;
  }
  return p;
}

static void mirror_put(void* p) {
  if (!p) return;
  std::lock_guard<std::mutex> lk(g_mirror_mu);
  if (g_mirror_free.size() < 16) g_mirror_free.push_back(p);
  else cudaFreeHost(p);
}

template <typename T>
static int alloc_dev(cudaStream_t s, T** p, int64_t count) {
  if (count <= 0) count = 1;
  return dev_alloc((void**)p, (size_t)count * sizeof(T), s);
}

static cudaError_t host_sync(Tree* t);
static int64_t round_cap(int64_t n) { return (n + 1023) / 1024 * 1024; }

// (Re)allocate every per-leaf buffer for `need` leaves, preserving the current keys, the
// snapshot and both bucket indices.
static int grow(Tree* t, int64_t need) {
  if (need <= t->cap) return LT_OK;
  if (need >= (1ll << 31) - 1024) return LT_ERR_CAPACITY;
  int64_t cap = round_cap(need + need / 4);
  if (cap >= (1ll << 31) - 1024) cap = round_cap(need);
  LT_CUDA(host_sync(t));
  const int dim = t->g.dim, nf = 2 * dim;
  uint64_t* nk[3] = {nullptr, nullptr, nullptr};
  uint8_t* mark = nullptr;
  uint64_t* fk[2] = {nullptr, nullptr};
  uint8_t* ft[2] = {nullptr, nullptr};
  // balance frontier: at most one entry per leaf that was split or flagged (< cap * 8 / 7 in total)
  const int64_t fcap = cap + cap / 4 + 1024;
  int32_t* nbr = nullptr;
  uint8_t* kind = nullptr;
  int32_t* msrc = nullptr;
  uint8_t* mkind = nullptr;
  int32_t* frows = nullptr;
  uint8_t* fbytes = nullptr;
  unsigned long long* tstate = nullptr;
  int rc = LT_OK;
  for (int b = 0; b < 3 && rc == LT_OK; ++b) rc = alloc_dev(t->stream, &nk[b], cap);
  if (rc == LT_OK) rc = alloc_dev(t->stream, &mark, cap);
  for (int b = 0; b < 2 && rc == LT_OK; ++b) {
    rc = alloc_dev(t->stream, &fk[b], fcap);
    if (rc == LT_OK) rc = alloc_dev(t->stream, &ft[b], fcap + 4);
  }
  if (rc == LT_OK) rc = alloc_dev(t->stream, &nbr, cap * nf);
  if (rc == LT_OK) rc = alloc_dev(t->stream, &kind, cap * nf);
  if (rc == LT_OK) rc = alloc_dev(t->stream, &msrc, cap);
  if (rc == LT_OK) rc = alloc_dev(t->stream, &mkind, cap);
  // face-table pool with fixed regions (lt_connect.cu face_regions): n_conf, n_hang <= dim*M
  // rows of 2 int32, n_bnd <= nf*M rows of 1 int32, one byte per row
  if (rc == LT_OK) rc = alloc_dev(t->stream, &frows, cap * (4 * dim + nf));
  if (rc == LT_OK) rc = alloc_dev(t->stream, &fbytes, cap * (2 * dim + nf));
  if (rc == LT_OK) rc = alloc_dev(t->stream, &tstate, 2 * (cap / 256 + 2));
  if (rc != LT_OK) {
    for (int b = 0; b < 3; ++b) free_dev(t->stream, nk[b]);
    free_dev(t->stream, mark); free_dev(t->stream, fk[0]); free_dev(t->stream, fk[1]); free_dev(t->stream, ft[0]); free_dev(t->stream, ft[1]); free_dev(t->stream, nbr); free_dev(t->stream, kind); free_dev(t->stream, msrc); free_dev(t->stream, mkind);
    free_dev(t->stream, frows); free_dev(t->stream, fbytes); free_dev(t->stream, tstate);
    return rc;
  }
  if (t->keys[t->cur] && t->n_valid && t->n > 0)
    LT_CUDA(cudaMemcpyAsync(nk[t->cur], t->keys[t->cur], (size_t)t->n * 8, cudaMemcpyDeviceToDevice, t->stream));
  if (t->keys[t->old] && t->have_old && t->n_old > 0)
    LT_CUDA(cudaMemcpyAsync(nk[t->old], t->keys[t->old], (size_t)t->n_old * 8, cudaMemcpyDeviceToDevice, t->stream));
  LT_CUDA(cudaMemsetAsync(mark, 0, (size_t)cap, t->stream));
  LT_CUDA(host_sync(t));
  for (int b = 0; b < 3; ++b) {
    free_dev(t->stream, t->keys[b]);
    t->keys[b] = nk[b];
  }
  free_dev(t->stream, t->mark); t->mark = mark;
  for (int b = 0; b < 2; ++b) {
    free_dev(t->stream, t->fkey[b]); t->fkey[b] = fk[b];
    free_dev(t->stream, t->ftag[b]); t->ftag[b] = ft[b];
  }
  t->fcap = fcap;
  free_dev(t->stream, t->nbr); t->nbr = nbr;
  free_dev(t->stream, t->kind); t->kind = kind;
  free_dev(t->stream, t->map_src); t->map_src = msrc;
  free_dev(t->stream, t->map_kind); t->map_kind = mkind;
  free_dev(t->stream, t->face_rows); t->face_rows = frows;
  free_dev(t->stream, t->face_bytes); t->face_bytes = fbytes;
  free_dev(t->stream, t->tile_state); t->tile_state = tstate;
  t->map_valid = false;
  t->map_ready = false;
  t->faces_valid = false;
  t->front_ok = false;  // the frontier buffers were reallocated
  t->cap = cap;
  return LT_OK;
}

// every wait of the host for the tree's stream goes through here (lt_host_syncs counts them)
static cudaError_t host_sync(Tree* t) {
  t->host_syncs++;
  return cudaStreamSynchronize(t->stream);
}

// copy the device scalars to the pinned mirror and wait
static int fetch_scalars(Tree* t) {
  LT_CUDA(cudaMemcpyAsync(t->h_s, t->d_s, sizeof(DevScalars), cudaMemcpyDeviceToHost, t->stream));
  LT_CUDA(host_sync(t));
  t->n = t->h_s->n;
  t->n_valid = true;
  if (t->parity_pending) {  // an lt_balance that did not wait: which key buffer holds its result
    if (t->h_s->parity) {
      const int c = t->cur;
      t->cur = t->tmp;
      t->tmp = c;
    }
    t->parity_pending = false;
  }
  return LT_OK;
}

static int take_status(Tree* t) {
  int st = t->h_s->status;
  if (st != 0) {
    cudaMemsetAsync(&t->d_s->status, 0, sizeof(int), t->stream);
    t->h_s->status = 0;
  }
  return st;
}

// the face query's own sticky word (k_connect may run beside lt_transfer on the side stream)
static int take_status_connect(Tree* t) {
  int st = t->h_s->status_c;
  if (st != 0) {
    cudaMemsetAsync(&t->d_s->status_c, 0, sizeof(int), t->stream);
    t->h_s->status_c = 0;
  }
  return st;
}

int check_device(const Tree* t) {
  int dev = -1;
  LT_CUDA(cudaGetDevice(&dev));
  return dev == t->device ? LT_OK : LT_ERR_ARG;
}

static void tic(Tree* t, int which) { cudaEventRecord(t->ev[2 * which], t->stream); }
static void toc(Tree* t, int which) {
  cudaEventRecord(t->ev[2 * which + 1], t->stream);
  t->ev_set[which] = true;
}

static int new_tree(int dim, int base, int maxl, const double* domain, const int* periodic, void* stream,
                    Tree** out, const int* nroot = nullptr) {
  if (!out) return LT_ERR_ARG;
  *out = nullptr;
  if (dim != 2 && dim != 3) return LT_ERR_ARG;
  if (base < 0 || maxl < base) return LT_ERR_ARG;
  // the brick of root cubes: the cube index takes tbits key bits above the path bits, and the
  // global integer coordinates (nroot[a] << maxl) must fit 31 bits
  int64_t ntrees = 1;
  for (int a = 0; a < dim; ++a) {
    const int na = nroot ? nroot[a] : 1;
    if (na < 1 || ((int64_t)na << maxl) > (1ll << 31)) return LT_ERR_ARG;
    ntrees *= na;
    if (ntrees > (1ll << 24)) return LT_ERR_ARG;
  }
  int tbits = 0;
  while ((1ll << tbits) < ntrees) ++tbits;
  if (dim * maxl + kLevelBits + tbits > 63 || maxl > 29) return LT_ERR_ARG;
  if ((int64_t)dim * base + tbits > 30) return LT_ERR_ARG;  // the base leaves must fit an int32 index
  int dev = 0;
  LT_CUDA(cudaGetDevice(&dev));
  lt_tree* t = new (std::nothrow) lt_tree();
  if (!t) return LT_ERR_OOM;
  memset((void*)t, 0, sizeof(lt_tree));
  t->device = dev;
  t->stream = (cudaStream_t)stream;
  cudaError_t e = cudaDeviceGetAttribute(&t->num_sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) {
    g_last_cuda_error = (int)e;
    delete t;
    return LT_ERR_CUDA;
  }
  Geo& g = t->g;
  g.dim = dim;
  g.base = base;
  g.maxl = maxl;
  // bucket index one level below the base tree (buckets of at most 2^(dim*(maxl-base-1)) keys),
  // of at most 2^24 cells
  g.ilevel = base + 1 <= maxl ? base + 1 : maxl;
  while (g.ilevel > 0 && dim * g.ilevel + tbits > 24) --g.ilevel;
  g.ishift = dim * (maxl - g.ilevel);
  g.nbuckets = (int)(ntrees << (dim * g.ilevel));
  g.tshift = dim * maxl;
  g.ntrees = (int)ntrees;
  g.keybits = dim * maxl + kLevelBits + tbits;
  for (int a = 0; a < 3; ++a) g.nroot[a] = (nroot && a < dim) ? nroot[a] : 1;
  g.periodic = 0;
  for (int a = 0; a < dim; ++a)
    if (periodic && periodic[a]) g.periodic |= 1 << a;
  g.total = (1ull << (dim * maxl)) - 1;
  for (int a = 0; a < dim; ++a) {
    t->domain[a] = domain ? domain[a] : 0.0;
    t->domain[dim + a] = domain ? domain[dim + a] : 1.0;
  }
  t->cur = 0;
  t->old = 1;
  t->tmp = 2;
  t->ops_p = -1;
  int rc = LT_OK;
  auto fail = [&](int code) {
    lt_free(t);
    return code;
  };
  for (int b = 0; b < 3; ++b)
    if ((rc = alloc_dev(t->stream, &t->first[b], (int64_t)g.nbuckets + 1)) != LT_OK) return fail(rc);
  if ((rc = alloc_dev(t->stream, &t->d_s, 1)) != LT_OK) return fail(rc);
  if ((rc = alloc_dev(t->stream, &t->d_sums, kMaxGrid)) != LT_OK) return fail(rc);
  if ((rc = alloc_dev(t->stream, &t->d_sums3, 3 * kMaxGrid)) != LT_OK) return fail(rc);
  if ((rc = alloc_dev(t->stream, &t->d_cmarks, 2 * kMaxGrid)) != LT_OK) return fail(rc);
  if (cudaMemsetAsync(t->d_cmarks, 0, 2 * kMaxGrid * sizeof(int), t->stream) != cudaSuccess) return fail(LT_ERR_CUDA);
  static_assert(sizeof(DevScalars) <= 256, "mirror layout");
  t->h_s = (DevScalars*)mirror_get();  // one pinned block: scalars | chunk sums
  if (!t->h_s) return fail(LT_ERR_OOM);
  t->h_sums = (int*)((char*)t->h_s + 256);
  memset(t->h_s, 0, sizeof(DevScalars));
  if (cudaMemsetAsync(t->d_s, 0, sizeof(DevScalars), t->stream) != cudaSuccess) return fail(LT_ERR_CUDA);
  for (int i = 0; i < 16; ++i)
    if (cudaEventCreate(&t->ev[i]) != cudaSuccess) return fail(LT_ERR_CUDA);
  *out = t;
  return LT_OK;
}

// Alg. 2 behind lt_build_complete_from_keys / lt_build_from_points: `work` holds n unsorted
// keys (device, owned by the caller).  Radix sort, linearise (Alg. 3), then the completed
// tree is written in Morton order straight into the tree's key buffer (lt_construct.cu).
static int complete_from_unsorted(Tree* t, uint64_t* work, int64_t n) {
  const int dim = t->g.dim, maxl = t->g.maxl;
  SortScratch sc = {nullptr, 0, nullptr, nullptr, 0, nullptr};
  int rc = sort_keys(work, n, dim * maxl + kLevelBits, &sc, t->stream, &t->launches);
  t->sort_tmp = sc.tmp; t->sort_cap = sc.cap; t->sort_hist = sc.hist; t->sort_status = sc.status;
  t->sort_status_cap = sc.status_cap;
  if (rc != LT_OK) return rc;
  uint64_t* lin = nullptr;
  uint32_t* offs = nullptr;
  if ((rc = alloc_dev(t->stream, &lin, n)) != LT_OK) return rc;
  auto done = [&](int code) {
    host_sync(t);
    free_dev(t->stream, lin);
    free_dev(t->stream, offs);
    return code;
  };
  int64_t m = 0, total = 0;
  rc = linearise_keys(dim, maxl, work, lin, n, &m, t->d_sums, &t->d_s->aux, (int*)t->h_sums, grid_for(t, 4),
                      t->stream, &t->launches);
  if (rc != LT_OK) return done(rc);
  if ((rc = alloc_dev(t->stream, &offs, m + 2)) != LT_OK) return done(rc);
  if ((rc = launch_complete_count(t, lin, m, offs, &total)) != LT_OK) return done(rc);
  const int st = take_status(t);
  if (st != LT_OK) return done(st);
  if (total >= (1ll << 31) - 1024) return done(LT_ERR_CAPACITY);
  if ((rc = grow(t, total)) != LT_OK) return done(rc);
  if ((rc = launch_complete_fill(t, lin, m, offs, total)) != LT_OK) return done(rc);
  t->n = total;
  t->n_valid = true;
  if ((rc = launch_build_index(t, t->cur)) != LT_OK) return done(rc);
  return done(LT_OK);
}

}  // namespace lt

using namespace lt;

// main stream waits for an lt_connect_begin that has not been collected yet
static int join_side(Tree* t) {
  if (t->connect_pending) {
    LT_CUDA(cudaStreamWaitEvent(t->stream, t->ev_side_join, 0));
    t->connect_pending = false;
  }
  return LT_OK;
}

extern "C" {

int lt_version(void) { return 200; }
int lt_debug_build(void) {
#ifdef LT_DEBUG
  return 1;
#else
  return 0;
#endif
}
int lt_last_cuda_error(void) { return g_last_cuda_error; }

const char* lt_strerror(int status) {
  switch (status) {
    case LT_OK: return "ok";
    case LT_ERR_ARG: return "bad argument";
    case LT_ERR_CUDA: return "CUDA runtime error (no device, or a launch failed)";
    case LT_ERR_OOM: return "out of device memory";
    case LT_ERR_CAPACITY: return "device buffer capacity exceeded";
    case LT_ERR_UNBALANCED: return "tree is not 2:1 face balanced";
    case LT_ERR_MAPPING: return "a new leaf is more than one level from the old tree";
    case LT_ERR_INCOMPLETE: return "keys do not tile the domain";
  }
  return "unknown status";
}

void lt_free(lt_tree* t) {
  if (!t) return;
  if (t->s_side) {
    cudaStreamSynchronize(t->s_side);
    cudaStreamDestroy(t->s_side);
    cudaEventDestroy(t->ev_side_fork);
    cudaEventDestroy(t->ev_side_join);
  }
  host_sync(t);
  for (int b = 0; b < 3; ++b) {
    free_dev(t->stream, t->keys[b]);
    free_dev(t->stream, t->first[b]);
  }
  free_dev(t->stream, t->d_s); free_dev(t->stream, t->d_sums); free_dev(t->stream, t->d_sums3);
  mirror_put(t->h_s);
  free_dev(t->stream, t->mark); free_dev(t->stream, t->d_cmarks);
  for (int b = 0; b < 2; ++b) {
    free_dev(t->stream, t->fkey[b]);
    free_dev(t->stream, t->ftag[b]);
  }
  free_dev(t->stream, t->nbr); free_dev(t->stream, t->kind);
  free_dev(t->stream, t->face_rows); free_dev(t->stream, t->face_bytes); free_dev(t->stream, t->tile_state);
  free_dev(t->stream, t->map_src); free_dev(t->stream, t->map_kind); free_dev(t->stream, t->d_ops);
  for (int r = 0; r < Tree::kRing; ++r) {
    free_dev(t->stream, t->ring_old[r]);
    free_dev(t->stream, t->ring_new[r]);
    if (t->ev_in[r]) cudaEventDestroy(t->ev_in[r]);
    if (t->ev_done[r]) cudaEventDestroy(t->ev_done[r]);
    if (t->ev_out[r]) cudaEventDestroy(t->ev_out[r]);
  }
  free_dev(t->stream, t->mortar_hits);
  free_dev(t->stream, t->d_bounds);
  if (t->h_bounds) cudaFreeHost(t->h_bounds);
  if (t->s_in) cudaStreamDestroy(t->s_in);
  if (t->s_out) cudaStreamDestroy(t->s_out);
  free_dev(t->stream, t->sort_tmp); free_dev(t->stream, t->sort_hist); free_dev(t->stream, t->sort_status);
  for (int i = 0; i < 16; ++i)
    if (t->ev[i]) cudaEventDestroy(t->ev[i]);
  delete t;
}

int lt_build(int dim, int base_level, int max_level, const double* domain, const int* periodic,
             void* cuda_stream, lt_tree** out) {
  return lt_build_brick(dim, nullptr, base_level, max_level, domain, periodic, cuda_stream, out);
}

int lt_roots(lt_tree* t, int* nroot) {
  if (!t || !nroot) return LT_ERR_ARG;
  for (int a = 0; a < 3; ++a) nroot[a] = t->g.nroot[a];
  return LT_OK;
}

int lt_build_brick(int dim, const int* nroot, int base_level, int max_level, const double* domain,
                   const int* periodic, void* cuda_stream, lt_tree** out) {
  Tree* t = nullptr;
  int rc = new_tree(dim, base_level, max_level, domain, periodic, cuda_stream, &t, nroot);
  if (rc != LT_OK) return rc;
  const int64_t nb = (int64_t)t->g.ntrees << (dim * base_level);
  if ((rc = grow(t, nb * 2)) != LT_OK) {
    lt_free((lt_tree*)t);
    return rc;
  }
  if ((rc = launch_build_uniform(t)) != LT_OK) {
    lt_free((lt_tree*)t);
    return rc;
  }
  t->n = nb;
  t->n_valid = true;
  *out = (lt_tree*)t;
  t->balanced_conn = 3;  // a uniform tree is balanced for every connectivity
  return LT_OK;
}

int lt_reserve(lt_tree* t, int64_t n_leaves) {
  if (t && join_side(t) != LT_OK) return LT_ERR_CUDA;
  if (!t || n_leaves < 0) return LT_ERR_ARG;
  if (!t->n_valid) {
    int rc = fetch_scalars(t);
    if (rc != LT_OK) return rc;
  }
  return grow(t, n_leaves);
}

int64_t lt_num_leaves(lt_tree* t) {
  if (!t) return LT_ERR_ARG;
  if (!t->n_valid) {
    int rc = fetch_scalars(t);
    if (rc != LT_OK) return rc;
  }
  return t->n;
}
int64_t lt_num_old_leaves(lt_tree* t) { return t && t->have_old ? t->n_old : 0; }
const uint64_t* lt_keys(lt_tree* t) {
  if (!t) return nullptr;
  if (!t->n_valid && fetch_scalars(t) != LT_OK) return nullptr;  // (settles which buffer is current)
  return t->keys[t->cur];
}
int lt_last_balance_iters(lt_tree* t) {
  if (!t) return LT_ERR_ARG;
  if (!t->n_valid) {
    int rc = fetch_scalars(t);
    if (rc != LT_OK) return rc;
  }
  return t->last_iters >= 0 ? t->last_iters : t->h_s->iters;
}
const uint64_t* lt_old_keys(lt_tree* t) { return t && t->have_old ? t->keys[t->old] : nullptr; }

int lt_domain(lt_tree* t, double* lo_hi) {
  if (!t || !lo_hi) return LT_ERR_ARG;
  for (int a = 0; a < 2 * t->g.dim; ++a) lo_hi[a] = t->domain[a];
  return LT_OK;
}
int lt_info(lt_tree* t, int* dim, int* base_level, int* max_level, int* periodic) {
  if (!t) return LT_ERR_ARG;
  if (dim) *dim = t->g.dim;
  if (base_level) *base_level = t->g.base;
  if (max_level) *max_level = t->g.maxl;
  if (periodic)
    for (int a = 0; a < 3; ++a) periodic[a] = (t->g.periodic >> a) & 1;
  return LT_OK;
}

int lt_set_option(lt_tree* t, int option, int value) {
  if (!t) return LT_ERR_ARG;
  if (option == LT_OPT_ADAPT_SORT) t->opt_adapt_sort = value != 0;
  else if (option == LT_OPT_BALANCE_FULL_SWEEPS) t->opt_full_sweeps = value != 0;
  else if (option == LT_OPT_DEBUG_BALANCE_SLACK) t->opt_debug_slack = value > 0 ? value : 0;
  else if (option == LT_OPT_HOST_SLAB_LEAVES) t->opt_host_slab = value > 0 ? value : 0;
  else if (option == LT_OPT_BALANCE_CONNECTIVITY) {
    if (value < 1 || value > t->g.dim) return LT_ERR_ARG;
    t->opt_balance_conn = value;
  }
  else return LT_ERR_ARG;
  return LT_OK;
}

int lt_sync(lt_tree* t) {
  if (!t) return LT_ERR_ARG;
  int rc = fetch_scalars(t);
  if (rc != LT_OK) return rc;
  // a face query still running on the side stream keeps its word for lt_connect_end
  const int st = take_status(t), stc = t->connect_pending ? LT_OK : take_status_connect(t);
  return st != LT_OK ? st : stc;
}

int lt_timings(lt_tree* t, float* out8) {
  if (!t || !out8) return LT_ERR_ARG;
  LT_CUDA(host_sync(t));
  for (int i = 0; i < 8; ++i) {
    out8[i] = 0.f;
    if (t->ev_set[i]) LT_CUDA(cudaEventElapsedTime(&out8[i], t->ev[2 * i], t->ev[2 * i + 1]));
  }
  return LT_OK;
}
int64_t lt_launch_count(lt_tree* t) { return t ? t->launches : 0; }
int64_t lt_host_syncs(lt_tree* t) { return t ? t->host_syncs : 0; }

int lt_balance_phases(lt_tree* t, float* out4) {
  if (!t || !out4) return LT_ERR_ARG;
  for (int k = 0; k < 4; ++k) out4[k] = 1e-6f * (float)t->h_s->bal_ns[k];  // mirror filled by lt_balance
  return LT_OK;
}

int lt_leaf_boxes(lt_tree* t, int32_t* d_level, uint32_t* d_xyz) {
  if (!t) return LT_ERR_ARG;
  int rc;
  if (!t->n_valid && (rc = fetch_scalars(t)) != LT_OK) return rc;
  return launch_leaf_boxes(t, d_level, d_xyz);
}

int lt_encode(int dim, int max_level, const uint32_t* d_xyz, const int32_t* d_level, int64_t n,
              uint64_t* d_keys, void* cuda_stream) {
  if ((dim != 2 && dim != 3) || n < 0 || !d_xyz || !d_level || !d_keys) return LT_ERR_ARG;
  if (dim * max_level + kLevelBits > 63 || max_level > 29 || max_level < 0) return LT_ERR_ARG;
  return launch_encode(dim, max_level, d_xyz, d_level, n, d_keys, (cudaStream_t)cuda_stream);
}
int lt_decode(int dim, int max_level, const uint64_t* d_keys, int64_t n, int32_t* d_level, uint32_t* d_xyz,
              void* cuda_stream) {
  if ((dim != 2 && dim != 3) || n < 0 || !d_keys) return LT_ERR_ARG;
  return launch_decode(dim, max_level, d_keys, n, d_level, d_xyz, (cudaStream_t)cuda_stream);
}

// ---------------------------------------------------------------------------- adapt
int lt_adapt(lt_tree* t, const int8_t* d_flags) {
  if (!t || !d_flags) return LT_ERR_ARG;
  int rc;
  if ((rc = join_side(t)) != LT_OK) return rc;
  if (!t->n_valid && (rc = fetch_scalars(t)) != LT_OK) return rc;
  bool front_ok = false;
  tic(t, 0);
  // (a grid of exactly the blocks k_adapt_scatter keeps resident -- 5 per SM, one wave instead of 1.6 --
  // was measured: slower, 0.177 -> 0.193 ms under ncu; the smaller chunks of the larger grid balance better)
  const int G = grid_for(t, 8);
  if ((rc = launch_adapt_count(t, d_flags, G)) != LT_OK) return rc;
  const int nc = 1 << t->g.dim;
  if (!t->opt_adapt_sort && t->cap >= nc * t->n) {
    // The buffers hold the worst case (every leaf refined): nothing to size, so the host does not wait
    // for the new count -- it stays on the device until a call needs it (lt_num_leaves, lt_connect_end ...).
    const int emit = t->balanced_conn >= 1;
    if ((rc = launch_adapt_scatter(t, d_flags, G, 0, emit)) != LT_OK) return rc;
    const int o = t->old;
    t->old = t->cur;
    t->cur = t->tmp;
    t->tmp = o;
    t->have_old = true;
    t->n_old = t->n;
    t->n_upper = nc * t->n;
    t->n_valid = false;
    t->map_valid = false;
    t->map_ready = false;
    t->faces_valid = false;
    t->front_ok = emit != 0;
    t->front_conn = t->balanced_conn;
    t->balanced_conn = 0;
    toc(t, 0);
    return LT_OK;
  }
  // the new size is needed on the host to size buffers: one small read-back
  LT_CUDA(cudaMemcpyAsync(t->h_sums, t->d_sums, (size_t)G * sizeof(unsigned long long), cudaMemcpyDeviceToHost,
                          t->stream));
  LT_CUDA(host_sync(t));
  int64_t n_b = 0, n_kept = 0;
  const unsigned long long* hs = (const unsigned long long*)t->h_sums;
  for (int b = 0; b < G; ++b) {
    n_b += (int64_t)(hs[b] & 0xffffffffull);
    n_kept += (int64_t)(hs[b] >> 32);
  }
  const int64_t n_in = t->n;
  const int64_t need = t->opt_adapt_sort ? n_kept + n_b : n_b;
  if ((rc = grow(t, need)) != LT_OK) return rc;
  if (!t->opt_adapt_sort) {
    // path B: ordered expansion cur -> tmp.  If the tree was balanced, the leaves created here
    // become the frontier of lt_balance's first sweep.
    const int emit = t->balanced_conn >= 1;
    if ((rc = launch_adapt_scatter(t, d_flags, G, 0, emit)) != LT_OK) return rc;
    front_ok = emit != 0;
    const int o = t->old;
    t->old = t->cur;
    t->cur = t->tmp;
    t->tmp = o;
    t->n = n_b;
  } else {
    // path A (Alg. 6 as printed): append -> radix sort -> linearise
    LT_CUDA(cudaMemsetAsync(&t->d_s->aux, 0, sizeof(int), t->stream));
    if ((rc = launch_adapt_scatter(t, d_flags, G, 1, 0)) != LT_OK) return rc;
    if ((rc = fetch_scalars(t)) != LT_OK) return rc;
    t->n = n_in;  // fetch_scalars read the (unchanged) device count
    const int64_t n_app = n_kept + t->h_s->aux;
    SortScratch sc = {t->sort_tmp, t->sort_cap, t->sort_hist, t->sort_status, t->sort_status_cap, nullptr};
    rc = sort_keys(t->keys[t->tmp], n_app, t->g.keybits, &sc, t->stream, &t->launches);
    t->sort_tmp = sc.tmp; t->sort_cap = sc.cap; t->sort_hist = sc.hist; t->sort_status = sc.status;
    t->sort_status_cap = sc.status_cap;
    if (rc != LT_OK) return rc;
    int64_t n_lin = 0;
    // the previous snapshot buffer receives the result (the snapshot is being replaced)
    rc = linearise_keys(t->g.dim, t->g.maxl, t->keys[t->tmp], t->keys[t->old], n_app, &n_lin, t->d_sums,
                        &t->d_s->aux, (int*)t->h_sums, G, t->stream, &t->launches);
    if (rc != LT_OK) return rc;
    const int o = t->old;
    t->old = t->cur;
    t->cur = o;
    t->n = n_lin;
    int nn = (int)n_lin;
    LT_CUDA(cudaMemcpyAsync(&t->d_s->n, &nn, sizeof(int), cudaMemcpyHostToDevice, t->stream));
    LT_CUDA(host_sync(t));
    if ((rc = launch_build_index(t, t->cur)) != LT_OK) return rc;
  }
  t->have_old = true;
  t->n_old = n_in;
  t->n_valid = true;
  t->map_valid = false;
  t->map_ready = false;
  t->faces_valid = false;
  t->front_ok = front_ok;
  t->front_conn = t->balanced_conn;
  t->balanced_conn = 0;
  toc(t, 0);
  return LT_OK;
}

// ---------------------------------------------------------------------------- balance
int lt_balance(lt_tree* t, int* iters) {
  if (!t) return LT_ERR_ARG;
  int rc;
  if ((rc = join_side(t)) != LT_OK) return rc;
  t->last_iters = -1;
  // Without a sweep count to hand back, and when the buffers hold the largest tree the ripple can
  // produce -- a tree that was balanced before lt_adapt is never refined by more than one level
  // (reading C-5): at most 2^dim * n_old leaves -- the call does not wait for the kernel: the leaf
  // count and the buffer the result ends in stay on the device until a later call fetches them.
  if (!iters && t->front_ok && !t->parity_pending && t->opt_debug_slack == 0 && !t->opt_full_sweeps &&
      (t->opt_balance_conn <= 1) && t->have_old && t->cap >= (int64_t)(1 << t->g.dim) * t->n_old) {
    tic(t, 1);
    t->front_ok = false;
    if ((rc = launch_balance(t, t->cap, 1)) != LT_OK) return rc;
    t->parity_pending = true;
    t->n_valid = false;
    t->n_upper = (int64_t)(1 << t->g.dim) * t->n_old;
    t->balanced_conn = 1;
    t->map_valid = false;
    t->map_ready = true;   // k_transfer reports a mapping error found by the kernel's tail (map_bad)
    t->faces_valid = false;
    toc(t, 1);
    return LT_OK;
  }
  if (!t->n_valid && (rc = fetch_scalars(t)) != LT_OK) return rc;
  tic(t, 1);
  const bool had_front = t->front_ok;  // consumed by this call whatever happens
  t->front_ok = false;
  int total_iters = 0;
  int64_t slack = t->opt_debug_slack;
  for (int attempt = 0;; ++attempt) {
    // (testing aid: pretend the buffers hold only n + slack leaves, to exercise the retry)
    const int64_t cap_told = slack > 0 && t->n + slack < t->cap ? t->n + slack : t->cap;
    const int conn = t->opt_balance_conn > 0 ? t->opt_balance_conn : 1;
    // (lt_adapt's list is the whole first frontier only if the tree it adapted was balanced with at least
    // this connectivity)
    const int use_front = attempt == 0 && had_front && conn <= t->front_conn && !t->opt_full_sweeps;
    if ((rc = launch_balance(t, cap_told, use_front)) != LT_OK) return rc;
    if ((rc = fetch_scalars(t)) != LT_OK) return rc;
    if (t->h_s->parity) {
      const int c = t->cur;
      t->cur = t->tmp;
      t->tmp = c;
    }
    total_iters += t->h_s->iters;
    const int st = take_status(t);
    if (st == LT_OK) break;
    // (an interrupted kernel leaves marks and per-chunk counters behind)
    LT_CUDA(cudaMemsetAsync(t->d_cmarks, 0, 2 * kMaxGrid * sizeof(int), t->stream));
    if (st != LT_ERR_CAPACITY || attempt >= 40) {
      cudaMemsetAsync(t->mark, 0, (size_t)t->cap, t->stream);
      return st;
    }
    // the analogue of the paper's "perform the balance algorithm again" when the
    // allocated cap is exceeded: grow and continue from the valid,
    // partially balanced tree
    LT_CUDA(cudaMemsetAsync(t->mark, 0, (size_t)t->cap, t->stream));
    if (cap_told < t->cap) {
      slack *= 2;
      continue;
    }
    if ((rc = grow(t, t->cap * 2)) != LT_OK) return rc == LT_ERR_OOM ? LT_ERR_CAPACITY : rc;
  }
  if (iters) *iters = total_iters;
  t->last_iters = total_iters;
  t->front_ok = false;
  t->balanced_conn = t->opt_balance_conn > 0 ? t->opt_balance_conn : 1;
  t->map_valid = false;
  // Alg. 7 ran in the tail of the kernel; a mapping error is left to lt_transfer's checked k_map
  t->map_ready = t->have_old && t->h_s->map_bad == 0;
  t->faces_valid = false;
  toc(t, 1);
  return LT_OK;
}

// ---------------------------------------------------------------------------- connect
static int collect_faces(Tree* t, lt_faces* out) {
  int rc;
  if ((rc = fetch_scalars(t)) != LT_OK) return rc;
  const int st = take_status_connect(t);
  if (st != LT_OK) return st;
  const int64_t nc = t->h_s->n_face[0], nh = t->h_s->n_face[1], nb = t->h_s->n_face[2];
  out->n_leaves = t->n;
  out->n_conf = nc;
  out->n_hang = nh;
  out->n_bnd = nb;
  out->nbr = t->nbr;
  out->kind = t->kind;
  {
    int32_t *conf, *hang, *bnd;
    uint8_t *conf_axis, *hang_info, *bnd_face;
    face_regions(t, &conf, &conf_axis, &hang, &hang_info, &bnd, &bnd_face);
    out->conf = conf;
    out->conf_axis = conf_axis;
    out->hang = hang;
    out->hang_info = hang_info;
    out->bnd = bnd;
    out->bnd_face = bnd_face;
  }
  t->faces_valid = true;
  return LT_OK;
}

int lt_connect(lt_tree* t, lt_faces* out) {
  if (!t || !out) return LT_ERR_ARG;
  int rc;
  if ((rc = join_side(t)) != LT_OK) return rc;
  if (!t->n_valid && (rc = fetch_scalars(t)) != LT_OK) return rc;
  tic(t, 2);
  tic(t, 6);
  if ((rc = launch_connect(t, t->stream, 0)) != LT_OK) return rc;
  toc(t, 6);
  rc = collect_faces(t, out);
  toc(t, 2);
  return rc;
}

// The face query depends only on the balanced tree, and so does the solution transfer: begin
// enqueues k_connect on a side stream (a quarter of the SM resources, so that the HBM-bound
// transfer kernel launched next on the main stream runs beside it), end joins and reads the counts.
int lt_connect_begin(lt_tree* t) {
  if (!t) return LT_ERR_ARG;
  int rc;
  if ((rc = join_side(t)) != LT_OK) return rc;
  // (no wait for a pending leaf count / result buffer: k_connect reads both on the device)
  if (!t->s_side) {
    LT_CUDA(cudaStreamCreateWithFlags(&t->s_side, cudaStreamNonBlocking));
    LT_CUDA(cudaEventCreateWithFlags(&t->ev_side_fork, cudaEventDisableTiming));
    LT_CUDA(cudaEventCreateWithFlags(&t->ev_side_join, cudaEventDisableTiming));
  }
  t->faces_valid = false;
  LT_CUDA(cudaEventRecord(t->ev_side_fork, t->stream));
  LT_CUDA(cudaStreamWaitEvent(t->s_side, t->ev_side_fork, 0));
  cudaEventRecord(t->ev[12], t->s_side);
  // 2 resident blocks per SM (k_connect handles two leaves per thread at 64 registers, so two of its blocks
  // and two blocks of the transfer share an SM's registers): measured best on config 5 -- 1: the query
  // outlasts the transfer (15.7 ms), 3: the transfer loses more than the query gains; LT_SIDE_BLOCKS
  // overrides for experiments
  static const int side_blocks = getenv("LT_SIDE_BLOCKS") ? atoi(getenv("LT_SIDE_BLOCKS")) : 2;
  // (a small mesh -- the transfer beside it takes well under a millisecond -- gets every block: there
  // the query itself would become the critical path)
  const int64_t n_est = t->n_valid ? t->n : (t->n_upper >> t->g.dim);  // (n_upper is the 2^dim-fold worst case)
  if ((rc = launch_connect(t, t->s_side, n_est > (4 << 20) ? side_blocks : 0)) != LT_OK) return rc;
  cudaEventRecord(t->ev[13], t->s_side);
  t->ev_set[6] = true;
  t->ev_set[2] = false;  // the call has no duration of its own in this mode
  LT_CUDA(cudaEventRecord(t->ev_side_join, t->s_side));
  t->connect_pending = true;
  return LT_OK;
}

int lt_connect_end(lt_tree* t, lt_faces* out) {
  if (!t || !out || !t->connect_pending) return LT_ERR_ARG;
  int rc;
  if ((rc = join_side(t)) != LT_OK) return rc;
  return collect_faces(t, out);
}

// ---------------------------------------------------------------------------- mortars
static int mortar_call(lt_tree* t, int which, const double* d_in, double* d_out, int p, int nvars) {
  if (!t || !d_in || !d_out || p < 0 || p > 7 || nvars < 1) return LT_ERR_ARG;
  if (!t->faces_valid) return LT_ERR_ARG;  // lt_connect must describe the current tree
  int rc;
  if ((rc = build_operators(t, p)) != LT_OK) return rc;
  tic(t, 7);
  // the gather works from the list of coarse-side hanging faces (rebuilt per call: d_s->aux,
  // its counter, is shared scratch)
  if (which == 1 && (rc = launch_mortar_hits(t)) != LT_OK) return rc;
  if ((rc = launch_mortar(t, which, d_in, d_out, p, nvars)) != LT_OK) return rc;
  toc(t, 7);
  return LT_OK;
}

int lt_face_interp(lt_tree* t, const double* d_u, double* d_u_face, int p, int nvars) {
  if (!t || !d_u || !d_u_face || d_u == d_u_face || p < 0 || p > 7 || nvars < 1) return LT_ERR_ARG;
  int rc;
  if (!t->n_valid && (rc = fetch_scalars(t)) != LT_OK) return rc;
  if ((rc = build_operators(t, p)) != LT_OK) return rc;
  tic(t, 7);
  if ((rc = launch_face_interp(t, d_u, d_u_face, p, nvars)) != LT_OK) return rc;
  toc(t, 7);
  return LT_OK;
}

int lt_mortar_project(lt_tree* t, const double* d_u_face, double* d_u_nb, int p, int nvars) {
  if (d_u_face == d_u_nb) return LT_ERR_ARG;
  return mortar_call(t, 0, d_u_face, d_u_nb, p, nvars);
}

int lt_mortar_gather(lt_tree* t, const double* d_f_mortar, double* d_f_face, int p, int nvars) {
  return mortar_call(t, 1, d_f_mortar, d_f_face, p, nvars);
}

// ---------------------------------------------------------------------------- transfer
int lt_transfer(lt_tree* t, const double* d_u_old, double* d_u_new, int p, int nvars) {
  if (!t || !d_u_old || !d_u_new || p < 0 || p > 7 || nvars < 1) return LT_ERR_ARG;
  // the kernels move x-pencils of an even number of doubles with 128-bit accesses
  if ((p + 1) % 2 == 0 && ((((uintptr_t)d_u_old) | ((uintptr_t)d_u_new)) & 15)) return LT_ERR_ARG;
  int rc;
  // (a leaf count still pending on the device is not needed here: the kernels read it there)
  if (!t->map_ready && !t->n_valid && (rc = fetch_scalars(t)) != LT_OK) return rc;
  if ((rc = build_operators(t, p)) != LT_OK) return rc;
  tic(t, 3);
  tic(t, 4);
  if (!t->map_ready && (rc = launch_map(t)) != LT_OK) return rc;
  toc(t, 4);
  tic(t, 5);
  if ((rc = launch_transfer(t, d_u_old, d_u_new, p, nvars)) != LT_OK) return rc;
  toc(t, 5);
  t->have_old = false;
  t->n_old = 0;
  t->map_valid = true;
  t->map_ready = false;
  toc(t, 3);
  return LT_OK;
}

int lt_map(lt_tree* t, const int32_t** d_src, const uint8_t** d_kind) {
  if (!t || !t->map_valid) return LT_ERR_ARG;
  if (d_src) *d_src = t->map_src;
  if (d_kind) *d_kind = t->map_kind;
  return LT_OK;
}

// Host arrays: the transfer is pipelined in slabs of consecutive new leaves.  Slab k needs the
// contiguous old range [o_k, o_k+1) (the map is monotone), so while the kernel works on slab
// k the copy-in stream uploads slab k+1 and the copy-out stream downloads slab k-1: both PCIe
// directions stay busy and only a ring of kRing slab pairs lives in device memory.
int lt_transfer_host(lt_tree* t, const double* h_u_old, double* h_u_new, int p, int nvars) {
  if (!t || !h_u_old || !h_u_new || p < 0 || p > 7 || nvars < 1) return LT_ERR_ARG;
  int rc;
  if (!t->n_valid && (rc = fetch_scalars(t)) != LT_OK) return rc;
  if ((rc = build_operators(t, p)) != LT_OK) return rc;
  int64_t E = nvars;
  for (int a = 0; a < t->g.dim; ++a) E *= (p + 1);
  const int64_t n_old = t->have_old ? t->n_old : t->n, n_new = t->n;
  constexpr int R = Tree::kRing;
  if (!t->s_in) {
    LT_CUDA(cudaStreamCreateWithFlags(&t->s_in, cudaStreamNonBlocking));
    LT_CUDA(cudaStreamCreateWithFlags(&t->s_out, cudaStreamNonBlocking));
    for (int r = 0; r < R; ++r) {
      LT_CUDA(cudaEventCreateWithFlags(&t->ev_in[r], cudaEventDisableTiming));
      LT_CUDA(cudaEventCreateWithFlags(&t->ev_done[r], cudaEventDisableTiming));
      LT_CUDA(cudaEventCreateWithFlags(&t->ev_out[r], cudaEventDisableTiming));
    }
  }
  // slabs of about 128 MB of new solution, a multiple of 1024 leaves, at most 4096 slabs
  int64_t slab = ((128ll << 20) / (E * 8) + 1023) / 1024 * 1024;
  if (slab < 1024) slab = 1024;
  if (t->opt_host_slab > 0) slab = t->opt_host_slab;
  while ((n_new + slab - 1) / slab > 4096) slab *= 2;
  const int S = (int)((n_new + slab - 1) / slab);
  if (t->bounds_cap < S + 1) {
    free_dev(t->stream, t->d_bounds);
    if (t->h_bounds) cudaFreeHost(t->h_bounds);
    t->d_bounds = nullptr; t->h_bounds = nullptr; t->bounds_cap = 0;
    if ((rc = alloc_dev(t->stream, &t->d_bounds, 2 * (int64_t)(S + 1))) != LT_OK) return rc;
    LT_CUDA(cudaMallocHost((void**)&t->h_bounds, 2 * (size_t)(S + 1) * sizeof(int64_t)));
    t->bounds_cap = S + 1;
  }
  tic(t, 3);
  tic(t, 4);
  if (!t->map_ready && (rc = launch_map(t)) != LT_OK) return rc;
  toc(t, 4);
  if ((rc = launch_slab_bounds(t, n_old, slab, S, t->d_bounds)) != LT_OK) return rc;
  LT_CUDA(cudaMemcpyAsync(t->h_bounds, t->d_bounds, 2 * (size_t)(S + 1) * sizeof(int64_t), cudaMemcpyDeviceToHost,
                          t->stream));
  if ((rc = fetch_scalars(t)) != LT_OK) return rc;
  int st = take_status(t);
  if (st != LT_OK) return st;
  const int64_t* B = t->h_bounds;
  int64_t max_new = 0, max_old = 0;
  for (int k = 0; k < S; ++k) {
    if (B[2 * k + 2] - B[2 * k] > max_new) max_new = B[2 * k + 2] - B[2 * k];
    if (B[2 * k + 3] - B[2 * k + 1] > max_old) max_old = B[2 * k + 3] - B[2 * k + 1];
  }
  if (t->ring_old_cap < max_old * E || t->ring_new_cap < max_new * E) {
    for (int r = 0; r < R; ++r) {
      free_dev(t->stream, t->ring_old[r]); t->ring_old[r] = nullptr;
      free_dev(t->stream, t->ring_new[r]); t->ring_new[r] = nullptr;
    }
    t->ring_old_cap = t->ring_new_cap = 0;
    for (int r = 0; r < R; ++r) {
      if ((rc = alloc_dev(t->stream, &t->ring_old[r], max_old * E)) != LT_OK) return rc;
      if ((rc = alloc_dev(t->stream, &t->ring_new[r], max_new * E)) != LT_OK) return rc;
    }
    t->ring_old_cap = max_old * E;
    t->ring_new_cap = max_new * E;
  }
  // the copy streams must not run ahead of the (stream-ordered) ring allocation
  LT_CUDA(cudaEventRecord(t->ev_done[0], t->stream));
  LT_CUDA(cudaStreamWaitEvent(t->s_in, t->ev_done[0], 0));
  LT_CUDA(cudaStreamWaitEvent(t->s_out, t->ev_done[0], 0));
  tic(t, 5);
  int used = 0;
  for (int k = 0; k < S; ++k) {
    const int64_t jk = B[2 * k], ok = B[2 * k + 1], jn = B[2 * k + 2], on = B[2 * k + 3];
    if (jn <= jk) continue;
    const int r = used % R;
    if (used >= R) LT_CUDA(cudaStreamWaitEvent(t->s_in, t->ev_done[r], 0));
    LT_CUDA(cudaMemcpyAsync(t->ring_old[r], h_u_old + ok * E, (size_t)(on - ok) * E * 8, cudaMemcpyHostToDevice, t->s_in));
    LT_CUDA(cudaEventRecord(t->ev_in[r], t->s_in));
    LT_CUDA(cudaStreamWaitEvent(t->stream, t->ev_in[r], 0));
    if (used >= R) LT_CUDA(cudaStreamWaitEvent(t->stream, t->ev_out[r], 0));
    if ((rc = launch_transfer(t, t->ring_old[r] - ok * E, t->ring_new[r] - jk * E, p, nvars, jk, jn)) != LT_OK) return rc;
    LT_CUDA(cudaEventRecord(t->ev_done[r], t->stream));
    LT_CUDA(cudaStreamWaitEvent(t->s_out, t->ev_done[r], 0));
    LT_CUDA(cudaMemcpyAsync(h_u_new + jk * E, t->ring_new[r], (size_t)(jn - jk) * E * 8, cudaMemcpyDeviceToHost, t->s_out));
    LT_CUDA(cudaEventRecord(t->ev_out[r], t->s_out));
    ++used;
  }
  for (int r = 0; r < R && r < used; ++r) LT_CUDA(cudaStreamWaitEvent(t->stream, t->ev_out[r], 0));
  toc(t, 5);
  t->have_old = false;
  t->n_old = 0;
  t->map_valid = true;
  t->map_ready = false;
  toc(t, 3);
  if ((rc = fetch_scalars(t)) != LT_OK) return rc;
  return take_status(t);
}

// ---------------------------------------------------------------------------- sort / build from keys
int lt_sort_keys(int dim, int max_level, uint64_t* d_keys, int64_t n, int linearise, int64_t* n_out,
                 void* cuda_stream) {
  if ((dim != 2 && dim != 3) || n < 0 || (n > 0 && !d_keys)) return LT_ERR_ARG;
  if (dim * max_level + kLevelBits > 63 || max_level < 0) return LT_ERR_ARG;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  SortScratch sc = {nullptr, 0, nullptr, nullptr, 0, nullptr};
  int64_t launches = 0;
  int rc = sort_keys(d_keys, n, dim * max_level + kLevelBits, &sc, s, &launches);
  int64_t m = n;
  if (rc == LT_OK && linearise && n > 0) {
    unsigned long long* d_sums = nullptr;
    int* d_total = nullptr;
    int* h_total = nullptr;
    uint64_t* d_out = nullptr;
    const int G = 148 * 4;
    if (alloc_dev(s, &d_sums, G) != LT_OK || alloc_dev(s, &d_total, 1) != LT_OK || alloc_dev(s, &d_out, n) != LT_OK ||
        cudaMallocHost((void**)&h_total, sizeof(int)) != cudaSuccess) {
      rc = LT_ERR_OOM;
    } else {
      rc = linearise_keys(dim, max_level, d_keys, d_out, n, &m, d_sums, d_total, h_total, G, s, &launches);
      if (rc == LT_OK && cudaMemcpyAsync(d_keys, d_out, (size_t)m * 8, cudaMemcpyDeviceToDevice, s) != cudaSuccess)
        rc = LT_ERR_CUDA;
    }
    cudaStreamSynchronize(s);
    free_dev(s, d_sums); free_dev(s, d_total); free_dev(s, d_out);
    if (h_total) cudaFreeHost(h_total);
  }
  if (cudaStreamSynchronize(s) != cudaSuccess && rc == LT_OK) rc = LT_ERR_CUDA;
  free_dev(s, sc.tmp); free_dev(s, sc.hist); free_dev(s, sc.status);
  if (n_out) *n_out = m;
  return rc;
}

int lt_build_from_keys(int dim, int base_level, int max_level, const double* domain, const int* periodic,
                       void* cuda_stream, const uint64_t* d_keys, int64_t n, lt_tree** out) {
  if (!d_keys || n < 1 || n >= (1ll << 30)) return LT_ERR_ARG;
  Tree* t = nullptr;
  int rc = new_tree(dim, base_level, max_level, domain, periodic, cuda_stream, &t);
  if (rc != LT_OK) return rc;
  auto fail = [&](int code) {
    lt_free((lt_tree*)t);
    return code;
  };
  if ((rc = grow(t, n)) != LT_OK) return fail(rc);
  if (cudaMemcpyAsync(t->keys[t->tmp], d_keys, (size_t)n * 8, cudaMemcpyDeviceToDevice, t->stream) != cudaSuccess)
    return fail(LT_ERR_CUDA);
  SortScratch sc = {nullptr, 0, nullptr, nullptr, 0, nullptr};
  rc = sort_keys(t->keys[t->tmp], n, dim * max_level + kLevelBits, &sc, t->stream, &t->launches);
  t->sort_tmp = sc.tmp; t->sort_cap = sc.cap; t->sort_hist = sc.hist; t->sort_status = sc.status;
  t->sort_status_cap = sc.status_cap;
  if (rc != LT_OK) return fail(rc);
  int64_t m = 0;
  rc = linearise_keys(dim, max_level, t->keys[t->tmp], t->keys[t->cur], n, &m, t->d_sums, &t->d_s->aux,
                      (int*)t->h_sums, grid_for(t, 4), t->stream, &t->launches);
  if (rc != LT_OK) return fail(rc);
  int nn = (int)m;
  if (cudaMemcpyAsync(&t->d_s->n, &nn, sizeof(int), cudaMemcpyHostToDevice, t->stream) != cudaSuccess)
    return fail(LT_ERR_CUDA);
  if (host_sync(t) != cudaSuccess) return fail(LT_ERR_CUDA);
  t->n = m;
  t->n_valid = true;
  if ((rc = launch_check_tiling(t)) != LT_OK) return fail(rc);
  if ((rc = fetch_scalars(t)) != LT_OK) return fail(rc);
  t->n = m;
  int st = take_status(t);
  if (st != LT_OK) return fail(st);
  if (t->h_s->volume != (1ull << (dim * max_level))) return fail(LT_ERR_INCOMPLETE);
  if ((rc = launch_build_index(t, t->cur)) != LT_OK) return fail(rc);
  *out = (lt_tree*)t;
  return LT_OK;
}

int lt_build_complete_from_keys(int dim, int base_level, int max_level, const double* domain, const int* periodic,
                                void* cuda_stream, const uint64_t* d_keys, int64_t n, lt_tree** out) {
  if (!d_keys || n < 1 || n >= (1ll << 30)) return LT_ERR_ARG;
  Tree* t = nullptr;
  int rc = new_tree(dim, base_level, max_level, domain, periodic, cuda_stream, &t);
  if (rc != LT_OK) return rc;
  uint64_t* work = nullptr;
  if ((rc = alloc_dev(t->stream, &work, n)) == LT_OK) {
    if (cudaMemcpyAsync(work, d_keys, (size_t)n * 8, cudaMemcpyDeviceToDevice, t->stream) != cudaSuccess)
      rc = LT_ERR_CUDA;
    else
      rc = complete_from_unsorted(t, work, n);
  }
  host_sync(t);
  free_dev(t->stream, work);
  if (rc != LT_OK) {
    lt_free((lt_tree*)t);
    return rc;
  }
  *out = (lt_tree*)t;
  return LT_OK;
}

int lt_build_from_points(int dim, int base_level, int max_level, const double* domain, const int* periodic,
                         void* cuda_stream, const double* d_xyz, int64_t n, lt_tree** out) {
  if (!d_xyz || !domain || n < 1 || n >= (1ll << 30)) return LT_ERR_ARG;
  if (dim == 2 || dim == 3)
    for (int a = 0; a < dim; ++a)
      if (!(domain[dim + a] > domain[a])) return LT_ERR_ARG;
  Tree* t = nullptr;
  int rc = new_tree(dim, base_level, max_level, domain, periodic, cuda_stream, &t);
  if (rc != LT_OK) return rc;
  uint64_t* work = nullptr;
  if ((rc = alloc_dev(t->stream, &work, n)) == LT_OK) {
    rc = launch_points_to_keys(dim, max_level, t->domain, d_xyz, n, work, grid_for(t, 8), t->stream, &t->launches);
    if (rc == LT_OK) rc = complete_from_unsorted(t, work, n);
  }
  host_sync(t);
  free_dev(t->stream, work);
  if (rc != LT_OK) {
    lt_free((lt_tree*)t);
    return rc;
  }
  *out = (lt_tree*)t;
  return LT_OK;
}

// ---------------------------------------------------------------------------- FR pieces (Eq. 1-6)
int lt_common_flux(lt_tree* t, const double* d_u_face, const double* d_u_nb, double* d_f_star, int p) {
  if (!t || !d_u_face || !d_u_nb || !d_f_star || p < 0 || p > 7) return LT_ERR_ARG;
  if (!t->faces_valid) return LT_ERR_ARG;
  tic(t, 7);
  int rc = launch_common_flux(t, d_u_face, d_u_nb, d_f_star, p);
  toc(t, 7);
  return rc;
}

int lt_face_flux(lt_tree* t, const double* d_u_face, double* d_f_star, int p) {
  if (!t || !d_u_face || !d_f_star || d_u_face == d_f_star || p < 0 || p > 7) return LT_ERR_ARG;
  if (!t->faces_valid) return LT_ERR_ARG;
  int rc;
  if ((rc = build_operators(t, p)) != LT_OK) return rc;
  tic(t, 7);
  rc = launch_face_flux(t, d_u_face, d_f_star, p);
  toc(t, 7);
  return rc;
}

int lt_fr_rhs(lt_tree* t, const double* d_u, const double* d_f_star, double* d_rhs, int p) {
  if (!t || !d_u || !d_f_star || !d_rhs || d_u == d_rhs || p < 0 || p > 7) return LT_ERR_ARG;
  int rc;
  if (!t->n_valid && (rc = fetch_scalars(t)) != LT_OK) return rc;
  if ((rc = build_fr_operators(t, p)) != LT_OK) return rc;
  tic(t, 7);
  rc = launch_fr_rhs(t, d_u, d_f_star, d_rhs, p);
  toc(t, 7);
  return rc;
}

int lt_fr_stage(lt_tree* t, int stage, double dt, const double* d_u_n, const double* d_u_stage, const double* d_f_star,
                double* d_u_out, int p) {
  if (!t || !d_u_n || !d_u_stage || !d_f_star || !d_u_out || stage < 1 || stage > 3 || p < 0 || p > 7) return LT_ERR_ARG;
  int rc;
  if (!t->n_valid && (rc = fetch_scalars(t)) != LT_OK) return rc;
  if ((rc = build_fr_operators(t, p)) != LT_OK) return rc;
  const double a = stage == 1 ? 0.0 : (stage == 2 ? 0.75 : 1.0 / 3.0);
  const double b = stage == 1 ? 1.0 : (stage == 2 ? 0.25 : 2.0 / 3.0);
  tic(t, 7);
  rc = launch_fr_rhs(t, d_u_stage, d_f_star, d_u_out, p, d_u_n, a, b, dt);
  toc(t, 7);
  return rc;
}

int lt_fr_stage_faces(lt_tree* t, int stage, double dt, const double* d_u_n, const double* d_u_stage,
                      const double* d_f_star, double* d_u_out, double* d_u_face_out, int p) {
  if (!t || !d_u_n || !d_u_stage || !d_f_star || !d_u_out || !d_u_face_out || stage < 1 || stage > 3 || p < 0 || p > 7)
    return LT_ERR_ARG;
  int rc;
  if (!t->n_valid && (rc = fetch_scalars(t)) != LT_OK) return rc;
  if ((rc = build_fr_operators(t, p)) != LT_OK) return rc;
  const double a = stage == 1 ? 0.0 : (stage == 2 ? 0.75 : 1.0 / 3.0);
  const double b = stage == 1 ? 1.0 : (stage == 2 ? 0.25 : 2.0 / 3.0);
  tic(t, 7);
  rc = launch_fr_rhs(t, d_u_stage, d_f_star, d_u_out, p, d_u_n, a, b, dt, d_u_face_out);
  toc(t, 7);
  return rc;
}

int lt_rk3_stage(lt_tree* t, int stage, double dt, const double* d_u_n, const double* d_u_stage, const double* d_rhs,
                 double* d_u_out, int p) {
  if (!t || !d_u_n || !d_u_stage || !d_rhs || !d_u_out || stage < 1 || stage > 3 || p < 0 || p > 7) return LT_ERR_ARG;
  int rc;
  if (!t->n_valid && (rc = fetch_scalars(t)) != LT_OK) return rc;
  int64_t n = t->n * (t->g.dim + 2);
  for (int a = 0; a < t->g.dim; ++a) n *= (p + 1);
  const double a = stage == 1 ? 0.0 : (stage == 2 ? 0.75 : 1.0 / 3.0);
  const double b = stage == 1 ? 1.0 : (stage == 2 ? 0.25 : 2.0 / 3.0);
  return launch_rk_update(t, n, a, b, dt, d_u_n, d_u_stage, d_rhs, d_u_out);
}

}  // extern "C"
