// lt_internal.h -- host-side state of a tree and the launcher prototypes shared by the
// translation units of liblt.  Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/lt.h"
#include "lt_dev.cuh"

// Test hook, not part of the public enum lt_option (value 3 is reserved there): v > 0 makes lt_balance
// pretend that its buffers hold only n + v leaves, to exercise the LT_ERR_CAPACITY retry.
#define LT_OPT_DEBUG_BALANCE_SLACK 3

namespace lt {

// Device-resident scalars of a tree (one allocation).
struct DevScalars {
  int n;                 // current leaf count
  int n_in;              // lt_adapt: the count of the tree being adapted (snapshot taken by pass 1)
  int status;            // sticky lt_status detected on the device (0 = ok)
  int iters;             // balance: sweeps that split >= 1 leaf
  int parity;            // balance: 0 = result in the buffer it started in, 1 = in the other
  int n_face[3];         // connect: n_conf, n_hang, n_bnd
  int aux;               // scratch counter (path-A append cursor, sort tickets)
  unsigned long long volume;  // build_from_keys: sum of leaf volumes
  int splits;            // balance: leaves split in total
  unsigned ticket;       // tile ticket of k_transfer (zeroed before each launch)
  unsigned ticket_c;     // tile ticket of k_connect (its own word: the two kernels may overlap)
  int nfront[2];         // balance frontier ping-pong counters; [0] also counts lt_adapt's list
  int fr_overflow;       // balance: the next frontier did not fit its buffer (-> full sweep)
  int map_bad;           // balance tail (Alg. 7): a new leaf is more than one level from T_old
  unsigned long long bal_ns[4];  // k_balance, device time per phase of the last launch: examine, chunk
                                 // offsets, split + frontier, Alg. 7 tail (lt_balance_phases)
  int status_c;          // sticky status of k_connect (its own word: the face query may run beside
                         // lt_transfer on the side stream, and each call reports only its own errors)
};

constexpr int kMaxGrid = 4096;  // upper bound on persistent grid sizes (chunk-sum arrays)

struct Tree {
  Geo g;
  double domain[6];
  cudaStream_t stream;
  int device, num_sms;

  int64_t cap;            // leaf capacity of every per-leaf buffer
  uint64_t* keys[3];      // cur / old (snapshot) / tmp rotate through these
  int* first[3];          // bucket index per key buffer, nbuckets + 1 entries
  int cur, old, tmp;
  bool have_old;
  int64_t n_old;
  int64_t n;              // host copy of the leaf count
  bool n_valid;
  bool parity_pending;    // an lt_balance that did not wait: h_s->parity decides cur / tmp at the next fetch
  int64_t n_upper;        // upper bound of the leaf count while !n_valid
  int last_iters;         // sweeps of the last synchronous lt_balance (-1: read them from h_s)

  DevScalars* d_s;
  DevScalars* h_s;        // pinned mirror
  unsigned long long* d_sums;  // [kMaxGrid] chunk sums (packed pairs)
  int* d_sums3;           // [3*kMaxGrid] connect chunk sums
  int* h_sums;            // pinned [3*kMaxGrid + ..]

  uint8_t* mark;          // [cap] balance marks: bit0 split, bit1 re-examine
  uint64_t* fkey[2];      // [fcap] balance frontier: entry keys (or positions) ...
  uint8_t* ftag[2];       // [fcap] ... and their tags (lt_tree.cu)
  int64_t fcap;
  int* d_cmarks;          // [2*kMaxGrid] balance: leaves marked per chunk

  // connectivity
  int32_t* nbr;
  uint8_t* kind;
  // face-table pool, fixed regions (face_regions() in lt_connect.cu):
  //   rows  = conf [dim*cap][2] | hang [dim*cap][2] | bnd [nf*cap]      (int32)
  //   bytes = conf_axis [dim*cap] | hang_info [dim*cap] | bnd_face [nf*cap]
  int32_t* face_rows;
  uint8_t* face_bytes;
  unsigned long long* tile_state;  // [2*(cap/256 + 2)] look-back status of k_connect

  // Alg. 7 map
  int32_t* map_src;
  uint8_t* map_kind;
  bool map_valid;         // lt_map may hand the arrays out (set by lt_transfer)
  bool map_ready;         // map_src / map_kind already hold T_old -> current tree (lt_balance's tail)
  bool faces_valid;       // nbr / kind describe the current tree (set by lt_connect)
  // lt_connect_begin / lt_connect_end: k_connect on a side stream, overlapping lt_transfer
  cudaStream_t s_side;
  cudaEvent_t ev_side_fork, ev_side_join;
  bool connect_pending;
  int balanced_conn;      // the tree is 2:1 balanced with this connectivity (0: unknown)
  int front_conn;         // balanced_conn of the tree the last lt_adapt started from
  bool front_ok;          // fkey[0] / ftag[0] / d_s->nfront[0] list the leaves created by the last lt_adapt
  int* mortar_hits;       // [hits][2 + 2^(dim-1)]: coarse-side hanging faces (e, f, fine neighbours)
  int64_t mortar_hits_cap;

  // transfer operators on the device for (dim, p): I^0,I^1,R^0,R^1, each [P1][P1]
  double* d_ops;
  int ops_p;

  // lt_transfer_host: ring of device staging slabs, copy-in / copy-out streams, slab bounds
  static constexpr int kRing = 3;
  double* ring_old[kRing]; double* ring_new[kRing]; int64_t ring_old_cap, ring_new_cap;
  cudaStream_t s_in, s_out;
  cudaEvent_t ev_in[kRing], ev_done[kRing], ev_out[kRing];
  int64_t* d_bounds; int64_t* h_bounds; int bounds_cap;

  // sort scratch
  uint64_t* sort_tmp; int64_t sort_cap; unsigned* sort_hist; unsigned* sort_status; int64_t sort_status_cap;

  int opt_adapt_sort, opt_full_sweeps, opt_debug_slack, opt_host_slab, opt_balance_conn;
  cudaEvent_t ev[16];
  bool ev_set[8];
  int64_t launches;
  int64_t host_syncs;     // times the host waited for the tree's stream (lt_host_syncs)
};

extern thread_local int g_last_cuda_error;
#define LT_CUDA(call)                                   \
  do {                                                  \
    cudaError_t e_ = (call);                            \
    if (e_ != cudaSuccess) {                            \
      lt::g_last_cuda_error = (int)e_;                  \
      cudaGetLastError();                               \
      return e_ == cudaErrorMemoryAllocation ? LT_ERR_OOM : LT_ERR_CUDA; \
    }                                                   \
  } while (0)

int grid_for(const Tree* t, int blocks_per_sm);
// LT_OK iff the tree's device is the current one (kernels, constant-memory uploads and pool
// allocations all go to the current device)
int check_device(const Tree* t);
// stream-ordered device memory (lt_api.cu): the device's default cudaMallocAsync pool
int dev_alloc(void** p, size_t bytes, cudaStream_t s);
void dev_free(void* p, cudaStream_t s);

// ---- lt_tree.cu
int launch_build_uniform(Tree* t);
int launch_build_index(Tree* t, int buf);
int launch_adapt_count(Tree* t, const int8_t* d_flags, int G);
int launch_adapt_scatter(Tree* t, const int8_t* d_flags, int G, int path_a, int emit_front);
int launch_balance(Tree* t, int64_t cap_told, int use_front);
int launch_leaf_boxes(Tree* t, int32_t* d_level, uint32_t* d_xyz);
int launch_encode(int dim, int maxl, const uint32_t* d_xyz, const int32_t* d_level, int64_t n, uint64_t* d_keys, cudaStream_t s);
int launch_decode(int dim, int maxl, const uint64_t* d_keys, int64_t n, int32_t* d_level, uint32_t* d_xyz, cudaStream_t s);
int launch_check_tiling(Tree* t);

// ---- lt_connect.cu
int launch_connect(Tree* t, cudaStream_t stream, int blocks_per_sm /* 0 = full occupancy */);
void face_regions(const Tree* t, int32_t** conf, uint8_t** conf_axis, int32_t** hang, uint8_t** hang_info,
                  int32_t** bnd, uint8_t** bnd_face);

// ---- lt_transfer.cu
int launch_map(Tree* t);
int launch_transfer(Tree* t, const double* d_u_old, double* d_u_new, int p, int nvars, int64_t jb = 0,
                    int64_t je = -1);
int launch_slab_bounds(Tree* t, int64_t n_old, int64_t slab, int S, int64_t* d_out);
int build_operators(Tree* t, int p);
int launch_face_interp(Tree* t, const double* d_u, double* d_uf, int p, int nvars);
int launch_mortar_hits(Tree* t);
int launch_mortar(Tree* t, int which, const double* d_in, double* d_out, int p, int nvars);
int launch_face_flux(Tree* t, const double* d_uf, double* d_fs, int p);

// ---- lt_construct.cu (Alg. 2)
int launch_points_to_keys(int dim, int maxl, const double* domain, const double* d_xyz, int64_t n, uint64_t* d_keys,
                          int G, cudaStream_t s, int64_t* launches);
int launch_complete_count(Tree* t, const uint64_t* d_in, int64_t n, uint32_t* d_offs, int64_t* total);
int launch_complete_fill(Tree* t, const uint64_t* d_in, int64_t n, const uint32_t* d_offs, int64_t total);

// ---- lt_fr.cu (Eq. 1-6, Alg. 8 step 3)
int build_fr_operators(Tree* t, int p);
int launch_common_flux(Tree* t, const double* d_uf, const double* d_unb, double* d_fs, int p);
int launch_fr_rhs(Tree* t, const double* d_u, const double* d_fs, double* d_R, int p, const double* d_un = nullptr,
                  double ca = 0.0, double cb = 0.0, double dt = 0.0, double* d_uf_out = nullptr);
int launch_rk_update(Tree* t, int64_t n, double a, double b, double dt, const double* un, const double* us,
                     const double* R, double* out);

// ---- lt_sort.cu
struct SortScratch {
  uint64_t* tmp; int64_t cap; unsigned* hist; unsigned* status; int64_t status_cap; int* counter;
};
int sort_keys(uint64_t* d_keys, int64_t n, int key_bits, SortScratch* sc, cudaStream_t s, int64_t* launches);
int linearise_keys(int dim, int maxl, const uint64_t* d_in, uint64_t* d_out, int64_t n, int64_t* n_out,
                   unsigned long long* d_sums, int* d_total, int* h_total, int G, cudaStream_t s, int64_t* launches);

}  // namespace lt

struct lt_tree : lt::Tree {};
