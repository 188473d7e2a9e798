// lt_connect.cu -- face connectivity (Alg. 5) for sm_100a, ONE kernel, one
// pass over the leaves:
//   - a tile of 256 consecutive leaves is claimed through a ticket; one thread per leaf
//     classifies first its dim parent-interior faces (sibling shortcut) and then its dim
//     exterior faces (same-level search key, bucketed lower bound, Eq. 7) into shared memory
//     -- two warp-uniform phases;
//   - nbr / kind (the paper's face array F) leave in slot order, coalesced;
//   - one thread per leaf counts its rows, a packed block scan orders them inside the tile,
//     a decoupled look-back over the earlier tiles orders the tiles, and the three face
//     tables are written in emission order (reading D-4) -- no atomics on the data, the
//     output is deterministic.
// Product code.
#include "lt_internal.h"

namespace lt {

constexpr int CT = 256;   // threads per block
constexpr int LPT = 2;    // leaves per thread: a tile is CT * LPT consecutive leaves (thread t: leaves t and CT + t)
constexpr int TL = CT * LPT;

// slot of a fine face inside the coarse face: the fine leaf's child-id bits on the
// tangential axes, ascending axis order ("the first contributor along one
// axis will be the one that has smaller coordinates"; reading D-3)
template <int DIM>
__device__ __forceinline__ int face_slot(int cid, int axis) {
  if (DIM == 2) return (cid >> (1 - axis)) & 1;
  if (axis == 0) return (cid >> 1) & 3;
  if (axis == 1) return (cid & 1) | (((cid >> 2) & 1) << 1);
  return cid & 3;
}

// Face f of leaf (m, l) at position i by search: same-level neighbour key (periodic wrap /
// domain boundary), bucketed lower bound (Eq. 7), classification.  Returns kind; *nb_out =
// neighbour index (or -1).
template <int DIM>
__device__ __forceinline__ int face_by_search(const Geo& g, const uint64_t* __restrict__ keys,
                                              const int* __restrict__ first, uint64_t m, int l, int f, int* status,
                                              int* nb_out) {
  const int a = f >> 1;
  *nb_out = -1;
  uint64_t mn;
  if (!face_neighbour<DIM>(g, m, l, f, &mn)) return 0;  // domain boundary
  const int j = locate(g, keys, first, mn);
  LT_DASSERT(j >= 0 && j < first[g.nbuckets]);
  const int lj = key_level(keys[j]);
  if (lj == l) {  // Eq. 7 case 1: the search key is in the tree -> conforming
    *nb_out = j;
    return 1;
  }
  if (lj == l - 1) {  // Eq. 7 case 2: the entry to the left is the parent -> hanging, fine side
    *nb_out = j;
    return 2 | (face_slot<DIM>(child_id<DIM>(g, m, l), a) << 4);
  }
  if (lj < l - 1) {
    set_status(status, LT_ERR_UNBALANCED);  // reading D-5
    return 0;
  }
  // Eq. 7 case 3: the search key is subdivided.  Record the slot-0 fine neighbour: the child
  // of the search key touching this face with tangential bits 0 (reading D-2).
  int j2 = j;
  if (!(f & 1)) {
    const uint64_t mn2 = mn | (1ull << (DIM * (g.maxl - l - 1) + a));
    j2 = locate(g, keys, first, mn2);
  }
  if (key_level(keys[j2]) != l + 1) set_status(status, LT_ERR_UNBALANCED);
  *nb_out = j2;
  return 3;
}

// The face of leaf i on axis a that is INTERIOR to its parent looks at a sibling.  If that
// sibling is a leaf and every sibling between the two is a leaf too, it sits exactly
// (cid' - cid) entries away: one key comparison decides, no search.
template <int DIM>
__device__ __forceinline__ bool face_by_sibling(const Geo& g, const uint64_t* __restrict__ keys, int n, int i,
                                                uint64_t m, int l, int cid, int a, int* nb_out) {
  const int sh = DIM * (g.maxl - l);
  const int j = i + ((cid ^ (1 << a)) - cid);
  if (j >= 0 && j < n && keys[j] == make_key(m ^ (1ull << (sh + a)), l)) {
    *nb_out = j;
    return true;
  }
  return false;
}

// Tile status words of the decoupled look-back, two independent channels per tile:
//   st[2t]   = flag << 62 | n_conf << 31 | n_hang        st[2t+1] = flag << 62 | n_bnd
// flag 1 = the tile's own counts, 2 = inclusive prefix over tiles 0..t.  No field carries
// into its neighbour because every partial sum is bounded by a final total < 2^31.
constexpr unsigned long long kFlagAgg = 1ull << 62, kFlagInc = 2ull << 62, kValMask = (1ull << 62) - 1;

// (one warp) exclusive prefix of channel ch over the tiles before `tile`, 32 predecessors per
// step; publishes the tile's inclusive prefix.
__device__ __forceinline__ unsigned long long lookback_warp(volatile unsigned long long* st, int tile, int ch,
                                                            unsigned long long own, int lane) {
  unsigned long long excl = 0;
  for (int t = tile - 1; t >= 0; t -= 32) {
    const int idx = t - lane;
    unsigned long long v = kFlagInc;  // before tile 0: an inclusive prefix of zero
    if (idx >= 0) {
      do { v = st[2 * (size_t)idx + ch]; } while ((v >> 62) == 0);
      LT_DASSERT((v >> 62) <= 2);  // look-back protocol: 0 not ready, 1 own counts, 2 inclusive prefix
    }
    const unsigned inc = __ballot_sync(0xffffffffu, (v >> 62) == 2);
    const int stop = inc ? __ffs(inc) - 1 : 31;  // nearest predecessor that is already inclusive
    unsigned long long c = lane <= stop ? (v & kValMask) : 0ull;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) c += __shfl_xor_sync(0xffffffffu, c, d);
    excl += c;
    if (inc) break;
  }
  if (lane == 0) st[2 * (size_t)tile + ch] = kFlagInc | (excl + own);
  return excl;
}

template <int DIM>
__global__ void __launch_bounds__(CT) k_connect(Geo g, const uint64_t* __restrict__ keys,
                                                const int* __restrict__ first,
                                                const uint64_t* __restrict__ keys_alt,
                                                const int* __restrict__ first_alt, DevScalars* s,
                                                int32_t* __restrict__ nbr, uint8_t* __restrict__ kind,
                                                int32_t* __restrict__ conf, uint8_t* __restrict__ conf_axis,
                                                int32_t* __restrict__ hang, uint8_t* __restrict__ hang_info,
                                                int32_t* __restrict__ bnd, uint8_t* __restrict__ bnd_face,
                                                unsigned long long* st, unsigned* ticket) {
  constexpr int NF = Dim<DIM>::NF;
  // per-leaf rows padded to an odd pitch: with NF = 6 (or 4) words per leaf the lanes of a warp, each
  // writing its own leaf's slot f, hit every other bank twice (12 M conflicts per 13.5 M-leaf query)
  constexpr int NP = NF + 1;
  __shared__ int s_nb[TL * NP];
  __shared__ uint8_t s_kd[TL * NP];
  __shared__ unsigned long long sm[33];
  __shared__ unsigned long long s_excl[2];
  __shared__ int s_tile;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int n = s->n;
  const int ntiles = (n + TL - 1) / TL;
  // keys_alt != nullptr: the lt_balance before this query did not wait for its kernel, and the
  // buffer its result ended in (DevScalars::parity) is only known here
  if (keys_alt != nullptr && s->parity) {
    keys = keys_alt;
    first = first_alt;
  }
  for (;;) {
    if (threadIdx.x == 0) s_tile = (int)atomicAdd(ticket, 1u);
    __syncthreads();
    const int tile = s_tile;
    LT_DASSERT(tile >= 0 && tile < ntiles + (int)gridDim.x);  // every block draws one ticket past the end
    if (tile >= ntiles) break;
    const int e0 = tile * TL;
    const int ne = min(TL, n - e0);
    // (Tried and rejected, round 2: sharing ONE search per face of the parent among the 2^(dim-1) members
    // of a complete sibling group -- the trick that pays in k_balance -- with key compares for the members'
    // own neighbours.  Bit-exact, but 2.2 instead of 1.5 ms alone and no better beside the transfer: the
    // probes it saves hit L1, the group detection, shuffles and divergence it adds do not come for free.)
    // (Also tried and rejected: the DIM exterior searches of a leaf in lock-step -- bucket bounds, every
    // binary-search round and the located keys of the three faces loaded together.  Bit-exact; the query
    // beside the transfer went from 7.3 to 6.6 ms, but the step did not move (15.42 -> 15.50 ms: what the
    // transfer loses depends on how many of its blocks the query displaces, not on how long).  A 4-ary
    // lock-step search that also takes in the interior-face fallbacks needs 127 registers; capped at 64 it
    // spills and is slower everywhere: 2.5 instead of 1.7 ms alone, 10.8 ms beside the transfer.)
    // ---- classify: a thread handles LPT leaves (two independent chains of dependent probes in flight per
    // thread, and half as many barriers, tickets and look-backs per leaf as with one), each in two
    // warp-uniform phases -- first the DIM faces interior to the parent (sibling shortcut, one compare),
    // then the DIM exterior faces (search) -- so that a warp never executes both code paths for every slot
    {
      constexpr int NC = Dim<DIM>::NC;
      uint64_t mq[LPT];
      int lq[LPT], cq[LPT];
#pragma unroll
      for (int h = 0; h < LPT; ++h) {
        const int li = h * CT + threadIdx.x;
        const uint64_t key = li < ne ? keys[e0 + li] : 0;
        lq[h] = key_level(key);
        mq[h] = key_morton(key);
        cq[h] = lq[h] > 0 ? (int)((mq[h] >> (DIM * (g.maxl - lq[h]))) & (uint64_t)(NC - 1)) : 0;
      }
#pragma unroll
      for (int a = 0; a < DIM; ++a) {
#pragma unroll
        for (int h = 0; h < LPT; ++h) {
          const int li = h * CT + threadIdx.x;
          if (li >= ne) continue;
          const int f = 2 * a + (((cq[h] >> a) & 1) ^ 1);
          int nb, kd = 1;
          if (lq[h] == 0 || !face_by_sibling<DIM>(g, keys, n, e0 + li, mq[h], lq[h], cq[h], a, &nb))
            kd = face_by_search<DIM>(g, keys, first, mq[h], lq[h], f, &s->status_c, &nb);
          s_nb[li * NP + f] = nb;
          s_kd[li * NP + f] = (uint8_t)kd;
        }
      }
#pragma unroll
      for (int a = 0; a < DIM; ++a) {
#pragma unroll
        for (int h = 0; h < LPT; ++h) {
          const int li = h * CT + threadIdx.x;
          if (li >= ne) continue;
          const int f = 2 * a + ((cq[h] >> a) & 1);
          int nb;
          const int kd = face_by_search<DIM>(g, keys, first, mq[h], lq[h], f, &s->status_c, &nb);
          s_nb[li * NP + f] = nb;
          s_kd[li * NP + f] = (uint8_t)kd;
        }
      }
    }
    __syncthreads();
    // F (the paper's face array) leaves in slot order, coalesced
#pragma unroll
    for (int r = 0; r < NF * LPT; ++r) {
      const int sl = r * CT + threadIdx.x;
      if (sl < ne * NF) {
        const size_t gs = (size_t)e0 * NF + sl;
        const int pl = (sl / NF) * NP + sl % NF;
        nbr[gs] = s_nb[pl];
        kind[gs] = s_kd[pl];
      }
    }
    // ---- rows of this thread's leaves, packed for ONE block scan: per half of the tile (h = 0: leaves
    // 0..CT-1, h = 1: the rest) conf (10 bits, <= DIM * CT) | hang (10 bits) | bnd (11 bits, <= NF * CT)
    static_assert(LPT == 2 && DIM * CT < 1024 && NF * CT < 2048, "packed row counts");
    unsigned long long cnt = 0;
#pragma unroll
    for (int h = 0; h < LPT; ++h) {
      const int li = h * CT + threadIdx.x;
      if (li < ne) {
        unsigned long long c = 0;
#pragma unroll
        for (int f = 0; f < NF; ++f) {
          const int kd = s_kd[li * NP + f];
          c += (unsigned long long)((kd == 1) & (f & 1)) | ((unsigned long long)((kd & 15) == 2) << 10) |
               ((unsigned long long)(kd == 0) << 20);
        }
        cnt |= c << (31 * h);
      }
    }
    unsigned long long tot;
    const unsigned long long ex = block_excl_scan<unsigned long long>(cnt, sm, &tot);
    const unsigned long long a_conf = tot & 0x3ff, a_hang = (tot >> 10) & 0x3ff, a_bnd = (tot >> 20) & 0x7ff;
    const unsigned long long t_conf = a_conf + ((tot >> 31) & 0x3ff), t_hang = a_hang + ((tot >> 41) & 0x3ff),
                             t_bnd = a_bnd + ((tot >> 51) & 0x7ff);
    // ---- order the tiles: publish the tile's own counts, then look back (warp 0: conf and
    // hang, warp 1: bnd)
    if (w < 2) {
      const unsigned long long own = w == 0 ? ((t_conf << 31) | t_hang) : t_bnd;
      volatile unsigned long long* vst = st;
      if (lane == 0 && tile > 0) vst[2 * (size_t)tile + w] = kFlagAgg | own;
      const unsigned long long excl = lookback_warp(vst, tile, w, own, lane);
      if (lane == 0) s_excl[w] = excl;
    }
    __syncthreads();
    const unsigned long long x0 = s_excl[0], x1 = s_excl[1];
    if (tile == ntiles - 1 && threadIdx.x == 0) {
      s->n_face[0] = (int)((x0 >> 31) + t_conf);
      s->n_face[1] = (int)((x0 & 0x7fffffffull) + t_hang);
      s->n_face[2] = (int)(x1 + t_bnd);
    }
    // ---- emit (leaf order, local faces 0..NF-1: reading D-4)
#pragma unroll
    for (int h = 0; h < LPT; ++h) {
      const int li = h * CT + threadIdx.x;
      if (li >= ne) continue;
      const int e = e0 + li;
      int64_t p_conf = (int64_t)(x0 >> 31) + (int64_t)((ex >> (31 * h)) & 0x3ff) + (h ? (int64_t)a_conf : 0);
      int64_t p_hang = (int64_t)(x0 & 0x7fffffffull) + (int64_t)((ex >> (31 * h + 10)) & 0x3ff) + (h ? (int64_t)a_hang : 0);
      int64_t p_bnd = (int64_t)x1 + (int64_t)((ex >> (31 * h + 20)) & 0x7ff) + (h ? (int64_t)a_bnd : 0);
      // the rows of the leaves before e: at most DIM conforming, DIM hanging and NF boundary rows each
      LT_DASSERT(p_conf >= 0 && p_conf <= (int64_t)DIM * e && p_hang >= 0 && p_hang <= (int64_t)DIM * e &&
                 p_bnd >= 0 && p_bnd <= (int64_t)NF * e);
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        const int kd = s_kd[li * NP + f];
        const int nb = s_nb[li * NP + f];
        if (kd == 1) {
          if (f & 1) {  // a conforming face is emitted by the element on its minus side
            reinterpret_cast<int2*>(conf)[p_conf] = make_int2(e, nb);
            conf_axis[p_conf] = (uint8_t)(f >> 1);
            ++p_conf;
          }
        } else if ((kd & 15) == 2) {  // hanging: emitted by the fine element
          reinterpret_cast<int2*>(hang)[p_hang] = make_int2(e, nb);
          hang_info[p_hang] = (uint8_t)(f | ((kd >> 4) << 3));
          ++p_hang;
        } else if (kd == 0) {
          bnd[p_bnd] = e;
          bnd_face[p_bnd] = (uint8_t)f;
          ++p_bnd;
        }
      }
    }
    __syncthreads();  // s_kd / s_nb / s_tile / s_excl are reused by the next tile
  }
}

// The three tables have fixed regions in the pool.  Each face slot emits at most one row; only
// a face exterior to the parent can see a coarser neighbour (an interior face looks at a
// sibling's cell, tiled by leaves at least as fine) and only odd faces emit conforming rows:
//   n_conf <= dim*M,  n_hang <= dim*M,  n_bnd <= nf*M.
void face_regions(const Tree* t, int32_t** conf, uint8_t** conf_axis, int32_t** hang, uint8_t** hang_info,
                  int32_t** bnd, uint8_t** bnd_face) {
  const size_t dc = (size_t)t->g.dim * (size_t)t->cap;
  *conf = t->face_rows;
  *hang = t->face_rows + 2 * dc;
  *bnd = t->face_rows + 4 * dc;
  *conf_axis = t->face_bytes;
  *hang_info = t->face_bytes + dc;
  *bnd_face = t->face_bytes + 2 * dc;
}

int launch_connect(Tree* t, cudaStream_t stream, int blocks_per_sm) {
  int32_t *conf, *hang, *bnd;
  uint8_t *conf_axis, *hang_info, *bnd_face;
  face_regions(t, &conf, &conf_axis, &hang, &hang_info, &bnd, &bnd_face);
  // (leaf count still on the device: its upper bound sizes the look-back words to clear)
  const int64_t ntiles = ((t->n_valid ? t->n : t->n_upper) + TL - 1) / TL;
  LT_CUDA(cudaMemsetAsync(t->tile_state, 0, (size_t)(ntiles + 1) * 2 * sizeof(unsigned long long), stream));
  LT_CUDA(cudaMemsetAsync(&t->d_s->ticket_c, 0, sizeof(unsigned), stream));
  const void* fn = t->g.dim == 2 ? (const void*)k_connect<2> : (const void*)k_connect<3>;
  static int occ[2] = {0, 0};  // resident blocks per SM (the query costs microseconds of host time)
  int& per_sm_cached = occ[t->g.dim - 2];
  if (per_sm_cached == 0) LT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_cached, fn, CT, 0));
  int per_sm = per_sm_cached;
  if (per_sm < 1) per_sm = 1;
  const uint64_t* keys_alt = t->parity_pending ? t->keys[t->tmp] : nullptr;
  const int* first_alt = t->parity_pending ? t->first[t->tmp] : nullptr;
  if (blocks_per_sm > 0 && blocks_per_sm < per_sm) per_sm = blocks_per_sm;
  const int G = t->num_sms * per_sm;
  if (t->g.dim == 2)
    k_connect<2><<<G, CT, 0, stream>>>(t->g, t->keys[t->cur], t->first[t->cur], keys_alt, first_alt, t->d_s, t->nbr, t->kind, conf,
                                          conf_axis, hang, hang_info, bnd, bnd_face, t->tile_state,
                                          &t->d_s->ticket_c);
  else
    k_connect<3><<<G, CT, 0, stream>>>(t->g, t->keys[t->cur], t->first[t->cur], keys_alt, first_alt, t->d_s, t->nbr, t->kind, conf,
                                          conf_axis, hang, hang_info, bnd, bnd_face, t->tile_state,
                                          &t->d_s->ticket_c);
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

}  // namespace lt
