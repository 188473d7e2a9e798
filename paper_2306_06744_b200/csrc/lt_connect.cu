// lt_connect.cu -- face connectivity (Alg. 5) for sm_100a: one thread per
// (leaf, local face) slot builds the same-level search key, locates it in the sorted leaf
// array (Eq. 7) and classifies the face; a second pass compacts the three face tables in
// emission order (reading D-4) through a scan -- no atomics, deterministic output.
// Product code.
#include "lt_internal.h"

namespace lt {

constexpr int CT = 256;

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

template <int DIM>
__global__ void __launch_bounds__(CT) k_connect_search(Geo g, const uint64_t* __restrict__ keys,
                                                       const int* __restrict__ first, DevScalars* s,
                                                       int32_t* __restrict__ nbr, uint8_t* __restrict__ kind,
                                                       int* __restrict__ sums3) {
  constexpr int NF = Dim<DIM>::NF;
  __shared__ unsigned long long sm[33];
  const int64_t nslots = (int64_t)s->n * NF;
  int64_t lo, hi;
  block_chunk(nslots, gridDim.x, blockIdx.x, CT, &lo, &hi);
  unsigned long long acc = 0;  // three 21-bit fields would overflow per chunk: use 3 x 20 bits per tile, flush per tile
  int c_conf = 0, c_hang = 0, c_bnd = 0;
  for (int64_t sidx = lo + threadIdx.x; sidx < hi; sidx += CT) {
    const int i = (int)(sidx / NF), f = (int)(sidx % NF);
    const uint64_t key = keys[i];
    const int l = key_level(key);
    const uint64_t m = key_morton(key);
    int kd = 0, nb = -1;
    uint64_t mn;
    if (face_neighbour<DIM>(g, m, l, f, &mn)) {
      const int j = locate(g, keys, first, mn);
      const int lj = key_level(keys[j]);
      if (lj == l) {  // Eq. 7 case 1: the search key is in the tree -> conforming
        kd = 1;
        nb = j;
      } else if (lj == l - 1) {  // Eq. 7 case 2: the entry to the left is the parent
        kd = 2 | (face_slot<DIM>(child_id<DIM>(g, m, l), f >> 1) << 4);
        nb = j;
      } else if (lj < l - 1) {
        set_status(&s->status, LT_ERR_UNBALANCED);  // reading D-5
      } else {
        // Eq. 7 case 3: the search key is subdivided.  Record the slot-0 fine neighbour:
        // the child of the search key touching this face with tangential bits 0 (D-2).
        int j2 = j;
        if (!(f & 1)) {
          const uint64_t mn2 = mn | (1ull << (DIM * (g.maxl - l - 1) + (f >> 1)));
          j2 = locate(g, keys, first, mn2);
        }
        if (key_level(keys[j2]) != l + 1) set_status(&s->status, LT_ERR_UNBALANCED);
        kd = 3;
        nb = j2;
      }
    }
    nbr[sidx] = nb;
    kind[sidx] = (uint8_t)kd;
    c_conf += (kd == 1) & (f & 1);
    c_hang += ((kd & 15) == 2);
    c_bnd += (kd == 0);
  }
  (void)acc;
  int t_conf = (int)block_sum<unsigned long long>(c_conf, sm);
  int t_hang = (int)block_sum<unsigned long long>(c_hang, sm);
  int t_bnd = (int)block_sum<unsigned long long>(c_bnd, sm);
  if (threadIdx.x == 0) {
    sums3[3 * blockIdx.x + 0] = t_conf;
    sums3[3 * blockIdx.x + 1] = t_hang;
    sums3[3 * blockIdx.x + 2] = t_bnd;
  }
}

// The three tables live back to back in one pool of nf*cap rows (every slot emits at most
// one row): conf rows [0, n_conf), hang rows [n_conf, n_conf + n_hang), then bnd.  The
// region offsets come from the chunk sums, so no host round trip separates the passes.
template <int DIM>
__global__ void __launch_bounds__(CT) k_connect_tables(DevScalars* __restrict__ s,
                                                       const int32_t* __restrict__ nbr,
                                                       const uint8_t* __restrict__ kind,
                                                       const int* __restrict__ sums3, int32_t* __restrict__ rows,
                                                       uint8_t* __restrict__ bytes) {
  constexpr int NF = Dim<DIM>::NF;
  __shared__ unsigned long long sm[33];
  const int64_t nslots = (int64_t)s->n * NF;
  // prefix of the three counters over the chunks before this one, and their totals
  unsigned long long b0 = 0, b1 = 0, b2 = 0, a0 = 0, a1 = 0, a2 = 0;
  for (int i = threadIdx.x; i < (int)gridDim.x; i += CT) {
    const unsigned long long c0 = sums3[3 * i], c1 = sums3[3 * i + 1], c2 = sums3[3 * i + 2];
    a0 += c0;
    a1 += c1;
    a2 += c2;
    if (i < (int)blockIdx.x) {
      b0 += c0;
      b1 += c1;
      b2 += c2;
    }
  }
  int64_t r_conf = (int64_t)block_sum(b0, sm);
  int64_t r_hang = (int64_t)block_sum(b1, sm);
  int64_t r_bnd = (int64_t)block_sum(b2, sm);
  const int64_t n_conf = (int64_t)block_sum(a0, sm), n_hang = (int64_t)block_sum(a1, sm);
  const int64_t n_bnd = (int64_t)block_sum(a2, sm);
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    s->n_face[0] = (int)n_conf;
    s->n_face[1] = (int)n_hang;
    s->n_face[2] = (int)n_bnd;
  }
  int32_t* __restrict__ conf = rows;
  int32_t* __restrict__ hang = rows + 2 * n_conf;
  int32_t* __restrict__ bnd = rows + 2 * (n_conf + n_hang);
  uint8_t* __restrict__ conf_axis = bytes;
  uint8_t* __restrict__ hang_info = bytes + n_conf;
  uint8_t* __restrict__ bnd_face = bytes + n_conf + n_hang;
  int64_t lo, hi;
  block_chunk(nslots, gridDim.x, blockIdx.x, CT, &lo, &hi);
  for (int64_t t0 = lo; t0 < hi; t0 += CT) {
    const int64_t sidx = t0 + threadIdx.x;
    int kd = 255, nb = 0, f = 0;
    if (sidx < hi) {
      kd = kind[sidx];
      nb = nbr[sidx];
      f = (int)(sidx % NF);
    }
    const bool is_conf = (kd == 1) && (f & 1), is_hang = (kd & 15) == 2 && kd != 255, is_bnd = kd == 0;
    unsigned long long v = (unsigned long long)is_conf | ((unsigned long long)is_hang << 21) |
                           ((unsigned long long)is_bnd << 42);
    unsigned long long tot;
    unsigned long long ex = block_excl_scan<unsigned long long>(v, sm, &tot);
    const int e = (int)(sidx / NF);
    if (is_conf) {
      int64_t p = r_conf + (int64_t)(ex & 0x1fffff);
      conf[2 * p] = e;
      conf[2 * p + 1] = nb;
      conf_axis[p] = (uint8_t)(f >> 1);
    } else if (is_hang) {
      int64_t p = r_hang + (int64_t)((ex >> 21) & 0x1fffff);
      hang[2 * p] = e;
      hang[2 * p + 1] = nb;
      hang_info[p] = (uint8_t)(f | ((kd >> 4) << 3));
    } else if (is_bnd) {
      int64_t p = r_bnd + (int64_t)((ex >> 42) & 0x1fffff);
      bnd[p] = e;
      bnd_face[p] = (uint8_t)f;
    }
    r_conf += (int64_t)(tot & 0x1fffff);
    r_hang += (int64_t)((tot >> 21) & 0x1fffff);
    r_bnd += (int64_t)((tot >> 42) & 0x1fffff);
  }
}

int launch_connect_search(Tree* t, int G) {
  if (t->g.dim == 2)
    k_connect_search<2><<<G, CT, 0, t->stream>>>(t->g, t->keys[t->cur], t->first[t->cur], t->d_s, t->nbr, t->kind,
                                                 t->d_sums3);
  else
    k_connect_search<3><<<G, CT, 0, t->stream>>>(t->g, t->keys[t->cur], t->first[t->cur], t->d_s, t->nbr, t->kind,
                                                 t->d_sums3);
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

int launch_connect_tables(Tree* t, int G) {
  if (t->g.dim == 2)
    k_connect_tables<2><<<G, CT, 0, t->stream>>>(t->d_s, t->nbr, t->kind, t->d_sums3, t->face_rows, t->face_bytes);
  else
    k_connect_tables<3><<<G, CT, 0, t->stream>>>(t->d_s, t->nbr, t->kind, t->d_sums3, t->face_rows, t->face_bytes);
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

}  // namespace lt
