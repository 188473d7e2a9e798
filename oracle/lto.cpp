// oracle/lto.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, sequential CPU oracle for the h-adaptation cycle of
// "An efficient GPU-based h-adaptation framework via linear trees for the flux
// reconstruction method" (arxiv 2306.06744; citations are PAPER.md:<line>).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference leg may load this.  It shares no code, header, table or constant
// generator with the CUDA library (paper_2306_06744_b200/csrc, include/lt.h).
//
// Form (BASELINE.json north_star): a pointer-based tree, std::sort, brute-force
// O(N^2) face adjacency for tiny meshes, point-location descent for large ones,
// dense mass / projection matrices built by over-integrated Gauss quadrature
// and solved by Gaussian elimination.  Every function cites the passage it
// follows; readings of silent/garbled passages are the ones listed in
// DESIGN.md (section "Readings").
//
// The domain may be a brick of root cubes (a forest of pointer trees, reading J-1 of DESIGN.md;
// PAPER.md:410 runs on a slab of 16 x 16 x 1 cubes): one cube reproduces the single-tree oracle bit for bit.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): see DESIGN.md section "Oracle
// pins".  No function here is "parity unpinned".
//
// Build: g++ -O2 -std=c++17 -shared -fPIC oracle/lto.cpp -o oracle/liblto.so
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

namespace {

constexpr int kLevelBits = 5;  // reading A-2: m_b fixed at 5

struct Node {
  int level = 0;
  uint32_t x[3] = {0, 0, 0};  // integer anchor in units of the finest cell
  Node* child[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  Node* parent = nullptr;
  int64_t idx = -1;   // position in the sorted leaf array (leaves only)
  bool mark = false;  // scratch
  bool is_leaf() const { return child[0] == nullptr; }
};

struct Faces {
  std::vector<int32_t> nbr;
  std::vector<uint8_t> kind;
  std::vector<int32_t> conf;
  std::vector<uint8_t> conf_axis;
  std::vector<int32_t> hang;
  std::vector<uint8_t> hang_info;
  std::vector<int32_t> bnd;
  std::vector<uint8_t> bnd_face;
};

struct Ops {  // dense transfer operators for one (dim, p)
  int dim = 0, p = -1, N = 0;
  std::vector<double> interp;  // [nc][N][N]  child c value n = sum_m interp[c][n][m] * parent m   (Eq. 8)
  std::vector<double> proj;    // [nc][N][N]  parent n = sum_c sum_m proj[c][n][m] * child c m     (Eq. 12)
  std::vector<double> mass;    // [N][N]   M   (Eq. 13)
  std::vector<double> S;       // [nc][N][N] S_c (Eq. 13)
};

struct Tree {
  int dim = 2, base = 0, maxl = 0, nc = 4, nf = 4;
  int periodic[3] = {0, 0, 0};
  // The domain is a brick of nroot[0] x nroot[1] (x nroot[2]) root cubes, i.e. a forest of pointer
  // trees (reading J-1 of DESIGN.md; PAPER.md:84 considers "perfect cubes" only, its 3-D runs use a
  // slab of 16 x 16 x 1 cubes).  roots[r], r = tx + nroot[0] * (ty + nroot[1] * tz); node
  // anchors are GLOBAL integer coordinates in [0, nroot[a] << maxl).  A single cube is the forest {1,1,1}.
  int nroot[3] = {1, 1, 1};
  std::vector<Node*> roots;
  std::vector<Node*> leaves;   // sorted by Morton ID
  std::vector<uint64_t> keys;  // their IDs
  // snapshot of the forest before the last adapt (T_o of Alg. 7)
  std::vector<Node*> old_roots;
  std::vector<Node*> old_leaves;
  std::vector<uint64_t> old_keys;
  bool have_old = false;
  std::vector<int32_t> map_src;
  std::vector<uint8_t> map_kind;
  Faces faces;
  Ops ops;
};

// ---------------------------------------------------------------- Alg. 1
// Morton encoding, PAPER.md:92-97 (Alg. 1) with readings A-1..A-3:
//  step 2: integer coordinates at the octant's own depth, xi = x >> (Dmax - D)
//  step 3: interleave, digit k = (z_k y_k x_k), x lowest                (:96)
//  step 4: pad dim*(Dmax - D) zero bits                                  (:97, garbled)
//  step 5: append the depth in m_b = 5 low bits                          (:97, :142)
uint64_t raw_id(int dim, int level, const uint32_t* xi_at_level) {
  uint64_t r = 0;
  for (int k = 0; k < level; ++k)
    for (int a = 0; a < dim; ++a)
      r |= (uint64_t)((xi_at_level[a] >> k) & 1u) << (dim * k + a);
  return r;  // "raw Morton ID": no padding, no depth
}

uint64_t encode(int dim, int maxl, int level, const uint32_t* x_finest) {
  uint32_t xi[3] = {0, 0, 0};
  for (int a = 0; a < dim; ++a) xi[a] = level == 0 ? 0u : (x_finest[a] >> (maxl - level));
  uint64_t r = raw_id(dim, level, xi);
  uint64_t padded = (maxl == level) ? r : (r << (dim * (maxl - level)));
  return (padded << kLevelBits) | (uint64_t)level;
}

void decode(int dim, int maxl, uint64_t key, int* level, uint32_t* x_finest) {
  *level = (int)(key & ((1u << kLevelBits) - 1));
  uint64_t r = key >> kLevelBits;
  for (int a = 0; a < 3; ++a) x_finest[a] = 0;
  for (int k = 0; k < maxl; ++k)
    for (int a = 0; a < dim; ++a)
      x_finest[a] |= (uint32_t)((r >> (dim * k + a)) & 1u) << k;
}

// Forest ID (reading J-1): the Morton ID of the octant inside its root cube (Alg. 1 on the
// coordinates relative to the cube) with the cube's index r placed above the dim * D_max path bits,
//   key = ((r << dim * D_max) | padded raw ID) << 5 | depth,
// so that ascending order is cube-major and a single cube (r = 0) keeps the paper's ID unchanged.
int root_index(const Tree* t, const uint32_t* x) {
  int r = 0, mul = 1;
  for (int a = 0; a < t->dim; ++a) {
    r += (int)(x[a] >> t->maxl) * mul;
    mul *= t->nroot[a];
  }
  return r;
}
uint64_t key_of(const Tree* t, const Node* n) {
  uint32_t rel[3] = {0, 0, 0};
  for (int a = 0; a < t->dim; ++a) rel[a] = n->x[a] & ((1u << t->maxl) - 1u);
  if (t->maxl == 0) rel[0] = rel[1] = rel[2] = 0;
  const uint64_t k = encode(t->dim, t->maxl, n->level, rel);
  return k | ((uint64_t)root_index(t, n->x) << (t->dim * t->maxl + kLevelBits));
}

// a is a strict ancestor of b (integer boxes; PAPER.md:84 half-open regions)
bool contains_strict(int dim, int maxl, int la, const uint32_t* xa, int lb, const uint32_t* xb) {
  if (la >= lb) return false;
  uint32_t wa = 1u << (maxl - la);
  for (int a = 0; a < dim; ++a)
    if (xb[a] < xa[a] || xb[a] >= xa[a] + wa) return false;
  return true;
}

// ---------------------------------------------------------------- tree basics
void free_subtree(Node* n) {
  if (!n) return;
  for (int c = 0; c < 8; ++c) free_subtree(n->child[c]);
  delete n;
}

// split: child k has anchor x0 + i*Delta/2, i = bits of k, x lowest (reading A-6)
void split(Tree* t, Node* n) {
  uint32_t h = 1u << (t->maxl - n->level - 1);
  for (int c = 0; c < t->nc; ++c) {
    Node* ch = new Node();
    ch->level = n->level + 1;
    for (int a = 0; a < t->dim; ++a) ch->x[a] = n->x[a] + (((c >> a) & 1) ? h : 0u);
    ch->parent = n;
    n->child[c] = ch;
  }
}

void merge(Tree* t, Node* n) {
  for (int c = 0; c < t->nc; ++c) {
    free_subtree(n->child[c]);
    n->child[c] = nullptr;
  }
}

Node* clone(const Node* n, Node* parent) {
  Node* m = new Node(*n);
  m->parent = parent;
  for (int c = 0; c < 8; ++c)
    if (n->child[c]) m->child[c] = clone(n->child[c], m);
  return m;
}

void dfs_leaves(Tree* t, Node* n, std::vector<Node*>& out) {
  if (n->is_leaf()) {
    out.push_back(n);
    return;
  }
  for (int c = 0; c < t->nc; ++c) dfs_leaves(t, n->child[c], out);
}

// list leaves by depth-first traversal, then std::sort on the 64-bit ID
void relist(Tree* t) {
  t->leaves.clear();
  for (Node* r : t->roots) dfs_leaves(t, r, t->leaves);
  std::vector<std::pair<uint64_t, Node*>> kv;
  kv.reserve(t->leaves.size());
  for (Node* n : t->leaves) kv.emplace_back(key_of(t, n), n);
  std::sort(kv.begin(), kv.end(), [](const auto& a, const auto& b) { return a.first < b.first; });
  t->keys.resize(kv.size());
  for (size_t i = 0; i < kv.size(); ++i) {
    t->keys[i] = kv[i].first;
    t->leaves[i] = kv[i].second;
    kv[i].second->idx = (int64_t)i;
  }
}

void list_into(Tree* t, const std::vector<Node*>& roots, std::vector<Node*>& lv, std::vector<uint64_t>& ks) {
  lv.clear();
  for (Node* r : roots) dfs_leaves(t, r, lv);
  std::sort(lv.begin(), lv.end(), [t](Node* a, Node* b) { return key_of(t, a) < key_of(t, b); });
  ks.resize(lv.size());
  for (size_t i = 0; i < lv.size(); ++i) {
    ks[i] = key_of(t, lv[i]);
    lv[i]->idx = (int64_t)i;
  }
}

// point location: pick the root cube that holds the integer point x, descend towards x, stop at a
// leaf or at depth `limit`
Node* locate(Tree* t, const std::vector<Node*>& roots, const uint32_t* x, int limit) {
  Node* n = roots[root_index(t, x)];
  while (!n->is_leaf() && n->level < limit) {
    int sh = t->maxl - n->level - 1;
    int c = 0;
    for (int a = 0; a < t->dim; ++a) c |= (int)((x[a] >> sh) & 1u) << a;
    n = n->child[c];
  }
  return n;
}

// same-level face neighbour anchor of `n` across local face f (reading D-1:
// 0=-x 1=+x 2=-y 3=+y 4=-z 5=+z), periodic wrap of integer coordinates
// (PAPER.md:267).  Returns false when the face is on a non-periodic boundary.
bool neighbour_anchor(const Tree* t, const Node* n, int f, uint32_t* nx) {
  int a = f >> 1;
  int64_t w = (int64_t)1 << (t->maxl - n->level);
  int64_t L = (int64_t)t->nroot[a] << t->maxl;  // width of the brick along a
  for (int b = 0; b < 3; ++b) nx[b] = n->x[b];
  int64_t v = (int64_t)n->x[a] + ((f & 1) ? w : -w);
  if (v < 0 || v >= L) {
    if (!t->periodic[a]) return false;
    v = (v + L) % L;
  }
  nx[a] = (uint32_t)v;
  return true;
}

// ---------------------------------------------------------------- Alg. 6
// Adaptation; readings B-1..B-4.
//  flags > 0 : refine (ignored at level == max_level)
//  flags < 0 : coarsen; honoured only when all 2^dim siblings are leaves and all
//              carry a coarsen flag (steps 3-4) and level > base_level
//  one level per call.
void adapt(Tree* t, const int8_t* flags) {
  // snapshot T_o for Alg. 7
  for (Node* r : t->old_roots) free_subtree(r);
  t->old_roots.clear();
  for (Node* r : t->roots) t->old_roots.push_back(clone(r, nullptr));
  list_into(t, t->old_roots, t->old_leaves, t->old_keys);
  t->have_old = true;

  std::vector<Node*> to_refine, to_merge;
  const int64_t M = (int64_t)t->leaves.size();
  for (int64_t i = 0; i < M; ++i) {
    Node* n = t->leaves[i];
    if (flags[i] > 0 && n->level < t->maxl) to_refine.push_back(n);
  }
  for (int64_t i = 0; i < M; ++i) {
    Node* n = t->leaves[i];
    Node* p = n->parent;
    if (!p || p->child[0] != n) continue;  // visit each sibling group once
    if (n->level <= t->base) continue;
    bool all = true;
    for (int c = 0; c < t->nc; ++c) {
      Node* s = p->child[c];
      if (!s->is_leaf() || !(flags[s->idx] < 0)) {
        all = false;
        break;
      }
    }
    if (all) to_merge.push_back(p);
  }
  for (Node* n : to_refine) split(t, n);
  for (Node* p : to_merge) merge(t, p);
  relist(t);
}

// ---------------------------------------------------------------- 2:1 balance
// PAPER.md:130-147, Alg. 4 (:153-161).  Face balance (reading C-1).  The result
// is the unique coarsest refinement in which face-adjacent leaves differ by at
// most one level (reading C-2); it is computed by Jacobi ripple sweeps (reading
// C-3): in one sweep every leaf L is examined against the tree as it stood at
// the start of the sweep; every face-neighbour leaf with level < level(L) - 1
// is marked; all marked leaves are split once.  Returns the number of sweeps
// that split at least one leaf.
// `conn` selects which neighbours count (reading C-1 / C-9): 1 = leaves sharing a face
// (BASELINE.json's contract); 2 = faces and edges -- the paper's own "strong" balance in
// 3-D, "any two adjacent octants that share either an edge or a face"; 3 =
// faces, edges and corners.  In 2-D a quadrant's edges ARE its faces, so 1 is already the
// paper's strong balance and 2 adds the corners.  A neighbour direction is an offset
// o in {-1,0,+1}^dim with 1 <= |o|_0 <= conn; the same-level neighbour anchor is x + o*w
// with periodic wrap per axis, directions leaving a non-periodic domain
// are skipped.
bool offset_anchor(const Tree* t, const Node* n, const int* o, uint32_t* nx) {
  const int64_t w = (int64_t)1 << (t->maxl - n->level);
  for (int b = 0; b < 3; ++b) nx[b] = n->x[b];
  for (int a = 0; a < t->dim; ++a) {
    if (!o[a]) continue;
    const int64_t L = (int64_t)t->nroot[a] << t->maxl;
    int64_t v = (int64_t)n->x[a] + o[a] * w;
    if (v < 0 || v >= L) {
      if (!t->periodic[a]) return false;
      v = (v + L) % L;
    }
    nx[a] = (uint32_t)v;
  }
  return true;
}

int balance(Tree* t, int64_t* n_split_total, int conn) {
  int iters = 0;
  int64_t total = 0;
  for (;;) {
    std::vector<Node*> marked;
    for (Node* L : t->leaves) {
      int o[3] = {0, 0, 0};
      for (o[0] = -1; o[0] <= 1; ++o[0])
        for (o[1] = -1; o[1] <= 1; ++o[1])
          for (o[2] = (t->dim == 3 ? -1 : 0); o[2] <= (t->dim == 3 ? 1 : 0); ++o[2]) {
            const int nnz = (o[0] != 0) + (o[1] != 0) + (o[2] != 0);
            if (nnz < 1 || nnz > conn) continue;
            uint32_t nx[3];
            if (!offset_anchor(t, L, o, nx)) continue;
            Node* N = locate(t, t->roots, nx, L->level);
            if (N->is_leaf() && N->level < L->level - 1 && !N->mark) {
              N->mark = true;
              marked.push_back(N);
            }
          }
    }
    if (marked.empty()) break;
    for (Node* N : marked) {
      N->mark = false;
      split(t, N);
    }
    total += (int64_t)marked.size();
    ++iters;
    relist(t);
  }
  if (n_split_total) *n_split_total = total;
  return iters;
}

// ---------------------------------------------------------------- Alg. 5
// Face connectivity.  Per (element, face) slot (reading D-2):
//   kind 0 boundary (nbr -1); 1 conforming; 2 | slot<<4 neighbour coarser;
//   3 neighbour finer (nbr = the slot-0 fine neighbour).
// slot (reading D-3) = position of the fine face inside the coarse face,
// tangential axes ascending, smaller coordinate first.
// Returns 0, or -1 if a level jump > 1 is met (reading D-5).
int slot_of(const Tree* t, const Node* fine, const Node* coarse, int axis) {
  uint32_t wf = 1u << (t->maxl - fine->level);
  int s = 0, bit = 0;
  for (int a = 0; a < t->dim; ++a) {
    if (a == axis) continue;
    uint32_t rel = (fine->x[a] - coarse->x[a]) / wf;  // 0 or 1: geometric position
    s |= (int)(rel & 1u) << bit;
    ++bit;
  }
  return s;
}

int connect_descent(Tree* t, std::vector<int32_t>& nbr, std::vector<uint8_t>& kind) {
  const int64_t M = (int64_t)t->leaves.size();
  nbr.assign((size_t)M * t->nf, -1);
  kind.assign((size_t)M * t->nf, 0);
  for (int64_t e = 0; e < M; ++e) {
    Node* L = t->leaves[e];
    for (int f = 0; f < t->nf; ++f) {
      uint32_t nx[3];
      size_t s = (size_t)e * t->nf + f;
      if (!neighbour_anchor(t, L, f, nx)) continue;  // boundary
      Node* N = locate(t, t->roots, nx, L->level);
      if (N->is_leaf()) {
        if (N->level == L->level) {
          kind[s] = 1;
          nbr[s] = (int32_t)N->idx;
        } else if (N->level == L->level - 1) {
          kind[s] = (uint8_t)(2 | (slot_of(t, L, N, f >> 1) << 4));
          nbr[s] = (int32_t)N->idx;
        } else {
          return -1;
        }
      } else {
        // finer neighbours: the child of N that touches the face and has
        // tangential bits 0 (reading D-2)
        int c = (f & 1) ? 0 : (1 << (f >> 1));
        Node* F = N->child[c];
        if (!F->is_leaf()) return -1;
        kind[s] = 3;
        nbr[s] = (int32_t)F->idx;
      }
    }
  }
  return 0;
}

// Brute force over all pairs (tiny meshes): two leaves are face neighbours
// across axis a iff their integer boxes abut along a (mod domain width if
// periodic) and overlap with positive (dim-1)-measure in the other axes.
int connect_bruteforce(Tree* t, std::vector<int32_t>& nbr, std::vector<uint8_t>& kind) {
  const int64_t M = (int64_t)t->leaves.size();
  nbr.assign((size_t)M * t->nf, -1);
  kind.assign((size_t)M * t->nf, 0);
  for (int64_t e = 0; e < M; ++e) {
    Node* A = t->leaves[e];
    int64_t wa = (int64_t)1 << (t->maxl - A->level);
    for (int f = 0; f < t->nf; ++f) {
      int ax = f >> 1;
      const int64_t Lw = (int64_t)t->nroot[ax] << t->maxl;  // width of the brick along ax
      size_t s = (size_t)e * t->nf + f;
      // plane coordinate the neighbour must start/end at
      int64_t plane = (f & 1) ? (int64_t)A->x[ax] + wa : (int64_t)A->x[ax];
      bool wrapped = false;
      if (f & 1) {
        if (plane == Lw) { plane = 0; wrapped = true; }
      } else {
        if (plane == 0) { plane = Lw; wrapped = true; }
      }
      if (wrapped && !t->periodic[ax]) continue;  // boundary
      std::vector<Node*> touching;
      for (int64_t g = 0; g < M; ++g) {
        Node* B = t->leaves[g];
        int64_t wb = (int64_t)1 << (t->maxl - B->level);
        int64_t bface = (f & 1) ? (int64_t)B->x[ax] : (int64_t)B->x[ax] + wb;
        if (bface != plane) continue;
        bool overlap = true;
        for (int a = 0; a < t->dim; ++a) {
          if (a == ax) continue;
          int64_t lo = std::max<int64_t>(A->x[a], B->x[a]);
          int64_t hi = std::min<int64_t>((int64_t)A->x[a] + wa, (int64_t)B->x[a] + wb);
          if (hi <= lo) overlap = false;
        }
        if (overlap) touching.push_back(B);
      }
      if (touching.empty()) return -2;  // incomplete tree
      if (touching.size() == 1) {
        Node* B = touching[0];
        if (B->level == A->level) {
          kind[s] = 1;
          nbr[s] = (int32_t)B->idx;
        } else if (B->level == A->level - 1) {
          kind[s] = (uint8_t)(2 | (slot_of(t, A, B, ax) << 4));
          nbr[s] = (int32_t)B->idx;
        } else {
          return -1;
        }
      } else {
        if ((int)touching.size() != (1 << (t->dim - 1))) return -1;
        Node* first = nullptr;
        for (Node* B : touching) {
          if (B->level != A->level + 1) return -1;
          bool is_first = true;  // smallest tangential coordinates
          for (int a = 0; a < t->dim; ++a)
            if (a != ax && B->x[a] != A->x[a]) is_first = false;
          if (is_first) first = B;
        }
        if (!first) return -1;
        kind[s] = 3;
        nbr[s] = (int32_t)first->idx;
      }
    }
  }
  return 0;
}

// Face tables in canonical order (reading D-4): leaves in array order, local
// faces 0..nf-1; a conforming face is emitted by the element on its minus side
// (local face odd) as (e, nbr), axis = f>>1; a hanging face by the fine element
// as (e_fine, e_coarse), info = f | slot<<3; a boundary face by its element.
void face_tables(Tree* t) {
  Faces& F = t->faces;
  F.conf.clear(); F.conf_axis.clear(); F.hang.clear(); F.hang_info.clear();
  F.bnd.clear(); F.bnd_face.clear();
  const int64_t M = (int64_t)t->leaves.size();
  for (int64_t e = 0; e < M; ++e)
    for (int f = 0; f < t->nf; ++f) {
      size_t s = (size_t)e * t->nf + f;
      int k = F.kind[s] & 0xF;
      if (k == 0) {
        F.bnd.push_back((int32_t)e);
        F.bnd_face.push_back((uint8_t)f);
      } else if (k == 1) {
        if (f & 1) {
          F.conf.push_back((int32_t)e);
          F.conf.push_back(F.nbr[s]);
          F.conf_axis.push_back((uint8_t)(f >> 1));
        }
      } else if (k == 2) {
        F.hang.push_back((int32_t)e);
        F.hang.push_back(F.nbr[s]);
        F.hang_info.push_back((uint8_t)(f | ((F.kind[s] >> 4) << 3)));
      }
    }
}

// ---------------------------------------------------------------- Alg. 7
// Old/new mapping, computed on the integer boxes: for each
// new leaf descend the OLD tree towards its anchor:
//   old leaf, same level      -> kind 0 copy,    src = old index
//   old leaf, one level above -> kind 1 | child<<4 refine, src = old index
//   old interior node at the new leaf's level whose children are all leaves
//                             -> kind 2 coarsen, src = old index of first child
// anything else -> error (reading: LT_ERR_MAPPING).
int build_map(Tree* t) {
  const int64_t M = (int64_t)t->leaves.size();
  t->map_src.assign((size_t)M, -1);
  t->map_kind.assign((size_t)M, 0);
  if (!t->have_old) {  // identity (state rule)
    for (int64_t j = 0; j < M; ++j) t->map_src[j] = (int32_t)j;
    return 0;
  }
  for (int64_t j = 0; j < M; ++j) {
    Node* L = t->leaves[j];
    Node* O = locate(t, t->old_roots, L->x, L->level);
    if (O->is_leaf()) {
      if (O->level == L->level) {
        t->map_kind[j] = 0;
        t->map_src[j] = (int32_t)O->idx;
      } else if (O->level == L->level - 1) {
        int sh = t->maxl - L->level;
        int c = 0;
        for (int a = 0; a < t->dim; ++a) c |= (int)((L->x[a] >> sh) & 1u) << a;
        t->map_kind[j] = (uint8_t)(1 | (c << 4));
        t->map_src[j] = (int32_t)O->idx;
      } else {
        return -1;
      }
    } else {
      for (int c = 0; c < t->nc; ++c)
        if (!O->child[c]->is_leaf()) return -1;
      for (int c = 1; c < t->nc; ++c)
        if (O->child[c]->idx != O->child[0]->idx + c) return -1;
      t->map_kind[j] = 2;
      t->map_src[j] = (int32_t)O->child[0]->idx;
    }
  }
  return 0;
}

// ---------------------------------------------------------------- quadrature
// n-point Gauss-Legendre rule on [-1,1]: Newton iteration on P_n via the
// three-term recurrence.  Pinned in tests against closed forms (n = 1,2,3),
// sum of weights and monomial exactness.
void gauss_legendre(int n, std::vector<double>& z, std::vector<double>& w) {
  z.assign(n, 0.0);
  w.assign(n, 0.0);
  for (int i = 0; i < n; ++i) {
    double x = -std::cos(M_PI * (i + 0.75) / (n + 0.5));
    for (int it = 0; it < 100; ++it) {
      double p0 = 1.0, p1 = x;
      for (int k = 2; k <= n; ++k) {
        double pk = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / k;
        p0 = p1;
        p1 = pk;
      }
      if (n == 1) { p0 = 1.0; p1 = x; }
      double dp = n * (x * p1 - p0) / (x * x - 1.0);
      double dx = p1 / dp;
      x -= dx;
      if (std::fabs(dx) < 1e-16) break;
    }
    double p0 = 1.0, p1 = x;
    for (int k = 2; k <= n; ++k) {
      double pk = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / k;
      p0 = p1;
      p1 = pk;
    }
    double dp = n * (x * p1 - p0) / (x * x - 1.0);
    z[i] = x;
    w[i] = 2.0 / ((1.0 - x * x) * dp * dp);
  }
  for (int i = 0; i < n / 2; ++i) {  // symmetrise
    double s = 0.5 * (z[n - 1 - i] - z[i]);
    z[i] = -s;
    z[n - 1 - i] = s;
    double ww = 0.5 * (w[i] + w[n - 1 - i]);
    w[i] = w[n - 1 - i] = ww;
  }
  if (n % 2) z[n / 2] = 0.0;
}

// 1-D Lagrange polynomial l_i through nodes z (Eq. 3) at x
double lagrange(const std::vector<double>& z, int i, double x) {
  double v = 1.0;
  for (size_t k = 0; k < z.size(); ++k)
    if ((int)k != i) v *= (x - z[k]) / (z[i] - z[k]);
  return v;
}

// tensor-product Lagrange basis function n (x fastest; reading E-5) at xi
double tensor_lagrange(const std::vector<double>& z, int dim, int n, const double* xi) {
  int P1 = (int)z.size();
  double v = 1.0;
  for (int a = 0; a < dim; ++a) {
    v *= lagrange(z, n % P1, xi[a]);
    n /= P1;
  }
  return v;
}

// Solve A X = B in place (A: n x n, B: n x m, row major), partial pivoting
void solve_dense(std::vector<double> A, int n, std::vector<double>& B, int m) {
  for (int k = 0; k < n; ++k) {
    int piv = k;
    for (int r = k + 1; r < n; ++r)
      if (std::fabs(A[(size_t)r * n + k]) > std::fabs(A[(size_t)piv * n + k])) piv = r;
    if (piv != k) {
      for (int c = 0; c < n; ++c) std::swap(A[(size_t)k * n + c], A[(size_t)piv * n + c]);
      for (int c = 0; c < m; ++c) std::swap(B[(size_t)k * m + c], B[(size_t)piv * m + c]);
    }
    double d = A[(size_t)k * n + k];
    for (int r = k + 1; r < n; ++r) {
      double f = A[(size_t)r * n + k] / d;
      if (f == 0.0) continue;
      for (int c = k; c < n; ++c) A[(size_t)r * n + c] -= f * A[(size_t)k * n + c];
      for (int c = 0; c < m; ++c) B[(size_t)r * m + c] -= f * B[(size_t)k * m + c];
    }
  }
  for (int k = n - 1; k >= 0; --k) {
    for (int c = 0; c < m; ++c) {
      double s = B[(size_t)k * m + c];
      for (int j = k + 1; j < n; ++j) s -= A[(size_t)k * n + j] * B[(size_t)j * m + c];
      B[(size_t)k * m + c] = s / A[(size_t)k * n + k];
    }
  }
}

// Transfer operators, PAPER.md:204-255 (section 4.2), readings E-1..E-4.
//  solution points: p+1 Gauss-Legendre points per direction (E-1)
//  interp[c] : Eq. 8 evaluated at child c's solution points; child c occupies
//              xi_a in [b_a - 1, b_a] with b_a = (c>>a)&1, i.e.
//              xi = (z + 2b - 1)/2                                     (:210, :230)
//  M, S_c    : Eq. 13 by (p+6)-point tensor Gauss quadrature, S_c integrated over
//              child c's region (reading E-3)
//  proj[c]   = M^{-1} S_c by dense Gaussian elimination               (Eq. 12)
void build_ops_dim(Ops& o, int dim, int p) {
  if (o.p == p && o.dim == dim) return;
  const int nc = 1 << dim, P1 = p + 1;
  int N = 1;
  for (int a = 0; a < dim; ++a) N *= P1;
  o.dim = dim; o.p = p; o.N = N;
  std::vector<double> z, w, qz, qw;
  gauss_legendre(P1, z, w);
  gauss_legendre(p + 6, qz, qw);
  const int Q = p + 6;
  int NQ = 1;
  for (int a = 0; a < dim; ++a) NQ *= Q;

  o.interp.assign((size_t)nc * N * N, 0.0);
  for (int c = 0; c < nc; ++c)
    for (int n = 0; n < N; ++n) {
      double xi[3];
      int r = n;
      for (int a = 0; a < dim; ++a) {
        int b = (c >> a) & 1;
        xi[a] = 0.5 * (z[r % P1] + 2.0 * b - 1.0);
        r /= P1;
      }
      for (int m = 0; m < N; ++m)
        o.interp[((size_t)c * N + n) * N + m] = tensor_lagrange(z, dim, m, xi);
    }

  // mass matrix over the parent, in parent reference coordinates
  o.mass.assign((size_t)N * N, 0.0);
  for (int q = 0; q < NQ; ++q) {
    double xi[3], wq = 1.0;
    int r = q;
    for (int a = 0; a < dim; ++a) {
      xi[a] = qz[r % Q];
      wq *= qw[r % Q];
      r /= Q;
    }
    std::vector<double> l(N);
    for (int n = 0; n < N; ++n) l[n] = tensor_lagrange(z, dim, n, xi);
    for (int j = 0; j < N; ++j)
      for (int i = 0; i < N; ++i) o.mass[(size_t)j * N + i] += wq * l[j] * l[i];
  }
  // S_c over child c: xi = (zeta + 2b - 1)/2, d xi = 2^-dim d zeta
  o.S.assign((size_t)nc * N * N, 0.0);
  const double jac = std::ldexp(1.0, -dim);
  for (int c = 0; c < nc; ++c)
    for (int q = 0; q < NQ; ++q) {
      double zeta[3], xi[3], wq = jac;
      int r = q;
      for (int a = 0; a < dim; ++a) {
        int b = (c >> a) & 1;
        zeta[a] = qz[r % Q];
        xi[a] = 0.5 * (zeta[a] + 2.0 * b - 1.0);
        wq *= qw[r % Q];
        r /= Q;
      }
      std::vector<double> lp(N), lc(N);
      for (int n = 0; n < N; ++n) {
        lp[n] = tensor_lagrange(z, dim, n, xi);
        lc[n] = tensor_lagrange(z, dim, n, zeta);
      }
      for (int j = 0; j < N; ++j)
        for (int i = 0; i < N; ++i) o.S[((size_t)c * N + j) * N + i] += wq * lp[j] * lc[i];
    }
  o.proj.assign((size_t)nc * N * N, 0.0);
  for (int c = 0; c < nc; ++c) {
    std::vector<double> B(o.S.begin() + (size_t)c * N * N, o.S.begin() + (size_t)(c + 1) * N * N);
    solve_dense(o.mass, N, B, N);
    std::copy(B.begin(), B.end(), o.proj.begin() + (size_t)c * N * N);
  }
}

void build_ops(Tree* t, int p) { build_ops_dim(t->ops, t->dim, p); }

// u[e][v][n] (reading E-5).  Rows [j0, j1) of the new tree are produced.
void transfer_rows(Tree* t, const double* u_old, double* u_new_rows, int nvars, int64_t j0, int64_t j1) {
  const Ops& o = t->ops;
  const int N = o.N, nc = t->nc;
  const size_t E = (size_t)nvars * N;
  for (int64_t j = j0; j < j1; ++j) {
    double* dst = u_new_rows + (size_t)(j - j0) * E;
    int kind = t->map_kind[j] & 0xF;
    int64_t src = t->map_src[j];
    if (kind == 0) {
      std::memcpy(dst, u_old + (size_t)src * E, E * sizeof(double));
    } else if (kind == 1) {
      int c = t->map_kind[j] >> 4;
      const double* I = &o.interp[(size_t)c * N * N];
      for (int v = 0; v < nvars; ++v) {
        const double* up = u_old + (size_t)src * E + (size_t)v * N;
        for (int n = 0; n < N; ++n) {
          double s = 0.0;
          for (int m = 0; m < N; ++m) s += I[(size_t)n * N + m] * up[m];
          dst[(size_t)v * N + n] = s;
        }
      }
    } else {
      for (int v = 0; v < nvars; ++v)
        for (int n = 0; n < N; ++n) {
          double s = 0.0;
          for (int c = 0; c < nc; ++c) {
            const double* R = &o.proj[(size_t)c * N * N];
            const double* uc = u_old + (size_t)(src + c) * E + (size_t)v * N;
            for (int m = 0; m < N; ++m) s += R[(size_t)n * N + m] * uc[m];
          }
          dst[(size_t)v * N + n] = s;
        }
    }
  }
}

// ---------------------------------------------------------------- Alg. 3
// Linearisation: reverse, std::unique with the binary
// predicate "two consecutive Morton IDs are overlapping", reverse back.
bool overlapping(int dim, int maxl, uint64_t a, uint64_t b) {
  int la, lb;
  uint32_t xa[3], xb[3];
  decode(dim, maxl, a, &la, xa);
  decode(dim, maxl, b, &lb, xb);
  if (a == b) return true;
  return contains_strict(dim, maxl, la, xa, lb, xb) || contains_strict(dim, maxl, lb, xb, la, xa);
}

int64_t sort_linearise(int dim, int maxl, uint64_t* keys, int64_t n) {
  std::sort(keys, keys + n);
  std::reverse(keys, keys + n);
  uint64_t* e = std::unique(keys, keys + n,
                            [=](uint64_t a, uint64_t b) { return overlapping(dim, maxl, a, b); });
  int64_t m = e - keys;
  std::reverse(keys, keys + m);
  return m;
}

bool complete_subtree(const Tree* t, const Node* n) {
  if (n->is_leaf()) return true;
  for (int c = 0; c < t->nc; ++c) {
    if (!n->child[c]) return false;
    if (!complete_subtree(t, n->child[c])) return false;
  }
  return true;
}

Tree* new_tree(int dim, int base, int maxl, const int* periodic, const int* nroot = nullptr) {
  if (dim != 2 && dim != 3) return nullptr;
  if (base < 0 || base > maxl) return nullptr;
  int64_t ntrees = 1;
  for (int a = 0; a < dim; ++a) {
    const int na = nroot ? nroot[a] : 1;
    if (na < 1 || ((int64_t)na << maxl) > ((int64_t)1 << 31)) return nullptr;
    ntrees *= na;
  }
  int tbits = 0;
  while (((int64_t)1 << tbits) < ntrees) ++tbits;
  if (dim * maxl + kLevelBits + tbits > 63 || maxl > 31) return nullptr;
  Tree* t = new Tree();
  t->dim = dim; t->base = base; t->maxl = maxl;
  t->nc = 1 << dim; t->nf = 2 * dim;
  for (int a = 0; a < dim; ++a) {
    t->periodic[a] = periodic ? periodic[a] : 0;
    t->nroot[a] = nroot ? nroot[a] : 1;
  }
  // one pointer tree per root cube, anchors in global integer coordinates
  for (int64_t r = 0; r < ntrees; ++r) {
    Node* n = new Node();
    int64_t q = r;
    for (int a = 0; a < dim; ++a) {
      n->x[a] = (uint32_t)((q % t->nroot[a]) << maxl);
      q /= t->nroot[a];
    }
    t->roots.push_back(n);
  }
  return t;
}

void refine_uniform(Tree* t, Node* n, int to_level) {
  if (n->level >= to_level) return;
  split(t, n);
  for (int c = 0; c < t->nc; ++c) refine_uniform(t, n->child[c], to_level);
}


// ---------------------------------------------------------------- Alg. 2
// Tree construction from scattered points and completion, PAPER.md:105-120 (section 3.1,
// Alg. 2).  The paper completes the sorted initial octants by splitting the largest common
// ancestor of consecutive octants and keeping the children that lie between them; the
// result it reaches is the plainly defined one computed here (readings G-2, G-3 of
// DESIGN.md): the COARSEST complete tree that refines the uniform depth-D_min tree
// (D_min = base_level) and has every input octant as a leaf -- or as
// an interior node when a finer input octant lies inside it (linearisation keeps the
// finer one, Alg. 3).  On a pointer tree that is: walk from the root to
// the octant and split every leaf met on the way.  Order of insertion does not matter.
void insert_octant(Tree* t, int lvl, const uint32_t* x) {  // single cube only (construction)
  Node* nd = t->roots[0];
  while (nd->level < lvl) {
    if (nd->is_leaf()) split(t, nd);
    int sh = t->maxl - nd->level - 1;
    int c = 0;
    for (int a = 0; a < t->dim; ++a) c |= (int)((x[a] >> sh) & 1u) << a;
    nd = nd->child[c];
  }
}

// Alg. 1 steps 1-2 / Alg. 2 step 1 for a scattered point: integer
// coordinate of the depth-D_max cell that contains it (half-open cells).
// Reading G-1: xi = floor((x - lo) / (hi - lo) * 2^D_max) evaluated in fp64 in exactly
// this order, clamped to [0, 2^D_max - 1] (points on or beyond the upper boundary fall
// into the last cell).
uint32_t point_cell(double x, double lo, double hi, int maxl) {
  double s = (x - lo) / (hi - lo);
  double v = std::floor(s * (double)((uint64_t)1 << maxl));
  double top = (double)(((uint64_t)1 << maxl) - 1);
  if (!(v >= 0.0)) v = 0.0;  // also catches NaN
  if (v > top) v = top;
  return (uint32_t)v;
}


// ---------------------------------------------------------------- Alg. 8 (mortars)
// Common-flux plumbing on nonconforming faces, PAPER.md:265-314 (section 4.3, Alg. 8 steps
// 2 and 4, Eq. 14-20); readings H-1..H-4 of DESIGN.md.
//  face points : the (p+1)^(dim-1) Gauss-Legendre points of the face, tangential axes in
//                ascending order, lower axis fastest; N = (k+1)^(dim-1) (Eq. 14)      (H-1)
//  mortars     : the 2^(dim-1) mortar faces of a coarse face coincide with the fine
//                neighbours' faces, mortar s = slot s of lt_connect (fine side <-> mortar
//                is "a direct copy", :273)                                              (H-2)
//  Eq. 17      : M^ u^ = S u,  M^_ji = int_Xi l^_j l^_i dz,  S_ji = int_Xi l^_j l_i(xi(z)) dz
//  Eq. 20      : M F = sum_s S^s F^s,  M_ji = int_Oc l_j l_i dxi,  S^s_ji = int_Oc^s l_j l^_i dxi
//                (the sum runs over the 2^(dim-1) mortars; "2^dim - 1" at :310 is a typo) (H-3)
// All integrals by (p+6)-point tensor Gauss quadrature, systems solved densely.
struct FaceOps {
  int fdim = -1, p = -1, N = 0;
  Ops coarse;                  // operators of the (dim-1)-dimensional face: .proj[s] = M^-1 S^s (Eq. 20)
  std::vector<double> to_mortar;  // [ns][N][N]  (M^)^-1 S of Eq. 17 for mortar s
};

void build_face_ops(FaceOps& fo, int dim, int p) {
  const int fdim = dim - 1;
  if (fo.fdim == fdim && fo.p == p) return;
  build_ops_dim(fo.coarse, fdim, p);
  const int P1 = p + 1, ns = 1 << fdim, Q = p + 6;
  int N = 1, NQ = 1;
  for (int a = 0; a < fdim; ++a) { N *= P1; NQ *= Q; }
  fo.fdim = fdim; fo.p = p; fo.N = N;
  std::vector<double> z, w, qz, qw;
  gauss_legendre(P1, z, w);
  gauss_legendre(Q, qz, qw);
  fo.to_mortar.assign((size_t)ns * N * N, 0.0);
  for (int s = 0; s < ns; ++s) {
    std::vector<double> Mh((size_t)N * N, 0.0), Sh((size_t)N * N, 0.0);
    for (int q = 0; q < NQ; ++q) {
      double zeta[3] = {0, 0, 0}, xi[3] = {0, 0, 0}, wq = 1.0;  // zeta: mortar coordinates, xi: coarse-face coordinates
      int r = q;
      for (int a = 0; a < fdim; ++a) {
        const int b = (s >> a) & 1;
        zeta[a] = qz[r % Q];
        xi[a] = 0.5 * (zeta[a] + 2.0 * b - 1.0);
        wq *= qw[r % Q];
        r /= Q;
      }
      std::vector<double> lh(N), lc(N);
      for (int n = 0; n < N; ++n) {
        lh[n] = tensor_lagrange(z, fdim, n, zeta);
        lc[n] = tensor_lagrange(z, fdim, n, xi);
      }
      for (int j = 0; j < N; ++j)
        for (int i = 0; i < N; ++i) {
          Mh[(size_t)j * N + i] += wq * lh[j] * lh[i];
          Sh[(size_t)j * N + i] += wq * lh[j] * lc[i];
        }
    }
    solve_dense(Mh, N, Sh, N);
    std::copy(Sh.begin(), Sh.end(), fo.to_mortar.begin() + (size_t)s * N * N);
  }
}

// Alg. 8 step 2 for every face slot (e, f); face arrays are [n_leaves][nf][nvars][N] (H-4):
//   kind 1 (conforming):        u_nb[e][f] = u_f[nbr][f^1]                   (copy)
//   kind 2 (neighbour coarser): u_nb[e][f] = (M^)^-1 S u_f[nbr][f^1] for mortar `slot` (Eq. 17)
//   kind 0 / 3:                 left untouched
void mortar_project(Tree* t, const FaceOps& fo, const double* uf, double* unb, int nvars) {
  const int nf = t->nf, N = fo.N;
  const size_t E = (size_t)nvars * N;
  const int64_t M = (int64_t)t->leaves.size();
  for (int64_t e = 0; e < M; ++e)
    for (int f = 0; f < nf; ++f) {
      const size_t sl = (size_t)e * nf + f;
      const int kd = t->faces.kind[sl] & 15, slot = t->faces.kind[sl] >> 4;
      if (kd != 1 && kd != 2) continue;
      const double* src = uf + ((size_t)t->faces.nbr[sl] * nf + (f ^ 1)) * E;
      double* dst = unb + sl * E;
      for (int v = 0; v < nvars; ++v)
        for (int n = 0; n < N; ++n) {
          if (kd == 1) {
            dst[(size_t)v * N + n] = src[(size_t)v * N + n];
          } else {
            double acc = 0.0;
            for (int m = 0; m < N; ++m) acc += fo.to_mortar[((size_t)slot * N + n) * N + m] * src[(size_t)v * N + m];
            dst[(size_t)v * N + n] = acc;
          }
        }
    }
}

// Alg. 8 step 4 for every coarse face slot (kind 3): F[e][f] = M^-1 sum_s S^s F^[e_s][f^1]
// (Eq. 20), e_s = the fine neighbour occupying mortar s.  Other slots are left untouched.
// Returns -1 if a fine neighbour is missing (tree not balanced).
int mortar_gather(Tree* t, const FaceOps& fo, const double* fm, double* ff, int nvars) {
  const int nf = t->nf, N = fo.N, ns = 1 << (t->dim - 1);
  const size_t E = (size_t)nvars * N;
  const int64_t M = (int64_t)t->leaves.size();
  for (int64_t e = 0; e < M; ++e)
    for (int f = 0; f < nf; ++f) {
      const size_t sl = (size_t)e * nf + f;
      if ((t->faces.kind[sl] & 15) != 3) continue;
      Node* L = t->leaves[e];
      uint32_t nx[3];
      if (!neighbour_anchor(t, L, f, nx)) return -1;
      Node* Nn = locate(t, t->roots, nx, L->level);
      if (Nn->is_leaf() || Nn->level != L->level) return -1;
      const int axis = f >> 1;
      std::vector<double> acc(E, 0.0);
      for (int s = 0; s < ns; ++s) {
        // the child of the neighbour cell that touches the face and sits at tangential position s
        int c = (f & 1) ? 0 : (1 << axis), bit = 0;
        for (int a = 0; a < t->dim; ++a) {
          if (a == axis) continue;
          c |= ((s >> bit) & 1) << a;
          ++bit;
        }
        Node* F = Nn->child[c];
        if (!F->is_leaf()) return -1;
        const double* src = fm + ((size_t)F->idx * nf + (f ^ 1)) * E;
        for (int v = 0; v < nvars; ++v)
          for (int n = 0; n < N; ++n) {
            double a2 = 0.0;
            for (int m = 0; m < N; ++m) a2 += fo.coarse.proj[((size_t)s * N + n) * N + m] * src[(size_t)v * N + m];
            acc[(size_t)v * N + n] += a2;
          }
      }
      std::copy(acc.begin(), acc.end(), ff + sl * E);
    }
  return 0;
}


// Alg. 8 step 1: "Interpolate the solution from interior solution points to local
// flux points."  The solution of an element is the tensor Lagrange expansion on its (p+1)^dim
// Gauss-Legendre points (Eq. 8 / reading E-1); the flux points of face f are the Gauss-Legendre
// points of the face (reading H-1), i.e. the reference point xi with xi_axis = -1 (f even) or +1
// (f odd) and the tangential coordinates z[n_t].  Evaluated directly:
//   u_f[e][f][v][n] = sum_m l_m(xi_n) u[e][v][m].
void face_interp(const Tree* t, int p, const double* u, double* uf, int nvars) {
  const int dim = t->dim, nf = t->nf, P1 = p + 1;
  int N = 1, Nf = 1;
  for (int a = 0; a < dim; ++a) N *= P1;
  for (int a = 0; a + 1 < dim; ++a) Nf *= P1;
  std::vector<double> z, w;
  gauss_legendre(P1, z, w);
  const int64_t M = (int64_t)t->leaves.size();
  for (int f = 0; f < nf; ++f) {
    const int axis = f >> 1;
    // row n of the face operator: values of the N volume basis functions at face point n
    std::vector<double> op((size_t)Nf * N);
    for (int n = 0; n < Nf; ++n) {
      double xi[3] = {0, 0, 0};
      int r = n;
      for (int a = 0; a < dim; ++a) {
        if (a == axis) {
          xi[a] = (f & 1) ? 1.0 : -1.0;
        } else {
          xi[a] = z[r % P1];
          r /= P1;
        }
      }
      for (int m = 0; m < N; ++m) op[(size_t)n * N + m] = tensor_lagrange(z, dim, m, xi);
    }
    for (int64_t e = 0; e < M; ++e)
      for (int v = 0; v < nvars; ++v) {
        const double* src = u + ((size_t)e * nvars + v) * N;
        double* dst = uf + (((size_t)e * nf + f) * nvars + v) * Nf;
        for (int n = 0; n < Nf; ++n) {
          double acc = 0.0;
          for (int m = 0; m < N; ++m) acc += op[(size_t)n * N + m] * src[m];
          dst[n] = acc;
        }
      }
  }
}


// ---------------------------------------------------------------- FR right-hand side (Eq. 1-6)
// The flux reconstruction update around the adaptation cycle, PAPER.md:51-76 (section 2.1) and
// Alg. 8 step 3 ("we use a Rusanov solver"); readings I-1..I-5 of DESIGN.md.
//  I-1  conservation law = compressible Euler (the paper's vortex test, Eq. 21),
//       conserved variables (rho, rho u, rho v[, rho w], E), gamma = 1.4,
//       p = (gamma-1)(E - rho |v|^2 / 2), flux along axis a:
//       F_a = (rho v_a, rho v v_a + p e_a, (E + p) v_a).
//  I-2  Rusanov common flux along +a between the minus-side state uL and the plus-side state uR:
//       F* = (F_a(uL) + F_a(uR))/2 - lambda (uR - uL)/2, lambda = max(|v_a| + c) over both, c^2 = gamma p / rho.
//  I-3  correction functions = Radau polynomials ("to recover the discontinuous Galerkin method",
//       PAPER.md:67): g_L = (-1)^(k+1) (P_(k+1) - P_k)/2 (g_L(-1) = 1, g_L(1) = 0), g_R(xi) = g_L(-xi).
//  I-4  Eq. 4-5 per axis: d f/dx = (2/dx) [ sum_j l_j'(z_i) f_j + g_L'(z_i)(F*_- - f(-1)) + g_R'(z_i)(F*_+ - f(1)) ],
//       f(+-1) = sum_j l_j(+-1) f_j (Eq. 3), dx = domain width / 2^level ("inferred from the encoded
//       information of each element"); R = - sum_a d F_a / d x_a.
//  I-5  F* lives in the face array at the element's own slot (e, 2a) / (e, 2a+1), always as the
//       flux along +a, at the face point whose tangential indices are those of the solution point.
double legendre(int n, double x) {
  double pm = 1.0, pc = x;
  if (n == 0) return 1.0;
  for (int k = 1; k < n; ++k) {
    double pn = ((2 * k + 1) * x * pc - k * pm) / (k + 1);
    pm = pc;
    pc = pn;
  }
  return pc;
}
double legendre_d(int n, double x) {  // P_n'(x) = n (x P_n - P_(n-1)) / (x^2 - 1), interior x
  if (n == 0) return 0.0;
  return n * (x * legendre(n, x) - legendre(n - 1, x)) / (x * x - 1.0);
}
double lagrange_d(const std::vector<double>& z, int j, double x) {  // l_j'(x)
  double s = 0.0;
  for (size_t m = 0; m < z.size(); ++m) {
    if ((int)m == j) continue;
    double t = 1.0 / (z[j] - z[m]);
    for (size_t k = 0; k < z.size(); ++k)
      if ((int)k != j && k != m) t *= (x - z[k]) / (z[j] - z[k]);
    s += t;
  }
  return s;
}

struct FrOps {
  int p = -1;
  std::vector<double> z, w, D, lm, lp, gl, gr;  // D[i][j] = l_j'(z_i); lm/lp[j] = l_j(-1/+1); gl/gr[i] = g_L'/g_R'(z_i)
};
void build_fr_ops(FrOps& o, int p) {
  if (o.p == p) return;
  const int P1 = p + 1;
  o.p = p;
  gauss_legendre(P1, o.z, o.w);
  o.D.assign((size_t)P1 * P1, 0.0);
  o.lm.assign(P1, 0.0); o.lp.assign(P1, 0.0); o.gl.assign(P1, 0.0); o.gr.assign(P1, 0.0);
  const double sgn = ((p + 1) % 2) ? -1.0 : 1.0;  // (-1)^(k+1), k = p
  for (int i = 0; i < P1; ++i) {
    for (int j = 0; j < P1; ++j) o.D[(size_t)i * P1 + j] = lagrange_d(o.z, j, o.z[i]);
    o.lm[i] = lagrange(o.z, i, -1.0);
    o.lp[i] = lagrange(o.z, i, 1.0);
    o.gl[i] = 0.5 * sgn * (legendre_d(p + 1, o.z[i]) - legendre_d(p, o.z[i]));
    o.gr[i] = -0.5 * sgn * (legendre_d(p + 1, -o.z[i]) - legendre_d(p, -o.z[i]));  // d/dxi g_L(-xi)
  }
}

constexpr double kGamma = 1.4;
void euler_flux(int dim, int a, const double* u, double* F) {
  const double rho = u[0], E = u[dim + 1];
  double v[3] = {0, 0, 0}, q = 0.0;
  for (int b = 0; b < dim; ++b) { v[b] = u[1 + b] / rho; q += v[b] * v[b]; }
  const double pr = (kGamma - 1.0) * (E - 0.5 * rho * q);
  F[0] = rho * v[a];
  for (int b = 0; b < dim; ++b) F[1 + b] = u[1 + b] * v[a] + (b == a ? pr : 0.0);
  F[dim + 1] = (E + pr) * v[a];
}
double wave_speed(int dim, int a, const double* u) {
  const double rho = u[0], E = u[dim + 1];
  double q = 0.0;
  for (int b = 0; b < dim; ++b) q += (u[1 + b] / rho) * (u[1 + b] / rho);
  const double pr = (kGamma - 1.0) * (E - 0.5 * rho * q);
  return std::fabs(u[1 + a] / rho) + std::sqrt(kGamma * pr / rho);
}
void rusanov(int dim, int a, const double* uL, const double* uR, double* F) {
  double FL[5], FR[5];
  euler_flux(dim, a, uL, FL);
  euler_flux(dim, a, uR, FR);
  const double lam = std::max(wave_speed(dim, a, uL), wave_speed(dim, a, uR));
  for (int v = 0; v < dim + 2; ++v) F[v] = 0.5 * (FL[v] + FR[v]) - 0.5 * lam * (uR[v] - uL[v]);
}

// Alg. 8 step 3 on every kind 1 / kind 2 slot: own trace u_f[e][f], neighbour trace u_nb[e][f]
// (mortar_project); the minus-side state is the own one on an odd face, the neighbour's on an even one.
void common_flux(Tree* t, int Nf, const double* uf, const double* unb, double* fs) {
  const int dim = t->dim, nf = t->nf, nv = dim + 2;
  const int64_t M = (int64_t)t->leaves.size();
  for (int64_t e = 0; e < M; ++e)
    for (int f = 0; f < nf; ++f) {
      const size_t sl = (size_t)e * nf + f;
      const int kd = t->faces.kind[sl] & 15;
      if (kd != 1 && kd != 2) continue;
      for (int n = 0; n < Nf; ++n) {
        double own[5], nb[5], F[5];
        for (int v = 0; v < nv; ++v) {
          own[v] = uf[(sl * nv + v) * Nf + n];
          nb[v] = unb[(sl * nv + v) * Nf + n];
        }
        if (f & 1) rusanov(dim, f >> 1, own, nb, F); else rusanov(dim, f >> 1, nb, own, F);
        for (int v = 0; v < nv; ++v) fs[(sl * nv + v) * Nf + n] = F[v];
      }
    }
}

// Eq. 2-5 for every element; width[a] = physical domain width along axis a.
void fr_rhs(Tree* t, const FrOps& o, const double* width, const double* u, const double* fs, double* R) {
  const int dim = t->dim, nf = t->nf, nv = dim + 2, P1 = o.p + 1;
  int N = 1, Nf = 1;
  for (int a = 0; a < dim; ++a) N *= P1;
  for (int a = 0; a + 1 < dim; ++a) Nf *= P1;
  const int64_t M = (int64_t)t->leaves.size();
  std::vector<double> F((size_t)N * nv);
  for (int64_t e = 0; e < M; ++e) {
    const double* ue = u + (size_t)e * nv * N;
    double* Re = R + (size_t)e * nv * N;
    for (int i = 0; i < nv * N; ++i) Re[i] = 0.0;
    for (int a = 0; a < dim; ++a) {
      // the brick is nroot[a] cubes wide along a (one cube: dx = width / 2^level)
      const double dx = width[a] / ((double)t->nroot[a] * (double)((uint64_t)1 << t->leaves[e]->level));
      int stride = 1;
      for (int b = 0; b < a; ++b) stride *= P1;
      for (int n = 0; n < N; ++n) {  // flux along a at every solution point
        double us[5], Fs[5];
        for (int v = 0; v < nv; ++v) us[v] = ue[(size_t)v * N + n];
        euler_flux(dim, a, us, Fs);
        for (int v = 0; v < nv; ++v) F[(size_t)v * N + n] = Fs[v];
      }
      for (int n = 0; n < N; ++n) {
        const int ia = (n / stride) % P1;          // index along a
        const int line = n - ia * stride;          // first point of the line through n
        int nt = 0, mul = 1, r = n;                // tangential face-point index (lower axis fastest)
        for (int b = 0; b < dim; ++b) {
          const int ib = r % P1;
          r /= P1;
          if (b == a) continue;
          nt += ib * mul;
          mul *= P1;
        }
        for (int v = 0; v < nv; ++v) {
          double d = 0.0, fm = 0.0, fp = 0.0;
          for (int j = 0; j < P1; ++j) {
            const double fj = F[(size_t)v * N + line + j * stride];
            d += o.D[(size_t)ia * P1 + j] * fj;
            fm += o.lm[j] * fj;
            fp += o.lp[j] * fj;
          }
          const double Fm = fs[((((size_t)e * nf + 2 * a) * nv) + v) * Nf + nt];
          const double Fp = fs[((((size_t)e * nf + 2 * a + 1) * nv) + v) * Nf + nt];
          d += o.gl[ia] * (Fm - fm) + o.gr[ia] * (Fp - fp);
          Re[(size_t)v * N + n] -= (2.0 / dx) * d;
        }
      }
    }
  }
}

// Eq. 6: the three-stage, third-order explicit Runge-Kutta method, one stage per call,
// written as printed:
//   stage 1:  u^1     = u^n + dt R(u^n)
//   stage 2:  u^2     = 3/4 u^n + 1/4 u^1 + 1/4 dt R(u^1)
//   stage 3:  u^(n+1) = 1/3 u^n + 2/3 u^2 + 2/3 dt R(u^2)
// un = u^n, us = the stage vector the right-hand side R was evaluated at (u^n, u^1, u^2; unused in
// stage 1, where it is u^n by definition), R = R(us).  Pinned by the scheme's amplification
// polynomial 1 + z + z^2/2 + z^3/6 on u' = lambda u and by third-order convergence
// (tests/test_oracle_fr.py).
int rk3_stage(int stage, double dt, int64_t n, const double* un, const double* us, const double* R, double* out) {
  if (stage == 1) {
    for (int64_t i = 0; i < n; ++i) out[i] = un[i] + dt * R[i];
  } else if (stage == 2) {
    for (int64_t i = 0; i < n; ++i) out[i] = 3.0 / 4.0 * un[i] + 1.0 / 4.0 * us[i] + 1.0 / 4.0 * dt * R[i];
  } else if (stage == 3) {
    for (int64_t i = 0; i < n; ++i) out[i] = 1.0 / 3.0 * un[i] + 2.0 / 3.0 * us[i] + 2.0 / 3.0 * dt * R[i];
  } else {
    return -1;
  }
  return 0;
}

}  // namespace

// ======================================================================= C ABI
extern "C" {

typedef struct Tree lto_tree;

uint64_t lto_encode(int dim, int maxl, int level, const uint32_t* x) { return encode(dim, maxl, level, x); }
uint64_t lto_raw_id(int dim, int maxl, int level, const uint32_t* x) {
  uint32_t xi[3] = {0, 0, 0};
  for (int a = 0; a < dim; ++a) xi[a] = level == 0 ? 0u : (x[a] >> (maxl - level));
  return raw_id(dim, level, xi);
}
void lto_decode(int dim, int maxl, uint64_t key, int* level, uint32_t* x) { decode(dim, maxl, key, level, x); }

int64_t lto_sort_linearise(int dim, int maxl, uint64_t* keys, int64_t n) {
  return sort_linearise(dim, maxl, keys, n);
}

void* lto_build(int dim, int base, int maxl, const int* periodic) {
  Tree* t = new_tree(dim, base, maxl, periodic);
  if (!t) return nullptr;
  refine_uniform(t, t->roots[0], base);
  relist(t);
  return t;
}

// Uniform depth-`base` forest on a brick of nroot[0] x nroot[1] (x nroot[2]) root cubes.
void* lto_build_brick(int dim, const int* nroot, int base, int maxl, const int* periodic) {
  Tree* t = new_tree(dim, base, maxl, periodic, nroot);
  if (!t) return nullptr;
  for (Node* r : t->roots) refine_uniform(t, r, base);
  relist(t);
  return t;
}

// unsorted keys -> sort + linearise (Alg. 3) -> pointer tree.  Returns NULL if
// the linearised set does not tile the domain.
void* lto_build_from_keys(int dim, int base, int maxl, const int* periodic, const uint64_t* keys, int64_t n) {
  Tree* t = new_tree(dim, base, maxl, periodic);
  if (!t) return nullptr;
  std::vector<uint64_t> k(keys, keys + n);
  int64_t m = sort_linearise(dim, maxl, k.data(), n);
  for (int64_t i = 0; i < m; ++i) {
    int lvl;
    uint32_t x[3];
    decode(dim, maxl, k[i], &lvl, x);
    Node* nd = t->roots[0];
    while (nd->level < lvl) {
      if (nd->is_leaf()) split(t, nd);
      int sh = maxl - nd->level - 1;
      int c = 0;
      for (int a = 0; a < dim; ++a) c |= (int)((x[a] >> sh) & 1u) << a;
      nd = nd->child[c];
    }
    nd->mark = true;  // a stored leaf
  }
  // completeness: every leaf of the pointer tree must be a stored key
  std::vector<Node*> lv;
  dfs_leaves(t, t->roots[0], lv);
  bool ok = (int64_t)lv.size() == m;
  for (Node* q : lv) {
    if (!q->mark) ok = false;
    q->mark = false;
  }
  if (!ok) {
    free_subtree(t->roots[0]);
    delete t;
    return nullptr;
  }
  relist(t);
  return t;
}

// Alg. 2 on octants: complete the key set (any order, duplicates / ancestors allowed)
// over the uniform depth-`base` tree.  NULL on bad arguments or a key above base level.
void* lto_build_complete(int dim, int base, int maxl, const int* periodic, const uint64_t* keys, int64_t n) {
  Tree* t = new_tree(dim, base, maxl, periodic);
  if (!t) return nullptr;
  refine_uniform(t, t->roots[0], base);
  for (int64_t i = 0; i < n; ++i) {
    int lvl;
    uint32_t x[3];
    decode(dim, maxl, keys[i], &lvl, x);
    if (lvl < base || lvl > maxl) {
      free_subtree(t->roots[0]);
      delete t;
      return nullptr;
    }
    insert_octant(t, lvl, x);
  }
  relist(t);
  return t;
}

// Alg. 2 from scattered points: xyz [n][dim] fp64, domain lo_hi = lo_x.., hi_x..; every
// point becomes its depth-D_max cell (point_cell), then completion as above.
void* lto_build_from_points(int dim, int base, int maxl, const int* periodic, const double* lo_hi,
                            const double* xyz, int64_t n) {
  Tree* t = new_tree(dim, base, maxl, periodic);
  if (!t) return nullptr;
  refine_uniform(t, t->roots[0], base);
  for (int64_t i = 0; i < n; ++i) {
    uint32_t x[3] = {0, 0, 0};
    for (int a = 0; a < dim; ++a) x[a] = point_cell(xyz[i * dim + a], lo_hi[a], lo_hi[dim + a], maxl);
    insert_octant(t, maxl, x);
  }
  relist(t);
  return t;
}

uint32_t lto_point_cell(double x, double lo, double hi, int maxl) { return point_cell(x, lo, hi, maxl); }

void lto_free(void* h) {
  Tree* t = (Tree*)h;
  if (!t) return;
  for (Node* r : t->roots) free_subtree(r);
  for (Node* r : t->old_roots) free_subtree(r);
  delete t;
}

int64_t lto_num_leaves(void* h) { return (int64_t)((Tree*)h)->leaves.size(); }
void lto_keys(void* h, uint64_t* out) {
  Tree* t = (Tree*)h;
  std::memcpy(out, t->keys.data(), t->keys.size() * sizeof(uint64_t));
}
// integer anchors (finest units, [M][3]) and levels of the leaves, array order
void lto_leaf_boxes(void* h, int32_t* level, uint32_t* xyz) {
  Tree* t = (Tree*)h;
  for (size_t i = 0; i < t->leaves.size(); ++i) {
    level[i] = t->leaves[i]->level;
    for (int a = 0; a < 3; ++a) xyz[3 * i + a] = t->leaves[i]->x[a];
  }
}
// 1 if the DFS order of the pointer tree equals the std::sort order of the IDs
int lto_dfs_is_sorted(void* h) {
  Tree* t = (Tree*)h;
  std::vector<Node*> lv;
  for (Node* r : t->roots) dfs_leaves(t, r, lv);
  if (lv.size() != t->leaves.size()) return 0;
  for (size_t i = 0; i < lv.size(); ++i)
    if (lv[i] != t->leaves[i]) return 0;
  return 1;
}

void lto_adapt(void* h, const int8_t* flags) { adapt((Tree*)h, flags); }
int lto_balance(void* h, int64_t* n_split) { return balance((Tree*)h, n_split, 1); }
int lto_balance_conn(void* h, int64_t* n_split, int conn) {
  if (conn < 1 || conn > ((Tree*)h)->dim) return -1;
  return balance((Tree*)h, n_split, conn);
}

// method: 0 = point-location descent, 1 = brute force O(N^2)
int lto_connect(void* h, int method) {
  Tree* t = (Tree*)h;
  int rc = method == 1 ? connect_bruteforce(t, t->faces.nbr, t->faces.kind)
                       : connect_descent(t, t->faces.nbr, t->faces.kind);
  if (rc != 0) return rc;
  face_tables(t);
  return 0;
}
void lto_face_counts(void* h, int64_t* out3) {
  Tree* t = (Tree*)h;
  out3[0] = (int64_t)t->faces.conf_axis.size();
  out3[1] = (int64_t)t->faces.hang_info.size();
  out3[2] = (int64_t)t->faces.bnd.size();
}
void lto_faces(void* h, int32_t* nbr, uint8_t* kind, int32_t* conf, uint8_t* conf_axis, int32_t* hang,
               uint8_t* hang_info, int32_t* bnd, uint8_t* bnd_face) {
  Faces& F = ((Tree*)h)->faces;
  auto cp = [](auto* dst, const auto& v) {
    if (dst && !v.empty()) std::memcpy(dst, v.data(), v.size() * sizeof(v[0]));
  };
  cp(nbr, F.nbr); cp(kind, F.kind); cp(conf, F.conf); cp(conf_axis, F.conf_axis);
  cp(hang, F.hang); cp(hang_info, F.hang_info); cp(bnd, F.bnd); cp(bnd_face, F.bnd_face);
}

// Alg. 7.  Returns 0 or -1 (a new leaf more than one level from T_o).
int lto_build_map(void* h) { return build_map((Tree*)h); }
void lto_map(void* h, int32_t* src, uint8_t* kind) {
  Tree* t = (Tree*)h;
  std::memcpy(src, t->map_src.data(), t->map_src.size() * sizeof(int32_t));
  std::memcpy(kind, t->map_kind.data(), t->map_kind.size());
}
int64_t lto_num_old_leaves(void* h) { return (int64_t)((Tree*)h)->old_keys.size(); }
void lto_old_keys(void* h, uint64_t* out) {
  Tree* t = (Tree*)h;
  std::memcpy(out, t->old_keys.data(), t->old_keys.size() * sizeof(uint64_t));
}

// Transfer rows [j0, j1) of the new tree (slab-wise so config 5 fits the host).
// Requires lto_build_map first.  u_old is the whole old array.
int lto_transfer_rows(void* h, const double* u_old, double* u_new_rows, int p, int nvars, int64_t j0, int64_t j1) {
  Tree* t = (Tree*)h;
  if (p < 0 || p > 7 || nvars < 1) return -1;
  if (t->map_src.size() != t->leaves.size()) return -1;
  build_ops(t, p);
  transfer_rows(t, u_old, u_new_rows, nvars, j0, j1);
  return 0;
}
// drop the snapshot (state rule: lt_transfer consumes it)
void lto_drop_snapshot(void* h) {
  Tree* t = (Tree*)h;
  for (Node* r : t->old_roots) free_subtree(r);
  t->old_roots.clear();
  t->old_leaves.clear();
  t->old_keys.clear();
  t->have_old = false;
}

// operator access for pins: which = 0 interp[nc][N][N], 1 proj[nc][N][N], 2 mass[N][N], 3 S[nc][N][N]
int lto_operators(int dim, int p, int which, double* out) {
  int per[3] = {0, 0, 0};
  Tree* t = new_tree(dim, 0, 1, per);
  if (!t) return -1;
  build_ops(t, p);
  const std::vector<double>* v = which == 0 ? &t->ops.interp : which == 1 ? &t->ops.proj
                                 : which == 2 ? &t->ops.mass : &t->ops.S;
  std::memcpy(out, v->data(), v->size() * sizeof(double));
  free_subtree(t->roots[0]);
  delete t;
  return 0;
}
// Alg. 8 steps 2 / 4 on the face arrays [n_leaves][nf][nvars][(p+1)^(dim-1)]; lto_connect
// must have run on the current tree.  which = 0: to_mortar (Eq. 17), 1: M^-1 S^s (Eq. 20).
int lto_mortar_project(void* h, const double* uf, double* unb, int p, int nvars) {
  Tree* t = (Tree*)h;
  if (t->faces.kind.size() != t->leaves.size() * (size_t)t->nf) return -2;
  FaceOps fo;
  build_face_ops(fo, t->dim, p);
  mortar_project(t, fo, uf, unb, nvars);
  return 0;
}
int lto_mortar_gather(void* h, const double* fm, double* ff, int p, int nvars) {
  Tree* t = (Tree*)h;
  if (t->faces.kind.size() != t->leaves.size() * (size_t)t->nf) return -2;
  FaceOps fo;
  build_face_ops(fo, t->dim, p);
  return mortar_gather(t, fo, fm, ff, nvars);
}
// FR solver pieces around the cycle (Eq. 1-6, Alg. 8 step 3); Euler equations, nvars = dim + 2.
int lto_common_flux(void* h, const double* uf, const double* unb, double* fs, int p) {
  Tree* t = (Tree*)h;
  if (t->faces.kind.size() != t->leaves.size() * (size_t)t->nf) return -2;
  int Nf = 1;
  for (int a = 0; a + 1 < t->dim; ++a) Nf *= p + 1;
  common_flux(t, Nf, uf, unb, fs);
  return 0;
}
int lto_fr_rhs(void* h, const double* width, const double* u, const double* fs, double* R, int p) {
  FrOps o;
  build_fr_ops(o, p);
  fr_rhs((Tree*)h, o, width, u, fs, R);
  return 0;
}
int lto_rk3_stage(int stage, double dt, int64_t n, const double* un, const double* us, const double* R, double* out) {
  return rk3_stage(stage, dt, n, un, us, R, out);
}
// which: 0 D [P1][P1], 1 l(-1) [P1], 2 l(+1) [P1], 3 g_L' [P1], 4 g_R' [P1]
int lto_fr_operators(int p, int which, double* out) {
  FrOps o;
  build_fr_ops(o, p);
  const std::vector<double>* v[5] = {&o.D, &o.lm, &o.lp, &o.gl, &o.gr};
  if (which < 0 || which > 4) return -1;
  std::memcpy(out, v[which]->data(), v[which]->size() * sizeof(double));
  return 0;
}
int lto_face_interp(void* h, const double* u, double* uf, int p, int nvars) {
  if (p < 0 || nvars < 1) return -1;
  face_interp((Tree*)h, p, u, uf, nvars);
  return 0;
}
int lto_face_operators(int dim, int p, int which, double* out) {
  if (dim != 2 && dim != 3) return -1;
  FaceOps fo;
  build_face_ops(fo, dim, p);
  const std::vector<double>& v = which == 0 ? fo.to_mortar : fo.coarse.proj;
  std::memcpy(out, v.data(), v.size() * sizeof(double));
  return 0;
}
void lto_gauss_legendre(int n, double* z, double* w) {
  std::vector<double> zz, ww;
  gauss_legendre(n, zz, ww);
  std::memcpy(z, zz.data(), n * sizeof(double));
  std::memcpy(w, ww.data(), n * sizeof(double));
}

}  // extern "C"
