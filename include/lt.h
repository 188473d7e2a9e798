/* lt.h -- C ABI of liblt: the single-GPU h-adaptation cycle over a linear quadtree /
 * octree (arxiv 2306.06744, "An efficient GPU-based h-adaptation framework via linear
 * trees for the flux reconstruction method").  Citations are PAPER.md:<line>.
 *
 * One adaptation cycle:
 *     lt_adapt -> lt_balance -> lt_connect -> lt_transfer
 * on a tree created by lt_build (uniform base tree) or lt_build_from_keys (unsorted,
 * possibly overlapping keys -> radix sort + linearise, Alg. 3).
 *
 * Conventions
 *   - "device" pointers are CUDA device memory of the GPU that was current when the
 *     tree was built; "host" pointers are ordinary host memory.  That GPU must be the
 *     current device at every later call on the tree (calls that upload operators check it
 *     and return LT_ERR_ARG otherwise).
 *   - Every call enqueues on the CUDA stream given at build time.  Calls that return a
 *     count or a status detected on the device synchronise that stream (stated per call).
 *   - Every int-returning call returns LT_OK (0) or a negative lt_status.  No exceptions,
 *     no aborts, no CPU fallback: without a CUDA device every call fails with LT_ERR_CUDA.
 *   - The tree owns every device array it hands out (keys, map, face arrays).  Such
 *     pointers stay valid until the next mutating call on the same tree (lt_adapt,
 *     lt_balance, lt_connect, lt_transfer, lt_reserve, lt_free).
 *
 * Key format (Alg. 1; readings A-1..A-3 of DESIGN.md)
 *     key = (interleave(x, y[, z]) << 5) | level
 *   x_a in [0, 2^max_level): integer anchor (minimum corner) in units of the
 *   finest cell, a multiple of 2^(max_level - level); bit k of axis a sits at interleaved
 *   position dim*k + a (x lowest); the depth occupies the 5 low bits, so the
 *   first child of a key is key + 1 (Eq. 7 case 3).  Leaves are stored in
 *   ascending uint64 order.
 *
 * Local face numbering (reading D-1): 0 = -x, 1 = +x, 2 = -y, 3 = +y,
 * 4 = -z, 5 = +z; the opposite face of f is f ^ 1.
 */
#ifndef LT_H_
#define LT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lt_tree lt_tree; /* opaque */

typedef enum {
  LT_OK = 0,
  LT_ERR_ARG = -1,        /* bad argument (dim, levels, p, nvars, NULL pointer, n too large)       */
  LT_ERR_CUDA = -2,       /* a CUDA runtime call failed (lt_last_cuda_error gives the code)        */
  LT_ERR_OOM = -3,        /* device allocation failed                                              */
  LT_ERR_CAPACITY = -4,   /* a device buffer would overflow and could not be grown                 */
  LT_ERR_UNBALANCED = -5, /* lt_connect met face neighbours more than one level apart (D-5)        */
  LT_ERR_MAPPING = -6,    /* lt_transfer met a new leaf more than one level from T_old (Alg. 7)    */
  LT_ERR_INCOMPLETE = -7  /* lt_build_from_keys: the linearised keys do not tile the domain        */
} lt_status;

/* Face connectivity (Alg. 5; format = readings D-2..D-4).
 * All pointers are device memory owned by the tree.  nf = 2*dim.
 *   nbr[e*nf+f], kind[e*nf+f]  -- the paper's face array F plus a type byte:
 *     kind & 15 == 0  boundary           nbr = -1
 *     kind & 15 == 1  conforming         nbr = the same-level neighbour
 *     kind & 15 == 2  neighbour coarser  nbr = the coarse neighbour; kind >> 4 = slot of
 *                     this fine face inside the coarse face: the leaf's child-id bits on
 *                     the tangential axes, ascending axis order, smaller coordinate first
 *
 *     kind & 15 == 3  neighbour finer    nbr = the slot-0 fine neighbour
 *   conf[i] = (e_minus, e_plus), conf_axis[i] in 0..dim-1: one row per conforming face,
 *     emitted by the element on its minus side (local face odd)
 *   hang[i] = (e_fine, e_coarse), hang_info[i] = f_fine | slot << 3: one row per fine face
 *     of a hanging face, emitted by the fine element ("search from the fine side",
 *     PAPER.md:188)
 *   bnd[i] = element, bnd_face[i] = local face: one row per boundary face.
 * Each list is in emission order: leaves in array order, local faces 0..nf-1. */
typedef struct {
  int64_t n_leaves, n_conf, n_hang, n_bnd;
  const int32_t* nbr;
  const uint8_t* kind;
  const int32_t* conf;
  const uint8_t* conf_axis;
  const int32_t* hang;
  const uint8_t* hang_info;
  const int32_t* bnd;
  const uint8_t* bnd_face;
} lt_faces;

/* ---- construction ------------------------------------------------------------------ */

/* Uniform tree of 2^(dim*base_level) leaves at depth base_level, written directly in
 * Morton order (Alg. 1).  dim in {2,3}; 0 <= base_level <= max_level; max_level <= 29
 * (2-D) / 19 (3-D) so that dim*max_level + 5 <= 63 bits.  base_level is D_min (leaves are
 * never coarsened above it), max_level is D_max.
 *   domain   host [2*dim]: lo_x.., hi_x.. -- stored for the caller (lt_domain); the tree
 *            works on integer coordinates only ("perfect cubes").  May be NULL.
 *   periodic host [dim]: non-zero = wrap neighbour coordinates on that axis.
 *            May be NULL (no periodic axis).
 *   cuda_stream  a cudaStream_t (NULL = the legacy default stream).
 * Asynchronous. */
int lt_build(int dim, int base_level, int max_level, const double* domain, const int* periodic,
             void* cuda_stream, lt_tree** out);

/* The same on a BRICK of nroot[0] x nroot[1] (x nroot[2]) root cubes (host [dim], NULL = one cube): a
 * forest of linear trees for domains that are not a cube, e.g. the paper's 3-D slab
 * [-12.5, 12.5]^2 x 1.5625 = 16 x 16 x 1 cubes, one element thick at D_min (PAPER.md:84
 * treats "perfect cubes" only; reading J-1).  Levels count from the root cubes; base_level
 * leaves per cube edge = 2^base_level.  The index r = tx + nroot[0] * (ty + nroot[1] * tz) of a leaf's
 * cube sits above the path bits of its ID,
 *     key = (((r << dim * max_level) | interleave(x - cube origin)) << 5) | level,
 * so leaves are stored cube by cube, in Morton order inside each cube, and one cube gives lt_build's
 * keys.  Needs dim * max_level + 5 + ceil(log2(#cubes)) <= 63 and nroot[a] * 2^max_level <= 2^31.
 * `domain` is the whole brick (its cubes have edge (hi_a - lo_a) / nroot[a], equal on all axes for a
 * conforming mesh); `periodic` wraps the whole brick.  lt_adapt, lt_balance, lt_connect, lt_transfer
 * and the mortar / FR calls work unchanged; lt_leaf_boxes returns anchors in global finest-cell
 * units, [0, nroot[a] * 2^max_level).  Construction from points / keys is defined on one cube. */
int lt_build_brick(int dim, const int* nroot, int base_level, int max_level, const double* domain,
                   const int* periodic, void* cuda_stream, lt_tree** out);
int lt_roots(lt_tree*, int* nroot /* host [3] */);

/* Tree from n unsorted device keys (any levels >= base_level; duplicates and ancestors
 * allowed): LSD radix sort over the used key bits, then linearisation (Alg. 3,
 * drop duplicates and every key that is an ancestor of its successor).
 * Fails with LT_ERR_INCOMPLETE if the result does not tile the domain.  Synchronises. */
int lt_build_from_keys(int dim, int base_level, int max_level, const double* domain,
                       const int* periodic, void* cuda_stream, const uint64_t* d_keys, int64_t n,
                       lt_tree** out);

/* Alg. 2 on octants: n unsorted device keys (levels in [base_level,
 * max_level]; duplicates and ancestors allowed) -> radix sort, linearise (Alg. 3), then
 * COMPLETION: the result is the coarsest complete tree that refines the uniform depth-
 * base_level tree (base_level = the paper's D_min) and keeps every
 * linearised input octant as a leaf (readings G-2, G-3).  The gaps between
 * consecutive octants, and before the first / after the last one, are filled in Morton
 * order by a closed form of the two neighbouring keys: no atomics, no append, no second
 * sort.  The tree is NOT 2:1 balanced: call lt_balance (Alg. 4) next.
 * LT_ERR_ARG if a key is outside [base_level, max_level] or misaligned; LT_ERR_CAPACITY if
 * the completed tree would exceed 2^31 - 1024 leaves.  Synchronises. */
int lt_build_complete_from_keys(int dim, int base_level, int max_level, const double* domain,
                                const int* periodic, void* cuda_stream, const uint64_t* d_keys,
                                int64_t n, lt_tree** out);

/* Alg. 2 from scattered points (PAPER.md:109 step 1): d_xyz device fp64 [n][dim].  Every point
 * becomes its depth-max_level cell, xi = floor((x - lo) / (hi - lo) * 2^max_level) evaluated
 * in fp64 in this order and clamped to [0, 2^max_level - 1] (reading G-1; cells are half-
 * open), then as lt_build_complete_from_keys.  domain (host [2*dim]) is
 * required, hi > lo on every axis.  Synchronises. */
int lt_build_from_points(int dim, int base_level, int max_level, const double* domain,
                         const int* periodic, void* cuda_stream, const double* d_xyz, int64_t n,
                         lt_tree** out);

void lt_free(lt_tree*);

/* Make room for `n_leaves` leaves in every tree-owned buffer (buffers also grow on
 * demand).  Synchronises when it has to reallocate. */
int lt_reserve(lt_tree*, int64_t n_leaves);

/* ---- the cycle --------------------------------------------------------------------- */

/* Alg. 6: d_flags device int8 [lt_num_leaves], > 0 refine
 * (ignored at max_level), < 0 coarsen (honoured only for complete sibling groups whose
 * 2^dim members are all leaves, all flagged < 0, level > base_level).  One level per
 * call.  Snapshots the pre-adapt keys as T_old (replacing any earlier snapshot).
 * The new leaves are written in Morton order by an order-preserving expansion (a leaf's
 * children occupy its Morton interval), so no sort is needed; set
 * lt_set_option(t, LT_OPT_ADAPT_SORT, 1) to realise it as the paper does (append, radix
 * sort, linearise) -- same result.  Synchronises once (reads the new leaf count to size
 * buffers) -- unless the buffers already hold the worst case, 2^dim * lt_num_leaves (lt_reserve): then
 * the call only enqueues, and the new count stays on the device until a later call needs it. */
int lt_adapt(lt_tree*, const int8_t* d_flags);

/* 2:1 face balance (Alg. 4; readings C-1..C-7): the unique coarsest
 * refinement in which leaves sharing a (dim-1)-face (periodic images included) differ by
 * at most one level, by Jacobi ripple sweeps run in ONE cooperative kernel (no host round
 * trip per sweep).  *iters (host, may be NULL) = number of sweeps that split >= 1 leaf.
 * If the tree was balanced when the preceding lt_adapt was called, the first sweep examines only
 * the leaves that call created (same result, sweep count and splits as a full sweep).
 * Synchronises at the end (reads leaf count / status).  On LT_ERR_CAPACITY (growth
 * impossible) the tree is a valid, partially balanced refinement of the input.
 * With iters == NULL, face connectivity, a tree that was balanced before the preceding lt_adapt and
 * buffers that hold 2^dim * lt_num_old_leaves leaves (the largest result possible, reading C-5) the
 * call only enqueues: lt_connect_begin, lt_transfer and lt_connect_end then run the rest of the cycle
 * with ONE host synchronisation (in lt_connect_end); lt_last_balance_iters returns the sweep count. */
int lt_balance(lt_tree*, int* iters);

/* Alg. 5: fills *out (host struct; device arrays inside).
 * LT_ERR_UNBALANCED if a level jump > 1 is met.  Synchronises. */
int lt_connect(lt_tree*, lt_faces* out);

/* The same query split in two so that it can overlap lt_transfer (both depend only on the
 * balanced tree): lt_connect_begin enqueues the connectivity kernel on a side stream owned by
 * the tree, ordered after everything already enqueued on the tree's stream, and returns at once;
 * lt_connect_end makes the tree's stream wait for it, synchronises and fills *out exactly as
 * lt_connect does.  Calls enqueued between the two (typically lt_transfer) run concurrently
 * with the face query; lt_adapt / lt_balance / lt_reserve / lt_free join it first.
 * lt_connect_end without a pending begin: LT_ERR_ARG. */
int lt_connect_begin(lt_tree*);
int lt_connect_end(lt_tree*, lt_faces* out);

/* Alg. 7 + section 4.2: maps T_old -> current tree and moves the
 * solution: copy (same ID), interpolation of the parent's Lagrange expansion at the
 * child's solution points (Eq. 8), L2 projection of the 2^dim children (Eq. 9-13).
 *   d_u_old device [n_old][nvars][N] fp64, d_u_new device [lt_num_leaves][nvars][N] fp64,
 *   N = (p+1)^dim Gauss-Legendre solution points, x fastest (readings E-1, E-5).
 *   The arrays must not overlap and must be 16-byte aligned (cudaMalloc / torch allocations
 *   are).  1 <= p+1 <= 8 (p = 0..7), nvars >= 1.
 * Without a snapshot this is a plain copy.  Drops the snapshot.  Asynchronous; a mapping
 * error is sticky and is returned by this call only if detected before it returns --
 * lt_sync reports it otherwise. */
int lt_transfer(lt_tree*, const double* d_u_old, double* d_u_new, int p, int nvars);

/* Same as lt_transfer with HOST arrays (pinned memory for full speed).  Pipelined in slabs of
 * consecutive new leaves: slab k reads one contiguous range of old leaves (the map is
 * monotone), so the upload of slab k+1, the kernel on slab k and the download of slab k-1
 * overlap on three streams and only a ring of three slab pairs is staged in device memory
 * (owned by the tree).  Synchronises. */
int lt_transfer_host(lt_tree*, const double* h_u_old, double* h_u_new, int p, int nvars);

/* ---- mortars on nonconforming faces (Alg. 8 steps 2 and 4) -------------
 * Face arrays: device fp64 [lt_num_leaves][nf][nvars][Nf], Nf = (p+1)^(dim-1) Gauss-Legendre
 * face points, tangential axes in ascending order, lower axis fastest (readings H-1, H-4).
 * The 2^(dim-1) mortars of a coarse face coincide with the faces of its fine neighbours
 * (mortar s = slot s of lt_connect; fine side <-> mortar is "a direct copy"),
 * so mortar data lives in the fine element's face slot.  Both calls need lt_connect on the
 * current tree (LT_ERR_ARG otherwise), 0 <= p <= 7, nvars >= 1.  Asynchronous.
 *
 * lt_mortar_project -- step 2, Eq. 14-17: for every face slot (e, f) the neighbour's trace as
 * seen from e:   kind 1: d_u_nb[e][f] = d_u_face[nbr][f^1]  (conforming, copy);
 *                kind 2: d_u_nb[e][f] = L2 projection of the coarse trace d_u_face[nbr][f^1]
 *                        onto mortar `slot` (Eq. 17);   kind 0 / 3: left untouched.
 * The arrays must not overlap.
 *
 * lt_mortar_gather -- step 4, Eq. 18-20: for every coarse face slot (kind 3)
 *   d_f_face[e][f] = M^-1 sum_s S^s d_f_mortar[e_s][f^1],  e_s = the fine neighbour on mortar s;
 * other slots are left untouched, so d_f_face may be d_f_mortar itself (in place).  The paper
 * scatters these contributions with atomicAdd; here each coarse face gathers its
 * mortars, which makes the result deterministic.  A missing fine neighbour sets the sticky
 * status LT_ERR_UNBALANCED (reported by lt_sync). */
int lt_mortar_project(lt_tree*, const double* d_u_face, double* d_u_nb, int p, int nvars);
int lt_mortar_gather(lt_tree*, const double* d_f_mortar, double* d_f_face, int p, int nvars);

/* Alg. 8 step 1: the solution at the face flux points,
 *   d_u_face[e][f][v][n_t] = sum_i l_i(-1 | +1) d_u[e][v][.. i on the face's axis ..],
 * d_u device [lt_num_leaves][nvars][(p+1)^dim] (layout of lt_transfer), d_u_face a face array as
 * above; l_i = the Lagrange basis on the Gauss-Legendre solution points.  Needs no connectivity.
 * The arrays must not overlap.  Asynchronous. */
int lt_face_interp(lt_tree*, const double* d_u, double* d_u_face, int p, int nvars);

/* ---- the flux-reconstruction update around the cycle (Eq. 1-6; Alg. 8 step 3) ---
 * Compressible Euler equations, conserved variables (rho, rho u, rho v[, rho w], E), nvars = dim + 2,
 * gamma = 1.4 (the paper's vortex test); readings I-1..I-5 of DESIGN.md.  Solution
 * arrays [lt_num_leaves][dim+2][(p+1)^dim], face arrays [lt_num_leaves][nf][dim+2][(p+1)^(dim-1)].
 *
 * lt_common_flux -- Alg. 8 step 3 ("a Rusanov solver"): on every kind 1 / kind 2 slot
 *   F* = (F_a(uL) + F_a(uR))/2 - max(|v_a| + c)(uR - uL)/2, the flux along +a (a = f >> 1); the minus-
 *   side state uL is the element's own trace d_u_face on an odd face and the neighbour's trace d_u_nb
 *   (lt_mortar_project) on an even one.  Kind 0 / 3 slots are left untouched (kind 3: lt_mortar_gather;
 *   boundary conditions other than periodic are the caller's).  d_f_star may be d_u_nb (in place).
 *   Needs lt_connect on the current tree.
 * lt_fr_rhs -- Eq. 2-5 with Radau correction functions: R = - sum_a (2/dx_a) [ D f_a +
 *   g_L' (F*_(a-) - f_a(-1)) + g_R' (F*_(a+) - f_a(+1)) ], dx_a = domain width / 2^level;
 *   d_f_star holds the common flux along +a in the element's own slots 2a and 2a+1.
 * lt_rk3_stage -- Eq. 6, stage = 1, 2, 3: d_u_out = a u_n + b (u_stage + dt R), (a, b) = (0, 1),
 *   (3/4, 1/4), (1/3, 2/3); d_u_out may be d_u_stage or d_u_n.
 * lt_fr_stage -- lt_fr_rhs and lt_rk3_stage in one pass: d_u_out = a u_n + b (u_stage + dt R(u_stage, F*));
 *   the right-hand side never goes to memory.  d_u_out may be d_u_stage or d_u_n.
 * All four are asynchronous. */
int lt_common_flux(lt_tree*, const double* d_u_face, const double* d_u_nb, double* d_f_star, int p);
/* lt_face_flux -- Alg. 8 steps 2 and 3 in ONE pass (= lt_mortar_project followed by lt_common_flux, the
 *   neighbour traces never go to memory): d_f_star[e][f] on every kind 1 / kind 2 slot from the traces
 *   d_u_face.  A conforming face is computed once, by the element on its minus side, and stored in both
 *   elements' slots (both sides compute the same flux along +a).  Kind 0 / 3 slots are left untouched
 *   (lt_mortar_gather fills kind 3).  The arrays must not overlap.  Needs lt_connect on the current
 *   tree.  Asynchronous. */
int lt_face_flux(lt_tree*, const double* d_u_face, double* d_f_star, int p);
int lt_fr_rhs(lt_tree*, const double* d_u, const double* d_f_star, double* d_rhs, int p);
int lt_rk3_stage(lt_tree*, int stage, double dt, const double* d_u_n, const double* d_u_stage,
                 const double* d_rhs, double* d_u_out, int p);
int lt_fr_stage(lt_tree*, int stage, double dt, const double* d_u_n, const double* d_u_stage,
                const double* d_f_star, double* d_u_out, int p);
/* lt_fr_stage_faces -- lt_fr_stage that also writes the traces of d_u_out at the face points
 *   (= lt_face_interp(d_u_out), Alg. 8 step 1 of the NEXT stage) while the element is still on chip;
 *   d_u_face_out may be d_f_star (an element reads and writes only its own face slots).  With
 *   lt_face_flux and lt_mortar_gather one RK stage is three passes:
 *       lt_face_flux(u_face -> f_star); lt_mortar_gather(f_star, in place);
 *       lt_fr_stage_faces(u_n, u_stage, f_star -> u_out, u_face). */
int lt_fr_stage_faces(lt_tree*, int stage, double dt, const double* d_u_n, const double* d_u_stage,
                      const double* d_f_star, double* d_u_out, double* d_u_face_out, int p);

/* ---- accessors --------------------------------------------------------------------- */

int64_t lt_num_leaves(lt_tree*);       /* synchronises only if the count is not cached   */
int lt_last_balance_iters(lt_tree*);   /* sweeps of the last lt_balance (also after lt_balance(t, NULL)); same rule */
int64_t lt_num_old_leaves(lt_tree*);   /* leaves of the snapshot T_old (0 if none)        */
const uint64_t* lt_keys(lt_tree*);     /* device, sorted                                  */
const uint64_t* lt_old_keys(lt_tree*); /* device, snapshot (NULL if none)                 */

/* Alg. 7's mapping arrays, valid after lt_transfer until the next mutating call:
 *   src[j]  old index of the leaf (copy / refined-from) or of the first child (fused-from)
 *   kind[j] 0 copy; 1 | child_id << 4 refine; 2 coarsen. */
int lt_map(lt_tree*, const int32_t** d_src, const uint8_t** d_kind);

/* Decode: d_level device int32 [n], d_xyz device uint32 [n][3]
 * (integer anchors in finest-cell units; unused axes 0).  Asynchronous. */
int lt_leaf_boxes(lt_tree*, int32_t* d_level, uint32_t* d_xyz);

/* Batch key codec on device arrays (Alg. 1).  d_xyz uint32 [n][3], d_level int32 [n]. */
int lt_encode(int dim, int max_level, const uint32_t* d_xyz, const int32_t* d_level, int64_t n,
              uint64_t* d_keys, void* cuda_stream);
int lt_decode(int dim, int max_level, const uint64_t* d_keys, int64_t n, int32_t* d_level,
              uint32_t* d_xyz, void* cuda_stream);

/* Ascending LSD radix sort of n device keys in place (8-bit digits over bits
 * [0, key_bits)), then, if linearise != 0, Alg. 3.  *n_out (host) = resulting count.
 * Synchronises. */
int lt_sort_keys(int dim, int max_level, uint64_t* d_keys, int64_t n, int linearise,
                 int64_t* n_out, void* cuda_stream);

/* The same sort (no linearisation) for callers that must not allocate (CUDA graph capture,
 * serving loops, harnesses that forbid cudaMalloc): the scratch of the radix passes (ping-pong
 * key buffer, per-tile digit table and its scan sums) is a static device array inside the library,
 * 8.26 MiB held by every GPU that loads liblt until exit.  d_keys: device uint64 [n], sorted
 * in place, ascending; n <= LT_SORT_STATIC_MAX_KEYS, else LT_ERR_CAPACITY (nothing is launched;
 * use lt_sort_keys).  Calls no cudaMalloc / cudaFree / allocating routine.  Asynchronous on
 * cuda_stream; the result is bit-identical to lt_sort_keys(..., linearise = 0).
 * All calls on one GPU share the array (it keeps the last call's contents; the call clears what
 * must start at zero): calls that overlap on the GPU -- different streams, or graph branches
 * without a dependency between them -- race.  Serialise them. */
#define LT_SORT_STATIC_MAX_KEYS (1 << 20)
int lt_sort_keys_static(int dim, int max_level, uint64_t* d_keys, int64_t n, void* cuda_stream);

int lt_domain(lt_tree*, double* lo_hi /* host [2*dim] */);
int lt_info(lt_tree*, int* dim, int* base_level, int* max_level, int* periodic /* host [3] */);

/* Wait for the tree's stream and return (and clear) the sticky device status.  The face query
 * keeps a status word of its own, so lt_connect / lt_connect_end report only connectivity errors
 * and a mapping error raised by an lt_transfer that ran beside the query is reported here. */
int lt_sync(lt_tree*);

typedef enum {
  LT_OPT_ADAPT_SORT = 1, /* 0 (default): ordered expansion; 1: append + sort + linearise */
  LT_OPT_BALANCE_FULL_SWEEPS = 2, /* 1: every sweep examines every leaf (debug)         */
  /* 3: reserved (a test hook of the library's own tests, see csrc/lt_internal.h) */
  LT_OPT_HOST_SLAB_LEAVES = 4,    /* v > 0: new leaves per slab of lt_transfer_host's copy /
                                     compute pipeline (default: about 128 MB of solution)   */
  LT_OPT_BALANCE_CONNECTIVITY = 5 /* which neighbours lt_balance keeps within one level:
                                     1 (default) leaves sharing a face; 2 + leaves sharing an
                                     edge -- the paper's "strong" balance in 3-D (
                                     in 2-D this adds the corner neighbours, a quadrant's edges
                                     being its faces); 3 (3-D) + leaves sharing only a corner.
                                     Values outside 1..dim: LT_ERR_ARG                       */
} lt_option;
int lt_set_option(lt_tree*, int option, int value);

/* Device times of the last cycle in milliseconds (CUDA events on the tree's stream):
 * out[0..3] = the calls lt_adapt, lt_balance, lt_connect, lt_transfer; out[4] = the Alg. 7
 * map kernel alone, out[5] = the solution-transfer kernel alone, out[6] = the connectivity
 * kernel alone, out[7] = the last mortar kernel (lt_mortar_project / lt_mortar_gather); 0 where not run.
 * Synchronises. */
int lt_timings(lt_tree*, float* out8);
/* Number of kernels liblt launched on this tree since it was built, and the number of times a call
 * made the host wait for the tree's stream (what a small mesh pays per cycle). */
int64_t lt_launch_count(lt_tree*);
int64_t lt_host_syncs(lt_tree*);
/* Where the last lt_balance spent its device time, in milliseconds, read from the GPU's global timer
 * between the grid-wide barriers of the cooperative kernel: out[0] examination sweeps, out[1] chunk
 * offsets, out[2] splitting + next frontier, out[3] the Alg. 7 map in the kernel's tail. */
int lt_balance_phases(lt_tree*, float* out4);

const char* lt_strerror(int status);
int lt_last_cuda_error(void); /* cudaError_t of the last failing runtime call (this thread) */
int lt_version(void);
/* 1 in the checked build (liblt_debug.so, compiled with -DLT_DEBUG: device-side assertions on every
 * located index, table write position, ticket and look-back word; a failing one traps the kernel and the
 * next synchronising call returns LT_ERR_CUDA), 0 in the release build. */
int lt_debug_build(void);

#ifdef __cplusplus
}
#endif
#endif /* LT_H_ */
