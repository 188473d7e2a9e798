// lt_transfer.cu -- old/new tree mapping (Alg. 7) and FR solution
// transfer (section 4.2) for sm_100a.  Product code.
//
// Transfer operators (readings E-1..E-4): with p+1 Gauss-Legendre solution points z_m per
// direction, child half b in {0,1} of a direction covers xi = (z + 2b - 1)/2, so
//   interpolation (Eq. 8)   I^b[m][i] = l_i((z_m + 2b - 1)/2)
//   L2 projection (Eq. 12)  R^b = M^-1 S^b; with GL nodes M = diag(w) exactly and
//                           R^b[j][i] = (w_i / (2 w_j)) I^b[i][j]
// and the dim-dimensional operators are tensor products of the 1-D ones, applied one
// direction at a time (sum factorisation).
//
// The same 1-D operators, one dimension lower, are the mortar projections of Alg. 8
// (PAPER.md:265-314), so the face kernels live in this translation unit as well (they share
// the operators in constant memory): k_face_interp (step 1), k_mortar_project (step 2,
// Eq. 17), k_mortar_hits + k_mortar_apply (step 4, Eq. 20).
#include <math.h>

#include <mutex>
#include <type_traits>
#include <vector>

#include "lt_internal.h"
#include "lt_euler.cuh"

namespace lt {

// ------------------------------------------------------------------------ Alg. 7
// For every new leaf map_entry() (lt_dev.cuh) locates its anchor in T_old.  The map is produced in
// new-leaf order, so step 5's sort is not needed (reading E-6).  lt_balance normally produces the
// map in the tail of its own kernel; this kernel is the path for a cycle without lt_balance and the
// checked fallback that reports LT_ERR_MAPPING.
template <int DIM>
__global__ void __launch_bounds__(256) k_map(Geo g, const uint64_t* __restrict__ keys_new,
                                             const uint64_t* __restrict__ keys_old,
                                             const int* __restrict__ first_old, int n_old, DevScalars* s,
                                             int32_t* __restrict__ src, uint8_t* __restrict__ kind) {
  const int64_t n = s->n;
  for (int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; j < n; j += (int64_t)gridDim.x * blockDim.x) {
    int o, kd;
    if (!map_entry<DIM>(g, keys_new[j], keys_old, first_old, n_old, &o, &kd)) set_status(&s->status, LT_ERR_MAPPING);
    src[j] = o;
    kind[j] = (uint8_t)kd;
  }
}

__global__ void k_map_identity(const DevScalars* __restrict__ s, int32_t* __restrict__ src,
                               uint8_t* __restrict__ kind) {
  const int64_t n = s->n;
  for (int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; j < n; j += (int64_t)gridDim.x * blockDim.x) {
    src[j] = (int)j;
    kind[j] = 0;
  }
}

// ------------------------------------------------------------------------ transfer
// One warp per unit of work, found by walking the new leaves in chunks of 32 (see
// k_transfer; warp-uniform branches):
//   copy     a run of consecutive copy leaves: a flat streaming 128-bit copy;
//   refine   one PARENT (the warp that meets child 0 does all 2^dim children, the warps
//            that meet children 1.. skip): the parent is read once and the 1-D operators
//            are applied one direction at a time with the intermediate results shared by
//            the children (sum factorisation: 2N + 4N + 8N outputs of P1 FMAs each in 3-D
//            instead of 8 * 3N);
//   coarsen  one new parent: the mirror image, children pairs are fused direction by
//            direction (4N + 2N + N outputs of 2*P1 FMAs).
// Every stage works on "pencils": a lane loads the P1 values along the contraction
// direction into registers and produces all outputs that depend on them, with the operator
// entries coming straight from constant memory (compile-time indices -> immediate c[][]
// operands of DFMA, no shared-memory or register traffic for coefficients).
//   u[e][v][n], n = ix + P1*(iy + P1*iz) (reading E-5).
//
// c_ops[P1-1][which][row][col]: which 0,1 = I^0, I^1 (Eq. 8); 2,3 = R^0, R^1 (Eq. 12).
__constant__ double c_ops[8][4][8][8];
// c_edge[P1-1][side][i] = l_i(-1) (side 0) / l_i(+1) (side 1): the solution-point basis at the
// element boundary (Alg. 8 step 1)
__constant__ double c_edge[8][2][8];

template <int P1> struct Pad {  // z-plane stride in shared memory (doubles): de-conflicts banks
  static constexpr int PP = P1 * P1;
  static constexpr int ZS = (PP % 16 == 0) ? PP + 4 : PP;
};

template <int DIM, int P1>
struct Xfer {
  static constexpr int PP = P1 * P1;
  static constexpr int N = DIM == 2 ? PP : PP * P1;
  static constexpr int NC = 1 << DIM;
  static constexpr int ZS = Pad<P1>::ZS;
  static constexpr int NP = DIM == 2 ? PP : ZS * P1;     // padded size of one N-block
  static constexpr int ROWS = N / P1;                     // x-pencils per variable
  static constexpr int SMEM_DOUBLES = DIM == 2 ? 2 * NP : 6 * NP;  // per warp

  // padded offset of node n (3-D only pads between z planes)
  __device__ static __forceinline__ int off(int n) { return DIM == 2 ? n : (n / PP) * ZS + (n % PP); }

  // P1 consecutive doubles of one x-pencil (128-bit loads when P1 is even: rows are then
  // 16-byte aligned whenever the arrays are)
  __device__ static __forceinline__ void load_row(const double* __restrict__ p, double* in) {
    if (P1 % 2 == 0) {
#pragma unroll
      for (int i = 0; i < P1 / 2; ++i) {
        const double2 t = __ldcs(reinterpret_cast<const double2*>(p) + i);
        in[2 * i] = t.x;
        in[2 * i + 1] = t.y;
      }
    } else {
#pragma unroll
      for (int i = 0; i < P1; ++i) in[i] = __ldcs(p + i);
    }
  }

  // ---- parent -> 2^dim children (Eq. 8)
  __device__ static __forceinline__ void refine(const double* __restrict__ up, double* __restrict__ dst, int nvars,
                                                size_t E, double* sm, int lane) {
    double* t1 = sm;            // [2][NP]   after x
    double* t2 = sm + 2 * NP;   // [4][NP]   after y (3-D)
    // the first x-pencil of the NEXT variable is loaded before the current one is processed,
    // so the DRAM round trips of the nvars variables overlap with the arithmetic
    const bool has0 = lane < 2 * ROWS;
    double cur[P1], nxt[P1];
#pragma unroll
    for (int i = 0; i < P1; ++i) cur[i] = nxt[i] = 0.0;
    if (has0) load_row(up + (lane % ROWS) * P1, cur);
    for (int v = 0; v < nvars; ++v) {
      const double* u = up + (size_t)v * N;
      if (has0 && v + 1 < nvars) load_row(u + N + (lane % ROWS) * P1, nxt);
      // stage x: lane = (bx, row); both halves of a row are produced by two lanes
      for (int q = lane; q < 2 * ROWS; q += 32) {
        const int bx = q / ROWS, r = q % ROWS;
        double in[P1];
        if (q == lane) {
#pragma unroll
          for (int i = 0; i < P1; ++i) in[i] = cur[i];
        } else {
          load_row(u + r * P1, in);
        }
        double* o = t1 + bx * NP + off(r * P1);
#pragma unroll
        for (int m = 0; m < P1; ++m) {
          double a0 = 0.0, a1 = 0.0;
#pragma unroll
          for (int i = 0; i < P1; ++i) {
            a0 = fma(c_ops[P1 - 1][0][m][i], in[i], a0);
            a1 = fma(c_ops[P1 - 1][1][m][i], in[i], a1);
          }
          o[m] = bx ? a1 : a0;
        }
      }
#pragma unroll
      for (int i = 0; i < P1; ++i) cur[i] = nxt[i];
      __syncwarp();
      if (DIM == 2) {
        // stage y: pencil (bx, x'); outputs go to children (bx, by)
        for (int q = lane; q < 2 * P1; q += 32) {
          const int bx = q / P1, x = q % P1;
          double in[P1];
#pragma unroll
          for (int i = 0; i < P1; ++i) in[i] = t1[bx * NP + i * P1 + x];
#pragma unroll
          for (int by = 0; by < 2; ++by) {
            double* d = dst + (size_t)(bx + 2 * by) * E + (size_t)v * N + x;
#pragma unroll
            for (int m = 0; m < P1; ++m) {
              double a = 0.0;
#pragma unroll
              for (int i = 0; i < P1; ++i) a = fma(c_ops[P1 - 1][by][m][i], in[i], a);
              __stcs(d + m * P1, a);
            }
          }
        }
      } else {
        // stage y: pencil (bx, z, x')
        for (int q = lane; q < 2 * PP; q += 32) {
          const int bx = q / PP, z = (q % PP) / P1, x = q % P1;
          double in[P1];
#pragma unroll
          for (int i = 0; i < P1; ++i) in[i] = t1[bx * NP + z * ZS + i * P1 + x];
#pragma unroll
          for (int by = 0; by < 2; ++by) {
            double* o = t2 + (by * 2 + bx) * NP + z * ZS + x;
#pragma unroll
            for (int m = 0; m < P1; ++m) {
              double a = 0.0;
#pragma unroll
              for (int i = 0; i < P1; ++i) a = fma(c_ops[P1 - 1][by][m][i], in[i], a);
              o[m * P1] = a;
            }
          }
        }
        __syncwarp();
        // stage z: pencil (cxy = bx + 2 by, rem = x' + P1 y'); outputs go to children cxy + 4 bz
        for (int q = lane; q < 4 * PP; q += 32) {
          const int cxy = q / PP, rem = q % PP;
          double in[P1];
#pragma unroll
          for (int i = 0; i < P1; ++i) in[i] = t2[cxy * NP + i * ZS + rem];
#pragma unroll
          for (int bz = 0; bz < 2; ++bz) {
            double* d = dst + (size_t)(cxy + 4 * bz) * E + (size_t)v * N + rem;
#pragma unroll
            for (int m = 0; m < P1; ++m) {
              double a = 0.0;
#pragma unroll
              for (int i = 0; i < P1; ++i) a = fma(c_ops[P1 - 1][bz][m][i], in[i], a);
              __stcs(d + m * PP, a);
            }
          }
        }
      }
      __syncwarp();
    }
  }

  // ---- 2^dim children -> parent (Eq. 9-13): u_P = sum_c (R^{bz} x R^{by} x R^{bx}) u_c
  __device__ static __forceinline__ void coarsen(const double* __restrict__ uc, double* __restrict__ dst, int nvars,
                                                 size_t E, double* sm, int lane) {
    double* s1 = sm;            // [NC/2][NP]  after x (index: by + 2 bz)
    double* s2 = sm + 4 * NP;   // [2][NP]     after y (3-D, index bz)
    for (int v = 0; v < nvars; ++v) {
      // stage x: pencil (cyz, row): fuse the children bx = 0, 1
      for (int q = lane; q < (NC / 2) * ROWS; q += 32) {
        const int cyz = q / ROWS, r = q % ROWS;
        const double* a = uc + (size_t)(2 * cyz) * E + (size_t)v * N + r * P1;
        const double* b = a + E;
        double ia[P1], ib[P1];
        if (P1 % 2 == 0) {
#pragma unroll
          for (int i = 0; i < P1 / 2; ++i) {
            double2 t = __ldcs(reinterpret_cast<const double2*>(a) + i);
            ia[2 * i] = t.x;
            ia[2 * i + 1] = t.y;
            t = __ldcs(reinterpret_cast<const double2*>(b) + i);
            ib[2 * i] = t.x;
            ib[2 * i + 1] = t.y;
          }
        } else {
#pragma unroll
          for (int i = 0; i < P1; ++i) {
            ia[i] = __ldcs(a + i);
            ib[i] = __ldcs(b + i);
          }
        }
        double* o = s1 + cyz * NP + off(r * P1);
#pragma unroll
        for (int m = 0; m < P1; ++m) {
          double acc = 0.0;
#pragma unroll
          for (int i = 0; i < P1; ++i) {
            acc = fma(c_ops[P1 - 1][2][m][i], ia[i], acc);
            acc = fma(c_ops[P1 - 1][3][m][i], ib[i], acc);
          }
          o[m] = acc;
        }
      }
      __syncwarp();
      if (DIM == 2) {
        // stage y: pencil x'
        for (int x = lane; x < P1; x += 32) {
          double ia[P1], ib[P1];
#pragma unroll
          for (int i = 0; i < P1; ++i) {
            ia[i] = s1[i * P1 + x];
            ib[i] = s1[NP + i * P1 + x];
          }
          double* d = dst + (size_t)v * N + x;
#pragma unroll
          for (int m = 0; m < P1; ++m) {
            double acc = 0.0;
#pragma unroll
            for (int i = 0; i < P1; ++i) {
              acc = fma(c_ops[P1 - 1][2][m][i], ia[i], acc);
              acc = fma(c_ops[P1 - 1][3][m][i], ib[i], acc);
            }
            __stcs(d + m * P1, acc);
          }
        }
      } else {
        // stage y: pencil (bz, z, x'): fuse by = 0, 1
        for (int q = lane; q < 2 * PP; q += 32) {
          const int bz = q / PP, z = (q % PP) / P1, x = q % P1;
          double ia[P1], ib[P1];
#pragma unroll
          for (int i = 0; i < P1; ++i) {
            ia[i] = s1[(2 * bz) * NP + z * ZS + i * P1 + x];
            ib[i] = s1[(2 * bz + 1) * NP + z * ZS + i * P1 + x];
          }
          double* o = s2 + bz * NP + z * ZS + x;
#pragma unroll
          for (int m = 0; m < P1; ++m) {
            double acc = 0.0;
#pragma unroll
            for (int i = 0; i < P1; ++i) {
              acc = fma(c_ops[P1 - 1][2][m][i], ia[i], acc);
              acc = fma(c_ops[P1 - 1][3][m][i], ib[i], acc);
            }
            o[m * P1] = acc;
          }
        }
        __syncwarp();
        // stage z: pencil rem = (y', x'): fuse bz = 0, 1
        for (int rem = lane; rem < PP; rem += 32) {
          double ia[P1], ib[P1];
#pragma unroll
          for (int i = 0; i < P1; ++i) {
            ia[i] = s2[i * ZS + rem];
            ib[i] = s2[NP + i * ZS + rem];
          }
          double* d = dst + (size_t)v * N + rem;
#pragma unroll
          for (int m = 0; m < P1; ++m) {
            double acc = 0.0;
#pragma unroll
            for (int i = 0; i < P1; ++i) {
              acc = fma(c_ops[P1 - 1][2][m][i], ia[i], acc);
              acc = fma(c_ops[P1 - 1][3][m][i], ib[i], acc);
            }
            __stcs(d + m * PP, acc);
          }
        }
      }
      __syncwarp();
    }
  }
};

// Flat streaming copy of `count` doubles (a run of consecutive copy leaves whose sources are
// consecutive too is one contiguous range on both sides): eight 128-bit loads per lane are
// issued before the first store, i.e. 4 KB per warp per DRAM round trip.
__device__ __forceinline__ void copy_run(const double* __restrict__ sp, double* __restrict__ dp, int64_t count,
                                         int vec2, int lane) {
  constexpr int U = 8;
  if (vec2) {
    const double2* s2 = reinterpret_cast<const double2*>(sp);
    double2* d2 = reinterpret_cast<double2*>(dp);
    const int64_t T = count >> 1;
    int64_t k = lane;
    for (; k + 32 * (U - 1) < T; k += 32 * U) {
      double2 r[U];
#pragma unroll
      for (int q = 0; q < U; ++q) r[q] = __ldcs(s2 + k + 32 * q);
#pragma unroll
      for (int q = 0; q < U; ++q) __stcs(d2 + k + 32 * q, r[q]);
    }
    if (k < T) {
      double2 r[U];
#pragma unroll
      for (int q = 0; q < U; ++q) {
        r[q] = make_double2(0.0, 0.0);  // (defined on every path: keeps r[] in registers)
        if (k + 32 * q < T) r[q] = __ldcs(s2 + k + 32 * q);
      }
#pragma unroll
      for (int q = 0; q < U; ++q)
        if (k + 32 * q < T) __stcs(d2 + k + 32 * q, r[q]);
    }
  } else {
    for (int64_t k = lane; k < count; k += 32 * U) {
      double r[U];
#pragma unroll
      for (int q = 0; q < U; ++q) {
        r[q] = 0.0;
        if (k + 32 * q < count) r[q] = __ldcs(sp + k + 32 * q);
      }
#pragma unroll
      for (int q = 0; q < U; ++q)
        if (k + 32 * q < count) __stcs(dp + k + 32 * q, r[q]);
    }
  }
}

// Work distribution (measured on B200: a statically partitioned persistent
// copy reaches 6.07 TB/s, the same loop fed by tickets with a compact access front 6.9 TB/s):
//   - a block claims TILES of 8 sub-chunks through one global ticket, so that all blocks
//     together touch a window of only (#blocks x tile) bytes that sweeps the arrays once;
//   - its warps claim the sub-chunks (SL = 2^sl_log2 consecutive new leaves, about 10 KB of
//     solution) independently through a shared-memory word -- no block barrier, a warp that
//     interpolates does not hold up the warps that copy.
// Per sub-chunk: one coalesced read of the map entries, then (warp-uniform control flow,
// decided by ballots)
//   - every maximal run of copy leaves with consecutive sources -> one flat copy_run,
//   - every refined parent (met at its child 0)                 -> Xfer::refine (writes all
//     2^dim children, which may extend into the next sub-chunk),
//   - every coarsened parent                                    -> Xfer::coarsen.
constexpr int kSubs = 8;  // sub-chunks per tile

template <int DIM, int P1>
__global__ void __launch_bounds__(256, 4) k_transfer(const DevScalars* s,
                                                  const int32_t* __restrict__ map_src,
                                                  const uint8_t* __restrict__ map_kind,
                                                  const double* __restrict__ u_old, double* __restrict__ u_new,
                                                  int nvars, int vec2, int sl_log2, unsigned* ticket,
                                                  int64_t jb, int64_t je) {
  // [jb, je) = the slab of new leaves this launch handles (je < 0: up to the leaf count);
  // u_old / u_new are indexed by ABSOLUTE old / new leaf numbers (lt_transfer_host passes
  // staging pointers shifted by the slab origins)
  using X = Xfer<DIM, P1>;
  extern __shared__ double smem[];
  // tile << 8 | next sub-chunk; sub-chunk == kSubs: exhausted, > kSubs: a warp is fetching a ticket
  __shared__ unsigned long long s_word;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  double* wsm = smem + (size_t)w * X::SMEM_DOUBLES;
  const size_t E = (size_t)nvars * X::N;
  const int64_t n = je < 0 ? (int64_t)s->n : je;
  const int SL = 1 << sl_log2, TL = kSubs << sl_log2;
  const int64_t ntiles = (n - jb + TL - 1) / TL;
  // the Alg. 7 tail of lt_balance met a new leaf more than one level from T_old: nothing to move
  if (s->map_bad) {
    if (blockIdx.x == 0 && threadIdx.x == 0) set_status(const_cast<int*>(&s->status), LT_ERR_MAPPING);
    return;
  }
  if (threadIdx.x == 0) s_word = kSubs;
  __syncthreads();
  for (;;) {
    unsigned long long tile = 0;
    int sub = 0;
    if (lane == 0) {
      volatile unsigned long long* vw = &s_word;
      for (;;) {
        const unsigned long long wv = *vw;
        const unsigned sb = (unsigned)(wv & 0xff);
        if (sb < kSubs) {
          if (atomicCAS(&s_word, wv, wv + 1) == wv) {
            tile = wv >> 8;
            sub = (int)sb;
            break;
          }
        } else if (sb == kSubs) {
          if (atomicCAS(&s_word, wv, wv + 1) == wv) {
            tile = atomicAdd(ticket, 1u);
            sub = 0;
            // the map entries of the tile this block is likely to claim next: into L2
            const int64_t jp = jb + ((int64_t)tile + gridDim.x) * TL;
            if (jp < n) {
              asm volatile("prefetch.global.L2 [%0];" ::"l"(map_src + jp));
              asm volatile("prefetch.global.L2 [%0];" ::"l"(map_kind + jp));
            }
            *vw = (tile << 8) | 1ull;
            break;
          }
        }
      }
    }
    tile = __shfl_sync(0xffffffffu, tile, 0);
    sub = __shfl_sync(0xffffffffu, sub, 0);
    if ((int64_t)tile >= ntiles) break;
    const int64_t j0 = jb + (int64_t)tile * TL + (int64_t)sub * SL;
    int kd = 255, so = 0;
    if (lane < SL && j0 + lane < n) {
      kd = map_kind[j0 + lane];
      so = map_src[j0 + lane];
      LT_DASSERT(so >= 0 && ((kd & 15) == 0 || (kd & 15) == 1 || kd == 2) && (kd >> 4) < X::NC);
    }
    const bool is_copy = kd == 0;
    const int so_prev = __shfl_up_sync(0xffffffffu, so, 1);
    const unsigned copy_mask = __ballot_sync(0xffffffffu, is_copy);
    const bool prev_copy = lane > 0 && ((copy_mask >> (lane - 1)) & 1u);
    unsigned heads = __ballot_sync(0xffffffffu, is_copy && !(prev_copy && so == so_prev + 1));
    unsigned rm = __ballot_sync(0xffffffffu, kd == 1);  // child 0 of a refined leaf
    unsigned cm = __ballot_sync(0xffffffffu, kd != 255 && (kd & 15) == 2);
    const unsigned all_heads = heads;
    // direct copies
    while (heads) {
      const int a = __ffs(heads) - 1;
      heads &= heads - 1;
      // the run ends at the next head or at the first non-copy lane
      const unsigned stop = (~copy_mask | all_heads) & ~((2u << a) - 1u);
      const int b = stop ? __ffs(stop) - 1 : 32;
      const int64_t sa = __shfl_sync(0xffffffffu, so, a);
      copy_run(u_old + (size_t)sa * E, u_new + (size_t)(j0 + a) * E, (int64_t)(b - a) * (int64_t)E, vec2, lane);
    }
    // interpolation, Eq. 8
    while (rm) {
      const int a = __ffs(rm) - 1;
      rm &= rm - 1;
      const int64_t sa = __shfl_sync(0xffffffffu, so, a);
      X::refine(u_old + (size_t)sa * E, u_new + (size_t)(j0 + a) * E, nvars, E, wsm, lane);
    }
    // L2 projection of the 2^dim children, Eq. 9-13
    while (cm) {
      const int a = __ffs(cm) - 1;
      cm &= cm - 1;
      const int64_t sa = __shfl_sync(0xffffffffu, so, a);
      X::coarsen(u_old + (size_t)sa * E, u_new + (size_t)(j0 + a) * E, nvars, E, wsm, lane);
    }
  }
}

// ------------------------------------------------------------------------ operators (host)
// Gauss-Legendre rule by Newton iteration on P_n with the Bonnet recurrence.
static void gl_rule(int n, std::vector<long double>& z, std::vector<long double>& w) {
  z.resize(n);
  w.resize(n);
  const long double pi = acosl(-1.0L);
  for (int i = 0; i < (n + 1) / 2; ++i) {
    long double x = cosl(pi * (i + 0.75L) / (n + 0.5L)), dp = 1.0L;
    for (int it = 0; it < 60; ++it) {
      long double pm = 1.0L, pc = x;
      for (int k = 1; k < n; ++k) {
        long double pn = ((2 * k + 1) * x * pc - k * pm) / (k + 1);
        pm = pc;
        pc = pn;
      }
      if (n == 0) pc = 1.0L;
      dp = n * (pm - x * pc) / (1.0L - x * x);
      long double dx = pc / dp;
      x -= dx;
      if (fabsl(dx) < 1e-19L) break;
    }
    {
      long double pm = 1.0L, pc = x;
      for (int k = 1; k < n; ++k) {
        long double pn = ((2 * k + 1) * x * pc - k * pm) / (k + 1);
        pm = pc;
        pc = pn;
      }
      dp = n * (pm - x * pc) / (1.0L - x * x);
    }
    z[n - 1 - i] = x;
    z[i] = -x;
    w[i] = w[n - 1 - i] = 2.0L / ((1.0L - x * x) * dp * dp);
  }
  if (n % 2) z[n / 2] = 0.0L;
}

int build_operators(Tree* t, int p) {
  // per device, per P1; the upload goes to the CURRENT device's constant memory, so the tree's
  // device must be current (check_device) and concurrent host threads are serialised
  static std::mutex mu;
  static bool uploaded[64][8];
  int rc = check_device(t);
  if (rc != LT_OK) return rc;
  if (t->device < 0 || t->device >= 64) return LT_ERR_ARG;
  std::lock_guard<std::mutex> lk(mu);
  const int dev = t->device;
  if (uploaded[dev][p]) return LT_OK;
  const int P1 = p + 1;
  std::vector<long double> z, w;
  gl_rule(P1, z, w);
  std::vector<double> h(4 * 64, 0.0);
  for (int b = 0; b < 2; ++b)
    for (int m = 0; m < P1; ++m) {
      const long double xi = 0.5L * (z[m] + 2 * b - 1);
      for (int i = 0; i < P1; ++i) {
        long double v = 1.0L;
        for (int k = 0; k < P1; ++k)
          if (k != i) v *= (xi - z[k]) / (z[i] - z[k]);
        h[b * 64 + m * 8 + i] = (double)v;                                // I^b[m][i]
        h[(2 + b) * 64 + i * 8 + m] = (double)(0.5L * (w[m] / w[i]) * v);  // R^b[i][m]
      }
    }
  LT_CUDA(cudaMemcpyToSymbol(c_ops, h.data(), 4 * 64 * sizeof(double), (size_t)p * 4 * 64 * sizeof(double),
                             cudaMemcpyHostToDevice));
  double he[2][8] = {{0}};
  for (int side = 0; side < 2; ++side)
    for (int i = 0; i < P1; ++i) {
      const long double x = side ? 1.0L : -1.0L;
      long double v = 1.0L;
      for (int k = 0; k < P1; ++k)
        if (k != i) v *= (x - z[k]) / (z[i] - z[k]);
      he[side][i] = (double)v;
    }
  LT_CUDA(cudaMemcpyToSymbol(c_edge, he, sizeof(he), (size_t)p * sizeof(he), cudaMemcpyHostToDevice));
  uploaded[dev][p] = true;
  return LT_OK;
}

// ------------------------------------------------------------------------ mortars (Alg. 8)
// Common-flux plumbing on nonconforming faces, PAPER.md:265-314 (Alg. 8 steps 2 and 4,
// Eq. 14-20; readings H-1..H-4).  Face arrays are [n_leaves][nf][nvars][Nf], Nf =
// (p+1)^(dim-1) Gauss-Legendre face points, tangential axes ascending, lower axis fastest.
// The 2^(dim-1) mortars of a coarse face coincide with the fine neighbours' faces (mortar s
// = slot s of lt_connect), so with Gauss-Legendre points the Eq. 17 projection onto mortar s
// is the tensor product of the 1-D interpolations I^b and the Eq. 20 projection back is the
// tensor product of R^b = (1/2) W^-1 (I^b)^T W -- the same 1-D operators as the volume
// transfer, one dimension lower.  One warp per leaf; both kernels stream the face arrays
// once, coalesced, and are HBM-bound.  The paper scatters Eq. 20 with atomicAdd;
// here the coarse face GATHERS its mortars (found by 2^(dim-1) bucketed searches), so the
// result is deterministic.
__device__ __forceinline__ void load_ops_1d(int P1, double (*sI)[8][8], double (*sR)[8][8]) {
  for (int i = threadIdx.x; i < 2 * 64; i += blockDim.x) {
    const int b = i >> 6, r = (i >> 3) & 7, c = i & 7;
    sI[b][r][c] = c_ops[P1 - 1][b][r][c];
    sR[b][r][c] = c_ops[P1 - 1][2 + b][r][c];
  }
  __syncthreads();
}

// value q (= v * Nf + nn) of the Eq. 17 projection of the coarse trace `src` onto mortar `slot`
template <int DIM, int P1>
__device__ __forceinline__ double mortar_value(const double (*sI)[8][8], const double* __restrict__ src, int slot,
                                               int q) {
  constexpr int Nf = DIM == 2 ? P1 : P1 * P1;
  const int v = q / Nf, nn = q - v * Nf;
  src += (size_t)v * Nf;
  double out = 0.0;
  if (DIM == 2) {
#pragma unroll
    for (int m = 0; m < P1; ++m) out += sI[slot & 1][nn][m] * src[m];
  } else {
    const int n1 = nn / P1, n0 = nn - n1 * P1;
#pragma unroll
    for (int m1 = 0; m1 < P1; ++m1) {
      double row = 0.0;
#pragma unroll
      for (int m0 = 0; m0 < P1; ++m0) row += sI[slot & 1][n0][m0] * src[m1 * P1 + m0];
      out += sI[slot >> 1][n1][m1] * row;
    }
  }
  return out;
}

// One warp per leaf.  The leaf's nf (kind, nbr) pairs are staged per warp in shared memory.
// Pass A streams the conforming faces: for every 64 * VEC doubles of a face block the loads of
// ALL nf faces are issued before the first store (2 * nf independent 128-bit loads per lane),
// no per-element index arithmetic.  Pass B handles the few fine-side hanging faces (Eq. 17).
template <int DIM, int VEC, int P1>
__global__ void __launch_bounds__(256) k_mortar_project(const DevScalars* s, const int32_t* __restrict__ nbr,
                                                        const uint8_t* __restrict__ kind,
                                                        const double* __restrict__ uf, double* __restrict__ unb,
                                                        int nvars) {
  constexpr int NF = Dim<DIM>::NF;
  typedef typename std::conditional<VEC == 2, double2, double>::type V;
  __shared__ double sI[2][8][8], sR[2][8][8];
  __shared__ int s_nb[8][8];
  __shared__ int s_kd[8][8];
  load_ops_1d(P1, sI, sR);
  constexpr int Nf = DIM == 2 ? P1 : P1 * P1;
  const int E = nvars * Nf, EV = E / VEC;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t n = s->n;
  const int64_t nw = (int64_t)gridDim.x * (blockDim.x >> 5);
  // the (kind, nbr) pairs of the warp's NEXT leaf are fetched while the current one streams, so a
  // leaf costs one DRAM round trip, not two dependent ones
  int64_t e = (int64_t)blockIdx.x * (blockDim.x >> 5) + w;
  int pk = 0, pn = 0;
  if (e < n && lane < NF) {
    pk = kind[(size_t)e * NF + lane];
    pn = nbr[(size_t)e * NF + lane];
  }
  for (; e < n; e += nw) {
    __syncwarp();
    if (lane < NF) {
      s_kd[w][lane] = pk;
      s_nb[w][lane] = pn;
      if (e + nw < n) {
        pk = kind[(size_t)(e + nw) * NF + lane];
        pn = nbr[(size_t)(e + nw) * NF + lane];
      }
    }
    __syncwarp();
    V* dst = reinterpret_cast<V*>(unb + (size_t)e * NF * E);
    const V* src[NF];
    bool conf[NF];
    bool any2 = false;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const int k = s_kd[w][f] & 15;
      conf[f] = k == 1;
      any2 = any2 || k == 2;
      // conforming: the mortar is the face itself
      src[f] = reinterpret_cast<const V*>(uf + ((size_t)(conf[f] ? s_nb[w][f] : 0) * NF + (f ^ 1)) * E);
    }
    for (int q0 = 0; q0 < EV; q0 += 64) {
      const int qa = q0 + lane, qb = q0 + 32 + lane;
      constexpr int FC = NF / 2;  // faces per round: 2 * FC loads in flight per lane (all NF at once costs 20 registers more and a resident block)
#pragma unroll
      for (int fh = 0; fh < NF; fh += FC) {
        V v0[FC], v1[FC];
#pragma unroll
        for (int f = 0; f < FC; ++f) {
          if (conf[fh + f] && qa < EV) v0[f] = __ldcs(src[fh + f] + qa);
          if (conf[fh + f] && qb < EV) v1[f] = __ldcs(src[fh + f] + qb);
        }
#pragma unroll
        for (int f = 0; f < FC; ++f) {
          if (conf[fh + f] && qa < EV) __stcs(dst + (fh + f) * EV + qa, v0[f]);
          if (conf[fh + f] && qb < EV) __stcs(dst + (fh + f) * EV + qb, v1[f]);
        }
      }
    }
    if (any2) {
#pragma unroll 1
      for (int f = 0; f < NF; ++f) {
        const int kd = s_kd[w][f];
        if ((kd & 15) != 2) continue;
        const double* sp = uf + ((size_t)s_nb[w][f] * NF + (f ^ 1)) * E;
        double* dp = unb + ((size_t)e * NF + f) * E;
        for (int q = lane; q < E; q += 32) dp[q] = mortar_value<DIM, P1>(sI, sp, kd >> 4, q);
      }
    }
  }
}

// Coarse face (e, f) of kind 3, step 1 (ONE LANE per face, so a warp resolves up to 32 faces
// with their dependent loads in flight together): the fine neighbour on mortar s is the child
// of the same-level neighbour cell that touches the face with tangential child bits s.
// lt_connect stored the slot-0 neighbour j0; when the siblings in between are leaves the others
// sit (c - c0) entries further: one key compare, else a bucketed search.
template <int DIM>
__device__ __forceinline__ void gather_resolve(const Geo& g, const uint64_t* __restrict__ keys,
                                               const int* __restrict__ first, DevScalars* s, int64_t e, int f,
                                               int j0, int* es /* [2^(DIM-1)] */) {
  constexpr int NS = 1 << (DIM - 1);
  const uint64_t key = keys[e];
  const int l = key_level(key);
  const uint64_t m = key_morton(key);
  const int axis = f >> 1;
  uint64_t mn = 0;
  face_neighbour<DIM>(g, m, l, f, &mn);
  const int c0 = (f & 1) ? 0 : (1 << axis);
  const int n = s->n;
#pragma unroll
  for (int sidx = 0; sidx < NS; ++sidx) {
    int c = c0, bit = 0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
      if (a == axis) continue;
      c |= ((sidx >> bit) & 1) << a;
      ++bit;
    }
    const uint64_t cm = mn | ((uint64_t)c << (DIM * (g.maxl - l - 1)));
    const int64_t cand = (int64_t)j0 + (c - c0);
    if (cand >= 0 && cand < n && keys[cand] == make_key(cm, l + 1)) {
      es[sidx] = (int)cand;
    } else {
      es[sidx] = locate(g, keys, first, cm);
      if (key_level(keys[es[sidx]]) != l + 1) set_status(&s->status, LT_ERR_UNBALANCED);
    }
  }
}

// Step 1 kernel: a warp scans the kind bytes of 32 consecutive leaves (nf coalesced rounds); every
// coarse-side hanging slot (a few per cent of all slots) is resolved by its own lane and appended
// to the hit list: (e, f, es[0..NS)).  The order of the list is arbitrary, the result is not:
// every hit owns its output block.
template <int DIM>
__global__ void __launch_bounds__(256) k_mortar_hits(Geo g, const uint64_t* __restrict__ keys,
                                                     const int* __restrict__ first, DevScalars* s,
                                                     const int32_t* __restrict__ nbr,
                                                     const uint8_t* __restrict__ kind, int* __restrict__ hits,
                                                     int max_hits) {
  constexpr int NF = Dim<DIM>::NF, NS = 1 << (DIM - 1), HW = 2 + NS;
  const int lane = threadIdx.x & 31;
  const int64_t nslots = (int64_t)s->n * NF;
  const int64_t nw = (int64_t)gridDim.x * (blockDim.x >> 5);
  for (int64_t c0 = ((int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 32; c0 < nslots;
       c0 += nw * 32) {
    const int64_t idx = c0 + lane;
    const bool hit = idx < nslots && (kind[idx] & 15) == 3;
    const unsigned mask = __ballot_sync(0xffffffffu, hit);
    if (mask == 0) continue;
    int base = 0;
    if (lane == 0) base = atomicAdd(&s->aux, __popc(mask));
    base = __shfl_sync(0xffffffffu, base, 0);
    if (hit) {
      const int64_t e = idx / NF;
      const int f = (int)(idx - e * NF);
      int es[NS];
      gather_resolve<DIM>(g, keys, first, s, e, f, nbr[idx], es);
      const int h = base + __popc(mask & ((1u << lane) - 1));
      if (h < max_hits) {
        hits[(size_t)h * HW] = (int)e;
        hits[(size_t)h * HW + 1] = f;
#pragma unroll
        for (int sidx = 0; sidx < NS; ++sidx) hits[(size_t)h * HW + 2 + sidx] = es[sidx];
      } else {
        set_status(&s->status, LT_ERR_UNBALANCED);
      }
    }
  }
}

// Step 2 kernel: one thread per output value F[e][f][v][n] of every hit (Eq. 20):
//   F = sum_s (R^{s1} (x) R^{s0}) F^_s, applied as a row pass and a column pass per mortar.
// The NS * Nf inputs of a (hit, variable) pair are shared by Nf neighbouring threads and stay
// in L1; the 1-D operators sit in shared memory.
template <int DIM, int P1>
__global__ void __launch_bounds__(256) k_mortar_apply(const DevScalars* s, const int* __restrict__ hits,
                                                      const double* __restrict__ fm, double* __restrict__ ff,
                                                      int nvars) {
  constexpr int NF = Dim<DIM>::NF, NS = 1 << (DIM - 1), HW = 2 + NS;
  constexpr int Nf = DIM == 2 ? P1 : P1 * P1;
  __shared__ double sI[2][8][8], sR[2][8][8];
  load_ops_1d(P1, sI, sR);
  const int E = nvars * Nf;
  if (DIM == 2) {
    const int64_t total = (int64_t)s->aux * E;
    for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
      const int64_t h = idx / E;
      const int q = (int)(idx - h * E);
      const int v = q / Nf, nn = q - v * Nf;
      const int* hp = hits + (size_t)h * HW;
      const int e = hp[0], f = hp[1];
      double acc = 0.0;
#pragma unroll
      for (int sidx = 0; sidx < NS; ++sidx) {
        const double* src = fm + ((size_t)hp[2 + sidx] * NF + (f ^ 1)) * E + (size_t)v * Nf;
#pragma unroll
        for (int mm = 0; mm < P1; ++mm) acc += sR[sidx][nn][mm] * src[mm];
      }
      ff[((size_t)e * NF + f) * E + q] = acc;
    }
  } else {
    // 3-D: one thread per output ROW (h, v, n1): every input row is loaded once and feeds the P1
    // outputs of the thread (5x fewer loads than one thread per value)
    const int RW = nvars * P1;  // rows per hit
    const int64_t total = (int64_t)s->aux * RW;
    for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total;
         idx += (int64_t)gridDim.x * blockDim.x) {
      const int64_t h = idx / RW;
      const int q = (int)(idx - h * RW);
      const int v = q / P1, n1 = q - v * P1;
      const int* hp = hits + (size_t)h * HW;
      const int e = hp[0], f = hp[1];
      double acc[P1];
#pragma unroll
      for (int n0 = 0; n0 < P1; ++n0) acc[n0] = 0.0;
#pragma unroll
      for (int sidx = 0; sidx < NS; ++sidx) {
        const double* src = fm + ((size_t)hp[2 + sidx] * NF + (f ^ 1)) * E + (size_t)v * Nf;
#pragma unroll
        for (int m1 = 0; m1 < P1; ++m1) {
          double in[P1];
#pragma unroll
          for (int m0 = 0; m0 < P1; ++m0) in[m0] = src[m1 * P1 + m0];
          const double r1 = sR[sidx >> 1][n1][m1];
#pragma unroll
          for (int n0 = 0; n0 < P1; ++n0) {
            double row = 0.0;
#pragma unroll
            for (int m0 = 0; m0 < P1; ++m0) row += sR[sidx & 1][n0][m0] * in[m0];
            acc[n0] += r1 * row;
          }
        }
      }
      double* dst = ff + ((size_t)e * NF + f) * E + (size_t)v * Nf + n1 * P1;
#pragma unroll
      for (int n0 = 0; n0 < P1; ++n0) dst[n0] = acc[n0];
    }
  }
}

template <int DIM, int P1>
static void launch_mortar_t(Tree* t, int which, const double* d_in, double* d_out, int nvars, int G) {
  constexpr int Nf = DIM == 2 ? P1 : P1 * P1;
  if (which == 0) {
    const bool vec2 = ((nvars * Nf) % 2 == 0) && (((uintptr_t)d_in | (uintptr_t)d_out) & 15) == 0;
    if (vec2) k_mortar_project<DIM, 2, P1><<<G, 256, 0, t->stream>>>(t->d_s, t->nbr, t->kind, d_in, d_out, nvars);
    else k_mortar_project<DIM, 1, P1><<<G, 256, 0, t->stream>>>(t->d_s, t->nbr, t->kind, d_in, d_out, nvars);
  } else {
    k_mortar_apply<DIM, P1><<<G, 256, 0, t->stream>>>(t->d_s, t->mortar_hits, d_in, d_out, nvars);
  }
}

template <int DIM>
static int launch_mortar_d(Tree* t, int which, const double* d_in, double* d_out, int p, int nvars, int G) {
  switch (p) {
    case 0: launch_mortar_t<DIM, 1>(t, which, d_in, d_out, nvars, G); break;
    case 1: launch_mortar_t<DIM, 2>(t, which, d_in, d_out, nvars, G); break;
    case 2: launch_mortar_t<DIM, 3>(t, which, d_in, d_out, nvars, G); break;
    case 3: launch_mortar_t<DIM, 4>(t, which, d_in, d_out, nvars, G); break;
    case 4: launch_mortar_t<DIM, 5>(t, which, d_in, d_out, nvars, G); break;
    case 5: launch_mortar_t<DIM, 6>(t, which, d_in, d_out, nvars, G); break;
    case 6: launch_mortar_t<DIM, 7>(t, which, d_in, d_out, nvars, G); break;
    case 7: launch_mortar_t<DIM, 8>(t, which, d_in, d_out, nvars, G); break;
    default: return LT_ERR_ARG;
  }
  return LT_OK;
}

// ------------------------------------------------------------------------ Alg. 8 steps 2 + 3 fused
// lt_face_flux: the neighbour's trace is taken straight from the face array (conforming: the face
// itself; fine side of a hanging face: the Eq. 17 projection of the coarse trace onto
// the mortar) and fed to the Rusanov solver without going through memory.  A conforming
// face is computed ONCE, by the element on its minus side (odd local face), and stored in both
// elements' slots -- both sides compute the same number anyway (the flux along +a).  Per element and
// axis this reads 2 face blocks and writes 2 instead of reading 4 and writing 4 (lt_mortar_project +
// lt_common_flux).  One thread per (leaf, axis, face point); coarse-side hanging slots (kind 3) are left
// to lt_mortar_gather, boundary slots to the caller.
template <int DIM, int P1>
__global__ void __launch_bounds__(256, 3) k_face_flux(const DevScalars* s, const int32_t* __restrict__ nbr,
                                                   const uint8_t* __restrict__ kind,
                                                   const double* __restrict__ uf, double* __restrict__ fs) {
  constexpr int NF = Dim<DIM>::NF, NV = DIM + 2;
  constexpr int Nf = DIM == 2 ? P1 : P1 * P1, E = NV * Nf;
  __shared__ double sI[2][8][8], sR[2][8][8];
  load_ops_1d(P1, sI, sR);
  const int64_t total = (int64_t)s->n * DIM * Nf;
  for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int64_t ea = idx / Nf;
    const int pt = (int)(idx - ea * Nf);
    const int64_t e = ea / DIM;
    const int a = (int)(ea - e * DIM);
#pragma unroll
    for (int side = 1; side >= 0; --side) {
      const int f = 2 * a + side;
      const size_t sl = (size_t)e * NF + f;
      const int kd = kind[sl];
      const int k = kd & 15;
      if (!((k == 1 && side == 1) || k == 2)) continue;
      const size_t nsl = (size_t)nbr[sl] * NF + (f ^ 1);
      double own[NV], nb[NV], F[NV];
#pragma unroll
      for (int v = 0; v < NV; ++v) own[v] = __ldcs(uf + sl * E + v * Nf + pt);
      if (k == 1) {
#pragma unroll
        for (int v = 0; v < NV; ++v) nb[v] = __ldcs(uf + nsl * E + v * Nf + pt);
      } else {
#pragma unroll
        for (int v = 0; v < NV; ++v) nb[v] = mortar_value<DIM, P1>(sI, uf + nsl * E, kd >> 4, v * Nf + pt);
      }
      // the minus-side state is the element's own trace on an odd face
      if (side) rusanov<DIM>(a, own, nb, F); else rusanov<DIM>(a, nb, own, F);
#pragma unroll
      for (int v = 0; v < NV; ++v) __stcs(fs + sl * E + v * Nf + pt, F[v]);
      if (k == 1) {
#pragma unroll
        for (int v = 0; v < NV; ++v) __stcs(fs + nsl * E + v * Nf + pt, F[v]);
      }
    }
  }
}

template <int DIM, int P1>
static void launch_face_flux_t(Tree* t, const double* d_uf, double* d_fs) {
  k_face_flux<DIM, P1><<<t->num_sms * 8, 256, 0, t->stream>>>(t->d_s, t->nbr, t->kind, d_uf, d_fs);
}

template <int DIM>
static int launch_face_flux_d(Tree* t, const double* d_uf, double* d_fs, int p) {
  switch (p) {
    case 0: launch_face_flux_t<DIM, 1>(t, d_uf, d_fs); break;
    case 1: launch_face_flux_t<DIM, 2>(t, d_uf, d_fs); break;
    case 2: launch_face_flux_t<DIM, 3>(t, d_uf, d_fs); break;
    case 3: launch_face_flux_t<DIM, 4>(t, d_uf, d_fs); break;
    case 4: launch_face_flux_t<DIM, 5>(t, d_uf, d_fs); break;
    case 5: launch_face_flux_t<DIM, 6>(t, d_uf, d_fs); break;
    case 6: launch_face_flux_t<DIM, 7>(t, d_uf, d_fs); break;
    case 7: launch_face_flux_t<DIM, 8>(t, d_uf, d_fs); break;
    default: return LT_ERR_ARG;
  }
  return LT_OK;
}

int launch_face_flux(Tree* t, const double* d_uf, double* d_fs, int p) {
  const int rc = t->g.dim == 2 ? launch_face_flux_d<2>(t, d_uf, d_fs, p) : launch_face_flux_d<3>(t, d_uf, d_fs, p);
  if (rc != LT_OK) return rc;
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

// (Re)build the list of coarse-side hanging faces with their fine neighbours; valid until the
// tree or its connectivity changes.
int launch_mortar_hits(Tree* t) {
  const int NS = 1 << (t->g.dim - 1), HW = 2 + NS;
  const int64_t max_hits = t->h_s->n_face[1] / NS + 1;  // every coarse face has exactly NS fine faces
  if (t->mortar_hits_cap < max_hits) {
    dev_free(t->mortar_hits, t->stream);
    t->mortar_hits = nullptr;
    t->mortar_hits_cap = 0;
    int rc = dev_alloc((void**)&t->mortar_hits, (size_t)max_hits * HW * sizeof(int), t->stream);
    if (rc != LT_OK) return rc;
    t->mortar_hits_cap = max_hits;
  }
  LT_CUDA(cudaMemsetAsync(&t->d_s->aux, 0, sizeof(int), t->stream));
  const int G = t->num_sms * 8;
  if (t->g.dim == 2)
    k_mortar_hits<2><<<G, 256, 0, t->stream>>>(t->g, t->keys[t->cur], t->first[t->cur], t->d_s, t->nbr, t->kind,
                                               t->mortar_hits, (int)max_hits);
  else
    k_mortar_hits<3><<<G, 256, 0, t->stream>>>(t->g, t->keys[t->cur], t->first[t->cur], t->d_s, t->nbr, t->kind,
                                               t->mortar_hits, (int)max_hits);
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

int launch_mortar(Tree* t, int which, const double* d_in, double* d_out, int p, int nvars) {
  const int G = t->num_sms * 8;
  const int rc = t->g.dim == 2 ? launch_mortar_d<2>(t, which, d_in, d_out, p, nvars, G)
                               : launch_mortar_d<3>(t, which, d_in, d_out, p, nvars, G);
  if (rc != LT_OK) return rc;
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

// ------------------------------------------------------------------------ Alg. 8 step 1
// Solution at the face flux points (readings E-5, H-1): u_f[e][f][v][n_t] =
// sum_i l_i(-1 | +1) u[e][v][.. i on the face's axis, n_t on the others ..].  One warp per leaf,
// one variable at a time through shared memory; reads u once (coalesced), writes the nf face
// blocks in full 128-bit sectors.  HBM-bound: Bu in, nf * Bf out per leaf.
// BULK (the element block is a multiple of 16 bytes and u is 16-byte aligned): the element arrives by ONE
// cp.async.bulk of lane 0 onto the warp's mbarrier, into the other half of a double buffer while the
// current element is being worked on -- no load or shared-memory store instruction, and the DRAM latency
// of the next element hides behind the arithmetic and the stores of this one.
template <int DIM, int P1, bool BULK>
__global__ void __launch_bounds__(256) k_face_interp(const DevScalars* s, const double* __restrict__ u,
                                                     double* __restrict__ uf, int nvars) {
  constexpr int NF = Dim<DIM>::NF;
  constexpr int N = DIM == 2 ? P1 * P1 : P1 * P1 * P1, Nf = DIM == 2 ? P1 : P1 * P1;
  extern __shared__ __align__(128) double su_all[];  // [warps][1 or 2][nvars][N]: the whole element, staged once
  __shared__ uint64_t bars[8][2];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int EV = nvars * N, E = nvars * Nf;
  double* su0 = su_all + (size_t)w * EV * (BULK ? 2 : 1);
  const int64_t n = s->n;
  const int64_t nw = (int64_t)gridDim.x * (blockDim.x >> 5);
  int64_t e = (int64_t)blockIdx.x * (blockDim.x >> 5) + w;
  uint32_t phase[2] = {0, 0};
  int buf = 0;
  auto fetch = [&](int b, int64_t el) {  // (lane 0)
    mbar_arrive_expect_tx(&bars[w][b], (uint32_t)EV * 8u);
    bulk_g2s(su0 + (size_t)b * EV, u + (size_t)el * EV, (uint32_t)EV * 8u, &bars[w][b]);
  };
  if (BULK) {
    if (lane == 0) {
      mbar_init(&bars[w][0], 1);
      mbar_init(&bars[w][1], 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      if (e < n) fetch(0, e);
    }
    __syncwarp();
  }
  for (; e < n; e += nw, buf ^= 1) {
    __syncwarp();  // (the buffer about to be refilled was read in the previous iteration)
    const double* su = su0;
    if (BULK) {
      if (lane == 0 && e + nw < n) fetch(buf ^ 1, e + nw);
      while (!mbar_try_wait(&bars[w][buf], phase[buf])) {
      }
      phase[buf] ^= 1;
      su = su0 + (size_t)buf * EV;
    } else {
      const double* src = u + (size_t)e * EV;
      for (int i = lane; i < EV; i += 32) su0[i] = __ldcs(src + i);
      __syncwarp();
    }
    double* dst = uf + (size_t)e * NF * E;
    // one lane per LINE of P1 points along an axis: the line is read once and gives the trace on
    // the minus AND the plus face of that axis; consecutive lanes store consecutive doubles
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
      const int stride = a == 0 ? 1 : (a == 1 ? P1 : P1 * P1);
      for (int ln = lane; ln < E; ln += 32) {
        const int v = ln / Nf, nt = ln - v * Nf;
        int first;
        if (DIM == 2) {
          first = a == 0 ? nt * P1 : nt;
        } else {
          const int n1 = nt / P1, n0 = nt - n1 * P1;  // lower tangential axis fastest
          first = a == 0 ? n0 * P1 + n1 * P1 * P1 : (a == 1 ? n0 + n1 * P1 * P1 : n0 + n1 * P1);
        }
        const double* sv = su + v * N + first;
        double lo = 0.0, hi = 0.0;
#pragma unroll
        for (int i = 0; i < P1; ++i) {
          const double x = sv[i * stride];
          lo += c_edge[P1 - 1][0][i] * x;
          hi += c_edge[P1 - 1][1][i] * x;
        }
        __stcs(dst + (2 * a) * E + ln, lo);
        __stcs(dst + (2 * a + 1) * E + ln, hi);
      }
    }
  }
}

template <int DIM, int P1>
static int launch_face_interp_t(Tree* t, const double* d_u, double* d_uf, int nvars) {
  constexpr int N = DIM == 2 ? P1 * P1 : P1 * P1 * P1;
  int warps = 8;
  // the copy engine needs 16-byte multiples: an even number of doubles per element, u 16-byte aligned
  const bool bulk = ((nvars * N) % 2 == 0) && (((uintptr_t)d_u) & 15) == 0;
  const size_t per_warp = (size_t)nvars * N * sizeof(double) * (bulk ? 2 : 1);
  while (warps > 1 && warps * per_warp > 64 * 1024) warps >>= 1;
  const size_t smem = warps * per_warp;
  if (smem > 200 * 1024) return LT_ERR_ARG;  // nvars * (p+1)^dim beyond one SM's shared memory
  auto fn = bulk ? k_face_interp<DIM, P1, true> : k_face_interp<DIM, P1, false>;
  LT_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0;
  LT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, warps * 32, smem));
  if (per_sm < 1) per_sm = 1;
  fn<<<t->num_sms * per_sm, warps * 32, smem, t->stream>>>(t->d_s, d_u, d_uf, nvars);
  return LT_OK;
}

template <int DIM>
static int launch_face_interp_d(Tree* t, const double* d_u, double* d_uf, int p, int nvars, int G) {
  switch (p) {
    case 0: return launch_face_interp_t<DIM, 1>(t, d_u, d_uf, nvars);
    case 1: return launch_face_interp_t<DIM, 2>(t, d_u, d_uf, nvars);
    case 2: return launch_face_interp_t<DIM, 3>(t, d_u, d_uf, nvars);
    case 3: return launch_face_interp_t<DIM, 4>(t, d_u, d_uf, nvars);
    case 4: return launch_face_interp_t<DIM, 5>(t, d_u, d_uf, nvars);
    case 5: return launch_face_interp_t<DIM, 6>(t, d_u, d_uf, nvars);
    case 6: return launch_face_interp_t<DIM, 7>(t, d_u, d_uf, nvars);
    case 7: return launch_face_interp_t<DIM, 8>(t, d_u, d_uf, nvars);
    default: return LT_ERR_ARG;
  }
  return LT_OK;
}

int launch_face_interp(Tree* t, const double* d_u, double* d_uf, int p, int nvars) {
  const int G = t->num_sms * 8;
  const int rc = t->g.dim == 2 ? launch_face_interp_d<2>(t, d_u, d_uf, p, nvars, G)
                               : launch_face_interp_d<3>(t, d_u, d_uf, p, nvars, G);
  if (rc != LT_OK) return rc;
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

int launch_map(Tree* t) {
  int G = grid_for(t, 8);
  LT_CUDA(cudaMemsetAsync(&t->d_s->map_bad, 0, sizeof(int), t->stream));  // (k_map reports through the status word)
  if (!t->have_old) {
    k_map_identity<<<G, 256, 0, t->stream>>>(t->d_s, t->map_src, t->map_kind);
  } else if (t->g.dim == 2) {
    k_map<2><<<G, 256, 0, t->stream>>>(t->g, t->keys[t->cur], t->keys[t->old], t->first[t->old], (int)t->n_old,
                                       t->d_s, t->map_src, t->map_kind);
  } else {
    k_map<3><<<G, 256, 0, t->stream>>>(t->g, t->keys[t->cur], t->keys[t->old], t->first[t->old], (int)t->n_old,
                                       t->d_s, t->map_src, t->map_kind);
  }
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

template <int DIM, int P1>
static int launch_transfer_t(Tree* t, const double* u_old, double* u_new, int nvars, int vec2, int64_t jb,
                             int64_t je) {
  using X = Xfer<DIM, P1>;
  int warps = 8;
  const size_t per_warp = (size_t)X::SMEM_DOUBLES * sizeof(double);
  while (warps > 1 && warps * per_warp > 96 * 1024) warps >>= 1;
  const size_t smem = warps * per_warp;
  auto fn = k_transfer<DIM, P1>;
  static int per_sm = 0;  // per instantiation: attribute and occupancy are queried once
  if (per_sm == 0) {
    LT_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    LT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, warps * 32, smem));
    if (per_sm < 1) per_sm = 1;
  }
  const int G = t->num_sms * per_sm;
  // sub-chunk = the power-of-two number of leaves closest below ~10 KB of solution, 1..32
  const size_t Bu = (size_t)nvars * X::N * sizeof(double);
  int sl_log2 = 0;
  while (sl_log2 < 5 && ((size_t)2 << sl_log2) * Bu <= 10240) ++sl_log2;
  LT_CUDA(cudaMemsetAsync(&t->d_s->ticket, 0, sizeof(unsigned), t->stream));
  fn<<<G, warps * 32, smem, t->stream>>>(t->d_s, t->map_src, t->map_kind, u_old, u_new, nvars, vec2, sl_log2,
                                         &t->d_s->ticket, jb, je);
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

template <int DIM>
static int launch_transfer_d(Tree* t, const double* u_old, double* u_new, int p, int nvars, int vec2, int64_t jb,
                             int64_t je) {
  switch (p) {
    case 0: return launch_transfer_t<DIM, 1>(t, u_old, u_new, nvars, vec2, jb, je);
    case 1: return launch_transfer_t<DIM, 2>(t, u_old, u_new, nvars, vec2, jb, je);
    case 2: return launch_transfer_t<DIM, 3>(t, u_old, u_new, nvars, vec2, jb, je);
    case 3: return launch_transfer_t<DIM, 4>(t, u_old, u_new, nvars, vec2, jb, je);
    case 4: return launch_transfer_t<DIM, 5>(t, u_old, u_new, nvars, vec2, jb, je);
    case 5: return launch_transfer_t<DIM, 6>(t, u_old, u_new, nvars, vec2, jb, je);
    case 6: return launch_transfer_t<DIM, 7>(t, u_old, u_new, nvars, vec2, jb, je);
    case 7: return launch_transfer_t<DIM, 8>(t, u_old, u_new, nvars, vec2, jb, je);
  }
  return LT_ERR_ARG;
}

int launch_transfer(Tree* t, const double* d_u_old, double* d_u_new, int p, int nvars, int64_t jb, int64_t je) {
  int N = 1;
  for (int a = 0; a < t->g.dim; ++a) N *= (p + 1);
  const int E = nvars * N;
  const int vec2 = (E % 2 == 0) && (((uintptr_t)d_u_old & 15) == 0) && (((uintptr_t)d_u_new & 15) == 0);
  return t->g.dim == 2 ? launch_transfer_d<2>(t, d_u_old, d_u_new, p, nvars, vec2, jb, je)
                       : launch_transfer_d<3>(t, d_u_old, d_u_new, p, nvars, vec2, jb, je);
}

// Slab boundaries for the pipelined host transfer: candidate k (k = 0..S) is moved forward to
// the next new leaf that does not sit inside a refined sibling group (children 1..nc-1 are
// written by the warp that owns child 0), so that slab [j_k, j_k+1) reads exactly the old
// leaves [o_k, o_k+1): the map is monotone and partitions T_old (Alg. 7).
__global__ void k_slab_bounds(const DevScalars* s, const int32_t* __restrict__ map_src,
                              const uint8_t* __restrict__ map_kind, int64_t n_old, int64_t slab, int S,
                              int64_t* __restrict__ out /* [S+1][2] */) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k > S) return;
  const int64_t n = s->n;
  int64_t j = (int64_t)k * slab;
  if (j > n || k == S) j = n;
  while (j < n && (map_kind[j] & 15) == 1 && (map_kind[j] >> 4) != 0) ++j;
  out[2 * k] = j;
  out[2 * k + 1] = j < n ? (int64_t)map_src[j] : n_old;
}

int launch_slab_bounds(Tree* t, int64_t n_old, int64_t slab, int S, int64_t* d_out) {
  k_slab_bounds<<<(S + 1 + 127) / 128, 128, 0, t->stream>>>(t->d_s, t->map_src, t->map_kind, n_old, slab, S, d_out);
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

}  // namespace lt
