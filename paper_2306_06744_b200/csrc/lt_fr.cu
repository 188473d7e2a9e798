// lt_fr.cu -- the flux-reconstruction pieces around the adaptation cycle (Eq. 1-6,
// and Alg. 8 step 3, PAPER.md:278 / :304) for sm_100a.  Product code: shares nothing with oracle/.
//
// Readings I-1..I-5 of DESIGN.md: compressible Euler, conserved variables (rho, rho v, E), gamma =
// 1.4; Rusanov common flux; Radau correction functions g_L = (-1)^(k+1) (P_(k+1) - P_k)/2,
// g_R(xi) = g_L(-xi); per axis
//   d f/dx = (2/dx) [ sum_j l_j'(z_i) f_j + g_L'(z_i)(F*_- - f(-1)) + g_R'(z_i)(F*_+ - f(1)) ]   (Eq. 4-5)
// with dx inferred from the element's level; SSP-RK3 of Eq. 6.
#include <math.h>
#include <string.h>

#include <mutex>
#include <vector>

#include "lt_internal.h"
#include "lt_euler.cuh"

namespace lt {

// c_fr[P1-1]: D[i][j] = l_j'(z_i) | l(-1)[j] | l(+1)[j] | g_L'(z_i) | g_R'(z_i) | D'
struct FrConst {
  double D[8][8];
  double lm[8], lp[8], gl[8], gr[8];
  double Dp[8][8];  // D'[i][j] = D[i][j] - gl[i] lm[j] - gr[i] lp[j] (k_fr_rhs)
};
__constant__ FrConst c_fr[8];

// Alg. 8 step 3: one thread per (slot, face point).  Own trace on an odd face = minus side.
template <int DIM>
__global__ void __launch_bounds__(256) k_common_flux(const DevScalars* s, const uint8_t* __restrict__ kind,
                                                     const double* __restrict__ uf, const double* unb,
                                                     double* fs, int Nf) {  // fs may be unb (in place)
  constexpr int NF = Dim<DIM>::NF, NV = DIM + 2;
  const int64_t total = (int64_t)s->n * NF * Nf;
  for (int64_t idx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; idx < total;
       idx += (int64_t)gridDim.x * blockDim.x) {
    const int64_t sl = idx / Nf;
    const int n = (int)(idx - sl * Nf);
    const int k = kind[sl] & 15;
    if (k != 1 && k != 2) continue;
    const int f = (int)(sl % NF), a = f >> 1;
    const size_t base = (size_t)sl * NV * Nf + n;
    double own[NV], nb[NV], FL[NV], FR[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      own[v] = uf[base + (size_t)v * Nf];
      nb[v] = unb[base + (size_t)v * Nf];
    }
    const double* L = (f & 1) ? own : nb;
    const double* R = (f & 1) ? nb : own;
    euler_flux<DIM>(a, L, FL);
    euler_flux<DIM>(a, R, FR);
    const double lam = fmax(wave_speed<DIM>(a, L), wave_speed<DIM>(a, R));
#pragma unroll
    for (int v = 0; v < NV; ++v) fs[base + (size_t)v * Nf] = 0.5 * (FL[v] + FR[v]) - 0.5 * lam * (R[v] - L[v]);
  }
}

// Eq. 2-5: one warp per element; u and the flux along the current axis live in shared memory.
// Lane l owns the entries i = l + 32 k of the element's [NV][N] block through the whole kernel: it
// loads them, accumulates their right-hand side (in registers when the block is at most 16 entries
// per lane), applies the RK stage and stores them.  For the derivative along axis a an entry (v, p)
// reads the P1 fluxes of ITS line -- the lanes of one line read the same words (broadcast), the
// lines of one instruction sit side by side -- which costs 1-2 shared-memory wavefronts per load.
// (Round 2 until here: one lane per LINE, R in shared memory.  The line starts are P1 or P1^2 doubles
// apart, so its loads and read-modify-writes took 8 wavefronts on two of the three axes: about 1080
// wavefronts per p = 3 element = 33 ms on 8.86 M elements, which was the measured time.  A padded
// and an index-rotated layout of that mapping were tried before and lost to occupancy / index
// arithmetic.)  Eq. 4-5 per axis are applied in the merged form
//   d_i = sum_j D'[i][j] f_j + g_L'(z_i) F*_- + g_R'(z_i) F*_+,   D' = D - g_L' (x) l(-1) - g_R' (x) l(+1)
// (identical algebra, 6 instead of 16 multiply-adds per entry for p = 3; D' is formed in long double).
template <int DIM, int P1>
struct FrShape {
  static constexpr int NV = DIM + 2;
  static constexpr int N = DIM == 2 ? P1 * P1 : P1 * P1 * P1;
  static constexpr int Nf = DIM == 2 ? P1 : P1 * P1;
  static constexpr int EV = NV * N;
  static constexpr int KN = (EV + 31) / 32;
  static constexpr bool REG = KN <= 16;  // a lane's accumulators in registers: k_fr_rhs, else k_fr_rhs_big
  // doubles of shared memory per warp: u | u_n | F | the 2 DIM face blocks, or u | F | R
  static constexpr int PER_WARP = REG ? 3 * EV + 2 * DIM * NV * Nf : 3 * EV;
  static constexpr int PER_WARP_EVEN = (PER_WARP + 1) & ~1;
};

// entry p of an element and axis a: index along the line, first point of the line, face-point index
template <int DIM, int P1>
__device__ __forceinline__ void line_of(int a, int p, int& idx, int& first, int& nt) {
  if (a == 0) {
    idx = p % P1;
    nt = p / P1;
    first = p - idx;
  } else if (a == 1) {
    const int q = p / P1;
    idx = q % P1;
    first = p - idx * P1;
    nt = DIM == 2 ? p % P1 : p % P1 + P1 * (q / P1);
  } else {
    idx = p / (P1 * P1);
    nt = p - idx * P1 * P1;
    first = nt;
  }
}

// 8-byte asynchronous copy global -> shared (LDGSTS): no alignment demand beyond the doubles' own
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)),
               "l"(gsrc)
               : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// The kernel for blocks of at most 16 entries per lane (2-D: every p; 3-D: p <= 3).  A warp keeps four
// buffers: u, u_n, the element's 2 DIM common-flux blocks, and F.  The three inputs of the warp's NEXT
// element are fetched by cp.async as soon as their buffer is dead -- u_n right after the accumulators
// are initialised, u after the last flux evaluation, the flux blocks after the last derivative -- so
// the DRAM latency hides behind the arithmetic and the stores of the current element (the synchronous
// version spent 9 of 14 issue-stall cycles waiting for global loads with 24 warps per SM).
// The stage of Eq. 6 is folded into the accumulator: acc = ca u_n + cb u_s, then acc -= cb dt (2/dx) d
// per axis (the same sum as ca u_n + cb (u_s + dt R) in another order).
template <int DIM, int P1>
__global__ void __launch_bounds__(256, 2) k_fr_rhs(Geo g, const uint64_t* __restrict__ keys, const DevScalars* s,
                                                   const double* u, const double* fs, double* R,
                                                   double w0, double w1, double w2, const double* un, double ca,
                                                   double cb, double dt, double* uf_out, int bulk) {
  // un == nullptr: R = right-hand side.  Otherwise the RK stage of Eq. 6 is applied on the fly:
  // R (= u_out) = ca * un + cb * (u + dt * rhs); u_out may be u or un (element-local access: a warp
  // prefetches only elements that it will write itself, later).
  // uf_out != nullptr (stage mode only): the traces of u_out at the face points (Alg. 8 step 1 of the
  // NEXT stage) are written as well, while u_out is still in shared memory; uf_out may be fs (an element
  // reads and writes only its own face slots).
  using S = FrShape<DIM, P1>;
  static_assert(S::REG, "k_fr_rhs_big handles the larger blocks");
  constexpr int NF = Dim<DIM>::NF, NV = S::NV, N = S::N, Nf = S::Nf, EV = S::EV, KN = S::KN;
  constexpr int E = NV * Nf, FB = NF * E;  // one face block, all face blocks of an element
  constexpr int CP = P1 + 2;               // operator table: row i = D'[i][0..P1-1] | g_L'(z_i) | g_R'(z_i)
  constexpr int CT = P1 * CP;              // then l(-1)[0..P1-1] | l(+1)[0..P1-1]
  // [warps]: f*[FB] | u[EV] | u_n[EV] | F[EV], every warp's part a multiple of 16 bytes (bulk-copy destinations)
  extern __shared__ __align__(16) double sm_gen[];
  __shared__ double sc[CT + 2 * P1];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  double* sfs = sm_gen + (size_t)w * S::PER_WARP_EVEN;
  double* su = sfs + FB;
  double* sn = su + EV;
  double* sF = sn + EV;
  {
    const FrConst& c = c_fr[P1 - 1];
    for (int t = threadIdx.x; t < CT + 2 * P1; t += blockDim.x) {
      if (t < CT) {
        const int i = t / CP, j = t - i * CP;
        sc[t] = j < P1 ? c.Dp[i][j] : (j == P1 ? c.gl[i] : c.gr[i]);
      } else {
        const int j = t - CT;
        sc[t] = j < P1 ? c.lm[j] : c.lp[j - P1];
      }
    }
  }
  __syncthreads();
  const int64_t n = s->n;
  const int64_t nw = (int64_t)gridDim.x * (blockDim.x >> 5);
  const bool stage = un != nullptr;
  // A block of the element is fetched by ONE cp.async.bulk of lane 0 (the copy engine: no LSU work, no
  // shared-memory store instructions) when its size is a multiple of 16 bytes and its array 16-byte aligned
  // (bulk bit 0: the flux blocks, always a multiple; bit 1: u and u_n, even EV only), else by 8-byte
  // cp.async of every lane.  The bulk copies of one element -- issued at different times -- all arrive on
  // the warp's mbarrier, whose phase completes when each has announced its bytes and delivered them.
  const bool bulk_f = (bulk & 1) != 0, bulk_u = (bulk & 2) != 0;
  __shared__ uint64_t bars[8];
  uint64_t* bar = &bars[w];
  uint32_t phase = 0;
  if (bulk && lane == 0) {
    mbar_init(bar, (bulk_f ? 1 : 0) + (bulk_u ? (stage ? 2 : 1) : 0));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncwarp();
  auto fetch = [&](double* dst, const double* src, int count, bool by_bulk) {
    if (by_bulk) {
      if (lane == 0) {
        mbar_arrive_expect_tx(bar, (uint32_t)count * 8u);
        bulk_g2s(dst, src, (uint32_t)count * 8u, bar);
      }
    } else {
      for (int i = lane; i < count; i += 32) cp_async8(dst + i, src + i);
    }
  };
  int64_t e = (int64_t)blockIdx.x * (blockDim.x >> 5) + w;
  if (e < n) {
    fetch(su, u + (size_t)e * EV, EV, bulk_u);
    if (stage) fetch(sn, un + (size_t)e * EV, EV, bulk_u);
    fetch(sfs, fs + (size_t)e * FB, FB, bulk_f);
  }
  cp_async_commit();
  for (; e < n; e += nw) {
    const int64_t e_next = e + nw;
    cp_async_wait_all();
    if (bulk) {
      while (!mbar_try_wait(bar, phase)) {
      }
      phase ^= 1;
    }
    __syncwarp();
    double acc[KN];
#pragma unroll
    for (int k = 0; k < KN; ++k) {
      const int i = lane + 32 * k;
      acc[k] = (stage && (EV % 32 == 0 || i < EV)) ? ca * sn[i] + cb * su[i] : 0.0;
    }
    if (stage && e_next < n) {  // (a lane overwrites only the entries of u_n that it has just read;
      if (bulk_u) __syncwarp();  //  the copy engine overwrites all of them: every lane has to be done)
      fetch(sn, un + (size_t)e_next * EV, EV, bulk_u);
      cp_async_commit();
    }
    const int level = key_level(keys[e]);
    const double inv2l = (double)(1ull << level);
    const double wgt = stage ? cb * dt : 1.0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
      const double scale = wgt * 2.0 * inv2l / (a == 0 ? w0 : (a == 1 ? w1 : w2));  // (cb dt) 2 / dx
      const int stride = a == 0 ? 1 : (a == 1 ? P1 : P1 * P1);
      __syncwarp();
      for (int p = lane; p < N; p += 32) {  // flux along a at every solution point
        double us[NV], Fp[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) us[v] = su[v * N + p];
        euler_flux<DIM>(a, us, Fp);
#pragma unroll
        for (int v = 0; v < NV; ++v) sF[v * N + p] = Fp[v];
      }
      __syncwarp();
      if (a == DIM - 1 && e_next < n) {  // u is dead: bring in the next element's
        fetch(su, u + (size_t)e_next * EV, EV, bulk_u);
        cp_async_commit();
      }
      const double* fsm = sfs + 2 * a * E;  // common flux on the - face: [v][nt]
      const double* fsp = fsm + E;          // and on the + face
#pragma unroll
      for (int k = 0; k < KN; ++k) {
        const int i = lane + 32 * k;
        if (EV % 32 == 0 || i < EV) {
          const int v = i / N, p = i - v * N;
          int idx, first, nt;
          line_of<DIM, P1>(a, p, idx, first, nt);
          const double* row = sc + idx * CP;
          const double* f = sF + v * N + first;
          double d = row[P1] * fsm[v * Nf + nt];
          d += row[P1 + 1] * fsp[v * Nf + nt];
#pragma unroll
          for (int j = 0; j < P1; ++j) d += row[j] * f[j * stride];
          acc[k] -= scale * d;
        }
      }
    }
    __syncwarp();
    if (e_next < n) {  // the flux blocks are dead
      fetch(sfs, fs + (size_t)e_next * FB, FB, bulk_f);
      cp_async_commit();
    }
    double* dst = R + (size_t)e * EV;
#pragma unroll
    for (int k = 0; k < KN; ++k) {
      const int i = lane + 32 * k;
      if (EV % 32 == 0 || i < EV) {
        __stcs(dst + i, acc[k]);
        if (uf_out != nullptr) sF[i] = acc[k];  // (sF is free after the last axis)
      }
    }
    if (uf_out != nullptr) {
      // Alg. 8 step 1 for the next stage: u_out at the face points.  Same entry -> line mapping; the
      // entry at position 0 of its line forms the trace on the - face, the one at position 1 the
      // trace on the + face (p = 0: the one point is both traces).
      __syncwarp();
      double* fd = uf_out + (size_t)e * FB;
#pragma unroll
      for (int a = 0; a < DIM; ++a) {
        const int stride = a == 0 ? 1 : (a == 1 ? P1 : P1 * P1);
#pragma unroll
        for (int k = 0; k < KN; ++k) {
          const int i = lane + 32 * k;
          if (EV % 32 == 0 || i < EV) {
            const int v = i / N, p = i - v * N;
            int idx, first, nt;
            line_of<DIM, P1>(a, p, idx, first, nt);
            if (P1 == 1) {
              __stcs(fd + (2 * a) * E + v * Nf + nt, acc[k]);
              __stcs(fd + (2 * a + 1) * E + v * Nf + nt, acc[k]);
            } else if (idx < 2) {
              const double* cf = sc + CT + idx * P1;
              const double* f = sF + v * N + first;
              double t = 0.0;
#pragma unroll
              for (int j = 0; j < P1; ++j) t += cf[j] * f[j * stride];
              __stcs(fd + (2 * a + idx) * E + v * Nf + nt, t);
            }
          }
        }
      }
    }
  }
}

// 3-D, p = 3 (the paper's order; 64 points, 320 entries): the element lives in REGISTERS.  With
// i = lane + 32 k the lane owns all five variables at its two points (x, y, z) = (lane & 3,
// (lane >> 2) & 3, (lane >> 4) + 2 h), h = 0, 1, so the point fluxes need no shared memory at all, and
// a line along x / y is four lanes that differ in lane bits 0-1 / 2-3, a line along z two lanes
// (bit 4) times the two points of each: the P1 fluxes of a line are exchanged by warp shuffles.  The
// generic kernel above is bound by the shared-memory data pipe (ncu: l1tex data-pipe wavefronts at
// 93-96 % of peak, 670 per element without and 900 with the traces, every 64-bit access of a warp
// costing two); here only the six common-flux blocks of the element go through shared memory (prefetched
// by cp.async), u and u_n of the warp's NEXT element are loaded into registers when the tail of the
// current one begins, and the traces of u_out are reduced over the line's lanes by shuffles.
// BULK: the element's six flux blocks are one contiguous run of 3840 bytes, fetched by ONE cp.async.bulk of
// the warp's lane 0 onto the warp's own mbarrier instead of 15 LDGSTS per lane (BULK = false when the
// caller's flux array is not 16-byte aligned).
template <bool BULK>
__global__ void __launch_bounds__(256, 2) k_fr_rhs_p3(const uint64_t* __restrict__ keys, const DevScalars* s,
                                                      const double* u, const double* fs, double* R, double w0,
                                                      double w1, double w2, const double* un, double ca, double cb,
                                                      double dt, double* uf_out) {
  constexpr int DIM = 3, P1 = 4, NV = 5, N = 64, Nf = 16, EV = 320, KN = 10, E = NV * Nf, FB = 6 * E;
  constexpr int CP = P1 + 2, CT = P1 * CP;
  constexpr unsigned FULL = 0xffffffffu;
  extern __shared__ __align__(128) double sm_p3[];  // [warps]: f*[FB]
  __shared__ double sc[CT + 2 * P1];  // D'[i][0..3] | g_L'(z_i) | g_R'(z_i) per row, then l(-1), l(+1)
  __shared__ uint64_t bars[8];        // one mbarrier per warp (BULK)
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  double* sfs = sm_p3 + (size_t)w * FB;
  uint64_t* bar = &bars[w];
  uint32_t phase = 0;
  if (BULK && lane == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  // the flux blocks of element `el` -> this warp's buffer (all lanes call it; the buffer must be dead)
  auto fetch_fluxes = [&](int64_t el) {
    if (BULK) {
      if (lane == 0) {
        mbar_arrive_expect_tx(bar, FB * 8);
        bulk_g2s(sfs, fs + (size_t)el * FB, FB * 8, bar);
      }
    } else {
      for (int i = lane; i < FB; i += 32) cp_async8(sfs + i, fs + (size_t)el * FB + i);
    }
  };
  {
    const FrConst& c = c_fr[P1 - 1];
    for (int t = threadIdx.x; t < CT + 2 * P1; t += blockDim.x) {
      if (t < CT) {
        const int i = t / CP, j = t - i * CP;
        sc[t] = j < P1 ? c.Dp[i][j] : (j == P1 ? c.gl[i] : c.gr[i]);
      } else {
        const int j = t - CT;
        sc[t] = j < P1 ? c.lm[j] : c.lp[j - P1];
      }
    }
  }
  __syncthreads();
  const int x = lane & 3, y = (lane >> 2) & 3, z0 = lane >> 4;
  const int64_t n = s->n;
  const int64_t nw = (int64_t)gridDim.x * (blockDim.x >> 5);
  const bool stage = un != nullptr;
  int64_t e = (int64_t)blockIdx.x * (blockDim.x >> 5) + w;
  double nu[KN], nn[KN];  // u and u_n of the element about to be processed
  if (e < n) {
    fetch_fluxes(e);
#pragma unroll
    for (int k = 0; k < KN; ++k) {
      nu[k] = __ldcs(u + (size_t)e * EV + lane + 32 * k);
      nn[k] = stage ? __ldcs(un + (size_t)e * EV + lane + 32 * k) : 0.0;
    }
  }
  cp_async_commit();
  for (; e < n; e += nw) {
    const int64_t e_next = e + nw;
    double uo[KN], acc[KN];
#pragma unroll
    for (int k = 0; k < KN; ++k) {
      uo[k] = nu[k];
      acc[k] = stage ? ca * nn[k] + cb * nu[k] : 0.0;
    }
    if (BULK) {
      while (!mbar_try_wait(bar, phase)) {
      }
      phase ^= 1;
    } else {
      cp_async_wait_all();
      __syncwarp();
    }
    const int level = key_level(keys[e]);
    const double inv2l = (double)(1ull << level);
    const double wgt = stage ? cb * dt : 1.0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
      const double scale = wgt * 2.0 * inv2l / (a == 0 ? w0 : (a == 1 ? w1 : w2));  // (cb dt) 2 / dx
      double F[KN];  // flux along a at the lane's two points: F[2 v + h]
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        double us[NV], Fp[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) us[v] = uo[2 * v + h];
        euler_flux<DIM>(a, us, Fp);
#pragma unroll
        for (int v = 0; v < NV; ++v) F[2 * v + h] = Fp[v];
      }
      const double* fsm = sfs + 2 * a * E;  // common flux on the - face: [v][nt]
      const double* fsp = fsm + E;          // and on the + face
      if (a < 2) {
        // the line = the four lanes that differ in bits sh, sh + 1; this lane is position idx
        const int idx = a == 0 ? x : y, sh = a == 0 ? 0 : 2;
        const double* row = sc + idx * CP;
        double cD[P1];
#pragma unroll
        for (int m = 0; m < P1; ++m) cD[m] = row[idx ^ m];
        const double cl = row[P1], cr = row[P1 + 1];
        // face point of the line: a = 0: y + 4 z, a = 1: x + 4 z (z = z0 + 2 h)
        const int nt0 = a == 0 ? (lane >> 2) : x + 4 * z0;
#pragma unroll
        for (int k = 0; k < KN; ++k) {
          const int v = k >> 1, h = k & 1, nt = nt0 + 8 * h;
          double d = cl * fsm[v * Nf + nt];
          d += cr * fsp[v * Nf + nt];
          d += cD[0] * F[k];
#pragma unroll
          for (int m = 1; m < P1; ++m) d += cD[m] * __shfl_xor_sync(FULL, F[k], m << sh);
          acc[k] -= scale * d;
        }
      } else {
        // the line = this lane and lane ^ 16, two points each: z = z0 + 2 h
        double cO[2][2], cP[2][2], cl[2], cr[2];  // [h of the entry][h of the source]: own / partner
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const double* row = sc + (z0 + 2 * h) * CP;
#pragma unroll
          for (int hh = 0; hh < 2; ++hh) {
            cO[h][hh] = row[z0 + 2 * hh];
            cP[h][hh] = row[(z0 ^ 1) + 2 * hh];
          }
          cl[h] = row[P1];
          cr[h] = row[P1 + 1];
        }
        const int nt = lane & 15;  // x + 4 y
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const double p0 = __shfl_xor_sync(FULL, F[2 * v], 16), p1 = __shfl_xor_sync(FULL, F[2 * v + 1], 16);
          const double fm = fsm[v * Nf + nt], fp = fsp[v * Nf + nt];
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            double d = cl[h] * fm;
            d += cr[h] * fp;
            d += cO[h][0] * F[2 * v];
            d += cO[h][1] * F[2 * v + 1];
            d += cP[h][0] * p0;
            d += cP[h][1] * p1;
            acc[2 * v + h] -= scale * d;
          }
        }
      }
    }
    __syncwarp();
    if (e_next < n) {  // the flux blocks are dead: the next element's; its u and u_n go to registers
      fetch_fluxes(e_next);
#pragma unroll
      for (int k = 0; k < KN; ++k) {
        nu[k] = __ldcs(u + (size_t)e_next * EV + lane + 32 * k);
        nn[k] = stage ? __ldcs(un + (size_t)e_next * EV + lane + 32 * k) : 0.0;
      }
    }
    cp_async_commit();
    double* dst = R + (size_t)e * EV;
#pragma unroll
    for (int k = 0; k < KN; ++k) __stcs(dst + lane + 32 * k, acc[k]);
    if (uf_out != nullptr) {
      // Alg. 8 step 1 for the next stage: u_out at the face points.  Every lane weighs its value with
      // l(-1) and l(+1) at its position; the sums over the line are formed by a butterfly in which half
      // of the lanes collect the - trace and the other half the + trace.
      double* fd = uf_out + (size_t)e * FB;
      const double* lm = sc + CT;
      const double* lp = lm + P1;
#pragma unroll
      for (int a = 0; a < 2; ++a) {
        const int idx = a == 0 ? x : y, sh = a == 0 ? 0 : 2;
        const double wm = lm[idx], wp = lp[idx];
        const bool odd = idx & 1;
        const int nt0 = a == 0 ? (lane >> 2) : x + 4 * z0;
#pragma unroll
        for (int k = 0; k < KN; ++k) {
          const int v = k >> 1, h = k & 1, nt = nt0 + 8 * h;
          const double pm = wm * acc[k], pp = wp * acc[k];
          double r = (odd ? pp : pm) + __shfl_xor_sync(FULL, odd ? pm : pp, 1 << sh);
          r += __shfl_xor_sync(FULL, r, 2 << sh);
          if (idx < 2) __stcs(fd + (2 * a + idx) * E + v * Nf + nt, r);
        }
      }
      {
        const double wm0 = lm[z0], wm1 = lm[z0 + 2], wp0 = lp[z0], wp1 = lp[z0 + 2];
        const int nt = lane & 15;
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          const double pm = wm0 * acc[2 * v] + wm1 * acc[2 * v + 1];
          const double pp = wp0 * acc[2 * v] + wp1 * acc[2 * v + 1];
          const double r = (z0 ? pp : pm) + __shfl_xor_sync(FULL, z0 ? pm : pp, 16);
          __stcs(fd + (4 + z0) * E + v * Nf + nt, r);
        }
      }
    }
  }
}


// 3-D p = 2 -- the order of the paper's own 3-D runs (Table 5) -- register-resident like
// k_fr_rhs_p3: lane i < 27 owns solution point i = x + 3 (y + 3 z) with all five variables, so the point
// fluxes need no shared memory; a line along axis a is the three lanes base + j * 3^a, whose fluxes are
// exchanged by warp shuffles (lanes 27-31 shuffle along and store nothing).  Only the six flux blocks
// (2160 bytes, one cp.async.bulk when BULK) go through shared memory; u and u_n of the warp's next element
// are loaded into registers when the tail of the current one begins.
template <bool BULK>
__global__ void __launch_bounds__(256, 2) k_fr_rhs_p2(const uint64_t* __restrict__ keys, const DevScalars* s,
                                                      const double* u, const double* fs, double* R, double w0,
                                                      double w1, double w2, const double* un, double ca, double cb,
                                                      double dt, double* uf_out) {
  constexpr int DIM = 3, P1 = 3, NV = 5, N = 27, Nf = 9, EV = 135, E = NV * Nf, FB = 6 * E;
  constexpr int CP = P1 + 2, CT = P1 * CP;
  constexpr unsigned FULL = 0xffffffffu;
  extern __shared__ __align__(128) double sm_p2[];  // [warps]: f*[FB]
  __shared__ double sc[CT + 2 * P1];  // D'[i][0..2] | g_L'(z_i) | g_R'(z_i) per row, then l(-1), l(+1)
  __shared__ uint64_t bars[8];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  double* sfs = sm_p2 + (size_t)w * FB;
  uint64_t* bar = &bars[w];
  uint32_t phase = 0;
  if (BULK && lane == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  auto fetch_fluxes = [&](int64_t el) {
    if (BULK) {
      if (lane == 0) {
        mbar_arrive_expect_tx(bar, FB * 8);
        bulk_g2s(sfs, fs + (size_t)el * FB, FB * 8, bar);
      }
    } else {
      for (int i = lane; i < FB; i += 32) cp_async8(sfs + i, fs + (size_t)el * FB + i);
    }
  };
  {
    const FrConst& c = c_fr[P1 - 1];
    for (int t = threadIdx.x; t < CT + 2 * P1; t += blockDim.x) {
      if (t < CT) {
        const int i = t / CP, j = t - i * CP;
        sc[t] = j < P1 ? c.Dp[i][j] : (j == P1 ? c.gl[i] : c.gr[i]);
      } else {
        const int j = t - CT;
        sc[t] = j < P1 ? c.lm[j] : c.lp[j - P1];
      }
    }
  }
  __syncthreads();
  const bool live = lane < N;
  const int pi = live ? lane : 0;  // (the idle lanes mirror point 0)
  const int cx = pi % 3, cy = (pi / 3) % 3, cz = pi / 9;
  const int64_t n = s->n;
  const int64_t nw = (int64_t)gridDim.x * (blockDim.x >> 5);
  const bool stage = un != nullptr;
  int64_t e = (int64_t)blockIdx.x * (blockDim.x >> 5) + w;
  double nu[NV], nn[NV];  // u and u_n of the element about to be processed
  if (e < n) {
    fetch_fluxes(e);
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      nu[v] = __ldcs(u + (size_t)e * EV + v * N + pi);
      nn[v] = stage ? __ldcs(un + (size_t)e * EV + v * N + pi) : 0.0;
    }
  }
  cp_async_commit();
  for (; e < n; e += nw) {
    const int64_t e_next = e + nw;
    double uo[NV], acc[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      uo[v] = nu[v];
      acc[v] = stage ? ca * nn[v] + cb * nu[v] : 0.0;
    }
    if (BULK) {
      while (!mbar_try_wait(bar, phase)) {
      }
      phase ^= 1;
    } else {
      cp_async_wait_all();
      __syncwarp();
    }
    const int level = key_level(keys[e]);
    const double inv2l = (double)(1ull << level);
    const double wgt = stage ? cb * dt : 1.0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
      const double scale = wgt * 2.0 * inv2l / (a == 0 ? w0 : (a == 1 ? w1 : w2));  // (cb dt) 2 / dx
      double F[NV];
      euler_flux<DIM>(a, uo, F);
      const int stride = a == 0 ? 1 : (a == 1 ? 3 : 9);
      const int idx = a == 0 ? cx : (a == 1 ? cy : cz);
      const int base = pi - idx * stride;
      const int nt = a == 0 ? cy + 3 * cz : (a == 1 ? cx + 3 * cz : cx + 3 * cy);  // lower tangential axis fastest
      const double* row = sc + idx * CP;
      const double* fsm = sfs + 2 * a * E;  // common flux on the - face: [v][nt]
      const double* fsp = fsm + E;          // and on the + face
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        double d = row[P1] * fsm[v * Nf + nt];
        d += row[P1 + 1] * fsp[v * Nf + nt];
#pragma unroll
        for (int j = 0; j < P1; ++j) d += row[j] * __shfl_sync(FULL, F[v], base + j * stride);
        acc[v] -= scale * d;
      }
    }
    __syncwarp();
    if (e_next < n) {  // the flux blocks are dead: the next element's; its u and u_n go to registers
      fetch_fluxes(e_next);
#pragma unroll
      for (int v = 0; v < NV; ++v) {
        nu[v] = __ldcs(u + (size_t)e_next * EV + v * N + pi);
        nn[v] = stage ? __ldcs(un + (size_t)e_next * EV + v * N + pi) : 0.0;
      }
    }
    cp_async_commit();
    if (live) {
      double* dst = R + (size_t)e * EV;
#pragma unroll
      for (int v = 0; v < NV; ++v) __stcs(dst + v * N + pi, acc[v]);
    }
    if (uf_out != nullptr) {
      // Alg. 8 step 1 for the next stage: u_out at the face points; the lane at position 0 of its line
      // forms the trace on the - face, the one at position 1 the trace on the + face
      double* fd = uf_out + (size_t)e * FB;
      const double* lm = sc + CT;
      const double* lp = lm + P1;
#pragma unroll
      for (int a = 0; a < DIM; ++a) {
        const int stride = a == 0 ? 1 : (a == 1 ? 3 : 9);
        const int idx = a == 0 ? cx : (a == 1 ? cy : cz);
        const int base = pi - idx * stride;
        const int nt = a == 0 ? cy + 3 * cz : (a == 1 ? cx + 3 * cz : cx + 3 * cy);
        const double* cf = idx == 0 ? lm : lp;
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          double t = 0.0;
#pragma unroll
          for (int j = 0; j < P1; ++j) t += cf[j] * __shfl_sync(FULL, acc[v], base + j * stride);
          if (live && idx < 2) __stcs(fd + (2 * a + idx) * E + v * Nf + nt, t);
        }
      }
    }
  }
}

// The same for larger blocks (3-D, p >= 4): right-hand side accumulated in shared memory, synchronous loads.
template <int DIM, int P1>
__global__ void __launch_bounds__(256) k_fr_rhs_big(Geo g, const uint64_t* __restrict__ keys, const DevScalars* s,
                                                    const double* u, const double* fs, double* R,
                                                    double w0, double w1, double w2, const double* un, double ca,
                                                    double cb, double dt, double* uf_out, int /*bulk: unused*/) {
  using S = FrShape<DIM, P1>;
  constexpr int NF = Dim<DIM>::NF, NV = S::NV, N = S::N, Nf = S::Nf, EV = S::EV;
  constexpr int E = NV * Nf;
  constexpr int CP = P1 + 2, CT = P1 * CP;
  extern __shared__ double sm_all[];  // [warps]: u[EV] | F[EV] | R[EV]
  __shared__ double sc[CT + 2 * P1];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  double* su = sm_all + (size_t)w * S::PER_WARP;
  double* sF = su + EV;
  double* sR = sF + EV;
  {
    const FrConst& c = c_fr[P1 - 1];
    for (int t = threadIdx.x; t < CT + 2 * P1; t += blockDim.x) {
      if (t < CT) {
        const int i = t / CP, j = t - i * CP;
        sc[t] = j < P1 ? c.Dp[i][j] : (j == P1 ? c.gl[i] : c.gr[i]);
      } else {
        const int j = t - CT;
        sc[t] = j < P1 ? c.lm[j] : c.lp[j - P1];
      }
    }
  }
  __syncthreads();
  const int64_t n = s->n;
  const int64_t nw = (int64_t)gridDim.x * (blockDim.x >> 5);
  for (int64_t e = (int64_t)blockIdx.x * (blockDim.x >> 5) + w; e < n; e += nw) {
    __syncwarp();
    const double* src = u + (size_t)e * EV;
    for (int i = lane; i < EV; i += 32) {
      su[i] = __ldcs(src + i);
      sR[i] = 0.0;
    }
    const int level = key_level(keys[e]);
    const double inv2l = (double)(1ull << level);
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
      const double scale = 2.0 * inv2l / (a == 0 ? w0 : (a == 1 ? w1 : w2));  // 2 / dx
      const int stride = a == 0 ? 1 : (a == 1 ? P1 : P1 * P1);
      __syncwarp();
      for (int p = lane; p < N; p += 32) {
        double us[NV], Fp[NV];
#pragma unroll
        for (int v = 0; v < NV; ++v) us[v] = su[v * N + p];
        euler_flux<DIM>(a, us, Fp);
#pragma unroll
        for (int v = 0; v < NV; ++v) sF[v * N + p] = Fp[v];
      }
      __syncwarp();
      const double* fsm = fs + ((size_t)e * NF + 2 * a) * E;
      const double* fsp = fsm + E;
      for (int i = lane; i < EV; i += 32) {
        const int v = i / N, p = i - v * N;
        int idx, first, nt;
        line_of<DIM, P1>(a, p, idx, first, nt);
        const double* row = sc + idx * CP;
        const double* f = sF + v * N + first;
        double d = row[P1] * fsm[v * Nf + nt];
        d += row[P1 + 1] * fsp[v * Nf + nt];
#pragma unroll
        for (int j = 0; j < P1; ++j) d += row[j] * f[j * stride];
        sR[i] -= scale * d;
      }
    }
    __syncwarp();
    double* dst = R + (size_t)e * EV;
    if (un == nullptr) {
      for (int i = lane; i < EV; i += 32) __stcs(dst + i, sR[i]);
    } else {
      const double* gn = un + (size_t)e * EV;
      for (int i = lane; i < EV; i += 32) {
        const double o = ca * gn[i] + cb * (su[i] + dt * sR[i]);
        dst[i] = o;
        sF[i] = o;
      }
      if (uf_out != nullptr) {
        __syncwarp();
        double* fd = uf_out + (size_t)e * NF * E;
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
          const int stride = a == 0 ? 1 : (a == 1 ? P1 : P1 * P1);
          for (int i = lane; i < EV; i += 32) {
            const int v = i / N, p = i - v * N;
            int idx, first, nt;
            line_of<DIM, P1>(a, p, idx, first, nt);
            if (idx < 2) {
              const double* cf = sc + CT + idx * P1;
              const double* f = sF + v * N + first;
              double t = 0.0;
#pragma unroll
              for (int j = 0; j < P1; ++j) t += cf[j] * f[j * stride];
              __stcs(fd + (2 * a + idx) * E + v * Nf + nt, t);
            }
          }
        }
      }
    }
  }
}

// Eq. 6: u_out = a u_n + b (u_s + dt R), (a, b) = (0, 1), (3/4, 1/4), (1/3, 2/3) for stages 1, 2, 3.
__global__ void __launch_bounds__(256) k_rk_update(int64_t n, double a, double b, double dt,
                                                   const double* un, const double* us,
                                                   const double* __restrict__ R, double* out) {  // out may be un / us
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    out[i] = a * un[i] + b * (us[i] + dt * R[i]);
}

// ---------------------------------------------------------------- operators (host, long double)
static long double legendre_ld(int n, long double x, long double* dp) {
  long double pm = 1.0L, pc = n == 0 ? 1.0L : x;
  for (int k = 1; k < n; ++k) {
    const long double pn = ((2 * k + 1) * x * pc - k * pm) / (k + 1);
    pm = pc;
    pc = pn;
  }
  if (dp) *dp = n == 0 ? 0.0L : n * (x * pc - (n == 1 ? 1.0L : pm)) / (x * x - 1.0L);
  return pc;
}

int build_fr_operators(Tree* t, int p) {
  // as build_operators: per device, uploaded to the current device, serialised across host threads
  static std::mutex mu;
  static bool uploaded[64][8];
  int rc = check_device(t);
  if (rc != LT_OK) return rc;
  if (t->device < 0 || t->device >= 64) return LT_ERR_ARG;
  std::lock_guard<std::mutex> lk(mu);
  const int dev = t->device;
  if (uploaded[dev][p]) return LT_OK;
  const int P1 = p + 1;
  // Gauss-Legendre nodes by Newton iteration on P_n
  std::vector<long double> z(P1);
  const long double pi = acosl(-1.0L);
  for (int i = 0; i < P1; ++i) {
    long double x = -cosl(pi * (i + 0.75L) / (P1 + 0.5L));
    for (int it = 0; it < 80; ++it) {
      long double dp;
      const long double pv = legendre_ld(P1, x, &dp);
      const long double dx = pv / dp;
      x -= dx;
      if (fabsl(dx) < 1e-20L) break;
    }
    z[i] = x;
  }
  FrConst h;
  memset(&h, 0, sizeof(h));
  long double Dl[8][8], lml[8], lpl[8], gll[8], grl[8];
  const long double sgn = ((p + 1) % 2) ? -1.0L : 1.0L;  // (-1)^(k+1), k = p
  for (int i = 0; i < P1; ++i) {
    for (int j = 0; j < P1; ++j) {  // l_j'(z_i)
      long double sacc = 0.0L;
      for (int m = 0; m < P1; ++m) {
        if (m == j) continue;
        long double tt = 1.0L / (z[j] - z[m]);
        for (int k = 0; k < P1; ++k)
          if (k != j && k != m) tt *= (z[i] - z[k]) / (z[j] - z[k]);
        sacc += tt;
      }
      Dl[i][j] = sacc;
      h.D[i][j] = (double)sacc;
    }
    long double lm = 1.0L, lp = 1.0L;
    for (int k = 0; k < P1; ++k)
      if (k != i) {
        lm *= (-1.0L - z[k]) / (z[i] - z[k]);
        lp *= (1.0L - z[k]) / (z[i] - z[k]);
      }
    lml[i] = lm;
    lpl[i] = lp;
    h.lm[i] = (double)lm;
    h.lp[i] = (double)lp;
    long double d1, d0, e1, e0;
    legendre_ld(p + 1, z[i], &d1);
    legendre_ld(p, z[i], &d0);
    legendre_ld(p + 1, -z[i], &e1);
    legendre_ld(p, -z[i], &e0);
    gll[i] = 0.5L * sgn * (d1 - d0);
    grl[i] = -0.5L * sgn * (e1 - e0);
    h.gl[i] = (double)gll[i];
    h.gr[i] = (double)grl[i];
  }
  for (int i = 0; i < P1; ++i)
    for (int j = 0; j < P1; ++j) h.Dp[i][j] = (double)(Dl[i][j] - gll[i] * lml[j] - grl[i] * lpl[j]);
  LT_CUDA(cudaMemcpyToSymbol(c_fr, &h, sizeof(h), (size_t)p * sizeof(FrConst), cudaMemcpyHostToDevice));
  uploaded[dev][p] = true;
  return LT_OK;
}

// ---------------------------------------------------------------- launchers
int launch_common_flux(Tree* t, const double* d_uf, const double* d_unb, double* d_fs, int p) {
  int Nf = 1;
  for (int a = 1; a < t->g.dim; ++a) Nf *= p + 1;
  const int G = t->num_sms * 8;
  if (t->g.dim == 2) k_common_flux<2><<<G, 256, 0, t->stream>>>(t->d_s, t->kind, d_uf, d_unb, d_fs, Nf);
  else k_common_flux<3><<<G, 256, 0, t->stream>>>(t->d_s, t->kind, d_uf, d_unb, d_fs, Nf);
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

template <int DIM, int P1, bool REG>
struct fr_rhs_kernel {
  static auto get() { return k_fr_rhs<DIM, P1>; }
};
template <int DIM, int P1>
struct fr_rhs_kernel<DIM, P1, false> {
  static auto get() { return k_fr_rhs_big<DIM, P1>; }
};

template <int DIM, int P1>
static int launch_fr_rhs_t(Tree* t, const double* d_u, const double* d_fs, double* d_R, const double* d_un, double ca,
                           double cb, double dt, double* d_uf_out) {
  using S = FrShape<DIM, P1>;
  // width of a root cube along each axis (a single cube: the domain width)
  const double w0 = (t->domain[DIM] - t->domain[0]) / t->g.nroot[0];
  const double w1 = (t->domain[DIM + 1] - t->domain[1]) / t->g.nroot[1];
  const double w2 = DIM == 3 ? (t->domain[DIM + 2] - t->domain[2]) / t->g.nroot[2] : 1.0;
  if (DIM == 3 && P1 == 4) {
    const size_t smem3 = (size_t)8 * 6 * S::NV * S::Nf * sizeof(double);
    static int per_sm3 = 0;
    if (per_sm3 == 0) {
      int q = 0;
      LT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&q, k_fr_rhs_p3<true>, 256, smem3));
      per_sm3 = q < 1 ? 1 : q;
    }
    if ((reinterpret_cast<uintptr_t>(d_fs) & 15) == 0)  // cp.async.bulk needs 16-byte aligned addresses
      k_fr_rhs_p3<true><<<t->num_sms * per_sm3, 256, smem3, t->stream>>>(t->keys[t->cur], t->d_s, d_u, d_fs, d_R, w0,
                                                                         w1, w2, d_un, ca, cb, dt, d_uf_out);
    else
      k_fr_rhs_p3<false><<<t->num_sms * per_sm3, 256, smem3, t->stream>>>(t->keys[t->cur], t->d_s, d_u, d_fs, d_R, w0,
                                                                          w1, w2, d_un, ca, cb, dt, d_uf_out);
    return LT_OK;
  }
  if (DIM == 3 && P1 == 3) {
    const size_t smem2 = (size_t)8 * 6 * S::NV * S::Nf * sizeof(double);
    static int per_sm2 = 0;
    if (per_sm2 == 0) {
      int q = 0;
      LT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&q, k_fr_rhs_p2<true>, 256, smem2));
      per_sm2 = q < 1 ? 1 : q;
    }
    if ((reinterpret_cast<uintptr_t>(d_fs) & 15) == 0)  // cp.async.bulk needs 16-byte aligned addresses
      k_fr_rhs_p2<true><<<t->num_sms * per_sm2, 256, smem2, t->stream>>>(t->keys[t->cur], t->d_s, d_u, d_fs, d_R, w0,
                                                                         w1, w2, d_un, ca, cb, dt, d_uf_out);
    else
      k_fr_rhs_p2<false><<<t->num_sms * per_sm2, 256, smem2, t->stream>>>(t->keys[t->cur], t->d_s, d_u, d_fs, d_R, w0,
                                                                          w1, w2, d_un, ca, cb, dt, d_uf_out);
    return LT_OK;
  }
  int warps = 8;
  const size_t per_warp = (size_t)S::PER_WARP_EVEN * sizeof(double);
  while (warps > 1 && warps * per_warp > 96 * 1024) warps >>= 1;
  const size_t smem = warps * per_warp;
  // which inputs the copy engine may fetch (16-byte multiples at 16-byte aligned addresses): bit 0 the flux
  // blocks, bit 1 u and u_n
  const auto al16 = [](const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15) == 0; };
  const int bulk = (al16(d_fs) ? 1 : 0) | ((S::EV % 2 == 0 && al16(d_u) && (d_un == nullptr || al16(d_un))) ? 2 : 0);
  auto fn = fr_rhs_kernel<DIM, P1, S::REG>::get();
  LT_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0;
  LT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, warps * 32, smem));
  if (per_sm < 1) per_sm = 1;
  fn<<<t->num_sms * per_sm, warps * 32, smem, t->stream>>>(t->g, t->keys[t->cur], t->d_s, d_u, d_fs, d_R, w0, w1,
                                                            w2, d_un, ca, cb, dt, d_uf_out, bulk);
  return LT_OK;
}

template <int DIM>
static int launch_fr_rhs_d(Tree* t, const double* d_u, const double* d_fs, double* d_R, int p, const double* d_un,
                           double ca, double cb, double dt, double* d_uf_out) {
  switch (p) {
    case 0: return launch_fr_rhs_t<DIM, 1>(t, d_u, d_fs, d_R, d_un, ca, cb, dt, d_uf_out);
    case 1: return launch_fr_rhs_t<DIM, 2>(t, d_u, d_fs, d_R, d_un, ca, cb, dt, d_uf_out);
    case 2: return launch_fr_rhs_t<DIM, 3>(t, d_u, d_fs, d_R, d_un, ca, cb, dt, d_uf_out);
    case 3: return launch_fr_rhs_t<DIM, 4>(t, d_u, d_fs, d_R, d_un, ca, cb, dt, d_uf_out);
    case 4: return launch_fr_rhs_t<DIM, 5>(t, d_u, d_fs, d_R, d_un, ca, cb, dt, d_uf_out);
    case 5: return launch_fr_rhs_t<DIM, 6>(t, d_u, d_fs, d_R, d_un, ca, cb, dt, d_uf_out);
    case 6: return launch_fr_rhs_t<DIM, 7>(t, d_u, d_fs, d_R, d_un, ca, cb, dt, d_uf_out);
    case 7: return launch_fr_rhs_t<DIM, 8>(t, d_u, d_fs, d_R, d_un, ca, cb, dt, d_uf_out);
  }
  return LT_ERR_ARG;
}

int launch_fr_rhs(Tree* t, const double* d_u, const double* d_fs, double* d_R, int p, const double* d_un, double ca,
                  double cb, double dt, double* d_uf_out) {
  const int rc = t->g.dim == 2 ? launch_fr_rhs_d<2>(t, d_u, d_fs, d_R, p, d_un, ca, cb, dt, d_uf_out)
                               : launch_fr_rhs_d<3>(t, d_u, d_fs, d_R, p, d_un, ca, cb, dt, d_uf_out);
  if (rc != LT_OK) return rc;
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

int launch_rk_update(Tree* t, int64_t n, double a, double b, double dt, const double* un, const double* us,
                     const double* R, double* out) {
  k_rk_update<<<t->num_sms * 8, 256, 0, t->stream>>>(n, a, b, dt, un, us, R, out);
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

}  // namespace lt
