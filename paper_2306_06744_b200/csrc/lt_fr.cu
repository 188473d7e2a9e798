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

// c_fr[P1-1]: D[i][j] = l_j'(z_i) | l(-1)[j] | l(+1)[j] | g_L'(z_i) | g_R'(z_i)
struct FrConst {
  double D[8][8];
  double lm[8], lp[8], gl[8], gr[8];
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

// Eq. 2-5: one warp per element.  u, the flux along the current axis and the accumulated R of the
// element live in shared memory; the common fluxes come from the element's own face slots.
template <int DIM, int P1>
__global__ void __launch_bounds__(256) k_fr_rhs(Geo g, const uint64_t* __restrict__ keys, const DevScalars* s,
                                                const double* u, const double* fs, double* R,
                                                double w0, double w1, double w2, const double* un, double ca,
                                                double cb, double dt, double* uf_out) {
  // un == nullptr: R = right-hand side.  Otherwise the RK stage of Eq. 6 is applied on the fly:
  // R (= u_out) = ca * un + cb * (u + dt * rhs); u_out may be u or un (element-local access).
  // uf_out != nullptr (stage mode only): the traces of u_out at the face points (Alg. 8 step 1 of the
  // NEXT stage) are written as well, while u_out is still in shared memory; uf_out may be fs (an element
  // reads and writes only its own face slots).
  // (A layout with padded x-lines and 1 / rho, p stored once per point was tried: it removes the bank
  // conflicts but needs 10.9 instead of 7.7 KB of shared memory per warp, i.e. 16 instead of 24 resident
  // warps per SM, and the kernel is latency-bound: 35.6 instead of 25.2 ms per stage on 8.86 M elements.
  // Rotating the x / y indices by iz instead (conflict-free on all three axes at no cost in shared memory)
  // was tried as well: 27.1 ms -- the extra index arithmetic costs more than the 4-way conflicts.)
  constexpr int NF = Dim<DIM>::NF, NV = DIM + 2;
  constexpr int N = DIM == 2 ? P1 * P1 : P1 * P1 * P1, Nf = DIM == 2 ? P1 : P1 * P1, EV = NV * N;
  extern __shared__ double sm_all[];  // [warps][3][NV][N]: u | F | R
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  double* su = sm_all + (size_t)w * 3 * EV;
  double* sF = su + EV;
  double* sR = sF + EV;
  const FrConst& c = c_fr[P1 - 1];
  const int64_t n = s->n;
  const int64_t nw = (int64_t)gridDim.x * (blockDim.x >> 5);
  for (int64_t e = (int64_t)blockIdx.x * (blockDim.x >> 5) + w; e < n; e += nw) {
    __syncwarp();
    const double* src = u + (size_t)e * EV;
    for (int i = lane; i < EV; i += 32) {
      su[i] = __ldcs(src + i);
      sR[i] = 0.0;
    }
    // fused stage: u_n is fetched now, so that its latency hides behind the arithmetic
    constexpr int KN = (EV + 31) / 32;
    constexpr bool PREF = KN <= 16;
    double pn[PREF ? KN : 1];
    if (PREF && un != nullptr) {
#pragma unroll
      for (int k = 0; k < KN; ++k) {
        const int i = lane + 32 * k;
        pn[k] = i < EV ? __ldcs(un + (size_t)e * EV + i) : 0.0;
      }
    }
    const int level = key_level(keys[e]);
    const double inv2l = (double)(1ull << level);
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
      const double scale = 2.0 * inv2l / (a == 0 ? w0 : (a == 1 ? w1 : w2));  // 2 / dx
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
      // one lane per LINE of P1 points along a: its P1 point fluxes are read once, f(-1), f(+1)
      // and the two common fluxes are formed once per line, then the P1 derivatives
      constexpr int LINES = NV * Nf;  // lines per element along one axis
      for (int ln = lane; ln < LINES; ln += 32) {
        const int v = ln / Nf, nt = ln - v * Nf;  // nt = tangential face-point index, lower axis fastest
        int first;                                // first point of the line
        if (DIM == 2) {
          first = a == 0 ? nt * P1 : nt;
        } else {
          const int n0 = nt % P1, n1 = nt / P1;
          first = a == 0 ? n0 * P1 + n1 * P1 * P1 : (a == 1 ? n0 + n1 * P1 * P1 : n0 + n1 * P1);
        }
        double fj[P1], fm = 0.0, fp = 0.0;
#pragma unroll
        for (int j = 0; j < P1; ++j) {
          fj[j] = sF[v * N + first + j * stride];
          fm += c.lm[j] * fj[j];
          fp += c.lp[j] * fj[j];
        }
        const double dm = fs[(((size_t)e * NF + 2 * a) * NV + v) * Nf + nt] - fm;
        const double dp = fs[(((size_t)e * NF + 2 * a + 1) * NV + v) * Nf + nt] - fp;
#pragma unroll
        for (int i = 0; i < P1; ++i) {
          double d = c.gl[i] * dm + c.gr[i] * dp;
#pragma unroll
          for (int j = 0; j < P1; ++j) d += c.D[i][j] * fj[j];
          sR[v * N + first + i * stride] -= scale * d;
        }
      }
    }
    __syncwarp();
    double* dst = R + (size_t)e * EV;
    if (un == nullptr) {
      for (int i = lane; i < EV; i += 32) __stcs(dst + i, sR[i]);
    } else {
      if (PREF) {
#pragma unroll
        for (int k = 0; k < KN; ++k) {
          const int i = lane + 32 * k;
          if (i < EV) {
            const double o = ca * pn[k] + cb * (su[i] + dt * sR[i]);
            __stcs(dst + i, o);
            sF[i] = o;  // (kept for the traces below; sF is free after the last axis)
          }
        }
      } else {
        const double* sn = un + (size_t)e * EV;
        for (int i = lane; i < EV; i += 32) {
          const double o = ca * sn[i] + cb * (su[i] + dt * sR[i]);
          dst[i] = o;
          sF[i] = o;
        }
      }
      if (uf_out != nullptr) {
        // Alg. 8 step 1 for the next stage: u_out at the face points, one lane per line, both end faces
        __syncwarp();
        constexpr int E = NV * Nf;
        double* fd = uf_out + (size_t)e * NF * E;
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
          const int stride = a == 0 ? 1 : (a == 1 ? P1 : P1 * P1);
          for (int ln = lane; ln < E; ln += 32) {
            const int v = ln / Nf, nt = ln - v * Nf;
            int first;
            if (DIM == 2) {
              first = a == 0 ? nt * P1 : nt;
            } else {
              const int n0 = nt % P1, n1 = nt / P1;
              first = a == 0 ? n0 * P1 + n1 * P1 * P1 : (a == 1 ? n0 + n1 * P1 * P1 : n0 + n1 * P1);
            }
            double lo = 0.0, hi = 0.0;
#pragma unroll
            for (int i = 0; i < P1; ++i) {
              const double x = sF[v * N + first + i * stride];
              lo += c.lm[i] * x;
              hi += c.lp[i] * x;
            }
            __stcs(fd + (2 * a) * E + ln, lo);
            __stcs(fd + (2 * a + 1) * E + ln, hi);
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
      h.D[i][j] = (double)sacc;
    }
    long double lm = 1.0L, lp = 1.0L;
    for (int k = 0; k < P1; ++k)
      if (k != i) {
        lm *= (-1.0L - z[k]) / (z[i] - z[k]);
        lp *= (1.0L - z[k]) / (z[i] - z[k]);
      }
    h.lm[i] = (double)lm;
    h.lp[i] = (double)lp;
    long double d1, d0, e1, e0;
    legendre_ld(p + 1, z[i], &d1);
    legendre_ld(p, z[i], &d0);
    legendre_ld(p + 1, -z[i], &e1);
    legendre_ld(p, -z[i], &e0);
    h.gl[i] = (double)(0.5L * sgn * (d1 - d0));
    h.gr[i] = (double)(-0.5L * sgn * (e1 - e0));
  }
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

template <int DIM, int P1>
static int launch_fr_rhs_t(Tree* t, const double* d_u, const double* d_fs, double* d_R, const double* d_un, double ca,
                           double cb, double dt, double* d_uf_out) {
  constexpr int N = DIM == 2 ? P1 * P1 : P1 * P1 * P1;
  int warps = 8;
  const size_t per_warp = (size_t)3 * (DIM + 2) * N * sizeof(double);
  while (warps > 1 && warps * per_warp > 96 * 1024) warps >>= 1;
  const size_t smem = warps * per_warp;
  auto fn = k_fr_rhs<DIM, P1>;
  LT_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0;
  LT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, warps * 32, smem));
  if (per_sm < 1) per_sm = 1;
  // width of a root cube along each axis (a single cube: the domain width)
  const double w0 = (t->domain[DIM] - t->domain[0]) / t->g.nroot[0];
  const double w1 = (t->domain[DIM + 1] - t->domain[1]) / t->g.nroot[1];
  const double w2 = DIM == 3 ? (t->domain[DIM + 2] - t->domain[2]) / t->g.nroot[2] : 1.0;
  fn<<<t->num_sms * per_sm, warps * 32, smem, t->stream>>>(t->g, t->keys[t->cur], t->d_s, d_u, d_fs, d_R, w0, w1,
                                                            w2, d_un, ca, cb, dt, d_uf_out);
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
