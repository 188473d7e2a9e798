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
#include <math.h>

#include <vector>

#include "lt_internal.h"

namespace lt {

// ------------------------------------------------------------------------ Alg. 7
// For every new leaf: locate its anchor in T_old (lower bound, Eq. 7):
//   same ID                       -> copy
//   old entry is its parent       -> refined-from
//   old entry is its first child  -> fused-from      (reading E-6)
// The map is produced in new-leaf order, so step 5's sort is not needed (reading E-6).
template <int DIM>
__global__ void __launch_bounds__(256) k_map(Geo g, const uint64_t* __restrict__ keys_new,
                                             const uint64_t* __restrict__ keys_old,
                                             const int* __restrict__ first_old, int n_old, DevScalars* s,
                                             int32_t* __restrict__ src, uint8_t* __restrict__ kind) {
  constexpr int NC = Dim<DIM>::NC;
  const int64_t n = s->n;
  for (int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; j < n; j += (int64_t)gridDim.x * blockDim.x) {
    const uint64_t key = keys_new[j];
    const int l = key_level(key);
    const uint64_t m = key_morton(key);
    const int o = locate(g, keys_old, first_old, m);
    const uint64_t ko = keys_old[o];
    const int lo = key_level(ko);
    int kd = 0;
    if (lo == l) {
      kd = 0;
    } else if (lo == l - 1) {
      kd = 1 | (child_id<DIM>(g, m, l) << 4);
    } else if (lo == l + 1) {
      // complete group of leaves: last sibling present at o + NC - 1
      const int sh = DIM * (g.maxl - l - 1);
      const uint64_t klast = make_key(m | ((uint64_t)(NC - 1) << sh), l + 1);
      if (o + NC - 1 >= n_old || keys_old[o + NC - 1] != klast) set_status(&s->status, LT_ERR_MAPPING);
      kd = 2;
    } else {
      set_status(&s->status, LT_ERR_MAPPING);
    }
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
// One warp per new element.  The three cases are warp-uniform branches.
//   u[e][v][n], n = ix + P1*(iy + P1*iz) (reading E-5); E = nvars * N doubles per element.
// A 1-D operator is applied along axis d to the flattened [v][n] block:
//   out[k] = sum_i op[q][i] * in[k + (i - q) * P1^d],  q = (k / P1^d) % P1.
template <int P1, int STRIDE>
__device__ __forceinline__ double apply_1d(const double* __restrict__ op, const double* __restrict__ in, int k) {
  const int q = (k / STRIDE) % P1;
  const double* row = op + q * P1;
  const double* col = in + (k - q * STRIDE);
  double acc = 0.0;
#pragma unroll
  for (int i = 0; i < P1; ++i) acc = fma(row[i], col[i * STRIDE], acc);
  return acc;
}

template <int DIM, int P1>
__global__ void __launch_bounds__(256) k_transfer(const DevScalars* __restrict__ s,
                                                  const int32_t* __restrict__ map_src,
                                                  const uint8_t* __restrict__ map_kind,
                                                  const double* __restrict__ u_old, double* __restrict__ u_new,
                                                  int E, const double* __restrict__ ops_g, int vec2) {
  constexpr int NC = Dim<DIM>::NC;
  constexpr int PP = P1 * P1;
  extern __shared__ double smem[];
  double* ops = smem;  // I^0, I^1, R^0, R^1
  for (int i = threadIdx.x; i < 4 * PP; i += blockDim.x) ops[i] = ops_g[i];
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  double* b0 = smem + 4 * PP + (size_t)w * 3 * E;
  double* b1 = b0 + E;
  double* b2 = b1 + E;
  const int64_t n = s->n;
  for (int64_t j = (int64_t)blockIdx.x * nw + w; j < n; j += (int64_t)gridDim.x * nw) {
    const int kd = map_kind[j];
    const int64_t so = map_src[j];
    double* dst = u_new + (size_t)j * E;
    if ((kd & 15) == 0) {  // direct copy
      const double* sp = u_old + (size_t)so * E;
      if (vec2) {
        const double2* s2 = reinterpret_cast<const double2*>(sp);
        double2* d2 = reinterpret_cast<double2*>(dst);
        for (int k = lane; k < E / 2; k += 32) __stcs(d2 + k, __ldcs(s2 + k));
      } else {
        for (int k = lane; k < E; k += 32) __stcs(dst + k, __ldcs(sp + k));
      }
    } else if ((kd & 15) == 1) {  // interpolation, Eq. 8
      const int cid = kd >> 4;
      const double* sp = u_old + (size_t)so * E;
      for (int k = lane; k < E; k += 32) b0[k] = sp[k];
      __syncwarp();
      const double* ox = ops + ((cid >> 0) & 1) * PP;
      const double* oy = ops + ((cid >> 1) & 1) * PP;
      for (int k = lane; k < E; k += 32) b1[k] = apply_1d<P1, 1>(ox, b0, k);
      __syncwarp();
      if (DIM == 2) {
        for (int k = lane; k < E; k += 32) __stcs(dst + k, apply_1d<P1, P1>(oy, b1, k));
      } else {
        const double* oz = ops + ((cid >> 2) & 1) * PP;
        for (int k = lane; k < E; k += 32) b0[k] = apply_1d<P1, P1>(oy, b1, k);
        __syncwarp();
        for (int k = lane; k < E; k += 32) __stcs(dst + k, apply_1d<P1, PP>(oz, b0, k));
      }
      __syncwarp();
    } else {  // L2 projection of the NC children, Eq. 9-13
      for (int k = lane; k < E; k += 32) b2[k] = 0.0;
      for (int c = 0; c < NC; ++c) {
        const double* sp = u_old + (size_t)(so + c) * E;
        for (int k = lane; k < E; k += 32) b0[k] = __ldcs(sp + k);
        __syncwarp();
        const double* ox = ops + (2 + ((c >> 0) & 1)) * PP;
        const double* oy = ops + (2 + ((c >> 1) & 1)) * PP;
        for (int k = lane; k < E; k += 32) b1[k] = apply_1d<P1, 1>(ox, b0, k);
        __syncwarp();
        if (DIM == 2) {
          for (int k = lane; k < E; k += 32) b2[k] += apply_1d<P1, P1>(oy, b1, k);
        } else {
          const double* oz = ops + (2 + ((c >> 2) & 1)) * PP;
          for (int k = lane; k < E; k += 32) b0[k] = apply_1d<P1, P1>(oy, b1, k);
          __syncwarp();
          for (int k = lane; k < E; k += 32) b2[k] += apply_1d<P1, PP>(oz, b0, k);
        }
        __syncwarp();
      }
      for (int k = lane; k < E; k += 32) __stcs(dst + k, b2[k]);
      __syncwarp();
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
  if (t->ops_p == p && t->d_ops) return LT_OK;
  const int P1 = p + 1, PP = P1 * P1;
  std::vector<long double> z, w;
  gl_rule(P1, z, w);
  std::vector<double> h(4 * PP);
  for (int b = 0; b < 2; ++b)
    for (int m = 0; m < P1; ++m) {
      const long double xi = 0.5L * (z[m] + 2 * b - 1);
      for (int i = 0; i < P1; ++i) {
        long double v = 1.0L;
        for (int k = 0; k < P1; ++k)
          if (k != i) v *= (xi - z[k]) / (z[i] - z[k]);
        h[b * PP + m * P1 + i] = (double)v;                                  // I^b[m][i]
        h[(2 + b) * PP + i * P1 + m] = (double)(0.5L * (w[m] / w[i]) * v);   // R^b[i][m]
      }
    }
  if (!t->d_ops) LT_CUDA(cudaMalloc(&t->d_ops, 4 * 64 * sizeof(double)));
  LT_CUDA(cudaMemcpyAsync(t->d_ops, h.data(), 4 * PP * sizeof(double), cudaMemcpyHostToDevice, t->stream));
  LT_CUDA(cudaStreamSynchronize(t->stream));  // h goes out of scope
  t->ops_p = p;
  return LT_OK;
}

int launch_map(Tree* t) {
  int G = grid_for(t, 8);
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
static int launch_transfer_t(Tree* t, const double* u_old, double* u_new, int E, int vec2) {
  const int PP = P1 * P1;
  int warps = 8;
  size_t per_warp = (size_t)3 * E * sizeof(double);
  const size_t budget = 200 * 1024 - 4 * PP * sizeof(double);
  while (warps > 1 && warps * per_warp > budget) warps >>= 1;
  if (warps * per_warp > budget) return LT_ERR_ARG;
  size_t smem = 4 * PP * sizeof(double) + warps * per_warp;
  auto fn = k_transfer<DIM, P1>;
  LT_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0;
  LT_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, warps * 32, smem));
  if (per_sm < 1) per_sm = 1;
  int G = t->num_sms * per_sm;
  fn<<<G, warps * 32, smem, t->stream>>>(t->d_s, t->map_src, t->map_kind, u_old, u_new, E, t->d_ops, vec2);
  t->launches++;
  LT_CUDA(cudaGetLastError());
  return LT_OK;
}

template <int DIM>
static int launch_transfer_d(Tree* t, const double* u_old, double* u_new, int p, int E, int vec2) {
  switch (p) {
    case 0: return launch_transfer_t<DIM, 1>(t, u_old, u_new, E, vec2);
    case 1: return launch_transfer_t<DIM, 2>(t, u_old, u_new, E, vec2);
    case 2: return launch_transfer_t<DIM, 3>(t, u_old, u_new, E, vec2);
    case 3: return launch_transfer_t<DIM, 4>(t, u_old, u_new, E, vec2);
    case 4: return launch_transfer_t<DIM, 5>(t, u_old, u_new, E, vec2);
    case 5: return launch_transfer_t<DIM, 6>(t, u_old, u_new, E, vec2);
    case 6: return launch_transfer_t<DIM, 7>(t, u_old, u_new, E, vec2);
    case 7: return launch_transfer_t<DIM, 8>(t, u_old, u_new, E, vec2);
  }
  return LT_ERR_ARG;
}

int launch_transfer(Tree* t, const double* d_u_old, double* d_u_new, int p, int nvars) {
  int N = 1;
  for (int a = 0; a < t->g.dim; ++a) N *= (p + 1);
  const int E = nvars * N;
  const int vec2 = (E % 2 == 0) && (((uintptr_t)d_u_old & 15) == 0) && (((uintptr_t)d_u_new & 15) == 0);
  return t->g.dim == 2 ? launch_transfer_d<2>(t, d_u_old, d_u_new, p, E, vec2)
                       : launch_transfer_d<3>(t, d_u_old, d_u_new, p, E, vec2);
}

}  // namespace lt
