// lt_euler.cuh -- the compressible Euler flux and the Rusanov common flux (readings I-1, I-2;
// PAPER.md:304) shared by the FR kernels of lt_fr.cu and the fused face pass of lt_transfer.cu.
// Product code: shares nothing with oracle/.
#pragma once
#include "lt_dev.cuh"

namespace lt {

constexpr double kGamma = 1.4;

template <int DIM>
__device__ __forceinline__ void euler_flux(int a, const double* u, double* F) {
  const double rho = u[0], E = u[DIM + 1], ir = 1.0 / rho;
  double v[DIM], q = 0.0;
#pragma unroll
  for (int b = 0; b < DIM; ++b) {
    v[b] = u[1 + b] * ir;
    q += v[b] * v[b];
  }
  const double pr = (kGamma - 1.0) * (E - 0.5 * rho * q);
  double va = v[0];
#pragma unroll
  for (int b = 1; b < DIM; ++b)
    if (b == a) va = v[b];
  F[0] = rho * va;
#pragma unroll
  for (int b = 0; b < DIM; ++b) F[1 + b] = u[1 + b] * va + (b == a ? pr : 0.0);
  F[DIM + 1] = (E + pr) * va;
}

template <int DIM>
__device__ __forceinline__ double wave_speed(int a, const double* u) {
  const double rho = u[0], E = u[DIM + 1], ir = 1.0 / rho;
  double q = 0.0, va = 0.0;
#pragma unroll
  for (int b = 0; b < DIM; ++b) {
    const double vb = u[1 + b] * ir;
    q += vb * vb;
    if (b == a) va = vb;
  }
  const double pr = (kGamma - 1.0) * (E - 0.5 * rho * q);
  return fabs(va) + sqrt(kGamma * pr * ir);
}

// F* = (F_a(uL) + F_a(uR))/2 - max(|v_a| + c)(uR - uL)/2, the flux along +a (reading I-2)
template <int DIM>
__device__ __forceinline__ void rusanov(int a, const double* L, const double* R, double* F) {
  constexpr int NV = DIM + 2;
  double FL[NV], FR[NV];
  euler_flux<DIM>(a, L, FL);
  euler_flux<DIM>(a, R, FR);
  const double lam = fmax(wave_speed<DIM>(a, L), wave_speed<DIM>(a, R));
#pragma unroll
  for (int v = 0; v < NV; ++v) F[v] = 0.5 * (FL[v] + FR[v]) - 0.5 * lam * (R[v] - L[v]);
}

}  // namespace lt
