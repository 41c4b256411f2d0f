// Device-inline physics of the ideal-MHD step (eqs (1)-(5), L170-183) in the
// readings of DESIGN.md: primitive reconstruction with an MC(beta) limiter (Q-R1, Q-R2),
// Rusanov flux with the speed of the mean face state (Q-F1, Q-F2), B = B0 + B1 split
// (Q-B1).  Variables: primitive W = (rho, u, B1, p), conserved U = (rho, rho u, B1, e).
#pragma once
#include <cuda_runtime.h>

namespace batl {

// O-4 / Q-R2: limited slope from the one-sided differences dm = W_c - W_{c-1}, dp = W_{c+1} - W_c
__device__ __forceinline__ double mc_limited(double dm, double dp, double beta) {
  const double lim = fmin(fmin(beta * fabs(dm), beta * fabs(dp)), 0.5 * fabs(dm + dp));
  return (dm * dp <= 0.0) ? 0.0 : copysign(lim, dm);
}

// analytic dipole at the origin: B0 = (3 (m.x) x / r^2 - m) / r^3
__device__ __forceinline__ void dipole_field(const double m[3], double x, double y, double z, double B0[3]) {
  const double r2 = x * x + y * y + z * z;
  if (r2 == 0.0) { B0[0] = B0[1] = B0[2] = 0.0; return; }
  const double r = sqrt(r2), r3 = r2 * r;
  const double md = m[0] * x + m[1] * y + m[2] * z;
  B0[0] = (3.0 * md * x / r2 - m[0]) / r3;
  B0[1] = (3.0 * md * y / r2 - m[1]) / r3;
  B0[2] = (3.0 * md * z / r2 - m[2]) / r3;
}

// physical flux through a face with normal e_D and the conserved state of W
// (eqs (1)-(4), L170-177; B0f = B0 at the face centre, Q-B1)
template <int D>
__device__ __forceinline__ void mhd_flux(const double W[8], const double B0f[3], double inv_gm1,
                                         double F[8], double U[8]) {
  const double rho = W[0], p = W[7];
  const double ux = W[1], uy = W[2], uz = W[3];
  const double bx = W[4], by = W[5], bz = W[6];
  const double un = W[1 + D], b1n = W[4 + D], b0n = B0f[D];
  const double b1sq = bx * bx + by * by + bz * bz;
  const double b0b1 = B0f[0] * bx + B0f[1] * by + B0f[2] * bz;
  const double ub1 = ux * bx + uy * by + uz * bz;
  const double u2 = ux * ux + uy * uy + uz * uz;
  const double e = p * inv_gm1 + 0.5 * rho * u2 + 0.5 * b1sq;     // eq. (5)
  const double ptot = p + 0.5 * b1sq + b0b1;
  const double mn = rho * un;
  const double bn = b1n + b0n;
  F[0] = mn;                                                       // eq. (1)
  F[1] = mn * ux - b1n * bx - b0n * bx - b1n * B0f[0];             // eq. (2)
  F[2] = mn * uy - b1n * by - b0n * by - b1n * B0f[1];
  F[3] = mn * uz - b1n * bz - b0n * bz - b1n * B0f[2];
  F[1 + D] += ptot;
  F[4] = un * (bx + B0f[0]) - bn * ux;                             // eq. (3)
  F[5] = un * (by + B0f[1]) - bn * uy;
  F[6] = un * (bz + B0f[2]) - bn * uz;
  F[7] = un * (e + ptot) - ub1 * bn;                               // eq. (4)
  U[0] = rho; U[1] = rho * ux; U[2] = rho * uy; U[3] = rho * uz;
  U[4] = bx; U[5] = by; U[6] = bz; U[7] = e;
}

// Rusanov flux (O-5): F^ = (F(WL)+F(WR))/2 - c_max (U(WR)-U(WL))/2, c_max = |u_n| + c_f of the
// mean state.  Also returns the face-averaged normal B1 (Q-S1) and c_max (O-8).
template <int D>
__device__ __forceinline__ void rusanov_flux(const double WL[8], const double WR[8], const double B0f[3],
                                             double gamma, double inv_gm1, double F[8], double& Bn, double& cmax,
                                             int flux_type = 0) {
  double FL[8], FR[8], UL[8], UR[8];
  mhd_flux<D>(WL, B0f, inv_gm1, FL, UL);
  mhd_flux<D>(WR, B0f, inv_gm1, FR, UR);
  const double rho = 0.5 * (WL[0] + WR[0]);
  const double p = 0.5 * (WL[7] + WR[7]);
  const double un = 0.5 * (WL[1 + D] + WR[1 + D]);
  const double bx = 0.5 * (WL[4] + WR[4]) + B0f[0];
  const double by = 0.5 * (WL[5] + WR[5]) + B0f[1];
  const double bz = 0.5 * (WL[6] + WR[6]) + B0f[2];
  const double bnt = (D == 0) ? bx : (D == 1) ? by : bz;
  const double a2 = gamma * p / rho;
  const double b2 = (bx * bx + by * by + bz * bz) / rho;
  const double bn2 = bnt * bnt / rho;
  const double s = a2 + b2;
  const double disc = fmax(s * s - 4.0 * a2 * bn2, 0.0);
  const double cf = sqrt(0.5 * (s + sqrt(disc)));
  const double c = fabs(un) + cf;
  if (flux_type == 1) {                                  // Q-F4: HLL with the bounds of the mean state
    const double sl = fmin(0.0, un - cf), sr = fmax(0.0, un + cf);
#pragma unroll
    for (int v = 0; v < 8; ++v) F[v] = (sr * FL[v] - sl * FR[v] + sl * sr * (UR[v] - UL[v])) / (sr - sl);
  } else {
#pragma unroll
    for (int v = 0; v < 8; ++v) F[v] = 0.5 * (FL[v] + FR[v]) - 0.5 * c * (UR[v] - UL[v]);
  }
  Bn = 0.5 * (WL[4 + D] + WR[4 + D]);
  cmax = c;
}

// order-preserving map positive double <-> uint64 for atomicMin
__device__ __forceinline__ void atomic_min_positive(unsigned long long* addr, double v) {
  if (v > 0.0) atomicMin(addr, (unsigned long long)__double_as_longlong(v));
}

}  // namespace batl
