// Device-side random numbers, samplers and small numeric helpers.  Compiled with -fmad=false: every
// fp64 operation below is one IEEE round-to-nearest operation in the order written (DESIGN.md
// "Arithmetic policy").  Written from SURVEY.md 8(c) "R"; shares no code with oracle/.
#pragma once
#include "common.cuh"

namespace bit1 {

// Philox4x32-10 (Salmon et al., SC'11).  Counter (pid, step_lo, step_hi, slot), key (seed_lo, seed_hi).
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const unsigned hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const unsigned hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u;
    k.y += 0xBB67AE85u;
  }
  return c;
}

__device__ __forceinline__ uint4 draw(const Params& P, unsigned pid, unsigned long long step, unsigned slot) {
  return philox4x32_10(make_uint4(pid, (unsigned)step, (unsigned)(step >> 32), slot),
                       make_uint2(P.seed_lo, P.seed_hi));
}

// two-word uniform in (0,1): (((a<<32|b)>>12)+0.5)*2^-52, exact (reading R-U)
__device__ __forceinline__ double u52(unsigned a, unsigned b) {
  const unsigned long long w = (((unsigned long long)a << 32) | (unsigned long long)b) >> 12;
  return ((double)w + 0.5) * 2.220446049250313080847263336181640625e-16;
}
// one-word uniform in (0,1): (a+0.5)*2^-32, exact
__device__ __forceinline__ double u32(unsigned a) {
  return ((double)a + 0.5) * 2.3283064365386962890625e-10;
}

// normal deviate from one word through the caller's piecewise-linear inverse CDF table (A18)
__device__ __forceinline__ double normal_from_word(const Params& P, unsigned a) {
  const double t = u32(a) * (double)P.n_norm;
  int i = (int)t;
  if (i > P.n_norm - 1) i = P.n_norm - 1;
  const double a0 = __ldg(P.inv_norm + i), a1 = __ldg(P.inv_norm + i + 1);
  return a0 + (t - (double)i) * (a1 - a0);
}

// isotropic unit vector: rejection on the unit disc, slots first..first+3, two attempts per block
static __device__ __noinline__ int direction(const Params& P, unsigned pid, unsigned long long step, unsigned first,
                                      double n[3]) {
  for (unsigned b = 0; b < 4; ++b) {
    const uint4 w = draw(P, pid, step, first + b);
    const unsigned ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
    for (int a = 0; a < 2; ++a) {
      const double p = 2.0 * u32(ww[2 * a]) - 1.0;
      const double q = 2.0 * u32(ww[2 * a + 1]) - 1.0;
      const double S = p * p + q * q;
      if (S > 0.0 && S < 1.0) {
        const double r = sqrt(1.0 - S);
        n[0] = 1.0 - 2.0 * S;
        n[1] = (2.0 * p) * r;
        n[2] = (2.0 * q) * r;
        return 0;
      }
    }
  }
  n[0] = 1.0; n[1] = 0.0; n[2] = 0.0;
  return 1;
}

// cross-section table, uniform in eV, clamped
__device__ __forceinline__ double sigma_lookup(const Params& P, const double* tab, double E_eV) {
  double t = E_eV / P.dE_eV;
  const double tmax = (double)(P.n_sig - 1);
  if (t > tmax) t = tmax;
  if (!(t >= 0.0)) t = 0.0;
  int i = (int)t;
  if (i > P.n_sig - 2) i = P.n_sig - 2;
  double fr = t - (double)i;
  if (fr > 1.0) fr = 1.0;
  const double a0 = __ldg(tab + i), a1 = __ldg(tab + i + 1);
  return a0 + fr * (a1 - a0);
}

// cell of a position: (int)(x*inv_dx) clamped to [0, nc-1]
// The clamps are taken on the integer: cvt.rzi.s32.f64 truncates toward zero, saturates and maps NaN to 0, and
// truncation is monotone, so max(0, min((int)t, nc-1)) equals the cast of the clamped double for every t.
__device__ __forceinline__ int cell_of(const Params& P, double x) {
  const int c = __double2int_rz(x * P.inv_dx);
  return max(0, min(c, P.nc - 1));
}

// CIC split of the fixed-point charge Q (SURVEY 8(c) "D"): a goes to node c+1, Q-a to node c, with
// F = 0 for f <= 0 (or NaN), 2^32 - 1 for f >= 1, else trunc(f * 2^32): exactly what the saturating conversion
// cvt.rzi.u32.f64 yields for every f (f * 2^32 is an exact scaling; NaN -> 0), in one instruction instead of
// two compares, a 64-bit conversion and a clamp.
__device__ __forceinline__ unsigned deposit_a(double x, int c, double inv_dx, unsigned Q) {
  const double f = x * inv_dx - (double)c;
  const unsigned F = __double2uint_rz(f * 4294967296.0);
  return (unsigned)(((unsigned long long)Q * (unsigned long long)F + 2147483648ull) >> 32);
}

// dbl(n): sign(n) * ((double)hi(|n|) * 2^64 + (double)lo(|n|))  (reading R-dbl)
__device__ __forceinline__ double dbl128(__int128 n) {
  const bool neg = n < 0;
  const unsigned __int128 a = neg ? (unsigned __int128)0 - (unsigned __int128)n : (unsigned __int128)n;
  const unsigned long long hi = (unsigned long long)(a >> 64), lo = (unsigned long long)a;
  const double d = (double)hi * 18446744073709551616.0 + (double)lo;
  return neg ? -d : d;
}

__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

}  // namespace bit1
