// mem_common.cuh -- pieces shared by every process kernel of the CUDA path.
//
// S1 of the hot path: Philox4x32-10 counter-based sampling keyed by
// (seed, event, point) (BASELINE.json:north_star (b)); the toy PDF (BASELINE.json:configs[0]);
// the double-Gaussian jet transfer function; the warp/block reduction of
// sum w and sum w^2 (Eq. 5-6).  Nothing here is shared with oracle/.
#pragma once
#include <cstdint>
#include <type_traits>

#include <cuda_runtime.h>

namespace memb200 {

constexpr int kThreads = 256;            // threads per block in the integrate kernels
constexpr int kWarps = kThreads / 32;
constexpr int64_t kChunk = 1 << 14;      // points per (event, chunk) block; fixes the reduction order
constexpr int kMaxDims = 8;
constexpr int kMaxBins = 64;
constexpr int kMaxAdaptChunks = 8;       // adaptation passes use at most this many blocks per event

// Everything the kernels need that does not depend on the event.  Filled on the host from
// mem_params (mem_api.cu: make_dev_const) and passed by value as a kernel argument, so every
// member is a constant-bank operand.
template <typename T>
struct DevConstR {
  // beams, O3
  T sqrt_s, inv_sqrt_s, S, inv_S;
  // toy PDF, O4
  T pdf_pow_x, pdf_pow_1mx;
  int pdf_fast;                         // 1 when pow_x == -1/2 and pow_1mx == 3
  int n_flav;
  T A_q2, A_g2;                    // pdf_A_q^2, pdf_A_g^2
  // jets, O5: E = E_jet (rlo + dr u); TF(E_jet; E) * E = c1 exp(-z1^2) + c2 exp(-z2^2),
  // z_k = a_k / x + b_k with x = E / E_jet
  T rlo, dr;
  T tf_a1, tf_b1, tf_c1, tf_a2, tf_b2, tf_c2;
  T tf_q2, tf_q1, tf_q0;           // z1^2 - z2^2 = q2 v^2 + q1 v + q0, v = 1/x
  // Breit-Wigner data, O6
  T mW, GW, mW2, mWGW, mWGW2;      // m, Gamma, m^2, m Gamma, (m Gamma)^2
  T tW_lo, tW_dt;                  // t window of m +- n Gamma
  T mt2, mtGt, mtGt2, tT_lo, tT_dt;
  T mZ2, mZGZ2;
  // couplings, O8
  T g4w;                           // g^4, g^2 = 4 sqrt2 G_F m_W^2
  T gz4;                           // g_Z^4
  T gs4;                           // g_s^4 = (4 pi alpha_s)^2
  T V_ud2, V_tb2;
  T z_cu, z_ct;                    // sum_q [..] coefficient of u^2 and of t^2 (config 2)
  // windows
  T nu_pz_max, nu_eta_max, met_sigma, met_nsigma;
  // VEGAS
  int vegas_bins;
  T vegas_alpha;
  int n_perm;                      // jet-parton assignments summed per point (>= 1)
  // NEXT-4 (mem_tth.cuh): upper edge of the parton-energy window, Higgs Breit-Wigner data, 2 ln(rhi/rlo),
  // hypothesis (0 = t tbar H, 1 = non-resonant t tbar b bbar) and every constant factor of the radiated system
  T rhi, mH2, mHGH, tH_lo, tH_dt, lnr, tth_c;
  int tth_hyp;
  // NEXT-3 grid PDFs: tables already interpolated in ln Q at the handle's fixed scale, [6][pdf_nx]
  // (species 0 = g, 1..5 = d,u,s,c,b), sample i at pdf_lxmin + i pdf_dx; nullptr = toy PDF
  const double* pdf_tab;
  int pdf_nx;
  double pdf_lxmin, pdf_dx, pdf_inv_dx;
};
using DevConst = DevConstR<double>;   // the fp64 path
using DevConstF = DevConstR<float>;   // fp32 integrand core of config 3 (reading A15)

// ---------------------------------------------------------------------------------------
// S1. Philox4x32-10 (Salmon et al. 2011; multipliers and Weyl constants are the published ones)
// ---------------------------------------------------------------------------------------
// The ten round keys (key + r * Weyl constant) are formed once on the host (make_philox in mem_api.cu) and reach the
// kernels as a by-value argument, i.e. as constant-bank operands of the round's XOR: no key arithmetic in the point loop.
// Each round's two 32 x 32 -> 64 products are written as 64-bit multiplies (one IMAD.WIDE each, high and low word at once).
struct Philox {
  uint32_t ka[10], kb[10];              // round keys of key word 0 and key word 1
  __device__ __forceinline__ void operator()(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                             uint32_t (&out)[4]) const {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
      const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
      const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0, hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
      c0 = hi1 ^ c1 ^ ka[r]; c1 = lo1; c2 = hi0 ^ c3 ^ kb[r]; c3 = lo0;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
  }
};
inline Philox make_philox(uint64_t seed) {
  Philox p;
  uint32_t a = (uint32_t)seed, b = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) { p.ka[r] = a; p.kb[r] = b; a += 0x9E3779B9u; b += 0xBB67AE85u; }
  return p;
}

// 52-bit uniform in (0,1): u = (k + 1/2) 2^-52, k = (a >> 6) 2^26 + (b >> 6).  Built without an
// integer->double conversion: 1.k (binary) = 1 + k 2^-52 is assembled in the mantissa, and
// adding -(1 - 2^-53) is exact because (2k + 1) 2^-53 is representable.
__device__ __forceinline__ double u52(uint32_t a, uint32_t b) {
  const uint32_t A = a >> 6;
  const uint32_t hi = 0x3FF00000u | (A >> 6);
  const uint32_t lo = __funnelshift_r(b, A, 6);        // low word of ((A : b) >> 6) = (A << 26) | (b >> 6)
  return __hiloint2double((int)hi, (int)lo) + (-0x1.fffffffffffffp-1);
}

// counter = (point low, point high, event, pass * 256 + word block); block j feeds dims 2j, 2j+1
template <int D>
__device__ __forceinline__ void draw_uniforms(const Philox& rng, uint64_t point, uint32_t event,
                                              uint32_t pass, double (&u)[D]) {
#pragma unroll
  for (int j = 0; 2 * j < D; ++j) {
    uint32_t r[4];
    rng((uint32_t)point, (uint32_t)(point >> 32), event, pass * 256u + (uint32_t)j, r);
    u[2 * j] = u52(r[0], r[1]);
    if (2 * j + 1 < D) u[2 * j + 1] = u52(r[2], r[3]);
  }
}

// fp32 variant (reading A15), plain Monte Carlo: single-precision uniforms straight from the same Philox words,
// u = (k + 1/2) 2^-23 with k the 23 leading bits of the first word of the dimension's pair -- exact in fp32 and in
// (0, 1); it is the fp64 uniform of the same counter truncated to 23 bits (they differ by less than 2^-23).
// The VEGAS passes map the fp64 uniform through the grid first and round the mapped point instead.
template <int D>
__device__ __forceinline__ void draw_uniforms(const Philox& rng, uint64_t point, uint32_t event, uint32_t pass,
                                              float (&u)[D]) {
#pragma unroll
  for (int j = 0; 2 * j < D; ++j) {
    uint32_t r[4];
    rng((uint32_t)point, (uint32_t)(point >> 32), event, pass * 256u + (uint32_t)j, r);
    u[2 * j] = fmaf(__uint2float_rn(r[0] >> 9), 0x1p-23f, 0x1p-24f);
    if (2 * j + 1 < D) u[2 * j + 1] = fmaf(__uint2float_rn(r[2] >> 9), 0x1p-23f, 0x1p-24f);
  }
}

// ---------------------------------------------------------------------------------------
// small fp64 helpers
// ---------------------------------------------------------------------------------------
// 1/x for normal, finite x well inside the exponent range (every use below): the MUFU seed
// (relative error ~2^-20, it reads only the high word) -> one cubic step (e^3 ~ 2^-60) -> one
// linear step for the last bits; error about 1 ulp.  No special-case branches.
__device__ __forceinline__ double rcp_fast(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  y = fma(y, fma(e, e, e), y);          // y (1 + e + e^2)
  e = fma(-x, y, 1.0);
  return fma(y, e, y);
}

// 1/sqrt(x) for normal, finite, positive x: MUFU seed (relative error ~2^-20) -> one cubic step
// y (1 + e/2 + 3 e^2/8), e = 1 - x y^2 (error ~e^3) -> one linear step; about 1 ulp, no special-case branch.
__device__ __forceinline__ double rsqrt_fast(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x * y, y, 1.0);
  y = fma(y * e, fma(0.375, e, 0.5), y);
  e = fma(-x * y, y, 1.0);
  return fma(0.5 * y, e, y);
}

// Polynomial coefficients live in the constant bank (c[3][..] operands of DFMA): as 64-bit literals each costs two
// UMOVs per use inside the point loop (there are more of them than uniform registers to hoist them into), and a
// DFMA with a constant-bank operand issues at the full FP64 rate (profiles/r01_microbench.md).
__constant__ double kTanS[6] = {-0x1.5555555555554p-3, 0x1.1111111110a86p-7, -0x1.a01a019e3e0afp-13,
                                0x1.71de373e0fee6p-19, -0x1.ae5fb0a5df712p-26, 0x1.5deb31d167e93p-33};
__constant__ double kTanC[6] = {0x1.5555555555555p-5, -0x1.6c16c16c168d0p-10, 0x1.a01a019f2bd7bp-16,
                                -0x1.27e4f9eb9238ep-22, 0x1.1eeb3bafbb15dp-29, -0x1.905db35e3086ap-37};
// exp_tab: 256/ln2, the rounding constant 1.5 2^52, -ln2/256 in two parts, 1/24, 1/6, 1/2
__constant__ double kExpC[7] = {0x1.71547652b82fep+8, 6755399441055744.0, -0x1.62e42fee00000p-9, -0x1.a39ef35793c76p-41,
                                1.0 / 24.0, 1.0 / 6.0, 0.5};

// tan(t) for the Breit-Wigner maps (O6): t = atan(..) lies strictly inside (-pi/2, pi/2), so no
// general range reduction (and none of libdevice's large-argument path) is needed.  |t| <= pi/4:
// tan = S(t)/C(t); otherwise with r = pi/2 - |t| (pi/2 in two parts): tan = C(r)/S(r).  S, C are
// degree-13 / degree-12 polynomials (Chebyshev interpolants in r^2 on 1.02 [0, (pi/4)^2]; the quotient
// is within 2.0e-17 of tan before rounding), one reciprocal.  tan_bw_n evaluates N arguments with
// the Horner steps interleaved so that each coefficient is fetched once for all of them.
template <int N>
__device__ __forceinline__ void tan_bw_n(const double (&t)[N], double (&out)[N]) {
  const double* kS = kTanS;
  const double* kC = kTanC;
  double r[N], z[N], ps[N], pc[N];
  bool big[N];
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const double a = fabs(t[j]);
    big[j] = a > 0.78539816339744830962;
    r[j] = big[j] ? (1.57079632679489655800e+00 - a) + 6.12323399573676603587e-17 : a;
    z[j] = r[j] * r[j];
    ps[j] = kS[5]; pc[j] = kC[5];
  }
#pragma unroll
  for (int i = 4; i >= 0; --i) {
#pragma unroll
    for (int j = 0; j < N; ++j) { ps[j] = fma(ps[j], z[j], kS[i]); pc[j] = fma(pc[j], z[j], kC[i]); }
  }
#pragma unroll
  for (int j = 0; j < N; ++j) {
    const double sn = fma(r[j] * z[j], ps[j], r[j]);
    const double cs = fma(z[j] * z[j], pc[j], fma(-0.5, z[j], 1.0));
    const double q = (big[j] ? cs : sn) * rcp_fast(big[j] ? sn : cs);
    out[j] = copysign(q, t[j]);
  }
}
// cos(x) for 0 <= x <= pi/3 (the trigonometric form of the resolvent cubic): 1 - 2 sin^2(x/2) with the
// sine polynomial of tan_bw_n on |x/2| <= pi/6; no range reduction, no large-argument path.
__device__ __forceinline__ double cos_third(double x) {
  const double* kS = kTanS;
  const double h = 0.5 * x, z = h * h;
  double ps = kS[5];
#pragma unroll
  for (int i = 4; i >= 0; --i) ps = fma(ps, z, kS[i]);
  const double sn = fma(h * z, ps, h);
  return fma(-2.0 * sn, sn, 1.0);
}

// sin(x) and cos(x) for 0 <= x < pi (config 1's Breit-Wigner complement angle and its window fraction): the
// polynomials of tan_bw_n at x/4 <= pi/4, then two angle doublings.  No range reduction, no large-argument path.
// cos(x/2) = 1 - 2 sin^2(x/4) cancels only next to x = pi, which the callers' windows exclude by >= 0.026
// (the transverse-mass edge cannot lie more than 38 widths below the W pole): relative error <= 1e-14 there, ~2 ulp elsewhere.
__device__ __forceinline__ void sincos_0pi(double x, double* sn, double* cs) {
  const double r = 0.25 * x, z = r * r;
  double ps = kTanS[5], pc = kTanC[5];
#pragma unroll
  for (int i = 4; i >= 0; --i) { ps = fma(ps, z, kTanS[i]); pc = fma(pc, z, kTanC[i]); }
  const double s1 = fma(r * z, ps, r);                                // sin(x/4)
  const double c1 = fma(z * z, pc, fma(-0.5, z, 1.0));                // cos(x/4)
  const double s2 = 2.0 * s1 * c1, c2 = fma(-2.0 * s1, s1, 1.0);      // x/2
  *sn = 2.0 * s2 * c2;
  *cs = fma(-2.0 * s2, s2, 1.0);
}

__device__ __forceinline__ double tan_bw(double t) {
  const double a[1] = {t};
  double o[1];
  tan_bw_n<1>(a, o);
  return o[0];
}

// exp(x) for the hot loops: x = k ln2/256 + r with |r| <= ln2/512, exp(x) = 2^(k >> 8) * T[k & 255] * (1 + p(r)),
// T[j] = 2^(j/256) (correctly rounded, own table), p = r + r^2 (1/2 + r (1/6 + r/24)) (remainder r^5/120 < 3.8e-17),
// 2^(k >> 8) through the exponent field.  9 FP64 instructions against libdevice's 17 per call; about 1 ulp.
// CHECK = false (the integrands): the caller guarantees |x| < 700 -- mem_create validates the transfer-function and
// window parameters that bound every argument (mem_api.cu: check_params).  CHECK = true: |x| >= 700 (or NaN)
// returns 0 or +inf without touching the exponent arithmetic.
__device__ const double kExpTab[256] = {
    0x1.0000000000000p+0, 0x1.00b1afa5abcbfp+0, 0x1.0163da9fb3335p+0, 0x1.02168143b0281p+0,
    0x1.02c9a3e778061p+0, 0x1.037d42e11bbccp+0, 0x1.04315e86e7f85p+0, 0x1.04e5f72f654b1p+0,
    0x1.059b0d3158574p+0, 0x1.0650a0e3c1f89p+0, 0x1.0706b29ddf6dep+0, 0x1.07bd42b72a836p+0,
    0x1.0874518759bc8p+0, 0x1.092bdf66607e0p+0, 0x1.09e3ecac6f383p+0, 0x1.0a9c79b1f3919p+0,
    0x1.0b5586cf9890fp+0, 0x1.0c0f145e46c85p+0, 0x1.0cc922b7247f7p+0, 0x1.0d83b23395decp+0,
    0x1.0e3ec32d3d1a2p+0, 0x1.0efa55fdfa9c5p+0, 0x1.0fb66affed31bp+0, 0x1.1073028d7233ep+0,
    0x1.11301d0125b51p+0, 0x1.11edbab5e2ab6p+0, 0x1.12abdc06c31ccp+0, 0x1.136a814f204abp+0,
    0x1.1429aaea92de0p+0, 0x1.14e95934f312ep+0, 0x1.15a98c8a58e51p+0, 0x1.166a45471c3c2p+0,
    0x1.172b83c7d517bp+0, 0x1.17ed48695bbc0p+0, 0x1.18af9388c8deap+0, 0x1.1972658375d2fp+0,
    0x1.1a35beb6fcb75p+0, 0x1.1af99f8138a1cp+0, 0x1.1bbe084045cd4p+0, 0x1.1c82f95281c6bp+0,
    0x1.1d4873168b9aap+0, 0x1.1e0e75eb44027p+0, 0x1.1ed5022fcd91dp+0, 0x1.1f9c18438ce4dp+0,
    0x1.2063b88628cd6p+0, 0x1.212be3578a819p+0, 0x1.21f49917ddc96p+0, 0x1.22bdda27912d1p+0,
    0x1.2387a6e756238p+0, 0x1.2451ffb82140ap+0, 0x1.251ce4fb2a63fp+0, 0x1.25e85711ece75p+0,
    0x1.26b4565e27cddp+0, 0x1.2780e341ddf29p+0, 0x1.284dfe1f56381p+0, 0x1.291ba7591bb70p+0,
    0x1.29e9df51fdee1p+0, 0x1.2ab8a66d10f13p+0, 0x1.2b87fd0dad990p+0, 0x1.2c57e39771b2fp+0,
    0x1.2d285a6e4030bp+0, 0x1.2df961f641589p+0, 0x1.2ecafa93e2f56p+0, 0x1.2f9d24abd886bp+0,
    0x1.306fe0a31b715p+0, 0x1.31432edeeb2fdp+0, 0x1.32170fc4cd831p+0, 0x1.32eb83ba8ea32p+0,
    0x1.33c08b26416ffp+0, 0x1.3496266e3fa2dp+0, 0x1.356c55f929ff1p+0, 0x1.36431a2de883bp+0,
    0x1.371a7373aa9cbp+0, 0x1.37f26231e754ap+0, 0x1.38cae6d05d866p+0, 0x1.39a401b7140efp+0,
    0x1.3a7db34e59ff7p+0, 0x1.3b57fbfec6cf4p+0, 0x1.3c32dc313a8e5p+0, 0x1.3d0e544ede173p+0,
    0x1.3dea64c123422p+0, 0x1.3ec70df1c5175p+0, 0x1.3fa4504ac801cp+0, 0x1.40822c367a024p+0,
    0x1.4160a21f72e2ap+0, 0x1.423fb2709468ap+0, 0x1.431f5d950a897p+0, 0x1.43ffa3f84b9d4p+0,
    0x1.44e086061892dp+0, 0x1.45c2042a7d232p+0, 0x1.46a41ed1d0057p+0, 0x1.4786d668b3237p+0,
    0x1.486a2b5c13cd0p+0, 0x1.494e1e192aed2p+0, 0x1.4a32af0d7d3dep+0, 0x1.4b17dea6db7d7p+0,
    0x1.4bfdad5362a27p+0, 0x1.4ce41b817c114p+0, 0x1.4dcb299fddd0dp+0, 0x1.4eb2d81d8abffp+0,
    0x1.4f9b2769d2ca7p+0, 0x1.508417f4531eep+0, 0x1.516daa2cf6642p+0, 0x1.5257de83f4eefp+0,
    0x1.5342b569d4f82p+0, 0x1.542e2f4f6ad27p+0, 0x1.551a4ca5d920fp+0, 0x1.56070dde910d2p+0,
    0x1.56f4736b527dap+0, 0x1.57e27dbe2c4cfp+0, 0x1.58d12d497c7fdp+0, 0x1.59c0827ff07ccp+0,
    0x1.5ab07dd485429p+0, 0x1.5ba11fba87a03p+0, 0x1.5c9268a5946b7p+0, 0x1.5d84590998b93p+0,
    0x1.5e76f15ad2148p+0, 0x1.5f6a320dceb71p+0, 0x1.605e1b976dc09p+0, 0x1.6152ae6cdf6f4p+0,
    0x1.6247eb03a5585p+0, 0x1.633dd1d1929fdp+0, 0x1.6434634ccc320p+0, 0x1.652b9febc8fb7p+0,
    0x1.6623882552225p+0, 0x1.671c1c70833f6p+0, 0x1.68155d44ca973p+0, 0x1.690f4b19e9538p+0,
    0x1.6a09e667f3bcdp+0, 0x1.6b052fa75173ep+0, 0x1.6c012750bdabfp+0, 0x1.6cfdcddd47645p+0,
    0x1.6dfb23c651a2fp+0, 0x1.6ef9298593ae5p+0, 0x1.6ff7df9519484p+0, 0x1.70f7466f42e87p+0,
    0x1.71f75e8ec5f74p+0, 0x1.72f8286ead08ap+0, 0x1.73f9a48a58174p+0, 0x1.74fbd35d7cbfdp+0,
    0x1.75feb564267c9p+0, 0x1.77024b1ab6e09p+0, 0x1.780694fde5d3fp+0, 0x1.790b938ac1cf6p+0,
    0x1.7a11473eb0187p+0, 0x1.7b17b0976cfdbp+0, 0x1.7c1ed0130c132p+0, 0x1.7d26a62ff86f0p+0,
    0x1.7e2f336cf4e62p+0, 0x1.7f3878491c491p+0, 0x1.80427543e1a12p+0, 0x1.814d2add106d9p+0,
    0x1.82589994cce13p+0, 0x1.8364c1eb941f7p+0, 0x1.8471a4623c7adp+0, 0x1.857f4179f5b21p+0,
    0x1.868d99b4492edp+0, 0x1.879cad931a436p+0, 0x1.88ac7d98a6699p+0, 0x1.89bd0a478580fp+0,
    0x1.8ace5422aa0dbp+0, 0x1.8be05bad61778p+0, 0x1.8cf3216b5448cp+0, 0x1.8e06a5e0866d9p+0,
    0x1.8f1ae99157736p+0, 0x1.902fed0282c8ap+0, 0x1.9145b0b91ffc6p+0, 0x1.925c353aa2fe2p+0,
    0x1.93737b0cdc5e5p+0, 0x1.948b82b5f98e5p+0, 0x1.95a44cbc8520fp+0, 0x1.96bdd9a7670b3p+0,
    0x1.97d829fde4e50p+0, 0x1.98f33e47a22a2p+0, 0x1.9a0f170ca07bap+0, 0x1.9b2bb4d53fe0dp+0,
    0x1.9c49182a3f090p+0, 0x1.9d674194bb8d5p+0, 0x1.9e86319e32323p+0, 0x1.9fa5e8d07f29ep+0,
    0x1.a0c667b5de565p+0, 0x1.a1e7aed8eb8bbp+0, 0x1.a309bec4a2d33p+0, 0x1.a42c980460ad8p+0,
    0x1.a5503b23e255dp+0, 0x1.a674a8af46052p+0, 0x1.a799e1330b358p+0, 0x1.a8bfe53c12e59p+0,
    0x1.a9e6b5579fdbfp+0, 0x1.ab0e521356ebap+0, 0x1.ac36bbfd3f37ap+0, 0x1.ad5ff3a3c2774p+0,
    0x1.ae89f995ad3adp+0, 0x1.afb4ce622f2ffp+0, 0x1.b0e07298db666p+0, 0x1.b20ce6c9a8952p+0,
    0x1.b33a2b84f15fbp+0, 0x1.b468415b749b1p+0, 0x1.b59728de5593ap+0, 0x1.b6c6e29f1c52ap+0,
    0x1.b7f76f2fb5e47p+0, 0x1.b928cf22749e4p+0, 0x1.ba5b030a1064ap+0, 0x1.bb8e0b79a6f1fp+0,
    0x1.bcc1e904bc1d2p+0, 0x1.bdf69c3f3a207p+0, 0x1.bf2c25bd71e09p+0, 0x1.c06286141b33dp+0,
    0x1.c199bdd85529cp+0, 0x1.c2d1cd9fa652cp+0, 0x1.c40ab5fffd07ap+0, 0x1.c544778fafb22p+0,
    0x1.c67f12e57d14bp+0, 0x1.c7ba88988c933p+0, 0x1.c8f6d9406e7b5p+0, 0x1.ca3405751c4dbp+0,
    0x1.cb720dcef9069p+0, 0x1.ccb0f2e6d1675p+0, 0x1.cdf0b555dc3fap+0, 0x1.cf3155b5bab74p+0,
    0x1.d072d4a07897cp+0, 0x1.d1b532b08c968p+0, 0x1.d2f87080d89f2p+0, 0x1.d43c8eacaa1d6p+0,
    0x1.d5818dcfba487p+0, 0x1.d6c76e862e6d3p+0, 0x1.d80e316c98398p+0, 0x1.d955d71ff6075p+0,
    0x1.da9e603db3285p+0, 0x1.dbe7cd63a8315p+0, 0x1.dd321f301b460p+0, 0x1.de7d5641c0658p+0,
    0x1.dfc97337b9b5fp+0, 0x1.e11676b197d17p+0, 0x1.e264614f5a129p+0, 0x1.e3b333b16ee12p+0,
    0x1.e502ee78b3ff6p+0, 0x1.e653924676d76p+0, 0x1.e7a51fbc74c83p+0, 0x1.e8f7977cdb740p+0,
    0x1.ea4afa2a490dap+0, 0x1.eb9f4867cca6ep+0, 0x1.ecf482d8e67f1p+0, 0x1.ee4aaa2188510p+0,
    0x1.efa1bee615a27p+0, 0x1.f0f9c1cb6412ap+0, 0x1.f252b376bba97p+0, 0x1.f3ac948dd7274p+0,
    0x1.f50765b6e4540p+0, 0x1.f6632798844f8p+0, 0x1.f7bfdad9cbe14p+0, 0x1.f91d802243c89p+0,
    0x1.fa7c1819e90d8p+0, 0x1.fbdba3692d514p+0, 0x1.fd3c22b8f71f1p+0, 0x1.fe9d96b2a23d9p+0
};
template <bool CHECK = false>
__device__ __forceinline__ double exp_tab(double x) {
  const double kf = fma(x, kExpC[0], kExpC[1]);                           // 256/ln2; 1.5 * 2^52 rounds to the nearest integer
  const int k = __double2loint(kf);
  const double kd = kf - kExpC[1];
  double r = fma(kd, kExpC[2], x);                                        // ln2/256, 32 leading bits (exact product)
  r = fma(kd, kExpC[3], r);                                               // ... and the rest
  const double r2 = r * r;
  double q = fma(r, kExpC[4], kExpC[5]);
  q = fma(q, r, kExpC[6]);
  const double pm1 = fma(q, r2, r);                                       // exp(r) - 1
  const double t = __ldg(kExpTab + (k & 255));
  const double y = fma(t, pm1, t);
  double res = __hiloint2double(__double2hiint(y) + ((k >> 8) << 20), __double2loint(y));
  if (CHECK) {
    const int hx = __double2hiint(x);
    if ((hx & 0x7fffffff) >= 0x4085e000) res = (hx < 0) ? 0.0 : __longlong_as_double(0x7ff0000000000000LL);
  }
  return res;
}

// toy PDF shape product f(x1) f(x2) / A^2 = (x1 x2)^pow_x ((1-x1)(1-x2))^pow_1mx (O4)
__device__ __forceinline__ double pdf_pair(const DevConst& c, double x1, double x2) {
  const double xx = x1 * x2, yy = (1.0 - x1) * (1.0 - x2);
  if (c.pdf_fast) return rsqrt_fast(xx) * (yy * yy * yy);
  return pow(xx, c.pdf_pow_x) * pow(yy, c.pdf_pow_1mx);
}

// Jet transfer functions (O5).  For x = E / E_jet, inv_x = 1 / x:
//   E * T(E_jet; E) = c1 exp(-z1^2) + c2 exp(-z2^2) = exp(-z1^2) (c1 + c2 exp(z1^2 - z2^2)),  z_k = a_k inv_x + b_k
// (the factor 1/E of the Gaussians cancels the E of the jet's measure E sin(theta) dE).  A product
// over jets therefore needs one exponential per jet plus ONE for the sum of the z1^2 (and any
// other Gaussian factor of the point, e.g. the MET transfer function): tf_accum() adds z1^2 to
// `esum` and multiplies `fac` by the bracket; the caller finishes with fac * exp(-esum).
template <typename T> struct TfAcc { T esum, fac; };

// ---------------------------------------------------------------------------------------
// fp32 counterparts (reading A15: the integrand core of config 3 in single precision; sampling,
// per-event constants, the overall constant C0 and the sums stay in fp64).  MUFU-based
// reciprocal / rsqrt / exp2; no --use_fast_math anywhere, these are chosen per call site.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ float rcp_fast(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));      // one MUFU, 1 ulp: ample for the 1e-4 bar
  return y;
}
// tan for the Breit-Wigner map in fp32: same scheme as tan_bw_n (no range reduction beyond pi/2 - |t|),
// degree-9 / degree-8 polynomials (Taylor coefficients; the remainders are below 2e-8 on |r| <= pi/4)
__device__ __forceinline__ float tan_bw(float t) {
  const float a = fabsf(t);
  const bool big = a > 0.78539816f;
  const float r = big ? (1.57079637f - a) - 4.37113883e-8f : a, z = r * r;
  float ps = 2.75573192e-6f, pc = 2.48015873e-5f;
  ps = fmaf(ps, z, -1.98412698e-4f); pc = fmaf(pc, z, -1.38888889e-3f);
  ps = fmaf(ps, z, 8.33333333e-3f);  pc = fmaf(pc, z, 4.16666667e-2f);
  ps = fmaf(ps, z, -1.66666667e-1f);
  const float sn = fmaf(r * z, ps, r), cs = fmaf(z * z, pc, fmaf(-0.5f, z, 1.0f));
  const float q = (big ? cs : sn) * rcp_fast(big ? sn : cs);
  return copysignf(q, t);
}
__device__ __forceinline__ double m_exp(double x) { return exp(x); }
__device__ __forceinline__ float m_exp(float x) { return __expf(x); }
__device__ __forceinline__ double m_tan(double x) { return tan_bw(x); }
__device__ __forceinline__ float m_tan(float x) { return tan_bw(x); }
__device__ __forceinline__ double m_rsqrt(double x) { return rsqrt_fast(x); }
__device__ __forceinline__ float m_rsqrt(float x) { return rsqrtf(x); }

// NEXT-3 (listing :274-306, reading A17): one species of the grid PDF at ln x = L.
// Cell index as in the listing: 0 below the grid, clamped to nx - 2 above (the edge cell is
// extrapolated); linear in ln x between the two samples (the ln Q direction was folded in on the host).
__device__ __forceinline__ double pdf_grid_1d(const double* __restrict__ tab, int nx, double lxmin, double dx,
                                              double inv_dx, double L) {
  int ix = 0;
  if (lxmin < L) ix = (int)((L - lxmin) * inv_dx);
  ix = ix < nx - 1 ? ix : nx - 2;
  const double c11 = fma(dx, (double)ix, lxmin), c22 = fma(dx, (double)(ix + 1), lxmin);
  return fma(__ldg(tab + ix), c22 - L, __ldg(tab + ix + 1) * (L - c11)) * inv_dx;
}

// Flavour sum of t tbar production: sum_ab f_a(x1) f_b(x2) |M_ab|^2 = Lgg Mgg + Lqq Mqq with
// Mqq = tau1^2 + tau2^2 + rho/2 (the colour factor 4/9 is folded into Lqq).  Toy mode (O4): every
// species has the same shape; grid mode: g g, and q qbar + qbar q for the first n_flav species.
// GRIDPDF = false compiles the toy branch only (the hot kernels are instantiated both ways and the
// launch picks one: carrying the table code costs 1-4 % even when it is not taken).
template <typename T> struct TtLumi { T gg, qq; };
// rsxx = (x1 x2)^(-1/2) when the caller has it already (toy PDF with the default exponents), else < 0
template <bool GRIDPDF, typename T>
__device__ __forceinline__ TtLumi<T> tt_lumi(const DevConstR<T>& c, T x1, T x2, T rsxx = T(-1)) {
  if (!GRIDPDF || c.pdf_tab == nullptr) {
    T ff;
    if (c.pdf_fast && rsxx > T(0)) { const T yy = (T(1) - x1) * (T(1) - x2); ff = rsxx * (yy * yy * yy); }
    else ff = pdf_pair(c, x1, x2);
    return {ff * c.A_g2, ff * ((T(2.0) * c.n_flav * (T(4.0) / T(9.0))) * c.A_q2)};
  }
  const double L1 = log((double)x1), L2 = log((double)x2);
  const double* t = c.pdf_tab;
  const double gg = pdf_grid_1d(t, c.pdf_nx, c.pdf_lxmin, c.pdf_dx, c.pdf_inv_dx, L1) *
                    pdf_grid_1d(t, c.pdf_nx, c.pdf_lxmin, c.pdf_dx, c.pdf_inv_dx, L2);
  double qq = 0.0;
  for (int f = 1; f <= c.n_flav; ++f)
    qq = fma(pdf_grid_1d(t + f * c.pdf_nx, c.pdf_nx, c.pdf_lxmin, c.pdf_dx, c.pdf_inv_dx, L1),
             pdf_grid_1d(t + f * c.pdf_nx, c.pdf_nx, c.pdf_lxmin, c.pdf_dx, c.pdf_inv_dx, L2), qq);
  return {(T)gg, (T)(qq * (2.0 * 4.0 / 9.0))};
}

// the outer exponential of a product of Gaussians: its argument may run below the range of exp (the result is then 0)
template <bool TAB> __device__ __forceinline__ double x_exp(double x) { return TAB ? exp_tab<true>(x) : exp(x); }
template <bool TAB> __device__ __forceinline__ float x_exp(float x) { return m_exp(x); }
// an exponential whose argument is bounded by construction (|eta_nu| <= nu_eta_max <= 50)
template <bool TAB> __device__ __forceinline__ double b_exp(double x) { return TAB ? exp_tab<false>(x) : exp(x); }
template <bool TAB> __device__ __forceinline__ float b_exp(float x) { return m_exp(x); }

// TAB: exp_tab instead of libdevice's exp (fp64 only).  Every integrate kernel is instantiated with TAB = true
// (mem_kernels.cuh); TAB = false is passed only at the fp32 variant's call sites, where the flag has no effect.
// Measured when it went in: configs 2 and 4 gain 5.7 % and 5.8 %, the VEGAS passes 3 %.
template <bool TAB = false, typename T>
__device__ __forceinline__ void tf_accum(const DevConstR<T>& c, T inv_x, TfAcc<T>& acc) {
  // fp64: z1^2 - z2^2 as a quadratic in inv_x (coefficients tf_q2, tf_q1, tf_q0 from the host): four FP64
  // instructions per jet besides the exponential instead of five
  const T z1 = fma(c.tf_a1, inv_x, c.tf_b1);
  acc.esum = fma(z1, z1, acc.esum);
  T arg;
  if constexpr (std::is_same<T, double>::value) {
    arg = fma(fma(c.tf_q2, inv_x, c.tf_q1), inv_x, c.tf_q0);
  } else {                                    // fp32: the expanded quadratic cancels too much
    const T z2 = fma(c.tf_a2, inv_x, c.tf_b2);
    arg = fma(-z2, z2, z1 * z1);
  }
  T e;
  if constexpr (TAB && std::is_same<T, double>::value) e = exp_tab(arg);
  else e = m_exp(arg);
  acc.fac *= fma(c.tf_c2, e, c.tf_c1);
}

__device__ __forceinline__ float pdf_pair(const DevConstF& c, float x1, float x2) {
  const float xx = x1 * x2, yy = (1.0f - x1) * (1.0f - x2);
  if (c.pdf_fast) return rsqrtf(xx) * (yy * yy * yy);
  return powf(xx, c.pdf_pow_x) * powf(yy, c.pdf_pow_1mx);
}


// ---------------------------------------------------------------------------------------
// S8. block reduction of (sum w, sum w^2): registers -> warp shuffle tree -> shared -> warp 0,
// fixed order, so results are bitwise reproducible.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// returns the block totals in thread 0
__device__ __forceinline__ void block_sum2(double& s1, double& s2, double* sh /* [2 * kWarps] */) {
  s1 = warp_sum(s1);
  s2 = warp_sum(s2);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) { sh[warp] = s1; sh[kWarps + warp] = s2; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) { a += sh[w]; b += sh[kWarps + w]; }
    s1 = a; s2 = b;
  }
}

}  // namespace memb200
