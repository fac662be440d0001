// sc_math.cuh -- device-side model arithmetic of the semi-coherent statistic (sm_100a).
//
// What is evaluated HERE runs only at the coarse nodes (one node per `stride` FFT bins, the paper's
// "sparse grid") and in the per-particle set-up; the dense per-bin loop lives in sc_stat.cu.
// Formulas: readings O2 (TaylorF2 phase), O3 (t(f)), O4 (orbit, single link, TDI-1 A/E) of SURVEY.md 8(c),
// restated in DESIGN.md; the paper itself names the models and prints no formula.
// This file shares nothing with oracle/ (which is test infrastructure).
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

namespace sc {

constexpr double kPi = 3.141592653589793238462643383279502884;
constexpr double kEulerGamma = 0.577215664901532860606512090082402431;
constexpr double kMsunSec = 4.925491025543576e-06;   // G Msun / c^3 [s]

// Run-time description of the problem handed to every kernel by value.
struct DevCfg {
  double T_obs, inv_T;          // observation time [s], df
  long long j0;                 // f_j = (j0 + j) / T_obs
  int n_bins;
  int window_mode, pn_order_x2, ecc_leading;
  double f_ref_ecc;
  double L, AU, alpha0, year;   // arm length, AU [s]; initial orbital phase [rad]; year [s]
  double sbn[3], cbn[3];        // sin, cos of beta_n = 2 pi (n-1)/3 + lambda0
  double f_amp_ref;             // amplitude normalisation: A(f) = (f / f_amp_ref)^(-7/6)
  int log2_stride, stride;      // coarse node spacing in bins (power of two, >= 4)
  int n_nodes;                  // nodes i = -kNodeOff .. n_intervals + 3
  int chan_set;                 // 0: the node amplitudes are (A, E); 1: (T, 0) -- the T pass of a three-channel handle;
                                // 2: (A, E, T) -- the fused three-channel kernel (k_dense3)
};
// Each coarse interval is cut into 4 fine sub-intervals (stride/4 bins) on which the amplitudes are local cubics.
constexpr int kNodeOff = 2;     // the quintic phase stencil reaches 2 nodes to the left, 3 to the right

// Per-particle constants (a1): SoA table, field-major, [kPcFields][P_pad].
enum PcField { PC_PIM = 0, PC_ETA, PC_TC, PC_TAU_HI, PC_TAU_LO, PC_CL, PC_SL, PC_CB, PC_SB, PC_C2P, PC_S2P, PC_CI,
               PC_ECC, kPcFields };

struct Particle {
  double piM, eta, tc, tau_hi, tau_lo, cl, sl, cb, sb, c2p, s2p, ci, ecc;
};

__device__ __forceinline__ Particle load_particle(const double* __restrict__ pc, int P_pad, int p) {
  Particle q;
  q.piM = pc[PC_PIM * (size_t)P_pad + p];       q.eta = pc[PC_ETA * (size_t)P_pad + p];
  q.tc = pc[PC_TC * (size_t)P_pad + p];         q.tau_hi = pc[PC_TAU_HI * (size_t)P_pad + p];
  q.tau_lo = pc[PC_TAU_LO * (size_t)P_pad + p]; q.cl = pc[PC_CL * (size_t)P_pad + p];
  q.sl = pc[PC_SL * (size_t)P_pad + p];         q.cb = pc[PC_CB * (size_t)P_pad + p];
  q.sb = pc[PC_SB * (size_t)P_pad + p];         q.c2p = pc[PC_C2P * (size_t)P_pad + p];
  q.s2p = pc[PC_S2P * (size_t)P_pad + p];       q.ci = pc[PC_CI * (size_t)P_pad + p];
  q.ecc = pc[PC_ECC * (size_t)P_pad + p];
  return q;
}

// O2/O3: the PN sums  S(v) = sum_k psi_k v^(k-5)  and  B(v) = 3 f d/df S  (so that dS/df = B/(3f)).
// SKIP0: S without its k = 0 (Newtonian) term, which eval_node adds in extended precision.
template <bool SKIP0 = false>
__device__ __forceinline__ void pn_sums(double eta, double v, int order, double& S, double& B) {
  const double lv = log(v);
  const double eta2 = eta * eta;
  const double P5 = kPi * (38645.0 / 756.0 - 65.0 * eta / 9.0);
  double psi[8];
  psi[0] = 1.0;
  psi[1] = 0.0;
  psi[2] = 3715.0 / 756.0 + 55.0 * eta / 9.0;
  psi[3] = -16.0 * kPi;
  psi[4] = 15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta2 / 72.0;
  psi[5] = P5 * (1.0 + 3.0 * lv);
  psi[6] = 11583231236531.0 / 4694215680.0 - 640.0 * kPi * kPi / 3.0 - 6848.0 * kEulerGamma / 21.0
           - (6848.0 / 21.0) * (1.3862943611198906 + lv)
           + (-15737765635.0 / 3048192.0 + 2255.0 * kPi * kPi / 12.0) * eta
           + 76055.0 * eta2 / 1728.0 - 127825.0 * eta2 * eta / 1296.0;
  psi[7] = kPi * (77096675.0 / 254016.0 + 378515.0 * eta / 1512.0 - 74045.0 * eta2 / 756.0);
  const double v2 = v * v;
  double vp = 1.0 / (v2 * v2 * v);   // v^-5
  S = 0.0; B = 0.0;
#pragma unroll
  for (int k = 0; k <= 7; ++k) {
    if (k <= order) {
      if (!(SKIP0 && k == 0)) S = fma(psi[k], vp, S);
      if (k == 5) B += 3.0 * P5;                                   // vp = 1 here
      else if (k == 6) B = fma(psi[6] - 6848.0 / 21.0, vp, B);      // vp = v
      else B = fma((double)(k - 5) * psi[k], vp, B);
    }
    vp *= v;
  }
}

// O3: t(f) [s], direct evaluation (used for the window search and at the nodes).
__device__ __forceinline__ double tf_direct(const DevCfg& c, const Particle& q, double f) {
  const double v = cbrt(q.piM * f);
  double S, B;
  pn_sums(q.eta, v, c.pn_order_x2, S, B);
  const double pref = 3.0 / (128.0 * q.eta) / (2.0 * kPi);        // phase prefactor in turns
  double t = q.tc + pref * B / (3.0 * f);
  if (c.ecc_leading) {
    const double e_t = -pref * q.ecc * pow(v, -34.0 / 3.0);        // eccentric phase term in turns, ~ f^(-34/9)
    t += e_t * (-34.0 / 9.0) / f;
  }
  return t;
}

// One coarse node: fast phase (integer + fractional turns), t_f, and the slowly varying complex amplitudes.
//   h_alpha(f) = amp_alpha(f) * f_amp_ref^(-7/6) * exp(-2 pi i Phi(f)),
//   Phi = Psi/(2 pi) + f k.p0(t_f)   (PN phase plus the Doppler phase of the constellation centroid),
//   amp_alpha = T_alpha * exp(+2 pi i f k.p0) * (f/f_amp_ref)^(-7/6)      (everything annual-period smooth).
struct NodeOut {
  int n_turns;        // integer part of Phi
  double frac;        // fractional part, |frac| <= 0.5
  double Ar, Ai, Er, Ei;
  double Tr, Ti;      // T = (X + Y + Z)/sqrt(3) (chan_set = 2 only)
};


// sin(x)/x given sin x from an angle-addition formula (absolute error ~1e-16): near x = 0 the quotient would lose
// relative accuracy, so the series takes over below 1e-2 (next term x^6/5040 < 2e-16).
__device__ __forceinline__ double sinc_from(double x, double sin_x) {
  const double x2 = x * x;
  return (x2 < 1.0e-4) ? fma(x2, fma(x2, 1.0 / 120.0, -1.0 / 6.0), 1.0) : sin_x / x;
}

// Double-double helpers for the Newtonian phase term (products by error-free transformation; the intrinsics keep the
// compiler from contracting them).
struct dd2 { double hi, lo; };
__device__ __forceinline__ dd2 dd_two_prod(double a, double b) { const double p = __dmul_rn(a, b); return {p, fma(a, b, -p)}; }
__device__ __forceinline__ dd2 dd_mul(dd2 a, dd2 b) {
  const double p = __dmul_rn(a.hi, b.hi);
  double e = fma(a.hi, b.hi, -p);
  e = fma(a.hi, b.lo, e);
  e = fma(a.lo, b.hi, e);
  const double s = __dadd_rn(p, e);
  return {s, __dadd_rn(e, -__dadd_rn(s, -p))};
}
// The Newtonian term of the phase, pref (pi M f)^(-5/3) turns, reaches 4e6 turns (c5: 0.01 Hz, M_c = 24 Msun): plain FP64
// (cbrt, five products, one reciprocal: ~4e-16 relative, independent from node to node) leaves 1e-8 rad per node, which is
// the whole error budget of the all-FP64 path at small Upsilon (found with the oracle's long-double mode: 1.05e-6 at
// Upsilon = 1.2e-3 on c5).  Here: u = (pi M / T) n as an exact product, y0 = u^(-5/3) in FP64, one Newton step on
// y^3 u^5 = 1 with the residual formed in double-double, and the product with pref split into integer turns + fraction.
// (Rounding of pi M / T and of pref is the same at every node: a 1e-16 relative shift of M_c, harmless.)
__device__ __forceinline__ void newtonian_turns(double piM_over_T, double n, double pref, double& int_turns, double& frac) {
  const dd2 u = dd_two_prod(piM_over_T, n);
  const double v0 = cbrt(u.hi);
  const double v02 = v0 * v0;
  const double y0 = 1.0 / (v02 * v02 * v0);
  const dd2 y2 = dd_two_prod(y0, y0);
  const dd2 y3 = dd_mul(y2, dd2{y0, 0.0});
  const dd2 u2 = dd_mul(u, u);
  const dd2 u5 = dd_mul(dd_mul(u2, u2), u);
  const dd2 pr = dd_mul(y3, u5);                                  // = 1 + r
  const double r = __dadd_rn(__dadd_rn(pr.hi, -1.0), pr.lo);
  const double y_lo = -y0 * r * (1.0 / 3.0);                      // y = y0 (1 - r/3)
  const dd2 a = dd_two_prod(pref, y0);
  int_turns = rint(a.hi);
  frac = __dadd_rn(a.hi, -int_turns) + fma(pref, y_lo, a.lo);
}

__device__ NodeOut eval_node(const DevCfg& c, const Particle& q, long long jglob /* j0 + bin position */) {
  NodeOut o;
  o.Tr = 0.0; o.Ti = 0.0;
  const double n = (double)jglob;
  const double f = n * c.inv_T;
  // --- O2 phase in turns.  The 2 pi f t_c term reaches ~5e6 turns: take its fractional part exactly,
  //     f t_c = n * (t_c/T) with t_c/T split as tau_hi + tau_lo and the product error recovered by FMA.
  const double p = n * q.tau_hi;
  const double perr = fma(n, q.tau_hi, -p);
  const double ip = rint(p);
  double frac = (p - ip) + (perr + n * q.tau_lo);
  const double v = cbrt(q.piM * f);
  double S, B;
  pn_sums<true>(q.eta, v, c.pn_order_x2, S, B);                   // S: the terms beyond the Newtonian one (<= 2e4 turns)
  const double pref = 3.0 / (128.0 * q.eta) / (2.0 * kPi);
  double i0, f0;
  newtonian_turns(q.piM * c.inv_T, n, pref, i0, f0);
  const double pn_t = pref * S;
  const double ipn = rint(pn_t);
  frac += (pn_t - ipn) + f0;
  double tf = q.tc + pref * B / (3.0 * f);
  if (c.ecc_leading) {
    const double e_t = -pref * q.ecc * pow(v, -34.0 / 3.0);
    frac += e_t;
    tf += e_t * (-34.0 / 9.0) / f;
  }
  // --- O4 orbit at t_f
  double sa, ca;
  sincos(2.0 * kPi * tf / c.year + c.alpha0, &sa, &ca);
  // Doppler phase of the centroid: f k.p0 = -f AU cos(beta) cos(alpha - lambda)
  frac += -f * c.AU * q.cb * (ca * q.cl + sa * q.sl) - 0.125;      // -pi/4 of the SPA
  const double ir = rint(frac);
  o.n_turns = (int)(ip + ipn + i0 + ir);
  o.frac = frac - ir;

  const double aue = c.L / (2.0 * 1.7320508075688772);             // AU * e
  double d[3][3];
#pragma unroll
  for (int m = 0; m < 3; ++m) {
    d[m][0] = aue * (sa * ca * c.sbn[m] - (1.0 + sa * sa) * c.cbn[m]);
    d[m][1] = aue * (sa * ca * c.cbn[m] - (1.0 + ca * ca) * c.sbn[m]);
    d[m][2] = -1.7320508075688772 * aue * (ca * c.cbn[m] + sa * c.sbn[m]);
  }
  const double kx = -q.cb * q.cl, ky = -q.cb * q.sl, kz = -q.sb;
  const double ux = -q.sb * q.cl, uy = -q.sb * q.sl, uz = q.cb;
  const double vx = -q.sl, vy = q.cl;
  const double pfl = kPi * f * c.L;
  // sin, cos of pi f L once per node: the six sinc arguments pfl (1 -+ k.n) and the delay D = e^{-2 i pfl} follow by the
  // angle-addition formulas (one sincos of pfl k.n per arm instead of two sines, none for D)
  double sp, cp;
  sincos(pfl, &sp, &cp);
  // arms (s, r) = (1,2), (2,3), (3,1): y_sr and y_rs share zeta and the phase factor
  double ysr[3][2], yrs[3][2];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const int s = a, r = (a + 1) % 3;
    double nx = d[r][0] - d[s][0], ny = d[r][1] - d[s][1], nz = d[r][2] - d[s][2];
    const double inv = rsqrt(nx * nx + ny * ny + nz * nz);
    nx *= inv; ny *= inv; nz *= inv;
    const double nu = nx * ux + ny * uy + nz * uz, nv = nx * vx + ny * vy, kn = nx * kx + ny * ky + nz * kz;
    const double ep = nu * nu - nv * nv, ex = 2.0 * nu * nv;
    const double Fp = q.c2p * ep + q.s2p * ex, Fx = -q.s2p * ep + q.c2p * ex;
    const double zr = 0.5 * (1.0 + q.ci * q.ci) * Fp, zi = -q.ci * Fx;
    const double kd = kx * (d[r][0] + d[s][0]) + ky * (d[r][1] + d[s][1]) + kz * (d[r][2] + d[s][2]);
    double es, ec;
    sincos(-kPi * f * (c.L + kd), &es, &ec);
    const double wr = ec * zr - es * zi, wi = ec * zi + es * zr;
    double sb, cb;
    sincos(pfl * kn, &sb, &cb);
    const double a_sr = pfl * sinc_from(pfl * (1.0 - kn), fma(sp, cb, -(cp * sb)));
    const double a_rs = pfl * sinc_from(pfl * (1.0 + kn), fma(sp, cb, cp * sb));
    ysr[a][0] = a_sr * wi; ysr[a][1] = -a_sr * wr;      // -i a (wr + i wi)
    yrs[a][0] = a_rs * wi; yrs[a][1] = -a_rs * wr;
  }
  const double Dr = fma(-2.0 * sp, sp, 1.0), Di = -2.0 * sp * cp;   // D = e^{-2 pi i f L} = cos 2 pfl - i sin 2 pfl
  const double gr = 1.0 - (Dr * Dr - Di * Di), gi = -2.0 * Dr * Di;
  // y12 = ysr[0], y21 = yrs[0], y23 = ysr[1], y32 = yrs[1], y31 = ysr[2], y13 = yrs[2]
  // X = (1-D^2)[(y31 + D y13) - (y21 + D y12)], Y, Z cyclic
  double XYZ[3][2];
#pragma unroll
  for (int m = 0; m < 3; ++m) {
    const int aIn = (m + 2) % 3;    // arm (c,a): y_ca = ysr[aIn], y_ac = yrs[aIn]
    const int aOut = m;             // arm (a,b): y_ab = ysr[aOut], y_ba = yrs[aOut]
    const double tr = (ysr[aIn][0] + Dr * yrs[aIn][0] - Di * yrs[aIn][1]) - (yrs[aOut][0] + Dr * ysr[aOut][0] - Di * ysr[aOut][1]);
    const double ti = (ysr[aIn][1] + Dr * yrs[aIn][1] + Di * yrs[aIn][0]) - (yrs[aOut][1] + Dr * ysr[aOut][1] + Di * ysr[aOut][0]);
    XYZ[m][0] = gr * tr - gi * ti;
    XYZ[m][1] = gr * ti + gi * tr;
  }
  const double fr = f / c.f_amp_ref;
  const double amp = 1.0 / (fr * cbrt(sqrt(fr)));                   // (f/f_ref)^(-7/6)
  const double s2 = 0.7071067811865476 * amp, s6 = 0.4082482904638631 * amp;
  if (c.chan_set == 1) {                                             // T = (X + Y + Z)/sqrt(3) in the first slot
    const double s3 = 0.5773502691896258 * amp;
    o.Ar = (XYZ[0][0] + XYZ[1][0] + XYZ[2][0]) * s3;
    o.Ai = (XYZ[0][1] + XYZ[1][1] + XYZ[2][1]) * s3;
    o.Er = 0.0; o.Ei = 0.0;
    return o;
  }
  if (c.chan_set == 2) {
    const double s3 = 0.5773502691896258 * amp;
    o.Tr = (XYZ[0][0] + XYZ[1][0] + XYZ[2][0]) * s3;
    o.Ti = (XYZ[0][1] + XYZ[1][1] + XYZ[2][1]) * s3;
  }
  o.Ar = (XYZ[2][0] - XYZ[0][0]) * s2;
  o.Ai = (XYZ[2][1] - XYZ[0][1]) * s2;
  o.Er = (XYZ[0][0] - 2.0 * XYZ[1][0] + XYZ[2][0]) * s6;
  o.Ei = (XYZ[0][1] - 2.0 * XYZ[1][1] + XYZ[2][1]) * s6;
  return o;
}

// Quintic through 6 equispaced phase nodes m = -2..3 (Y_m = Phi_m - Phi_0 in turns, Y_0 = 0):
// monomial coefficients in bins, b[1..5] (b[0] = 0), h = 1/stride.
__device__ __forceinline__ void quintic_coeffs(const double Y[6], double h, double b[6]) {
  const double ym2 = Y[0], ym1 = Y[1], y1 = Y[3], y2 = Y[4], y3 = Y[5];
  const double a1 = ym2 * (1.0 / 20.0) - ym1 * 0.5 + y1 - y2 * 0.25 + y3 * (1.0 / 30.0);
  const double a2 = -ym2 * (1.0 / 24.0) + ym1 * (2.0 / 3.0) + y1 * (2.0 / 3.0) - y2 * (1.0 / 24.0);
  const double a3 = -ym2 * (1.0 / 24.0) - ym1 * (1.0 / 24.0) - y1 * (7.0 / 12.0) + y2 * (7.0 / 24.0) - y3 * (1.0 / 24.0);
  const double a4 = ym2 * (1.0 / 24.0) - ym1 * (1.0 / 6.0) - y1 * (1.0 / 6.0) + y2 * (1.0 / 24.0);
  const double a5 = -ym2 * (1.0 / 120.0) + ym1 * (1.0 / 24.0) + y1 * (1.0 / 12.0) - y2 * (1.0 / 24.0) + y3 * (1.0 / 120.0);
  const double h2 = h * h;
  b[0] = 0.0; b[1] = a1 * h; b[2] = a2 * h2; b[3] = a3 * h2 * h; b[4] = a4 * h2 * h2; b[5] = a5 * h2 * h2 * h;
}

// Forward differences of sum_k b_k u^k at u = 0 for unit steps: d_j = j! * sum_k S2(k, j) b_k.
__device__ __forceinline__ void forward_diffs(const double b[6], double d[6]) {
  d[1] = b[1] + b[2] + b[3] + b[4] + b[5];
  d[2] = 2.0 * b[2] + 6.0 * b[3] + 14.0 * b[4] + 30.0 * b[5];
  d[3] = 6.0 * b[3] + 36.0 * b[4] + 150.0 * b[5];
  d[4] = 24.0 * b[4] + 240.0 * b[5];
  d[5] = 120.0 * b[5];
}

// In-place Taylor shift of sum_k b_k u^k to sum_k b'_k (u - u0)^k.
__device__ __forceinline__ void taylor_shift(double b[6], double u0) {
#pragma unroll
  for (int i = 0; i < 5; ++i)
#pragma unroll
    for (int j = 4; j >= i; --j) b[j] = fma(u0, b[j + 1], b[j]);
}

// Quintic Lagrange weights of the 6 nodes m = -2..3 at s = -1/4, 0, 1/4, 1/2, 3/4, 1, 5/4 (all dyadic: exact in FP32).
__device__ constexpr double kSampleW[7][6] = {
    {-117.0 / 8192, 1365.0 / 8192, 4095.0 / 4096, -819.0 / 4096, 455.0 / 8192, -63.0 / 8192},
    {0, 0, 1, 0, 0, 0},
    {77.0 / 8192, -693.0 / 8192, 3465.0 / 4096, 1155.0 / 4096, -495.0 / 8192, 63.0 / 8192},
    {3.0 / 256, -25.0 / 256, 75.0 / 128, 75.0 / 128, -25.0 / 256, 3.0 / 256},
    {63.0 / 8192, -495.0 / 8192, 1155.0 / 4096, 3465.0 / 4096, -693.0 / 8192, 77.0 / 8192},
    {0, 0, 0, 1, 0, 0},
    {-63.0 / 8192, 455.0 / 8192, -819.0 / 4096, 4095.0 / 4096, 1365.0 / 8192, -117.0 / 8192}};

// Amplitude on fine sub-interval q (0..3) of a coarse interval: the quintic through the 6 coarse nodes is sampled
// at s = (q-1)/4 .. (q+2)/4 and replaced by the cubic through those 4 samples, in t = (u - q stride/4)/(stride/4).
template <typename R>
__device__ __forceinline__ void fine_cubic(const R node[6], int q, R& a0, R& a1, R& a2, R& a3) {
  R smp[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    R acc = R(0.0);
#pragma unroll
    for (int m = 0; m < 6; ++m) acc = fma((R)kSampleW[q + i][m], node[m], acc);
    smp[i] = acc;
  }
  a0 = smp[1];
  a1 = -smp[0] * R(1.0 / 3.0) - smp[1] * R(0.5) + smp[2] - smp[3] * R(1.0 / 6.0);
  a2 = smp[0] * R(0.5) - smp[1] + smp[2] * R(0.5);
  a3 = -smp[0] * R(1.0 / 6.0) + smp[1] * R(0.5) - smp[2] * R(0.5) + smp[3] * R(1.0 / 6.0);
}

// The same map as fine_cubic written as one 4 x 6 matrix per sub-interval q: cubic coefficient k = sum_m kFineM[q][k][m]
// node[m] (the product of the cubic-fit matrix and the sampling weights above, exact rationals).  Row 0 sums to 1 and
// rows 1..3 sum to 0, so the rows may be applied to node[m] - node[2] (see fine_cubic2 in sc_stat.cu).
__device__ constexpr float kFineM[4][4][6] = {
  {{0.0, 0.0, 1.0, 0.0, 0.0, 0.0},
   {25.0 / 2048, -761.0 / 6144, -87.0 / 1024, 257.0 / 1024, -385.0 / 6144, 17.0 / 2048},
   {-5.0 / 2048, 21.0 / 512, -79.0 / 1024, 21.0 / 512, -5.0 / 2048, 0.0},
   {-3.0 / 8192, -43.0 / 24576, 33.0 / 4096, -41.0 / 4096, 115.0 / 24576, -5.0 / 8192}},
  {{77.0 / 8192, -693.0 / 8192, 3465.0 / 4096, 1155.0 / 4096, -495.0 / 8192, 63.0 / 8192},
   {47.0 / 8192, -371.0 / 8192, -2671.0 / 12288, 1245.0 / 4096, -437.0 / 8192, 155.0 / 24576},
   {-29.0 / 8192, 293.0 / 8192, -217.0 / 4096, 45.0 / 4096, 95.0 / 8192, -15.0 / 8192},
   {1.0 / 8192, -29.0 / 8192, 127.0 / 12288, -45.0 / 4096, 37.0 / 8192, -11.0 / 24576}},
  {{3.0 / 256, -25.0 / 256, 75.0 / 128, 75.0 / 128, -25.0 / 256, 3.0 / 256},
   {-1.0 / 768, 17.0 / 1024, -75.0 / 256, 449.0 / 1536, -1.0 / 64, 1.0 / 1024},
   {-13.0 / 4096, 103.0 / 4096, -45.0 / 2048, -45.0 / 2048, 103.0 / 4096, -13.0 / 4096},
   {11.0 / 24576, -37.0 / 8192, 45.0 / 4096, -127.0 / 12288, 29.0 / 8192, -1.0 / 8192}},
  {{63.0 / 8192, -495.0 / 8192, 1155.0 / 4096, 3465.0 / 4096, -693.0 / 8192, 77.0 / 8192},
   {-53.0 / 8192, 1315.0 / 24576, -1241.0 / 4096, 881.0 / 4096, 1157.0 / 24576, -51.0 / 8192},
   {-15.0 / 8192, 95.0 / 8192, 45.0 / 4096, -217.0 / 4096, 293.0 / 8192, -29.0 / 8192},
   {5.0 / 8192, -115.0 / 24576, 41.0 / 4096, -33.0 / 4096, 43.0 / 24576, 3.0 / 8192}}};
// The same matrix in FP64 (the FP64 edge decision of the per-particle-segment path).
__device__ constexpr double kFineMd[4][4][6] = {
  {{0.0, 0.0, 1.0, 0.0, 0.0, 0.0},
   {25.0 / 2048, -761.0 / 6144, -87.0 / 1024, 257.0 / 1024, -385.0 / 6144, 17.0 / 2048},
   {-5.0 / 2048, 21.0 / 512, -79.0 / 1024, 21.0 / 512, -5.0 / 2048, 0.0},
   {-3.0 / 8192, -43.0 / 24576, 33.0 / 4096, -41.0 / 4096, 115.0 / 24576, -5.0 / 8192}},
  {{77.0 / 8192, -693.0 / 8192, 3465.0 / 4096, 1155.0 / 4096, -495.0 / 8192, 63.0 / 8192},
   {47.0 / 8192, -371.0 / 8192, -2671.0 / 12288, 1245.0 / 4096, -437.0 / 8192, 155.0 / 24576},
   {-29.0 / 8192, 293.0 / 8192, -217.0 / 4096, 45.0 / 4096, 95.0 / 8192, -15.0 / 8192},
   {1.0 / 8192, -29.0 / 8192, 127.0 / 12288, -45.0 / 4096, 37.0 / 8192, -11.0 / 24576}},
  {{3.0 / 256, -25.0 / 256, 75.0 / 128, 75.0 / 128, -25.0 / 256, 3.0 / 256},
   {-1.0 / 768, 17.0 / 1024, -75.0 / 256, 449.0 / 1536, -1.0 / 64, 1.0 / 1024},
   {-13.0 / 4096, 103.0 / 4096, -45.0 / 2048, -45.0 / 2048, 103.0 / 4096, -13.0 / 4096},
   {11.0 / 24576, -37.0 / 8192, 45.0 / 4096, -127.0 / 12288, 29.0 / 8192, -1.0 / 8192}},
  {{63.0 / 8192, -495.0 / 8192, 1155.0 / 4096, 3465.0 / 4096, -693.0 / 8192, 77.0 / 8192},
   {-53.0 / 8192, 1315.0 / 24576, -1241.0 / 4096, 881.0 / 4096, 1157.0 / 24576, -51.0 / 8192},
   {-15.0 / 8192, 95.0 / 8192, 45.0 / 4096, -217.0 / 4096, 293.0 / 8192, -29.0 / 8192},
   {5.0 / 8192, -115.0 / 24576, 41.0 / 4096, -33.0 / 4096, 43.0 / 24576, 3.0 / 8192}}};

// Cubic through 4 equispaced nodes m = -1..2 in s = u/stride: a0 + a1 s + a2 s^2 + a3 s^3.
template <typename R>
__device__ __forceinline__ void cubic_coeffs(R cm1, R c0, R c1, R c2, R& a0, R& a1, R& a2, R& a3) {
  a0 = c0;
  a1 = -cm1 * R(1.0 / 3.0) - c0 * R(0.5) + c1 - c2 * R(1.0 / 6.0);
  a2 = cm1 * R(0.5) - c0 + c1 * R(0.5);
  a3 = -cm1 * R(1.0 / 6.0) + c0 * R(0.5) - c1 * R(0.5) + c2 * R(1.0 / 6.0);
}

// Philox4x32-10 (Salmon et al., SC'11), restated from the published algorithm.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

}  // namespace sc
