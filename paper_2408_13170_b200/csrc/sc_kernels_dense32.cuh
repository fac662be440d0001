// sc_kernels_dense32.cuh -- a4 + a5, FP32-amplitude flavour of the hot loop: packed FP32x2 (FFMA2) bin pairs, FP64 phase.
// Part of libscstat.so (one translation unit: sc_stat.cu includes the kernel files in pipeline order).
#pragma once
#include "sc_common.cuh"

namespace {

// ------------------------------------------------------------------------------------------------ a4 + a5, FP32x2
// The FP32-amplitude flavour of the hot loop, written for the packed FP32 pipe of sm_100a (FFMA2 / FMUL2 / FADD2:
// one issue slot carries two FP32 operations).  Each lane (= particle) walks its chunk two bins at a time: the low
// half of every packed register belongs to the even bin 2m, the high half to the odd bin 2m+1, so the whole
// per-bin arithmetic (amplitude cubics, the complex multiply-accumulate with the data, |h|^2) is element-wise and
// needs no swizzle.  Segment edges on odd bins split a pair between two segments (the pair is evaluated once).
// Phase: per fine sub-interval the 6-node quintic is economised (Chebyshev) to a cubic and advanced by forward
// differences, 3 FP64 adds per bin; the fraction of a turn is read from the low word of phi + 1.5 * 2^20.
typedef unsigned long long u64;
__device__ __forceinline__ u64 f2pack(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void f2unpack(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 f2fma(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ u64 f2mul(u64 a, u64 b) { u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 f2add(u64 a, u64 b) { u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 f2neg(u64 a) { float lo, hi; f2unpack(a, lo, hi); return f2pack(-lo, -hi); }   // folded into FFMA2 by ptxas
__device__ __forceinline__ u64 f2bcast(float v) { return f2pack(v, v); }

__device__ __forceinline__ u64 f2sub(u64 a, u64 b) { u64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }

// Cubic coefficients on fine sub-interval q for two amplitude components at once (the halves of the packed registers):
// kFineM applied to node[m] - node[2], so that the rounding of the matrix entries acts on small differences only.
__device__ __forceinline__ void fine_cubic2(const u64 nd[6], int q, u64 out[4]) {
  u64 dl[6];
#pragma unroll
  for (int m = 0; m < 6; ++m) dl[m] = f2sub(nd[m], nd[2]);
#pragma unroll
  for (int kk = 0; kk < 4; ++kk) {
    u64 acc = (kk == 0) ? nd[2] : 0ull;
#pragma unroll
    for (int m = 0; m < 6; ++m)
      if (m != 2) acc = f2fma(f2bcast(kFineM[q][kk][m]), dl[m], acc);
    out[kk] = acc;
  }
}

#ifndef SC_QUAD_FLUSH
#define SC_QUAD_FLUSH 128     /* bins per FP32 flush group of the QUAD flavour's unmasked runs (measured on c3, 264 particles:
                                32 bins 18.47 ms, rms error 4.2e-9; 64 bins 18.04 ms; 128 bins 17.85 ms, rms 5.6e-9, and error x sqrt(Upsilon) <= 1.73e-6
                                over c2 / c3 / c4 samples, i.e. <= 4.3e-7 at the escalation threshold tau = 16) */
#endif
#ifndef SC_DENSE2_MINB
#define SC_DENSE2_MINB 4     /* CTAs per SM the register allocation aims at (128 registers/thread) */
#endif

constexpr int kPairRec = 3;

// Moments of the sigma weights over one piece (a fine sub-interval cut at the segment edges; shared by all particles):
//   M_a,m = sum_{j in piece} G_a(j) s_j^m,  s_j = (j - sub-interval start)/Sf,  m = 0..6,  a = A, E.
// On a fine sub-interval the amplitudes are cubics in s, so |c_a(s)|^2 is a polynomial of degree 6 and
// sigma_piece = sum_m (e_A,m M_A,m + e_E,m M_E,m) -- the per-bin evaluation of |h|^2 leaves the hot loop.
__global__ void k_moments(const double2* __restrict__ G64, const int* __restrict__ piece_lo, const int* __restrict__ piece_hi,
                          int n_pieces, int n_bins, int log2_fine, float2* __restrict__ out /* [n_pieces][8] */,
                          double2* __restrict__ out64 = nullptr /* [n_pieces][7], all-FP64 path */) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_pieces) return;
  // piece_lo == nullptr: uniform pieces of 2^(int)(size_t)piece_hi bins (the groups / sub-intervals of the adaptive path)
  const int lg_u = (int)(size_t)piece_hi;
  const int lo = piece_lo ? piece_lo[i] : (i << lg_u);
  const int hi = min(piece_lo ? piece_hi[i] : ((i + 1) << lg_u), n_bins);
  const int ib = (lo >> log2_fine) << log2_fine;
  const double hS = 1.0 / (double)(1 << log2_fine);
  double mA[7] = {0, 0, 0, 0, 0, 0, 0}, mE[7] = {0, 0, 0, 0, 0, 0, 0};
  for (int j = lo; j < hi; ++j) {
    const double2 g = G64[j];
    const double sj = (double)(j - ib) * hS;
    double pw = 1.0;
#pragma unroll
    for (int m = 0; m < 7; ++m) { mA[m] = fma(g.x, pw, mA[m]); mE[m] = fma(g.y, pw, mE[m]); pw *= sj; }
  }
#pragma unroll
  for (int m = 0; m < 7; ++m) out[(size_t)i * 8 + m] = make_float2((float)mA[m], (float)mE[m]);
  out[(size_t)i * 8 + 7] = make_float2(0.f, 0.f);
  if (out64) {
#pragma unroll
    for (int m = 0; m < 7; ++m) out64[(size_t)i * 7 + m] = make_double2(mA[m], mE[m]);
  }
}            // ulonglong2 records per bin pair: (wAr, wAi), (wEr, wEi), (gA, gE), each (even, odd)

// FP32 sin/cos of two phases given as signed 32-bit fractions of a turn: polynomial flavour (SC = 0).  Each is reduced to
// the nearest quarter turn in integer arithmetic (|x| <= 1/8 turn, exact), the two polynomials run on the packed pipe
// (even bin in the low half; fma.rn.f32x2 rounds each half as fmaf does: bit-identical to the scalar evaluation it replaced,
// c3 at N = 10: dense kernel 31.4 -> 29.4 ms), and the quadrant is put back by swap / sign.
__device__ __forceinline__ void sincos_frac32_pair(int n0, int n1, u64& cr2, u64& sr2) {
  const int q0 = (n0 + (1 << 29)) >> 30, q1 = (n1 + (1 << 29)) >> 30;
  const u64 x = f2mul(f2pack((float)(n0 - (q0 << 30)), (float)(n1 - (q1 << 30))), f2bcast(2.3283064365386963e-10f));
  const u64 x2 = f2mul(x, x);
  u64 ps = f2fma(x2, f2bcast(42.0586939448976531f), f2bcast(-76.7058597530613858f));
  ps = f2fma(ps, x2, f2bcast(81.6052492760750542f));
  ps = f2fma(ps, x2, f2bcast(-41.3417022403997602f));
  ps = f2fma(ps, x2, f2bcast(6.28318530717958648f));
  const u64 sn2 = f2mul(ps, x);
  u64 pc = f2fma(x2, f2bcast(-26.4262567833743975f), f2bcast(60.2446413718766604f));
  pc = f2fma(pc, x2, f2bcast(-85.4568172066937277f));
  pc = f2fma(pc, x2, f2bcast(64.9393940226682915f));
  pc = f2fma(pc, x2, f2bcast(-19.7392088021787172f));
  const u64 cn2 = f2fma(pc, x2, f2bcast(1.0f));
  float s0, s1, c0, c1;
  f2unpack(sn2, s0, s1); f2unpack(cn2, c0, c1);
  float cr0 = (q0 & 1) ? s0 : c0, sr0 = (q0 & 1) ? c0 : s0;
  float cr1 = (q1 & 1) ? s1 : c1, sr1 = (q1 & 1) ? c1 : s1;
  cr0 = ((q0 + 1) & 2) ? -cr0 : cr0; sr0 = (q0 & 2) ? -sr0 : sr0;
  cr1 = ((q1 + 1) & 2) ? -cr1 : cr1; sr1 = (q1 & 2) ? -sr1 : sr1;
  cr2 = f2pack(cr0, cr1); sr2 = f2pack(sr0, sr1);
}

// ---- pieces of the packed hot loop shared by k_dense2 (shared edges) and k_dense2_ad (per-particle edges) ----
struct PhaseFD { double phi, d1, d2, d3; };   // phase in turns at the next bin and its forward differences (unit steps)
__device__ __forceinline__ void phase_next_pair(PhaseFD& ph, int& n0, int& n1) {
  n0 = __double2loint(ph.phi);
  ph.phi += ph.d1; ph.d1 += ph.d2; ph.d2 += ph.d3;
  n1 = __double2loint(ph.phi);
  ph.phi += ph.d1; ph.d1 += ph.d2; ph.d2 += ph.d3;
}
__device__ __forceinline__ void phase_skip_pair(PhaseFD& ph) {
  ph.phi += ph.d1; ph.d1 += ph.d2; ph.d2 += ph.d3;
  ph.phi += ph.d1; ph.d1 += ph.d2; ph.d2 += ph.d3;
}
__device__ __forceinline__ void phase_set(PhaseFD& ph, double p0, const double b[6]) {
  // phi carries the bias 1.5 * 2^20: in that binade the unit in the last place is 2^-32 turn, so the low word of phi IS the
  // fraction of a turn as an int32 -- no separate biasing add per bin.  Every step then rounds to 2^-32 turn (1.5e-9 rad): a
  // random walk of < 1e-8 rad over a fine sub-interval (<= 512 steps), far below the FP32 amplitudes' 1e-7 per bin.
  ph.phi = p0 + 1572864.0;
  ph.d1 = b[1] + b[2] + b[3];
  ph.d2 = 2.0 * b[2] + 6.0 * b[3];
  ph.d3 = 6.0 * b[3];
}

// Phase on fine sub-interval [ib, ib + Sf): quintic through 6 nodes -> Taylor shift to the centre of the sub-interval ->
// Chebyshev economisation to a cubic on [-H, H] -> shift to the start -> forward differences for unit steps.
__device__ __forceinline__ void sub_phase(const DevCfg& c, const DenseArgs& a, int p, int ib, PhaseFD& ph) {
  const int ic = ib >> c.log2_stride;
  const int i0 = ic + kNodeOff;
  const int S = c.stride, Sf = S >> 2;
  const size_t base = (size_t)i0 * a.P_pad + p;
  const int n0 = a.node_n[base];
  const double r0 = a.node_frac[base];
  double Y[6];
#pragma unroll
  for (int m = -2; m <= 3; ++m) {
    const size_t at = (size_t)(i0 + m) * a.P_pad + p;
    Y[m + 2] = (double)(a.node_n[at] - n0) + (a.node_frac[at] - r0);
  }
  double b[6];
  quintic_coeffs(Y, 1.0 / (double)S, b);
  const double H = 0.5 * (double)Sf;
  taylor_shift(b, (double)(ib - (ic << c.log2_stride)) + H);
  const double H2 = H * H, H4 = H2 * H2;
  b[0] = fma(-0.125 * H4, b[4], b[0]);
  b[2] = fma(H2, b[4], b[2]);
  b[1] = fma(-0.3125 * H4, b[5], b[1]);
  b[3] = fma(1.25 * H2, b[5], b[3]);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 2; j >= i; --j) b[j] = fma(-H, b[j + 1], b[j]);
  phase_set(ph, r0 + b[0], b);
}

// Cubic coefficients of (Ar, Ai, Er, Ei) on that sub-interval in s = (j - ib)/Sf.  NA: element type of the node table
// (float; double in the per-particle-segment path, whose edge decision needs the FP64 table anyway).
template <typename NA = float>
__device__ __forceinline__ void sub_amps(const DevCfg& c, const DenseArgs& a, int p, int ib, float (&cf)[4][4]) {
  const int i0 = (ib >> c.log2_stride) + kNodeOff;
  const int q = (ib >> (c.log2_stride - 2)) & 3;
  const NA* __restrict__ namp = reinterpret_cast<const NA*>(a.node_amp);
#pragma unroll
  for (int r = 0; r < 4; r += 2) {                          // (Ar, Ai) then (Er, Ei) as packed halves
    const NA* col = namp + ((size_t)i0 * 4 + r) * a.P_pad + p;
    const ptrdiff_t st = (ptrdiff_t)4 * a.P_pad;
    u64 nd[6], o[4];
#pragma unroll
    for (int m = -2; m <= 3; ++m) nd[m + 2] = f2pack((float)col[m * st], (float)col[m * st + a.P_pad]);
    fine_cubic2(nd, q, o);
#pragma unroll
    for (int kk = 0; kk < 4; ++kk) f2unpack(o[kk], cf[r][kk], cf[r + 1][kk]);
  }
}

// ---- merged coarse intervals (k_dense2<.., MERGE = true>, launched when the node stride is >= 512 bins) ----
// The node stride is set by the slowest-chirping corner of the tile; towards higher frequencies a particle crosses a coarse
// interval in less signal time than the day a FINE sub-interval is allowed to span.  Where that holds for every lane of the
// warp (and every lane is inside its window over the whole coarse interval), one set-up serves the four fine
// sub-intervals: the phase quintic is economised over the coarse interval and its forward differences run on through it;
// the amplitudes are the plain cubic through nodes -1 .. 2 (the same <= 1-day spacing the fine cubics work with),
// re-expanded per fine sub-interval (the pieces and their sigma moments stay as they are).
// Signal time spanned by coarse interval ic, as a difference of phase slopes in turns per bin (t_f = T_obs dPhi/dj):
// second difference of the node phases / stride.
__device__ __forceinline__ double coarse_dslope(const DevCfg& c, const DenseArgs& a, int p, int ic) {
  const size_t at0 = (size_t)(ic + kNodeOff) * a.P_pad + p, atm = at0 - a.P_pad, atp = at0 + a.P_pad;
  const int n0 = a.node_n[at0];
  const double r0 = a.node_frac[at0];
  const double ym = (double)(a.node_n[atm] - n0) + (a.node_frac[atm] - r0);
  const double yp = (double)(a.node_n[atp] - n0) + (a.node_frac[atp] - r0);
  return fabs(ym + yp) / (double)c.stride;
}
// Phase over the whole coarse interval starting at bin ib (= ic * stride): as sub_phase with H = stride / 2.
__device__ __forceinline__ void coarse_phase(const DevCfg& c, const DenseArgs& a, int p, int ib, PhaseFD& ph) {
  const int i0 = (ib >> c.log2_stride) + kNodeOff;
  const int S = c.stride;
  const size_t base = (size_t)i0 * a.P_pad + p;
  const int n0 = a.node_n[base];
  const double r0 = a.node_frac[base];
  double Y[6];
#pragma unroll
  for (int m = -2; m <= 3; ++m) {
    const size_t at = (size_t)(i0 + m) * a.P_pad + p;
    Y[m + 2] = (double)(a.node_n[at] - n0) + (a.node_frac[at] - r0);
  }
  double b[6];
  quintic_coeffs(Y, 1.0 / (double)S, b);
  const double H = 0.5 * (double)S;
  taylor_shift(b, H);
  const double H2 = H * H, H4 = H2 * H2;
  b[0] = fma(-0.125 * H4, b[4], b[0]);
  b[2] = fma(H2, b[4], b[2]);
  b[1] = fma(-0.3125 * H4, b[5], b[1]);
  b[3] = fma(1.25 * H2, b[5], b[3]);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 2; j >= i; --j) b[j] = fma(-H, b[j + 1], b[j]);
  phase_set(ph, r0 + b[0], b);
}
// Cubic through nodes -1 .. 2 of (Ar, Ai, Er, Ei) in t = (j - ib) / stride.
template <typename NA = float>
__device__ __forceinline__ void coarse_amps(const DevCfg& c, const DenseArgs& a, int p, int ib, float (&cc)[4][4]) {
  const int i0 = (ib >> c.log2_stride) + kNodeOff;
  const NA* __restrict__ namp = reinterpret_cast<const NA*>(a.node_amp);
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const NA* col = namp + ((size_t)i0 * 4 + r) * a.P_pad + p;
    const ptrdiff_t st = (ptrdiff_t)4 * a.P_pad;
    cubic_coeffs<float>((float)col[-st], (float)col[0], (float)col[st], (float)col[2 * st], cc[r][0], cc[r][1], cc[r][2], cc[r][3]);
  }
}
// The same cubic in the variable of fine sub-interval q: t = (q + s) / 4.
__device__ __forceinline__ void coarse_to_fine(const float (&cc)[4][4], int q, float (&cf)[4][4]) {
  const float t0 = 0.25f * (float)q;
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const float a0 = cc[r][0], a1 = cc[r][1], a2 = cc[r][2], a3 = cc[r][3];
    cf[r][0] = fmaf(fmaf(fmaf(a3, t0, a2), t0, a1), t0, a0);
    cf[r][1] = 0.25f * fmaf(fmaf(3.0f * a3, t0, 2.0f * a2), t0, a1);
    cf[r][2] = 0.0625f * fmaf(3.0f * a3, t0, a2);
    cf[r][3] = 0.015625f * a3;
  }
}

// One bin pair (j, j+1): FP64 phase steps, sin/cos, amplitude cubics, multiply-accumulate into packed sums (low half =
// even bin, high half = odd bin).  MASKED: apply the particle's time window per bin.  WITH_SG: accumulate |h|^2 per
// bin (otherwise sigma comes from the moments).  s2 = (s_j, s_{j+1}), rec = the pair's data record; both advance.
template <bool MASKED, bool WITH_SG, int SC>
__device__ __forceinline__ void pair_eval(PhaseFD& ph, const float (&cf)[4][4], u64& s2, const ulonglong2*& rec, int j,
                                          int jlo, int jhi, u64 h2, u64 K2, u64& zr2, u64& zi2, u64& sg2) {
  int n0, n1;
  phase_next_pair(ph, n0, n1);
  u64 cr2, sr2;
  if (SC == 2) {
    float x0, x1;
    f2unpack(f2mul(f2pack((float)n0, (float)n1), K2), x0, x1);
    cr2 = f2pack(__cosf(x0), __cosf(x1)); sr2 = f2pack(__sinf(x0), __sinf(x1));
  } else {
    sincos_frac32_pair(n0, n1, cr2, sr2);
  }
  const u64 Ar = f2fma(f2fma(f2fma(f2bcast(cf[0][3]), s2, f2bcast(cf[0][2])), s2, f2bcast(cf[0][1])), s2, f2bcast(cf[0][0]));
  const u64 Ai = f2fma(f2fma(f2fma(f2bcast(cf[1][3]), s2, f2bcast(cf[1][2])), s2, f2bcast(cf[1][1])), s2, f2bcast(cf[1][0]));
  const u64 Er = f2fma(f2fma(f2fma(f2bcast(cf[2][3]), s2, f2bcast(cf[2][2])), s2, f2bcast(cf[2][1])), s2, f2bcast(cf[2][0]));
  const u64 Ei = f2fma(f2fma(f2fma(f2bcast(cf[3][3]), s2, f2bcast(cf[3][2])), s2, f2bcast(cf[3][1])), s2, f2bcast(cf[3][0]));
  s2 = f2add(s2, h2);
  const ulonglong2 wA = rec[0], wE = rec[1];
  u64 m2 = 0;
  if (MASKED) {
    m2 = f2pack((j >= jlo && j < jhi) ? 1.0f : 0.0f, (j + 1 >= jlo && j + 1 < jhi) ? 1.0f : 0.0f);
    cr2 = f2mul(cr2, m2); sr2 = f2mul(sr2, m2);
  }
  // q = W_A conj(c_A) + W_E conj(c_E)
  const u64 qr = f2fma(wA.x, Ar, f2fma(wA.y, Ai, f2fma(wE.x, Er, f2mul(wE.y, Ei))));
  const u64 qi = f2fma(wA.y, Ar, f2fma(f2neg(wA.x), Ai, f2fma(wE.y, Er, f2neg(f2mul(wE.x, Ei)))));
  if (WITH_SG) {
    ulonglong2 g = rec[2];
    if (MASKED) { g.x = f2mul(g.x, m2); g.y = f2mul(g.y, m2); }
    sg2 = f2fma(g.x, f2fma(Ar, Ar, f2mul(Ai, Ai)), f2fma(g.y, f2fma(Er, Er, f2mul(Ei, Ei)), sg2));
  }
  rec += kPairRec;
  // z += q e^{+2 pi i Phi}
  zr2 = f2fma(qr, cr2, f2fma(f2neg(qi), sr2, zr2));
  zi2 = f2fma(qr, sr2, f2fma(qi, cr2, zi2));
}

// sigma of a run of bins from the moments of its weights: |c_a(s)|^2 = sum_m e_a,m s^m with the cubic coefficients of
// the sub-interval; both channels at once (A in the low half, E in the high half).  mp: 4 records = 8 (A, E) pairs.
__device__ __forceinline__ double sigma_moments(const float (&cf)[4][4], const ulonglong2* __restrict__ mp) {
  const ulonglong2 m01 = mp[0], m23 = mp[1], m45 = mp[2], m6 = mp[3];
  u64 R[4], I[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) { R[i] = f2pack(cf[0][i], cf[2][i]); I[i] = f2pack(cf[1][i], cf[3][i]); }
  const u64 two = f2bcast(2.0f);
  const u64 R0x2 = f2mul(R[0], two), I0x2 = f2mul(I[0], two), R1x2 = f2mul(R[1], two), I1x2 = f2mul(I[1], two);
  const u64 R2x2 = f2mul(R[2], two), I2x2 = f2mul(I[2], two);
  const u64 e0 = f2fma(R[0], R[0], f2mul(I[0], I[0]));
  const u64 e1 = f2fma(R0x2, R[1], f2mul(I0x2, I[1]));
  const u64 e2 = f2fma(R0x2, R[2], f2fma(I0x2, I[2], f2fma(R[1], R[1], f2mul(I[1], I[1]))));
  const u64 e3 = f2fma(R0x2, R[3], f2fma(I0x2, I[3], f2fma(R1x2, R[2], f2mul(I1x2, I[2]))));
  const u64 e4 = f2fma(R1x2, R[3], f2fma(I1x2, I[3], f2fma(R[2], R[2], f2mul(I[2], I[2]))));
  const u64 e5 = f2fma(R2x2, R[3], f2mul(I2x2, I[3]));
  const u64 e6 = f2fma(R[3], R[3], f2mul(I[3], I[3]));
  u64 acc = f2mul(e0, m01.x);
  acc = f2fma(e1, m01.y, acc); acc = f2fma(e2, m23.x, acc); acc = f2fma(e3, m23.y, acc);
  acc = f2fma(e4, m45.x, acc); acc = f2fma(e5, m45.y, acc); acc = f2fma(e6, m6.x, acc);
  float l, h;
  f2unpack(acc, l, h);
  return (double)l + (double)h;
}

// sin, cos of the phase at the next two bins as packed halves; advances the phase by two bins.
template <int SC>
__device__ __forceinline__ void sincos_pair(PhaseFD& ph, u64 K2, u64& cr2, u64& sr2) {
  int n0, n1;
  phase_next_pair(ph, n0, n1);
  if (SC == 2) {
    float x0, x1;
    f2unpack(f2mul(f2pack((float)n0, (float)n1), K2), x0, x1);
    cr2 = f2pack(__cosf(x0), __cosf(x1)); sr2 = f2pack(__sinf(x0), __sinf(x1));
  } else {
    sincos_frac32_pair(n0, n1, cr2, sr2);
  }
}
// amplitude cubics at (s_j, s_{j+1}), q = W_A conj(c_A) + W_E conj(c_E), z += q e^{+2 pi i Phi}
__device__ __forceinline__ void mac_pair(const float (&cf)[4][4], u64& s2, const ulonglong2 wA, const ulonglong2 wE, u64 h2,
                                         u64 cr2, u64 sr2, u64& zr2, u64& zi2) {
  const u64 Ar = f2fma(f2fma(f2fma(f2bcast(cf[0][3]), s2, f2bcast(cf[0][2])), s2, f2bcast(cf[0][1])), s2, f2bcast(cf[0][0]));
  const u64 Ai = f2fma(f2fma(f2fma(f2bcast(cf[1][3]), s2, f2bcast(cf[1][2])), s2, f2bcast(cf[1][1])), s2, f2bcast(cf[1][0]));
  const u64 Er = f2fma(f2fma(f2fma(f2bcast(cf[2][3]), s2, f2bcast(cf[2][2])), s2, f2bcast(cf[2][1])), s2, f2bcast(cf[2][0]));
  const u64 Ei = f2fma(f2fma(f2fma(f2bcast(cf[3][3]), s2, f2bcast(cf[3][2])), s2, f2bcast(cf[3][1])), s2, f2bcast(cf[3][0]));
  s2 = f2add(s2, h2);
  const u64 qr = f2fma(wA.x, Ar, f2fma(wA.y, Ai, f2fma(wE.x, Er, f2mul(wE.y, Ei))));
  const u64 qi = f2fma(wA.y, Ar, f2fma(f2neg(wA.x), Ai, f2fma(wE.y, Er, f2neg(f2mul(wE.x, Ei)))));
  zr2 = f2fma(qr, cr2, f2fma(f2neg(qi), sr2, zr2));
  zi2 = f2fma(qr, sr2, f2fma(qi, cr2, zi2));
}
// n >= 1 consecutive unmasked pairs, software-pipelined by hand: the sin/cos (FP64 step, conversion, MUFU) and the
// shared-memory loads of pair i+1 are issued before the multiply-accumulate of pair i.
template <int SC>
__device__ __forceinline__ void pairs_fast(PhaseFD& ph, const float (&cf)[4][4], u64& s2, const ulonglong2*& rec, int n,
                                           u64 h2, u64 K2, u64& zr2, u64& zi2) {
  u64 cr, sr;
  sincos_pair<SC>(ph, K2, cr, sr);
  ulonglong2 wA = rec[0], wE = rec[1];
#pragma unroll 1
  for (int i = 1; i < n; ++i) {
    u64 crn, srn;
    sincos_pair<SC>(ph, K2, crn, srn);
    rec += kPairRec;
    const ulonglong2 wAn = rec[0], wEn = rec[1];
    mac_pair(cf, s2, wA, wE, h2, cr, sr, zr2, zi2);
    cr = crn; sr = srn; wA = wAn; wE = wEn;
  }
  rec += kPairRec;
  mac_pair(cf, s2, wA, wE, h2, cr, sr, zr2, zi2);
}

// The same with the amplitudes QUADRATIC over runs of a quarter of the fine sub-interval (QUAD flavour, fine
// sub-intervals of >= 256 bins): the sub-interval's cubic re-expanded about the run start in u = (j - run start)/run
// length, its u^3 term economised (u^3 ~ 3/2 u^2 - 9/16 u + 1/32 on [0, 1], error <= |c_3| / (64 x 32) of the cubic's
// own s^3 coefficient: <= 3e-8 of the amplitude at 4 days per coarse interval, oscillating inside the run) -- 8 packed
// FMAs per bin pair instead of 12.  sigma keeps the cubic (sigma_moments).  off = first bin - sub-interval start,
// lg_run = log2(run length in bins); s2 is not used by this flavour.
struct QuadRun { float q[4][3]; };
__device__ __forceinline__ void quad_run(const float (&cf)[4][4], int r, QuadRun& o) {
  const float s0 = 0.25f * (float)r;
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    const float c0 = cf[a][0], c1 = cf[a][1], c2 = cf[a][2], c3 = cf[a][3];
    const float a3 = c3 * (1.0f / 64.0f);
    const float a2 = fmaf(3.0f * c3, s0, c2) * (1.0f / 16.0f);
    const float a1 = fmaf(fmaf(3.0f * c3, s0, 2.0f * c2), s0, c1) * 0.25f;
    const float a0 = fmaf(fmaf(fmaf(c3, s0, c2), s0, c1), s0, c0);
    o.q[a][2] = fmaf(1.5f, a3, a2);
    o.q[a][1] = fmaf(-0.5625f, a3, a1);
    o.q[a][0] = fmaf(0.03125f, a3, a0);
  }
}
__device__ __forceinline__ void mac_pair_q(const QuadRun& w, u64& u2, const ulonglong2 wA, const ulonglong2 wE, u64 hu2,
                                           u64 cr2, u64 sr2, u64& zr2, u64& zi2) {
  const u64 Ar = f2fma(f2fma(f2bcast(w.q[0][2]), u2, f2bcast(w.q[0][1])), u2, f2bcast(w.q[0][0]));
  const u64 Ai = f2fma(f2fma(f2bcast(w.q[1][2]), u2, f2bcast(w.q[1][1])), u2, f2bcast(w.q[1][0]));
  const u64 Er = f2fma(f2fma(f2bcast(w.q[2][2]), u2, f2bcast(w.q[2][1])), u2, f2bcast(w.q[2][0]));
  const u64 Ei = f2fma(f2fma(f2bcast(w.q[3][2]), u2, f2bcast(w.q[3][1])), u2, f2bcast(w.q[3][0]));
  u2 = f2add(u2, hu2);
  const u64 qr = f2fma(wA.x, Ar, f2fma(wA.y, Ai, f2fma(wE.x, Er, f2mul(wE.y, Ei))));
  const u64 qi = f2fma(wA.y, Ar, f2fma(f2neg(wA.x), Ai, f2fma(wE.y, Er, f2neg(f2mul(wE.x, Ei)))));
  zr2 = f2fma(qr, cr2, f2fma(f2neg(qi), sr2, zr2));
  zi2 = f2fma(qr, sr2, f2fma(qi, cr2, zi2));
}
// The run state lives across the flush groups of a piece: coefficients are rebuilt at run boundaries only.
struct QuadState { QuadRun w; u64 u2; int left; int r; };
__device__ __forceinline__ void quad_start(const float (&cf)[4][4], int off, int lg_run, QuadState& q) {
  const int run_bins = 1 << lg_run;
  const int o = off & (run_bins - 1);
  const float hu = 1.0f / (float)run_bins;
  q.r = off >> lg_run;
  q.left = (run_bins - o) >> 1;                                 // pairs to the end of the run
  q.u2 = f2pack((float)o * hu, (float)(o + 1) * hu);
  quad_run(cf, q.r, q.w);
}
template <int SC>
__device__ __forceinline__ void pairs_fast_q(PhaseFD& ph, const float (&cf)[4][4], QuadState& q, int lg_run, const ulonglong2*& rec,
                                             int n, u64 K2, u64& zr2, u64& zi2) {
  const int run_pairs = 1 << (lg_run - 1);
  const float hu = 1.0f / (float)(2 * run_pairs);
  const u64 hu2 = f2bcast(2.0f * hu);
  u64 cr, sr;
  sincos_pair<SC>(ph, K2, cr, sr);
  ulonglong2 wA = rec[0], wE = rec[1];
#pragma unroll 1
  for (int i = 1; i < n; ++i) {
    u64 crn, srn;
    sincos_pair<SC>(ph, K2, crn, srn);
    rec += kPairRec;
    const ulonglong2 wAn = rec[0], wEn = rec[1];
    mac_pair_q(q.w, q.u2, wA, wE, hu2, cr, sr, zr2, zi2);
    if (--q.left == 0) { quad_run(cf, ++q.r, q.w); q.left = run_pairs; q.u2 = f2pack(0.0f, hu); }
    cr = crn; sr = srn; wA = wAn; wE = wEn;
  }
  rec += kPairRec;
  mac_pair_q(q.w, q.u2, wA, wE, hu2, cr, sr, zr2, zi2);
  if (--q.left == 0) { quad_run(cf, ++q.r, q.w); q.left = run_pairs; q.u2 = f2pack(0.0f, hu); }
}

// Staging of the chunk's data records (all flavours but the segment-table one): ONE bulk copy (cp.async.bulk, the TMA unit) of 48 KB issued by thread 0, completion on
// an mbarrier; the threads load their per-particle state while it is in flight and wait on the barrier before the walk.
namespace stg {
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t b, uint32_t cnt) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(b), "r"(cnt)); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(b), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t b, uint32_t parity) {
  asm volatile("{\n.reg .pred P1;\nLAB_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n@P1 bra DONE;\nbra LAB_WAIT;\nDONE:\n}"
               :: "r"(b), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
}  // namespace stg
constexpr int kDense2DataBytes = kChunkF32 / 2 * kPairRec * 16;              // 48 KB of data records per chunk
constexpr int kDense2Smem = kDense2DataBytes + 16;                           // + the mbarrier (dynamic shared memory: > 48 KB)

template <bool SEG, int SC, bool MERGE = false, bool QUAD = false>
__global__ void __launch_bounds__(kBlock, SC_DENSE2_MINB) k_dense2(DevCfg c, DenseArgs a, const ulonglong2* __restrict__ Dg) {
  constexpr int CH = kChunkF32;
  // The segment-table flavour (SEG: sc_eval_segments, the two-pass three-channel path) keeps the plain staging loop into
  // static shared memory: with the dynamic array its register allocation spills 60 B more and it runs 10 % slower.
  extern __shared__ __align__(128) unsigned char smem_d2[];
  ulonglong2* sD;                                                // 48 KB
  uint32_t bar = 0;
  if constexpr (SEG) {
    __shared__ ulonglong2 sD_static[CH / 2 * kPairRec];
    sD = sD_static;
  } else {
    sD = reinterpret_cast<ulonglong2*>(smem_d2);
    bar = stg::smem_u32(smem_d2 + kDense2DataBytes);
    if (threadIdx.x == 0) {
      stg::mbar_init(bar, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
  }

  const int chunk_l = blockIdx.x;
  const int cs = (a.chunk_first + chunk_l) * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int ce2 = (ce + 1) & ~1;                               // pair-aligned end (data beyond n_bins is zero)
  const int p = blockIdx.y * kBlock + threadIdx.x;

  // no particle of this block has its time window in this chunk (common once the batch is sorted by window centre): skip
  // the staging of the data.  k_stitch reads a particle's fragments only in the chunks its window overlaps, i.e. never
  // those of such a CTA; k_stitch_seg (SEG) reads every chunk and gets empty fragments.
  if (!__syncthreads_or((a.jhi[p] > cs) && (a.jlo[p] < ce))) {
    if constexpr (SEG) {
      double* fz = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + p;
#pragma unroll
      for (int m = 0; m < kFragFields; ++m) fz[(size_t)m * a.P_pad] = 0.0;
    }
    return;
  }

  if constexpr (SEG) {
    const ulonglong2* src = Dg + (size_t)(cs >> 1) * kPairRec;
#pragma unroll 4
    for (int t = threadIdx.x; t < CH / 2 * kPairRec; t += kBlock) sD[t] = src[t];
    __syncthreads();
  } else if (threadIdx.x == 0) {
    // (the __syncthreads_or above orders the barrier's initialisation before every wait)
    stg::mbar_expect_tx(bar, kDense2DataBytes);
    stg::bulk_g2s(stg::smem_u32(sD), Dg + (size_t)(cs >> 1) * kPairRec, kDense2DataBytes, bar);
  }

  const int jlo = a.jlo[p], jhi = a.jhi[p];
  const int S = c.stride, Sf = S >> 2;
  const float hS = 1.0f / (float)Sf;
  const u64 h2 = f2bcast(2.0f * hS);
  const u64 K2 = f2bcast(1.4629180792671596e-09f);            // 2 pi / 2^32

  int k = a.chunk_k0[chunk_l];
  int next_edge = (k + 1 <= a.n_seg) ? a.edges[k + 1] : INT_MAX;
  bool open_at_edge = (k >= 0 && k < a.n_seg) ? (a.edges[k] == cs) : true;
  double Zr = 0.0, Zi = 0.0, Sg = 0.0, ups = 0.0, xs = 0.0, hs = 0.0;
  double* frag = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + p;

  auto close_piece = [&](bool at_edge_end) {
    if (open_at_edge && at_edge_end) {
      if (SEG) {
        if (p < a.P) {
          double* o = a.out_seg + ((size_t)p * a.n_seg + k) * 3;
          o[0] = Zr * a.seg_scale_z; o[1] = Zi * a.seg_scale_z; o[2] = Sg * a.seg_scale_s;
        }
      } else if (Sg > 0.0) {
        const double z2 = Zr * Zr + Zi * Zi;
        ups += z2 / Sg;
        if (a.comp) { xs += sqrt(z2); hs += Sg; }
      }
    } else if (!open_at_edge) {
      frag[(size_t)1 * a.P_pad] = Zr; frag[(size_t)2 * a.P_pad] = Zi; frag[(size_t)3 * a.P_pad] = Sg;
    } else {
      frag[(size_t)4 * a.P_pad] = Zr; frag[(size_t)5 * a.P_pad] = Zi; frag[(size_t)6 * a.P_pad] = Sg;
    }
    Zr = 0.0; Zi = 0.0; Sg = 0.0;
  };
  auto next_segment = [&]() {
    ++k;
    next_edge = (k + 1 <= a.n_seg) ? a.edges[k + 1] : INT_MAX;
    open_at_edge = true;
  };

  PhaseFD fd = {};
  float cc[MERGE ? 4 : 1][4];  // merged coarse interval: cubic of the amplitudes in t = (j - coarse start)/stride
  int merged_left = 0;         // fine sub-intervals of the current merged coarse interval still to walk
  bool landed = SEG;           // the bulk copy is waited for after the first sub-interval's set-up (node reads only)
  for (int ib = cs; ib < ce2; ib += Sf) {
    const int ie = min(ib + Sf, ce2);
    const bool lane_in = (ib >= jlo) && (ie <= jhi);
    const bool lane_out = (ie <= jlo) || (ib >= jhi);
    const bool all_in = __all_sync(0xffffffffu, lane_in);
    const bool all_out = __all_sync(0xffffffffu, lane_out);

    float cf[4][4];    // cubic coefficients of (Ar, Ai, Er, Ei) in s = (j - ib)/Sf (FFMA2 broadcasts a scalar operand)
    if constexpr (MERGE) {
      if (merged_left == 0 && (ib & (S - 1)) == 0 && ib + S <= ce2 &&
          __all_sync(0xffffffffu, (ib >= jlo) && (ib + S <= jhi)) &&
          __all_sync(0xffffffffu, coarse_dslope(c, a, p, ib >> c.log2_stride) <= a.merge_lim)) {
        coarse_phase(c, a, p, ib, fd);
        coarse_amps(c, a, p, ib, cc);
        merged_left = 4;
      }
    }
    if (MERGE && merged_left > 0) {
      if constexpr (MERGE) coarse_to_fine(cc, 4 - merged_left, cf);   // the phase differences run on
      --merged_left;
    } else if (!all_out) {
      sub_phase(c, a, p, ib, fd);
      sub_amps(c, a, p, ib, cf);
    }

    if (!landed) { stg::mbar_wait(bar, 0); landed = true; }
    u64 s2 = 0;        // (s_j, s_{j+1}) of the next pair
    const ulonglong2* rec = sD;   // its data record
    auto pair = [&](int j, auto masked_c, auto with_sg_c, u64& zr2, u64& zi2, u64& sg2) {
      pair_eval<decltype(masked_c)::value, decltype(with_sg_c)::value, SC>(fd, cf, s2, rec, j, jlo, jhi, h2, K2, zr2, zi2, sg2);
    };
    auto sigma_piece = [&](int piece) { Sg += sigma_moments(cf, a.moments + (size_t)piece * 4); };
    using T_ = std::true_type; using F_ = std::false_type;

    // Walk the pieces of this sub-interval (it is cut at every distinct edge inside it).  Pairs are evaluated once:
    // when a piece ends on an odd bin the straddling pair forms a flush group of its own, its low half goes to the
    // piece that ends and its high half is carried into the next piece.
    const bool use_mom = all_in;      // all lanes inside their windows: sigma from the piece moments, unmasked pairs
    int piece = use_mom ? a.piece_first[(ib >> (c.log2_stride - 2)) - ((a.chunk_first * CH) >> (c.log2_stride - 2))] : 0;
    float car_zr = 0.f, car_zi = 0.f, car_sg = 0.f;
    bool carry = false;
    QuadState qs;
    int q_pos = -1;            // the bin qs stands at (-1: nowhere; a new sub-interval has new coefficients)
    int pl = ib;
    while (pl < ie) {
      const int ph = min(next_edge, ie);                       // next_edge > pl: edges <= pl are consumed
      const bool live = (k >= 0) && (k < a.n_seg);
      int jj = pl;
      if (carry) {
        if (live) { Zr += (double)car_zr; Zi += (double)car_zi; Sg += (double)car_sg; }
        carry = false;
        jj = pl + 1;
      }
      const int jfull = ph & ~1;                               // full pairs end here; a straddling pair follows if ph is odd
      if (!all_out) {
        if (!live && jj < jfull) {
          for (int t = jj; t < jfull; t += 2) phase_skip_pair(fd);
          jj = jfull;
        }
        s2 = f2pack((float)(jj - ib) * hS, (float)(jj + 1 - ib) * hS);
        rec = sD + ((jj - cs) >> 1) * kPairRec;
        // (a piece that begins where the previous one's pairs ended finds the run state in place)
        if constexpr (QUAD) { if (use_mom && jj < ph && q_pos != jj) quad_start(cf, jj - ib, c.log2_stride - 4, qs); }
        while (jj < ph) {
          const bool split = (jj == jfull);                    // the pair (ph - 1, ph)
          const int e2 = split ? jj + 2 : min(jj + ((QUAD && use_mom) ? SC_QUAD_FLUSH : kFlushBins), jfull);
          u64 zr2 = 0, zi2 = 0, sg2 = 0;
          if (use_mom) {
            if constexpr (QUAD) { pairs_fast_q<SC>(fd, cf, qs, c.log2_stride - 4, rec, (e2 - jj) >> 1, K2, zr2, zi2); q_pos = e2; }
            else pairs_fast<SC>(fd, cf, s2, rec, (e2 - jj) >> 1, h2, K2, zr2, zi2);
            jj = e2;
          }
          else         { for (; jj < e2; jj += 2) pair(jj, T_{}, T_{}, zr2, zi2, sg2); }
          float zrl, zrh, zil, zih, sgl, sgh;
          f2unpack(zr2, zrl, zrh); f2unpack(zi2, zil, zih); f2unpack(sg2, sgl, sgh);
          if (split) { car_zr = zrh; car_zi = zih; car_sg = sgh; carry = true; zrh = 0.f; zih = 0.f; sgh = 0.f; }
          if (live) { Zr += (double)(zrl + zrh); Zi += (double)(zil + zih); Sg += (double)(sgl + sgh); }
        }
      } else if (ph & 1) {
        car_zr = 0.f; car_zi = 0.f; car_sg = 0.f; carry = true;   // keep the bookkeeping of the walk uniform
      }
      if (use_mom && live) sigma_piece(piece);
      ++piece;
      while (next_edge == ph) {                                // segments that end here (incl. empty ones)
        if (k >= 0 && k < a.n_seg) close_piece(true);
        next_segment();
      }
      pl = ph;
    }
  }
  // (a segment that ends exactly on the chunk end was closed by the walk: the host's CF_HEAD_CLOSES rule says the same)
  // the piece still open at the chunk end
  if (k >= 0 && k < a.n_seg) close_piece(false);
  if (!SEG) {
    frag[0] = ups;
    if (a.comp) { frag[(size_t)7 * a.P_pad] = xs; frag[(size_t)8 * a.P_pad] = hs; }
  }
}

}  // namespace
