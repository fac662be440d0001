// sc_kernels_dense64.cuh -- a4 + a5, all-FP64 flavour of the hot loop (few segments) and the shared DenseArgs.
// Part of libscstat.so (one translation unit: sc_stat.cu includes the kernel files in pipeline order).
#pragma once
#include "sc_common.cuh"

namespace {

// ------------------------------------------------------------------------------------------------ a4 + a5
// sin, cos of 2 pi x for |x| <= 1/8 turn (Taylor in x^2, coefficients (2 pi)^k / k!).
__device__ __forceinline__ void sincos_2pi_small(float x, float& s, float& c) {
  const float x2 = x * x;
  float ps = fmaf(x2, 42.0586939448976531f, -76.7058597530613858f);  // (2pi)^9/9!, -(2pi)^7/7!
  ps = fmaf(ps, x2, 81.6052492760750542f);                            // (2pi)^5/5!
  ps = fmaf(ps, x2, -41.3417022403997602f);                           // -(2pi)^3/3!
  ps = fmaf(ps, x2, 6.28318530717958648f);
  s = ps * x;
  float pc = fmaf(x2, -26.4262567833743975f, 60.2446413718766604f);  // -(2pi)^10/10!, (2pi)^8/8!
  pc = fmaf(pc, x2, -85.4568172066937277f);                           // -(2pi)^6/6!
  pc = fmaf(pc, x2, 64.9393940226682915f);                            // (2pi)^4/4!
  pc = fmaf(pc, x2, -19.7392088021787172f);                           // -(2pi)^2/2!
  c = fmaf(pc, x2, 1.0f);
}
// Taylor coefficients (2 pi)^k / k! in the constant bank: a DFMA takes them as c[bank][offset] operands (64-bit literals
// would be rebuilt in uniform registers, two UMOV each, on every bin of the issue-bound all-FP64 loop).
__constant__ double kSinC[7] = {3.8199525848482821277, -15.094642576822990392, 42.058693944897653145, -76.705859753061385842,
                                81.605249276075054203, -41.341702240399760234, 6.2831853071795864769};   // x^13 .. x^1
__constant__ double kCosC[7] = {-1.7143907110886720654, 7.9035363713184688042, -26.426256783374397453, 60.244641371876660363,
                                -85.456817206693727736, 64.939394022668291491, -19.739208802178717238};  // x^14 .. x^2
__device__ __forceinline__ void sincos_2pi_small(double x, double& s, double& c) {
  const double x2 = x * x;
  // |x| <= 1/8 turn: the first omitted terms are (pi/4)^15/15! = 2e-14 (sin) and (pi/4)^16/16! = 1e-15 (cos)
  double ps = fma(x2, kSinC[0], kSinC[1]);
#pragma unroll
  for (int i = 2; i < 7; ++i) ps = fma(ps, x2, kSinC[i]);
  s = ps * x;
  double pc = fma(x2, kCosC[0], kCosC[1]);
#pragma unroll
  for (int i = 2; i < 7; ++i) pc = fma(pc, x2, kCosC[i]);
  c = fma(pc, x2, 1.0);
}

template <typename R> struct DataT;
template <> struct DataT<double> { using W = double4; using G = double2; static constexpr int chunk = kChunkF64; };

struct DenseArgs {
  const int* edges;            // [n_seg + 1]
  int n_seg;
  int chunk_first;             // first chunk launched (global chunk index)
  const int* chunk_k0;         // [n_chunks_launched] last k with e_k <= chunk start (-1 .. n_seg)
  const int* node_n;           // [n_nodes][P_pad]
  const double* node_frac;
  const void* node_amp;        // R [n_nodes][4][P_pad]
  const int* jlo; const int* jhi;
  int P_pad;
  double* frag;                // [n_chunks_launched][kFragFields][P_pad]
  double* out_seg;             // SEG mode: [P][n_seg][3] (already offset to this batch), else nullptr
  int P;                       // particles in this batch
  double seg_scale_z, seg_scale_s;
  int comp;                    // also accumulate sum_k |z_k| and sum_k sigma_k (Eq. 8, 9 components)
  // k_dense2 only: pieces = fine sub-intervals cut at the segment edges, with the moments of the sigma weights
  const int* piece_first;      // [n_sub_launched + 1] first piece of each launched fine sub-interval
  const ulonglong2* moments;   // [n_pieces][4] = 8 packed (A, E) pairs: sum_j g_a(j) s_j^m, m = 0..6, pad
  const ulonglong2* momentsT;  // k_dense3 only: the same for (T, 0)
  double merge_lim;            // k_dense2<.., MERGE>: a coarse interval every lane crosses in less signal time than this
                               // (as a slope difference, turns per bin) is set up once for its four fine sub-intervals
  // k_dense only: FP64 moments of the sigma weights per piece, [n_pieces][7] (A, E) pairs, or nullptr (per-bin sigma)
  const double2* moments64;
  // escalation pass (k_dense only): device-side particle count and this batch's offset; nullptr otherwise
  const int* esc_count; int esc_pb;
};

// sigma of one piece from the FP64 moments of its weights: on a fine sub-interval the amplitudes are cubics in s, so
// |c_a(s)|^2 = sum_m e_a,m s^m (m = 0..6) and sigma_piece = sum_m (e_A,m M_A,m + e_E,m M_E,m) -- 7 FP64 operations per bin
// leave the loop for ~45 per piece.
__device__ __forceinline__ double sigma_moments64(const double (&cf)[4][4], const double2* __restrict__ M) {
  double sig = 0.0;
#pragma unroll
  for (int ch = 0; ch < 2; ++ch) {
    const double* R = cf[2 * ch];
    const double* I = cf[2 * ch + 1];
    double e[7];
    e[0] = fma(R[0], R[0], I[0] * I[0]);
    e[1] = 2.0 * fma(R[0], R[1], I[0] * I[1]);
    e[2] = fma(2.0, fma(R[0], R[2], I[0] * I[2]), fma(R[1], R[1], I[1] * I[1]));
    e[3] = 2.0 * (fma(R[0], R[3], I[0] * I[3]) + fma(R[1], R[2], I[1] * I[2]));
    e[4] = fma(2.0, fma(R[1], R[3], I[1] * I[3]), fma(R[2], R[2], I[2] * I[2]));
    e[5] = 2.0 * fma(R[2], R[3], I[2] * I[3]);
    e[6] = fma(R[3], R[3], I[3] * I[3]);
#pragma unroll
    for (int m = 0; m < 7; ++m) sig = fma(e[m], ch == 0 ? M[m].x : M[m].y, sig);
  }
  return sig;
}

// sin, cos of 2 pi x for any |x| < 2^49 turns: nearest quarter turn removed exactly, polynomials on |x| <= 1/8 turn.
__device__ __forceinline__ void sincos_turns(double x, double& sr, double& cr) {
  const double t = fma(x, 4.0, kMagic);
  const int quad = __double2loint(t);
  x = fma(t - kMagic, -0.25, x);
  double sn, cn;
  sincos_2pi_small(x, sn, cn);
  const bool swp = quad & 1;
  cr = swp ? sn : cn; sr = swp ? cn : sn;
  cr = ((quad + 1) & 2) ? -cr : cr;
  sr = (quad & 2) ? -sr : sr;
}

// Phase on fine sub-interval [ib, ib + Sf) as a cubic in unit bin steps from ib: quintic through 6 nodes -> Taylor shift to
// the centre -> Chebyshev economisation to a cubic on [-H, H] (dropped: |b4| H^4 / 8 + |b5| H^5 / 16 turns, < 1e-11 rad
// at the <= 2-day node spacing of this path) -> shift to the start.  Returns the phase at ib [turns] and its forward
// differences d1 = Phi(1) - Phi(0), d2, d3 (constant).
__device__ __forceinline__ void sub_phase_cubic(const DevCfg& c, const int* __restrict__ node_n,
                                                const double* __restrict__ node_frac, int P_pad, int p, int ib,
                                                double& p0, double& d1, double& d2, double& d3) {
  const int ic = ib >> c.log2_stride;
  const int i0 = ic + kNodeOff;
  const int S = c.stride, Sf = S >> 2;
  const size_t base = (size_t)i0 * P_pad + p;
  const int n0 = node_n[base];
  const double r0 = node_frac[base];
  double Y[6];
#pragma unroll
  for (int m = -2; m <= 3; ++m) {
    const size_t at = (size_t)(i0 + m) * P_pad + p;
    Y[m + 2] = (double)(node_n[at] - n0) + (node_frac[at] - r0);
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
  p0 = r0 + b[0];
  d1 = b[1] + b[2] + b[3];
  d2 = 2.0 * b[2] + 6.0 * b[3];
  d3 = 6.0 * b[3];
}

// All-FP64 flavour (few segments, N_seg < 8 by default): one bin per step, FP64 amplitudes and accumulation.  The phase
// factor e^{2 pi i Phi_j} is carried by a rotation recurrence instead of being evaluated per bin: with the sub-interval's
// cubic phase, E_j = e^{2 pi i Phi_j}, R_j = e^{2 pi i d1_j}, Q_j = e^{2 pi i d2_j} obey E_{j+1} = E_j R_j, R_{j+1} = R_j Q_j,
// Q_{j+1} = Q_j (1 + 2 pi i d3) -- 10 FP64 operations per bin against 23 for five forward differences, the range reduction
// and two polynomials.  E, R, Q are re-seeded with FP64 sin/cos at every fine sub-interval (<= 256 bins), over which the
// recurrences' rounding grows to < 1e-10 rad (Q's error enters E as n^3/6 x 1.1e-16).
constexpr size_t kDense64Smem = (size_t)kChunkF64 * (sizeof(double4) + sizeof(double2) + sizeof(float4));
template <bool SEG, bool ESC = false>
__global__ void __launch_bounds__(kBlock) k_dense(DevCfg c, DenseArgs a, const double4* __restrict__ Wg,
                                                  const double2* __restrict__ Gg) {
  using R = double;
  using WT = typename DataT<R>::W;
  using GT = typename DataT<R>::G;
  constexpr int CH = DataT<R>::chunk;
  // dynamic shared memory (kDense64Smem = 64 KB per CTA, 3 CTAs per SM): the chunk's whitened data in FP64, the sigma
  // weights, and an FP32 copy of the data for the correction term of the anchored path
  extern __shared__ __align__(16) unsigned char smem_raw[];
  WT* sW = reinterpret_cast<WT*>(smem_raw);
  GT* sG = reinterpret_cast<GT*>(sW + CH);
  float4* sW32 = reinterpret_cast<float4*>(sG + CH);

  const int chunk_l = blockIdx.x;                              // launched-chunk index
  const int cs = (a.chunk_first + chunk_l) * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int esc_lim = ESC ? min(*a.esc_count - a.esc_pb, a.P_pad) : 0;
  if (ESC && (int)(blockIdx.y * kBlock) >= esc_lim) return;
  if (ESC) {
    // escalation pass: the CTA strides over particle blocks; none of them may live in this chunk (short windows, batch
    // sorted by window centre) -- then every block gets its empty fragments and the data is not staged
    bool any = false;
    for (int pblk = blockIdx.y; pblk * kBlock < esc_lim; pblk += gridDim.y) {
      const int pp = pblk * kBlock + threadIdx.x;
      any = any || ((a.jhi[pp] > cs) && (a.jlo[pp] < ce));
    }
    if (!__syncthreads_or(any)) {
      for (int pblk = blockIdx.y; pblk * kBlock < esc_lim; pblk += gridDim.y) {
        double* fz = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + pblk * kBlock + threadIdx.x;
#pragma unroll
        for (int m = 0; m < kFragFields; ++m) fz[(size_t)m * a.P_pad] = 0.0;
      }
      return;
    }
  }
  if (!ESC) {                                                  // as in k_dense2: nothing of this block lives in this chunk
    const int p0 = blockIdx.y * kBlock + threadIdx.x;
    if (!__syncthreads_or((a.jhi[p0] > cs) && (a.jlo[p0] < ce))) {   // (see k_dense2: only k_stitch_seg reads these fragments)
      if constexpr (SEG) {
        double* fz = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + p0;
#pragma unroll
        for (int m = 0; m < kFragFields; ++m) fz[(size_t)m * a.P_pad] = 0.0;
      }
      return;
    }
  }

  for (int t = threadIdx.x; t < ce - cs; t += kBlock) {
    const WT w = Wg[cs + t];
    sW[t] = w; sG[t] = Gg[cs + t];
    sW32[t] = make_float4((float)w.x, (float)w.y, (float)w.z, (float)w.w);
  }
  __syncthreads();

  // one pass over the block's 128 particles; in the escalation pass the blocks stride over the selected particles
  for (int pblk = blockIdx.y; ; pblk += gridDim.y) {
  if (ESC && pblk * kBlock >= esc_lim) return;
  const int p = pblk * kBlock + threadIdx.x;                   // particle within the batch (P_pad is a multiple of kBlock)

  const int jlo = a.jlo[p], jhi = a.jhi[p];
  if (ESC && !__any_sync(0xffffffffu, (jhi > cs) && (jlo < ce))) {   // no lane of this warp lives here (no barrier below)
    double* fz = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + p;
#pragma unroll
    for (int m = 0; m < kFragFields; ++m) fz[(size_t)m * a.P_pad] = 0.0;
    continue;
  }
  const int S = c.stride, Sf = S >> 2;
  const R hS = R(1.0) / R(Sf);
  const R* __restrict__ namp = reinterpret_cast<const R*>(a.node_amp);

  int k = a.chunk_k0[chunk_l];
  int next_edge = (k + 1 <= a.n_seg) ? a.edges[k + 1] : INT_MAX;
  bool open_at_edge = (k >= 0 && k < a.n_seg) ? (a.edges[k] == cs) : true;
  double Zr = 0.0, Zi = 0.0, Sg = 0.0, ups = 0.0, xs = 0.0, hs = 0.0;
  double* frag = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + p;

  auto close_piece = [&](bool at_edge_end) {
    // at_edge_end: the piece ends at e_{k+1}.  open_at_edge: it began at e_k.
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
    } else if (!open_at_edge) {          // began in an earlier chunk: head fragment (closed or running through)
      frag[(size_t)1 * a.P_pad] = Zr; frag[(size_t)2 * a.P_pad] = Zi; frag[(size_t)3 * a.P_pad] = Sg;
    } else {                             // began here, continues into the next chunk: tail fragment
      frag[(size_t)4 * a.P_pad] = Zr; frag[(size_t)5 * a.P_pad] = Zi; frag[(size_t)6 * a.P_pad] = Sg;
    }
    Zr = 0.0; Zi = 0.0; Sg = 0.0;
  };

  double Pr = 1.0, Pi = 0.0, Rr = 1.0, Ri = 0.0, Qr = 1.0, Qi = 0.0, eps = 0.0;   // rotation recurrence: P = E_j (see above)
  auto rot_step = [&]() {
    const double pr = fma(Pr, Rr, -(Pi * Ri)), pi = fma(Pr, Ri, Pi * Rr);
    const double rr = fma(Rr, Qr, -(Ri * Qi)), ri = fma(Rr, Qi, Ri * Qr);
    const double qr = fma(-eps, Qi, Qr), qi = fma(eps, Qr, Qi);
    Pr = pr; Pi = pi; Rr = rr; Ri = ri; Qr = qr; Qi = qi;
  };
  for (int ib = cs; ib < ce; ib += Sf) {
    const int ie = min(ib + Sf, ce);
    const bool lane_in = (ib >= jlo) && (ie <= jhi);
    const bool lane_out = (ie <= jlo) || (ib >= jhi);
    const bool all_in = __all_sync(0xffffffffu, lane_in);
    const bool all_out = __all_sync(0xffffffffu, lane_out);

    R cf[4][4];        // cubic coefficients of (Ar, Ai, Er, Ei) in t = (u - u_sub)/fine_stride
    if (!all_out) {
      const int ic = ib >> c.log2_stride;                      // coarse interval
      const int i0 = ic + kNodeOff;                            // table row of its left node
      const int q = (ib >> (c.log2_stride - 2)) & 3;           // fine sub-interval within the coarse one
      if (lane_out) {
        // a lane outside its window here may see stencil nodes beyond k_nodes' reach (written as zeros): its bins are
        // masked, but the recurrence must stay finite (0 x Inf), so it idles on the unit circle
        Pr = 1.0; Pi = 0.0; Rr = 1.0; Ri = 0.0; Qr = 1.0; Qi = 0.0; eps = 0.0;
      } else {
        double p0, d1, d2, d3;
        sub_phase_cubic(c, a.node_n, a.node_frac, a.P_pad, p, ib, p0, d1, d2, d3);
        sincos_turns(p0, Pi, Pr);
        sincos_turns(d1, Ri, Rr);
        sincos_turns(d2, Qi, Qr);
        eps = 6.283185307179586477 * d3;
      }
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const R* col = namp + ((size_t)i0 * 4 + r) * a.P_pad + p;
        const ptrdiff_t st = (ptrdiff_t)4 * a.P_pad;
        R nd[6];
#pragma unroll
        for (int m = -2; m <= 3; ++m) nd[m + 2] = col[m * st];
        fine_cubic<R>(nd, q, cf[r][0], cf[r][1], cf[r][2], cf[r][3]);
      }
    }
    R s = R(0.0);
    // Anchored form of the amplitudes for the fast path below: c(s) = g0 + delta(d), d = s - 1/2, with the value at the
    // centre of the sub-interval in FP64 and the cubic correction delta = d (g1 + d (g2 + d g3)) in FP32 (|delta| is a few
    // 1e-2 of |c| over a <= 0.5-day sub-interval, so its FP32 rounding is ~1e-9 of the amplitude).
    R g0[4];
    float g1[4], g2[4], g3[4];
    if (!all_out)
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      g0[r] = fma(cf[r][3], 0.125, fma(cf[r][2], 0.25, fma(cf[r][1], 0.5, cf[r][0])));
      g1[r] = (float)fma(cf[r][3], 0.75, cf[r][1] + cf[r][2]);
      g2[r] = (float)fma(cf[r][3], 1.5, cf[r][2]);
      g3[r] = (float)cf[r][3];
    }

    // one bin: phase factor from the recurrence, amplitude cubics, multiply-accumulate
    auto bin = [&](int j, bool masked, bool with_sg, R& zr, R& zi, R& sg) {
      const R cr = Pr, sr = Pi;
      rot_step();
      // amplitudes
      const R Ar = fma(fma(fma(cf[0][3], s, cf[0][2]), s, cf[0][1]), s, cf[0][0]);
      const R Ai = fma(fma(fma(cf[1][3], s, cf[1][2]), s, cf[1][1]), s, cf[1][0]);
      const R Er = fma(fma(fma(cf[2][3], s, cf[2][2]), s, cf[2][1]), s, cf[2][0]);
      const R Ei = fma(fma(fma(cf[3][3], s, cf[3][2]), s, cf[3][1]), s, cf[3][0]);
      s += hS;
      const WT w = sW[j - cs];
      // q = W_A conj(c_A) + W_E conj(c_E)
      R qr = fma(w.x, Ar, fma(w.y, Ai, fma(w.z, Er, w.w * Ei)));
      R qi = fma(w.y, Ar, fma(-w.x, Ai, fma(w.w, Er, -(w.z * Ei))));
      R ss = R(0.0);
      if (with_sg) {
        const GT g = sG[j - cs];
        ss = fma(g.x, fma(Ar, Ar, Ai * Ai), g.y * fma(Er, Er, Ei * Ei));
      }
      if (masked) {
        const bool in = (j >= jlo) && (j < jhi);
        qr = in ? qr : R(0.0); qi = in ? qi : R(0.0); ss = in ? ss : R(0.0);
      }
      // z += q e^{+2 pi i Phi}
      zr = fma(qr, cr, fma(-qi, sr, zr));
      zi = fma(qr, sr, fma(qi, cr, zi));
      sg += ss;
    };

    // all lanes inside their windows and moments available: sigma per piece from the moments, not per bin
    const bool use_mom = all_in && (a.moments64 != nullptr);
    int piece = use_mom ? a.piece_first[(ib >> (c.log2_stride - 2)) - ((a.chunk_first * CH) >> (c.log2_stride - 2))] : 0;
    int j = ib;
    while (j < ie) {
      const int b = min(next_edge, ie);
      const bool live = (k >= 0) && (k < a.n_seg);
      if (b > j) {
        if (all_out) {
          // nothing to add; the recurrence is re-seeded at the next sub-interval
        } else if (!live) {
          for (int jj = j; jj < b; ++jj) { rot_step(); s += hS; }
        } else if (use_mom) {
          // Fast path (every lane of the warp inside its window, sigma from the moments): with c = g0 + delta,
          //   z_piece = conj(g0_A) T_A + conj(g0_E) T_E + sum_j [w_A conj(delta_A) + w_E conj(delta_E)] P_j,  T_a = sum_j w_a P_j.
          // T_a is accumulated in FP64 (8 operations per bin, with the recurrence 18 in all against 37 for the direct
          // form); the correction sum runs on the otherwise idle FP32 pipe and is folded into FP64 every kFlushBins bins.
          double TAr = 0.0, TAi = 0.0, TEr = 0.0, TEi = 0.0;
          float d = (float)(j - ib) * (float)hS - 0.5f;          // exact: multiples of 1/Sf
          const float hSf = (float)hS;
          for (int jj = j; jj < b;) {
            const int e2 = min(jj + kFlushBins, b);
            float zr = 0.f, zi = 0.f;
            for (; jj < e2; ++jj) {
              const WT w = sW[jj - cs];
              const float4 v = sW32[jj - cs];
              const float pr = (float)Pr, pi = (float)Pi;
              TAr = fma(w.x, Pr, fma(-w.y, Pi, TAr)); TAi = fma(w.x, Pi, fma(w.y, Pr, TAi));
              TEr = fma(w.z, Pr, fma(-w.w, Pi, TEr)); TEi = fma(w.z, Pi, fma(w.w, Pr, TEi));
              rot_step();
              const float dAr = d * fmaf(fmaf(g3[0], d, g2[0]), d, g1[0]), dAi = d * fmaf(fmaf(g3[1], d, g2[1]), d, g1[1]);
              const float dEr = d * fmaf(fmaf(g3[2], d, g2[2]), d, g1[2]), dEi = d * fmaf(fmaf(g3[3], d, g2[3]), d, g1[3]);
              d += hSf;
              const float qr = fmaf(v.x, dAr, fmaf(v.y, dAi, fmaf(v.z, dEr, v.w * dEi)));
              const float qi = fmaf(v.y, dAr, fmaf(-v.x, dAi, fmaf(v.w, dEr, -(v.z * dEi))));
              zr = fmaf(qr, pr, fmaf(-qi, pi, zr));
              zi = fmaf(qr, pi, fmaf(qi, pr, zi));
            }
            Zr += (double)zr; Zi += (double)zi;
          }
          Zr += fma(g0[0], TAr, fma(g0[1], TAi, fma(g0[2], TEr, g0[3] * TEi)));
          Zi += fma(g0[0], TAi, fma(-g0[1], TAr, fma(g0[2], TEi, -(g0[3] * TEr))));
          s = (R)(b - ib) * hS;
          Sg += sigma_moments64(cf, a.moments64 + (size_t)piece * 7);
        } else {
          for (int jj = j; jj < b;) {
            const int e2 = min(jj + kFlushBins, b);
            R zr = R(0.0), zi = R(0.0), sg = R(0.0);
            if (all_in)      { for (; jj < e2; ++jj) bin(jj, false, true, zr, zi, sg); }
            else             { for (; jj < e2; ++jj) bin(jj, true, true, zr, zi, sg); }
            Zr += (double)zr; Zi += (double)zi; Sg += (double)sg;
          }
        }
        ++piece;
        j = b;
      }
      if (j == next_edge) {
        if (live) close_piece(true);
        ++k;
        next_edge = (k + 1 <= a.n_seg) ? a.edges[k + 1] : INT_MAX;
        open_at_edge = true;
      }
    }
  }
  // the piece still open at the chunk end
  if (k >= 0 && k < a.n_seg) close_piece(false);
  if (!SEG) {
    frag[0] = ups;
    if (a.comp) { frag[(size_t)7 * a.P_pad] = xs; frag[(size_t)8 * a.P_pad] = hs; }
  }
  if (!ESC) return;
  }
}

}  // namespace
