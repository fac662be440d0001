// sc_kernels_dense32x3.cuh -- a4 + a5 for three TDI channels A, E, T (Eq. 1 and Eq. 7 sum over all three)
// in ONE pass: the FP32-amplitude hot loop of k_dense2 with a third channel in the pair loop.  Part of libscstat.so.
//
// Same mapping and walk as k_dense2 (lane = particle, warp walks the bins of its chunk, segment edges shared, pieces
// finalised in registers, fragments stitched by k_stitch); what changes is the per-bin arithmetic:
//   q_j = W_A conj(c_A) + W_E conj(c_E) + W_T conj(c_T),   sigma_j = G_A |c_A|^2 + G_E |c_E|^2 + G_T |c_T|^2,
// 18 + 12 + 4 packed FMAs per bin pair instead of 12 + 8 + 4, against twice the whole loop (phase, sin/cos included) for a
// second pass plus per-segment tables.  The node tables carry six amplitude fields (k_nodes<.., 6>, DevCfg.chan_set = 2), the
// chunk's data three records per bin pair (wA, wE, wT); the sigma weights of the rare masked bins (band edges) are read
// from global memory.  T's data and weights are rescaled to the (A, E) handle's power-of-two scale s0 when the fused tables
// are built (k_fuse3), so that one scale converts the sums back to definition units.
#pragma once
#include "sc_common.cuh"

namespace {

constexpr int kPairRec3 = 3;   // shared-memory records per bin pair: (wAr, wAi), (wEr, wEi), (wTr, wTi), each (even bin, odd bin)

// Fused data tables of a three-channel handle: D3 = per bin pair (wA, wE, wT); Gp = per bin pair (gA, gE), (gT, 0);
// GT64 = (gT, 0) per bin in FP64 for the sigma moments.  r = s0_T / s0_AE (a power of two: exact).
__global__ void k_fuse3(const float4* __restrict__ D_ae, const float4* __restrict__ D_t, const double2* __restrict__ G_t,
                        int n_pairs_pad, int n_bins, float r, float4* __restrict__ D3, float4* __restrict__ Gp,
                        double2* __restrict__ GT64) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n_pairs_pad) return;
  const float4 wt = D_t[3 * (size_t)m], gt = D_t[3 * (size_t)m + 2];
  D3[3 * (size_t)m] = D_ae[3 * (size_t)m];
  D3[3 * (size_t)m + 1] = D_ae[3 * (size_t)m + 1];
  D3[3 * (size_t)m + 2] = make_float4(wt.x * r, wt.y * r, wt.z * r, wt.w * r);
  Gp[2 * (size_t)m] = D_ae[3 * (size_t)m + 2];
  Gp[2 * (size_t)m + 1] = make_float4(gt.x * r * r, gt.y * r * r, 0.f, 0.f);
  const double r2 = (double)r * (double)r;
  if (2 * m < n_bins) GT64[2 * m] = make_double2(G_t[2 * m].x * r2, 0.0);
  if (2 * m + 1 < n_bins) GT64[2 * m + 1] = make_double2(G_t[2 * m + 1].x * r2, 0.0);
}

// Cubic coefficients of (Ar, Ai, Er, Ei, Tr, Ti) on the fine sub-interval starting at ib, in s = (j - ib)/Sf (see sub_amps).
template <typename NT = float>   // element type of the node table (double in the per-particle-segment path)
__device__ __forceinline__ void sub_amps3(const DevCfg& c, const DenseArgs& a, int p, int ib, float (&cf)[6][4]) {
  const int i0 = (ib >> c.log2_stride) + kNodeOff;
  const int q = (ib >> (c.log2_stride - 2)) & 3;
  const NT* __restrict__ namp = reinterpret_cast<const NT*>(a.node_amp);
#pragma unroll
  for (int r = 0; r < 6; r += 2) {
    const NT* col = namp + ((size_t)i0 * 6 + r) * a.P_pad + p;
    const ptrdiff_t st = (ptrdiff_t)6 * a.P_pad;
    u64 nd[6], o[4];
#pragma unroll
    for (int m = -2; m <= 3; ++m) nd[m + 2] = f2pack((float)col[m * st], (float)col[m * st + a.P_pad]);
    fine_cubic2(nd, q, o);
#pragma unroll
    for (int kk = 0; kk < 4; ++kk) f2unpack(o[kk], cf[r][kk], cf[r + 1][kk]);
  }
}

__device__ __forceinline__ u64 horner2(const float (&c4)[4], u64 s2) {
  return f2fma(f2fma(f2fma(f2bcast(c4[3]), s2, f2bcast(c4[2])), s2, f2bcast(c4[1])), s2, f2bcast(c4[0]));
}

// amplitude cubics of the three channels at (s_j, s_{j+1}), q = sum_a W_a conj(c_a), z += q e^{+2 pi i Phi}
__device__ __forceinline__ void mac_pair3(const float (&cf)[6][4], u64& s2, const ulonglong2 wA, const ulonglong2 wE,
                                          const ulonglong2 wT, u64 h2, u64 cr2, u64 sr2, u64& zr2, u64& zi2) {
  const u64 Ar = horner2(cf[0], s2), Ai = horner2(cf[1], s2), Er = horner2(cf[2], s2), Ei = horner2(cf[3], s2);
  const u64 Tr = horner2(cf[4], s2), Ti = horner2(cf[5], s2);
  s2 = f2add(s2, h2);
  const u64 qr = f2fma(wA.x, Ar, f2fma(wA.y, Ai, f2fma(wE.x, Er, f2fma(wE.y, Ei, f2fma(wT.x, Tr, f2mul(wT.y, Ti))))));
  const u64 qi = f2fma(wA.y, Ar, f2fma(f2neg(wA.x), Ai, f2fma(wE.y, Er, f2fma(f2neg(wE.x), Ei, f2fma(wT.y, Tr, f2neg(f2mul(wT.x, Ti)))))));
  zr2 = f2fma(qr, cr2, f2fma(f2neg(qi), sr2, zr2));
  zi2 = f2fma(qr, sr2, f2fma(qi, cr2, zi2));
}

// One bin pair with the particle's time window applied per bin and sigma per bin (band-edge sub-intervals).
// rec: the pair's three data records (shared memory); grec: its two weight records (global memory).
template <int SC>
__device__ __forceinline__ void pair_eval3(PhaseFD& ph, const float (&cf)[6][4], u64& s2, const ulonglong2*& rec,
                                           const ulonglong2* __restrict__ grec, int j, int jlo, int jhi, u64 h2, u64 K2,
                                           u64& zr2, u64& zi2, u64& sg2) {
  u64 cr2, sr2;
  sincos_pair<SC>(ph, K2, cr2, sr2);
  const u64 m2 = f2pack((j >= jlo && j < jhi) ? 1.0f : 0.0f, (j + 1 >= jlo && j + 1 < jhi) ? 1.0f : 0.0f);
  cr2 = f2mul(cr2, m2); sr2 = f2mul(sr2, m2);
  const u64 Ar = horner2(cf[0], s2), Ai = horner2(cf[1], s2), Er = horner2(cf[2], s2), Ei = horner2(cf[3], s2);
  const u64 Tr = horner2(cf[4], s2), Ti = horner2(cf[5], s2);
  const ulonglong2 gAE = grec[0], gT = grec[1];
  sg2 = f2fma(f2mul(gAE.x, m2), f2fma(Ar, Ar, f2mul(Ai, Ai)),
              f2fma(f2mul(gAE.y, m2), f2fma(Er, Er, f2mul(Ei, Ei)), f2fma(f2mul(gT.x, m2), f2fma(Tr, Tr, f2mul(Ti, Ti)), sg2)));
  u64 s2c = s2;
  // (the multiply-accumulate re-evaluates the cubics: this path is rare, the code stays in one place)
  mac_pair3(cf, s2c, rec[0], rec[1], rec[2], h2, cr2, sr2, zr2, zi2);
  s2 = s2c;
  rec += kPairRec3;
}

// sigma of a run of bins from the moments of its weights, three channels: (A, E) packed as in sigma_moments, then (T, 0)
__device__ __forceinline__ double sigma_moments3(const float (&cf)[6][4], const ulonglong2* __restrict__ mp, const ulonglong2* __restrict__ mpT) {
  const float cT[4][4] = {{cf[4][0], cf[4][1], cf[4][2], cf[4][3]}, {cf[5][0], cf[5][1], cf[5][2], cf[5][3]},
                          {0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
  return sigma_moments(*reinterpret_cast<const float(*)[4][4]>(&cf[0]), mp) + sigma_moments(cT, mpT);
}

// n >= 1 consecutive unmasked pairs, software-pipelined like pairs_fast
template <int SC>
__device__ __forceinline__ void pairs_fast3(PhaseFD& ph, const float (&cf)[6][4], u64& s2, const ulonglong2*& rec, int n,
                                            u64 h2, u64 K2, u64& zr2, u64& zi2) {
  u64 cr, sr;
  sincos_pair<SC>(ph, K2, cr, sr);
  ulonglong2 wA = rec[0], wE = rec[1], wT = rec[2];
#pragma unroll 1
  for (int i = 1; i < n; ++i) {
    u64 crn, srn;
    sincos_pair<SC>(ph, K2, crn, srn);
    rec += kPairRec3;
    const ulonglong2 wAn = rec[0], wEn = rec[1], wTn = rec[2];
    mac_pair3(cf, s2, wA, wE, wT, h2, cr, sr, zr2, zi2);
    cr = crn; sr = srn; wA = wAn; wE = wEn; wT = wTn;
  }
  rec += kPairRec3;
  mac_pair3(cf, s2, wA, wE, wT, h2, cr, sr, zr2, zi2);
}

// QUAD flavour for six amplitude parts (see pairs_fast_q in sc_kernels_dense32.cuh): quadratic amplitudes over runs of a
// quarter sub-interval, 12 packed FMAs per bin pair instead of 18.  Used by k_dense2_ad<.., 6> and by k_dense3<.., QUAD>.
struct QuadState3 { float q[6][3]; u64 u2; int left; int r; };
__device__ __forceinline__ void quad_run3(const float (&cf)[6][4], int r, QuadState3& o) {
  const float s0 = 0.25f * (float)r;
#pragma unroll
  for (int a = 0; a < 6; ++a) {
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
__device__ __forceinline__ void quad_start3(const float (&cf)[6][4], int off, int lg_run, QuadState3& q) {
  const int run_bins = 1 << lg_run;
  const int o = off & (run_bins - 1);
  const float hu = 1.0f / (float)run_bins;
  q.r = off >> lg_run;
  q.left = (run_bins - o) >> 1;
  q.u2 = f2pack((float)o * hu, (float)(o + 1) * hu);
  quad_run3(cf, q.r, q);
}
__device__ __forceinline__ u64 quad2(const float (&w)[3], u64 u2) { return f2fma(f2fma(f2bcast(w[2]), u2, f2bcast(w[1])), u2, f2bcast(w[0])); }
__device__ __forceinline__ void mac_pair3_q(QuadState3& w, const ulonglong2 wA, const ulonglong2 wE, const ulonglong2 wT, u64 hu2,
                                            u64 cr2, u64 sr2, u64& zr2, u64& zi2) {
  const u64 Ar = quad2(w.q[0], w.u2), Ai = quad2(w.q[1], w.u2), Er = quad2(w.q[2], w.u2), Ei = quad2(w.q[3], w.u2);
  const u64 Tr = quad2(w.q[4], w.u2), Ti = quad2(w.q[5], w.u2);
  w.u2 = f2add(w.u2, hu2);
  const u64 qr = f2fma(wA.x, Ar, f2fma(wA.y, Ai, f2fma(wE.x, Er, f2fma(wE.y, Ei, f2fma(wT.x, Tr, f2mul(wT.y, Ti))))));
  const u64 qi = f2fma(wA.y, Ar, f2fma(f2neg(wA.x), Ai, f2fma(wE.y, Er, f2fma(f2neg(wE.x), Ei, f2fma(wT.y, Tr, f2neg(f2mul(wT.x, Ti)))))));
  zr2 = f2fma(qr, cr2, f2fma(f2neg(qi), sr2, zr2));
  zi2 = f2fma(qr, sr2, f2fma(qi, cr2, zi2));
}
template <int SC>
__device__ __forceinline__ void pairs_fast3_q(PhaseFD& ph, const float (&cf)[6][4], QuadState3& q, int lg_run, const ulonglong2*& rec,
                                              int n, u64 K2, u64& zr2, u64& zi2) {
  const int run_pairs = 1 << (lg_run - 1);
  const float hu = 1.0f / (float)(2 * run_pairs);
  const u64 hu2 = f2bcast(2.0f * hu);
  u64 cr, sr;
  sincos_pair<SC>(ph, K2, cr, sr);
  ulonglong2 wA = rec[0], wE = rec[1], wT = rec[2];
#pragma unroll 1
  for (int i = 1; i < n; ++i) {
    u64 crn, srn;
    sincos_pair<SC>(ph, K2, crn, srn);
    rec += kPairRec3;
    const ulonglong2 wAn = rec[0], wEn = rec[1], wTn = rec[2];
    mac_pair3_q(q, wA, wE, wT, hu2, cr, sr, zr2, zi2);
    if (--q.left == 0) { quad_run3(cf, ++q.r, q); q.left = run_pairs; q.u2 = f2pack(0.0f, hu); }
    cr = crn; sr = srn; wA = wAn; wE = wEn; wT = wTn;
  }
  rec += kPairRec3;
  mac_pair3_q(q, wA, wE, wT, hu2, cr, sr, zr2, zi2);
  if (--q.left == 0) { quad_run3(cf, ++q.r, q); q.left = run_pairs; q.u2 = f2pack(0.0f, hu); }
}

#ifndef SC_DENSE3_MINB
#define SC_DENSE3_MINB 4     /* CTAs per SM: 128 registers/thread with ~150 B of spills beats 168 registers at 3 CTAs (28.6 vs 32.0 ms on c3) */
#endif
#ifndef SC_DENSE3_QUAD_MINB
#define SC_DENSE3_QUAD_MINB 3   /* QUAD flavour: 24 cubic + 18 quadratic coefficients live -- 168 registers at 3 CTAs per SM 25.6 ms on c3,
                                   128 registers at 4 CTAs (232 B of spills) 29.7 ms, 255 registers at 2 CTAs 26.5 ms; cubic flavour 26.9 ms */
#endif
template <bool SEG, int SC, bool QUAD = false>
__global__ void __launch_bounds__(kBlock, QUAD ? SC_DENSE3_QUAD_MINB : SC_DENSE3_MINB) k_dense3(DevCfg c, DenseArgs a, const ulonglong2* __restrict__ Dg,
                                                                   const ulonglong2* __restrict__ Gp) {
  constexpr int CH = kChunkF32;
  __shared__ ulonglong2 sD[CH / 2 * kPairRec3];                // 48 KB

  const int chunk_l = blockIdx.x;
  const int cs = (a.chunk_first + chunk_l) * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int ce2 = (ce + 1) & ~1;                               // pair-aligned end (data beyond n_bins is zero)
  const int p = blockIdx.y * kBlock + threadIdx.x;

  if (!__syncthreads_or((a.jhi[p] > cs) && (a.jlo[p] < ce))) {     // (see k_dense2: only k_stitch_seg reads these fragments)
    if constexpr (SEG) {
      double* fz = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + p;
#pragma unroll
      for (int m = 0; m < kFragFields; ++m) fz[(size_t)m * a.P_pad] = 0.0;
    }
    return;
  }
  {
    const ulonglong2* src = Dg + (size_t)(cs >> 1) * kPairRec3;
#pragma unroll 4
    for (int t = threadIdx.x; t < CH / 2 * kPairRec3; t += kBlock) sD[t] = src[t];
  }
  __syncthreads();

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
  for (int ib = cs; ib < ce2; ib += Sf) {
    const int ie = min(ib + Sf, ce2);
    const bool lane_in = (ib >= jlo) && (ie <= jhi);
    const bool lane_out = (ie <= jlo) || (ib >= jhi);
    const bool all_in = __all_sync(0xffffffffu, lane_in);
    const bool all_out = __all_sync(0xffffffffu, lane_out);

    float cf[6][4];    // cubic coefficients of (Ar, Ai, Er, Ei, Tr, Ti) in s = (j - ib)/Sf
    if (!all_out) {
      sub_phase(c, a, p, ib, fd);
      sub_amps3(c, a, p, ib, cf);
    }
    u64 s2 = 0;        // (s_j, s_{j+1}) of the next pair
    const ulonglong2* rec = sD;   // its data records
    auto sigma_piece = [&](int piece) { Sg += sigma_moments3(cf, a.moments + (size_t)piece * 4, a.momentsT + (size_t)piece * 4); };
    const bool use_mom = all_in;      // all lanes inside their windows: sigma from the piece moments, unmasked pairs
    int piece = use_mom ? a.piece_first[(ib >> (c.log2_stride - 2)) - ((a.chunk_first * CH) >> (c.log2_stride - 2))] : 0;
    float car_zr = 0.f, car_zi = 0.f, car_sg = 0.f;
    bool carry = false;
    QuadState3 qs;
    int q_pos = -1;            // the bin qs stands at (see k_dense2)
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
        rec = sD + ((jj - cs) >> 1) * kPairRec3;
        if constexpr (QUAD) { if (use_mom && jj < ph && q_pos != jj) quad_start3(cf, jj - ib, c.log2_stride - 4, qs); }
        while (jj < ph) {
          const bool split = (jj == jfull);                    // the pair (ph - 1, ph)
          const int e2 = split ? jj + 2 : min(jj + ((QUAD && use_mom) ? SC_QUAD_FLUSH : kFlushBins), jfull);
          u64 zr2 = 0, zi2 = 0, sg2 = 0;
          if (use_mom) {
            if constexpr (QUAD) { pairs_fast3_q<SC>(fd, cf, qs, c.log2_stride - 4, rec, (e2 - jj) >> 1, K2, zr2, zi2); q_pos = e2; }
            else pairs_fast3<SC>(fd, cf, s2, rec, (e2 - jj) >> 1, h2, K2, zr2, zi2);
            jj = e2;
          }
          else {
            for (; jj < e2; jj += 2) pair_eval3<SC>(fd, cf, s2, rec, Gp + (size_t)(jj >> 1) * 2, jj, jlo, jhi, h2, K2, zr2, zi2, sg2);
          }
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
  if (k >= 0 && k < a.n_seg) close_piece(false);
  if (!SEG) {
    frag[0] = ups;
    if (a.comp) { frag[(size_t)7 * a.P_pad] = xs; frag[(size_t)8 * a.P_pad] = hs; }
  }
}

}  // namespace
