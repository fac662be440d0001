// sc_kernels_adaptive.cuh -- per-particle equal-SNR^2 segments (App. A).
// Part of libscstat.so (one translation unit: sc_stat.cu includes the kernel files in pipeline order).
#pragma once
#include "sc_common.cuh"

namespace {

// ------------------------------------------------------------------------------------------------ per-particle segments
// Equal squared-SNR segments re-evaluated for every particle (App. A):
//   s_j = sum_a |h_a(f_j)|^2 / S_a(f_j),  C = sum_j s_j,  e_0 = 0, e_N = n_bins,
//   e_n = min{ j : sum_{j' < j} s_j' >= C n / N }   (n = 1 .. N-1),
// then Upsilon_N on those edges.  Three steps, all with lane = particle:
//   k_sigma_chunks   sigma of every (chunk, particle) from the moments of the weights (no per-bin work inside the window)
//   k_scan_chunks    prefix sum over chunks -> cumulative sigma at every chunk start, and C
//   k_dense2_ad      the hot loop of k_dense2 with a running cumulative sigma per lane: groups of <= 32 bins in which
//                    no lane of the warp reaches its next target (decided from the group's moments) take the unmasked
//                    packed path; the others are walked bin by bin and the segments are closed where the running sum
//                    crosses the target.  The number of edges closed inside a chunk is fixed by the scanned sums
//                    (k0 = K(cbase[chunk]), k1 = K(cbase[chunk + 1])), so neighbouring chunks always agree.
constexpr int kFragAd = 10;    // partial Upsilon, head (zr, zi, sg), tail (zr, zi, sg), head-closes flag, partial sum|z|, sum sigma

struct AdaptArgs {
  int n_seg, n_chunks;
  const double* cbase;         // [n_chunks + 1][P_pad]: cumulative sigma at the chunk starts; row n_chunks = C
  const ulonglong2* gmom;      // [n_groups][4] moments of the weights over groups of 2^lg_group bins
  const ulonglong2* smom;      // [n_sub][4]    ... over the fine sub-intervals
  int lg_group;
  int* out_edges;              // [P][n_seg + 1] of this batch, or nullptr
  double* chunk_sigma;         // = cbase (written by k_sigma_chunks before the scan)
  const int* pmap;             // window sort: table slot -> particle of the batch (rows of out_edges), or nullptr
};

__device__ __forceinline__ double seg_target(double C, int n, int N) { return C * (double)n / (double)N; }
// K(c) = max{ n in [0, N-1] : C n / N <= c }: the segment that contains the first bin whose cumulative sum is c.
__device__ __forceinline__ int seg_index(double cum, double C, int N) {
  if (!(C > 0.0)) return 0;
  int n = (int)(cum / C * (double)N);
  n = min(max(n, 0), N - 1);
  while (n + 1 <= N - 1 && seg_target(C, n + 1, N) <= cum) ++n;
  while (n > 0 && seg_target(C, n, N) > cum) --n;
  return n;
}

__global__ void __launch_bounds__(kBlock) k_sigma_chunks(DevCfg c, DenseArgs a, AdaptArgs ad, const float4* __restrict__ D32) {
  constexpr int CH = kChunkF32;
  const int chunk = blockIdx.x;
  const int cs = chunk * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int ce2 = (ce + 1) & ~1;
  const int p = blockIdx.y * kBlock + threadIdx.x;
  const int jlo = a.jlo[p], jhi = a.jhi[p];
  if (!__syncthreads_or((jhi > cs) && (jlo < ce))) {          // no particle of this block lives in this chunk
    ad.chunk_sigma[(size_t)(chunk + 1) * a.P_pad + p] = 0.0;
    return;
  }
  const int Sf = c.stride >> 2;
  const float hS = 1.0f / (float)Sf;
  double tot = 0.0;
  for (int ib = cs; ib < ce2; ib += Sf) {
    const int ie = min(ib + Sf, ce2);
    const bool lane_in = (ib >= jlo) && (ie <= jhi);
    const bool lane_out = (ie <= jlo) || (ib >= jhi);
    const bool all_in = __all_sync(0xffffffffu, lane_in);
    const bool all_out = __all_sync(0xffffffffu, lane_out);
    if (all_out) continue;
    float cf[4][4];
    sub_amps(c, a, p, ib, cf);
    if (all_in) {
      tot += sigma_moments(cf, ad.smom + (size_t)(ib >> (c.log2_stride - 2)) * 4);
    } else {
      // a window border of some lane falls in this sub-interval: bin by bin, masked (two sub-intervals per particle)
      for (int j = ib; j < ie; ++j) {
        const float sj = (float)(j - ib) * hS;
        const float Ar = fmaf(fmaf(fmaf(cf[0][3], sj, cf[0][2]), sj, cf[0][1]), sj, cf[0][0]);
        const float Ai = fmaf(fmaf(fmaf(cf[1][3], sj, cf[1][2]), sj, cf[1][1]), sj, cf[1][0]);
        const float Er = fmaf(fmaf(fmaf(cf[2][3], sj, cf[2][2]), sj, cf[2][1]), sj, cf[2][0]);
        const float Ei = fmaf(fmaf(fmaf(cf[3][3], sj, cf[3][2]), sj, cf[3][1]), sj, cf[3][0]);
        const float4 g = D32[(size_t)(j >> 1) * kPairRec + 2];            // (gA even, gA odd, gE even, gE odd)
        const float gA = (j & 1) ? g.y : g.x, gE = (j & 1) ? g.w : g.z;
        const float sg = fmaf(gA, fmaf(Ar, Ar, Ai * Ai), gE * fmaf(Er, Er, Ei * Ei));
        if (j >= jlo && j < jhi) tot += (double)sg;
      }
    }
  }
  ad.chunk_sigma[(size_t)(chunk + 1) * a.P_pad + p] = tot;
}

__global__ void k_scan_chunks(double* __restrict__ cbase, int n_chunks, int P_pad) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= P_pad) return;
  double acc = 0.0;
  cbase[p] = 0.0;
  constexpr int kU = 8;                          // loads of kU chunks in flight; the sum itself stays in chunk order
  for (int i0 = 1; i0 <= n_chunks; i0 += kU) {
    double v[kU];
#pragma unroll
    for (int u = 0; u < kU; ++u) v[u] = cbase[(size_t)min(i0 + u, n_chunks) * P_pad + p];
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      if (i0 + u > n_chunks) break;
      acc += v[u];
      cbase[(size_t)(i0 + u) * P_pad + p] = acc;
    }
  }
}

template <int SC, bool MERGE = false>
__global__ void __launch_bounds__(kBlock, SC_DENSE2_MINB) k_dense2_ad(DevCfg c, DenseArgs a, AdaptArgs ad,
                                                                      const ulonglong2* __restrict__ Dg) {
  constexpr int CH = kChunkF32;
  __shared__ ulonglong2 sD[CH / 2 * kPairRec];
  const int chunk = blockIdx.x;
  const int cs = chunk * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int ce2 = (ce + 1) & ~1;
  const int p = blockIdx.y * kBlock + threadIdx.x;
  const int jlo = a.jlo[p], jhi = a.jhi[p];
  // no particle of this block lives in this chunk: its cumulative sigma does not move here, so no edge falls into the
  // chunk (k == k1 below) -- the fragments of "nothing happened", without staging the data
  if (!__syncthreads_or((jhi > cs) && (jlo < ce))) {
    double* fz = a.frag + (size_t)chunk * kFragAd * a.P_pad + p;
#pragma unroll
    for (int m = 0; m < kFragAd; ++m) fz[(size_t)m * a.P_pad] = 0.0;
    return;
  }
  {
    const ulonglong2* src = Dg + (size_t)(cs >> 1) * kPairRec;
#pragma unroll 4
    for (int t = threadIdx.x; t < CH / 2 * kPairRec; t += kBlock) sD[t] = src[t];
  }
  __syncthreads();

  const int Sf = c.stride >> 2;
  const float hS = 1.0f / (float)Sf;
  const u64 h2 = f2bcast(2.0f * hS);
  const u64 K2 = f2bcast(1.4629180792671596e-09f);
  const int N = ad.n_seg;
  const int Gs = 1 << ad.lg_group;

  const double C = ad.cbase[(size_t)ad.n_chunks * a.P_pad + p];
  const double cb0 = ad.cbase[(size_t)chunk * a.P_pad + p];
  const double cb1 = ad.cbase[(size_t)(chunk + 1) * a.P_pad + p];
  int k = seg_index(cb0, C, N);                 // segment open at the chunk start
  const int k1 = seg_index(cb1, C, N);          // edges k+1 .. k1 are closed inside this chunk, no more, no fewer
  double t_next = (k < k1) ? seg_target(C, k + 1, N) - cb0 : INFINITY;
  double crel = 0.0, c_open = 0.0;              // cumulative sigma relative to the chunk start; its value where the open piece began
  double Zr = 0.0, Zi = 0.0, ups = 0.0, xs = 0.0, hs = 0.0;
  bool closed_any = false;
  double* frag = a.frag + (size_t)chunk * kFragAd * a.P_pad + p;
  const int pq = ad.pmap ? ad.pmap[p] : p;      // particle of the batch in this table slot

  auto close_at = [&](int j) {                  // edge k+1 lies at bin j
    const double Sg = crel - c_open;
    if (!closed_any) {                          // the piece that was open at the chunk start: head fragment
      frag[(size_t)1 * a.P_pad] = Zr; frag[(size_t)2 * a.P_pad] = Zi; frag[(size_t)3 * a.P_pad] = Sg;
      closed_any = true;
    } else if (Sg > 0.0) {
      const double z2 = Zr * Zr + Zi * Zi;
      ups += z2 / Sg;
      if (a.comp) { xs += sqrt(z2); hs += Sg; }
    }
    Zr = 0.0; Zi = 0.0; c_open = crel;
    ++k;
    if (ad.out_edges && pq < a.P) ad.out_edges[(size_t)pq * (N + 1) + k] = j;
    t_next = (k < k1) ? seg_target(C, k + 1, N) - cb0 : INFINITY;
  };

  PhaseFD ph = {};
  float cc[MERGE ? 4 : 1][4];
  int merged_left = 0;
  for (int ib = cs; ib < ce2; ib += Sf) {
    const int ie = min(ib + Sf, ce2);
    const bool lane_in = (ib >= jlo) && (ie <= jhi);
    const bool lane_out = (ie <= jlo) || (ib >= jhi);
    const bool all_in = __all_sync(0xffffffffu, lane_in);
    const bool all_out = __all_sync(0xffffffffu, lane_out);
    if (all_out) continue;
    float cf[4][4];
    // merged coarse intervals as in k_dense2 (the group and sub-interval moments stay those of the fine sub-intervals)
    if constexpr (MERGE) {
      if (merged_left == 0 && (ib & (c.stride - 1)) == 0 && ib + c.stride <= ce2 &&
          __all_sync(0xffffffffu, (ib >= jlo) && (ib + c.stride <= jhi)) &&
          __all_sync(0xffffffffu, coarse_dslope(c, a, p, ib >> c.log2_stride) <= a.merge_lim)) {
        coarse_phase(c, a, p, ib, ph);
        coarse_amps(c, a, p, ib, cc);
        merged_left = 4;
      }
    }
    if (MERGE && merged_left > 0) {
      if constexpr (MERGE) coarse_to_fine(cc, 4 - merged_left, cf);
      --merged_left;
    } else {
      sub_phase(c, a, p, ib, ph);
      sub_amps(c, a, p, ib, cf);
    }
    u64 s2 = f2pack(0.0f, hS);
    const ulonglong2* rec = sD + ((ib - cs) >> 1) * kPairRec;
    // First ask the question for the whole sub-interval (its moments are those k_sigma_chunks used): if no lane reaches its
    // next target in it, all its groups take the unmasked path and the group moments are not needed at all.
    if (all_in && ie - ib == Sf) {
      const double sg_s = sigma_moments(cf, ad.smom + (size_t)(ib >> (c.log2_stride - 2)) * 4);
      const bool cross_s = (k < k1) && (crel + sg_s * 1.0001 >= t_next);
      if (!__any_sync(0xffffffffu, cross_s)) {
        for (int gs = ib; gs < ie; gs += Gs) {
          u64 zr2 = 0, zi2 = 0;
          pairs_fast<SC>(ph, cf, s2, rec, Gs >> 1, h2, K2, zr2, zi2);
          float zrl, zrh, zil, zih;
          f2unpack(zr2, zrl, zrh); f2unpack(zi2, zil, zih);
          Zr += (double)(zrl + zrh); Zi += (double)(zil + zih);
        }
        crel += sg_s;
        continue;
      }
    }
    for (int gs = ib; gs < ie; gs += Gs) {
      const int ge = min(gs + Gs, ie);
      const double sg_m = sigma_moments(cf, ad.gmom + (size_t)(gs >> ad.lg_group) * 4);
      // would the running sum reach this lane's next target inside the group?  (margin: the per-bin and the moment sums
      // differ by FP32 rounding; a group flagged needlessly only takes the slower path)
      const bool cross = (k < k1) && (crel + sg_m * 1.0001 >= t_next);
      const bool slow = !all_in || __any_sync(0xffffffffu, cross);
      if (!slow) {
        u64 zr2 = 0, zi2 = 0;
        pairs_fast<SC>(ph, cf, s2, rec, (ge - gs) >> 1, h2, K2, zr2, zi2);
        float zrl, zrh, zil, zih;
        f2unpack(zr2, zrl, zrh); f2unpack(zi2, zil, zih);
        Zr += (double)(zrl + zrh); Zi += (double)(zil + zih);
        crel += sg_m;
      } else {
        for (int jj = gs; jj < ge; jj += 2) {
          u64 zr2 = 0, zi2 = 0, sg2 = 0;
          pair_eval<true, true, SC>(ph, cf, s2, rec, jj, jlo, jhi, h2, K2, zr2, zi2, sg2);
          float zrl, zrh, zil, zih, sgl, sgh;
          f2unpack(zr2, zrl, zrh); f2unpack(zi2, zil, zih); f2unpack(sg2, sgl, sgh);
          while (k < k1 && crel >= t_next) close_at(jj);          // e_n = first bin whose cumulative sum reached the target
          Zr += (double)zrl; Zi += (double)zil; crel += (double)sgl;
          while (k < k1 && crel >= t_next) close_at(jj + 1);
          Zr += (double)zrh; Zi += (double)zih; crel += (double)sgh;
        }
      }
    }
  }
  while (k < k1) close_at(ce);                  // targets the scanned sums place in this chunk (rounding): at its end
  const double Sg = crel - c_open;
  if (!closed_any) {
    frag[(size_t)1 * a.P_pad] = Zr; frag[(size_t)2 * a.P_pad] = Zi; frag[(size_t)3 * a.P_pad] = Sg;
    frag[(size_t)4 * a.P_pad] = 0.0; frag[(size_t)5 * a.P_pad] = 0.0; frag[(size_t)6 * a.P_pad] = 0.0;
  } else {
    frag[(size_t)4 * a.P_pad] = Zr; frag[(size_t)5 * a.P_pad] = Zi; frag[(size_t)6 * a.P_pad] = Sg;
  }
  frag[(size_t)7 * a.P_pad] = closed_any ? 1.0 : 0.0;
  frag[0] = ups;
  if (a.comp) { frag[(size_t)8 * a.P_pad] = xs; frag[(size_t)9 * a.P_pad] = hs; }
}

__global__ void k_stitch_ad(const double* __restrict__ frag, int n_chunks, int P_pad, int P, double scale,
                            double* __restrict__ out, double* __restrict__ comp3, double x_scale, double h_scale,
                            int* __restrict__ out_edges, int n_seg, int n_bins, const int* __restrict__ pmap = nullptr,
                            const int* __restrict__ jlo = nullptr, const int* __restrict__ jhi = nullptr, int chunk_len = 1) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= (pmap ? P_pad : P)) return;
  const int q = pmap ? pmap[p] : p;             // window sort: slot p holds particle q of the batch
  if (q >= P) return;
  // chunks wholly outside the particle's window hold the fragments of "nothing happened": only [c_lo, c_hi] is folded
  int c_lo = 0, c_hi = n_chunks - 1;
  if (jlo) {
    const int lo = jlo[p], hi = jhi[p];
    if (hi <= lo) { c_lo = 0; c_hi = -1; }
    else { c_lo = max(lo / chunk_len, 0); c_hi = min((hi - 1) / chunk_len, n_chunks - 1); }
  }
  double ups = 0.0, zr = 0.0, zi = 0.0, sg = 0.0, xs = 0.0, hs = 0.0;
  auto finish = [&]() {
    if (sg > 0.0) {
      const double z2 = zr * zr + zi * zi;
      ups += z2 / sg;
      if (comp3) { xs += sqrt(z2); hs += sg; }
    }
  };
  // serial fold in chunk order (bitwise reproducible), loads of kU chunks in flight (as in k_stitch)
  constexpr int kU = 8;
  for (int c0 = c_lo; c0 <= c_hi; c0 += kU) {
    double v[kU][8], w8[kU], w9[kU];
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      const double* f = frag + (size_t)min(c0 + u, c_hi) * kFragAd * P_pad + p;
#pragma unroll
      for (int m = 0; m < 8; ++m) v[u][m] = f[(size_t)m * P_pad];
      w8[u] = comp3 ? f[(size_t)8 * P_pad] : 0.0; w9[u] = comp3 ? f[(size_t)9 * P_pad] : 0.0;
    }
#pragma unroll
    for (int u = 0; u < kU; ++u) {
      if (c0 + u > c_hi) break;
      zr += v[u][1]; zi += v[u][2]; sg += v[u][3];
      if (v[u][7] != 0.0) {
        finish();
        zr = v[u][4]; zi = v[u][5]; sg = v[u][6];
      }
      ups += v[u][0];
      if (comp3) { xs += w8[u]; hs += w9[u]; }
    }
  }
  finish();                                     // the last segment closes at e_N = n_bins
  if (out) out[q] = ups * scale;
  if (comp3) { comp3[3 * (size_t)q] = ups * scale; comp3[3 * (size_t)q + 1] = xs * x_scale; comp3[3 * (size_t)q + 2] = hs * h_scale; }
  if (out_edges) { out_edges[(size_t)q * (n_seg + 1)] = 0; out_edges[(size_t)q * (n_seg + 1) + n_seg] = n_bins; }
}

}  // namespace
