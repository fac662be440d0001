// sc_kernels_adaptive.cuh -- per-particle equal-SNR^2 segments (App. A).
// Part of libscstat.so (one translation unit: sc_stat.cu includes the kernel files in pipeline order).
#pragma once
#include "sc_common.cuh"

namespace {

// ------------------------------------------------------------------------------------------------ per-particle segments
// Equal squared-SNR segments re-evaluated for every particle (App. A):
//   s_j = sum_a |h_a(f_j)|^2 / S_a(f_j),  C = sum_j s_j,  e_0 = 0, e_N = n_bins,
//   e_n = min{ j : sum_{j' < j} s_j' >= C n / N }   (n = 1 .. N-1),
// then Upsilon_N on those edges.  Floating point decides these integers, so the decision is taken in FP64 like the
// definition's (FP64 node amplitudes, FP64 moments of the weights, FP64 per-bin walk where a target falls): the edges equal
// the FP64 oracle's except where a cumulative sum comes within the interpolation error (~1e-12 relative) of a target.
// Four steps, all with lane = particle:
//   k_sigma_chunks64 sigma of every (chunk, particle) in FP64 from the moments of the weights over the fine sub-intervals
//   k_scan_chunks    prefix sum over chunks -> cumulative sigma at every chunk start, and C
//   k_edges64        per (chunk, particle): the edges whose targets C n / N fall into the chunk -- sub-interval by
//                    sub-interval from the moments, group by group (32 bins) inside the sub-interval that holds a target,
//                    bin by bin inside that group.  The number of edges of a chunk is fixed by the scanned sums
//                    (k0 = K(cbase[chunk]), k1 = K(cbase[chunk + 1])), so neighbouring chunks always agree.
//   k_dense2_ad      the hot loop of k_dense2 on those integer edges (FP32 amplitudes): groups of <= 32 bins in which no
//                    lane of the warp has an edge take the unmasked packed path; the others are walked bin by bin.
constexpr int kFragAd = 10;    // partial Upsilon, head (zr, zi, sg), tail (zr, zi, sg), head-closes flag, partial sum|z|, sum sigma

struct AdaptArgs {
  int n_seg, n_chunks;
  const double* cbase;         // [n_chunks + 1][P_pad]: cumulative sigma at the chunk starts; row n_chunks = C
  const ulonglong2* gmom;      // [n_groups][4] moments of the weights over groups of 2^lg_group bins
  const ulonglong2* smom;      // [n_sub][4]    ... over the fine sub-intervals
  int lg_group;
  int* out_edges;              // [P][n_seg + 1] of this batch (the caller's array or scratch): written by k_edges64
  double* chunk_sigma;         // = cbase (written by k_sigma_chunks64 before the scan)
  const int* pmap;             // window sort: table slot -> particle of the batch (rows of out_edges), or nullptr
  const double2* smom64;       // [n_sub][7]    FP64 moments of the weights over the fine sub-intervals
  const double2* gmom64;       // [n_groups][7] ... over the groups
  const double2* G64;          // [n_bins] sigma weights per bin (FP64)
  double* sub_sigma;           // [n_chunks * CH / Sf][P_pad]: sigma of every fine sub-interval (k_sigma_chunks64 -> k_edges64)
  // three-channel handles (NA = 6): the same tables for the T weights, as (T, 0) pairs
  const ulonglong2* gmomT; const ulonglong2* smomT; const double2* smom64T; const double2* GT64;
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

// The six FP64 nodes (m = -2 .. 3) of the four amplitude components around coarse interval ic, kept in registers while a
// lane walks the chunk: the four fine sub-intervals of a coarse interval share them, and the next coarse interval needs
// one new node per component (read per sub-interval they cost 25 GB of L2 traffic per pass on c3).
template <int NA> struct Nodes64 { double v[NA][6]; };      // NA = 4: (A, E); 6: (A, E, T)
template <int NA>
__device__ __forceinline__ void nodes64_load(const DevCfg& c, const DenseArgs& a, int p, int ic, Nodes64<NA>& n) {
  const double* __restrict__ namp = reinterpret_cast<const double*>(a.node_amp);
#pragma unroll
  for (int r = 0; r < NA; ++r) {
    const double* col = namp + ((size_t)(ic + kNodeOff) * NA + r) * a.P_pad + p;
    const ptrdiff_t st = (ptrdiff_t)NA * a.P_pad;
#pragma unroll
    for (int m = -2; m <= 3; ++m) n.v[r][m + 2] = col[m * st];
  }
}
template <int NA>
__device__ __forceinline__ void nodes64_advance(const DevCfg& c, const DenseArgs& a, int p, int ic_new, Nodes64<NA>& n) {
  const double* __restrict__ namp = reinterpret_cast<const double*>(a.node_amp);
#pragma unroll
  for (int r = 0; r < NA; ++r) {
#pragma unroll
    for (int m = 0; m < 5; ++m) n.v[r][m] = n.v[r][m + 1];
    n.v[r][5] = namp[((size_t)(ic_new + kNodeOff + 3) * NA + r) * a.P_pad + p];
  }
}
// FP64 cubic coefficients of (Ar, Ai, Er, Ei[, Tr, Ti]) on fine sub-interval q of the coarse interval whose nodes are n.
template <int NA>
__device__ __forceinline__ void sub_amps64(const Nodes64<NA>& n, int q, double (&cf)[NA][4]) {
#pragma unroll
  for (int r = 0; r < NA; ++r)
#pragma unroll
    for (int kk = 0; kk < 4; ++kk) {
      double acc = 0.0;
#pragma unroll
      for (int m = 0; m < 6; ++m) acc = fma(kFineMd[q][kk][m], n.v[r][m], acc);
      cf[r][kk] = acc;
    }
}
// s_j = sum_a G_a(j) |c_a(s_j)|^2 in FP64 (the integrand of <h|h>, up to the common scale).
template <int NA>
__device__ __forceinline__ double sigma_bin64(const double (&cf)[NA][4], double sj, double2 g, double gT) {
  const double Ar = fma(fma(fma(cf[0][3], sj, cf[0][2]), sj, cf[0][1]), sj, cf[0][0]);
  const double Ai = fma(fma(fma(cf[1][3], sj, cf[1][2]), sj, cf[1][1]), sj, cf[1][0]);
  const double Er = fma(fma(fma(cf[2][3], sj, cf[2][2]), sj, cf[2][1]), sj, cf[2][0]);
  const double Ei = fma(fma(fma(cf[3][3], sj, cf[3][2]), sj, cf[3][1]), sj, cf[3][0]);
  double s = fma(g.x, fma(Ar, Ar, Ai * Ai), g.y * fma(Er, Er, Ei * Ei));
  if (NA == 6) {
    const double Tr = fma(fma(fma(cf[NA - 2][3], sj, cf[NA - 2][2]), sj, cf[NA - 2][1]), sj, cf[NA - 2][0]);
    const double Ti = fma(fma(fma(cf[NA - 1][3], sj, cf[NA - 1][2]), sj, cf[NA - 1][1]), sj, cf[NA - 1][0]);
    s = fma(gT, fma(Tr, Tr, Ti * Ti), s);
  }
  return s;
}
// sigma over a run of bins from the FP64 moments of its weights, all channels
template <int NA>
__device__ __forceinline__ double sigma_mom64(const double (&cf)[NA][4], const double2* __restrict__ M, const double2* __restrict__ MT) {
  double s = sigma_moments64(*reinterpret_cast<const double(*)[4][4]>(&cf[0]), M);
  if (NA == 6) {
    const double cT[4][4] = {{cf[NA - 2][0], cf[NA - 2][1], cf[NA - 2][2], cf[NA - 2][3]},
                             {cf[NA - 1][0], cf[NA - 1][1], cf[NA - 1][2], cf[NA - 1][3]}, {0, 0, 0, 0}, {0, 0, 0, 0}};
    s += sigma_moments64(cT, MT);
  }
  return s;
}
// sigma of the fine sub-interval [ib, ie) for this lane: from the moments when the lane's window covers it, bin by bin
// (masked) when a window border falls inside.  The same function serves k_sigma_chunks64 and k_edges64, so the second
// pass reproduces the chunk sums of the first bit for bit.
template <int NA>
__device__ __forceinline__ double sigma_sub64(const DevCfg& c, const AdaptArgs& ad, const double (&cf)[NA][4], int ib, int ie,
                                              int jlo, int jhi, int n_bins) {
  const int Sf = c.stride >> 2;
  const size_t isub = (size_t)(ib >> (c.log2_stride - 2));
  if (ib >= jlo && ie <= jhi && ie - ib == Sf) return sigma_mom64<NA>(cf, ad.smom64 + isub * 7, NA == 6 ? ad.smom64T + isub * 7 : nullptr);
  const double hS = 1.0 / (double)Sf;
  double tot = 0.0;
  for (int j = max(ib, jlo); j < min(min(ie, jhi), n_bins); ++j)
    tot += sigma_bin64<NA>(cf, (double)(j - ib) * hS, ad.G64[j], NA == 6 ? ad.GT64[j].x : 0.0);
  return tot;
}

template <int NA = 4>
__global__ void __launch_bounds__(kBlock, NA == 6 ? 3 : 4) k_sigma_chunks64(DevCfg c, DenseArgs a, AdaptArgs ad) {
  constexpr int CH = kChunkF32;
  const int chunk = blockIdx.x;
  const int cs = chunk * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int p = blockIdx.y * kBlock + threadIdx.x;
  const int jlo = a.jlo[p], jhi = a.jhi[p];
  if (!__syncthreads_or((jhi > cs) && (jlo < ce))) {          // no particle of this block lives in this chunk
    ad.chunk_sigma[(size_t)(chunk + 1) * a.P_pad + p] = 0.0;
    return;
  }
  const int Sf = c.stride >> 2;
  double tot = 0.0;
  Nodes64<NA> nd;
  int ic_have = -1;
  for (int ib = cs; ib < ce; ib += Sf) {
    const int ie = min(ib + Sf, ce);
    const bool lane_out = (ie <= jlo) || (ib >= jhi);
    const int ic = ib >> c.log2_stride;
    if (ic != ic_have) { if (ic_have < 0) nodes64_load(c, a, p, ic, nd); else nodes64_advance(c, a, p, ic, nd); ic_have = ic; }
    double sg = 0.0;
    if (!lane_out) {                                           // (a lane outside its window holds zeros or unused nodes)
      double cf[NA][4];
      sub_amps64<NA>(nd, (ib >> (c.log2_stride - 2)) & 3, cf);
      sg = sigma_sub64<NA>(c, ad, cf, ib, ie, jlo, jhi, c.n_bins);
    }
    ad.sub_sigma[(size_t)(ib >> (c.log2_stride - 2)) * a.P_pad + p] = sg;
    tot += sg;
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

// The edges of every particle whose targets fall into this chunk (see the file header).  Edge n lies at the first bin j
// whose cumulative sum C_j = sum_{j' < j} s_j' has reached C n / N; inside chunk `chunk` that is a j in (cs, ce].
// Each lane walks its sub-interval sums (as k_sigma_chunks64 left them) until one holds a target; that sub-interval is then
// resolved by the WHOLE WARP for that lane: the lane's cubic coefficients are broadcast, the 32 lanes evaluate 32 bins at
// a time in FP64 and a warp scan gives the cumulative sums (a lane walking its own bins alone would run at 1/32 efficiency).
__device__ __forceinline__ double shfl_d(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }
template <int NA = 4>
__global__ void __launch_bounds__(kBlock, NA == 6 ? 4 : 6) k_edges64(DevCfg c, DenseArgs a, AdaptArgs ad) {
  constexpr int CH = kChunkF32;
  const int chunk = blockIdx.x;
  const int cs = chunk * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int p = blockIdx.y * kBlock + threadIdx.x;
  const int lane = threadIdx.x & 31;
  const int jlo = a.jlo[p], jhi = a.jhi[p];
  const int N = ad.n_seg;
  const double C = ad.cbase[(size_t)ad.n_chunks * a.P_pad + p];
  const double cb0 = ad.cbase[(size_t)chunk * a.P_pad + p];
  const double cb1 = ad.cbase[(size_t)(chunk + 1) * a.P_pad + p];
  int k = seg_index(cb0, C, N);
  const int k1 = seg_index(cb1, C, N);
  if (!__any_sync(0xffffffffu, k < k1)) return;               // no lane of this warp has an edge in this chunk
  const int pq = ad.pmap ? ad.pmap[p] : p;
  int* erow = (pq < a.P) ? ad.out_edges + (size_t)pq * (N + 1) : nullptr;
  const int Sf = c.stride >> 2;
  const double hS = 1.0 / (double)Sf;
  double t_next = (k < k1) ? seg_target(C, k + 1, N) - cb0 : INFINITY;
  double crel = 0.0;
  Nodes64<NA> nd;
  int ic_have = -1;
  for (int ib = cs; ib < ce; ib += Sf) {
    const int ie = min(ib + Sf, ce);
    if (!__any_sync(0xffffffffu, k < k1)) break;               // every lane has placed its edges of this chunk
    const int ic = ib >> c.log2_stride;
    if (ic != ic_have) { if (ic_have < 0) nodes64_load(c, a, p, ic, nd); else nodes64_advance(c, a, p, ic, nd); ic_have = ic; }
    // sigma of the sub-interval as k_sigma_chunks64 summed it (bit for bit: the scanned chunk sums are sums of these)
    const double sg_s = (k < k1) ? ad.sub_sigma[(size_t)(ib >> (c.log2_stride - 2)) * a.P_pad + p] : 0.0;
    const bool cross = (k < k1) && (crel + sg_s >= t_next);    // a target of this lane falls into this sub-interval
    unsigned todo = __ballot_sync(0xffffffffu, cross);
    if (!cross) crel += sg_s;
    if (!todo) continue;
    double cf[NA][4];
    sub_amps64<NA>(nd, (ib >> (c.log2_stride - 2)) & 3, cf);
    while (todo) {
      const int L = __ffs(todo) - 1;
      todo &= todo - 1;
      // lane L's problem, held by every lane
      double g[NA][4];
#pragma unroll
      for (int r = 0; r < NA; ++r)
#pragma unroll
        for (int m = 0; m < 4; ++m) g[r][m] = shfl_d(cf[r][m], L);
      const double C_L = shfl_d(C, L), cb0_L = shfl_d(cb0, L);
      double crel_L = shfl_d(crel, L), t_L = shfl_d(t_next, L);
      int k_L = __shfl_sync(0xffffffffu, k, L);
      const int k1_L = __shfl_sync(0xffffffffu, k1, L), jlo_L = __shfl_sync(0xffffffffu, jlo, L), jhi_L = __shfl_sync(0xffffffffu, jhi, L);
      int* erow_L = (int*)__shfl_sync(0xffffffffu, (unsigned long long)erow, L);
      auto close_L = [&](int j) {
        ++k_L;
        if (lane == 0 && erow_L) erow_L[k_L] = j;
        t_L = (k_L < k1_L) ? seg_target(C_L, k_L + 1, N) - cb0_L : INFINITY;
      };
      // (the sigma weights of kPre rounds are fetched together: the rounds are serial, their loads need not be)
      constexpr int kPre = 4;
      for (int jb = ib; jb < ie && k_L < k1_L; jb += 32 * kPre) {
      double2 gw[kPre];
      double gt[kPre];
#pragma unroll
      for (int u = 0; u < kPre; ++u) {
        const int j = jb + 32 * u + lane;
        const bool in = (j < ie) && (j >= jlo_L) && (j < jhi_L);
        gw[u] = in ? ad.G64[j] : make_double2(0.0, 0.0);
        gt[u] = (NA == 6 && in) ? ad.GT64[j].x : 0.0;
      }
#pragma unroll
      for (int u = 0; u < kPre; ++u) {
        const int j0 = jb + 32 * u;
        if (j0 >= ie || k_L >= k1_L) break;
        const int j = j0 + lane;
        double sj = 0.0;
        if (j < ie && j >= jlo_L && j < jhi_L) sj = sigma_bin64<NA>(g, (double)(j - ib) * hS, gw[u], gt[u]);
        double inc = sj;                                       // inclusive warp scan, fixed order
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const double up = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += up; }
        const double excl = inc - sj;                          // sum of the bins of this round before bin j
        const double tot = shfl_d(inc, 31);
        // e_n = first bin whose cumulative sum (before adding it) has reached the target; several targets may fall here
        while (k_L < k1_L) {
          const unsigned hit = __ballot_sync(0xffffffffu, (j < ie) && (crel_L + excl >= t_L));
          if (!hit) break;
          close_L(j0 + __ffs(hit) - 1);
        }
        crel_L += tot;
      }
      }
      while (k_L < k1_L && crel_L >= t_L) close_L(ie);
      if (lane == L) { crel = crel_L; t_next = t_L; k = k_L; }
    }
  }
  while (k < k1) { ++k; if (erow) erow[k] = ce; }   // targets the scanned sums place in this chunk (rounding): at its end
}

// NA = 6 (three-channel handles): the pair loop, the masked pairs and the moments of k_dense3; Dg = the fused records
// (wA, wE, wT), Gp = the sigma weights per bin pair (masked pairs only); no merged coarse intervals.
// QUAD (fine sub-intervals >= 256 bins): the unmasked runs evaluate the amplitudes as quadratics over runs of
// a quarter sub-interval (pairs_fast_q of sc_kernels_dense32.cuh); the run state lives across the 32-bin groups.
template <int SC, bool MERGE = false, int NA = 4, bool QUAD = false>
__global__ void __launch_bounds__(kBlock, NA == 6 ? SC_DENSE3_MINB : SC_DENSE2_MINB)
k_dense2_ad(DevCfg c, DenseArgs a, AdaptArgs ad, const ulonglong2* __restrict__ Dg, const ulonglong2* __restrict__ Gp = nullptr) {
  static_assert(!(MERGE && NA == 6), "merged coarse intervals are a two-channel variant");

  constexpr int CH = kChunkF32;
  constexpr int kRec = (NA == 6) ? kPairRec3 : kPairRec;
  __shared__ ulonglong2 sD[CH / 2 * kRec];
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
    const ulonglong2* src = Dg + (size_t)(cs >> 1) * kRec;
#pragma unroll 4
    for (int t = threadIdx.x; t < CH / 2 * kRec; t += kBlock) sD[t] = src[t];
  }
  __syncthreads();

  const int Sf = c.stride >> 2;
  const float hS = 1.0f / (float)Sf;
  const u64 h2 = f2bcast(2.0f * hS);
  const u64 K2 = f2bcast(1.4629180792671596e-09f);
  const int N = ad.n_seg;
  // the channel-count-specific pieces of the walk
  auto sig_mom = [&](const float (&cfx)[NA][4], const ulonglong2* m, const ulonglong2* mT, size_t idx) -> double {
    if constexpr (NA == 6) return sigma_moments3(cfx, m + idx * 4, mT + idx * 4);
    else return sigma_moments(cfx, m + idx * 4);
  };
  typename std::conditional<NA == 6, QuadState3, QuadState>::type qs;
  int q_off = -1;                               // bins from the sub-interval start where qs stands (-1: nowhere)
  const int lg_run = c.log2_stride - 4;
  // off = first bin of the run of pairs, counted from the sub-interval start
  auto run_pairs = [&](PhaseFD& phx, const float (&cfx)[NA][4], u64& s2x, const ulonglong2*& recx, int n, u64& zr2, u64& zi2, int off) {
    if constexpr (QUAD && NA == 6) {
      if (q_off != off) quad_start3(cfx, off, lg_run, qs);
      pairs_fast3_q<SC>(phx, cfx, qs, lg_run, recx, n, K2, zr2, zi2);
      q_off = off + 2 * n;
    } else if constexpr (QUAD) {
      if (q_off != off) quad_start(cfx, off, lg_run, qs);
      pairs_fast_q<SC>(phx, cfx, qs, lg_run, recx, n, K2, zr2, zi2);
      q_off = off + 2 * n;
    }
    else if constexpr (NA == 6) pairs_fast3<SC>(phx, cfx, s2x, recx, n, h2, K2, zr2, zi2);
    else pairs_fast<SC>(phx, cfx, s2x, recx, n, h2, K2, zr2, zi2);
  };
  const int Gs = 1 << ad.lg_group;

  const double C = ad.cbase[(size_t)ad.n_chunks * a.P_pad + p];
  const double cb0 = ad.cbase[(size_t)chunk * a.P_pad + p];
  const double cb1 = ad.cbase[(size_t)(chunk + 1) * a.P_pad + p];
  int k = seg_index(cb0, C, N);                 // segment open at the chunk start
  const int k1 = seg_index(cb1, C, N);          // edges k+1 .. k1 lie in (cs, ce] (k_edges64 placed them), no more, no fewer
  const int pq = ad.pmap ? ad.pmap[p] : p;      // particle of the batch in this table slot
  const int* erow = ad.out_edges + (size_t)min(pq, a.P - 1) * (N + 1);
  int j_next = (k < k1 && pq < a.P) ? erow[k + 1] : INT_MAX;   // bin of the next edge of this lane
  double crel = 0.0, c_open = 0.0;              // sigma (FP32 amplitudes) since the chunk start; its value where the open piece began
  double Zr = 0.0, Zi = 0.0, ups = 0.0, xs = 0.0, hs = 0.0;
  bool closed_any = false;
  double* frag = a.frag + (size_t)chunk * kFragAd * a.P_pad + p;

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
    j_next = (k < k1) ? erow[k + 1] : INT_MAX;
    (void)j;
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
    float cf[NA][4];
    // merged coarse intervals as in k_dense2 (the group and sub-interval moments stay those of the fine sub-intervals)
    if constexpr (MERGE) {
      if (merged_left == 0 && (ib & (c.stride - 1)) == 0 && ib + c.stride <= ce2 &&
          __all_sync(0xffffffffu, (ib >= jlo) && (ib + c.stride <= jhi)) &&
          __all_sync(0xffffffffu, coarse_dslope(c, a, p, ib >> c.log2_stride) <= a.merge_lim)) {
        coarse_phase(c, a, p, ib, ph);
        coarse_amps<double>(c, a, p, ib, cc);
        merged_left = 4;
      }
    }
    if (MERGE && merged_left > 0) {
      if constexpr (MERGE) coarse_to_fine(cc, 4 - merged_left, cf);
      --merged_left;
    } else {
      sub_phase(c, a, p, ib, ph);
      if constexpr (NA == 6) sub_amps3<double>(c, a, p, ib, cf);
      else sub_amps<double>(c, a, p, ib, cf);
    }
    u64 s2 = f2pack(0.0f, hS);
    q_off = -1;                                 // new coefficients
    const ulonglong2* rec = sD + ((ib - cs) >> 1) * kRec;
    // First ask the question for the whole sub-interval (its moments are those k_sigma_chunks used): if no lane reaches its
    // next target in it, all its groups take the unmasked path and the group moments are not needed at all.
    if (all_in && ie - ib == Sf) {
      const bool cross_s = j_next < ie;          // (an edge AT ie is closed by the first bin of the next sub-interval)
      if (!__any_sync(0xffffffffu, cross_s)) {
        const double sg_s = sig_mom(cf, ad.smom, ad.smomT, (size_t)(ib >> (c.log2_stride - 2)));
        for (int gs = ib; gs < ie; gs += Gs) {
          u64 zr2 = 0, zi2 = 0;
          run_pairs(ph, cf, s2, rec, Gs >> 1, zr2, zi2, gs - ib);
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
      const bool slow = !all_in || __any_sync(0xffffffffu, j_next < ge);   // a lane has an edge inside this group
      if (!slow) {
        const double sg_m = sig_mom(cf, ad.gmom, ad.gmomT, (size_t)(gs >> ad.lg_group));
        u64 zr2 = 0, zi2 = 0;
        run_pairs(ph, cf, s2, rec, (ge - gs) >> 1, zr2, zi2, gs - ib);
        float zrl, zrh, zil, zih;
        f2unpack(zr2, zrl, zrh); f2unpack(zi2, zil, zih);
        Zr += (double)(zrl + zrh); Zi += (double)(zil + zih);
        crel += sg_m;
      } else {
        if constexpr (QUAD) s2 = f2pack((float)(gs - ib) * hS, (float)(gs + 1 - ib) * hS);   // (the quadratic runs do not advance it)
        for (int jj = gs; jj < ge; jj += 2) {
          u64 zr2 = 0, zi2 = 0, sg2 = 0;
          if constexpr (NA == 6) pair_eval3<SC>(ph, cf, s2, rec, Gp + (size_t)(jj >> 1) * 2, jj, jlo, jhi, h2, K2, zr2, zi2, sg2);
          else pair_eval<true, true, SC>(ph, cf, s2, rec, jj, jlo, jhi, h2, K2, zr2, zi2, sg2);
          float zrl, zrh, zil, zih, sgl, sgh;
          f2unpack(zr2, zrl, zrh); f2unpack(zi2, zil, zih); f2unpack(sg2, sgl, sgh);
          while (j_next <= jj) close_at(jj);                      // edges at this bin (several: empty segments)
          Zr += (double)zrl; Zi += (double)zil; crel += (double)sgl;
          while (j_next <= jj + 1) close_at(jj + 1);
          Zr += (double)zrh; Zi += (double)zih; crel += (double)sgh;
        }
      }
    }
  }
  while (k < k1) close_at(ce);                  // edges at the chunk end
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
