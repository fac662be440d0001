// sc_kernels_dense32tc.cuh -- a4 + a5, FP32-amplitude hot loop with the amplitude correction on the 5th-generation tensor
// cores (tcgen05.mma kind::tf32, accumulators in TMEM).  Part of libscstat.so (one translation unit).
//
// What goes where.  On a fine sub-interval the node amplitudes are cubics; about its centre (x = s - 1/2, |x| <= 1/2)
//     c_a(x) = g0_a + g1_a x + g2_a x^2 + g3_a x^3,           a = A, E (complex),
// so the per-bin factor q_j = sum_a W_a(j) conj(c_a(x_j)) of z = sum_j q_j e^{2 pi i Phi_j} splits into
//     q_j = sum_a W_a(j) conj(g0_a)                            -- 8 FP32 FMAs per bin on the CUDA cores, as before, and
//     u_j = sum_a sum_{m=1..3} conj(g_m,a) [W_a(j) x_j^m]      -- a correction of relative size <= a few 1e-2.
// u is a dense contraction: [128 particles x K] times [K x bins], with the bracket shared by ALL particles (the bin grid
// and the sub-interval grid are shared).  K = 12 real coefficients per output component; written as a 3xTF32 split
// (hi*hi + lo*hi + hi*lo for m = 1, 2; hi*hi for m = 3: 28 of K = 32 columns used) the error of u is < 2^-22 |u| <= 1e-8 |q|,
// far below the FP32 rounding of the leading term.  The 12 amplitude FMAs per bin of the Horner form leave the FP32 pipe
// (26 -> 13 packed-pipe lane slots per bin); everything that is NOT a contraction -- FP64 phase, sin/cos, the rotation
// z += q e^{2 pi i Phi}, the segment bookkeeping -- stays where it was (k_dense2).
//
// Mechanics per CTA (128 particles x one chunk of 2048 bins, 4 CTAs per SM, 128 TMEM columns each):
//   * the data side of the contraction is precomputed once per data stream and node spacing by k_tc_image: per 32-bin tile a
//     4 KB K-major operand image (canonical no-swizzle core-matrix order) followed by the tile's 16 bin-pair records;
//     one cp.async.bulk (UBLKCP) per tile into a 4-stage ring, completion on an mbarrier;
//   * per fine sub-interval every thread writes its particle's two coefficient rows (real and imaginary output) as
//     TF32 hi/lo into the A operand tiles in shared memory;
//   * one elected lane issues 8 tcgen05.mma (M = 128, N = 32, K = 8) per tile into one of two TMEM buffers and commits to an
//     mbarrier; the lane that issues is the LAST of the four warps to have released the buffer (an acq_rel counter in
//     shared memory), so no warp ever waits for another except through the data it needs;
//   * each thread reads its own row (TMEM lane = particle) with tcgen05.ld as the bin pairs come up.
// Sub-intervals that are not "all 128 lanes inside their time windows" take the k_dense2 code path with the records read
// from global memory (band edges; a few per cent of the work on the short-window configurations).
#pragma once
#include "sc_common.cuh"

namespace {

namespace tc {
constexpr int kTileBins = 32;
constexpr int kImgBytes = 4096;                          // operand image of one tile: 32 bins x K = 32 TF32
constexpr int kRecBytes = kTileBins / 2 * kPairRec * 16;  // its 16 bin-pair records (768 B)
constexpr int kTileBytes = kImgBytes + kRecBytes;         // 4864 B per tile in global memory and per ring stage
constexpr int kStages = 4;
constexpr int kOffA = 0;                                  // A_r (16 KB), A_i (16 KB)
constexpr int kOffT = 32768;                              // ring
constexpr int kOffBar = kOffT + kStages * kTileBytes;     // b_full[4], d_full[2]
constexpr int kOffU = kOffBar + 48;                       // tmem base, cntA, cntD[2], fast mask[2], merge mask, n_list
constexpr int kOffList = kOffU + 32;                      // tile list (uint8 x 64)
constexpr int kSmemBytes = kOffList + 64;
// instruction descriptor: D = F32, A = B = TF32, both K-major, N = 32, M = 128
constexpr uint32_t kIdesc = (1u << 4) | (2u << 7) | (2u << 10) | ((32u >> 3) << 17) | ((128u >> 4) << 24);

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, uint32_t cnt) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(b)), "r"(cnt));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, uint32_t parity) {
  asm volatile("{\n.reg .pred P1;\nLAB_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n@P1 bra DONE;\nbra LAB_WAIT;\nDONE:\n}"
               :: "r"(smem_u32(b)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               :: "r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// K-major, no swizzle: a core matrix is 8 rows x 16 B, contiguous; LBO = distance between the two core matrices of one
// K = 8 step, SBO = distance between 8-row groups.  Here LBO = 128 B, SBO = 1024 B for both operands.
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46);
}
__device__ __forceinline__ void mma_tf32(uint32_t d_tmem, uint64_t da, uint64_t db, uint32_t acc) {
  asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
               :: "r"(d_tmem), "l"(da), "l"(db), "r"(kIdesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void mma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ uint32_t atom_add_acqrel(uint32_t* p, uint32_t v) {
  uint32_t o;
  asm volatile("atom.acq_rel.cta.shared::cta.add.u32 %0, [%1], %2;" : "=r"(o) : "r"(smem_u32(p)), "r"(v) : "memory");
  return o;
}
__device__ __forceinline__ float tf32_rna(float v) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(v));
  return __uint_as_float(r);
}
__device__ __forceinline__ void tld2(uint32_t taddr, uint32_t& a, uint32_t& b) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(a), "=r"(b) : "r"(taddr));
}
// the wait names the registers it protects, so that no use of them can be scheduled above it
__device__ __forceinline__ void tld_wait(uint32_t& a, uint32_t& b, uint32_t& c, uint32_t& d) {
  asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(a), "+r"(b), "+r"(c), "+r"(d) :: "memory");
}
}  // namespace tc

// The data side of the contraction (see the header), one CTA of 32 threads per 32-bin tile; thread n = bin.  Row n of the
// K-major image, K index = 4 * chunk + component (component order wAr, wAi, wEr, wEi):
//   chunk 0: hi(P1)  1: hi(P1)  2: lo(P1)  3: hi(P2)  4: hi(P2)  5: lo(P2)  6: hi(P3)  7: 0,   Pm = W x^m,
// against the coefficient rows  hi(g1) lo(g1) hi(g1) hi(g2) lo(g2) hi(g2) hi(g3) 0  written by k_dense2_tc.
__global__ void __launch_bounds__(32) k_tc_image(const float4* __restrict__ D32, int lg_fine, long long n_tiles,
                                                 uint4* __restrict__ img) {
  const long long tile = blockIdx.x;
  if (tile >= n_tiles) return;
  const int n = threadIdx.x;
  const long long j = tile * tc::kTileBins + n;
  const float4 ra = D32[(size_t)(j >> 1) * kPairRec], re = D32[(size_t)(j >> 1) * kPairRec + 1];
  const bool odd = (j & 1);
  const float w[4] = {odd ? ra.y : ra.x, odd ? ra.w : ra.z, odd ? re.y : re.x, odd ? re.w : re.z};
  const int Sf = 1 << lg_fine;
  const double x = (double)(j & (Sf - 1)) / (double)Sf - 0.5;
  uint4* row = img + (size_t)tile * (tc::kTileBytes / 16) + (n >> 3) * 64 + (n & 7);   // + chunk * 8
  float hi[3][4], lo[3][4];
  double xm = 1.0;
#pragma unroll
  for (int m = 0; m < 3; ++m) {
    xm *= x;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const float P = (float)((double)w[r] * xm);
      hi[m][r] = tc::tf32_rna(P);
      lo[m][r] = tc::tf32_rna(P - hi[m][r]);
    }
  }
  auto pack = [](const float (&v)[4]) { return make_uint4(__float_as_uint(v[0]), __float_as_uint(v[1]), __float_as_uint(v[2]), __float_as_uint(v[3])); };
  row[0 * 8] = pack(hi[0]); row[1 * 8] = pack(hi[0]); row[2 * 8] = pack(lo[0]);
  row[3 * 8] = pack(hi[1]); row[4 * 8] = pack(hi[1]); row[5 * 8] = pack(lo[1]);
  row[6 * 8] = pack(hi[2]); row[7 * 8] = make_uint4(0u, 0u, 0u, 0u);
  // the tile's 16 bin-pair records (48 x 16 B) behind the image
  const uint4* src = reinterpret_cast<const uint4*>(D32) + (size_t)tile * (tc::kRecBytes / 16);
  uint4* dst = img + (size_t)tile * (tc::kTileBytes / 16) + tc::kImgBytes / 16;
  for (int t = n; t < tc::kRecBytes / 16; t += 32) dst[t] = src[t];
}

// q = W conj(g0) + u for one bin pair, z += q e^{2 pi i Phi}.  G[0..3] = (g0Ar, g0Ai, g0Er, g0Ei), G[4] = -g0Ai, G[5] = -g0Ei
// as broadcast pairs; ur2, ui2 the tensor-core correction (even bin, odd bin).
__device__ __forceinline__ void mac_pair_tc(const u64 (&G)[6], const ulonglong2 wA, const ulonglong2 wE, u64 ur2, u64 ui2,
                                            u64 cr2, u64 sr2, u64& zr2, u64& zi2) {
  const u64 qr = f2fma(wA.x, G[0], f2fma(wA.y, G[1], f2fma(wE.x, G[2], f2fma(wE.y, G[3], ur2))));
  const u64 qi = f2fma(wA.y, G[0], f2fma(wA.x, G[4], f2fma(wE.y, G[2], f2fma(wE.x, G[5], ui2))));
  zr2 = f2fma(qr, cr2, f2fma(f2neg(qi), sr2, zr2));
  zi2 = f2fma(qr, sr2, f2fma(qi, cr2, zi2));
}

// n >= 1 consecutive pairs inside one tile, software-pipelined like pairs_fast: the sin/cos, the record loads and the
// TMEM loads of pair i+1 are issued before the multiply-accumulate of pair i.
template <int SC>
__device__ __forceinline__ void pairs_fast_tc(PhaseFD& ph, const u64 (&G)[6], const ulonglong2* rec, uint32_t taddr, int n,
                                              u64 K2, u64& zr2, u64& zi2) {
  u64 cr, sr;
  sincos_pair<SC>(ph, K2, cr, sr);
  ulonglong2 wA = rec[0], wE = rec[1];
  uint32_t u0, u1, v0, v1;
  tc::tld2(taddr, u0, u1); tc::tld2(taddr + 32, v0, v1);
#pragma unroll 1
  for (int i = 1; i < n; ++i) {
    u64 crn, srn;
    sincos_pair<SC>(ph, K2, crn, srn);
    rec += kPairRec;
    const ulonglong2 wAn = rec[0], wEn = rec[1];
    tc::tld_wait(u0, u1, v0, v1);
    const u64 ur2 = f2pack(__uint_as_float(u0), __uint_as_float(u1)), ui2 = f2pack(__uint_as_float(v0), __uint_as_float(v1));
    taddr += 2;
    tc::tld2(taddr, u0, u1); tc::tld2(taddr + 32, v0, v1);
    mac_pair_tc(G, wA, wE, ur2, ui2, cr, sr, zr2, zi2);
    cr = crn; sr = srn; wA = wAn; wE = wEn;
  }
  tc::tld_wait(u0, u1, v0, v1);
  mac_pair_tc(G, wA, wE, f2pack(__uint_as_float(u0), __uint_as_float(u1)), f2pack(__uint_as_float(v0), __uint_as_float(v1)),
              cr, sr, zr2, zi2);
}

template <bool SEG, int SC, bool MERGE = false>
__global__ void __launch_bounds__(kBlock, 4) k_dense2_tc(DevCfg c, DenseArgs a, const ulonglong2* __restrict__ Dg,
                                                         const uint4* __restrict__ Tg) {
  constexpr int CH = kChunkF32;
  extern __shared__ __align__(128) unsigned char smem[];
  uint4* sAr = reinterpret_cast<uint4*>(smem + tc::kOffA);
  uint4* sAi = sAr + 1024;
  unsigned char* sT = smem + tc::kOffT;
  uint64_t* b_full = reinterpret_cast<uint64_t*>(smem + tc::kOffBar);
  uint64_t* d_full = b_full + tc::kStages;
  uint32_t* sU = reinterpret_cast<uint32_t*>(smem + tc::kOffU);
  uint8_t* tlist = smem + tc::kOffList;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int chunk_l = blockIdx.y;                              // particle block fastest: the CTAs in flight share their tiles in L2
  const int cs = (a.chunk_first + chunk_l) * CH;
  const int ce = min(cs + CH, c.n_bins);
  const int ce2 = (ce + 1) & ~1;                               // pair-aligned end (data beyond n_bins is zero)
  const int p = blockIdx.x * kBlock + tid;

  if (!__syncthreads_or((a.jhi[p] > cs) && (a.jlo[p] < ce))) {
    double* fz = a.frag + (size_t)chunk_l * kFragFields * a.P_pad + p;
#pragma unroll
    for (int m = 0; m < kFragFields; ++m) fz[(size_t)m * a.P_pad] = 0.0;
    return;
  }

  if (tid == 0) {
#pragma unroll
    for (int i = 0; i < tc::kStages + 2; ++i) tc::mbar_init(b_full + i, 1);
    sU[1] = 0u; sU[2] = 0u; sU[3] = 0u; sU[4] = 0xffffffffu; sU[5] = 0xffffffffu; sU[6] = 0xffffffffu; sU[7] = 0u;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    __syncwarp();
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(tc::smem_u32(&sU[0])), "r"(128u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = sU[0];
  const uint32_t tm_lane = tmem + ((uint32_t)(warp * 32) << 16);

  const int jlo = a.jlo[p], jhi = a.jhi[p];
  const int S = c.stride, Sf = S >> 2, lgSf = c.log2_stride - 2;
  const int n_sub = CH >> lgSf;                                // <= 64 (Sf >= 32)
  const float hS = 1.0f / (float)Sf;
  const u64 h2 = f2bcast(2.0f * hS);
  const u64 K2 = f2bcast(1.4629180792671596e-09f);            // 2 pi / 2^32

  // which fine sub-intervals have all 128 lanes inside their windows (the tensor-core path), which coarse intervals merge
  {
    uint32_t m0 = 0u, m1 = 0u;
    for (int i = 0; i < n_sub; ++i) {
      const int ib = cs + (i << lgSf);
      if (ib >= ce2) break;
      if (ib >= jlo && min(ib + Sf, ce2) <= jhi) { if (i < 32) m0 |= 1u << i; else m1 |= 1u << (i - 32); }
    }
    uint32_t mm = 0u;
    if constexpr (MERGE) {
      const int n_co = CH >> c.log2_stride;                    // <= 4 (stride >= 512)
      for (int ic = 0; ic < n_co; ++ic) {
        const int ib = cs + (ic << c.log2_stride);
        const bool win = (ib >= jlo) && (ib + S <= jhi) && (ib + S <= ce2);
        if (win && coarse_dslope(c, a, p, ib >> c.log2_stride) <= a.merge_lim) mm |= 1u << ic;
      }
    }
    m0 = __reduce_and_sync(0xffffffffu, m0); m1 = __reduce_and_sync(0xffffffffu, m1); mm = __reduce_and_sync(0xffffffffu, mm);
    if (lane == 0) { atomicAnd(&sU[4], m0); atomicAnd(&sU[5], m1); atomicAnd(&sU[6], mm); }
  }
  __syncthreads();
  const unsigned long long fastmask = (unsigned long long)sU[4] | ((unsigned long long)sU[5] << 32);
  const uint32_t mergemask = MERGE ? sU[6] : 0u;
  const uint4* Tc = Tg + (size_t)(cs >> 5) * (tc::kTileBytes / 16);   // this chunk's tiles
  if (tid == 0) {
    int n = 0;
    for (int i = 0; i < n_sub; ++i) {
      if (!((fastmask >> i) & 1ull)) continue;
      const int ib = cs + (i << lgSf);
      const int nt = (min(ib + Sf, ce2) - ib + 31) >> 5;
      for (int t = 0; t < nt; ++t) tlist[n++] = (uint8_t)(((i << lgSf) >> 5) + t);
    }
    sU[7] = (uint32_t)n;
    for (int g = 0; g < min(n, 2); ++g) {
      tc::mbar_expect_tx(&b_full[g], tc::kTileBytes);
      tc::bulk_g2s(sT + g * tc::kTileBytes, Tc + (size_t)tlist[g] * (tc::kTileBytes / 16), tc::kTileBytes, &b_full[g]);
    }
  }
  __syncthreads();
  const int n_list = (int)sU[7];

  // MMAs of tile g (index into the tile list) into TMEM buffer g & 1, then the load of tile g + 2.  One lane.
  auto issue = [&](int g) {
    const int stg = g & 3, buf = g & 1;
    tc::mbar_wait(&b_full[stg], (uint32_t)((g >> 2) & 1));
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t aR = tc::smem_u32(sAr), aI = tc::smem_u32(sAi), bB = tc::smem_u32(sT + stg * tc::kTileBytes);
#pragma unroll
    for (int k = 0; k < 4; ++k) tc::mma_tf32(tmem + buf * 64, tc::make_desc(aR + k * 256), tc::make_desc(bB + k * 256), k > 0);
#pragma unroll
    for (int k = 0; k < 4; ++k) tc::mma_tf32(tmem + buf * 64 + 32, tc::make_desc(aI + k * 256), tc::make_desc(bB + k * 256), k > 0);
    tc::mma_commit(&d_full[buf]);
    if (g + 2 < n_list) {
      const int s2 = (g + 2) & 3;
      tc::mbar_expect_tx(&b_full[s2], tc::kTileBytes);
      tc::bulk_g2s(sT + s2 * tc::kTileBytes, Tc + (size_t)tlist[g + 2] * (tc::kTileBytes / 16), tc::kTileBytes, &b_full[s2]);
    }
  };

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
  int g_base = 0;              // tiles of the list that belong to earlier sub-intervals
  for (int ib = cs; ib < ce2; ib += Sf) {
    const int ie = min(ib + Sf, ce2);
    const int i_sub = (ib - cs) >> lgSf;
    const bool fast = (fastmask >> i_sub) & 1ull;              // CTA-uniform
    const bool lane_in = (ib >= jlo) && (ie <= jhi);
    const bool lane_out = (ie <= jlo) || (ib >= jhi);
    const bool all_in = fast || __all_sync(0xffffffffu, lane_in);
    const bool all_out = !fast && __all_sync(0xffffffffu, lane_out);

    float cf[4][4];    // cubic coefficients of (Ar, Ai, Er, Ei) in s = (j - ib)/Sf
    const bool merged = MERGE && ((mergemask >> ((ib - cs) >> c.log2_stride)) & 1u);
    if (merged) {
      if constexpr (MERGE) {
        if ((ib & (S - 1)) == 0) { coarse_phase(c, a, p, ib, fd); coarse_amps(c, a, p, ib, cc); }
        coarse_to_fine(cc, (ib >> lgSf) & 3, cf);              // the phase differences run on
      }
    } else if (!all_out) {
      sub_phase(c, a, p, ib, fd);
      sub_amps(c, a, p, ib, cf);
    }

    // tensor-core path: coefficient rows about the centre of the sub-interval, then the first two tiles
    u64 G[6] = {0, 0, 0, 0, 0, 0};
    const int n_t = fast ? ((ie - ib + 31) >> 5) : 0;
    int n_left = 0;            // tiles of this sub-interval this warp has released
    int cur_t = -1;            // tile whose MMAs this warp has waited for
    if (fast) {
      float g1[4], g2[4], g3[4];
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const float c0 = cf[r][0], c1 = cf[r][1], c2 = cf[r][2], c3 = cf[r][3];
        const float g0 = fmaf(0.5f, c1, c0) + fmaf(0.125f, c3, 0.25f * c2);
        g1[r] = fmaf(0.75f, c3, c1 + c2); g2[r] = fmaf(1.5f, c3, c2); g3[r] = c3;
        G[r] = f2bcast(g0);
        if (r == 1) G[4] = f2bcast(-g0);
        if (r == 3) G[5] = f2bcast(-g0);
      }
      const int at = (tid >> 3) * 64 + (tid & 7);
      auto rows = [&](const float (&v)[4], int kc_hi0, int kc_lo, int kc_hi1) {
        float h[4], l[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) { h[r] = tc::tf32_rna(v[r]); l[r] = tc::tf32_rna(v[r] - h[r]); }
        const uint4 hr = make_uint4(__float_as_uint(h[0]), __float_as_uint(h[1]), __float_as_uint(h[2]), __float_as_uint(h[3]));
        const uint4 hi_ = make_uint4(__float_as_uint(-h[1]), __float_as_uint(h[0]), __float_as_uint(-h[3]), __float_as_uint(h[2]));
        sAr[at + kc_hi0 * 8] = hr; sAi[at + kc_hi0 * 8] = hi_;
        if (kc_lo >= 0) {
          const uint4 lr = make_uint4(__float_as_uint(l[0]), __float_as_uint(l[1]), __float_as_uint(l[2]), __float_as_uint(l[3]));
          const uint4 li = make_uint4(__float_as_uint(-l[1]), __float_as_uint(l[0]), __float_as_uint(-l[3]), __float_as_uint(l[2]));
          sAr[at + kc_lo * 8] = lr; sAi[at + kc_lo * 8] = li;
          sAr[at + kc_hi1 * 8] = hr; sAi[at + kc_hi1 * 8] = hi_;
        }
      };
      rows(g1, 0, 1, 2); rows(g2, 3, 4, 5); rows(g3, 6, -1, -1);
      sAr[at + 7 * 8] = make_uint4(0u, 0u, 0u, 0u); sAi[at + 7 * 8] = make_uint4(0u, 0u, 0u, 0u);
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncwarp();
      if (lane == 0) {
        const uint32_t old = tc::atom_add_acqrel(&sU[1], 1u);
        if ((old & 3u) == 3u) { issue(g_base); if (n_t > 1) issue(g_base + 1); }
      }
      __syncwarp();
    }
    auto leave = [&](int u) {                                  // this warp is done with tile u of the sub-interval
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      __syncwarp();
      if (lane == 0) {
        const int g = g_base + u;
        const uint32_t old = tc::atom_add_acqrel(&sU[2 + (g & 1)], 1u);
        if ((old & 3u) == 3u && u + 2 < n_t) issue(g + 2);
      }
      __syncwarp();
    };
    auto enter = [&](int t) {                                  // wait for the MMAs of tile t
      while (n_left < t) leave(n_left++);
      const int g = g_base + t;
      tc::mbar_wait(&d_full[g & 1], (uint32_t)((g >> 1) & 1));
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    };

    u64 s2 = 0;        // (s_j, s_{j+1}) of the next pair
    const ulonglong2* rec = Dg;   // its data record
    auto pair = [&](int j, auto masked_c, auto with_sg_c, u64& zr2, u64& zi2, u64& sg2) {
      pair_eval<decltype(masked_c)::value, decltype(with_sg_c)::value, SC>(fd, cf, s2, rec, j, jlo, jhi, h2, K2, zr2, zi2, sg2);
    };
    auto sigma_piece = [&](int piece) { Sg += sigma_moments(cf, a.moments + (size_t)piece * 4); };
    using T_ = std::true_type;

    const bool use_mom = all_in;      // all lanes inside their windows: sigma from the piece moments, unmasked pairs
    int piece = use_mom ? a.piece_first[(ib >> lgSf) - ((a.chunk_first * CH) >> lgSf)] : 0;
    float car_zr = 0.f, car_zi = 0.f, car_sg = 0.f;
    bool carry = false;
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
        if (!fast) {
          s2 = f2pack((float)(jj - ib) * hS, (float)(jj + 1 - ib) * hS);
          rec = Dg + (size_t)(jj >> 1) * kPairRec;
        }
        while (jj < ph) {
          const bool split = (jj == jfull);                    // the pair (ph - 1, ph)
          int e2 = split ? jj + 2 : min(jj + kFlushBins, jfull);
          u64 zr2 = 0, zi2 = 0, sg2 = 0;
          if (fast) {
            e2 = min(e2, (jj & ~31) + 32);                     // a flush group stays inside one tile
            const int t = (jj - ib) >> 5, g = g_base + t, off = jj & 31;
            if (t != cur_t) { enter(t); cur_t = t; }
            const ulonglong2* trec = reinterpret_cast<const ulonglong2*>(sT + (g & 3) * tc::kTileBytes + tc::kImgBytes) + (off >> 1) * kPairRec;
            pairs_fast_tc<SC>(fd, G, trec, tm_lane + (uint32_t)((g & 1) * 64 + off), (e2 - jj) >> 1, K2, zr2, zi2);
            jj = e2;
          } else if (use_mom) { pairs_fast<SC>(fd, cf, s2, rec, (e2 - jj) >> 1, h2, K2, zr2, zi2); jj = e2; }
          else                { for (; jj < e2; jj += 2) pair(jj, T_{}, T_{}, zr2, zi2, sg2); }
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
    if (fast) {
      // every MMA of this sub-interval has completed before this warp rewrites its coefficient rows
      if (cur_t != n_t - 1) enter(n_t - 1);
      while (n_left < n_t) leave(n_left++);
      g_base += n_t;
    }
  }
  if (k >= 0 && k < a.n_seg) close_piece(false);
  if (!SEG) {
    frag[0] = ups;
    if (a.comp) { frag[(size_t)7 * a.P_pad] = xs; frag[(size_t)8 * a.P_pad] = hs; }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"(128u) : "memory");
  }
}

}  // namespace
