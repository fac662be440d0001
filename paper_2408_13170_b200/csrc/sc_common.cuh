// sc_common.cuh -- constants shared by the kernel files of libscstat.so (see sc_stat.cu for the pipeline).
#pragma once
#include "../../include/sc_stat.h"
#include "sc_math.cuh"

#include <climits>
#include <cstdint>
#include <type_traits>

using namespace sc;

namespace {

constexpr int kBlock = 128;            // threads per CTA of the dense kernel = particles per CTA
constexpr int kChunkF32 = 2048;        // bins per CTA, FP32 amplitude path (24 B/bin of shared memory)
constexpr int kChunkF64 = 1024;        // bins per CTA, all-FP64 path (48 B/bin)
constexpr int kFlushBins = 32;         // FP32 partial sums are folded into the FP64 accumulators this often
constexpr int kFragFields = 9;         // partial Upsilon, head (zr, zi, sg), tail (zr, zi, sg), partial sum|z|, partial sum sigma
constexpr double kMagic = 6755399441055744.0;   // 1.5 * 2^52: (x + kMagic) - kMagic = rint(x), low word = int

// chunk flags (host-built from the edges, shared by all particles)
enum : uint8_t { CF_HEAD = 1, CF_HEAD_CLOSES = 2, CF_TAIL = 4 };

}  // namespace
