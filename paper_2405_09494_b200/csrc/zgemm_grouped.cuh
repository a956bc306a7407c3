// Grouped / ragged batched complex-FP64 GEMM engine (declarations) and the tiling rule that the host plan and
// the device kernels share.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "gwsig_plan.h"

#if defined(__CUDACC__)
#define ZG_HD __host__ __device__ __forceinline__
#else
#define ZG_HD inline
#endif

// ---- tiling rule -----------------------------------------------------------------------------------------
// A problem C[M x N] is cut into tiles of bm rows (ZG_BM = 128 or ZG_BM3 = 64, by engine) and of at most ZG_NG_MAX = 4 column groups of 8:
// the G = ceil(N / 8) column groups are dealt evenly to tiles_n = ceil(G / 4) tiles (tile j owns groups
// [j G / tiles_n, (j + 1) G / tiles_n)), so a ragged N costs no tensor-pipe time beyond its last group of 8.
// Tiles of a problem are numbered batch-major, then m, then n (n fastest).
constexpr int ZG_BM = 128;                // tile height of the 4-product kernel (and the default of the plan)
constexpr int ZG_BM3 = 64;                // tile height of the 3M kernel (two CTAs per SM, eight MMA warps each)
constexpr int ZG_NG_MAX = 4;
constexpr int ZG_BN = 8 * ZG_NG_MAX;
constexpr int ZG_BUCKET_SHIFT = 6;        // tile -> problem lookup: one table entry per 64 tiles

ZG_HD int zg_tiles_m(int M, int bm) { return (M + bm - 1) / bm; }
ZG_HD int zg_tiles_n(int N) { return ((N + 7) / 8 + ZG_NG_MAX - 1) / ZG_NG_MAX; }
ZG_HD void zg_ntile(int N, int tiles_n, int tn, int& n0, int& ncols) {
  const int G = (N + 7) / 8;
  const int g0 = (tn * G) / tiles_n, g1 = ((tn + 1) * G) / tiles_n;      // G < 2^27 / tiles_n: no overflow
  n0 = 8 * g0;
  const int n1 = 8 * g1 < N ? 8 * g1 : N;
  ncols = n1 - n0;
}

struct ZgParams {
  const double2* A;
  const double2* B;
  double2* C;
  const gwsig_problem* prob;   // device, ordered by tile_begin
  const gwsig_seg* seg;        // device
  const int* bucket;           // device: bucket[t >> ZG_BUCKET_SHIFT] = index of the problem holding tile (t & ~63)
  int nprob;
  long long total_tiles;
  int t0;                      // first tau of the chunk (multiplies *_tstride)
  int bm;                      // tile height the plan was built for (ZG_BM or ZG_BM3)
  int use_bulk;                // 3M kernel: move whole-row operands with cp.async.bulk (UBLKCP) instead of 16-byte cp.async
  unsigned long long* counter; // device, zeroed before launch (dynamic tile scheduler)
};

// enqueue one grouped GEMM; engine: 0 = DMMA tensor path, 1 = reference DFMA path.
// GWSIG_FLAG_ACCUM problems add into C with FP64 atomics (several problems / split-K parts may share a C block).
cudaError_t zg_launch(int engine, const ZgParams& p, int num_sms, cudaStream_t stream);
