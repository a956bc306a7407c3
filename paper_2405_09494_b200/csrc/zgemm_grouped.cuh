// Grouped / ragged batched complex-FP64 GEMM engine (declarations).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "gwsig_plan.h"

struct ZgParams {
  const double2* A;
  const double2* B;
  double2* C;
  const gwsig_problem* prob;   // device
  const gwsig_seg* seg;        // device
  int nprob;
  long long total_tiles;
  int t0;                      // first tau of the chunk (multiplies *_tstride)
  unsigned long long* counter; // device, zeroed before launch (dynamic tile scheduler)
};

struct ZgTile { int bm, bn; };

// tile shape the engine uses for a given shape class; the plan must tile with the same numbers
ZgTile zg_tile_shape(int shape_class);

// enqueue one grouped GEMM; engine: 0 = DMMA tensor path, 1 = reference DFMA path
cudaError_t zg_launch(int engine, int shape_class, const ZgParams& p, int num_sms, cudaStream_t stream);
