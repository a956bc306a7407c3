// Grouped / ragged batched complex-FP64 GEMM on the FP64 tensor pipe (sm_100a).
//
// Serves the three contraction stages of the GW self-energy (Algorithm 4 lines 5, 7, 8 of
// arXiv 2405.09494) and the block-basis unfold (Eq. 28).
// Descriptors: include/gwsig_plan.h.  Design notes: DESIGN.md section 5.
//
//  * persistent CTAs, dynamic tile scheduler (one atomic per tile, heaviest problems first)
//  * operands staged global -> shared with 16-byte cp.async (one complex128 per copy, so every
//    two-level ragged index is addressable and ragged edges are zero-filled), STAGES-deep ring
//  * shared tiles are k-major with leading dimension = 2 (mod 8) complex elements: the
//    one-double2-per-lane fragment loads of mma.m8n8k4.f64 are bank-conflict free
//  * complex product = 4 real DMMA per 8x8x4 tile: re += ar*br, re += (-ai)*bi, im += ar*bi, im += ai*br
#include <cuda_runtime.h>
#include <stdint.h>

#include "zgemm_grouped.cuh"

namespace {

__device__ __forceinline__ long long idx2(const gwsig_idx2& d, int i) {
  if (d.div == GWSIG_NODIV) return (long long)i * d.lo;
  int q = i / d.div;
  return (long long)q * d.hi + (long long)(i - q * d.div) * d.lo;
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src, bool valid) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
  int bytes = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem_src), "r"(bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

// D(8x8) += A(8x4) * B(4x8), FP64 tensor core.  SASS: DMMA.8x8x4
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// linear tile id -> problem (binary search on tile_begin), batch entry, tile coordinates
struct TileInfo {
  int prob, batch, tm, tn;
};
__device__ __forceinline__ TileInfo decode_tile(const ZgParams& p, long long tile) {
  int lo = 0, hi = p.nprob - 1;
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    if (__ldg(&p.prob[mid].tile_begin) <= tile) lo = mid; else hi = mid - 1;
  }
  const gwsig_problem& P = p.prob[lo];
  long long local = tile - P.tile_begin;
  int per = P.tiles_m * P.tiles_n;
  TileInfo t;
  t.prob = lo;
  t.batch = (int)(local / per);
  int r = (int)(local - (long long)t.batch * per);
  t.tm = r / P.tiles_n;
  t.tn = r - t.tm * P.tiles_n;
  return t;
}

// ------------------------------------------------------------------------------------------
// tensor-core engine
// ------------------------------------------------------------------------------------------
template <int BM, int BN, int WARPS_M, int WARPS_N, int STAGES>
__global__ void __launch_bounds__(WARPS_M* WARPS_N * 32) zgemm_grouped_dmma(ZgParams p) {
  constexpr int BK = 8;
  constexpr int NT = WARPS_M * WARPS_N * 32;
  constexpr int WTM = BM / WARPS_M, WTN = BN / WARPS_N;
  constexpr int MI = WTM / 8, NI = WTN / 8;
  constexpr int LDA = BM + 2, LDB = BN + 2;          // = 2 (mod 8): conflict-free fragment loads
  constexpr int A_PER = (BM * BK) / NT, B_PER = (BN * BK) / NT;
  static_assert((BM * BK) % NT == 0 && (BN * BK) % NT == 0, "tile / thread mismatch");
  static_assert(BM % 8 == 0 && BN % 8 == 0 && LDA % 8 == 2 && LDB % 8 == 2, "layout");

  extern __shared__ double2 zg_smem[];
  double2* As = zg_smem;                           // [STAGES][BK][LDA]
  double2* Bs = zg_smem + STAGES * BK * LDA;       // [STAGES][BK][LDB]
  __shared__ unsigned long long s_tile;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / WARPS_N) * WTM, wn0 = (warp % WARPS_N) * WTN;
  const int fr = lane >> 2, fk = lane & 3;         // fragment row / k index of this lane

  while (true) {
    __syncthreads();                                // previous tile fully consumed (smem, s_tile)
    if (tid == 0) s_tile = atomicAdd(p.counter, 1ULL);
    __syncthreads();
    const long long tile = (long long)s_tile;
    if (tile >= p.total_tiles) break;

    const TileInfo ti = decode_tile(p, tile);
    const gwsig_problem& P = p.prob[ti.prob];
    const int M = P.M, N = P.N, flags = P.flags;
    const int m0 = ti.tm * BM, n0 = ti.tn * BN;
    const long long a_boff = (long long)ti.batch * P.a_bstride + (long long)p.t0 * P.a_tstride;
    const long long b_boff = (long long)ti.batch * P.b_bstride + (long long)p.t0 * P.b_tstride;
    const bool kmajor = (flags & GWSIG_FLAG_A_KMAJOR) != 0;
    const bool conjA = (flags & GWSIG_FLAG_CONJ_A) != 0, conjB = (flags & GWSIG_FLAG_CONJ_B) != 0;

    // this thread's slots in the A and B tiles
    int a_ml[A_PER], a_kl[A_PER], b_nl[B_PER], b_kl[B_PER];
#pragma unroll
    for (int e = 0; e < A_PER; ++e) {
      int lin = tid + e * NT;
      if (kmajor) { a_kl[e] = lin % BK; a_ml[e] = lin / BK; }
      else        { a_ml[e] = lin % BM; a_kl[e] = lin / BM; }
    }
#pragma unroll
    for (int e = 0; e < B_PER; ++e) {
      int lin = tid + e * NT;
      b_nl[e] = lin % BN; b_kl[e] = lin / BN;
    }

    // how many 8-row / 8-column MMA sub-tiles of this warp hold real data
    const int mi_act = min(MI, max(0, (M - m0 - wm0 + 7) >> 3));
    const int ni_act = min(NI, max(0, (N - n0 - wn0 + 7) >> 3));

    double cre[MI][NI][2], cim[MI][NI][2];
#pragma unroll
    for (int i = 0; i < MI; ++i)
#pragma unroll
      for (int j = 0; j < NI; ++j) { cre[i][j][0] = cre[i][j][1] = 0.0; cim[i][j][0] = cim[i][j][1] = 0.0; }

    // ---- flattened (segment, k0) iteration space; the loader runs STAGES-1 iterations ahead ----
    const int nseg = P.seg_count;
    int total_iters = 0;
    for (int s = 0; s < nseg; ++s) total_iters += (__ldg(&p.seg[P.seg_begin + s].K) + BK - 1) / BK;

    int ld_seg = -1, ld_k0 = 0, ld_K = 0;            // loader position
    const double2* a_ptr[A_PER];
    const double2* b_ptr[B_PER];
    bool a_ok[A_PER], b_ok[B_PER];
    gwsig_idx2 ak, bk;
    ak.div = bk.div = GWSIG_NODIV; ak.hi = ak.lo = bk.hi = bk.lo = 0;

    auto next_segment = [&]() {
      do { ++ld_seg; ld_K = __ldg(&p.seg[P.seg_begin + ld_seg].K); } while (ld_K == 0);   // skip empty segments
      ld_k0 = 0;
      const gwsig_seg& S = p.seg[P.seg_begin + ld_seg];
      ak = S.ak;
      bk = S.bk;
#pragma unroll
      for (int e = 0; e < A_PER; ++e) {
        int m = m0 + a_ml[e];
        a_ok[e] = m < M;
        a_ptr[e] = p.A + S.a_off + a_boff + (a_ok[e] ? idx2(S.am, m) : 0);
      }
#pragma unroll
      for (int e = 0; e < B_PER; ++e) {
        int n = n0 + b_nl[e];
        b_ok[e] = n < N;
        b_ptr[e] = p.B + S.b_off + b_boff + (b_ok[e] ? idx2(S.bn, n) : 0);
      }
    };

    auto issue_loads = [&](int stage) {
      if (ld_seg < 0 || ld_k0 >= ld_K) next_segment();
      double2* as = As + stage * BK * LDA;
      double2* bs = Bs + stage * BK * LDB;
#pragma unroll
      for (int e = 0; e < A_PER; ++e) {
        int k = ld_k0 + a_kl[e];
        bool ok = a_ok[e] && k < ld_K;
        cp_async16(as + a_kl[e] * LDA + a_ml[e], ok ? (const void*)(a_ptr[e] + idx2(ak, k)) : (const void*)p.A, ok);
      }
#pragma unroll
      for (int e = 0; e < B_PER; ++e) {
        int k = ld_k0 + b_kl[e];
        bool ok = b_ok[e] && k < ld_K;
        cp_async16(bs + b_kl[e] * LDB + b_nl[e], ok ? (const void*)(b_ptr[e] + idx2(bk, k)) : (const void*)p.B, ok);
      }
      ld_k0 += BK;
    };

    int issued = 0;
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
      if (issued < total_iters) { issue_loads(s); ++issued; }
      cp_async_commit();
    }

    for (int it = 0; it < total_iters; ++it) {
      cp_async_wait<STAGES - 2>();
      __syncthreads();
      if (issued < total_iters) { issue_loads((it + STAGES - 1) % STAGES); ++issued; }
      cp_async_commit();

      const double2* as = As + (it % STAGES) * BK * LDA;
      const double2* bs = Bs + (it % STAGES) * BK * LDB;
#pragma unroll
      for (int kk = 0; kk < BK / 4; ++kk) {
        double2 af[MI], bf[NI];
#pragma unroll
        for (int i = 0; i < MI; ++i)
          if (i < mi_act) {
            af[i] = as[(kk * 4 + fk) * LDA + wm0 + i * 8 + fr];
            if (conjA) af[i].y = -af[i].y;
          }
#pragma unroll
        for (int j = 0; j < NI; ++j)
          if (j < ni_act) {
            bf[j] = bs[(kk * 4 + fk) * LDB + wn0 + j * 8 + fr];
            if (conjB) bf[j].y = -bf[j].y;
          }
#pragma unroll
        for (int i = 0; i < MI; ++i)
          if (i < mi_act) {
            const double nai = -af[i].y;
#pragma unroll
            for (int j = 0; j < NI; ++j)
              if (j < ni_act) {
                dmma884(cre[i][j][0], cre[i][j][1], af[i].x, bf[j].x);
                dmma884(cim[i][j][0], cim[i][j][1], af[i].x, bf[j].y);
                dmma884(cre[i][j][0], cre[i][j][1], nai, bf[j].y);
                dmma884(cim[i][j][0], cim[i][j][1], af[i].y, bf[j].x);
              }
          }
      }
    }
    cp_async_wait<0>();

    // ---- epilogue: registers -> C (two-level addressing, optional accumulate) ------------------
    double2* cbase = p.C + P.c_off + (long long)ti.batch * P.c_bstride + (long long)p.t0 * P.c_tstride;
    const bool accum = (flags & GWSIG_FLAG_ACCUM) != 0;
    long long cn_off[NI][2];
    bool cn_ok[NI][2];
#pragma unroll
    for (int j = 0; j < NI; ++j)
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        int n = n0 + wn0 + j * 8 + fk * 2 + c;
        cn_ok[j][c] = n < N;
        cn_off[j][c] = cn_ok[j][c] ? idx2(P.cn, n) : 0;
      }
#pragma unroll
    for (int i = 0; i < MI; ++i) {
      int m = m0 + wm0 + i * 8 + fr;
      if (m >= M) continue;
      long long cm_off = idx2(P.cm, m);
#pragma unroll
      for (int j = 0; j < NI; ++j)
#pragma unroll
        for (int c = 0; c < 2; ++c)
          if (cn_ok[j][c]) {
            double2* dst = cbase + cm_off + cn_off[j][c];
            double2 v = make_double2(cre[i][j][c], cim[i][j][c]);
            if (accum) { double2 o = *dst; v.x += o.x; v.y += o.y; }
            *dst = v;
          }
    }
  }
}

// ------------------------------------------------------------------------------------------
// reference engine: same plan, one thread per output element, plain DFMA, no shared memory
// ------------------------------------------------------------------------------------------
template <int BM, int BN>
__global__ void __launch_bounds__(256) zgemm_grouped_reference(ZgParams p) {
  for (long long tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x) {
    const TileInfo ti = decode_tile(p, tile);
    const gwsig_problem& P = p.prob[ti.prob];
    const bool conjA = (P.flags & GWSIG_FLAG_CONJ_A) != 0, conjB = (P.flags & GWSIG_FLAG_CONJ_B) != 0;
    const long long a_boff = (long long)ti.batch * P.a_bstride + (long long)p.t0 * P.a_tstride;
    const long long b_boff = (long long)ti.batch * P.b_bstride + (long long)p.t0 * P.b_tstride;
    double2* cbase = p.C + P.c_off + (long long)ti.batch * P.c_bstride + (long long)p.t0 * P.c_tstride;
    for (int e = threadIdx.x; e < BM * BN; e += blockDim.x) {
      int m = ti.tm * BM + e / BN, n = ti.tn * BN + e % BN;
      if (m >= P.M || n >= P.N) continue;
      double sr = 0.0, si = 0.0;
      for (int s = 0; s < P.seg_count; ++s) {
        const gwsig_seg& S = p.seg[P.seg_begin + s];
        const double2* a = p.A + S.a_off + a_boff + idx2(S.am, m);
        const double2* b = p.B + S.b_off + b_boff + idx2(S.bn, n);
        for (int k = 0; k < S.K; ++k) {
          double2 x = a[idx2(S.ak, k)], y = b[idx2(S.bk, k)];
          if (conjA) x.y = -x.y;
          if (conjB) y.y = -y.y;
          sr += x.x * y.x - x.y * y.y;
          si += x.x * y.y + x.y * y.x;
        }
      }
      double2* dst = cbase + idx2(P.cm, m) + idx2(P.cn, n);
      if (P.flags & GWSIG_FLAG_ACCUM) { sr += dst->x; si += dst->y; }
      *dst = make_double2(sr, si);
    }
  }
}

template <int BM, int BN, int WM, int WN, int STAGES>
cudaError_t launch_dmma(const ZgParams& p, int num_sms, cudaStream_t stream) {
  auto kern = zgemm_grouped_dmma<BM, BN, WM, WN, STAGES>;
  constexpr int smem = STAGES * 8 * ((BM + 2) + (BN + 2)) * (int)sizeof(double2);
  static bool configured = false;
  static int occ = 1;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, WM * WN * 32, smem);
    if (e != cudaSuccess) return e;
    if (occ < 1) occ = 1;
    configured = true;
  }
  long long grid = (long long)num_sms * occ;
  if (grid > p.total_tiles) grid = p.total_tiles;
  if (grid < 1) return cudaSuccess;
  kern<<<(unsigned)grid, WM * WN * 32, smem, stream>>>(p);
  return cudaGetLastError();
}

}  // namespace

ZgTile zg_tile_shape(int shape_class) {
  switch (shape_class) {
    case 1: return ZgTile{64, 32};
    default: return ZgTile{64, 64};
  }
}

cudaError_t zg_launch(int engine, int shape_class, const ZgParams& p, int num_sms, cudaStream_t stream) {
  if (p.total_tiles <= 0) return cudaSuccess;
  if (engine == 1) {
    long long grid = p.total_tiles < 65535LL * 16 ? p.total_tiles : 65535LL * 16;
    if (shape_class == 1) zgemm_grouped_reference<64, 32><<<(unsigned)grid, 256, 0, stream>>>(p);
    else zgemm_grouped_reference<64, 64><<<(unsigned)grid, 256, 0, stream>>>(p);
    return cudaGetLastError();
  }
  if (shape_class == 1) return launch_dmma<64, 32, 4, 2, 3>(p, num_sms, stream);
  return launch_dmma<64, 64, 4, 2, 3>(p, num_sms, stream);
}
