// Grouped / ragged batched complex-FP64 GEMM on the FP64 tensor pipe (sm_100a).
//
// TWO tensor-core kernels share the loader, the tile scheduler and the descriptors:
//   zgemm_grouped_dmma3m (engine 0, default): Karatsuba / "3M" complex product -- three REAL products
//       P1 = Ar Br, P2 = Ai Bi, P3 = (Ar+Ai)(Br+Bi),  re = P1 - P2,  im = P3 - P1 - P2  (25 % fewer DMMA than 4M),
//       one product per group of four MMA warps (12 MMA warps, 32 accumulator doubles each), accumulators handed to
//       four EPILOGUE warps through shared memory so that the MMA warps never touch global memory or index arithmetic:
//       loader warps -> MMA warps -> epilogue warps, decoupled by mbarriers (details above the kernel)
//   zgemm_grouped_dmma   (engine 2): the conventional four-product kernel (engine v3 of round 1), described below.
//
// Serves the three contraction stages of the GW self-energy (Algorithm 4 lines 5, 7, 8 of
// arXiv 2405.09494).  Descriptors: include/gwsig_plan.h.  Design: DESIGN.md section 5.
//
//  * persistent CTAs (2 per SM), dynamic tile scheduler over a cost-sorted tile list; the tile counter is
//    fetched one tile ahead and a tile is mapped to its problem through a 64-tile bucket table
//  * warp-specialised: FOUR PRODUCER WARPS do all index arithmetic (two-level ragged addressing) and stage
//    operands global -> shared with 16-byte cp.async (one complex128 per copy), signalling a STAGES-deep ring
//    of mbarriers (cp.async.mbarrier.arrive.noinc); the FOUR CONSUMER WARPS only wait, load fragments and
//    issue DMMA, then release the slot.  setmaxnreg moves the producers' registers to the consumers.
//  * tile = 128 rows x (<= 4 column groups of 8).  The 16 row groups of a tile are dealt round-robin to the
//    four consumer warps (warp w owns groups w, w+4, w+8, w+12), every warp owns all column groups: ragged
//    edges leave no warp idle, and the main loop is instantiated for every (row groups, column groups) count
//    of a warp -- 16 variants of straight-line, unpredicated DMMA -- so padding never reaches the tensor pipe
//    beyond the last group of 8 (rows, columns) or 4 (k)
//  * shared tiles are k-major with leading dimension = 2 (mod 8) complex elements: the
//    one-double2-per-lane fragment loads of mma.m8n8k4.f64 are bank-conflict free
//  * complex product = 4 real DMMA per 8x8x4 tile: re += ar*br, im += ar*bi, re += (-ai)*bi, im += ai*br,
//    issued in four passes over the warp tile so that dependent DMMAs are far apart
//  * GWSIG_FLAG_ACCUM tiles add into C with red.global.add.f64 (split-K parts of stage 3 share a Sigma block)
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "zgemm_grouped.cuh"

namespace {

// two-level index: one shared copy of the division code (the kernel's hot code has to stay small: all SMs of a GPC
// share one instruction cache behind their 32 KB L1.5, and warp-specialised CTAs run several code regions at once)
__device__ __noinline__ long long idx2_div(long long hi, long long lo, int div, int i) {
  int q = i / div;
  return (long long)q * hi + (long long)(i - q * div) * lo;
}
__device__ __forceinline__ long long idx2(const gwsig_idx2& d, int i) {
  if (d.div == GWSIG_NODIV) return (long long)i * d.lo;
  return idx2_div(d.hi, d.lo, d.div, i);
}

__device__ __forceinline__ void cp_async16(unsigned smem_dst, const void* gmem_src, bool valid) {
  int bytes = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(smem_dst), "l"(gmem_src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared.b64 st, [%0];\n\t}\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_cp_async(unsigned bar) {   // fires when this thread's prior cp.async land
  asm volatile("cp.async.mbarrier.arrive.noinc.shared.b64 [%0];\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(unsigned bar, unsigned parity) {
  unsigned ok;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "mbarrier.try_wait.parity.shared.b64 p, [%1], %2;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}\n"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok != 0;
}
// a wait that cannot complete (a protocol bug) traps after ~2^26 polls instead of hanging the GPU until the job is killed
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  unsigned spins = 0;
  while (!mbar_try_wait(bar, parity))
    if (++spins > (1u << 26)) __trap();
}

// D(8x8) += A(8x4) * B(4x8), FP64 tensor core.  SASS: DMMA.8x8x4
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ double xor_hi(double x, unsigned m) {      // sign flips on the integer pipe
  return __hiloint2double(__double2hiint(x) ^ (int)m, __double2loint(x));
}
__device__ __forceinline__ void red_add(double* addr, double v) {
  asm volatile("red.global.add.f64 [%0], %1;\n" ::"l"(addr), "d"(v) : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;\n" ::"r"(id), "r"(nthreads) : "memory");
}

// linear tile id -> problem (bucket table + short forward scan on tile_begin), batch entry, tile coordinates
struct TileInfo {
  int prob, batch, tm, tn;
};
__device__ __forceinline__ TileInfo decode_tile(const ZgParams& p, long long tile) {
  int lo = __ldg(&p.bucket[tile >> ZG_BUCKET_SHIFT]);
  while (lo + 1 < p.nprob && __ldg(&p.prob[lo + 1].tile_begin) <= tile) ++lo;
  const gwsig_problem& P = p.prob[lo];
  const unsigned local = (unsigned)(tile - __ldg(&P.tile_begin));      // tiles of one problem < 2^32 (checked by the plan)
  const unsigned tn_ = (unsigned)__ldg(&P.tiles_n);
  const unsigned per = (unsigned)__ldg(&P.tiles_m) * tn_;
  TileInfo t;
  t.prob = lo;
  t.batch = (int)(local / per);
  const unsigned r = local - (unsigned)t.batch * per;
  t.tm = (int)(r / tn_);
  t.tn = (int)(r - (unsigned)t.tm * tn_);
  return t;
}

struct SlotHdr {
  int ctl;            // bit0: first slot of a tile, bit1: last slot of a tile, bit2: no more work
  int nk4;            // k4-steps of this slot that hold data (1 or 2)
  int trec;           // index of the tile record (valid when bit0)
  int pad_;
};
struct __align__(16) TileRec {   // what the consumers need to know about a tile (written by the producer)
  int mrows, ncols;   // rows / columns of this tile that exist
  int flags, pad_;
  long long c_off;    // element offset of C(m = 0, n = 0) incl. batch / tau offsets
  int m0, n0;
  gwsig_idx2 cm, cn;
};

constexpr int kProducerWarps = 4;
constexpr int kConsumerWarps = 4;
constexpr int kProducerRegs = 56;
constexpr int kConsumerRegs = 200;
constexpr int BK = 8;
constexpr int LDA = ZG_BM + 2, LDB = ZG_BN + 2;          // = 2 (mod 8): conflict-free fragment loads
constexpr int kStages = 5;
static_assert(LDA % 8 == 2 && LDB % 8 == 2, "layout");

// ------------------------------------------------------------------------------------------
// loader (producer) side, shared by both kernels: kProducerWarps warps stage tiles global -> shared
// ------------------------------------------------------------------------------------------
struct RingCtl {
  unsigned full0, empty0;        // shared addresses of the full / empty mbarrier arrays
  SlotHdr* hdr;
  TileRec* trec;
  int ntrec;
  long long* next_tile;
};

__device__ __forceinline__ void producer_loop(const ZgParams& p, double2* As, double2* Bs, const RingCtl& rc, int pw, int lane) {
  const unsigned full0 = rc.full0, empty0 = rc.empty0;
  SlotHdr* hdr = rc.hdr;
  TileRec* trec = rc.trec;
  long long* next_tile = rc.next_tile;
  int stage = 0;
  unsigned phase = 0;
  const bool leader = pw == 0 && lane == 0;
  const unsigned as0 = (unsigned)__cvta_generic_to_shared(As), bs0 = (unsigned)__cvta_generic_to_shared(Bs);
  int tslot = 0, tbuf = 0;
  long long pre = 0;                                  // tile id fetched one tile ahead (leader only)
  if (leader) pre = (long long)atomicAdd(p.counter, 1ULL);
  while (true) {
    if (leader) next_tile[tbuf] = pre;
    named_bar_sync(1, kProducerWarps * 32);
    const long long tile = next_tile[tbuf];
    tbuf ^= 1;
    if (tile >= p.total_tiles) break;
    if (leader) pre = (long long)atomicAdd(p.counter, 1ULL);       // lands while this tile is being staged
    const TileInfo ti = decode_tile(p, tile);
    const gwsig_problem& P = p.prob[ti.prob];
    const int M = __ldg(&P.M), N = __ldg(&P.N), flags = __ldg(&P.flags);
    const int m0 = ti.tm * ZG_BM;
    int n0, ncols;
    zg_ntile(N, __ldg(&P.tiles_n), ti.tn, n0, ncols);
    const int mrows = min(ZG_BM, M - m0);
    const long long a_boff = (long long)ti.batch * __ldg(&P.a_bstride) + (long long)p.t0 * __ldg(&P.a_tstride);
    const long long b_boff = (long long)ti.batch * __ldg(&P.b_bstride) + (long long)p.t0 * __ldg(&P.b_tstride);
    const int seg_begin = __ldg(&P.seg_begin), nseg = __ldg(&P.seg_count);
    const bool kmajor = (flags & GWSIG_FLAG_A_KMAJOR) != 0;
    bool first = true;
    for (int s = 0; s < nseg; ++s) {
      const gwsig_seg& S = p.seg[seg_begin + s];
      const int K = __ldg(&S.K);
      if (K == 0) continue;
      const bool last_seg = s == nseg - 1;
      const gwsig_idx2 ak = S.ak, bk = S.bk;
      const double2* abase = p.A + __ldg(&S.a_off) + a_boff;
      const bool b_ok = lane < ncols;
      const double2* b_col = p.B + __ldg(&S.b_off) + b_boff + (b_ok ? idx2(S.bn, n0 + lane) : 0);
      // A row offsets of this lane (32-bit: element offsets inside a tile stay < 2^31, checked by the plan).
      //   A contiguous along m: lane <-> tile rows lane + 32 r (r < 4); this warp stages k-rows 2 pw, 2 pw + 1
      //   A contiguous along k: lane <-> (k = lane & 7, tile rows 4 (lane >> 3) + pw + 16 j, j < 8)
      const gwsig_idx2 am = S.am;
      const int kl = lane & 7, mr = 4 * (lane >> 3) + pw;
      int a_roff[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int ml = kmajor ? mr + 16 * j : lane + 32 * j;
        a_roff[j] = ((kmajor || j < 4) && ml < mrows) ? (int)idx2(am, m0 + ml) : -1;
      }
      for (int k0 = 0; k0 < K; k0 += BK) {
        mbar_wait(empty0 + 8 * stage, phase ^ 1);
        const unsigned as = as0 + (unsigned)(stage * BK * LDA) * 16u;
        const unsigned bs = bs0 + (unsigned)(stage * BK * LDB) * 16u;
        const bool two = k0 + 4 < K;                      // the slot's second k4 step holds data
        if (!kmajor) {
#pragma unroll
          for (int h2 = 0; h2 < 2; ++h2) {
            const int kk = 2 * pw + h2;
            const int k = k0 + kk;
            if (kk < 4 || two) {
              const bool kok = k < K;
              const double2* ap = abase + (kok ? idx2(ak, k) : 0);
#pragma unroll
              for (int r = 0; r < 4; ++r)
                if (a_roff[r] >= 0) cp_async16(as + (unsigned)(kk * LDA + lane + 32 * r) * 16u, kok ? ap + a_roff[r] : abase, kok);
            }
          }
        } else if (kl < 4 || two) {
          const int k = k0 + kl;
          const bool kok = k < K;
          const double2* ap = abase + (kok ? idx2(ak, k) : 0);
#pragma unroll
          for (int j = 0; j < 8; ++j)
            if (a_roff[j] >= 0) cp_async16(as + (unsigned)(kl * LDA + mr + 16 * j) * 16u, kok ? ap + a_roff[j] : abase, kok);
        }
        if (b_ok) {
#pragma unroll
          for (int h2 = 0; h2 < 2; ++h2) {
            const int kk = 2 * pw + h2;
            const int k = k0 + kk;
            if (kk < 4 || two) {
              const bool kok = k < K;
              cp_async16(bs + (unsigned)(kk * LDB + lane) * 16u, b_col + (kok ? idx2(bk, k) : 0), kok);
            }
          }
        }
        mbar_arrive_cp_async(full0 + 8 * stage);
        if (leader) {                                     // slot header, then a releasing arrive
          SlotHdr& h = hdr[stage];
          const bool last = last_seg && k0 + BK >= K;
          h.ctl = (first ? 1 : 0) | (last ? 2 : 0);
          h.nk4 = two ? 2 : 1;
          if (first) {
            TileRec& t = trec[tslot];
            t.mrows = mrows; t.ncols = ncols; t.flags = flags; t.m0 = m0; t.n0 = n0;
            t.c_off = __ldg(&P.c_off) + (long long)ti.batch * __ldg(&P.c_bstride) + (long long)p.t0 * __ldg(&P.c_tstride);
            t.cm = P.cm; t.cn = P.cn;
            h.trec = tslot;
          }
          mbar_arrive(full0 + 8 * stage);
        }
        if (first) { first = false; if (++tslot == rc.ntrec) tslot = 0; }
        if (++stage == kStages) { stage = 0; phase ^= 1; }
      }
    }
  }
  // tell the consumers there is no more work
  mbar_wait(empty0 + 8 * stage, phase ^ 1);
  mbar_arrive_cp_async(full0 + 8 * stage);
  if (leader) { hdr[stage].ctl = 4; mbar_arrive(full0 + 8 * stage); }
  asm volatile("cp.async.wait_all;\n" ::: "memory");
}

// ------------------------------------------------------------------------------------------
// consumer side: one warp tile = MI row groups (8 rows each, 32 rows apart) x NI column groups, accumulators
// acc[i][j] = {re(c0), re(c1), im(c0), im(c1)} of the 8x8 DMMA tile (i, j)
// ------------------------------------------------------------------------------------------
template <int MI, int NI>
__device__ __forceinline__ void consume_k4(double (&acc)[4][4][4], const double2* as, const double2* bs, unsigned mask_n,
                                           unsigned mask_y, unsigned mask_b) {
  double2 af[MI], bf[NI];
  double an[MI];                              // -Im(a) (after the optional conjugation)
#pragma unroll
  for (int i = 0; i < MI; ++i) af[i] = as[i * 32];
#pragma unroll
  for (int j = 0; j < NI; ++j) bf[j] = bs[j * 8];
#pragma unroll
  for (int i = 0; i < MI; ++i) {
    an[i] = xor_hi(af[i].y, mask_n);
    af[i].y = xor_hi(af[i].y, mask_y);
  }
  if (mask_b) {
#pragma unroll
    for (int j = 0; j < NI; ++j) bf[j].y = xor_hi(bf[j].y, mask_b);
  }
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NI; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i].x, bf[j].x);
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NI; ++j) dmma884(acc[i][j][2], acc[i][j][3], af[i].x, bf[j].y);
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NI; ++j) dmma884(acc[i][j][0], acc[i][j][1], an[i], bf[j].y);
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NI; ++j) dmma884(acc[i][j][2], acc[i][j][3], af[i].y, bf[j].x);
}

template <int MI, int NI>
__device__ __forceinline__ void consume_slot(double (&acc)[4][4][4], const double2* as, const double2* bs, int nk4,
                                             unsigned mask_n, unsigned mask_y, unsigned mask_b) {
#pragma unroll 1
  for (int kk = 0; kk < nk4; ++kk) consume_k4<MI, NI>(acc, as + kk * 4 * LDA, bs + kk * 4 * LDB, mask_n, mask_y, mask_b);
}

// registers -> C (two-level addressing); rows (warp + 4 i) * 8 + fr, columns j * 8 + 2 fk + c of the tile.
// One instance for all variants (bounds are run-time, accumulator indices compile-time).  Lane L computes the offset of
// tile column L and of the warp's L-th row once; the lanes then fetch the ones they need by shuffle (one idx2 site each).
__device__ __forceinline__ void store_tile(const double (&acc)[4][4][4], const TileRec& t, double2* C, int warp, int lane) {
  const int fr = lane >> 2, fk = lane & 3;
  const int mrows = t.mrows, ncols = t.ncols;
  double2* cbase = C + t.c_off;
  const bool accum = (t.flags & GWSIG_FLAG_ACCUM) != 0;
  const long long my_col = lane < ncols ? idx2(t.cn, t.n0 + lane) : -1;
  const int my_row_l = warp * 8 + 32 * (lane >> 3) + (lane & 7);
  const long long my_row = my_row_l < mrows ? idx2(t.cm, t.m0 + my_row_l) : -1;
  long long coff[4][2], roff[4];
#pragma unroll
  for (int j = 0; j < 4; ++j)
#pragma unroll
    for (int c = 0; c < 2; ++c) coff[j][c] = __shfl_sync(0xffffffffu, my_col, j * 8 + fk * 2 + c);
#pragma unroll
  for (int i = 0; i < 4; ++i) roff[i] = __shfl_sync(0xffffffffu, my_row, i * 8 + fr);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    if (roff[i] < 0) continue;
    double2* crow = cbase + roff[i];
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
      for (int c = 0; c < 2; ++c)
        if (coff[j][c] >= 0) {
          double2* dst = crow + coff[j][c];
          if (accum) {
            red_add(&dst->x, acc[i][j][c]);
            red_add(&dst->y, acc[i][j][2 + c]);
          } else {
            *dst = make_double2(acc[i][j][c], acc[i][j][2 + c]);
          }
        }
  }
}

#define ZG_VARIANTS(F)                                                                                   \
  case 0: F(1, 1) break;  case 1: F(1, 2) break;  case 2: F(1, 3) break;  case 3: F(1, 4) break;       \
  case 4: F(2, 1) break;  case 5: F(2, 2) break;  case 6: F(2, 3) break;  case 7: F(2, 4) break;       \
  case 8: F(3, 1) break;  case 9: F(3, 2) break;  case 10: F(3, 3) break; case 11: F(3, 4) break;      \
  case 12: F(4, 1) break; case 13: F(4, 2) break; case 14: F(4, 3) break; case 15: F(4, 4) break;

// ------------------------------------------------------------------------------------------
// the kernel: warps 0..3 consume, warps 4..7 produce
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__((kConsumerWarps + kProducerWarps) * 32, 2) zgemm_grouped_dmma(ZgParams p) {
  extern __shared__ double2 zg_smem[];
  double2* As = zg_smem;                             // [kStages][BK][LDA]
  double2* Bs = zg_smem + kStages * BK * LDA;        // [kStages][BK][LDB]
  __shared__ __align__(8) unsigned long long bars[2 * kStages];
  __shared__ SlotHdr hdr[kStages];
  __shared__ TileRec trec[kStages + 1];       // the producers are at most kStages tiles ahead of any consumer
  __shared__ long long next_tile[2];          // tile id broadcast among the producer warps (double buffered)

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned full0 = (unsigned)__cvta_generic_to_shared(&bars[0]);
  const unsigned empty0 = (unsigned)__cvta_generic_to_shared(&bars[kStages]);
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kStages; ++s) { mbar_init(full0 + 8 * s, kProducerWarps * 32 + 1); mbar_init(empty0 + 8 * s, kConsumerWarps); }
  }
  __syncthreads();

  int stage = 0;
  unsigned phase = 0;

  if (warp >= kConsumerWarps) {
    // ================================= PRODUCERS ================================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(kProducerRegs));
    RingCtl rc;
    rc.full0 = full0; rc.empty0 = empty0; rc.hdr = hdr; rc.trec = trec; rc.ntrec = kStages + 1; rc.next_tile = next_tile;
    producer_loop(p, As, Bs, rc, warp - kConsumerWarps, lane);
  } else {
    // ================================= CONSUMERS ================================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(kConsumerRegs));
    const int fr = lane >> 2, fk = lane & 3;         // fragment row / k index of this lane
    double acc[4][4][4];
    int tslot = 0, variant = -1;
    unsigned mask_n = 0x80000000u, mask_y = 0, mask_b = 0;
    while (true) {
      mbar_wait(full0 + 8 * stage, phase);
      const int ctl = hdr[stage].ctl;
      if (ctl & 4) break;
      if (ctl & 1) {
        tslot = hdr[stage].trec;
        const TileRec& t = trec[tslot];
        const int mg = (t.mrows + 7) >> 3, ng = (t.ncols + 7) >> 3;
        const int mi = mg > warp ? (mg - warp + 3) >> 2 : 0;
        variant = mi > 0 ? (mi - 1) * 4 + (ng - 1) : -1;
        const bool conjA = (t.flags & GWSIG_FLAG_CONJ_A) != 0;
        mask_n = conjA ? 0u : 0x80000000u;
        mask_y = conjA ? 0x80000000u : 0u;
        mask_b = (t.flags & GWSIG_FLAG_CONJ_B) ? 0x80000000u : 0u;
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[i][j][c] = 0.0;
      }
      if (variant >= 0) {
        const double2* as = As + stage * BK * LDA + fk * LDA + warp * 8 + fr;
        const double2* bs = Bs + stage * BK * LDB + fk * LDB + fr;
        const int nk4 = hdr[stage].nk4;
#define ZG_F(MI_, NI_) consume_slot<MI_, NI_>(acc, as, bs, nk4, mask_n, mask_y, mask_b);
        switch (variant) { ZG_VARIANTS(ZG_F) default: break; }
#undef ZG_F
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty0 + 8 * stage);
      if (++stage == kStages) { stage = 0; phase ^= 1; }

      // ---- epilogue after the last slot of a tile ----------
      if ((ctl & 2) && variant >= 0) {
        const TileRec& t = trec[tslot];
        store_tile(acc, t, p.C, warp, lane);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// the 3M kernel: warps 0..11 MMA (three product groups of four), 12..15 loaders, 16..19 epilogue
//
//   complex C += A B  as three real products (Karatsuba):  P1 = Ar Br,  P2 = Ai Bi,  P3 = (Ar + Ai)(Br + Bi),
//   re C = P1 - P2,  im C = P3 - P1 - P2.  MMA warp (g, w) accumulates product g for row groups w, w+4, w+8, w+12
//   of the 128-row tile and all (<= 4) column groups: 32 accumulator doubles.  Warp id mod 4 = w is the SM
//   sub-partition, so every sub-partition hosts one warp of each product: three independent DMMA streams per FP64
//   pipe.  conj(A) / conj(B): the sign of Ai / Bi enters the operand sums of P3 (XOR on the integer pipe) and the
//   sign of P2 in the epilogue.  At the end of a tile the MMA warps drop their accumulators into a shared staging
//   buffer [3][128][33] and go straight on with the next tile; the epilogue warps combine the three planes, do the
//   two-level C addressing and store (or red.add) with full-line global accesses in the orientation C is
//   contiguous in.  Register budget per CTA: 12 x 32 x 128 + 4 x 32 x 40 + 4 x 32 x 56 = 61440 = 640 x 96 at launch.
// ------------------------------------------------------------------------------------------
constexpr int kMmaWarps = 12;
constexpr int kEpiWarps = 4;
constexpr int kMmaRegs = 128, kLoaderRegs3 = 40, kEpiRegs = 56;
constexpr int kThreads3 = (kMmaWarps + kProducerWarps + kEpiWarps) * 32;
constexpr int kLaunchRegs3 = 96;                       // what __launch_bounds__(640, 1) gives every thread: 65536 / 640 -> 96
// setmaxnreg only moves registers INSIDE the CTA's launch-time allocation: an inc beyond it waits forever
static_assert(32 * (kMmaWarps * kMmaRegs + kProducerWarps * kLoaderRegs3 + kEpiWarps * kEpiRegs) <= kThreads3 * kLaunchRegs3,
              "setmaxnreg budget exceeds the launch-time register allocation of the CTA");
constexpr int STG_LD = ZG_BN + 1;                      // odd pitch (doubles): conflict-free in both epilogue orientations
constexpr int kTrec3 = kStages + 3;                    // loaders <= kStages tiles ahead of the MMA warps, epilogue one behind

template <int MI, int NI>
__device__ __forceinline__ void mma3_k4(double (&acc)[4][4][2], const double2* as, const double2* bs, int grp, unsigned sa,
                                        unsigned sb) {
  double2 af[MI], bf[NI];
  double a[MI], b[NI];
#pragma unroll
  for (int i = 0; i < MI; ++i) af[i] = as[i * 32];
#pragma unroll
  for (int j = 0; j < NI; ++j) bf[j] = bs[j * 8];
  if (grp == 0) {
#pragma unroll
    for (int i = 0; i < MI; ++i) a[i] = af[i].x;
#pragma unroll
    for (int j = 0; j < NI; ++j) b[j] = bf[j].x;
  } else if (grp == 1) {
#pragma unroll
    for (int i = 0; i < MI; ++i) a[i] = af[i].y;
#pragma unroll
    for (int j = 0; j < NI; ++j) b[j] = bf[j].y;
  } else {
#pragma unroll
    for (int i = 0; i < MI; ++i) a[i] = af[i].x + xor_hi(af[i].y, sa);
#pragma unroll
    for (int j = 0; j < NI; ++j) b[j] = bf[j].x + xor_hi(bf[j].y, sb);
  }
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NI; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
}

template <int MI, int NI>
__device__ __forceinline__ void mma3_slot(double (&acc)[4][4][2], const double2* as, const double2* bs, int nk4, int grp,
                                          unsigned sa, unsigned sb) {
#pragma unroll 1
  for (int kk = 0; kk < nk4; ++kk) mma3_k4<MI, NI>(acc, as + kk * 4 * LDA, bs + kk * 4 * LDB, grp, sa, sb);
}

struct __align__(8) StageCtl {      // handshake MMA warps -> epilogue warps
  int trec;                          // tile record of the staged tile
  int ctl;                           // 4: no more tiles
};

__global__ void __launch_bounds__(kThreads3, 1) zgemm_grouped_dmma3m(ZgParams p) {
  extern __shared__ double2 zg_smem[];
  double2* As = zg_smem;                             // [kStages][BK][LDA]
  double2* Bs = zg_smem + kStages * BK * LDA;        // [kStages][BK][LDB]
  double* Stg = reinterpret_cast<double*>(zg_smem + kStages * BK * (LDA + LDB));   // [3][ZG_BM][STG_LD]
  __shared__ __align__(8) unsigned long long bars[2 * kStages + 2];
  __shared__ SlotHdr hdr[kStages];
  __shared__ TileRec trec[kTrec3];
  __shared__ long long next_tile[2];
  __shared__ StageCtl sctl;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned full0 = (unsigned)__cvta_generic_to_shared(&bars[0]);
  const unsigned empty0 = (unsigned)__cvta_generic_to_shared(&bars[kStages]);
  const unsigned stg_full = (unsigned)__cvta_generic_to_shared(&bars[2 * kStages]);
  const unsigned stg_empty = (unsigned)__cvta_generic_to_shared(&bars[2 * kStages + 1]);
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kStages; ++s) { mbar_init(full0 + 8 * s, kProducerWarps * 32 + 1); mbar_init(empty0 + 8 * s, kMmaWarps); }
    mbar_init(stg_full, kMmaWarps);
    mbar_init(stg_empty, kEpiWarps);
  }
  __syncthreads();

  if (warp >= kMmaWarps + kProducerWarps) {
    // ================================= EPILOGUE WARPS ===========================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(kEpiRegs));
    const int ew = warp - kMmaWarps - kProducerWarps;
    unsigned tpar = 0;
    while (true) {
      mbar_wait(stg_full, tpar);
      if (sctl.ctl & 4) break;
      const TileRec& t = trec[sctl.trec];
      const int mrows = t.mrows, ncols = t.ncols;
      const bool accum = (t.flags & GWSIG_FLAG_ACCUM) != 0;
      const bool flip = ((t.flags & GWSIG_FLAG_CONJ_A) != 0) != ((t.flags & GWSIG_FLAG_CONJ_B) != 0);   // sign of Ai Bi
      double2* cbase = p.C + t.c_off;
      const int row = 32 * ew + lane;
      const long long my_roff = row < mrows ? idx2(t.cm, t.m0 + row) : -1;
      const long long my_coff = lane < ncols ? idx2(t.cn, t.n0 + lane) : -1;
      const double* s1 = Stg, *s2 = Stg + ZG_BM * STG_LD, *s3 = Stg + 2 * ZG_BM * STG_LD;
      if (t.cm.lo == 1) {
        // C contiguous along m (X, Y): lane <-> row, walk the columns; 32 lanes write 32 consecutive rows
        const double* q1 = s1 + row * STG_LD, *q2 = s2 + row * STG_LD, *q3 = s3 + row * STG_LD;
        for (int c = 0; c < ncols; ++c) {
          const long long coff = __shfl_sync(0xffffffffu, my_coff, c);
          if (my_roff >= 0) {
            const double p1 = q1[c], p2 = flip ? -q2[c] : q2[c], p3 = q3[c];
            const double re = p1 - p2, im = p3 - p1 - p2;
            double2* dst = cbase + my_roff + coff;
            if (accum) { red_add(&dst->x, re); red_add(&dst->y, im); }
            else *dst = make_double2(re, im);
          }
        }
      } else {
        // C contiguous along n (Sigma blocks): lane <-> column, walk this warp's 32 rows
        const int rend = min(32, mrows - 32 * ew);
        for (int rr = 0; rr < rend; ++rr) {
          const long long roff = __shfl_sync(0xffffffffu, my_roff, rr);
          if (my_coff >= 0) {
            const int r = 32 * ew + rr;
            const double p1 = s1[r * STG_LD + lane], p2r = s2[r * STG_LD + lane], p3 = s3[r * STG_LD + lane];
            const double p2 = flip ? -p2r : p2r;
            const double re = p1 - p2, im = p3 - p1 - p2;
            double2* dst = cbase + roff + my_coff;
            if (accum) { red_add(&dst->x, re); red_add(&dst->y, im); }
            else *dst = make_double2(re, im);
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(stg_empty);
      tpar ^= 1;
    }
  } else if (warp >= kMmaWarps) {
    // ================================= LOADER WARPS =============================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(kLoaderRegs3));
    RingCtl rc;
    rc.full0 = full0; rc.empty0 = empty0; rc.hdr = hdr; rc.trec = trec; rc.ntrec = kTrec3; rc.next_tile = next_tile;
    producer_loop(p, As, Bs, rc, warp - kMmaWarps, lane);
  } else {
    // ================================= MMA WARPS ================================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(kMmaRegs));
    const int grp = warp >> 2, wq = warp & 3;
    const int fr = lane >> 2, fk = lane & 3;
    double acc[4][4][2];
    int stage = 0, tslot = 0, variant = -1, mi = 0, ng = 0;
    unsigned phase = 0, tpar = 0, sa = 0, sb = 0;
    while (true) {
      mbar_wait(full0 + 8 * stage, phase);
      const int ctl = hdr[stage].ctl;
      if (ctl & 4) break;
      if (ctl & 1) {
        tslot = hdr[stage].trec;
        const TileRec& t = trec[tslot];
        const int mg = (t.mrows + 7) >> 3;
        ng = (t.ncols + 7) >> 3;
        mi = mg > wq ? (mg - wq + 3) >> 2 : 0;
        variant = mi > 0 ? (mi - 1) * 4 + (ng - 1) : -1;
        sa = (t.flags & GWSIG_FLAG_CONJ_A) ? 0x80000000u : 0u;
        sb = (t.flags & GWSIG_FLAG_CONJ_B) ? 0x80000000u : 0u;
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }
      }
      if (variant >= 0) {
        const double2* as = As + stage * BK * LDA + fk * LDA + wq * 8 + fr;
        const double2* bs = Bs + stage * BK * LDB + fk * LDB + fr;
        const int nk4 = hdr[stage].nk4;
#define ZG_F(MI_, NI_) mma3_slot<MI_, NI_>(acc, as, bs, nk4, grp, sa, sb);
        switch (variant) { ZG_VARIANTS(ZG_F) default: break; }
#undef ZG_F
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty0 + 8 * stage);
      if (++stage == kStages) { stage = 0; phase ^= 1; }

      if (ctl & 2) {
        // ---- hand the accumulators of this product to the epilogue warps -----------------------
        mbar_wait(stg_empty, tpar ^ 1);                 // staging buffer free (passes at once for the first tile)
        double* sg = Stg + grp * (ZG_BM * STG_LD) + (wq * 8 + fr) * STG_LD + 2 * fk;
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
          for (int j = 0; j < 4; ++j)
            if (i < mi && j < ng) {
              sg[i * 32 * STG_LD + j * 8] = acc[i][j][0];
              sg[i * 32 * STG_LD + j * 8 + 1] = acc[i][j][1];
            }
        if (warp == 0 && lane == 0) { sctl.trec = tslot; sctl.ctl = 0; }
        __syncwarp();
        if (lane == 0) mbar_arrive(stg_full);
        tpar ^= 1;
      }
    }
    // no more tiles: release the epilogue warps
    mbar_wait(stg_empty, tpar ^ 1);
    if (warp == 0 && lane == 0) sctl.ctl = 4;
    __syncwarp();
    if (lane == 0) mbar_arrive(stg_full);
  }
}

// ------------------------------------------------------------------------------------------
// reference engine: same plan, one thread per output element, plain DFMA, no shared memory
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) zgemm_grouped_reference(ZgParams p) {
  for (long long tile = blockIdx.x; tile < p.total_tiles; tile += gridDim.x) {
    const TileInfo ti = decode_tile(p, tile);
    const gwsig_problem& P = p.prob[ti.prob];
    const bool conjA = (P.flags & GWSIG_FLAG_CONJ_A) != 0, conjB = (P.flags & GWSIG_FLAG_CONJ_B) != 0;
    const long long a_boff = (long long)ti.batch * P.a_bstride + (long long)p.t0 * P.a_tstride;
    const long long b_boff = (long long)ti.batch * P.b_bstride + (long long)p.t0 * P.b_tstride;
    double2* cbase = p.C + P.c_off + (long long)ti.batch * P.c_bstride + (long long)p.t0 * P.c_tstride;
    int n0, ncols;
    zg_ntile(P.N, P.tiles_n, ti.tn, n0, ncols);
    const int m0 = ti.tm * ZG_BM, mrows = min(ZG_BM, P.M - m0);
    for (int e = threadIdx.x; e < mrows * ncols; e += blockDim.x) {
      int m = m0 + e / ncols, n = n0 + e % ncols;
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
      if (P.flags & GWSIG_FLAG_ACCUM) { atomicAdd(&dst->x, sr); atomicAdd(&dst->y, si); }
      else *dst = make_double2(sr, si);
    }
  }
}

}  // namespace

namespace {
struct LaunchCfg { bool ok3 = false, ok4 = false; int occ4 = 1; };
LaunchCfg g_cfg[64];                 // per device: the shared-memory opt-in is a per-device function attribute
std::mutex g_cfg_mu;
}  // namespace

cudaError_t zg_launch(int engine, const ZgParams& p, int num_sms, cudaStream_t stream) {
  if (p.total_tiles <= 0) return cudaSuccess;
  if (engine == 1) {
    long long grid = p.total_tiles < 65535LL * 16 ? p.total_tiles : 65535LL * 16;
    zgemm_grouped_reference<<<(unsigned)grid, 256, 0, stream>>>(p);
    return cudaGetLastError();
  }
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lk(g_cfg_mu);
  LaunchCfg& cfg = g_cfg[dev];
  if (engine == 0) {
    // 3M kernel: 12 MMA + 4 loader + 4 epilogue warps, one persistent CTA per SM
    constexpr int smem = kStages * BK * (LDA + LDB) * (int)sizeof(double2) + 3 * ZG_BM * STG_LD * (int)sizeof(double);
    if (!cfg.ok3) {
      e = cudaFuncSetAttribute(zgemm_grouped_dmma3m, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
      if (e != cudaSuccess) return e;
      cfg.ok3 = true;
    }
    long long grid = num_sms;
    if (grid > p.total_tiles) grid = p.total_tiles;
    if (grid < 1) return cudaSuccess;
    zgemm_grouped_dmma3m<<<(unsigned)grid, kThreads3, smem, stream>>>(p);
    return cudaGetLastError();
  }
  // 4M kernel: 4 consumer + 4 producer warps, 128 registers / thread at launch (2 CTAs / SM), redistributed 200 / 56
  constexpr int smem = kStages * BK * (LDA + LDB) * (int)sizeof(double2);
  constexpr int threads = (kConsumerWarps + kProducerWarps) * 32;
  if (!cfg.ok4) {
    e = cudaFuncSetAttribute(zgemm_grouped_dmma, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(zgemm_grouped_dmma, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&cfg.occ4, zgemm_grouped_dmma, threads, smem);
    if (e != cudaSuccess) return e;
    if (cfg.occ4 < 1) cfg.occ4 = 1;
    cfg.ok4 = true;
  }
  long long grid = (long long)num_sms * cfg.occ4;
  if (grid > p.total_tiles) grid = p.total_tiles;
  if (grid < 1) return cudaSuccess;
  zgemm_grouped_dmma<<<(unsigned)grid, threads, smem, stream>>>(p);
  return cudaGetLastError();
}
