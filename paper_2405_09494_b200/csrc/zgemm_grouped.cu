// Grouped / ragged batched complex-FP64 GEMM on the FP64 tensor pipe (sm_100a).
//
// TWO tensor-core kernels share the tile scheduler and the descriptors:
//   zgemm_grouped_dmma3m (engine 3; the default engine runs stages 1 and 2 on it): Karatsuba / "3M" complex product -- three
//       REAL products P1 = Ar Br, P2 = Ai Bi, P3 = (Ar+Ai)(Br+Bi),  re = P1 - P2,  im = P3 - P1 - P2  (25 % fewer DMMA than 4M);
//       two CTAs per SM of 8 MMA warps (one 8-row group of a 64-row tile each) + 2 loader warps; details above the kernel
//   zgemm_grouped_dmma   (engine 2; the default engine runs stage 3 and the Eq. 28 unfold on it): the conventional
//       four-product kernel (engine v3 of round 1), described below.
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

// two-level index i -> (i / div) * hi + (i % div) * lo.  The quotient comes from a single-precision reciprocal with a one-step
// fix-up (exact for i, div < 2^22, which the plan checks): ten inline instructions instead of the 40-instruction integer
// division, which used to sit on the loaders' per-tile critical path and, with a two-level k index (stage 3), in every k-row.
__device__ __forceinline__ long long idx2(const gwsig_idx2& d, int i) {
  if (d.div == GWSIG_NODIV) return (long long)i * d.lo;
  const int div = d.div;
  int q = __float2int_rz(__int2float_rn(i) * __frcp_rn(__int2float_rn(div)));
  int r = i - q * div;
  if (r < 0) { --q; r += div; }
  else if (r >= div) { ++q; r -= div; }
  return (long long)q * d.hi + (long long)r * d.lo;
}

// 16-byte asynchronous copy global -> shared; !valid writes 16 zero bytes and reads nothing (the ignore-src predicate form: one
// LDGSTS; with a variable src-size operand ptxas spends six more instructions per copy on the size arithmetic)
__device__ __forceinline__ void cp_async16(unsigned smem_dst, const void* gmem_src, bool valid) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.eq.b32 p, %2, 0;\n\tcp.async.cg.shared.global [%0], [%1], 16, p;\n\t}\n" ::"r"(smem_dst), "l"(gmem_src),
               "r"((int)valid)
               : "memory");
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
      "mbarrier.try_wait.parity.shared.b64 p, [%1], %2, 0x989680;\n\t"     // suspend-time hint: sleep in hardware, do not spin
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
// Column map of the B fragment.  A DMMA hands lane (fr, fk) the accumulator columns 2 fk, 2 fk + 1 of an 8-column group; were
// those the tile's columns 2 fk, 2 fk + 1, one store instruction (fixed c) would write 16-byte pieces 32 bytes apart: half
// sectors, twice the L2 write slots of the payload.  The lane that feeds B column n of the group therefore loads TILE column
// zg_bcol(n), so that accumulator column 2 fk is tile column fk and 2 fk + 1 is tile column 4 + ((fk + 1) & 3): a store
// instruction then covers four adjacent complex numbers (64 contiguous bytes) per row.  (The odd distance between the tile
// columns of a lane pair keeps the 16-byte fragment loads bank-conflict free with LDB = 2 mod 8.)
__device__ __forceinline__ int zg_bcol(int n) { return (n & 1) ? 4 + (((n >> 1) + 1) & 3) : (n >> 1); }
__device__ __forceinline__ int zg_ccol(int fk, int c) { return c ? 4 + ((fk + 1) & 3) : fk; }     // tile column (within the group) of accumulator c

__device__ __forceinline__ void red_add(double* addr, double v) {
  asm volatile("red.global.add.f64 [%0], %1;\n" ::"l"(addr), "d"(v) : "memory");
}
__device__ __forceinline__ void st_pred(double2* addr, double re, double im, bool on) {      // predicated 16-byte store: no branch
  asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %3, 0;\n\t@q st.global.v2.f64 [%0], {%1, %2};\n\t}\n" ::"l"(addr), "d"(re), "d"(im), "r"((int)on)
               : "memory");
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

struct __align__(16) SlotHdr {
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

// registers -> C (two-level addressing); rows (warp + 4 i) * 8 + fr, columns j * 8 + zg_ccol(fk, c) of the tile.
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
    for (int c = 0; c < 2; ++c) coff[j][c] = __shfl_sync(0xffffffffu, my_col, j * 8 + zg_ccol(fk, c));
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
        const double2* bs = Bs + stage * BK * LDB + fk * LDB + zg_bcol(fr);
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
// the 3M kernel: warps 0..7 MMA, warps 8..9 loaders; two CTAs per SM
//
//   complex C += A B  as three real products (Karatsuba):  P1 = Ar Br,  P2 = Ai Bi,  P3 = (Ar + Ai)(Br + Bi),
//   re C = P1 - P2,  im C = P3 - P1 - P2:  3 real DMMA per complex 8x8x4 block instead of 4.
//   MMA warp w owns row group w (8 rows) of the 64-row tile and all (<= 4) column groups, all three products: 24 accumulator
//   doubles; it stores its own rows at the end of a tile (8 complex numbers per lane) and goes straight on.  conj(A) /
//   conj(B) flip the sign of Ai / Bi on the integer pipe (XOR) before the operand sums.
//   Two CTAs per SM (20 warps x 96 registers = the whole register file, no setmaxnreg): every SM sub-partition hosts two MMA
//   warps of each CTA, and the two CTAs are at unrelated points of unrelated tiles, so one CTA's barrier round trips,
//   fragment-load latency, tile switches and stores are covered by the other's DMMA stream (measured: sixteen MMA warps of
//   ONE CTA run in lock step and leave the pipe idle at every step and slot boundary).
//   Two loader warps per CTA feed a ring of kStages3 = 4 slots of BK3 = 16 k-rows (four k4 steps per barrier round trip,
//   100 KB of shared memory per CTA).  The plan lays X and Y out so that every operand is contiguous along its tile dimension.
// ------------------------------------------------------------------------------------------
constexpr int kMmaWarps = ZG_BM3 / 8;     // 8: one row group each
constexpr int kLoaderWarps3 = 2;
constexpr int LDA3 = ZG_BM3 + 2;          // = 2 (mod 8): conflict-free fragment loads
static_assert(LDA3 % 8 == 2, "layout");
constexpr int kThreads3 = (kMmaWarps + kLoaderWarps3) * 32;
constexpr int BK3 = 16;
constexpr int kStages3 = 4;
constexpr int kTrec3 = kStages3 + 2;
constexpr int kChunk3 = 4;             // consecutive tile ids a CTA takes per scheduler fetch
constexpr unsigned kFullCount3 = 32 + 1;      // the 32 lanes of the slot's owner warp (cp.async-triggered arrive) + its lane 0's expect_tx
static_assert(kStages3 % kLoaderWarps3 == 0, "loader warp lw owns ring stages lw, lw + kLoaderWarps3, ...");

__device__ __forceinline__ void bulk_g2s(unsigned smem_dst, const void* gmem_src, unsigned bytes, unsigned bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_dst),
               "l"(gmem_src), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.expect_tx.shared.b64 st, [%0], %1;\n\t}\n" ::"r"(bar), "r"(bytes) : "memory");
}

// step a two-level index by one: offset(i + 1) from offset(i) without a division
struct KStep {
  long long off, wrap;       // current offset; what to add when the fast index wraps (hi - div * lo)
  long long lo;
  int r, div;
};
__device__ __forceinline__ KStep kstep_init(const gwsig_idx2& d, int k) {
  KStep s;
  s.lo = d.lo; s.div = d.div;
  if (d.div == GWSIG_NODIV) { s.r = 0; s.off = (long long)k * d.lo; s.wrap = 0; }
  else { const int q = k / d.div; s.r = k - q * d.div; s.off = (long long)q * d.hi + (long long)s.r * d.lo; s.wrap = d.hi - (long long)d.div * d.lo; }
  return s;
}
__device__ __forceinline__ void kstep_next(KStep& s) {        // branch-free: div = GWSIG_NODIV (INT_MAX) never wraps
  const bool w = ++s.r == s.div;
  s.off += s.lo + (w ? s.wrap : 0);
  s.r = w ? 0 : s.r;
}
__device__ __forceinline__ void cp_async16_sz(unsigned smem_dst, const void* gmem_src, unsigned bytes) {   // bytes = 0: zero-fill, no read
  cp_async16(smem_dst, gmem_src, bytes != 0u);
}

// per loader warp: the descriptor of the problem its tile ids are running through and the segment being staged, copied to
// shared memory ONCE per problem (per segment for multi-segment problems).  Tile ids run through a problem n-tile by n-tile, so
// what used to be a chain of dependent L2 round trips per tile (bucket table, forward scan, problem, segment) is paid once per
// problem; per tile the fields come from shared memory.
struct __align__(16) LoaderCache {
  gwsig_problem P;     // 144 bytes
  gwsig_seg S;         // 120 bytes
  long long pad_;
};
static_assert(sizeof(gwsig_problem) == 144 && sizeof(gwsig_seg) == 120, "descriptor layout");

// Loader warp lw OWNS the ring slots whose global index is lw (mod kLoaderWarps3): every loader warp walks the same tile /
// segment / slot sequence but only fills its own slots, so it has kLoaderWarps3 slot times for one slot's address
// arithmetic.  Operands move as one 16-byte cp.async per element, lane <-> tile row / column (tile rows lane, lane + 32);
// with ZgParams::use_bulk an operand whose tile dimension is ONE contiguous run (single-level index with unit stride: X / Y
// and W rows in stage 2, V2 rows in stage 3) moves as one bulk copy per k-row instead, issued by lane 0 (UBLKCP).
template <bool kBulk>
__device__ __forceinline__ void loader3(const ZgParams& p, double2* As, double2* Bs, unsigned full0, unsigned empty0, SlotHdr* hdr,
                                        TileRec* trec, long long* next_tile, LoaderCache& lc, int lw, int lane) {
  const unsigned as0 = (unsigned)__cvta_generic_to_shared(As), bs0 = (unsigned)__cvta_generic_to_shared(Bs);
  const bool leader = lw == 0 && lane == 0;
  int stage = 0, tslot = 0, tbuf = 0;
  unsigned phase = 0;             // parity of the ring round of the next slot (all loader warps count alike)
  int gslot = 0;                  // global slot index modulo kLoaderWarps3
  long long pre = 0;
  if (leader) pre = (long long)atomicAdd(p.counter, 1ULL);
  long long c_begin = 0, c_end = 0;                                                // tile id range of the cached problem (empty at first)
  int c_prob = 0, c_tn = 1, c_per = 1;
  int key_prob = -1, key_batch = -1, key_tm = -1;                                  // what pa[] / sza[] were computed for
  const double2* pa[2] = {nullptr, nullptr};
  unsigned sza[2] = {0u, 0u};
  while (true) {
    // tiles are taken kChunk3 consecutive ids at a time: neighbours belong to the same problem (n fastest), so their
    // descriptor loads hit L1 and the chain of dependent L2 round trips is paid once per chunk, not once per tile
    if (leader) next_tile[tbuf] = pre;
    named_bar_sync(1, kLoaderWarps3 * 32);
    const long long chunk0 = next_tile[tbuf] * kChunk3;
    tbuf ^= 1;
    if (chunk0 >= p.total_tiles) break;
    if (leader) pre = (long long)atomicAdd(p.counter, 1ULL);        // lands while this chunk is being staged
    for (long long tile = chunk0; tile < chunk0 + kChunk3 && tile < p.total_tiles; ++tile) {
      // consecutive tile ids run through one problem n-tile by n-tile: the problem's fields are decoded when the id leaves the
      // cached problem's range only (bucket table, forward scan and the descriptor are a chain of dependent loads)
      if (tile < c_begin || tile >= c_end) {
        int lo = __ldg(&p.bucket[tile >> ZG_BUCKET_SHIFT]);
        while (lo + 1 < p.nprob && __ldg(&p.prob[lo + 1].tile_begin) <= tile) ++lo;
        __syncwarp();                                   // every lane is done with the previous problem's copy
        if (lane < 18) reinterpret_cast<long long*>(&lc.P)[lane] = __ldg(reinterpret_cast<const long long*>(&p.prob[lo]) + lane);
        __syncwarp();
        if (lc.P.seg_count == 1) {
          if (lane < 15) reinterpret_cast<long long*>(&lc.S)[lane] = __ldg(reinterpret_cast<const long long*>(&p.seg[lc.P.seg_begin]) + lane);
          __syncwarp();
        }
        c_prob = lo;
        c_tn = lc.P.tiles_n;
        c_per = lc.P.tiles_m * c_tn;
        c_begin = lc.P.tile_begin;
        c_end = c_begin + (long long)lc.P.nbatch * c_per;
        key_prob = -1;
      }
      const gwsig_problem& P = lc.P;
      TileInfo ti;
      {
        const unsigned local = (unsigned)(tile - c_begin);
        ti.prob = c_prob;
        ti.batch = (int)(local / (unsigned)c_per);
        const unsigned r = local - (unsigned)ti.batch * (unsigned)c_per;
        ti.tm = (int)(r / (unsigned)c_tn);
        ti.tn = (int)(r - (unsigned)ti.tm * (unsigned)c_tn);
      }
      const int M = P.M, N = P.N, flags = P.flags;
      const int m0 = ti.tm * ZG_BM3;
      int n0, ncols;
      zg_ntile(N, c_tn, ti.tn, n0, ncols);
      const int mrows = min(ZG_BM3, M - m0);
      const long long a_boff = (long long)ti.batch * P.a_bstride + (long long)p.t0 * P.a_tstride;
      const long long b_boff = (long long)ti.batch * P.b_bstride + (long long)p.t0 * P.b_tstride;
      const int seg_begin = P.seg_begin, nseg = P.seg_count;
      // the A row pointers of a one-segment problem depend on (problem, batch entry, m-tile) only: kept across its n-tiles
      const bool a_cached = !kBulk && nseg == 1 && c_prob == key_prob && ti.batch == key_batch && ti.tm == key_tm;
      bool first = true;
      for (int s = 0; s < nseg; ++s) {
        if (nseg > 1) {                                 // multi-segment problem (split-K lists): stage this segment's descriptor
          __syncwarp();
          if (lane < 15) reinterpret_cast<long long*>(&lc.S)[lane] = __ldg(reinterpret_cast<const long long*>(&p.seg[seg_begin + s]) + lane);
          __syncwarp();
        }
        const gwsig_seg& S = lc.S;
        const int K = S.K;
        if (K == 0) continue;
        const bool last_seg = s == nseg - 1;
        const int nslots = (K + BK3 - 1) / BK3;
        const int j0 = (lw - gslot + kLoaderWarps3) % kLoaderWarps3;       // this warp's first slot of the segment
        if (j0 < nslots) {
          const bool a_row = kBulk && S.am.div == GWSIG_NODIV && S.am.lo == 1, b_row = kBulk && S.bn.div == GWSIG_NODIV && S.bn.lo == 1;
          const double2* abase = p.A + S.a_off + a_boff + (a_row ? m0 : 0);
          const double2* bbase = p.B + S.b_off + b_boff + (b_row ? n0 : 0);
          // per-lane source pointers of tile rows lane, lane + 32 and tile column lane; lanes outside the tile point at the
          // operand base and copy zero bytes (cp.async zero-fills: no branch in the slot loop, nothing read)
          unsigned szb;
          if (!a_cached) {
#pragma unroll
            for (int j = 0; j < 2; ++j) {
              const bool v = !a_row && lane + 32 * j < mrows;
              pa[j] = abase + (v ? idx2(S.am, m0 + lane + 32 * j) : 0);
              sza[j] = v ? 16u : 0u;
            }
            key_prob = nseg == 1 ? c_prob : -1; key_batch = ti.batch; key_tm = ti.tm;
          }
          const bool vb = !b_row && lane < ncols;
          const double2* pb = bbase + (vb ? idx2(S.bn, n0 + lane) : 0);
          szb = vb ? 16u : 0u;
          const gwsig_idx2 ak = S.ak, bk = S.bk;
          for (int j = j0; j < nslots; j += kLoaderWarps3) {
            const int k0 = j * BK3;
            const int st = (stage + j) % kStages3;
            const unsigned ph = phase ^ (unsigned)(((stage + j) / kStages3) & 1);     // ring round of this slot
            const unsigned bar_full = full0 + 8 * st;
            mbar_wait(empty0 + 8 * st, ph ^ 1);
            const unsigned as = as0 + (unsigned)(st * BK3 * LDA3) * 16u, bs = bs0 + (unsigned)(st * BK3 * LDB) * 16u;
            const int nkv = min(BK3, K - k0);                   // k-rows that hold data
            const int nk4 = (nkv + 3) >> 2;
            const bool firstslot = first && j == 0;
            if (lane == 0) {                                    // slot header, then the releasing arrive that announces the bulk bytes
              SlotHdr& h = hdr[st];
              const bool last = last_seg && j == nslots - 1;
              h.ctl = (firstslot ? 1 : 0) | (last ? 2 : 0);
              h.nk4 = nk4;
              if (firstslot) {
                TileRec& t = trec[tslot];
                t.mrows = mrows; t.ncols = ncols; t.flags = flags; t.m0 = m0; t.n0 = n0;
                t.c_off = P.c_off + (long long)ti.batch * P.c_bstride + (long long)p.t0 * P.c_tstride;
                t.cm = P.cm; t.cn = P.cn;
                h.trec = tslot;
              }
              mbar_arrive_expect_tx(bar_full, (unsigned)(nkv * ((a_row ? mrows : 0) + (b_row ? ncols : 0)) * 16));
            }
            if (!a_row && !b_row && ak.div == GWSIG_NODIV && bk.div == GWSIG_NODIV) {
              // stages 1 and 2: both k indices are single-level, three pointers advance by constant strides
              const double2* qa0 = pa[0] + (long long)k0 * ak.lo;
              const double2* qa1 = pa[1] + (long long)k0 * ak.lo;
              const double2* qb = pb + (long long)k0 * bk.lo;
              unsigned arow = as + (unsigned)lane * 16u, brow = bs + (unsigned)lane * 16u;
              const long long sa_ = ak.lo, sb_ = bk.lo;
#pragma unroll 4
              for (int kk = 0; kk < 4 * nk4; ++kk) {
                const bool kok = kk < nkv;
                cp_async16_sz(arow, qa0, kok ? sza[0] : 0u);
                cp_async16_sz(arow + 32u * 16u, qa1, kok ? sza[1] : 0u);
                cp_async16_sz(brow, qb, kok ? szb : 0u);
                arow += (unsigned)LDA3 * 16u; brow += (unsigned)LDB * 16u;
                if (kok) { qa0 += sa_; qa1 += sa_; qb += sb_; }       // (never step past the last row: the pointers stay valid)
              }
              mbar_arrive_cp_async(bar_full);
              continue;
            }
            if (!a_row && !b_row && ak.div == bk.div) {
              // stage 3 (and every pair of operands cut from the same [P'][b][.] layout): A and B step through k with the SAME
              // fast-index period, so one (quotient, remainder) walk serves both offsets
              KStep ka = kstep_init(ak, k0);
              long long offb = ak.div == GWSIG_NODIV ? (long long)k0 * bk.lo : (long long)(k0 / ak.div) * bk.hi + (long long)(k0 % ak.div) * bk.lo;
              const long long wrapb = ak.div == GWSIG_NODIV ? 0 : bk.hi - (long long)bk.div * bk.lo;
              unsigned arow = as + (unsigned)lane * 16u, brow = bs + (unsigned)lane * 16u;
#pragma unroll 4
              for (int kk = 0; kk < 4 * nk4; ++kk) {
                const bool kok = kk < nkv;
                cp_async16_sz(arow, pa[0] + ka.off, kok ? sza[0] : 0u);
                cp_async16_sz(arow + 32u * 16u, pa[1] + ka.off, kok ? sza[1] : 0u);
                cp_async16_sz(brow, pb + offb, kok ? szb : 0u);
                arow += (unsigned)LDA3 * 16u; brow += (unsigned)LDB * 16u;
                const bool w = ++ka.r == ka.div;
                ka.off += ka.lo + (w ? ka.wrap : 0);
                offb += bk.lo + (w ? wrapb : 0);
                ka.r = w ? 0 : ka.r;
              }
              mbar_arrive_cp_async(bar_full);
              continue;
            }
            KStep ka = kstep_init(ak, k0), kb = kstep_init(bk, k0);
            if (!a_row && !b_row) {
              // the common path: three cp.async per k-row and lane, no branches
              unsigned arow = as + (unsigned)lane * 16u, brow = bs + (unsigned)lane * 16u;
#pragma unroll 4
              for (int kk = 0; kk < 4 * nk4; ++kk) {
                const bool kok = kk < nkv;                      // rows of the last k4 step beyond K are zero-filled
                cp_async16_sz(arow, pa[0] + ka.off, kok ? sza[0] : 0u);
                cp_async16_sz(arow + 32u * 16u, pa[1] + ka.off, kok ? sza[1] : 0u);
                cp_async16_sz(brow, pb + kb.off, kok ? szb : 0u);
                arow += (unsigned)LDA3 * 16u; brow += (unsigned)LDB * 16u;
                kstep_next(ka); kstep_next(kb);
              }
            } else {
              for (int kk = 0; kk < 4 * nk4; ++kk) {
                const bool kok = kk < nkv;
                const unsigned arow = as + (unsigned)(kk * LDA3) * 16u, brow = bs + (unsigned)(kk * LDB) * 16u;
                if (a_row) {
                  if (kok) { if (lane == 0) bulk_g2s(arow, abase + ka.off, (unsigned)mrows * 16u, bar_full); }
                  else for (int m = lane; m < mrows; m += 32) As[(st * BK3 + kk) * LDA3 + m] = make_double2(0.0, 0.0);
                } else {
                  cp_async16_sz(arow + (unsigned)lane * 16u, pa[0] + ka.off, kok ? sza[0] : 0u);
                  cp_async16_sz(arow + (unsigned)(lane + 32) * 16u, pa[1] + ka.off, kok ? sza[1] : 0u);
                }
                if (b_row) {
                  if (kok) { if (lane == 0) bulk_g2s(brow, bbase + kb.off, (unsigned)ncols * 16u, bar_full); }
                  else if (lane < ncols) Bs[(st * BK3 + kk) * LDB + lane] = make_double2(0.0, 0.0);
                } else {
                  cp_async16_sz(brow + (unsigned)lane * 16u, pb + kb.off, kok ? szb : 0u);
                }
                kstep_next(ka); kstep_next(kb);
              }
            }
            mbar_arrive_cp_async(bar_full);    // this lane's arrival, once its cp.async (if any) have landed; its zero stores precede it
          }
        }
        if (first) { first = false; if (++tslot == kTrec3) tslot = 0; }
        const int adv = stage + nslots;
        phase ^= (unsigned)((adv / kStages3) & 1);
        stage = adv % kStages3;
        gslot = (gslot + nslots) % kLoaderWarps3;
      }
    }
  }
  // the slot after the last one carries the end mark: its owner tells the MMA warps there is no more work
  if (lw == gslot) {
    mbar_wait(empty0 + 8 * stage, phase ^ 1);
    if (lane == 0) { hdr[stage].ctl = 4; mbar_arrive_expect_tx(full0 + 8 * stage, 0); }
    mbar_arrive_cp_async(full0 + 8 * stage);
  }
  asm volatile("cp.async.wait_all;\n" ::: "memory");
}

// the k4 steps of one slot for one MMA warp: NI column groups, products P1, P2, P3 in acc[j][0..2].  The fragment registers
// double as the P1 / P2 operands (sign flips in place), only the operand sums of P3 need registers of their own, so the warp
// stays inside the 96 registers a 20-warp CTA gives every thread; P1 is issued before the operand sums so that the FP64 adds
// queue behind the warp's own DMMAs, and the other three warps of the sub-partition cover the fragment-load latency.
template <int NI, bool kFlip>
__device__ __forceinline__ void mma3_slot(double (&acc)[4][3][2], const double2* as, const double2* bs, int nk4, unsigned sa, unsigned sb) {
#pragma unroll 1
  for (int kk = 0; kk < nk4; ++kk) {
    double2 af = as[kk * 4 * LDA3], bf[NI];
#pragma unroll
    for (int j = 0; j < NI; ++j) bf[j] = bs[kk * 4 * LDB + j * 8];
    if (kFlip) {                       // conj(A) / conj(B): stage 2 has neither, and five XORs per 12 DMMA are issue slots
      af.y = xor_hi(af.y, sa);
#pragma unroll
      for (int j = 0; j < NI; ++j) bf[j].y = xor_hi(bf[j].y, sb);
    }
#pragma unroll
    for (int j = 0; j < NI; ++j) dmma884(acc[j][0][0], acc[j][0][1], af.x, bf[j].x);
    const double asum = af.x + af.y;
    double bsum[NI];
#pragma unroll
    for (int j = 0; j < NI; ++j) bsum[j] = bf[j].x + bf[j].y;
#pragma unroll
    for (int j = 0; j < NI; ++j) dmma884(acc[j][1][0], acc[j][1][1], af.y, bf[j].y);
#pragma unroll
    for (int j = 0; j < NI; ++j) dmma884(acc[j][2][0], acc[j][2][1], asum, bsum[j]);
  }
}

// accumulators of one row group -> C: re = P1 - P2, im = P3 - P1 - P2; lane (fr, fk) holds row fr, columns 8 j + zg_ccol(fk, c).
// Lane L computes the offset of tile column L once (32 bits: checked by the plan); the eight shuffles that hand every lane
// its own column offsets are issued back to back, and the stores carry no branch but their own predicate: with K = n_alpha
// <= 26 in stage 1 a tile is two slots of DMMA work, and this epilogue is what the MMA warps spend the rest of their time in.
__device__ __forceinline__ void store_rows3(const double (&acc)[4][3][2], const TileRec& t, double2* C, int rg, int lane) {
  const int fr = lane >> 2, fk = lane & 3;
  const int ncols = t.ncols;
  const int my_col = lane < ncols ? (int)idx2(t.cn, t.n0 + lane) : 0;
  const int row = rg * 8 + fr;
  const bool rok = row < t.mrows;
  double2* rowp = C + t.c_off + (rok ? idx2(t.cm, t.m0 + row) : 0);
  int coff[4][2];
#pragma unroll
  for (int j = 0; j < 4; ++j)
#pragma unroll
    for (int c = 0; c < 2; ++c) coff[j][c] = __shfl_sync(0xffffffffu, my_col, j * 8 + zg_ccol(fk, c));
  if (t.flags & GWSIG_FLAG_ACCUM) {
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
      for (int c = 0; c < 2; ++c)
        if (rok && j * 8 + zg_ccol(fk, c) < ncols) {
          double2* dst = rowp + coff[j][c];
          red_add(&dst->x, acc[j][0][c] - acc[j][1][c]);
          red_add(&dst->y, acc[j][2][c] - acc[j][0][c] - acc[j][1][c]);
        }
  } else {
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const double re = acc[j][0][c] - acc[j][1][c], im = acc[j][2][c] - acc[j][0][c] - acc[j][1][c];
        st_pred(rowp + coff[j][c], re, im, rok && j * 8 + zg_ccol(fk, c) < ncols);
      }
  }
}

template <bool kBulk>
__global__ void __launch_bounds__(kThreads3, 2) zgemm_grouped_dmma3m(ZgParams p) {
  extern __shared__ double2 zg_smem[];
  double2* As = zg_smem;                              // [kStages3][BK3][LDA3]
  double2* Bs = zg_smem + kStages3 * BK3 * LDA3;      // [kStages3][BK3][LDB]
  __shared__ __align__(8) unsigned long long bars[2 * kStages3];
  __shared__ SlotHdr hdr[kStages3];
  __shared__ TileRec trec[kTrec3];
  __shared__ long long next_tile[2];
  __shared__ LoaderCache lcache[kLoaderWarps3];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned full0 = (unsigned)__cvta_generic_to_shared(&bars[0]);
  const unsigned empty0 = (unsigned)__cvta_generic_to_shared(&bars[kStages3]);
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < kStages3; ++s) { mbar_init(full0 + 8 * s, kFullCount3); mbar_init(empty0 + 8 * s, kMmaWarps); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();

  if (warp >= kMmaWarps) {
    loader3<kBulk>(p, As, Bs, full0, empty0, hdr, trec, next_tile, lcache[warp - kMmaWarps], warp - kMmaWarps, lane);
  } else {
    // ================================= MMA WARPS ================================================
    const int fr = lane >> 2, fk = lane & 3;
    double acc[4][3][2];
    int stage = 0, tslot = 0, ng = 0;
    bool active = false;
    unsigned phase = 0, sa = 0, sb = 0;
    while (true) {
      mbar_wait(full0 + 8 * stage, phase);
      const int4 h4 = *reinterpret_cast<const int4*>(&hdr[stage]);      // ctl, nk4, trec in one 16-byte load
      const int ctl = h4.x;
      if (ctl & 4) break;
      if (ctl & 1) {
        tslot = h4.z;
        const TileRec& t = trec[tslot];
        active = warp * 8 < t.mrows;
        ng = (t.ncols + 7) >> 3;
        sa = (t.flags & GWSIG_FLAG_CONJ_A) ? 0x80000000u : 0u;
        sb = (t.flags & GWSIG_FLAG_CONJ_B) ? 0x80000000u : 0u;
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
          for (int q = 0; q < 3; ++q) { acc[j][q][0] = 0.0; acc[j][q][1] = 0.0; }
      }
      if (active) {
        const double2* as = As + stage * BK3 * LDA3 + fk * LDA3 + warp * 8 + fr;
        const double2* bs = Bs + stage * BK3 * LDB + fk * LDB + zg_bcol(fr);
        const int nk4 = h4.y;
        if (sa | sb) {
          if (ng == 4) mma3_slot<4, true>(acc, as, bs, nk4, sa, sb);
          else if (ng == 3) mma3_slot<3, true>(acc, as, bs, nk4, sa, sb);
          else if (ng == 2) mma3_slot<2, true>(acc, as, bs, nk4, sa, sb);
          else mma3_slot<1, true>(acc, as, bs, nk4, sa, sb);
        } else {
          if (ng == 4) mma3_slot<4, false>(acc, as, bs, nk4, sa, sb);
          else if (ng == 3) mma3_slot<3, false>(acc, as, bs, nk4, sa, sb);
          else if (ng == 2) mma3_slot<2, false>(acc, as, bs, nk4, sa, sb);
          else mma3_slot<1, false>(acc, as, bs, nk4, sa, sb);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty0 + 8 * stage);
      if (++stage == kStages3) { stage = 0; phase ^= 1; }
      if ((ctl & 2) && active) store_rows3(acc, trec[tslot], p.C, warp, lane);
    }
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
    const int m0 = ti.tm * p.bm, mrows = min(p.bm, P.M - m0);
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
struct LaunchCfg { bool ok3 = false, ok4 = false; int occ3 = 1, occ4 = 1; };
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
  if (engine == 3) {
    // 3M kernel: 8 MMA + 2 loader warps, two persistent CTAs per SM (96 registers per thread), 64-row tiles
    constexpr int smem = kStages3 * BK3 * (LDA3 + LDB) * (int)sizeof(double2);
    if (p.bm != ZG_BM3) return cudaErrorInvalidValue;
    if (!cfg.ok3) {
      for (int b = 0; b < 2; ++b) {          // both instantiations: without / with the bulk-copy loader path (option bulk_copies)
        const void* fn = b ? (const void*)zgemm_grouped_dmma3m<true> : (const void*)zgemm_grouped_dmma3m<false>;
        e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        if (e != cudaSuccess) return e;
      }
      e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&cfg.occ3, zgemm_grouped_dmma3m<false>, kThreads3, smem);
      if (e != cudaSuccess) return e;
      if (cfg.occ3 < 1) cfg.occ3 = 1;
      cfg.ok3 = true;
    }
    long long nchunks = (p.total_tiles + kChunk3 - 1) / kChunk3;
    long long grid = (long long)num_sms * cfg.occ3;
    if (grid > nchunks) grid = nchunks;
    if (grid < 1) return cudaSuccess;
    if (p.use_bulk) zgemm_grouped_dmma3m<true><<<(unsigned)grid, kThreads3, smem, stream>>>(p);
    else zgemm_grouped_dmma3m<false><<<(unsigned)grid, kThreads3, smem, stream>>>(p);
    return cudaGetLastError();
  }
  // 4M kernel: 4 consumer + 4 producer warps, 128 registers / thread at launch (2 CTAs / SM), redistributed 200 / 56
  constexpr int smem = kStages * BK * (LDA + LDB) * (int)sizeof(double2);
  constexpr int threads = (kConsumerWarps + kProducerWarps) * 32;
  if (p.bm != ZG_BM) return cudaErrorInvalidValue;
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
