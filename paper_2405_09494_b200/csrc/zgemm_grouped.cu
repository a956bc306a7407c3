// Grouped / ragged batched complex-FP64 GEMM on the FP64 tensor pipe (sm_100a).
//
// Serves the three contraction stages of the GW self-energy (Algorithm 4 lines 5, 7, 8 of
// arXiv 2405.09494).  Descriptors: include/gwsig_plan.h.  Design: DESIGN.md section 5.
//
//  * persistent CTAs, dynamic tile scheduler over a cost-sorted tile list (heaviest problems first)
//  * warp-specialised, two warpgroups per CTA: FOUR PRODUCER WARPS do all index arithmetic (two-level ragged
//    addressing) and stage operands global -> shared with 16-byte cp.async (one complex128 per copy; ragged
//    edges are zero-filled), signalling a STAGES-deep ring of mbarriers (cp.async.mbarrier.arrive.noinc);
//    the FOUR CONSUMER WARPS only wait, load fragments and issue DMMA, then release the slot.
//    setmaxnreg moves the producers' registers to the consumers (48 / 208), two CTAs are resident per SM, so
//    every SM sub-partition holds two consumer warps working on independent tiles (one tile's epilogue
//    overlaps the other's main loop)
//  * ragged edges cost no tensor-pipe time: a consumer warp skips the 8-row / 8-column groups of its
//    warp tile that lie outside the problem
//  * shared tiles are k-major with leading dimension = 2 (mod 8) complex elements: the
//    one-double2-per-lane fragment loads of mma.m8n8k4.f64 are bank-conflict free
//  * complex product = 4 real DMMA per 8x8x4 tile: re += ar*br, im += ar*bi, re += (-ai)*bi, im += ai*br,
//    issued in two passes over the warp tile so that dependent DMMAs are MI*NI*2 instructions apart
#include <cuda_runtime.h>
#include <stdint.h>

#include "zgemm_grouped.cuh"

namespace {

__device__ __forceinline__ long long idx2(const gwsig_idx2& d, int i) {
  if (d.div == GWSIG_NODIV) return (long long)i * d.lo;
  int q = i / d.div;
  return (long long)q * d.hi + (long long)(i - q * d.div) * d.lo;
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
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_LOOP:\n\t"
      "mbarrier.try_wait.parity.shared.b64 p, [%0], %1;\n\t"
      "@p bra WAIT_DONE;\n\t"
      "bra WAIT_LOOP;\n\t"
      "WAIT_DONE:\n\t}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
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
  long long local = tile - __ldg(&P.tile_begin);
  int tn_ = __ldg(&P.tiles_n);
  int per = __ldg(&P.tiles_m) * tn_;
  TileInfo t;
  t.prob = lo;
  t.batch = (int)(local / per);
  int r = (int)(local - (long long)t.batch * per);
  t.tm = r / tn_;
  t.tn = r - t.tm * tn_;
  return t;
}

// ------------------------------------------------------------------------------------------
// tensor-core engine, warp-specialised
//   consumer warpgroup (warps 0..3): WGM x WGN warps, each owning an (8 MI) x (8 NI) complex tile
//   producer warpgroup (warps 4..7): owns the tile scheduler (one atomicAdd per tile) and every descriptor
//   read; tells the consumers what a pipeline slot holds through a small header in shared memory.
//   Within a slot of BK = 8 k-rows producer warp w stages rows 2w, 2w+1 (A contiguous along m) or the
//   tile rows = w (mod 4) (A contiguous along k).
// ------------------------------------------------------------------------------------------
struct SlotHdr {
  int ctl;            // bit0: first slot of a tile, bit1: last slot of a tile, bit2: no more work
  int nk4;            // k4-steps of this slot that hold data (1 or 2)
  int trec;           // index of the tile record (valid when bit0)
  int pad_;
};
struct __align__(16) TileRec {   // what the consumers need to know about a tile (written by the producer)
  int m_rem, n_rem;   // M - m0, N - n0
  int flags, pad_;
  long long c_off;    // element offset of C(m = 0, n = 0) incl. batch / tau offsets
  int m0, n0;
  gwsig_idx2 cm, cn;
};

constexpr int kProducerWarps = 4;
constexpr int kProducerRegs = 48;
constexpr int kConsumerRegs = 208;

__device__ __forceinline__ double flip_sign(double x) {      // integer pipe: keeps the FP64 pipe for DMMA
  return __hiloint2double(__double2hiint(x) ^ (int)0x80000000, __double2loint(x));
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;\n" ::"r"(id), "r"(nthreads) : "memory");
}

template <int MI, int NI, int WGM, int WGN, int STAGES>
__global__ void __launch_bounds__((WGM* WGN + kProducerWarps) * 32, 2) zgemm_grouped_dmma(ZgParams p) {
  static_assert(WGM * WGN == 4, "one consumer warpgroup");
  constexpr int BK = 8;
  constexpr int BM = WGM * MI * 8, BN = WGN * NI * 8;
  constexpr int NCW = WGM * WGN;                     // consumer warps
  constexpr int LDA = BM + 2, LDB = BN + 2;          // = 2 (mod 8): conflict-free fragment loads
  constexpr int RA = (BM + 31) / 32, RB = (BN + 31) / 32;
  constexpr int RAK = BM / 16;                       // rows per lane and producer warp in the k-major A mapping
  static_assert(LDA % 8 == 2 && LDB % 8 == 2 && BM % 16 == 0, "layout");

  extern __shared__ double2 zg_smem[];
  double2* As = zg_smem;                             // [STAGES][BK][LDA]
  double2* Bs = zg_smem + STAGES * BK * LDA;         // [STAGES][BK][LDB]
  __shared__ __align__(8) unsigned long long bars[2 * STAGES];
  __shared__ SlotHdr hdr[STAGES];
  __shared__ TileRec trec[STAGES + 1];        // the producers are at most STAGES tiles ahead of any consumer
  __shared__ long long next_tile[2];          // tile id broadcast among the producer warps (double buffered)

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned full0 = (unsigned)__cvta_generic_to_shared(&bars[0]);
  const unsigned empty0 = (unsigned)__cvta_generic_to_shared(&bars[STAGES]);
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) { mbar_init(full0 + 8 * s, kProducerWarps * 32 + 1); mbar_init(empty0 + 8 * s, NCW); }
  }
  __syncthreads();

  int stage = 0;
  unsigned phase = 0;

  if (warp >= NCW) {
    // ================================= PRODUCERS ================================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(kProducerRegs));
    const int pw = warp - NCW;                          // producer warp 0..3
    const unsigned as0 = (unsigned)__cvta_generic_to_shared(As), bs0 = (unsigned)__cvta_generic_to_shared(Bs);
    int tslot = 0, tbuf = 0;
    while (true) {
      if (pw == 0 && lane == 0) next_tile[tbuf] = (long long)atomicAdd(p.counter, 1ULL);
      named_bar_sync(1, kProducerWarps * 32);
      const long long tile = next_tile[tbuf];
      tbuf ^= 1;
      if (tile >= p.total_tiles) break;
      const TileInfo ti = decode_tile(p, tile);
      const gwsig_problem& P = p.prob[ti.prob];
      const int M = __ldg(&P.M), N = __ldg(&P.N), flags = __ldg(&P.flags);
      const int m0 = ti.tm * BM, n0 = ti.tn * BN;
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
        const double2* b_col[RB];
        bool b_ok[RB];
        {
          const gwsig_idx2 bn = S.bn;
          const double2* bbase = p.B + __ldg(&S.b_off) + b_boff;
#pragma unroll
          for (int r = 0; r < RB; ++r) {
            int nl = lane + 32 * r;
            b_ok[r] = nl < BN && n0 + nl < N;
            b_col[r] = bbase + (b_ok[r] ? idx2(bn, n0 + nl) : 0);
          }
        }
        auto publish = [&](int k0) {                      // producer warp 0, lane 0: slot header, then a releasing arrive
          if (pw == 0 && lane == 0) {
            SlotHdr& h = hdr[stage];
            const bool last = last_seg && k0 + BK >= K;
            h.ctl = (first ? 1 : 0) | (last ? 2 : 0);
            h.nk4 = (K - k0 > 4) ? 2 : 1;
            if (first) {
              TileRec& t = trec[tslot];
              t.m_rem = M - m0; t.n_rem = N - n0; t.flags = flags; t.m0 = m0; t.n0 = n0;
              t.c_off = __ldg(&P.c_off) + (long long)ti.batch * __ldg(&P.c_bstride) + (long long)p.t0 * __ldg(&P.c_tstride);
              t.cm = P.cm; t.cn = P.cn;
              h.trec = tslot;
            }
            mbar_arrive(full0 + 8 * stage);
          }
          if (first) { first = false; if (++tslot == STAGES + 1) tslot = 0; }
        };
        // B rows of this warp: kk = 2 pw, 2 pw + 1 (both A layouts)
        auto stage_b = [&](int k0, unsigned bs) {
#pragma unroll
          for (int h2 = 0; h2 < 2; ++h2) {
            const int kk = 2 * pw + h2;
            const int k = k0 + kk;
            const bool kok = k < K;
            const long long kb = kok ? idx2(bk, k) : 0;
#pragma unroll
            for (int r = 0; r < RB; ++r)
              if (lane + 32 * r < BN)
                cp_async16(bs + (unsigned)(kk * LDB + lane + 32 * r) * 16u, b_col[r] + kb, kok && b_ok[r]);
          }
        };
        if (!kmajor) {
          // ---- A contiguous along m: lane <-> rows lane, lane+32 of the tile; this warp stages k-rows 2 pw, 2 pw + 1 ----
          const gwsig_idx2 am = S.am;
          const double2* a_row[RA];
          bool a_ok[RA];
#pragma unroll
          for (int r = 0; r < RA; ++r) {
            int ml = lane + 32 * r;
            a_ok[r] = ml < BM && m0 + ml < M;
            a_row[r] = abase + (a_ok[r] ? idx2(am, m0 + ml) : 0);
          }
          for (int k0 = 0; k0 < K; k0 += BK) {
            mbar_wait(empty0 + 8 * stage, phase ^ 1);
            const unsigned as = as0 + (unsigned)(stage * BK * LDA) * 16u;
            const unsigned bs = bs0 + (unsigned)(stage * BK * LDB) * 16u;
#pragma unroll
            for (int h2 = 0; h2 < 2; ++h2) {
              const int kk = 2 * pw + h2;
              const int k = k0 + kk;
              const bool kok = k < K;
              const long long ka = kok ? idx2(ak, k) : 0;
#pragma unroll
              for (int r = 0; r < RA; ++r)
                if (lane + 32 * r < BM)
                  cp_async16(as + (unsigned)(kk * LDA + lane + 32 * r) * 16u, a_row[r] + ka, kok && a_ok[r]);
            }
            stage_b(k0, bs);
            mbar_arrive_cp_async(full0 + 8 * stage);
            publish(k0);
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
        } else {
          // ---- A contiguous along k: lane <-> (k = lane & 7, tile rows 4 (lane >> 3) + pw + 16 j) ----
          const gwsig_idx2 am = S.am;
          const int kl = lane & 7, mr = 4 * (lane >> 3) + pw;
          int a_roff[RAK];                              // element offsets inside a tile stay < 2^31 (checked by the plan)
#pragma unroll
          for (int j = 0; j < RAK; ++j) {
            int m = m0 + mr + 16 * j;
            a_roff[j] = m < M ? (int)idx2(am, m) : -1;
          }
          for (int k0 = 0; k0 < K; k0 += BK) {
            mbar_wait(empty0 + 8 * stage, phase ^ 1);
            const unsigned as = as0 + (unsigned)(stage * BK * LDA) * 16u;
            const unsigned bs = bs0 + (unsigned)(stage * BK * LDB) * 16u;
            {
              const int k = k0 + kl;
              const bool kok = k < K;
              const double2* ap = abase + (kok ? idx2(ak, k) : 0);
#pragma unroll
              for (int j = 0; j < RAK; ++j) {
                const bool ok = kok && a_roff[j] >= 0;
                cp_async16(as + (unsigned)(kl * LDA + mr + 16 * j) * 16u, ok ? ap + a_roff[j] : abase, ok);
              }
            }
            stage_b(k0, bs);
            mbar_arrive_cp_async(full0 + 8 * stage);
            publish(k0);
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
        }
      }
    }
    // tell the consumers there is no more work
    mbar_wait(empty0 + 8 * stage, phase ^ 1);
    mbar_arrive_cp_async(full0 + 8 * stage);
    if (pw == 0 && lane == 0) { hdr[stage].ctl = 4; mbar_arrive(full0 + 8 * stage); }
    asm volatile("cp.async.wait_all;\n" ::: "memory");
  } else {
    // ================================= CONSUMERS ================================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(kConsumerRegs));
    const int wm0 = (warp / WGN) * (MI * 8), wn0 = (warp % WGN) * (NI * 8);
    const int fr = lane >> 2, fk = lane & 3;         // fragment row / k index of this lane
    double cre[MI][NI][2], cim[MI][NI][2];
    int tslot = 0, mi_eff = 0, ni_eff = 0;           // 8-row / 8-column groups of the warp tile that hold data
    bool conjA = false, conjB = false;
    while (true) {
      mbar_wait(full0 + 8 * stage, phase);
      const SlotHdr& h = hdr[stage];
      const int ctl = h.ctl;
      if (ctl & 4) break;
      if (ctl & 1) {
        tslot = h.trec;
        const TileRec& t = trec[tslot];
        mi_eff = min(MI, max(0, (t.m_rem - wm0 + 7) >> 3));
        ni_eff = min(NI, max(0, (t.n_rem - wn0 + 7) >> 3));
        if (mi_eff == 0 || ni_eff == 0) mi_eff = ni_eff = 0;
        conjA = (t.flags & GWSIG_FLAG_CONJ_A) != 0; conjB = (t.flags & GWSIG_FLAG_CONJ_B) != 0;
#pragma unroll
        for (int i = 0; i < MI; ++i)
#pragma unroll
          for (int j = 0; j < NI; ++j) { cre[i][j][0] = cre[i][j][1] = 0.0; cim[i][j][0] = cim[i][j][1] = 0.0; }
      }
      if (mi_eff > 0) {
        const double2* as = As + stage * BK * LDA + wm0 + fr;
        const double2* bs = Bs + stage * BK * LDB + wn0 + fr;
        const int nk4 = h.nk4;
#pragma unroll
        for (int kk = 0; kk < BK / 4; ++kk) {
          if (kk < nk4) {
            double2 af[MI], bf[NI];
            double an[MI];                            // -Im(a) (after the optional conjugation)
#pragma unroll
            for (int i = 0; i < MI; ++i)
              if (i < mi_eff) af[i] = as[(kk * 4 + fk) * LDA + i * 8];
#pragma unroll
            for (int j = 0; j < NI; ++j)
              if (j < ni_eff) bf[j] = bs[(kk * 4 + fk) * LDB + j * 8];
#pragma unroll
            for (int i = 0; i < MI; ++i) {
              const double neg = flip_sign(af[i].y);
              an[i] = conjA ? af[i].y : neg;
              af[i].y = conjA ? neg : af[i].y;
            }
            if (conjB) {
#pragma unroll
              for (int j = 0; j < NI; ++j) bf[j].y = flip_sign(bf[j].y);
            }
            // four passes over the warp tile: dependent DMMAs are >= mi_eff*ni_eff instructions apart
#pragma unroll
            for (int i = 0; i < MI; ++i)
              if (i < mi_eff) {
#pragma unroll
                for (int j = 0; j < NI; ++j)
                  if (j < ni_eff) dmma884(cre[i][j][0], cre[i][j][1], af[i].x, bf[j].x);
              }
#pragma unroll
            for (int i = 0; i < MI; ++i)
              if (i < mi_eff) {
#pragma unroll
                for (int j = 0; j < NI; ++j)
                  if (j < ni_eff) dmma884(cim[i][j][0], cim[i][j][1], af[i].x, bf[j].y);
              }
#pragma unroll
            for (int i = 0; i < MI; ++i)
              if (i < mi_eff) {
#pragma unroll
                for (int j = 0; j < NI; ++j)
                  if (j < ni_eff) dmma884(cre[i][j][0], cre[i][j][1], an[i], bf[j].y);
              }
#pragma unroll
            for (int i = 0; i < MI; ++i)
              if (i < mi_eff) {
#pragma unroll
                for (int j = 0; j < NI; ++j)
                  if (j < ni_eff) dmma884(cim[i][j][0], cim[i][j][1], af[i].y, bf[j].x);
              }
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(empty0 + 8 * stage);
      if (++stage == STAGES) { stage = 0; phase ^= 1; }

      // ---- epilogue after the last slot of a tile: registers -> C (two-level addressing) ----------
      if ((ctl & 2) && mi_eff > 0) {
        const TileRec& t = trec[tslot];
        const int m_rem = t.m_rem, n_rem = t.n_rem, m0 = t.m0, n0 = t.n0;
        const gwsig_idx2 cm = t.cm, cn = t.cn;
        double2* cbase = p.C + t.c_off;
        const bool accum = (t.flags & GWSIG_FLAG_ACCUM) != 0;
        long long cn_off[NI][2];
#pragma unroll
        for (int j = 0; j < NI; ++j)
#pragma unroll
          for (int c = 0; c < 2; ++c) {
            int nl = wn0 + j * 8 + fk * 2 + c;
            cn_off[j][c] = nl < n_rem ? idx2(cn, n0 + nl) : -1;
          }
#pragma unroll
        for (int i = 0; i < MI; ++i) {
          int ml = wm0 + i * 8 + fr;
          if (ml < m_rem) {
            double2* crow = cbase + idx2(cm, m0 + ml);
#pragma unroll
            for (int j = 0; j < NI; ++j)
#pragma unroll
              for (int c = 0; c < 2; ++c)
                if (cn_off[j][c] >= 0) {
                  double2* dst = crow + cn_off[j][c];
                  double2 v = make_double2(cre[i][j][c], cim[i][j][c]);
                  if (accum) { double2 o = *dst; v.x += o.x; v.y += o.y; }
                  *dst = v;
                }
          }
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// reference engine: same plan, one thread per output element, plain DFMA, no shared memory
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) zgemm_grouped_reference(ZgParams p, int BM, int BN) {
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

template <int MI, int NI, int WGM, int WGN, int STAGES>
cudaError_t launch_dmma(const ZgParams& p, int num_sms, cudaStream_t stream) {
  auto kern = zgemm_grouped_dmma<MI, NI, WGM, WGN, STAGES>;
  constexpr int BM = WGM * MI * 8, BN = WGN * NI * 8;
  constexpr int smem = STAGES * 8 * ((BM + 2) + (BN + 2)) * (int)sizeof(double2);
  constexpr int threads = (WGM * WGN + kProducerWarps) * 32;
  static bool configured = false;
  static int occ = 1;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, threads, smem);
    if (e != cudaSuccess) return e;
    if (occ < 1) occ = 1;
    configured = true;
  }
  long long grid = (long long)num_sms * occ;
  if (grid > p.total_tiles) grid = p.total_tiles;
  if (grid < 1) return cudaSuccess;
  kern<<<(unsigned)grid, threads, smem, stream>>>(p);
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
  const ZgTile ts = zg_tile_shape(shape_class);
  if (engine == 1) {
    long long grid = p.total_tiles < 65535LL * 16 ? p.total_tiles : 65535LL * 16;
    zgemm_grouped_reference<<<(unsigned)grid, 256, 0, stream>>>(p, ts.bm, ts.bn);
    return cudaGetLastError();
  }
  // 4 consumer + 4 producer warps, 128 registers / thread at launch (2 CTAs / SM), redistributed 208 / 48 by setmaxnreg.
  // class 0: warp tiles 32x32 complex (2x2 warps -> 64x64); class 1: warp tiles 32x16 (2x2 warps -> 64x32)
  if (shape_class == 1) return launch_dmma<4, 2, 2, 2, 6>(p, num_sms, stream);
  return launch_dmma<4, 4, 2, 2, 5>(p, num_sms, stream);
}
