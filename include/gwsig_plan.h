/* gwsig_plan.h -- descriptors of the grouped / ragged batched complex GEMM that all three
 * contraction stages (Algorithm 4 lines 5, 7, 8) and the block-basis unfold
 * (Eq. 28) are lowered to.  Plain C structs: the host plan writes them, the CUDA
 * engine reads them, gwsig_plan_get() hands them to the host-logic tests.
 *
 * One PROBLEM is   C[M x N] (+)= sum over its SEGMENTS s of  op(A_s)[M x K_s] . B_s[K_s x N],
 * repeated for nbatch batch entries (tau).  Every index of every operand is addressed by a
 * two-level rule   offset(i) = (i / div) * hi + (i % div) * lo   (complex elements), which covers
 * compound indices such as m = (Q, i), n = (tau, b), k = (Q', b) of ragged irrep blocks.
 * div = GWSIG_NODIV means single level: offset(i) = i * lo.
 *
 * element address of A for (batch, m, k) in segment s:
 *     A_base + s.a_off + batch * a_bstride + t0 * a_tstride + am(m) + ak(k)
 * (same pattern for B with bk, bn and for C with cm, cn); t0 is the first tau of the chunk being
 * processed, passed at launch, so one descriptor set serves every tau chunk of equal length.
 */
#ifndef GWSIG_PLAN_H
#define GWSIG_PLAN_H

#include <stdint.h>

#define GWSIG_NODIV 0x7fffffff

#define GWSIG_FLAG_CONJ_A 1      /* use conj(A) (stage 1: V^{k,k-q} = conj-transpose of V2)          */
#define GWSIG_FLAG_ACCUM 2       /* C += instead of C =  (stage 3 accumulates over pushes)           */
#define GWSIG_FLAG_A_KMAJOR 4    /* A is contiguous along k (loader hint only)                        */
#define GWSIG_FLAG_CONJ_B 8      /* use conj(B) (unfold step 2: T . O^dagger)                         */

typedef struct {
  int64_t hi, lo;
  int32_t div, pad_;
} gwsig_idx2; /* 24 bytes */

typedef struct {
  int64_t a_off, b_off;
  gwsig_idx2 am, ak, bk, bn;
  int32_t K, pad_;
} gwsig_seg; /* 120 bytes */

typedef struct {
  int64_t c_off;
  int64_t a_bstride, b_bstride, c_bstride; /* per batch entry (tau inside the chunk)              */
  int64_t a_tstride, b_tstride, c_tstride; /* per unit of t0 (first tau of the chunk)             */
  int64_t tile_begin;                      /* first linear tile id of this problem                */
  gwsig_idx2 cm, cn;
  int32_t M, N;
  int32_t seg_begin, seg_count;
  int32_t nbatch, flags;
  int32_t tiles_m, tiles_n;
} gwsig_problem; /* 144 bytes */

#endif /* GWSIG_PLAN_H */
