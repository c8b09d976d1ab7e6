// C = A B for 17 x 17 complex matrices in shared memory, by ONE WARP on the FP64 tensor cores
// (mma.sync.m8n8k4.f64), the scheme of block_back.cu: the 16 x 16 x 16 core is 2 x 2 output tiles x 4 k-steps x 4
// real products = 64 DMMA with no padding; the border (k = 16 term, last row, last column, corner) runs on the
// SIMT pipe from the same fragments.  The whole product is formed in registers before anything is stored, so
// C may be A or B.  Used by sancho_rubio.cu for the eight n x n products of a decimation pass.
#pragma once
#include "block_ops.cuh"

namespace negf {
namespace blk {

__device__ __forceinline__ void dmma884(double (&d)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d[0]), "+d"(d[1])
               : "d"(a), "d"(b));
}

// A, B, C row-major with leading dimensions lda, ldb, ldc (in elements).  All 32 lanes call it.
__device__ __forceinline__ void cgemm17_warp(const c64* A, int lda, const c64* B, int ldb, c64* C, int ldc,
                                             int lane) {
  const unsigned full = 0xffffffffu;
  const int g = lane >> 2, q4 = lane & 3;
  double cre[2][2][2], cim[2][2][2];
#pragma unroll
  for (int mt = 0; mt < 2; ++mt)
#pragma unroll
    for (int nt = 0; nt < 2; ++nt) cre[mt][nt][0] = cre[mt][nt][1] = cim[mt][nt][0] = cim[mt][nt][1] = 0.0;
  c64 colp[2] = {make_double2(0.0, 0.0), make_double2(0.0, 0.0)};   // C[8 mt + g][16], partial over q4
  c64 rowp[2] = {make_double2(0.0, 0.0), make_double2(0.0, 0.0)};   // C[16][8 nt + g], partial over q4
  c64 cornp = make_double2(0.0, 0.0);                               // C[16][16], partial over q4
#pragma unroll
  for (int ks = 0; ks < 4; ++ks) {
    const int kr = 4 * ks + q4;
    const c64 b0 = B[kr * ldb + g], b1 = B[kr * ldb + 8 + g];       // B fragments, nt = 0, 1
    const c64 b16 = B[kr * ldb + 16];
    const c64 a16 = A[16 * lda + kr];                               // A[16][kr]
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
      const c64 av = A[(8 * mt + g) * lda + kr];
      const double nai = -av.y;
      dmma884(cre[mt][0], av.x, b0.x);
      dmma884(cre[mt][0], nai, b0.y);
      dmma884(cim[mt][0], av.x, b0.y);
      dmma884(cim[mt][0], av.y, b0.x);
      dmma884(cre[mt][1], av.x, b1.x);
      dmma884(cre[mt][1], nai, b1.y);
      dmma884(cim[mt][1], av.x, b1.y);
      dmma884(cim[mt][1], av.y, b1.x);
      cfma(colp[mt], av, b16);
    }
    cfma(rowp[0], a16, b0);
    cfma(rowp[1], a16, b1);
    cfma(cornp, a16, b16);
  }
  // k = 16 terms and the quad reductions of the border sums
  auto quad_sum = [&](c64 v) {
    v.x += __shfl_xor_sync(full, v.x, 1);
    v.y += __shfl_xor_sync(full, v.y, 1);
    v.x += __shfl_xor_sync(full, v.x, 2);
    v.y += __shfl_xor_sync(full, v.y, 2);
    return v;
  };
  const c64 b1616 = B[16 * ldb + 16];
  const c64 acorner = A[16 * lda + 16];
  c64 colv[2], rowv[2];
#pragma unroll
  for (int mt = 0; mt < 2; ++mt) {
    const c64 ar16 = A[(8 * mt + g) * lda + 16];                    // A[8 mt + g][16]
#pragma unroll
    for (int nt = 0; nt < 2; ++nt)
#pragma unroll
      for (int i2 = 0; i2 < 2; ++i2) {
        const c64 bl = B[16 * ldb + 8 * nt + 2 * q4 + i2];
        cre[mt][nt][i2] = fma(ar16.x, bl.x, cre[mt][nt][i2]);
        cre[mt][nt][i2] = fma(-ar16.y, bl.y, cre[mt][nt][i2]);
        cim[mt][nt][i2] = fma(ar16.x, bl.y, cim[mt][nt][i2]);
        cim[mt][nt][i2] = fma(ar16.y, bl.x, cim[mt][nt][i2]);
      }
    colv[mt] = quad_sum(colp[mt]);
    cfma(colv[mt], ar16, b1616);
  }
#pragma unroll
  for (int nt = 0; nt < 2; ++nt) {
    rowv[nt] = quad_sum(rowp[nt]);
    cfma(rowv[nt], acorner, B[16 * ldb + 8 * nt + g]);
  }
  c64 cornv = quad_sum(cornp);
  cfma(cornv, acorner, b1616);
  __syncwarp();                                                     // every lane has read A and B
#pragma unroll
  for (int mt = 0; mt < 2; ++mt)
#pragma unroll
    for (int nt = 0; nt < 2; ++nt)
#pragma unroll
      for (int i2 = 0; i2 < 2; ++i2)
        C[(8 * mt + g) * ldc + 8 * nt + 2 * q4 + i2] = make_double2(cre[mt][nt][i2], cim[mt][nt][i2]);
  if (q4 == 0) {
    C[g * ldc + 16] = colv[0];
    C[(8 + g) * ldc + 16] = colv[1];
    C[16 * ldc + g] = rowv[0];
    C[16 * ldc + 8 + g] = rowv[1];
  }
  if (lane == 0) C[16 * ldc + 16] = cornv;
  __syncwarp();
}

}  // namespace blk
}  // namespace negf
