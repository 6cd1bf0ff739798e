// Tile-packed operator format of a level ("TP-CSR") -- the HBM layout the solve-phase row kernels
// stream.  Shared by the packer (amg_pack.cu) and the kernels (amg_kernels.cuh).
//
// A level's rows are cut into tiles of consecutive rows (boundaries on aggregate starts).  Each
// tile owns ONE contiguous, 16-byte aligned blob, fetched by a single bulk-async copy (TMA):
//
//   section A  val   f64[nnz]      matrix values, row-major, ascending columns within a row
//              col   u16[nnz]      LOCAL column: < nrows -> row r0+col of this tile,
//                                  >= nrows -> entry (col - nrows) of the tile's halo list
//              roff  u16[nrows+1]  local row offsets into val / col
//              halo  i32[nhalo]    level index of every distinct out-of-tile column, ascending
//              aoff  u16[nagg+1]   local first row of every aggregate of the tile (restriction)
//   section B  dinv  f64[nrows]    smoother diagonal
//   section C  aggl  u16[nrows]    local aggregate of every row   (prolongation)
//              hagg  i32[nhalo]    coarse index of every halo column (prolongation)
//
// SpMV / residual+restriction copy A, the Jacobi sweeps A+B, the prolongation-fused sweep A+B+C:
// always one prefix of the blob.  Every sub-array starts on a 16-byte boundary.
// 10 bytes per nonzero instead of CSR's 12, and the out-of-tile x values are fetched once per
// distinct column into shared memory, so the inner loop reads shared memory only.
#pragma once
#include <stdint.h>

#ifndef __host__
#define __host__
#define __device__
#endif

struct alignas(16) PackDesc {   // 32 bytes per tile, read by the issuing thread one tile ahead
  uint32_t off16;               // blob offset in 16-byte units
  int32_t r0;                   // first row
  int32_t I0;                   // first coarse row (aggregate) of the tile
  int32_t nnz;
  uint16_t nrows, nhalo, nagg, pad0;
  int32_t pad1, pad2;
};

struct PackLayout {             // byte offsets inside the blob; all multiples of 16
  int o_val, o_col, o_roff, o_halo, o_aoff, endA;
  int o_dinv, endB;
  int o_aggl, o_hagg, endC;
};

__host__ __device__ inline int tp_up(int x, int m) { return (x + m - 1) / m * m; }

__host__ __device__ inline PackLayout tp_layout(int nnz, int nrows, int nhalo, int nagg) {
  PackLayout p;
  p.o_val = 0;
  p.o_col = p.o_val + tp_up(nnz, 2) * 8;
  p.o_roff = p.o_col + tp_up(nnz, 8) * 2;
  p.o_halo = p.o_roff + tp_up(nrows + 1, 8) * 2;
  p.o_aoff = p.o_halo + tp_up(nhalo, 4) * 4;
  p.endA = p.o_aoff + tp_up(nagg + 1, 8) * 2;
  p.o_dinv = p.endA;
  p.endB = p.o_dinv + tp_up(nrows, 2) * 8;
  p.o_aggl = p.endB;
  p.o_hagg = p.o_aggl + tp_up(nrows, 8) * 2;
  p.endC = p.o_hagg + tp_up(nhalo, 4) * 4;
  return p;
}

// Shared-memory bytes one ring stage needs for a tile, for the most demanding operation (the
// prolongation-fused sweep): blob prefix A+B+C, then xs[nrows+nhalo] (+2: the 16-byte rounding
// of the x slice), h2[nhalo], b[nrows] (+2), ec[nagg] (+2).  The partitioner keeps this below
// the stage size; other operations need less.
__host__ __device__ inline int tp_stage_need(int nnz, int nrows, int nhalo, int nagg) {
  const PackLayout p = tp_layout(nnz, nrows, nhalo, nagg);
  return p.endC + 8 * (tp_up(nrows + nhalo + 2, 2) + tp_up(nhalo, 2) + tp_up(nrows + 2, 2) + tp_up(nagg + 2, 2));
}
