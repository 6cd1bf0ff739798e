// Tile-packed operator format of a level ("sorted-ELL tiles") -- the HBM layout the solve-phase
// row kernels stream (DESIGN.md §5/§6).  Shared by the packer (amg_setup.cu) and the kernels
// (amg_kernels.cuh); nothing here is part of the C ABI.
//
// A level's rows (aggregate-contiguous numbering) are cut into tiles of consecutive rows with
// boundaries on aggregate starts.  Each tile owns ONE contiguous, 16-byte aligned blob that a single
// bulk-async copy (TMA) brings into a ring stage:
//
//   slices  int2[nsl]      {first slot, width} of every slice of 32 storage rows
//   perm    u16[32 nsl]    storage row -> tile-local row (0xFFFF: padding).  Storage rows are the
//                          tile's rows sorted by descending length (stable), so the 32 rows of a
//                          slice have (almost) the same length and the padding stays at a few %
//   col     u16[nslots]    TILE-LOCAL column of every slot: < nr -> row r0+col of this tile,
//                          >= nr -> entry (col - nr) of the tile's halo list.  Slice-major; inside a
//                          slice k-major: slot = first + 32 k + lane  (conflict-free shared-memory reads)
//   val     f64[nslots]    matrix values, same order; padding slots are {col 0, val 0}
//           (f32[nslots] with the mixed-precision hierarchy, TileDesc::vb = 4: 6 bytes per entry)
//   -- or, for a level stored as 8-bit codes into a value dictionary (TileDesc::vb = 1), col and val merged:
//   cw      u32[nslots]    tile-local column | code << 16 (code 255 = 0.0: padding); 4 bytes per entry
//
// and a range [halo_off, halo_off + nhalo) of the level's halo arrays
//
//   halo_idx  i32[]        level index of every distinct out-of-tile column of the tile, ascending
//   halo_cagg i32[]        its coarse index (prolongation-fused sweep only)
//
// 10 bytes per stored entry instead of CSR's 12 (+4 per row), no row pointers.  The x values a
// tile needs -- its own rows and its halo columns, once per distinct column -- are assembled in
// shared memory by dedicated warps that run several tiles AHEAD of the row walk (they read the
// halo lists straight from global memory and do not depend on the ring), so the inner loop reads
// shared memory only.  Within a row the entries keep their CSR order (ascending column of the
// level numbering), so a row sum is accumulated in the same order as by the CSR kernels and by
// the oracle.
#pragma once
#include <stdint.h>

struct alignas(16) TileDesc {  // 48 bytes per tile
  int32_t r0, nr;              // rows [r0, r0 + nr)
  int32_t I0, nA;              // coarse rows [I0, I0 + nA); nA = 0 on the coarsest level
  int32_t nsl, nslots;         // slices; stored slots (= sum of 32 * width)
  int32_t nhalo;
  uint32_t blob16;             // blob offset in 16-byte units
  int32_t halo_off;            // first entry of the tile in the level's halo arrays
  int32_t vb;                  // bytes per stored value: 8 (fp64) or 4 (fp32, mixed-precision hierarchy)
  int32_t pad1, pad2;
};

__host__ __device__ inline int tp_up(int x, int m) { return (x + m - 1) / m * m; }

struct BlobLayout {  // byte offsets inside the blob; all multiples of 16
  int o_perm, o_col, o_val, end;
};
__host__ __device__ inline BlobLayout tp_blob(int nsl, int nslots, int vb) {
  BlobLayout p;
  p.o_perm = tp_up(8 * nsl, 16);
  p.o_col = p.o_perm + 64 * nsl;
  if (vb == 1) {  // value dictionary: ONE u32 per slot, tile-local column | code << 16 (one shared-memory read per entry)
    p.o_val = p.o_col;
    p.end = p.o_col + tp_up(4 * nslots, 16);
    return p;
  }
  p.o_val = p.o_col + tp_up(2 * nslots, 16);
  p.end = p.o_val + tp_up(vb * nslots, 16);
  return p;
}

// Placement of a tile inside its ring stage, after the TP_DESC_BYTES stage header.  Row-vector
// slices are rounded out to 16-byte boundaries of their source arrays (bulk copies need 16-byte
// aligned addresses and sizes): ra2 / Ia4 are the rounded-down first elements.
constexpr int TP_DESC_BYTES = 128;
struct StageLayout {
  int ra2, nrv;    // first staged row of the f64 row vectors (even), entries staged (even)
  int Ia4, nap;    // agg_ptr slice (nA + 1 entries from I0)
  int Ia2, nec;    // coarse-vector slice (nA entries from I0)
  int o_b, o_d, o_agg, o_dc, o_out, end;  // byte offsets (blob at 0)
};
// flags: which operands the operation stages in the ring
enum { TP_B = 1, TP_D = 2, TP_DC = 8, TP_AGGPTR = 16, TP_OUT = 64 };
__host__ __device__ inline StageLayout tp_stage(const TileDesc& d, int flags) {
  StageLayout t;
  const BlobLayout p = tp_blob(d.nsl, d.nslots, d.vb);
  const int r1 = d.r0 + d.nr;
  t.ra2 = d.r0 & ~1;
  t.nrv = tp_up(r1 - t.ra2, 2);
  t.Ia4 = d.I0 & ~3;
  t.nap = tp_up(d.I0 + d.nA + 1 - t.Ia4, 4);
  t.Ia2 = d.I0 & ~1;
  t.nec = tp_up(d.I0 + d.nA - t.Ia2, 2);
  int o = p.end;
  t.o_b = o;
  if (flags & TP_B) o += 8 * t.nrv;
  t.o_d = o;
  if (flags & TP_D) o += 8 * t.nrv;
  t.o_agg = o;
  if (flags & TP_AGGPTR) o += 4 * t.nap;
  t.o_dc = o;
  if (flags & TP_DC) o += 8 * t.nec;
  t.o_out = o;
  if (flags & TP_OUT) o += 8 * tp_up(d.nr, 2);
  t.end = o;
  return t;
}
constexpr int TP_FLAGS_SWEEP = TP_B | TP_D;                            // Jacobi sweeps
constexpr int TP_FLAGS_RESTRICT = TP_B | TP_AGGPTR | TP_DC | TP_OUT;   // residual + restriction (+ x1 of the coarse level)
// shared-memory bytes one ring stage needs for a tile, for the most demanding operations
__host__ __device__ inline int tp_stage_need(const TileDesc& d) {
  const int a = tp_stage(d, TP_FLAGS_SWEEP).end, b = tp_stage(d, TP_FLAGS_RESTRICT).end;
  return TP_DESC_BYTES + (a > b ? a : b);
}
// bytes of the tile's x slot (side ring): [x of the tile's rows | x of its halo columns]
__host__ __device__ inline int tp_xslot_need(const TileDesc& d) { return 8 * (d.nr + d.nhalo); }
