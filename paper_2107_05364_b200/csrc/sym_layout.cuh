// sym_layout.cuh — F3: storage of the pair-symmetric half of the tensor ("MagTense
// utilizes the fact that the tensor is symmetric ... reducing the scaling to ... almost N^2/2").
//
// On a mesh of congruent axis-aligned cuboids the block of a pair depends on c_i - c_j only and is
// even in it (Q2, pin P9), so N_ij = N_ji: only blocks with j >= i need to be kept, and each
// serves two rows of the product.  The half is kept at tile granularity, in the order the field kernel
// reads it:
//   row block I   = rows [32 I, 32 I + 32)
//   column tile J = columns [TW J, TW J + TW), TW = 32 W, W = 16 / sizeof(T) (128 fp32 / 64 fp64 columns)
//   row block I keeps the tiles J = Jd(I) .. ntc-1, Jd(I) = 32 I / TW (the tile holding its diagonal)
//   inside a tile: [plane 0..5][g 0..3][warp 0..7][lane 0..31][e 0..W-1] with
//       row    it = 8 g + lane / 4
//       column jt = 4 W warp + W (lane % 4) + e
//   so that one warp-wide 16-byte load is 512 contiguous bytes and a tile is 96 KiB.
// Entries of the diagonal tile left of the row block's own 32 x 32 diagonal block (column block
// jb = j / 32 < I) are not part of the half: they are stored as zero and never used.
#pragma once
#include <stdint.h>

template <typename T> struct SymCfg {
  static constexpr int W = 16 / (int)sizeof(T);  // columns per lane
  static constexpr int TW = 32 * W;              // columns per tile
  static constexpr int RB = 32;                  // rows per row block
  static constexpr int kBlocksPerTile = TW / 32; // 32-column blocks per tile (= W)
  static constexpr int64_t kTileElems = (int64_t)6 * RB * TW;
};

__host__ __device__ inline int64_t sym_row_blocks(int64_t n) { return (n + 31) / 32; }
__host__ __device__ inline int64_t sym_col_tiles(int64_t n, int tw) { return (n + tw - 1) / tw; }
// number of tiles kept by row blocks 0 .. I-1 (bpt = 32-column blocks per tile)
__host__ __device__ inline int64_t sym_tile_prefix(int64_t I, int64_t ntc, int bpt) {
  const int64_t q = I / bpt, r = I % bpt;
  return I * ntc - ((int64_t)bpt * q * (q - 1) / 2 + r * q);
}
__host__ __device__ inline int64_t sym_total_tiles(int64_t n, int tw) {
  return sym_tile_prefix(sym_row_blocks(n), sym_col_tiles(n, tw), tw / 32);
}
// element offset inside a tile
__host__ __device__ inline int sym_elem_offset(int plane, int it, int jt, int w_cols) {
  const int g = it >> 3, warp = jt / (4 * w_cols), lane = ((it & 7) << 2) | ((jt / w_cols) & 3), e = jt % w_cols;
  return ((((plane * 4 + g) * 8 + warp) * 32 + lane) * w_cols) + e;
}
