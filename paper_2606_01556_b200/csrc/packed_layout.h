// packed_layout.h -- byte offsets of the sections inside the opaque packed-weight blob
// (host-side arithmetic shared by the packer, both kernels' launchers and twq_packed_bytes).
//
//   R4   [N/8][K/G][8][G/2] u8   4-bit residual codes, two per byte (low nibble = even k).  One
//                                (8-channel tile, K-group) block is 4*G contiguous bytes: the decode kernel
//                                streams whole tiles with 1-D bulk copies and reads a block with one
//                                warp-wide 16-byte load; the tcgen05 kernel fetches 16 such blocks of one
//                                group (128 channels x G/2 bytes) as one 4-D TMA box.
//   sw16 [N/8][K/G][8] f16       residual group scales, same tiling (FP16 as the format stores them)
//   L1T  [r][K] f16              L1 transposed: K-major A operand of the tcgen05 stage-1 MMA
//   L1D  [K/32][r][32] f16       L1 in 32-wide K slabs: a cluster rank's K slice is one contiguous range
//                                (1-D bulk copies) and an MMA fragment row is 64 contiguous bytes (decode kernel)
//   L2T  [N][r] f16              L2 transposed: K-major operand of stage 2 (reduction over r)
// Every section is 256-byte aligned.
#pragma once
#include <stddef.h>

namespace twq {

struct PackedLayout {
    size_t off_r4, off_sw16, off_l1t, off_l1d, off_l2t, total;
};

inline size_t align256(size_t x) { return (x + 255) & ~static_cast<size_t>(255); }

inline PackedLayout packed_layout(int N, int K, int r, int G) {
    PackedLayout l;
    size_t o = 0;
    l.off_r4 = o;
    o = align256(o + static_cast<size_t>(N) * (K / 2));
    l.off_sw16 = o;
    o = align256(o + static_cast<size_t>(K / G) * N * 2);
    l.off_l1t = o;
    o = align256(o + static_cast<size_t>(r) * K * 2);
    l.off_l1d = o;
    o = align256(o + static_cast<size_t>(r) * K * 2);
    l.off_l2t = o;
    o = align256(o + static_cast<size_t>(N) * r * 2);
    l.total = o;
    return l;
}

}  // namespace twq
