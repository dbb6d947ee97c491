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
//
// The q4lr blob (twq_pack_weights_q4lr: both low-rank factors 4-bit) keeps R4 and sw16 and replaces the
// FP16 sections by
//   U    [K/G][ r x G/2 u8 codes | r f16 scales ]   per K-group: the codes of U = L1^T ([r][G/2], row j = rank index,
//                                two per byte) followed by that group's r scales; a cluster rank's K slice is one
//                                contiguous range and a j tile of a group is 8 rows x G/2 bytes like a block of R4
//   V    [N/8][nh][8][grs/2] u8  codes of V = L2^T, groups of gr rank indices (gr = r for r <= 128, else 128), each row
//                                zero-padded to grs = gr rounded up to 32 codes (one MMA K-step)
//   sv16 [N/8][nh][8] f16        scales of V
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

struct PackedLayoutQ4 {
    size_t off_r4, off_sw16, off_u, off_v, off_sv16, total;
    int gr, grs, nh;
    size_t u_group_bytes;
};

inline PackedLayoutQ4 packed_layout_q4lr(int N, int K, int r, int G) {
    PackedLayoutQ4 l;
    l.gr = r <= 128 ? r : 128;
    l.grs = (l.gr + 31) / 32 * 32;
    l.nh = l.gr > 0 ? r / l.gr : 0;
    l.u_group_bytes = static_cast<size_t>(r) * (G / 2) + static_cast<size_t>(r) * 2;
    size_t o = 0;
    l.off_r4 = o;
    o = align256(o + static_cast<size_t>(N) * (K / 2));
    l.off_sw16 = o;
    o = align256(o + static_cast<size_t>(K / G) * N * 2);
    l.off_u = o;
    o = align256(o + static_cast<size_t>(K / G) * l.u_group_bytes);
    l.off_v = o;
    o = align256(o + static_cast<size_t>(N) * l.nh * (l.grs / 2));
    l.off_sv16 = o;
    o = align256(o + static_cast<size_t>(N) * l.nh * 2);
    l.total = o;
    return l;
}

}  // namespace twq
