// packed_layout.h -- byte offsets of the sections inside the opaque packed-weight blob
// (host-side arithmetic shared by the packer, the fused kernel's launcher and
// twq_packed_bytes).  Sections: R4 [N][K/2] u8 | swT [K/G][N] f32 | L1T [r][K] f16 | L2T [N][r] f16.
#pragma once
#include <stddef.h>

namespace twq {

struct PackedLayout {
    size_t off_r4, off_swT, off_l1t, off_l2t, total;
};

inline size_t align256(size_t x) { return (x + 255) & ~static_cast<size_t>(255); }

inline PackedLayout packed_layout(int N, int K, int r, int G) {
    PackedLayout l;
    size_t o = 0;
    l.off_r4 = o;
    o = align256(o + static_cast<size_t>(N) * (K / 2));
    l.off_swT = o;
    o = align256(o + static_cast<size_t>(K / G) * N * 4);
    l.off_l1t = o;
    o = align256(o + static_cast<size_t>(r) * K * 2);
    l.off_l2t = o;
    o = align256(o + static_cast<size_t>(N) * r * 2);
    l.total = o;
    return l;
}

}  // namespace twq
