// layout.cuh — HBM layout of the link store.
//
// Parity-split structure-of-arrays in 16-byte vectors (the Float4 scheme of PAPER.md:359 generalised,
// with the parity-priority index order of PAPER.md:366):
//
//     links[parity p][mu][chunk c][checkerboard site cb]        one chunk = 16 bytes (float4 | double2)
//
// p = parity (t+x+y+z)&1 of the link's origin x (Eq. (32));
// cb = lexicographic index ((t*Nx + x)*Ny + y)*Nz + z divided by 2 (z fastest);
// chunk c holds reals [c*PER16, (c+1)*PER16) of the row-major (i,j,re/im) link, of which only the
// first RECON = 18 or 12 are stored.  SP-18 is 72 bytes = four float4 chunks plus
// one float2 tail plane.  A warp reading one chunk of consecutive sites moves 512 contiguous bytes.
#pragma once
#include <cstdint>

namespace gf {

template <class R, int RECON>
struct Layout {
    static constexpr int LINK_BYTES = RECON * (int)sizeof(R);
    static constexpr int NV16 = LINK_BYTES / 16;          // full 16-byte chunks per link
    static constexpr int TAIL8 = (LINK_BYTES % 16) / 8;   // 1 only for SP-18
    static constexpr int PER16 = 16 / (int)sizeof(R);     // reals per chunk
    // byte offset of chunk plane 0 of link direction mu in parity p; Vh = V/2 sites per parity
    __host__ __device__ static int64_t link_offset(int p, int mu, int64_t Vh) {
        return (int64_t)(p * 4 + mu) * LINK_BYTES * Vh;
    }
    // the same for one-matrix-per-site fields (tracked gauge transform): field[p][chunk][cb]
    __host__ __device__ static int64_t site_offset(int p, int64_t Vh) { return (int64_t)p * LINK_BYTES * Vh; }
    __host__ __device__ static int64_t links_bytes(int64_t Vh) { return (int64_t)8 * LINK_BYTES * Vh; }
    __host__ __device__ static int64_t field_bytes(int64_t Vh) { return (int64_t)2 * LINK_BYTES * Vh; }
};

}  // namespace gf
