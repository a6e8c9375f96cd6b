// fftb_slab.cuh -- the data-movement stage of the slab-distributed transform (sm_100a).
//
// PAPER.md:231 ("small CUDA codelets that pack and rotate the data locally on the GPU before communicating") and
// :241-243 (the plane-wave variant sends only the pruned stick data): with R ranks, rank r owns the sticks of a
// contiguous range of k1 columns and the z-planes of one slab.  Between the z pass (all z of the own sticks) and the
// plane pass (all sticks of the own planes) every rank hands every other rank a block
//     rows = the receiver's (inverse) / the sender's (forward) z-planes,  columns = the sender's / receiver's sticks,
// both of which are CONTIGUOUS runs of the plane-major intermediate A[band][z][stick].  So "pack, rotate, all-to-all,
// unpack" is one kernel of row copies with one segment per peer.  The destination of a segment is either a staging
// buffer ([peer][band][row][column], handed to an NCCL all-to-all by the caller) or -- with peer-mapped pointers over
// NVLink -- the peer's intermediate itself, in which case the same kernel IS the exchange.
#pragma once
#include <cuda_runtime.h>

namespace fftb {

constexpr int SLAB_MAXR = 16;
struct SlabSeg {
    long long src_off, src_sb, src_sr; // first element, band stride, row stride (elements) on the source side
    long long dst_off, dst_sb, dst_sr; // ... on the destination side
    int rows, cols, peer;
};
struct SlabSegs {
    SlabSeg s[SLAB_MAXR];
    void *dst[SLAB_MAXR]; // destination base of peer i (all equal when the blocks go to one staging buffer)
    int n;
};

// grid = (row blocks, bands, segments); a CTA copies rows blockIdx.x, blockIdx.x + gridDim.x, ... of one band of one segment
template <typename C> __global__ void __launch_bounds__(256) slab_rows_k(const __grid_constant__ SlabSegs sg, const C *__restrict__ src)
{
    const SlabSeg &g = sg.s[blockIdx.z];
    C *__restrict__ dst = reinterpret_cast<C *>(sg.dst[g.peer]);
    const long long b = blockIdx.y;
    for (int row = blockIdx.x; row < g.rows; row += gridDim.x) {
        const C *s = src + g.src_off + b * g.src_sb + (long long)row * g.src_sr;
        C *d = dst + g.dst_off + b * g.dst_sb + (long long)row * g.dst_sr;
        for (int c = threadIdx.x; c < g.cols; c += blockDim.x) d[c] = s[c];
    }
}

} // namespace fftb
