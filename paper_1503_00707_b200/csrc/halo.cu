// halo.cu -- ghost-cell exchange of a partitioned mesh (Fig. 5): gather the
// octant chunks a peer rank needs into one contiguous buffer (pack) and scatter a received buffer into the ghost slabs
// (unpack).  Only the upwind chunks cross: for a face on axis a the four octants whose xi_a points from the ghost cell
// into the inner cell (sign-group property).  The transfer itself (ncclSend / ncclRecv, or a copy
// when the ranks are emulated on one device) is the caller's.
#include "kernels.cuh"

namespace ufs {
namespace {

// one CTA per chunk; a chunk is `nvec` 16-byte vectors
template <bool PACK>
__global__ void __launch_bounds__(256) k_halo_copy(const int32_t* __restrict__ chunks, uint4* __restrict__ f, uint4* __restrict__ buf, int nvec) {
    const int64_t c = chunks[blockIdx.x];
    uint4* a = f + c * nvec;
    uint4* b = buf + (int64_t)blockIdx.x * nvec;
    for (int i = threadIdx.x; i < nvec; i += blockDim.x) {
        if (PACK) b[i] = a[i];
        else a[i] = b[i];
    }
}

}  // namespace

cudaError_t launch_halo_copy(bool pack, const int32_t* chunks, int64_t n_chunks, void* f, void* buf, int64_t chunk_bytes, cudaStream_t st) {
    if (n_chunks == 0) return cudaSuccess;
    const int nvec = (int)(chunk_bytes / 16);
    if (pack) k_halo_copy<true><<<(unsigned)n_chunks, 256, 0, st>>>(chunks, reinterpret_cast<uint4*>(f), reinterpret_cast<uint4*>(buf), nvec);
    else k_halo_copy<false><<<(unsigned)n_chunks, 256, 0, st>>>(chunks, reinterpret_cast<uint4*>(f), reinterpret_cast<uint4*>(buf), nvec);
    return cudaGetLastError();
}

}  // namespace ufs
