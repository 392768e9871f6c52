// halo.cu -- ghost-cell exchange of a partitioned mesh (Fig. 5): gather the
// octant chunks a peer rank needs into one contiguous buffer (pack) and scatter a received buffer into the ghost slabs
// (unpack).  Only the upwind chunks cross: for a face on axis a the four octants whose xi_a points from the ghost cell
// into the inner cell (sign-group property).  Behind the chunks the buffer carries the cells' 36 carried
// velocity sums (the Maxwellian of an inner cell needs its upwind sources' flux moments): the ghost rows then
// hold the owner's own sums, as in the unpartitioned run.  The transfer itself (ncclSend / ncclRecv, or a copy
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

// the 36 carried velocity sums of each listed cell travel behind its chunks: row i of the tail <-> sums row slabs[i]
template <bool PACK>
__global__ void __launch_bounds__(256) k_halo_sums(const int32_t* __restrict__ slabs, int64_t n, double* __restrict__ sums, double* __restrict__ tail) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n * SUMS_STRIDE) return;
    const int64_t row = i / SUMS_STRIDE;
    const int j = (int)(i % SUMS_STRIDE);
    double* a = sums + (int64_t)slabs[row] * SUMS_STRIDE + j;
    if (PACK) tail[i] = *a;
    else *a = tail[i];
}

}  // namespace

cudaError_t launch_halo_sums(bool pack, const int32_t* slabs, int64_t n_slabs, double* sums, void* tail, cudaStream_t st) {
    if (n_slabs == 0) return cudaSuccess;
    const int64_t n = n_slabs * SUMS_STRIDE;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    if (pack) k_halo_sums<true><<<blocks, 256, 0, st>>>(slabs, n_slabs, sums, reinterpret_cast<double*>(tail));
    else k_halo_sums<false><<<blocks, 256, 0, st>>>(slabs, n_slabs, sums, reinterpret_cast<double*>(tail));
    return cudaGetLastError();
}

cudaError_t launch_halo_copy(bool pack, const int32_t* chunks, int64_t n_chunks, void* f, void* buf, int64_t chunk_bytes, cudaStream_t st) {
    if (n_chunks == 0) return cudaSuccess;
    const int nvec = (int)(chunk_bytes / 16);
    if (pack) k_halo_copy<true><<<(unsigned)n_chunks, 256, 0, st>>>(chunks, reinterpret_cast<uint4*>(f), reinterpret_cast<uint4*>(buf), nvec);
    else k_halo_copy<false><<<(unsigned)n_chunks, 256, 0, st>>>(chunks, reinterpret_cast<uint4*>(f), reinterpret_cast<uint4*>(buf), nvec);
    return cudaGetLastError();
}

}  // namespace ufs
