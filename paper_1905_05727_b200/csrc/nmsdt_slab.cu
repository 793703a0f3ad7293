// nmsdt_slab.cu -- halo-column movement of the x-slab decomposition (include/nmsdt.h sim_slab_*).
//
// The only data a slab needs from its neighbours per step are two columns of the 7 planes per side before the x-sweep
// (stencil radius 2, O4; 7 x ny x 2 doubles = 0.46 MB at ny = 4096).  One kernel moves such a block between two strided
// layouts; the three uses differ only in the layouts:
//   pack   : own edge columns            -> dense block [7][ny][2]      (staging transport, e.g. NCCL send/recv)
//   unpack : dense block                 -> own ghost columns
//   push   : own edge columns            -> the NEIGHBOUR's ghost columns (peer memory over NVLink: plain stores through a
//            pointer that is valid in this process -- same process, or mapped with cudaIpcOpenMemHandle)
#include "nmsdt_host.h"

namespace nmsdt {

// element (f, j, m) of a block: base[f * fstride + j * pitch + m], m = 0, 1
__global__ void __launch_bounds__(128) k_slab_move(SlabView src, SlabView dst, int ny)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int f = blockIdx.y;
    if (j >= ny) return;
    const double* a = src.base + (long long)f * src.fstride + (long long)j * src.pitch;
    double* b = dst.base + (long long)f * dst.fstride + (long long)j * dst.pitch;
    const double v0 = a[0], v1 = a[1];
    b[0] = v0; b[1] = v1;
}

void launch_slab_move(const SlabView& src, const SlabView& dst, int ny, cudaStream_t s)
{
    dim3 grid((ny + 127) / 128, 7);
    k_slab_move<<<grid, 128, 0, s>>>(src, dst, ny);
}

} // namespace nmsdt
