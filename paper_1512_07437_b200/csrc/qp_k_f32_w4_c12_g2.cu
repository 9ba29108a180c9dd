// fp32 pair kernels, split class (C=12, W=4): the 4 warps of a CTA share one long pair (anti-diagonal wavefront
// pipelined over 4 neighbouring column blocks). GP=2 insert-state pairs in the partition-function model.
#include "qp_kernel.cuh"
namespace qp {
template cudaError_t launch_pair<float, 2, 12, kModeCsr, 4>(const KArgs<float>&, int, cudaStream_t);
template cudaError_t launch_pair<float, 2, 12, kModeFull, 4>(const KArgs<float>&, int, cudaStream_t);
}
