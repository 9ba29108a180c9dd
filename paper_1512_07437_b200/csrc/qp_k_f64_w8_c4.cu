// fp64 pair kernels, split class (C=4, W=8): the distance-only re-evaluation of near-identical pairs after an fp32
// pass (few pairs, so the 8 warps of a CTA share each of them to cut its latency)
#include "qp_kernel.cuh"
namespace qp {
template cudaError_t launch_pair<double, 2, 4, kModeDist, 8>(const KArgs<double>&, int, cudaStream_t);
template cudaError_t launch_pair<double, 1, 4, kModeDist, 8>(const KArgs<double>&, int, cudaStream_t);   // GP = 1

}
