// fp64 pair kernels, stripe width C=4 (QP_FP64 mode and the refinement pass of near-identical pairs)
#include "qp_kernel.cuh"
namespace qp {
template cudaError_t launch_pair<double, 2, 4>(const KArgs<double>&, int, cudaStream_t);
}
