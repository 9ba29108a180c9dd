// fp32 pair kernels, stripe width C=14 (GP = insert-state pairs of the partition-function model)
#include "qp_kernel.cuh"
namespace qp {
template cudaError_t launch_pair<float, 1, 14>(const KArgs<float>&, int, cudaStream_t);
template cudaError_t launch_pair<float, 2, 14>(const KArgs<float>&, int, cudaStream_t);
}
