// fp32 pair kernels, packed class with stripe width C=3 (one warp per pair). GP = insert-state pairs of the
// partition-function model; MODE 0 = CSR + distance, 1 = the same plus the optional dense_P / logZ test outputs
#include "qp_kernel.cuh"
namespace qp {
template cudaError_t launch_pair<float, 1, 3, kModeCsr, 1>(const KArgs<float>&, int, cudaStream_t);
template cudaError_t launch_pair<float, 2, 3, kModeCsr, 1>(const KArgs<float>&, int, cudaStream_t);
template cudaError_t launch_pair<float, 1, 3, kModeFull, 1>(const KArgs<float>&, int, cudaStream_t);
template cudaError_t launch_pair<float, 2, 3, kModeFull, 1>(const KArgs<float>&, int, cudaStream_t);
}
