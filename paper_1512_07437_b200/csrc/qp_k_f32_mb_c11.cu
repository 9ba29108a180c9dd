// fp32 pair kernels, packed TWO-BLOCK class with stripe width C=11 (one warp per pair of 513..1024 columns; the warp
// runs the pair's two 32*C-column blocks one after the other). GP = insert-state pairs of the partition-function model
#include "qp_kernel.cuh"
namespace qp {
template cudaError_t launch_pair<float, 1, 11, kModeCsr | kModeMB, 1>(const KArgs<float>&, int, cudaStream_t);
template cudaError_t launch_pair<float, 2, 11, kModeCsr | kModeMB, 1>(const KArgs<float>&, int, cudaStream_t);
template cudaError_t launch_pair<float, 1, 11, kModeFull | kModeMB, 1>(const KArgs<float>&, int, cudaStream_t);
template cudaError_t launch_pair<float, 2, 11, kModeFull | kModeMB, 1>(const KArgs<float>&, int, cudaStream_t);
}
