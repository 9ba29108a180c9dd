// fp64 pair kernels, packed class with stripe width C=2: QP_FP64 mode (all outputs)
#include "qp_kernel.cuh"
namespace qp {
template cudaError_t launch_pair<double, 2, 2, kModeFull, 1>(const KArgs<double>&, int, cudaStream_t);
}
