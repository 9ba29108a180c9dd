// fp64 pair kernels, stripe width C=8: QP_FP64 mode (all outputs) and the distance-only re-evaluation of
// near-identical pairs after an fp32 pass
#include "qp_kernel.cuh"
namespace qp {
template cudaError_t launch_pair<double, 2, 8, kModeFull>(const KArgs<double>&, int, cudaStream_t);
template cudaError_t launch_pair<double, 2, 8, kModeDist>(const KArgs<double>&, int, cudaStream_t);
}
