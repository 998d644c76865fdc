// sc_fast.cu -- fast kernels (placeholder: not built yet; the generic kernel serves every ring).
#include "sc_internal.cuh"
#include <vector>
namespace sc {
struct FastPlan {};
FastPlan *fast_plan_create(const Dev &, const std::vector<double> &, const std::vector<double> &, int, int *polar_rings, cudaError_t *err) {
    *polar_rings = 0; *err = cudaSuccess; return nullptr;
}
void fast_plan_destroy(FastPlan *) {}
cudaError_t fast_convolve(FastPlan *, const Dev &, const Maps &, int, cudaStream_t, int *launches) { *launches = 0; return cudaSuccess; }
}  // namespace sc
