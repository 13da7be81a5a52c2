// placeholder until the z-marching kernels land
#include "ahs_internal.cuh"
namespace ahs {
template <typename T> bool march_supported(int) { return false; }
template <typename T> int launch_step_march(const FieldPtrs<T>&, int, const StepCoef&, cudaStream_t) { return AHS_ERR_STATE; }
template <typename T> int launch_diag_march(const DiagPtrs<T>&, int, const DiagCoef&, DiagPartial*, int, DiagPartial*, cudaStream_t) { return AHS_ERR_STATE; }
template bool march_supported<float>(int);
template bool march_supported<double>(int);
template int launch_step_march<float>(const FieldPtrs<float>&, int, const StepCoef&, cudaStream_t);
template int launch_step_march<double>(const FieldPtrs<double>&, int, const StepCoef&, cudaStream_t);
template int launch_diag_march<float>(const DiagPtrs<float>&, int, const DiagCoef&, DiagPartial*, int, DiagPartial*, cudaStream_t);
template int launch_diag_march<double>(const DiagPtrs<double>&, int, const DiagCoef&, DiagPartial*, int, DiagPartial*, cudaStream_t);
}
