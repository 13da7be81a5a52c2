// ahs_diag_march.cu -- diagnostics for lattices served by the z-marching step kernel.
// Until the staged marching version lands this forwards to the one-thread-per-site kernel (ahs_diag_generic.cu).
#include "ahs_internal.cuh"

namespace ahs {

template <typename T>
int launch_diag_march(const DiagPtrs<T>& f, int N, const DiagCoef& c, DiagPartial* partials, int max_partials, DiagPartial* result, cudaStream_t st)
{
    return launch_diag_generic<T>(f, N, c, partials, max_partials, result, st);
}

template int launch_diag_march<float>(const DiagPtrs<float>&, int, const DiagCoef&, DiagPartial*, int, DiagPartial*, cudaStream_t);
template int launch_diag_march<double>(const DiagPtrs<double>&, int, const DiagCoef&, DiagPartial*, int, DiagPartial*, cudaStream_t);

}  // namespace ahs
