// Team-per-station kernel (unfold_t4k.cuh): the instantiations that read int16 ADC counts and write fp32
// (aera_unfold_batch_i16 at N = 1024, 4096, 8192, 16384).
#include "unfold_t4k.cuh"

namespace aera {

cudaError_t launch_unfold_t4k_i16(const PlanDev &p, long n_units, int n_stations, const void *traces, void *efield, void *amp,
                                  int32_t *idx, const void *minv, cudaStream_t s, const UnfoldExt &x)
{
    return launch_t4k_typed<float, true>(p, n_units, n_stations, traces, efield, amp, idx, minv, s, x);
}

} // namespace aera
