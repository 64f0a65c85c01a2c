// Team-per-station kernel (unfold_t4k.cuh): the fp32 instantiations (N = 1024, 4096, 8192, 16384; float or int16 traces).
#include "unfold_t4k.cuh"

namespace aera {

cudaError_t launch_unfold_t4k_f32(const PlanDev &p, long n_units, int n_stations, const void *traces, void *efield, void *amp,
                                  int32_t *idx, const void *minv, cudaStream_t s, const UnfoldExt &x)
{
    if (x.input_i16) return launch_unfold_t4k_i16(p, n_units, n_stations, traces, efield, amp, idx, minv, s, x);
    return launch_t4k_typed<float>(p, n_units, n_stations, traces, efield, amp, idx, minv, s, x);
}

} // namespace aera
