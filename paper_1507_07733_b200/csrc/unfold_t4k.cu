// Team-per-station kernel (unfold_t4k.cuh): the fp64 instantiations and the dispatch by precision. The fp32 ones are
// compiled in unfold_t4k_f32.cu (two translation units: the build runs them side by side).
#include "unfold_t4k.cuh"

namespace aera {

int t4k_team_warps(int dtype, const PlanDev &p)
{
    if (p.k_lo < 1 || p.k_hi >= p.N / 2) return 0;
    if (p.N == 4096 && (dtype == AERA_F64 || dtype == AERA_F32)) return 4;
    if (p.N == 2048 && dtype == AERA_F64) return 2;
    if (p.N == 1024 && (dtype == AERA_F64 || dtype == AERA_F32)) return 1;
    if (p.N == 8192 && (dtype == AERA_F64 || dtype == AERA_F32)) return 8;
    if (p.N == 16384 && dtype == AERA_F32) return 16;
    return 0;
}
bool t4k_supported(int dtype, const PlanDev &p) { return t4k_team_warps(dtype, p) != 0; }

cudaError_t launch_unfold_t4k(int dtype, const PlanDev &p, long n_events, int n_stations, const void *traces, void *efield,
                              void *amp, int32_t *idx, const void *minv, cudaStream_t s, const UnfoldExt &x)
{
    const long n_units = n_events * (long)n_stations;
    if (n_units <= 0) return cudaSuccess;
    ProfScope prof(KID_UNFOLD, s);
    const cudaError_t e = dtype == AERA_F64 ? launch_t4k_typed<double>(p, n_units, n_stations, traces, efield, amp, idx, minv, s, x)
                                            : launch_unfold_t4k_f32(p, n_units, n_stations, traces, efield, amp, idx, minv, s, x);
    count_launches(1);
    return e;
}

} // namespace aera
