// lbm_inplace_launch.cu — instantiations and launch of the in-place streaming step (lbm_inplace.cuh); a translation unit of
// its own so that it compiles beside lbm_api.cu (paper_2607_04516_b200/build.py runs the two nvcc jobs in parallel).
#include "lbm_inplace.cuh"
#include "lbm_thermal.cuh"
#include "lbm_inplace_launch.h"

namespace lbmk {
namespace {

#ifndef IP_MINB
#define IP_MINB 10
#endif

inline unsigned blocks_for(long long n, int block) { return (unsigned)((n + block - 1) / block); }

template <typename real, typename S, int MINB, bool DAMP, bool PERX, bool TURB>
cudaError_t launch_as(const IpLaunch &L, const Params<real> &P)
{
    constexpr int BLOCK = 128;
    dim3 grid(blocks_for((long long)P.nxy, BLOCK), (unsigned)P.nz);
    const int turb_planes = TURB ? (int)((blocks_for(P.F, BLOCK) + grid.x - 1) / grid.x) : 0;
    grid.y += turb_planes;
    const IpPtrs<S> T = make_ip_ptrs<S>((S *)L.G, L.parity, P);
    const Turb<real> tb{(const real *)L.fum, L.modes, L.nmodes, L.t};
    cudaLaunchConfig_t cfg{}; // programmatic dependent launch, as for the two-buffer step (lbm_api.cu launch_step_as)
    cfg.gridDim = grid; cfg.blockDim = dim3(BLOCK); cfg.dynamicSmemBytes = 0; cfg.stream = L.stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    real *ms = (real *)L.msum;
    const real *fur = (const real *)L.fur;
    real *fuw = (real *)L.fuw;
    constexpr int MINB_S = MINB == 10 ? 9 : MINB; // sampling steps hold three more values per thread
    if (L.sample) return cudaLaunchKernelEx(&cfg, ip_step_kernel<real, S, true, BLOCK, MINB_S, DAMP, PERX, TURB>, L.flags, L.links, ms, fur, fuw, P, T, tb, turb_planes);
    return cudaLaunchKernelEx(&cfg, ip_step_kernel<real, S, false, BLOCK, MINB, DAMP, PERX, TURB>, L.flags, L.links, ms, fur, fuw, P, T, tb, turb_planes);
}

// fused flow + thermal step, the flow lattice in place (lbm_thermal.cuh ip_thermal_step_kernel); S = real there
template <typename real, bool PERX, bool DAMP>
cudaError_t launch_thermal_as(const IpLaunch &L, const Params<real> &P, bool turb)
{
    constexpr int BLOCK = 128, MINB = std::is_same<real, float>::value ? 8 : 2;
    dim3 grid(blocks_for((long long)P.nxy, BLOCK), (unsigned)P.nz);
    const int turb_planes = (DAMP && turb) ? (int)((blocks_for(P.F, BLOCK) + grid.x - 1) / grid.x) : 0;
    grid.y += turb_planes;
    const IpPtrs<real> I = make_ip_ptrs<real>((real *)L.G, L.parity, P);
    const ThermalPtrs<real> T = make_thermal_ptrs<real>((const real *)L.G, (real *)L.G, (const real *)L.HA, (real *)L.HB, P); // flow entries unused
    const OpenFaces<real> O{(const real *)L.fur, (real *)L.fuw, (const real *)L.ftr, (real *)L.ftw};
    const Turb<real> tb{(const real *)L.fum, L.modes, L.nmodes, L.t};
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = dim3(BLOCK); cfg.dynamicSmemBytes = 0; cfg.stream = L.stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    real *HB = (real *)L.HB, *ms = (real *)L.msum;
    if (L.sample) return cudaLaunchKernelEx(&cfg, ip_thermal_step_kernel<real, true, BLOCK, MINB, PERX, DAMP>, HB, L.flags, L.links, ms, P, T, O, tb, turb_planes, I);
    return cudaLaunchKernelEx(&cfg, ip_thermal_step_kernel<real, false, BLOCK, MINB, PERX, DAMP>, HB, L.flags, L.links, ms, P, T, O, tb, turb_planes, I);
}
template <typename real>
cudaError_t launch_thermal(const IpLaunch &L)
{
    const Params<real> &P = *(const Params<real> *)L.params;
    const bool ext = L.damp || L.turb; // the open-boundary-stack instantiation (zones + fluctuation block rows)
    if (P.perx != 0) return ext ? launch_thermal_as<real, true, true>(L, P, L.turb) : launch_thermal_as<real, true, false>(L, P, false);
    return ext ? launch_thermal_as<real, false, true>(L, P, L.turb) : launch_thermal_as<real, false, false>(L, P, false);
}

template <typename real, typename S>
cudaError_t launch(const IpLaunch &L)
{
    const Params<real> &P = *(const Params<real> *)L.params;
    constexpr int M = std::is_same<real, float>::value ? IP_MINB : 4;
    constexpr int M9 = std::is_same<real, float>::value ? (IP_MINB == 10 ? 9 : IP_MINB) : 4; // two more indices / table values: one CTA per SM less
    const bool perx = P.perx != 0;
    if (L.turb) {
        if (L.damp) return perx ? launch_as<real, S, M9, true, true, true>(L, P) : launch_as<real, S, M9, true, false, true>(L, P);
        return perx ? launch_as<real, S, M9, false, true, true>(L, P) : launch_as<real, S, M, false, false, true>(L, P);
    }
    if (L.damp) return perx ? launch_as<real, S, M9, true, true, false>(L, P) : launch_as<real, S, M9, true, false, false>(L, P);
    return perx ? launch_as<real, S, M9, false, true, false>(L, P) : launch_as<real, S, M, false, false, false>(L, P);
}

} // namespace

cudaError_t ip_launch(const IpLaunch &L)
{
    if (L.HB) return L.prec == 1 ? launch_thermal<double>(L) : launch_thermal<float>(L); // thermal lattice on (never with 16-bit storage)
    if (L.prec == 1) return launch<double, double>(L);
    if (L.prec == 2) return launch<float, __half>(L);
    return launch<float, float>(L);
}

} // namespace lbmk
