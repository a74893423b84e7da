// lbm_inplace_launch.h — host-side interface between the launch layer (lbm_api.cu) and the in-place step kernels, which are
// compiled as a translation unit of their own (lbm_inplace_launch.cu) so that the two halves of the library build in parallel.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace lbmk {

struct IpLaunch {
    int prec;              // 0 = <float, float>, 1 = <double, double>, 2 = <float, __half>   (include/lbm.h LBM_PREC_*)
    bool sample, damp, turb;
    int parity;            // parity of this step = the layout the state is in
    void *G;               // the one population buffer
    const uint8_t *flags;
    const uint32_t *links;
    void *msum;            // mean sums (reals), may be null when !sample
    const void *fur;       // face-velocity side array: the half to read, the half to write (reals)
    void *fuw;
    const void *params;    // const Params<real> * of the handle
    const void *fum;       // inflow fluctuations: mean boundary velocity, mode table, number of modes, time of the step after next
    const double *modes;
    int nmodes;
    double t;
    // thermal lattice on (lbm_set_thermal): its two buffers stay double (HA = the one that goes with the current state, HB = the
    // one this step writes) and the thermal companion of the side array (halves to read / to write); null while it is off
    const void *HA;
    void *HB;
    const void *ftr;
    void *ftw;
    cudaStream_t stream;
};

// launches one step; returns the cudaError_t of the launch
cudaError_t ip_launch(const IpLaunch &L);

} // namespace lbmk
