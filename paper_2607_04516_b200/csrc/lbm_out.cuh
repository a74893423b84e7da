// lbm_out.cuh — a7: macroscopic fields and time means of the stored state, and the parity exports.
// Outputs are un-padded C-order [nz][ny][nx] arrays; the internal state is halo-padded (lbm_core.cuh).
#pragma once
#include "lbm_core.cuh"

namespace lbmk {

// theta - theta_ref of the stored thermal state of cell p (lbm_thermal.cuh: 7 shifted populations, directions 0..6)
template <typename real>
__device__ __forceinline__ real stored_theta_shift(const real *__restrict__ H, long long stride, int p)
{
    return H[p] + ((H[stride + p] + H[2 * stride + p]) + (H[3 * stride + p] + H[4 * stride + p]) + (H[5 * stride + p] + H[6 * stride + p]));
}

// local macros of the stored state (DESIGN.md §3 step 7)
template <typename real, typename S, typename out_t, int IPM = 0>
__global__ void macros_kernel(const S *__restrict__ A, const uint8_t *__restrict__ flags, out_t *__restrict__ rho,
                              out_t *__restrict__ ux, out_t *__restrict__ uy, out_t *__restrict__ uz, Params<real> P,
                              const real *__restrict__ H, const uint32_t *__restrict__ links, const Box bx)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    int x, y, z;
    if (!box_cell(bx, c, x, y, z)) return; // outputs are the box's own C-order arrays (the whole lattice: the box is the lattice)
    const int p = pidx(P, x, y, z);
    const uint8_t fl = flags[p];
    const int cls = fl & CLASS_MASK;
    real g[Q];
    Macro<real> m{real(1), real(0), real(0), real(0)};
    if (cls != SOLID) {
        if constexpr (IPM == 0) load_cell(g, A, P.stride, p);
        else load_cell_any<real, S, 1>(g, A, P, p, x, y, z, fl, (fl & SLOW_BIT) ? links[p] : 0u); // in-place streaming: the state lies at its destinations
        if (H) P.Fz += P.gbeta * stored_theta_shift(H, P.stride, p); // Boussinesq: the buoyancy the cell's collision used
        m = local_macros(g, cls, P, damp_at(P, x, y, z));
    }
    if (rho) rho[c] = out_t(m.rho);
    if (ux) ux[c] = out_t(m.ux);
    if (uy) uy[c] = out_t(m.uy);
    if (uz) uz[c] = out_t(m.uz);
}

template <typename real, typename out_t>
__global__ void mean_out_kernel(const real *__restrict__ msum, out_t *__restrict__ ux, out_t *__restrict__ uy, out_t *__restrict__ uz,
                                double inv_count, Params<real> P, const Box bx)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    int x, y, z;
    if (!box_cell(bx, c, x, y, z)) return;
    const int p = pidx(P, x, y, z);
    if (ux) ux[c] = out_t(double(msum[p]) * inv_count);
    if (uy) uy[c] = out_t(double(msum[P.stride + p]) * inv_count);
    if (uz) uz[c] = out_t(double(msum[2 * P.stride + p]) * inv_count);
}

// class bits only (SLOW / EDGE bits are internal)
template <typename real>
__global__ void flags_out_kernel(const uint8_t *__restrict__ flags, uint8_t *__restrict__ out, Params<real> P)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    int x, y, z;
    cell_xyz(P, c, x, y, z);
    out[c] = flags[pidx(P, x, y, z)] & CLASS_MASK;
}

template <typename real>
__global__ void links_out_kernel(const uint32_t *__restrict__ links, const uint8_t *__restrict__ flags, uint32_t *__restrict__ out,
                                 Params<real> P)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    int x, y, z;
    cell_xyz(P, c, x, y, z);
    const int p = pidx(P, x, y, z);
    out[c] = (flags[p] & CLASS_MASK) == FLUID ? links[p] : 0u; // SOLID cells keep an internal mailbox mask there
}

} // namespace lbmk
