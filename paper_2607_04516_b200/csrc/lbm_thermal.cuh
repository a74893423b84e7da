// lbm_thermal.cuh — SURVEY.md §8(f) rank 3: the D3Q7 thermal lattice with Boussinesq coupling (Table 1
// "Optional D3Q7 or D3Q19 thermal lattice with Boussinesq coupling"; density-current workload PAPER.md:121;
// DESIGN.md §4 reading 23), fused with the flow step: ONE kernel pulls the 19 flow and the 7 thermal populations,
// forms theta, adds g beta (theta - theta_ref) e_z to the body force of the flow collision, relaxes the thermal
// populations towards h_eq(theta, u) of that collision's velocity, and stores both.
//
// The seven thermal directions are directions 0..6 of the flow lattice, and the thermal populations live on the same
// halo-padded box (lbm_core.cuh) with the same write-side boundary rule: a population that leaves towards a SOLID /
// WALL target goes into the bounce-back mailbox, towards a FREE_SLIP ghost into the mirrored slot (both = zero heat
// flux), towards a PERIODIC ghost into the far halo.  So the read side is again a pure gather, the link word of the
// cell serves both lattices (bits 1..6), and the sector-completion mask of a surface solid is valid for both.
// Stored shifted: t_i = h_i - wT_i theta_ref (an isothermal state at rest is exactly 0).
// Traffic per FLUID cell: (19 + 7) x 4 B read + (19 + 7) x 4 B write + 1 flag byte = 209 B.
#pragma once
#include "lbm_core.cuh"
#include "lbm_step.cuh"

namespace lbmk {

constexpr int QT = 7;

// theta - theta_ref of a stored / pulled thermal state
template <typename real>
__device__ __forceinline__ real theta_shift(const real (&t)[QT])
{
    return t[0] + ((t[1] + t[2]) + (t[3] + t[4]) + (t[5] + t[6]));
}

// shifted linear equilibrium: wT_i (dth + 4 theta c_i.u), wT_0 = 1/4, wT_1..6 = 1/8, c_sT^2 = 1/4
template <typename real>
__device__ __forceinline__ void thermal_equilibrium(real (&e)[QT], real dth, real theta_ref, real ux, real uy, real uz)
{
    const real th = theta_ref + dth;
    const real a = real(0.125) * dth;
    const real bx = real(0.5) * th * ux, by = real(0.5) * th * uy, bz = real(0.5) * th * uz;
    e[0] = real(0.25) * dth;
    e[1] = a + bx; e[2] = a - bx;
    e[3] = a + by; e[4] = a - by;
    e[5] = a + bz; e[6] = a - bz;
}

// all stores of one cell's thermal state: own 7 slots, wall mailboxes (bits 1..6 of the link word), ghost slots
template <typename real>
__device__ __forceinline__ void store_cell_thermal(real *__restrict__ HB, const Params<real> &P, int p, int x, int y, int z, uint8_t fl,
                                                   uint32_t lk, const real (&t)[QT])
{
#pragma unroll
    for (int i = 0; i < QT; ++i) HB[(long long)i * P.stride + p] = t[i];
    if (fl & SLOW_BIT) {
        // pull direction i = 1..6 crosses face k = i - 1 when the cell lies on it (1: x-, 2: x+, 3: y-, 4: y+, 5: z-, 6: z+).
        // A WALL face held at theta_w returns the population anti-bounced: -t_j + 2 wT_j (theta_w - theta_ref), wT_j = 1/8
        // (DESIGN.md §4 reading 26); every other wall link (buildings, adiabatic walls) bounces it back unchanged.
        static_for<1, QT>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            if ((lk >> i) & 1u) {
                real v = t[dir_opp(i)];
                if (P.thd) { // rare: only handles with held walls pay for the test
                    const bool at = i == 1 ? x == 0 : i == 2 ? x == P.nx - 1 : i == 3 ? y == 0 : i == 4 ? y == P.ny - 1 : i == 5 ? z == 0 : z == P.nz - 1;
                    if (at && ((P.thd >> (i - 1)) & 1)) v = real(0.125) * P.thw[i - 1] - v;
                }
                HB[(long long)i * P.stride + (p - poff<i>(P))] = v;
            }
        });
    }
    if (fl & EDGE_BIT)
        ghost_stores(P, x, y, z, lk, [&](int i, int pt, auto jc) {
            constexpr int j = decltype(jc)::value;
            if constexpr (j < QT) HB[(long long)i * P.stride + pt] = t[j]; // an axis direction reflects into an axis direction
        });
}

// Per-launch address table of the 26 streams, as StepPtrs for the plain kernel: src = buffer + i stride - off_i (the pull of
// direction i is src[i][p]), dst = buffer + i stride.  One 64-bit add per access instead of a 64-bit multiply-add chain.
template <typename real>
struct ThermalPtrs {
    const real *gsrc[Q];
    real *gdst[Q];
    const real *tsrc[QT];
    real *tdst[QT];
};
template <typename real>
inline ThermalPtrs<real> make_thermal_ptrs(const real *A, real *B, const real *HA, real *HB, const Params<real> &P)
{
    ThermalPtrs<real> t;
    for (int i = 0; i < Q; ++i) {
        const long long off = dir_cx(i) + (long long)dir_cy(i) * P.px + (long long)dir_cz(i) * P.pxy;
        t.gsrc[i] = A + ((long long)i * P.stride - off);
        t.gdst[i] = B + (long long)i * P.stride;
        if (i < QT) {
            t.tsrc[i] = HA + ((long long)i * P.stride - off);
            t.tdst[i] = HB + (long long)i * P.stride;
        }
    }
    return t;
}

template <typename real, bool MEAN, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB)
thermal_step_kernel(real *__restrict__ B, real *__restrict__ HB, const uint8_t *__restrict__ flags, const uint32_t *__restrict__ links,
                    real *__restrict__ msum, const Params<real> P, const ThermalPtrs<real> T)
{
    const unsigned c2 = blockIdx.x * BLOCK + threadIdx.x;
    if (c2 >= (unsigned)P.nxy) return;
    const int y = P.nx_magic ? (int)__umulhi(c2, P.nx_magic) : (int)(c2 / (unsigned)P.nx);
    const int x = (int)c2 - y * P.nx;
    const int z = blockIdx.y == 0 ? P.nz - 1 : (int)blockIdx.y - 1; // the all-slow top plane first, not as the tail (lbm_step.cuh)
    const int p = pidx(P, x, y, z);
    // as in step_kernel's SPEC instantiations: all 26 pulls are issued before the flag byte has arrived (no dependent
    // round trip; a SOLID cell then costs its reads), pinned by volatile asm so that the flag test cannot move above them
    real g[Q], t[QT];
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        g[i] = ld_pinned(T.gsrc[i] + p);
    });
    static_for<0, QT>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        t[i] = ld_pinned(T.tsrc[i] + p);
    });
    const uint8_t fl = ld_pinned(flags + p);
    // the collision pair of one FLUID cell: buoyancy from the pulled theta into the flow collision, thermal BGK towards
    // h_eq(theta, u) of that collision's velocity
    auto collide_both = [&]() {
        const real dth = theta_shift(t);
        const Macro<real> m = collide<real, false, true>(g, P, Damp<real>{}, P.gbeta * dth);
        real e[QT];
        thermal_equilibrium(e, dth, P.theta_ref, m.ux, m.uy, m.uz);
#pragma unroll
        for (int i = 0; i < QT; ++i) t[i] = t[i] - P.omega_t * (t[i] - e[i]);
        return m;
    };
    // fast path, warp-uniform: every lane a plain FLUID cell (no wall link, no ghost slot, nothing to complete)
    if (__all_sync(__activemask(), fl == 0)) {
        const Macro<real> m = collide_both();
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            T.gdst[i][p] = g[i];
        });
        static_for<0, QT>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            T.tdst[i][p] = t[i];
        });
        if constexpr (MEAN) {
            msum[p] += m.ux;
            msum[P.stride + p] += m.uy;
            msum[2 * P.stride + p] += m.uz;
        }
        return;
    }
    const int cls = fl & CLASS_MASK;
    uint32_t lk = 0;
    if (fl & (SLOW_BIT | SURF_BIT)) lk = links[p];
    if (cls == SOLID) {
        // surface solid: completes the 32-byte sectors its live neighbours write, with zeros, in both lattices
        if (fl & SURF_BIT) {
            static_for<0, Q>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                if ((lk >> i) & 1u) {
                    B[(long long)i * P.stride + p] = real(0);
                    if constexpr (i < QT) HB[(long long)i * P.stride + p] = real(0);
                }
            });
        }
        return;
    }
    if (cls != FLUID) return; // no EQ cells while the thermal lattice is on (lbm_set_thermal refuses EQ faces)
    const Macro<real> m = collide_both();
    store_cell(B, P, p, x, y, z, fl, lk, g);
    store_cell_thermal(HB, P, p, x, y, z, fl, lk, t);
    if constexpr (MEAN) {
        msum[p] += m.ux;
        msum[P.stride + p] += m.uy;
        msum[2 * P.stride + p] += m.uz;
    }
}

// H0 = h_eq(theta0, u0) into both buffers (lbm_set_theta); NULL theta = theta_ref, NULL component = 0
template <typename real, typename in_t>
__global__ void thermal_init_kernel(real *__restrict__ HA, real *__restrict__ HB, const uint8_t *__restrict__ flags,
                                    const uint32_t *__restrict__ links, const in_t *__restrict__ theta, const in_t *__restrict__ ux,
                                    const in_t *__restrict__ uy, const in_t *__restrict__ uz, Params<real> P)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    int x, y, z;
    cell_xyz(P, c, x, y, z);
    const int p = pidx(P, x, y, z);
    const uint8_t fl = flags[p];
    if ((fl & CLASS_MASK) != FLUID) return;
    // theta - theta_ref formed in the input's precision (FP64 input on an FP32 handle keeps the small perturbation)
    const real dth = theta ? real(theta[c] - in_t(P.theta_ref)) : real(0);
    real t[QT];
    thermal_equilibrium(t, dth, P.theta_ref, ux ? real(ux[c]) : real(0), uy ? real(uy[c]) : real(0), uz ? real(uz[c]) : real(0));
    const uint32_t lk = links[p];
    store_cell_thermal(HA, P, p, x, y, z, fl, lk, t);
    store_cell_thermal(HB, P, p, x, y, z, fl, lk, t);
}

// ---- checkpoint of the thermal lattice (lbm_get_thermal_state / lbm_set_thermal_state) -----------------------------------
// h [7][nz][ny][nx] double, NOT shifted; non-FLUID cells export the rest state wT_i theta_ref and ignore their input.
__host__ __device__ inline double weight_t_f64(int i) { return i == 0 ? 0.25 : 0.125; }

template <typename real>
__global__ void thermal_state_out_kernel(const real *__restrict__ H, const uint8_t *__restrict__ flags, double *__restrict__ h, Params<real> P)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    int x, y, z;
    cell_xyz(P, c, x, y, z);
    const int p = pidx(P, x, y, z);
    const bool live = (flags[p] & CLASS_MASK) == FLUID;
#pragma unroll
    for (int i = 0; i < QT; ++i)
        h[(long long)i * P.N + c] = (live ? double(H[(long long)i * P.stride + p]) : 0.0) + weight_t_f64(i) * double(P.theta_ref);
}

template <typename real>
__global__ void thermal_state_in_kernel(real *__restrict__ HA, real *__restrict__ HB, const uint8_t *__restrict__ flags,
                                        const uint32_t *__restrict__ links, const double *__restrict__ h, Params<real> P)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    int x, y, z;
    cell_xyz(P, c, x, y, z);
    const int p = pidx(P, x, y, z);
    const uint8_t fl = flags[p];
    if ((fl & CLASS_MASK) != FLUID) return;
    real t[QT];
#pragma unroll
    for (int i = 0; i < QT; ++i) t[i] = real(h[(long long)i * P.N + c] - weight_t_f64(i) * double(P.theta_ref));
    const uint32_t lk = links[p];
    store_cell_thermal(HA, P, p, x, y, z, fl, lk, t);
    store_cell_thermal(HB, P, p, x, y, z, fl, lk, t);
}

// theta of the stored state (lbm_get_theta); SOLID cells report theta_ref
template <typename real, typename out_t>
__global__ void theta_out_kernel(const real *__restrict__ H, const uint8_t *__restrict__ flags, out_t *__restrict__ theta, Params<real> P)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    int x, y, z;
    cell_xyz(P, c, x, y, z);
    const int p = pidx(P, x, y, z);
    real t[QT];
#pragma unroll
    for (int i = 0; i < QT; ++i) t[i] = H[(long long)i * P.stride + p];
    const bool live = (flags[p] & CLASS_MASK) == FLUID;
    theta[c] = out_t(P.theta_ref) + (live ? out_t(theta_shift(t)) : out_t(0));
}

} // namespace lbmk
