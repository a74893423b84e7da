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
#include "lbm_inplace.cuh"

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
                HB[(long long)i * P.stride + (p - poff<i>(P) + xwrap<i>(P, x))] = v;
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

// Open faces (DESIGN.md §4 reading 27).  The face-velocity side array of the flow lattice (lbm_core.cuh: fu[2 halves][3][F]) has a
// thermal companion ft[2 halves][F] holding theta - theta_ref per face slot: an EQ_FIXED cell re-expands f_eq(1, u_b) and
// h_eq(theta_b, u_b) from its slot every step, an EQ_OUTFLOW cell f_eq(1, u) and h_eq(theta, u) of what its inward neighbour
// published while writing the previous state (u as in the plain kernel, theta = the neighbour's pulled theta, which its thermal
// collision conserves).  r = the half written together with the state being read, w = the half this launch writes.
template <typename real>
struct OpenFaces { const real *fur; real *fuw; const real *ftr; real *ftw; };

// DAMP: the open-boundary-stack instantiation, launched only while damping zones or inflow fluctuations are configured together
// with the thermal lattice, so the plain thermal kernel carries none of it:
//  * damping zones (lbm_set_damping): the relaxation acceleration sigma (u_t - u) and the buoyancy enter the same implicit
//    half-force solve (collide<real, true, true>; outside the zones sigma = 0 takes the undamped branch);
//  * synthetic inflow fluctuations (lbm_set_inflow_turbulence): the first turb_planes block rows carry the face slots, exactly as
//    in step_body (lbm_step.cuh) — the boundary velocity of the step after this one goes into the half of the side array this
//    launch writes; an EQ_FIXED cell re-expands BOTH equilibria from its slot's velocity every step, so its thermal state
//    follows u_b + u' with no further code (DESIGN.md §4 reading 28).  turb_planes = 0 while there are no modes.
// IP: the FLOW lattice streams in place (one buffer; lbm_inplace.cuh: loads through I.rd, every outgoing population over the
// address its opposite was read from, wall links through I.nx, ghost slots by slot and cell); the seven thermal populations
// stay double-buffered (they are 7 of 26 values per cell), so everything thermal below is the same in both schemes.
template <typename real, bool MEAN, int BLOCK, bool PERX, bool DAMP, bool IP>
__device__ __forceinline__ void thermal_step_body(real *__restrict__ B, real *__restrict__ HB, const uint8_t *__restrict__ flags,
                                                  const uint32_t *__restrict__ links, real *__restrict__ msum, const Params<real> &P,
                                                  const ThermalPtrs<real> &T, const OpenFaces<real> &O, const Turb<real> &tb,
                                                  const int turb_planes, const IpPtrs<real> &I)
{
    int zb = blockIdx.y;
    if constexpr (DAMP) {
        if (zb < turb_planes) {
            asm volatile("griddepcontrol.launch_dependents;");
            asm volatile("griddepcontrol.wait;" ::: "memory"); // the half written here is the one the previous launch reads
            const int s = (zb * (int)gridDim.x + (int)blockIdx.x) * BLOCK + (int)threadIdx.x;
            if (s < P.F) fluct_slot<real, false, real>(s, nullptr, nullptr, nullptr, O.fuw, nullptr, flags, tb, P);
            return;
        }
        zb -= turb_planes;
    }
    const unsigned c2 = blockIdx.x * BLOCK + threadIdx.x;
    if (c2 >= (unsigned)P.nxy) return;
    const int y = P.nx_magic ? (int)__umulhi(c2, P.nx_magic) : (int)(c2 / (unsigned)P.nx);
    const int x = (int)c2 - y * P.nx;
    const int z = zb == 0 ? P.nz - 1 : zb - 1; // the all-slow top plane first, not as the tail (lbm_step.cuh)
    const int p = pidx(P, x, y, z);
    asm volatile("griddepcontrol.launch_dependents;");   // programmatic dependent launch, as in step_body (lbm_step.cuh)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    int pL = p, pR = p; // PERX: read-side wrap of the pulls across periodic x faces (lbm_core.cuh xwrap), as in step_body
    if constexpr (PERX) {
        if (x == 0) pL = p + P.nx;
        if (x == P.nx - 1) pR = p - P.nx;
    }
    auto psrc = [&](auto ic) {
        constexpr int i = decltype(ic)::value;
        if constexpr (PERX && dir_cx(i) == 1) return pL;
        else if constexpr (PERX && dir_cx(i) == -1) return pR;
        else return p;
    };
    real g[Q], t[QT];
    auto ipat = [&](auto ic) { // IP: the cell index that goes with I.rd[i] / I.nx[i] (lbm_inplace.cuh)
        constexpr int i = decltype(ic)::value;
        if constexpr (PERX && i > 0 && (i & 1) == 0 && dir_cx(i) == -1) return pR;
        else return p;
    };
    // IP: the outgoing flow population j overwrites the address the incoming opp(j) was read from
    auto ip_store_all = [&]() {
        static_for<0, Q>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            I.rd[dir_opp(j)][ipat(std::integral_constant<int, dir_opp(j)>{})] = g[j];
        });
    };
    // as in step_kernel's SPEC instantiations: all 26 pulls are issued before the flag byte has arrived (no dependent
    // round trip; a SOLID cell then costs its reads), pinned by volatile asm so that the flag test cannot move above them
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        if constexpr (IP) g[i] = ld_pinned(I.rd[i] + ipat(ic));
        else g[i] = ld_pinned(T.gsrc[i] + psrc(ic));
    });
    static_for<0, QT>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        t[i] = ld_pinned(T.tsrc[i] + psrc(ic));
    });
    const uint8_t fl = ld_pinned(flags + p);
    // the collision pair of one FLUID cell: buoyancy from the pulled theta into the flow collision, thermal BGK towards
    // h_eq(theta, u) of that collision's velocity
    auto collide_both = [&]() {
        const real dth = theta_shift(t);
        Macro<real> m;
        if constexpr (DAMP) m = collide<real, true, true>(g, P, damp_at(P, x, y, z), P.gbeta * dth); // table look-ups: L1 / L2 resident
        else m = collide<real, false, true>(g, P, Damp<real>{}, P.gbeta * dth);
        real e[QT];
        thermal_equilibrium(e, dth, P.theta_ref, m.ux, m.uy, m.uz);
#pragma unroll
        for (int i = 0; i < QT; ++i) t[i] = t[i] - P.omega_t * (t[i] - e[i]);
        return m;
    };
    // ONE instance of the collision pair serves both paths (a second inlined copy put the body further beyond the instruction
    // cache): the link word of a wall-link / surface cell is requested first, so that it travels while the collision runs
    const int cls = fl & CLASS_MASK;
    uint32_t lk = 0;
    if (fl & (SLOW_BIT | SURF_BIT)) lk = links[p];
    Macro<real> m{real(1), real(0), real(0), real(0)};
    real dth = real(0); // the pulled theta: what a feeding cell publishes (its collision conserves it)
    if (cls == FLUID) {
        dth = theta_shift(t);
        m = collide_both();
    }
    // fast path, warp-uniform: every lane a plain FLUID cell (no wall link, no ghost slot, nothing to complete)
    if (__all_sync(__activemask(), fl == 0)) {
        if constexpr (IP) ip_store_all();
        else
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
    if (cls == SOLID) {
        // surface solid: completes the 32-byte sectors its live neighbours write, with zeros, in both lattices
        if (fl & SURF_BIT) {
            static_for<0, Q>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                if ((lk >> i) & 1u) {
                    if constexpr (!IP) B[(long long)i * P.stride + p] = real(0); // (in place: the flow sectors were read whole)
                    if constexpr (i < QT) HB[(long long)i * P.stride + p] = real(0);
                }
            });
        }
        return;
    }
    if (cls == FLUID) {
        if (fl & FEED_BIT)
            outflow_feed(P, x, y, z, m.ux, m.uy, m.uz, [&](int sl, int comp, real v) {
                O.fuw[comp * P.F + sl] = v;
                if (comp == 0) O.ftw[sl] = dth;
            });
    } else { // EQ_FIXED / EQ_OUTFLOW: both equilibria of the slot's (theta, u), re-stored every step like the plain kernel's EQ cells
        const int sl = eq_slot(P, cls, x, y, z);
        const real u0 = O.fur[sl], u1 = O.fur[P.F + sl], u2 = O.fur[2 * P.F + sl], db = O.ftr[sl];
        m = Macro<real>{real(1), u0, u1, u2};
        equilibrium(g, real(0), u0, u1, u2);
        thermal_equilibrium(t, db, P.theta_ref, u0, u1, u2);
    }
    // own slots and wall mailboxes of both lattices (store_cell / store_cell_thermal with the EDGE part masked off), then ONE
    // ghost-store sequence for both: the face logic per direction is shared, which halves that code (the fused body is larger
    // than the instruction cache)
    if constexpr (IP) {
        ip_store_all(); // towards a dead cell this fills the link's unused slot
        if (fl & SLOW_BIT)
            static_for<1, Q>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                if ((lk >> i) & 1u) I.nx[i][ipat(ic)] = g[dir_opp(i)];
            });
    } else store_cell(B, P, p, x, y, z, (uint8_t)(fl & ~EDGE_BIT), lk, g);
    store_cell_thermal(HB, P, p, x, y, z, (uint8_t)(fl & ~EDGE_BIT), lk, t);
    if (fl & EDGE_BIT)
        ghost_stores(P, x, y, z, lk, [&](int i, int pt, auto jc) {
            constexpr int j = decltype(jc)::value;
            if constexpr (IP) { // ghost slot (i, pt) = "cell pt + c_i receives direction i" (lbm_core.cuh ip_visit)
                int cell = pt;
                if (i & 1) cell = pt + poff_rt(P, i) + ((dir_cx(i) == 1 && P.perx && x == P.nx - 1) ? -P.nx : 0);
                I.G[(long long)ip_slot(I.qn, i) * P.stride + cell] = g[j];
            } else B[(long long)i * P.stride + pt] = g[j];
            if constexpr (j < QT) HB[(long long)i * P.stride + pt] = t[j]; // an axis direction reflects into an axis direction
        });
    if constexpr (MEAN) {
        msum[p] += m.ux;
        msum[P.stride + p] += m.uy;
        msum[2 * P.stride + p] += m.uz;
    }
}

template <typename real, bool MEAN, int BLOCK, int MINB, bool PERX = false, bool DAMP = false>
__global__ void __launch_bounds__(BLOCK, MINB)
thermal_step_kernel(real *__restrict__ B, real *__restrict__ HB, const uint8_t *__restrict__ flags, const uint32_t *__restrict__ links,
                    real *__restrict__ msum, const Params<real> P, const ThermalPtrs<real> T, const OpenFaces<real> O,
                    const Turb<real> tb = Turb<real>{}, const int turb_planes = 0)
{
    IpPtrs<real> none; // not touched by the two-buffer instantiation
    thermal_step_body<real, MEAN, BLOCK, PERX, DAMP, false>(B, HB, flags, links, msum, P, T, O, tb, turb_planes, none);
}

// the same step with the flow lattice on ONE buffer (lbm_create_ex precision | LBM_STREAM_INPLACE)
template <typename real, bool MEAN, int BLOCK, int MINB, bool PERX, bool DAMP>
__global__ void __launch_bounds__(BLOCK, MINB)
ip_thermal_step_kernel(real *__restrict__ HB, const uint8_t *__restrict__ flags, const uint32_t *__restrict__ links, real *__restrict__ msum,
                       const Params<real> P, const ThermalPtrs<real> T, const OpenFaces<real> O, const Turb<real> tb, const int turb_planes,
                       const IpPtrs<real> I)
{
    thermal_step_body<real, MEAN, BLOCK, PERX, DAMP, true>(nullptr, HB, flags, links, msum, P, T, O, tb, turb_planes, I);
}

// Publish what a feeding cell (one layer inside an EQ_OUTFLOW face) hands to the outflow cells for the next step, from the
// CURRENT states A (flow) and its thermal shift dth: the local velocity with the cell's buoyancy in the force, and theta; both
// halves of both side arrays (set-up paths).
template <typename real>
__device__ __forceinline__ void thermal_feed_both(const real *__restrict__ A, real *__restrict__ fu, real *__restrict__ ft, Params<real> P,
                                                  int p, int x, int y, int z, int cls, real dth, uint8_t fl, uint32_t lk)
{
    real g[Q];
    load_cell_any(g, A, P, p, x, y, z, fl, (fl & SLOW_BIT) ? lk : 0u); // the flow state, whichever streaming scheme holds it
    P.Fz += P.gbeta * dth;
    const Macro<real> m = local_macros(g, cls, P, damp_at(P, x, y, z));
    outflow_feed(P, x, y, z, m.ux, m.uy, m.uz, [&](int sl, int comp, real v) {
        fu[comp * P.F + sl] = v;
        fu[(3 + comp) * P.F + sl] = v;
        if (comp == 0) { ft[sl] = dth; ft[P.F + sl] = dth; }
    });
}

// H0 = h_eq(theta0, u0) into both buffers (lbm_set_theta); NULL theta = theta_ref, NULL component = 0.  FLUID and EQ_OUTFLOW
// cells; EQ_FIXED cells keep their boundary state h_eq(theta_b, u_b) (as lbm_set_macros keeps f_eq(1, u_b)).
template <typename real, typename in_t>
__global__ void thermal_init_kernel(real *__restrict__ HA, real *__restrict__ HB, const uint8_t *__restrict__ flags,
                                    const uint32_t *__restrict__ links, const in_t *__restrict__ theta, const in_t *__restrict__ ux,
                                    const in_t *__restrict__ uy, const in_t *__restrict__ uz, Params<real> P,
                                    const real *__restrict__ A, real *__restrict__ fu, real *__restrict__ ft)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    int x, y, z;
    cell_xyz(P, c, x, y, z);
    const int p = pidx(P, x, y, z);
    const uint8_t fl = flags[p];
    const int cls = fl & CLASS_MASK;
    if (cls != FLUID && cls != EQ_OUTFLOW) return;
    // theta - theta_ref formed in the input's precision (FP64 input on an FP32 handle keeps the small perturbation)
    const real dth = theta ? real(theta[c] - in_t(P.theta_ref)) : real(0);
    real t[QT];
    thermal_equilibrium(t, dth, P.theta_ref, ux ? real(ux[c]) : real(0), uy ? real(uy[c]) : real(0), uz ? real(uz[c]) : real(0));
    const uint32_t lk = links[p];
    store_cell_thermal(HA, P, p, x, y, z, fl, lk, t);
    store_cell_thermal(HB, P, p, x, y, z, fl, lk, t);
    if ((fl & FEED_BIT) && P.F > 0) thermal_feed_both(A, fu, ft, P, p, x, y, z, cls, dth, fl, lk);
}

// Prescribed temperature of the EQ_FIXED cells (lbm_set_inlet_theta; reading 27): one thread per face slot; theta_b[nz] by level,
// or NULL = keep the slot's value (refresh after the boundary velocity changed, or after lbm_set_thermal).  Writes the slot
// (both halves) and the cell's thermal state h_eq(theta_b, u_b) in both buffers, u_b from the flow's side array.
template <typename real, typename in_t>
__global__ void thermal_inlet_kernel(real *__restrict__ HA, real *__restrict__ HB, const uint8_t *__restrict__ flags,
                                     const in_t *__restrict__ theta_b, const real *__restrict__ fu, real *__restrict__ ft, Params<real> P)
{
    const int sl = blockIdx.x * blockDim.x + threadIdx.x;
    int k, x, y, z;
    if (sl >= P.F || !fixed_slot_cell(P, flags, sl, k, x, y, z)) return;
    const real dth = theta_b ? real(theta_b[z] - in_t(P.theta_ref)) : ft[sl];
    ft[sl] = dth; ft[P.F + sl] = dth;
    real t[QT];
    thermal_equilibrium(t, dth, P.theta_ref, fu[sl], fu[P.F + sl], fu[2 * P.F + sl]);
    const int p = pidx(P, x, y, z);
    store_cell_thermal(HA, P, p, x, y, z, flags[p], 0u, t);
    store_cell_thermal(HB, P, p, x, y, z, flags[p], 0u, t);
}

// ---- checkpoint of the thermal lattice (lbm_get_thermal_state / lbm_set_thermal_state) -----------------------------------
// h [7][nz][ny][nx] double, NOT shifted; SOLID cells export the rest state wT_i theta_ref and ignore their input; EQ_FIXED
// cells export their boundary state and keep it on input (it belongs to the prescribed theta_b, u_b).
__host__ __device__ inline double weight_t_f64(int i) { return i == 0 ? 0.25 : 0.125; }

template <typename real>
__global__ void thermal_state_out_kernel(const real *__restrict__ H, const uint8_t *__restrict__ flags, double *__restrict__ h, Params<real> P)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    int x, y, z;
    cell_xyz(P, c, x, y, z);
    const int p = pidx(P, x, y, z);
    const bool live = (flags[p] & CLASS_MASK) != SOLID;
#pragma unroll
    for (int i = 0; i < QT; ++i)
        h[(long long)i * P.N + c] = (live ? double(H[(long long)i * P.stride + p]) : 0.0) + weight_t_f64(i) * double(P.theta_ref);
}

template <typename real>
__global__ void thermal_state_in_kernel(real *__restrict__ HA, real *__restrict__ HB, const uint8_t *__restrict__ flags,
                                        const uint32_t *__restrict__ links, const double *__restrict__ h, Params<real> P,
                                        const real *__restrict__ A, real *__restrict__ fu, real *__restrict__ ft)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    int x, y, z;
    cell_xyz(P, c, x, y, z);
    const int p = pidx(P, x, y, z);
    const uint8_t fl = flags[p];
    const int cls = fl & CLASS_MASK;
    if (cls != FLUID && cls != EQ_OUTFLOW) return;
    real t[QT];
#pragma unroll
    for (int i = 0; i < QT; ++i) t[i] = real(h[(long long)i * P.N + c] - weight_t_f64(i) * double(P.theta_ref));
    const uint32_t lk = links[p];
    store_cell_thermal(HA, P, p, x, y, z, fl, lk, t);
    store_cell_thermal(HB, P, p, x, y, z, fl, lk, t);
    if ((fl & FEED_BIT) && P.F > 0) thermal_feed_both(A, fu, ft, P, p, x, y, z, cls, theta_shift(t), fl, lk);
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
    const bool live = (flags[p] & CLASS_MASK) != SOLID;
    theta[c] = out_t(P.theta_ref) + (live ? out_t(theta_shift(t)) : out_t(0));
}

} // namespace lbmk
