// lbm_step.cuh — a5/a6 (+ the fused part of a7): the per-step fused stream-collide kernel for sm_100a.
//
// One cell per thread, threads linear over the interior cells of one z plane (a warp = 32 consecutive interior cells,
// at most two contiguous row segments; no idle lanes).  Every FLUID cell pulls A[i][p - off_i] for all 19 directions with
// no case distinction: bounce-back, free-slip and periodic faces were resolved by the WRITER of the previous step
// (lbm_core.cuh, "mailboxes"), so the read side is a pure 19-stream gather and the only divergent code is a few
// extra predicated stores in cells that have a wall link or lie on a domain face.
// Traffic per FLUID cell: 19 x 4 B read + 19 x 4 B write + 1 flag byte (+ 4 B link word only where SLOW_BIT is set).
//
// SPEC: issue the 19 population loads before the flag byte has arrived (no dependent round trip; SOLID cells then
//       cost their 76 B of reads).  The FP32 product kernels are SPEC; the FP64 reference twin is not.
// TURB: the launch carries the synthetic inflow fluctuations in extra leading block rows (lbm_set_inflow_turbulence).
// DAMP: the damping-zone instantiation (lbm_set_damping); launched only while zones are configured, so the plain
//       kernel carries none of it.
#pragma once
#include "lbm_core.cuh"
#include "lbm_setup.cuh"
#include <cooperative_groups.h>

namespace lbmk {

// A load the compiler may not sink below a later branch (volatile asm keeps its place): the 19 pulls of the
// speculative kernels are issued before the flag byte is tested.
__device__ __forceinline__ float ld_pinned(const float *p)
{
    float v;
    asm volatile("ld.volatile.global.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ double ld_pinned(const double *p)
{
    double v;
    asm volatile("ld.volatile.global.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ float ld_pinned(const __half *p)
{
    unsigned short v;
    asm volatile("ld.volatile.global.u16 %0, [%1];" : "=h"(v) : "l"(p));
    return __half2float(__ushort_as_half(v));
}
__device__ __forceinline__ uint8_t ld_pinned(const uint8_t *p)
{
    uint32_t v;
    asm volatile("ld.global.u8 %0, [%1];" : "=r"(v) : "l"(p));
    return (uint8_t)v;
}

// Per-launch address table: src[i] = A + i stride - off_i (so the pull of direction i is src[i][p]), dst[i] = B + i stride.
// One 64-bit multiply-add per access instead of rebuilding i * stride - off_i in every thread.
template <typename S>
struct StepPtrs {
    const S *src[Q];
    S *dst[Q];
};
template <typename S, typename real>
inline StepPtrs<S> make_step_ptrs(const S *A, S *B, const Params<real> &P)
{
    StepPtrs<S> t;
    for (int i = 0; i < Q; ++i) {
        const long long off = dir_cx(i) + (long long)dir_cy(i) * P.px + (long long)dir_cz(i) * P.pxy;
        t.src[i] = A + ((long long)i * P.stride - off);
        t.dst[i] = B + (long long)i * P.stride;
    }
    return t;
}

// The step of one thread (one cell, or one face slot in a TURB block row).  A plain device function so that it can be
// called once per launch (step_kernel) or in a loop with grid-wide barriers (step_loop_kernel, lattices that fit L2).
template <typename real, typename S, bool MEAN, bool SPEC, int BLOCK, bool DAMP, bool TURB, bool PERX>
__device__ __forceinline__ void step_body(const S *__restrict__ A, S *__restrict__ B, const uint8_t *__restrict__ flags,
                                          const uint32_t *__restrict__ links, real *__restrict__ msum, const real *__restrict__ fur,
                                          real *__restrict__ fuw, const Params<real> &P, const StepPtrs<S> &T, const Turb<real> &tb,
                                          const int turb_planes)
{
    int zb = blockIdx.y;
    if constexpr (TURB) {
        // the first turb_planes block rows carry the inflow fluctuations instead of lattice cells: one thread per face slot,
        // boundary velocity of the step AFTER this one (tb.t) into the half this launch writes — the EQ_FIXED cells of the
        // next launch read it from there.  They are dispatched first and run beside the memory-bound lattice blocks.
        if (zb < turb_planes) {
            asm volatile("griddepcontrol.launch_dependents;");
            asm volatile("griddepcontrol.wait;" ::: "memory"); // the half written here is the one the previous launch reads
            const int s = (zb * (int)gridDim.x + (int)blockIdx.x) * BLOCK + (int)threadIdx.x;
            if (s < P.F) fluct_slot<real, false, S>(s, nullptr, nullptr, nullptr, fuw, nullptr, flags, tb, P);
            return;
        }
        zb -= turb_planes;
    }
    const unsigned c2 = blockIdx.x * BLOCK + threadIdx.x; // cell of the z plane, linear over interior (y, x)
    if (c2 >= (unsigned)P.nxy) return;
    const int y = P.nx_magic ? (int)__umulhi(c2, P.nx_magic) : (int)(c2 / (unsigned)P.nx);
    const int x = (int)c2 - y * P.nx;
    // Block rows are dispatched in order; the planes whose cells all take the slow path (the top plane under a FREE_SLIP /
    // PERIODIC lid: a ghost store sequence per cell) must not be the tail of the launch, where nothing is left to overlap
    // them with: the last plane goes first, everything else one later.
    const int z = zb == 0 ? P.nz - 1 : zb - 1;
    const int p = pidx(P, x, y, z);
    // Programmatic dependent launch: the next step's launch may be set up while this one drains (launch_dependents, issued at
    // once: the dependent grid is admitted only when every CTA of this one has started), and this grid's threads do their
    // index arithmetic before the previous step has finished — but touch no memory until it has (wait).  Both are no-ops for
    // a launch without the attribute.
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    // PERX (both x faces PERIODIC): the pulls with c_x = +1 / -1 of the first / last cell of a row wrap to the other end of
    // their source row (lbm_core.cuh xwrap); an instantiation of its own, so that the other lattices carry no second index
    int pL = p, pR = p;
    if constexpr (PERX) {
        if (x == 0) pL = p + P.nx;
        if (x == P.nx - 1) pR = p - P.nx;
    }
    auto psrc = [&](auto ic) { // cell index of the pull source slot of direction i, before the table's - off_i
        constexpr int i = decltype(ic)::value;
        if constexpr (PERX && dir_cx(i) == 1) return pL;
        else if constexpr (PERX && dir_cx(i) == -1) return pR;
        else return p;
    };

    real g[Q];
    uint8_t fl;
    real fu0 = real(0), fu1 = real(0), fu2 = real(0); // face velocity of an EQ cell
    real ms0 = real(0), ms1 = real(0), ms2 = real(0); // running mean sums (MEAN && SPEC: prefetched)
    Damp<real> dmp{real(0), real(0), real(0), real(0)}; // damping coefficient / target of the cell (DAMP && SPEC: prefetched)
    if constexpr (SPEC) {
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            g[i] = real(ld_pinned(T.src[i] + psrc(ic)));
        });
        // a cell on an EQ face fetches its face velocity now, from geometry alone (EQ_FIXED wins, as in the voxeliser);
        // if the flag then says SOLID the three values are simply not used
        // (one unsigned compare per axis: c - 1 >= n - 2 <=> c == 0 or c == n - 1; interior warps skip the owner search)
        const bool onface = ((unsigned)(x - 1) >= (unsigned)(P.nx - 2)) | ((unsigned)(y - 1) >= (unsigned)(P.ny - 2)) |
                            ((unsigned)(z - 1) >= (unsigned)(P.nz - 2));
        if (P.F > 0 && onface) {
            int k = eq_owner(P, FACE_EQ_FIXED, x, y, z);
            if (k < 0) k = eq_owner(P, FACE_EQ_OUTFLOW, x, y, z);
            if (k >= 0) {
                const int sl = outflow_slot(P, k, x, y, z);
                fu0 = ld_pinned(fur + sl); fu1 = ld_pinned(fur + P.F + sl); fu2 = ld_pinned(fur + 2 * P.F + sl);
            }
        }
        // sampling steps: the three running sums are fetched with the pulls (their latency hides behind the collision
        // instead of a dependent read-modify-write at the end; SOLID cells simply do not use them)
        if constexpr (DAMP) dmp = damp_at(P, x, y, z); // table look-ups in flight with the pulls
        if constexpr (MEAN) { ms0 = ld_pinned(msum + p); ms1 = ld_pinned(msum + P.stride + p); ms2 = ld_pinned(msum + 2 * P.stride + p); }
        fl = ld_pinned(flags + p); // volatile asm statements keep their order: the flag test cannot move above the pulls
    } else {
        fl = flags[p];
    }
    if constexpr (SPEC) {
        // Fast path, warp-uniform: every lane a plain FLUID cell (no wall link, no ghost slot, nothing to complete) — the
        // bulk of the lattice — or an EQ cell / a feeding cell without wall link or ghost slot (the inlet and outflow cells
        // at the two ends of every row).  Straight-line collide (or equilibrium re-expansion) + 19 stores, none of the
        // per-feature tests below.
        const bool plain = (fl & (SLOW_BIT | EDGE_BIT | SURF_BIT)) == 0 && (fl & CLASS_MASK) != SOLID && (fl & CLASS_MASK) != GHOST;
        if (__all_sync(__activemask(), plain)) {
            Macro<real> m;
            if ((fl & CLASS_MASK) == FLUID) {
                if constexpr (DAMP) m = collide<real, true>(g, P, dmp);
                else m = collide(g, P);
            } else {
                m = Macro<real>{real(1), fu0, fu1, fu2};
                equilibrium(g, real(0), fu0, fu1, fu2);
            }
            static_for<0, Q>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                st_s(T.dst[i] + p, g[i]);
            });
            if (fl & FEED_BIT) outflow_feed(P, x, y, z, m.ux, m.uy, m.uz, [&](int sl, int comp, real v) { fuw[comp * P.F + sl] = v; });
            if constexpr (MEAN) {
                msum[p] = ms0 + m.ux;
                msum[P.stride + p] = ms1 + m.uy;
                msum[2 * P.stride + p] = ms2 + m.uz;
            }
            return;
        }
    }
    const int cls = fl & CLASS_MASK;
    // link word: wall links of a FLUID cell / zero-fill mask of a surface SOLID cell; one predicated load for both,
    // issued as soon as the flag is there and consumed only after the collision
    uint32_t lk = 0;
    if (fl & (SLOW_BIT | SURF_BIT)) lk = links[p];
    if (cls == SOLID && !(fl & SURF_BIT)) return;
    Macro<real> m{real(1), real(0), real(0), real(0)};
    const bool merged_solid = cls == SOLID; // a surface solid: it only completes sectors, with zeros
    if (merged_solid) {
#pragma unroll
        for (int i = 0; i < Q; ++i) g[i] = real(0);
    }
    if (cls == FLUID) {
        if constexpr (!SPEC) {
            static_for<0, Q>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                g[i] = ld_s<real>(T.src[i] + psrc(ic));
            });
        }
        if constexpr (DAMP) m = collide<real, true>(g, P, SPEC ? dmp : damp_at(P, x, y, z));
        else m = collide(g, P);
    } else if (cls != SOLID) { // EQ_FIXED (a3) / EQ_OUTFLOW (a6): f_eq(1, u) of the cell's face velocity (lbm_core.cuh)
        if constexpr (!SPEC) {
            const int sl = eq_slot(P, cls, x, y, z);
            fu0 = fur[sl]; fu1 = fur[P.F + sl]; fu2 = fur[2 * P.F + sl];
        }
        m = Macro<real>{real(1), fu0, fu1, fu2};
        equilibrium(g, real(0), m.ux, m.uy, m.uz);
    }
    // ONE store sequence for the whole warp.  A surface solid takes part in it with zeros, predicated by its completion
    // mask: a solid cell whose 32-byte sector is written by others (live cells, neighbours' mailboxes) completes it, so
    // that the sector leaves L2 fully written — no DRAM read-modify-write, same bytes written either way.  Warps without
    // such a lane (the common case, a warp-uniform branch) store unpredicated.  A second, divergent store sequence for
    // the solid lanes cost 2 % of the step.
    const uint32_t wm = merged_solid ? lk : 0x7FFFFu;
    if (__any_sync(__activemask(), merged_solid)) {
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            if ((wm >> i) & 1u) st_s(T.dst[i] + p, g[i]);
        });
    } else {
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            st_s(T.dst[i] + p, g[i]);
        });
    }
    if (merged_solid) return;
    if (fl & SLOW_BIT) {
        // wall links (lbm_core.cuh wall_stores, with the launch's address table): slot (i, p - off_i) <- g[opp(i)]
        static_for<1, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            if ((lk >> i) & 1u) st_s(T.dst[i] + (psrc(ic) - poff<i>(P)), g[dir_opp(i)]);
        });
    }
    if (fl & EDGE_BIT)
        ghost_stores(P, x, y, z, lk, [&](int i, int pt, auto jc) { st_s(B + ((long long)i * P.stride + pt), g[decltype(jc)::value]); });
    if (fl & FEED_BIT) outflow_feed(P, x, y, z, m.ux, m.uy, m.uz, [&](int sl, int comp, real v) { fuw[comp * P.F + sl] = v; });
    if constexpr (MEAN) {
        if constexpr (SPEC) {
            msum[p] = ms0 + m.ux;
            msum[P.stride + p] = ms1 + m.uy;
            msum[2 * P.stride + p] = ms2 + m.uz;
        } else {
            msum[p] += m.ux;
            msum[P.stride + p] += m.uy;
            msum[2 * P.stride + p] += m.uz;
        }
    }
}

template <typename real, typename S, bool MEAN, bool SPEC, int BLOCK, int MINB, bool DAMP = false, bool TURB = false, bool PERX = false>
__global__ void __launch_bounds__(BLOCK, MINB)
step_kernel(const S *__restrict__ A, S *__restrict__ B, const uint8_t *__restrict__ flags, const uint32_t *__restrict__ links,
            real *__restrict__ msum, const real *__restrict__ fur, real *__restrict__ fuw, const Params<real> P, const StepPtrs<S> T,
            const Turb<real> tb = Turb<real>{}, const int turb_planes = 0)
{
    step_body<real, S, MEAN, SPEC, BLOCK, DAMP, TURB, PERX>(A, B, flags, links, msum, fur, fuw, P, T, tb, turb_planes);
}

// Several steps in ONE cooperative launch, a grid-wide barrier between them: for lattices whose whole grid is resident
// at once (<= 10 CTAs x 148 SMs x 128 cells; config 1) a step is a few microseconds of work and one dependent launch per
// step would dominate (8.2 us per step measured).  2 * pairs steps: A -> B with table T0, then B -> A with table T1.
// Every pull, the flag byte and the face velocities are read with ld.volatile / from read-only data, the barrier orders
// the stores of one step before the loads of the next.  No time mean, no inflow fluctuations on this path (the host
// falls back to single launches for those steps).
template <typename real, typename S, int BLOCK, int MINB, bool DAMP, bool PERX>
__global__ void __launch_bounds__(BLOCK, MINB)
step_loop_kernel(S *__restrict__ A, S *__restrict__ B, const uint8_t *__restrict__ flags, const uint32_t *__restrict__ links,
                 real *__restrict__ fu0, real *__restrict__ fu1, const Params<real> P, const StepPtrs<S> T0, const StepPtrs<S> T1,
                 const int pairs)
{
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    const Turb<real> tb{};
    for (int s = 0; s < pairs; ++s) {
        step_body<real, S, false, true, BLOCK, DAMP, false, PERX>(A, B, flags, links, nullptr, fu0, fu1, P, T0, tb, 0);
        grid.sync();
        step_body<real, S, false, true, BLOCK, DAMP, false, PERX>(B, A, flags, links, nullptr, fu1, fu0, P, T1, tb, 0);
        grid.sync();
    }
}

} // namespace lbmk
