// lbm_inplace.cuh — a5/a6 (+ the fused part of a7) with IN-PLACE streaming: the same fused stream-collide step on ONE
// population buffer.  Half the memory of the two-buffer scheme, the same 153 B per
// cell and step (76 B read + 76 B written + 1 flag byte) and the same arithmetic (collide / equilibrium of lbm_core.cuh).
//
// Scheme (lbm_core.cuh, "in-place streaming"): the two slots 2k-1, 2k of cell y belong to the link (y - c_k, y).  A step of
// parity q reads, per pair k, the cell's own slot ip_slot(q, 2k-1) (direction +c_k, pushed there by the neighbour) and slot
// ip_slot(q, 2k) of the neighbour x + c_k (direction -c_k, still at home there), and after the collision writes the outgoing
// +c_k population over the second address and the outgoing -c_k population over the first: every address is read and then
// written by the same thread and by nobody else, and the next step finds everything with the two slots' roles swapped
// (parity q ^ 1).  Known in the literature as the "esoteric pull" access pattern; here it carries this library's write-side
// boundary rule, so the read side stays a pure 19-address gather for every face type: populations that leave towards a SOLID
// cell (halfway bounce-back) or a GHOST halo cell (free-slip, periodic y / z) are stored where their receiving cell will read
// them next step — slots of links with a dead end, which nobody reads during this step.  PERIODIC x faces wrap on both sides
// of the same address (read and write of the pair's neighbour slot by the last cell of a row go to the row's first cell).
// No sector completion by surface solids: every sector that is written was read by the same warp a moment before, so it is
// whole in L2 when it is written back.
#pragma once
#include "lbm_core.cuh"
#include "lbm_setup.cuh"
#include "lbm_step.cuh"

namespace lbmk {

// Per-launch address tables.  rd[i] + c (c = the cell's padded index, or its row-wrapped one for the c_x = -1 directions of a
// PERIODIC-x lattice) = where a cell reads its incoming direction i in this launch's parity, and where it then stores its
// outgoing opp(i).  nx[i] = the same table for the next parity: where a wall link puts direction i for the cell itself.
template <typename S>
struct IpPtrs {
    S *rd[Q];
    S *nx[Q];
    S *G;    // the population buffer (ghost slots: slot and cell are known only at run time)
    int qn;  // parity of the next step
};
template <typename S, typename real>
inline IpPtrs<S> make_ip_ptrs(S *G, int q, const Params<real> &P)
{
    IpPtrs<S> t;
    for (int i = 0; i < Q; ++i) {
        const long long off = dir_cx(i) + (long long)dir_cy(i) * P.px + (long long)dir_cz(i) * P.pxy;
        const bool even = i > 0 && (i & 1) == 0;
        t.rd[i] = G + ((long long)ip_slot(q, i) * P.stride - (even ? off : 0));
        t.nx[i] = G + ((long long)ip_slot(q ^ 1, i) * P.stride - (even ? off : 0));
    }
    t.G = G;
    t.qn = q ^ 1;
    return t;
}

// TURB: the launch carries the synthetic inflow fluctuations in extra leading block rows, exactly as the two-buffer kernel does
// (lbm_step.cuh): one thread per face slot publishes the boundary velocity of the step after this one into the half of the side
// array this launch writes.
template <typename real, typename S, bool MEAN, int BLOCK, bool DAMP, bool PERX, bool TURB>
__device__ __forceinline__ void ip_step_body(const uint8_t *__restrict__ flags, const uint32_t *__restrict__ links, real *__restrict__ msum,
                                             const real *__restrict__ fur, real *__restrict__ fuw, const Params<real> &P, const IpPtrs<S> &T,
                                             const Turb<real> &tb, const int turb_planes)
{
    int zb = blockIdx.y;
    if constexpr (TURB) {
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
    const int z = zb == 0 ? P.nz - 1 : zb - 1; // the all-slow top plane first (lbm_step.cuh)
    const int p = pidx(P, x, y, z);
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    int pR = p;
    if constexpr (PERX) {
        if (x == P.nx - 1) pR = p - P.nx;
    }
    auto at = [&](auto ic) { // cell index that goes with rd[i] / nx[i]
        constexpr int i = decltype(ic)::value;
        if constexpr (PERX && i > 0 && (i & 1) == 0 && dir_cx(i) == -1) return pR;
        else return p;
    };

    real g[Q];
    real fu0 = real(0), fu1 = real(0), fu2 = real(0);
    real ms0 = real(0), ms1 = real(0), ms2 = real(0);
    Damp<real> dmp{real(0), real(0), real(0), real(0)};
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        g[i] = real(ld_pinned(T.rd[i] + at(ic)));
    });
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
    if constexpr (DAMP) dmp = damp_at(P, x, y, z);
    if constexpr (MEAN) { ms0 = ld_pinned(msum + p); ms1 = ld_pinned(msum + P.stride + p); ms2 = ld_pinned(msum + 2 * P.stride + p); }
    const uint8_t fl = ld_pinned(flags + p);
    const int cls = fl & CLASS_MASK;
    // the outgoing population j overwrites the address the incoming opp(j) was read from
    auto store_all = [&]() {
        static_for<0, Q>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            st_s(T.rd[dir_opp(j)] + at(std::integral_constant<int, dir_opp(j)>{}), g[j]);
        });
    };
    auto finish = [&](const Macro<real> &m) {
        if (fl & FEED_BIT) outflow_feed(P, x, y, z, m.ux, m.uy, m.uz, [&](int sl, int comp, real v) { fuw[comp * P.F + sl] = v; });
        if constexpr (MEAN) {
            msum[p] = ms0 + m.ux;
            msum[P.stride + p] = ms1 + m.uy;
            msum[2 * P.stride + p] = ms2 + m.uz;
        }
    };
    // fast path, warp-uniform: plain FLUID cells and EQ / feeding cells without wall link or ghost slot
    const bool plain = (fl & (SLOW_BIT | EDGE_BIT)) == 0 && cls != SOLID && cls != GHOST;
    if (__all_sync(__activemask(), plain)) {
        Macro<real> m;
        if (cls == FLUID) {
            if constexpr (DAMP) m = collide<real, true>(g, P, dmp);
            else m = collide(g, P);
        } else {
            m = Macro<real>{real(1), fu0, fu1, fu2};
            equilibrium(g, real(0), fu0, fu1, fu2);
        }
        store_all();
        finish(m);
        return;
    }
    uint32_t lk = 0;
    if (fl & SLOW_BIT) lk = links[p];
    if (cls == SOLID || cls == GHOST) return;
    Macro<real> m{real(1), fu0, fu1, fu2};
    if (cls == FLUID) {
        if constexpr (DAMP) m = collide<real, true>(g, P, dmp);
        else m = collide(g, P);
    } else equilibrium(g, real(0), fu0, fu1, fu2); // EQ_FIXED (a3) / EQ_OUTFLOW (a6)
    store_all(); // towards a dead cell this fills the link's unused slot
    if (fl & SLOW_BIT) {
        // wall link i: the cell's own outgoing opp(i) is what it reads as direction i next step
        static_for<1, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            if ((lk >> i) & 1u) st_s(T.nx[i] + at(ic), g[dir_opp(i)]);
        });
    }
    if (fl & EDGE_BIT)
        ghost_stores(P, x, y, z, lk, [&](int i, int pt, auto jc) {
            int cell = pt; // ghost slot (i, pt) of the two-buffer scheme = "cell pt + c_i receives direction i" (lbm_core.cuh ip_visit)
            if (i & 1) cell = pt + poff_rt(P, i) + ((dir_cx(i) == 1 && P.perx && x == P.nx - 1) ? -P.nx : 0);
            st_s(T.G + ((long long)ip_slot(T.qn, i) * P.stride + cell), g[decltype(jc)::value]);
        });
    finish(m);
}

template <typename real, typename S, bool MEAN, int BLOCK, int MINB, bool DAMP = false, bool PERX = false, bool TURB = false>
__global__ void __launch_bounds__(BLOCK, MINB)
ip_step_kernel(const uint8_t *__restrict__ flags, const uint32_t *__restrict__ links, real *__restrict__ msum, const real *__restrict__ fur,
               real *__restrict__ fuw, const Params<real> P, const IpPtrs<S> T, const Turb<real> tb, const int turb_planes)
{
    ip_step_body<real, S, MEAN, BLOCK, DAMP, PERX, TURB>(flags, links, msum, fur, fuw, P, T, tb, turb_planes);
}

} // namespace lbmk
