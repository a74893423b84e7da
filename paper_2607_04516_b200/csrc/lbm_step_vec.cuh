// lbm_step_vec.cuh — a5/a6 (+ the fused part of a7): the fused stream-collide kernel with V x-cells per thread and
// 64/128-bit loads and stores (north_star: "SoA, FP32, coalesced and 128-bit-vectorised loads and stores";
// SURVEY.md §7 step 7).  Same arithmetic, same storage, same write-side boundary rule as lbm_step.cuh; what changes is
// how the 38 streams are moved:
//
//   * a thread owns V consecutive cells of one row (V = 4: one float4 per population; rows start 32-byte aligned and
//     nx % V == 0, so every access is naturally aligned);
//   * ALL 19 pulls are aligned vector loads at the thread's own x: the c_x = +-1 part of the pull offset is applied in
//     registers — a population with c_x = +1 needs the value one cell to the left, i.e. the thread's own elements
//     0..V-2 and the left neighbour lane's element V-1 (one __shfl_up); lane 0 of a warp and the first thread of a row
//     fetch that one value with a scalar load (the x = -1 halo slot at a row start);
//   * the V flag bytes are one word; a warp whose cells are all plain FLUID / EQ / FEED cells (no wall link, no ghost
//     slot, no solid) stores 19 vectors per thread; other warps store vectors where all V cells of the thread write a
//     slot and predicated scalars elsewhere, then the mailbox / ghost stores of lbm_core.cuh.
//
// Per 32 cells this issues ~9.5 load/store instructions instead of 38 and a quarter of the address arithmetic.
// S = storage type of the populations (float; __half: lbm_set_storage), arithmetic always FP32.
#pragma once
#include "lbm_step.cuh"
#include "lbm_packed.cuh"
#include <cuda_fp16.h>

namespace lbmk {

// V consecutive stored values <-> V floats.  The loads are volatile asm statements: they keep their order, so the pulls
// stay ahead of the flag test (ptxas otherwise sinks them below it: a second dependent round trip).
template <typename S, int V>
struct VecIO;

template <>
struct VecIO<float, 4> {
    static __device__ __forceinline__ void ld(const float *p, float (&v)[4])
    {
        asm volatile("ld.global.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]) : "l"(p));
    }
    static __device__ __forceinline__ void st(float *p, const float (&v)[4])
    {
        *reinterpret_cast<float4 *>(p) = make_float4(v[0], v[1], v[2], v[3]);
    }
};
template <>
struct VecIO<float, 2> {
    static __device__ __forceinline__ void ld(const float *p, float (&v)[2])
    {
        asm volatile("ld.global.v2.f32 {%0, %1}, [%2];" : "=f"(v[0]), "=f"(v[1]) : "l"(p));
    }
    static __device__ __forceinline__ void st(float *p, const float (&v)[2]) { *reinterpret_cast<float2 *>(p) = make_float2(v[0], v[1]); }
};
template <>
struct VecIO<float, 8> { // the mean sums of the 8-cell kernel: two 128-bit accesses
    static __device__ __forceinline__ void ld(const float *p, float (&v)[8])
    {
        asm volatile("ld.global.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]) : "l"(p));
        asm volatile("ld.global.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]) : "l"(p + 4));
    }
    static __device__ __forceinline__ void st(float *p, const float (&v)[8])
    {
        reinterpret_cast<float4 *>(p)[0] = make_float4(v[0], v[1], v[2], v[3]);
        reinterpret_cast<float4 *>(p)[1] = make_float4(v[4], v[5], v[6], v[7]);
    }
};
template <>
struct VecIO<__half, 2> {
    static __device__ __forceinline__ void ld(const __half *p, float (&v)[2])
    {
        uint32_t a;
        asm volatile("ld.global.b32 %0, [%1];" : "=r"(a) : "l"(p));
        const float2 f = __half22float2(*reinterpret_cast<const __half2 *>(&a));
        v[0] = f.x; v[1] = f.y;
    }
    static __device__ __forceinline__ void st(__half *p, const float (&v)[2])
    {
        const __half2 h = __floats2half2_rn(v[0], v[1]);
        *reinterpret_cast<uint32_t *>(p) = *reinterpret_cast<const uint32_t *>(&h);
    }
};
template <>
struct VecIO<__half, 4> {
    static __device__ __forceinline__ void ld(const __half *p, float (&v)[4])
    {
        uint32_t a, b;
        asm volatile("ld.global.v2.b32 {%0, %1}, [%2];" : "=r"(a), "=r"(b) : "l"(p));
        const float2 lo = __half22float2(*reinterpret_cast<const __half2 *>(&a)), hi = __half22float2(*reinterpret_cast<const __half2 *>(&b));
        v[0] = lo.x; v[1] = lo.y; v[2] = hi.x; v[3] = hi.y;
    }
    static __device__ __forceinline__ void st(__half *p, const float (&v)[4])
    {
        const __half2 lo = __floats2half2_rn(v[0], v[1]), hi = __floats2half2_rn(v[2], v[3]);
        uint2 w;
        w.x = *reinterpret_cast<const uint32_t *>(&lo);
        w.y = *reinterpret_cast<const uint32_t *>(&hi);
        *reinterpret_cast<uint2 *>(p) = w;
    }
};
template <>
struct VecIO<__half, 8> {
    static __device__ __forceinline__ void ld(const __half *p, float (&v)[8])
    {
        uint32_t w[4];
        asm volatile("ld.global.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "l"(p));
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float2 f = __half22float2(*reinterpret_cast<const __half2 *>(&w[k]));
            v[2 * k] = f.x; v[2 * k + 1] = f.y;
        }
    }
    static __device__ __forceinline__ void st(__half *p, const float (&v)[8])
    {
        uint4 w;
        uint32_t *wp = reinterpret_cast<uint32_t *>(&w);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const __half2 h = __floats2half2_rn(v[2 * k], v[2 * k + 1]);
            wp[k] = *reinterpret_cast<const uint32_t *>(&h);
        }
        *reinterpret_cast<uint4 *>(p) = w;
    }
};

// one stored value, pinned like the vector loads
__device__ __forceinline__ float ld1_pinned(const float *p)
{
    float v;
    asm volatile("ld.global.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ float ld1_pinned(const __half *p)
{
    unsigned short v;
    asm volatile("ld.global.u16 %0, [%1];" : "=h"(v) : "l"(p));
    return __half2float(__ushort_as_half(v));
}
// the V flag bytes of a thread as one word (byte k = cell k)
template <int V>
__device__ __forceinline__ uint64_t ld_flags(const uint8_t *p)
{
    if constexpr (V == 8) {
        unsigned long long v;
        asm volatile("ld.global.u64 %0, [%1];" : "=l"(v) : "l"(p));
        return v;
    } else if constexpr (V == 4) {
        uint32_t v;
        asm volatile("ld.global.u32 %0, [%1];" : "=r"(v) : "l"(p));
        return v;
    } else {
        unsigned short v;
        asm volatile("ld.global.u16 %0, [%1];" : "=h"(v) : "l"(p));
        return v;
    }
}

__device__ __forceinline__ float to_store(float v, float *) { return v; }
__device__ __forceinline__ __half to_store(float v, __half *) { return __float2half_rn(v); }

// Address table of the vector kernel: src[i] = A + i stride - (c_y px + c_z pxy) — NO c_x part (applied in registers).
template <typename S>
struct VecPtrs {
    const S *src[Q];
    S *dst[Q];
};
template <typename S, typename real>
inline VecPtrs<S> make_vec_ptrs(const S *A, S *B, const Params<real> &P)
{
    VecPtrs<S> t;
    for (int i = 0; i < Q; ++i) {
        const long long off = (long long)dir_cy(i) * P.px + (long long)dir_cz(i) * P.pxy;
        t.src[i] = A + ((long long)i * P.stride - off);
        t.dst[i] = B + (long long)i * P.stride;
    }
    return t;
}
// thread -> (row, first cell): nq = threads per plane = nx ny / V, qpr = threads per row, qmagic = ceil(2^32 / qpr)
// (0: divide), exact for every index below nq + 1024 (checked by the host)
struct VecGeom { unsigned nq, qpr, qmagic; };

// rare per-cell work of the slow path, out of line (the cell's populations go through local memory): keeps the V-fold
// unrolled kernel body small
template <typename S>
__device__ __noinline__ void ghost_cell(S *__restrict__ B, const Params<float> &P, int x, int y, int z, uint32_t lk, const float *gl)
{
    ghost_stores(P, x, y, z, lk, [&](int i, int pt, auto jc) { B[(long long)i * P.stride + pt] = to_store(gl[decltype(jc)::value], (S *)nullptr); });
}
__device__ __noinline__ void feed_cell(float *__restrict__ fuw, const Params<float> &P, int x, int y, int z, float ux, float uy, float uz)
{
    outflow_feed(P, x, y, z, ux, uy, uz, [&](int sl, int comp, float v) { fuw[comp * P.F + sl] = v; });
}

template <typename S, int V, bool MEAN, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB)
step_vec_kernel(const uint8_t *__restrict__ flags, const uint32_t *__restrict__ links, float *__restrict__ msum,
                const float *__restrict__ fur, float *__restrict__ fuw, const __grid_constant__ Params<float> P,
                const __grid_constant__ VecPtrs<S> T, const VecGeom G)
{
    using IO = VecIO<S, V>;
    constexpr unsigned FULL = 0xffffffffu;
    constexpr uint32_t ALL = 0x7FFFFu;
    const unsigned lane = threadIdx.x & 31u;
    unsigned c = blockIdx.x * BLOCK + threadIdx.x;
    if (c - lane >= G.nq) return; // the whole warp lies beyond the plane
    // a thread beyond the plane stays (the shuffles need every lane), as a copy of the last thread that stores nothing
    const bool valid = c < G.nq;
    if (!valid) c = G.nq - 1;
    const int y = G.qmagic ? (int)__umulhi(c, G.qmagic) : (int)(c / G.qpr);
    const int x0 = ((int)c - y * (int)G.qpr) * V;
    const int z = blockIdx.y;
    const int p0 = pidx(P, x0, y, z);

    // ---- all loads, before anything is waited for -------------------------------------------------------------------
    float g[V][Q];
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        float a[V];
        IO::ld(T.src[i] + p0, a);
#pragma unroll
        for (int k = 0; k < V; ++k) g[k][i] = a[k];
    });
    // the one value a c_x = +-1 population needs from beyond the thread's own cells, where no neighbour lane has it
    const bool edgeL = lane == 0u || x0 == 0, edgeR = lane == 31u || x0 + V == P.nx;
    float e[Q];
    static_for<1, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        e[i] = 0.0f;
        if constexpr (dir_cx(i) == 1) { if (edgeL) e[i] = ld1_pinned(T.src[i] + (p0 - 1)); }
        else if constexpr (dir_cx(i) == -1) { if (edgeR) e[i] = ld1_pinned(T.src[i] + (p0 + V)); }
    });
    // face velocity of an EQ cell at a row end, from geometry alone (EQ_FIXED wins, as in the voxeliser); EQ cells on y / z
    // faces (whole rows, rare) fetch theirs when the flag is known
    float fuL[3] = {0.0f, 0.0f, 0.0f}, fuR[3] = {0.0f, 0.0f, 0.0f};
    auto face_vel = [&](int x, float (&fu)[3]) {
        int k = eq_owner(P, FACE_EQ_FIXED, x, y, z);
        if (k < 0) k = eq_owner(P, FACE_EQ_OUTFLOW, x, y, z);
        if (k >= 0) {
            const int sl = outflow_slot(P, k, x, y, z);
            fu[0] = ld1_pinned(fur + sl); fu[1] = ld1_pinned(fur + P.F + sl); fu[2] = ld1_pinned(fur + 2 * P.F + sl);
        }
    };
    if (P.F > 0 && x0 == 0) face_vel(0, fuL);
    if (P.F > 0 && x0 + V == P.nx) face_vel(P.nx - 1, fuR);
    float ms[3][V];
    if constexpr (MEAN) {
        VecIO<float, V>::ld(msum + p0, ms[0]);
        VecIO<float, V>::ld(msum + P.stride + p0, ms[1]);
        VecIO<float, V>::ld(msum + 2 * P.stride + p0, ms[2]);
    }
    const uint64_t fw = ld_flags<V>(flags + p0);

    // ---- the c_x shift, in registers -------------------------------------------------------------------------------------
    static_for<1, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        if constexpr (dir_cx(i) == 1) {
            const float left = __shfl_up_sync(FULL, g[V - 1][i], 1);
#pragma unroll
            for (int k = V - 1; k > 0; --k) g[k][i] = g[k - 1][i];
            g[0][i] = edgeL ? e[i] : left;
        } else if constexpr (dir_cx(i) == -1) {
            const float right = __shfl_down_sync(FULL, g[0][i], 1);
#pragma unroll
            for (int k = 0; k < V - 1; ++k) g[k][i] = g[k + 1][i];
            g[V - 1][i] = edgeR ? e[i] : right;
        }
    });

    // ---- classes -------------------------------------------------------------------------------------------------------
    // "bad" bytes: SLOW / EDGE / SURF bit, or class SOLID (1) / GHOST (4).  A warp without any stores 19 vectors per thread.
    constexpr uint64_t ONES = 0x0101010101010101ull;
    const uint64_t badw = (fw & (ONES * (uint64_t)(SLOW_BIT | EDGE_BIT | SURF_BIT | 4))) | ((fw & ~(fw >> 1)) & ONES);
    const bool slow_warp = !__all_sync(FULL, badw == 0);
    uint32_t lk[V];
#pragma unroll
    for (int k = 0; k < V; ++k) lk[k] = 0;
    if (slow_warp) {
#pragma unroll
        for (int k = 0; k < V; ++k)
            if ((fw >> (8 * k)) & (SLOW_BIT | SURF_BIT)) lk[k] = links[p0 + k];
    }
    uint32_t wm[V];      // slots cell k writes: all 19 if live, the completion mask of a surface solid, none otherwise
    uint32_t wand = ALL; // slots ALL cells of the thread write: these go out as one vector
    // V = 2 with 16-bit storage: the two cells collide together in packed FP32 pairs (lbm_packed.cuh: FFMA2 / FADD2 / FMUL2)
    // whenever at least one of them is FLUID; the result of a cell that is not is replaced below (its inputs may be anything:
    // nothing traps, nothing of it is kept).  Measured: 221.5 M instead of 278.6 M warp instructions per step of
    // config 3 and +2 % on the 16-bit path; on FP32 storage the packed pairs cost spills at 80 registers (-6 %), so it stays scalar.
    constexpr bool PACKED = V == 2 && std::is_same<S, __half>::value;
    Macro<float> mk[2];
    if constexpr (PACKED) {
        const bool any_fluid = ((fw & CLASS_MASK) == FLUID) | (((fw >> 8) & CLASS_MASK) == FLUID);
        if (any_fluid) collide2(g[0], g[1], P, mk[0], mk[1]);
    }
    static_for<0, V>([&](auto kc) {
        constexpr int k = decltype(kc)::value;
        const uint32_t fl = (uint32_t)(fw >> (8 * k)) & 0xFFu;
        const int cls = fl & CLASS_MASK;
        Macro<float> m{1.0f, 0.0f, 0.0f, 0.0f};
        if (cls == FLUID) {
            if constexpr (PACKED) m = mk[k];
            else m = collide(g[k], P);
            wm[k] = ALL;
        } else if (cls == SOLID || cls == GHOST) {
#pragma unroll
            for (int i = 0; i < Q; ++i) g[k][i] = 0.0f;
            wm[k] = (fl & SURF_BIT) ? lk[k] : 0u;
        } else { // EQ_FIXED (a3) / EQ_OUTFLOW (a6): f_eq(1, u) of the cell's face velocity (lbm_core.cuh)
            float u0, u1, u2;
            if (k == 0 && x0 == 0) { u0 = fuL[0]; u1 = fuL[1]; u2 = fuL[2]; }
            else if (k == V - 1 && x0 + V == P.nx) { u0 = fuR[0]; u1 = fuR[1]; u2 = fuR[2]; }
            else {
                const int sl = eq_slot(P, cls, x0 + k, y, z);
                u0 = fur[sl]; u1 = fur[P.F + sl]; u2 = fur[2 * P.F + sl];
            }
            m = Macro<float>{1.0f, u0, u1, u2};
            equilibrium(g[k], 0.0f, u0, u1, u2);
            wm[k] = ALL;
        }
        if (!valid) wm[k] = 0u;
        wand &= wm[k];
        if ((fl & FEED_BIT) && cls != SOLID && valid) feed_cell(fuw, P, x0 + k, y, z, m.ux, m.uy, m.uz);
        if constexpr (MEAN) {
            if (cls != SOLID) { ms[0][k] += m.ux; ms[1][k] += m.uy; ms[2][k] += m.uz; }
        }
    });

    // ---- own slots ---------------------------------------------------------------------------------------------------
    if (!slow_warp) {
        if (valid) {
            static_for<0, Q>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                float a[V];
#pragma unroll
                for (int k = 0; k < V; ++k) a[k] = g[k][i];
                IO::st(T.dst[i] + p0, a);
            });
        }
    } else {
        // a surface solid takes part with zeros where its completion mask says so: the sector leaves L2 fully written
        static_for<0, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            if ((wand >> i) & 1u) {
                float a[V];
#pragma unroll
                for (int k = 0; k < V; ++k) a[k] = g[k][i];
                IO::st(T.dst[i] + p0, a);
            } else {
#pragma unroll
                for (int k = 0; k < V; ++k)
                    if ((wm[k] >> i) & 1u) T.dst[i][p0 + k] = to_store(g[k][i], (S *)nullptr);
            }
        });
        // mailboxes of the wall links and ghost slots (lbm_core.cuh), cell by cell
        static_for<0, V>([&](auto kc) {
            constexpr int k = decltype(kc)::value;
            const uint32_t fl = (uint32_t)(fw >> (8 * k)) & 0xFFu;
            if (!valid || (fl & CLASS_MASK) == SOLID) return;
            if (fl & SLOW_BIT) {
                static_for<1, Q>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    if ((lk[k] >> i) & 1u) T.dst[i][p0 + k - poff<i>(P)] = to_store(g[k][dir_opp(i)], (S *)nullptr);
                });
            }
            if (fl & EDGE_BIT) {
                float gl[Q];
#pragma unroll
                for (int i = 0; i < Q; ++i) gl[i] = g[k][i];
                ghost_cell<S>(T.dst[0], P, x0 + k, y, z, lk[k], gl);
            }
        });
    }
    if constexpr (MEAN) {
        if (valid) {
            VecIO<float, V>::st(msum + p0, ms[0]);
            VecIO<float, V>::st(msum + P.stride + p0, ms[1]);
            VecIO<float, V>::st(msum + 2 * P.stride + p0, ms[2]);
        }
    }
}

} // namespace lbmk
