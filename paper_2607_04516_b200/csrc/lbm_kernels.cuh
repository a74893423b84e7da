// lbm_kernels.cuh — device code of the D3Q19 LBM-LES path for sm_100a.
//
// Storage: populations SoA  g[i][z][y][x]  with g_i = f_i - w_i ("shifted": the rest state is exactly 0 and the
// stored numbers are O(Ma), which keeps FP32 rounding two orders below the 1e-5 parity bar).  Two buffers A/B
// (pull scheme: read A at x - c_i, write B at x).  One flag byte per cell: bits 0-1 = class, bit 7 = "this FLUID
// cell has a wall link or lies on a domain face" (needs the resolving path).  Algorithm: DESIGN.md §3.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>

namespace lbmk {

constexpr int Q = 19;
enum : int { FLUID = 0, SOLID = 1, EQ_FIXED = 2, EQ_OUTFLOW = 3 };
enum : int { PERIODIC = 0, WALL = 1, FREE_SLIP = 2, FACE_EQ_FIXED = 3, FACE_EQ_OUTFLOW = 4 };
constexpr uint8_t CLASS_MASK = 3;
constexpr uint8_t SLOW_BIT = 0x80; // FLUID cell with at least one wall link
constexpr uint8_t EDGE_BIT = 0x40; // FLUID cell on a domain face (periodic / free-slip / wall resolution needed)

// ---- lattice (DESIGN.md §3 step 1): pair k = 1..9 holds directions 2k-1 (+) and 2k (-) -------------------------
// pair vectors: 1:(1,0,0) 2:(0,1,0) 3:(0,0,1) 4:(1,1,0) 5:(1,0,1) 6:(0,1,1) 7:(1,-1,0) 8:(1,0,-1) 9:(0,1,-1)
__host__ __device__ constexpr int pair_cx(int k) { return (k == 1 || k == 4 || k == 5 || k == 7 || k == 8) ? 1 : 0; }
__host__ __device__ constexpr int pair_cy(int k) { return (k == 2 || k == 4 || k == 6 || k == 9) ? 1 : (k == 7 ? -1 : 0); }
__host__ __device__ constexpr int pair_cz(int k) { return (k == 3 || k == 5 || k == 6) ? 1 : ((k == 8 || k == 9) ? -1 : 0); }
__host__ __device__ constexpr int dir_cx(int i) { return i == 0 ? 0 : ((i & 1) ? pair_cx((i + 1) / 2) : -pair_cx(i / 2)); }
__host__ __device__ constexpr int dir_cy(int i) { return i == 0 ? 0 : ((i & 1) ? pair_cy((i + 1) / 2) : -pair_cy(i / 2)); }
__host__ __device__ constexpr int dir_cz(int i) { return i == 0 ? 0 : ((i & 1) ? pair_cz((i + 1) / 2) : -pair_cz(i / 2)); }
__host__ __device__ constexpr int dir_opp(int i) { return i == 0 ? 0 : ((i & 1) ? i + 1 : i - 1); }
__host__ __device__ constexpr int dir_find(int cx, int cy, int cz)
{
    for (int i = 0; i < Q; ++i)
        if (dir_cx(i) == cx && dir_cy(i) == cy && dir_cz(i) == cz) return i;
    return -1;
}

template <int B, int E, class F>
__host__ __device__ __forceinline__ void static_for(F &&f)
{
    if constexpr (B < E) {
        f(std::integral_constant<int, B>{});
        static_for<B + 1, E>(f);
    }
}

// ---- parameters ------------------------------------------------------------------------------------------------
template <typename real>
struct Params {
    int nx, ny, nz, nxy;
    int N;            // cells
    long long stride; // elements between consecutive populations (>= N, multiple of 64)
    int face[6];
    real tau0, Kles;  // Kles = 18 sqrt(2) Cs^2
    real fcor, h, inv1ph2; // h = fcor/2, 1/(1+h^2)
    real Fx, Fy, Fz;
};

template <typename real>
struct Macro { real rho, ux, uy, uz; };

// ---- cache-hinted global access ----------------------------------------------------------------------------------
// Every population is read exactly once and written exactly once per step: stream them.
// HINT: 0 = ld.cs / st.cs, 1 = default / default, 2 = default ld / st.cs, 3 = ld.cs / default st
template <int HINT, typename real>
__device__ __forceinline__ real ld_pop(const real *p)
{
    if constexpr (HINT == 0 || HINT == 3) return __ldcs(p);
    else return *p;
}
template <int HINT, typename real>
__device__ __forceinline__ void st_pop(real *p, real v)
{
    if constexpr (HINT == 0 || HINT == 2) __stcs(p, v);
    else *p = v;
}

// ---- collision (DESIGN.md §3 steps 4b-4e) on shifted populations ---------------------------------------------------
// In: pulled g[19].  Out: post-collision g[19]; returns the (rho,u) the collision used.
template <typename real>
__device__ __forceinline__ Macro<real> collide(real (&g)[Q], const Params<real> &P)
{
    real s[10], d[10];
#pragma unroll
    for (int k = 1; k <= 9; ++k) { s[k] = g[2 * k - 1] + g[2 * k]; d[k] = g[2 * k - 1] - g[2 * k]; }
    // 4b: moments of the shifted populations (sum_i w_i = 1, sum_i w_i c_i = 0 drop out exactly)
    const real drho = g[0] + (((s[1] + s[2]) + (s[3] + s[4])) + ((s[5] + s[6]) + (s[7] + s[8])) + s[9]);
    const real mx = (d[1] + d[4]) + (d[5] + d[7]) + d[8];
    const real my = (d[2] + d[4]) + (d[6] - d[7]) + d[9];
    const real mz = (d[3] + d[5]) + (d[6] - d[8]) - d[9];
    const real Mxx = (s[1] + s[4]) + (s[5] + s[7]) + s[8];
    const real Myy = (s[2] + s[4]) + (s[6] + s[7]) + s[9];
    const real Mzz = (s[3] + s[5]) + (s[6] + s[8]) + s[9];
    const real Mxy = s[4] - s[7], Mxz = s[5] - s[8], Myz = s[6] - s[9];
    const real rho = real(1) + drho;
    const real inv = real(1) / rho;
    // 4c: implicit half-force velocity
    const real bx = mx * inv + real(0.5) * P.Fx, by = my * inv + real(0.5) * P.Fy, bz = mz * inv + real(0.5) * P.Fz;
    const real ux = (bx + P.h * by) * P.inv1ph2;
    const real uy = (by - P.h * bx) * P.inv1ph2;
    const real uz = bz;
    const real Fdx = rho * (P.Fx + P.fcor * uy), Fdy = rho * (P.Fy - P.fcor * ux), Fdz = rho * P.Fz;
    // 4d: Pi = sum c c (f - feq) = M - (drho/3) I - rho u u   (second moment of the shifted equilibrium is exact)
    const real third = real(1) / real(3);
    const real Pxx = Mxx - third * drho - rho * ux * ux;
    const real Pyy = Myy - third * drho - rho * uy * uy;
    const real Pzz = Mzz - third * drho - rho * uz * uz;
    const real Pxy = Mxy - rho * ux * uy, Pxz = Mxz - rho * ux * uz, Pyz = Myz - rho * uy * uz;
    const real Qn = sqrt(Pxx * Pxx + Pyy * Pyy + Pzz * Pzz + real(2) * (Pxy * Pxy + Pxz * Pxz + Pyz * Pyz));
    const real tau = real(0.5) * (P.tau0 + sqrt(P.tau0 * P.tau0 + P.Kles * Qn * inv));
    const real omega = real(1) / tau;
    const real phi = real(1) - real(0.5) * omega;
    // 4e: BGK + Guo source, pair by pair
    const real uF = ux * Fdx + uy * Fdy + uz * Fdz;
    const real A0 = drho - real(1.5) * rho * (ux * ux + uy * uy + uz * uz);
    const real keep = real(1) - omega;
    {
        const real w0 = real(1) / real(3);
        g[0] = keep * g[0] + omega * (w0 * A0) - w0 * phi * real(3) * uF;
    }
    static_for<1, 10>([&](auto kc) {
        constexpr int k = decltype(kc)::value;
        constexpr int cx = pair_cx(k), cy = pair_cy(k), cz = pair_cz(k);
        const real w = (k <= 3) ? real(1) / real(18) : real(1) / real(36);
        const real cu = real(cx) * ux + real(cy) * uy + real(cz) * uz;
        const real cF = real(cx) * Fdx + real(cy) * Fdy + real(cz) * Fdz;
        const real even = omega * (w * (A0 + real(4.5) * rho * cu * cu)) + w * phi * (real(9) * cu * cF - real(3) * uF);
        const real odd = omega * (w * real(3) * rho * cu) + w * phi * real(3) * cF;
        g[2 * k - 1] = keep * g[2 * k - 1] + (even + odd);
        g[2 * k] = keep * g[2 * k] + (even - odd);
    });
    return Macro<real>{rho, ux, uy, uz};
}

// shifted equilibrium at density 1: g_eq,i = w_i (3 cu + 4.5 cu^2 - 1.5 u^2)  (+ w_i drho when rho != 1)
template <typename real>
__device__ __forceinline__ void equilibrium(real (&g)[Q], real drho, real ux, real uy, real uz)
{
    const real rho = real(1) + drho;
    const real A0 = drho - real(1.5) * rho * (ux * ux + uy * uy + uz * uz);
    g[0] = (real(1) / real(3)) * A0;
    static_for<1, 10>([&](auto kc) {
        constexpr int k = decltype(kc)::value;
        constexpr int cx = pair_cx(k), cy = pair_cy(k), cz = pair_cz(k);
        const real w = (k <= 3) ? real(1) / real(18) : real(1) / real(36);
        const real cu = real(cx) * ux + real(cy) * uy + real(cz) * uz;
        const real even = w * (A0 + real(4.5) * rho * cu * cu);
        const real odd = w * real(3) * rho * cu;
        g[2 * k - 1] = even + odd;
        g[2 * k] = even - odd;
    });
}

// local macros of a stored (post-collision) state (DESIGN.md §3 step 7)
template <typename real>
__device__ __forceinline__ Macro<real> local_macros(const real (&g)[Q], int cls, const Params<real> &P)
{
    if (cls == SOLID) return Macro<real>{real(1), real(0), real(0), real(0)};
    real s[10], d[10];
#pragma unroll
    for (int k = 1; k <= 9; ++k) { s[k] = g[2 * k - 1] + g[2 * k]; d[k] = g[2 * k - 1] - g[2 * k]; }
    const real drho = g[0] + (((s[1] + s[2]) + (s[3] + s[4])) + ((s[5] + s[6]) + (s[7] + s[8])) + s[9]);
    const real mx = (d[1] + d[4]) + (d[5] + d[7]) + d[8];
    const real my = (d[2] + d[4]) + (d[6] - d[7]) + d[9];
    const real mz = (d[3] + d[5]) + (d[6] - d[8]) - d[9];
    const real rho = real(1) + drho;
    const real inv = real(1) / rho;
    if (cls == FLUID) {
        const real bx = mx * inv - real(0.5) * P.Fx, by = my * inv - real(0.5) * P.Fy, bz = mz * inv - real(0.5) * P.Fz;
        return Macro<real>{rho, (bx - P.h * by) * P.inv1ph2, (by + P.h * bx) * P.inv1ph2, bz};
    }
    return Macro<real>{rho, mx * inv, my * inv, mz * inv};
}

template <typename real>
__device__ __forceinline__ void load_cell(real (&g)[Q], const real *__restrict__ A, long long stride, int cell)
{
#pragma unroll
    for (int i = 0; i < Q; ++i) g[i] = A[(long long)i * stride + cell];
}

// ---- pull resolution (DESIGN.md §3 step 4a) -------------------------------------------------------------------------
// Geometry part, no memory access: for FLUID cell (x,y,z) and direction I, returns true if a WALL face is crossed;
// else the source cell and source direction after periodic wrap / free-slip mirroring.  Axis order z, y, x.
template <int I, typename real>
__device__ __forceinline__ bool resolve_geom(const Params<real> &P, int x, int y, int z, int &src_cell, int &src_dir)
{
    constexpr int cx = dir_cx(I), cy = dir_cy(I), cz = dir_cz(I);
    int sx = x - cx, sy = y - cy, sz = z - cz;
    bool wall = false, fx = false, fy = false, fz = false;
    if constexpr (cz != 0) {
        const bool lo = sz < 0, hi = sz >= P.nz;
        if (lo | hi) {
            const int ft = lo ? P.face[4] : P.face[5];
            if (ft == PERIODIC) sz = lo ? P.nz - 1 : 0;
            else if (ft == FREE_SLIP) { sz = z; fz = true; }
            else wall = true; // WALL (EQ faces are never crossed from a FLUID cell)
        }
    }
    if constexpr (cy != 0) {
        const bool lo = sy < 0, hi = sy >= P.ny;
        if (lo | hi) {
            const int ft = lo ? P.face[2] : P.face[3];
            if (ft == PERIODIC) sy = lo ? P.ny - 1 : 0;
            else if (ft == FREE_SLIP) { sy = y; fy = true; }
            else wall = true;
        }
    }
    if constexpr (cx != 0) {
        const bool lo = sx < 0, hi = sx >= P.nx;
        if (lo | hi) {
            const int ft = lo ? P.face[0] : P.face[1];
            if (ft == PERIODIC) sx = lo ? P.nx - 1 : 0;
            else if (ft == FREE_SLIP) { sx = x; fx = true; }
            else wall = true;
        }
    }
    // mirrored direction: a compile-time candidate per flip combination, selected by the three flip bits
    const int key = (fx ? 1 : 0) | (fy ? 2 : 0) | (fz ? 4 : 0);
    int j = I;
    static_for<1, 8>([&](auto kc) {
        constexpr int kk = decltype(kc)::value;
        constexpr bool possible = !((kk & 1) && cx == 0) && !((kk & 2) && cy == 0) && !((kk & 4) && cz == 0);
        if constexpr (possible) {
            constexpr int cand = dir_find((kk & 1) ? -cx : cx, (kk & 2) ? -cy : cy, (kk & 4) ? -cz : cz);
            if (key == kk) j = cand;
        }
    });
    src_dir = j;
    src_cell = wall ? (z * P.ny + y) * P.nx + x : (sz * P.ny + sy) * P.nx + sx;
    return wall;
}

// Bit i set <=> pulling direction i takes the bounce-back branch.  All neighbour flag loads are independent of one
// another (no branch between them), so they are issued as one batch.
template <typename real>
__device__ __forceinline__ uint32_t link_mask_edge(const Params<real> &P, const uint8_t *__restrict__ flags, int x, int y, int z)
{
    uint32_t bits = 0;
    static_for<1, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        int s, j;
        const bool wall = resolve_geom<i>(P, x, y, z, s, j);
        const uint8_t f = flags[s]; // own (FLUID) cell when a wall face was crossed
        bits |= ((wall || (f & CLASS_MASK) == SOLID) ? 1u : 0u) << i;
    });
    return bits;
}
template <typename real>
__device__ __forceinline__ uint32_t link_mask_interior(const Params<real> &P, const uint8_t *__restrict__ flags, int cell)
{
    uint32_t bits = 0;
    static_for<1, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        const int off = dir_cx(i) + dir_cy(i) * P.nx + dir_cz(i) * P.nxy;
        bits |= (((flags[cell - off] & CLASS_MASK) == SOLID) ? 1u : 0u) << i;
    });
    return bits;
}

template <typename real>
__device__ __forceinline__ uint32_t link_mask(const Params<real> &P, const uint8_t *__restrict__ flags, int x, int y, int z)
{
    return link_mask_edge(P, flags, x, y, z);
}

// which face's normal an EQ_OUTFLOW cell uses: first EQ_OUTFLOW face it lies on, order x-,x+,y-,y+,z-,z+
template <typename real>
__device__ __forceinline__ int outflow_neighbour(const Params<real> &P, int x, int y, int z)
{
    if (x == 0 && P.face[0] == FACE_EQ_OUTFLOW) return (P.nx > 1) ? (z * P.ny + y) * P.nx + 1 : -1;
    if (x == P.nx - 1 && P.face[1] == FACE_EQ_OUTFLOW) return (P.nx > 1) ? (z * P.ny + y) * P.nx + x - 1 : -1;
    if (y == 0 && P.face[2] == FACE_EQ_OUTFLOW) return (P.ny > 1) ? (z * P.ny + 1) * P.nx + x : -1;
    if (y == P.ny - 1 && P.face[3] == FACE_EQ_OUTFLOW) return (P.ny > 1) ? (z * P.ny + y - 1) * P.nx + x : -1;
    if (z == 0 && P.face[4] == FACE_EQ_OUTFLOW) return (P.nz > 1) ? (1 * P.ny + y) * P.nx + x : -1;
    if (z == P.nz - 1 && P.face[5] == FACE_EQ_OUTFLOW) return (P.nz > 1) ? ((z - 1) * P.ny + y) * P.nx + x : -1;
    return -1;
}

// ---- a1: voxelise -----------------------------------------------------------------------------------------------------
template <typename real>
__global__ void voxelise_kernel(const int32_t *__restrict__ height, uint8_t *__restrict__ flags, Params<real> P)
{
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= P.N) return;
    const int x = cell % P.nx, y = (cell / P.nx) % P.ny, z = cell / P.nxy;
    int h = height ? height[y * P.nx + x] : 0;
    h = min(max(h, 0), P.nz);
    int cls = FLUID;
    if (z < h) cls = SOLID;
    else {
        const bool on[6] = {x == 0, x == P.nx - 1, y == 0, y == P.ny - 1, z == 0, z == P.nz - 1};
        bool fixed = false, outflow = false;
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            fixed |= on[k] && P.face[k] == FACE_EQ_FIXED;
            outflow |= on[k] && P.face[k] == FACE_EQ_OUTFLOW;
        }
        cls = fixed ? EQ_FIXED : (outflow ? EQ_OUTFLOW : FLUID);
    }
    flags[cell] = (uint8_t)cls;
}

// ---- a2: link classification: sets SLOW_BIT; optionally exports the 18-bit masks ---------------------------------------
template <typename real>
__global__ void classify_kernel(uint8_t *__restrict__ flags_out, const uint8_t *__restrict__ flags, uint32_t *__restrict__ links,
                                Params<real> P)
{
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= P.N) return;
    const int x = cell % P.nx, y = (cell / P.nx) % P.ny, z = cell / P.nxy;
    const uint8_t cls = flags[cell] & CLASS_MASK;
    uint32_t bits = 0;
    if (cls == FLUID) bits = link_mask(P, flags, x, y, z);
    if (links) links[cell] = bits;
    if (flags_out) {
        const bool edge = x == 0 || x == P.nx - 1 || y == 0 || y == P.ny - 1 || z == 0 || z == P.nz - 1;
        flags_out[cell] = cls | ((cls == FLUID && bits != 0) ? SLOW_BIT : 0) | ((cls == FLUID && edge) ? EDGE_BIT : 0);
    }
}

// ---- a3: inlet write -------------------------------------------------------------------------------------------------
// mode 0: profile prof[3][nz] by level; mode 1: plane uvw[3][n2][n1] of one face
template <typename real, typename in_t>
__global__ void inlet_kernel(real *__restrict__ A, real *__restrict__ B, const uint8_t *__restrict__ flags,
                             const in_t *__restrict__ pu, const in_t *__restrict__ pv, const in_t *__restrict__ pw,
                             int mode, int face, Params<real> P)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    int cell;
    long long src;
    if (mode == 0) {
        cell = t;
        if (cell >= P.N) return;
        src = cell / P.nxy;
    } else {
        const int axis = face >> 1;
        const int n1 = axis == 0 ? P.ny : P.nx;
        const int n2 = axis == 2 ? P.ny : P.nz;
        if (t >= n1 * n2) return;
        const int j1 = t % n1, j2 = t / n1;
        const int nn[3] = {P.nx, P.ny, P.nz};
        const int fixed = (face & 1) ? nn[axis] - 1 : 0;
        int x, y, z;
        if (axis == 0) { x = fixed; y = j1; z = j2; }
        else if (axis == 1) { x = j1; y = fixed; z = j2; }
        else { x = j1; y = j2; z = fixed; }
        cell = (z * P.ny + y) * P.nx + x;
        src = t;
    }
    if ((flags[cell] & CLASS_MASK) != EQ_FIXED) return;
    const real ux = real(pu[src]), uy = pv ? real(pv[src]) : real(0), uz = pw ? real(pw[src]) : real(0);
    real g[Q];
    equilibrium(g, real(0), ux, uy, uz);
#pragma unroll
    for (int i = 0; i < Q; ++i) {
        A[(long long)i * P.stride + cell] = g[i];
        B[(long long)i * P.stride + cell] = g[i];
    }
}

// ---- a8: precursor plane -> main inlet (config 5) -----------------------------------------------------------------------
template <typename real>
__global__ void feed_kernel(real *__restrict__ dA, real *__restrict__ dB, const uint8_t *__restrict__ dflags, Params<real> D,
                            const real *__restrict__ sA, const uint8_t *__restrict__ sflags, Params<real> S, int sx)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= D.ny * D.nz) return;
    const int y = t % D.ny, z = t / D.ny;
    const int dcell = (z * D.ny + y) * D.nx;
    if ((dflags[dcell] & CLASS_MASK) != EQ_FIXED) return;
    const int scell = (z * S.ny + (y % S.ny)) * S.nx + sx;
    real g[Q];
    load_cell(g, sA, S.stride, scell);
    const Macro<real> m = local_macros(g, sflags[scell] & CLASS_MASK, S);
    equilibrium(g, real(0), m.ux, m.uy, m.uz);
#pragma unroll
    for (int i = 0; i < Q; ++i) {
        dA[(long long)i * D.stride + dcell] = g[i];
        dB[(long long)i * D.stride + dcell] = g[i];
    }
}

// ---- a4: init ------------------------------------------------------------------------------------------------------------
template <typename real, typename in_t>
__global__ void init_kernel(real *__restrict__ A, real *__restrict__ B, const uint8_t *__restrict__ flags,
                            const in_t *__restrict__ rho, const in_t *__restrict__ ux, const in_t *__restrict__ uy,
                            const in_t *__restrict__ uz, Params<real> P)
{
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= P.N) return;
    const int cls = flags[cell] & CLASS_MASK;
    if (cls == EQ_FIXED) return;
    real drho = rho ? real(rho[cell] - in_t(1)) : real(0);
    real u = ux ? real(ux[cell]) : real(0), v = uy ? real(uy[cell]) : real(0), w = uz ? real(uz[cell]) : real(0);
    if (cls == SOLID) { drho = 0; u = v = w = 0; }
    real g[Q];
    equilibrium(g, drho, u, v, w);
#pragma unroll
    for (int i = 0; i < Q; ++i) {
        A[(long long)i * P.stride + cell] = g[i];
        B[(long long)i * P.stride + cell] = g[i];
    }
}

// ---- a5/a6: fused stream-collide, one cell per thread (variant 0) ----------------------------------------------------------
template <typename real, bool MEAN, int HINT, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB)
step_kernel(const real *__restrict__ A, real *__restrict__ B, const uint8_t *__restrict__ flags, real *__restrict__ msum,
            Params<real> P)
{
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= P.N) return;
    const uint8_t fl = flags[cell];
    const int cls = fl & CLASS_MASK;
    if (cls == SOLID) return;
    real g[Q];
    if (cls == EQ_FIXED) {
        if constexpr (MEAN) {
            load_cell(g, A, P.stride, cell);
            const Macro<real> m = local_macros(g, EQ_FIXED, P);
            msum[cell] += m.ux;
            msum[P.stride + cell] += m.uy;
            msum[2 * P.stride + cell] += m.uz;
        }
        return;
    }
    Macro<real> m;
    if (cls == EQ_OUTFLOW) {
        const int x = cell % P.nx, y = (cell / P.nx) % P.ny, z = cell / P.nxy;
        const int nb = outflow_neighbour(P, x, y, z);
        m = Macro<real>{real(1), real(0), real(0), real(0)};
        if (nb >= 0) {
            load_cell(g, A, P.stride, nb);
            m = local_macros(g, flags[nb] & CLASS_MASK, P);
        }
        equilibrium(g, real(0), m.ux, m.uy, m.uz);
    } else {
        if (!(fl & (SLOW_BIT | EDGE_BIT))) {
            static_for<0, Q>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                const int off = dir_cx(i) + dir_cy(i) * P.nx + dir_cz(i) * P.nxy;
                g[i] = ld_pop<HINT>(A + ((long long)i * P.stride + (cell - off)));
            });
        } else if (!(fl & EDGE_BIT)) {
            // interior cell next to a solid: neighbours are plain offsets, some links bounce back
            const uint32_t bb = link_mask_interior(P, flags, cell);
            g[0] = ld_pop<HINT>(A + cell);
            static_for<1, Q>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                const int off = dir_cx(i) + dir_cy(i) * P.nx + dir_cz(i) * P.nxy;
                const bool b = (bb >> i) & 1u;
                const long long pop = b ? (long long)dir_opp(i) * P.stride : (long long)i * P.stride;
                g[i] = ld_pop<HINT>(A + (pop + (b ? cell : cell - off)));
            });
        } else {
            // cell on a domain face: periodic wrap / free-slip mirror / wall, then solidity of the resolved source
            const int x = cell % P.nx, y = (cell / P.nx) % P.ny, z = cell / P.nxy;
            const uint32_t bb = link_mask_edge(P, flags, x, y, z);
            g[0] = ld_pop<HINT>(A + cell);
            static_for<1, Q>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                int s, j;
                resolve_geom<i>(P, x, y, z, s, j);
                const bool b = (bb >> i) & 1u;
                g[i] = ld_pop<HINT>(A + ((long long)(b ? dir_opp(i) : j) * P.stride + (b ? cell : s)));
            });
        }
        m = collide(g, P);
    }
#pragma unroll
    for (int i = 0; i < Q; ++i) st_pop<HINT>(B + ((long long)i * P.stride + cell), g[i]);
    if constexpr (MEAN) {
        msum[cell] += m.ux;
        msum[P.stride + cell] += m.uy;
        msum[2 * P.stride + cell] += m.uz;
    }
}

// ---- a5/a6: fused stream-collide, FOUR x-consecutive cells per thread, 128-bit loads and stores (default for FP32) --------
// Thread t owns cells c = 4t .. 4t+3 of the linear [z][y][x] index (nx % 4 == 0, so c, nx and nx*ny are multiples of 4
// and every population row is 16-byte aligned).  Pull of direction i for the four cells = elements (c - off_i .. c+3 - off_i):
//   c_x = 0 : one aligned 128-bit load at c - off_yz;
//   c_x = +1: the same aligned load, shifted right by one element: element -1 comes from the left lane (__shfl_up),
//             lane 0 fetches it with one scalar load;  c_x = -1: mirror image with __shfl_down / lane 31.
// This is the plain interior streaming.  Cells whose flag byte has SLOW_BIT / EDGE_BIT then overwrite the affected
// directions (bounce-back from the stored link mask, periodic / free-slip / wall resolution on domain faces); static
// cells (SOLID, EQ_FIXED, EQ_OUTFLOW) are not stored.  EQ face cells are served by the first `face_blocks` blocks of the
// same launch (face_worker).  The arrays are padded by >= nx*ny + nx + 8 elements at both ends, so the unconditional
// vector loads of cells next to the domain faces stay inside the allocation (their values are replaced above).
template <typename real>
struct alignas(4 * sizeof(real)) Vec4 { real x, y, z, w; };

template <int J, typename real>
__device__ __forceinline__ real &comp(Vec4<real> &v)
{
    if constexpr (J == 0) return v.x;
    else if constexpr (J == 1) return v.y;
    else if constexpr (J == 2) return v.z;
    else return v.w;
}
template <typename real>
__device__ __forceinline__ void set_comp(Vec4<real> &v, int j, real val)
{
    v.x = j == 0 ? val : v.x;
    v.y = j == 1 ? val : v.y;
    v.z = j == 2 ? val : v.z;
    v.w = j == 3 ? val : v.w;
}

template <int HINT, typename real>
__device__ __forceinline__ Vec4<real> ld_vec(const real *p)
{
    const Vec4<real> *q = reinterpret_cast<const Vec4<real> *>(p);
    if constexpr (std::is_same<real, float>::value && (HINT == 0 || HINT == 3)) {
        const float4 t = __ldcs(reinterpret_cast<const float4 *>(p));
        return Vec4<real>{t.x, t.y, t.z, t.w};
    } else return *q;
}
template <int HINT, typename real>
__device__ __forceinline__ void st_vec(real *p, const Vec4<real> &v)
{
    if constexpr (std::is_same<real, float>::value && (HINT == 0 || HINT == 2)) __stcs(reinterpret_cast<float4 *>(p), make_float4(v.x, v.y, v.z, v.w));
    else *reinterpret_cast<Vec4<real> *>(p) = v;
}

// EQ face cells (a6 and the EQ part of a7): worker thread w walks the planes of the faces that need per-step work.
// A cell on several such faces is served from the first one in the order x-,x+,y-,y+,z-,z+ whose type matches its class.
template <typename real, bool MEAN>
__device__ __forceinline__ void face_worker(const real *__restrict__ A, real *__restrict__ B, const uint8_t *__restrict__ flags,
                                            real *__restrict__ msum, const Params<real> &P, long long w)
{
    int k = 0;
    long long cnt = 0;
    for (; k < 6; ++k) {
        const int ft = P.face[k];
        if (!(ft == FACE_EQ_OUTFLOW || (MEAN && ft == FACE_EQ_FIXED))) continue;
        const int axis = k >> 1;
        cnt = (long long)(axis == 0 ? P.ny : P.nx) * (axis == 2 ? P.ny : P.nz);
        if (w < cnt) break;
        w -= cnt;
    }
    if (k == 6) return;
    const int axis = k >> 1;
    const int n1 = axis == 0 ? P.ny : P.nx;
    const int j1 = (int)(w % n1), j2 = (int)(w / n1);
    const int nn[3] = {P.nx, P.ny, P.nz};
    const int fixed = (k & 1) ? nn[axis] - 1 : 0;
    int x, y, z;
    if (axis == 0) { x = fixed; y = j1; z = j2; }
    else if (axis == 1) { x = j1; y = fixed; z = j2; }
    else { x = j1; y = j2; z = fixed; }
    const int cell = (z * P.ny + y) * P.nx + x;
    const int cls = flags[cell] & CLASS_MASK;
    const int want = cls == EQ_OUTFLOW ? FACE_EQ_OUTFLOW : (cls == EQ_FIXED ? FACE_EQ_FIXED : -1);
    if (want < 0 || P.face[k] != want) return;
    const bool on[6] = {x == 0, x == P.nx - 1, y == 0, y == P.ny - 1, z == 0, z == P.nz - 1};
    for (int q = 0; q < k; ++q)
        if (on[q] && P.face[q] == want) return; // an earlier face owns this cell
    real g[Q];
    Macro<real> m{real(1), real(0), real(0), real(0)};
    if (cls == EQ_OUTFLOW) {
        const int nb = outflow_neighbour(P, x, y, z);
        if (nb >= 0) {
            load_cell(g, A, P.stride, nb);
            m = local_macros(g, flags[nb] & CLASS_MASK, P);
        }
        equilibrium(g, real(0), m.ux, m.uy, m.uz);
#pragma unroll
        for (int i = 0; i < Q; ++i) B[(long long)i * P.stride + cell] = g[i];
    } else {
        load_cell(g, A, P.stride, cell);
        m = local_macros(g, EQ_FIXED, P);
    }
    if constexpr (MEAN) {
        msum[cell] += m.ux;
        msum[P.stride + cell] += m.uy;
        msum[2 * P.stride + cell] += m.uz;
    }
}

// number of worker threads face_worker needs
template <typename real>
inline long long face_work_items(const Params<real> &P, bool mean)
{
    long long n = 0;
    for (int k = 0; k < 6; ++k) {
        const int ft = P.face[k];
        if (!(ft == FACE_EQ_OUTFLOW || (mean && ft == FACE_EQ_FIXED))) continue;
        const int axis = k >> 1;
        n += (long long)(axis == 0 ? P.ny : P.nx) * (axis == 2 ? P.ny : P.nz);
    }
    return n;
}

template <typename real, bool MEAN, int HINT, int BLOCK, int MINB>
__global__ void __launch_bounds__(BLOCK, MINB)
step4_kernel(const real *__restrict__ A, real *__restrict__ B, const uint8_t *__restrict__ flags, const uint32_t *__restrict__ links,
             real *__restrict__ msum, Params<real> P, int face_blocks)
{
    using V = Vec4<real>;
    if ((int)blockIdx.x < face_blocks) {
        face_worker<real, MEAN>(A, B, flags, msum, P, (long long)blockIdx.x * BLOCK + threadIdx.x);
        return;
    }
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const long long t = (long long)(blockIdx.x - face_blocks) * BLOCK + threadIdx.x;
    const bool inside = 4 * t < P.N;
    const int c = inside ? (int)(4 * t) : P.N - 4;
    const uint32_t word = inside ? *reinterpret_cast<const uint32_t *>(flags + c) : 0x01010101u;
    // byte j of nf: 1 = cell j is static (class != FLUID)
    const uint32_t nf = (word | (word >> 1)) & 0x01010101u;
    if (__all_sync(FULL, nf == 0x01010101u)) return;
    // a lane's aligned vectors are needed by itself, by the right lane (its cell 0, c_x = +1) and the left lane (its cell 3)
    const uint32_t nf_r = __shfl_down_sync(FULL, nf, 1), nf_l = __shfl_up_sync(FULL, nf, 1);
    const bool need = nf != 0x01010101u || (lane < 31 && !(nf_r & 1u)) || (lane > 0 && !(nf_l >> 24));
    const bool need_lo = lane == 0 && !(nf & 1u);         // element c-1 (c_x = +1 directions)
    const bool need_hi = lane == 31 && !(nf >> 24);       // element c+4 (c_x = -1 directions)

    V v[Q];
    real e[Q];
    const real *a = A + c;
    static_for<0, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int cx = dir_cx(i), cy = dir_cy(i), cz = dir_cz(i);
        const real *p = a + ((long long)i * P.stride - (cy * P.nx + cz * P.nxy));
        v[i] = need ? ld_vec<HINT>(p) : V{real(0), real(0), real(0), real(0)};
        if constexpr (cx == 1) e[i] = need_lo ? ld_pop<HINT>(p - 1) : real(0);
        if constexpr (cx == -1) e[i] = need_hi ? ld_pop<HINT>(p + 4) : real(0);
    });
    static_for<1, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int cx = dir_cx(i);
        if constexpr (cx == 1) {
            real prev = __shfl_up_sync(FULL, v[i].w, 1);
            if (lane == 0) prev = e[i];
            v[i] = V{prev, v[i].x, v[i].y, v[i].z};
        }
        if constexpr (cx == -1) {
            real next = __shfl_down_sync(FULL, v[i].x, 1);
            if (lane == 31) next = e[i];
            v[i] = V{v[i].y, v[i].z, v[i].w, next};
        }
    });

    // cells with wall links or on a domain face: overwrite what plain streaming got wrong
    if (word & 0xC0C0C0C0u) {
#pragma unroll 1
        for (int j = 0; j < 4; ++j) {
            const uint32_t fb = (word >> (8 * j)) & 0xFFu;
            if (!(fb & (SLOW_BIT | EDGE_BIT))) continue;
            const int cell = c + j;
            const uint32_t bb = links[cell];
            if (!(fb & EDGE_BIT)) {
                static_for<1, Q>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    if ((bb >> i) & 1u) set_comp(v[i], j, A[(long long)dir_opp(i) * P.stride + cell]);
                });
            } else {
                const int x = cell % P.nx, y = (cell / P.nx) % P.ny, z = cell / P.nxy;
                static_for<1, Q>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    int s, jd;
                    resolve_geom<i>(P, x, y, z, s, jd);
                    const bool b = (bb >> i) & 1u;
                    set_comp(v[i], j, A[(long long)(b ? dir_opp(i) : jd) * P.stride + (b ? cell : s)]);
                });
            }
        }
    }

    V mu[3];
    static_for<0, 4>([&](auto jc) {
        constexpr int j = decltype(jc)::value;
        real g[Q];
#pragma unroll
        for (int i = 0; i < Q; ++i) g[i] = comp<j>(v[i]);
        const Macro<real> m = collide(g, P);
#pragma unroll
        for (int i = 0; i < Q; ++i) comp<j>(v[i]) = g[i];
        if constexpr (MEAN) { comp<j>(mu[0]) = m.ux; comp<j>(mu[1]) = m.uy; comp<j>(mu[2]) = m.uz; }
    });

    real *b = B + c;
    if (nf == 0) {
#pragma unroll
        for (int i = 0; i < Q; ++i) st_vec<HINT>(b + (long long)i * P.stride, v[i]);
        if constexpr (MEAN) {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                V *mp = reinterpret_cast<V *>(msum + (long long)k * P.stride + c);
                V s = *mp;
                s.x += mu[k].x; s.y += mu[k].y; s.z += mu[k].z; s.w += mu[k].w;
                *mp = s;
            }
        }
    } else {
        static_for<0, 4>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            if (!((nf >> (8 * j)) & 1u)) {
#pragma unroll
                for (int i = 0; i < Q; ++i) b[(long long)i * P.stride + j] = comp<j>(v[i]);
                if constexpr (MEAN) {
#pragma unroll
                    for (int k = 0; k < 3; ++k) msum[(long long)k * P.stride + c + j] += comp<j>(mu[k]);
                }
            }
        });
    }
}

// ---- a7: macros / mean / state ---------------------------------------------------------------------------------------------
template <typename real, typename out_t>
__global__ void macros_kernel(const real *__restrict__ A, const uint8_t *__restrict__ flags, out_t *__restrict__ rho,
                              out_t *__restrict__ ux, out_t *__restrict__ uy, out_t *__restrict__ uz, Params<real> P)
{
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= P.N) return;
    const int cls = flags[cell] & CLASS_MASK;
    real g[Q];
    Macro<real> m{real(1), real(0), real(0), real(0)};
    if (cls != SOLID) {
        load_cell(g, A, P.stride, cell);
        m = local_macros(g, cls, P);
    }
    if (rho) rho[cell] = out_t(m.rho);
    if (ux) ux[cell] = out_t(m.ux);
    if (uy) uy[cell] = out_t(m.uy);
    if (uz) uz[cell] = out_t(m.uz);
}

// standalone sample (used when a sample is due at a step the fused kernel did not produce, e.g. step 0)
template <typename real>
__global__ void mean_sample_kernel(const real *__restrict__ A, const uint8_t *__restrict__ flags, real *__restrict__ msum, Params<real> P)
{
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= P.N) return;
    const int cls = flags[cell] & CLASS_MASK;
    if (cls == SOLID) return;
    real g[Q];
    load_cell(g, A, P.stride, cell);
    const Macro<real> m = local_macros(g, cls, P);
    msum[cell] += m.ux;
    msum[P.stride + cell] += m.uy;
    msum[2 * P.stride + cell] += m.uz;
}

template <typename real, typename out_t>
__global__ void mean_out_kernel(const real *__restrict__ msum, out_t *__restrict__ ux, out_t *__restrict__ uy, out_t *__restrict__ uz,
                                double inv_count, Params<real> P)
{
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= P.N) return;
    if (ux) ux[cell] = out_t(double(msum[cell]) * inv_count);
    if (uy) uy[cell] = out_t(double(msum[P.stride + cell]) * inv_count);
    if (uz) uz[cell] = out_t(double(msum[2 * P.stride + cell]) * inv_count);
}

// class bits only (the SLOW bit is internal)
__global__ void flags_out_kernel(const uint8_t *__restrict__ flags, uint8_t *__restrict__ out, int N)
{
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell < N) out[cell] = flags[cell] & CLASS_MASK;
}

__host__ __device__ inline double weight_f64(int i) { return i == 0 ? 1.0 / 3.0 : (i <= 6 ? 1.0 / 18.0 : 1.0 / 36.0); }

template <typename real>
__global__ void state_out_kernel(const real *__restrict__ A, double *__restrict__ f, Params<real> P)
{
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= P.N) return;
#pragma unroll
    for (int i = 0; i < Q; ++i) f[(long long)i * P.N + cell] = double(A[(long long)i * P.stride + cell]) + weight_f64(i);
}

template <typename real>
__global__ void state_in_kernel(real *__restrict__ A, real *__restrict__ B, const double *__restrict__ f, Params<real> P)
{
    const int cell = blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= P.N) return;
#pragma unroll
    for (int i = 0; i < Q; ++i) {
        const real v = real(f[(long long)i * P.N + cell] - weight_f64(i));
        A[(long long)i * P.stride + cell] = v;
        B[(long long)i * P.stride + cell] = v;
    }
}

} // namespace lbmk
