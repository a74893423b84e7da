// lbm_core.cuh — lattice, layout, per-cell arithmetic and the write-side boundary rule of the D3Q19 LBM-LES path
// (sm_100a).  Algorithm statement: DESIGN.md §3 (restating PAPER.md:61, Table 1).
//
// Storage.  Populations SoA g[i][Z][Y][X] on a HALO-PADDED box: one halo layer on every side, interior rows starting
// at padded x = 8, x pitch rounded up to 32 cells (every row is 128-byte aligned).  g_i = f_i - w_i ("shifted": the rest
// state is exactly 0, stored numbers are O(Ma), FP32 rounding stays two orders below the 1e-5 parity bar).
// Two buffers A/B, pull scheme: every FLUID cell reads A[i][p - off_i] for ALL i with no case distinction.
// Storage type S of the populations: the arithmetic type `real` (float / double), or __half with FP32 arithmetic
// (lbm_create_ex precision 2; binary16 of the shifted population, rounded to nearest even at every store).
// Rows start on a 32-byte sector: interior x = 0 sits at padded x = P.xoff (8 cells; 16 for __half).
//
// What makes that possible is a write-side boundary rule ("mailboxes").  A population j that leaves cell x
// towards a cell that cannot be pulled from is stored, by x itself, where the pull of the next step will look:
//   * target is SOLID (building, WALL face, or halo whose image is solid): slot (opp(j), x + c_j) <- g_j
//     — halfway bounce-back: next step x pulls opp(j) from x - c_opp(j) = x + c_j  (DESIGN.md §3 step 4a);
//   * target is a GHOST halo cell of a FREE_SLIP face: slot (flip(j), x with the out axes stepped into the halo)
//     <- g_j — specular reflection; of a PERIODIC face: slot (j, x with the out axes moved to the far halo) <- g_j.
// Every halo slot has exactly one writer, so there is no race; SOLID cells never run, so their slots are free.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>
#include <cuda_fp16.h>

namespace lbmk {

constexpr int Q = 19;
// cell classes (3 bits).  GHOST exists only in the halo.
enum : int { FLUID = 0, SOLID = 1, EQ_FIXED = 2, EQ_OUTFLOW = 3, GHOST = 4 };
enum : int { PERIODIC = 0, WALL = 1, FREE_SLIP = 2, FACE_EQ_FIXED = 3, FACE_EQ_OUTFLOW = 4 };
constexpr uint8_t CLASS_MASK = 7;
constexpr uint8_t SLOW_BIT = 0x80; // FLUID cell with at least one wall link (mailbox stores needed)
constexpr uint8_t EDGE_BIT = 0x40; // non-solid cell on a domain face that has at least one ghost slot to store
constexpr uint8_t FEED_BIT = 0x20; // non-solid cell one layer inside an EQ_OUTFLOW face: publishes its velocity (a6)
constexpr uint8_t SURF_BIT = 0x10; // SOLID cell sharing a 32-byte sector with a cell that is rewritten every step

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

// ---- parameters and layout ---------------------------------------------------------------------------------------
template <typename real>
struct Params {
    int nx, ny, nz;   // interior cells
    int px, py, pxy;  // padded x pitch (multiple of 32, >= nx + xoff + 1), padded rows per plane (ny + 2), px * py
    int perx;         // both x faces PERIODIC: the pull across them wraps on the READ side (xwrap below), no x ghost slots
    int xoff, sec;    // padded x of interior x = 0 (one 32-byte sector of storage elements), cells per 32-byte sector (8; 16 for __half)
    int Np;           // padded cells = pxy * (nz + 2)
    int N;            // interior cells
    int nxy;          // nx * ny
    unsigned nx_magic; // ceil(2^32 / nx) when umulhi(n, nx_magic) == n / nx for all n < nxy + 1024, else 0 (use a division)
    long long stride; // elements between consecutive populations (>= Np, multiple of 64)
    int face[6];
    int foff[6];      // first slot of each EQ face (FIXED or OUTFLOW) in the face-velocity side buffer, slots = face-plane cells
    int F;            // slots in total (0 if there is no EQ face)
    real tau0, Kles;       // Kles = 18 sqrt(2) Cs^2
    real fx, fy, fz;       // Coriolis vector f = 2 Omega; the scalar f_cor of lbm_create is fz
    real hx, hy, hz, inv1ph2; // h = f/2, 1/(1+|h|^2)
    real Fx, Fy, Fz;
    // damping zones (lbm_set_damping; PAPER.md:175 top sponge + lateral buffer nudging): nullptr = none, else the per-axis
    // coefficient tables sx[nx], sy[ny], sz[nz] (each the larger of the axis' two face ramps) followed by the target
    // profile ut[3][nz];  sigma(x,y,z) = max(sx[x], sy[y], sz[z])
    const real *damp;
    int dlo[3], dhi[3]; // cells with dlo <= (x,y,z) < dhi lie outside every zone: no table look-up there
    // thermal lattice (lbm_set_thermal, lbm_thermal.cuh): buoyancy coefficient g beta, reference theta, 1 / tau_theta;
    // all 0 while it is off
    real gbeta, theta_ref, omega_t;
    // fixed-temperature WALL faces of the thermal lattice (lbm_set_thermal_walls; DESIGN.md §4 reading 26): bit k of thd = face k
    // is held, thw[k] = 2 (theta_w - theta_ref) of that face (the anti-bounce-back mailbox value is -t_j + wT_j thw[k])
    int thd;
    real thw[6];
    // in-place streaming (lbm_create_ex precision | LBM_STREAM_INPLACE): -1 = two buffers (A/B pull, everything
    // above), else the handle has ONE population buffer and ipq = parity of the step that reads the current state next
    int ipq;
};

// Interior x = 0 sits at padded x = P.xoff (8 cells of 4 or 8 bytes, 16 cells of 2): every interior row starts on a
// 32-byte sector boundary (and ends on one when nx % P.sec == 0), so full-row stores never leave partially written
// sectors, which would cost a DRAM fill read each.
template <typename S>
constexpr int xoff_for() { return sizeof(S) == 2 ? 16 : 8; }
// padded linear index of interior cell (x,y,z); also valid for halo coordinates -1 and n
template <typename real>
__host__ __device__ __forceinline__ int pidx(const Params<real> &P, int x, int y, int z)
{
    return ((z + 1) * P.py + (y + 1)) * P.px + (x + P.xoff);
}
// offset (in cells) of the pull source of direction i relative to the cell: source = p - poff
template <int I, typename real>
__host__ __device__ __forceinline__ int poff(const Params<real> &P)
{
    return dir_cx(I) + dir_cy(I) * P.px + dir_cz(I) * P.pxy;
}

// PERIODIC x faces.  A ghost slot in the x halo would be a single element in an otherwise untouched 32-byte sector (a DRAM
// read-modify-write per row and direction: 2.4 - 6 % of the step), so the wrap across the x faces is done by
// the READER instead: the pull of a direction with c_x = +1 by a cell at x = 0 comes from x = nx - 1 of the same source row
// (index + nx), with c_x = -1 at x = nx - 1 from x = 0 (index - nx).  Everything addressed relative to a pull source moves
// with it: the bounce-back mailbox of such a link lies in the wrapped cell, and a population that leaves through a periodic
// x face AND a y / z face goes to the y / z halo slot of its own x column.  xwrap = cells to add to p - off_i.
template <int I, typename real>
__host__ __device__ __forceinline__ int xwrap(const Params<real> &P, int x)
{
    if constexpr (dir_cx(I) == 1) return (P.perx && x == 0) ? P.nx : 0;
    else if constexpr (dir_cx(I) == -1) return (P.perx && x == P.nx - 1) ? -P.nx : 0;
    else return 0;
}

// c . a for a lattice vector known at compile time: only the non-zero components are touched (no 0 * x terms,
// which IEEE arithmetic may not fold away)
template <int CX, int CY, int CZ, typename real>
__device__ __forceinline__ real cdot(real ax, real ay, real az)
{
    static_assert(CX != 0 || CY != 0 || CZ != 0, "zero vector");
    if constexpr (CX != 0 && CY == 0 && CZ == 0) return CX > 0 ? ax : -ax;
    else if constexpr (CX == 0 && CY != 0 && CZ == 0) return CY > 0 ? ay : -ay;
    else if constexpr (CX == 0 && CY == 0 && CZ != 0) return CZ > 0 ? az : -az;
    else if constexpr (CZ == 0) return (CX > 0) ? (CY > 0 ? ax + ay : ax - ay) : (CY > 0 ? ay - ax : -ax - ay);
    else if constexpr (CY == 0) return (CX > 0) ? (CZ > 0 ? ax + az : ax - az) : (CZ > 0 ? az - ax : -ax - az);
    else return (CY > 0) ? (CZ > 0 ? ay + az : ay - az) : (CZ > 0 ? az - ay : -ay - az);
}

template <typename real>
struct Macro { real rho, ux, uy, uz; };

// damping coefficient and target velocity of one cell (DESIGN.md §4 reading 20): a_d(u) = sg (ut - u)
template <typename real>
struct Damp { real sg, utx, uty, utz; };
template <typename real>
__device__ __forceinline__ Damp<real> damp_at(const Params<real> &P, int x, int y, int z)
{
    if (!P.damp || (x >= P.dlo[0] && x < P.dhi[0] && y >= P.dlo[1] && y < P.dhi[1] && z >= P.dlo[2] && z < P.dhi[2]))
        return Damp<real>{real(0), real(0), real(0), real(0)};
    const real *d = P.damp;
    const real sg = fmax(fmax(d[x], d[P.nx + y]), d[P.nx + P.ny + z]);
    const real *t = d + (P.nx + P.ny + P.nz);
    return Damp<real>{sg, t[z], t[P.nz + z], t[2 * P.nz + z]};
}

// ---- collision (DESIGN.md §3 steps 4b-4e) on shifted populations ---------------------------------------------------
// In: pulled g[19].  Out: post-collision g[19]; returns the (rho,u) the collision used.
// BUOY: fb = an extra acceleration along z of this cell (the Boussinesq buoyancy g beta (theta - theta_ref) of the thermal
// lattice, lbm_thermal.cuh), added to P.Fz — passed as a value so that P stays the kernel parameter (constant bank).
template <typename real, bool DAMP = false, bool BUOY = false>
__device__ __forceinline__ Macro<real> collide(real (&g)[Q], const Params<real> &P, const Damp<real> dm = Damp<real>{}, const real fb = real(0))
{
    const real PFz = BUOY ? P.Fz + fb : P.Fz;
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
    // 4c: implicit half-force velocity.  a(u) = F - f x u, so rho u = m + rho a(u)/2 reads u + h x u = b with h = f/2,
    // b = m/rho + F/2, whose solution is u = (b - h x b + h (h.b)) / (1 + |h|^2)
    const real bx = mx * inv + real(0.5) * P.Fx, by = my * inv + real(0.5) * P.Fy, bz = mz * inv + real(0.5) * PFz;
    real ux, uy, uz, Fdx, Fdy, Fdz;
    bool damped = false;
    if constexpr (DAMP) damped = dm.sg > real(0);
    if (damped) {
        // inside a damping zone a(u) gains sg (ut - u):  A u + h x u = b' with A = 1 + sg/2, b' = b + (sg/2) ut, whose
        // solution is u = (A^2 b' - A h x b' + h (h.b')) / (A (A^2 + |h|^2))
        const real hs = real(0.5) * dm.sg, A = real(1) + hs;
        const real cx = bx + hs * dm.utx, cy = by + hs * dm.uty, cz = bz + hs * dm.utz;
        const real hb = P.hx * cx + P.hy * cy + P.hz * cz;
        const real den = real(1) / (A * (A * A + (P.hx * P.hx + P.hy * P.hy + P.hz * P.hz)));
        const real A2 = A * A;
        ux = (A2 * cx - A * (P.hy * cz - P.hz * cy) + P.hx * hb) * den;
        uy = (A2 * cy - A * (P.hz * cx - P.hx * cz) + P.hy * hb) * den;
        uz = (A2 * cz - A * (P.hx * cy - P.hy * cx) + P.hz * hb) * den;
        Fdx = rho * (P.Fx - (P.fy * uz - P.fz * uy) + dm.sg * (dm.utx - ux));
        Fdy = rho * (P.Fy - (P.fz * ux - P.fx * uz) + dm.sg * (dm.uty - uy));
        Fdz = rho * (PFz - (P.fx * uy - P.fy * ux) + dm.sg * (dm.utz - uz));
    } else {
        const real hb = P.hx * bx + P.hy * by + P.hz * bz;
        ux = (bx - (P.hy * bz - P.hz * by) + P.hx * hb) * P.inv1ph2;
        uy = (by - (P.hz * bx - P.hx * bz) + P.hy * hb) * P.inv1ph2;
        uz = (bz - (P.hx * by - P.hy * bx) + P.hz * hb) * P.inv1ph2;
        Fdx = rho * (P.Fx - (P.fy * uz - P.fz * uy));
        Fdy = rho * (P.Fy - (P.fz * ux - P.fx * uz));
        Fdz = rho * (PFz - (P.fx * uy - P.fy * ux));
    }
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
    // 4e: BGK + Guo source.  With base = omega A0 - 3 phi uF, P1 = omega rho u, P2 = phi Fd and, per weight group,
    //   E0 = w base,  v = w (4.5 P1 + 9 P2),  o = 3 w (P1 + P2):
    //   even_k = E0 + (c_k.u)(c_k.v),  odd_k = c_k.o,  g'_{k+-} = (1 - omega) g_{k+-} + even_k +- odd_k
    // which is the expansion of  g - omega (g - g_eq) + (1 - omega/2) w [3 (c - u).Fd + 9 (c.u)(c.Fd)]  pair by pair.
    const real uF = ux * Fdx + uy * Fdy + uz * Fdz;
    const real A0 = drho - real(1.5) * rho * (ux * ux + uy * uy + uz * uz);
    const real keep = real(1) - omega;
    const real base = omega * A0 - real(3) * phi * uF;
    const real orho = omega * rho;
    const real P1x = orho * ux, P1y = orho * uy, P1z = orho * uz;
    const real P2x = phi * Fdx, P2y = phi * Fdy, P2z = phi * Fdz;
    g[0] = keep * g[0] + third * base;
    // group a: w = 1/18 (axis pairs 1..3); group b: w = 1/36 (diagonal pairs 4..9) = half of group a
    const real E0a = base * (real(1) / real(18)), E0b = base * (real(1) / real(36));
    const real vax = real(0.25) * P1x + real(0.5) * P2x, vay = real(0.25) * P1y + real(0.5) * P2y, vaz = real(0.25) * P1z + real(0.5) * P2z;
    const real oax = (P1x + P2x) * (real(1) / real(6)), oay = (P1y + P2y) * (real(1) / real(6)), oaz = (P1z + P2z) * (real(1) / real(6));
    const real vbx = real(0.5) * vax, vby = real(0.5) * vay, vbz = real(0.5) * vaz;
    const real obx = real(0.5) * oax, oby = real(0.5) * oay, obz = real(0.5) * oaz;
    static_for<1, 10>([&](auto kc) {
        constexpr int k = decltype(kc)::value;
        constexpr int cx = pair_cx(k), cy = pair_cy(k), cz = pair_cz(k);
        const real E0 = (k <= 3) ? E0a : E0b;
        const real vx = (k <= 3) ? vax : vbx, vy = (k <= 3) ? vay : vby, vz = (k <= 3) ? vaz : vbz;
        const real ox = (k <= 3) ? oax : obx, oy = (k <= 3) ? oay : oby, oz = (k <= 3) ? oaz : obz;
        const real cu = cdot<cx, cy, cz>(ux, uy, uz);
        const real cv = cdot<cx, cy, cz>(vx, vy, vz);
        const real co = cdot<cx, cy, cz>(ox, oy, oz);
        const real even = E0 + cu * cv;
        g[2 * k - 1] = keep * g[2 * k - 1] + (even + co);
        g[2 * k] = keep * g[2 * k] + (even - co);
    });
    return Macro<real>{rho, ux, uy, uz};
}

// shifted equilibrium: g_eq,i = w_i (drho + rho (3 cu + 4.5 cu^2 - 1.5 u^2))
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
        const real cu = cdot<cx, cy, cz>(ux, uy, uz);
        const real even = w * (A0 + real(4.5) * rho * cu * cu);
        const real odd = w * real(3) * rho * cu;
        g[2 * k - 1] = even + odd;
        g[2 * k] = even - odd;
    });
}

// local macros of a stored (post-collision) state (DESIGN.md §3 step 7); dm = the cell's damping (damp_at)
template <typename real>
__device__ __forceinline__ Macro<real> local_macros(const real (&g)[Q], int cls, const Params<real> &P, const Damp<real> dm = Damp<real>{})
{
    if (cls == SOLID || cls == GHOST) return Macro<real>{real(1), real(0), real(0), real(0)};
    real s[10], d[10];
#pragma unroll
    for (int k = 1; k <= 9; ++k) { s[k] = g[2 * k - 1] + g[2 * k]; d[k] = g[2 * k - 1] - g[2 * k]; }
    const real drho = g[0] + (((s[1] + s[2]) + (s[3] + s[4])) + ((s[5] + s[6]) + (s[7] + s[8])) + s[9]);
    const real mx = (d[1] + d[4]) + (d[5] + d[7]) + d[8];
    const real my = (d[2] + d[4]) + (d[6] - d[7]) + d[9];
    const real mz = (d[3] + d[5]) + (d[6] - d[8]) - d[9];
    const real rho = real(1) + drho;
    const real inv = real(1) / rho;
    if (cls == FLUID && dm.sg > real(0)) {
        // m*/rho - F/2 - (sg/2) ut = A u - h x u with A = 1 - sg/2  =>  u = (A^2 b + A h x b + h (h.b)) / (A (A^2 + |h|^2))
        const real hs = real(0.5) * dm.sg, A = real(1) - hs, A2 = A * A;
        const real bx = mx * inv - real(0.5) * P.Fx - hs * dm.utx, by = my * inv - real(0.5) * P.Fy - hs * dm.uty,
                   bz = mz * inv - real(0.5) * P.Fz - hs * dm.utz;
        const real hb = P.hx * bx + P.hy * by + P.hz * bz;
        const real den = real(1) / (A * (A2 + (P.hx * P.hx + P.hy * P.hy + P.hz * P.hz)));
        return Macro<real>{rho, (A2 * bx + A * (P.hy * bz - P.hz * by) + P.hx * hb) * den,
                           (A2 * by + A * (P.hz * bx - P.hx * bz) + P.hy * hb) * den,
                           (A2 * bz + A * (P.hx * by - P.hy * bx) + P.hz * hb) * den};
    }
    if (cls == FLUID) {
        // m*/rho - F/2 = u - h x u  =>  u = (b + h x b + h (h.b)) / (1 + |h|^2)
        const real bx = mx * inv - real(0.5) * P.Fx, by = my * inv - real(0.5) * P.Fy, bz = mz * inv - real(0.5) * P.Fz;
        const real hb = P.hx * bx + P.hy * by + P.hz * bz;
        return Macro<real>{rho, (bx + (P.hy * bz - P.hz * by) + P.hx * hb) * P.inv1ph2,
                           (by + (P.hz * bx - P.hx * bz) + P.hy * hb) * P.inv1ph2,
                           (bz + (P.hx * by - P.hy * bx) + P.hz * hb) * P.inv1ph2};
    }
    return Macro<real>{rho, mx * inv, my * inv, mz * inv};
}

// one stored population <-> the arithmetic type (S = real: a plain access; S = __half: widen / round to nearest even)
template <typename real, typename S>
__device__ __forceinline__ real ld_s(const S *p)
{
    if constexpr (std::is_same<S, __half>::value) return real(__half2float(*p));
    else return real(*p);
}
template <typename real, typename S>
__device__ __forceinline__ void st_s(S *p, real v)
{
    if constexpr (std::is_same<S, __half>::value) *p = __float2half_rn(float(v));
    else *p = S(v);
}

template <typename real, typename S>
__device__ __forceinline__ void load_cell(real (&g)[Q], const S *__restrict__ A, long long stride, int p)
{
#pragma unroll
    for (int i = 0; i < Q; ++i) g[i] = ld_s<real>(A + ((long long)i * stride + p));
}

// ---- the write-side boundary rule ------------------------------------------------------------------------------------
// st(i, pt, jc): "slot (direction i, padded cell pt) <- g[jc]" with jc an integral_constant (register indexing).
// Wall links: bit i of lk set <=> the pull source of direction i is SOLID <=> population opp(i) leaves towards it.
template <typename real, class St>
__device__ __forceinline__ void wall_stores(const Params<real> &P, int p, int x, uint32_t lk, St &&st)
{
    static_for<1, Q>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        if ((lk >> i) & 1u) st(i, p - poff<i>(P) + xwrap<i>(P, x), std::integral_constant<int, dir_opp(i)>{});
    });
}

// Ghost slots of a non-solid cell (x,y,z) on a domain face: for every direction j that leaves the box, unless it is
// a wall link (then wall_stores owns it) or an out axis is a WALL / EQ face (nobody pulls from there).
template <typename real, class St>
__device__ __forceinline__ void ghost_stores(const Params<real> &P, int x, int y, int z, uint32_t lk, St &&st)
{
    static_for<1, Q>([&](auto jc) {
        constexpr int j = decltype(jc)::value;
        constexpr int cx = dir_cx(j), cy = dir_cy(j), cz = dir_cz(j);
        bool out = false, ok = true, fx = false, fy = false, fz = false;
        int hx = x, hy = y, hz = z;
        if constexpr (cx != 0) {
            const bool lo = x + cx < 0, hi = x + cx >= P.nx;
            if (lo | hi) {
                const int ft = lo ? P.face[0] : P.face[1];
                if (ft == PERIODIC) { /* read-side wrap (xwrap): the slot stays in the cell's own x column and exists only if a
                                         y / z face is crossed as well */ }
                else if (ft == FREE_SLIP) { out = true; hx = x + cx; fx = true; }
                else { out = true; ok = false; }
            }
        }
        if constexpr (cy != 0) {
            const bool lo = y + cy < 0, hi = y + cy >= P.ny;
            if (lo | hi) {
                out = true;
                const int ft = lo ? P.face[2] : P.face[3];
                if (ft == PERIODIC) hy = y - cy * P.ny;
                else if (ft == FREE_SLIP) { hy = y + cy; fy = true; }
                else ok = false;
            }
        }
        if constexpr (cz != 0) {
            const bool lo = z + cz < 0, hi = z + cz >= P.nz;
            if (lo | hi) {
                out = true;
                const int ft = lo ? P.face[4] : P.face[5];
                if (ft == PERIODIC) hz = z - cz * P.nz;
                else if (ft == FREE_SLIP) { hz = z + cz; fz = true; }
                else ok = false;
            }
        }
        if (out && ok && !((lk >> dir_opp(j)) & 1u)) {
            // reflected direction: a compile-time candidate per flip combination
            const int key = (fx ? 1 : 0) | (fy ? 2 : 0) | (fz ? 4 : 0);
            int i = j;
            static_for<1, 8>([&](auto kc) {
                constexpr int kk = decltype(kc)::value;
                constexpr bool possible = !((kk & 1) && cx == 0) && !((kk & 2) && cy == 0) && !((kk & 4) && cz == 0);
                if constexpr (possible) {
                    constexpr int cand = dir_find((kk & 1) ? -cx : cx, (kk & 2) ? -cy : cy, (kk & 4) ? -cz : cz);
                    if (key == kk) i = cand;
                }
            });
            st(i, pidx(P, hx, hy, hz), jc);
        }
    });
}

// All stores of one cell's post-collision state into buffer B: own 19 slots, wall mailboxes, ghost slots.
template <typename real, typename S>
__device__ __forceinline__ void store_cell(S *__restrict__ B, const Params<real> &P, int p, int x, int y, int z, uint8_t fl,
                                           uint32_t lk, const real (&g)[Q])
{
#pragma unroll
    for (int i = 0; i < Q; ++i) st_s(B + ((long long)i * P.stride + p), g[i]);
    if (fl & (SLOW_BIT | EDGE_BIT)) {
        auto st = [&](int i, int pt, auto jc) { st_s(B + ((long long)i * P.stride + pt), g[decltype(jc)::value]); };
        if (fl & SLOW_BIT) wall_stores(P, p, x, lk, st);
        if (fl & EDGE_BIT) ghost_stores(P, x, y, z, lk, st);
    }
}

// ---- in-place streaming: one population buffer --------------------------------------------------------------
// Every link between a cell y and its neighbour y - c_k (pair k = 1..9) owns the two slots 2k-1 and 2k of cell y.  In a state of
// parity q a cell x' finds its incoming population of direction i
//     i odd  (= +c_k):  in slot ip_slot(q, i) of x' itself          (the neighbour x' - c_k pushed it there),
//     i even (= -c_k):  in slot ip_slot(q, i) of x' + c_k            (the neighbour x' + c_k kept it at home),
// with ip_slot(0, i) = i and ip_slot(1, i) = opp(i).  A step of parity q reads these 19 addresses and writes its outgoing
// population j to the address it read opp(j) from — which is exactly where x' = x + c_j looks for direction j in parity q ^ 1.
// Nobody else touches those two addresses during the step, so one buffer is enough.  The write-side boundary rule carries
// over unchanged: a population that cannot go to x + c_j (wall link, ghost slot) is put where its receiving cell x' will look
// for its receiving direction i next step; that slot belongs to a link whose other end is SOLID / GHOST (a cell that never
// runs), so nobody reads it during this step either.  The slot of the link that the dead end would have used stays unused, and
// a live cell may store its outgoing population towards a dead cell there unconditionally (never read).
__host__ __device__ constexpr int ip_slot(int q, int i) { return q ? dir_opp(i) : i; }

// element index (slot * stride + cell) at which cell p (interior x coordinate x) reads its incoming direction I in parity q
template <int I, typename real>
__device__ __forceinline__ long long ip_read_at(const Params<real> &P, int q, int p, int x)
{
    if constexpr (I == 0 || (I & 1)) return (long long)ip_slot(q, I) * P.stride + p;
    else return (long long)ip_slot(q, I) * P.stride + (p - poff<I>(P) + xwrap<I>(P, x));
}
// cell offset of direction i, i known only at run time (ghost slots: the reflected direction)
template <typename real>
__device__ __forceinline__ int poff_rt(const Params<real> &P, int i)
{
    return dir_cx(i) + dir_cy(i) * P.px + dir_cz(i) * P.pxy;
}
// Visit the addresses that hold the post-collision state of cell p = (x,y,z) in a state of parity q: f(jc, e) is called with
// direction j (integral_constant) and element index e, first with the plain destination of every direction, then once more
// for every redirected direction (wall links, ghost slots) — a later call overrides an earlier one.  A store visitor writes
// g[j] to every address it is shown (the plain destination of a redirected direction is an unused slot); a load visitor
// reads g[j] from the last one.
template <typename real, class F>
__device__ __forceinline__ void ip_visit(const Params<real> &P, int q, int p, int x, int y, int z, uint8_t fl, uint32_t lk, F &&f)
{
    f(std::integral_constant<int, 0>{}, (long long)p);
    static_for<1, Q>([&](auto jc) {
        constexpr int j = decltype(jc)::value;
        // arrives at x + c_j with direction j: odd j is kept by the receiving cell itself, even j stays at home (= x)
        if constexpr (j & 1) {
            const int wrap = (dir_cx(j) == 1 && P.perx && x == P.nx - 1) ? -P.nx : 0;
            f(jc, (long long)ip_slot(q, j) * P.stride + (p + poff<j>(P) + wrap));
        } else f(jc, (long long)ip_slot(q, j) * P.stride + p);
    });
    if (fl & SLOW_BIT) {
        // wall link i: population opp(i) comes back to this cell as direction i
        static_for<1, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            if ((lk >> i) & 1u) f(std::integral_constant<int, dir_opp(i)>{}, ip_read_at<i>(P, q, p, x));
        });
    }
    if (fl & EDGE_BIT) {
        // ghost slot (i, pt) of the two-buffer scheme = "the cell pt + c_i receives direction i"
        ghost_stores(P, x, y, z, lk, [&](int i, int pt, auto jc) {
            int cell = pt;
            if (i & 1) cell = pt + poff_rt(P, i) + ((dir_cx(i) == 1 && P.perx && x == P.nx - 1) ? -P.nx : 0);
            f(jc, (long long)ip_slot(q, i) * P.stride + cell);
        });
    }
}

// the stored (post-collision) state of a cell, whichever streaming scheme the handle uses; A = the current buffer.
// IPM: -1 = decided at run time (P.ipq; the small set-up kernels), 0 = two buffers, 1 = in place — the whole-lattice kernels
// (init, macros) are instantiated per scheme, so that the two-buffer instantiation carries none of the in-place code (with the
// run-time branch macros_kernel took 448 us instead of 243 us on config 3: registers)
template <typename real, typename S, int IPM = -1>
__device__ __forceinline__ void load_cell_any(real (&g)[Q], const S *__restrict__ A, const Params<real> &P, int p, int x, int y, int z,
                                              uint8_t fl, uint32_t lk)
{
    if constexpr (IPM == 0) load_cell(g, A, P.stride, p);
    else {
        if (IPM < 0 && P.ipq < 0) { load_cell(g, A, P.stride, p); return; }
        ip_visit(P, P.ipq, p, x, y, z, fl, lk, [&](auto jc, long long e) { g[decltype(jc)::value] = ld_s<real>(A + e); });
    }
}
template <typename real, typename S, int IPM = -1>
__device__ __forceinline__ void store_cell_any(S *__restrict__ A, const Params<real> &P, int p, int x, int y, int z, uint8_t fl,
                                               uint32_t lk, const real (&g)[Q])
{
    if constexpr (IPM == 0) store_cell(A, P, p, x, y, z, fl, lk, g);
    else {
        if (IPM < 0 && P.ipq < 0) { store_cell(A, P, p, x, y, z, fl, lk, g); return; }
        ip_visit(P, P.ipq, p, x, y, z, fl, lk, [&](auto jc, long long e) { st_s(A + e, g[decltype(jc)::value]); });
    }
}

// ---- a3 / a6: EQ face cells -------------------------------------------------------------------------------------------
// Both kinds of EQ cell hold f_eq(1, u) of a velocity that lives in a small side array fu[2 halves][3][F], one slot per
// face-plane cell of every EQ face:
//   EQ_FIXED   u = u_b, written (both halves) when the inlet profile / plane is set (DESIGN.md §3 step 5);
//   EQ_OUTFLOW u = u_loc(G_k, c - n) (step 6), n = outward normal of the cell's owner face.  u_loc(G_k, nb) is the
//              velocity the cell nb itself holds while it writes G_k (its collision velocity if FLUID), so nb
//              publishes it ("feeds") into the half that belongs to the buffer it writes, and the outflow cell reads
//              3 values next step instead of gathering nb's 19 populations.  Slots never fed (nb SOLID, box one
//              cell thick) stay 0 = the u = 0 the rule prescribes.
// Every EQ cell re-stores its 19 populations each step: a static cell inside a row would leave its 32-byte sector
// partially written, and on this HBM a partially written sector costs far more than the bytes (measured: two static
// cells per 400-cell row cost 10 % of the step).
// Owner face of an EQ cell = the first face of the matching type it lies on (order x-,x+,y-,y+,z-,z+).
template <typename real>
__device__ __forceinline__ int eq_owner(const Params<real> &P, int ftype, int x, int y, int z)
{
    if (x == 0 && P.face[0] == ftype) return 0;
    if (x == P.nx - 1 && P.face[1] == ftype) return 1;
    if (y == 0 && P.face[2] == ftype) return 2;
    if (y == P.ny - 1 && P.face[3] == ftype) return 3;
    if (z == 0 && P.face[4] == ftype) return 4;
    if (z == P.nz - 1 && P.face[5] == ftype) return 5;
    return -1;
}
template <typename real>
__device__ __forceinline__ int outflow_owner(const Params<real> &P, int x, int y, int z)
{
    return eq_owner(P, FACE_EQ_OUTFLOW, x, y, z);
}
template <typename real>
__device__ __forceinline__ int outflow_slot(const Params<real> &P, int k, int x, int y, int z)
{
    const int axis = k >> 1;
    const int j1 = axis == 0 ? y : x, j2 = axis == 2 ? y : z, n1 = axis == 0 ? P.ny : P.nx;
    return P.foff[k] + j2 * n1 + j1;
}
// slot of an EQ cell of class cls (EQ_FIXED / EQ_OUTFLOW); 0 if it has none (cannot happen for a voxelised EQ cell)
template <typename real>
__device__ __forceinline__ int eq_slot(const Params<real> &P, int cls, int x, int y, int z)
{
    const int k = eq_owner(P, cls == EQ_FIXED ? FACE_EQ_FIXED : FACE_EQ_OUTFLOW, x, y, z);
    return k < 0 ? 0 : outflow_slot(P, k, x, y, z);
}
// is (x,y,z) one layer inside some EQ_OUTFLOW face? (superset test used for FEED_BIT)
template <typename real>
__device__ __forceinline__ bool outflow_feeder(const Params<real> &P, int x, int y, int z)
{
    const int c[3] = {x, y, z}, n[3] = {P.nx, P.ny, P.nz};
    bool f = false;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const int a = k >> 1;
        f |= P.face[k] == FACE_EQ_OUTFLOW && n[a] > 1 && c[a] == ((k & 1) ? n[a] - 2 : 1);
    }
    return f;
}
// publish velocity u of cell (x,y,z) to every outflow cell whose inward neighbour it is; w(slot, component, value)
template <typename real, class W>
__device__ __forceinline__ void outflow_feed(const Params<real> &P, int x, int y, int z, real ux, real uy, real uz, W &&w)
{
    const int n[3] = {P.nx, P.ny, P.nz};
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const int a = k >> 1;
        int c[3] = {x, y, z};
        if (P.face[k] != FACE_EQ_OUTFLOW || n[a] < 2 || c[a] != ((k & 1) ? n[a] - 2 : 1)) continue;
        c[a] = (k & 1) ? n[a] - 1 : 0;
        if (outflow_owner(P, c[0], c[1], c[2]) != k) continue;
        const int s = outflow_slot(P, k, c[0], c[1], c[2]);
        w(s, 0, ux); w(s, 1, uy); w(s, 2, uz);
    }
}

// interior cell c = (z*ny + y)*nx + x  ->  coordinates (set-up and output kernels; not on the hot path)
template <typename real>
__device__ __forceinline__ void cell_xyz(const Params<real> &P, int c, int &x, int &y, int &z)
{
    x = c % P.nx;
    const int r = c / P.nx;
    y = r % P.ny;
    z = r / P.ny;
}

// a sub-box lo <= (x,y,z) < lo + bn of the lattice (the whole lattice: lo = 0, bn = n); cell c of the box, C order [bz][by][bx]
struct Box { int lo[3], bn[3]; };
__device__ __forceinline__ bool box_cell(const Box &bx, int c, int &x, int &y, int &z)
{
    if (c >= bx.bn[0] * bx.bn[1] * bx.bn[2]) return false;
    x = bx.lo[0] + c % bx.bn[0];
    const int r = c / bx.bn[0];
    y = bx.lo[1] + r % bx.bn[1];
    z = bx.lo[2] + r / bx.bn[1];
    return true;
}

__host__ __device__ inline double weight_f64(int i) { return i == 0 ? 1.0 / 3.0 : (i <= 6 ? 1.0 / 18.0 : 1.0 / 36.0); }

} // namespace lbmk
