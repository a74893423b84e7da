// lbm_setup.cuh — one-off kernels: voxelise (a1), link classification (a2), inlet write (a3), init (a4), precursor feed
// (a8), checkpoint in/out.  Rows of SURVEY.md §8(a); arithmetic of DESIGN.md §3.  Layout: lbm_core.cuh.
#pragma once
#include "lbm_core.cuh"

namespace lbmk {

// ---- a1: voxelise the padded box ---------------------------------------------------------------------------------------
// Interior: SOLID iff z < clamp(h[y][x], 0, nz), or mask[z][y][x] >= thresh when a solid mask is merged in (PAPER.md:51
// Boolean merge of base / terrain / building layers; the mask is a user's or the vote count of the mesh voxeliser,
// lbm_mesh.cuh); non-solid cells on an EQ face take the EQ class (EQ_FIXED wins).
// Halo: SOLID behind a WALL or EQ face (never pulled from / bounce-back), else the class follows the in-box image
// cell (PERIODIC: wrapped, FREE_SLIP: clamped): image solid -> SOLID (DESIGN.md §3 step 4a "mirrored source SOLID ->
// bounce-back"), else GHOST.  x padding beyond the halo: SOLID.
template <typename real>
__global__ void voxelise_kernel(const int32_t *__restrict__ height, const uint8_t *__restrict__ mask, int thresh,
                                uint8_t *__restrict__ flags, Params<real> P)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P.Np) return;
    int x = p % P.px - P.xoff, y = (p / P.px) % P.py - 1, z = p / P.pxy - 1;
    if (x < -1 || x > P.nx) { flags[p] = SOLID; return; }
    const int n[3] = {P.nx, P.ny, P.nz};
    int c[3] = {x, y, z};
    bool halo = false, dead = false;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const bool lo = c[a] < 0, hi = c[a] >= n[a];
        if (lo | hi) {
            halo = true;
            const int ft = lo ? P.face[2 * a] : P.face[2 * a + 1];
            if (ft == PERIODIC) c[a] = lo ? n[a] - 1 : 0;
            else if (ft == FREE_SLIP) c[a] = lo ? 0 : n[a] - 1;
            else dead = true;
        }
    }
    if (dead) { flags[p] = SOLID; return; }
    int h = height ? height[c[1] * P.nx + c[0]] : 0;
    h = min(max(h, 0), P.nz);
    if (mask && mask[((long long)c[2] * P.ny + c[1]) * P.nx + c[0]] >= thresh) h = P.nz;
    int cls;
    if (c[2] < h) cls = SOLID;
    else if (halo) cls = GHOST;
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
    flags[p] = (uint8_t)cls;
}

// ---- a2: link classification ---------------------------------------------------------------------------------------------
// FLUID cell: bit i (1..18) of links[p] <=> the pull source of direction i is SOLID in the padded box — exactly
// "step 4a takes the bounce-back branch" (DESIGN.md §3 step 9).  SOLID cell: bit i <=> the cell stores 0 into its slot i
// every step to complete a 32-byte sector that others write (internal; lbm_get_links reports 0 for it).
// Adds SLOW / EDGE / FEED / SURF bits to the flag byte in place (class bits are never changed, and readers mask them,
// so in-place is race-free).
template <typename real>
__global__ void classify_kernel(uint8_t *__restrict__ flags, uint32_t *__restrict__ links, Params<real> P)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    int x, y, z;
    cell_xyz(P, c, x, y, z);
    const int p = pidx(P, x, y, z);
    const int cls = flags[p] & CLASS_MASK;
    uint32_t bits = 0;
    uint8_t extra = 0;
    if (cls == FLUID) {
        static_for<1, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            bits |= (((flags[p - poff<i>(P)] & CLASS_MASK) == SOLID) ? 1u : 0u) << i;
        });
        if (bits) extra |= SLOW_BIT;
    } else if (cls == SOLID) {
        // slot i of this cell must be zero-filled every step iff some cell of its 32-byte sector is written in
        // population i (a live cell, or a solid cell whose slot i is a neighbour's mailbox) and this one is not
        const int s0 = p & ~(P.sec - 1); // the cells of the 32-byte sector (8 for FP32; also used for FP64: a superset; 16 for __half)
        uint32_t written = 0, own = 0;
        for (int q = s0; q < s0 + P.sec; ++q) {
            const int cq = flags[q] & CLASS_MASK;
            const int xq = q % P.px - P.xoff; // the sector lies in the cell's own row; at a row end it reaches into the x halo
            if (P.perx && (xq < 0 || xq >= P.nx)) continue; // PERIODIC x: nothing is ever stored in the x halo (xwrap)
            if (cq == FLUID || cq == EQ_OUTFLOW || cq == EQ_FIXED) written |= 0x7FFFFu;
            else if (cq == SOLID) {
                uint32_t mb = 0;
                static_for<1, Q>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    // the cell whose mailbox slot (i, q) is: the one that pulls direction i from q, across a periodic x face too
                    int t = q + poff<i>(P);
                    if (P.perx) {
                        if (dir_cx(i) == 1 && xq == P.nx - 1) t -= P.nx;
                        if (dir_cx(i) == -1 && xq == 0) t += P.nx;
                    }
                    if (t >= 0 && t < P.Np) mb |= (((flags[t] & CLASS_MASK) == FLUID) ? 1u : 0u) << i;
                });
                written |= mb;
                if (q == p) own = mb;
            }
        }
        bits = written & ~own;
        if (bits) extra |= SURF_BIT;
    }
    links[p] = bits;
    if (cls != SOLID) {
        // EDGE_BIT only where the ghost rule really stores something (not e.g. on the WALL ground or mid-face EQ cells)
        const bool edge = x == 0 || x == P.nx - 1 || y == 0 || y == P.ny - 1 || z == 0 || z == P.nz - 1;
        int nghost = 0;
        if (edge) ghost_stores(P, x, y, z, bits, [&](int, int, auto) { ++nghost; });
        if (nghost) extra |= EDGE_BIT;
        if (outflow_feeder(P, x, y, z)) extra |= FEED_BIT;
    }
    flags[p] = (uint8_t)(cls | extra);
}

// The same classification with the 3 x 3 x 3 class neighbourhood staged through shared memory: a CTA owns a tile of
// 32 (padded x, sector-aligned) x 4 x 4 cells and loads the classes of the tile and its one-cell halo once (1 224 bytes), so a
// flag byte is read ~2.4 times from L2 instead of 18 (FLUID) or up to 16 x 18 (SOLID) times: 277 -> ~60 us on config 3.
// Everything a cell looks at lies inside that box: its own 18 neighbours, the cells of its 32-byte sector (the tile's x range is
// a multiple of the sector) and their neighbours.  Only the read-side wrap of PERIODIC x faces reaches further (the other end of
// the row): that rare access goes to global memory.  Cells outside the padded row (X = -1, X = px) count as SOLID, which is what
// the linear index of classify_kernel finds there (row padding).  Same output bit for bit (tests/test_gpu_parity.py).
constexpr int CT_X = 32, CT_Y = 4, CT_Z = 4;
template <typename real>
__global__ void __launch_bounds__(CT_X *CT_Y *CT_Z)
classify_tiled_kernel(uint8_t *__restrict__ flags, uint32_t *__restrict__ links, Params<real> P)
{
    __shared__ uint8_t tile[CT_Z + 2][CT_Y + 2][CT_X + 2];
    const int X0 = blockIdx.x * CT_X, Y0 = 1 + blockIdx.y * CT_Y, Z0 = 1 + blockIdx.z * CT_Z; // padded coordinates of the tile origin
    const int pz = P.nz + 2;
    // one warp per row of the box (36 rows of 34 bytes, 16 warps): lane l loads tx = l + 1, lanes 0 / 1 also tx = 0 / 33
    const int lane = threadIdx.x, warp = threadIdx.z * CT_Y + threadIdx.y;
    int solid_seen = 0;
    for (int r = warp; r < (CT_Z + 2) * (CT_Y + 2); r += CT_Y * CT_Z) {
        const int tz = r / (CT_Y + 2), ty = r - tz * (CT_Y + 2);
        const int Y = Y0 - 1 + ty, Z = Z0 - 1 + tz;
        const bool row_ok = Y >= 0 && Y < P.py && Z >= 0 && Z < pz;
        const uint8_t *row = flags + (long long)(Z * P.py + Y) * P.px;
        const int X = X0 + lane;
        uint8_t c = (row_ok && X < P.px) ? (row[X] & CLASS_MASK) : (uint8_t)SOLID;
        tile[tz][ty][lane + 1] = c;
        solid_seen |= c == SOLID;
        if (lane < 2) {
            const int Xe = lane == 0 ? X0 - 1 : X0 + CT_X;
            c = (row_ok && Xe >= 0 && Xe < P.px) ? (row[Xe] & CLASS_MASK) : (uint8_t)SOLID;
            tile[tz][ty][lane == 0 ? 0 : CT_X + 1] = c;
            solid_seen |= c == SOLID;
        }
    }
    const int any_solid = __syncthreads_or(solid_seen); // also the barrier between the tile's writers and readers
    const int lx = threadIdx.x, ly = threadIdx.y, lz = threadIdx.z;
    const int x = X0 + lx - P.xoff, y = Y0 + ly - 1, z = Z0 + lz - 1;
    const bool inside = x >= 0 && x < P.nx && y < P.ny && z < P.nz;
    const int p = pidx(P, x, y, z);
    // the bulk of the lattice: no SOLID cell within reach of the tile and no domain face in it -> every cell is a plain FLUID
    // cell without wall link, ghost slot or feed (block-uniform test)
    // ("face" = the face layer or the layer inside it: a feeding cell sits one layer inside an EQ_OUTFLOW face)
    const bool on_face = X0 - P.xoff <= 1 || X0 + CT_X - 1 - P.xoff >= P.nx - 2 || Y0 - 1 <= 1 || Y0 + CT_Y - 2 >= P.ny - 2 ||
                         Z0 - 1 <= 1 || Z0 + CT_Z - 2 >= P.nz - 2;
    if (!any_solid && !on_face) {
        if (inside) {
            links[p] = 0u;
            flags[p] = tile[lz + 1][ly + 1][lx + 1];
        }
        return;
    }
    auto at = [&](int ax, int ay, int az) -> int { return tile[az + 1][ay + 1][ax + 1]; }; // class at tile-local coordinates
    const int cls = at(lx, ly, lz);
    // Which of its 19 slots does somebody write every step?  A live cell: all of them.  A SOLID cell (also one in the x halo
    // behind a WALL / EQ face): the slots that are a neighbour's bounce-back mailbox.  Each thread derives that for its own cell
    // once and shares it; a surface solid then ORs the entries of its 32-byte sector (the tile's x range is sector-aligned).
    __shared__ uint32_t wmask[CT_Z][CT_Y][CT_X];
    uint32_t w = 0;
    const bool row_in = y < P.ny && z < P.nz;
    if (row_in && x >= -1 && x <= P.nx && !(P.perx && (x < 0 || x >= P.nx))) { // PERIODIC x: nothing is ever stored in the x halo (xwrap)
        if (cls == FLUID || cls == EQ_OUTFLOW || cls == EQ_FIXED) w = 0x7FFFFu;
        else if (cls == SOLID) {
            static_for<1, Q>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                // the cell whose mailbox slot (i, this cell) is: the one that pulls direction i from here, across a periodic x face too
                int ct;
                if (P.perx && ((dir_cx(i) == 1 && x == P.nx - 1) || (dir_cx(i) == -1 && x == 0))) {
                    const int t = p + poff<i>(P) + (dir_cx(i) == 1 ? -P.nx : P.nx);
                    ct = (t >= 0 && t < P.Np) ? (flags[t] & CLASS_MASK) : SOLID;
                } else ct = at(lx + dir_cx(i), ly + dir_cy(i), lz + dir_cz(i));
                w |= ((ct == FLUID) ? 1u : 0u) << i;
            });
        }
    }
    wmask[lz][ly][lx] = w;
    __syncthreads();
    if (!inside) return;
    uint32_t bits = 0;
    uint8_t extra = 0;
    if (cls == FLUID) {
        static_for<1, Q>([&](auto ic) {
            constexpr int i = decltype(ic)::value;
            bits |= ((at(lx - dir_cx(i), ly - dir_cy(i), lz - dir_cz(i)) == SOLID) ? 1u : 0u) << i;
        });
        if (bits) extra |= SLOW_BIT;
    } else if (cls == SOLID) {
        const int s0 = lx & ~(P.sec - 1); // the cells of the 32-byte sector, tile-local (X0 is a multiple of the sector)
        uint32_t written = 0;
        for (int qx = s0; qx < s0 + P.sec; ++qx) written |= wmask[lz][ly][qx];
        bits = written & ~w; // w = this cell's own mailbox slots: their owners write them
        if (bits) extra |= SURF_BIT;
    }
    links[p] = bits;
    if (cls != SOLID) {
        const bool edge = x == 0 || x == P.nx - 1 || y == 0 || y == P.ny - 1 || z == 0 || z == P.nz - 1;
        int nghost = 0;
        if (edge) ghost_stores(P, x, y, z, bits, [&](int, int, auto) { ++nghost; });
        if (nghost) extra |= EDGE_BIT;
        if (outflow_feeder(P, x, y, z)) extra |= FEED_BIT;
    }
    flags[p] = (uint8_t)(cls | extra);
}

// store one cell's state into BOTH buffers (boundary cells rewritten while a run is under way: whichever buffer is current
// must hold them) or, with B == nullptr, into A only (whole-lattice writes, after which A is the current buffer: the first
// step rewrites every slot of B that is ever read — own slots, mailboxes, ghost slots, EQ cells, sector completions — so
// filling B too would be 76 B per cell of wasted writes), and publish its velocity to the outflow cells it feeds (both
// halves of the double-buffered side array)
template <typename real, typename S, int IPM = -1>
__device__ __forceinline__ void store_cell_both(S *__restrict__ A, S *__restrict__ B, real *__restrict__ fu, const Params<real> &P,
                                                int p, int x, int y, int z, uint8_t fl, uint32_t lk, const real (&g)[Q])
{
    store_cell_any<real, S, IPM>(A, P, p, x, y, z, fl, lk, g);
    if (IPM != 1 && B && P.ipq < 0) store_cell(B, P, p, x, y, z, fl, lk, g); // B == nullptr: whole-lattice writes (init, checkpoint) fill the current buffer only; in-place streaming: there is one buffer
    const int cls = fl & CLASS_MASK;
    if ((fl & FEED_BIT) || cls == EQ_FIXED) {
        const Macro<real> m = local_macros(g, cls, P, damp_at(P, x, y, z));
        auto w = [&](int s, int comp, real v) {
            fu[comp * P.F + s] = v;
            fu[(3 + comp) * P.F + s] = v;
        };
        if (fl & FEED_BIT) outflow_feed(P, x, y, z, m.ux, m.uy, m.uz, w);
        if (cls == EQ_FIXED) { // the boundary velocity the step kernel re-expands every step
            const int s = eq_slot(P, EQ_FIXED, x, y, z);
            w(s, 0, m.ux); w(s, 1, m.uy); w(s, 2, m.uz);
        }
    }
}

// the boundary velocity of an EQ_FIXED cell exactly as prescribed (store_cell_both publishes the moments of the
// equilibrium, which carry rounding noise: a prescribed 0 could become -1e-19 and flip the active-inflow test)
template <typename real>
__device__ __forceinline__ void publish_fixed(real *__restrict__ fu, const Params<real> &P, int x, int y, int z, real ux, real uy, real uz)
{
    const int s = eq_slot(P, EQ_FIXED, x, y, z);
    fu[s] = ux; fu[P.F + s] = uy; fu[2 * P.F + s] = uz;
    fu[3 * P.F + s] = ux; fu[4 * P.F + s] = uy; fu[5 * P.F + s] = uz;
}

// ---- a3: inlet write -------------------------------------------------------------------------------------------------
template <typename real>
__device__ __forceinline__ bool fixed_slot_cell(const Params<real> &P, const uint8_t *__restrict__ flags, int sl, int &k, int &x, int &y,
                                                int &z);

// mode 0: profile prof[nz] per component by level, one thread per face-velocity slot (= per face-plane cell of every EQ
// face; a cell is handled by the slot of its owner face); mode 1: plane uvw[3][n2][n1] of one face, one thread per plane cell
template <typename real, typename S, typename in_t>
__global__ void inlet_kernel(S *__restrict__ A, S *__restrict__ B, real *__restrict__ fu, const uint8_t *__restrict__ flags,
                             const in_t *__restrict__ pu, const in_t *__restrict__ pv, const in_t *__restrict__ pw,
                             int mode, int face, Params<real> P)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    int x, y, z;
    long long src;
    if (mode == 0) {
        int k;
        if (t >= P.F || !fixed_slot_cell(P, flags, t, k, x, y, z)) return;
        src = z;
    } else {
        const int axis = face >> 1;
        const int n1 = axis == 0 ? P.ny : P.nx;
        const int n2 = axis == 2 ? P.ny : P.nz;
        if (t >= n1 * n2) return;
        const int j1 = t % n1, j2 = t / n1;
        const int nn[3] = {P.nx, P.ny, P.nz};
        const int fixed = (face & 1) ? nn[axis] - 1 : 0;
        if (axis == 0) { x = fixed; y = j1; z = j2; }
        else if (axis == 1) { x = j1; y = fixed; z = j2; }
        else { x = j1; y = j2; z = fixed; }
        src = t;
    }
    const int p = pidx(P, x, y, z);
    const uint8_t fl = flags[p];
    if ((fl & CLASS_MASK) != EQ_FIXED) return;
    const real ux = real(pu[src]), uy = pv ? real(pv[src]) : real(0), uz = pw ? real(pw[src]) : real(0);
    real g[Q];
    equilibrium(g, real(0), ux, uy, uz);
    store_cell_both(A, B, fu, P, p, x, y, z, fl, 0u, g);
    publish_fixed(fu, P, x, y, z, ux, uy, uz);
}

// ---- synthetic inflow fluctuations (lbm_set_inflow_turbulence; Table 1) -------------------
// One thread per face-velocity slot.  For an EQ_FIXED cell whose MEAN velocity (fum) points into the domain
// (ub . n < -1e-7, n = outward normal of the owner face) the boundary velocity of time t is
//     u_b = ub + sum_n a_n cos(kappa_n . x + psi_n - omega_n t),     a_n = 2 sqrt(E(|kappa_n|) dkappa_n) sigma_n,
// x = cell indices (DESIGN.md §4 reading 21); all other EQ_FIXED cells keep the mean.  modes = [n][8] doubles:
// kappa[3], a[3], psi, omega (amplitudes folded on the host).  The phase is formed and reduced to [-pi, pi] in FP64 (t
// reaches 1e4-1e5 steps, an FP32 phase would lose 1e-3 rad), the cosine is taken in the handle's precision.
// The value goes to the side array: the step kernel re-expands f_eq(1, u_b) from it (a3).
template <typename real>
struct Turb { const real *fum; const double *modes; int n; double t; };

// one slot: boundary velocity of time t -> dst0 / dst1 (the halves to publish to; dst1 may be null)
template <typename real, bool CELLS, typename S = real>
__device__ __forceinline__ void fluct_slot(int s, S *__restrict__ A, S *__restrict__ B, real *__restrict__ fu, real *__restrict__ dst0,
                                           real *__restrict__ dst1, const uint8_t *__restrict__ flags, const Turb<real> &tb, const Params<real> &P)
{
    int k = 5;
    while (k > 0 && s < P.foff[k]) --k; // the last face whose first slot is <= s (faces without slots share their successor's offset)
    if (P.face[k] != FACE_EQ_FIXED) return;
    const int axis = k >> 1;
    const int n1 = axis == 0 ? P.ny : P.nx;
    const int r = s - P.foff[k], j1 = r % n1, j2 = r / n1;
    const int fixed = (k & 1) ? (axis == 0 ? P.nx : (axis == 1 ? P.ny : P.nz)) - 1 : 0;
    int x, y, z;
    if (axis == 0) { x = fixed; y = j1; z = j2; }
    else if (axis == 1) { x = j1; y = fixed; z = j2; }
    else { x = j1; y = j2; z = fixed; }
    if (eq_owner(P, FACE_EQ_FIXED, x, y, z) != k) return; // an edge cell belongs to the first EQ_FIXED face it lies on
    const int p = pidx(P, x, y, z);
    const uint8_t fl = flags[p];
    if ((fl & CLASS_MASK) != EQ_FIXED) return;
    real u0 = tb.fum[s], u1 = tb.fum[P.F + s], u2 = tb.fum[2 * P.F + s];
    const real ua = axis == 0 ? u0 : (axis == 1 ? u1 : u2);
    const double un = (k & 1) ? (double)ua : -(double)ua;
    if (un < -1e-7) { // "active inflow": inward by more than rounding noise (DESIGN.md §4 reading 21); compared in FP64 like the oracle
        real a0 = real(0), a1 = real(0), a2 = real(0);
        const double xd = (double)x, yd = (double)y, zd = (double)z;
        for (int n = 0; n < tb.n; ++n) {
            const double *m = tb.modes + 8 * n;
            double ph = fma(m[0], xd, fma(m[1], yd, fma(m[2], zd, fma(-m[7], tb.t, m[6]))));
            real c;
            if constexpr (sizeof(real) == 8) c = cos(ph);
            else {
                ph = fma(-6.283185307179586, rint(ph * 0.15915494309189535), ph);
                c = cosf((float)ph);
            }
            a0 = fma(c, real(m[3]), a0); a1 = fma(c, real(m[4]), a1); a2 = fma(c, real(m[5]), a2);
        }
        u0 += a0; u1 += a1; u2 += a2;
    }
    if constexpr (CELLS) {
        real g[Q];
        equilibrium(g, real(0), u0, u1, u2);
        store_cell_both(A, B, fu, P, p, x, y, z, fl, 0u, g);
    }
    dst0[s] = u0; dst0[P.F + s] = u1; dst0[2 * P.F + s] = u2;
    if (dst1) { dst1[s] = u0; dst1[P.F + s] = u1; dst1[2 * P.F + s] = u2; }
}

// stand-alone form (set-up, switch-off, re-initialisation): both halves; CELLS = also the cells' populations in both buffers.
// During a run the step kernel itself carries the slots (lbm_step.cuh, TURB blocks): no extra launch.
template <typename real, typename S, bool CELLS>
__global__ void fluct_kernel(S *__restrict__ A, S *__restrict__ B, real *__restrict__ fu, const uint8_t *__restrict__ flags,
                             const Turb<real> tb, Params<real> P)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P.F) return;
    fluct_slot<real, CELLS, S>(s, A, B, fu, fu, fu + 3 * (size_t)P.F, flags, tb, P);
}

// Re-publish the velocities the outflow cells will read next step from the CURRENT state (both halves of the side
// array).  Needed when something that enters the local macro inversion changes between steps (lbm_set_damping): the
// rule is u_loc(G_k, c - n) evaluated with the parameters in force when the step runs (DESIGN.md §3 step 6).
template <typename real, typename S>
__global__ void refeed_kernel(const S *__restrict__ A, real *__restrict__ fu, const uint8_t *__restrict__ flags,
                              const uint32_t *__restrict__ links, Params<real> P, const real *__restrict__ H = nullptr)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    int x, y, z;
    cell_xyz(P, c, x, y, z);
    const int p = pidx(P, x, y, z);
    const uint8_t fl = flags[p];
    if (!(fl & FEED_BIT)) return;
    real g[Q];
    load_cell_any(g, A, P, p, x, y, z, fl, (fl & SLOW_BIT) ? links[p] : 0u);
    if (H) // thermal lattice on (H = its current state, 7 shifted populations): the cell's buoyancy belongs to its force (lbm_thermal.cuh)
        P.Fz += P.gbeta * (H[p] + ((H[P.stride + p] + H[2 * P.stride + p]) + (H[3 * P.stride + p] + H[4 * P.stride + p]) +
                                   (H[5 * P.stride + p] + H[6 * P.stride + p])));
    const Macro<real> m = local_macros(g, fl & CLASS_MASK, P, damp_at(P, x, y, z));
    outflow_feed(P, x, y, z, m.ux, m.uy, m.uz, [&](int s, int comp, real v) {
        fu[comp * P.F + s] = v;
        fu[(3 + comp) * P.F + s] = v;
    });
}

// ---- a8: precursor plane -> main inlet (config 5) -----------------------------------------------------------------------
template <typename real, typename S>
__global__ void feed_kernel(S *__restrict__ dA, S *__restrict__ dB, real *__restrict__ dfu, const uint8_t *__restrict__ dflags,
                            Params<real> D,
                            const S *__restrict__ sA, const uint8_t *__restrict__ sflags, const uint32_t *__restrict__ slinks,
                            Params<real> Ps, int sx)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= D.ny * D.nz) return;
    const int y = t % D.ny, z = t / D.ny;
    const int dp = pidx(D, 0, y, z);
    const uint8_t fl = dflags[dp];
    if ((fl & CLASS_MASK) != EQ_FIXED) return;
    const int sp = pidx(Ps, sx, y % Ps.ny, z);
    real g[Q];
    const uint8_t sfl = sflags[sp];
    load_cell_any(g, sA, Ps, sp, sx, y % Ps.ny, z, sfl, (sfl & SLOW_BIT) ? slinks[sp] : 0u);
    const Macro<real> m = local_macros(g, sfl & CLASS_MASK, Ps, damp_at(Ps, sx, y % Ps.ny, z));
    equilibrium(g, real(0), m.ux, m.uy, m.uz);
    store_cell_both(dA, dB, dfu, D, dp, 0, y, z, fl, 0u, g);
    publish_fixed(dfu, D, 0, y, z, m.ux, m.uy, m.uz);
}

// ---- a4: init ------------------------------------------------------------------------------------------------------------
// G0 = f_eq(rho0, u0) in FLUID and EQ_OUTFLOW cells (EQ_FIXED keep their boundary state; SOLID cells hold mailboxes)
template <typename real, typename S, typename in_t, int IPM>
__global__ void init_kernel(S *__restrict__ A, S *__restrict__ B, real *__restrict__ fu, const uint8_t *__restrict__ flags,
                            const uint32_t *__restrict__ links, const in_t *__restrict__ rho, const in_t *__restrict__ ux,
                            const in_t *__restrict__ uy, const in_t *__restrict__ uz, Params<real> P)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    int x, y, z;
    cell_xyz(P, c, x, y, z);
    const int p = pidx(P, x, y, z);
    const uint8_t fl = flags[p];
    const int cls = fl & CLASS_MASK;
    if (cls == EQ_FIXED || cls == SOLID) return;
    const real drho = rho ? real(rho[c] - in_t(1)) : real(0);
    const real u = ux ? real(ux[c]) : real(0), v = uy ? real(uy[c]) : real(0), w = uz ? real(uz[c]) : real(0);
    real g[Q];
    equilibrium(g, drho, u, v, w);
    store_cell_both<real, S, IPM>(A, B, fu, P, p, x, y, z, fl, links[p], g);
}

// ---- checkpoint ------------------------------------------------------------------------------------------------------------
// f [19][bz][by][bx] double, NOT shifted, of the box lo <= (x,y,z) < lo + bn (the whole lattice: lo = 0, bn = n).  SOLID cells
// export the rest state w_i (their slots are mailboxes).
template <typename real, typename S>
__global__ void state_out_kernel(const S *__restrict__ A, const uint8_t *__restrict__ flags, const uint32_t *__restrict__ links,
                                 double *__restrict__ f, Params<real> P, const Box bx)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    int x, y, z;
    if (!box_cell(bx, c, x, y, z)) return;
    const long long NB = (long long)bx.bn[0] * bx.bn[1] * bx.bn[2];
    const int p = pidx(P, x, y, z);
    const uint8_t fl = flags[p];
    const bool solid = (fl & CLASS_MASK) == SOLID;
    real g[Q];
    if (!solid) load_cell_any(g, A, P, p, x, y, z, fl, (fl & SLOW_BIT) ? links[p] : 0u);
#pragma unroll
    for (int i = 0; i < Q; ++i) f[(long long)i * NB + c] = (solid ? 0.0 : double(g[i])) + weight_f64(i);
}

template <typename real, typename S>
__global__ void state_in_kernel(S *__restrict__ A, S *__restrict__ B, real *__restrict__ fu, const uint8_t *__restrict__ flags,
                                const uint32_t *__restrict__ links, const double *__restrict__ f, Params<real> P, const Box bx)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    int x, y, z;
    if (!box_cell(bx, c, x, y, z)) return;
    const long long NB = (long long)bx.bn[0] * bx.bn[1] * bx.bn[2];
    const int p = pidx(P, x, y, z);
    const uint8_t fl = flags[p];
    if ((fl & CLASS_MASK) == SOLID) return;
    real g[Q];
#pragma unroll
    for (int i = 0; i < Q; ++i) g[i] = real(f[(long long)i * NB + c] - weight_f64(i));
    store_cell_both(A, B, fu, P, p, x, y, z, fl, links[p], g);
}

// ---- global flux-balancing correction of the open-boundary velocities -----------------------------------------------------
// PAPER.md:55 ("the minimal normal velocity adjustment required to enforce near-zero net volume flow")
// ("a global flux-balancing correction is applied over the full set of open boundaries"), sign PAPER.md:185 (positive =
// outflow).  Open-boundary cells = EQ_FIXED cells, each owned by the first EQ_FIXED face it lies on; their velocities
// live in the face-velocity buffer.  Phi = sum u_b . n; correction u_b <- u_b - (Phi / N) n, then f_eq(1, u_b) again.
// One thread per face-velocity slot; (k, x, y, z) of slot sl, false if the slot is not an EQ_FIXED cell's own slot.
template <typename real>
__device__ __forceinline__ bool fixed_slot_cell(const Params<real> &P, const uint8_t *__restrict__ flags, int sl, int &k, int &x, int &y,
                                                int &z)
{
    k = -1;
    for (int q = 0; q < 6; ++q)
        if ((P.face[q] == FACE_EQ_FIXED || P.face[q] == FACE_EQ_OUTFLOW) && sl >= P.foff[q]) k = q;
    if (k < 0 || P.face[k] != FACE_EQ_FIXED) return false;
    const int axis = k >> 1, idx = sl - P.foff[k];
    const int n1 = axis == 0 ? P.ny : P.nx, n2 = axis == 2 ? P.ny : P.nz;
    if (idx >= n1 * n2) return false;
    const int j1 = idx % n1, j2 = idx / n1;
    const int nn[3] = {P.nx, P.ny, P.nz};
    const int fixed = (k & 1) ? nn[axis] - 1 : 0;
    if (axis == 0) { x = fixed; y = j1; z = j2; }
    else if (axis == 1) { x = j1; y = fixed; z = j2; }
    else { x = j1; y = j2; z = fixed; }
    if ((flags[pidx(P, x, y, z)] & CLASS_MASK) != EQ_FIXED) return false;
    return eq_owner(P, FACE_EQ_FIXED, x, y, z) == k;
}

// acc[0] += sum of u_b . n, acc[1] += number of open-boundary cells
template <typename real>
__global__ void flux_sum_kernel(const real *__restrict__ fu, const uint8_t *__restrict__ flags, double *__restrict__ acc, Params<real> P)
{
    const int sl = blockIdx.x * blockDim.x + threadIdx.x;
    double un = 0.0, cnt = 0.0;
    int k, x, y, z;
    if (sl < P.F && fixed_slot_cell(P, flags, sl, k, x, y, z)) {
        un = (double)fu[(k >> 1) * P.F + sl] * ((k & 1) ? 1.0 : -1.0);
        cnt = 1.0;
    }
    for (int o = 16; o > 0; o >>= 1) {
        un += __shfl_down_sync(0xffffffffu, un, o);
        cnt += __shfl_down_sync(0xffffffffu, cnt, o);
    }
    if ((threadIdx.x & 31) == 0 && cnt != 0.0) { atomicAdd(&acc[0], un); atomicAdd(&acc[1], cnt); }
}

template <typename real, typename S>
__global__ void flux_apply_kernel(S *__restrict__ A, S *__restrict__ B, real *__restrict__ fu, const uint8_t *__restrict__ flags,
                                  const double *__restrict__ acc, Params<real> P)
{
    const int sl = blockIdx.x * blockDim.x + threadIdx.x;
    int k, x, y, z;
    if (sl >= P.F || !fixed_slot_cell(P, flags, sl, k, x, y, z)) return;
    if (acc[1] == 0.0) return;
    const double shift = acc[0] / acc[1];
    real u[3] = {fu[sl], fu[P.F + sl], fu[2 * P.F + sl]};
    u[k >> 1] = real((double)u[k >> 1] - shift * ((k & 1) ? 1.0 : -1.0));
    real g[Q];
    equilibrium(g, real(0), u[0], u[1], u[2]);
    const int p = pidx(P, x, y, z);
    store_cell_both(A, B, fu, P, p, x, y, z, flags[p], 0u, g);
#pragma unroll
    for (int c = 0; c < 3; ++c) { fu[c * P.F + sl] = u[c]; fu[(3 + c) * P.F + sl] = u[c]; } // the exact corrected velocity
}

} // namespace lbmk
