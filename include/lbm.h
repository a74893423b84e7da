/*
 * lbm.h — C ABI of the B200-native D3Q19 LBM-LES stream-collide library
 *         (paper_2607_04516_b200/liblbm_b200.so, built for sm_100a).
 *
 * What the calls are.  The paper's problem statement for the solver (§2, Table 1
 * PAPER.md:77-89, boundary set-up PAPER.md:175-179): a voxelised solid mask on a uniform Cartesian
 * lattice, boundary wind data on the outer faces, N explicit
 * lattice-Boltzmann steps, then the macroscopic fields and their time averages
 * ("per-step macroscopic reconstruction"; averaging window PAPER.md:388).  The arithmetic of
 * every call is the algorithm statement in DESIGN.md §3 (steps 1-9), which restates the methods the paper
 * names (D3Q19, BGK, Smagorinsky-Lilly from non-equilibrium moments, Guo-forced Coriolis, equilibrium
 * velocity boundaries, no-slip solids: Table 1) — the paper prints no formula.
 *
 * Conventions (all calls)
 *   - Every function returns LBM_OK (0) or a negative LBM_E* code; nothing throws or aborts.  After an
 *     error lbm_last_error(h) describes it.  A NULL handle gives LBM_EINVAL.
 *   - Arrays are C order [z][y][x] (x fastest); nx,ny,nz are cell counts.  "real" below is float for the
 *     plain entry points and double for the *_f64 twins; both work on FP32 and FP64 handles.
 *   - Input arrays are borrowed for the duration of the call and copied.  Output arrays are allocated by
 *     the caller.  Array arguments may be HOST or DEVICE pointers unless stated; the library asks the
 *     CUDA runtime which (cudaPointerGetAttributes).  Host arrays are copied on the handle's stream and
 *     the call returns after the copy has completed.
 *   - lbm_step is asynchronous on the handle's stream.  Getters that write to host memory synchronise;
 *     getters that write to device memory are stream-ordered (call lbm_sync before reading elsewhere).
 *   - The handle owns its device memory unless lbm_create_ex was given a caller-owned workspace, which the
 *     caller must keep alive until lbm_destroy.
 *   - There is no CPU fallback: without a CUDA device every call that needs one returns LBM_ECUDA.
 */
#ifndef LBM_B200_H
#define LBM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lbm lbm_t; /* opaque; owned by the library */

enum { LBM_OK = 0, LBM_EINVAL = -1, LBM_ENOMEM = -2, LBM_ECUDA = -3, LBM_ESTATE = -4 };

/* face types, used in face_type[6] = {x-, x+, y-, y+, z-, z+}  (DESIGN.md §3 step 4a, 5, 6) */
enum {
    LBM_PERIODIC   = 0, /* wrap; must be set on both faces of an axis                                  */
    LBM_WALL       = 1, /* halfway bounce-back, wall half a cell outside the last node                 */
    LBM_FREE_SLIP  = 2, /* halfway specular reflection                                                 */
    LBM_EQ_FIXED   = 3, /* face cells hold f_eq(1, u_b): the "equilibrium-based velocity" face PAPER.md:175 */
    LBM_EQ_OUTFLOW = 4  /* face cells hold f_eq(1, u of the inward neighbour at the previous step)     */
};

/* cell classes returned by lbm_get_flags (DESIGN.md §3 step 3, 9) */
enum { LBM_FLUID = 0, LBM_SOLID = 1, LBM_CELL_EQ_FIXED = 2, LBM_CELL_EQ_OUTFLOW = 3 };

/* Precision of a handle: what the arithmetic runs in and how the 19 populations per cell are stored.
 *   LBM_PREC_F32      FP32 arithmetic, FP32 storage: 153 B per cell and step (BASELINE.json north_star; the headline path)
 *   LBM_PREC_F64      FP64 arithmetic and storage: the reference twin of the same kernels (1 = the old `fp64 != 0`)
 *   LBM_PREC_F32_S16  FP32 arithmetic, 16-bit population storage: what is stored
 *                     of population i is the shifted value f_i - w_i rounded to IEEE binary16 (round to nearest even)
 *                     every time it is written — 77 B per cell and step, half the memory.  Every call works the same;
 *                     lbm_get_state returns the stored (rounded) values, lbm_set_state rounds its input.  Not combinable
 *                     with the thermal lattice (lbm_set_thermal returns LBM_EINVAL). */
enum { LBM_PREC_F32 = 0, LBM_PREC_F64 = 1, LBM_PREC_F32_S16 = 2 };

/* Streaming scheme, OR-ed into the `precision` argument of lbm_workspace_bytes / lbm_create_ex ("in-place
 * streaming").  Default (bit clear): two population buffers, A -> B pull.  LBM_STREAM_INPLACE: ONE population
 * buffer — every step reads and overwrites the same 19 addresses per cell, the two slots of a lattice link swapping roles from
 * step to step — so a lattice takes about half the memory (config 5's 2.9e8 cells: 24 GB instead of 46 GB; 1.2e9 FP32 cells fit
 * one B200), for the same 153 B per cell and step and the same arithmetic: every call works the same and returns the same
 * values (lbm_get_state / lbm_set_state exchange the same post-collision populations).  Combinable with all three precisions,
 * every face type, damping zones, flux correction, synthetic inflow fluctuations, the time mean, lbm_feed_inlet (either side) and
 * the thermal lattice (whose seven populations per cell stay double-buffered: 19 + 14 instead of 38 + 14 stored values per cell);
 * lbm_set_variant has no effect (one launch shape: one cell per thread, one launch per step). */
#define LBM_STREAM_INPLACE 16

/* Bytes of device workspace a handle of this size needs (two population buffers of 19 stored values per cell — one with
 * LBM_STREAM_INPLACE —, one flag byte and one link word per cell, optional 3 reals per cell of time-mean sums, small
 * profile/plane scratch).  precision: LBM_PREC_* [| LBM_STREAM_INPLACE]; anything else returns LBM_EINVAL. */
int lbm_workspace_bytes(int nx, int ny, int nz, int want_mean, int precision, size_t *out);

/* Create an FP32 handle that allocates its own workspace (cudaMalloc) and uses the default stream.
 * nu0: molecular viscosity (tau0 = 3 nu0 + 1/2); Cs: Smagorinsky constant; f_cor: Coriolis parameter about z
 * (acceleration f_cor (u_y, -u_x, 0)); F[3]: uniform acceleration (pressure-gradient drive), host pointer,
 * NULL = 0.  All in lattice units.  Faces default to {EQ_FIXED, EQ_OUTFLOW, PERIODIC, PERIODIC, WALL,
 * FREE_SLIP} (BASELINE.json configs[0]).  Mean sums are allocated (want_mean = 1). */
int lbm_create(int nx, int ny, int nz, double nu0, double Cs, double f_cor, const double F[3], lbm_t **out);

/* Same, with a caller-owned DEVICE workspace of at least lbm_workspace_bytes() bytes (256-byte aligned;
 * NULL = allocate), a cudaStream_t passed as void* (NULL = default stream), and the precision (LBM_PREC_*, optionally
 * | LBM_STREAM_INPLACE).
 * want_mean = 0 omits the time-mean sums (lbm_mean_config then returns LBM_ESTATE). */
int lbm_create_ex(int nx, int ny, int nz, double nu0, double Cs, double f_cor, const double F[3],
                  void *dev_workspace, size_t workspace_bytes, void *cuda_stream, int precision, int want_mean,
                  lbm_t **out);

int lbm_destroy(lbm_t *h);

/* Face types, order x-,x+,y-,y+,z-,z+.  Invalidates the flags: call lbm_set_flags afterwards. */
int lbm_set_boundaries(lbm_t *h, const int face_type[6]);

/* Full Coriolis rotation vector (Table 1: "full rotation vector in the local ENU frame ...
 * evaluated directly within the GPU kernel"): f = 2 Omega in lattice units (rad per step), host pointer; the
 * acceleration is -f x u, applied through Guo forcing with the implicit half-force velocity (DESIGN.md §3 step 4c).
 * lbm_create's scalar f_cor is the vector (0, 0, f_cor).  Takes effect at the next lbm_step; may be called at any time. */
int lbm_set_coriolis(lbm_t *h, const double f[3]);

/* Voxelise ("solid mask"; heightmap form per north_star): cell (x,y,z) is SOLID iff
 * z < clamp(height[y][x], 0, nz); non-solid cells on an EQ face take the EQ class (EQ_FIXED wins);
 * then classify the wall links of every FLUID cell.  Integer work, done on the device.
 * height: int32 [ny][nx], host or device; NULL = flat ground (all 0).
 * Resets the populations to the rest state (rho = 1, u = 0) and the step counter and mean sums to 0. */
int lbm_set_flags(lbm_t *h, const int32_t *height);

/* a1 with a general solid mask merged in ("The final solid mask is assembled by the Boolean merging of a
 * fixed-thickness base layer, the terrain layer, and the building layer"): SOLID <=> z < clamp(height[y][x], 0, nz) OR
 * solid[z][y][x] != 0.  solid: uint8 [nz][ny][nx], host or device, borrowed for the call; NULL = lbm_set_flags.  Overhangs,
 * bridges and hollow shapes are allowed: the link classification and the step kernel work from the flags alone. */
int lbm_set_flags_mask(lbm_t *h, const int32_t *height, const uint8_t *solid);

/* a1 in the paper's own form: voxelise a triangle mesh on the device ("casting axis-aligned rays through grid
 * columns and computing ray-triangle intersections, using an odd-even parity rule along each column ... corroborate
 * independent passes along different ray directions for solid labeling"), then merge it with the heightmap layer as above.
 * tri: float [n_tri][3 vertices][x,y,z] in lattice units (cell (x,y,z) has its centre at (x+1/2, y+1/2, z+1/2); the ground
 * face is z = 0), host or device, borrowed.  Reading (DESIGN.md §4 reading 22), exact integer arithmetic: vertices snapped
 * to 1/256 cell (rint), must lie in [-1024, 2048) cells; pass d casts rays along axis d through the cell centres; a
 * triangle is hit iff the ray's foot point lies inside its projection (taken counter-clockwise, top-left rule on edges,
 * zero-area projections skipped); a crossing flips every cell whose centre is at or beyond it; SOLID iff at least
 * min_votes (1..3; 2 = majority) of the three passes end odd.  Orientation of the triangles is irrelevant; the mesh
 * should be closed (a hole corrupts only the rays through it, which the vote out-numbers).  n_tri = 0: heightmap only.
 * LBM_EINVAL: min_votes out of range, NULL tri, a vertex not finite or out of range.  Synchronises. */
int lbm_set_flags_mesh(lbm_t *h, const int32_t *height, int n_tri, const float *tri, int min_votes);

/* The same mesh voxeliser (DESIGN.md §4 reading 22; same tie rules, same kernels) WITHOUT a handle and
 * WITHOUT any allocation: for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it).  The scratch of the ray-cast passes lives in a file-scope device array inside the library, sized
 * for boxes of at most LBM_STATIC_VOXEL_MAX_CELLS cells (2^21 = 128^3; 4 MiB held by every GPU that loads the library until
 * the process exits); nx ny nz beyond that returns LBM_EINVAL with a message naming the limit — use lbm_set_flags_mesh there.
 * dev_tri: float [n_tri][3][3], DEVICE memory; dev_solid: uint8 [nz][ny][nx], DEVICE memory, 1 = SOLID (at least min_votes
 * of the three passes odd), 0 otherwise — both the caller's (host pointers are refused: staging them would allocate).
 * cuda_stream: a cudaStream_t passed as void* (NULL = default stream).  Runs on the CURRENT device; calls no cudaMalloc,
 * cudaFree or allocating library routine.  Synchronises the stream (the out-of-range-vertex flag is read back).
 * Every call shares the one scratch array, which keeps the last call's contents (the call clears what must start at zero):
 * calls that OVERLAP on the GPU — other streams, other host threads — race; serialise them.
 * err: optional host buffer of err_len bytes for the message (no handle to keep it).  LBM_EINVAL: size beyond the limit, bad
 * sizes / min_votes / NULL or host pointers, a vertex not finite or out of range.  LBM_ECUDA: a CUDA call failed. */
#define LBM_STATIC_VOXEL_MAX_CELLS 2097152
int lbm_voxelise_mesh_static(int nx, int ny, int nz, int n_tri, const float *dev_tri, int min_votes, uint8_t *dev_solid,
                             void *cuda_stream, char *err, size_t err_len);

/* Boundary wind profile ("macroscopic boundary states"): every EQ_FIXED cell at level z is set
 * to f_eq(1, (u[z], v[z], w[z])).  Each array [nz]; v, w may be NULL (= 0).  Needs flags. */
int lbm_set_inlet_profile(lbm_t *h, const float *u, const float *v, const float *w);
int lbm_set_inlet_profile_f64(lbm_t *h, const double *u, const double *v, const double *w);

/* Per-cell boundary state of one face: uvw is [3][n2][n1] with (n2,n1) = (nz,ny) on x faces, (nz,nx) on
 * y faces, (ny,nx) on z faces.  Only the EQ_FIXED cells of that face are written. */
int lbm_set_inlet_plane(lbm_t *h, int face, const float *uvw);
int lbm_set_inlet_plane_f64(lbm_t *h, int face, const double *uvw);

/* Global flux-balancing correction of the prescribed open-boundary velocities ("the minimal normal velocity
 * adjustment required to enforce near-zero net volume flow"; "applied over the full set of open boundaries").
 * Open-boundary cells = the EQ_FIXED cells, each owned by the first EQ_FIXED face it lies on (order x-,x+,y-,y+,z-,z+),
 * n = that face's outward normal.  Phi = sum u_b . n over them (positive = outflow); every such cell gets
 * u_b <- u_b - (Phi / N) n and is rewritten to f_eq(1, u_b).  EQ_OUTFLOW faces take no part (their velocity is not
 * prescribed).  flux_before / flux_after: host pointers, may be NULL; the call synchronises.  Call after the inlet
 * profile / planes have been set; a later lbm_set_inlet_* or lbm_feed_inlet overwrites the corrected values. */
int lbm_balance_flux(lbm_t *h, double *flux_before, double *flux_after);

/* Damping zones: top sponge layer and boundary-adjacent buffer nudging towards the target boundary state (PAPER.md:175
 * "relaxation-based damping regions adjacent to the upper and lateral boundaries, including a top sponge layer and
 * boundary-adjacent buffer nudging toward the target boundary state"; Table 1 PAPER.md:86 "sponge and buffer damping").
 * The paper prints neither form nor coefficients (S7 missing); reading (DESIGN.md §4 reading 20): a Rayleigh relaxation
 * acceleration a_d(u) = sigma(x) (u_t(z) - u) joins the body force of FLUID cells and is integrated by the same implicit
 * half-force rule as the Coriolis term (unconditionally stable; per step a uniform defect shrinks by
 * (1 - sigma/2) / (1 + sigma/2)).  width[k] (cells, >= 0) and peak[k] (0 <= peak <= 1) for the faces x-,x+,y-,y+,z-,z+:
 * a cell d = 0, 1, ... cells away from the layer adjacent to face k sees  peak[k] sin^2((pi/2)(1 - d/width[k]))  while
 * d < width[k];  sigma(x) = the largest of the six.  target: HOST array [3][nz] = u_t, v_t, w_t per level (e.g. the
 * inlet profile), copied.  All width or peak zero: damping off (target may be NULL).  The zones cost no HBM traffic
 * (coefficients come from three small per-axis tables); lbm_get_macros / lbm_get_mean stay exact inside them.
 * Returns LBM_EINVAL for a negative width, a peak outside [0, 1] or a non-finite / device target.  Synchronises. */
int lbm_set_damping(lbm_t *h, const int width[6], const double peak[6], const double *target);

/* Synthetic inflow fluctuations ("On-the-fly synthetic turbulent fluctuations are superposed on this mean
 * field", the mean being "held fixed throughout the LBM-LES integration"; Table 1 PAPER.md:86 "synthetic von Karman
 * fluctuations on active inflow cells").  The formulation is in the paper's Supplementary S7 (missing); reading
 * (DESIGN.md §4 reading 21) = random Fourier modes with the von Karman-Pao spectrum:
 *     u'(x, t) = 2 sum_n uhat_n cos(kappa_n . x + psi_n - omega_n t) sigma_n,   uhat_n = sqrt(E(|kappa_n|) dkappa_n),
 *     E(k) = 1.453 (u_rms^2 / k_e) (k/k_e)^4 / [1 + (k/k_e)^2]^(17/6) exp(-2 (k/k_eta)^2)      (k_eta = 0: no cut-off),
 * x = cell indices, t = step number, all in lattice units.  The random draws are the caller's: modes = HOST array
 * [n_modes][9] = kappa[3], sigma[3] (unit, normal to kappa), psi, omega, dkappa  (omega = kappa . U_c gives a frozen
 * pattern carried with U_c).  Active inflow cells = EQ_FIXED cells whose mean velocity points into the domain
 * (u_b . n < -1e-7 lattice units — inward by more than rounding noise —, n = outward normal of the owner face); after k steps such a cell holds f_eq(1, u_b + u'(x, k)); every
 * other EQ_FIXED cell keeps the mean.  The mean is the boundary state in force when the call is made: while
 * fluctuations are on, lbm_set_inlet_profile / _plane, lbm_feed_inlet and lbm_balance_flux return LBM_ESTATE.
 * n_modes = 0 switches them off and restores the mean (modes may be NULL).  lbm_set_flags switches them off too.
 * Cost per step: no extra launch — the face slots ride in extra leading block rows of the step launch itself (n_modes
 * cosines per active cell), no lattice traffic.
 * LBM_EINVAL: n_modes < 0 or > LBM_MAX_INFLOW_MODES, k_e <= 0, u_rms < 0, k_eta < 0, dkappa < 0, non-finite or device
 * table.  Needs flags (else LBM_ESTATE).  Synchronises. */
#define LBM_MAX_INFLOW_MODES 1024
int lbm_set_inflow_turbulence(lbm_t *h, int n_modes, const double *modes, double u_rms, double k_e, double k_eta);

/* Thermal lattice with Boussinesq coupling (Table 1 "Optional D3Q7 or D3Q19 thermal
 * lattice with Boussinesq coupling", density-current workload PAPER.md:121; DESIGN.md §4 reading 23).  A D3Q7 BGK
 * advection-diffusion lattice (rest vector + six axis vectors, weights 1/4 and 1/8, c_sT^2 = 1/4, linear equilibrium
 * h_eq,i = wT_i theta (1 + 4 c_i.u), tau_theta = 4 alpha + 1/2) stepped in the same kernel as the flow: each FLUID
 * cell pulls its 7 thermal populations by the rule of the flow pull (bounce-back on walls / solids and specular
 * reflection on FREE_SLIP faces = zero heat flux; periodic wrap), theta = sum_i h_i, the flow collision sees the
 * acceleration F + g_beta (theta - theta_ref) e_z (+z = up), and the thermal populations relax towards h_eq(theta, u)
 * with the velocity of that collision.  lbm_get_macros then reports the velocity corrected by the same buoyancy.
 * lbm_set_thermal switches it on with theta = theta_ref at rest; it allocates 2 x 7 population arrays of the handle's
 * precision (library-owned, freed by lbm_destroy).  Open faces (DESIGN.md §4 reading 27): an EQ_FIXED cell holds
 * h_eq(theta_b, u_b) beside f_eq(1, u_b), with theta_b = theta_ref until lbm_set_inlet_theta prescribes it; an EQ_OUTFLOW
 * cell holds the equilibria of the theta and u its inward neighbour had at the previous step (zero gradient).  Damping zones
 * (lbm_set_damping) combine with it: the relaxation acceleration and the buoyancy enter the same implicit half-force solve.
 * So do the synthetic inflow fluctuations (lbm_set_inflow_turbulence): an active inflow cell holds h_eq(theta_b, u_b + u') beside
 * f_eq(1, u_b + u'), one boundary velocity for both lattices (DESIGN.md §4 reading 28); theta_b itself does not fluctuate.
 * 16-bit storage must be off (LBM_EINVAL); with LBM_STREAM_INPLACE the flow lattice streams in place and the thermal one stays double-buffered.  alpha > 0 (lattice units); LBM_ENOMEM / LBM_ECUDA if the allocation fails.  Synchronises. */
int lbm_set_thermal(lbm_t *h, double alpha, double g_beta, double theta_ref);
/* Prescribed temperature of the EQ_FIXED cells by level (reading 27): theta_b[nz], host or device; the cells' thermal state
 * becomes h_eq(theta_b(z), u_b) at once and is re-expanded from it every step.  A later lbm_set_inlet_profile / _plane,
 * lbm_feed_inlet or lbm_balance_flux keeps theta_b and refreshes the cells for the new u_b.  Needs lbm_set_thermal and flags
 * (else LBM_ESTATE); a new lbm_set_flags* resets theta_b to theta_ref. */
int lbm_set_inlet_theta(lbm_t *h, const float *theta_b);
int lbm_set_inlet_theta_f64(lbm_t *h, const double *theta_b);
/* Initial thermal state H0 = h_eq(theta, u): theta, ux, uy, uz each [nz][ny][nx], host or device; NULL theta =
 * theta_ref, NULL component = 0; SOLID cells are skipped, EQ_FIXED cells keep their boundary state.  Call it AFTER
 * lbm_set_macros (what the cells next to an outflow face hand to it is derived from both states).  Needs lbm_set_thermal
 * and flags (else LBM_ESTATE); a new lbm_set_flags* leaves the thermal state stale until this is called again. */
int lbm_set_theta(lbm_t *h, const float *theta, const float *ux, const float *uy, const float *uz);
int lbm_set_theta_f64(lbm_t *h, const double *theta, const double *ux, const double *uy, const double *uz);
/* theta = sum_i h_i of the current state, [nz][ny][nx], host or device; SOLID cells report theta_ref.  Synchronises. */
int lbm_get_theta(lbm_t *h, float *theta);
int lbm_get_theta_f64(lbm_t *h, double *theta);
/* Fixed-temperature walls (DESIGN.md §4 reading 26): on[k] != 0 holds domain face k (order x-,x+,y-,y+,z-,z+), which must be
 * a WALL face (else LBM_EINVAL), at temperature theta_w[k] by halfway anti-bounce-back — a thermal population leaving
 * towards it returns as -h_i + 2 wT_i theta_w, theta = theta_w half a cell outside the last node; all other walls and the
 * buildings stay adiabatic.  Host arrays.  The change applies to the populations stored from the next step on (the
 * mailboxes written by the last step / by lbm_set_theta keep the rule in force when they were written: call it before
 * lbm_set_theta for an exact start).  Needs lbm_set_thermal (else LBM_ESTATE).  With it the thermal lattice covers heated
 * / cooled ground and lids — e.g. Rayleigh-Benard convection, the closed-form pin of the coupled loop. */
int lbm_set_thermal_walls(lbm_t *h, const int on[6], const double theta_w[6]);
/* Checkpoint of the thermal lattice: the 7 thermal populations h_i (NOT shifted), double, [7][nz][ny][nx], directions
 * 0..6 of the flow lattice; host or device.  Together with lbm_get_state / lbm_set_state and lbm_set_step a thermal run
 * restarts exactly.  Non-FLUID cells export the rest state wT_i theta_ref and ignore their input.  Needs
 * lbm_set_thermal and flags (else LBM_ESTATE). */
int lbm_get_thermal_state(lbm_t *h, double *hpop);
int lbm_set_thermal_state(lbm_t *h, const double *hpop);

/* Config-5 coupling, device to device, stream-ordered on dst's stream: local macros of src on the plane
 * x = src_x_plane are written as f_eq(1, u) into the EQ_FIXED cells of dst's x- face, tiling y modulo
 * src's ny; nz must match; SOLID src cells feed u = 0.  Both handles must share precision. */
int lbm_feed_inlet(lbm_t *dst, const lbm_t *src, int src_x_plane);

/* Initial state G0 = f_eq(rho, u) (DESIGN.md §3 step 3).  NULL rho = 1; NULL component = 0.  SOLID cells get
 * rho = 1, u = 0; EQ_FIXED cells keep their boundary state.  Resets the step counter; the mean sums and their sample count
 * are left alone (lbm_mean_reset clears them; a new lbm_set_flags* does too).  Needs flags. */
int lbm_set_macros(lbm_t *h, const float *rho, const float *ux, const float *uy, const float *uz);
int lbm_set_macros_f64(lbm_t *h, const double *rho, const double *ux, const double *uy, const double *uz);

/* n fused stream-collide steps (DESIGN.md §3 steps 4 and 6): pull with bounce-back / specular / periodic
 * resolution, moments, Coriolis + F with the implicit half-force velocity, Smagorinsky tau from the local
 * non-equilibrium stress, BGK + Guo source, store; outflow cells refreshed; on sampling steps the time-mean
 * sums are updated in the same kernel.  Asynchronous.  Needs flags (else LBM_ESTATE). */
int lbm_step(lbm_t *h, int n);

/* Time mean (DESIGN.md §3 step 8): after step k (k counted from the last set_macros/set_flags), if
 * every > 0, k >= start_step and (k - start_step) % every == 0, u is added to the sums. */
int lbm_mean_config(lbm_t *h, long start_step, int every);
int lbm_mean_reset(lbm_t *h);

/* Local macroscopic fields of the current state (DESIGN.md §3 step 7); any pointer may be NULL. */
int lbm_get_macros(lbm_t *h, float *rho, float *ux, float *uy, float *uz);
int lbm_get_macros_f64(lbm_t *h, double *rho, double *ux, double *uy, double *uz);

/* The same fields for the box lo[a] <= c_a < hi[a] only (axes x, y, z; 0 <= lo < hi <= n, else LBM_EINVAL): outputs are the
 * box's own C-order arrays [hi[2]-lo[2]][hi[1]-lo[1]][hi[0]-lo[0]], host or device, any may be NULL.  What the paper's
 * application reads back is of this kind — a horizontal plane at pedestrian height ("wind speeds ... at a pedestrian
 * height of 2 m"), a vertical profile above a station (PAPER.md:137-148 lidar comparison) — and on a 1.2e9-cell lattice the four
 * whole fields would be 19 GB. */
int lbm_get_macros_box(lbm_t *h, const int lo[3], const int hi[3], float *rho, float *ux, float *uy, float *uz);
int lbm_get_macros_box_f64(lbm_t *h, const int lo[3], const int hi[3], double *rho, double *ux, double *uy, double *uz);

/* mean = sum / n_samples (0 where n_samples == 0 and in SOLID cells); n_samples is a host pointer, may be NULL */
int lbm_get_mean(lbm_t *h, float *ux, float *uy, float *uz, long *n_samples);
int lbm_get_mean_f64(lbm_t *h, double *ux, double *uy, double *uz, long *n_samples);
/* the time mean of a box (as lbm_get_macros_box) */
int lbm_get_mean_box(lbm_t *h, const int lo[3], const int hi[3], float *ux, float *uy, float *uz, long *n_samples);

/* Parity exports.  flags: uint8 [nz][ny][nx] cell classes.  links: uint32 [nz][ny][nx], bit i (1..18) set
 * iff pulling direction i into that FLUID cell takes the bounce-back branch; 0 for non-FLUID cells. */
int lbm_get_flags(lbm_t *h, uint8_t *flags);
int lbm_get_links(lbm_t *h, uint32_t *links);

/* Checkpoint: populations f_i (NOT shifted), double, [19][nz][ny][nx], direction order of DESIGN.md §3
 * step 1.  set_state leaves the step counter, the mean sums and the thermal state alone (lbm_set_step, lbm_mean_reset,
 * lbm_set_thermal_state).  The boundary velocity of an EQ_FIXED cell becomes the velocity moment of the populations
 * given for it (the cell is re-expanded from that velocity every step); prescribe the profile / plane again afterwards
 * to impose an exact u_b.  SOLID cells export the rest state and ignore their input. */
int lbm_get_state(lbm_t *h, double *f);
int lbm_set_state(lbm_t *h, const double *f);

/* The same checkpoint for the box lo[a] <= c_a < hi[a] (axes x, y, z; 0 <= lo < hi <= n, else LBM_EINVAL):
 * f [19][hi[2]-lo[2]][hi[1]-lo[1]][hi[0]-lo[0]] doubles, host or device.  For lattices whose whole state (152 B per cell in
 * this format) does not fit beside the lattice itself — 2.9e8 cells and more, or anything on LBM_STREAM_INPLACE scale — a run is
 * checkpointed and restored slab by slab, and a sampled sub-box can be handed to a reference solver.  lbm_set_state_box writes the
 * cells of the box into the CURRENT state (wall-link and ghost copies of their populations included) and leaves every other cell,
 * the step counter and the mean sums alone; boxes that together cover the lattice restore exactly what lbm_set_state restores. */
int lbm_get_state_box(lbm_t *h, const int lo[3], const int hi[3], double *f);
int lbm_set_state_box(lbm_t *h, const int lo[3], const int hi[3], const double *f);

long lbm_get_step(const lbm_t *h);
int lbm_set_step(lbm_t *h, long step);
int lbm_sync(lbm_t *h);
const char *lbm_last_error(const lbm_t *h);

/* Kernel launches issued by this handle since creation (bench.py's gpu_launches). */
long lbm_launch_count(const lbm_t *h);

/* The lattice as the library defines it: c[19][3], opposite[19] (host arrays).  For tests. */
int lbm_lattice(int *c, int *opposite);

/* Launch shape of the FP32 stream-collide step, for A/B measurements.  Every variant computes the same arithmetic on
 * the same stored state (tests/test_gpu_parity.py runs each against the oracle):
 *   0  default: 4 x-cells per thread with 128-bit loads / stores where nx % 4 == 0, else one cell per thread; lattices
 *      whose whole grid is resident at once run several steps per cooperative launch;
 *   1  one cell per thread, 32-bit accesses, one launch per step;
 *   2  2 x-cells per thread, 64-bit accesses (32-bit with 16-bit storage; nx % 2 == 0, else as 1), one launch per step;
 *   3  4 x-cells per thread, 128-bit accesses (64-bit with 16-bit storage; nx % 4 == 0, else as 1), one launch per step.
 * Lattices with PERIODIC x faces always run one cell per thread (the read-side wrap lives there).
 * FP64 handles, damping zones, inflow fluctuations and the thermal lattice have one launch shape each and ignore it.
 * Returns LBM_EINVAL for an unknown variant. */
int lbm_set_variant(lbm_t *h, int variant);

#ifdef __cplusplus
}
#endif
#endif /* LBM_B200_H */
