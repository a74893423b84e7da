/*
 * lbm_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of the D3Q19 LBM-LES step that
 * the CUDA library in paper_2607_04516_b200/ must reproduce.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.  It shares no code, header, table or helper with the CUDA path.
 *
 * What it follows.  The paper (§2.2; Table 1) names
 * the ingredients — weakly compressible D3Q19, single-relaxation-time BGK,
 * Smagorinsky-Lilly with the effective relaxation time "computed locally from
 * nonequilibrium moments", Coriolis through Guo forcing, equilibrium-based
 * velocity boundaries, no-slip solids — but prints no equation (all deferred to
 * supplementary S4-S7, not available).  Each function
 * therefore writes out the textbook definition of the named method, in the
 * reading fixed by DESIGN.md "Readings" (= SURVEY.md §8(c)); the step numbers
 * in comments (1..9) are the steps of that algorithm statement.
 *
 * Structure is deliberately naive: array-of-structures G[cell][19], one
 * explicit resolve() per pulled population, no link masks, no blocking, no
 * fusion beyond "one pass = one time step".  OpenMP on the outer z loop only.
 *
 * Pins: tests/test_oracle_*.py (closed forms, invariants, brute force) — see
 * DESIGN.md "Oracle pins".  Parity unpinned: the urban LES statistics of
 * configs 3-5 (no closed form exists; SURVEY.md §8(c) last row).
 * The optional thermal lattice + Boussinesq coupling (heq(),
 * oracle_set_thermal / _set_theta / _get_theta and the thermal branch of
 * oracle_step; reading 23) is pinned by tests/test_oracle_thermal.py:
 * closed forms and the density-current front positions the paper prints
 * (tests/golden/density_current_fronts.txt).
 * The optional 16-bit population storage (round_to_half, to_storage, oracle_set_storage16) is pinned by
 * tests/test_oracle_storage16.py: numpy's float16 cast on a value sweep, the state lying on the half grid after every
 * kind of write, and closed-form error budgets (Taylor-Green decay, Poiseuille, mass drift).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* cell classes (step 3) */
enum { C_FLUID = 0, C_SOLID = 1, C_EQ_FIXED = 2, C_EQ_OUTFLOW = 3 };
/* face types */
enum { F_PERIODIC = 0, F_WALL = 1, F_FREE_SLIP = 2, F_EQ_FIXED = 3, F_EQ_OUTFLOW = 4 };

#define Q 19

/* step 1: lattice.  0 = rest; then opposite pairs adjacent, odd index = the
 * sign listed first: 1,2=(+-1,0,0) 3,4=(0,+-1,0) 5,6=(0,0,+-1) 7,8=+-(1,1,0)
 * 9,10=+-(1,0,1) 11,12=+-(0,1,1) 13,14=+-(1,-1,0) 15,16=+-(1,0,-1)
 * 17,18=+-(0,1,-1). */
static const int CI[Q][3] = {
    {0, 0, 0},
    {1, 0, 0},  {-1, 0, 0},
    {0, 1, 0},  {0, -1, 0},
    {0, 0, 1},  {0, 0, -1},
    {1, 1, 0},  {-1, -1, 0},
    {1, 0, 1},  {-1, 0, -1},
    {0, 1, 1},  {0, -1, -1},
    {1, -1, 0}, {-1, 1, 0},
    {1, 0, -1}, {-1, 0, 1},
    {0, 1, -1}, {0, -1, 1},
};

static double weight(int i) { return i == 0 ? 1.0 / 3.0 : (i <= 6 ? 1.0 / 18.0 : 1.0 / 36.0); }

/* Thermal lattice D3Q7: the rest vector and the six axis vectors = directions 0..6 of CI;
 * weights 1/4 and 1/8, lattice sound speed squared 1/4 (sum_i wT_i c_ia c_ib = delta_ab / 4). */
#define QT 7
static double weight_t(int i) { return i == 0 ? 0.25 : 0.125; }
/* linear advection-diffusion equilibrium h_eq,i = wT_i theta (1 + c_i.u / c_sT^2) = wT_i theta (1 + 4 c_i.u) */
static void heq(double theta, const double u[3], double out[QT])
{
    for (int i = 0; i < QT; ++i) {
        double cu = CI[i][0] * u[0] + CI[i][1] * u[1] + CI[i][2] * u[2];
        out[i] = weight_t(i) * theta * (1.0 + 4.0 * cu);
    }
}

static int dir_index(int cx, int cy, int cz)
{
    for (int i = 0; i < Q; ++i)
        if (CI[i][0] == cx && CI[i][1] == cy && CI[i][2] == cz) return i;
    return -1;
}

static int opposite_search(int i) { return dir_index(-CI[i][0], -CI[i][1], -CI[i][2]); }

/* the two searches above, tabulated once (filled from them, nothing else) */
static int OPP[Q];
static int DIR[3][3][3]; /* [cx+1][cy+1][cz+1] -> i, or -1 */
static int tables_ready = 0;
static void init_tables(void)
{
    if (tables_ready) return;
    for (int i = 0; i < Q; ++i) OPP[i] = opposite_search(i);
    for (int a = -1; a <= 1; ++a)
        for (int b = -1; b <= 1; ++b)
            for (int c = -1; c <= 1; ++c) DIR[a + 1][b + 1][c + 1] = dir_index(a, b, c);
    tables_ready = 1;
}
static int opposite(int i) { return OPP[i]; }

typedef struct oracle {
    int nx, ny, nz;
    double nu0, Cs, fv[3], F[3]; /* fv = Coriolis vector f = 2 Omega (lattice units); scalar f_cor = fv[2] */
    int face[6]; /* x-,x+,y-,y+,z-,z+ */
    int have_flags;
    uint8_t *cls; /* [z][y][x] */
    double *G;    /* [cell][19], post-collision state G_k (step 3) */
    double *Gn;   /* next */
    double *ub;   /* [cell][3] prescribed velocity of EQ_FIXED cells */
    double *sig;  /* [cell] damping coefficient sigma(x) of the sponge / buffer zones (NULL = none) */
    double *ut;   /* [3][nz] target state u_t(z) the damping relaxes towards */
    int nmodes;   /* synthetic inflow turbulence: number of Fourier modes (0 = off) */
    double *modes; /* [nmodes][9] = kappa[3], sigma[3], psi, omega, dkappa */
    double *uhat; /* [nmodes] mode amplitudes sqrt(E(|kappa|) dkappa) */
    long step;
    double *msum; /* [cell][3] */
    long mcount, mstart;
    int mevery;
    /* thermal lattice (Table 1 "Optional D3Q7 ... thermal lattice with Boussinesq coupling"; DESIGN.md §4
     * reading 23): off unless oracle_set_thermal was called */
    int thermal;
    double alpha, gbeta, theta_ref; /* diffusivity, g*beta (buoyancy per unit theta, along +z), reference theta */
    double *H, *Hn;                 /* [cell][7] post-collision thermal populations, directions 0..6 of CI */
    double *thb;                    /* [cell] prescribed temperature of EQ_FIXED cells (reading 27); theta_ref unless set */
    int thd[6];                     /* WALL faces held at a fixed temperature (Dirichlet; reading 26): 1 = on */
    double thw[6];                  /* ... their temperatures theta_w */
    /* 16-bit population storage: 0 = populations kept in FP64 (default),
     * 1 = every population is rounded to IEEE binary16 at the moment it is written into the state */
    int store16;
} oracle_t;

static long cell_of(const oracle_t *o, int x, int y, int z)
{
    return ((long)z * o->ny + y) * o->nx + x;
}

/* ---- 16-bit population storage (SURVEY.md §8(f) row 5 "16-bit DDF storage") --------------------------
 * The paper does not say how its populations are stored (PAPER.md:181-185 silent; SURVEY.md §6 infers from the printed
 * wall-clock that they were not plain FP32).  Reading: arithmetic is unchanged; what is STORED for
 * population i is the shifted value G_i - w_i rounded to IEEE 754 binary16 (1 sign, 5 exponent, 10 fraction bits;
 * subnormals kept; round to nearest, ties to even), at the moment it is written.  The rest state is stored exactly (0).
 * round_to_half writes the definition out: spacing 2^(E-10) for 2^E <= |x| < 2^(E+1), E clamped at -14 (below that the
 * spacing stays 2^-24), overflow to infinity from 65520 on. */
static double round_to_half(double x)
{
    if (x == 0.0 || x != x) return x;
    double a = fabs(x);
    if (a >= 65520.0) return x > 0 ? INFINITY : -INFINITY; /* halfway between the largest half (65504) and 2^16 */
    int e;
    frexp(a, &e);                 /* a = m 2^e with 1/2 <= m < 1: leading bit has exponent e - 1 */
    int E = e - 1;
    if (E < -14) E = -14;         /* subnormal range */
    double ulp = ldexp(1.0, E - 10);
    double q = nearbyint(a / ulp); /* a / ulp is exact (power of two); default rounding mode = ties to even */
    return x > 0 ? q * ulp : -(q * ulp);
}
int oracle_round_half(int n, const double *in, double *out)
{
    for (int i = 0; i < n; ++i) out[i] = round_to_half(in[i]);
    return 0;
}
/* what the state keeps of a freshly computed set of populations g[19] (in place) */
static void to_storage(const oracle_t *o, double *g)
{
    if (!o->store16) return;
    for (int i = 0; i < Q; ++i) g[i] = weight(i) + round_to_half(g[i] - weight(i));
}

/* step 2: second-order equilibrium */
static void feq(double rho, const double u[3], double out[Q])
{
    double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    for (int i = 0; i < Q; ++i) {
        double cu = CI[i][0] * u[0] + CI[i][1] * u[1] + CI[i][2] * u[2];
        out[i] = weight(i) * rho * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * uu);
    }
}

/* step 4b-4e on one cell: pulled populations f[] -> post-collision g[].
 * Also returns the (rho,u,tau) the collision used. */
/* Solve the 3x3 system M x = r by Cramer's rule (M is I +- C/2 with C skew: always regular). */
static void solve3(const double M[3][3], const double r[3], double x[3])
{
    double det = M[0][0] * (M[1][1] * M[2][2] - M[1][2] * M[2][1])
               - M[0][1] * (M[1][0] * M[2][2] - M[1][2] * M[2][0])
               + M[0][2] * (M[1][0] * M[2][1] - M[1][1] * M[2][0]);
    for (int k = 0; k < 3; ++k) {
        double N[3][3];
        for (int a = 0; a < 3; ++a)
            for (int c = 0; c < 3; ++c) N[a][c] = (c == k) ? r[a] : M[a][c];
        double dk = N[0][0] * (N[1][1] * N[2][2] - N[1][2] * N[2][1])
                  - N[0][1] * (N[1][0] * N[2][2] - N[1][2] * N[2][0])
                  + N[0][2] * (N[1][0] * N[2][1] - N[1][1] * N[2][0]);
        x[k] = dk / det;
    }
}

/* Coriolis acceleration of the full rotation vector (Table 1: "full rotation vector in the
 * local ENU frame"): a_cor(u) = -2 Omega x u = -fv x u = C u with fv = 2 Omega and
 *     C = [[0, fz, -fy], [-fz, 0, fx], [fy, -fx, 0]].
 * fv = (0, 0, f) gives the scalar reading a_cor = f (u_y, -u_x, 0) of DESIGN.md §4 reading 5. */
static void coriolis_matrix(const double fv[3], double Cm[3][3])
{
    Cm[0][0] = 0.0;    Cm[0][1] = fv[2];  Cm[0][2] = -fv[1];
    Cm[1][0] = -fv[2]; Cm[1][1] = 0.0;    Cm[1][2] = fv[0];
    Cm[2][0] = fv[1];  Cm[2][1] = -fv[0]; Cm[2][2] = 0.0;
}

/* Damping zones ("relaxation-based damping regions adjacent to the upper and lateral boundaries,
 * including a top sponge layer and boundary-adjacent buffer nudging toward the target boundary state"; Table 1
 * PAPER.md:86 "sponge and buffer damping").  Reading (DESIGN.md §4 reading 20): a Rayleigh relaxation acceleration
 * a_d(u) = sigma(x) (u_t - u) towards the target state u_t, added to the body force and integrated by the same
 * implicit half-force rule as the Coriolis term.  sigma = 0 is the undamped step. */
static void collide(const double f[Q], double nu0, double Cs, const double fv[3], const double F[3],
                    double sigma, const double ut[3],
                    double g[Q], double *rho_out, double u_out[3], double *tau_out)
{
    /* 4b moments */
    double rho = 0.0, m[3] = {0, 0, 0};
    for (int i = 0; i < Q; ++i) {
        rho += f[i];
        for (int a = 0; a < 3; ++a) m[a] += CI[i][a] * f[i];
    }
    /* 4c implicit half-force velocity: rho u = m + rho a(u)/2, a(u) = F + C u + sigma (u_t - u)
     * => ((1 + sigma/2) I - C/2) u = m/rho + F/2 + (sigma/2) u_t */
    double Cm[3][3], M[3][3];
    coriolis_matrix(fv, Cm);
    for (int a = 0; a < 3; ++a)
        for (int c = 0; c < 3; ++c) M[a][c] = (a == c ? 1.0 + 0.5 * sigma : 0.0) - 0.5 * Cm[a][c];
    double b[3];
    for (int a = 0; a < 3; ++a) b[a] = m[a] / rho + 0.5 * F[a] + 0.5 * sigma * (ut ? ut[a] : 0.0);
    double u[3];
    solve3(M, b, u);
    double Fd[3]; /* force density rho a(u) */
    for (int a = 0; a < 3; ++a)
        Fd[a] = rho * (F[a] + Cm[a][0] * u[0] + Cm[a][1] * u[1] + Cm[a][2] * u[2] + sigma * ((ut ? ut[a] : 0.0) - u[a]));
    /* 4d LES: Pi = sum c c (f - feq); Q = Frobenius norm over all 9 entries */
    double fe[Q];
    feq(rho, u, fe);
    double Pi[3][3] = {{0}};
    for (int i = 0; i < Q; ++i)
        for (int a = 0; a < 3; ++a)
            for (int c = 0; c < 3; ++c) Pi[a][c] += CI[i][a] * CI[i][c] * (f[i] - fe[i]);
    double QQ = 0.0;
    for (int a = 0; a < 3; ++a)
        for (int c = 0; c < 3; ++c) QQ += Pi[a][c] * Pi[a][c];
    QQ = sqrt(QQ);
    double tau0 = 3.0 * nu0 + 0.5;
    double tau = 0.5 * (tau0 + sqrt(tau0 * tau0 + 18.0 * sqrt(2.0) * Cs * Cs * QQ / rho));
    /* 4e BGK + Guo source */
    for (int i = 0; i < Q; ++i) {
        double cu = CI[i][0] * u[0] + CI[i][1] * u[1] + CI[i][2] * u[2];
        double cF = CI[i][0] * Fd[0] + CI[i][1] * Fd[1] + CI[i][2] * Fd[2];
        double cmuF = (CI[i][0] - u[0]) * Fd[0] + (CI[i][1] - u[1]) * Fd[1] + (CI[i][2] - u[2]) * Fd[2];
        double S = (1.0 - 1.0 / (2.0 * tau)) * weight(i) * (3.0 * cmuF + 9.0 * cu * cF);
        g[i] = f[i] - (f[i] - fe[i]) / tau + S;
    }
    if (rho_out) *rho_out = rho;
    if (u_out) { u_out[0] = u[0]; u_out[1] = u[1]; u_out[2] = u[2]; }
    if (tau_out) *tau_out = tau;
}

/* step 4a: where does population i of FLUID cell (x,y,z) come from?
 * returns 1 = bounce-back branch (take G(x, opposite(i))), 0 = take G(*s, *j),
 * -1 = an EQ face was crossed (cannot happen for a FLUID cell; reported). */
static int resolve(const oracle_t *o, int x, int y, int z, int i, long *s, int *j)
{
    int p[3] = {x - CI[i][0], y - CI[i][1], z - CI[i][2]};
    int c[3] = {CI[i][0], CI[i][1], CI[i][2]};
    int n[3] = {o->nx, o->ny, o->nz};
    int wall = 0;
    static const int order[3] = {2, 1, 0}; /* z, then y, then x */
    for (int k = 0; k < 3; ++k) {
        int a = order[k];
        int ft;
        if (p[a] < 0) ft = o->face[2 * a];
        else if (p[a] >= n[a]) ft = o->face[2 * a + 1];
        else continue;
        if (ft == F_PERIODIC) p[a] = (p[a] + n[a]) % n[a];
        else if (ft == F_FREE_SLIP) { p[a] = p[a] < 0 ? 0 : n[a] - 1; c[a] = -c[a]; }
        else if (ft == F_WALL) wall = 1;
        else return -1;
    }
    if (wall) return 1;
    *s = cell_of(o, p[0], p[1], p[2]);
    if (o->cls[*s] == C_SOLID) return 1;
    *j = DIR[c[0] + 1][c[1] + 1][c[2] + 1];
    return 0;
}

/* step 7: local macros of the stored state at one cell */
static void local_macros(const oracle_t *o, const double *Gs, long cell, double *rho, double u[3])
{
    int cl = o->cls ? o->cls[cell] : C_FLUID;
    if (cl == C_SOLID) { *rho = 1.0; u[0] = u[1] = u[2] = 0.0; return; }
    const double *g = Gs + cell * Q;
    double r = 0.0, m[3] = {0, 0, 0};
    for (int i = 0; i < Q; ++i) {
        r += g[i];
        for (int a = 0; a < 3; ++a) m[a] += CI[i][a] * g[i];
    }
    *rho = r;
    if (cl == C_FLUID) {
        /* invert m* = rho u + rho a(u)/2, a(u) = F + C u + sigma (u_t - u)
         * =>  ((1 - sigma/2) I + C/2) u = m* / rho - F/2 - (sigma/2) u_t   (regular for sigma < 2) */
        double Cm[3][3], M[3][3];
        coriolis_matrix(o->fv, Cm);
        double sg = o->sig ? o->sig[cell] : 0.0;
        long zc = cell / ((long)o->nx * o->ny);
        for (int a = 0; a < 3; ++a)
            for (int c = 0; c < 3; ++c) M[a][c] = (a == c ? 1.0 - 0.5 * sg : 0.0) + 0.5 * Cm[a][c];
        double Fl[3] = {o->F[0], o->F[1], o->F[2]};
        if (o->thermal && Gs == o->G) {
            /* Boussinesq: the buoyancy the cell's collision used is g beta (theta - theta_ref) with theta = sum_i h_i,
             * which the thermal collision conserves: read it back from the stored thermal state */
            double th = 0.0;
            for (int i = 0; i < QT; ++i) th += o->H[cell * QT + i];
            Fl[2] += o->gbeta * (th - o->theta_ref);
        }
        double b[3];
        for (int a = 0; a < 3; ++a) b[a] = m[a] / r - 0.5 * Fl[a] - 0.5 * sg * (o->ut ? o->ut[a * o->nz + zc] : 0.0);
        solve3(M, b, u);
    } else {
        u[0] = m[0] / r; u[1] = m[1] / r; u[2] = m[2] / r;
    }
}

/* ------------------------------------------------------------------ C API */

int oracle_lattice(int *c /*[19][3]*/, double *w /*[19]*/, int *opp /*[19]*/)
{
    init_tables();
    for (int i = 0; i < Q; ++i) {
        for (int a = 0; a < 3; ++a) c[3 * i + a] = CI[i][a];
        w[i] = weight(i);
        opp[i] = opposite(i);
    }
    return 0;
}

int oracle_feq(double rho, const double *u, double *out) { feq(rho, u, out); return 0; }

int oracle_collide_cell(const double *f, double nu0, double Cs, double fcor, const double *F,
                        double *g, double *rho, double *u, double *tau)
{
    const double fv[3] = {0.0, 0.0, fcor};
    collide(f, nu0, Cs, fv, F, 0.0, NULL, g, rho, u, tau);
    return 0;
}

/* same with the full Coriolis vector fv = 2 Omega */
int oracle_collide_cell_vec(const double *f, double nu0, double Cs, const double *fv, const double *F,
                            double *g, double *rho, double *u, double *tau)
{
    collide(f, nu0, Cs, fv, F, 0.0, NULL, g, rho, u, tau);
    return 0;
}

/* same inside a damping zone: coefficient sigma, target velocity ut[3] */
int oracle_collide_cell_damped(const double *f, double nu0, double Cs, const double *fv, const double *F,
                               double sigma, const double *ut, double *g, double *rho, double *u, double *tau)
{
    collide(f, nu0, Cs, fv, F, sigma, ut, g, rho, u, tau);
    return 0;
}

oracle_t *oracle_create(int nx, int ny, int nz, double nu0, double Cs, double fcor, const double *F)
{
    if (nx < 1 || ny < 1 || nz < 1) return NULL;
    init_tables();
    oracle_t *o = (oracle_t *)calloc(1, sizeof(oracle_t));
    if (!o) return NULL;
    o->nx = nx; o->ny = ny; o->nz = nz;
    o->nu0 = nu0; o->Cs = Cs; o->fv[0] = 0.0; o->fv[1] = 0.0; o->fv[2] = fcor;
    for (int a = 0; a < 3; ++a) o->F[a] = F ? F[a] : 0.0;
    /* default faces = config 1 */
    o->face[0] = F_EQ_FIXED; o->face[1] = F_EQ_OUTFLOW;
    o->face[2] = F_PERIODIC; o->face[3] = F_PERIODIC;
    o->face[4] = F_WALL;     o->face[5] = F_FREE_SLIP;
    long N = (long)nx * ny * nz;
    o->cls = (uint8_t *)calloc(N, 1);
    o->G = (double *)malloc(sizeof(double) * N * Q);
    o->Gn = (double *)malloc(sizeof(double) * N * Q);
    o->ub = (double *)calloc(N * 3, sizeof(double));
    if (!o->cls || !o->G || !o->Gn || !o->ub) { free(o->cls); free(o->G); free(o->Gn); free(o->ub); free(o); return NULL; }
    o->mstart = 0; o->mevery = 0;
    return o;
}

void oracle_destroy(oracle_t *o)
{
    if (!o) return;
    free(o->cls); free(o->G); free(o->Gn); free(o->ub); free(o->msum); free(o->sig); free(o->ut); free(o->modes); free(o->uhat); free(o->H); free(o->Hn); free(o->thb); free(o);
}

/* Damping zones (see collide()).  width[k] (cells) and peak[k] for the six faces x-,x+,y-,y+,z-,z+; a cell at
 * distance d = 0, 1, ... (in cells) from the layer of cells adjacent to face k lies in that face's zone if d < width[k]
 * and sees the ramp  peak[k] * sin^2( (pi/2) (1 - d / width[k]) )  (peak at the face layer, smoothly to 0 at d = width);
 * sigma(x) = the LARGEST of the six (zones do not add up in edges and corners).  ut = [3][nz] target profile u_t(z).
 * All widths 0 switch the damping off.  0 <= peak[k] <= 1 (sigma < 2 keeps the macro inversion regular). */
int oracle_set_damping(oracle_t *o, const int *width, const double *peak, const double *ut)
{
    if (!o || !width || !peak) return -1;
    int any = 0;
    for (int k = 0; k < 6; ++k) {
        if (width[k] < 0 || peak[k] < 0.0 || peak[k] > 1.0) return -1;
        if (width[k] > 0 && peak[k] > 0.0) any = 1;
    }
    free(o->sig); free(o->ut); o->sig = NULL; o->ut = NULL;
    if (!any) return 0;
    if (!ut) return -1;
    long N = (long)o->nx * o->ny * o->nz;
    o->sig = (double *)calloc(N, sizeof(double));
    o->ut = (double *)malloc(sizeof(double) * 3 * o->nz);
    if (!o->sig || !o->ut) return -4;
    memcpy(o->ut, ut, sizeof(double) * 3 * o->nz);
    const double half_pi = 2.0 * atan(1.0);
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                int d[6] = {x, o->nx - 1 - x, y, o->ny - 1 - y, z, o->nz - 1 - z};
                double s = 0.0;
                for (int k = 0; k < 6; ++k) {
                    if (width[k] <= 0 || d[k] >= width[k]) continue;
                    double r = sin(half_pi * (1.0 - (double)d[k] / (double)width[k]));
                    double v = peak[k] * r * r;
                    if (v > s) s = v;
                }
                o->sig[cell_of(o, x, y, z)] = s;
            }
    return 0;
}

int oracle_get_damping(const oracle_t *o, double *sigma)
{
    long N = (long)o->nx * o->ny * o->nz;
    for (long c = 0; c < N; ++c) sigma[c] = o->sig ? o->sig[c] : 0.0;
    return 0;
}

/* Coriolis vector f = 2 Omega in lattice units; replaces the scalar given at creation */
int oracle_set_coriolis(oracle_t *o, const double *fv)
{
    if (!o || !fv) return -1;
    for (int a = 0; a < 3; ++a) o->fv[a] = fv[a];
    return 0;
}

int oracle_set_boundaries(oracle_t *o, const int *face_type)
{
    for (int a = 0; a < 3; ++a) {
        int lo = face_type[2 * a], hi = face_type[2 * a + 1];
        if (lo < 0 || lo > 4 || hi < 0 || hi > 4) return -1;
        if ((lo == F_PERIODIC) != (hi == F_PERIODIC)) return -1;
    }
    for (int k = 0; k < 6; ++k) o->face[k] = face_type[k];
    o->have_flags = 0;
    return 0;
}

/* step 9: SOLID <=> z < clamp(h,0,nz); non-solid cells of an EQ face take the
 * EQ class, EQ_FIXED winning over EQ_OUTFLOW where two EQ faces meet. */
static int set_flags_impl(oracle_t *o, const int32_t *height, const uint8_t *solid);
int oracle_set_flags(oracle_t *o, const int32_t *height) { return set_flags_impl(o, height, NULL); }

/* the same with a general solid mask merged in ("The final solid mask is assembled by the Boolean merging of
 * a fixed-thickness base layer, the terrain layer, and the building layer"): SOLID <=> z < clamp(h) OR solid[z][y][x] != 0 */
int oracle_set_flags_mask(oracle_t *o, const int32_t *height, const uint8_t *solid) { return set_flags_impl(o, height, solid); }

static int set_flags_impl(oracle_t *o, const int32_t *height, const uint8_t *solid)
{
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                int h = height ? height[(long)y * o->nx + x] : 0;
                if (h < 0) h = 0;
                if (h > o->nz) h = o->nz;
                if (solid && solid[cell_of(o, x, y, z)]) h = o->nz; /* merged in: this cell is solid whatever the column height */
                int cl = C_FLUID;
                if (z < h) cl = C_SOLID;
                else {
                    int on[6] = {x == 0, x == o->nx - 1, y == 0, y == o->ny - 1, z == 0, z == o->nz - 1};
                    int fixed = 0, outflow = 0;
                    for (int k = 0; k < 6; ++k) {
                        if (on[k] && o->face[k] == F_EQ_FIXED) fixed = 1;
                        if (on[k] && o->face[k] == F_EQ_OUTFLOW) outflow = 1;
                    }
                    if (fixed) cl = C_EQ_FIXED;
                    else if (outflow) cl = C_EQ_OUTFLOW;
                }
                o->cls[cell_of(o, x, y, z)] = (uint8_t)cl;
            }
    o->have_flags = 1;
    return 0;
}

int oracle_get_flags(const oracle_t *o, uint8_t *out)
{
    memcpy(out, o->cls, (size_t)o->nx * o->ny * o->nz);
    return 0;
}

/* step 9: link bit i of a FLUID cell = "step 4a took the bounce-back branch" */
int oracle_get_links(const oracle_t *o, uint32_t *out)
{
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                long cell = cell_of(o, x, y, z);
                uint32_t bits = 0;
                if (o->cls[cell] == C_FLUID)
                    for (int i = 1; i < Q; ++i) {
                        long s; int j;
                        int r = resolve(o, x, y, z, i, &s, &j);
                        if (r < 0) return -2;
                        if (r == 1) bits |= (1u << i);
                    }
                out[cell] = bits;
            }
    return 0;
}

/* ---- synthetic inflow turbulence ------------------------------------------------------------------------------
 * PAPER.md:160 "On-the-fly synthetic turbulent fluctuations are superposed on this mean field" (which is "held fixed
 * throughout the LBM-LES integration"); Table 1 PAPER.md:86 "synthetic von Karman fluctuations on active inflow
 * cells".  The formulation is in Supplementary S7 (missing); reading (DESIGN.md §4 reading 21) = the textbook random
 * Fourier mode synthesis (Kraichnan 1970; the form in Davidson's synthetic-inlet notes, the author PAPER.md:209 cites):
 *     u'(x, t) = 2 sum_n uhat_n cos(kappa_n . x + psi_n - omega_n t) sigma_n,      sigma_n . kappa_n = 0,
 *     uhat_n = sqrt(E(|kappa_n|) dkappa_n),
 * with the von Karman-Pao energy spectrum
 *     E(k) = alpha (u_rms^2 / k_e) (k/k_e)^4 / [1 + (k/k_e)^2]^(17/6) exp(-2 (k/k_eta)^2),   alpha = 1.453.
 * x = cell indices (lattice units), t = step number.  The random draws (kappa_n, sigma_n, psi_n, omega_n, dkappa_n)
 * are INPUTS.  An EQ_FIXED cell is an "active inflow cell" when its mean velocity points into the domain,
 * ub . n < -1e-7 with n the outward normal of its owner face (the threshold, lattice units, keeps a normal component
 * that is zero up to rounding — e.g. a top face with w = 0 after the flux correction of a balanced profile — from
 * being "inflow" or not by the sign of its noise; DESIGN.md §4 reading 21); only those carry u'.  After k steps such a cell holds
 * f_eq(1, ub + u'(x, k)). */
static double vk_spectrum(double k, double u_rms, double k_e, double k_eta)
{
    const double alpha = 1.453;
    double r = k / k_e;
    double E = alpha * (u_rms * u_rms / k_e) * pow(r, 4.0) / pow(1.0 + r * r, 17.0 / 6.0);
    if (k_eta > 0.0) E *= exp(-2.0 * (k / k_eta) * (k / k_eta));
    return E;
}
int oracle_vk_spectrum(int n, const double *k, double u_rms, double k_e, double k_eta, double *E)
{
    for (int i = 0; i < n; ++i) E[i] = vk_spectrum(k[i], u_rms, k_e, k_eta);
    return 0;
}

static int fixed_face(const oracle_t *o, int x, int y, int z);

/* u'(x, t) of the stored modes */
static void fluctuation(const oracle_t *o, int x, int y, int z, double t, double up[3])
{
    up[0] = up[1] = up[2] = 0.0;
    for (int n = 0; n < o->nmodes; ++n) {
        const double *m = o->modes + 9 * n;
        double phase = m[0] * x + m[1] * y + m[2] * z + m[6] - m[7] * t;
        double c = 2.0 * o->uhat[n] * cos(phase);
        for (int a = 0; a < 3; ++a) up[a] += c * m[3 + a];
    }
}

/* boundary velocity of EQ_FIXED cell (x,y,z) at time t: mean + fluctuation on active inflow cells */
static void boundary_velocity(const oracle_t *o, int x, int y, int z, double t, double u[3])
{
    long cell = cell_of(o, x, y, z);
    for (int a = 0; a < 3; ++a) u[a] = o->ub[3 * cell + a];
    if (o->nmodes <= 0) return;
    int k = fixed_face(o, x, y, z);
    if (k < 0) return;
    double un = (k % 2 ? 1.0 : -1.0) * u[k / 2]; /* ub . n, n outward */
    if (!(un < -1e-7)) return;
    double up[3];
    fluctuation(o, x, y, z, t, up);
    for (int a = 0; a < 3; ++a) u[a] += up[a];
}

static void write_fixed_cells_at(oracle_t *o, double t)
{
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                long cell = cell_of(o, x, y, z);
                if (o->cls[cell] != C_EQ_FIXED) continue;
                double u[3], g[Q];
                boundary_velocity(o, x, y, z, t, u);
                feq(1.0, u, g);
                to_storage(o, g);
                memcpy(o->G + cell * Q, g, sizeof g);
                memcpy(o->Gn + cell * Q, g, sizeof g);
                if (o->thermal) { /* reading 28: the thermal state of the cell is the equilibrium of the SAME velocity */
                    double h[QT];
                    heq(o->thb[cell], u, h);
                    memcpy(o->H + cell * QT, h, sizeof h);
                    memcpy(o->Hn + cell * QT, h, sizeof h);
                }
            }
}

/* modes = [n][9]: kappa[3], sigma[3], psi, omega, dkappa.  n = 0 switches the fluctuations off (cells return to the
 * mean).  The EQ_FIXED cells are rewritten for the current step at once. */
int oracle_set_inflow_turbulence(oracle_t *o, int n, const double *modes, double u_rms, double k_e, double k_eta)
{
    if (!o || n < 0 || (n > 0 && (!modes || !(k_e > 0.0) || u_rms < 0.0 || k_eta < 0.0))) return -1;
    if (!o->have_flags) return -3;
    free(o->modes); free(o->uhat); o->modes = NULL; o->uhat = NULL; o->nmodes = 0;
    if (n > 0) {
        o->modes = (double *)malloc(sizeof(double) * 9 * n);
        o->uhat = (double *)malloc(sizeof(double) * n);
        if (!o->modes || !o->uhat) return -4;
        memcpy(o->modes, modes, sizeof(double) * 9 * n);
        for (int i = 0; i < n; ++i) {
            const double *m = modes + 9 * i;
            double k = sqrt(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
            if (!(m[8] >= 0.0)) return -1;
            o->uhat[i] = sqrt(vk_spectrum(k, u_rms, k_e, k_eta) * m[8]);
        }
        o->nmodes = n;
    }
    write_fixed_cells_at(o, (double)o->step);
    return 0;
}

/* Thermal lattice on open faces (DESIGN.md §4 reading 27): an EQ_FIXED cell holds the thermal equilibrium of its prescribed
 * temperature and velocity, h_eq(theta_b, u_b), as it holds f_eq(1, u_b) for the flow. */
static void write_eq_fixed_thermal(oracle_t *o, long cell)
{
    if (!o->thermal) return;
    double h[QT];
    heq(o->thb[cell], o->ub + 3 * cell, h);
    memcpy(o->H + cell * QT, h, sizeof h);
    memcpy(o->Hn + cell * QT, h, sizeof h);
}

static void write_eq_fixed_cell(oracle_t *o, long cell)
{
    double g[Q];
    feq(1.0, o->ub + 3 * cell, g);
    to_storage(o, g);
    memcpy(o->G + cell * Q, g, sizeof g);
    memcpy(o->Gn + cell * Q, g, sizeof g);
    write_eq_fixed_thermal(o, cell);
}

/* step 5 (profile form): every EQ_FIXED cell gets f_eq(1, (u[z],v[z],w[z])) */
int oracle_set_inlet_profile(oracle_t *o, const double *u, const double *v, const double *w)
{
    if (!o->have_flags || o->nmodes > 0) return -3; /* the mean is fixed while fluctuations ride on it */
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                long cell = cell_of(o, x, y, z);
                if (o->cls[cell] != C_EQ_FIXED) continue;
                o->ub[3 * cell + 0] = u ? u[z] : 0.0;
                o->ub[3 * cell + 1] = v ? v[z] : 0.0;
                o->ub[3 * cell + 2] = w ? w[z] : 0.0;
                write_eq_fixed_cell(o, cell);
            }
    return 0;
}

/* step 5 (plane form): EQ_FIXED cells of one face get f_eq(1, uvw[:,j2,j1]);
 * uvw is [3][n2][n1] with (n2,n1) = (nz,ny) for x faces, (nz,nx) for y faces,
 * (ny,nx) for z faces. */
int oracle_set_inlet_plane(oracle_t *o, int face, const double *uvw)
{
    if (!o->have_flags || o->nmodes > 0) return -3;
    if (face < 0 || face > 5) return -1;
    int axis = face / 2;
    int n[3] = {o->nx, o->ny, o->nz};
    int fixed = (face % 2) ? n[axis] - 1 : 0;
    int a1 = axis == 0 ? 1 : 0;           /* fast in-plane axis */
    int a2 = axis == 2 ? 1 : 2;           /* slow in-plane axis */
    long plane = (long)n[a1] * n[a2];
    for (int j2 = 0; j2 < n[a2]; ++j2)
        for (int j1 = 0; j1 < n[a1]; ++j1) {
            int p[3];
            p[axis] = fixed; p[a1] = j1; p[a2] = j2;
            long cell = cell_of(o, p[0], p[1], p[2]);
            if (o->cls[cell] != C_EQ_FIXED) continue;
            for (int a = 0; a < 3; ++a) o->ub[3 * cell + a] = uvw[a * plane + (long)j2 * n[a1] + j1];
            write_eq_fixed_cell(o, cell);
        }
    return 0;
}

/* step 3 / a4: G0 = f_eq(rho0,u0); NULL rho => 1; NULL velocity component => 0.
 * SOLID cells: rho=1,u=0.  EQ_FIXED cells keep their prescribed state. */
int oracle_set_macros(oracle_t *o, const double *rho, const double *ux, const double *uy, const double *uz)
{
    if (!o->have_flags) return -3;
    long N = (long)o->nx * o->ny * o->nz;
    for (long cell = 0; cell < N; ++cell) {
        int cl = o->cls[cell];
        if (cl == C_EQ_FIXED) { write_eq_fixed_cell(o, cell); continue; }
        double r = rho ? rho[cell] : 1.0;
        double u[3] = {ux ? ux[cell] : 0.0, uy ? uy[cell] : 0.0, uz ? uz[cell] : 0.0};
        if (cl == C_SOLID) { r = 1.0; u[0] = u[1] = u[2] = 0.0; }
        double g[Q];
        feq(r, u, g);
        to_storage(o, g);
        memcpy(o->G + cell * Q, g, sizeof g);
        memcpy(o->Gn + cell * Q, g, sizeof g);
    }
    o->step = 0;
    if (o->nmodes > 0) write_fixed_cells_at(o, 0.0); /* the step counter restarts: inflow cells carry u'(x, 0) */
    return 0;
}

/* which face's normal an EQ_OUTFLOW cell uses: the first EQ_OUTFLOW face it
 * lies on, in the order x-,x+,y-,y+,z-,z+ (DESIGN.md §4 reading 24) */
static int outflow_face(const oracle_t *o, int x, int y, int z)
{
    int on[6] = {x == 0, x == o->nx - 1, y == 0, y == o->ny - 1, z == 0, z == o->nz - 1};
    for (int k = 0; k < 6; ++k)
        if (on[k] && o->face[k] == F_EQ_OUTFLOW) return k;
    return -1;
}

static void sample_mean(oracle_t *o)
{
    long N = (long)o->nx * o->ny * o->nz;
    if (!o->msum) o->msum = (double *)calloc(N * 3, sizeof(double));
#pragma omp parallel for schedule(static)
    for (long cell = 0; cell < N; ++cell) {
        double r, u[3];
        local_macros(o, o->G, cell, &r, u);
        for (int a = 0; a < 3; ++a) o->msum[3 * cell + a] += u[a];
    }
    o->mcount += 1;
}

/* Global flux-balancing correction of the prescribed open-boundary velocities ("mass flux consistency
 * correction ... the minimal normal velocity adjustment required to enforce near-zero net volume flow"
 * "a global flux-balancing correction is applied over the full set of open boundaries"; sign convention PAPER.md:185
 * "positive values indicate an outflow").  Open-boundary cells = the EQ_FIXED cells; each belongs to the first
 * EQ_FIXED face it lies on (order x-,x+,y-,y+,z-,z+) and n is that face's outward normal.
 *   Phi = sum over those cells of u_b . n        (unit cell faces, lattice units)
 *   minimal (least-squares) adjustment with sum(delta u . n) = -Phi: the same shift on every cell,
 *   u_b <- u_b - (Phi / N) n,   then G = f_eq(1, u_b) again.
 * Returns the net flux before and after (after is recomputed from the corrected cells). */
static int fixed_face(const oracle_t *o, int x, int y, int z)
{
    int on[6] = {x == 0, x == o->nx - 1, y == 0, y == o->ny - 1, z == 0, z == o->nz - 1};
    for (int k = 0; k < 6; ++k)
        if (on[k] && o->face[k] == F_EQ_FIXED) return k;
    return -1;
}

int oracle_balance_flux(oracle_t *o, double *flux_before, double *flux_after)
{
    if (!o || !o->have_flags || o->nmodes > 0) return -3;
    double phi = 0.0, phi2 = 0.0;
    long n = 0;
    for (int pass = 0; pass < 3; ++pass) {
        for (int z = 0; z < o->nz; ++z)
            for (int y = 0; y < o->ny; ++y)
                for (int x = 0; x < o->nx; ++x) {
                    long cell = cell_of(o, x, y, z);
                    if (o->cls[cell] != C_EQ_FIXED) continue;
                    int k = fixed_face(o, x, y, z);
                    if (k < 0) continue;
                    double nrm[3] = {0, 0, 0};
                    nrm[k / 2] = (k & 1) ? 1.0 : -1.0;
                    double rho, u[3];
                    local_macros(o, o->G, cell, &rho, u);
                    double un = u[0] * nrm[0] + u[1] * nrm[1] + u[2] * nrm[2];
                    if (pass == 0) { phi += un; n += 1; }
                    else if (pass == 1) {
                        double shift = phi / (double)n;
                        double ub[3] = {u[0] - shift * nrm[0], u[1] - shift * nrm[1], u[2] - shift * nrm[2]};
                        feq(1.0, ub, o->G + cell * Q);
                        to_storage(o, o->G + cell * Q);
                        memcpy(o->Gn + cell * Q, o->G + cell * Q, sizeof(double) * Q);
                        for (int a = 0; a < 3; ++a) o->ub[3 * cell + a] = ub[a];
                    } else phi2 += un;
                }
        if (pass == 0 && n == 0) break;
    }
    if (flux_before) *flux_before = phi;
    if (flux_after) *flux_after = phi2;
    return 0;
}

/* Fixed-temperature walls of the thermal lattice (DESIGN.md §4 reading 26).  The paper's thermal workload is a closed
 * adiabatic box and its Table 1 only names the lattice; a wall held at a temperature is the
 * textbook halfway anti-bounce-back rule for an advection-diffusion lattice: a thermal population that leaves a cell
 * towards a WALL face k held at theta_w returns as  h_ibar <- -h_i + 2 wT_i theta_w  (wall at rest), which puts
 * theta = theta_w half a cell outside the last node, where halfway bounce-back puts the no-slip wall.  Only domain faces
 * of type WALL can be held; buildings and all other faces stay adiabatic (plain bounce-back / specular reflection).
 * Which face does the pull of direction i (1..6, an axis direction) of cell (x,y,z) cross?  -1 if none that is held. */
static int fixed_temperature_face(const oracle_t *o, int x, int y, int z, int i)
{
    if (i < 1 || i > 6) return -1;
    int p[3] = {x - CI[i][0], y - CI[i][1], z - CI[i][2]};
    int n[3] = {o->nx, o->ny, o->nz};
    for (int a = 0; a < 3; ++a) {
        int k = -1;
        if (p[a] < 0) k = 2 * a;
        else if (p[a] >= n[a]) k = 2 * a + 1;
        if (k >= 0 && o->face[k] == F_WALL && o->thd[k]) return k;
    }
    return -1;
}

/* on[6] (x-,x+,y-,y+,z-,z+): 1 = hold that face at theta_w[k].  The face must be a WALL face (-1 otherwise). */
int oracle_set_thermal_walls(oracle_t *o, const int *on, const double *theta_w)
{
    if (!o || !on || !theta_w || !o->thermal) return -3;
    for (int k = 0; k < 6; ++k)
        if (on[k] && o->face[k] != F_WALL) return -1;
    for (int k = 0; k < 6; ++k) { o->thd[k] = on[k] ? 1 : 0; o->thw[k] = theta_w[k]; }
    return 0;
}

int oracle_step(oracle_t *o, int nsteps)
{
    if (!o->have_flags) return -3;
    int bad = 0;
    for (int it = 0; it < nsteps; ++it) {
#pragma omp parallel for schedule(static)
        for (int z = 0; z < o->nz; ++z)
            for (int y = 0; y < o->ny; ++y)
                for (int x = 0; x < o->nx; ++x) {
                    long cell = cell_of(o, x, y, z);
                    int cl = o->cls[cell];
                    double *gn = o->Gn + cell * Q;
                    if (cl == C_FLUID) {
                        /* step 4a pull */
                        double f[Q];
                        for (int i = 0; i < Q; ++i) {
                            long s = 0; int j = 0;
                            int r = resolve(o, x, y, z, i, &s, &j);
                            if (r < 0) {
#pragma omp atomic write
                                bad = 1;
                                r = 1;
                            }
                            f[i] = r ? o->G[cell * Q + opposite(i)] : o->G[s * Q + j];
                        }
                        double ut[3] = {0, 0, 0};
                        if (o->ut) for (int a = 0; a < 3; ++a) ut[a] = o->ut[a * o->nz + z];
                        if (!o->thermal) {
                            collide(f, o->nu0, o->Cs, o->fv, o->F, o->sig ? o->sig[cell] : 0.0, ut, gn, NULL, NULL, NULL);
                            to_storage(o, gn);
                        } else {
                            /* thermal lattice (reading 23): pull the 7 thermal populations by the same rule 4a
                             * (bounce-back on walls / solids and specular reflection on free-slip faces = no heat flux),
                             * theta = sum_i h_i; the flow collision sees F + g beta (theta - theta_ref) e_z; the thermal
                             * BGK relaxes towards h_eq(theta, u) with the velocity u of that flow collision */
                            double h[QT], theta = 0.0;
                            for (int i = 0; i < QT; ++i) {
                                long s = 0; int j = 0;
                                int r = resolve(o, x, y, z, i, &s, &j);
                                if (r < 0) {
#pragma omp atomic write
                                    bad = 1;
                                    r = 1;
                                }
                                h[i] = r ? o->H[cell * QT + opposite(i)] : o->H[s * QT + j];
                                /* a WALL face held at theta_w (reading 26): anti-bounce-back, the population comes
                                 * back with the opposite sign plus twice the wall's equilibrium share */
                                int kf = r ? fixed_temperature_face(o, x, y, z, i) : -1;
                                if (kf >= 0) h[i] = -o->H[cell * QT + opposite(i)] + 2.0 * weight_t(i) * o->thw[kf];
                                theta += h[i];
                            }
                            double Fb[3] = {o->F[0], o->F[1], o->F[2] + o->gbeta * (theta - o->theta_ref)};
                            double u[3];
                            collide(f, o->nu0, o->Cs, o->fv, Fb, o->sig ? o->sig[cell] : 0.0, ut, gn, NULL, u, NULL);
                            double he[QT], tau_t = 4.0 * o->alpha + 0.5;
                            heq(theta, u, he);
                            for (int i = 0; i < QT; ++i) o->Hn[cell * QT + i] = h[i] - (h[i] - he[i]) / tau_t;
                        }
                    } else if (cl == C_EQ_OUTFLOW) {
                        /* step 6 */
                        int k = outflow_face(o, x, y, z);
                        int p[3] = {x, y, z};
                        p[k / 2] += (k % 2) ? -1 : +1; /* x - n, n outward */
                        int n[3] = {o->nx, o->ny, o->nz};
                        double r, u[3] = {0, 0, 0};
                        double th_nb = o->theta_ref;
                        if (p[k / 2] >= 0 && p[k / 2] < n[k / 2]) {
                            long nb = cell_of(o, p[0], p[1], p[2]);
                            local_macros(o, o->G, nb, &r, u);
                            if (o->thermal && o->cls[nb] != C_SOLID) {
                                th_nb = 0.0;
                                for (int i = 0; i < QT; ++i) th_nb += o->H[nb * QT + i];
                            }
                        }
                        feq(1.0, u, gn);
                        to_storage(o, gn);
                        /* reading 27: the outflow cell also copies the temperature of its inward neighbour (zero gradient) */
                        if (o->thermal) heq(th_nb, u, o->Hn + cell * QT);
                    } else if (cl == C_EQ_FIXED && o->nmodes > 0) {
                        /* step 5 with fluctuations: the state of step k+1 carries u'(x, k+1) */
                        double u[3];
                        boundary_velocity(o, x, y, z, (double)(o->step + 1), u);
                        feq(1.0, u, gn);
                        to_storage(o, gn);
                        /* reading 28: with the thermal lattice on, the cell holds h_eq(theta_b, u_b + u') beside
                         * f_eq(1, u_b + u') — one boundary velocity for both lattices, as reading 27 has it for the mean */
                        if (o->thermal) heq(o->thb[cell], u, o->Hn + cell * QT);
                    } else {
                        /* SOLID: inert; EQ_FIXED (step 5): unchanged */
                        memcpy(gn, o->G + cell * Q, sizeof(double) * Q);
                    }
                    if (o->thermal && cl != C_FLUID && cl != C_EQ_OUTFLOW && !(cl == C_EQ_FIXED && o->nmodes > 0))
                        memcpy(o->Hn + cell * QT, o->H + cell * QT, sizeof(double) * QT);
                }
        double *t = o->G; o->G = o->Gn; o->Gn = t;
        if (o->thermal) { t = o->H; o->H = o->Hn; o->Hn = t; }
        o->step += 1;
        /* step 8 */
        if (o->mevery > 0 && o->step >= o->mstart && (o->step - o->mstart) % o->mevery == 0) sample_mean(o);
    }
    return bad ? -2 : 0;
}

int oracle_get_macros(const oracle_t *o, double *rho, double *ux, double *uy, double *uz)
{
    long N = (long)o->nx * o->ny * o->nz;
#pragma omp parallel for schedule(static)
    for (long cell = 0; cell < N; ++cell) {
        double r, u[3];
        local_macros(o, o->G, cell, &r, u);
        if (rho) rho[cell] = r;
        if (ux) ux[cell] = u[0];
        if (uy) uy[cell] = u[1];
        if (uz) uz[cell] = u[2];
    }
    return 0;
}

int oracle_mean_config(oracle_t *o, long start_step, int every)
{
    o->mstart = start_step; o->mevery = every;
    return 0;
}

int oracle_mean_reset(oracle_t *o)
{
    long N = (long)o->nx * o->ny * o->nz;
    if (o->msum) memset(o->msum, 0, sizeof(double) * N * 3);
    o->mcount = 0;
    return 0;
}

/* step 8: mean = sum / count (SOLID cells contribute and return 0) */
int oracle_get_mean(const oracle_t *o, double *ux, double *uy, double *uz, long *n_samples)
{
    long N = (long)o->nx * o->ny * o->nz;
    if (n_samples) *n_samples = o->mcount;
    for (long cell = 0; cell < N; ++cell) {
        double inv = o->mcount > 0 ? 1.0 / (double)o->mcount : 0.0;
        double s0 = o->msum ? o->msum[3 * cell + 0] : 0.0;
        double s1 = o->msum ? o->msum[3 * cell + 1] : 0.0;
        double s2 = o->msum ? o->msum[3 * cell + 2] : 0.0;
        if (ux) ux[cell] = s0 * inv;
        if (uy) uy[cell] = s1 * inv;
        if (uz) uz[cell] = s2 * inv;
    }
    return 0;
}

/* raw populations, [19][nz][ny][nx] in the order of step 1 */
int oracle_get_state(const oracle_t *o, double *f)
{
    long N = (long)o->nx * o->ny * o->nz;
    for (int i = 0; i < Q; ++i)
        for (long cell = 0; cell < N; ++cell) f[(long)i * N + cell] = o->G[cell * Q + i];
    return 0;
}

int oracle_set_state(oracle_t *o, const double *f)
{
    long N = (long)o->nx * o->ny * o->nz;
    for (long cell = 0; cell < N; ++cell) {
        double g[Q];
        for (int i = 0; i < Q; ++i) g[i] = f[(long)i * N + cell];
        to_storage(o, g);
        memcpy(o->G + cell * Q, g, sizeof g);
        memcpy(o->Gn + cell * Q, g, sizeof g);
    }
    return 0;
}

/* 16-bit population storage on (1) / off (0); see round_to_half.  Takes effect for every population written from now
 * on (set it before the state is initialised).  Not combinable with the thermal lattice (-1). */
int oracle_set_storage16(oracle_t *o, int on)
{
    if (!o || (on && o->thermal)) return -1;
    o->store16 = on ? 1 : 0;
    return 0;
}

long oracle_get_step(const oracle_t *o) { return o->step; }
int oracle_set_step(oracle_t *o, long s) { o->step = s; return 0; }

/* ------------------------------------------------------------------ thermal lattice (reading 23) */

/* Switch the D3Q7 thermal lattice on: diffusivity alpha (tau_theta = 4 alpha + 1/2), buoyancy coefficient gbeta
 * (acceleration g beta (theta - theta_ref) along +z), reference theta.  The thermal state is set to theta_ref at rest.
 * On open faces (reading 27) EQ_FIXED cells take h_eq(theta_b, u_b) with theta_b = theta_ref until oracle_set_inlet_theta. */
int oracle_set_thermal(oracle_t *o, double alpha, double gbeta, double theta_ref)
{
    if (o->store16) return -1;
    if (!(alpha > 0.0)) return -1;
    long N = (long)o->nx * o->ny * o->nz;
    if (!o->H) {
        o->H = (double *)malloc(sizeof(double) * N * QT);
        o->Hn = (double *)malloc(sizeof(double) * N * QT);
        if (!o->H || !o->Hn) return -4;
    }
    if (!o->thb) {
        o->thb = (double *)malloc(sizeof(double) * N);
        if (!o->thb) return -4;
    }
    o->alpha = alpha; o->gbeta = gbeta; o->theta_ref = theta_ref; o->thermal = 1;
    for (long cell = 0; cell < N; ++cell) {
        o->thb[cell] = theta_ref;
        for (int i = 0; i < QT; ++i) o->H[cell * QT + i] = o->Hn[cell * QT + i] = weight_t(i) * theta_ref;
        if (o->have_flags && o->cls[cell] == C_EQ_FIXED) write_eq_fixed_thermal(o, cell);
    }
    /* reading 28: inflow cells that carry fluctuations hold the thermal equilibrium of the velocity they have now */
    if (o->have_flags && o->nmodes > 0) write_fixed_cells_at(o, (double)o->step);
    return 0;
}

/* Prescribed temperature of the EQ_FIXED cells by level, theta_b(z) [nz] (reading 27): their thermal state becomes
 * h_eq(theta_b, u_b).  Call it after the velocity profile / plane (a later velocity call keeps theta_b). */
int oracle_set_inlet_theta(oracle_t *o, const double *theta_b)
{
    if (!o->thermal || !o->have_flags || !theta_b) return -3;
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                long cell = cell_of(o, x, y, z);
                if (o->cls[cell] != C_EQ_FIXED) continue;
                o->thb[cell] = theta_b[z];
                write_eq_fixed_thermal(o, cell);
            }
    if (o->nmodes > 0) write_fixed_cells_at(o, (double)o->step); /* reading 28: ... of the velocity the cells have now */
    return 0;
}

/* H0 = h_eq(theta0, u0); NULL velocity component => 0; SOLID cells: theta_ref at rest; EQ_FIXED cells keep their boundary state. */
int oracle_set_theta(oracle_t *o, const double *theta, const double *ux, const double *uy, const double *uz)
{
    if (!o->thermal) return -3;
    long N = (long)o->nx * o->ny * o->nz;
    for (long cell = 0; cell < N; ++cell) {
        double th = theta ? theta[cell] : o->theta_ref;
        double u[3] = {ux ? ux[cell] : 0.0, uy ? uy[cell] : 0.0, uz ? uz[cell] : 0.0};
        if (o->cls[cell] == C_EQ_FIXED) continue; /* keeps its boundary state h_eq(theta_b, u_b), as in oracle_set_macros */
        if (o->cls[cell] == C_SOLID) { th = o->theta_ref; u[0] = u[1] = u[2] = 0.0; }
        double h[QT];
        heq(th, u, h);
        memcpy(o->H + cell * QT, h, sizeof h);
        memcpy(o->Hn + cell * QT, h, sizeof h);
    }
    return 0;
}

/* theta = sum_i h_i of the stored state; SOLID cells report theta_ref */
int oracle_get_theta(const oracle_t *o, double *theta)
{
    if (!o->thermal) return -3;
    long N = (long)o->nx * o->ny * o->nz;
    for (long cell = 0; cell < N; ++cell) {
        double th = 0.0;
        for (int i = 0; i < QT; ++i) th += o->H[cell * QT + i];
        theta[cell] = o->cls[cell] == C_SOLID ? o->theta_ref : th;
    }
    return 0;
}

/* the 7 thermal populations h_i of the stored state, [7][nz][ny][nx] (directions 0..6 of the flow lattice); SOLID cells report
 * the rest state wT_i theta_ref — the format of the library's lbm_get_thermal_state */
int oracle_get_thermal_state(const oracle_t *o, double *h)
{
    if (!o->thermal) return -3;
    long N = (long)o->nx * o->ny * o->nz;
    for (long cell = 0; cell < N; ++cell)
        for (int i = 0; i < QT; ++i)
            h[(long)i * N + cell] = o->cls[cell] == C_SOLID ? weight_t(i) * o->theta_ref : o->H[cell * QT + i];
    return 0;
}

int oracle_heq(double theta, const double *u, double *out) { heq(theta, u, out); return 0; }
