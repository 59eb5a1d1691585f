/* lbm_oracle.c — fp64 CPU ORACLE for the fused D3Q19 LES + forest-canopy LBM step.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or constant generator with paper_2206_15454_b200/ (the CUDA path) and
 * neither imports the other.
 *
 * What it is: the algorithm of arxiv 2206.15454 (Shao et al.) written out step by step in the
 * paper's order and notation — Algorithm 1 with Eqs. 1-16 — in plain
 * double precision, two full lattices (fa = state, fb = next), pull streaming, fixed summation
 * order i = 0..18, OpenMP over (z,y) rows only.  No blocking, fusion, vectorisation tricks or
 * shifted populations.  Readings of ambiguous passages are the ones tabulated in DESIGN.md
 * ("Readings", R1..) and cited at each site below.
 *
 * Pins (tests/test_oracle_pins.py, tests/test_paper_cases.py, -m "not gpu"): lattice identities (P0),
 * rest state (P1), mass conservation (P2), Poiseuille (P3), Taylor-Green (P4), exact momentum
 * increment (P5), uniform-flow drag recurrence (P6), tau_total self-consistency (P7), mirror
 * equivalence (P8), analytic plane statistics (P9), z-mirror/translation symmetry (P12), brute-force
 * push streaming (P13), Couette flow under the forced-equilibrium lid (P14), solid cells: brute-force
 * push with random solids, solid layers == wall faces, mass (P15), the Pi_neq assembly inside the
 * collision: relaxation of a known non-equilibrium part (P16), run-time removal of solids (P17),
 * per-cell forest codes (P18), row-table SGS models (P19), splitmix64 known answers, LAD closed forms, Table I / II / III numbers,
 * the text's qualitative statements about the three ABL cases.
 * PARITY UNPINNED (no printed value or closed form in the paper fixes them; both sides share the
 * reading): (R4) no rho factor in the drag of Eq. 13, (R5) streamwise-only vs vector drag direction,
 * (R8) no forcing correction in Pi_neq, (R9) Eq. 10 rather than Eq. 12 as printed where they differ
 * (rho != 1), (R27) the bit layout of the forest code, (R28) f_eq(1, 0) in cells freed from a solid, (R29) which
 * "other SGS models" (the paper names none).
 *
 * Units: lattice units, dx = dt = 1, c = 1, c_s^2 = 1/3, filter width Delta = dx = 1.
 * Layout: cell = x + nx*(y + ny*z), x streamwise, y wall-normal, z spanwise; f[i*N + cell].
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define Q 19
#define NSTAT 10

/* D3Q19 velocity set, weights, opposite and y-mirror maps.  PAPER.md:L39 names "D3Q19" only;
 * this is the standard lattice (reading R2).  Index i : c_i. */
static const int C[Q][3] = {
    {0, 0, 0},
    {1, 0, 0},  {-1, 0, 0},  {0, 1, 0},  {0, -1, 0}, {0, 0, 1},  {0, 0, -1},
    {1, 1, 0},  {-1, -1, 0}, {1, -1, 0}, {-1, 1, 0},
    {1, 0, 1},  {-1, 0, -1}, {1, 0, -1}, {-1, 0, 1},
    {0, 1, 1},  {0, -1, -1}, {0, 1, -1}, {0, -1, 1}};
static const double W[Q] = {
    1.0 / 3.0,
    1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0,
    1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0,
    1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0};
/* opp(i): c_opp = -c_i */
static const int OPP[Q] = {0, 2, 1, 4, 3, 6, 5, 8, 7, 10, 9, 12, 11, 14, 13, 16, 15, 18, 17};
/* m(i): c_y -> -c_y (specular reflection at a y-face) */
static const int MIR[Q] = {0, 1, 2, 4, 3, 5, 6, 9, 10, 7, 8, 11, 12, 13, 14, 18, 17, 16, 15};

/* bc_flags bit layout: the oracle keeps its own copy of the constants. */
enum {
    ORC_BOTTOM_MASK = 0x3,  /* bits 0-1: 0 bounce-back wall, 1 periodic-y */
    ORC_TOP_SHIFT = 2,      /* bits 2-3: 0 bounce-back, 1 free-slip, 2 periodic-y, 3 forced-eq */
    ORC_DRAG_VECTOR = 1 << 4, /* bit 4: 0 streamwise-only drag (paper), 1 vector drag */
    ORC_SOLID_MASK = 1 << 5   /* bit 5: per-cell solid mask present */
};

typedef struct orc_s {
    int nx, ny, nz;
    long long N;
    double nu, Csmag, Fb[3], Cd, tau0;
    double *lad;          /* [ny] a(y_j), 0 = not forest */
    unsigned bc;
    double Utop[3];       /* forced-equilibrium lid velocity (NEXT #1) */
    unsigned char *solid; /* [N] 1 = solid (NEXT #2), NULL = none */
    uint32_t *fcode;      /* [N] per-cell forest code (NEXT #2), NULL = none; 0 = use lad[y] */
    double a_fm;          /* a_fm of Eq. 14 for the coded cells */
    double *sgs_C;        /* [ny] per-row Smagorinsky constant C_smag,j (other SGS models), NULL = Csmag */
    double *sgs_Sbar;     /* [ny] per-row mean-shear magnitude |<S>|_j (shear-improved model), NULL = 0 */
    double *fa, *fb;      /* [Q][N] */
    double *acc;          /* [ny][NSTAT] running sums */
    double *rowsum;       /* [nz][ny][NSTAT] scratch */
    long long nsamples;
    int stats_every;
    long long stats_phase;
    long long t;
} orc_t;

/* ---------------------------------------------------------------------------------------- */
/* Unit functions (also exported so the pins can exercise them in isolation)                 */
/* ---------------------------------------------------------------------------------------- */

void orc_tables(int *c /*[19][3]*/, double *w, int *opp, int *mir)
{
    for (int i = 0; i < Q; ++i) {
        c[3 * i] = C[i][0]; c[3 * i + 1] = C[i][1]; c[3 * i + 2] = C[i][2];
        w[i] = W[i]; opp[i] = OPP[i]; mir[i] = MIR[i];
    }
}

/* Eq. 3: f_i^eq = w_i rho [1 + c.u/cs2 + (c.u)^2/(2 cs4) - u.u/(2 cs2)], cs2 = 1/3 */
void orc_feq(double rho, const double *u, double *feq)
{
    double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    for (int i = 0; i < Q; ++i) {
        double cu = C[i][0] * u[0] + C[i][1] * u[1] + C[i][2] * u[2];
        feq[i] = W[i] * rho * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * uu);
    }
}

/* Eq. 4: F_i = (1 - 1/(2 tau)) w_i [ (c_i - u)/cs2 + (c_i.u) c_i / cs4 ] . F */
void orc_guo(double tau, const double *u, const double *F, double *Fi)
{
    for (int i = 0; i < Q; ++i) {
        double cu = C[i][0] * u[0] + C[i][1] * u[1] + C[i][2] * u[2];
        double s = 0.0;
        for (int a = 0; a < 3; ++a)
            s += (3.0 * (C[i][a] - u[a]) + 9.0 * cu * C[i][a]) * F[a];
        Fi[i] = (1.0 - 1.0 / (2.0 * tau)) * W[i] * s;
    }
}

/* Eqs. 10-12, reading R9: tau_total = tau0 + 3 C_smag |S| with |S| of Eq. 10
 * (delta = Delta = dx = 1, c = 1, C == C_smag)
 *   => tau_total = ( tau0 + sqrt( tau0^2 + 18 sqrt(2) C_smag Q^{1/2} / rho ) ) / 2.
 * Pneq is the full symmetric tensor given as [xx, yy, zz, xy, yz, xz]; Eq. 11 contracts all
 * nine entries (off-diagonals twice). */
double orc_tau_total(double tau0, double Csmag, double rho, const double *Pneq)
{
    double QQ = Pneq[0] * Pneq[0] + Pneq[1] * Pneq[1] + Pneq[2] * Pneq[2] +
                2.0 * (Pneq[3] * Pneq[3] + Pneq[4] * Pneq[4] + Pneq[5] * Pneq[5]);
    double Qh = sqrt(QQ); /* Eq. 11 */
    return 0.5 * (tau0 + sqrt(tau0 * tau0 + 18.0 * sqrt(2.0) * Csmag * Qh / rho));
}

/* Other SGS models ("the standard Smagorinsky model is used ... A future work is to
 * implement other SGS models").  The paper names none; two published eddy-
 * viscosity closures that keep the local form of Eq. 10, nu_t = C Delta^2 x (a strain-rate measure),
 * are restated here (reading R29).  With |S| the strain-rate magnitude that Eq. 10 takes
 * from Pi_neq - Eq. 10 is tau_total = tau0 + 3 C |S| solved for tau_total, which fixes
 * |S| = 3 Q^{1/2} / (sqrt(2) rho tau_total) -
 *   wall-damped Smagorinsky (van Driest damping): nu_t = C_j |S|, C_j = C_smag D(y+_j)^2,
 *       D = 1 - exp(-y+/A+): a per-row constant (orc_sgs_van_driest);
 *   shear-improved Smagorinsky (Leveque, Toschi, Shao, Bertoglio 2007): nu_t = C (|S| - |<S>|),
 *       never negative, <S> the mean shear - in a plane-homogeneous flow a per-row number
 *       Sbar_j = |d<u>/dy| (orc_sgs_mean_shear).
 * Both: tau_total = tau0 + 3 C_j (|S| - Sbar_j)_+.  While the bracket is positive this is the
 * quadratic of Eq. 10 with tau0 replaced by tau0' = tau0 - 3 C_j Sbar_j,
 *   tau_total = ( tau0' + sqrt( tau0'^2 + 18 sqrt(2) C_j Q^{1/2} / rho ) ) / 2,
 * and the bracket is positive exactly when that root exceeds tau0; otherwise nu_t = 0 and
 * tau_total = tau0.  C_j = C_smag, Sbar_j = 0 is Eq. 10 itself. */
double orc_tau_total_rows(double tau0, double C_j, double Sbar_j, double rho, const double *Pneq)
{
    double QQ = Pneq[0] * Pneq[0] + Pneq[1] * Pneq[1] + Pneq[2] * Pneq[2] +
                2.0 * (Pneq[3] * Pneq[3] + Pneq[4] * Pneq[4] + Pneq[5] * Pneq[5]);
    double Qh = sqrt(QQ); /* Eq. 11 */
    double tau0p = tau0 - 3.0 * C_j * Sbar_j;
    double tau = 0.5 * (tau0p + sqrt(tau0p * tau0p + 18.0 * sqrt(2.0) * C_j * Qh / rho));
    return (tau > tau0) ? tau : tau0;
}

/* van Driest damping of the Smagorinsky constant: C_j = Cs^2 [1 - exp(-y+_j / A+)]^2, y+_j =
 * d_j u_tau / nu with d_j the distance of the cell centre j + 1/2 from the nearest no-slip wall
 * (bottom wall only, or both walls of a channel). */
void orc_sgs_van_driest(int ny, double Cs, double u_tau, double nu, double A_plus, int both_walls, double *C_out)
{
    for (int j = 0; j < ny; ++j) {
        double d = j + 0.5;
        if (both_walls && ny - d < d) d = ny - d;
        double D = 1.0 - exp(-(d * u_tau / nu) / A_plus);
        C_out[j] = Cs * Cs * D * D;
    }
}

/* Mean-shear magnitude of a plane-averaged profile: |<S>| = sqrt(2 <S>:<S>) with <S>_xy =
 * (1/2) d<u>/dy, <S>_yz = (1/2) d<w>/dy  =>  Sbar_j = sqrt( (d<u>/dy)^2 + (d<w>/dy)^2 ).
 * Central differences between cell centres; at a no-slip wall the profile is extended with its
 * mirror image of opposite sign (u = 0 on the face), at a free-slip or lid face with its mirror
 * image (zero gradient).  stats = the [ny][10] table of orc_stats_read (columns 0 and 2).
 * top_wall: 1 = no-slip wall at the top face, 0 = zero-gradient top. */
void orc_sgs_mean_shear(const double *stats, int ny, int top_wall, double *Sbar_out)
{
    for (int j = 0; j < ny; ++j) {
        double d[2];
        for (int a = 0; a < 2; ++a) {
            int col = a ? 2 : 0;
            double below = (j > 0) ? stats[(j - 1) * NSTAT + col] : -stats[col];
            double above = (j < ny - 1) ? stats[(j + 1) * NSTAT + col]
                                        : (top_wall ? -stats[(ny - 1) * NSTAT + col] : stats[(ny - 1) * NSTAT + col]);
            d[a] = 0.5 * (above - below);
        }
        Sbar_out[j] = sqrt(d[0] * d[0] + d[1] * d[1]);
    }
}

/* Counter-based uniform generator in [0,1) shared by specification with the CUDA path
 * (DESIGN.md "Input recipe"): the splitmix64 output function applied to
 * state = seed + (ctr+1)*0x9E3779B97F4A7C15, top 53 bits. */
uint64_t orc_mix64(uint64_t seed, uint64_t ctr)
{
    uint64_t z = seed + (ctr + 1ULL) * 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
double orc_rand01(uint64_t seed, uint64_t ctr)
{
    return (double)(orc_mix64(seed, ctr) >> 11) * (1.0 / 9007199254740992.0);
}

/* Eqs. 14-15, reading R14: shape s(eta) = r^n exp[n(1-r)],
 * r = (1-eta_m)/(1-eta), n = 6 for eta < eta_m, 1/2 otherwise; evaluated at cell centres
 * eta_j = (j+1/2)/h, normalised so that sum_j a_j = LAI; a_j = 0 for j >= h. */
double orc_lad_shape(double eta, double eta_m)
{
    if (eta >= 1.0) return 0.0;
    double r = (1.0 - eta_m) / (1.0 - eta);
    double n = (eta < eta_m) ? 6.0 : 0.5;
    return pow(r, n) * exp(n * (1.0 - r));
}
void orc_lad_profile(int h, int ny, double LAI, double eta_m, double *out)
{
    double sum = 0.0;
    for (int j = 0; j < ny; ++j) {
        out[j] = (j < h) ? orc_lad_shape((j + 0.5) / h, eta_m) : 0.0;
        sum += out[j];
    }
    for (int j = 0; j < ny; ++j) out[j] = (sum > 0.0) ? LAI * out[j] / sum : 0.0;
}

/* ---------------------------------------------------------------------------------------- */
/* Handle                                                                                    */
/* ---------------------------------------------------------------------------------------- */

orc_t *orc_create(int nx, int ny, int nz, double nu, double Cs, const double *body_force,
                  double Cd, const double *lad_profile, unsigned bc_flags)
{
    if (nx < 1 || ny < 1 || nz < 1 || !(nu > 0.0)) return NULL;
    unsigned bot = bc_flags & ORC_BOTTOM_MASK, top = (bc_flags >> ORC_TOP_SHIFT) & 3u;
    if ((bot == 1) != (top == 2)) return NULL; /* periodic-y needs both faces */
    orc_t *o = (orc_t *)calloc(1, sizeof(orc_t));
    o->nx = nx; o->ny = ny; o->nz = nz; o->N = (long long)nx * ny * nz;
    o->nu = nu;
    o->Csmag = Cs * Cs;          /* reading R9: paper's C_smag == Cs^2 (Table I 0.01 <-> Cs 0.1) */
    o->tau0 = 3.0 * nu + 0.5;    /* reading R3: nu = cs2 (tau0 - 1/2) */
    for (int a = 0; a < 3; ++a) o->Fb[a] = body_force ? body_force[a] : 0.0;
    o->Cd = Cd;
    o->lad = (double *)calloc(ny, sizeof(double));
    if (lad_profile) memcpy(o->lad, lad_profile, ny * sizeof(double));
    o->bc = bc_flags;
    o->fa = (double *)malloc(sizeof(double) * Q * o->N);
    o->fb = (double *)malloc(sizeof(double) * Q * o->N);
    o->acc = (double *)calloc((size_t)ny * NSTAT, sizeof(double));
    o->rowsum = (double *)calloc((size_t)nz * ny * NSTAT, sizeof(double));
    if (!o->fa || !o->fb) { free(o->fa); free(o->fb); free(o); return NULL; }
    /* rest state */
    for (int i = 0; i < Q; ++i)
        for (long long n = 0; n < o->N; ++n) o->fa[i * o->N + n] = W[i];
    return o;
}

void orc_destroy(orc_t *o)
{
    if (!o) return;
    free(o->lad); free(o->solid); free(o->fcode); free(o->sgs_C); free(o->sgs_Sbar); free(o->fa); free(o->fb); free(o->acc); free(o->rowsum);
    free(o);
}

void orc_set_top_velocity(orc_t *o, const double *U) { for (int a = 0; a < 3; ++a) o->Utop[a] = U[a]; }

/* Per-cell forest code: "The code for each forest cell contains ... h: height
 * of the forest ...; y: distance in the vertical direction between the lower bounding box of the
 * forest object and the current cell; y_m: distance ... between the lower bounding box of the
 * forest and the maximum value of the LAD distribution.  This information is stored into the
 * forest cell's code using a bit mask".  Layout chosen here (the paper gives none; DESIGN.md
 * reading R27): bits 0-9 y (cells), bits 10-19 h (cells, 0 = not a forest cell), bits 20-31 y_m in
 * eighths of a cell (0 = no maximum: constant LAD a_fm, Table II case 1).
 * LAD of a coded cell, Eq. 14 (L107) with Eq. 15 (L112) at the cell centre eta = (y + 1/2)/h,
 * eta_m = y_m/h: a_f = a_fm * shape(eta, eta_m). */
uint32_t orc_forest_code(int h, int y, double y_m)
{
    uint32_t ym8 = (uint32_t)floor(y_m * 8.0 + 0.5);
    return ((uint32_t)y & 1023u) | (((uint32_t)h & 1023u) << 10) | ((ym8 & 4095u) << 20);
}
double orc_forest_code_lad(uint32_t code, double a_fm)
{
    int y = (int)(code & 1023u), h = (int)((code >> 10) & 1023u);
    double y_m = (double)((code >> 20) & 4095u) / 8.0;
    if (h == 0 || y >= h) return 0.0;
    if (y_m == 0.0) return a_fm;
    return a_fm * orc_lad_shape((y + 0.5) / h, y_m / h);
}
void orc_set_forest_codes(orc_t *o, const uint32_t *code /* [N] or NULL */, double a_fm)
{
    free(o->fcode); o->fcode = NULL; o->a_fm = a_fm;
    if (code) {
        o->fcode = (uint32_t *)malloc(sizeof(uint32_t) * o->N);
        memcpy(o->fcode, code, sizeof(uint32_t) * o->N);
    }
}

/* Per-row SGS tables (see orc_tau_total_rows): C_j and / or Sbar_j, [ny] each; NULL, NULL restores
 * the standard model of the paper. */
void orc_set_sgs_rows(orc_t *o, const double *C_row, const double *Sbar_row)
{
    free(o->sgs_C); free(o->sgs_Sbar); o->sgs_C = NULL; o->sgs_Sbar = NULL;
    if (C_row) {
        o->sgs_C = (double *)malloc(sizeof(double) * o->ny);
        memcpy(o->sgs_C, C_row, sizeof(double) * o->ny);
    }
    if (Sbar_row) {
        o->sgs_Sbar = (double *)malloc(sizeof(double) * o->ny);
        memcpy(o->sgs_Sbar, Sbar_row, sizeof(double) * o->ny);
    }
}

/* Install (or with NULL remove) the solid cells AT RUN TIME, keeping the flow (PAPER.md:L226:
 * "Once the turbulence is developed, the boxes are removed from the computational domain.  The
 * flow remains in the turbulent status afterwards").  Cells that stay fluid keep their
 * populations; a cell that is solid carries the rest state f = w, so a cell that turns fluid
 * starts from f_eq(1, 0) (reading R28). */
void orc_set_solid(orc_t *o, const unsigned char *mask /* [N] or NULL */)
{
    free(o->solid); o->solid = NULL;
    if (mask) {
        o->solid = (unsigned char *)malloc(o->N);
        memcpy(o->solid, mask, o->N);
        /* solid cells carry the rest state and are never updated */
        for (long long n = 0; n < o->N; ++n)
            if (o->solid[n]) for (int i = 0; i < Q; ++i) o->fa[i * o->N + n] = W[i];
    }
}

/* O1: state 0 = f^eq(rho, u) per Eq. 3, no non-equilibrium part (reading R17). */
void orc_set_macros(orc_t *o, const double *rho /*[N]*/, const double *u /*[3][N]*/)
{
    for (long long n = 0; n < o->N; ++n) {
        double uu[3] = {u[n], u[o->N + n], u[2 * o->N + n]}, feq[Q];
        double r = rho[n];
        if (o->solid && o->solid[n]) { r = 1.0; uu[0] = uu[1] = uu[2] = 0.0; }
        orc_feq(r, uu, feq);
        for (int i = 0; i < Q; ++i) o->fa[i * o->N + n] = feq[i];
    }
    o->t = 0;
}

/* Initial macroscopic field (reading R16): rho = 1,
 * u = U(y_j) e_x + noise_frac * U_ref * (2 r - 1) per component, r = rand01(seed, 3*cell + comp).
 * kind 0: U = U_ref ((j+1/2)/ny)^(1/7); kind 1: U = U_ref 4 eta (1 - eta); kind 2: U = 0. */
void orc_init_field(const orc_t *o, int kind, double U_ref, double noise_frac, uint64_t seed,
                    double *rho, double *u)
{
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y) {
            double eta = (y + 0.5) / o->ny, U = 0.0;
            if (kind == 0) U = U_ref * pow(eta, 1.0 / 7.0);
            else if (kind == 1) U = U_ref * 4.0 * eta * (1.0 - eta);
            for (int x = 0; x < o->nx; ++x) {
                long long n = x + (long long)o->nx * (y + (long long)o->ny * z);
                rho[n] = 1.0;
                for (int a = 0; a < 3; ++a) {
                    double r = orc_rand01(seed, 3ULL * (uint64_t)n + (uint64_t)a);
                    u[a * o->N + n] = (a == 0 ? U : 0.0) + noise_frac * U_ref * (2.0 * r - 1.0);
                }
            }
        }
}

void orc_stats_reset(orc_t *o);

void orc_init(orc_t *o, int kind, double U_ref, double noise_frac, uint64_t seed)
{
    double *rho = (double *)malloc(sizeof(double) * o->N);
    double *u = (double *)malloc(sizeof(double) * 3 * o->N);
    orc_init_field(o, kind, U_ref, noise_frac, seed, rho, u);
    orc_set_macros(o, rho, u);
    free(rho); free(u);
    orc_stats_reset(o);
}

void orc_get_populations(const orc_t *o, double *f) { memcpy(f, o->fa, sizeof(double) * Q * o->N); }
void orc_set_populations(orc_t *o, const double *f) { memcpy(o->fa, f, sizeof(double) * Q * o->N); }

/* ---------------------------------------------------------------------------------------- */
/* O2: stream (pull) with boundary links                                                     */
/* ---------------------------------------------------------------------------------------- */

/* Incoming populations f_i(x) of one cell from the post-collision state fa.
 * Eq. 1 LHS, Alg. 1 "Stream" (L150); periodic x,z (L177, L216); halfway
 * bounce-back at wall faces (readings R11, R12); specular reflection at a free-slip top (R13). */
static void stream_cell(const orc_t *o, int x, int y, int z, double *f)
{
    const int nx = o->nx, ny = o->ny, nz = o->nz;
    const long long N = o->N;
    const unsigned bot = o->bc & ORC_BOTTOM_MASK, top = (o->bc >> ORC_TOP_SHIFT) & 3u;
    const long long cell = x + (long long)nx * (y + (long long)ny * z);
    for (int i = 0; i < Q; ++i) {
        int xs = (x - C[i][0] + nx) % nx;
        int zs = (z - C[i][2] + nz) % nz;
        int ys = y - C[i][1];
        if (ys < 0) {
            if (bot == 1) ys = ny - 1;                      /* periodic-y */
            else { f[i] = o->fa[OPP[i] * N + cell]; continue; } /* wall: f_i <- f*_opp(i), same cell */
        } else if (ys >= ny) {
            if (top == 2) ys = 0;                           /* periodic-y */
            else if (top == 1) {                            /* free-slip: f_i <- f*_m(i)(x-cx, y, z-cz) */
                long long s = xs + (long long)nx * (y + (long long)ny * zs);
                if (o->solid && o->solid[s]) f[i] = o->fa[OPP[i] * N + cell];
                else f[i] = o->fa[MIR[i] * N + s];
                continue;
            } else if (top == 3) {                          /* forced equilibrium lid */
                double feq[Q];
                orc_feq(1.0, o->Utop, feq);
                f[i] = feq[i];
                continue;
            } else { f[i] = o->fa[OPP[i] * N + cell]; continue; }
        }
        long long s = xs + (long long)nx * (ys + (long long)ny * zs);
        if (o->solid && o->solid[s]) f[i] = o->fa[OPP[i] * N + cell]; /* bounce-back off a solid cell */
        else f[i] = o->fa[i * N + s];
    }
}

/* O3-O5: moments, predictor velocity, forest drag, corrected velocity, total force. */
static void macros_cell(const orc_t *o, long long cell, int y, const double *f, double *rho_out, double *u,
                        double *F, double *Pi /* [xx,yy,zz,xy,yz,xz] or NULL */)
{
    double rho = 0.0, m[3] = {0, 0, 0};
    for (int i = 0; i < Q; ++i) {                           /* Eqs. 5, 6 */
        rho += f[i];
        for (int a = 0; a < 3; ++a) m[a] += f[i] * C[i][a];
    }
    if (Pi) {                                               /* Eq. 7 */
        for (int k = 0; k < 6; ++k) Pi[k] = 0.0;
        for (int i = 0; i < Q; ++i) {
            Pi[0] += f[i] * C[i][0] * C[i][0]; Pi[1] += f[i] * C[i][1] * C[i][1];
            Pi[2] += f[i] * C[i][2] * C[i][2]; Pi[3] += f[i] * C[i][0] * C[i][1];
            Pi[4] += f[i] * C[i][1] * C[i][2]; Pi[5] += f[i] * C[i][0] * C[i][2];
        }
    }
    /* Alg. 1: local velocity with the driving body force, Eq. 6 (reading R7) */
    double us[3];
    for (int a = 0; a < 3; ++a) us[a] = (m[a] + 0.5 * o->Fb[a]) / rho;
    double Ff[3] = {0, 0, 0};
    double a_j = o->lad[y];
    /* Alg. 1 "if forest cell": a coded cell takes its LAD from its own code (L129-135) */
    if (o->fcode && o->fcode[cell]) a_j = orc_forest_code_lad(o->fcode[cell], o->a_fm);
    if (a_j > 0.0) {
        /* Alg. 1, Eq. 13: F_f = -C_D a_f(y) |u| u, no rho factor (R4);
         * streamwise component only (R5) unless the vector form is flagged. */
        double mag = sqrt(us[0] * us[0] + us[1] * us[1] + us[2] * us[2]);
        Ff[0] = -o->Cd * a_j * mag * us[0];
        if (o->bc & ORC_DRAG_VECTOR) {
            Ff[1] = -o->Cd * a_j * mag * us[1];
            Ff[2] = -o->Cd * a_j * mag * us[2];
        }
    }
    /* Alg. 1: correct the velocity with the forest force (explicit, one pass; R6) */
    for (int a = 0; a < 3; ++a) {
        u[a] = us[a] + 0.5 * Ff[a] / rho;
        F[a] = o->Fb[a] + Ff[a];
    }
    *rho_out = rho;
}

/* O7-O9: Smagorinsky relaxation time and forced BGK collision of one cell. */
static void collide_cell(const orc_t *o, int y, double rho, const double *u, const double *F,
                         const double *Pi, const double *f, double *fstar)
{
    /* Pi_neq = Pi - Pi_eq, Pi_eq = rho cs2 I + rho u u (reading R8) */
    double Pneq[6];
    Pneq[0] = Pi[0] - (rho / 3.0 + rho * u[0] * u[0]);
    Pneq[1] = Pi[1] - (rho / 3.0 + rho * u[1] * u[1]);
    Pneq[2] = Pi[2] - (rho / 3.0 + rho * u[2] * u[2]);
    Pneq[3] = Pi[3] - rho * u[0] * u[1];
    Pneq[4] = Pi[4] - rho * u[1] * u[2];
    Pneq[5] = Pi[5] - rho * u[0] * u[2];
    double tau;
    if (o->sgs_C || o->sgs_Sbar)                                 /* other SGS models (L307) */
        tau = orc_tau_total_rows(o->tau0, o->sgs_C ? o->sgs_C[y] : o->Csmag, o->sgs_Sbar ? o->sgs_Sbar[y] : 0.0, rho, Pneq);
    else
        tau = orc_tau_total(o->tau0, o->Csmag, rho, Pneq);       /* Eq. 12 */
    double feq[Q], Fi[Q];
    orc_feq(rho, u, feq);                                        /* Eq. 3 */
    orc_guo(tau, u, F, Fi);                                      /* Eq. 4 with tau_total (R10) */
    /* Eq. 1 with Eq. 2 relaxing TOWARDS equilibrium (reading R1) */
    for (int i = 0; i < Q; ++i) fstar[i] = f[i] - (f[i] - feq[i]) / tau + Fi[i];
}

/* Streamed (pre-collision) populations of every cell, no collision: used by the streaming pins. */
void orc_stream_only(const orc_t *o, double *fout /*[Q][N]*/)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                long long cell = x + (long long)o->nx * (y + (long long)o->ny * z);
                double f[Q];
                if (o->solid && o->solid[cell]) { for (int i = 0; i < Q; ++i) f[i] = o->fa[i * o->N + cell]; }
                else stream_cell(o, x, y, z, f);
                for (int i = 0; i < Q; ++i) fout[i * o->N + cell] = f[i];
            }
}

/* O6: sample S_k = (rho, u) = stream(state k) -> O3-O5; state unchanged (reading R19). */
void orc_get_macros(const orc_t *o, double *rho /*[N]*/, double *u /*[3][N]*/)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y)
            for (int x = 0; x < o->nx; ++x) {
                long long cell = x + (long long)o->nx * (y + (long long)o->ny * z);
                double f[Q], r, uu[3], F[3];
                if (o->solid && o->solid[cell]) { rho[cell] = 1.0; u[cell] = u[o->N + cell] = u[2 * o->N + cell] = 0.0; continue; }
                stream_cell(o, x, y, z, f);
                macros_cell(o, cell, y, f, &r, uu, F, NULL);
                rho[cell] = r;
                u[cell] = uu[0]; u[o->N + cell] = uu[1]; u[2 * o->N + cell] = uu[2];
            }
}

void orc_stats_accumulate(orc_t *o, int every) { o->stats_every = every; o->stats_phase = 0; }
void orc_stats_reset(orc_t *o)
{
    memset(o->acc, 0, sizeof(double) * o->ny * NSTAT);
    o->nsamples = 0; o->stats_phase = 0;
}

/* One time step: Algorithm 1's loop body over all cells. */
static void step_once(orc_t *o)
{
    const int sample = (o->stats_every > 0) && (o->stats_phase % o->stats_every == 0);
#pragma omp parallel for collapse(2) schedule(static)
    for (int z = 0; z < o->nz; ++z)
        for (int y = 0; y < o->ny; ++y) {
            double rs[NSTAT] = {0};
            for (int x = 0; x < o->nx; ++x) {
                long long cell = x + (long long)o->nx * (y + (long long)o->ny * z);
                double f[Q], fstar[Q], rho, u[3], F[3], Pi[6];
                if (o->solid && o->solid[cell]) {
                    for (int i = 0; i < Q; ++i) o->fb[i * o->N + cell] = o->fa[i * o->N + cell];
                    continue;
                }
                stream_cell(o, x, y, z, f);              /* Stream */
                macros_cell(o, cell, y, f, &rho, u, F, Pi);    /* u, F_f, corrected u */
                if (sample) {                            /* O10: time + x-z plane averaging (L200, L251) */
                    rs[0] += u[0]; rs[1] += u[1]; rs[2] += u[2];
                    rs[3] += u[0] * u[0]; rs[4] += u[1] * u[1]; rs[5] += u[2] * u[2];
                    rs[6] += u[0] * u[1]; rs[7] += u[1] * u[2]; rs[8] += u[0] * u[2];
                    rs[9] += rho;
                }
                collide_cell(o, y, rho, u, F, Pi, f, fstar); /* Collide with the body force */
                for (int i = 0; i < Q; ++i) o->fb[i * o->N + cell] = fstar[i];
            }
            if (sample)
                for (int k = 0; k < NSTAT; ++k) o->rowsum[((long long)z * o->ny + y) * NSTAT + k] = rs[k];
        }
    if (sample) {
        for (int z = 0; z < o->nz; ++z)
            for (int y = 0; y < o->ny; ++y)
                for (int k = 0; k < NSTAT; ++k)
                    o->acc[y * NSTAT + k] += o->rowsum[((long long)z * o->ny + y) * NSTAT + k];
        o->nsamples++;
    }
    if (o->stats_every > 0) o->stats_phase++;
    double *tmp = o->fa; o->fa = o->fb; o->fb = tmp;
    o->t++;
}

void orc_step(orc_t *o, int n) { for (int k = 0; k < n; ++k) step_once(o); }

/* Read-out: <a>_j = sum a / (nsamples nx nz); <a'b'>_j = <ab>_j - <a>_j <b>_j.
 * Columns: <u>,<v>,<w>,<u'u'>,<v'v'>,<w'w'>,<u'v'>,<v'w'>,<u'w'>,<rho>. */
long long orc_stats_read(const orc_t *o, double *out /*[ny][10]*/)
{
    double cnt = (double)o->nsamples * o->nx * o->nz;
    for (int y = 0; y < o->ny; ++y) {
        const double *a = o->acc + y * NSTAT;
        double *r = out + y * NSTAT;
        if (o->nsamples == 0) { for (int k = 0; k < NSTAT; ++k) r[k] = 0.0; continue; }
        double mu = a[0] / cnt, mv = a[1] / cnt, mw = a[2] / cnt;
        r[0] = mu; r[1] = mv; r[2] = mw;
        r[3] = a[3] / cnt - mu * mu; r[4] = a[4] / cnt - mv * mv; r[5] = a[5] / cnt - mw * mw;
        r[6] = a[6] / cnt - mu * mv; r[7] = a[7] / cnt - mv * mw; r[8] = a[8] / cnt - mu * mw;
        r[9] = a[9] / cnt;
    }
    return o->nsamples;
}

/* raw sums, for pins that want them */
void orc_stats_raw(const orc_t *o, double *acc /*[ny][10]*/) { memcpy(acc, o->acc, sizeof(double) * o->ny * NSTAT); }

long long orc_time(const orc_t *o) { return o->t; }
double orc_tau0(const orc_t *o) { return o->tau0; }
