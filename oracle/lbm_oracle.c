/*
 * lbm_oracle.c -- plain, slow, obviously-correct CPU lattice Boltzmann reference.
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the parity oracle for the CUDA library in
 * paper_1311_2404_b200/.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code,
 * headers, tables or helpers with the CUDA path and must never be reachable from the
 * product path.
 *
 * What it computes: the explicit lattice Boltzmann iteration of arXiv 1311.2404 (Sailfish),
 * step by step in the paper's order, in fp64, with two full copies of the lattice
 * (collide into f*, then stream into f), no fusion, no blocking, no vectorisation.
 * P:<n> cites line n of /root/reference/PAPER.md.
 *
 *   state      f_i(x,t) = pre-collision, post-streaming populations (what Alg. 1 line 4
 *              loads); SOLID nodes keep their initial values for ever.
 *   moments    rho = sum_i f_i, rho u = sum_i f_i e_i                     P:85  eq. (1)
 *   forcing    rho v = sum_i e_i f_i + F/2, F = rho g (acceleration g)    P:247 eq. (16)
 *   f^eq       rho w_i (1 + 3 e.v + 9/2 (e.v)^2 - 3/2 v^2)                P:111 eq. (3)
 *   weights    D2Q9 4/9 1/9 1/36 ; D3Q19 1/3 1/18 1/36                    P:96-105 Table 1
 *   LBGK       f* = f + (f^eq - f)/tau                                    P:371 Alg. 1 l.13
 *              (eq. (2) as printed at P:89 has the opposite sign; Alg. 1 is the form that
 *              relaxes towards equilibrium -- DESIGN.md reading A1)
 *   MRT        f* = f + M^-1 S (M f^eq - M f), S diagonal                 P:140 eq. (4)
 *              (M "see d'Humieres [11]": defined below by polynomials of e_i,
 *              DESIGN.md reading A5; m^eq = M f^eq, reading A6)
 *   Guo term   f* += (1 - 1/(2 tau)) w_i [3 (e_i - v) + 9 (e_i.v) e_i].F  P:251 eq. (17)
 *              (c_s^2 = 1/3).  MRT: M^-1 (I - S/2) M applied to the bracket (A16).
 *   streaming  f_i(x,t+1) = f*_i(x - e_i), periodic on every axis          P:89 eq. (2) lhs
 *   bounce-back if x - e_i is SOLID: f_i(x,t+1) = f*_ibar(x), e_ibar = -e_i  P:237 (half-way,
 *              reflected in the same step; reading A8)
 *   Shan-Chen  F_A(x) = -G psi(rho_A(x)) sum_i w_i psi(rho_B(x+e_i)) e_i   P:183 eq. (10),
 *              sign per DESIGN.md reading A11; common velocity
 *              u' = (j_A/tau_A + j_B/tau_B)/(rho_A/tau_A + rho_B/tau_B)    P:188;
 *              v_s = u' + F_s/(2 rho_s), then f^eq / LBGK / Guo per component (A13);
 *              macro fields are computed for all nodes first
 *   full-way BB  wall node (dry): f* = f reversed, no relaxation; back in the fluid at t+2     P:237 Fig. 2 (1), A20
 *   velocity BC  f* = f^eq(rho, u_bc), rho from the node's own populations, missing ones
 *              are bounce-back copies (the half-way rule behind a SOLID node)              P:239, A21
 *   EDM        F_i = f^eq(rho, u + F/rho) - f^eq(rho, u), any collision operator          P:253-258 eq. (18), A22
 *   regularized f^neq -> w_i/(2 c_s^4)(e e - c_s^2 delta):Pi^neq, then LBGK               P:130, A23
 *   Smagorinsky tau = tau_0 + (sqrt(tau_0^2 + 4 c_s^-4 C_S^2 |Q|) - tau_0)/2                P:164-173 eq. (8)-(9), A23
 *   init       f_i(x,0) = f^eq_i(rho0(x), u0(x))
 *   macro      rho = sum f_i, velocity v of eq. (16)
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): Table 1 weights and isotropy, exact
 * equilibrium moments, collision fixed point, mass conservation, uniform-force closed form,
 * Poiseuille parabola + second-order convergence, Taylor-Green decay rate, MRT == LBGK for
 * equal rates, MRT matrix orthogonality and d'Humieres' closed-form equilibrium moments,
 * MRT shear-wave viscosity, brute-force stream map on tiny lattices, Shan-Chen conservation
 * laws / G = 0 / linear-gradient force, full-way wall (hand-tracked arrow, steady Poiseuille equals
 * the half-way profile), velocity node (uniform-flow fixed point, Couette flow), and one step with
 * all four node types against an independent whole-array numpy implementation.
 * Round 2 (tests/test_oracle_pins_r2.py): Smagorinsky shear-wave decay predicted from eq. (9);
 * Smagorinsky + Guo with C_S > 0 (exact momentum balance, numpy step); MRT + Guo with unequal rates
 * (one collision in physical moments: trace / deviator / heat flux with their own rates and
 * (1 - s_k/2) source prefactors; numpy step with np.linalg.inv; Poiseuille curvature); Shan-Chen
 * with non-FLUID nodes (closed-form force beside a dry plane, numpy step with all node types,
 * per-component mass with SOLID + WALL_FULLWAY nodes).
 * PARITY UNPINNED (no printed value in the paper): the physical sign of the
 * Shan-Chen coupling (reading A11) and the c3 rate s_m = 1.98 (a parameter, not arithmetic).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { ORC_D2Q9 = 0, ORC_D3Q19 = 1 };
enum { ORC_BGK = 0, ORC_MRT = 1, ORC_SC2 = 2, ORC_REG = 3, ORC_LES = 4 };
enum { ORC_PSI_RHO = 0, ORC_PSI_1MEXP = 1 };
#define ORC_QMAX 19
/* node types (P:446 reduced; readings A8, A20, A21) */
enum { ORC_FORCE_GUO = 0, ORC_FORCE_EDM = 1 };
enum { ORC_FLUID = 0, ORC_SOLID = 1, ORC_WALL_FULLWAY = 2, ORC_VELOCITY = 3 };

typedef struct {
    int32_t lattice, model;
    int32_t nx, ny, nz;
    double tau[2];
    double rates[ORC_QMAX];
    double force[3]; /* body acceleration g; F = rho g */
    double sc_G;
    int32_t sc_psi;
    double bc_velocity[3]; /* velocity imposed on ORC_VELOCITY nodes (reading A21) */
    int32_t force_scheme;  /* ORC_FORCE_GUO (eq. 17) | ORC_FORCE_EDM (eq. 18) */
    double smagorinsky_cs; /* C_S of eq. (9), ORC_LES only */
} orc_params;

/* ---- velocity sets (reading A2; weights from Table 1) ------------- */
static const int E_D2Q9[9][3] = {
    {0, 0, 0}, {1, 0, 0}, {0, 1, 0}, {-1, 0, 0}, {0, -1, 0},
    {1, 1, 0}, {-1, 1, 0}, {-1, -1, 0}, {1, -1, 0}};
static const int E_D3Q19[19][3] = {
    {0, 0, 0},
    {1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0}, {0, 0, 1}, {0, 0, -1},
    {1, 1, 0}, {-1, 1, 0}, {1, -1, 0}, {-1, -1, 0},
    {1, 0, 1}, {-1, 0, 1}, {1, 0, -1}, {-1, 0, -1},
    {0, 1, 1}, {0, -1, 1}, {0, 1, -1}, {0, -1, -1}};

typedef struct {
    int Q, D;
    int e[ORC_QMAX][3];
    double w[ORC_QMAX];
    int opp[ORC_QMAX];
} lattice_t;

static int lattice_fill(int lattice, lattice_t *L)
{
    memset(L, 0, sizeof *L);
    if (lattice == ORC_D2Q9) {
        L->Q = 9; L->D = 2;
        for (int i = 0; i < 9; i++) for (int a = 0; a < 3; a++) L->e[i][a] = E_D2Q9[i][a];
    } else if (lattice == ORC_D3Q19) {
        L->Q = 19; L->D = 3;
        for (int i = 0; i < 19; i++) for (int a = 0; a < 3; a++) L->e[i][a] = E_D3Q19[i][a];
    } else {
        return -1;
    }
    for (int i = 0; i < L->Q; i++) {
        int n2 = L->e[i][0] * L->e[i][0] + L->e[i][1] * L->e[i][1] + L->e[i][2] * L->e[i][2];
        /* Table 1: weight by link length 0, 1, sqrt 2 */
        if (lattice == ORC_D2Q9) L->w[i] = (n2 == 0) ? 4.0 / 9.0 : (n2 == 1) ? 1.0 / 9.0 : 1.0 / 36.0;
        else                     L->w[i] = (n2 == 0) ? 1.0 / 3.0 : (n2 == 1) ? 1.0 / 18.0 : 1.0 / 36.0;
        L->opp[i] = -1;
        for (int k = 0; k < L->Q; k++)
            if (L->e[k][0] == -L->e[i][0] && L->e[k][1] == -L->e[i][1] && L->e[k][2] == -L->e[i][2])
                L->opp[i] = k;
    }
    return 0;
}

/* ---- equilibrium, eq. (3) P:111 ------------------------------------------------------- */
static void feq(const lattice_t *L, double rho, const double v[3], double *out)
{
    double vv = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    for (int i = 0; i < L->Q; i++) {
        double ev = L->e[i][0] * v[0] + L->e[i][1] * v[1] + L->e[i][2] * v[2];
        out[i] = rho * L->w[i] * (1.0 + 3.0 * ev + 4.5 * ev * ev - 1.5 * vv);
    }
}

/* ---- MRT moment matrix, reading A5 (rows are polynomials of e_i) ------------ */
static void mrt_matrix(const lattice_t *L, int lattice, double *M /* Q x Q, row-major */)
{
    for (int i = 0; i < L->Q; i++) {
        double x = L->e[i][0], y = L->e[i][1], z = L->e[i][2];
        double n2 = x * x + y * y + z * z, n4 = n2 * n2;
        double r[ORC_QMAX];
        if (lattice == ORC_D2Q9) {
            r[0] = 1.0;
            r[1] = -4.0 + 3.0 * n2;
            r[2] = 4.0 - 10.5 * n2 + 4.5 * n4;
            r[3] = x;
            r[4] = (-5.0 + 3.0 * n2) * x;
            r[5] = y;
            r[6] = (-5.0 + 3.0 * n2) * y;
            r[7] = x * x - y * y;
            r[8] = x * y;
        } else {
            r[0] = 1.0;
            r[1] = 19.0 * n2 - 30.0;
            r[2] = (21.0 * n4 - 53.0 * n2 + 24.0) / 2.0;
            r[3] = x;
            r[4] = (5.0 * n2 - 9.0) * x;
            r[5] = y;
            r[6] = (5.0 * n2 - 9.0) * y;
            r[7] = z;
            r[8] = (5.0 * n2 - 9.0) * z;
            r[9] = 3.0 * x * x - n2;
            r[10] = (3.0 * n2 - 5.0) * (3.0 * x * x - n2);
            r[11] = y * y - z * z;
            r[12] = (3.0 * n2 - 5.0) * (y * y - z * z);
            r[13] = x * y;
            r[14] = y * z;
            r[15] = x * z;
            r[16] = (y * y - z * z) * x;
            r[17] = (z * z - x * x) * y;
            r[18] = (x * x - y * y) * z;
        }
        for (int k = 0; k < L->Q; k++) M[k * L->Q + i] = r[k];
    }
}

/* general inverse by Gauss-Jordan with partial pivoting (no use of row orthogonality) */
static int mat_inverse(int n, const double *A, double *Ainv)
{
    double a[ORC_QMAX][2 * ORC_QMAX];
    for (int r = 0; r < n; r++)
        for (int c = 0; c < n; c++) { a[r][c] = A[r * n + c]; a[r][n + c] = (r == c) ? 1.0 : 0.0; }
    for (int c = 0; c < n; c++) {
        int p = c;
        for (int r = c + 1; r < n; r++) if (fabs(a[r][c]) > fabs(a[p][c])) p = r;
        if (fabs(a[p][c]) < 1e-14) return -1;
        if (p != c) for (int k = 0; k < 2 * n; k++) { double t = a[c][k]; a[c][k] = a[p][k]; a[p][k] = t; }
        double d = a[c][c];
        for (int k = 0; k < 2 * n; k++) a[c][k] /= d;
        for (int r = 0; r < n; r++) {
            if (r == c) continue;
            double m = a[r][c];
            if (m != 0.0) for (int k = 0; k < 2 * n; k++) a[r][k] -= m * a[c][k];
        }
    }
    for (int r = 0; r < n; r++) for (int c = 0; c < n; c++) Ainv[r * n + c] = a[r][n + c];
    return 0;
}

/* ---- context --------------------------------------------------------------------------- */
typedef struct {
    orc_params p;
    lattice_t L;
    int64_t N;
    int ncomp;
    uint8_t *mask;        /* N, node type ORC_FLUID / SOLID / WALL_FULLWAY / VELOCITY */
    double *f[2];         /* per component: Q*N, canonical pre-collision state */
    double *fs[2];        /* per component: Q*N, post-collision f*            */
    double *rho[2];       /* Shan-Chen: per-component density field           */
    double *mom[2];       /* Shan-Chen: per-component momentum field, 3*N     */
    double M[ORC_QMAX * ORC_QMAX], Minv[ORC_QMAX * ORC_QMAX];
} orc_ctx;

static int64_t node_index(const orc_ctx *c, int x, int y, int z)
{
    return ((int64_t)z * c->p.ny + y) * c->p.nx + x;
}
static int wrap(int a, int n) { return ((a % n) + n) % n; }

static double psi_of(int kind, double rho)
{
    return (kind == ORC_PSI_1MEXP) ? 1.0 - exp(-rho) : rho;
}

/* ---- exported helpers used by the pins -------------------------------------------------- */
int orc_lattice_Q(int lattice) { lattice_t L; return lattice_fill(lattice, &L) ? -1 : L.Q; }
int orc_lattice_D(int lattice) { lattice_t L; return lattice_fill(lattice, &L) ? -1 : L.D; }
int orc_lattice_tables(int lattice, int32_t *e /* Q*3 */, double *w, int32_t *opp)
{
    lattice_t L;
    if (lattice_fill(lattice, &L)) return -1;
    for (int i = 0; i < L.Q; i++) {
        for (int a = 0; a < 3; a++) e[i * 3 + a] = L.e[i][a];
        w[i] = L.w[i];
        opp[i] = L.opp[i];
    }
    return 0;
}
int orc_feq(int lattice, double rho, const double *v3, double *out)
{
    lattice_t L;
    if (lattice_fill(lattice, &L)) return -1;
    feq(&L, rho, v3, out);
    return 0;
}
int orc_mrt_matrix(int lattice, double *M, double *Minv)
{
    lattice_t L;
    if (lattice_fill(lattice, &L)) return -1;
    mrt_matrix(&L, lattice, M);
    return mat_inverse(L.Q, M, Minv);
}
int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- life cycle -------------------------------------------------------------------------- */
void orc_destroy(orc_ctx *c)
{
    if (!c) return;
    free(c->mask);
    for (int s = 0; s < 2; s++) { free(c->f[s]); free(c->fs[s]); free(c->rho[s]); free(c->mom[s]); }
    free(c);
}

orc_ctx *orc_create(const orc_params *p)
{
    orc_ctx *c = (orc_ctx *)calloc(1, sizeof *c);
    if (!c) return NULL;
    c->p = *p;
    if (lattice_fill(p->lattice, &c->L) || p->nx < 1 || p->ny < 1 || p->nz < 1 ||
        (p->lattice == ORC_D2Q9 && p->nz != 1) || p->model < ORC_BGK || p->model > ORC_LES ||
        (p->model == ORC_REG && p->force_scheme == ORC_FORCE_GUO &&
         (p->force[0] != 0 || p->force[1] != 0 || p->force[2] != 0))) { /* reading A23 */
        free(c);
        return NULL;
    }
    c->N = (int64_t)p->nx * p->ny * p->nz;
    c->ncomp = (p->model == ORC_SC2) ? 2 : 1;
    c->mask = (uint8_t *)calloc((size_t)c->N, 1);
    int ok = c->mask != NULL;
    for (int s = 0; s < c->ncomp && ok; s++) {
        c->f[s] = (double *)calloc((size_t)(c->N * c->L.Q), sizeof(double));
        c->fs[s] = (double *)calloc((size_t)(c->N * c->L.Q), sizeof(double));
        ok = c->f[s] && c->fs[s];
        if (p->model == ORC_SC2 && ok) {
            c->rho[s] = (double *)calloc((size_t)c->N, sizeof(double));
            c->mom[s] = (double *)calloc((size_t)(3 * c->N), sizeof(double));
            ok = c->rho[s] && c->mom[s];
        }
    }
    if (ok && p->model == ORC_MRT) {
        mrt_matrix(&c->L, p->lattice, c->M);
        ok = mat_inverse(c->L.Q, c->M, c->Minv) == 0;
    }
    if (!ok) { orc_destroy(c); return NULL; }
    return c;
}

int orc_set_geometry(orc_ctx *c, const uint8_t *mask)
{
    /* 0, 2, 3 as named; every other value is a dry SOLID node */
    for (int64_t n = 0; n < c->N; n++)
        c->mask[n] = (mask[n] == ORC_FLUID || mask[n] == ORC_WALL_FULLWAY || mask[n] == ORC_VELOCITY) ? mask[n] : ORC_SOLID;
    return 0;
}

/* f_i(x,0) = f^eq_i(rho0, u0), u0 used as given (reading A15).
 * rho: N, u: D*N component planes. */
int orc_init_equilibrium(orc_ctx *c, int comp, const double *rho, const double *u)
{
    if (comp < 0 || comp >= c->ncomp) return -1;
    const int Q = c->L.Q, D = c->L.D;
    for (int64_t n = 0; n < c->N; n++) {
        double v[3] = {0, 0, 0}, fe[ORC_QMAX];
        for (int a = 0; a < D; a++) v[a] = u[a * c->N + n];
        feq(&c->L, rho[n], v, fe);
        for (int i = 0; i < Q; i++) c->f[comp][i * c->N + n] = fe[i];
    }
    return 0;
}

int orc_set_distributions(orc_ctx *c, int comp, const double *f)
{
    if (comp < 0 || comp >= c->ncomp) return -1;
    memcpy(c->f[comp], f, sizeof(double) * (size_t)(c->N * c->L.Q));
    return 0;
}
int orc_get_distributions(const orc_ctx *c, int comp, double *f)
{
    if (comp < 0 || comp >= c->ncomp) return -1;
    memcpy(f, c->f[comp], sizeof(double) * (size_t)(c->N * c->L.Q));
    return 0;
}

/* Streaming map, reading A8: map[i*N + x] = slot (i'*N + x') whose post-collision
 * value becomes f_i(x,t+1): (i, x - e_i) if that node is FLUID, else (ibar, x); -1 on SOLID x. */
int orc_stream_map(const orc_ctx *c, int64_t *map)
{
    const int nx = c->p.nx, ny = c->p.ny, nz = c->p.nz, Q = c->L.Q;
    for (int z = 0; z < nz; z++)
        for (int y = 0; y < ny; y++)
            for (int x = 0; x < nx; x++) {
                int64_t n = node_index(c, x, y, z);
                for (int i = 0; i < Q; i++) {
                    if (c->mask[n] == ORC_SOLID) { map[i * c->N + n] = -1; continue; }
                    int64_t m = node_index(c, wrap(x - c->L.e[i][0], nx), wrap(y - c->L.e[i][1], ny),
                                           wrap(z - c->L.e[i][2], nz));
                    map[i * c->N + n] = c->mask[m] == ORC_SOLID ? (int64_t)c->L.opp[i] * c->N + n : (int64_t)i * c->N + m;
                }
            }
    return 0;
}

/* ---- one collision at one node ------------------------------------------------------------
 * in:  f (Q values), rho, v (velocity entering f^eq and the source), F (force density), tau
 * out: fstar */
static void collide_node(const orc_ctx *c, const double *f, double rho, const double v[3],
                         const double ub[3], const double F[3], double tau, double *fstar)
{
    const lattice_t *L = &c->L;
    const int Q = L->Q;
    double fe[ORC_QMAX], src[ORC_QMAX];
    double freg_store[ORC_QMAX];
    if (c->p.model == ORC_REG) {
        /* Regularized LBGK, P:130 (reading A23): replace f^neq = f - f^eq by its projection
         * f^reg_i = w_i / (2 c_s^4) (e_ia e_ib - c_s^2 delta_ab) Pi^neq_ab,
         * Pi^neq_ab = sum_i f^neq_i (e_ia e_ib - c_s^2 delta_ab), c_s^2 = 1/3; then collide as LBGK.
         * The equilibrium is taken at the bare velocity (a force enters through the EDM only). */
        double Pi[3][3] = {{0}};
        feq(L, rho, ub, fe);
        for (int i = 0; i < Q; i++)
            for (int a = 0; a < 3; a++)
                for (int b = 0; b < 3; b++)
                    Pi[a][b] += (f[i] - fe[i]) * (L->e[i][a] * L->e[i][b] - (a == b ? 1.0 / 3.0 : 0.0));
        for (int i = 0; i < Q; i++) {
            double s = 0;
            for (int a = 0; a < 3; a++)
                for (int b = 0; b < 3; b++) s += (L->e[i][a] * L->e[i][b] - (a == b ? 1.0 / 3.0 : 0.0)) * Pi[a][b];
            freg_store[i] = fe[i] + 4.5 * L->w[i] * s;
        }
        f = freg_store; /* "after this regularization step, the collision ... proceeds as in LBGK" */
    }
    if (c->p.model == ORC_LES) {
        /* Smagorinsky subgrid model, eq. (8)-(9) P:164-173: tau = tau_0 + tau_t,
         * tau_t = ( sqrt(tau_0^2 + 4 c_s^-4 C_S^2 |Q|) - tau_0 ) / 2, Q_ab = sum_i e_ia e_ib (f_i - f^eq_i),
         * |Q| = (Q_ab Q_ab)^(1/2); f^eq at the velocity the collision uses (Guo: v, EDM: u). */
        double Qt[3][3] = {{0}}, q2 = 0;
        feq(L, rho, c->p.force_scheme == ORC_FORCE_EDM ? ub : v, fe);
        for (int i = 0; i < Q; i++)
            for (int a = 0; a < 3; a++)
                for (int b = 0; b < 3; b++) Qt[a][b] += L->e[i][a] * L->e[i][b] * (f[i] - fe[i]);
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++) q2 += Qt[a][b] * Qt[a][b];
        double cs = c->p.smagorinsky_cs;
        tau = tau + 0.5 * (sqrt(tau * tau + 4.0 * 9.0 * cs * cs * sqrt(q2)) - tau);
    }
    if (c->p.force_scheme == ORC_FORCE_EDM) {
        /* Exact Difference Method, eq. (18) P:253-258 (reading A22): relax towards f^eq(rho, u) at
         * the bare velocity u = ub (sum e f / rho; the common velocity u' for Shan-Chen) and add
         * F_i = f^eq(rho, u + F/rho) - f^eq(rho, u), unscaled, for any collision operator. */
        double u2[3], fe2[ORC_QMAX];
        for (int a = 0; a < 3; a++) u2[a] = ub[a] + F[a] / rho;
        feq(L, rho, ub, fe);
        feq(L, rho, u2, fe2);
        if (c->p.model == ORC_MRT) {
            double m[ORC_QMAX], me[ORC_QMAX], d[ORC_QMAX];
            for (int k = 0; k < Q; k++) {
                double a = 0, b = 0;
                for (int i = 0; i < Q; i++) { a += c->M[k * Q + i] * f[i]; b += c->M[k * Q + i] * fe[i]; }
                m[k] = a; me[k] = b;
            }
            for (int k = 0; k < Q; k++) d[k] = c->p.rates[k] * (me[k] - m[k]);
            for (int i = 0; i < Q; i++) {
                double a = 0;
                for (int k = 0; k < Q; k++) a += c->Minv[i * Q + k] * d[k];
                fstar[i] = f[i] + a + (fe2[i] - fe[i]);
            }
        } else {
            for (int i = 0; i < Q; i++) fstar[i] = f[i] + (fe[i] - f[i]) / tau + (fe2[i] - fe[i]);
        }
        return;
    }
    feq(L, rho, v, fe); /* eq. (3) */
    /* bracket of eq. (17): w_i [3 (e_i - v) + 9 (e_i.v) e_i] . F */
    for (int i = 0; i < Q; i++) {
        double ev = L->e[i][0] * v[0] + L->e[i][1] * v[1] + L->e[i][2] * v[2];
        double s = 0.0;
        for (int a = 0; a < 3; a++) s += (3.0 * (L->e[i][a] - v[a]) + 9.0 * ev * L->e[i][a]) * F[a];
        src[i] = L->w[i] * s;
    }
    if (c->p.model == ORC_MRT) {
        /* eq. (4): f* = f + M^-1 S (M f^eq - M f); source M^-1 (I - S/2) M src (A16) */
        double m[ORC_QMAX], me[ORC_QMAX], ms[ORC_QMAX], d[ORC_QMAX];
        for (int k = 0; k < Q; k++) {
            double a = 0, b = 0, s = 0;
            for (int i = 0; i < Q; i++) {
                a += c->M[k * Q + i] * f[i];
                b += c->M[k * Q + i] * fe[i];
                s += c->M[k * Q + i] * src[i];
            }
            m[k] = a; me[k] = b; ms[k] = s;
        }
        for (int k = 0; k < Q; k++) d[k] = c->p.rates[k] * (me[k] - m[k]) + (1.0 - 0.5 * c->p.rates[k]) * ms[k];
        for (int i = 0; i < Q; i++) {
            double a = 0;
            for (int k = 0; k < Q; k++) a += c->Minv[i * Q + k] * d[k];
            fstar[i] = f[i] + a;
        }
    } else {
        for (int i = 0; i < Q; i++) {
            fstar[i] = f[i] + (fe[i] - f[i]) / tau;          /* Alg. 1 l.13 */
            fstar[i] += (1.0 - 1.0 / (2.0 * tau)) * src[i];  /* eq. (17)    */
        }
    }
}

/* ---- boundary nodes that replace the collision (readings A20, A21) -------------------------
 * WALL_FULLWAY (Fig. 2 (1)): a dry node that only stores the populations streamed into it
 *   and scatters them back: f*_i = f_ibar, no relaxation; they return to the fluid one step later.
 * VELOCITY (equilibrium velocity boundary): the node is wet; its incoming populations are
 *   the streamed ones, the missing ones (from SOLID neighbours) equal their opposites, which is
 *   exactly the half-way rule of stream(); rho is computed from them and the post-collision
 *   state is f^eq(rho, u_bc).
 * Returns 1 if the node type was handled here. */
static int special_node(const orc_ctx *c, int type, const double *f, double rho, double *fstar)
{
    if (type == ORC_WALL_FULLWAY) {
        for (int i = 0; i < c->L.Q; i++) fstar[i] = f[c->L.opp[i]];
        return 1;
    }
    if (type == ORC_VELOCITY) {
        feq(&c->L, rho, c->p.bc_velocity, fstar);
        return 1;
    }
    return 0;
}

/* ---- streaming with half-way bounce-back: f <- stream(f*) (step 5 of DESIGN.md) ---------- */
static void stream(orc_ctx *c, int comp)
{
    const int nx = c->p.nx, ny = c->p.ny, nz = c->p.nz, Q = c->L.Q;
    const double *fs = c->fs[comp];
    double *f = c->f[comp];
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; z++)
        for (int y = 0; y < ny; y++)
            for (int x = 0; x < nx; x++) {
                int64_t n = node_index(c, x, y, z);
                if (c->mask[n] == ORC_SOLID) continue;
                for (int i = 0; i < Q; i++) {
                    int64_t m = node_index(c, wrap(x - c->L.e[i][0], nx), wrap(y - c->L.e[i][1], ny),
                                           wrap(z - c->L.e[i][2], nz));
                    f[i * c->N + n] = c->mask[m] == ORC_SOLID ? fs[c->L.opp[i] * c->N + n] : fs[i * c->N + m];
                }
            }
}

static void step_single(orc_ctx *c)
{
    const int Q = c->L.Q;
    const int64_t N = c->N;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < N; n++) {
        if (c->mask[n] == ORC_SOLID) continue;
        double f[ORC_QMAX], fstar[ORC_QMAX];
        double rho = 0, j[3] = {0, 0, 0}, F[3], v[3], ub[3];
        for (int i = 0; i < Q; i++) {
            f[i] = c->f[0][i * N + n];
            rho += f[i];                                               /* eq. (1) */
            for (int a = 0; a < 3; a++) j[a] += f[i] * c->L.e[i][a];
        }
        if (special_node(c, c->mask[n], f, rho, fstar)) {
            for (int i = 0; i < Q; i++) c->fs[0][i * N + n] = fstar[i];
            continue;
        }
        for (int a = 0; a < 3; a++) {
            F[a] = rho * c->p.force[a];                                /* F = rho g (A4) */
            v[a] = (j[a] + 0.5 * F[a]) / rho;                          /* eq. (16)       */
            ub[a] = j[a] / rho;                                        /* eq. (1)        */
        }
        collide_node(c, f, rho, v, ub, F, c->p.tau[0], fstar);
        for (int i = 0; i < Q; i++) c->fs[0][i * N + n] = fstar[i];
    }
    stream(c, 0);
}

/* Shan-Chen force on component s at node (x,y,z) from the density field of the other one,
 * eq. (10) with the sign of reading A11; psi = 0 on SOLID nodes (A14). */
static void sc_force_node(const orc_ctx *c, int s, int x, int y, int z, double F[3])
{
    const int nx = c->p.nx, ny = c->p.ny, nz = c->p.nz;
    const int o = 1 - s;
    int64_t n = node_index(c, x, y, z);
    double acc[3] = {0, 0, 0};
    for (int i = 0; i < c->L.Q; i++) {
        int64_t m = node_index(c, wrap(x + c->L.e[i][0], nx), wrap(y + c->L.e[i][1], ny),
                               wrap(z + c->L.e[i][2], nz));
        int dry = c->mask[m] == ORC_SOLID || c->mask[m] == ORC_WALL_FULLWAY; /* A14 */
        double ps = dry ? 0.0 : psi_of(c->p.sc_psi, c->rho[o][m]);
        for (int a = 0; a < 3; a++) acc[a] += c->L.w[i] * ps * c->L.e[i][a];
    }
    double p0 = psi_of(c->p.sc_psi, c->rho[s][n]);
    for (int a = 0; a < 3; a++) F[a] = -c->p.sc_G * p0 * acc[a];
}

static void sc_macro_fields(orc_ctx *c)
{
    const int Q = c->L.Q;
    const int64_t N = c->N;
    for (int s = 0; s < 2; s++) {
#pragma omp parallel for schedule(static)
        for (int64_t n = 0; n < N; n++) {
            double rho = 0, j[3] = {0, 0, 0};
            if (c->mask[n] != ORC_SOLID)
                for (int i = 0; i < Q; i++) {
                    double fi = c->f[s][i * N + n];
                    rho += fi;
                    for (int a = 0; a < 3; a++) j[a] += fi * c->L.e[i][a];
                }
            c->rho[s][n] = rho;
            for (int a = 0; a < 3; a++) c->mom[s][a * N + n] = j[a];
        }
    }
}

static void step_sc2(orc_ctx *c)
{
    const int nx = c->p.nx, ny = c->p.ny, nz = c->p.nz, Q = c->L.Q;
    const int64_t N = c->N;
    sc_macro_fields(c);                                                /* (i) */
#pragma omp parallel for schedule(static)
    for (int z = 0; z < nz; z++)
        for (int y = 0; y < ny; y++)
            for (int x = 0; x < nx; x++) {
                int64_t n = node_index(c, x, y, z);
                if (c->mask[n] == ORC_SOLID) continue;
                if (c->mask[n] != ORC_FLUID) {
                    for (int s = 0; s < 2; s++) {
                        double f[ORC_QMAX], fstar[ORC_QMAX];
                        for (int i = 0; i < Q; i++) f[i] = c->f[s][i * N + n];
                        special_node(c, c->mask[n], f, c->rho[s][n], fstar);
                        for (int i = 0; i < Q; i++) c->fs[s][i * N + n] = fstar[i];
                    }
                    continue;
                }
                const double tA = c->p.tau[0], tB = c->p.tau[1];
                double den = c->rho[0][n] / tA + c->rho[1][n] / tB, up[3];
                for (int a = 0; a < 3; a++)                            /* (ii) */
                    up[a] = (c->mom[0][a * N + n] / tA + c->mom[1][a * N + n] / tB) / den;
                for (int s = 0; s < 2; s++) {
                    double F[3], v[3], f[ORC_QMAX], fstar[ORC_QMAX];
                    double rs = c->rho[s][n];
                    sc_force_node(c, s, x, y, z, F);                   /* (iii) */
                    for (int a = 0; a < 3; a++) {
                        F[a] += rs * c->p.force[a];
                        v[a] = up[a] + F[a] / (2.0 * rs);              /* (iv)  */
                    }
                    for (int i = 0; i < Q; i++) f[i] = c->f[s][i * N + n];
                    collide_node(c, f, rs, v, up, F, c->p.tau[s], fstar); /* (v) */
                    for (int i = 0; i < Q; i++) c->fs[s][i * N + n] = fstar[i];
                }
            }
    stream(c, 0);
    stream(c, 1);
}

int orc_step(orc_ctx *c, int n)
{
    for (int t = 0; t < n; t++) {
        if (c->p.model == ORC_SC2) step_sc2(c);
        else step_single(c);
    }
    return 0;
}

/* rho = sum f_i; velocity = v of eq. (16) (includes g/2) for single-component models;
 * for SC2 the bare component velocity j_s/rho_s.  SOLID nodes: rho = 0, u = 0. */
int orc_macro(const orc_ctx *c, int comp, double *rho_out, double *u_out)
{
    if (comp < 0 || comp >= c->ncomp) return -1;
    const int Q = c->L.Q, D = c->L.D;
    const int64_t N = c->N;
    for (int64_t n = 0; n < N; n++) {
        double rho = 0, j[3] = {0, 0, 0};
        if (c->mask[n] == ORC_SOLID || c->mask[n] == ORC_WALL_FULLWAY) { /* dry nodes */
            rho_out[n] = 0.0;
            for (int a = 0; a < D; a++) u_out[a * N + n] = 0.0;
            continue;
        }
        for (int i = 0; i < Q; i++) {
            double fi = c->f[comp][i * N + n];
            rho += fi;
            for (int a = 0; a < 3; a++) j[a] += fi * c->L.e[i][a];
        }
        rho_out[n] = rho;
        for (int a = 0; a < D; a++) {
            double g = (c->p.model == ORC_SC2) ? 0.0 : c->p.force[a];
            u_out[a * N + n] = (j[a] + 0.5 * rho * g) / rho;
        }
    }
    return 0;
}

/* Shan-Chen force field of component `comp` from the current state (for the pins). F: 3*N */
int orc_sc_force(orc_ctx *c, int comp, double *F_out)
{
    if (c->p.model != ORC_SC2 || comp < 0 || comp > 1) return -1;
    sc_macro_fields(c);
    for (int z = 0; z < c->p.nz; z++)
        for (int y = 0; y < c->p.ny; y++)
            for (int x = 0; x < c->p.nx; x++) {
                int64_t n = node_index(c, x, y, z);
                double F[3] = {0, 0, 0};
                if (c->mask[n] == ORC_FLUID) sc_force_node(c, comp, x, y, z, F);
                for (int a = 0; a < 3; a++) F_out[a * c->N + n] = F[a];
            }
    return 0;
}
