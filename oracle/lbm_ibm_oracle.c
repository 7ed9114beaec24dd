/*
 * fp64 CPU ORACLE for the LBM-IBM time step of Beny & Latt (arXiv 1904.02108).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no code
 * with the CUDA path (paper_1904_02108_b200/csrc) and neither includes the other.
 *
 * It follows the paper step by step, in the paper's order and notation; all loops are plain, all
 * arithmetic is double.  "P:NN" cites /root/reference/PAPER.md line NN; "Rn" cites the reading
 * of that number in DESIGN.md (section "Readings of the paper").
 *
 * Parity pins (tests/test_oracle_pins.py, run with -m "not gpu"):
 *   orc_delta_w .............. K1 closed-form values + moment identities
 *   orc_interpolate/spread ... K2 (constants/linears exact), K3 brute force over ALL lattice cells,
 *                              K4 adjointness, K6 zeroth/first force moments
 *   orc_mdf .................. K5 geometric-series closed form, K7 U^N = U^0 + G bookkeeping
 *   orc_step (collide/stream/bounce-back/force) .. K8 rest state + mass + momentum balance,
 *                              K9 exact discrete Poiseuille profile, K10 shear-wave decay,
 *                              K12 lattice symmetry
 *   kinematics ............... K11 rigid rotation invariants
 *   coupled propeller fields . PARITY UNPINNED against the paper (it prints no field values);
 *                              pinned only through K1..K13.
 *
 * Canonical state = populations at the time-step boundary, post-stream / pre-collision
 * ("At the beginning of each iteration ... computed from the populations").
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define Q 19

/* D3Q19 structural vectors e_i and weights t_i (P:35, P:45 defer to Krueger et al.; R2):
 * e_0 = 0 (t = 1/3), 6 axis vectors (t = 1/18), 12 face diagonals (t = 1/36). */
static const int E[Q][3] = {
    {0, 0, 0},
    {1, 0, 0}, {-1, 0, 0}, {0, 1, 0}, {0, -1, 0}, {0, 0, 1}, {0, 0, -1},
    {1, 1, 0}, {-1, -1, 0}, {1, -1, 0}, {-1, 1, 0},
    {1, 0, 1}, {-1, 0, -1}, {1, 0, -1}, {-1, 0, 1},
    {0, 1, 1}, {0, -1, -1}, {0, 1, -1}, {0, -1, 1}};
static const double T[Q] = {
    1.0 / 3.0,
    1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0, 1.0 / 18.0,
    1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0,
    1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0, 1.0 / 36.0};
static const int OPP[Q] = {0, 2, 1, 4, 3, 6, 5, 8, 7, 10, 9, 12, 11, 14, 13, 16, 15, 18, 17};

typedef struct {
    double omega, axis[3], center[3];
    long long first, count; /* marker range of this body */
} orc_body_t;

typedef struct orc {
    int nx, ny, nz;
    int wall[3]; /* 0 periodic, 1 half-way bounce-back on both faces of that axis (R15, R16) */
    double tau, gb[3];
    int forcing; /* 0 = Guo (R3, hot path), 1 = the paper's velocity shift U + tau*G */
    long long cells, step;
    double *f, *f2;     /* [Q][cells] populations: canonical state, and scratch for streaming */
    double *rho, *U;    /* [cells], [3][cells]  moments of the canonical state, eq.(1) */
    double *Um;         /* [3][cells] the iterated field U^m of the MDF loop */
    double *G;          /* [3][cells] IBM force (acceleration, R4) of the last step */
    /* Lagrangian points */
    long long nm, cap;
    double *p, *vel, *s;    /* rest position [nm][3], extra velocity [nm][3], area [nm] */
    double *x, *uk;         /* current position, prescribed velocity u_k  [nm][3] */
    double *uint, *g, *du;  /* interpolated u^m(k), g^m(k), Delta u(k)     [nm][3] */
    int *body;
    int nbodies, bcap;
    orc_body_t *bodies;
} orc_t;

/* ------------------------------------------------------------------------------------------ */
/* Peskin 4-point kernel, P:84 with the garbled second branch read as the standard form (R6):
 *   w(r) = 1/8 (3 - 2|r| + sqrt( 1 + 4|r| - 4 r^2))   |r| <= 1
 *        = 1/8 (5 - 2|r| - sqrt(-7 + 12|r| - 4 r^2))   1 <= |r| <= 2
 *        = 0 otherwise                                                                       */
double orc_delta_w(double r)
{
    double a = fabs(r);
    if (a <= 1.0) return 0.125 * (3.0 - 2.0 * a + sqrt(1.0 + 4.0 * a - 4.0 * a * a));
    if (a <= 2.0) return 0.125 * (5.0 - 2.0 * a - sqrt(-7.0 + 12.0 * a - 4.0 * a * a));
    return 0.0;
}

static long long cell_index(const orc_t *o, int X, int Y, int Z)
{
    return ((long long)Z * o->ny + Y) * o->nx + X;
}

/* wrap an index on a periodic axis; on a wall axis an out-of-range index is an error (R17) */
static int wrap_idx(int i, int n, int wall, int *bad)
{
    if (i >= 0 && i < n) return i;
    if (wall) { *bad = 1; return 0; }
    i %= n;
    if (i < 0) i += n;
    return i;
}

/* The 4x4x4 neighbourhood of point x: cells floor(x)-1 .. floor(x)+2 per axis (R7: identical to
 * the paper's 5^3 "round(x) +- 2" block because w(2) = 0), with weights
 * W(X,Y,Z) = w(x-X) w(y-Y) w(z-Z).  Distances use the unwrapped cell coordinate. */
static int stencil(const orc_t *o, const double *x, int idx[3][4], double w[3][4])
{
    int n[3] = {o->nx, o->ny, o->nz};
    int bad = 0;
    for (int a = 0; a < 3; ++a) {
        int c = (int)floor(x[a]);
        for (int j = 0; j < 4; ++j) {
            int X = c - 1 + j;
            w[a][j] = orc_delta_w(x[a] - (double)X);
            idx[a][j] = wrap_idx(X, n[a], o->wall[a], &bad);
        }
    }
    return bad;
}

/* u(k) = sum_{XYZ} U(X,Y,Z) w(x-X) w(y-Y) w(z-Z) */
static void interpolate_point(const orc_t *o, const double *U, const double *x, double *u)
{
    int idx[3][4];
    double w[3][4];
    stencil(o, x, idx, w);
    u[0] = u[1] = u[2] = 0.0;
    for (int jz = 0; jz < 4; ++jz)
        for (int jy = 0; jy < 4; ++jy)
            for (int jx = 0; jx < 4; ++jx) {
                double weight = w[0][jx] * w[1][jy] * w[2][jz];
                long long c = cell_index(o, idx[0][jx], idx[1][jy], idx[2][jz]);
                u[0] += U[c] * weight;
                u[1] += U[o->cells + c] * weight;
                u[2] += U[2 * o->cells + c] * weight;
            }
}

/* F(X,Y,Z) += v * w(x-X) w(y-Y) w(z-Z) for one point.
 * Only target cells with zlo <= Z < zhi are written (the whole lattice for zlo=0, zhi=nz). */
static void spread_point(const orc_t *o, double *F, const double *x, const double *v, int zlo, int zhi)
{
    int idx[3][4];
    double w[3][4];
    stencil(o, x, idx, w);
    for (int jz = 0; jz < 4; ++jz) {
        if (idx[2][jz] < zlo || idx[2][jz] >= zhi) continue;
        for (int jy = 0; jy < 4; ++jy)
            for (int jx = 0; jx < 4; ++jx) {
                double weight = w[0][jx] * w[1][jy] * w[2][jz];
                long long c = cell_index(o, idx[0][jx], idx[1][jy], idx[2][jz]);
                F[c] += v[0] * weight;
                F[o->cells + c] += v[1] * weight;
                F[2 * o->cells + c] += v[2] * weight;
            }
    }
}

/* F += sum_k scale_k v_k W_k over all points, k ascending for every cell.  The z-slabs are
 * independent (each cell is written by exactly one slab, still in ascending k), so running the
 * slabs on different cores gives bit-identical sums to the single loop over k. */
static void spread_all(const orc_t *o, double *F, const double *v, const double *scale)
{
    int nslab = 1;
#ifdef _OPENMP
    nslab = omp_get_max_threads();
#endif
    if (nslab > o->nz) nslab = o->nz;
#pragma omp parallel for schedule(static, 1)
    for (int sl = 0; sl < nslab; ++sl) {
        int zlo = (int)((long long)o->nz * sl / nslab), zhi = (int)((long long)o->nz * (sl + 1) / nslab);
        for (long long k = 0; k < o->nm; ++k) {
            /* skip points none of whose four z-planes (wrapped) falls in this slab */
            int cz = (int)floor(o->x[3 * k + 2]), hit = 0;
            for (int j = -1; j <= 2; ++j) {
                int Z = ((cz + j) % o->nz + o->nz) % o->nz;
                hit |= (Z >= zlo && Z < zhi);
            }
            if (!hit) continue;
            double sc = scale ? scale[k] : 1.0;
            double vv[3] = {v[3 * k] * sc, v[3 * k + 1] * sc, v[3 * k + 2] * sc};
            spread_point(o, F, &o->x[3 * k], vv, zlo, zhi);
        }
    }
}

/* ------------------------------------------------------------------------------------------ */
orc_t *orc_create(int nx, int ny, int nz, double tau, const int wall[3], const double gb[3], int forcing)
{
    if (nx < 1 || ny < 1 || nz < 1 || !(tau > 0.5)) return NULL;
    orc_t *o = (orc_t *)calloc(1, sizeof(orc_t));
    o->nx = nx; o->ny = ny; o->nz = nz; o->tau = tau; o->forcing = forcing;
    for (int a = 0; a < 3; ++a) { o->wall[a] = wall[a]; o->gb[a] = gb[a]; }
    o->cells = (long long)nx * ny * nz;
    size_t c = (size_t)o->cells;
    o->f = (double *)malloc(sizeof(double) * Q * c);
    o->f2 = (double *)malloc(sizeof(double) * Q * c);
    o->rho = (double *)malloc(sizeof(double) * c);
    o->U = (double *)malloc(sizeof(double) * 3 * c);
    o->Um = (double *)malloc(sizeof(double) * 3 * c);
    o->G = (double *)calloc(3 * c, sizeof(double));
    if (!o->f || !o->f2 || !o->rho || !o->U || !o->Um || !o->G) return NULL;
    /* initial state: rest, rho = 1, u = 0 (R18): f_i = Eq_i(1, 0) = t_i */
    for (int i = 0; i < Q; ++i)
        for (size_t k = 0; k < c; ++k) o->f[(size_t)i * c + k] = T[i];
    return o;
}

void orc_destroy(orc_t *o)
{
    if (!o) return;
    free(o->f); free(o->f2); free(o->rho); free(o->U); free(o->Um); free(o->G);
    free(o->p); free(o->vel); free(o->s); free(o->x); free(o->uk); free(o->uint); free(o->g);
    free(o->du); free(o->body); free(o->bodies);
    free(o);
}

/* Eq(i, rho, u) = t_i rho [1 + 3 e_i.u + 9/2 (e_i.u)^2 - 3/2 u.u]    (eq.(3); rho per R1) */
static double equilibrium(int i, double rho, const double *u)
{
    double eu = E[i][0] * u[0] + E[i][1] * u[1] + E[i][2] * u[2];
    double uu = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    return T[i] * rho * (1.0 + 3.0 * eu + 4.5 * eu * eu - 1.5 * uu);
}

/* f = Eq(rho0, u0) with u0 the bare velocity (R18). rho0 may be NULL (=1), u0 may be NULL (=0);
 * layouts rho0[nz][ny][nx], u0[3][nz][ny][nx]. */
void orc_set_fields(orc_t *o, const double *rho0, const double *u0)
{
    size_t c = (size_t)o->cells;
    for (size_t k = 0; k < c; ++k) {
        double rho = rho0 ? rho0[k] : 1.0;
        double u[3] = {0, 0, 0};
        if (u0) { u[0] = u0[k]; u[1] = u0[c + k]; u[2] = u0[2 * c + k]; }
        for (int i = 0; i < Q; ++i) o->f[(size_t)i * c + k] = equilibrium(i, rho, u);
    }
    memset(o->G, 0, sizeof(double) * 3 * c);
}

/* raw population access for tests (mass / momentum sums, symmetry checks) */
double *orc_populations(orc_t *o) { return o->f; }
long long orc_step_count(const orc_t *o) { return o->step; }

/* ------------------------------------------------------------------------------------------ */
static void reserve_markers(orc_t *o, long long n)
{
    if (n <= o->cap) return;
    long long cap = o->cap ? o->cap : 1024;
    while (cap < n) cap *= 2;
    o->p = (double *)realloc(o->p, sizeof(double) * 3 * cap);
    o->vel = (double *)realloc(o->vel, sizeof(double) * 3 * cap);
    o->s = (double *)realloc(o->s, sizeof(double) * cap);
    o->x = (double *)realloc(o->x, sizeof(double) * 3 * cap);
    o->uk = (double *)realloc(o->uk, sizeof(double) * 3 * cap);
    o->uint = (double *)realloc(o->uint, sizeof(double) * 3 * cap);
    o->g = (double *)realloc(o->g, sizeof(double) * 3 * cap);
    o->du = (double *)realloc(o->du, sizeof(double) * 3 * cap);
    o->body = (int *)realloc(o->body, sizeof(int) * cap);
    o->cap = cap;
}

/* One call defines ONE rigid body (appends); pos[n][3], vel[n][3] or NULL, area[n]; returns the
 * body id.  Inputs are the float32 values that cross the product's C ABI, widened to double. */
int orc_set_markers(orc_t *o, const float *pos, const float *vel, const float *area, long long n)
{
    if (n < 0) return -1;
    reserve_markers(o, o->nm + n);
    if (o->nbodies == o->bcap) {
        o->bcap = o->bcap ? 2 * o->bcap : 16;
        o->bodies = (orc_body_t *)realloc(o->bodies, sizeof(orc_body_t) * o->bcap);
    }
    orc_body_t *b = &o->bodies[o->nbodies];
    memset(b, 0, sizeof(*b));
    b->axis[2] = 1.0;
    b->first = o->nm; b->count = n;
    for (long long k = 0; k < n; ++k) {
        long long m = o->nm + k;
        for (int a = 0; a < 3; ++a) {
            o->p[3 * m + a] = (double)pos[3 * k + a];
            o->x[3 * m + a] = (double)pos[3 * k + a];
            o->vel[3 * m + a] = vel ? (double)vel[3 * k + a] : 0.0;
            o->uk[3 * m + a] = 0.0; o->du[3 * m + a] = 0.0; o->g[3 * m + a] = 0.0; o->uint[3 * m + a] = 0.0;
        }
        o->s[m] = (double)area[k];
        o->body[m] = o->nbodies;
    }
    o->nm += n;
    return o->nbodies++;
}

/* applies to the body most recently defined */
int orc_set_kinematics(orc_t *o, double omega, const double axis[3], const double center[3])
{
    if (o->nbodies == 0) return -1;
    double nrm = sqrt(axis[0] * axis[0] + axis[1] * axis[1] + axis[2] * axis[2]);
    if (!(nrm > 0.0)) return -2;
    orc_body_t *b = &o->bodies[o->nbodies - 1];
    b->omega = omega;
    for (int a = 0; a < 3; ++a) { b->axis[a] = axis[a] / nrm; b->center[a] = center[a]; }
    return 0;
}

void orc_clear_markers(orc_t *o) { o->nm = 0; o->nbodies = 0; }

/* Rodrigues rotation matrix about unit axis a by angle th */
static void rodrigues(const double *a, double th, double R[3][3])
{
    double c = cos(th), s = sin(th), v = 1.0 - c;
    R[0][0] = c + a[0] * a[0] * v;        R[0][1] = a[0] * a[1] * v - a[2] * s; R[0][2] = a[0] * a[2] * v + a[1] * s;
    R[1][0] = a[1] * a[0] * v + a[2] * s; R[1][1] = c + a[1] * a[1] * v;        R[1][2] = a[1] * a[2] * v - a[0] * s;
    R[2][0] = a[2] * a[0] * v - a[1] * s; R[2][1] = a[2] * a[1] * v + a[0] * s; R[2][2] = c + a[2] * a[2] * v;
}

/* O2 kinematics (Alg.1; R12, R13, R14): step n -> n+1 uses
 *   x_k = c + R(omega (n+1)) (p_k - c)           always from the rest position, then wrapped into
 *                                                [0,n) on periodic axes,
 *   u_k = (R(omega (n+1)) - R(omega n)) (p_k - c) + vel_k     chord velocity x(t) - x(t-1).       */
void orc_kinematics(orc_t *o)
{
    int n[3] = {o->nx, o->ny, o->nz};
    for (int b = 0; b < o->nbodies; ++b) {
        const orc_body_t *B = &o->bodies[b];
        double R1[3][3], R0[3][3];
        rodrigues(B->axis, B->omega * (double)(o->step + 1), R1);
        rodrigues(B->axis, B->omega * (double)(o->step), R0);
        for (long long k = B->first; k < B->first + B->count; ++k) {
            double d[3], x1[3], x0[3];
            for (int a = 0; a < 3; ++a) d[a] = o->p[3 * k + a] - B->center[a];
            for (int a = 0; a < 3; ++a) {
                x1[a] = R1[a][0] * d[0] + R1[a][1] * d[1] + R1[a][2] * d[2];
                x0[a] = R0[a][0] * d[0] + R0[a][1] * d[1] + R0[a][2] * d[2];
            }
            for (int a = 0; a < 3; ++a) {
                double xa = B->center[a] + x1[a];
                if (!o->wall[a]) xa -= (double)n[a] * floor(xa / (double)n[a]);
                o->x[3 * k + a] = xa;
                o->uk[3 * k + a] = (x1[a] - x0[a]) + o->vel[3 * k + a];
            }
        }
    }
}

/* O1 moments, eq.(1):  rho = sum_i f_i,  U = (1/rho) sum_i e_i f_i  on every cell */
void orc_moments(orc_t *o)
{
    long long c = o->cells;
#pragma omp parallel for schedule(static)
    for (long long k = 0; k < c; ++k) {
        double rho = 0.0, j[3] = {0, 0, 0};
        for (int i = 0; i < Q; ++i) {
            double fi = o->f[(long long)i * c + k];
            rho += fi;
            j[0] += E[i][0] * fi; j[1] += E[i][1] * fi; j[2] += E[i][2] * fi;
        }
        o->rho[k] = rho;
        o->U[k] = j[0] / rho; o->U[c + k] = j[1] / rho; o->U[2 * c + k] = j[2] / rho;
    }
}

/* O4/O5  immersedBoundary(object, U) -> G  (section 3):
 *   U^0 = U, Delta u = 0
 *   for m = 0 .. N-1:   u^m(k) = sum U^m W_k
 *                       g^m(k) = u_k - u^m(k)
 *                       Delta u(k) += g^m(k) s(k)                (R9: also for m = 0)
 *                       if m < N-1:  U^{m+1} = U^m + sum_k s_k g^m_k W_k   (s_k per R8)
 *   G = sum_k Delta u(k) W_k                                     (R10, R11)
 * also_last_u != 0 additionally performs the U update of the last iteration (used by pin K7).
 * Reads o->U (left untouched), iterates on o->Um, writes o->G.  Returns <0 if a stencil crosses
 * a wall (R17). */
int orc_mdf(orc_t *o, int N, int also_last_u)
{
    long long c = o->cells;
    memcpy(o->Um, o->U, sizeof(double) * 3 * c);
    memset(o->G, 0, sizeof(double) * 3 * c);
    for (long long k = 0; k < o->nm; ++k) {
        int idx[3][4]; double w[3][4];
        if (stencil(o, &o->x[3 * k], idx, w)) return -3;
        o->du[3 * k] = o->du[3 * k + 1] = o->du[3 * k + 2] = 0.0;
        o->g[3 * k] = o->g[3 * k + 1] = o->g[3 * k + 2] = 0.0;
    }
    for (int m = 0; m < N; ++m) {
#pragma omp parallel for schedule(static)
        for (long long k = 0; k < o->nm; ++k) {
            interpolate_point(o, o->Um, &o->x[3 * k], &o->uint[3 * k]);
            for (int a = 0; a < 3; ++a) {
                o->g[3 * k + a] = o->uk[3 * k + a] - o->uint[3 * k + a];
                o->du[3 * k + a] += o->g[3 * k + a] * o->s[k];
            }
        }
        if (m < N - 1 || also_last_u) spread_all(o, o->Um, o->g, o->s);
    }
    if (N > 0) spread_all(o, o->G, o->du, NULL);
    return 0;
}

/* O6 collision, in place on the canonical state (eq.(2) with the force of P:56):
 *   a = G + g_body                                                   (acceleration, R4)
 *   forcing 0 (Guo, R3):  u* = U + a/2
 *        f_i <- f_i - (f_i - Eq_i(rho,u*))/tau + (1 - 1/(2 tau)) t_i rho [3 (e_i - u*).a + 9 (e_i.u*)(e_i.a)]
 *   forcing 1 (paper):  f_i <- f_i - (f_i - Eq_i(rho, U + tau a))/tau                      */
void orc_collide(orc_t *o)
{
    long long c = o->cells;
    double tau = o->tau;
#pragma omp parallel for schedule(static)
    for (long long k = 0; k < c; ++k) {
        double rho = o->rho[k];
        double U[3] = {o->U[k], o->U[c + k], o->U[2 * c + k]};
        double a[3] = {o->G[k] + o->gb[0], o->G[c + k] + o->gb[1], o->G[2 * c + k] + o->gb[2]};
        if (o->forcing == 0) {
            double us[3] = {U[0] + 0.5 * a[0], U[1] + 0.5 * a[1], U[2] + 0.5 * a[2]};
            for (int i = 0; i < Q; ++i) {
                double e[3] = {(double)E[i][0], (double)E[i][1], (double)E[i][2]};
                double eu = e[0] * us[0] + e[1] * us[1] + e[2] * us[2];
                double ea = e[0] * a[0] + e[1] * a[1] + e[2] * a[2];
                double ema = (e[0] - us[0]) * a[0] + (e[1] - us[1]) * a[1] + (e[2] - us[2]) * a[2];
                double S = (1.0 - 1.0 / (2.0 * tau)) * T[i] * rho * (3.0 * ema + 9.0 * eu * ea);
                double *fi = &o->f[(long long)i * c + k];
                *fi = *fi - (*fi - equilibrium(i, rho, us)) / tau + S;
            }
        } else {
            double ug[3] = {U[0] + tau * a[0], U[1] + tau * a[1], U[2] + tau * a[2]};
            for (int i = 0; i < Q; ++i) {
                double *fi = &o->f[(long long)i * c + k];
                *fi = *fi + (equilibrium(i, rho, ug) - *fi) / tau;
            }
        }
    }
}

/* O7 streaming, eq.(4):  f_i(x + e_i, n+1) = f_i'(x), indices wrapped on periodic axes.
 * Half-way bounce-back (R15, R16): if x + e_i leaves the domain through a wall axis, then
 * f_ibar(x, n+1) = f_i'(x) instead, even if the link also crosses a periodic face. */
void orc_stream(orc_t *o)
{
    long long c = o->cells;
    int nx = o->nx, ny = o->ny, nz = o->nz;
#pragma omp parallel for schedule(static)
    for (int Z = 0; Z < nz; ++Z)
        for (int Y = 0; Y < ny; ++Y)
            for (int X = 0; X < nx; ++X) {
                long long k = cell_index(o, X, Y, Z);
                for (int i = 0; i < Q; ++i) {
                    int X2 = X + E[i][0], Y2 = Y + E[i][1], Z2 = Z + E[i][2];
                    int hits_wall = (o->wall[0] && (X2 < 0 || X2 >= nx)) ||
                                    (o->wall[1] && (Y2 < 0 || Y2 >= ny)) ||
                                    (o->wall[2] && (Z2 < 0 || Z2 >= nz));
                    double v = o->f[(long long)i * c + k];
                    if (hits_wall) {
                        o->f2[(long long)OPP[i] * c + k] = v;
                    } else {
                        X2 = (X2 + nx) % nx; Y2 = (Y2 + ny) % ny; Z2 = (Z2 + nz) % nz;
                        o->f2[(long long)i * c + cell_index(o, X2, Y2, Z2)] = v;
                    }
                }
            }
    double *t = o->f; o->f = o->f2; o->f2 = t;
}

/* One time step n -> n+1 in the paper's order (pseudo-code P:60-66):
 *  1. U, rho (eq. 1)   2. G = immersedBoundary(object, U)   3.-5. forced collision   6. streaming */
int orc_step(orc_t *o, int nsteps, int mdf_iters)
{
    for (int s = 0; s < nsteps; ++s) {
        orc_moments(o);
        if (o->nm > 0 && mdf_iters > 0) {
            orc_kinematics(o);
            int rc = orc_mdf(o, mdf_iters, 0);
            if (rc) return rc;
        } else {
            memset(o->G, 0, sizeof(double) * 3 * (size_t)o->cells);
        }
        orc_collide(o);
        orc_stream(o);
        o->step += 1;
    }
    return 0;
}

/* O8 read-out: rho and bare U (eq. 1) of the state after the last completed step; force = G of
 * the last step (zero before any step). Any pointer may be NULL. */
void orc_read_fields(orc_t *o, double *rho, double *u, double *force)
{
    size_t c = (size_t)o->cells;
    orc_moments(o);
    if (rho) memcpy(rho, o->rho, sizeof(double) * c);
    if (u) memcpy(u, o->U, sizeof(double) * 3 * c);
    if (force) memcpy(force, o->G, sizeof(double) * 3 * c);
}

/* marker read-out: positions x(t), Delta u(k), last g(k), prescribed u_k, and the reference
 * binning O3: cell key = (floor(z) ny + floor(y)) nx + floor(x). Any pointer may be NULL. */
void orc_read_markers(orc_t *o, double *x, double *du, double *g, double *uk, long long *key)
{
    for (long long k = 0; k < o->nm; ++k) {
        for (int a = 0; a < 3; ++a) {
            if (x) x[3 * k + a] = o->x[3 * k + a];
            if (du) du[3 * k + a] = o->du[3 * k + a];
            if (g) g[3 * k + a] = o->g[3 * k + a];
            if (uk) uk[3 * k + a] = o->uk[3 * k + a];
        }
        if (key) {
            long long cx = (long long)floor(o->x[3 * k]), cy = (long long)floor(o->x[3 * k + 1]),
                      cz = (long long)floor(o->x[3 * k + 2]);
            key[k] = (cz * o->ny + cy) * o->nx + cx;
        }
    }
}

/* ---- stand-alone pieces, exposed so the pins can exercise them on arbitrary inputs ---------- */

/* set the Eulerian velocity field that interpolation / MDF read (layout [3][nz][ny][nx]) */
void orc_set_U(orc_t *o, const double *U) { memcpy(o->U, U, sizeof(double) * 3 * (size_t)o->cells); }
void orc_get_Um(orc_t *o, double *U) { memcpy(U, o->Um, sizeof(double) * 3 * (size_t)o->cells); }

/* place the markers at their rest positions with prescribed velocity vel (omega = 0 kinematics) */
void orc_markers_at_rest(orc_t *o)
{
    for (long long k = 0; k < 3 * o->nm; ++k) { o->x[k] = o->p[k]; o->uk[k] = o->vel[k]; }
}

/* u[nm][3] = interpolation of field U[3][cells] at the current marker positions */
void orc_interpolate(orc_t *o, const double *U, double *u)
{
    for (long long k = 0; k < o->nm; ++k) interpolate_point(o, U, &o->x[3 * k], &u[3 * k]);
}

/* F[3][cells] += sum_k v[k] W_k */
void orc_spread(orc_t *o, const double *v, double *F)
{
    spread_all(o, F, v, NULL);
}

/* O3 reference binning: stable sort of markers by cell key, ties by original index.
 * key[] are the integer cell keys to sort (the test passes the keys derived from the positions
 * the GPU reports, R20); perm[i] = original index of the i-th marker in sorted order. */
void orc_reference_sort(const long long *key, long long n, long long *perm)
{
    /* plain insertion into a stable order via merge sort on (key, index) pairs */
    long long *a = (long long *)malloc(sizeof(long long) * (size_t)n);
    long long *b = (long long *)malloc(sizeof(long long) * (size_t)n);
    for (long long i = 0; i < n; ++i) a[i] = i;
    for (long long width = 1; width < n; width *= 2) {
        for (long long lo = 0; lo < n; lo += 2 * width) {
            long long mid = lo + width < n ? lo + width : n;
            long long hi = lo + 2 * width < n ? lo + 2 * width : n;
            long long i = lo, j = mid, k = lo;
            while (i < mid && j < hi) {
                /* take from the left run on ties: stability */
                if (key[a[j]] < key[a[i]]) b[k++] = a[j++]; else b[k++] = a[i++];
            }
            while (i < mid) b[k++] = a[i++];
            while (j < hi) b[k++] = a[j++];
        }
        long long *t = a; a = b; b = t;
    }
    for (long long i = 0; i < n; ++i) perm[i] = a[i];
    free(a); free(b);
}
