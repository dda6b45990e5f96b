/*
 * hfft_oracle.c -- CPU ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, binary128 (__float128) restatement of the generalized Newell
 * demagnetization tensor of Heistracher et al., arXiv 1910.07054, and of the
 * direct real-space field sum.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may call this.  It shares no
 * code, header, table or constant with the CUDA library.
 *
 * Citations are PAPER.md:<line> (+ equation).  Readings of garbled / silent
 * passages are the ones listed in DESIGN.md ("Readings", A1..A16).
 *
 * What is here
 *   newell_f, newell_g          Eq.10, Eq.16
 *   F2,F1,F / G2,G1,G           Eq.9,27,28 / Eq.15,30,31 (nested, paper order)
 *   Nxx, Nxy                    Eq.5, Eq.11 (4th term
 *                               read as Y+dy -- reading A1)
 *   six components              "by permutation of the variables" PAPER.md:46
 *   hfft_oracle_tensor_row      Eq.19 lattice tensor N_{ij}(p dx, q dy) for one
 *                               target layer i (memoised phi lattice, see below)
 *   hfft_oracle_direct_row      Eq.18 direct sum, including the self term
 *
 *
 * Pins: tests/test_oracle_*.py (run with -m "not gpu").  No function here is
 * "parity unpinned".
 */
#include <quadmath.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef __float128 q;

/* ------------------------------------------------------------------ */
/* Eq.10.  Each term whose polynomial prefactor is 0    */
/* is taken as 0 (the limit; reading A5).  atan takes the principal     */
/* value of the quotient (reading A6).                                  */
/* ------------------------------------------------------------------ */
static q newell_f(q x, q y, q z)
{
    q R = sqrtq(x * x + y * y + z * z);
    q s = 0;
    q p1 = y / 2 * (z * z - x * x);
    if (p1 != 0) s += p1 * asinhq(y / sqrtq(x * x + z * z));
    q p2 = z / 2 * (y * y - x * x);
    if (p2 != 0) s += p2 * asinhq(z / sqrtq(x * x + y * y));
    q p3 = x * y * z;
    if (p3 != 0) s -= p3 * atanq(y * z / (x * R));
    s += (2 * x * x - y * y - z * z) * R / 6;
    return s;
}

/* Eq.16. Same conventions. */
static q newell_g(q x, q y, q z)
{
    q R = sqrtq(x * x + y * y + z * z);
    q s = 0;
    q p1 = x * y * z;
    if (p1 != 0) s += p1 * asinhq(z / sqrtq(x * x + y * y));
    q p2 = y / 6 * (3 * z * z - y * y);
    if (p2 != 0) s += p2 * asinhq(x / sqrtq(y * y + z * z));
    q p3 = x / 6 * (3 * z * z - x * x);
    if (p3 != 0) s += p3 * asinhq(y / sqrtq(x * x + z * z));
    q p4 = z * z * z / 6;
    if (p4 != 0) s -= p4 * atanq(x * y / (z * R));
    q p5 = z * y * y / 2;
    if (p5 != 0) s -= p5 * atanq(x * z / (y * R));
    q p6 = z * x * x / 2;
    if (p6 != 0) s -= p6 * atanq(y * z / (x * R));
    s -= x * y * R / 3;
    return s;
}

/* ------------------------------------------------------------------ */
/* Generic pair of cuboids: target size (dx,dy,dz), source (dxp,dyp,dzp) */
/* ------------------------------------------------------------------ */
typedef struct { q dx, dy, dz, dxp, dyp, dzp; } sizes_t;

/* Eq.9 PAPER.md:75 -- "the last three terms cancel out": F2 -> f */
static q F2(q X, q Y, q Z) { return newell_f(X, Y, Z); }

/* Eq.27 */
static q F1(q X, q Y, q Z, const sizes_t *s)
{
    return F2(X, Y + s->dy, Z) - F2(X, Y, Z)
         - F2(X, Y + s->dy - s->dyp, Z) + F2(X, Y - s->dyp, Z);
}

/* Eq.28 */
static q Fbig(q X, q Y, q Z, const sizes_t *s)
{
    return F1(X, Y, Z + s->dz, s) - F1(X, Y, Z, s)
         - F1(X, Y, Z + s->dz - s->dzp, s) + F1(X, Y, Z - s->dzp, s);
}

static const q PI_Q = 3.141592653589793238462643383279502884197Q;

/* Eq.5, |tau| = dx dy dz of the TARGET (reading A7) */
static q Nxx(q X, q Y, q Z, const sizes_t *s)
{
    q tau = s->dx * s->dy * s->dz;
    return (Fbig(X, Y, Z, s) - Fbig(X + s->dx, Y, Z, s)
          - Fbig(X - s->dxp, Y, Z, s) + Fbig(X + s->dx - s->dxp, Y, Z, s))
         / (4 * PI_Q * tau);
}

/* Eq.15 PAPER.md:118 -- "the second term cancels out": G2 -> g */
static q G2(q X, q Y, q Z) { return newell_g(X, Y, Z); }

/* Eq.30 */
static q G1(q X, q Y, q Z, const sizes_t *s)
{
    return G2(X, Y, Z + s->dz) - G2(X, Y, Z)
         - G2(X, Y, Z + s->dz - s->dzp) + G2(X, Y, Z - s->dzp);
}

/* Eq.31 */
static q Gbig(q X, q Y, q Z, const sizes_t *s)
{
    return G1(X + s->dx, Y, Z, s) - G1(X + s->dx, Y - s->dyp, Z, s)
         - G1(X, Y, Z, s) + G1(X, Y - s->dyp, Z, s);
}

/* Eq.11 PAPER.md:99.  The printed 4th term G(X-dx', Y-dy, Z) is read as
 * G(X-dx', Y+dy, Z): the target faces sit at y=Y and y=Y+dy exactly as in the
 * 3rd term (reading A1; pinned by the 6-D quadrature and N_xy = N_yx tests). */
static q Nxy(q X, q Y, q Z, const sizes_t *s)
{
    q tau = s->dx * s->dy * s->dz;
    return (Gbig(X, Y, Z, s) - Gbig(X - s->dxp, Y, Z, s)
          - Gbig(X, Y + s->dy, Z, s) + Gbig(X - s->dxp, Y + s->dy, Z, s))
         / (4 * PI_Q * tau);
}

/* "The remaining components can then be obtained by permutation of the
 * variables": relabel the axes of offset and of both sizes. */
static void tensor_point_q(const q X[3], const q D[3], const q Dp[3], q N[6])
{
    sizes_t s;
    /* xx: identity */
    s = (sizes_t){D[0], D[1], D[2], Dp[0], Dp[1], Dp[2]};
    N[0] = Nxx(X[0], X[1], X[2], &s);
    N[3] = Nxy(X[0], X[1], X[2], &s);
    /* yy: swap x<->y */
    s = (sizes_t){D[1], D[0], D[2], Dp[1], Dp[0], Dp[2]};
    N[1] = Nxx(X[1], X[0], X[2], &s);
    /* zz: swap x<->z */
    s = (sizes_t){D[2], D[1], D[0], Dp[2], Dp[1], Dp[0]};
    N[2] = Nxx(X[2], X[1], X[0], &s);
    /* xz: swap y<->z */
    s = (sizes_t){D[0], D[2], D[1], Dp[0], Dp[2], Dp[1]};
    N[4] = Nxy(X[0], X[2], X[1], &s);
    /* yz: (x,y,z) -> (y,z,x) */
    s = (sizes_t){D[1], D[2], D[0], Dp[1], Dp[2], Dp[0]};
    N[5] = Nxy(X[1], X[2], X[0], &s);
}

/* ------------------------------------------------------------------ */
/* exact (hi,lo) double-pair I/O so tests can look at all 113 bits      */
/* ------------------------------------------------------------------ */
static q from_pair(double hi, double lo) { return (q)hi + (q)lo; }
static void to_pair(q v, double *hi, double *lo)
{
    double h = (double)v;
    *hi = h;
    *lo = (double)(v - (q)h);
}

void hfft_oracle_f(const double hi[3], const double lo[3], double out[2])
{
    to_pair(newell_f(from_pair(hi[0], lo[0]), from_pair(hi[1], lo[1]), from_pair(hi[2], lo[2])),
            &out[0], &out[1]);
}

void hfft_oracle_g(const double hi[3], const double lo[3], double out[2])
{
    to_pair(newell_g(from_pair(hi[0], lo[0]), from_pair(hi[1], lo[1]), from_pair(hi[2], lo[2])),
            &out[0], &out[1]);
}

/* N(X,Y,Z; D target, Dp source) -> 6 components (xx,yy,zz,xy,xz,yz) */
void hfft_oracle_tensor_point(const double X[3], const double D[3], const double Dp[3],
                              double N_hi[6], double N_lo[6])
{
    q Xq[3] = {X[0], X[1], X[2]}, Dq[3] = {D[0], D[1], D[2]}, Dpq[3] = {Dp[0], Dp[1], Dp[2]};
    q N[6];
    tensor_point_q(Xq, Dq, Dpq, N);
    for (int c = 0; c < 6; ++c) to_pair(N[c], &N_hi[c], &N_lo[c]);
}

/* Same 64-term sums but with f, g evaluated in plain double: only used by the
 * test that shows binary128 is needed (pin P9). */
static double f_d(double x, double y, double z)
{
    double R = sqrt(x * x + y * y + z * z), s = 0;
    double p1 = y / 2 * (z * z - x * x);
    if (p1 != 0) s += p1 * asinh(y / sqrt(x * x + z * z));
    double p2 = z / 2 * (y * y - x * x);
    if (p2 != 0) s += p2 * asinh(z / sqrt(x * x + y * y));
    double p3 = x * y * z;
    if (p3 != 0) s -= p3 * atan(y * z / (x * R));
    s += (2 * x * x - y * y - z * z) * R / 6;
    return s;
}
double hfft_oracle_nxx_fp64(const double X[3], const double D[3], const double Dp[3])
{
    double acc = 0;
    const double ux[4] = {0, D[0], -Dp[0], D[0] - Dp[0]};          /* Eq.5 */
    const double sx[4] = {1, -1, -1, 1};
    const double vy[4] = {D[1], 0, D[1] - Dp[1], -Dp[1]};           /* Eq.27 */
    const double wz[4] = {D[2], 0, D[2] - Dp[2], -Dp[2]};           /* Eq.28 */
    const double sg[4] = {1, -1, -1, 1};
    for (int a = 0; a < 4; ++a)
        for (int c = 0; c < 4; ++c)
            for (int b = 0; b < 4; ++b)
                acc += sx[a] * sg[b] * sg[c] * f_d(X[0] + ux[a], X[1] + vy[b], X[2] + wz[c]);
    return acc / (4 * M_PI * D[0] * D[1] * D[2]);
}

/* ------------------------------------------------------------------ */
/* Lattice tensor for a layer stack (Eq.19, section 3      */
/* PAPER.md:153-155): common dx, dy; layer k has thickness dz[k]; layers */
/* are stacked contiguously in array order (reading A9); lower faces at  */
/* zeta_0 = 0, zeta_{k+1} = zeta_k + dz_k; Z_ij = zeta_i - zeta_j (A8).  */
/*                                                                      */
/* Every argument of f / g in the 64-term sums of N_ij(p dx, q dy) lies  */
/* on the lattice (P dx, Q dy, zeta_a - zeta_b), P in [-nx,nx],          */
/* Q in [-ny,ny], a in {i,i+1}, b in [0,nz].  phi() below memoises       */
/* f/g on that lattice; |P|,|Q| are stored and the sign restored from   */
/* the parity of Eq.10/16 in that argument.  Pinned entry by entry,      */
/* negative offsets included, against hfft_oracle_tensor_point by        */
/* tests/test_oracle_newell.py::test_tensor_row_equals_tensor_point_on_  */
/* every_entry (comment only; arithmetic unchanged).                     */
/* ------------------------------------------------------------------ */
typedef struct {
    int nx, ny, nz;
    q dx, dy;
    const q *zeta;          /* nz+1 */
    int a0;                 /* first target interface held (i) */
    q *tab;                 /* [6][2][nz+1][ny+1][nx+1] */
} lattice_t;

/* component c evaluated at lattice point; permutation as in tensor_point_q:
 * 0: f(x,y,z) 1: f(y,x,z) 2: f(z,y,x) 3: g(x,y,z) 4: g(x,z,y) 5: g(y,z,x) */
static q phi_eval(int c, q x, q y, q z)
{
    switch (c) {
    case 0: return newell_f(x, y, z);
    case 1: return newell_f(y, x, z);
    case 2: return newell_f(z, y, x);
    case 3: return newell_g(x, y, z);
    case 4: return newell_g(x, z, y);
    default: return newell_g(y, z, x);
    }
}

static inline size_t lat_index(const lattice_t *L, int c, int a, int b, int Q, int P)
{
    return ((((size_t)c * 2 + (size_t)(a - L->a0)) * (size_t)(L->nz + 1) + (size_t)b)
            * (size_t)(L->ny + 1) + (size_t)Q) * (size_t)(L->nx + 1) + (size_t)P;
}

/* parity of phi_c in x and in y: f even in every argument; g(x,y,z) odd in its
 * first two arguments, even in the third (Eq.10, Eq.16). */
static const int PAR_X[6] = {+1, +1, +1, -1, -1, +1};  /* g(y,z,x): x is 3rd arg -> even */
static const int PAR_Y[6] = {+1, +1, +1, -1, +1, -1};  /* g(x,z,y): y is 3rd arg -> even */

static inline q phi(const lattice_t *L, int c, int P, int Q, int a, int b)
{
    int sg = 1;
    if (P < 0) { P = -P; sg *= PAR_X[c]; }
    if (Q < 0) { Q = -Q; sg *= PAR_Y[c]; }
    q v = L->tab[lat_index(L, c, a, b, Q, P)];
    return sg > 0 ? v : -v;
}

/* A lattice point: x = P dx, y = Q dy, z = zeta_a - zeta_b. */
typedef struct { int P, Q, a, b; } lpt;

/* "+D" / "-D'" along a physical axis.  In-plane D = D' = one cell; along z,
 * Z + dz_i moves the target interface a -> a+1 and Z - dz_j moves the source
 * interface b -> b+1 (Z_ij = zeta_i - zeta_j, reading A8). */
static lpt shift(lpt t, int axis, int plusD, int minusDp)
{
    if (axis == 0) t.P += plusD - minusDp;
    else if (axis == 1) t.Q += plusD - minusDp;
    else { t.a += plusD; t.b += minusDp; }
    return t;
}

/* roles r[0..2]: which physical axis plays the paper's x, y, z for component c
 * (same permutations as tensor_point_q). */
static const int ROLE[6][3] = {{0, 1, 2}, {1, 0, 2}, {2, 1, 0}, {0, 1, 2}, {0, 2, 1}, {1, 2, 0}};

typedef struct { const lattice_t *L; int c; const int *r; } lctx;

static q leaf(const lctx *k, lpt t) { return phi(k->L, k->c, t.P, t.Q, t.a, t.b); }

/* Eq.27 PAPER.md:249-255 (F2 -> f) */
static q F1_l(const lctx *k, lpt t)
{
    int y = k->r[1];
    return leaf(k, shift(t, y, 1, 0)) - leaf(k, t)
         - leaf(k, shift(t, y, 1, 1)) + leaf(k, shift(t, y, 0, 1));
}
/* Eq.28 */
static q F_l(const lctx *k, lpt t)
{
    int z = k->r[2];
    return F1_l(k, shift(t, z, 1, 0)) - F1_l(k, t)
         - F1_l(k, shift(t, z, 1, 1)) + F1_l(k, shift(t, z, 0, 1));
}
/* Eq.5 PAPER.md:52 (without the 1/(4 pi tau) factor) */
static q Nxx_l(const lctx *k, lpt t)
{
    int x = k->r[0];
    return F_l(k, t) - F_l(k, shift(t, x, 1, 0))
         - F_l(k, shift(t, x, 0, 1)) + F_l(k, shift(t, x, 1, 1));
}
/* Eq.30 PAPER.md:274-280 (G2 -> g) */
static q G1_l(const lctx *k, lpt t)
{
    int z = k->r[2];
    return leaf(k, shift(t, z, 1, 0)) - leaf(k, t)
         - leaf(k, shift(t, z, 1, 1)) + leaf(k, shift(t, z, 0, 1));
}
/* Eq.31 */
static q G_l(const lctx *k, lpt t)
{
    int x = k->r[0], y = k->r[1];
    return G1_l(k, shift(t, x, 1, 0)) - G1_l(k, shift(shift(t, x, 1, 0), y, 0, 1))
         - G1_l(k, t) + G1_l(k, shift(t, y, 0, 1));
}
/* Eq.11 PAPER.md:99 with the 4th term read as Y+dy (reading A1) */
static q Nxy_l(const lctx *k, lpt t)
{
    int x = k->r[0], y = k->r[1];
    return G_l(k, t) - G_l(k, shift(t, x, 0, 1))
         - G_l(k, shift(t, y, 1, 0)) + G_l(k, shift(shift(t, x, 0, 1), y, 1, 0));
}

/* One component of N_ij(p dx, q dy): the same nested sums as Nxx()/Nxy() above,
 * on lattice indices, leaves read from the memo. |tau| = dx dy dz_i (target). */
static q lattice_component(const lattice_t *L, int c, int p, int qy, int i, int j)
{
    lctx k = {L, c, ROLE[c]};
    lpt t = {p, qy, i, j};
    q acc = (c < 3) ? Nxx_l(&k, t) : Nxy_l(&k, t);
    q tau = L->dx * L->dy * (L->zeta[i + 1] - L->zeta[i]);
    return acc / (4 * PI_Q * tau);
}

/* N for target layer i, all source layers j, all in-plane offsets:
 * out[j][c][q + ny-1][p + nx-1], p in [-(nx-1), nx-1], q likewise; fp64
 * (rounded once from binary128).  Returns 0, or -1 on allocation failure. */
int hfft_oracle_tensor_row(int nx, int ny, int nz, double dx, double dy, const double *dz,
                           int i, double *out)
{
    q *zeta = (q *)malloc(sizeof(q) * (size_t)(nz + 1));
    if (!zeta) return -1;
    zeta[0] = 0;
    for (int k = 0; k < nz; ++k) zeta[k + 1] = zeta[k] + (q)dz[k];

    lattice_t L = {nx, ny, nz, (q)dx, (q)dy, zeta, i, NULL};
    size_t plane = (size_t)(ny + 1) * (size_t)(nx + 1);
    size_t ntab = 6u * 2u * (size_t)(nz + 1) * plane;
    L.tab = (q *)malloc(sizeof(q) * ntab);
    if (!L.tab) { free(zeta); return -1; }

    /* fill the memo: one f or g evaluation per lattice point and component */
    long total = (long)(6 * 2 * (nz + 1)) * (long)(ny + 1);
#pragma omp parallel for schedule(dynamic, 4)
    for (long t = 0; t < total; ++t) {
        int Q = (int)(t % (ny + 1));
        long r = t / (ny + 1);
        int b = (int)(r % (nz + 1)); r /= (nz + 1);
        int a = (int)(r % 2) + i;
        int c = (int)(r / 2);
        q z = zeta[a] - zeta[b];
        q y = (q)Q * L.dy;
        for (int P = 0; P <= nx; ++P)
            L.tab[lat_index(&L, c, a, b, Q, P)] = phi_eval(c, (q)P * L.dx, y, z);
    }

    int wx = 2 * nx - 1, wy = 2 * ny - 1;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
    for (int j = 0; j < nz; ++j)
        for (int c = 0; c < 6; ++c)
            for (int qy = -(ny - 1); qy <= ny - 1; ++qy)
                for (int p = -(nx - 1); p <= nx - 1; ++p)
                    out[(((size_t)j * 6 + (size_t)c) * (size_t)wy + (size_t)(qy + ny - 1)) * (size_t)wx
                        + (size_t)(p + nx - 1)] = (double)lattice_component(&L, c, p, qy, i, j);
    free(L.tab);
    free(zeta);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Eq.18 PAPER.md:144 (with Eq.19): direct sum for target layer i,      */
/*   H_a(a1,a2,i) = - sum_j sum_{b2,b1} sum_b N^{ab}_{ij}(a1-b1, a2-b2)  */
/*                    * M_b(b1,b2,j),   M = Ms_j m  (reading A12),       */
/* "the sum goes over all points including i".            */
/* Nrow: [nz][6][2ny-1][2nx-1] from hfft_oracle_tensor_row.              */
/* M:    [3][nz][ny][nx].   cells: ncells flat indices a2*nx+a1.         */
/* H:    [ncells][3].  long double accumulators.                          */
/* ------------------------------------------------------------------ */
static const int COMP[3][3] = {{0, 3, 4}, {3, 1, 5}, {4, 5, 2}};

int hfft_oracle_direct_row(int nx, int ny, int nz, const double *Nrow, const double *M,
                           int ncells, const int *cells, double *H)
{
    size_t wx = (size_t)(2 * nx - 1), wy = (size_t)(2 * ny - 1);
#pragma omp parallel for schedule(dynamic, 8)
    for (int t = 0; t < ncells; ++t) {
        int a1 = cells[t] % nx, a2 = cells[t] / nx;
        long double acc[3] = {0, 0, 0};
        for (int j = 0; j < nz; ++j)
            for (int b2 = 0; b2 < ny; ++b2)
                for (int b1 = 0; b1 < nx; ++b1) {
                    size_t off = (size_t)(a2 - b2 + ny - 1) * wx + (size_t)(a1 - b1 + nx - 1);
                    for (int a = 0; a < 3; ++a)
                        for (int b = 0; b < 3; ++b) {
                            double n = Nrow[((size_t)j * 6 + (size_t)COMP[a][b]) * wy * wx + off];
                            double m = M[(((size_t)b * (size_t)nz + (size_t)j) * (size_t)ny + (size_t)b2)
                                         * (size_t)nx + (size_t)b1];
                            acc[a] -= (long double)n * (long double)m;
                        }
                }
        for (int a = 0; a < 3; ++a) H[(size_t)t * 3 + (size_t)a] = (double)acc[a];
    }
    return 0;
}

int hfft_oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
