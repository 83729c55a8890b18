/*
 * oracle/lcs_oracle.c  --  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, sequential, single-threaded fp64 CPU statement of the particle hot path of
 * LCS.jl (arxiv/paper_2604_11008): trilinear gather, drag (+gravity) advance, 27-way
 * classification, and the ordered sequential pack / compaction / append that the
 * prefix-scan particle communication of the paper reproduces in parallel.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this. It shares no code, header, table or constant with the CUDA path under
 * paper_2604_11008_b200/; every constant below is restated here from the paper or DESIGN.md.
 *
 * Citations are PAPER.md:<line> (the only reference file) and DESIGN.md "Readings" (R-n) where
 * the paper is silent.  Build: gcc -O2 -ffp-contract=off -fno-fast-math -mfma -shared -fPIC.
 * (-ffp-contract=off: a fused multiply-add happens only where fma() is written.)
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   orc_exp_neg            libm exp within 2 ulp; exact at z=0; monotone
 *   orc_pow_0687           libm pow within 2e-14 relative; exact at R = 0 and R = 1; monotone
 *   orc_push (drag_model 1) one-step closed form with frozen f; settling speed w f(w) = tau g; Stokes limit
 *   orc_cell / orc_owner   face coordinates and nextafter neighbours; interval brute force
 *   orc_interp             constant / nodal / tri-affine closed forms; O(dx^2) convergence; seam
 *   orc_push (advance)     closed-form drag relaxation V(t), X(t) under constant U and g
 *   orc_push (classify)    hand-placed particles for all 27 codes, seams, Px in {1,2,3}
 *   orc_rk2_stage1/2       Heun amplification factor 1 - z + z^2/2 and the position polynomial under constant U, g;
 *                          second-order convergence to the exact solution; decomposition independence (1x1x1 = 2x2x2 = 3x2x1
 *                          by id, which fails unless all 17 arrays travel with the particle); containment
 *   orc_classify_axis      hand-placed particles per axis incl. the seam and P_a in {1,2,3}; after the three sweeps every
 *                          particle is in its owner's slab and the slabs hold the same id sets as the direct 27-way migrate
 *   orc_migrate            paper's worked example; global-sort brute force;
 *                          conservation; containment; idempotence
 *   orc_rk2_stage x drag 1 Heun written out with libm pow, f re-evaluated from the slip of each stage
 *   orc_pair_count         hand-countable lattices, pairs across the periodic seam, shell edges, uniform random
 *                          particles -> g = 1 within the statistical error, independence of the decomposition
 *   contents after a sticky error: parity unpinned (by design)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { ORC_OK = 0, ORC_ERR_ARG = 1, ORC_ERR_CAPACITY = 2, ORC_ERR_JUMP = 3, ORC_ERR_RANGE = 4,
       ORC_ERR_STATE = 5, ORC_ERR_NOMEM = 6 };

#define ORC_STAY 13 /* code (0+1) + 3*(0+1) + 9*(0+1), R-13 */

typedef struct orc {
    int N, Px, Py, Pz, P, nx, ny, nz;
    int64_t cap;
    double L, inv_dx, K_tau, L_below, g[3];
    double inv_nu;                      /* 1 / nu, computed once (rule R6) */
    int drag_model;                     /* 0 = Stokes (f = 1); 1 = f = 1 + 0.15 Re_p^0.687, R-23 */
    const double *u, *v, *w;            /* borrowed, N^3 each, x fastest */
    double *f[7];                       /* x y z vx vy vz d : P*cap each (SoA) */
    int64_t *id;                        /* P*cap */
    double *ex[9];                      /* RK2 only: x0 y0 z0 vx0 vy0 vz0 and dV/dt of stage 1; NULL until used */
    uint8_t *code;                      /* P*cap, destination code of the last push */
    int64_t *send_slot;                 /* P*cap, storage position in the (s,c) send buffer, -1 = stay */
    int64_t *count;                     /* P   */
    int64_t *cnt;                       /* P*27 */
    int status;                         /* sticky */
    int pushed;                         /* a push happened since the last migrate */
    int64_t n_migrated_last;
} orc_t;

/* ---- exp(y) for |y| <= 708: the specified evaluation of DESIGN.md R-3 (range reduction by ln2 hi/lo, degree-14
 * Taylor polynomial in Horner form with fma, exact scaling).  Shared by exp(-z) and by the power of R-23. ---- */
static double exp_spec(double y)
{
    static const double inv_fact[15] = {
        1.0, 1.0, 1.0 / 2.0, 1.0 / 6.0, 1.0 / 24.0, 1.0 / 120.0, 1.0 / 720.0, 1.0 / 5040.0,
        1.0 / 40320.0, 1.0 / 362880.0, 1.0 / 3628800.0, 1.0 / 39916800.0, 1.0 / 479001600.0,
        1.0 / 6227020800.0, 1.0 / 87178291200.0 };
    double k = rint(y * 1.4426950408889634);        /* round to nearest even */
    double r = fma(-k, 6.93147180369123816490e-01, y);
    r = fma(-k, 1.90821492927058770002e-10, r);
    double p = inv_fact[14];
    for (int j = 13; j >= 0; --j) p = fma(p, r, inv_fact[j]);
    return ldexp(p, (int)k);
}

/* ---- exp(-z), z >= 0.  DESIGN.md R-3 (specified so two independent implementations agree). ---- */
double orc_exp_neg(double z)
{
    if (!(z <= 708.0)) return (z != z) ? z : 0.0;   /* z > 708 -> 0 ; NaN propagates */
    return exp_spec(-z);
}

/* ---- R^0.687 for the drag factor of PAPER.md:59 (Eq. 7), R-23: exp(0.687 ln R) with the logarithm
 * specified too.  R below the smallest normal number (in particular R = 0: no slip) gives 0, so f = 1. ---- */
double orc_pow_0687(double R)
{
    static const double inv_odd[11] = {             /* 1/(2k+1), k = 0..10: atanh series of ln m */
        1.0, 1.0 / 3.0, 1.0 / 5.0, 1.0 / 7.0, 1.0 / 9.0, 1.0 / 11.0, 1.0 / 13.0, 1.0 / 15.0, 1.0 / 17.0,
        1.0 / 19.0, 1.0 / 21.0 };
    if (!(R >= 2.2250738585072014e-308)) return (R != R) ? R : 0.0;
    if (R > 1.7976931348623157e308) return R;       /* +inf */
    int e;
    double m = 2.0 * frexp(R, &e);                  /* R = m 2^(e-1), m in [1, 2) */
    e -= 1;
    if (m > 1.4142135623730951) { m = 0.5 * m; e += 1; }   /* m in (sqrt(1/2), sqrt(2)] */
    double s = (m - 1.0) / (m + 1.0);
    double t = s * s;
    double q = inv_odd[10];
    for (int k = 9; k >= 0; --k) q = fma(q, t, inv_odd[k]);
    double lm = (2.0 * s) * q;                      /* ln m = 2 atanh(s) */
    double ed = (double)e;
    double lnR = fma(ed, 6.93147180369123816490e-01, fma(ed, 1.90821492927058770002e-10, lm));
    return exp_spec(0.687 * lnR);
}

/* drag factor f(Re_p) = 1 + 0.15 Re_p^0.687 (Eq. 7), Re_p = d |V - U| / nu (Eq. 8 with 2r = d) */
double orc_drag_factor(const orc_t *o, double d, double dvx, double dvy, double dvz)
{
    if (o->drag_model == 0) return 1.0;
    double s2 = fma(dvz, dvz, fma(dvy, dvy, dvx * dvx));
    double w = sqrt(s2);
    double Re = (d * w) * o->inv_nu;
    return fma(0.15, orc_pow_0687(Re), 1.0);
}

/* ---- geometry ---- */
static inline int64_t cell_of(const orc_t *o, double a)
{   /* integer cell containing a (half-open cells, R-15), clamped */
    int64_t i = (int64_t)floor(a * o->inv_dx);
    if (i < 0) i = 0;
    if (i > o->N - 1) i = o->N - 1;
    return i;
}
int64_t orc_cell(const orc_t *o, double a) { return cell_of(o, a); }

int64_t orc_owner(const orc_t *o, double x, double y, double z)
{   /* s = px + Px*(py + Py*pz), x fastest (R-13) */
    int64_t px = cell_of(o, x) / o->nx, py = cell_of(o, y) / o->ny, pz = cell_of(o, z) / o->nz;
    return px + (int64_t)o->Px * (py + (int64_t)o->Py * pz);
}

static inline int64_t floor_div(int64_t a, int64_t b)   /* b > 0 */
{
    int64_t q = a / b;
    if ((a % b) != 0 && a < 0) --q;
    return q;
}

static inline int64_t pmod(int64_t a, int64_t b) { int64_t m = a % b; return m < 0 ? m + b : m; }

int64_t orc_receiver(const orc_t *o, int64_t s, int c)
{   /* receiver of (s,c): neighbour in direction (dx,dy,dz), periodic */
    int64_t px = s % o->Px, py = (s / o->Px) % o->Py, pz = s / ((int64_t)o->Px * o->Py);
    int dx = c % 3 - 1, dy = (c / 3) % 3 - 1, dz = c / 9 - 1;
    return pmod(px + dx, o->Px) + (int64_t)o->Px * (pmod(py + dy, o->Py) + (int64_t)o->Py * pmod(pz + dz, o->Pz));
}

/* tau_p = (2/9)(rho_p/rho)(r^2/nu) = (rho_p/rho) d^2 / (18 nu), d = 2r */
double orc_tau(const orc_t *o, double d) { return (o->K_tau * d) * d; }

/* ---- a1: trilinear interpolation from the eight surrounding cell-centre values ---- */
static inline double lerp(double p, double q, double f) { return fma(f, q - p, p); }

typedef struct { int64_t i0, i1; double f; } stencil1d;

static inline stencil1d stencil_axis(const orc_t *o, double a)
{   /* cell centre i sits at (i+0.5)*dx; periodic stencil indices (R-9) */
    stencil1d s;
    double ga = fma(a, o->inv_dx, -0.5);
    double fl = floor(ga);
    int64_t i0 = (int64_t)fl;
    s.f = ga - fl;
    s.i0 = (i0 < 0) ? i0 + o->N : i0;
    s.i1 = (i0 + 1 >= o->N) ? i0 + 1 - o->N : i0 + 1;
    return s;
}

static inline double tri(const double *F, int64_t N, stencil1d sx, stencil1d sy, stencil1d sz)
{
#define AT(i, j, k) F[(i) + N * ((j) + N * (k))]
    double c00 = lerp(AT(sx.i0, sy.i0, sz.i0), AT(sx.i1, sy.i0, sz.i0), sx.f);
    double c10 = lerp(AT(sx.i0, sy.i1, sz.i0), AT(sx.i1, sy.i1, sz.i0), sx.f);
    double c01 = lerp(AT(sx.i0, sy.i0, sz.i1), AT(sx.i1, sy.i0, sz.i1), sx.f);
    double c11 = lerp(AT(sx.i0, sy.i1, sz.i1), AT(sx.i1, sy.i1, sz.i1), sx.f);
#undef AT
    double c0 = lerp(c00, c10, sy.f);
    double c1 = lerp(c01, c11, sy.f);
    return lerp(c0, c1, sz.f);
}

int orc_interp(const orc_t *o, int64_t n, const double *x, const double *y, const double *z,
               double *ou, double *ov, double *ow)
{
    if (!o->u) return ORC_ERR_STATE;
    for (int64_t p = 0; p < n; ++p) {
        stencil1d sx = stencil_axis(o, x[p]), sy = stencil_axis(o, y[p]), sz = stencil_axis(o, z[p]);
        ou[p] = tri(o->u, o->N, sx, sy, sz);
        ov[p] = tri(o->v, o->N, sx, sy, sz);
        ow[p] = tri(o->w, o->N, sx, sy, sz);
    }
    return ORC_OK;
}

/* ---- life cycle ---- */
orc_t *orc_create(int N, int Px, int Py, int Pz, int64_t cap, double nu, double rho_ratio,
                  const double *g)
{
    if (N < 2 || Px < 1 || Py < 1 || Pz < 1 || cap < 1) return NULL;
    if (N % Px || N % Py || N % Pz) return NULL;
    orc_t *o = (orc_t *)calloc(1, sizeof(orc_t));
    if (!o) return NULL;
    o->N = N; o->Px = Px; o->Py = Py; o->Pz = Pz; o->P = Px * Py * Pz;
    o->nx = N / Px; o->ny = N / Py; o->nz = N / Pz; o->cap = cap;
    o->L = 6.283185307179586;                       /* 2*pi*L0, L0 = 1 */
    o->inv_dx = (double)N / o->L;
    o->K_tau = rho_ratio / (18.0 * nu);
    o->inv_nu = 1.0 / nu;
    o->drag_model = 0;
    o->L_below = nextafter(o->L, 0.0);
    o->g[0] = g[0]; o->g[1] = g[1]; o->g[2] = g[2];
    size_t slots = (size_t)o->P * (size_t)cap;
    for (int a = 0; a < 7; ++a) o->f[a] = (double *)malloc(slots * sizeof(double));
    o->id = (int64_t *)malloc(slots * sizeof(int64_t));
    o->code = (uint8_t *)malloc(slots);
    o->send_slot = (int64_t *)malloc(slots * sizeof(int64_t));
    o->count = (int64_t *)calloc((size_t)o->P, sizeof(int64_t));
    o->cnt = (int64_t *)calloc((size_t)o->P * 27, sizeof(int64_t));
    int ok = o->id && o->code && o->send_slot && o->count && o->cnt;
    for (int a = 0; a < 7; ++a) ok = ok && o->f[a];
    if (!ok) { /* leak on this path is acceptable for test infrastructure */ return NULL; }
    memset(o->code, ORC_STAY, slots);
    return o;
}

int orc_set_drag_model(orc_t *o, int model)
{
    if (model != 0 && model != 1) return ORC_ERR_ARG;
    o->drag_model = model;
    return ORC_OK;
}

void orc_destroy(orc_t *o)
{
    if (!o) return;
    for (int a = 0; a < 7; ++a) free(o->f[a]);
    for (int a = 0; a < 9; ++a) free(o->ex[a]);
    free(o->id); free(o->code); free(o->send_slot); free(o->count); free(o->cnt);
    free(o);
}

int orc_set_fluid(orc_t *o, const double *u, const double *v, const double *w)
{
    if (!u || !v || !w) return ORC_ERR_ARG;
    o->u = u; o->v = v; o->w = w;
    return ORC_OK;
}

/* particles in any order, binned stably into their owner's slab (R-12) */
int orc_set_particles(orc_t *o, int64_t n, const double *x, const double *y, const double *z,
                      const double *vx, const double *vy, const double *vz, const double *d,
                      const int64_t *id)
{
    const double *in[7] = { x, y, z, vx, vy, vz, d };
    memset(o->count, 0, (size_t)o->P * sizeof(int64_t));
    memset(o->cnt, 0, (size_t)o->P * 27 * sizeof(int64_t));
    o->pushed = 0; o->status = ORC_OK; o->n_migrated_last = 0;
    for (int64_t p = 0; p < n; ++p) {
        if (!(x[p] >= 0.0 && x[p] < o->L && y[p] >= 0.0 && y[p] < o->L && z[p] >= 0.0 && z[p] < o->L)) {
            o->status = ORC_ERR_RANGE; return o->status;
        }
        int64_t s = orc_owner(o, x[p], y[p], z[p]);
        if (o->count[s] == o->cap) { o->status = ORC_ERR_CAPACITY; return o->status; }
        int64_t slot = s * o->cap + o->count[s]++;
        for (int a = 0; a < 7; ++a) o->f[a][slot] = in[a][p];
        o->id[slot] = id[p];
        o->code[slot] = ORC_STAY;
    }
    for (int64_t s = 0; s < o->P; ++s) o->cnt[s * 27 + ORC_STAY] = o->count[s];   /* all codes = stay */
    return ORC_OK;
}

/* load an already binned (packed) state, with codes: subdomain 0's particles, then 1's, ... */
int orc_load_packed(orc_t *o, const int64_t *counts, const double *x, const double *y, const double *z,
                    const double *vx, const double *vy, const double *vz, const double *d,
                    const int64_t *id, const uint8_t *code)
{
    const double *in[7] = { x, y, z, vx, vy, vz, d };
    int64_t q = 0;
    o->status = ORC_OK;
    memset(o->cnt, 0, (size_t)o->P * 27 * sizeof(int64_t));
    for (int64_t s = 0; s < o->P; ++s) {
        if (counts[s] < 0 || counts[s] > o->cap) { o->status = ORC_ERR_CAPACITY; return o->status; }
        o->count[s] = counts[s];
        for (int64_t i = 0; i < counts[s]; ++i, ++q) {
            int64_t slot = s * o->cap + i;
            for (int a = 0; a < 7; ++a) o->f[a][slot] = in[a][q];
            o->id[slot] = id[q];
            uint8_t c = code ? code[q] : ORC_STAY;
            if (c > 26) { o->status = ORC_ERR_ARG; return o->status; }
            o->code[slot] = c;
            o->cnt[s * 27 + c] += 1;
        }
    }
    o->pushed = (code != NULL);
    return ORC_OK;
}

/* ---- a1-a4: gather, advance, classify, count.  One RK2 *stage* of the paper
 *      with the exponential integrator of DESIGN.md R-1 for Eq. 5-6, f = 1. ---- */
int orc_push(orc_t *o, double dt)
{
    if (!o->u) return ORC_ERR_STATE;
    if (o->status) return o->status;
    const int64_t Nn = o->N;
    const int64_t na[3] = { o->nx, o->ny, o->nz };
    memset(o->cnt, 0, (size_t)o->P * 27 * sizeof(int64_t));
    for (int64_t s = 0; s < o->P; ++s) {
        const int64_t pa[3] = { s % o->Px, (s / o->Px) % o->Py, s / ((int64_t)o->Px * o->Py) };
        for (int64_t i = 0; i < o->count[s]; ++i) {
            const int64_t slot = s * o->cap + i;
            /* a1 gather */
            stencil1d sx = stencil_axis(o, o->f[0][slot]);
            stencil1d sy = stencil_axis(o, o->f[1][slot]);
            stencil1d sz = stencil_axis(o, o->f[2][slot]);
            double U[3];
            U[0] = tri(o->u, Nn, sx, sy, sz);
            U[1] = tri(o->v, Nn, sx, sy, sz);
            U[2] = tri(o->w, Nn, sx, sy, sz);
            /* a2 advance: exact solution of dV/dt = -(V-U)/tau + g, dX/dt = V with U frozen */
            double d = o->f[6][slot];
            double tau = (o->K_tau * d) * d;
            if (o->drag_model == 1)                            /* f frozen at the start of the step, tau_eff = tau_p / f */
                tau = tau / orc_drag_factor(o, d, o->f[3][slot] - U[0], o->f[4][slot] - U[1], o->f[5][slot] - U[2]);
            double zz = dt / tau;
            double alpha = orc_exp_neg(zz);
            double b = tau * (1.0 - alpha);
            int du[3];
            for (int a = 0; a < 3; ++a) {
                double vt = fma(tau, o->g[a], U[a]);          /* terminal velocity */
                double wv = o->f[3 + a][slot] - vt;
                double vnew = fma(wv, alpha, vt);
                double disp = fma(wv, b, dt * vt);
                double xu = o->f[a][slot] + disp;
                int wrap = 0;                                  /* periodic box */
                if (xu < 0.0) { xu = xu + o->L; wrap = -1; if (xu >= o->L) xu = o->L_below; }
                else if (xu >= o->L) { xu = xu - o->L; wrap = +1; }
                /* a3 classify: "boundary-crossing check", integer after one floor */
                int64_t dd;
                if (!(xu >= 0.0 && xu < o->L)) {               /* non-finite or > one period */
                    o->status = ORC_ERR_JUMP; dd = 0;
                } else {
                    int64_t ic = cell_of(o, xu);
                    int64_t icu = ic + (int64_t)wrap * Nn;     /* unwrapped cell index (R-14) */
                    dd = floor_div(icu, na[a]) - pa[a];
                    if (dd < -1 || dd > 1) { o->status = ORC_ERR_JUMP; dd = dd < -1 ? -1 : 1; }
                }
                du[a] = (int)dd;
                o->f[a][slot] = xu;
                o->f[3 + a][slot] = vnew;
            }
            int c = (du[0] + 1) + 3 * (du[1] + 1) + 9 * (du[2] + 1);
            o->code[slot] = (uint8_t)c;
            o->cnt[s * 27 + c] += 1;                           /* a4 */
        }
    }
    o->pushed = 1;
    return o->status;
}

/* ---- the paper's two-stage RK2 with per-stage migration ("explicit two-stage
 * Runge-Kutta", :150-164 the 17 arrays, :175-177 one communication per stage; R-25: Heun).
 *   stage 1: K1 = (U(X0) - V0)/tau + g ; X1 = X0 + dt V0 ; V1 = V0 + dt K1 ; keep X0, V0, K1 ; classify X1 ; migrate
 *   stage 2: K2 = (U(X1) - V1)/tau + g ; X  = X0 + dt/2 (V0 + V1) ; V = V0 + dt/2 (K1 + K2) ; classify X ; migrate
 * tau = tau_p / f with f evaluated at the start of each stage (f = 1 for drag_model 0).  The destination of a stage is
 * the minimum-image direction from the slab the particle sits in to the owner of its new position, per axis (the
 * particle of stage 2 no longer sits in the slab of X0, so the wrap of X0 + ... says nothing about it). ---- */
static int min_image_code(orc_t *o, int64_t s, const double *pos3)
{
    const int64_t Pa[3] = { o->Px, o->Py, o->Pz };
    const int64_t na[3] = { o->nx, o->ny, o->nz };
    const int64_t pa[3] = { s % o->Px, (s / o->Px) % o->Py, s / ((int64_t)o->Px * o->Py) };
    const int w[3] = { 1, 3, 9 };
    int c = ORC_STAY;
    for (int a = 0; a < 3; ++a) {
        int64_t dd = 0;
        if (!(pos3[a] >= 0.0 && pos3[a] < o->L)) o->status = ORC_ERR_JUMP;
        else {
            dd = cell_of(o, pos3[a]) / na[a] - pa[a];
            if (Pa[a] >= 3) { if (dd > 1) dd -= Pa[a]; else if (dd < -1) dd += Pa[a]; }
            if (dd < -1 || dd > 1) { o->status = ORC_ERR_JUMP; dd = dd < -1 ? -1 : 1; }
        }
        c += (int)dd * w[a];
    }
    return c;
}

static double wrap_once(const orc_t *o, double xu)
{
    if (xu < 0.0) { xu = xu + o->L; if (xu >= o->L) xu = o->L_below; }
    else if (xu >= o->L) xu = xu - o->L;
    return xu;                                      /* still outside [0, L): min_image_code raises ORC_ERR_JUMP */
}

static int rk2_stage(orc_t *o, double dt, int stage)
{
    if (!o->u) return ORC_ERR_STATE;
    if (o->status) return o->status;
    const size_t slots = (size_t)o->P * (size_t)o->cap;
    for (int a = 0; a < 9; ++a)
        if (!o->ex[a]) { o->ex[a] = (double *)calloc(slots, sizeof(double)); if (!o->ex[a]) return ORC_ERR_NOMEM; }
    if (stage == 2 && o->pushed) return ORC_ERR_STATE;          /* stage 1's codes must have been migrated */
    memset(o->cnt, 0, (size_t)o->P * 27 * sizeof(int64_t));
    const double hdt = 0.5 * dt;
    for (int64_t s = 0; s < o->P; ++s)
        for (int64_t i = 0; i < o->count[s]; ++i) {
            const int64_t slot = s * o->cap + i;
            stencil1d sx = stencil_axis(o, o->f[0][slot]);
            stencil1d sy = stencil_axis(o, o->f[1][slot]);
            stencil1d sz = stencil_axis(o, o->f[2][slot]);
            double U[3] = { tri(o->u, o->N, sx, sy, sz), tri(o->v, o->N, sx, sy, sz), tri(o->w, o->N, sx, sy, sz) };
            double d = o->f[6][slot];
            double tau = (o->K_tau * d) * d;
            if (o->drag_model == 1)
                tau = tau / orc_drag_factor(o, d, o->f[3][slot] - U[0], o->f[4][slot] - U[1], o->f[5][slot] - U[2]);
            double pos[3];
            for (int a = 0; a < 3; ++a) {
                double v = o->f[3 + a][slot];
                double k = (U[a] - v) / tau + o->g[a];              /* Eq. 6 + g (R-4) */
                if (stage == 1) {
                    double x = o->f[a][slot];
                    o->ex[a][slot] = x; o->ex[3 + a][slot] = v; o->ex[6 + a][slot] = k;
                    pos[a] = wrap_once(o, fma(dt, v, x));           /* X1 = X0 + dt V0 */
                    o->f[3 + a][slot] = fma(dt, k, v);              /* V1 = V0 + dt K1 */
                } else {
                    double x0 = o->ex[a][slot], v0 = o->ex[3 + a][slot], k1 = o->ex[6 + a][slot];
                    pos[a] = wrap_once(o, fma(hdt, v0 + v, x0));    /* X = X0 + dt/2 (V0 + V1) */
                    o->f[3 + a][slot] = fma(hdt, k1 + k, v0);       /* V = V0 + dt/2 (K1 + K2) */
                }
                o->f[a][slot] = pos[a];
            }
            int c = min_image_code(o, s, pos);
            o->code[slot] = (uint8_t)c;
            o->cnt[s * 27 + c] += 1;
        }
    o->pushed = 1;
    return o->status;
}

int orc_rk2_stage1(orc_t *o, double dt) { return rk2_stage(o, dt, 1); }
int orc_rk2_stage2(orc_t *o, double dt) { return rk2_stage(o, dt, 2); }

/* ---- axis-by-axis exchange (SURVEY.md 8(f) NEXT #3; PAPER.md:114-118 "mask", :191 "per direction", :243 "all three
 * communications"; R-24).  One sweep = classify along ONE axis from the particle's current position relative
 * to the slab it sits in, then the same ordered pack / compaction / append as orc_migrate with the three codes of that
 * axis.  The direction is the minimum-image difference of subdomain indices: with P_a >= 3 a difference of +-(P_a - 1)
 * is the periodic neighbour -+1; with P_a = 2 the difference is already in {-1, 0, +1}; with P_a = 1 nothing moves. ---- */
int orc_classify_axis(orc_t *o, int axis)
{
    if (axis < 0 || axis > 2) return ORC_ERR_ARG;
    if (o->status) return o->status;
    const int64_t Pa[3] = { o->Px, o->Py, o->Pz };
    const int64_t na[3] = { o->nx, o->ny, o->nz };
    const int w[3] = { 1, 3, 9 };
    memset(o->cnt, 0, (size_t)o->P * 27 * sizeof(int64_t));
    for (int64_t s = 0; s < o->P; ++s) {
        const int64_t pa[3] = { s % o->Px, (s / o->Px) % o->Py, s / ((int64_t)o->Px * o->Py) };
        for (int64_t i = 0; i < o->count[s]; ++i) {
            const int64_t slot = s * o->cap + i;
            const double a = o->f[axis][slot];
            int64_t dd = 0;
            if (!(a >= 0.0 && a < o->L)) o->status = ORC_ERR_JUMP;
            else {
                dd = cell_of(o, a) / na[axis] - pa[axis];
                if (Pa[axis] >= 3) {
                    if (dd > 1) dd -= Pa[axis];
                    else if (dd < -1) dd += Pa[axis];
                }
                if (dd < -1 || dd > 1) { o->status = ORC_ERR_JUMP; dd = dd < -1 ? -1 : 1; }
            }
            const int c = ORC_STAY + (int)dd * w[axis];
            o->code[slot] = (uint8_t)c;
            o->cnt[s * 27 + c] += 1;
        }
    }
    o->pushed = 1;
    return o->status;
}

/* ---- a5-a8: the Fortran LCS sequential packing made 27-way, then ordered append. ---- */
int orc_migrate(orc_t *o)
{
    if (o->status) return o->status;
    const int64_t P = o->P, cap = o->cap;
    int64_t nmig = 0;
    for (int64_t s = 0; s < P; ++s)
        for (int c = 0; c < 27; ++c) if (c != ORC_STAY) nmig += o->cnt[s * 27 + c];
    /* send buffers: one segment per (s,c); seg_start by plain accumulation in (s,c) order */
    int64_t *seg_start = (int64_t *)malloc((size_t)P * 27 * sizeof(int64_t));
    int64_t *counter = (int64_t *)calloc((size_t)P * 27, sizeof(int64_t));   /* per-direction counter */
    double *sb[7]; int64_t *sbid;
    double *sbe[9];                                   /* the RK2 arrays travel with the particle */
    const int rk2 = o->ex[0] != NULL;
    size_t m = (size_t)(nmig > 0 ? nmig : 1);
    for (int a = 0; a < 7; ++a) sb[a] = (double *)malloc(m * sizeof(double));
    sbid = (int64_t *)malloc(m * sizeof(int64_t));
    for (int a = 0; a < 9; ++a) sbe[a] = rk2 ? (double *)malloc(m * sizeof(double)) : NULL;
    int64_t *stay = (int64_t *)malloc((size_t)P * sizeof(int64_t));
    int64_t *fill = (int64_t *)malloc((size_t)P * sizeof(int64_t));
    {
        int64_t acc = 0;
        for (int64_t s = 0; s < P; ++s)
            for (int c = 0; c < 27; ++c) {
                seg_start[s * 27 + c] = acc;
                if (c != ORC_STAY) acc += o->cnt[s * 27 + c];
            }
    }
    /* all particles are scanned in order; each migrant increments its destination's counter */
    for (int64_t s = 0; s < P; ++s) {
        int64_t nstay = 0;
        for (int64_t i = 0; i < o->count[s]; ++i) {
            int64_t slot = s * cap + i;
            int c = o->code[slot];
            if (c == ORC_STAY) {
                int64_t dst = s * cap + nstay;
                o->send_slot[slot] = -1;
                if (dst != slot) {
                    for (int a = 0; a < 7; ++a) o->f[a][dst] = o->f[a][slot];
                    if (rk2) for (int a = 0; a < 9; ++a) o->ex[a][dst] = o->ex[a][slot];
                    o->id[dst] = o->id[slot];
                }
                ++nstay;
            } else {
                int64_t k = counter[s * 27 + c]++;
                int64_t dst = seg_start[s * 27 + c] + k;
                o->send_slot[slot] = k;
                for (int a = 0; a < 7; ++a) sb[a][dst] = o->f[a][slot];
                if (rk2) for (int a = 0; a < 9; ++a) sbe[a][dst] = o->ex[a][slot];
                sbid[dst] = o->id[slot];
            }
        }
        stay[s] = nstay;
    }
    /* append: receiver r = stayers ++ for s ascending, c ascending: segment (s,c) (R-12) */
    for (int64_t r = 0; r < P; ++r) fill[r] = stay[r];
    int overflow = 0;
    for (int64_t s = 0; s < P && !overflow; ++s)
        for (int c = 0; c < 27; ++c) {
            if (c == ORC_STAY) continue;
            int64_t len = counter[s * 27 + c];
            int64_t r = orc_receiver(o, s, c);
            if (fill[r] + len > cap) { overflow = 1; break; }
            int64_t src = seg_start[s * 27 + c], dst = r * cap + fill[r];
            for (int a = 0; a < 7; ++a) memcpy(o->f[a] + dst, sb[a] + src, (size_t)len * sizeof(double));
            if (rk2) for (int a = 0; a < 9; ++a) memcpy(o->ex[a] + dst, sbe[a] + src, (size_t)len * sizeof(double));
            memcpy(o->id + dst, sbid + src, (size_t)len * sizeof(int64_t));
            fill[r] += len;
        }
    if (overflow) o->status = ORC_ERR_CAPACITY;
    else {
        for (int64_t r = 0; r < P; ++r) {
            o->count[r] = fill[r];
            memset(o->code + r * cap, ORC_STAY, (size_t)fill[r]);
        }
        memset(o->cnt, 0, (size_t)P * 27 * sizeof(int64_t));
        for (int64_t r = 0; r < P; ++r) o->cnt[r * 27 + ORC_STAY] = o->count[r];
        o->n_migrated_last = nmig;
    }
    o->pushed = 0;
    for (int a = 0; a < 7; ++a) free(sb[a]);
    for (int a = 0; a < 9; ++a) free(sbe[a]);
    free(sbid); free(seg_start); free(counter); free(stay); free(fill);
    return o->status;
}

/* ---- accessors ---- */
int64_t orc_total(const orc_t *o)
{
    int64_t n = 0;
    for (int64_t s = 0; s < o->P; ++s) n += o->count[s];
    return n;
}
int orc_status(const orc_t *o) { return o->status; }
int64_t orc_n_migrated_last(const orc_t *o) { return o->n_migrated_last; }
void orc_get_counts(const orc_t *o, int64_t *counts) { memcpy(counts, o->count, (size_t)o->P * sizeof(int64_t)); }
void orc_get_cnt_table(const orc_t *o, int64_t *cnt) { memcpy(cnt, o->cnt, (size_t)o->P * 27 * sizeof(int64_t)); }

/* packed: subdomain 0's particles in slot order, then subdomain 1's, ...  Any pointer may be NULL. */
void orc_get_particles(const orc_t *o, int64_t *counts, double *x, double *y, double *z, double *vx,
                       double *vy, double *vz, double *d, int64_t *id, uint8_t *code)
{
    double *out[7] = { x, y, z, vx, vy, vz, d };
    int64_t q = 0;
    for (int64_t s = 0; s < o->P; ++s) {
        if (counts) counts[s] = o->count[s];
        size_t len = (size_t)o->count[s];
        const size_t base = (size_t)s * (size_t)o->cap;
        for (int a = 0; a < 7; ++a) if (out[a]) memcpy(out[a] + q, o->f[a] + base, len * sizeof(double));
        if (id) memcpy(id + q, o->id + base, len * sizeof(int64_t));
        if (code) memcpy(code + q, o->code + base, len);
        q += (int64_t)len;
    }
}

/* storage positions assigned by the last orc_migrate to the first n pre-migrate slots of subdomain s:
 * 0-based index inside the (s, code) send buffer, -1 for a stayer (PAPER.md:117-124, 1-based there) */
void orc_get_last_send_slots(const orc_t *o, int64_t s, int64_t n, int64_t *out)
{
    memcpy(out, o->send_slot + (size_t)s * (size_t)o->cap, (size_t)n * sizeof(int64_t));
}

/* ---- statistics hook: the pair count behind the radial distribution function g(r)
 * ("radial distribution function at contact g(r=R) ... unity indicates a uniform distribution"; the
 * statistic the heterogeneous run offloads to a GPU).  Plain definition, O(n^2): the number of
 * unordered pairs {i, j}, i != j, of ALL particles in the box whose periodic (minimum-image) separation r satisfies
 * r_lo <= r < r_hi.  The paper gives no formula for it; R-26 fixes the arithmetic so that two independent
 * implementations agree on every pair, also at the edges of the shell:
 *   per axis  d = a_i - a_j;  if (d > L/2) d = d - L;  else if (d < -L/2) d = d + L;        (L/2 = 0.5 * L, exact)
 *   r2 = fma(dz, dz, fma(dy, dy, dx * dx));   counted iff  r_lo * r_lo <= r2  and  r2 < r_hi * r_hi.
 * (d and -d give the same r2 bit for bit, so the count does not depend on which of the two particles comes first.)
 * g over the shell = count / (n (n-1) / 2 * V_shell / L^3), V_shell = 4/3 pi (r_hi^3 - r_lo^3): left to the caller.
 * Pins: tests/test_oracle_pairs.py (hand-countable lattice, seam pairs, uniform random -> g = 1 within the
 * statistical error, shell edges). ---- */
int64_t orc_pair_count(const orc_t *o, double r_lo, double r_hi)
{
    if (!(r_lo >= 0.0) || !(r_hi > r_lo)) return -1;
    const double half = 0.5 * o->L;
    const double lo2 = r_lo * r_lo, hi2 = r_hi * r_hi;
    int64_t n = 0, pairs = 0;
    for (int64_t s = 0; s < o->P; ++s) n += o->count[s];
    double *xs = (double *)malloc((size_t)(n > 0 ? n : 1) * 3 * sizeof(double));
    if (!xs) return -1;
    int64_t q = 0;
    for (int64_t s = 0; s < o->P; ++s)
        for (int64_t i = 0; i < o->count[s]; ++i, ++q)
            for (int a = 0; a < 3; ++a) xs[3 * q + a] = o->f[a][s * o->cap + i];
    for (int64_t i = 0; i < n; ++i)
        for (int64_t j = i + 1; j < n; ++j) {
            double d[3];
            for (int a = 0; a < 3; ++a) {
                d[a] = xs[3 * i + a] - xs[3 * j + a];
                if (d[a] > half) d[a] = d[a] - o->L;
                else if (d[a] < -half) d[a] = d[a] + o->L;
            }
            const double r2 = fma(d[2], d[2], fma(d[1], d[1], d[0] * d[0]));
            if (lo2 <= r2 && r2 < hi2) ++pairs;
        }
    free(xs);
    return pairs;
}
