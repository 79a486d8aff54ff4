/*
 * krp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded fp64 CPU statement of the polarized Monte-Carlo
 * transport + per-event imaging path of Kratos-polrad (arxiv 2512.01283),
 * written from /root/reference/PAPER.md (cited below as PAPER.md:<line>) and
 * the readings listed in DESIGN.md ("Readings of the paper", R1..).
 *
 * It shares no code with the CUDA path (paper_2512_01283_b200/csrc).  Only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call it.
 *
 * Precision: fp64 everywhere, with five deliberate fp32 quantisations that
 * are part of the method's *state definition* (R12), made so that
 * integer decisions (which cell an event falls in) are taken on the same
 * numbers by both implementations:
 *   - the lookup tables are the caller's fp32 arrays, read as they are;
 *   - the per-cell unit field direction B^ is stored rounded to fp32;
 *   - the packet direction n^ is stored rounded to fp32 after emission and
 *     after every scattering;
 *   - the cell-local position of a packet is stored rounded to fp32 at
 *     emission and at every event (the event record holds fp32 positions and
 *     the next flight starts from the record);
 *   - the normalised Stokes components (q,u,v) are stored rounded to fp32 at
 *     every event and after every scattering (the 48-byte event record and the
 *     packet queue hold fp32 Stokes vectors).
 *
 * The last two of these entered after the first kernel existed; the build with
 * -DORA_STATE_FP32=0 (libkrp_oracle_pure.so) leaves them out and serves as the
 * control: tests/test_oracle_control.py runs every pin on it and compares the two
 * builds' maps, tests/test_gpu_parity.py reports the CUDA path's agreement with it.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): every exported function
 * below is pinned to a closed form, an invariant, a library routine
 * (scipy.linalg.expm, cuRAND host Philox) or brute force; see the table in
 * DESIGN.md section "Oracle pins" (round 2 added: the second-moment map img2,
 * the (U,V) block and S34 terms of F(Theta), the emission map).  "Parity
 * unpinned": the absolute image unit (R14) and the sign convention of V (R6).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORA_PI 3.14159265358979323846264338327950288

/* Control build (R12, "pure-state control"): -DORA_STATE_FP32=0 turns OFF the two state
 * roundings that were added after the first kernel existed -- the cell-local position at emission
 * and at every event, and (q,u,v) at every event and after every scattering -- so that the state
 * between steps is pure fp64 (tables, B^ and n^ stay fp32 as in the oracle's first commit).  The
 * pins run on both builds; tests report how the CUDA path and the rounded build compare with it. */
#ifndef ORA_STATE_FP32
#define ORA_STATE_FP32 1
#endif
#if ORA_STATE_FP32
#define ORA_STATE(x) ((double)(float)(x))
#else
#define ORA_STATE(x) (x)
#endif
int ora_state_is_fp32(void) { return ORA_STATE_FP32; }

/* ------------------------------------------------------------------ */
/* S0  Random numbers: Philox4x32-10 (Salmon et al. 2011), counter     */
/*     based; schedule in DESIGN.md R11.                               */
/* ------------------------------------------------------------------ */
void ora_philox(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* uniform in (0,1) from the top 23 bits: (2k+1)/2^24, k < 2^23, is exact in
 * fp32 and fp64 and never 0 or 1 (R11).  (24 bits + 1/2 would need a 25-bit
 * significand and would round to 1.0f in fp32.) */
double ora_u01(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }

/* uniform in (0,1) from 27 + 25 = 52 bits of two words: (2k+1)/2^53 is exact
 * in fp64 and never 0 or 1 (volume-source cell pick, R11). */
double ora_u53(uint32_t x0, uint32_t x1)
{
    return ((double)(x0 >> 5) * 33554432.0 + (double)(x1 >> 7) + 0.5) * (1.0 / 4503599627370496.0);
}

static void draw(uint64_t seed, uint64_t id, uint32_t k, uint32_t b, uint32_t w[4])
{
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { (uint32_t)id, (uint32_t)(id >> 32), k, b };
    ora_philox(key, ctr, w);
}

/* ------------------------------------------------------------------ */
/* A1  Hamilton quaternions, eq. 1.  q = (w, x, y, z).  */
/* ------------------------------------------------------------------ */
void ora_quat_mul(const double a[4], const double b[4], double o[4])
{
    double w = a[0]*b[0] - a[1]*b[1] - a[2]*b[2] - a[3]*b[3];
    double x = a[0]*b[1] + a[1]*b[0] + a[2]*b[3] - a[3]*b[2];
    double y = a[0]*b[2] - a[1]*b[3] + a[2]*b[0] + a[3]*b[1];
    double z = a[0]*b[3] + a[1]*b[2] - a[2]*b[1] + a[3]*b[0];
    o[0] = w; o[1] = x; o[2] = y; o[3] = z;
}

/* A2  q_B(theta_B, phi_B), eq. 2.  |B| = 0 gives q_B = 1 (R10). */
void ora_quat_from_B(const double b[3], double q[4])
{
    double rho = hypot(b[0], b[1]);
    double th = atan2(rho, b[2]);
    double ph = (rho > 0.0) ? atan2(b[1], b[0]) : 0.0;
    if (rho == 0.0 && b[2] == 0.0) { th = 0.0; ph = 0.0; }
    q[0] =  cos(ph / 2) * cos(th / 2);
    q[1] = -sin(ph / 2) * sin(th / 2);
    q[2] =  cos(ph / 2) * sin(th / 2);
    q[3] =  sin(ph / 2) * cos(th / 2);
}

/* A3  (0, v_GF) = q* (0, v) q, eq. 3. */
void ora_rot_to_gf(const double q[4], const double v[3], double o[3])
{
    double qc[4] = { q[0], -q[1], -q[2], -q[3] };
    double pv[4] = { 0.0, v[0], v[1], v[2] }, t[4], r[4];
    ora_quat_mul(qc, pv, t);
    ora_quat_mul(t, q, r);
    o[0] = r[1]; o[1] = r[2]; o[2] = r[3];
}

/* inverse of eq. 3: (0, v) = q (0, v_GF) q*. */
void ora_rot_to_lab(const double q[4], const double v[3], double o[3])
{
    double qc[4] = { q[0], -q[1], -q[2], -q[3] };
    double pv[4] = { 0.0, v[0], v[1], v[2] }, t[4], r[4];
    ora_quat_mul(q, pv, t);
    ora_quat_mul(t, qc, r);
    o[0] = r[1]; o[1] = r[2]; o[2] = r[3];
}

static double dot3(const double a[3], const double b[3]) { return a[0]*b[0] + a[1]*b[1] + a[2]*b[2]; }
static void cross3(const double a[3], const double b[3], double o[3])
{
    double x = a[1]*b[2] - a[2]*b[1], y = a[2]*b[0] - a[0]*b[2], z = a[0]*b[1] - a[1]*b[0];
    o[0] = x; o[1] = y; o[2] = z;
}

/* A4  spherical basis of a propagation direction, eq. 4-5.
 *     Pole rule R10: n_x^2 + n_y^2 < 1e-24 takes phi = 0. */
void ora_basis(const double n[3], double th[3], double ph[3])
{
    double s2 = n[0]*n[0] + n[1]*n[1];
    double r = sqrt(s2 + n[2]*n[2]);
    double cp = 1.0, sp = 0.0;
    double s = sqrt(s2);
    if (s2 >= 1e-24) { cp = n[0] / s; sp = n[1] / s; }
    double ct = n[2] / r, st = s / r;
    th[0] = ct * cp; th[1] = ct * sp; th[2] = -st;
    ph[0] = -sp;     ph[1] = cp;      ph[2] = 0.0;
}

/* A5  angle eta between phi^_GF and phi^' (eq. 6) with the
 *     sign restored (R2): sin(eta) = (phi^_GF x phi^') . n_GF.            */
void ora_eta_gf(const double q[4], const double n[3], double* ce, double* se)
{
    double th[3], ph[3], phg[3], ng[3], thp[3], php[3], c[3];
    ora_basis(n, th, ph);
    ora_rot_to_gf(q, ph, phg);
    ora_rot_to_gf(q, n, ng);
    ora_basis(ng, thp, php);
    *ce = dot3(phg, php);
    cross3(phg, php, c);
    double nn = sqrt(dot3(ng, ng));
    *se = dot3(c, ng) / nn;
}

/* A5  (Q,U) rotation by 2 eta, eq. 7; I and V invariant. */
void ora_rotate_qu(double S[4], double ce, double se)
{
    double c2 = ce*ce - se*se, s2 = 2.0 * se * ce;
    double Q = S[1], U = S[2];
    S[1] =  c2 * Q + s2 * U;
    S[2] = -s2 * Q + c2 * U;
}

/* A12 source-free in-cell solution, PAPER.md:302-318 (App. A) with the
 *     matrix of R1.  Evaluated through exp(-(a1 -+ a2) dtau) so that nothing
 *     overflows at dtau = 1e3.                                            */
void ora_appA(double S[4], double a1, double a2, double a3, double dtau)
{
    double eA = exp(-(a1 - a2) * dtau), eB = exp(-(a1 + a2) * dtau), e1 = exp(-a1 * dtau);
    double I0 = S[0], Q0 = S[1], U0 = S[2], V0 = S[3];
    double cb = cos(a3 * dtau), sb = sin(a3 * dtau);
    S[0] = 0.5 * ((I0 - Q0) * eA + (I0 + Q0) * eB);
    S[1] = 0.5 * ((Q0 - I0) * eA + (Q0 + I0) * eB);
    S[2] = e1 * (U0 * cb - V0 * sb);
    S[3] = e1 * (U0 * sb + V0 * cb);
}

/* T4  in-cell event location (R7): smallest t > 0 with
 *       I_e/2 [(1-q) e^{-(a1-a2)t} + (1+q) e^{-(a1+a2)t}] = target.
 *     f is decreasing and convex, Newton from t = 0 converges monotonically. */
double ora_event_solve(double Ie, double q, double a1, double a2, double target)
{
    if (a2 == 0.0) return log(Ie / target) / a1;
    double t = 0.0;
    for (int it = 0; it < 200; ++it) {
        double eA = exp(-(a1 - a2) * t), eB = exp(-(a1 + a2) * t);
        double f  = 0.5 * Ie * ((1 - q) * eA + (1 + q) * eB) - target;
        double fp = -0.5 * Ie * ((1 - q) * (a1 - a2) * eA + (1 + q) * (a1 + a2) * eB);
        double dt = -f / fp;
        t += dt;
        if (fabs(dt) <= 1e-15 * fmax(t, 1e-300)) break;
    }
    return t;
}

/* ------------------------------------------------------------------ */
/* Model = grid + tables + source                                      */
/* ------------------------------------------------------------------ */
typedef struct ora_model {
    int nx, ny, nz;
    int64_t ncell;
    double lo[3], d[3];
    const float* kr;      /* borrowed, [nz][ny][nx], kappa*rho per unit length */
    float* bhat;          /* owned, [ncell][3], fp32-rounded unit B; NULL = none */
    int n_ang; float* mueller;     /* owned copies of the caller's fp32 tables */
    double* cdf;                   /* [n_ang] Theta CDF built here in fp64 */
    int n_inc; float* opac;
    double w_min; int max_scatter;
    int src_kind, emit_records;
    double src_pos[3], src_dir[3];
    double* src_cdf;      /* owned, [ncell] running sum of cell weights, or NULL */
    int64_t src_cell; int src_idx[3]; double src_p[3];
    int periodic;         /* bit a set: axis a is periodic, reading R20 */
    const struct ora_ztable* ztab;   /* borrowed; non-NULL: scatter and peel with the full Z(Omega;Omega') (NEXT-2, R21) */
} ora_model;
struct ora_ztable;
void ora_model_set_ztable(ora_model* m, const struct ora_ztable* z) { m->ztab = z; }
int ora_scatter_z(const struct ora_ztable* z, const double b[3], const double n_in[3], const double S_in[4],
                  uint64_t seed, uint64_t id, uint32_t k, double n_out[3], double S_out[4], double* tau_next);
void ora_peel_z(const struct ora_ztable* z, const double b[3], const double n_in[3], const double S_in[4], const double n_obs[3],
                double S_out[4]);

/* Periodic boundary conditions (the cylinder test: "our use of periodic boundary conditions").
 * Reading R20: a packet or an imaging ray that leaves through a face of a periodic axis re-enters through the opposite
 * face at the same cell-local position; after ORA_MAX_WRAPS such crossings it counts as having left the grid (a ray
 * that runs parallel to the open faces of an empty periodic box would never end). */
#define ORA_MAX_WRAPS 4096
void ora_model_set_periodic(ora_model* m, int mask) { m->periodic = mask & 7; }

void ora_model_free(ora_model* m)
{
    if (!m) return;
    free(m->bhat); free(m->mueller); free(m->cdf); free(m->opac); free(m->src_cdf); free(m);
}

/* D4/R13: Mueller table on n_ang nodes Theta_j = j*180/(n_ang-1) degrees,
 * rows (S11,S12,S33,S34); opacity table on n_inc nodes mu_m = m/(n_inc-1),
 * mu = |cos(angle between n^ and B^)|, rows (a1,a2,a3,albedo).            */
ora_model* ora_model_create(int nx, int ny, int nz, const double bounds[6],
                            const float* density, const float* bfield,
                            int n_ang, const float* mueller, int n_inc, const float* opac,
                            double w_min, int max_scatter)
{
    ora_model* m = (ora_model*)calloc(1, sizeof(ora_model));
    m->nx = nx; m->ny = ny; m->nz = nz; m->ncell = (int64_t)nx * ny * nz;
    for (int a = 0; a < 3; ++a) m->lo[a] = bounds[2*a];
    m->d[0] = (bounds[1] - bounds[0]) / nx;
    m->d[1] = (bounds[3] - bounds[2]) / ny;
    m->d[2] = (bounds[5] - bounds[4]) / nz;
    m->kr = density;
    if (bfield) {
        m->bhat = (float*)malloc(sizeof(float) * 3 * m->ncell);
        for (int64_t c = 0; c < m->ncell; ++c) {
            double bx = bfield[3*c], by = bfield[3*c+1], bz = bfield[3*c+2];
            double r = sqrt(bx*bx + by*by + bz*bz);
            if (r > 0.0) { bx /= r; by /= r; bz /= r; } else { bx = 0; by = 0; bz = 1; }
            m->bhat[3*c] = (float)bx; m->bhat[3*c+1] = (float)by; m->bhat[3*c+2] = (float)bz;
        }
    }
    m->n_ang = n_ang;
    m->mueller = (float*)malloc(sizeof(float) * 4 * n_ang);
    memcpy(m->mueller, mueller, sizeof(float) * 4 * n_ang);
    m->n_inc = n_inc;
    m->opac = (float*)malloc(sizeof(float) * 4 * n_inc);
    memcpy(m->opac, opac, sizeof(float) * 4 * n_inc);
    m->w_min = w_min; m->max_scatter = max_scatter;
    /* Theta CDF: trapezoid of g_j = S11_j sin(Theta_j) on the table nodes (R13) */
    m->cdf = (double*)malloc(sizeof(double) * n_ang);
    double dth = ORA_PI / (n_ang - 1);
    m->cdf[0] = 0.0;
    for (int j = 1; j < n_ang; ++j) {
        double g0 = (double)mueller[4*(j-1)] * sin((j-1) * dth);
        double g1 = (double)mueller[4*j] * sin(j * dth);
        m->cdf[j] = m->cdf[j-1] + 0.5 * (g0 + g1);
    }
    double tot = m->cdf[n_ang-1];
    for (int j = 0; j < n_ang; ++j) m->cdf[j] /= tot;
    m->cdf[n_ang-1] = 1.0;
    /* default source: point, isotropic, at the box centre */
    m->src_kind = 0;
    return m;
}

/* krp_source: kind bit0 = positions uniform/weighted in volume (else point),
 * bit1 = collimated along dir (else isotropic).  cell_weight: [ncell] or NULL. */
void ora_source_set(ora_model* m, int kind, const double pos[3], const double dir[3],
                    const float* cell_weight, int emit_records)
{
    m->src_kind = kind; m->emit_records = emit_records;
    for (int a = 0; a < 3; ++a) { m->src_pos[a] = pos[a]; m->src_dir[a] = dir[a]; }
    if (kind & 2) {
        /* reading R23: light propagates "along direction (theta, phi)", a unit vector, and the march measures
         * path length in units of |n|; the caller's `dir` "need not be normalised" (include/krp.h), so it is
         * divided by its length here, in fp64, before the fp32 rounding of R12 at emission */
        double nn = sqrt(dir[0] * dir[0] + dir[1] * dir[1] + dir[2] * dir[2]);
        if (nn > 0.0) for (int a = 0; a < 3; ++a) m->src_dir[a] = dir[a] / nn;
    }
    int n[3] = { m->nx, m->ny, m->nz };
    for (int a = 0; a < 3; ++a) {
        double x = (pos[a] - m->lo[a]) / m->d[a];
        int i = (int)floor(x);
        if (i < 0) i = 0;
        if (i > n[a] - 1) i = n[a] - 1;
        /* reading R24: a source position outside the box is moved to the nearest point of the box, coordinate by coordinate
         * (the paper is silent: the sources of its tests lie inside their grids; a packet has to start in a cell) */
        double p = x - i;
        if (p < 0.0) p = 0.0;
        if (p > 1.0) p = 1.0;
        m->src_idx[a] = i; m->src_p[a] = p;
    }
    free(m->src_cdf); m->src_cdf = NULL;
    if ((kind & 1) && cell_weight) {
        m->src_cdf = (double*)malloc(sizeof(double) * m->ncell);
        double acc = 0.0;
        for (int64_t c = 0; c < m->ncell; ++c) { acc += (double)cell_weight[c]; m->src_cdf[c] = acc; }
    }
}

/* linear interpolation of the Mueller table at Theta (degrees), R13 */
void ora_mueller_at(const ora_model* m, double theta_deg, double F[4])
{
    double x = theta_deg * (m->n_ang - 1) / 180.0;
    int j = (int)floor(x);
    if (j < 0) j = 0;
    if (j > m->n_ang - 2) j = m->n_ang - 2;
    double w = x - j;
    for (int s = 0; s < 4; ++s)
        F[s] = (1 - w) * (double)m->mueller[4*j + s] + w * (double)m->mueller[4*(j+1) + s];
}

/* linear interpolation of the opacity table at mu = |cos vartheta|, R8/R13 */
void ora_opac_at(const ora_model* m, double mu, double a[4])
{
    if (m->n_inc == 1) { for (int s = 0; s < 4; ++s) a[s] = m->opac[s]; return; }
    if (mu < 0) mu = -mu;
    if (mu > 1) mu = 1;
    double x = mu * (m->n_inc - 1);
    int j = (int)floor(x);
    if (j > m->n_inc - 2) j = m->n_inc - 2;
    double w = x - j;
    for (int s = 0; s < 4; ++s)
        a[s] = (1 - w) * (double)m->opac[4*j + s] + w * (double)m->opac[4*(j+1) + s];
}

static void cell_bhat(const ora_model* m, int64_t c, double b[3])
{
    if (m->bhat) { b[0] = m->bhat[3*c]; b[1] = m->bhat[3*c+1]; b[2] = m->bhat[3*c+2]; }
    else { b[0] = 0; b[1] = 0; b[2] = 1; }
}

static double mu_of(const double n[3], const double b[3])
{
    return fabs(dot3(n, b)) / sqrt(dot3(n, n) * dot3(b, b));
}

/* A11/R11b  distance to the cell's exit face from the cell-local position
 * p in [0,1]^3 (units of the cell size); ties resolved x before y before z. */
double ora_dda_exit(const ora_model* m, const double p[3], const double n[3], int* axis)
{
    double best = INFINITY; int ax = -1;
    for (int a = 0; a < 3; ++a) {
        double t;
        if (n[a] > 0)      t = (1.0 - p[a]) * m->d[a] / n[a];
        else if (n[a] < 0) t = p[a] * m->d[a] / (-n[a]);
        else continue;
        if (t < best) { best = t; ax = a; }
    }
    *axis = ax;
    return best;
}

/* move ds along n inside the cell; if axis >= 0 also cross that face.
 * Returns 0 when the packet leaves the grid. */
static int advance_w(const ora_model* m, int idx[3], double p[3], const double n[3], double ds, int axis, int* wraps)
{
    int nn[3] = { m->nx, m->ny, m->nz };
    for (int a = 0; a < 3; ++a) {
        if (a == axis) continue;
        p[a] += n[a] * ds / m->d[a];
        if (p[a] < 0) p[a] = 0;
        if (p[a] > 1) p[a] = 1;
    }
    if (axis >= 0) {
        if (n[axis] > 0) { idx[axis] += 1; p[axis] = 0.0; }
        else             { idx[axis] -= 1; p[axis] = 1.0; }
        if (idx[axis] < 0 || idx[axis] >= nn[axis]) {
            if (!((m->periodic >> axis) & 1) || !wraps || *wraps >= ORA_MAX_WRAPS) return 0;
            ++*wraps;                                                  /* R20 */
            idx[axis] = idx[axis] < 0 ? nn[axis] - 1 : 0;
        }
    }
    return 1;
}
static int advance(const ora_model* m, int idx[3], double p[3], const double n[3], double ds, int axis)
{
    return advance_w(m, idx, p, n, ds, axis, NULL);
}

static int64_t cell_of(const ora_model* m, const int idx[3])
{
    return ((int64_t)idx[2] * m->ny + idx[1]) * m->nx + idx[0];
}

/* S3  one cell: lab -> grain frame (eq. 2,3,6,7), App. A over dtau, back. */
void ora_cell_step(const ora_model* m, const double b[3], const double n[3], double S[4], double dtau)
{
    double a[4];
    ora_opac_at(m, mu_of(n, b), a);
    if (a[1] == 0.0 && a[2] == 0.0) {           /* exact no-op of the rotation */
        double e = exp(-a[0] * dtau);
        for (int s = 0; s < 4; ++s) S[s] *= e;
        return;
    }
    double q[4], ce, se;
    ora_quat_from_B(b, q);
    ora_eta_gf(q, n, &ce, &se);
    ora_rotate_qu(S, ce, se);
    ora_appA(S, a[0], a[1], a[2], dtau);
    ora_rotate_qu(S, ce, -se);
}

/* March from (idx,p) along n to the grid edge with no survival test
 * (imaging leg; also used by the slab pins).  Optionally logs
 * the visited cells and segment lengths.  Returns the number of cell steps. */
int64_t ora_march(const ora_model* m, const int idx0[3], const double p0[3], const double n[3],
                  double S[4], int64_t log_cap, int64_t* log_cell, double* log_ds)
{
    int idx[3] = { idx0[0], idx0[1], idx0[2] };
    double p[3] = { p0[0], p0[1], p0[2] };
    int64_t steps = 0;
    int wraps = 0;
    for (;;) {
        int axis; double ds = ora_dda_exit(m, p, n, &axis);
        int64_t c = cell_of(m, idx);
        if (steps < log_cap) { if (log_cell) log_cell[steps] = c; if (log_ds) log_ds[steps] = ds; }
        ++steps;
        double kr = m->kr[c];
        if (kr > 0) { double b[3]; cell_bhat(m, c, b); ora_cell_step(m, b, n, S, kr * ds); }
        if (!advance_w(m, idx, p, n, ds, axis, &wraps)) break;
    }
    return steps;
}

/* ------------------------------------------------------------------ */
/* S5  scattering                                                      */
/* ------------------------------------------------------------------ */
/* Theta (degrees) from the piecewise-linear CDF of S11 sin(Theta), R13 */
double ora_sample_theta(const ora_model* m, double u)
{
    int lo = 0, hi = m->n_ang - 1;            /* cdf[lo] <= u < cdf[hi] */
    while (hi - lo > 1) { int mid = (lo + hi) / 2; if (m->cdf[mid] <= u) lo = mid; else hi = mid; }
    double w = m->cdf[lo+1] - m->cdf[lo];
    double f = (w > 0) ? (u - m->cdf[lo]) / w : 0.5;
    return (lo + f) * 180.0 / (m->n_ang - 1);
}

/* rejection test for the azimuth (after Whitney & Wolff 2002) */
int ora_phi_accept(double p12, double q, double u, double phi, double uacc)
{
    double bound = 1.0 + fabs(p12) * sqrt(q*q + u*u);
    return uacc * bound < 1.0 + p12 * (q * cos(2*phi) + u * sin(2*phi));
}

/* Deterministic part of S5: given the angles, rotate lab -> grain frame,
 * scatter with F(Theta), rotate back.  S is normalised (1,q,u,v) in the lab
 * reference of n_in on entry and of n_out on exit.  n_out is rounded to
 * fp32 (R12) BEFORE the exit reference is taken.                           */
void ora_scatter_angles(const ora_model* m, const double b[3], const double n_in[3],
                        const double S_in[4], double theta_deg, double phi,
                        double n_out[3], double S_out[4])
{
    double q[4], ce, se, ng[3], thp[3], php[3];
    ora_quat_from_B(b, q);
    ora_rot_to_gf(q, n_in, ng);
    double nn = sqrt(dot3(ng, ng));
    for (int a = 0; a < 3; ++a) ng[a] /= nn;
    double S[4] = { S_in[0], S_in[1], S_in[2], S_in[3] };
    ora_eta_gf(q, n_in, &ce, &se);
    ora_rotate_qu(S, ce, se);                               /* reference theta^' */
    ora_basis(ng, thp, php);
    double ct = cos(theta_deg * ORA_PI / 180.0), st = sin(theta_deg * ORA_PI / 180.0);
    double cp = cos(phi), sp = sin(phi);
    double epar[3], nout_g[3], eout[3], sh[3];
    for (int a = 0; a < 3; ++a) epar[a] = cp * thp[a] + sp * php[a];
    for (int a = 0; a < 3; ++a) nout_g[a] = ct * ng[a] + st * epar[a];
    ora_rotate_qu(S, cp, sp);                               /* reference e_par */
    double F[4];
    ora_mueller_at(m, theta_deg, F);
    double I = F[0]*S[0] + F[1]*S[1], Q = F[1]*S[0] + F[0]*S[1];
    double U = F[2]*S[2] + F[3]*S[3], V = -F[3]*S[2] + F[2]*S[3];
    S[0] = 1.0; S[1] = Q / I; S[2] = U / I; S[3] = V / I;
    /* scattering-plane reference of the outgoing ray -> theta^'' of n'_GF */
    for (int a = 0; a < 3; ++a) eout[a] = ct * epar[a] - st * ng[a];
    cross3(ng, epar, sh);
    double th2[3], ph2[3];
    ora_basis(nout_g, th2, ph2);
    ora_rotate_qu(S, dot3(eout, th2), dot3(th2, sh));
    /* back to the lab: direction by the inverse of eq. 3, then fp32 state */
    double nl[3];
    ora_rot_to_lab(q, nout_g, nl);
    for (int a = 0; a < 3; ++a) n_out[a] = (double)(float)nl[a];
    ora_eta_gf(q, n_out, &ce, &se);
    ora_rotate_qu(S, ce, -se);
    for (int s = 0; s < 4; ++s) S_out[s] = S[s];
}

/* Full S5 with the draws of event k of packet id (schedule R11).
 * Returns the number of azimuth rounds used. */
int ora_scatter(const ora_model* m, const double b[3], const double n_in[3], const double S_in[4],
                uint64_t seed, uint64_t id, uint32_t k, double n_out[3], double S_out[4], double* tau_next)
{
    uint32_t w[4];
    draw(seed, id, k, 0, w);
    double theta = ora_sample_theta(m, ora_u01(w[0]));
    *tau_next = -log(ora_u01(w[3]));
    double F[4];
    ora_mueller_at(m, theta, F);
    double p12 = F[1] / F[0];
    /* Stokes in the grain-frame reference decides the azimuth */
    double q[4], ce, se, S[4] = { S_in[0], S_in[1], S_in[2], S_in[3] };
    ora_quat_from_B(b, q);
    ora_eta_gf(q, n_in, &ce, &se);
    ora_rotate_qu(S, ce, se);
    double phi = 2 * ORA_PI * ora_u01(w[1]);
    int rounds = 1;
    int ok = ora_phi_accept(p12, S[1], S[2], phi, ora_u01(w[2]));
    for (uint32_t blk = 1; !ok && rounds < 64; ++blk) {
        draw(seed, id, k, blk, w);
        for (int h = 0; h < 2 && !ok && rounds < 64; ++h) {
            phi = 2 * ORA_PI * ora_u01(w[2*h]);
            ok = ora_phi_accept(p12, S[1], S[2], phi, ora_u01(w[2*h+1]));
            ++rounds;
        }
    }
    ora_scatter_angles(m, b, n_in, S_in, theta, phi, n_out, S_out);
    return rounds;
}

/* ------------------------------------------------------------------ */
/* S1-S5  transport                                                    */
/* ------------------------------------------------------------------ */
typedef struct ora_stats {
    uint64_t packets, events, records, steps_transport, steps_image, contributions, dropped, overflow;
    double w_emitted, w_escaped, w_absorbed, w_cut;
} ora_stats;

typedef struct ora_events {          /* caller-allocated SoA, capacity cap */
    int64_t cap, n;
    int64_t* cell; double* p; double* n_in; double* S; uint64_t* id; int32_t* k;
} ora_events;

static void push_event(ora_events* ev, ora_stats* st, int64_t cell, const double p[3], const double n[3],
                       const double S[4], double scale, uint64_t id, int k)
{
    if (ev->n >= ev->cap) { st->overflow++; return; }
    int64_t i = ev->n++;
    ev->cell[i] = cell; ev->id[i] = id; ev->k[i] = k;
    for (int a = 0; a < 3; ++a) { ev->p[3*i+a] = p[a]; ev->n_in[3*i+a] = n[a]; }
    for (int s = 0; s < 4; ++s) ev->S[4*i+s] = scale * S[s];
}

typedef struct ora_observer { double theta, phi, center[3], half_w, half_h; } ora_observer;

/* step 1 of the paper's two-step form (defined at the end of this file): optional hook of flight() */
struct ora_deposit;
static void deposit_segment(const ora_model* m, struct ora_deposit* dep, int64_t c, const double n[3], const double S_lab[4],
                            const double a[4], double ce, double se, int rotated, double T, double W);

/* One flight (S2-S4): start with I = 1; after every cell compare I with
 * e^{-tau*}; locate the event inside the cell with ora_event_solve.
 * Returns 1 at an event (S normalised to (1,q,u,v), idx/p at the event),
 * 0 when the packet left the grid. */
static int flight(const ora_model* m, int idx[3], double p[3], const double n[3], double S[4],
                  double tau_star, ora_stats* st, struct ora_deposit* dep, double W)
{
    double target = exp(-tau_star);
    int wraps = 0;
    for (;;) {
        int axis; double ds = ora_dda_exit(m, p, n, &axis);
        int64_t c = cell_of(m, idx);
        st->steps_transport++;
        double kr = m->kr[c];
        if (kr > 0) {
            double b[3], a[4];
            cell_bhat(m, c, b);
            ora_opac_at(m, mu_of(n, b), a);
            double dtau = kr * ds;
            if (a[1] == 0.0 && a[2] == 0.0) {
                double Iout = S[0] * exp(-a[0] * dtau);
                if (Iout <= target) {
                    double t = ora_event_solve(S[0], 0.0, a[0], 0.0, target);
                    if (dep) deposit_segment(m, dep, c, n, S, a, 1.0, 0.0, 0, t, W);
                    advance(m, idx, p, n, t / kr, -1);
                    for (int a2 = 0; a2 < 3; ++a2) p[a2] = ORA_STATE(p[a2]);   /* R12 */
                    double I = S[0];
                    for (int s = 0; s < 4; ++s) S[s] /= I;
                    return 1;
                }
                if (dep) deposit_segment(m, dep, c, n, S, a, 1.0, 0.0, 0, dtau, W);
                double e = exp(-a[0] * dtau);
                for (int s = 0; s < 4; ++s) S[s] *= e;
            } else {
                double q[4], ce, se, Sg[4], So[4];
                ora_quat_from_B(b, q);
                ora_eta_gf(q, n, &ce, &se);
                for (int s = 0; s < 4; ++s) Sg[s] = S[s];
                ora_rotate_qu(Sg, ce, se);
                for (int s = 0; s < 4; ++s) So[s] = Sg[s];
                ora_appA(So, a[0], a[1], a[2], dtau);
                if (So[0] <= target) {
                    double t = ora_event_solve(Sg[0], Sg[1] / Sg[0], a[0], a[1], target);
                    if (dep) deposit_segment(m, dep, c, n, S, a, ce, se, 1, t, W);
                    ora_appA(Sg, a[0], a[1], a[2], t);
                    double I = Sg[0];
                    for (int s = 0; s < 4; ++s) Sg[s] /= I;
                    ora_rotate_qu(Sg, ce, -se);
                    for (int s = 0; s < 4; ++s) S[s] = Sg[s];
                    advance(m, idx, p, n, t / kr, -1);
                    for (int a2 = 0; a2 < 3; ++a2) p[a2] = ORA_STATE(p[a2]);   /* R12 */
                    return 1;
                }
                if (dep) deposit_segment(m, dep, c, n, S, a, ce, se, 1, dtau, W);
                ora_rotate_qu(So, ce, -se);
                for (int s = 0; s < 4; ++s) S[s] = So[s];
            }
        }
        if (!advance_w(m, idx, p, n, ds, axis, &wraps)) return 0;
    }
}

/* S1 emission of packet id (draw schedule R11).  Exported as ora_emit / ora_emit_full for the pins.
 * Thermal emission by aligned grains (kind bit2, with bit0; PAPER.md:95-97 eq. 8, :145; reading R22): the source term of
 * eq. 8 is alpha_abs B with alpha_abs = (1 - omega) alpha (R19), i.e. per unit extinction depth the grain-frame vector
 * (1 - omega(mu)) (alpha1(mu), alpha2(mu), 0, 0) B.  A packet of the Monte-Carlo step therefore leaves its cell in a
 * direction drawn with density proportional to (1 - omega(mu)) alpha1(mu), mu = |n . B^| (rejection from isotropic
 * candidates against the table's maximum; candidate k uses block 0 (k = 0) or block 2 + k of event 0: words
 * (cos theta, phi, accept, tau* [block 0 only]); at most 64 candidates, the last one is taken), and carries
 * (1, alpha2/alpha1, 0, 0) in the grain-frame reference, turned into the lab reference of n (eq. 6-7). */
static void emit_full(const ora_model* m, uint64_t seed, uint64_t id, int idx[3], double p[3], double n[3], double* tau_star, double S[4])
{
    uint32_t w[4];
    draw(seed, id, 0, 0, w);
    *tau_star = -log(ora_u01(w[2]));
    S[0] = 1; S[1] = S[2] = S[3] = 0;
    if (m->src_kind & 1) {
        uint32_t w1[4], w2[4];
        draw(seed, id, 0, 1, w1);
        draw(seed, id, 0, 2, w2);
        double u = ora_u53(w1[0], w1[1]);
        int64_t c;
        if (m->src_cdf) {
            double x = u * m->src_cdf[m->ncell - 1];
            int64_t lo = -1, hi = m->ncell - 1;          /* smallest c with cdf[c] > x */
            while (hi - lo > 1) { int64_t mid = lo + (hi - lo) / 2; if (m->src_cdf[mid] > x) hi = mid; else lo = mid; }
            c = hi;
        } else {
            c = (int64_t)floor(u * (double)m->ncell);
            if (c > m->ncell - 1) c = m->ncell - 1;
        }
        idx[0] = (int)(c % m->nx); idx[1] = (int)((c / m->nx) % m->ny); idx[2] = (int)(c / ((int64_t)m->nx * m->ny));
        for (int a = 0; a < 3; ++a) p[a] = ora_u01(w2[a]);
    } else {
        for (int a = 0; a < 3; ++a) { idx[a] = m->src_idx[a]; p[a] = ORA_STATE(m->src_p[a]); }   /* R12 */
    }
    if (m->src_kind & 2) {
        for (int a = 0; a < 3; ++a) n[a] = m->src_dir[a];
        for (int a = 0; a < 3; ++a) n[a] = (double)(float)n[a];          /* R12 */
        return;
    }
    int thermal = (m->src_kind & 4) && (m->src_kind & 1);
    double b[3] = { 0, 0, 1 }, emax = 0.0;
    if (thermal) {
        cell_bhat(m, cell_of(m, idx), b);
        for (int j = 0; j < m->n_inc; ++j) {
            double e = (1.0 - (double)m->opac[4*j+3]) * (double)m->opac[4*j];
            if (e > emax) emax = e;
        }
    }
    for (int k = 0; ; ++k) {
        if (k > 0) draw(seed, id, 0, 2 + k, w);
        double ct = 1.0 - 2.0 * ora_u01(w[0]);
        double st = sqrt(1.0 - ct * ct);
        double ph = 2 * ORA_PI * ora_u01(w[1]);
        n[0] = st * cos(ph); n[1] = st * sin(ph); n[2] = ct;
        for (int a = 0; a < 3; ++a) n[a] = (double)(float)n[a];          /* R12 */
        if (!thermal) return;
        double a[4];
        ora_opac_at(m, mu_of(n, b), a);
        if (ora_u01(w[k == 0 ? 3 : 2]) * emax < (1.0 - a[3]) * a[0] || k >= 63) {
            S[1] = a[1] / a[0];
            if (a[1] != 0.0) {
                double q[4], ce, se;
                ora_quat_from_B(b, q);
                ora_eta_gf(q, n, &ce, &se);
                ora_rotate_qu(S, ce, -se);
            }
            for (int s2 = 1; s2 < 4; ++s2) S[s2] = ORA_STATE(S[s2]);      /* R12: queue state */
            return;
        }
    }
}

static void emit(const ora_model* m, uint64_t seed, uint64_t id, int idx[3], double p[3], double n[3], double* tau_star)
{
    double S[4];
    emit_full(m, seed, id, idx, p, n, tau_star, S);
}

void ora_emit_full(const ora_model* m, uint64_t seed, uint64_t id, int idx[3], double p[3], double n[3], double* tau_star, double S[4])
{
    emit_full(m, seed, id, idx, p, n, tau_star, S);
}

void ora_emit(const ora_model* m, uint64_t seed, uint64_t id, int idx[3], double p[3], double n[3], double* tau_star)
{
    emit(m, seed, id, idx, p, n, tau_star);
}

/* Transport packets [id0, id0+n).  esc_* (optional, capacity esc_cap): the
 * state of every packet that leaves the grid -- direction, W*(1,q,u,v) in
 * the lab reference of that direction, id -- used by the naive-estimator pin
 * (PAPER.md:115).  Returns the number of escape records written.          */
int64_t ora_transport2(const ora_model* m, uint64_t id0, uint64_t n_packets, uint64_t seed,
                       ora_events* ev, ora_stats* st,
                       int64_t esc_cap, double* esc_n, double* esc_S, uint64_t* esc_id, int32_t* esc_k,
                       struct ora_deposit* dep)
{
    int64_t nesc = 0;
    for (uint64_t id = id0; id < id0 + n_packets; ++id) {
        int idx[3]; double p[3], n[3], tau_star;
        double W = 1.0, S[4];
        emit_full(m, seed, id, idx, p, n, &tau_star, S);
        st->packets++; st->w_emitted += W;
        if (m->emit_records) { push_event(ev, st, cell_of(m, idx), p, n, S, W, id, 0); st->records++; }
        int k = 0;
        for (;;) {
            if (!flight(m, idx, p, n, S, tau_star, st, dep, W)) {
                st->w_escaped += W;
                if (nesc < esc_cap) {
                    for (int a = 0; a < 3; ++a) esc_n[3*nesc+a] = n[a];
                    /* a surviving packet keeps its weight: Stokes renormalised to I = 1 (R7) */
                    for (int s = 0; s < 4; ++s) esc_S[4*nesc+s] = W * S[s] / S[0];
                    esc_id[nesc] = id; esc_k[nesc] = k;
                    ++nesc;
                }
                break;
            }
            ++k;
            for (int s = 1; s < 4; ++s) S[s] = ORA_STATE(S[s]);              /* R12: event record state */
            int64_t c = cell_of(m, idx);
            double b[3], a[4];
            cell_bhat(m, c, b);
            ora_opac_at(m, mu_of(n, b), a);
            double om = a[3];
            push_event(ev, st, c, p, n, S, om * W, id, k);
            st->events++;
            st->w_absorbed += (1 - om) * W;
            W *= om;
            if (W < m->w_min || k >= m->max_scatter) { st->w_cut += W; break; }
            double n2[3], S2[4];
            if (m->ztab) ora_scatter_z(m->ztab, b, n, S, seed, id, (uint32_t)k, n2, S2, &tau_star);
            else ora_scatter(m, b, n, S, seed, id, (uint32_t)k, n2, S2, &tau_star);
            for (int a2 = 0; a2 < 3; ++a2) n[a2] = n2[a2];
            for (int s = 0; s < 4; ++s) S[s] = ORA_STATE(S2[s]);             /* R12: queue state */
        }
    }
    return nesc;
}

int64_t ora_transport(const ora_model* m, uint64_t id0, uint64_t n_packets, uint64_t seed,
                      ora_events* ev, ora_stats* st,
                      int64_t esc_cap, double* esc_n, double* esc_S, uint64_t* esc_id, int32_t* esc_k)
{
    return ora_transport2(m, id0, n_packets, seed, ev, st, esc_cap, esc_n, esc_S, esc_id, esc_k, NULL);
}

/* ------------------------------------------------------------------ */
/* S6  imaging                                                         */
/* ------------------------------------------------------------------ */
/* I1 peel-off: Stokes sent toward n_obs by a scattering of the incoming
 * state (n_in, S in the lab reference of n_in), eq. 10-11.
 * Result in the reference theta^_obs, including the 1/(4 pi).             */
void ora_peel(const ora_model* m, const double n_in[3], const double S_in[4], const double n_obs[3], double S_out[4])
{
    double th[3], ph[3], tho[3], pho[3], sh[3], epar[3], eout[3];
    ora_basis(n_in, th, ph);
    ora_basis(n_obs, tho, pho);
    double mu = dot3(n_in, n_obs) / sqrt(dot3(n_in, n_in) * dot3(n_obs, n_obs));
    if (mu > 1) mu = 1;
    if (mu < -1) mu = -1;
    cross3(n_in, n_obs, sh);
    double sn = sqrt(dot3(sh, sh));
    if (sn < 1e-12) { for (int a = 0; a < 3; ++a) sh[a] = ph[a]; }
    else            { for (int a = 0; a < 3; ++a) sh[a] /= sn; }
    cross3(sh, n_in, epar);
    double S[4] = { S_in[0], S_in[1], S_in[2], S_in[3] };
    ora_rotate_qu(S, dot3(th, epar), dot3(ph, epar));
    double F[4];
    ora_mueller_at(m, acos(mu) * 180.0 / ORA_PI, F);
    double I = F[0]*S[0] + F[1]*S[1], Q = F[1]*S[0] + F[0]*S[1];
    double U = F[2]*S[2] + F[3]*S[3], V = -F[3]*S[2] + F[2]*S[3];
    S[0] = I; S[1] = Q; S[2] = U; S[3] = V;
    cross3(sh, n_obs, eout);
    ora_rotate_qu(S, dot3(eout, tho), dot3(tho, sh));
    for (int s = 0; s < 4; ++s) S_out[s] = S[s] / (4 * ORA_PI);
}

/* Image every event toward every observer.  img/img2: [n_obs][4][ny][nx]
 * sums and sums of squares.  flags bit0: also image emission records (k=0)
 * as isotropic unpolarized emitters.                                     */
void ora_image(const ora_model* m, const ora_events* ev, const ora_observer* obs, int n_obs,
               int npx, int npy, int flags, double* img, double* img2, ora_stats* st)
{
    for (int64_t e = 0; e < ev->n; ++e) {
        int64_t c = ev->cell[e];
        int idx[3] = { (int)(c % m->nx), (int)((c / m->nx) % m->ny), (int)(c / ((int64_t)m->nx * m->ny)) };
        const double* p = ev->p + 3*e;
        const double* nin = ev->n_in + 3*e;
        const double* Se = ev->S + 4*e;
        for (int o = 0; o < n_obs; ++o) {
            double no[3] = { sin(obs[o].theta) * cos(obs[o].phi), sin(obs[o].theta) * sin(obs[o].phi), cos(obs[o].theta) };
            double tho[3], pho[3], S[4];
            ora_basis(no, tho, pho);
            if (ev->k[e] == 0) {
                if (!(flags & 1)) continue;
                S[0] = Se[0] / (4 * ORA_PI); S[1] = S[2] = S[3] = 0.0;
            } else if (m->ztab) {
                double b[3];
                cell_bhat(m, c, b);
                ora_peel_z(m->ztab, b, nin, Se, no, S);
            } else {
                ora_peel(m, nin, Se, no, S);
            }
            st->steps_image += (uint64_t)ora_march(m, idx, p, no, S, 0, NULL, NULL);
            double x[3];
            for (int a = 0; a < 3; ++a) x[a] = m->lo[a] + (idx[a] + p[a]) * m->d[a] - obs[o].center[a];
            double xi =  dot3(x, pho) / obs[o].half_w;
            double yi = -dot3(x, tho) / obs[o].half_h;
            int ix = (int)floor((xi + 1.0) * npx / 2.0), iy = (int)floor((yi + 1.0) * npy / 2.0);
            if (ix < 0 || ix >= npx || iy < 0 || iy >= npy) { st->dropped++; continue; }
            st->contributions++;
            for (int s = 0; s < 4; ++s) {
                int64_t at = (((int64_t)o * 4 + s) * npy + iy) * npx + ix;
                img[at] += S[s];
                if (img2) img2[at] += S[s] * S[s];
            }
        }
    }
}

/* ================================================================== */
/* NEXT-1 / NEXT-3: the paper's own two-step form (PAPER.md:113-123,   */
/* eq. 11) and the in-cell solution WITH source terms (App. A,         */
/* PAPER.md:296-328).  DESIGN.md section 12 states the readings.       */
/* ================================================================== */

/* A12 with sources: PAPER.md:302-328 (eq. A2-A3) with the matrix of R1.  src = (S1..S4) is the source per unit
 * extinction optical depth, constant in the cell, in the same (grain-frame) reference as S.  The printed solution
 * is the source-free one applied to S - S_s, plus S_s, with the stationary vector S_s of eq. A3. */
void ora_appA_src(double S[4], double a1, double a2, double a3, const double src[4], double dtau)
{
    double Is = (a1 * src[0] - a2 * src[1]) / (a1 * a1 - a2 * a2);
    double Qs = (a1 * src[1] - a2 * src[0]) / (a1 * a1 - a2 * a2);
    double Us = (a1 * src[2] - a3 * src[3]) / (a1 * a1 + a3 * a3);
    double Vs = (a1 * src[3] + a3 * src[2]) / (a1 * a1 + a3 * a3);
    double D[4] = { S[0] - Is, S[1] - Qs, S[2] - Us, S[3] - Vs };
    ora_appA(D, a1, a2, a3, dtau);
    S[0] = Is + D[0]; S[1] = Qs + D[1]; S[2] = Us + D[2]; S[3] = Vs + D[3];
}

/* 16-point Gauss-Legendre nodes and weights on [-1,1], by Newton on P_16 (textbook construction) */
static void gl16(double x[16], double w[16])
{
    const int n = 16;
    for (int i = 0; i < n; ++i) {
        double z = cos(ORA_PI * (i + 0.75) / (n + 0.5)), pp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 0; j < n; ++j) { double p3 = p2; p2 = p1; p1 = ((2.0 * j + 1.0) * z * p2 - j * p3) / (j + 1.0); }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            double dz = p1 / pp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        x[i] = z; w[i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

/* Step 1 of the two-step scheme, one path segment ("each path integration segment (i.e., not only
 * at scattering events) contributes to a scattering source function stored on the grid", S_pp = Z(Omega_cam;Omega_pp) I_pp).
 * Reading R18: the deposit is the track-length form of the very estimator the event form uses.  A packet
 * that is alive at extinction depth tau inside the segment has the normalised state s^(tau) = S~(tau)/I~(tau) (R7; S~ the
 * source-free App. A solution from the state Sg at the start of the segment, grain-frame reference) and collides at the
 * rate r(tau) = -I~'/I~ = alpha1 + alpha2 q^_g(tau) per unit depth, every collision sending out omega W Z s^.  The
 * expected collision output of the segment is therefore omega W Z J with
 *        J = int_0^T r(tau) s^(tau) dtau ,
 * which this function returns (4 components, grain-frame reference; J[0] = expected number of collisions).  J[0] and
 * J[1] have closed forms (pins); U and V do not, so all four are evaluated by composite 16-point Gauss-Legendre
 * quadrature on sub-intervals of (|alpha2| + |alpha3|) h <= 0.5 (integrand analytic: error far below 1e-15). */
void ora_segment_integral(const double Sg[4], double a1, double a2, double a3, double T, double J[4])
{
    static double gx[16], gw[16]; static int have = 0;
    if (!have) { gl16(gx, gw); have = 1; }
    for (int s = 0; s < 4; ++s) J[s] = 0.0;
    if (!(T > 0.0)) return;
    int nsub = (int)ceil((fabs(a2) + fabs(a3)) * T / 0.5);
    if (nsub < 1) nsub = 1;
    double h = T / nsub;
    for (int k = 0; k < nsub; ++k) {
        for (int i = 0; i < 16; ++i) {
            double tau = (k + 0.5 * (gx[i] + 1.0)) * h;
            double S[4] = { Sg[0], Sg[1], Sg[2], Sg[3] };
            /* e^{+alpha1 tau} is divided out analytically: only ratios of the solution enter */
            ora_appA(S, 0.0, a2, a3, tau);
            double r = a1 + a2 * S[1] / S[0];
            for (int s = 0; s < 4; ++s) J[s] += 0.5 * h * gw[i] * r * S[s] / S[0];
        }
    }
}

/* what step 1 accumulates: sgrid[ncell][n_obs][4], the expected collision output toward every camera in the reference
 * theta^_obs, including omega W and the 1/(4 pi) of the peel-off, NOT attenuated (step 2 does that) and not divided by
 * the cell volume; coll[ncell] (optional) = expected number of collisions times W (pin against the event counts). */
typedef struct ora_deposit {
    const ora_observer* obs; int n_obs;
    double* sgrid; double* coll;
    uint64_t segments;
} ora_deposit;

static void deposit_segment(const ora_model* m, ora_deposit* dep, int64_t c, const double n[3], const double S_lab[4],
                            const double a[4], double ce, double se, int rotated, double T, double W)
{
    /* S_lab: state at the start of the segment in the lab reference of n; (ce, se): eta of eq. 6-7 when the cell is dichroic */
    double Sg[4] = { S_lab[0], S_lab[1], S_lab[2], S_lab[3] }, J[4];
    if (rotated) ora_rotate_qu(Sg, ce, se);
    ora_segment_integral(Sg, a[0], a[1], a[2], T, J);
    if (rotated) ora_rotate_qu(J, ce, -se);
    if (dep->coll) dep->coll[c] += W * J[0];
    double Jw[4] = { a[3] * W * J[0], a[3] * W * J[1], a[3] * W * J[2], a[3] * W * J[3] };
    for (int o = 0; o < dep->n_obs; ++o) {
        double no[3] = { sin(dep->obs[o].theta) * cos(dep->obs[o].phi), sin(dep->obs[o].theta) * sin(dep->obs[o].phi), cos(dep->obs[o].theta) };
        double out[4];
        ora_peel(m, n, Jw, no, out);
        for (int s = 0; s < 4; ++s) dep->sgrid[((int64_t)c * dep->n_obs + o) * 4 + s] += out[s];
    }
    dep->segments++;
}

/* step 1 for packets [id0, id0+n): the ordinary transport (same packets, same events) with every path segment also
 * deposited into sgrid / coll (either may be NULL) */
void ora_transport_deposit(const ora_model* m, uint64_t id0, uint64_t n_packets, uint64_t seed, ora_events* ev, ora_stats* st,
                           const ora_observer* obs, int n_obs, double* sgrid, double* coll, uint64_t* n_segments)
{
    ora_deposit dep = { obs, n_obs, sgrid, coll, 0 };
    ora_transport2(m, id0, n_packets, seed, ev, st, 0, NULL, NULL, NULL, NULL, &dep);
    if (n_segments) *n_segments = dep.segments;
}

/* Step 2: "a deterministic ray-tracing step by integrating eq. (8) along lines of sight toward the
 * camera ... with the same cell-by-cell analytic integration": one ray per pixel, through the pixel centre, from the far
 * side of the grid toward the observer, App. A WITH source terms in every cell.  Sources per unit extinction depth in
 * cell c (reference theta^_obs, rotated into the grain frame for the solve):
 *    scattering   sgrid[c][o][:] / (V_c kappa rho_c)        (step 1; V_c = cell volume)
 *    thermal      (1 - omega) (alpha1, alpha2, 0, 0)_GF B_c  (eq. 8: alpha_abs B with B ~ (1,0,0,0); reading R19:
 *                 alpha_abs = (1 - omega) alpha; emis[c] = B_c, may be NULL)
 * The pixel receives radiance times the pixel's area (R14: image units are sums of packet contributions per pixel).
 * img[n_obs][4][npy][npx] is added to. */
void ora_image_rays(const ora_model* m, const double* sgrid, const float* emis, const ora_observer* obs, int n_obs,
                    int npx, int npy, double* img, ora_stats* st)
{
    const int nn[3] = { m->nx, m->ny, m->nz };
    const double vol = m->d[0] * m->d[1] * m->d[2];
    for (int o = 0; o < n_obs; ++o) {
        double no[3] = { sin(obs[o].theta) * cos(obs[o].phi), sin(obs[o].theta) * sin(obs[o].phi), cos(obs[o].theta) };
        double tho[3], pho[3];
        ora_basis(no, tho, pho);
        const double apix = (2.0 * obs[o].half_w / npx) * (2.0 * obs[o].half_h / npy);
        for (int iy = 0; iy < npy; ++iy) for (int ix = 0; ix < npx; ++ix) {
            /* pixel centre on the image plane (R14: x along phi^_obs, y along -theta^_obs) */
            double xi = ((ix + 0.5) * 2.0 / npx - 1.0) * obs[o].half_w, yi = ((iy + 0.5) * 2.0 / npy - 1.0) * obs[o].half_h;
            double x0[3];
            for (int a = 0; a < 3; ++a) x0[a] = obs[o].center[a] + xi * pho[a] - yi * tho[a];
            /* the line x0 + s n_obs against the box: slab method */
            double s_in = -INFINITY, s_out = INFINITY; int miss = 0;
            for (int a = 0; a < 3; ++a) {
                double lo = m->lo[a], hi = m->lo[a] + nn[a] * m->d[a];
                if ((m->periodic >> a) & 1) continue;                     /* R20: a periodic axis does not clip the line ... */
                if (no[a] == 0.0) { if (x0[a] < lo || x0[a] >= hi) miss = 1; continue; }
                double t0 = (lo - x0[a]) / no[a], t1 = (hi - x0[a]) / no[a];
                if (t0 > t1) { double t = t0; t0 = t1; t1 = t; }
                if (t0 > s_in) s_in = t0;
                if (t1 < s_out) s_out = t1;
            }
            if (miss || !(s_in < s_out) || s_in == -INFINITY) continue;
            int idx[3]; double p[3];
            for (int a = 0; a < 3; ++a) {
                double x = (x0[a] + s_in * no[a] - m->lo[a]) / m->d[a];
                if ((m->periodic >> a) & 1) x -= floor(x / nn[a]) * nn[a];  /* ... its coordinate is taken modulo the box */
                int i = (int)floor(x);
                if (i < 0) i = 0;
                if (i > nn[a] - 1) i = nn[a] - 1;
                double f = x - i;
                idx[a] = i; p[a] = f < 0 ? 0 : (f > 1 ? 1 : f);
            }
            double S[4] = { 0, 0, 0, 0 };
            int wraps = 0;
            for (;;) {
                int axis; double ds = ora_dda_exit(m, p, no, &axis);
                int64_t c = cell_of(m, idx);
                if (st) st->steps_image++;
                double kr = m->kr[c];
                if (kr > 0) {
                    double b[3], a[4], src[4] = { 0, 0, 0, 0 };
                    cell_bhat(m, c, b);
                    ora_opac_at(m, mu_of(no, b), a);
                    if (sgrid) for (int s = 0; s < 4; ++s) src[s] = sgrid[((int64_t)c * n_obs + o) * 4 + s] / (vol * kr);
                    double q[4], ce = 1.0, se = 0.0;
                    int rot = !(a[1] == 0.0 && a[2] == 0.0);
                    if (rot) { ora_quat_from_B(b, q); ora_eta_gf(q, no, &ce, &se); ora_rotate_qu(S, ce, se); ora_rotate_qu(src, ce, se); }
                    if (emis) { src[0] += (1.0 - a[3]) * a[0] * (double)emis[c]; src[1] += (1.0 - a[3]) * a[1] * (double)emis[c]; }
                    ora_appA_src(S, a[0], a[1], a[2], src, kr * ds);
                    if (rot) ora_rotate_qu(S, ce, -se);
                }
                if (!advance_w(m, idx, p, no, ds, axis, &wraps)) break;
            }
            if (st) st->contributions++;
            for (int s = 0; s < 4; ++s) img[(((int64_t)o * 4 + s) * npy + iy) * npx + ix] += apix * S[s];
        }
    }
}

/* ================================================================== */
/* NEXT-2: the full aligned-grain scattering matrix Z(Omega; Omega')   */
/* in the grain frame (PAPER.md:103-105 eq. 10, :107-109, :129).       */
/* Reading R21.  The dipole formulas of the     */
/* paper's grain model are not in the paper's text, so Z is a user     */
/* table ("interpolation tables"):                        */
/*   Z[i][o][d][4][4], incidence angle vartheta_in = i 180/(n_ti-1),   */
/*   outgoing polar angle vartheta_out = o 180/(n_to-1), azimuth       */
/*   difference dphi = phi_out - phi_in = d 360/n_dp (periodic), all   */
/*   in the Grain Frame (z_GF = B^); both Stokes vectors referenced to */
/*   (theta^', phi^') of their own direction in that frame (eq. 4-5).  */
/*   Trilinear interpolation in the three angles.                      */
/* ================================================================== */
typedef struct ora_ztable {
    int n_ti, n_to, n_dp;
    float* Z;            /* owned copy of the caller's fp32 table */
    double* norm;        /* [n_ti][4]: (1/4pi) closed-surface integral of row 1 of Z over outgoing directions, per incidence node */
    double* bound;       /* [n_ti]: max over outgoing nodes of Z11 + sqrt(Z12^2 + Z13^2 + Z14^2) */
} ora_ztable;

void ora_ztable_free(ora_ztable* z) { if (z) { free(z->Z); free(z->norm); free(z->bound); free(z); } }

ora_ztable* ora_ztable_create(int n_ti, int n_to, int n_dp, const float* Z)
{
    ora_ztable* z = (ora_ztable*)calloc(1, sizeof(ora_ztable));
    z->n_ti = n_ti; z->n_to = n_to; z->n_dp = n_dp;
    size_t n = (size_t)n_ti * n_to * n_dp * 16;
    z->Z = (float*)malloc(sizeof(float) * n);
    memcpy(z->Z, Z, sizeof(float) * n);
    z->norm = (double*)calloc((size_t)n_ti * 4, sizeof(double));
    z->bound = (double*)calloc((size_t)n_ti, sizeof(double));
    /* per incidence node: trapezoid in vartheta_out of sin(vartheta_out) x (mean over the dphi nodes), times 1/2
     * (= (1/4pi) int dOmega), for the four elements of row 1; and the bound of the rejection sampler */
    double dth = ORA_PI / (n_to - 1);
    for (int i = 0; i < n_ti; ++i) {
        for (int o = 0; o < n_to; ++o) {
            double w = (o == 0 || o == n_to - 1 ? 0.5 : 1.0) * sin(o * dth) * dth * 0.5;
            for (int d = 0; d < n_dp; ++d) {
                const float* e = z->Z + (((size_t)i * n_to + o) * n_dp + d) * 16;
                for (int s = 0; s < 4; ++s) z->norm[4 * i + s] += w * (double)e[s] / n_dp;
                double b = (double)e[0] + sqrt((double)e[1] * e[1] + (double)e[2] * e[2] + (double)e[3] * e[3]);
                if (b > z->bound[i]) z->bound[i] = b;
            }
        }
    }
    return z;
}

/* trilinear interpolation; angles in degrees, dphi any real (periodic) */
void ora_ztable_at(const ora_ztable* z, double ti_deg, double to_deg, double dphi_deg, double M[16])
{
    double xi = ti_deg * (z->n_ti - 1) / 180.0, xo = to_deg * (z->n_to - 1) / 180.0;
    double xd = dphi_deg * z->n_dp / 360.0;
    xd -= floor(xd / z->n_dp) * z->n_dp;
    int i = (int)floor(xi), o = (int)floor(xo), d = (int)floor(xd);
    if (i < 0) i = 0;
    if (i > z->n_ti - 2) i = z->n_ti - 2;
    if (o < 0) o = 0;
    if (o > z->n_to - 2) o = z->n_to - 2;
    if (d > z->n_dp - 1) d = z->n_dp - 1;
    double wi = xi - i, wo = xo - o, wd = xd - d;
    int d1 = (d + 1) % z->n_dp;
    for (int k = 0; k < 16; ++k) M[k] = 0.0;
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) for (int c = 0; c < 2; ++c) {
        double w = (a ? wi : 1 - wi) * (b ? wo : 1 - wo) * (c ? wd : 1 - wd);
        const float* e = z->Z + (((size_t)(i + a) * z->n_to + (o + b)) * z->n_dp + (c ? d1 : d)) * 16;
        for (int k = 0; k < 16; ++k) M[k] += w * (double)e[k];
    }
}

/* (1/4pi) int dOmega_out of the scattered intensity for the grain-frame state S (any normalisation), incidence angle ti:
 * linear interpolation of the per-node integrals.  It normalises the phase function: the probability density of the
 * outgoing direction is I_out / (4 pi N). */
double ora_ztable_norm(const ora_ztable* z, double ti_deg, const double Sg[4])
{
    double xi = ti_deg * (z->n_ti - 1) / 180.0;
    int i = (int)floor(xi);
    if (i < 0) i = 0;
    if (i > z->n_ti - 2) i = z->n_ti - 2;
    double w = xi - i, N = 0.0;
    for (int s = 0; s < 4; ++s) N += ((1 - w) * z->norm[4 * i + s] + w * z->norm[4 * (i + 1) + s]) * Sg[s];
    return N;
}

static void angles_gf(const double v[3], double* polar_deg, double* azim_deg)
{
    double r = sqrt(dot3(v, v));
    double c = v[2] / r;
    if (c > 1) c = 1;
    if (c < -1) c = -1;
    *polar_deg = acos(c) * 180.0 / ORA_PI;
    *azim_deg = (v[0] * v[0] + v[1] * v[1] >= 1e-24) ? atan2(v[1], v[0]) * 180.0 / ORA_PI : 0.0;
}

/* Peel-off with the full Z: Stokes vector sent toward n_obs by a scattering of the state S_in (lab reference of n_in) on a
 * grain aligned with b: into the grain frame (eq. 2, 3, 6, 7), Z s, back to the reference theta^_obs; divided by 4 pi N so
 * that its I component integrates to S_in[0] over all observer directions. */
void ora_peel_z(const struct ora_ztable* z, const double b[3], const double n_in[3], const double S_in[4], const double n_obs[3],
                double S_out[4])
{
    double q[4], ce, se, ng[3], og[3], ti, pi_, to, po, M[16];
    ora_quat_from_B(b, q);
    ora_rot_to_gf(q, n_in, ng);
    ora_rot_to_gf(q, n_obs, og);
    double S[4] = { S_in[0], S_in[1], S_in[2], S_in[3] };
    ora_eta_gf(q, n_in, &ce, &se);
    ora_rotate_qu(S, ce, se);
    angles_gf(ng, &ti, &pi_);
    angles_gf(og, &to, &po);
    ora_ztable_at(z, ti, to, po - pi_, M);
    double N = ora_ztable_norm(z, ti, S);
    double R[4];
    for (int r = 0; r < 4; ++r) R[r] = (M[4*r] * S[0] + M[4*r+1] * S[1] + M[4*r+2] * S[2] + M[4*r+3] * S[3]) / (4 * ORA_PI * N) * S[0];
    /* (the event's weight rides on S[0]: the phase function is normalised for the state s = S/S[0]; N is linear in S) */
    ora_eta_gf(q, n_obs, &ce, &se);
    ora_rotate_qu(R, ce, -se);
    for (int r = 0; r < 4; ++r) S_out[r] = R[r];
}

/* Scattering with the full Z (S5 with reading R21).  Rejection sampling of the outgoing direction (after
 * Whitney & Wolff 2002): candidates isotropic in the grain frame, cos(vartheta_out) = 1 - 2u, dphi = 2 pi u', accepted when
 * u'' * bound < I_out(candidate) = row 1 of Z . s, bound = the larger of the two bracketing incidence nodes' bounds.
 * Draws (R11): block 0 of event k = (cos, dphi, accept, next tau*), block b >= 1 = (cos, dphi, accept, -), at most 256
 * candidates (the last one is taken).  Returns the number of candidates used. */
int ora_scatter_z(const struct ora_ztable* z, const double b[3], const double n_in[3], const double S_in[4],
                  uint64_t seed, uint64_t id, uint32_t k, double n_out[3], double S_out[4], double* tau_next)
{
    double q[4], ce, se, ng[3], ti, pi_;
    ora_quat_from_B(b, q);
    ora_rot_to_gf(q, n_in, ng);
    double S[4] = { 1.0, S_in[1] / S_in[0], S_in[2] / S_in[0], S_in[3] / S_in[0] };
    ora_eta_gf(q, n_in, &ce, &se);
    ora_rotate_qu(S, ce, se);
    angles_gf(ng, &ti, &pi_);
    double xi = ti * (z->n_ti - 1) / 180.0;
    int i = (int)floor(xi);
    if (i < 0) i = 0;
    if (i > z->n_ti - 2) i = z->n_ti - 2;
    double bound = z->bound[i] > z->bound[i + 1] ? z->bound[i] : z->bound[i + 1];
    uint32_t w[4];
    double M[16], to = 0, dp = 0;
    int rounds = 0;
    for (uint32_t blk = 0; ; ++blk) {
        draw(seed, id, k, blk, w);
        if (blk == 0) *tau_next = -log(ora_u01(w[3]));
        double ct = 1.0 - 2.0 * ora_u01(w[0]);
        to = acos(ct) * 180.0 / ORA_PI;
        dp = 360.0 * ora_u01(w[1]);
        ora_ztable_at(z, ti, to, dp, M);
        double Iout = M[0] * S[0] + M[1] * S[1] + M[2] * S[2] + M[3] * S[3];
        ++rounds;
        if (ora_u01(w[2]) * bound < Iout || rounds >= 256) break;
    }
    double R[4];
    for (int r = 0; r < 4; ++r) R[r] = M[4*r] * S[0] + M[4*r+1] * S[1] + M[4*r+2] * S[2] + M[4*r+3] * S[3];
    double I = R[0];
    R[0] = 1.0; R[1] /= I; R[2] /= I; R[3] /= I;
    /* outgoing direction in the grain frame, then to the lab (inverse of eq. 3), fp32 state (R12) */
    double tr = to * ORA_PI / 180.0, pr = (pi_ + dp) * ORA_PI / 180.0;
    double og[3] = { sin(tr) * cos(pr), sin(tr) * sin(pr), cos(tr) }, nl[3];
    ora_rot_to_lab(q, og, nl);
    for (int a = 0; a < 3; ++a) n_out[a] = (double)(float)nl[a];
    ora_eta_gf(q, n_out, &ce, &se);
    ora_rotate_qu(R, ce, -se);
    for (int s = 0; s < 4; ++s) S_out[s] = R[s];
    return rounds;
}
