// krp_device.cuh -- device-side building blocks of the polarized MCRT hot path (sm_100a).
//
// Citations: PAPER.md:<line> is the extracted text of arxiv 2512.01283; R<n> are the readings
// in DESIGN.md.  Nothing here is shared with oracle/ (the fp64 CPU checker).
//
// Precision plan: the imaging march is fp32; whatever decides *where* a
// packet scatters is fp64 (scalar mode: the optical depth still to go, from fp32 segments; general
// mode: segments, alpha_i(mu), depth, normalised intensity and the Stokes vector); scattering
// geometry (once per event) is fp64 and the new direction is stored rounded to fp32 (R12).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define KRP_PI_D 3.14159265358979323846264338327950288
#define KRP_TERM_BIT 0x80000000u
#define KRP_MAX_OBS_PACK 8

// ------------------------------------------------------------------------------------------
// by-value kernel parameters
// ------------------------------------------------------------------------------------------
// full scattering matrix Z(Omega;Omega') of aligned grains in the grain frame (R21)
struct KrpZt {
    const float* zt;       // [ni][no][nd][16], or NULL
    const double* norm;    // [ni][4]  (1/4pi) integral of row 1 over outgoing directions
    const double* bound;   // [ni]     bound of the rejection sampler
    int ni, no, nd;
};

struct KrpModel {
    int nx, ny, nz;
    uint32_t ncell;
    // Padded layout: the cell arrays carry a one-cell halo on every side whose
    // kappa*rho is -1, so that a ray leaves the grid exactly when it loads a negative kappa*rho.  Cell ids
    // inside the library are indices into this padded array: ((iz+1)*py + iy+1)*px + ix+1.
    int px, py;            // padded pitches: px = nx+2, py = ny+2
    uint32_t pxy;          // px*py
    uint32_t px_m, px_s, py_m, py_s;   // division by px, py as multiply-high + shifts (krp_fastdiv)
    float d[3];            // cell size per axis
    double lo[3], dd[3];   // lower corner and cell size in fp64 (projection to the image)
    double inv_dd[3];      // 1/dd
    const float* kr;       // SCALAR mode: kappa*rho per padded cell
    const float4* cell;    // general mode: {kappa*rho, B^x, B^y, B^z} per padded cell
    const float4* opac;    // [n_inc] {alpha1, alpha2, alpha3, albedo} on mu_m = m/(n_inc-1)
    const float4* opA;     // [n_inc-1] intercepts and
    const float4* opB;     // [n_inc-1] slopes of the same table: value = opA[j] + opB[j]*x on x = mu*(n_inc-1) in [j, j+1]
    const double4* opA_d;  // the same in fp64 (general-mode flight)
    const double4* opB_d;
    int n_inc;
    double xs;             // n_inc - 1 as fp64 (x = mu*xs)
    float guard;           // 1 + rho + 1e-3: margin of the fp32 depth sum that arms the fp64 event test of the general flight
    const float4* mueller; // [n_ang] {S11,S12,S33,S34}
    int n_ang;
    double inv_nang1;      // 1/(n_ang-1)
    float nang1_over_pi;   // (n_ang-1)/pi: scattering angle in radians -> units of the table spacing
    const double* cdf;     // [n_ang] Theta CDF of S11 sin(Theta)
    float a1c, omc;        // SCALAR mode constants
    float rho;             // max |alpha2|/alpha1 over the table
    float w_min;
    int max_scatter;
    int scalar;
    uint32_t npad;         // padded cells (px * py * (nz+2)); the cell arrays have a margin of pxy elements on either side
    int periodic;          // bit a: axis a is periodic (R20); only with the 16-byte cell layout
    // full scattering matrix Z(Omega;Omega') of aligned grains in the grain frame (R21), or zt = NULL: F(Theta) of `mueller`
    KrpZt z;
    // source
    int src_kind, emit_records;
    float src_n[3];
    uint32_t src_cell;     // padded id
    float src_p[3];
    const double* src_cdf; // [ncell] running sum of cell weights (unpadded order) or NULL
    double src_emax;       // thermal source (kind bit 2, R22): max over the table nodes of (1 - omega) alpha1
};

// Bounds check of every cell gather, compiled in with -DKRP_CHECK only (profiles/r2_bounds_check.md; compute-sanitizer is
// closed on this pool): an index outside the allocation (padded array plus its margin of one plane on either side, which the
// look-ahead loads may touch) traps, and the next synchronising call of the library returns KRP_ERR_CUDA.
#ifdef KRP_CHECK
#define KRP_CK(g, c) do { const long long c_ = (long long)(int)(c); if (c_ < -(long long)(g).pxy || c_ >= (long long)(g).npad + (long long)(g).pxy) __trap(); } while (0)
#else
#define KRP_CK(g, c) do { } while (0)
#endif

__device__ __forceinline__ uint32_t krp_pad_id(const KrpModel& g, int ix, int iy, int iz)
{
    return ((uint32_t)(iz + 1) * (uint32_t)g.py + (uint32_t)(iy + 1)) * (uint32_t)g.px + (uint32_t)(ix + 1);
}
// floor(x / d) for any 32-bit x, with m = floor(2^32 (2^l - d) / d) + 1, l = ceil(log2 d), s = l - 1
// (round-up method of Granlund & Montgomery; d >= 2 here because d is a padded pitch >= 3)
__device__ __forceinline__ uint32_t krp_fastdiv(uint32_t x, uint32_t m, uint32_t s)
{
    const uint32_t t = __umulhi(x, m);
    return (((x - t) >> 1) + t) >> s;
}
// padded coordinates (0..n+1 per axis) of a padded id
__device__ __forceinline__ void krp_pad_coords(const KrpModel& g, uint32_t c, int& hx, int& hy, int& hz)
{
    const uint32_t t = krp_fastdiv(c, g.px_m, g.px_s);
    hx = (int)(c - t * (uint32_t)g.px);
    const uint32_t z = krp_fastdiv(t, g.py_m, g.py_s);
    hy = (int)(t - z * (uint32_t)g.py);
    hz = (int)z;
}

// Periodic boundaries (R20).  `c` is a halo cell, reached from an interior cell by crossing one face: exactly
// one of its padded coordinates is out of range.  If that axis is periodic, c becomes the cell behind the opposite face and
// off[axis] takes the jump (so that unwrapped coordinates can still be formed); returns false when the axis is open.
#define KRP_MAX_WRAPS 4096
__device__ __forceinline__ bool krp_wrap(const KrpModel& g, uint32_t& c, int off[3])
{
    int hx, hy, hz;
    krp_pad_coords(g, c, hx, hy, hz);
    if (hx == 0)              { if (!(g.periodic & 1)) return false; c += (uint32_t)g.nx; off[0] -= g.nx; }
    else if (hx == g.nx + 1)  { if (!(g.periodic & 1)) return false; c -= (uint32_t)g.nx; off[0] += g.nx; }
    else if (hy == 0)         { if (!(g.periodic & 2)) return false; c += (uint32_t)(g.ny * g.px); off[1] -= g.ny; }
    else if (hy == g.ny + 1)  { if (!(g.periodic & 2)) return false; c -= (uint32_t)(g.ny * g.px); off[1] += g.ny; }
    else if (hz == 0)         { if (!(g.periodic & 4)) return false; c += (uint32_t)g.nz * g.pxy; off[2] -= g.nz; }
    else if (hz == g.nz + 1)  { if (!(g.periodic & 4)) return false; c -= (uint32_t)g.nz * g.pxy; off[2] += g.nz; }
    else return false;
    return true;
}

struct KrpStatsDev {
    unsigned long long packets, events, records, steps_transport, steps_image, contributions, dropped, overflow;
    double w_emitted, w_escaped, w_absorbed, w_cut;
};

struct KrpCtl {
    unsigned long long n_events;   // fill of the event buffer (may run past ev_cap while a kernel is appending)
    unsigned long long ev_begin;   // first event of the current wave
    unsigned long long ev_cap;
    unsigned int q_count[2];       // fill of the two packet queues
    unsigned int work[2];          // dynamic work counters of the flight kernels
    unsigned int n_sorted;         // events in the sorted order of the current imaging pass
    unsigned int img_work[KRP_MAX_OBS_PACK];   // per-observer warp-tile counters of the imaging pass
    unsigned long long sg_segments;            // path segments deposited into the source grid (two-step form)
    unsigned int n_hits;                       // general mode: flights of the current wave that ended in an event (hit queue fill)
    KrpStatsDev stats;
};

// packet queue / event buffer, structure of arrays
struct KrpRecords {
    float4* pc;                 // {p_x, p_y, p_z (cell-local, [0,1]), cell index bits}
    float4* nk;                 // {n_x, n_y, n_z, k bits}
    float4* S;                  // {W, q, u, v}: weight and normalised Stokes, lab reference of n
    double* tau;                // queue only: optical depth to the next event
    unsigned long long* id;     // global packet id
};

// general mode: what a marching lane leaves behind when its flight reaches the cell of its event -- the state at the
// entry of that cell.  A converged kernel (krp_k_event_general) locates the event and writes the record.
struct KrpHits {
    uint2* ic;                  // {queue item, padded cell id}
    double2* Di;                // {scalar depth still to go D, normalised intensity i}
    double2* qu;                // {q, u} lab reference
    double2* vr;                // {v, distance to the next x face}
    double2* ryz;               // {distance to the next y face, to the next z face}
};

struct KrpObserverDev {
    float n[3], th[3], ph[3];
    float dt[3];                // path length between faces per axis, d/|n| (inf when n = 0)
    int stride[3];              // signed stride in the padded array per axis (0 when n = 0)
    double thd[3], phd[3], center[3], inv_hw, inv_hh;
};


// ------------------------------------------------------------------------------------------
// S0  Philox4x32-10 (Salmon et al. 2011), counter = (id_lo, id_hi, k, block), key = seed (R11)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 krp_philox(uint64_t seed, uint64_t id, uint32_t k, uint32_t blk)
{
    uint32_t c0 = (uint32_t)id, c1 = (uint32_t)(id >> 32), c2 = k, c3 = blk;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
        uint32_t h0 = __umulhi(M0, c0), l0 = M0 * c0;
        uint32_t h1 = __umulhi(M1, c2), l1 = M1 * c2;
        c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}
// (2j+1)/2^24 from the top 23 bits: exact in fp32 and fp64, never 0 or 1 (R11)
__device__ __forceinline__ double krp_u01(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }
// 52-bit uniform from two words (volume-source cell pick)
__device__ __forceinline__ double krp_u53(uint32_t x0, uint32_t x1)
{
    return ((double)(x0 >> 5) * 33554432.0 + (double)(x1 >> 7) + 0.5) * (1.0 / 4503599627370496.0);
}

// ------------------------------------------------------------------------------------------
// A4  spherical basis of a direction (eq. 4-5), pole rule R10
// ------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ void krp_basis(const T n[3], T th[3], T ph[3])
{
    T s2 = n[0] * n[0] + n[1] * n[1];
    T rr = sqrt(s2 + n[2] * n[2]);
    T s = sqrt(s2);
    T cp = T(1), sp = T(0);
    if (s2 >= T(1e-24)) { cp = n[0] / s; sp = n[1] / s; }
    T ct = n[2] / rr, st = s / rr;
    th[0] = ct * cp; th[1] = ct * sp; th[2] = -st;
    ph[0] = -sp; ph[1] = cp; ph[2] = T(0);
}

// ------------------------------------------------------------------------------------------
// A11  cell-interface-to-interface march, R11b, in two forms.
//
// KrpRay (flights): per axis the distance still to go to the next face, re-based every step, so
// its rounding error is that of a cell-local coordinate whatever the length of the flight (what
// decides the event cell has to stay within ~1e-7 of a cell).
//
// KrpRayA (imaging): per axis the absolute path length at the next face; one subtraction gives the
// segment, one predicated add advances the axis crossed.
//
// Both walk the padded array: the ray has left the grid when the cell it loads has kappa*rho < 0.
// Ties: x before y before z.
// ------------------------------------------------------------------------------------------
#define KRP_INF_F __int_as_float(0x7f800000)

struct KrpRay {
    float rx, ry, rz;   // distance to the next x/y/z face
    float tx, ty, tz;   // d/|n| per axis (inf when n = 0)
    int sx, sy, sz;     // signed stride in the padded array
    uint32_t c;         // padded cell id
};

__device__ __forceinline__ void krp_ray_axis(float n, float p, float d, int stride, float& r, float& t, int& s)
{
    if (n > 0.f)      { t = d / n;  r = (1.f - p) * t; s = stride; }
    else if (n < 0.f) { t = d / -n; r = p * t;         s = -stride; }
    else              { t = KRP_INF_F; r = t; s = 0; }
}

__device__ __forceinline__ void krp_ray_init(const KrpModel& g, uint32_t cell, const float p[3], const float n[3], KrpRay& r)
{
    krp_ray_axis(n[0], p[0], g.d[0], 1, r.rx, r.tx, r.sx);
    krp_ray_axis(n[1], p[1], g.d[1], g.px, r.ry, r.ty, r.sy);
    krp_ray_axis(n[2], p[2], g.d[2], (int)g.pxy, r.rz, r.tz, r.sz);
    r.c = cell;
}

// length of the segment inside the current cell
__device__ __forceinline__ float krp_ray_ds(const KrpRay& r) { return fminf(r.rx, fminf(r.ry, r.rz)); }

// cross the exit face (the caller detects the grid edge from the next cell's kappa*rho)
__device__ __forceinline__ void krp_ray_step(KrpRay& r, float ds)
{
    const bool ax = (r.rx <= r.ry) & (r.rx <= r.rz);
    const bool ay = (!ax) & (r.ry <= r.rz);
    r.rx -= ds; r.ry -= ds; r.rz -= ds;
    if (ax)      { r.rx = r.tx; r.c += (uint32_t)r.sx; }
    else if (ay) { r.ry = r.ty; r.c += (uint32_t)r.sy; }
    else         { r.rz = r.tz; r.c += (uint32_t)r.sz; }
}

// Event position in fp64 without accumulated rounding: the flight started at
// cell-local p0 (fp32 state, R12) of padded cell c0 and has its event in padded cell c, `t_len` beyond the
// point where it entered c through the face of axis `axis` (-1: still in the first cell).  The entry path
// length is a single fp64 expression, (plane - p0) d / n on that axis; the result is rounded to fp32 the way
// the state is defined.
__device__ __forceinline__ void krp_event_pos(const KrpModel& g, const float n[3], const float p0[3], uint32_t c0,
                                              uint32_t c, int axis, double t_len, float pe[3])
{
    int h0[3], h[3];
    krp_pad_coords(g, c0, h0[0], h0[1], h0[2]);
    krp_pad_coords(g, c, h[0], h[1], h[2]);
    double s = t_len;
    if (axis >= 0) {
        const double plane = (double)(h[axis] - h0[axis]) + (n[axis] > 0.f ? 0.0 : 1.0);
        s += (plane - (double)p0[axis]) * g.dd[axis] / (double)n[axis];
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        double x = (double)p0[a] + (double)n[a] * s * g.inv_dd[a] - (double)(h[a] - h0[a]);
        pe[a] = (float)fmin(fmax(x, 0.0), 1.0);
    }
}

// path length of a flight from its start (cell c0, local p0) to its event (cell c, local pe), fp64: what the flight
// kernels hand to the deposit step of the two-step form (krp_twostep.cuh)
__device__ __forceinline__ double krp_path_length(const KrpModel& g, const float n[3], const float p0[3], uint32_t c0,
                                                  const float pe[3], uint32_t c)
{
    int h0[3], h[3];
    krp_pad_coords(g, c0, h0[0], h0[1], h0[2]);
    krp_pad_coords(g, c, h[0], h[1], h[2]);
    double s = 0.0, nn = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        s += (double)n[a] * ((double)(h[a] - h0[a]) + ((double)pe[a] - (double)p0[a])) * g.dd[a];
        nn += (double)n[a] * (double)n[a];
    }
    return s / nn;
}

// The same re-based march with the distances in fp64: used by the general-mode flight, where the optical
// depth consumed in every cell decides the integer outcome "which cell holds the event" and has to be taken
// in the oracle's precision.
struct KrpRayD {
    double rx, ry, rz;
    double tx, ty, tz;
    int sx, sy, sz;
    uint32_t c;
};

__device__ __forceinline__ void krp_rayd_axis(float n, float p, double d, int stride, double& r, double& t, int& s)
{
    // one division per axis: the distance to the first face is that fraction of the face spacing (1e-16 from the other order)
    // (branch-free: as two branches the lanes going up and those going down each ran their own division, a sixth of the
    // flight kernel's instructions on C3, whose flights are 1.2 cells long.  d / |n| = +inf for n = 0.)
    const double tt = d / fabs((double)n);
    const double f = n > 0.f ? 1.0 - (double)p : (double)p;
    t = tt;
    r = n != 0.f ? f * tt : tt;
    s = n > 0.f ? stride : (n < 0.f ? -stride : 0);
}

__device__ __forceinline__ void krp_rayd_init(const KrpModel& g, uint32_t cell, const float p[3], const float n[3], KrpRayD& r)
{
    krp_rayd_axis(n[0], p[0], g.dd[0], 1, r.rx, r.tx, r.sx);
    krp_rayd_axis(n[1], p[1], g.dd[1], g.px, r.ry, r.ty, r.sy);
    krp_rayd_axis(n[2], p[2], g.dd[2], (int)g.pxy, r.rz, r.tz, r.sz);
    r.c = cell;
}

__device__ __forceinline__ double krp_rayd_ds(const KrpRayD& r) { return fmin(r.rx, fmin(r.ry, r.rz)); }

__device__ __forceinline__ void krp_rayd_step(KrpRayD& r, double ds)
{
    bool ax = (r.rx <= r.ry) & (r.rx <= r.rz);
    bool ay = (!ax) & (r.ry <= r.rz);
    bool az = !(ax | ay);
    r.rx = ax ? r.tx : r.rx - ds;
    r.ry = ay ? r.ty : r.ry - ds;
    r.rz = az ? r.tz : r.rz - ds;
    int s = ax ? r.sx : (ay ? r.sy : r.sz);
    r.c += (uint32_t)s;
}

// cell-local position (fp64 distances) after moving `moved` from the point where r was taken
__device__ __forceinline__ float krp_locald(float n, double r, double inv_d, double moved, float p0)
{
    if (n == 0.f) return p0;
    double f = (r - moved) * fabs((double)n) * inv_d;      // 1/t = |n|/d
    f = fmin(fmax(f, 0.0), 1.0);
    return (float)(n > 0.f ? 1.0 - f : f);
}

struct KrpRayA {
    float t;            // path length at the entry of the current cell
    float tx, ty, tz;   // path length at the next x/y/z face
    uint32_t c;         // padded cell id
};

// ------------------------------------------------------------------------------------------
// D4  table look-ups, linear in the node variable (R13)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ float4 krp_opac_at(const float4* __restrict__ tab, int n_inc, float mu)
{
    mu = fminf(mu, 1.f);
    float x = mu * (float)(n_inc - 1);
    int j = min((int)x, n_inc - 2);
    float w = x - (float)j;
    float4 a = tab[j], b = tab[j + 1];
    float w0 = 1.f - w;
    return make_float4(w0 * a.x + w * b.x, w0 * a.y + w * b.y, w0 * a.z + w * b.z, w0 * a.w + w * b.w);
}

template <typename T>
__device__ __forceinline__ void krp_mueller_at(const float4* __restrict__ tab, int n_ang, T theta_deg, T F[4])
{
    T x = theta_deg * (T)(n_ang - 1) / T(180);
    int j = (int)floor(x);
    j = max(0, min(j, n_ang - 2));
    T w = x - (T)j, w0 = T(1) - w;
    float4 a = tab[j], b = tab[j + 1];
    F[0] = w0 * (T)a.x + w * (T)b.x; F[1] = w0 * (T)a.y + w * (T)b.y;
    F[2] = w0 * (T)a.z + w * (T)b.z; F[3] = w0 * (T)a.w + w * (T)b.w;
}

// ------------------------------------------------------------------------------------------
// A5  reference-frame angle between the lab basis (theta^, phi^) of n and the grain-frame
// basis of the same ray (eq. 6-7, sign restored per R2).  theta^' expressed
// in the lab is ((n.B)n - B)/sin(vartheta), so with a = theta^.B and b = phi^.B:
// cos(eta) = -a/s, sin(eta) = -b/s, s^2 = a^2 + b^2; only 2*eta enters eq. 7.
// ------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ void krp_eta2(T a, T b, T& c2, T& s2)
{
    T ss = a * a + b * b;
    if (ss < T(1e-24)) { c2 = T(1); s2 = T(0); return; }
    T inv = T(1) / ss;
    c2 = (a * a - b * b) * inv;
    s2 = T(2) * a * b * inv;
}

// fp64 form with the reciprocal by Newton from the fp32 one (two steps: relative error < 1e-16), cheaper than a division
__device__ __forceinline__ void krp_eta2_d(double a, double b, double& c2, double& s2)
{
    const double aa = a * a, bb = b * b, ss = aa + bb;
    if (__double2hiint(ss) < 0x3af357c2) { c2 = 1.0; s2 = 0.0; return; }     // ss < 1e-24, on the high word (ss >= 0)
    float rf;       // 1/ss: the hardware approximation (2^-23) and two Newton steps (1e-14, 1e-28); ss is in [1e-24, 1]
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rf) : "f"((float)ss));
    double r = (double)rf;
    r = r * (2.0 - ss * r);
    r = r * (2.0 - ss * r);
    c2 = (aa - bb) * r;
    s2 = 2.0 * a * b * r;
}

// sinh(x) and cosh(x)-1 without cancellation for small x; |x| < ~80
__device__ __forceinline__ void krp_sinh_coshm1(float x, float& sh, float& chm1)
{
    float ax = fabsf(x);
    if (ax < 0.35f) {
        float x2 = x * x;
        sh = x * (1.f + x2 * (1.f / 6.f + x2 * (1.f / 120.f + x2 * (1.f / 5040.f))));
        chm1 = x2 * (0.5f + x2 * (1.f / 24.f + x2 * (1.f / 720.f + x2 * (1.f / 40320.f))));
    } else {
        float e = expf(ax), ie = 1.f / e;
        sh = copysignf(0.5f * (e - ie), x);
        chm1 = 0.5f * (e + ie) - 1.f;
    }
}

// ------------------------------------------------------------------------------------------
// A12  source-free App. A solution (matrix of R1) over dtau in the grain-
// frame reference, written for a Stokes vector carried as  e^{-A} (i, q, u, v):
//   thin step  (|alpha2 dtau| < 0.35): returns the increment of i (so the caller can
//       accumulate it in fp64), updates q,u,v, and the scalar depth grows by alpha1*dtau;
//   thick step: the common factor e^{-|alpha2 dtau|} is moved into the scalar depth so that
//       nothing overflows at dtau ~ 1e3.
// On return `depth` is what was added to A.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ bool krp_appA(float i, float& qg, float& ug, float& v, float4 op, float dtau,
                                         float& di, float& i_new, float& depth)
{
    float x = op.y * dtau, y = op.z * dtau;
    float sy = 0.f, cy = 1.f;
    if (y != 0.f) sincosf(y, &sy, &cy);
    float ax = fabsf(x);
    bool thick = ax >= 0.35f;
    if (!thick) {
        float sh, chm1;
        krp_sinh_coshm1(x, sh, chm1);
        di = i * chm1 - qg * sh;
        float qn = qg + (qg * chm1 - i * sh);
        float un = ug * cy - v * sy;
        float vn = ug * sy + v * cy;
        qg = qn; ug = un; v = vn;
        i_new = i + di;
        depth = op.x * dtau;
    } else {
        float E = expf(-2.f * ax);
        float s = x > 0.f ? 1.f : -1.f;
        float ip = 0.5f * ((i - s * qg) + (i + s * qg) * E);
        float qp = 0.5f * ((qg - s * i) + (qg + s * i) * E);
        float f = expf(-ax);
        float un = f * (ug * cy - v * sy);
        float vn = f * (ug * sy + v * cy);
        i_new = ip; qg = qp; ug = un; v = vn;
        di = 0.f;
        depth = op.x * dtau - ax;
    }
    return thick;
}

// ------------------------------------------------------------------------------------------
// warp-aggregated reservation of one slot per calling lane in a 64-bit / 32-bit counter
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long krp_reserve64(unsigned long long* counter)
{
    unsigned m = __activemask();
    int lane = threadIdx.x & 31;
    int leader = __ffs(m) - 1;
    unsigned long long base = 0;
    if (lane == leader) base = atomicAdd(counter, (unsigned long long)__popc(m));
    base = __shfl_sync(m, base, leader);
    return base + (unsigned long long)__popc(m & ((1u << lane) - 1u));
}
__device__ __forceinline__ unsigned int krp_reserve32(unsigned int* counter)
{
    unsigned m = __activemask();
    int lane = threadIdx.x & 31;
    int leader = __ffs(m) - 1;
    unsigned int base = 0;
    if (lane == leader) base = atomicAdd(counter, (unsigned int)__popc(m));
    base = __shfl_sync(m, base, leader);
    return base + (unsigned int)__popc(m & ((1u << lane) - 1u));
}

__device__ __forceinline__ double krp_warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ unsigned long long krp_warp_sum(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
