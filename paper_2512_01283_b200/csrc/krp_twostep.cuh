// krp_twostep.cuh -- the paper's own two-step imaging (eq. 11) and thermal
// emission in the ray step (eq. 8; NEXT-3):
//   step 1  krp_k_deposit     every path segment of every flight deposits its expected collision output toward every
//                             camera into the grid-resident S(Omega_cam, x)            (reading R18)
//   step 2  krp_k_image_rays  one ray per pixel through the grid toward the camera, App. A WITH source terms
//                              in every cell: scattering source from S, thermal source (1-omega) alpha B
//
// B200 design against the paper's (one packet per warp, shared-memory reductions before global atomics):
// S is laid out [cell][camera][4 Stokes] in fp32, so that all cameras of a cell share one or two 128-byte lines, and a
// deposit is ONE vector reduction per camera (red.global.add.v4.f32, sm_90+) that the L2 slice applies in place -- no
// shared-memory staging of the sums.  A flight is re-marched by one lane, which holds the peel-off geometry of its flight
// toward every camera in shared memory.  The flights themselves are the ordinary ones (same packets, same events): the
// flight kernels only hand over each flight's path length.
#pragma once
#include "krp_kernels.cuh"

#define KRP_SG_MAX_OBS 16          // cameras of one source grid (two per lane of a group of 8)

__device__ __forceinline__ void krp_red_v4(float* addr, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" :: "l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

// normalised grain-frame state (q^, u^, v^) at depth t inside a segment that starts with (1, q0, u0, v0): source-free
// App. A divided by its intensity (R7)
__device__ __forceinline__ void krp_state_at(float q0, float u0, float v0, float a2, float a3, float t, float& q, float& u, float& v)
{
    const float x = a2 * t, y = a3 * t;
    float sy, cy;
    __sincosf(y, &sy, &cy);
    const float em = -expm1f(-2.f * fabsf(x));               // 1 - e^{-2|x|}; cosh, sinh below are in units of e^{|x|}/2, which cancels
    const float ch = 2.f - em, shh = copysignf(em, x);
    const float inv = 2.f * __frcp_rn(ch - q0 * shh);        // 2 / (cosh - q0 sinh) in those units times e^{-|x|}
    q = (q0 * ch - shh) * 0.5f * inv;
    const float f = __expf(-fabsf(x)) * inv;                 // 1 / (cosh x - q0 sinh x)
    u = (u0 * cy - v0 * sy) * f;
    v = (u0 * sy + v0 * cy) * f;
}

// J = int_0^T r s^ dtau of one segment (reading R18) from r s^ = s^' + K s^ :
//   J_I = a1 T - ln g(T),  g(T) = cosh(a2 T) - q0 sinh(a2 T)  (closed form)
//   J_Q = q^(T) - q0 + a2 T + a1 int q^,  int q^ = -ln g(T) / a2   (closed form; a2 -> 0: a1 T q0)
//   J_U = u^(T) - u0 + a1 int u^ + a3 int v^,  J_V = v^(T) - v0 - a3 int u^ + a1 int v^, the two integrals by 3-point
//         Gauss-Legendre on pieces of (|a2| + |a3|) h <= 0.35 (relative error below 1e-6 per piece)
// (q0,u0,v0) normalised grain-frame state at the start; returns also the state at the end.
__device__ __forceinline__ void krp_segment_integral(float q0, float u0, float v0, float a1, float a2, float a3, float T,
                                                     float J[4], float& qT, float& uT, float& vT)
{
    krp_state_at(q0, u0, v0, a2, a3, T, qT, uT, vT);
    const float x = a2 * T;
    // -ln g(T): g = cosh x - q0 sinh x = e^{|x|} (1 + e^{-2|x|} - q0 sgn(x)(1 - e^{-2|x|})) / 2
    float mlg;
    if (fabsf(x) < 0.1f) {
        const float x2 = x * x;
        const float gm1 = x2 * fmaf(x2, 1.f / 24.f, 0.5f) - q0 * fmaf(x * x2, 1.f / 6.f, x);
        mlg = -log1pf(gm1);
    } else {
        const float e = __expf(-2.f * fabsf(x));
        mlg = -(fabsf(x) + __logf(0.5f * ((1.f + e) - q0 * copysignf(1.f - e, x))));
    }
    J[0] = a1 * T + mlg;
    const float int_q = fabsf(a2) > 1e-6f * a1 ? mlg / a2 : q0 * T;
    J[1] = (qT - q0) + x + a1 * int_q;
    float iu = 0.f, iv = 0.f;
    {
        const float span = (fabsf(a2) + fabsf(a3)) * T;
        const int np = span > 0.35f ? (int)ceilf(span * (1.f / 0.35f)) : 1;
        const float h = T / (float)np;
        const float gx[3] = { 0.1127016653792583f, 0.5f, 0.8872983346207417f }, gw[3] = { 5.f / 18.f, 8.f / 18.f, 5.f / 18.f };
        for (int k = 0; k < np; ++k)
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                float q, u, v;
                krp_state_at(q0, u0, v0, a2, a3, ((float)k + gx[j]) * h, q, u, v);
                iu = fmaf(gw[j] * h, u, iu); iv = fmaf(gw[j] * h, v, iv);
            }
    }
    J[2] = (uT - u0) + a1 * iu + a3 * iv;
    J[3] = (vT - v0) - a3 * iu + a1 * iv;
}


// ------------------------------------------------------------------------------------------
// step 1: deposit.  Work item = one flight of the wave (queue entry `item`, or the on-the-fly emission of the first
// order), re-marched in fp32 over its known path length flen[item] (+inf: to the grid edge).  One flight per lane; the
// peel-off geometry of the flight toward every camera (8 floats each) sits in shared memory, [camera][thread], so that
// a segment costs the march and the segment integral once and per camera two 16-byte shared loads, ~20 FMAs and one
// vector reduction.  (The first version marched every flight redundantly in G = 8 lanes, one camera per lane: C5 deposit
// 1565 ms per 2^22 packets, profiles/r2e.)
// ------------------------------------------------------------------------------------------
// Sort key of a flight for the deposit: the number of cell faces it crosses (from its path length; for an escape, from the
// distance to the box), so that the 32 flights of a warp are equally long -- re-marched in queue order the lanes of a warp held
// flights of 1 to 500 cells and 8.3 of 32 threads were active (profiles/r2w).  Entries beyond the queue's fill get key 0 and sort last.
__global__ void __launch_bounds__(256) krp_k_deposit_keys(KrpModel g, KrpCtl* ctl, KrpRecords q, int in, KrpEmitSrc es,
                                                          const double* __restrict__ flen, unsigned int n_cap,
                                                          unsigned short* __restrict__ keys, unsigned int* __restrict__ vals)
{
    const unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_cap) return;
    vals[i] = i;
    if (i >= ctl->q_count[in]) { keys[i] = 0; return; }
    float4 pc, nk, S0; double tau; unsigned long long id;
    krp_item_load(g, q, es, i, pc, nk, S0, tau, id);
    double L = flen[i];
    const float n[3] = { nk.x, nk.y, nk.z }, p[3] = { pc.x, pc.y, pc.z };
    if (L > 3.0e38) {                     // escape: distance to the box along n
        int h[3];
        krp_pad_coords(g, __float_as_uint(pc.w), h[0], h[1], h[2]);
        const int nn[3] = { g.nx, g.ny, g.nz };
        L = 3.0e38;
        for (int a = 0; a < 3; ++a) {
            if (n[a] == 0.f) continue;
            const double x = (double)(h[a] - 1) + (double)p[a];
            const double t = (n[a] > 0.f ? (double)nn[a] - x : x) * g.dd[a] / fabs((double)n[a]);
            L = fmin(L, t);
        }
    }
    const double steps = L * (fabs((double)n[0]) * g.inv_dd[0] + fabs((double)n[1]) * g.inv_dd[1] + fabs((double)n[2]) * g.inv_dd[2]);
    keys[i] = (unsigned short)(1.0 + fmin(steps, 65000.0));
}

template <bool SCALAR>
__global__ void __launch_bounds__(128) krp_k_deposit(KrpModel g, KrpCtl* ctl, KrpRecords q, int in, KrpEmitSrc es,
                                                     const double* __restrict__ flen, const unsigned int* __restrict__ order,
                                                     const KrpObserverDev* __restrict__ obs,
                                                     int n_obs, float* __restrict__ sgrid, unsigned long long* __restrict__ n_seg)
{
    extern __shared__ float4 s_pg[];                 // [n_obs][2][blockDim.x]
    const unsigned int n_items = ctl->q_count[in];
    unsigned long long segs = 0;
    for (unsigned int slot = blockIdx.x * blockDim.x + threadIdx.x; slot < n_items; slot += gridDim.x * blockDim.x) {
        const unsigned int item = order[slot];           // flights in the order of their length (longest first)
        float4 pc, nk, S0; double tau; unsigned long long id;
        krp_item_load(g, q, es, item, pc, nk, S0, tau, id);
        const float n[3] = { nk.x, nk.y, nk.z };
        const double Ld = flen[item];
        const float L = Ld > 3.0e38 ? KRP_INF_F : (float)Ld;
        for (int o = 0; o < n_obs; ++o) {
            KrpPeelGeom pg;
            krp_peel_setup(g, n, obs[o], pg);
            s_pg[(2 * o) * blockDim.x + threadIdx.x] = make_float4(pg.c2i, pg.s2i, pg.c2o, pg.s2o);
            s_pg[(2 * o + 1) * blockDim.x + threadIdx.x] = make_float4(pg.F[0], pg.F[1], pg.F[2], pg.F[3]);
        }
        // lab basis of n for the grain-frame rotation (general mode)
        float th[3] = { 0.f, 0.f, 0.f }, ph[3] = { 0.f, 0.f, 0.f };
        if (!SCALAR) krp_basis<float>(n, th, ph);
        const float inv_n = rsqrtf(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
        // absolute path-length march: t_a = path length at the next face of axis a
        float tx, ty, tz, dtx, dty, dtz; int sx, sy, sz;
        krp_ray_axis(n[0], pc.x, g.d[0], 1, tx, dtx, sx);
        krp_ray_axis(n[1], pc.y, g.d[1], g.px, ty, dty, sy);
        krp_ray_axis(n[2], pc.z, g.d[2], (int)g.pxy, tz, dtz, sz);
        uint32_t c = __float_as_uint(pc.w);
        float t = 0.f;
        float qs = S0.y, us = S0.z, vs = S0.w;       // normalised lab state (1, q, u, v) of the live packet
        const float W = S0.x;
        for (;;) {
            float kr, bx = 0.f, by = 0.f, bz = 1.f;
            KRP_CK(g, c);
            if (SCALAR) kr = __ldg(g.kr + c);
            else { const float4 cl = __ldg(g.cell + c); kr = cl.x; bx = cl.y; by = cl.z; bz = cl.w; }
            if (kr < 0.f) break;                                  // halo
            const float tn = fminf(tx, fminf(ty, tz));
            const bool last = tn >= L;
            const float len = (last ? L : tn) - t;
            if (kr > 0.f) ++segs;                                 // counted like the oracle's: also a segment of zero length
            if (kr > 0.f && len > 0.f) {
                float a1, a2, a3, om, c2 = 1.f, s2 = 0.f;
                if (SCALAR) { a1 = g.a1c; a2 = 0.f; a3 = 0.f; om = g.omc; }
                else {
                    const float mu = fminf(fabsf(n[0] * bx + n[1] * by + n[2] * bz) * inv_n * rsqrtf(bx * bx + by * by + bz * bz), 1.f);
                    const float x = mu * (float)(g.n_inc - 1);
                    const int j = min((int)x, g.n_inc - 2);
                    const float4 ta = g.opA[j], tb = g.opB[j];
                    a1 = fmaf(tb.x, x, ta.x); a2 = fmaf(tb.y, x, ta.y); a3 = fmaf(tb.z, x, ta.z); om = fmaf(tb.w, x, ta.w);
                    if (a2 != 0.f || a3 != 0.f)
                        krp_eta2<float>(th[0] * bx + th[1] * by + th[2] * bz, ph[0] * bx + ph[1] * by + ph[2] * bz, c2, s2);
                }
                const float T = kr * len;
                float J[4];
                if (a2 == 0.f && a3 == 0.f) {                    // the state does not change: J = a1 T s^
                    const float f = a1 * T;
                    J[0] = f; J[1] = f * qs; J[2] = f * us; J[3] = f * vs;
                } else {
                    const float qg = c2 * qs + s2 * us, ug = c2 * us - s2 * qs;          // eq. 7
                    float Jg[4], qT, uT, vT;
                    krp_segment_integral(qg, ug, vs, a1, a2, a3, T, Jg, qT, uT, vT);
                    J[0] = Jg[0]; J[1] = c2 * Jg[1] - s2 * Jg[2]; J[2] = s2 * Jg[1] + c2 * Jg[2]; J[3] = Jg[3];
                    qs = c2 * qT - s2 * uT; us = s2 * qT + c2 * uT; vs = vT;
                }
                const float w = om * W;
                J[0] *= w; J[1] *= w; J[2] *= w; J[3] *= w;
                float* cell_s = sgrid + (size_t)c * n_obs * 4;
                for (int o = 0; o < n_obs; ++o) {
                    const float4 r = s_pg[(2 * o) * blockDim.x + threadIdx.x], F = s_pg[(2 * o + 1) * blockDim.x + threadIdx.x];
                    const float qq = r.x * J[1] + r.y * J[2], uu = -r.y * J[1] + r.x * J[2];          // into the scattering plane
                    const float I2 = F.x * J[0] + F.y * qq, Q2 = F.y * J[0] + F.x * qq;
                    const float U2 = F.z * uu + F.w * J[3], V2 = -F.w * uu + F.z * J[3];
                    krp_red_v4(cell_s + 4 * o, I2, r.z * Q2 + r.w * U2, -r.w * Q2 + r.z * U2, V2);       // to theta^_cam
                }
            }
            if (last) break;
            // cross the face (ties: x before y before z)
            t = tn;
            if (tx <= ty && tx <= tz) { tx += dtx; c += (uint32_t)sx; }
            else if (ty <= tz)        { ty += dty; c += (uint32_t)sy; }
            else                      { tz += dtz; c += (uint32_t)sz; }
        }
    }
    segs = krp_warp_sum(segs);
    if ((threadIdx.x & 31) == 0 && segs) atomicAdd(n_seg, segs);
}

// ------------------------------------------------------------------------------------------
// step 2: one ray per pixel, fp64.  The line through the pixel centre along n_obs is clipped against the
// box (slab method), then marched cell by cell from the far side toward the observer; in every cell the Stokes vector
// and the source are turned into the grain-frame reference (eq. 6-7), advanced by App. A with source terms
// (S = S_s + e^{-K dtau}(S_0 - S_s), K S_s = src, PAPER.md:302-328 with the matrix of R1) and turned back.
// Sources per unit extinction depth: sgrid[c][o][:] / (V_cell kappa rho) and (1 - omega)(alpha1, alpha2, 0, 0) B_c.
// The pixel receives radiance times its area (R14).  One launch per observer; one thread per pixel, no atomics.
// ------------------------------------------------------------------------------------------
struct KrpRayObs { double n[3], th[3], ph[3], center[3], half_w, half_h; };

template <bool SCALAR>
__global__ void __launch_bounds__(128) krp_k_image_rays(KrpModel g, KrpCtl* ctl, KrpRayObs ob, int o, int n_obs, int npx, int npy,
                                                        const float* __restrict__ sgrid, const float* __restrict__ emis,
                                                        double* __restrict__ img)
{
    const int pix = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long steps = 0, hit = 0;
    if (pix < npx * npy) {
        const int ix = pix % npx, iy = pix / npx;
        const double xi = (((double)ix + 0.5) * 2.0 / (double)npx - 1.0) * ob.half_w;
        const double yi = (((double)iy + 0.5) * 2.0 / (double)npy - 1.0) * ob.half_h;
        double x0[3];
        for (int a = 0; a < 3; ++a) x0[a] = ob.center[a] + xi * ob.ph[a] - yi * ob.th[a];
        const int nn[3] = { g.nx, g.ny, g.nz };
        const double inf = __longlong_as_double(0x7ff0000000000000ll);
        double s_in = -inf, s_out = inf;
        bool miss = false;
        for (int a = 0; a < 3; ++a) {
            const double lo = g.lo[a], hi = g.lo[a] + (double)nn[a] * g.dd[a];
            if ((g.periodic >> a) & 1) continue;          // R20: a periodic axis does not clip the line, its coordinate is taken modulo the box
            if (ob.n[a] == 0.0) { if (x0[a] < lo || x0[a] >= hi) miss = true; continue; }
            double t0 = (lo - x0[a]) / ob.n[a], t1 = (hi - x0[a]) / ob.n[a];
            if (t0 > t1) { const double t = t0; t0 = t1; t1 = t; }
            s_in = fmax(s_in, t0); s_out = fmin(s_out, t1);
        }
        if (!miss && s_in < s_out && s_in != -inf) {
            hit = 1;
            int nwrap = 0;
            // entry cell and cell-local position; per axis the distance to the next face and the face spacing (re-based march)
            int idx[3]; double r[3], tt[3]; int sgn[3];
            for (int a = 0; a < 3; ++a) {
                double x = (x0[a] + s_in * ob.n[a] - g.lo[a]) * g.inv_dd[a];
                if ((g.periodic >> a) & 1) x -= floor(x / (double)nn[a]) * (double)nn[a];
                int i = (int)floor(x);
                i = max(0, min(i, nn[a] - 1));
                const double p = fmin(fmax(x - (double)i, 0.0), 1.0);
                idx[a] = i;
                if (ob.n[a] > 0.0)      { tt[a] = g.dd[a] / ob.n[a];  r[a] = (1.0 - p) * tt[a]; sgn[a] = 1; }
                else if (ob.n[a] < 0.0) { tt[a] = g.dd[a] / -ob.n[a]; r[a] = p * tt[a];         sgn[a] = -1; }
                else                    { tt[a] = inf; r[a] = inf; sgn[a] = 0; }
            }
            const double vol = g.dd[0] * g.dd[1] * g.dd[2];
            double S[4] = { 0.0, 0.0, 0.0, 0.0 };
            for (;;) {
                const int ax = (r[0] <= r[1] && r[0] <= r[2]) ? 0 : (r[1] <= r[2] ? 1 : 2);      // ties: x before y before z
                const double ds = r[ax];
                const uint32_t c = krp_pad_id(g, idx[0], idx[1], idx[2]);
                ++steps;
                double kr, b[3] = { 0.0, 0.0, 1.0 };
                if (SCALAR) kr = (double)g.kr[c];
                else { const float4 cl = g.cell[c]; kr = (double)cl.x; b[0] = cl.y; b[1] = cl.z; b[2] = cl.w; }
                if (kr > 0.0) {
                    double a1, a2, a3, om;
                    if (SCALAR) { a1 = (double)g.a1c; a2 = 0.0; a3 = 0.0; om = (double)g.omc; }
                    else {
                        const double mu = fmin(fabs(ob.n[0] * b[0] + ob.n[1] * b[1] + ob.n[2] * b[2]) / sqrt(b[0] * b[0] + b[1] * b[1] + b[2] * b[2]), 1.0);
                        const double x = mu * g.xs;
                        const int j = min((int)x, g.n_inc - 2);
                        const double4 ta = g.opA_d[j], tb = g.opB_d[j];
                        a1 = fma(tb.x, x, ta.x); a2 = fma(tb.y, x, ta.y); a3 = fma(tb.z, x, ta.z); om = fma(tb.w, x, ta.w);
                    }
                    double src[4] = { 0.0, 0.0, 0.0, 0.0 };
                    if (sgrid) {
                        const float4 sg = *reinterpret_cast<const float4*>(sgrid + ((size_t)c * n_obs + o) * 4);
                        const double f = 1.0 / (vol * kr);
                        src[0] = f * (double)sg.x; src[1] = f * (double)sg.y; src[2] = f * (double)sg.z; src[3] = f * (double)sg.w;
                    }
                    double c2 = 1.0, s2 = 0.0;
                    const bool rot = a2 != 0.0 || a3 != 0.0;
                    if (rot) {
                        krp_eta2<double>(ob.th[0] * b[0] + ob.th[1] * b[1] + ob.th[2] * b[2], ob.ph[0] * b[0] + ob.ph[1] * b[1] + ob.ph[2] * b[2], c2, s2);
                        krp_rot_qu(S[1], S[2], c2, s2);
                        krp_rot_qu(src[1], src[2], c2, s2);
                    }
                    if (emis) { const double B = (double)emis[c]; src[0] += (1.0 - om) * a1 * B; src[1] += (1.0 - om) * a2 * B; }
                    // stationary vector (eq. A3) and the source-free solution of the difference
                    const double dIQ = 1.0 / (a1 * a1 - a2 * a2), dUV = 1.0 / (a1 * a1 + a3 * a3);
                    const double Is = (a1 * src[0] - a2 * src[1]) * dIQ, Qs = (a1 * src[1] - a2 * src[0]) * dIQ;
                    const double Us = (a1 * src[2] - a3 * src[3]) * dUV, Vs = (a1 * src[3] + a3 * src[2]) * dUV;
                    const double dtau = kr * ds;
                    const double dI = S[0] - Is, dQ = S[1] - Qs, dU = S[2] - Us, dV = S[3] - Vs;
                    const double em = exp(-(a1 - a2) * dtau), ep = exp(-(a1 + a2) * dtau), e1 = exp(-a1 * dtau);
                    double sy, cy;
                    sincos(a3 * dtau, &sy, &cy);
                    S[0] = Is + 0.5 * ((dI - dQ) * em + (dI + dQ) * ep);
                    S[1] = Qs + 0.5 * ((dQ - dI) * em + (dQ + dI) * ep);
                    S[2] = Us + e1 * (dU * cy - dV * sy);
                    S[3] = Vs + e1 * (dU * sy + dV * cy);
                    if (rot) krp_rot_qu(S[1], S[2], c2, -s2);
                }
                // cross the face; leaving the grid ends the ray
                idx[ax] += sgn[ax];
                if (idx[ax] < 0 || idx[ax] >= nn[ax]) {
                    if (!((g.periodic >> ax) & 1) || nwrap >= KRP_MAX_WRAPS) break;
                    ++nwrap;
                    idx[ax] = idx[ax] < 0 ? nn[ax] - 1 : 0;
                }
                for (int a = 0; a < 3; ++a) r[a] = (a == ax) ? tt[a] : r[a] - ds;
            }
            const double apix = (2.0 * ob.half_w / (double)npx) * (2.0 * ob.half_h / (double)npy);
            const size_t plane = (size_t)npx * npy;
            double* at = img + (size_t)o * 4 * plane + pix;
            at[0] += apix * S[0]; at[plane] += apix * S[1]; at[2 * plane] += apix * S[2]; at[3 * plane] += apix * S[3];
        }
    }
    steps = krp_warp_sum(steps); hit = krp_warp_sum(hit);
    if ((threadIdx.x & 31) == 0) {
        if (steps) atomicAdd(&ctl->stats.steps_image, steps);
        if (hit) atomicAdd(&ctl->stats.contributions, hit);
    }
}

// [nz][ny][nx] -> padded order (halo 0), for the per-cell thermal source
__global__ void krp_k_pad_scalar(KrpModel g, const float* __restrict__ in, uint32_t npad, float* __restrict__ out)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= npad) return;
    int hx, hy, hz;
    krp_pad_coords(g, c, hx, hy, hz);
    const bool halo = hx == 0 || hy == 0 || hz == 0 || hx == g.nx + 1 || hy == g.ny + 1 || hz == g.nz + 1;
    out[c] = halo ? 0.f : in[((size_t)(hz - 1) * g.ny + (hy - 1)) * g.nx + (hx - 1)];
}

// padded source grid -> the caller's [nz][ny][nx][n_obs][4] order
__global__ void krp_k_sgrid_unpad(KrpModel g, const float4* __restrict__ sg, int n_obs, float4* __restrict__ out)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (size_t)g.ncell * n_obs) return;
    const uint32_t lin = (uint32_t)(i / n_obs); const int o = (int)(i % n_obs);
    const uint32_t t = lin / (uint32_t)g.nx; const int ix = (int)(lin - t * (uint32_t)g.nx);
    const uint32_t iz = t / (uint32_t)g.ny; const int iy = (int)(t - iz * (uint32_t)g.ny);
    out[i] = sg[(size_t)krp_pad_id(g, ix, iy, (int)iz) * n_obs + o];
}

// ------------------------------------------------------------------------------------------
// frequency bins: kappa*rho of a bin = factor x the model's.  base holds the model's values in the
// padded order (halo -1); the cell arrays take base x factor.
// ------------------------------------------------------------------------------------------
__global__ void krp_k_save_base(uint32_t npad, const float* __restrict__ kr, const float4* __restrict__ cell, float* __restrict__ base)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c < npad) base[c] = kr ? kr[c] : cell[c].x;
}
__global__ void krp_k_rescale(uint32_t npad, const float* __restrict__ base, float factor, float* __restrict__ kr, float4* __restrict__ cell)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= npad) return;
    const float b = base[c], v = b < 0.f ? b : b * factor;
    if (kr) kr[c] = v;
    if (cell) cell[c].x = v;
}
