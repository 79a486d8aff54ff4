// krp_kernels.cuh -- the kernels of the hot path: emit, flight (cell march to the next
// event), scatter, image.  See DESIGN.md "Kernels".  Transport is a wavefront pipeline:
//   emit -> [ wave_prep -> flight -> scatter ] x waves
// Flights never execute scattering code; lanes that reach an event append the packet to the event
// buffer, and the scatter kernel (fp64 geometry, all lanes busy) turns the wave's events into the
// next queue.  The event buffer is what the imaging kernels consume (ordered by cell bin first).
#pragma once
#include "krp_device.cuh"

#ifndef KRP_IMG_CHUNK
#define KRP_IMG_CHUNK 128     // events a warp of the imaging kernels takes per atomic (a multiple of 32)
#endif
#ifndef KRP_IMAGE_SCALAR_MIN_BLOCKS
#define KRP_IMAGE_SCALAR_MIN_BLOCKS 8
#endif
#ifndef KRP_IMAGE_MIN_BLOCKS
#define KRP_IMAGE_MIN_BLOCKS 6
#endif

// ------------------------------------------------------------------------------------------
// T1/T2  emission: draws of block 0 = (cos theta, phi, tau*, spare); blocks 1-2
// place a volume-source packet (R11, R17).  One thread per packet.
// ------------------------------------------------------------------------------------------
// Direction bins of an isotropic point source (T7): packets whose flights start in the same cell are queued in
// the order of their direction (128 bins in cos(theta) x 256 in phi, read off the uniform words, 32 counters
// per bin against contention), so that the 32 flights of a warp walk through the same cells -- their gathers hit
// the same lines and they leave the grid together.  The queue order has no meaning for the results.
// A large batch is ordered in sub-batches of 2^sub_shift packets (the sub-batch is the leading key): the slots one
// sub-batch writes then span a few tens of MB, so that the 4-byte writes of a bin meet in L2 before they go to DRAM.
#define KRP_DIR_BINS (1u << 20)
#define KRP_DIR_SUBS_MAX 16u
#define KRP_DIR_SUB_SHIFT 23u
__device__ __forceinline__ unsigned int krp_dir_bin(uint4 w, unsigned int i, unsigned int sub_shift)
{
    return ((i >> sub_shift) << 20) | ((((w.x >> 25) << 8) | (w.y >> 24)) << 5) | (i & 31u);
}
__global__ void __launch_bounds__(256) krp_k_emit_count(unsigned long long id0, unsigned int n, unsigned long long seed,
                                                        unsigned int* __restrict__ dir_bins, unsigned int sub_shift)
{
    unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    atomicAdd(dir_bins + krp_dir_bin(krp_philox(seed, id0 + i, 0u, 0u), i, sub_shift), 1u);
}

// order[slot] = index of the packet within the batch, slot taken from the scanned direction bins
__global__ void __launch_bounds__(256) krp_k_emit_order(KrpCtl* ctl, unsigned long long id0, unsigned int n, unsigned long long seed,
                                                        unsigned int* __restrict__ dir_bins, unsigned int* __restrict__ order,
                                                        unsigned int sub_shift)
{
    unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) {
        ctl->q_count[0] = n; ctl->q_count[1] = 0;
        atomicAdd(&ctl->stats.packets, (unsigned long long)n);
        atomicAdd(&ctl->stats.w_emitted, (double)n);
    }
    if (i >= n) return;
    order[atomicAdd(dir_bins + krp_dir_bin(krp_philox(seed, id0 + i, 0u, 0u), i, sub_shift), 1u)] = i;
}

// Where a flight kernel takes its queue entries from: the packet queue, or (first scattering order of an isotropic
// point source) the emission itself, computed on the fly for packet id0 + order[item] -- the 64-byte queue entry of
// a fresh packet is never written or read.
struct KrpEmitSrc {
    const unsigned int* order;     // NULL: read the queue
    unsigned long long id0, seed;
};
__device__ __forceinline__ void krp_item_load(const KrpModel& g, const KrpRecords& q, const KrpEmitSrc& es, unsigned int item,
                                              float4& pc, float4& nk, float4& S0, double& tau, unsigned long long& id)
{
    if (es.order) {
        id = es.id0 + es.order[item];
        const uint4 w = krp_philox(es.seed, id, 0u, 0u);
        tau = -log(krp_u01(w.z));
        const double ct = 1.0 - 2.0 * krp_u01(w.x);
        const double st = sqrt(1.0 - ct * ct);
        double sp, cp;
        sincospi(2.0 * krp_u01(w.y), &sp, &cp);
        nk = make_float4((float)(st * cp), (float)(st * sp), (float)ct, __uint_as_float(0u));   // R12
        pc = make_float4(g.src_p[0], g.src_p[1], g.src_p[2], __uint_as_float(g.src_cell));
        S0 = make_float4(1.f, 0.f, 0.f, 0.f);
    } else {
        pc = q.pc[item]; nk = q.nk[item]; S0 = q.S[item]; tau = q.tau[item]; id = q.id[item];
    }
}

__global__ void __launch_bounds__(256) krp_k_emit(KrpModel g, KrpCtl* ctl, KrpRecords q, KrpRecords ev,
                                                  unsigned long long id0, unsigned int n, unsigned long long seed,
                                                  unsigned int* __restrict__ dir_bins)
{
    unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) {
        ctl->q_count[0] = n; ctl->q_count[1] = 0;
        atomicAdd(&ctl->stats.packets, (unsigned long long)n);
        atomicAdd(&ctl->stats.w_emitted, (double)n);
    }
    if (i >= n) return;
    unsigned long long id = id0 + i;
    uint4 w = krp_philox(seed, id, 0u, 0u);
    double tau = -log(krp_u01(w.z));
    float nn[3];
    if (g.src_kind & 2) {
        nn[0] = g.src_n[0]; nn[1] = g.src_n[1]; nn[2] = g.src_n[2];
    } else {
        double ct = 1.0 - 2.0 * krp_u01(w.x);
        double st = sqrt(1.0 - ct * ct);
        double sp, cp;
        sincospi(2.0 * krp_u01(w.y), &sp, &cp);
        nn[0] = (float)(st * cp); nn[1] = (float)(st * sp); nn[2] = (float)ct;   // R12
    }
    uint32_t cell; float p[3];
    if (g.src_kind & 1) {
        uint4 w1 = krp_philox(seed, id, 0u, 1u), w2 = krp_philox(seed, id, 0u, 2u);
        double u = krp_u53(w1.x, w1.y);
        if (g.src_cdf) {
            double x = u * g.src_cdf[g.ncell - 1];
            long long lo = -1, hi = (long long)g.ncell - 1;      // smallest c with cdf[c] > x
            while (hi - lo > 1) { long long mid = lo + (hi - lo) / 2; if (g.src_cdf[mid] > x) hi = mid; else lo = mid; }
            cell = (uint32_t)hi;
        } else {
            double c = floor(u * (double)g.ncell);
            cell = (uint32_t)fmin(c, (double)(g.ncell - 1));
        }
        {   // linear (x fastest) -> padded id
            const uint32_t t = cell / (uint32_t)g.nx;
            const int ix = (int)(cell - t * (uint32_t)g.nx);
            const uint32_t iz = t / (uint32_t)g.ny;
            cell = krp_pad_id(g, ix, (int)(t - iz * (uint32_t)g.ny), (int)iz);
        }
        p[0] = (float)krp_u01(w2.x); p[1] = (float)krp_u01(w2.y); p[2] = (float)krp_u01(w2.z);
    } else {
        cell = g.src_cell; p[0] = g.src_p[0]; p[1] = g.src_p[1]; p[2] = g.src_p[2];
    }
    float4 pc = make_float4(p[0], p[1], p[2], __uint_as_float(cell));
    float qe = 0.f, ue = 0.f;
    if ((g.src_kind & 5) == 5 && !(g.src_kind & 2) && !g.scalar) {
        // Thermal emission of aligned grains (R22; eq. 8): direction with density (1 - omega(mu)) alpha1(mu),
        // mu = |n . B^| of the emitting cell, by rejection from isotropic candidates (candidate 0: block 0, accept = word 3;
        // candidate k: block 2 + k, accept = word 2; at most 64), Stokes (1, alpha2/alpha1, 0, 0) in the grain-frame reference
        const float4 cl = g.cell[cell];
        const double b[3] = { cl.y, cl.z, cl.w };
        const double inv_b = 1.0 / sqrt(b[0] * b[0] + b[1] * b[1] + b[2] * b[2]);
        uint4 wk = w;
        for (int k = 0; ; ++k) {
            if (k > 0) {
                wk = krp_philox(seed, id, 0u, (uint32_t)(2 + k));
                const double ct = 1.0 - 2.0 * krp_u01(wk.x), st = sqrt(1.0 - ct * ct);
                double sp, cp;
                sincospi(2.0 * krp_u01(wk.y), &sp, &cp);
                nn[0] = (float)(st * cp); nn[1] = (float)(st * sp); nn[2] = (float)ct;   // R12
            }
            const double nd[3] = { nn[0], nn[1], nn[2] };
            const double mu = fmin(fabs(nd[0] * b[0] + nd[1] * b[1] + nd[2] * b[2]) * inv_b / sqrt(nd[0] * nd[0] + nd[1] * nd[1] + nd[2] * nd[2]), 1.0);
            const double x = mu * g.xs;
            const int j = min((int)x, g.n_inc - 2);
            const double4 ta = g.opA_d[j], tb = g.opB_d[j];
            const double a1 = fma(tb.x, x, ta.x), a2 = fma(tb.y, x, ta.y), om = fma(tb.w, x, ta.w);
            if (krp_u01(k == 0 ? wk.w : wk.z) * g.src_emax < (1.0 - om) * a1 || k >= 63) {
                double th[3], ph[3], c2 = 1.0, s2 = 0.0;
                krp_basis<double>(nd, th, ph);
                if (a2 != 0.0) krp_eta2<double>(th[0] * b[0] + th[1] * b[1] + th[2] * b[2], ph[0] * b[0] + ph[1] * b[1] + ph[2] * b[2], c2, s2);
                const double qg = a2 / a1;
                qe = (float)(c2 * qg); ue = (float)(s2 * qg);       // back to the lab reference of n (eq. 7 with -eta), fp32 state (R12)
                break;
            }
        }
    }
    const unsigned int slot = dir_bins ? atomicAdd(dir_bins + krp_dir_bin(w, i, 31u), 1u) : i;   // scanned counters: first slot of the bin
    q.pc[slot] = pc;
    q.nk[slot] = make_float4(nn[0], nn[1], nn[2], __uint_as_float(0u));
    q.S[slot] = make_float4(1.f, qe, ue, 0.f);
    q.tau[slot] = tau;
    q.id[slot] = id;
    if (g.emit_records) {
        unsigned long long slot = krp_reserve64(&ctl->n_events);
        if (slot < ctl->ev_cap) {
            ev.pc[slot] = pc;
            ev.nk[slot] = make_float4(nn[0], nn[1], nn[2], __uint_as_float(0u));
            ev.S[slot] = make_float4(1.f, 0.f, 0.f, 0.f);
            ev.id[slot] = id;
            atomicAdd(&ctl->stats.records, 1ull);
        } else {
            atomicAdd(&ctl->stats.overflow, 1ull);
        }
    }
}

// one thread: open a wave.  Events appended from here on belong to this wave.
__global__ void krp_k_wave_prep(KrpCtl* ctl, int in)
{
    if (ctl->n_events > ctl->ev_cap) ctl->n_events = ctl->ev_cap;
    ctl->ev_begin = ctl->n_events;
    ctl->q_count[1 - in] = 0;
    ctl->work[0] = 0;
    ctl->n_hits = 0;
}


// ------------------------------------------------------------------------------------------
// T3/T4/T5, scalar mode: the opacity table does not depend on direction and alpha2 = alpha3 = 0,
// so a cell is 4 bytes (kappa*rho), the Stokes vector only scales and the event is where the
// optical depth alpha1*kappa*rho*s reaches tau* (PAPER.md:107-109).  One flight per queue entry:
// march cell to cell until the event or the grid edge; at an event append the pre-scatter record.
// The march is fp32; the depth still to go is kept in fp64.
// ------------------------------------------------------------------------------------------
// per-thread tallies of a flight kernel, reduced once per warp at the end
struct KrpFlightTally {
    unsigned long long steps, n_ev, n_over;
    double w_esc, w_abs, w_cut;
};
__device__ __forceinline__ void krp_tally_flush(KrpFlightTally& t, KrpCtl* ctl)
{
    t.steps = krp_warp_sum(t.steps); t.n_ev = krp_warp_sum(t.n_ev); t.n_over = krp_warp_sum(t.n_over);
    t.w_esc = krp_warp_sum(t.w_esc); t.w_abs = krp_warp_sum(t.w_abs); t.w_cut = krp_warp_sum(t.w_cut);
    if ((threadIdx.x & 31) == 0) {
        if (t.steps) atomicAdd(&ctl->stats.steps_transport, t.steps);
        if (t.n_ev) atomicAdd(&ctl->stats.events, t.n_ev);
        if (t.n_over) atomicAdd(&ctl->stats.overflow, t.n_over);
        if (t.w_esc != 0.0) atomicAdd(&ctl->stats.w_escaped, t.w_esc);
        if (t.w_abs != 0.0) atomicAdd(&ctl->stats.w_absorbed, t.w_abs);
        if (t.w_cut != 0.0) atomicAdd(&ctl->stats.w_cut, t.w_cut);
    }
}

// T5: event record (pre-scatter state), albedo weighting, termination (R12).  Called by the lanes whose flight
// ended in an event; the slot is reserved with one atomic for all of them.
__device__ __forceinline__ void krp_event_append(const KrpModel& g, KrpCtl* ctl, const KrpRecords& ev, unsigned long long id,
                                                 uint32_t cell, const float pe[3], const float n[3], uint32_t k, float W,
                                                 float omega, float qs, float us, float vs, KrpFlightTally& t)
{
    const float Wn = omega * W;
    const uint32_t kn = k + 1u;
    const bool term = (Wn < g.w_min) || ((int)kn >= g.max_scatter);
    t.w_abs += (double)W - (double)Wn;
    const unsigned long long slot = krp_reserve64(&ctl->n_events);
    if (slot < ctl->ev_cap) {
        ev.pc[slot] = make_float4(pe[0], pe[1], pe[2], __uint_as_float(cell));
        ev.nk[slot] = make_float4(n[0], n[1], n[2], __uint_as_float(kn | (term ? KRP_TERM_BIT : 0u)));
        ev.S[slot] = make_float4(Wn, qs, us, vs);
        ev.id[slot] = id;
        ++t.n_ev;
        if (term) t.w_cut += (double)Wn;
    } else {
        ++t.n_over;
        t.w_cut += (double)Wn;
    }
}

// Flight kernels are persistent: a lane whose flight has ended (event or escape) takes the next queue entry
// at the next refill point, KRP_FLIGHT_BURST cell steps apart, so that the lanes of a warp stay busy although
// flight lengths are exponentially distributed (T7, north_star "warp-level compaction of live packets").
#ifndef KRP_FLIGHT_BURST
#define KRP_FLIGHT_BURST 16
#endif

// Work distribution of the persistent flight kernels: a warp reserves KRP_FLIGHT_CHUNK consecutive queue
// entries with one atomic and hands them to its idle lanes by rank, so the global counter sees one atomic per
// chunk instead of one per refill.  wbase/wleft are warp-uniform.  Returns true when the calling lane got `item`.
#ifndef KRP_FLIGHT_CHUNK
#define KRP_FLIGHT_CHUNK 128
#endif
__device__ __forceinline__ bool krp_take_work(unsigned int* counter, unsigned int n_items, bool idle, unsigned int& wbase,
                                              unsigned int& wleft, bool& more, unsigned int& item, const unsigned int CHUNK = KRP_FLIGHT_CHUNK)
{
    const int lane = threadIdx.x & 31;
    bool got = false;
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        const unsigned want = __ballot_sync(0xffffffffu, idle && !got);
        if (want == 0u) break;
        if (wleft == 0u && more) {
            unsigned int b = 0;
            if (lane == 0) b = atomicAdd(counter, CHUNK);
            b = __shfl_sync(0xffffffffu, b, 0);
            if (b >= n_items) { more = false; }
            else { wbase = b; wleft = min(CHUNK, n_items - b); }
        }
        if (wleft == 0u) break;
        const unsigned rank = __popc(want & ((1u << lane) - 1u));
        if (idle && !got && rank < wleft) { item = wbase + rank; got = true; }
        const unsigned used = min((unsigned)__popc(want), wleft);
        wbase += used; wleft -= used;
    }
    return got;
}

enum { KRP_IDLE = 0, KRP_RUN = 1, KRP_HIT = 2, KRP_ESC = 3 };

// one re-based step in registers: returns the length of the segment in the current cell and the axis of the face
// crossed (ties x before y before z), moves to the next cell
__device__ __forceinline__ float krp_ray_advance(KrpRay& r, int& axis)
{
    float ds;
    asm("{\n\t.reg .pred px, py, pz;\n\t"
        "min.f32 %0, %1, %2, %3;\n\t"
        "setp.le.f32 px, %1, %0;\n\t"
        "setp.le.and.f32 py, %2, %0, !px;\n\t"
        "setp.gt.and.f32 pz, %2, %0, !px;\n\t"
        "sub.f32 %1, %1, %0;\n\tsub.f32 %2, %2, %0;\n\tsub.f32 %3, %3, %0;\n\t"
        "selp.s32 %5, 1, 2, py;\n\tselp.s32 %5, 0, %5, px;\n\t"
        "@px mov.f32 %1, %6;\n\t@px add.s32 %4, %4, %9;\n\t"
        "@py mov.f32 %2, %7;\n\t@py add.s32 %4, %4, %10;\n\t"
        "@pz mov.f32 %3, %8;\n\t@pz add.s32 %4, %4, %11;\n\t}"
        : "=&f"(ds), "+f"(r.rx), "+f"(r.ry), "+f"(r.rz), "+r"(r.c), "=&r"(axis)
        : "f"(r.tx), "f"(r.ty), "f"(r.tz), "r"(r.sx), "r"(r.sy), "r"(r.sz));
    return ds;
}

// Persistent form with a refill point that never waits for memory (T7).  Per warp, in shared memory: a stage of the
// next 64 queue entries (loaded coalesced, one wait per 64 flights) and a ring of finished event records (flushed 32 at
// a time: one atomic and coalesced stores per 32 events).  At a refill point a lane whose flight has ended builds its
// record from registers, drops it in the ring and starts the next staged entry; the only memory access on its way back
// into the march is the first cell gather.  Everything is warp-local: no block barrier.
#define KRP_STAGE 64
struct KrpWarpShared {
    float4 s_pc[KRP_STAGE], s_nk[KRP_STAGE], s_S[KRP_STAGE];      // staged queue entries
    double s_tau[KRP_STAGE];
    unsigned long long s_id[KRP_STAGE];
    float4 r_pc[64], r_nk[64], r_S[64];                            // ring of event records
    unsigned long long r_id[64];
};

__global__ void __launch_bounds__(256, 3) krp_k_flight_scalar(KrpModel g, KrpCtl* ctl, KrpRecords q, int in, KrpRecords ev, int n_burst, KrpEmitSrc es)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    KrpWarpShared& sh = reinterpret_cast<KrpWarpShared*>(s_raw)[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const unsigned int n_items = ctl->q_count[in];
    KrpFlightTally tl = { 0, 0, 0, 0.0, 0.0, 0.0 };
    int status = KRP_IDLE;
    bool more = true;
    unsigned int stage_n = 0, stage_pos = 0, ring_n = 0;           // warp-uniform
    // the flight in progress
    float n[3] = { 0.f, 0.f, 1.f }, p0[3] = { 0.f, 0.f, 0.f }, kr = 0.f;
    float4 S0 = make_float4(0.f, 0.f, 0.f, 0.f);
    unsigned long long id = 0;
    uint32_t c0 = 0, k = 0;
    int ax = -1;
    KrpRay ray = {};
    double D = 0.0;
    for (;;) {
        // ---- refill point -------------------------------------------------------------------------------------
        bool rec = false;
        float4 rpc, rnk, rS;
        if (status == KRP_HIT || status == KRP_ESC) {
            int h0[3], h1[3];
            krp_pad_coords(g, c0, h0[0], h0[1], h0[2]);
            krp_pad_coords(g, ray.c, h1[0], h1[1], h1[2]);
            const int crossings = abs(h1[0] - h0[0]) + abs(h1[1] - h0[1]) + abs(h1[2] - h0[2]);
            if (status == KRP_HIT) {
                const double moved = D / ((double)g.a1c * (double)kr);
                float pe[3];
                krp_event_pos(g, n, p0, c0, ray.c, ax, moved, pe);
                tl.steps += (unsigned long long)(crossings + 1);
                const float Wn = g.omc * S0.x;
                const uint32_t kn = k + 1u;
                const bool term = (Wn < g.w_min) || ((int)kn >= g.max_scatter);
                tl.w_abs += (double)S0.x - (double)Wn;
                if (term) tl.w_cut += (double)Wn;            // (an overflowing record is accounted at the flush)
                rpc = make_float4(pe[0], pe[1], pe[2], __uint_as_float(ray.c));
                rnk = make_float4(n[0], n[1], n[2], __uint_as_float(kn | (term ? KRP_TERM_BIT : 0u)));
                rS = make_float4(Wn, S0.y, S0.z, S0.w);
                rec = true;
            } else {
                tl.steps += (unsigned long long)crossings;
                tl.w_esc += (double)S0.x;
            }
            status = KRP_IDLE;
        }
        {   // records of this point go to the ring (it has room for 32: it is flushed as soon as it holds 32)
            const unsigned m = __ballot_sync(0xffffffffu, rec);
            if (rec) {
                const unsigned slot = ring_n + __popc(m & ((1u << lane) - 1u));
                sh.r_pc[slot] = rpc; sh.r_nk[slot] = rnk; sh.r_S[slot] = rS; sh.r_id[slot] = id;
            }
            ring_n += __popc(m);
            __syncwarp();
        }
        // ---- take new work from the stage; re-stage when it runs dry ---------------------------------------------
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            const unsigned want = __ballot_sync(0xffffffffu, status == KRP_IDLE);
            if (want == 0u) break;
            if (stage_pos == stage_n && more) {
                unsigned int base = 0;
                if (lane == 0) base = atomicAdd(&ctl->work[0], (unsigned int)KRP_STAGE);
                base = __shfl_sync(0xffffffffu, base, 0);
                if (base >= n_items) { more = false; }
                else {
                    stage_n = min((unsigned int)KRP_STAGE, n_items - base); stage_pos = 0;
                    for (unsigned int j = lane; j < stage_n; j += 32) {
                        float4 pc_, nk_, S_; double tau_; unsigned long long id_;
                        krp_item_load(g, q, es, base + j, pc_, nk_, S_, tau_, id_);
                        sh.s_pc[j] = pc_; sh.s_nk[j] = nk_; sh.s_S[j] = S_; sh.s_tau[j] = tau_; sh.s_id[j] = id_;
                    }
                    __syncwarp();
                }
            }
            const unsigned avail = stage_n - stage_pos;
            if (avail == 0u) break;
            const unsigned rank = __popc(want & ((1u << lane) - 1u));
            if (status == KRP_IDLE && rank < avail) {
                const unsigned j = stage_pos + rank;
                const float4 pc_ = sh.s_pc[j], nk_ = sh.s_nk[j];
                S0 = sh.s_S[j]; D = sh.s_tau[j]; id = sh.s_id[j];
                n[0] = nk_.x; n[1] = nk_.y; n[2] = nk_.z; k = __float_as_uint(nk_.w);
                p0[0] = pc_.x; p0[1] = pc_.y; p0[2] = pc_.z; c0 = __float_as_uint(pc_.w);
                krp_ray_init(g, c0, p0, n, ray);
                ax = -1;
                KRP_CK(g, ray.c);
                kr = __ldg(g.kr + ray.c);
                status = KRP_RUN;
            }
            stage_pos += min((unsigned)__popc(want), avail);
            __syncwarp();
        }
        const bool any_run = __any_sync(0xffffffffu, status == KRP_RUN);
        // ---- flush 32 records (or, at the end, what is left): one atomic, coalesced stores ---------------------------
        while (ring_n >= 32u || (!any_run && ring_n > 0u)) {
            const unsigned int cnt = min(ring_n, 32u);
            unsigned long long base = 0;
            if (lane == 0) base = atomicAdd(&ctl->n_events, (unsigned long long)cnt);
            base = __shfl_sync(0xffffffffu, base, 0);
            if ((unsigned)lane < cnt) {
                const unsigned long long slot = base + lane;
                const float4 a = sh.r_pc[lane], b = sh.r_nk[lane], c = sh.r_S[lane];
                if (slot < ctl->ev_cap) {
                    ev.pc[slot] = a; ev.nk[slot] = b; ev.S[slot] = c; ev.id[slot] = sh.r_id[lane];
                    ++tl.n_ev;
                } else {
                    ++tl.n_over;
                    if (!(__float_as_uint(b.w) & KRP_TERM_BIT)) tl.w_cut += (double)c.x;     // a lost packet counts as cut
                }
            }
            __syncwarp();
            {   // move the rest to the front
                const bool mv = ring_n > 32u && (unsigned)lane < ring_n - 32u;
                float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a, c = a;
                unsigned long long d = 0;
                if (mv) { a = sh.r_pc[32 + lane]; b = sh.r_nk[32 + lane]; c = sh.r_S[32 + lane]; d = sh.r_id[32 + lane]; }
                __syncwarp();
                if (mv) { sh.r_pc[lane] = a; sh.r_nk[lane] = b; sh.r_S[lane] = c; sh.r_id[lane] = d; }
            }
            ring_n -= cnt;
            __syncwarp();
        }
        if (!any_run) break;
        // ---- burst ---------------------------------------------------------------------------------------------------
#pragma unroll 1
        for (int burst = 0; burst < n_burst; ++burst) {
            if (status == KRP_RUN) {
                const float dt1 = g.a1c * kr * krp_ray_ds(ray);
                if ((double)dt1 >= D) {
                    status = KRP_HIT;                // event inside this cell, located at the refill point
                } else {
                    D -= (double)dt1;
                    krp_ray_advance(ray, ax);
                    KRP_CK(g, ray.c);
                    kr = __ldg(g.kr + ray.c);
                    if (kr < 0.f) status = KRP_ESC;  // halo: the packet left the grid
                }
            }
        }
    }
    krp_tally_flush(tl, ctl);
}

// The same flight with a static assignment (one queue entry per thread and grid stride, the warp's 32 flights
// start and are closed together): no refill logic at all.  Cheaper when flights are short (C2: a point source
// inside a dense ring, most flights end within a few cells), selected with flight_burst = 1.
__global__ void __launch_bounds__(256, 4) krp_k_flight_scalar_static(KrpModel g, KrpCtl* ctl, KrpRecords q, int in, KrpRecords ev, KrpEmitSrc es, double* __restrict__ flen)
{
    const unsigned int n_items = ctl->q_count[in];
    KrpFlightTally tl = { 0, 0, 0, 0.0, 0.0, 0.0 };
    for (unsigned int item = blockIdx.x * blockDim.x + threadIdx.x; item < n_items; item += gridDim.x * blockDim.x) {
        float4 pc, nk, S0; double D; unsigned long long id;
        krp_item_load(g, q, es, item, pc, nk, S0, D, id);
        const float n[3] = { nk.x, nk.y, nk.z };
        const float p0[3] = { pc.x, pc.y, pc.z };
        const uint32_t c0 = __float_as_uint(pc.w);
        KrpRay ray;
        krp_ray_init(g, c0, p0, n, ray);
        // The march runs two cells ahead of the optical-depth test, so that two gathers are in flight: the stages hold
        // the cell id, the axis of its entry face, its segment length and its kappa*rho.  The look-ahead may step one
        // cell past the halo cell that ends the flight (inside the allocation's margin); its value is never used.
        bool hit = false;
        int ax_cur = -1, ax_nxt, ax_new;
        uint32_t c_cur = ray.c;
        KRP_CK(g, c_cur);
        float kr_cur = __ldg(g.kr + c_cur);
        float ds_cur = krp_ray_advance(ray, ax_nxt);
        uint32_t c_nxt = ray.c;
        KRP_CK(g, c_nxt);
        float kr_nxt = __ldg(g.kr + c_nxt);
        float ds_nxt = krp_ray_advance(ray, ax_new);
#pragma unroll 2
        for (;;) {
            const uint32_t c_new = ray.c;
            KRP_CK(g, (int)c_new);
            const float kr_new = __ldg(g.kr + (int)c_new);       // signed: the look-ahead may sit before the array's first cell
            const float dt1 = g.a1c * kr_cur * ds_cur;
            if ((double)dt1 >= D) { hit = true; break; }      // event inside the current cell
            D -= (double)dt1;
            if (kr_nxt < 0.f) { c_cur = c_nxt; break; }        // halo: the packet left the grid
            c_cur = c_nxt; ax_cur = ax_nxt; kr_cur = kr_nxt; ds_cur = ds_nxt;
            c_nxt = c_new; ax_nxt = ax_new; kr_nxt = kr_new;
            ds_nxt = krp_ray_advance(ray, ax_new);
        }
        int h0[3], h1[3];
        krp_pad_coords(g, c0, h0[0], h0[1], h0[2]);
        krp_pad_coords(g, c_cur, h1[0], h1[1], h1[2]);
        const int crossings = abs(h1[0] - h0[0]) + abs(h1[1] - h0[1]) + abs(h1[2] - h0[2]);
        if (!hit) {
            tl.steps += (unsigned long long)crossings; tl.w_esc += (double)S0.x;
            if (flen) flen[item] = __longlong_as_double(0x7ff0000000000000ll);       // two-step form: deposit to the grid edge
            continue;
        }
        tl.steps += (unsigned long long)(crossings + 1);
        const double moved = D / ((double)g.a1c * (double)kr_cur);
        float pe[3];
        krp_event_pos(g, n, p0, c0, c_cur, ax_cur, moved, pe);
        if (flen) flen[item] = krp_path_length(g, n, p0, c0, pe, c_cur);
        krp_event_append(g, ctl, ev, id, c_cur, pe, n, __float_as_uint(nk.w), S0.x, g.omc, S0.y, S0.z, S0.w, tl);
    }
    krp_tally_flush(tl, ctl);
}

// ------------------------------------------------------------------------------------------
// T4  in-cell event location (R7), general mode, fp64 (the root decides where the event lies).  With the
// Stokes vector carried as e^{-A}(i,q,u,v) and D = tau* - A the scalar depth still to go at cell entry,
// the event is at the t solving
//   alpha1 t - ln( cosh(alpha2 t) - (q_g/i) sinh(alpha2 t) ) = D + ln i  =: R ,
// whose left side is increasing and concave: Newton from R/alpha1 lands left of the root after one step
// and then rises monotonically.  alpha2 = 0 is the closed form t = R/alpha1.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ double krp_event_solve_d(double R, double qq, double a1, double a2, double tmax);

// 1/sqrt(1+e) for |e| << 1 (unit vectors stored in fp32 have |v|^2 = 1 + O(1e-7))
__device__ __forceinline__ double krp_rsqrt_near1(double vv)
{
    double e = vv - 1.0;
    return 1.0 + e * (-0.5 + e * (0.375 - 0.3125 * e));
}

// spherical basis (eq. 4-5, pole rule R10) of a direction that is unit to within fp32 rounding, fp64, with one
// division and one square root: |n| is divided out by the series of krp_rsqrt_near1
__device__ __forceinline__ void krp_basis_unit_d(const double n[3], double th[3], double ph[3])
{
    const double s2 = n[0] * n[0] + n[1] * n[1];
    const double inv_r = krp_rsqrt_near1(s2 + n[2] * n[2]);
    const double s = sqrt(s2);
    double cp = 1.0, sp = 0.0;
    if (s2 >= 1e-24) { const double is = 1.0 / s; cp = n[0] * is; sp = n[1] * is; }
    const double ct = n[2] * inv_r, st = s * inv_r;
    th[0] = ct * cp; th[1] = ct * sp; th[2] = -st;
    ph[0] = -sp; ph[1] = cp; ph[2] = 0.0;
}

// ------------------------------------------------------------------------------------------
// T3/T4/T5, general mode (direction-dependent, dichroic opacity; 16-byte cells).  Everything that
// decides in which cell the event falls -- segment lengths, alpha1(mu), the scalar depth D and the
// normalised intensity i -- is carried in fp64 (an integer decided by
// floating point is taken in the oracle's precision; in a clumpy medium a difference in the last
// bit of an event position is amplified by the density contrast at every later scattering).  That
// includes the Stokes vector: i depends on the grain-frame Q of every cell crossed, and in optically
// thin cells (C5 at 512^3: kappa*rho*dx ~ 0.02) an error of 1e-10 in ln i moves the event by an fp32
// ulp of the cell-local coordinate, so q,u,v and the reference rotation are fp64 here too (the
// imaging march, which decides no integer but the pixel, is fp32).
// ------------------------------------------------------------------------------------------
struct KrpCellCoef {
    double a1, a2, a3, dtau, dt1;   // alpha_i(mu), kappa*rho*ds, alpha1*kappa*rho*ds
    float omega;                    // albedo(mu)
};

__device__ __forceinline__ void krp_cell_coef(const KrpModel& g, const float4 cl, const double nd[3], double xs,
                                              double ds, KrpCellCoef& c)
{
    const double bx = cl.y, by = cl.z, bz = cl.w;
    const double mu = fabs(nd[0] * bx + nd[1] * by + nd[2] * bz) * krp_rsqrt_near1(bx * bx + by * by + bz * bz);
    const double x = mu * xs;        // mu <= 1 up to rounding: the index is clamped, the last segment extends by that much
    const int j = min((int)x, g.n_inc - 2);
    // the table as fp64 intercept + slope per segment (same piecewise-linear function, R13)
    const double4 ta = g.opA_d[j], tb = g.opB_d[j];
    c.a1 = fma(tb.x, x, ta.x);
    c.a2 = fma(tb.y, x, ta.y);
    c.a3 = fma(tb.z, x, ta.z);
    c.omega = (float)fma(tb.w, x, ta.w);
    c.dtau = (double)cl.x * ds;
    c.dt1 = c.a1 * c.dtau;
}

// sinh(x), cosh(x)-1 and sin(y), cos(y)-1 in fp64 for |x|, |y| < 0.35: Taylor series, 4 terms below 0.02 (remainder
// < 1e-19 relative), 8 terms (to x^15 / x^16) otherwise.  The coefficients sit in constant memory: a DFMA takes one
// operand straight from a constant bank, whereas a 64-bit literal costs two moves to build every time it is used
// (a third of the instructions of the flight loop before); the range tests look at the high word only.
__constant__ double KRP_SER[14] = {
    1.0 / 6, 1.0 / 120, 1.0 / 5040, 1.0 / 362880, 1.0 / 39916800, 1.0 / 6227020800.0, 1.0 / 1307674368000.0,       // odd: x^3 .. x^15
    1.0 / 24, 1.0 / 720, 1.0 / 40320, 1.0 / 3628800, 1.0 / 479001600, 1.0 / 87178291200.0, 1.0 / 20922789888000.0  // even: x^4 .. x^16
};
__device__ __forceinline__ bool krp_abs_below(double x, int hi) { return (__double2hiint(x) & 0x7fffffff) < hi; }
#define KRP_HI_0P35 0x3fd66666      // high word of 0.35
#define KRP_HI_4EM4 0x3f3a36e2      // high word of 4e-4

__device__ __forceinline__ void krp_sinh_coshm1_d(double x, double& sh, double& chm1)
{
    const double z = x * x;
    const double* c = KRP_SER;
    if (__double2hiint(z) < KRP_HI_4EM4) {
        sh = x * (1.0 + z * (c[0] + z * (c[1] + z * c[2])));
        chm1 = z * (0.5 + z * (c[7] + z * (c[8] + z * c[9])));
    } else {
        asm volatile("");      // keeps the long series a real branch (ptxas otherwise evaluates both and selects)
        sh = x * (1.0 + z * (c[0] + z * (c[1] + z * (c[2] + z * (c[3] + z * (c[4] + z * (c[5] + z * c[6])))))));
        chm1 = z * (0.5 + z * (c[7] + z * (c[8] + z * (c[9] + z * (c[10] + z * (c[11] + z * (c[12] + z * c[13])))))));
    }
}
__device__ __forceinline__ void krp_sin_cosm1_d(double y, double& sy, double& cym1)
{
    const double z = y * y;
    const double* c = KRP_SER;
    if (__double2hiint(z) < KRP_HI_4EM4) {
        sy = y * (1.0 - z * (c[0] - z * (c[1] - z * c[2])));
        cym1 = -z * (0.5 - z * (c[7] - z * (c[8] - z * c[9])));
    } else {
        asm volatile("");
        sy = y * (1.0 - z * (c[0] - z * (c[1] - z * (c[2] - z * (c[3] - z * (c[4] - z * (c[5] - z * c[6])))))));
        cym1 = -z * (0.5 - z * (c[7] - z * (c[8] - z * (c[9] - z * (c[10] - z * (c[11] - z * (c[12] - z * c[13])))))));
    }
}

// (defined here, after the series it uses)  In a thin cell (|alpha2 tmax| < 0.35, every cell of C4 and C5) the
// hyperbolic functions and the logarithm of the Newton step come from short series instead of the library routines.
__device__ __forceinline__ double krp_event_solve_d(double R, double qq, double a1, double a2, double tmax)
{
    double t = R / a1;
    if (a2 != 0.0) {
#pragma unroll 1
        for (int it = 0; it < 40; ++it) {
            const double x = a2 * t;
            double sh, chm1;
            if (krp_abs_below(x, KRP_HI_0P35)) krp_sinh_coshm1_d(x, sh, chm1);
            else {      // one exponential and one division for both (no cancellation from |x| = 0.35 on)
                asm volatile("");
                const double e = exp(fabs(x)), ie = 1.0 / e;
                sh = copysign(0.5 * (e - ie), x); chm1 = 0.5 * (e + ie) - 1.0;
            }
            const double gm1 = chm1 - qq * sh;
            double lg;
            if (fabs(gm1) < 0.01) {       // ln(1+g) = g - g^2/2 + ... to g^8 (remainder < 1e-19)
                lg = gm1 * (1.0 - gm1 * (0.5 - gm1 * (1.0 / 3 - gm1 * (0.25 - gm1 * (0.2 - gm1 * (1.0 / 6 - gm1 * (1.0 / 7 - gm1 * 0.125)))))));
            } else {
                asm volatile("");
                lg = log1p(gm1);
            }
            const double h = a1 * t - lg - R;
            const double hp = a1 - a2 * (sh - qq * (1.0 + chm1)) / (1.0 + gm1);
            const double dt = h / hp;
            t = fmin(fmax(t - dt, 0.0), tmax);
            if (fabs(dt) <= 1e-13 * t) break;      // quadratic convergence: the step after this one would be ~1e-26 t
        }
    }
    return fmin(fmax(t, 0.0), tmax);
}

// Source-free App. A step over the whole cell on the grain-frame state (i, qg, ug, v), fp64, with the common factor
// e^{-alpha1 dtau} (thin) or e^{-(alpha1 - |alpha2|) dtau} (thick) left to the scalar depth; `depth` is what the
// scalar depth grows by.
__device__ __forceinline__ void krp_appA_d(double i, double qg, double ug, double v, const KrpCellCoef& c,
                                           double& i_n, double& qg_n, double& ug_n, double& v_n, double& depth)
{
    const double x = c.a2 * c.dtau, y = c.a3 * c.dtau;
    double sy, cym1;
    if (krp_abs_below(y, KRP_HI_0P35)) krp_sin_cosm1_d(y, sy, cym1);
    else { double cy; sincos(y, &sy, &cy); cym1 = cy - 1.0; }
    const double un = ug + (ug * cym1 - v * sy), vn = v + (ug * sy + v * cym1);
    if (krp_abs_below(x, KRP_HI_0P35)) {
        double sh, chm1;
        krp_sinh_coshm1_d(x, sh, chm1);
        i_n = i + (i * chm1 - qg * sh);
        qg_n = qg + (qg * chm1 - i * sh);
        ug_n = un; v_n = vn;
        depth = c.dt1;
    } else {
        // thick cell: factor e^{-|alpha2 dtau|} moved into the scalar depth (no overflow at dtau ~ 1e3)
        const double ax = fabs(x), f = exp(-ax), E = f * f, sg = x > 0.0 ? 1.0 : -1.0;      // one exponential for both factors
        i_n = 0.5 * ((i - sg * qg) + (i + sg * qg) * E);
        qg_n = 0.5 * ((qg - sg * i) + (qg + sg * i) * E);
        ug_n = f * un; v_n = f * vn;
        depth = c.dt1 - ax;
    }
}

// the same evolved to depth t inside the cell, thin or thick, normalised to I = 1 (R7)
__device__ __forceinline__ void krp_appA_to_d(double i, double qg, double ug, double v, double a2, double a3, double t,
                                              double& qt, double& ut, double& vt)
{
    const double x = a2 * t, y = a3 * t;
    double sy, cy, sh, ch;
    if (fabs(y) < 0.35) { double cym1; krp_sin_cosm1_d(y, sy, cym1); cy = 1.0 + cym1; }
    else { asm volatile(""); sincos(y, &sy, &cy); }
    if (fabs(x) < 0.35) { double chm1; krp_sinh_coshm1_d(x, sh, chm1); ch = 1.0 + chm1; }
    else { const double e = exp(fabs(x)), ie = 1.0 / e; sh = copysign(0.5 * (e - ie), x); ch = 0.5 * (e + ie); }
    const double it = i * ch - qg * sh;
    const double inv = 1.0 / it;
    qt = (qg * ch - i * sh) * inv;
    ut = (ug * cy - v * sy) * inv;
    vt = (ug * sy + v * cy) * inv;
}

// Two builds: blocks of up to 128 threads, five per SM (20 warps, 96 registers: the default, measured best of 16, 18, 20, 24 and 32
// warps per SM on C4 and C5) and blocks of up to 256 threads, three per SM (24 warps, 80 registers) for krp_tune's larger blocks.
template <int TPB, int MINB>
__global__ void __launch_bounds__(TPB, MINB) krp_k_flight_general(KrpModel g, KrpCtl* ctl, KrpRecords q, int in, KrpHits hits, int n_burst, KrpEmitSrc es, double* __restrict__ flen)
{
    const unsigned int n_items = ctl->q_count[in];
    KrpFlightTally tl = { 0, 0, 0, 0.0, 0.0, 0.0 };
    const double xs = g.xs;
    const float inv_guard = 1.f / g.guard;
    // queue entries a warp reserves per visit to the launch's work counter: long flights (refill every 8 or 16 steps) take 32, so
    // that the last entries of a wave spread over all warps (C4 flights 35.9 -> 34.8 ms, C5 66.6 -> 65.2); flights of a cell or two,
    // which refill after every step, would queue on that one address (C3: 7.32 ms with 128, 7.56 with 32, 8.58 with 16)
    const unsigned int chunk = n_burst == 1 ? (unsigned int)KRP_FLIGHT_CHUNK : 32u;
    int status = KRP_IDLE;
    bool more = true;
    unsigned int item = 0, wbase = 0, wleft = 0;
    // state of the flight in progress (all fp64: it decides where the event falls)
    double nd[3] = { 0.0, 0.0, 1.0 }, th[3] = { 0.0, 0.0, 0.0 }, ph[3] = { 0.0, 0.0, 0.0 };
    double D = 0.0, i = 1.0, qs = 0.0, us = 0.0, vs = 0.0;
    float arm = 0.f;        // tau*/guard minus the fp32 sum of alpha1 dtau: the fp64 event test is armed once it is <= 0
    unsigned int nsteps = 0, nwrap = 0;
    KrpRayD ray = {};
    float4 cl = make_float4(0.f, 0.f, 0.f, 1.f), cl_f = cl;
    bool fresh = false;
    for (;;) {
        // refill point: a lane whose flight reached the cell of its event leaves the entry state in the hit queue (one
        // reservation for all such lanes of the warp) -- event location, record and albedo weighting run in their own,
        // fully converged kernel (krp_k_event_general) instead of inside the marching warp
        if (status == KRP_HIT) {
            const unsigned int slot = krp_reserve32(&ctl->n_hits);
            hits.ic[slot] = make_uint2(item, ray.c);
            hits.Di[slot] = make_double2(D, i);
            hits.qu[slot] = make_double2(qs, us);
            hits.vr[slot] = make_double2(vs, ray.rx);
            hits.ryz[slot] = make_double2(ray.ry, ray.rz);
            tl.steps += nsteps;
            status = KRP_IDLE;
        } else if (status == KRP_ESC) {
            if (flen) flen[item] = __longlong_as_double(0x7ff0000000000000ll);
            tl.steps += nsteps;
            tl.w_esc += es.order ? 1.0 : (double)q.S[item].x;
            status = KRP_IDLE;
        }
        if (krp_take_work(&ctl->work[0], n_items, status == KRP_IDLE, wbase, wleft, more, item, chunk)) {
            float4 pc, nk, S0; double tau0; unsigned long long id_;
            krp_item_load(g, q, es, item, pc, nk, S0, tau0, id_);
            const float n[3] = { nk.x, nk.y, nk.z }, p0[3] = { pc.x, pc.y, pc.z };
            krp_rayd_init(g, __float_as_uint(pc.w), p0, n, ray);
            // the first cell of the new flight goes to registers of its own and is taken over one step later: the warp's other
            // flights march on while it is in flight (a register is scoreboarded per warp, whoever's lanes wait for it)
            KRP_CK(g, ray.c);
            asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(cl_f.x), "=f"(cl_f.y), "=f"(cl_f.z), "=f"(cl_f.w) : "l"(g.cell + ray.c));
            fresh = true;
            nd[0] = n[0]; nd[1] = n[1]; nd[2] = n[2];
            krp_basis_unit_d(nd, th, ph);
            {   // n^ = n/|n| once per flight (|n|^2 = 1 + O(1e-7)): mu = |n^ . B| / |B| in every cell
                const double inv_n = krp_rsqrt_near1(nd[0] * nd[0] + nd[1] * nd[1] + nd[2] * nd[2]);
                nd[0] *= inv_n; nd[1] *= inv_n; nd[2] *= inv_n;
            }
            D = tau0; i = 1.0;
            qs = S0.y; us = S0.z; vs = S0.w;      // lab reference
            arm = (float)tau0 * inv_guard; nsteps = 0; nwrap = 0;
            status = KRP_RUN;
        }
        if (!__any_sync(0xffffffffu, status == KRP_RUN)) break;
#pragma unroll 1
        for (int burst = 0; burst < n_burst; ++burst) {
            if (status != KRP_RUN) continue;
            if (fresh) {
                if (burst == 0 && n_burst > 1) continue;
                cl = cl_f; fresh = false;
            }
            // face crossed next (ties x before y before z), decided once per step: segment length, next cell and the
            // re-based distances all follow from the two predicates
            const bool ax = (ray.rx <= ray.ry) & (ray.rx <= ray.rz);
            const bool ay = !ax & (ray.ry <= ray.rz);
            const double ds = ax ? ray.rx : (ay ? ray.ry : ray.rz);
            ++nsteps;
            // the next cell is requested now, so that its latency overlaps the fp64 update of this one
            const uint32_t c_next = ray.c + (uint32_t)(ax ? ray.sx : (ay ? ray.sy : ray.sz));
            float4 cn;      // a load the compiler may neither duplicate nor move: it has to be in flight during the update below
            KRP_CK(g, c_next);
            asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(cn.x), "=f"(cn.y), "=f"(cn.z), "=f"(cn.w) : "l"(g.cell + c_next));
            if (cl.x > 0.f) {
                KrpCellCoef cc;
                krp_cell_coef(g, cl, nd, xs, ds, cc);
                arm -= (float)cc.dt1;
                const bool near_end = arm <= 0.f;
                if (cc.a2 == 0.0 && cc.a3 == 0.0) {
                    if (near_end && cc.dt1 >= D + log(i)) { status = KRP_HIT; continue; }
                    D -= cc.dt1;
                } else {
                    const double bx = cl.y, by = cl.z, bz = cl.w;
                    double c2, s2;
                    krp_eta2_d(th[0] * bx + th[1] * by + th[2] * bz, ph[0] * bx + ph[1] * by, c2, s2);      // phi^_z = 0
                    const double qg_e = c2 * qs + s2 * us, ug_e = -s2 * qs + c2 * us;          // eq. 7
                    double i_new, qg, ug, vg, depth;
                    krp_appA_d(i, qg_e, ug_e, vs, cc, i_new, qg, ug, vg, depth);
                    const double Dn = D - depth;
                    // The event test is ln i_new + Dn <= 0.  The fp64 log (~110 instructions, which a warp would execute for the
                    // one or two lanes that are near their event: 27 % of all warp-steps on C4, profiles/r2g) is bracketed first:
                    // for |u| <= 1/4, u = i_new - 1, the series P4 = u - u^2/2 + u^3/3 - u^4/4 has |ln(1+u) - P4| <= |u|^5/(5 (1 - |u|))
                    // <= 4/15 |u|^5, so the decision is settled unless P4 + Dn lies within that band of zero -- only then the log itself
                    if (near_end) {
                        const double u = i_new - 1.0;
                        bool hit;
                        if (fabs(u) <= 0.25) {
                            const double u2 = u * u;
                            const double p4 = u + u2 * (-0.5 + u * (1.0 / 3.0 - 0.25 * u));
                            const double band = (4.0 / 15.0) * u2 * u2 * fabs(u);
                            const double v = p4 + Dn;
                            if (v > band) hit = false;
                            else if (v < -band) hit = true;
                            else hit = log(i_new) + Dn <= 0.0;
                        } else {
                            hit = log(i_new) + Dn <= 0.0;
                        }
                        if (hit) { status = KRP_HIT; continue; }   // state stays at cell entry
                    }
                    qs = c2 * qg - s2 * ug; us = s2 * qg + c2 * ug; vs = vg;
                    i = i_new; D = Dn;
                }
            }
            ray.rx = ax ? ray.tx : ray.rx - ds;
            ray.ry = ay ? ray.ty : ray.ry - ds;
            ray.rz = (ax | ay) ? ray.rz - ds : ray.tz;
            ray.c = c_next;
            cl = cn;
            if (cl.x < 0.f) {                        // halo: the packet left the grid -- or crosses a periodic face (R20)
                int off[3] = { 0, 0, 0 };
                if (g.periodic && nwrap < KRP_MAX_WRAPS && krp_wrap(g, ray.c, off)) {
                    ++nwrap;
                    KRP_CK(g, ray.c);
                    asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(cl.x), "=f"(cl.y), "=f"(cl.z), "=f"(cl.w) : "l"(g.cell + ray.c));
                } else status = KRP_ESC;
            }
        }
    }
    krp_tally_flush(tl, ctl);
}
// T4/T5, general mode: one thread per flight that ended in an event.  From the state at the entry of the event cell:
// solve for the depth t of the event (krp_event_solve_d), evolve the Stokes vector to t and normalise it to I = 1 (R7),
// place the event, write the record (slot = first event of the wave + hit index: coalesced, no atomic), weight by the albedo.
// 64 registers (8 blocks per SM): a hit is three dependent reads away from its arithmetic (hit -> queue entry -> cell) and the kernel
// waits for them (43 % of its stall samples on C3, profiles/r2r) -- warps in flight count for more than the 250 bytes of spills.
// Measured on C3, flights + events per 2^22 packets: 118 registers (no bound) 8.29 ms, 96: 7.85, 80: 7.79, 64: 7.32; requesting the
// next hit's queue entry and cell from L2 one iteration ahead made every variant slower (64 registers: 8.04 ms).
__global__ void __launch_bounds__(128, 8) krp_k_event_general(KrpModel g, KrpCtl* ctl, KrpRecords q, int in, KrpHits hits, KrpRecords ev,
                                                           KrpEmitSrc es, double* __restrict__ flen)
{
    const unsigned int n_hits = ctl->n_hits;
    const unsigned long long ev_begin = ctl->ev_begin, ev_cap = ctl->ev_cap;
    KrpFlightTally tl = { 0, 0, 0, 0.0, 0.0, 0.0 };
    for (unsigned int h = blockIdx.x * blockDim.x + threadIdx.x; h < n_hits; h += gridDim.x * blockDim.x) {
        const uint2 ic = hits.ic[h];
        const double2 Di = hits.Di[h], qu = hits.qu[h], vr = hits.vr[h], ryz = hits.ryz[h];
        const unsigned int item = ic.x; const uint32_t cell = ic.y;
        const double D = Di.x, i = Di.y;
        double qs = qu.x, us = qu.y, vs = vr.x;
        const double rx = vr.y, ry = ryz.x, rz = ryz.y;
        float4 pc, nk, S0; double tau_; unsigned long long id;
        krp_item_load(g, q, es, item, pc, nk, S0, tau_, id);
        const float n[3] = { nk.x, nk.y, nk.z };
        // the flight's direction constants, exactly as the marching kernel set them up
        double nd[3] = { n[0], n[1], n[2] }, th[3], ph[3];
        krp_basis_unit_d(nd, th, ph);
        {
            const double inv_n = krp_rsqrt_near1(nd[0] * nd[0] + nd[1] * nd[1] + nd[2] * nd[2]);
            nd[0] *= inv_n; nd[1] *= inv_n; nd[2] *= inv_n;
        }
        const float4 cl = g.cell[cell];
        const double ds = fmin(rx, fmin(ry, rz));
        KrpCellCoef cc;
        krp_cell_coef(g, cl, nd, g.xs, ds, cc);
        const double R = D + log(i);
        double moved;
        if (cc.a2 == 0.0 && cc.a3 == 0.0) {
            moved = (R / cc.a1) / (double)cl.x;
            const double inv = 1.0 / i;
            qs *= inv; us *= inv; vs *= inv;
        } else {
            const double bx = cl.y, by = cl.z, bz = cl.w;
            double c2, s2;
            krp_eta2_d(th[0] * bx + th[1] * by + th[2] * bz, ph[0] * bx + ph[1] * by, c2, s2);      // phi^_z = 0
            const double qg_e = c2 * qs + s2 * us, ug_e = -s2 * qs + c2 * us;
            const double t = krp_event_solve_d(R, qg_e / i, cc.a1, cc.a2, cc.dtau);
            double qt, ut, vt;
            krp_appA_to_d(i, qg_e, ug_e, vs, cc.a2, cc.a3, t, qt, ut, vt);
            qs = c2 * qt - s2 * ut; us = s2 * qt + c2 * ut; vs = vt;
            moved = t / (double)cl.x;
        }
        float pe[3];
        pe[0] = krp_locald(n[0], rx, g.inv_dd[0], moved, pc.x);
        pe[1] = krp_locald(n[1], ry, g.inv_dd[1], moved, pc.y);
        pe[2] = krp_locald(n[2], rz, g.inv_dd[2], moved, pc.z);
        if (flen) { const float p0[3] = { pc.x, pc.y, pc.z }; flen[item] = krp_path_length(g, n, p0, __float_as_uint(pc.w), pe, cell); }
        // T5: record, albedo weighting, termination (R12)
        const float W = S0.x, Wn = cc.omega * W;
        const uint32_t kn = __float_as_uint(nk.w) + 1u;
        const bool term = (Wn < g.w_min) || ((int)kn >= g.max_scatter);
        tl.w_abs += (double)W - (double)Wn;
        const unsigned long long slot = ev_begin + h;
        if (slot < ev_cap) {
            ev.pc[slot] = make_float4(pe[0], pe[1], pe[2], __uint_as_float(cell));
            ev.nk[slot] = make_float4(n[0], n[1], n[2], __uint_as_float(kn | (term ? KRP_TERM_BIT : 0u)));
            ev.S[slot] = make_float4(Wn, (float)qs, (float)us, (float)vs);
            ev.id[slot] = id;
            ++tl.n_ev;
            if (term) tl.w_cut += (double)Wn;
        } else {
            ++tl.n_over;
            tl.w_cut += (double)Wn;
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) atomicAdd(&ctl->n_events, (unsigned long long)n_hits);   // may run past ev_cap: clamped by the readers
    krp_tally_flush(tl, ctl);
}

// ------------------------------------------------------------------------------------------
// quaternion helpers (eq. 1-3): q = (w, a);  q* v q  and  q v q*  for a pure
// quaternion v, expanded from the Hamilton product:  v -+ 2w (a x v) + 2 a x (a x v).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void krp_cross(const double a[3], const double b[3], double o[3])
{
    o[0] = a[1] * b[2] - a[2] * b[1]; o[1] = a[2] * b[0] - a[0] * b[2]; o[2] = a[0] * b[1] - a[1] * b[0];
}
__device__ __forceinline__ double krp_dot(const double a[3], const double b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

__device__ __forceinline__ void krp_quat_rotate(const double q[4], const double v[3], double sign, double o[3])
{
    const double a[3] = { q[1], q[2], q[3] };
    double c1[3], c2[3];
    krp_cross(a, v, c1);
    krp_cross(a, c1, c2);
    for (int j = 0; j < 3; ++j) o[j] = v[j] + 2.0 * (sign * q[0] * c1[j] + c2[j]);
}

// (Q,U) -> reference turned by eta (eq. 7), given cos(2 eta), sin(2 eta)
__device__ __forceinline__ void krp_rot_qu(double& Q, double& U, double c2, double s2)
{
    double q = c2 * Q + s2 * U, u = -s2 * Q + c2 * U;
    Q = q; U = u;
}

// ------------------------------------------------------------------------------------------
// NEXT-2: full scattering matrix Z(vartheta_in, vartheta_out, dphi) in the grain frame (R21): trilinear interpolation of
// `rows` rows (row 1 alone decides the acceptance of a candidate direction), angles in degrees, dphi periodic
// ------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ void krp_zt_at(const KrpZt g, T ti_deg, T to_deg, T dphi_deg, int rows, T M[16])
{
    const T xi = ti_deg * (T)(g.ni - 1) / T(180), xo = to_deg * (T)(g.no - 1) / T(180);
    T xd = dphi_deg * (T)g.nd / T(360);
    xd -= floor(xd / (T)g.nd) * (T)g.nd;
    int i = max(0, min((int)floor(xi), g.ni - 2)), o = max(0, min((int)floor(xo), g.no - 2)), d = min((int)floor(xd), g.nd - 1);
    const T wi = xi - (T)i, wo = xo - (T)o, wd = xd - (T)d;
    const int d1 = (d + 1) % g.nd;
    for (int k = 0; k < 4 * rows; ++k) M[k] = T(0);
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b)
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const T w = (a ? wi : T(1) - wi) * (b ? wo : T(1) - wo) * (c ? wd : T(1) - wd);
                const float4* e = reinterpret_cast<const float4*>(g.zt + (((size_t)(i + a) * g.no + (o + b)) * g.nd + (c ? d1 : d)) * 16);
                for (int r = 0; r < rows; ++r) {
                    const float4 v = __ldg(e + r);
                    M[4 * r] += w * (T)v.x; M[4 * r + 1] += w * (T)v.y; M[4 * r + 2] += w * (T)v.z; M[4 * r + 3] += w * (T)v.w;
                }
            }
}

// I1 with the full Z (R21): both directions into the grain frame of the event cell (z_GF = B^, x_GF, y_GF = theta^, phi^ of B^:
// eq. 2 is R_z(phi_B) R_y(theta_B)), Stokes reference lab -> grain frame (eq. 6-7), Z s / (4 pi N), back to theta^_obs.
__device__ __forceinline__ void krp_peel_z(const KrpZt g, const float bh[3], const float n[3], float4 Se, const float on[3], const float oth[3], const float oph[3], float S[4])
{
    float thB[3], phB[3], th[3], ph[3];
    krp_basis<float>(bh, thB, phB);
    krp_basis<float>(n, th, ph);
    const float inv_b = rsqrtf(bh[0] * bh[0] + bh[1] * bh[1] + bh[2] * bh[2]);
    const float ngx = n[0] * thB[0] + n[1] * thB[1] + n[2] * thB[2], ngy = n[0] * phB[0] + n[1] * phB[1], ngz = (n[0] * bh[0] + n[1] * bh[1] + n[2] * bh[2]) * inv_b;
    const float ogx = on[0] * thB[0] + on[1] * thB[1] + on[2] * thB[2], ogy = on[0] * phB[0] + on[1] * phB[1],
                ogz = (on[0] * bh[0] + on[1] * bh[1] + on[2] * bh[2]) * inv_b;
    const float r2d = 57.29577951308232f;
    const float ti = atan2f(sqrtf(ngx * ngx + ngy * ngy), ngz) * r2d, to = atan2f(sqrtf(ogx * ogx + ogy * ogy), ogz) * r2d;
    const float pi_ = (ngx * ngx + ngy * ngy >= 1e-24f) ? atan2f(ngy, ngx) * r2d : 0.f;
    const float po = (ogx * ogx + ogy * ogy >= 1e-24f) ? atan2f(ogy, ogx) * r2d : 0.f;
    float c2, s2;
    krp_eta2<float>(th[0] * bh[0] + th[1] * bh[1] + th[2] * bh[2], ph[0] * bh[0] + ph[1] * bh[1], c2, s2);
    const float I = Se.x, Q = Se.x * (c2 * Se.y + s2 * Se.z), U = Se.x * (c2 * Se.z - s2 * Se.y), V = Se.x * Se.w;   // eq. 7
    float M[16];
    krp_zt_at<float>(g, ti, to, po - pi_, 4, M);
    // N: linear interpolation of the per-node integrals of row 1
    float N;
    {
        const float xi = ti * (float)(g.ni - 1) * (1.f / 180.f);
        const int i = max(0, min((int)xi, g.ni - 2));
        const float w = xi - (float)i;
        const double* a = g.norm + 4 * i;
        N = ((1.f - w) * (float)a[0] + w * (float)a[4]) * I + ((1.f - w) * (float)a[1] + w * (float)a[5]) * Q
          + ((1.f - w) * (float)a[2] + w * (float)a[6]) * U + ((1.f - w) * (float)a[3] + w * (float)a[7]) * V;
    }
    const float f = 0.07957747154594767f * I / N;
    float R[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) R[r] = f * (M[4 * r] * I + M[4 * r + 1] * Q + M[4 * r + 2] * U + M[4 * r + 3] * V);
    krp_eta2<float>(oth[0] * bh[0] + oth[1] * bh[1] + oth[2] * bh[2], oph[0] * bh[0] + oph[1] * bh[1] + oph[2] * bh[2], c2, s2);
    S[0] = R[0]; S[1] = c2 * R[1] - s2 * R[2]; S[2] = s2 * R[1] + c2 * R[2]; S[3] = R[3];
}

// ------------------------------------------------------------------------------------------
// T6  scattering (step S5 of DESIGN.md).  One thread per event
// of the wave, fp64.  Draws of block 0 of event k: (Theta, phi candidate, accept, next tau*);
// blocks >= 1: two more (phi, accept) pairs each, at most 64 rounds.
// ------------------------------------------------------------------------------------------
// T6 for one event: from the stored pre-scatter state (direction n, Stokes (Q,U,V) of the record, lab reference of n) to the
// outgoing direction in fp32 (R12), the scattered Stokes vector in the lab reference of that direction, and the next tau*.
// kb = scattering order of the event (the Philox counter word), cell = padded cell id of the event.
template <bool ZT>      // ZT: the outgoing direction and Stokes vector come from the full Z table (NEXT-2), else from F(Theta)
__device__ __forceinline__ void krp_scatter_one(const KrpModel& g, unsigned long long seed, unsigned long long id, uint32_t kb,
                                                const float4 nk, uint32_t cell, const float4 Se,
                                                float nf[3], double& Q, double& U, double& V, double& tau_next)
{
    double b[3] = { 0.0, 0.0, 1.0 };
    if (!g.scalar) { float4 cl = g.cell[cell]; b[0] = cl.y; b[1] = cl.z; b[2] = cl.w; }   // cell is a padded id
    const double n[3] = { nk.x, nk.y, nk.z };
    // A2: q_B from the direction angles of B (eq. 2).  Without a field (scalar mode) B^ = z^, q_B = 1: the grain
    // frame is the lab frame and every step below that involves q_B or eta is the identity
    double qB[4] = { 1.0, 0.0, 0.0, 0.0 };
    double ng[3] = { n[0], n[1], n[2] };
    double th[3], ph[3], c2 = 1.0, s2 = 0.0;
    Q = Se.y; U = Se.z; V = Se.w;
    if (!g.scalar) {
        // half angles of theta_B in [0, pi] and phi_B in (-pi, pi] from their cosines and sines (no atan2, no sincos):
        // cos(a/2) = sqrt((1 + cos a)/2), sin(a/2) = sin a / (2 cos(a/2)) on the side where that does not cancel
        const double rho2 = b[0] * b[0] + b[1] * b[1], rho = sqrt(rho2);
        const double inv_r = krp_rsqrt_near1(rho2 + b[2] * b[2]);       // B^ is unit to fp32 rounding
        const double cth = b[2] * inv_r, sth = rho * inv_r;
        double ch_t, sh_t, ch_p = 1.0, sh_p = 0.0;
        if (cth >= 0.0) { ch_t = sqrt(0.5 * (1.0 + cth)); sh_t = sth / (2.0 * ch_t); }
        else            { sh_t = sqrt(0.5 * (1.0 - cth)); ch_t = sth / (2.0 * sh_t); }
        if (rho > 0.0) {
            const double ir = 1.0 / rho, cph = b[0] * ir, sph = b[1] * ir;
            if (cph >= 0.0) { ch_p = sqrt(0.5 * (1.0 + cph)); sh_p = sph / (2.0 * ch_p); }
            else            { sh_p = copysign(sqrt(0.5 * (1.0 - cph)), sph); ch_p = sph / (2.0 * sh_p); }
        }
        qB[0] = ch_p * ch_t; qB[1] = -sh_p * sh_t; qB[2] = ch_p * sh_t; qB[3] = sh_p * ch_t;
        // A3: direction in the grain frame (eq. 3)
        krp_quat_rotate(qB, n, -1.0, ng);
        // A5: Stokes reference lab -> grain frame
        krp_basis_unit_d(n, th, ph);
        krp_eta2<double>(krp_dot(th, b), krp_dot(ph, b), c2, s2);
        krp_rot_qu(Q, U, c2, s2);
    }
    {
        double r = krp_rsqrt_near1(krp_dot(ng, ng));       // a rotation of a direction that is unit to fp32 rounding
        ng[0] *= r; ng[1] *= r; ng[2] *= r;
    }
    double nog[3];
    if (ZT) {
        // NEXT-2 (R21): outgoing direction by rejection sampling against the full Z: candidates isotropic in the
        // grain frame, block 0 of event k = (cos, dphi, accept, next tau*), block b >= 1 = (cos, dphi, accept, -), at most 256
        const double r2d = 57.29577951308232087680;
        const double ti = acos(fmin(fmax(ng[2], -1.0), 1.0)) * r2d;
        const double pin = (ng[0] * ng[0] + ng[1] * ng[1] >= 1e-24) ? atan2(ng[1], ng[0]) * r2d : 0.0;
        double bound;
        {
            const double xi = ti * (double)(g.z.ni - 1) / 180.0;
            const int i = max(0, min((int)floor(xi), g.z.ni - 2));
            bound = fmax(g.z.bound[i], g.z.bound[i + 1]);
        }
        double to = 0.0, dp = 0.0;
        tau_next = 0.0;
        int rounds = 0;
        for (uint32_t blk = 0; ; ++blk) {
            const uint4 w = krp_philox(seed, id, kb, blk);
            if (blk == 0u) tau_next = -log(krp_u01(w.w));
            to = acos(1.0 - 2.0 * krp_u01(w.x)) * r2d;
            dp = 360.0 * krp_u01(w.y);
            double M1[16];
            krp_zt_at<double>(g.z, ti, to, dp, 1, M1);
            const double Iout = M1[0] + M1[1] * Q + M1[2] * U + M1[3] * V;
            ++rounds;
            if (krp_u01(w.z) * bound < Iout || rounds >= 256) break;
        }
        double M[16];
        krp_zt_at<double>(g.z, ti, to, dp, 4, M);
        {
            const double I2 = M[0] + M[1] * Q + M[2] * U + M[3] * V, inv = 1.0 / I2;
            const double Q2 = M[4] + M[5] * Q + M[6] * U + M[7] * V, U2 = M[8] + M[9] * Q + M[10] * U + M[11] * V,
                         V2 = M[12] + M[13] * Q + M[14] * U + M[15] * V;
            Q = Q2 * inv; U = U2 * inv; V = V2 * inv;      // referenced to theta^ of the outgoing direction in the grain frame
        }
        double st, ct, sp, cp;
        sincos(to * (KRP_PI_D / 180.0), &st, &ct);
        sincos((pin + dp) * (KRP_PI_D / 180.0), &sp, &cp);
        nog[0] = st * cp; nog[1] = st * sp; nog[2] = ct;
    } else {
    // draws
    uint4 w = krp_philox(seed, id, kb, 0u);
    tau_next = -log(krp_u01(w.w));
    double theta;   // Theta from the piecewise-linear CDF (R13), in units of the table spacing 180 deg/(n_ang-1)
    {
        double u = krp_u01(w.x);
        int lo = 0, hi = g.n_ang - 1;
        while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (g.cdf[mid] <= u) lo = mid; else hi = mid; }
        double wd = g.cdf[lo + 1] - g.cdf[lo];
        double f = wd > 0.0 ? (u - g.cdf[lo]) / wd : 0.5;
        theta = (double)lo + f;
    }
    // Theta in units of the table spacing: the Mueller row is linear in it (R13), Theta/180 deg = theta/(n_ang-1)
    double F[4];
    {
        const int j = max(0, min((int)theta, g.n_ang - 2));
        const double w1 = theta - (double)j, w0 = 1.0 - w1;
        const float4 a = g.mueller[j], b2 = g.mueller[j + 1];
        F[0] = w0 * (double)a.x + w1 * (double)b2.x; F[1] = w0 * (double)a.y + w1 * (double)b2.y;
        F[2] = w0 * (double)a.z + w1 * (double)b2.z; F[3] = w0 * (double)a.w + w1 * (double)b2.w;
    }
    const double p12 = F[1] / F[0];
    const double bound = 1.0 + fabs(p12) * sqrt(Q * Q + U * U);
    double sphi, cphi;
    sincospi(2.0 * krp_u01(w.y), &sphi, &cphi);           // phi = 2 pi u: no range reduction needed
    bool ok;
    {
        double c2p = cphi * cphi - sphi * sphi, s2p = 2.0 * sphi * cphi;
        ok = krp_u01(w.z) * bound < 1.0 + p12 * (Q * c2p + U * s2p);
    }
    int rounds = 1;
    for (uint32_t blk = 1; !ok && rounds < 64; ++blk) {
        uint4 x = krp_philox(seed, id, kb, blk);
        uint32_t cand[2] = { x.x, x.z }, acc[2] = { x.y, x.w };
        for (int h = 0; h < 2 && !ok && rounds < 64; ++h) {
            sincospi(2.0 * krp_u01(cand[h]), &sphi, &cphi);
            double c2p = cphi * cphi - sphi * sphi, s2p = 2.0 * sphi * cphi;
            ok = krp_u01(acc[h]) * bound < 1.0 + p12 * (Q * c2p + U * s2p);
            ++rounds;
        }
    }
    // scattering in the grain frame
    double thp[3], php[3];
    krp_basis_unit_d(ng, thp, php);
    double st, ct;
    sincospi(theta * g.inv_nang1, &st, &ct);
    double epar[3], eout[3], shat[3];
    for (int j = 0; j < 3; ++j) epar[j] = cphi * thp[j] + sphi * php[j];
    for (int j = 0; j < 3; ++j) nog[j] = ct * ng[j] + st * epar[j];
    krp_rot_qu(Q, U, cphi * cphi - sphi * sphi, 2.0 * sphi * cphi);      // reference e_par
    {
        double I2 = F[0] + F[1] * Q, Q2 = F[1] + F[0] * Q;                  // F(Theta) (1,Q,U,V)
        double U2 = F[2] * U + F[3] * V, V2 = -F[3] * U + F[2] * V;
        const double inv = 1.0 / I2;
        Q = Q2 * inv; U = U2 * inv; V = V2 * inv;
    }
    for (int j = 0; j < 3; ++j) eout[j] = ct * epar[j] - st * ng[j];
    krp_cross(ng, epar, shat);
    double th2[3], ph2[3];
    krp_basis_unit_d(nog, th2, ph2);
    {
        double ce = krp_dot(eout, th2), se = krp_dot(th2, shat);
        krp_rot_qu(Q, U, ce * ce - se * se, 2.0 * se * ce);                // reference theta^ of n'_GF
    }
    }
    // back to the lab: inverse of eq. 3, direction stored in fp32 (R12)
    double nl[3] = { nog[0], nog[1], nog[2] };
    if (!g.scalar) krp_quat_rotate(qB, nog, 1.0, nl);
    nf[0] = (float)nl[0]; nf[1] = (float)nl[1]; nf[2] = (float)nl[2];
    if (!g.scalar) {
        const double nd[3] = { nf[0], nf[1], nf[2] };
        krp_basis_unit_d(nd, th, ph);
        krp_eta2<double>(krp_dot(th, b), krp_dot(ph, b), c2, s2);
        krp_rot_qu(Q, U, c2, -s2);
    }}

template <bool ZT>
__global__ void __launch_bounds__(128, ZT ? 4 : 8) krp_k_scatter(KrpModel g, KrpCtl* ctl, KrpRecords ev, KrpRecords qo, int out,
                                                     unsigned long long seed)
{
    const unsigned long long e0 = ctl->ev_begin;
    unsigned long long e1 = ctl->n_events;
    if (e1 > ctl->ev_cap) e1 = ctl->ev_cap;
    for (unsigned long long e = e0 + blockIdx.x * blockDim.x + threadIdx.x; e < e1; e += (unsigned long long)gridDim.x * blockDim.x) {
        const float4 nk = ev.nk[e];
        const uint32_t kb = __float_as_uint(nk.w);
        if ((kb & KRP_TERM_BIT) || kb == 0u) continue;
        const float4 pc = ev.pc[e], Se = ev.S[e];
        const unsigned long long id = ev.id[e];
        const uint32_t cell = __float_as_uint(pc.w);
        float nf[3];
        double Q, U, V, tau_next;
        krp_scatter_one<ZT>(g, seed, id, kb, nk, cell, Se, nf, Q, U, V, tau_next);
        unsigned int slot = krp_reserve32(&ctl->q_count[out]);
        qo.pc[slot] = pc;
        qo.nk[slot] = make_float4(nf[0], nf[1], nf[2], __uint_as_float(kb));
        qo.S[slot] = make_float4(Se.x, (float)Q, (float)U, (float)V);
        qo.tau[slot] = tau_next;
        qo.id[slot] = id;
    }
}

// T3-T7, scalar mode, small batches: one thread follows a packet from its queue entry to its end -- flight, event record,
// scattering, next flight -- the shape the paper gives its own kernel.  A batch of 10^5 packets (BASELINE
// configs[0]) fills the GPU once; as a wavefront it is 14 orders x 3 launches of a few microseconds of work each, i.e. launch
// latency (0.72 ms per job of 10^5 packets against 0.30 ms), and the later orders hold a handful of packets.  Same arithmetic as
// the wave path in the same order per packet (flight of krp_k_flight_scalar_static, krp_event_append, krp_scatter_one): the
// records are bit-identical, only their order in the buffer differs.  Used for batches of at most krp_tune_fused() packets
// (default 2^20; the wavefront wins from ~1.5e6 packets on, where its direction-ordered first flights and converged
// scattering kernels outweigh its launches: profiles/r2r_README.md).
// 80 registers, six blocks of 128 per SM: 10^5 packets are resident at once (C1, one packet per thread: 0.165 ms at 150
// registers and three blocks, two rounds; 0.130 ms at 80; 0.143 ms at 64).
__global__ void __launch_bounds__(128, 6) krp_k_packets_scalar(KrpModel g, KrpCtl* ctl, KrpRecords q, int in, KrpRecords ev,
                                                            unsigned long long seed, int max_flights)
{
    const unsigned int n_items = ctl->q_count[in];
    KrpFlightTally tl = { 0, 0, 0, 0.0, 0.0, 0.0 };
    // Persistent lanes: a lane whose packet has ended takes the next queue entry at the top of the loop, where the warp is
    // converged (one scattering order per turn: flight, record, scattering), so the lanes of a warp stay busy although most
    // packets end after one or two events and a few live through all orders (6.8 of 32 lanes active with one packet per
    // thread, profiles/r2s).
    unsigned int wbase = 0, wleft = 0, item = 0;
    bool more = true, alive = false;
    float4 pc = make_float4(0.f, 0.f, 0.f, 0.f), nk = pc, S0 = pc;
    double D = 0.0;
    unsigned long long id = 0;
    int f = 0;
    for (;;) {
        if (krp_take_work(&ctl->work[0], n_items, !alive, wbase, wleft, more, item, 32u)) {      // 32 per visit: a small batch spreads over all warps
            pc = q.pc[item]; nk = q.nk[item]; S0 = q.S[item];
            D = q.tau[item];
            id = q.id[item];
            alive = true; f = 0;
        }
        if (!__any_sync(0xffffffffu, alive)) break;
        if (alive) {
            const float n[3] = { nk.x, nk.y, nk.z };
            const float p0[3] = { pc.x, pc.y, pc.z };
            const uint32_t c0 = __float_as_uint(pc.w);
            KrpRay ray;
            krp_ray_init(g, c0, p0, n, ray);
            uint32_t c_cur = ray.c;
            int ax_cur = -1;
            KRP_CK(g, c_cur);
            float kr_cur = __ldg(g.kr + c_cur);
            bool hit = false;
            for (;;) {
                int ax_n;
                const float ds = krp_ray_advance(ray, ax_n);
                KRP_CK(g, ray.c);
                const float kr_nxt = __ldg(g.kr + ray.c);          // requested before the depth test of the current cell
                const float dt1 = g.a1c * kr_cur * ds;
                if ((double)dt1 >= D) { hit = true; break; }       // event inside the current cell
                D -= (double)dt1;
                c_cur = ray.c;
                if (kr_nxt < 0.f) break;                           // halo: the packet left the grid
                ax_cur = ax_n; kr_cur = kr_nxt;
            }
            int h0[3], h1[3];
            krp_pad_coords(g, c0, h0[0], h0[1], h0[2]);
            krp_pad_coords(g, c_cur, h1[0], h1[1], h1[2]);
            const int crossings = abs(h1[0] - h0[0]) + abs(h1[1] - h0[1]) + abs(h1[2] - h0[2]);
            alive = false;
            if (!hit) { tl.steps += (unsigned long long)crossings; tl.w_esc += (double)S0.x; }
            else {
                tl.steps += (unsigned long long)(crossings + 1);
                const double moved = D / ((double)g.a1c * (double)kr_cur);
                float pe[3];
                krp_event_pos(g, n, p0, c0, c_cur, ax_cur, moved, pe);
                const uint32_t k = __float_as_uint(nk.w);
                krp_event_append(g, ctl, ev, id, c_cur, pe, n, k, S0.x, g.omc, S0.y, S0.z, S0.w, tl);
                // what krp_event_append stored: weight after the albedo, order, termination (R12)
                const float Wn = g.omc * S0.x;
                const uint32_t kn = k + 1u;
                if (!((Wn < g.w_min) || ((int)kn >= g.max_scatter)) && ++f < max_flights) {
                    const float4 Se = make_float4(Wn, S0.y, S0.z, S0.w);
                    float nf[3];
                    double Q, U, V, tau_next;
                    krp_scatter_one<false>(g, seed, id, kn, make_float4(n[0], n[1], n[2], __uint_as_float(kn)), c_cur, Se, nf, Q, U, V, tau_next);
                    pc = make_float4(pe[0], pe[1], pe[2], __uint_as_float(c_cur));
                    nk = make_float4(nf[0], nf[1], nf[2], __uint_as_float(kn));
                    S0 = make_float4(Wn, (float)Q, (float)U, (float)V);
                    D = tau_next;
                    alive = true;
                }
            }
        }
    }
    krp_tally_flush(tl, ctl);
}

// ------------------------------------------------------------------------------------------
// I1  peel-off (PAPER.md:121 S_pp = Z(Omega_cam;Omega_pp) I_pp, eq. 10-11): Stokes vector sent
// toward the observer by a scattering of the stored incoming state, in the reference
// theta^_obs, times 1/(4 pi).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void krp_rot_qu_f(float& Q, float& U, float ce, float se)
{
    float c2 = ce * ce - se * se, s2 = 2.f * se * ce;
    float q = c2 * Q + s2 * U, u = -s2 * Q + c2 * U;
    Q = q; U = u;
}

// The geometry of one peel-off, which depends on the incoming direction and the observer only: rotation of the Stokes
// reference into the scattering plane (cos, sin of twice the angle), F(Theta_obs) times 1/(4 pi), rotation to theta^_obs.
struct KrpPeelGeom { float c2i, s2i, F[4], c2o, s2o; };

__device__ __forceinline__ void krp_peel_setup(const KrpModel& g, const float n[3], const KrpObserverDev& ob, KrpPeelGeom& pg)
{
    // spherical basis of n (eq. 4-5, R10) and the unit normal of the scattering plane with the hardware reciprocal
    // square root (2 ulp): this runs once per (event, observer), and IEEE divisions and square roots were a fifth of it
    float th[3], ph[3];
    {
        const float s2 = n[0] * n[0] + n[1] * n[1];
        const float inv_rr = rsqrtf(s2 + n[2] * n[2]);
        float cp = 1.f, sp = 0.f, s = 0.f;
        if (s2 >= 1e-24f) { const float inv_s = rsqrtf(s2); s = s2 * inv_s; cp = n[0] * inv_s; sp = n[1] * inv_s; }
        const float ct = n[2] * inv_rr, st = s * inv_rr;
        th[0] = ct * cp; th[1] = ct * sp; th[2] = -st;
        ph[0] = -sp; ph[1] = cp; ph[2] = 0.f;
    }
    float mu = n[0] * ob.n[0] + n[1] * ob.n[1] + n[2] * ob.n[2];
    mu = fminf(fmaxf(mu, -1.f), 1.f);
    float sh[3] = { n[1] * ob.n[2] - n[2] * ob.n[1], n[2] * ob.n[0] - n[0] * ob.n[2], n[0] * ob.n[1] - n[1] * ob.n[0] };
    const float ss = sh[0] * sh[0] + sh[1] * sh[1] + sh[2] * sh[2];
    float sn = 0.f;
    if (ss < 1e-24f) { sh[0] = ph[0]; sh[1] = ph[1]; sh[2] = ph[2]; }
    else { const float r = rsqrtf(ss); sn = ss * r; sh[0] *= r; sh[1] *= r; sh[2] *= r; }
    // e_par = s^ x n_in: reference of the incoming ray in the scattering plane
    float ep[3] = { sh[1] * n[2] - sh[2] * n[1], sh[2] * n[0] - sh[0] * n[2], sh[0] * n[1] - sh[1] * n[0] };
    {
        const float ce = th[0] * ep[0] + th[1] * ep[1] + th[2] * ep[2], se = ph[0] * ep[0] + ph[1] * ep[1] + ph[2] * ep[2];
        pg.c2i = ce * ce - se * se; pg.s2i = 2.f * se * ce;
    }
    // scattering angle from atan2(|n x n_obs|, n.n_obs): well conditioned at both poles
    // (in units of the table spacing: the Mueller row is linear in it, R13)
    const float x = atan2f(sn, mu) * g.nang1_over_pi;
    {
        const int j = max(0, min((int)x, g.n_ang - 2));
        const float w = x - (float)j, w0 = 1.f - w;
        const float4 a = g.mueller[j], b = g.mueller[j + 1];
        const float c = 0.07957747154594767f;   // 1/(4 pi)
        pg.F[0] = c * (w0 * a.x + w * b.x); pg.F[1] = c * (w0 * a.y + w * b.y); pg.F[2] = c * (w0 * a.z + w * b.z); pg.F[3] = c * (w0 * a.w + w * b.w);
    }
    // e_out = s^ x n_obs, then to theta^_obs
    float eo[3] = { sh[1] * ob.n[2] - sh[2] * ob.n[1], sh[2] * ob.n[0] - sh[0] * ob.n[2], sh[0] * ob.n[1] - sh[1] * ob.n[0] };
    {
        const float ce = eo[0] * ob.th[0] + eo[1] * ob.th[1] + eo[2] * ob.th[2], se = ob.th[0] * sh[0] + ob.th[1] * sh[1] + ob.th[2] * sh[2];
        pg.c2o = ce * ce - se * se; pg.s2o = 2.f * se * ce;
    }
}

// (I,Q,U,V) in the lab reference of the incoming direction -> Stokes vector sent toward the observer, reference theta^_obs
__device__ __forceinline__ void krp_peel_apply(const KrpPeelGeom& pg, float I, float Q, float U, float V, float S[4])
{
    const float q = pg.c2i * Q + pg.s2i * U, u = -pg.s2i * Q + pg.c2i * U;
    const float I2 = pg.F[0] * I + pg.F[1] * q, Q2 = pg.F[1] * I + pg.F[0] * q;
    const float U2 = pg.F[2] * u + pg.F[3] * V, V2 = -pg.F[3] * u + pg.F[2] * V;
    S[0] = I2; S[1] = pg.c2o * Q2 + pg.s2o * U2; S[2] = -pg.s2o * Q2 + pg.c2o * U2; S[3] = V2;
}

__device__ __forceinline__ void krp_peel(const KrpModel& g, const float n[3], float4 Se, const KrpObserverDev& ob, float S[4])
{
    KrpPeelGeom pg;
    krp_peel_setup(g, n, ob, pg);
    krp_peel_apply(pg, Se.x, Se.x * Se.y, Se.x * Se.z, Se.x * Se.w, S);
}

// ------------------------------------------------------------------------------------------
// I0  ordering of the event buffer for imaging: a counting sort of the event
// indices by bin = padded cell id >> shift, entirely on the device (the event count never visits the
// host).  Rays of one observer are parallel, so the 32 rays of a warp that start in neighbouring cells
// walk through neighbouring cells for their whole length: their gathers share cache lines and they
// leave the grid after nearly the same number of steps.  Every bin has 2^sub_bits counters, picked by the low
// bits of the event index, so that the many events of a hot cell (next to a point source) do not queue on one
// atomic; the order inside a bin is arbitrary anyway.
//   krp_k_sort_count    histogram of the bins
//   (exclusive scan of the histogram: cub::DeviceScan, in krp_api.cu)
//   krp_k_sort_scatter  perm[slot] = event index, slot reserved in the event's bin
// ------------------------------------------------------------------------------------------
// Both kernels walk the buffer in aligned groups of 32 events, one group per warp and visit; the lanes of a group that
// fall into the same bin are counted (and given their slots) by one atomic of their first lane (__match_any_sync), on the
// bin's sub-counter number (group index mod 2^sub_bits): the events next to a point source, which are a large share of
// every group, would otherwise queue on the one L2 slice that holds their bin's counters.
// The bins are taken block-major: the grid is cut into blocks of 2^B cells per edge and a bin is one run of 2^ls cells
// along x inside a block (a 128-byte line of cells), numbered block by block.  The minor order keeps the 32 rays of a
// warp in neighbouring cells, as before; the major order keeps the rays that are marched at the same time (a few
// hundred thousand, i.e. the events of a few blocks) inside one beam of cells along the line of sight, a few tens of
// MB that stay in L2 -- in plain cell order the rays of one z-plane of start cells sweep the whole grid above it and
// every window of the order streamed the observer's whole coefficient array from DRAM (C5: 228 GB per launch for a
// 2 GiB array, profiles/r1d).
struct KrpSortGeom { int B, ls; uint32_t nbx, nby; };
__device__ __forceinline__ unsigned int krp_sort_bin(const KrpModel& g, const KrpSortGeom& sg, uint32_t cell)
{
    if (sg.B == 0) return cell >> sg.ls;       // plain cell order (scalar mode: the 4-byte grid sits in L2 whatever the order)
    int hx, hy, hz;
    krp_pad_coords(g, cell, hx, hy, hz);
    const uint32_t m = (1u << sg.B) - 1u;
    const uint32_t blk = (((uint32_t)hz >> sg.B) * sg.nby + ((uint32_t)hy >> sg.B)) * sg.nbx + ((uint32_t)hx >> sg.B);
    const uint32_t in = ((((uint32_t)hz & m) << sg.B) | ((uint32_t)hy & m)) << (sg.B - sg.ls) | (((uint32_t)hx & m) >> sg.ls);
    return (blk << (3 * sg.B - sg.ls)) | in;
}

__global__ void __launch_bounds__(256) krp_k_sort_count(KrpModel g, KrpCtl* ctl, KrpRecords ev, KrpSortGeom sg, int sub_bits, int flags,
                                                        unsigned int* __restrict__ bins)
{
    unsigned long long n_ev = ctl->n_events;
    if (n_ev > ctl->ev_cap) n_ev = ctl->ev_cap;
    const unsigned int sub_mask = (1u << sub_bits) - 1u;
    const unsigned int lane = threadIdx.x & 31u;
    for (unsigned long long e0 = blockIdx.x * (unsigned long long)blockDim.x + (threadIdx.x & ~31u); e0 < n_ev;
         e0 += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long e = e0 + lane;
        // emission records take part only with direct light (flags bit 1: the buffer holds none, no need to look)
        bool valid = e < n_ev;
        if (valid && !(flags & 3) && (__float_as_uint(ev.nk[e].w) & ~KRP_TERM_BIT) == 0u) valid = false;
        const unsigned int bin = valid ? krp_sort_bin(g, sg, __float_as_uint(ev.pc[e].w)) : 0xffffffffu;
        const unsigned int peers = __match_any_sync(0xffffffffu, bin);
        if (valid && lane == (unsigned int)(__ffs(peers) - 1))
            atomicAdd(bins + ((bin << sub_bits) | ((unsigned int)(e0 >> 5) & sub_mask)), (unsigned int)__popc(peers));
    }
}

// after the scan `bins` holds the first slot of every bin; the last thread publishes the total
__global__ void __launch_bounds__(256) krp_k_sort_scatter(KrpModel g, KrpCtl* ctl, KrpRecords ev, KrpSortGeom sg, int sub_bits, int flags,
                                                          unsigned int* __restrict__ bins, unsigned int* __restrict__ perm)
{
    unsigned long long n_ev = ctl->n_events;
    if (n_ev > ctl->ev_cap) n_ev = ctl->ev_cap;
    const unsigned int sub_mask = (1u << sub_bits) - 1u;
    const unsigned int lane = threadIdx.x & 31u;
    for (unsigned long long e0 = blockIdx.x * (unsigned long long)blockDim.x + (threadIdx.x & ~31u); e0 < n_ev;
         e0 += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned long long e = e0 + lane;
        bool valid = e < n_ev;
        if (valid && !(flags & 3) && (__float_as_uint(ev.nk[e].w) & ~KRP_TERM_BIT) == 0u) valid = false;
        const unsigned int bin = valid ? krp_sort_bin(g, sg, __float_as_uint(ev.pc[e].w)) : 0xffffffffu;
        const unsigned int peers = __match_any_sync(0xffffffffu, bin);
        const int first = __ffs(peers) - 1;
        unsigned int base = 0u;
        if (valid && lane == (unsigned int)first)
            base = atomicAdd(bins + ((bin << sub_bits) | ((unsigned int)(e0 >> 5) & sub_mask)), (unsigned int)__popc(peers));
        base = __shfl_sync(0xffffffffu, base, first);
        if (valid) perm[base + __popc(peers & ((1u << lane) - 1u))] = (unsigned int)e;
    }
}

// one thread: open an imaging pass.  n_sorted = events that take part = last bin's end after the scatter,
// which the host cannot know; it is read from the scanned histogram's sentinel entry (bins[n_bins] = total).
__global__ void krp_k_image_prep(KrpCtl* ctl, const unsigned int* __restrict__ bins, unsigned int n_bins)
{
    ctl->n_sorted = bins[n_bins];
    for (int o = 0; o < KRP_MAX_OBS_PACK; ++o) ctl->img_work[o] = 0;
}
// the same without an order: every buffered event takes part in the order of the buffer (perm = NULL in the
// imaging kernel, which then skips emission records itself when they are not wanted)
__global__ void krp_k_image_prep_plain(KrpCtl* ctl)
{
    unsigned long long n_ev = ctl->n_events;
    if (n_ev > ctl->ev_cap) n_ev = ctl->ev_cap;
    ctl->n_sorted = (unsigned int)n_ev;
    for (int o = 0; o < KRP_MAX_OBS_PACK; ++o) ctl->img_work[o] = 0;
}
__global__ void krp_k_image_rewind(KrpCtl* ctl)
{
    for (int o = 0; o < KRP_MAX_OBS_PACK; ++o) ctl->img_work[o] = 0;
}

// ------------------------------------------------------------------------------------------
// I1-I3  imaging.  One launch per observer, whose constants (direction, bases, per-axis face spacing
// and stride) are kernel parameters, i.e. constant-bank operands of the march; a warp repeatedly takes
// the next 32 events of the sorted order from the launch's counter.  Per ray: peel-off, attenuation march to the grid edge with the same in-cell solution and
// no survival test, orthographic projection, fp64 accumulation into
// img[obs][4][npy][npx] (R14) with one atomic per distinct pixel of the warp.
//
// The march carries the absolute path length at the next face of each axis (KrpRayA): per step one
// min3, one subtraction, one 4- or 16-byte gather, the in-cell update, one predicated add per axis.
// The Stokes vector is e^{-A}(i,q,u,v); thin cells (|alpha2 dtau|, |alpha3 dtau| < 0.1) take the
// series of sinh, cosh-1, sin, cos-1 in "delta form"  S += R(-eta) dP R(eta) S, which needs no
// special case where n is parallel to B (the rotation is undefined there and dP vanishes).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void krp_appA_delta_thin(float x, float y, float i, float qg, float ug, float v,
                                                    float& di, float& dqg, float& dug, float& dv)
{
    const float x2 = x * x, y2 = y * y;
    const float sh = fmaf(x * x2, 1.f / 6.f, x);                   // sinh x,     |x| < 0.1: rel. error < 1e-6
    const float chm1 = x2 * fmaf(x2, 1.f / 24.f, 0.5f);            // cosh x - 1
    const float sy = fmaf(y * y2, -1.f / 6.f, y);                  // sin y
    const float cym1 = y2 * fmaf(y2, 1.f / 24.f, -0.5f);           // cos y - 1
    di = i * chm1 - qg * sh;
    dqg = qg * chm1 - i * sh;
    dug = ug * cym1 - v * sy;
    dv = ug * sy + v * cym1;
}

// one step of the absolute-path-length march: returns the length of the segment in the current cell and moves
// to the next one (ties: x before y before z).  dt and stride are launch constants (constant-bank operands).
// ------------------------------------------------------------------------------------------
// I0b  per-observer cell coefficients.  All rays of one observer share the direction, so what the in-cell
// solution needs from a cell -- alpha_i(mu) with mu = |n_obs . B^| (R8, R13) and the angle eta between the
// observer's reference and the grain frame (eq. 6-7, R2) -- depends on the cell only.  They are tabulated
// once per observer set as float4 {kappa*rho*alpha1, kappa*rho*alpha2, kappa*rho*alpha3, 2*eta} in the padded
// order (halo: first component -1), which takes the two table look-ups, nine dot-product terms and the
// reciprocal out of the march and halves its traffic through the L1 data pipe (profiles/: the shared-memory
// table reads were 49 % of that pipe on C5).  Used when n_obs such arrays fit in device memory.
// ------------------------------------------------------------------------------------------
// Encoding of the first component: >= 0  kappa*rho*alpha1 of a cell the march may treat with the short series (thin for
// every possible segment: max(|kappa rho alpha2|, |kappa rho alpha3|) x cell diagonal < 0.1); finite and < 0  minus that value
// for a cell that needs the full in-cell solution; -inf  halo.  The march's hot loop then runs on one sign test per cell.
__global__ void __launch_bounds__(256) krp_k_obs_cells(KrpModel g, const KrpObserverDev ob, uint32_t npad, float4* __restrict__ out)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= npad) return;
    const float4 cl = g.cell[c];
    float4 o = make_float4(cl.x < 0.f ? -KRP_INF_F : cl.x, 0.f, 0.f, 0.f);
    if (cl.x > 0.f) {
        const int nseg = g.n_inc - 1;
        const float mu = fminf(fabsf(ob.n[0] * cl.y + ob.n[1] * cl.z + ob.n[2] * cl.w), 1.f);
        const float x = mu * (float)nseg;
        const int j = min((int)x, nseg - 1);
        const float4 ta = g.opA[j], tb = g.opB[j];
        const float a = ob.th[0] * cl.y + ob.th[1] * cl.z + ob.th[2] * cl.w;
        const float b = ob.ph[0] * cl.y + ob.ph[1] * cl.z + ob.ph[2] * cl.w;
        const float aa = a * a, bb = b * b;
        o.x = cl.x * fmaf(tb.x, x, ta.x);
        o.y = cl.x * fmaf(tb.y, x, ta.y);
        o.z = cl.x * fmaf(tb.z, x, ta.z);
        o.w = aa + bb < 1e-24f ? 0.f : atan2f(2.f * a * b, aa - bb);   // cos 2eta ~ a^2 - b^2, sin 2eta ~ 2ab (R2)
        const float diag = sqrtf(g.d[0] * g.d[0] + g.d[1] * g.d[1] + g.d[2] * g.d[2]);
        if (fmaxf(fabsf(o.y), fabsf(o.z)) * diag >= 0.1f) o.x = -o.x;
    }
    out[c] = o;
}

struct KrpRayAConst { float dtx, dty, dtz; int sx, sy, sz; float n[3], th[3], ph[3]; float xs; int nseg; };
// The launch constants of the march, held in registers for the whole kernel: they are read back from shared
// memory through volatile loads, which ptxas (unlike a kernel parameter) will not re-load inside the loop.
__device__ __forceinline__ KrpRayAConst krp_raya_const(const KrpObserverDev& ob, int nseg, KrpRayAConst* sh)
{
    if (threadIdx.x == 0) {
        sh->dtx = ob.dt[0]; sh->dty = ob.dt[1]; sh->dtz = ob.dt[2];
        sh->sx = ob.stride[0]; sh->sy = ob.stride[1]; sh->sz = ob.stride[2];
        for (int a = 0; a < 3; ++a) { sh->n[a] = ob.n[a]; sh->th[a] = ob.th[a]; sh->ph[a] = ob.ph[a]; }
        sh->nseg = nseg; sh->xs = (float)nseg;
    }
    __syncthreads();
    volatile KrpRayAConst* v = sh;
    KrpRayAConst k;
    k.dtx = v->dtx; k.dty = v->dty; k.dtz = v->dtz; k.sx = v->sx; k.sy = v->sy; k.sz = v->sz;
    for (int a = 0; a < 3; ++a) { k.n[a] = v->n[a]; k.th[a] = v->th[a]; k.ph[a] = v->ph[a]; }
    k.xs = v->xs; k.nseg = v->nseg;
    return k;
}
// One step: min3 (FMNMX3), one subtraction, three compares, one predicated FADD + IADD per axis.
// Returns the segment length in the current cell; t_next is the path length at its exit face.
__device__ __forceinline__ float krp_raya_step(KrpRayA& r, const KrpRayAConst& k)
{
    float ds, tn;
    asm("{\n\t.reg .pred px, py, pz;\n\t"
        "min.f32 %1, %2, %3, %4;\n\t"
        "sub.f32 %0, %1, %6;\n\t"
        "setp.le.f32 px, %2, %1;\n\t"
        "setp.le.and.f32 py, %3, %1, !px;\n\t"
        "setp.gt.and.f32 pz, %3, %1, !px;\n\t"
        "@px add.f32 %2, %2, %7;\n\t@px add.s32 %5, %5, %10;\n\t"
        "@py add.f32 %3, %3, %8;\n\t@py add.s32 %5, %5, %11;\n\t"
        "@pz add.f32 %4, %4, %9;\n\t@pz add.s32 %5, %5, %12;\n\t}"
        : "=&f"(ds), "=&f"(tn), "+f"(r.tx), "+f"(r.ty), "+f"(r.tz), "+r"(r.c)
        : "f"(r.t), "f"(k.dtx), "f"(k.dty), "f"(k.dtz), "r"(k.sx), "r"(k.sy), "r"(k.sz));
    r.t = tn;
    return ds;
}

template <bool SCALAR, bool PRE, bool ZT>      // ZT: peel-off with the full Z of aligned grains (NEXT-2) instead of F(Theta)
__global__ void __launch_bounds__(256, SCALAR ? KRP_IMAGE_SCALAR_MIN_BLOCKS : (ZT ? 4 : KRP_IMAGE_MIN_BLOCKS)) krp_k_image(KrpModel g, KrpCtl* ctl, KrpRecords ev,
                                                   const unsigned int* __restrict__ perm, const KrpObserverDev ob,
                                                   const float4* __restrict__ obs_cell,
                                                   int slot, int obs_index, int npx, int npy, int flags, double* __restrict__ img)
{
    extern __shared__ float4 s_tab[];                // [2*(n_inc-1)]: intercepts, slopes of the opacity table
    const int nseg = g.n_inc - 1;
    if (!SCALAR && !PRE) {
        for (int j = threadIdx.x; j < nseg; j += blockDim.x) { s_tab[j] = g.opA[j]; s_tab[nseg + j] = g.opB[j]; }
        __syncthreads();
    }
    const unsigned int n_ev = ctl->n_sorted;
    const int lane = threadIdx.x & 31;
    __shared__ KrpRayAConst s_rc;
    const KrpRayAConst rc = krp_raya_const(ob, nseg, &s_rc);
    unsigned long long steps = 0, n_con = 0, n_drop = 0;
    // SCALAR mode: a warp takes KRP_IMG_CHUNK consecutive events of the order per visit to the launch's counter (32 when the
    // events are few, for the balance of the tail): with 32 per visit a large launch of short rays queues on that one address
    // (3.4 x 10^5 atomics per 10^7 rays; C2's imaging 8.9 -> 8.1 ms).  General mode keeps 32: its rays are long, and the
    // warps of an SM then work on one narrow window of the order and share its cells in L1/L2 (C5: 512 ms, 564 ms with 128).
    const unsigned int chunk = (SCALAR && n_ev >= (1u << 21)) ? (unsigned int)KRP_IMG_CHUNK : 32u;
    unsigned int cbase = 0, cleft = 0;
    for (;;) {
        if (cleft == 0u) {
            if (lane == 0) cbase = atomicAdd(&ctl->img_work[slot], chunk);
            cbase = __shfl_sync(0xffffffffu, cbase, 0);
            cleft = chunk;
        }
        const unsigned int base = cbase;
        cbase += 32u; cleft -= 32u;
        if (base >= n_ev) break;            // so are all later chunks
        bool live = base + lane < n_ev;
        int pixel = -1;
        float out[4] = { 0.f, 0.f, 0.f, 0.f };
        const unsigned int e = live ? (perm ? perm[base + lane] : base + lane) : 0u;
        float4 nk = make_float4(0.f, 0.f, 1.f, 0.f);
        if (live) {
            nk = ev.nk[e];
            // without an order (perm = NULL) emission records are still in the list: they take part only with direct light
            if (!perm && (__float_as_uint(nk.w) & ~KRP_TERM_BIT) == 0u && !(flags & 1)) live = false;
        }
        if (live) {
            const float4 pc = ev.pc[e], Se = ev.S[e];
            const uint32_t k = __float_as_uint(nk.w) & ~KRP_TERM_BIT;
            float S[4];
            const uint32_t c0 = __float_as_uint(pc.w);
            if (k == 0u) { S[0] = Se.x * 0.07957747154594767f; S[1] = S[2] = S[3] = 0.f; }
            else {
                const float n[3] = { nk.x, nk.y, nk.z };
                if (ZT) {                    // full Z of aligned grains: the peel-off depends on the field of the event cell (R21)
                    KRP_CK(g, c0);
                    const float4 cb = __ldg(g.cell + c0);
                    const float bh[3] = { cb.y, cb.z, cb.w };
                    krp_peel_z(g.z, bh, n, Se, rc.n, rc.th, rc.ph, S);
                } else krp_peel(g, n, Se, ob, S);
            }
            // ray set-up
            KrpRayA r;
            r.t = 0.f; r.c = c0;
            r.tx = ob.n[0] > 0.f ? (1.f - pc.x) * ob.dt[0] : (ob.n[0] < 0.f ? pc.x * ob.dt[0] : KRP_INF_F);
            r.ty = ob.n[1] > 0.f ? (1.f - pc.y) * ob.dt[1] : (ob.n[1] < 0.f ? pc.y * ob.dt[1] : KRP_INF_F);
            r.tz = ob.n[2] > 0.f ? (1.f - pc.z) * ob.dt[2] : (ob.n[2] < 0.f ? pc.z * ob.dt[2] : KRP_INF_F);
            float A = 0.f;
            int woff[3] = { 0, 0, 0 }, nwrap = 0;       // periodic boundaries: cells jumped per axis, faces re-entered
            if (SCALAR) {
                // two gathers in flight: the cell after next is requested before the next one is tested
                float tau = 0.f;
                KRP_CK(g, r.c);
                float kr_c = __ldg(g.kr + r.c);            // current cell (inside the grid)
                float ds_c = krp_raya_step(r, rc);
                KRP_CK(g, r.c);
                float kr_n = __ldg(g.kr + r.c);            // next cell
                uint32_t c_n = r.c;
#pragma unroll 2
                for (;;) {
                    const float ds_n = krp_raya_step(r, rc);
                    KRP_CK(g, (int)r.c);
                    const float kr_nn = __ldg(g.kr + (int)r.c); // look-ahead (may lie one cell past the halo, on either side: margin, signed index)
                    tau = fmaf(kr_c, ds_c, tau);
                    if (kr_n < 0.f) break;
                    kr_c = kr_n; ds_c = ds_n; kr_n = kr_nn; c_n = r.c;
                }
                r.c = c_n;                                 // the halo cell that ended the ray
                A = g.a1c * tau;
            } else if (PRE) {
                // march over the observer's own coefficient array {kr a1 (sign: thin / thick / halo), kr a2, kr a3, 2 eta}
                float i = S[0], qs = S[1], us = S[2], vs = S[3];
                KRP_CK(g, r.c);
                float4 cl = __ldg(obs_cell + r.c);
                // One loop, one sign test per cell: >= 0 thin whatever the segment (also empty cells: the update is then the
                // identity), < 0 rare -- a cell that may be thick, or the halo.  The rare cases sit behind a forward branch inside the
                // same loop, so that the lanes of a warp re-join at the next cell (as two nested loops a lane that met a thick cell
                // waited for all others to finish their rays: 25.9 of 32 threads active, profiles/r2m).
#pragma unroll 2
                for (;;) {
                    if (cl.x < 0.f) {
                        if (cl.x == -KRP_INF_F) {               // halo: the ray has left the grid -- or crosses a periodic face (R20)
                            // (a ray that has gone dark stops here as well: beyond A = 104 the carried vector would only grow, R20 allows 4096 periods)
                            KRP_CK(g, r.c);
                            if (g.periodic && A <= 104.f && nwrap < KRP_MAX_WRAPS && krp_wrap(g, r.c, woff)) { ++nwrap; cl = __ldg(obs_cell + r.c); continue; }
                            break;
                        }
                        // a cell that may be thick: full in-cell solution
                        const float ds = krp_raya_step(r, rc);
                        KRP_CK(g, r.c);
                        const float4 cn = __ldg(obs_cell + r.c);
                        float s2, c2;
                        __sincosf(cl.w, &s2, &c2);
                        float qg2 = c2 * qs + s2 * us, ug2 = c2 * us - s2 * qs, vg2 = vs, di, i_new, depth;
                        krp_appA(i, qg2, ug2, vg2, make_float4(-cl.x, cl.y, cl.z, 0.f), ds, di, i_new, depth);
                        i = i_new; A += depth; vs = vg2;
                        qs = c2 * qg2 - s2 * ug2; us = s2 * qg2 + c2 * ug2;
                        cl = cn;
                        if (A > 104.f) break;                   // e^{-A} is exactly 0 in fp32 from here on
                        continue;
                    }
                    const float ds = krp_raya_step(r, rc);
                    KRP_CK(g, r.c);
                    const float4 cn = __ldg(obs_cell + r.c);    // next cell, in flight during the update below
                    const float xx = cl.y * ds, yy = cl.z * ds;
                    float s2, c2;
                    __sincosf(cl.w, &s2, &c2);
                    const float qg = c2 * qs + s2 * us, ug = c2 * us - s2 * qs;   // eq. 7
                    // delta form S += R(-eta) dP R(eta) S with the two-term series (|xx|, |yy| < 0.1), written as chains of
                    // FFMAs: 16 for the update, the increments never materialised
                    const float x2 = xx * xx, y2 = yy * yy;
                    const float sh = fmaf(xx * x2, 1.f / 6.f, xx), chm1 = x2 * fmaf(x2, 1.f / 24.f, 0.5f);
                    const float sy = fmaf(yy * y2, -1.f / 6.f, yy), cym1 = y2 * fmaf(y2, 1.f / 24.f, -0.5f);
                    const float dqg = fmaf(qg, chm1, -(i * sh)), dug = fmaf(ug, cym1, -(vs * sy));
                    i = fmaf(-qg, sh, fmaf(i, chm1, i));
                    vs = fmaf(ug, sy, fmaf(vs, cym1, vs));
                    qs = fmaf(c2, dqg, fmaf(-s2, dug, qs));
                    us = fmaf(s2, dqg, fmaf(c2, dug, us));
                    A = fmaf(cl.x, ds, A);
                    cl = cn;
                }
                S[0] = i; S[1] = qs; S[2] = us; S[3] = vs;
            } else {
                float i = S[0], qs = S[1], us = S[2], vs = S[3];
                KRP_CK(g, r.c);
                float4 cl = __ldg(g.cell + r.c);
                for (;;) {
                do {
                    const float ds = krp_raya_step(r, rc);
                    KRP_CK(g, r.c);
                    const float4 cn = __ldg(g.cell + r.c);      // next cell, in flight during the update below
                    if (cl.x > 0.f) {
                        const float mu = fminf(fabsf(rc.n[0] * cl.y + rc.n[1] * cl.z + rc.n[2] * cl.w), 1.f);
                        const float x = mu * rc.xs;
                        const int j = min((int)x, rc.nseg - 1);
                        const float4 ta = s_tab[j], tb = s_tab[rc.nseg + j];
                        const float dtau = cl.x * ds;
                        const float a1 = fmaf(tb.x, x, ta.x), a2 = fmaf(tb.y, x, ta.y), a3 = fmaf(tb.z, x, ta.z);
                        const float xx = a2 * dtau, yy = a3 * dtau;
                        const float a = rc.th[0] * cl.y + rc.th[1] * cl.z + rc.th[2] * cl.w;
                        const float b = rc.ph[0] * cl.y + rc.ph[1] * cl.z + rc.ph[2] * cl.w;
                        const float aa = a * a, bb = b * b;
                        const float inv = __fdividef(1.f, fmaxf(aa + bb, 1e-30f));
                        const float c2 = (aa - bb) * inv, s2 = 2.f * a * b * inv;     // cos 2eta, sin 2eta (R2)
                        const float qg = c2 * qs + s2 * us, ug = c2 * us - s2 * qs;   // eq. 7
                        if (fmaxf(fabsf(xx), fabsf(yy)) < 0.1f) {
                            float di, dqg, dug, dv;
                            krp_appA_delta_thin(xx, yy, i, qg, ug, vs, di, dqg, dug, dv);
                            i += di; vs += dv;
                            qs += c2 * dqg - s2 * dug;
                            us += s2 * dqg + c2 * dug;
                            A = fmaf(a1, dtau, A);
                        } else {
                            // thick cell (rare outside C3): full in-cell solution; where n is parallel to B the
                            // rotation is undefined and, alpha2 = alpha3 = 0 there in any physical table, irrelevant
                            const bool pole = aa + bb < 1e-24f;
                            const float c2t = pole ? 1.f : c2, s2t = pole ? 0.f : s2;
                            float qg2 = c2t * qs + s2t * us, ug2 = c2t * us - s2t * qs, vg2 = vs, di, i_new, depth;
                            krp_appA(i, qg2, ug2, vg2, make_float4(a1, a2, a3, 0.f), dtau, di, i_new, depth);
                            i = i_new; A += depth; vs = vg2;
                            qs = c2t * qg2 - s2t * ug2; us = s2t * qg2 + c2t * ug2;
                            if (A > 104.f) { cl = cn; A = KRP_INF_F; break; }      // e^{-A} is exactly 0 in fp32 from here on
                        }
                    }
                    cl = cn;
                } while (cl.x >= 0.f);
                if (A > 104.f || !(g.periodic && nwrap < KRP_MAX_WRAPS && krp_wrap(g, r.c, woff))) break;
                KRP_CK(g, r.c);
                ++nwrap; cl = __ldg(g.cell + r.c);           // periodic face (R20): go on from the opposite side
                }
                S[0] = i; S[1] = qs; S[2] = us; S[3] = vs;
            }
            const float att = expf(-A);
            // steps taken = face crossings on the way from c0 to the last cell loaded
            int h0[3], h1[3];
            krp_pad_coords(g, c0, h0[0], h0[1], h0[2]);
            krp_pad_coords(g, r.c, h1[0], h1[1], h1[2]);
            steps += (unsigned long long)(abs(h1[0] + woff[0] - h0[0]) + abs(h1[1] + woff[1] - h0[1]) + abs(h1[2] + woff[2] - h0[2]));
            // I3: orthographic projection of the event position (fp64, once per ray)
            const double x[3] = { g.lo[0] + ((double)(h0[0] - 1) + (double)pc.x) * g.dd[0] - ob.center[0],
                                  g.lo[1] + ((double)(h0[1] - 1) + (double)pc.y) * g.dd[1] - ob.center[1],
                                  g.lo[2] + ((double)(h0[2] - 1) + (double)pc.z) * g.dd[2] - ob.center[2] };
            const double xi = (x[0] * ob.phd[0] + x[1] * ob.phd[1] + x[2] * ob.phd[2]) * ob.inv_hw;
            const double yi = -(x[0] * ob.thd[0] + x[1] * ob.thd[1] + x[2] * ob.thd[2]) * ob.inv_hh;
            const int ix = (int)floor((xi + 1.0) * (double)npx / 2.0), iy = (int)floor((yi + 1.0) * (double)npy / 2.0);
            if (ix < 0 || ix >= npx || iy < 0 || iy >= npy) { ++n_drop; }
            else {
                ++n_con;
                pixel = iy * npx + ix;
                out[0] = att * S[0]; out[1] = att * S[1]; out[2] = att * S[2]; out[3] = att * S[3];
            }
        }
        // I3: one atomic per distinct pixel of the warp: the values of every group of equal pixels are summed (fp64)
        // into its lowest lane
        const unsigned peers = __match_any_sync(0xffffffffu, pixel);
        const int leader = __ffs(peers) - 1;
        double acc[4] = { (double)out[0], (double)out[1], (double)out[2], (double)out[3] };
        {
            // tree over the lanes of each group, by their rank in it: in every round the lanes of even rank add the
            // partial sum of the next lane of their group still in play, those of odd rank leave: at most five
            // rounds (a group of 32), where collecting one peer at a time took up to 31
            int rank = __popc(peers & ((1u << lane) - 1u));
            bool in_play = pixel >= 0;
            unsigned above = in_play ? peers & (0xfffffffeu << lane) : 0u;     // lanes of the group above this one, still in play
            while (__any_sync(0xffffffffu, above != 0u)) {
                const int src = above ? __ffs(above) - 1 : lane;
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    const double v = __shfl_sync(0xffffffffu, acc[s], src);
                    if (above) acc[s] += v;
                }
                const unsigned stay = __ballot_sync(0xffffffffu, in_play && !(rank & 1));
                if (rank & 1) in_play = false;                              // added to its neighbour below
                above = in_play ? above & stay : 0u;
                rank >>= 1;
            }
        }
        if (pixel >= 0 && lane == leader) {
            const size_t plane = (size_t)npx * npy;
            double* at = img + (size_t)obs_index * 4 * plane + pixel;
            atomicAdd(at, acc[0]);
            atomicAdd(at + plane, acc[1]);
            atomicAdd(at + 2 * plane, acc[2]);
            atomicAdd(at + 3 * plane, acc[3]);
        }
    }
    steps = krp_warp_sum(steps); n_con = krp_warp_sum(n_con); n_drop = krp_warp_sum(n_drop);
    if (lane == 0) {
        if (steps) atomicAdd(&ctl->stats.steps_image, steps);
        if (n_con) atomicAdd(&ctl->stats.contributions, n_con);
        if (n_drop) atomicAdd(&ctl->stats.dropped, n_drop);
    }
}

// end of imaging: the event buffer is consumed
__global__ void krp_k_events_clear(KrpCtl* ctl) { ctl->n_events = 0; ctl->ev_begin = 0; }

// ------------------------------------------------------------------------------------------
// T0  setup kernels (not on the timed path)
// ------------------------------------------------------------------------------------------
__global__ void krp_k_pack(KrpModel g, const float* __restrict__ density, const float* __restrict__ bfield, uint32_t npad,
                           float4* __restrict__ cell, float* __restrict__ kr, int* __restrict__ bad)
{
    uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= npad) return;
    int hx, hy, hz;
    krp_pad_coords(g, c, hx, hy, hz);
    const bool halo = hx == 0 || hy == 0 || hz == 0 || hx == g.nx + 1 || hy == g.ny + 1 || hz == g.nz + 1;
    float d = -1.f;                                   // halo: negative kappa*rho marks the outside of the grid
    double bx = 0.0, by = 0.0, bz = 1.0;
    if (!halo) {
        const size_t lin = ((size_t)(hz - 1) * g.ny + (hy - 1)) * g.nx + (hx - 1);
        d = density[lin];
        if (!(d >= 0.f) || isinf(d)) { atomicAdd(bad, 1); d = 0.f; }
        if (bfield) {
            bx = bfield[3 * lin]; by = bfield[3 * lin + 1]; bz = bfield[3 * lin + 2];
            double r = sqrt(bx * bx + by * by + bz * bz);
            if (r > 0.0) { bx /= r; by /= r; bz /= r; } else { bx = 0.0; by = 0.0; bz = 1.0; }
        }
    }
    if (kr) kr[c] = d;
    if (cell) cell[c] = make_float4(d, (float)bx, (float)by, (float)bz);
}

__global__ void krp_k_f2d(const float* __restrict__ w, uint32_t n, double* __restrict__ o)
{
    uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c < n) o[c] = (double)w[c];
}
