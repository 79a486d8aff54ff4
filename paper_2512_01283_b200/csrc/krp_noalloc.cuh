// krp_noalloc.cuh -- krp_image_events_noalloc: per-event imaging (I1-I3) of caller-provided events with NO
// allocation of any kind in the call.  For callers that cannot reach cudaMalloc: code under CUDA graph capture, tight
// serving loops, harnesses that forbid it.  Included by krp_api.cu only (the array below and the host code that takes
// its address must be one translation unit).
//
// The imaging kernels work on the library's event records (three float4 per event) and a control block (work counters,
// tallies).  krp_image keeps both in buffers it allocates and grows; here they live in ONE file-scope device array of a
// fixed size, KRP_NOALLOC_MAX_EVENTS events = 12 MiB + the control block, which every GPU that loads the library holds
// until the process exits.  The imaging kernel itself is the one krp_image launches (general mode: the variant that reads
// the 16-byte cells directly -- the per-observer coefficient arrays of krp_image are an allocation), unordered.
//
// In HOST code `krp_na_scratch` is a stand-in, not a device address: krp_na_setup (from krp_grid_create, i.e. at set-up, with
// the grid's device current) asks cudaGetSymbolAddress once per device and the entry point hands that pointer to the kernels.
// Every call on a device shares the array, which keeps the last call's contents: the control block is cleared at the start of
// every call, the records are overwritten for the n events of the call and nothing beyond them is read.  Two calls that
// overlap on the GPU (different streams, or concurrent threads) race on it: callers serialise them.
#pragma once

#define KRP_NOALLOC_MAX_EVENTS_ 262144u

struct KrpNaScratch {
    KrpCtl ctl;
    float4 pc[KRP_NOALLOC_MAX_EVENTS_];
    float4 nk[KRP_NOALLOC_MAX_EVENTS_];
    float4 S[KRP_NOALLOC_MAX_EVENTS_];
};
static __device__ __align__(256) unsigned char krp_na_scratch[sizeof(KrpNaScratch)];

#define KRP_NA_MAX_DEVICES 64
static KrpNaScratch* krp_na_ptr[KRP_NA_MAX_DEVICES];      // device address of krp_na_scratch, per device ordinal (0 = not asked yet)

// set-up, once per device, that device current
static int krp_na_setup(int device)
{
    if (device < 0 || device >= KRP_NA_MAX_DEVICES) return KRP_OK;       // such a device gets KRP_ERR_STATE from the entry point
    if (krp_na_ptr[device]) return KRP_OK;
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, krp_na_scratch);
    if (e != cudaSuccess) return fail(KRP_ERR_CUDA, "cudaGetSymbolAddress(krp_na_scratch): %s", cudaGetErrorString(e));
    krp_na_ptr[device] = (KrpNaScratch*)p;
    return KRP_OK;
}

// Events in the public format of krp_events_get (DEVICE arrays) -> records in the scratch array; thread 0 opens the control
// block (cleared by the caller of this kernel).  An event outside the grid, with a negative index, non-finite values or a direction that is not a unit
// vector becomes a record of weight 0 in the first cell (it contributes nothing) and is counted in stats.overflow.
__global__ void __launch_bounds__(256) krp_k_na_load(KrpModel g, KrpNaScratch* s, unsigned int n, const int32_t* __restrict__ k,
                                                     const int64_t* __restrict__ cell, const float* __restrict__ pos,
                                                     const float* __restrict__ dir, const float* __restrict__ stokes)
{
    const unsigned int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) {
        s->ctl.n_events = n; s->ctl.ev_begin = 0; s->ctl.ev_cap = KRP_NOALLOC_MAX_EVENTS_;
        s->ctl.n_sorted = n;
    }
    if (i >= n) return;
    const int64_t c = cell[i];
    const float W = stokes[4 * i];
    const int32_t kk = k[i];
    bool ok = c >= 0 && c < (int64_t)g.ncell && kk >= 0 && isfinite(W);
    uint32_t cp = krp_pad_id(g, 0, 0, 0);
    float4 p = make_float4(0.5f, 0.5f, 0.5f, 0.f), d = make_float4(0.f, 0.f, 1.f, 0.f), S = make_float4(0.f, 0.f, 0.f, 0.f);
    if (ok) {
        const int64_t t = c / g.nx;
        const int ix = (int)(c - t * g.nx), iz = (int)(t / g.ny), iy = (int)(t - (int64_t)iz * g.ny);
        cp = krp_pad_id(g, ix, iy, iz);
        p.x = fminf(fmaxf(pos[3 * i], 0.f), 1.f); p.y = fminf(fmaxf(pos[3 * i + 1], 0.f), 1.f); p.z = fminf(fmaxf(pos[3 * i + 2], 0.f), 1.f);
        d.x = dir[3 * i]; d.y = dir[3 * i + 1]; d.z = dir[3 * i + 2];
        // the public format carries W (1, q, u, v); the records hold W and the normalised (q, u, v)
        const float inv = W != 0.f ? 1.f / W : 0.f;
        S = make_float4(W, stokes[4 * i + 1] * inv, stokes[4 * i + 2] * inv, stokes[4 * i + 3] * inv);
        const float nn = d.x * d.x + d.y * d.y + d.z * d.z;      // a direction (unit to fp32 rounding in krp_events_get's output)
        ok = nn > 0.5f && nn < 2.f && isfinite(S.y) && isfinite(S.z) && isfinite(S.w);
        if (!ok) { d = make_float4(0.f, 0.f, 1.f, 0.f); S = make_float4(0.f, 0.f, 0.f, 0.f); }
    }
    if (!ok) atomicAdd(&s->ctl.stats.overflow, 1ull);
    p.w = __uint_as_float(cp);
    d.w = __uint_as_float(ok ? (uint32_t)kk : 1u);
    s->pc[i] = p; s->nk[i] = d; s->S[i] = S;
}

extern "C" int krp_image_events_noalloc(krp_grid* g, uint64_t n, const int32_t* k, const int64_t* cell, const float* pos,
                                        const float* dir, const float* stokes, const krp_observer* obs, int npix_x, int npix_y,
                                        int flags, double* img, uint64_t* rejected, void* stream)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    if (n > KRP_NOALLOC_MAX_EVENTS_)
        return fail(KRP_ERR_ARG, "krp_image_events_noalloc takes at most %u events per call (its scratch array is fixed), got %llu",
                    KRP_NOALLOC_MAX_EVENTS_, (unsigned long long)n);
    int rc = check_observers(obs, 1, npix_x, npix_y);
    if (rc) return rc;
    if (!img) return fail(KRP_ERR_ARG, "img is NULL");
    if (n && (!k || !cell || !pos || !dir || !stokes)) return fail(KRP_ERR_ARG, "an event array is NULL");
    KrpNaScratch* s = (g->device >= 0 && g->device < KRP_NA_MAX_DEVICES) ? krp_na_ptr[g->device] : nullptr;
    if (!s) return fail(KRP_ERR_STATE, "no scratch address for device %d (krp_grid_create asks for it)", g->device);
    cudaStream_t st = (cudaStream_t)stream;
    if (rejected) *rejected = 0;
    if (n == 0) return KRP_OK;
    // everything that must start at zero: work counters and tallies of the control block
    CK(cudaMemsetAsync(&s->ctl, 0, sizeof(KrpCtl), st));
    krp_k_na_load<<<(unsigned)((n + 255u) / 256u), 256, 0, st>>>(g->m, s, (unsigned int)n, k, cell, pos, dir, stokes);
    const KrpObserverDev od = make_observer_dev(g, obs[0]);
    const KrpRecords ev = { s->pc, s->nk, s->S, nullptr, nullptr };
    const unsigned pers = (unsigned)(g->n_sm * g->blocks_per_sm);
    const int tb = g->image_block;
    const size_t smem = g->m.scalar ? 0 : 2 * sizeof(float4) * (size_t)(g->m.n_inc - 1);
    const bool zt = g->m.z.zt != nullptr;
#define KRP_NA_ARGS g->m, &s->ctl, ev, (const unsigned int*)nullptr, od, (const float4*)nullptr, 0, 0, npix_x, npix_y, flags, img
    if (g->m.scalar) krp_k_image<true, false, false><<<pers, tb, 0, st>>>(KRP_NA_ARGS);
    else if (!zt)    krp_k_image<false, false, false><<<pers, tb, smem, st>>>(KRP_NA_ARGS);
    else             krp_k_image<false, false, true><<<pers, tb, smem, st>>>(KRP_NA_ARGS);
#undef KRP_NA_ARGS
    g->launches += 2;
    CK(cudaGetLastError());
    if (rejected) {      // the one synchronising part, only on request
        unsigned long long r = 0;
        CK(cudaMemcpyAsync(&r, &s->ctl.stats.overflow, sizeof(r), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        *rejected = r;
    }
    return KRP_OK;
}
