// krp_api.cu -- the C ABI of include/krp.h: argument checks, device memory, table building,
// kernel launches on the caller's stream.  No arithmetic of the method lives on the host
// except the one-off table preparation (Theta CDF, observer bases).
#include "../../include/krp.h"
#include "krp_kernels.cuh"
#include "krp_twostep.cuh"

#include <cub/device/device_scan.cuh>
#include <cub/device/device_radix_sort.cuh>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#ifndef KRP_SORT_BLOCK_LOG2
#define KRP_SORT_BLOCK_LOG2 6      // blocks of 64^3 cells in the imaging order (C5 imaging: 16^3 383 ms, 32^3 364 ms, 64^3 357 ms; profiles/r2q_README.md)
#endif

static thread_local char g_err[512] = "";

static int fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CK(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess)                                                                     \
            return fail(e_ == cudaErrorMemoryAllocation ? KRP_ERR_OOM : KRP_ERR_CUDA, "%s: %s", #call, \
                        cudaGetErrorString(e_));                                                   \
    } while (0)

// One set of lookup tables on the device with the model constants derived from it: one per frequency bin
// (eq. 8 holds per frequency bin; include/krp.h krp_freq_define)
struct TableSet {
    float4* d_opac = nullptr; float4* d_opA = nullptr; float4* d_opB = nullptr;
    double4* d_opA_d = nullptr; double4* d_opB_d = nullptr;
    float4* d_mueller = nullptr; double* d_cdf = nullptr;
    int n_inc = 0, n_ang = 0, max_scatter = 0, max_waves = 0;
    float a1c = 0, omc = 0, rho = 0, w_min = 0;
    bool constant = true, dichroic = false;
    float kscale = 1.f;             // density factor of the bin: kappa*rho of the bin = kscale x the model's
    double* d_img = nullptr;        // the bin's maps (same observer set and size for all bins)
};

static void free_tables(TableSet& t);
static int apply_scale(struct krp_grid* g, float k, cudaStream_t st);

struct krp_grid {
    KrpModel m;
    std::vector<TableSet> bins;     // frequency bins (at least one)
    int cur_bin = 0;
    float* d_base = nullptr;        // kappa*rho of the model in the padded order (kept once a bin scales the density)
    float cur_scale = 1.f;
    int device = 0, n_sm = 0;
    // owned device memory
    float* d_kr = nullptr;          // = d_kr_alloc + margin
    float4* d_cell = nullptr;       // = d_cell_alloc + margin
    float* d_kr_alloc = nullptr;
    float4* d_cell_alloc = nullptr;
    float* d_stage_den = nullptr;   // staging of host inputs (krp_grid_create / krp_grid_update with KRP_MEM_HOST)
    float* d_stage_b = nullptr;
    bool staged = false;            // krp_grid_stage: the staging buffers hold (or are receiving) a snapshot not yet packed
    cudaEvent_t stage_ev = nullptr;
    int* d_bad = nullptr;
    bool has_bfield = false;
    bool obs_cells_stale = false;   // cells changed since the per-observer coefficient arrays were built (or never built)
    bool obs_cells_failed = false;  // the arrays did not fit for the current observer set
    uint32_t npad = 0;
    // imaging order (counting sort of the events by cell bin)
    unsigned int* d_bins = nullptr;
    uint32_t n_bins = 0;
    KrpSortGeom sort_geom = { 5, 3, 1, 1 };
    int sub_bits = 0;
    unsigned int* d_perm = nullptr;
    uint64_t perm_cap = 0;
    void* d_scan = nullptr;
    size_t scan_bytes = 0;
    // emission order of a point source (direction bins)
    unsigned int* d_dir_bins = nullptr;
    void* d_dir_scan = nullptr;
    size_t dir_scan_bytes = 0;
    size_t dir_bins_cap = 0;         // counters d_dir_bins holds
    int dir_sort = 1;
    long long fused_max = 1048576;      // scalar mode: batches up to this many packets go through krp_k_packets_scalar (krp_tune_fused)
    unsigned int* d_order = nullptr;
    uint64_t order_cap = 0;
    double* d_src_cdf = nullptr;
    KrpCtl* d_ctl = nullptr;
    KrpRecords q[2] = {};
    uint64_t q_cap = 0;
    KrpHits hits = {};              // general mode: hit queue of the current wave (capacity q_cap)
    KrpRecords ev = {};
    uint64_t ev_cap = 0;
    bool ev_reserved = false;
    KrpObserverDev* d_obs = nullptr;
    // ordering of the events before imaging: policy 0 never, 1 by the measured ray length, 2 always
    int order_policy = 1;
    bool order_events = true, order_decided = false;
    unsigned long long pk_since_image = 0;                     // packets transported since the last krp_image
    double acc_pn = 0.0, req_pn = 0.0, prev_pn = 0.0;          // sum over passes of packets x observers: running, at the last counter request, at the last evaluation
    double events_per_packet = -1.0;                           // measured with the ordering decision (policy 1)
    unsigned long long* h_ray_stats = nullptr;          // pinned: steps_image, contributions, dropped
    unsigned long long ray_stats_prev[3] = { 0, 0, 0 };
    cudaEvent_t ray_stats_ev = nullptr;
    bool ray_stats_pending = false;
    // refill distance of the general flight chosen from the measured flight length (read back without waiting, then frozen)
    unsigned long long* h_flight_stats = nullptr;       // pinned: packets, events, records, steps_transport
    cudaEvent_t flight_stats_ev = nullptr;
    bool flight_stats_pending = false, burst_auto = true, burst_decided = false;
    float4* d_obs_cells = nullptr;  // [n_obs][npad] per-observer cell coefficients (general mode), or NULL
    int obs_pre = 1;
    double* d_img = nullptr;
    int n_obs = 0, npx = 0, npy = 0;
    std::vector<krp_observer> obs_host;
    std::vector<KrpObserverDev> obs_dev;
    // the paper's two-step form: source grid S(Omega_cam, x), its cameras, per-flight path lengths
    float* d_sgrid = nullptr;
    int sg_n_obs = 0;
    std::vector<krp_observer> sg_obs_host;
    KrpObserverDev* d_sg_obs = nullptr;
    double* d_flen = nullptr;
    uint64_t flen_cap = 0;
    unsigned short* d_dkeys[2] = { nullptr, nullptr };      // deposit: flights sorted by length (keys, item indices, cub scratch)
    unsigned int* d_dvals[2] = { nullptr, nullptr };
    void* d_dsort = nullptr;
    size_t dsort_bytes = 0;
    float* d_emis = nullptr;        // padded thermal source of krp_image_rays
    float* d_zt = nullptr; double* d_zt_norm = nullptr; double* d_zt_bound = nullptr;   // full Z of aligned grains (krp_zmatrix_set)
    uint64_t next_id = 0;
    uint64_t launches = 0;
    int transport_block = 256, image_block = 256, blocks_per_sm = 8;   // general mode: transport_block 128 (krp_grid_create)
    int bps_tuned = 0;
    int ev_has_emission = 0;        // emission records (k = 0) may be in the event buffer
    int burst = KRP_FLIGHT_BURST;   // cell steps between refill points of the flight kernels
    // optional per-launch timing (krp_timing_*)
    bool timing = false;
    std::vector<cudaEvent_t> t_ev;          // pairs: start, stop
    std::vector<int> t_cls;                 // class of every recorded pair
};

// brackets one launch (or a short run of launches of the same class) with events when timing is on
struct TimedLaunch {
    krp_grid* g; cudaStream_t st; cudaEvent_t stop = nullptr;
    TimedLaunch(krp_grid* g_, cudaStream_t st_, int cls) : g(g_), st(st_)
    {
        if (!g->timing || g->t_cls.size() >= 4096) return;
        const size_t k = g->t_cls.size();
        if (g->t_ev.size() < 2 * (k + 1)) {
            cudaEvent_t a = nullptr, b = nullptr;
            if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) return;
            g->t_ev.push_back(a); g->t_ev.push_back(b);
        }
        cudaEventRecord(g->t_ev[2 * k], st);
        stop = g->t_ev[2 * k + 1];
        g->t_cls.push_back(cls);
    }
    ~TimedLaunch() { if (stop) cudaEventRecord(stop, st); }
};

extern "C" const char* krp_last_error(void) { return g_err; }
#ifndef KRP_BUILD_ID
#define KRP_BUILD_ID "unstamped"
#endif
extern "C" const char* krp_version(void) { return "krp 0.2 sm_100a " KRP_BUILD_ID; }

static void free_hits(KrpHits& h)
{
    cudaFree(h.ic); cudaFree(h.Di); cudaFree(h.qu); cudaFree(h.vr); cudaFree(h.ryz);
    h = KrpHits{};
}

static int alloc_hits(KrpHits& h, uint64_t cap)
{
    CK(cudaMalloc(&h.ic, cap * sizeof(uint2)));
    CK(cudaMalloc(&h.Di, cap * sizeof(double2)));
    CK(cudaMalloc(&h.qu, cap * sizeof(double2)));
    CK(cudaMalloc(&h.vr, cap * sizeof(double2)));
    CK(cudaMalloc(&h.ryz, cap * sizeof(double2)));
    return KRP_OK;
}

static void free_records(KrpRecords& r)
{
    cudaFree(r.pc); cudaFree(r.nk); cudaFree(r.S); cudaFree(r.tau); cudaFree(r.id);
    r = KrpRecords{};
}

static int alloc_records(KrpRecords& r, uint64_t cap, bool with_tau)
{
    CK(cudaMalloc(&r.pc, cap * sizeof(float4)));
    CK(cudaMalloc(&r.nk, cap * sizeof(float4)));
    CK(cudaMalloc(&r.S, cap * sizeof(float4)));
    if (with_tau) CK(cudaMalloc(&r.tau, cap * sizeof(double)));
    CK(cudaMalloc(&r.id, cap * sizeof(unsigned long long)));
    return KRP_OK;
}

extern "C" int krp_grid_destroy(krp_grid* g)
{
    if (!g) return KRP_OK;
    cudaFree(g->d_kr_alloc); cudaFree(g->d_cell_alloc); cudaFree(g->d_stage_den); cudaFree(g->d_stage_b); if (g->stage_ev) cudaEventDestroy(g->stage_ev); cudaFree(g->d_bad); cudaFree(g->d_base);
    if (!g->bins.empty()) g->bins[g->cur_bin].d_img = nullptr;      // the current bin's maps are g->d_img, freed below
    for (TableSet& t : g->bins) free_tables(t);
    cudaFree(g->d_src_cdf); cudaFree(g->d_ctl); cudaFree(g->d_obs); cudaFree(g->d_img); cudaFree(g->d_obs_cells);
    cudaFree(g->d_bins); cudaFree(g->d_perm); cudaFree(g->d_scan);
    cudaFree(g->d_dir_bins); cudaFree(g->d_dir_scan); cudaFree(g->d_order);
    cudaFree(g->d_sgrid); cudaFree(g->d_sg_obs); cudaFree(g->d_flen); cudaFree(g->d_emis);
    cudaFree(g->d_dkeys[0]); cudaFree(g->d_dkeys[1]); cudaFree(g->d_dvals[0]); cudaFree(g->d_dvals[1]); cudaFree(g->d_dsort);
    cudaFree(g->d_zt); cudaFree(g->d_zt_norm); cudaFree(g->d_zt_bound);
    free_records(g->q[0]); free_records(g->q[1]); free_records(g->ev); free_hits(g->hits);
    for (cudaEvent_t e : g->t_ev) cudaEventDestroy(e);
    if (g->h_ray_stats) cudaFreeHost(g->h_ray_stats);
    if (g->h_flight_stats) cudaFreeHost(g->h_flight_stats);
    if (g->flight_stats_ev) cudaEventDestroy(g->flight_stats_ev);
    if (g->ray_stats_ev) cudaEventDestroy(g->ray_stats_ev);
    delete g;
    return KRP_OK;
}

static int check_tables(const krp_tables* t)
{
    if (!t) return fail(KRP_ERR_ARG, "tables is NULL");
    if (t->n_ang < 2 || !t->mueller) return fail(KRP_ERR_ARG, "tables: n_ang must be >= 2 and mueller non-NULL");
    if (t->n_inc < 1 || t->n_inc > 1024 || !t->opacity) return fail(KRP_ERR_ARG, "tables: n_inc must be in 1..1024 and opacity non-NULL");
    if (!(t->w_min >= 0.f)) return fail(KRP_ERR_ARG, "tables: w_min must be >= 0");
    if (t->max_scatter < 1) return fail(KRP_ERR_ARG, "tables: max_scatter must be >= 1");
    if (t->periodic < 0 || t->periodic > 7) return fail(KRP_ERR_ARG, "tables: periodic must be a mask of the bits 1 (x), 2 (y), 4 (z)");
    for (int j = 0; j < t->n_ang; ++j) {
        const float* f = t->mueller + 4 * j;
        for (int s = 0; s < 4; ++s)
            if (!std::isfinite(f[s])) return fail(KRP_ERR_ARG, "tables: mueller[%d][%d] is not finite", j, s);
        if (!(f[0] > 0.f)) return fail(KRP_ERR_ARG, "tables: S11 must be positive (node %d)", j);
        double lhs = (double)f[0] * f[0] * (1.0 + 1e-6), rhs = (double)f[1] * f[1] + (double)f[2] * f[2] + (double)f[3] * f[3];
        if (lhs < rhs) return fail(KRP_ERR_ARG, "tables: S11^2 < S12^2+S33^2+S34^2 at node %d", j);
    }
    for (int j = 0; j < t->n_inc; ++j) {
        const float* a = t->opacity + 4 * j;
        for (int s = 0; s < 4; ++s)
            if (!std::isfinite(a[s])) return fail(KRP_ERR_ARG, "tables: opacity[%d][%d] is not finite", j, s);
        if (!(a[0] > std::fabs(a[1]))) return fail(KRP_ERR_ARG, "tables: alpha1 must exceed |alpha2| (node %d)", j);
        if (!(a[3] >= 0.f && a[3] <= 1.f)) return fail(KRP_ERR_ARG, "tables: albedo outside [0,1] (node %d)", j);
    }
    return KRP_OK;
}

static void free_tables(TableSet& t)
{
    cudaFree(t.d_opac); cudaFree(t.d_opA); cudaFree(t.d_opB); cudaFree(t.d_opA_d); cudaFree(t.d_opB_d); cudaFree(t.d_mueller);
    cudaFree(t.d_cdf); cudaFree(t.d_img);
    t = TableSet{};
}

// T0: upload one table set and derive the constants the kernels need from it
static int build_tables(const krp_tables* tables, TableSet& t, cudaStream_t st)
{
    // opacity table: n_inc = 1 becomes two equal rows so that the kernels always interpolate
    const int n_inc = tables->n_inc == 1 ? 2 : tables->n_inc;
    std::vector<float> op(4 * (size_t)n_inc);
    for (int j = 0; j < n_inc; ++j)
        memcpy(&op[4 * j], tables->opacity + 4 * (tables->n_inc == 1 ? 0 : j), 4 * sizeof(float));
    t.constant = true; t.dichroic = false;
    float rho = 0.f;
    for (int j = 0; j < n_inc; ++j) {
        for (int s = 0; s < 4; ++s) t.constant = t.constant && (op[4 * j + s] == op[s]);
        t.dichroic = t.dichroic || op[4 * j + 1] != 0.f || op[4 * j + 2] != 0.f;
        rho = std::fmax(rho, std::fabs(op[4 * j + 1]) / op[4 * j]);
    }
    t.a1c = op[0]; t.omc = op[3]; t.rho = rho;
    t.n_inc = n_inc; t.n_ang = tables->n_ang;
    t.w_min = tables->w_min; t.max_scatter = tables->max_scatter;
    // number of waves that can contain live packets: the weight after k scatterings is <= omega_max^k
    {
        float om_max = 0.f;
        for (int j = 0; j < n_inc; ++j) om_max = std::fmax(om_max, op[4 * j + 3]);
        int waves = tables->max_scatter;
        if (om_max <= 0.f) waves = 1;
        else if (om_max < 1.f && tables->w_min > 0.f) {
            double kk = std::ceil(std::log((double)tables->w_min) / std::log((double)om_max)) + 1.0;
            if (kk < waves) waves = (int)std::fmax(kk, 1.0);
        }
        t.max_waves = waves;
    }
    CK(cudaMalloc(&t.d_opac, sizeof(float4) * n_inc));
    CK(cudaMemcpyAsync(t.d_opac, op.data(), sizeof(float4) * n_inc, cudaMemcpyHostToDevice, st));
    // the same table as intercept + slope per segment of x = mu*(n_inc-1): value = A_j + B_j x on [j, j+1]
    std::vector<float> A(4 * (size_t)(n_inc - 1)), B(4 * (size_t)(n_inc - 1));
    std::vector<double> Ad(4 * (size_t)(n_inc - 1)), Bd(4 * (size_t)(n_inc - 1));
    for (int j = 0; j + 1 < n_inc; ++j)
        for (int s = 0; s < 4; ++s) {
            double a = op[4 * j + s], b = op[4 * (j + 1) + s];
            B[4 * j + s] = (float)(b - a); A[4 * j + s] = (float)(a - (b - a) * j);
            Bd[4 * j + s] = b - a; Ad[4 * j + s] = a - (b - a) * j;
        }
    CK(cudaMalloc(&t.d_opA, sizeof(float4) * (n_inc - 1)));
    CK(cudaMalloc(&t.d_opB, sizeof(float4) * (n_inc - 1)));
    CK(cudaMemcpyAsync(t.d_opA, A.data(), sizeof(float4) * (n_inc - 1), cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(t.d_opB, B.data(), sizeof(float4) * (n_inc - 1), cudaMemcpyHostToDevice, st));
    CK(cudaMalloc(&t.d_opA_d, sizeof(double4) * (n_inc - 1)));
    CK(cudaMalloc(&t.d_opB_d, sizeof(double4) * (n_inc - 1)));
    CK(cudaMemcpyAsync(t.d_opA_d, Ad.data(), sizeof(double4) * (n_inc - 1), cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(t.d_opB_d, Bd.data(), sizeof(double4) * (n_inc - 1), cudaMemcpyHostToDevice, st));
    CK(cudaMalloc(&t.d_mueller, sizeof(float4) * t.n_ang));
    CK(cudaMemcpyAsync(t.d_mueller, tables->mueller, sizeof(float4) * t.n_ang, cudaMemcpyHostToDevice, st));
    // Theta CDF: trapezoid of S11 sin(Theta) on the nodes, fp64 (R13)
    std::vector<double> cdf(t.n_ang);
    {
        const double h = KRP_PI_D / (t.n_ang - 1);
        double acc = 0.0, prev = 0.0;
        cdf[0] = 0.0;
        for (int j = 1; j < t.n_ang; ++j) {
            double cur = (double)tables->mueller[4 * j] * std::sin(j * h);
            acc += 0.5 * (prev + cur);
            cdf[j] = acc;
            prev = cur;
        }
        for (int j = 0; j < t.n_ang; ++j) cdf[j] /= acc;
        cdf[t.n_ang - 1] = 1.0;
    }
    CK(cudaMalloc(&t.d_cdf, sizeof(double) * t.n_ang));
    CK(cudaMemcpyAsync(t.d_cdf, cdf.data(), sizeof(double) * t.n_ang, cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));          // the host vectors are locals
    return KRP_OK;
}

// make bin b's tables the ones the kernels see
static void apply_tables(krp_grid* g, int b)
{
    KrpModel& m = g->m;
    const TableSet& t = g->bins[b];
    m.opac = t.d_opac; m.opA = t.d_opA; m.opB = t.d_opB; m.opA_d = t.d_opA_d; m.opB_d = t.d_opB_d;
    m.mueller = t.d_mueller; m.cdf = t.d_cdf;
    m.n_inc = t.n_inc; m.n_ang = t.n_ang;
    m.a1c = t.a1c; m.omc = t.omc; m.rho = t.rho;
    m.xs = (double)(t.n_inc - 1); m.guard = 1.f + t.rho + 1e-3f; m.inv_nang1 = 1.0 / (double)(t.n_ang - 1);
    m.nang1_over_pi = (float)((double)(t.n_ang - 1) / 3.14159265358979323846);
    m.w_min = t.w_min; m.max_scatter = t.max_scatter;
    g->cur_bin = b;
}

// T0: (re)pack the caller's density / field arrays into the padded cell array of g (halo included)
// host arrays -> the model's staging buffers (kept for later calls), asynchronously on st
static int stage_copy(krp_grid* g, const float* density, const float* bfield, cudaStream_t st)
{
    KrpModel& m = g->m;
    if (!g->d_stage_den) CK(cudaMalloc(&g->d_stage_den, sizeof(float) * (size_t)m.ncell));
    CK(cudaMemcpyAsync(g->d_stage_den, density, sizeof(float) * (size_t)m.ncell, cudaMemcpyHostToDevice, st));
    if (bfield && !m.scalar) {
        if (!g->d_stage_b) CK(cudaMalloc(&g->d_stage_b, sizeof(float) * 3 * (size_t)m.ncell));
        CK(cudaMemcpyAsync(g->d_stage_b, bfield, sizeof(float) * 3 * (size_t)m.ncell, cudaMemcpyHostToDevice, st));
    }
    return KRP_OK;
}

static int upload_cells(krp_grid* g, const float* density, const float* bfield, int mem, cudaStream_t st)
{
    KrpModel& m = g->m;
    const float* d_den = density;
    const float* d_b = bfield;
    const bool want_b = bfield && !m.scalar;
    if (mem == KRP_MEM_HOST) {
        g->staged = false;      // a staged snapshot that was never packed is overwritten
        int rc = stage_copy(g, density, bfield, st);
        if (rc) return rc;
        d_den = g->d_stage_den;
        if (want_b) d_b = g->d_stage_b;
    }
    if (!g->d_bad) CK(cudaMalloc(&g->d_bad, sizeof(int)));
    CK(cudaMemsetAsync(g->d_bad, 0, sizeof(int), st));
    const int tb = 256;
    const unsigned nb = (unsigned)((g->npad + tb - 1) / tb);
    krp_k_pack<<<nb, tb, 0, st>>>(m, d_den, want_b ? d_b : nullptr, g->npad, g->d_cell, g->d_kr, g->d_bad);
    CK(cudaGetLastError());
    g->launches++;
    int bad = 0;
    CK(cudaMemcpyAsync(&bad, g->d_bad, sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (bad) return fail(KRP_ERR_ARG, "density has %d negative, NaN or infinite cells", bad);
    g->obs_cells_stale = true;
    if (g->d_base) {       // frequency bins scale the density: keep the new model values and re-apply the current factor
        const float k = g->cur_scale;
        krp_k_save_base<<<nb, tb, 0, st>>>(g->npad, g->d_kr, g->d_cell, g->d_base);
        g->launches++;
        g->cur_scale = 1.f;
        return apply_scale(g, k, st);
    }
    return KRP_OK;
}

static int krp_na_setup(int device);      // krp_noalloc.cuh (end of this file)

extern "C" int krp_grid_create(krp_grid** out, int nx, int ny, int nz, const double bounds[6], const float* density,
                               const float* bfield, int mem, const krp_tables* tables, void* stream)
{
    if (!out) return fail(KRP_ERR_ARG, "out is NULL");
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1) return fail(KRP_ERR_ARG, "grid dims must be positive (%d,%d,%d)", nx, ny, nz);
    if ((uint64_t)(nx + 2) * (ny + 2) * (nz + 2) >= (1ull << 31)) return fail(KRP_ERR_ARG, "grid has too many cells (limit 2^31 with halo)");
    if (!bounds) return fail(KRP_ERR_ARG, "bounds is NULL");
    for (int a = 0; a < 3; ++a)
        if (!(bounds[2 * a + 1] > bounds[2 * a]) || !std::isfinite(bounds[2 * a]) || !std::isfinite(bounds[2 * a + 1]))
            return fail(KRP_ERR_ARG, "bounds must be finite and increasing on axis %d", a);
    if (!density) return fail(KRP_ERR_ARG, "density is NULL");
    if (mem != KRP_MEM_DEVICE && mem != KRP_MEM_HOST) return fail(KRP_ERR_ARG, "mem must be KRP_MEM_DEVICE or KRP_MEM_HOST");
    int rc = check_tables(tables);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;

    krp_grid* g = new (std::nothrow) krp_grid();
    if (!g) return fail(KRP_ERR_OOM, "host allocation failed");
    struct Guard { krp_grid* g; ~Guard() { if (g) krp_grid_destroy(g); } } guard{ g };

    CK(cudaGetDevice(&g->device));
    CK(cudaDeviceGetAttribute(&g->n_sm, cudaDevAttrMultiProcessorCount, g->device));
    rc = krp_na_setup(g->device);      // address of the fixed scratch array of krp_image_events_noalloc on this device
    if (rc) return rc;
    KrpModel& m = g->m;
    memset(&m, 0, sizeof(m));
    m.nx = nx; m.ny = ny; m.nz = nz; m.ncell = (uint32_t)((uint64_t)nx * ny * nz);
    m.px = nx + 2; m.py = ny + 2; m.pxy = (uint32_t)m.px * (uint32_t)m.py;
    g->npad = m.pxy * (uint32_t)(nz + 2);
    m.npad = g->npad;
    {
        auto magic = [](uint32_t d, uint32_t& mm, uint32_t& ss) {
            uint32_t l = 0;
            while ((1ull << l) < d) ++l;
            mm = (uint32_t)(((1ull << 32) * ((1ull << l) - d)) / d + 1);
            ss = l - 1;
        };
        magic((uint32_t)m.px, m.px_m, m.px_s);
        magic((uint32_t)m.py, m.py_m, m.py_s);
    }
    const int dims[3] = { nx, ny, nz };
    for (int a = 0; a < 3; ++a) {
        m.lo[a] = bounds[2 * a];
        m.dd[a] = (bounds[2 * a + 1] - bounds[2 * a]) / dims[a];
        m.d[a] = (float)m.dd[a];
        m.inv_dd[a] = 1.0 / m.dd[a];
    }
    // tables of the first (and, until krp_freq_define, only) frequency bin
    g->bins.resize(1);
    rc = build_tables(tables, g->bins[0], st);
    if (rc) return rc;
    m.periodic = tables->periodic;
    m.scalar = (g->bins[0].constant && !g->bins[0].dichroic && bfield == nullptr && !m.periodic) ? 1 : 0;
    apply_tables(g, 0);
    // scalar flights are short: static assignment; general flights are long: persistent lanes, refill every 32 steps
    g->burst = m.scalar ? 1 : 32;
    if (!m.scalar) g->transport_block = 128;
    if (m.scalar)
        CK(cudaFuncSetAttribute(krp_k_flight_scalar, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(8 * sizeof(KrpWarpShared))));
    g->order_events = g->order_policy != 0;

    // cells: packed into the padded layout (one-cell halo with kappa*rho = -1).  A margin of one padded plane on
    // either side keeps the look-ahead loads of the marches (one cell past the halo cell that ends a ray) inside
    // the allocation; its content is never used.
    {
        const size_t margin = m.pxy, n_alloc = (size_t)g->npad + 2 * margin;
        if (m.scalar) {
            CK(cudaMalloc(&g->d_kr_alloc, sizeof(float) * n_alloc));
            CK(cudaMemsetAsync(g->d_kr_alloc, 0xff, sizeof(float) * n_alloc, st));
            g->d_kr = g->d_kr_alloc + margin;
        } else {
            CK(cudaMalloc(&g->d_cell_alloc, sizeof(float4) * n_alloc));
            CK(cudaMemsetAsync(g->d_cell_alloc, 0xff, sizeof(float4) * n_alloc, st));
            g->d_cell = g->d_cell_alloc + margin;
        }
    }
    g->has_bfield = bfield != nullptr;
    rc = upload_cells(g, density, bfield, mem, st);
    if (rc) return rc;
    m.kr = g->d_kr; m.cell = g->d_cell;
    // bins of the imaging order: blocks of 64^3 cells, inside a block one cache line of cells along x per bin
    // (32 x 4 B or 8 x 16 B), at most 2^25 bins
    {
        KrpSortGeom& sg = g->sort_geom;
        sg.B = KRP_SORT_BLOCK_LOG2; sg.ls = m.scalar ? 5 : 3;
        const uint32_t bm = (1u << sg.B) - 1u;
        sg.nbx = ((uint32_t)m.px + bm) >> sg.B; sg.nby = ((uint32_t)m.py + bm) >> sg.B;
        const uint64_t nblk = (uint64_t)sg.nbx * sg.nby * (((uint32_t)nz + 2u + bm) >> sg.B);
        while (sg.ls < sg.B && (nblk << (3 * sg.B - sg.ls)) >= (1ull << 25)) sg.ls++;
        if ((nblk << (3 * sg.B - sg.ls)) >= (1ull << 31)) return fail(KRP_ERR_ARG, "grid too large for the imaging order");
        g->n_bins = (uint32_t)(nblk << (3 * sg.B - sg.ls)) + 1;
        if (m.scalar) {       // plain cell order, one 128-byte line of cells per bin
            sg.B = 0; sg.ls = 5;
            while ((g->npad >> sg.ls) >= (1u << 25)) sg.ls++;
            g->n_bins = (g->npad >> sg.ls) + 1;
        }
    }
    // sub-counters per bin against atomic contention in hot cells.  A grid of few bins (up to 2^17: C1, C2) collects hundreds
    // of events per bin and takes up to 128 counters per bin (four lines, 2^24 counters at most; measured on C2: 16 per bin
    // 0.85 ms, 64 0.86 ms, 128 0.57 ms, 256 0.61 ms); a large grid has a few events per bin and pays for every extra counter in the
    // scan (C4: 1 per bin 0.63 ms, 2 0.76 ms, 4 0.88 ms): about 2^21 counters in all, at most 64 per bin
    const bool few_bins = g->n_bins <= (1u << 17);
    const int sub_max = few_bins ? 7 : 6, cap_log2 = few_bins ? 24 : 21;
    g->sub_bits = 0;
    while (g->sub_bits < sub_max && ((uint64_t)g->n_bins << (g->sub_bits + 1)) <= (1ull << cap_log2)) g->sub_bits++;
    g->n_bins <<= g->sub_bits;
    CK(cudaMalloc(&g->d_bins, sizeof(unsigned int) * ((size_t)g->n_bins + 1)));
    CK(cub::DeviceScan::ExclusiveSum(nullptr, g->scan_bytes, g->d_bins, g->d_bins, (int)(g->n_bins + 1), st));
    CK(cudaMalloc(&g->d_scan, g->scan_bytes ? g->scan_bytes : 16));

    CK(cudaMalloc(&g->d_ctl, sizeof(KrpCtl)));
    CK(cudaMemsetAsync(g->d_ctl, 0, sizeof(KrpCtl), st));
    CK(cudaStreamSynchronize(st));
    // default source: isotropic point source at the centre of the box
    krp_source src;
    memset(&src, 0, sizeof(src));
    for (int a = 0; a < 3; ++a) src.pos[a] = 0.5 * (bounds[2 * a] + bounds[2 * a + 1]);
    src.dir[2] = 1.0;
    guard.g = nullptr;
    rc = krp_source_set(g, &src, stream);
    if (rc) { krp_grid_destroy(g); return rc; }
    *out = g;
    return KRP_OK;
}

extern "C" int krp_grid_update(krp_grid* g, const float* density, const float* bfield, int mem, void* stream)
{
    if (!g || !density) return fail(KRP_ERR_ARG, "grid or density is NULL");
    if (mem != KRP_MEM_DEVICE && mem != KRP_MEM_HOST) return fail(KRP_ERR_ARG, "mem must be KRP_MEM_DEVICE or KRP_MEM_HOST");
    if ((bfield != nullptr) != g->has_bfield) return fail(KRP_ERR_ARG, "bfield must be given exactly when the grid was created with one");
    return upload_cells(g, density, bfield, mem, (cudaStream_t)stream);
}

extern "C" int krp_grid_stage(krp_grid* g, const float* density, const float* bfield, void* copy_stream)
{
    if (!g || !density) return fail(KRP_ERR_ARG, "grid or density is NULL");
    if ((bfield != nullptr) != g->has_bfield) return fail(KRP_ERR_ARG, "bfield must be given exactly when the grid was created with one");
    if (!g->stage_ev) CK(cudaEventCreateWithFlags(&g->stage_ev, cudaEventDisableTiming));
    int rc = stage_copy(g, density, bfield, (cudaStream_t)copy_stream);
    if (rc) return rc;
    CK(cudaEventRecord(g->stage_ev, (cudaStream_t)copy_stream));
    g->staged = true;
    return KRP_OK;
}

extern "C" int krp_grid_update_staged(krp_grid* g, void* stream)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    if (!g->staged) return fail(KRP_ERR_STATE, "no staged snapshot: call krp_grid_stage first");
    CK(cudaStreamWaitEvent((cudaStream_t)stream, g->stage_ev, 0));
    g->staged = false;
    return upload_cells(g, g->d_stage_den, g->has_bfield ? g->d_stage_b : nullptr, KRP_MEM_DEVICE, (cudaStream_t)stream);
}

extern "C" int krp_source_set(krp_grid* g, const krp_source* src, void* stream)
{
    if (!g || !src) return fail(KRP_ERR_ARG, "grid or source is NULL");
    if (src->kind < 0 || src->kind > 7 || ((src->kind & 4) && (src->kind & 3) != 1))
        return fail(KRP_ERR_ARG, "source kind must be in 0..3, or 5 (thermal emission: volume source, isotropic candidates)");
    cudaStream_t st = (cudaStream_t)stream;
    KrpModel& m = g->m;
    if (src->kind & 2) {
        double nn = src->dir[0] * src->dir[0] + src->dir[1] * src->dir[1] + src->dir[2] * src->dir[2];
        if (!(nn > 0.0) || !std::isfinite(nn)) return fail(KRP_ERR_ARG, "collimated source needs a non-zero finite dir");
    }
    m.src_kind = src->kind; m.emit_records = src->emit_records ? 1 : 0;
    if (src->kind & 4) {
        if (m.emit_records) return fail(KRP_ERR_ARG, "a thermal source has no emission records: its direct light is krp_image_rays' thermal term");
        // max over the table nodes of (1 - omega) alpha1, from the fp32 table in fp64 (R22)
        const TableSet& t = g->bins[g->cur_bin];
        std::vector<float> op(4 * (size_t)t.n_inc);
        CK(cudaMemcpy(op.data(), t.d_opac, sizeof(float4) * t.n_inc, cudaMemcpyDeviceToHost));
        double emax = 0.0;
        for (int j = 0; j < t.n_inc; ++j) emax = std::fmax(emax, (1.0 - (double)op[4 * j + 3]) * (double)op[4 * j]);
        m.src_emax = emax;
    }
    const int dims[3] = { m.nx, m.ny, m.nz };
    int idx[3];
    // R23: `dir` need not be normalised -- divided by its length in fp64 here, rounded to fp32 (R12) below
    const double dir_len = (src->kind & 2) ? std::sqrt(src->dir[0] * src->dir[0] + src->dir[1] * src->dir[1] + src->dir[2] * src->dir[2]) : 1.0;
    for (int a = 0; a < 3; ++a) {
        if (!std::isfinite(src->pos[a])) return fail(KRP_ERR_ARG, "source pos is not finite");
        double x = (src->pos[a] - m.lo[a]) / m.dd[a];
        int i = (int)std::floor(x);
        i = i < 0 ? 0 : (i > dims[a] - 1 ? dims[a] - 1 : i);
        double p = x - i;
        p = p < 0.0 ? 0.0 : (p > 1.0 ? 1.0 : p);     // sources outside the box start on its surface
        idx[a] = i; m.src_p[a] = (float)p;
        m.src_n[a] = (float)((src->kind & 2) ? src->dir[a] / dir_len : src->dir[a]);
    }
    m.src_cell = ((uint32_t)(idx[2] + 1) * (uint32_t)m.py + (uint32_t)(idx[1] + 1)) * (uint32_t)m.px + (uint32_t)(idx[0] + 1);
    cudaFree(g->d_src_cdf); g->d_src_cdf = nullptr; m.src_cdf = nullptr;
    if ((src->kind & 1) && src->cell_weight) {
        double* tmp = nullptr;
        CK(cudaMalloc(&tmp, sizeof(double) * (size_t)m.ncell));
        CK(cudaMalloc(&g->d_src_cdf, sizeof(double) * (size_t)m.ncell));
        const int tb = 256;
        krp_k_f2d<<<(unsigned)((m.ncell + tb - 1) / tb), tb, 0, st>>>(src->cell_weight, m.ncell, tmp);
        CK(cudaGetLastError());
        void* scratch = nullptr; size_t bytes = 0;
        CK(cub::DeviceScan::InclusiveSum(scratch, bytes, tmp, g->d_src_cdf, (int)m.ncell, st));
        CK(cudaMalloc(&scratch, bytes));
        CK(cub::DeviceScan::InclusiveSum(scratch, bytes, tmp, g->d_src_cdf, (int)m.ncell, st));
        CK(cudaStreamSynchronize(st));
        cudaFree(scratch); cudaFree(tmp);
        g->launches += 2;
        m.src_cdf = g->d_src_cdf;
    }
    return KRP_OK;
}

static int ensure_events(krp_grid* g, uint64_t cap)
{
    if (g->ev_cap >= cap) return KRP_OK;
    // growing keeps nothing: only legal while the buffer is empty (checked by the callers)
    free_records(g->ev);
    g->ev_cap = 0;
    int rc = alloc_records(g->ev, cap, false);
    if (rc) { free_records(g->ev); return rc; }
    g->ev_cap = cap;
    return KRP_OK;
}

extern "C" int krp_events_reserve(krp_grid* g, uint64_t max_events)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    if (max_events < 1) return fail(KRP_ERR_ARG, "max_events must be positive");
    CK(cudaDeviceSynchronize());
    KrpCtl c;
    CK(cudaMemcpy(&c, g->d_ctl, sizeof(c), cudaMemcpyDeviceToHost));
    if (c.n_events != 0) return fail(KRP_ERR_STATE, "events_reserve with a non-empty event buffer");
    if (max_events != g->ev_cap) { free_records(g->ev); g->ev_cap = 0; }
    int rc = ensure_events(g, max_events);
    if (rc) return rc;
    g->ev_reserved = true;
    unsigned long long cap = g->ev_cap;
    CK(cudaMemcpy(&g->d_ctl->ev_cap, &cap, sizeof(cap), cudaMemcpyHostToDevice));
    return KRP_OK;
}

extern "C" int krp_packet_id_set(krp_grid* g, uint64_t next_id)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    g->next_id = next_id;
    return KRP_OK;
}

extern "C" int krp_transport(krp_grid* g, uint64_t n_packets, uint64_t seed, void* stream)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    if (n_packets == 0) return KRP_OK;
    if (n_packets > 0x7fffffffull) return fail(KRP_ERR_ARG, "n_packets per call is limited to 2^31-1; batch the run");
    cudaStream_t st = (cudaStream_t)stream;
    if (g->q_cap < n_packets) {
        CK(cudaStreamSynchronize(st));
        free_records(g->q[0]); free_records(g->q[1]); free_hits(g->hits); g->q_cap = 0;
        for (int s = 0; s < 2; ++s) {
            int rc = alloc_records(g->q[s], n_packets, true);
            if (rc) { free_records(g->q[0]); free_records(g->q[1]); return rc; }
        }
        if (!g->m.scalar) {
            int rc = alloc_hits(g->hits, n_packets);
            if (rc) { free_records(g->q[0]); free_records(g->q[1]); free_hits(g->hits); return rc; }
        }
        g->q_cap = n_packets;
    }
    if (!g->ev_reserved && g->ev_cap < 4 * n_packets) {
        // default capacity; only grown while the buffer is empty
        CK(cudaStreamSynchronize(st));
        KrpCtl c;
        CK(cudaMemcpy(&c, g->d_ctl, sizeof(c), cudaMemcpyDeviceToHost));
        if (c.n_events == 0 || g->ev_cap == 0) {
            uint64_t cap = 4 * n_packets;
            if (cap < (1ull << 20)) cap = 1ull << 20;
            int rc = ensure_events(g, cap);
            if (rc) return rc;
            unsigned long long c64 = g->ev_cap;
            CK(cudaMemcpy(&g->d_ctl->ev_cap, &c64, sizeof(c64), cudaMemcpyHostToDevice));
        }
    }
    if (g->d_sgrid && g->flen_cap < n_packets) {
        CK(cudaStreamSynchronize(st));
        cudaFree(g->d_flen); g->d_flen = nullptr; g->flen_cap = 0;
        cudaFree(g->d_dkeys[0]); cudaFree(g->d_dkeys[1]); cudaFree(g->d_dvals[0]); cudaFree(g->d_dvals[1]); cudaFree(g->d_dsort);
        g->d_dkeys[0] = g->d_dkeys[1] = nullptr; g->d_dvals[0] = g->d_dvals[1] = nullptr; g->d_dsort = nullptr;
        CK(cudaMalloc(&g->d_flen, sizeof(double) * n_packets));
        for (int k = 0; k < 2; ++k) {
            CK(cudaMalloc(&g->d_dkeys[k], sizeof(unsigned short) * n_packets));
            CK(cudaMalloc(&g->d_dvals[k], sizeof(unsigned int) * n_packets));
        }
        CK(cub::DeviceRadixSort::SortPairsDescending(nullptr, g->dsort_bytes, g->d_dkeys[0], g->d_dkeys[1], g->d_dvals[0], g->d_dvals[1], (int)n_packets, 0, 16, st));
        CK(cudaMalloc(&g->d_dsort, g->dsort_bytes ? g->dsort_bytes : 16));
        g->flen_cap = n_packets;
    }
    double* flen = g->d_sgrid ? g->d_flen : nullptr;
    // General flight: cell steps between two refill points, from the mean flight length of the batches so far (counters read back
    // without waiting; decided once, results do not depend on it).  Flights of one or two cells (C3: thick cells, 1.2 steps per
    // flight) take a new queue entry after every step: 10.8 -> 8.8 ms per 2^22 packets; long flights (C4, C5: ~67 steps) refill
    // every 16 steps (profiles/r2q_README.md).
    if (!g->m.scalar && g->burst_auto && !g->burst_decided && g->flight_stats_pending && cudaEventQuery(g->flight_stats_ev) == cudaSuccess) {
        g->flight_stats_pending = false;
        const unsigned long long flights = g->h_flight_stats[0] + g->h_flight_stats[1], steps = g->h_flight_stats[3];
        if (flights >= 10000ull) {
            const double len = (double)steps / (double)flights;
            g->burst = len < 3.0 ? 1 : (len < 24.0 ? 8 : 16);
            g->burst_decided = true;
        }
    }
    const unsigned n = (unsigned)n_packets;
    if (g->m.emit_records) g->ev_has_emission = 1;
    if (g->m.scalar && !flen && !g->m.z.zt && (long long)n_packets <= g->fused_max && g->bins[g->cur_bin].max_waves > 1) {
        // small batch, scalar mode: emission, then one kernel that follows every packet to its end (3 launches instead of 3 per order)
        { TimedLaunch tl(g, st, KRP_T_EMIT);
          krp_k_emit<<<(n + 255u) / 256u, 256, 0, st>>>(g->m, g->d_ctl, g->q[0], g->ev, g->next_id, n, seed, nullptr); }
        krp_k_wave_prep<<<1, 1, 0, st>>>(g->d_ctl, 0);
        { TimedLaunch tl(g, st, KRP_T_FLIGHT);
          const unsigned need_p = (n + 127u) / 128u, pers_p = (unsigned)g->n_sm * 6u;
          krp_k_packets_scalar<<<need_p < pers_p ? need_p : pers_p, 128, 0, st>>>(g->m, g->d_ctl, g->q[0], 0, g->ev, seed, g->bins[g->cur_bin].max_waves); }
        g->launches += 3;
        CK(cudaGetLastError());
        g->next_id += n_packets;
        g->pk_since_image += n_packets;
        return KRP_OK;
    }
    const int tb = g->transport_block;
    const unsigned grid_all = (n + 255u) / 256u;
    KrpEmitSrc es0 = { nullptr, g->next_id, seed };     // first scattering order
    {
        TimedLaunch tl(g, st, KRP_T_EMIT);
        if (g->m.src_kind == 0 && !g->m.emit_records && g->dir_sort && n >= (1u << 16)) {
            // isotropic point source: the first flights take the packets in the order of their direction and
            // compute the emission themselves (count, scan, order); nothing is written to the queue
            // sub-batches of 2^23 packets (32 MiB of slots each; measured on C2 against 2^21, 2^22 and one batch)
            unsigned sub_shift = KRP_DIR_SUB_SHIFT;
            while (((n - 1u) >> sub_shift) + 1u > KRP_DIR_SUBS_MAX) ++sub_shift;
            const size_t n_bins = (size_t)(((n - 1u) >> sub_shift) + 1u) * KRP_DIR_BINS;
            if (g->dir_bins_cap < n_bins) {
                CK(cudaStreamSynchronize(st));
                cudaFree(g->d_dir_bins); cudaFree(g->d_dir_scan); g->d_dir_bins = nullptr; g->d_dir_scan = nullptr; g->dir_bins_cap = 0;
                CK(cudaMalloc(&g->d_dir_bins, sizeof(unsigned int) * n_bins));
                CK(cub::DeviceScan::ExclusiveSum(nullptr, g->dir_scan_bytes, g->d_dir_bins, g->d_dir_bins, (int)n_bins, st));
                CK(cudaMalloc(&g->d_dir_scan, g->dir_scan_bytes ? g->dir_scan_bytes : 16));
                g->dir_bins_cap = n_bins;
            }
            if (g->order_cap < n_packets) {
                CK(cudaStreamSynchronize(st));
                cudaFree(g->d_order); g->d_order = nullptr; g->order_cap = 0;
                CK(cudaMalloc(&g->d_order, sizeof(unsigned int) * n_packets));
                g->order_cap = n_packets;
            }
            CK(cudaMemsetAsync(g->d_dir_bins, 0, sizeof(unsigned int) * n_bins, st));
            krp_k_emit_count<<<grid_all, 256, 0, st>>>(g->next_id, n, seed, g->d_dir_bins, sub_shift);
            CK(cub::DeviceScan::ExclusiveSum(g->d_dir_scan, g->dir_scan_bytes, g->d_dir_bins, g->d_dir_bins, (int)n_bins, st));
            krp_k_emit_order<<<grid_all, 256, 0, st>>>(g->d_ctl, g->next_id, n, seed, g->d_dir_bins, g->d_order, sub_shift);
            g->launches += 3;
            es0.order = g->d_order;
        } else {
            krp_k_emit<<<grid_all, 256, 0, st>>>(g->m, g->d_ctl, g->q[0], g->ev, g->next_id, n, seed, nullptr);
        }
    }
    g->launches++;
    unsigned pers = (unsigned)(g->n_sm * g->blocks_per_sm);
    unsigned need = (n + tb - 1) / tb;
    unsigned grid_f = need < pers ? need : pers;
    // general flight: persistent lanes, one resident set of blocks (640 threads per SM up to 128 per block, else 768) unless
    // krp_tune set blocks_per_sm
    const unsigned pers_g = (unsigned)g->n_sm * (unsigned)(g->bps_tuned ? g->blocks_per_sm : (tb <= 128 ? 640 / tb : 768 / tb));
    const unsigned grid_g = need < pers_g ? need : pers_g;
    unsigned grid_s = (n + 127u) / 128u;
    if (grid_s > pers * 2) grid_s = pers * 2;
    for (int w = 0; w < g->bins[g->cur_bin].max_waves; ++w) {
        const int in = w & 1;
        krp_k_wave_prep<<<1, 1, 0, st>>>(g->d_ctl, in);
        { TimedLaunch tl(g, st, KRP_T_FLIGHT);
        const KrpEmitSrc es = w == 0 ? es0 : KrpEmitSrc{ nullptr, 0, 0 };
        if (g->m.scalar && (g->burst == 1 || flen)) krp_k_flight_scalar_static<<<grid_f, tb, 0, st>>>(g->m, g->d_ctl, g->q[in], in, g->ev, es, flen);
        else if (g->m.scalar) krp_k_flight_scalar<<<grid_f, tb, (size_t)(tb / 32) * sizeof(KrpWarpShared), st>>>(g->m, g->d_ctl, g->q[in], in, g->ev, g->burst, es);
        else {
            if (tb <= 128) krp_k_flight_general<128, 5><<<grid_g, tb, 0, st>>>(g->m, g->d_ctl, g->q[in], in, g->hits, g->burst, es, flen);
            else           krp_k_flight_general<256, 3><<<grid_g, tb, 0, st>>>(g->m, g->d_ctl, g->q[in], in, g->hits, g->burst, es, flen);
            // the flights that reached their event cell: event location, record, albedo weighting, all lanes busy
            krp_k_event_general<<<grid_s, 128, 0, st>>>(g->m, g->d_ctl, g->q[in], in, g->hits, g->ev, es, flen);
            g->launches++;
        } }
        g->launches += 2;
        if (flen) {
            // step 1 of the two-step form: the flights of this wave, re-marched over their path lengths, deposit into S
            TimedLaunch tl(g, st, KRP_T_DEPOSIT);
            const KrpEmitSrc es = w == 0 ? es0 : KrpEmitSrc{ nullptr, 0, 0 };
            // flights of the wave sorted by the number of cells they cross (the queue's capacity is sorted: its fill is known on the device only)
            const unsigned n_cap = (unsigned)g->flen_cap < n ? (unsigned)g->flen_cap : n;
            krp_k_deposit_keys<<<(n_cap + 255u) / 256u, 256, 0, st>>>(g->m, g->d_ctl, g->q[in], in, es, flen, n_cap, g->d_dkeys[0], g->d_dvals[0]);
            CK(cub::DeviceRadixSort::SortPairsDescending(g->d_dsort, g->dsort_bytes, g->d_dkeys[0], g->d_dkeys[1], g->d_dvals[0], g->d_dvals[1], (int)n_cap, 0, 16, st));
            g->launches += 2;
            const unsigned need_d = (n + 127u) / 128u;
            const unsigned pers_d = (unsigned)g->n_sm * 8u;
            const unsigned grid_d = need_d < pers_d ? need_d : pers_d;
            const size_t smem_d = (size_t)g->sg_n_obs * 2 * 128 * sizeof(float4);
            if (g->m.scalar) krp_k_deposit<true><<<grid_d, 128, smem_d, st>>>(g->m, g->d_ctl, g->q[in], in, es, flen, g->d_dvals[1], g->d_sg_obs, g->sg_n_obs, g->d_sgrid, &g->d_ctl->sg_segments);
            else             krp_k_deposit<false><<<grid_d, 128, smem_d, st>>>(g->m, g->d_ctl, g->q[in], in, es, flen, g->d_dvals[1], g->d_sg_obs, g->sg_n_obs, g->d_sgrid, &g->d_ctl->sg_segments);
            g->launches++;
        }
        if (w + 1 < g->bins[g->cur_bin].max_waves) {
            TimedLaunch tl(g, st, KRP_T_SCATTER);
            if (g->m.z.zt) krp_k_scatter<true><<<grid_s, 128, 0, st>>>(g->m, g->d_ctl, g->ev, g->q[1 - in], 1 - in, seed);
            else         krp_k_scatter<false><<<grid_s, 128, 0, st>>>(g->m, g->d_ctl, g->ev, g->q[1 - in], 1 - in, seed);
            g->launches++;
        }
    }
    CK(cudaGetLastError());
    g->next_id += n_packets;
    g->pk_since_image += n_packets;
    if (!g->m.scalar && g->burst_auto && !g->burst_decided && !g->flight_stats_pending) {
        if (!g->h_flight_stats) {
            CK(cudaMallocHost(&g->h_flight_stats, 4 * sizeof(unsigned long long)));
            CK(cudaEventCreateWithFlags(&g->flight_stats_ev, cudaEventDisableTiming));
        }
        CK(cudaMemcpyAsync(g->h_flight_stats, &g->d_ctl->stats.packets, 4 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
        CK(cudaEventRecord(g->flight_stats_ev, st));
        g->flight_stats_pending = true;
    }
    return KRP_OK;
}

static void host_basis(const double n[3], double th[3], double ph[3])
{
    double s2 = n[0] * n[0] + n[1] * n[1], s = std::sqrt(s2), r = std::sqrt(s2 + n[2] * n[2]);
    double cp = 1.0, sp = 0.0;
    if (s2 >= 1e-24) { cp = n[0] / s; sp = n[1] / s; }
    double ct = n[2] / r, st = s / r;
    th[0] = ct * cp; th[1] = ct * sp; th[2] = -st;
    ph[0] = -sp; ph[1] = cp; ph[2] = 0.0;
}

// observer bases and launch constants of one camera
static KrpObserverDev make_observer_dev(const krp_grid* g, const krp_observer& ob)
{
    KrpObserverDev od;
    memset(&od, 0, sizeof(od));
    double st_ = std::sin(ob.theta), ct_ = std::cos(ob.theta);
    double n[3] = { st_ * std::cos(ob.phi), st_ * std::sin(ob.phi), ct_ }, th[3], ph[3];
    host_basis(n, th, ph);
    for (int a = 0; a < 3; ++a) {
        od.n[a] = (float)n[a]; od.th[a] = (float)th[a]; od.ph[a] = (float)ph[a];
        od.thd[a] = th[a]; od.phd[a] = ph[a]; od.center[a] = ob.center[a];
    }
    od.inv_hw = 1.0 / ob.half_w; od.inv_hh = 1.0 / ob.half_h;
    const int strides[3] = { 1, g->m.px, (int)g->m.pxy };
    for (int a = 0; a < 3; ++a) {
        const float nf = od.n[a];
        od.dt[a] = nf != 0.f ? g->m.d[a] / std::fabs(nf) : INFINITY;
        od.stride[a] = nf > 0.f ? strides[a] : (nf < 0.f ? -strides[a] : 0);
    }
    return od;
}

static int check_observers(const krp_observer* obs, int n_obs, int npix_x, int npix_y)
{
    if (!obs || n_obs < 1) return fail(KRP_ERR_ARG, "need at least one observer");
    if (npix_x < 1 || npix_y < 1) return fail(KRP_ERR_ARG, "pixel counts must be positive");
    for (int o = 0; o < n_obs; ++o)
        if (!(obs[o].half_w > 0.0) || !(obs[o].half_h > 0.0) || !std::isfinite(obs[o].theta) || !std::isfinite(obs[o].phi))
            return fail(KRP_ERR_ARG, "observer %d: half extents must be positive and angles finite", o);
    return KRP_OK;
}

// maps and per-observer data of an observer set (krp_image, krp_image_rays): (re)built when the set or the pixel counts change
static int setup_maps(krp_grid* g, const krp_observer* obs, int n_obs, int npix_x, int npix_y, cudaStream_t st, bool want_obs_cells)
{
    bool same = g->d_img && g->n_obs == n_obs && g->npx == npix_x && g->npy == npix_y &&
                memcmp(g->obs_host.data(), obs, sizeof(krp_observer) * n_obs) == 0;
    if (!same) {
        CK(cudaStreamSynchronize(st));
        cudaFree(g->d_img); g->d_img = nullptr;
        size_t bytes = sizeof(double) * 4 * (size_t)n_obs * npix_x * npix_y;
        CK(cudaMalloc(&g->d_img, bytes));
        CK(cudaMemsetAsync(g->d_img, 0, bytes, st));
        std::vector<KrpObserverDev> od(n_obs);
        for (int o = 0; o < n_obs; ++o) od[o] = make_observer_dev(g, obs[o]);
        g->obs_dev = od;
        g->obs_host.assign(obs, obs + n_obs);
        cudaFree(g->d_obs_cells); g->d_obs_cells = nullptr;
        g->obs_cells_failed = false;
        g->n_obs = n_obs; g->npx = npix_x; g->npy = npix_y;
    }
    // I0b: per-observer cell coefficients (general mode), when n_obs arrays of 16 B per padded cell fit
    if (want_obs_cells && !g->d_obs_cells && !g->m.scalar && g->obs_pre && !g->obs_cells_failed) {
        size_t free_b = 0, total_b = 0;
        CK(cudaMemGetInfo(&free_b, &total_b));
        const size_t need = sizeof(float4) * (size_t)g->npad * (size_t)n_obs;
        if (need + (4ull << 30) < free_b && cudaMalloc(&g->d_obs_cells, need) == cudaSuccess) {
            g->obs_cells_stale = true;
        } else {
            cudaGetLastError();
            g->d_obs_cells = nullptr;
            g->obs_cells_failed = true;      // not retried until the observer set changes
        }
    }
    return KRP_OK;
}

extern "C" int krp_image(krp_grid* g, const krp_observer* obs, int n_obs, int npix_x, int npix_y, int flags, void* stream)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    int rc = check_observers(obs, n_obs, npix_x, npix_y);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    rc = setup_maps(g, obs, n_obs, npix_x, npix_y, st, true);
    if (rc) return rc;
    if (g->d_obs_cells && g->obs_cells_stale) {
        // the cells changed (krp_grid_update) since the coefficient arrays were built
        const unsigned nb = (unsigned)((g->npad + 255u) / 256u);
        for (int o = 0; o < n_obs; ++o)
            krp_k_obs_cells<<<nb, 256, 0, st>>>(g->m, g->obs_dev[o], g->npad, g->d_obs_cells + (size_t)o * g->npad);
        CK(cudaGetLastError());
        g->launches += (uint64_t)n_obs;
        g->obs_cells_stale = false;
    }
    if (g->ev_cap == 0) return KRP_OK;   // nothing was ever transported
    if (g->ev_cap >= (1ull << 32)) return fail(KRP_ERR_ARG, "krp_image handles at most 2^32-1 buffered events per call");
    if (g->perm_cap < g->ev_cap) {
        CK(cudaStreamSynchronize(st));
        cudaFree(g->d_perm); g->d_perm = nullptr; g->perm_cap = 0;
        CK(cudaMalloc(&g->d_perm, sizeof(unsigned int) * g->ev_cap));
        g->perm_cap = g->ev_cap;
    }
    // I0: order the events by cell bin (count, scan, scatter) -- unless the rays of this model are so short that the
    // order does not pay: the decision follows the cell steps per ray of the previous imaging passes, read back
    // without waiting (a pinned copy of the counters taken after every pass; the first passes are ordered)
    const unsigned pers = (unsigned)(g->n_sm * g->blocks_per_sm);
    if (g->h_ray_stats && g->ray_stats_pending && cudaEventQuery(g->ray_stats_ev) == cudaSuccess) {
        // (the counters may have been reset by krp_stats_reset in between: then they count from zero)
        auto delta = [&](int j) { return g->h_ray_stats[j] >= g->ray_stats_prev[j] ? g->h_ray_stats[j] - g->ray_stats_prev[j] : g->h_ray_stats[j]; };
        const unsigned long long steps = delta(0), rays = delta(1) + delta(2);
        // decided once, on the first pass that has marched a fair number of rays, then kept: step times stay reproducible from
        // run to run also for models near the threshold
        if (rays >= 100000ull && !g->order_decided) {
            g->order_events = g->order_policy == 2 || (g->order_policy == 1 && (double)steps / (double)rays >= 12.0);
            g->order_decided = true;
            if (g->req_pn > g->prev_pn) g->events_per_packet = (double)rays / (g->req_pn - g->prev_pn);
        }
        g->ray_stats_prev[0] = g->h_ray_stats[0]; g->ray_stats_prev[1] = g->h_ray_stats[1]; g->ray_stats_prev[2] = g->h_ray_stats[2];
        g->prev_pn = g->req_pn;
        g->ray_stats_pending = false;
    }
    // ... nor when the events are few and the cell array small: a pass of fewer than 2^18 events over an array of at most 12 MiB,
    // a tenth of L2 (its rays find their cells there in any order; at 15 MiB -- C5 at 96^3 -- the order still wins by 9 %) costs more to order than the order saves (C1, 10^5 packets on 32^3 cells:
    // ordering + imaging 74 -> 49 us; C2 at 2^17 packets: 224 -> 175 us; at 2^20 packets the order wins, 458 against 506 us; on the
    // 512^3 grid of C5 it wins at any size).  Host-side estimate, the same for every pass of equal size: packets since the last
    // pass x the events per packet measured with the decision above.
    const size_t cell_bytes = (size_t)g->npad * (g->m.scalar ? sizeof(float) : sizeof(float4));
    const bool few = g->order_policy == 1 && g->events_per_packet >= 0.0 && cell_bytes <= ((size_t)12 << 20) &&
                     (double)g->pk_since_image * g->events_per_packet < 262144.0;
    const bool order_now = g->order_events && !few;
    g->acc_pn += (double)g->pk_since_image * (double)n_obs;
    g->pk_since_image = 0;
    const unsigned int* perm = order_now ? g->d_perm : nullptr;
    { TimedLaunch tlo(g, st, KRP_T_ORDER);
    if (order_now) {
        CK(cudaMemsetAsync(g->d_bins, 0, sizeof(unsigned int) * ((size_t)g->n_bins + 1), st));
        const int sflags = flags | (g->ev_has_emission ? 0 : 2);       // bit 1: no emission records to look for
        krp_k_sort_count<<<pers, 256, 0, st>>>(g->m, g->d_ctl, g->ev, g->sort_geom, g->sub_bits, sflags, g->d_bins);
        CK(cub::DeviceScan::ExclusiveSum(g->d_scan, g->scan_bytes, g->d_bins, g->d_bins, (int)(g->n_bins + 1), st));
        krp_k_image_prep<<<1, 1, 0, st>>>(g->d_ctl, g->d_bins, g->n_bins);
        krp_k_sort_scatter<<<pers, 256, 0, st>>>(g->m, g->d_ctl, g->ev, g->sort_geom, g->sub_bits, sflags, g->d_bins, g->d_perm);
        g->launches += 5;   // count, scan (2 kernels), prep, scatter
    } else {
        krp_k_image_prep_plain<<<1, 1, 0, st>>>(g->d_ctl);
        g->launches++;
    } }
    // I1-I3: one launch per observer (its constants are kernel parameters); launches rotate over
    // KRP_MAX_OBS_PACK work counters, rewound when the rotation wraps
    const int tb = g->image_block;
    const size_t smem = g->m.scalar ? 0 : 2 * sizeof(float4) * (size_t)(g->m.n_inc - 1);
    for (int o = 0; o < n_obs; ++o) {
        const int slot = o % KRP_MAX_OBS_PACK;
        if (o > 0 && slot == 0) { krp_k_image_rewind<<<1, 1, 0, st>>>(g->d_ctl); g->launches++; }
        TimedLaunch tli(g, st, KRP_T_IMAGE);
        const bool zt = g->m.z.zt != nullptr;
        float4* oc = g->d_obs_cells ? g->d_obs_cells + (size_t)o * g->npad : nullptr;
#define KRP_IMG_ARGS g->m, g->d_ctl, g->ev, perm, g->obs_dev[o], oc, slot, o, npix_x, npix_y, flags, g->d_img
        if (g->m.scalar)          krp_k_image<true, false, false><<<pers, tb, 0, st>>>(KRP_IMG_ARGS);
        else if (oc && !zt)       krp_k_image<false, true, false><<<pers, tb, 0, st>>>(KRP_IMG_ARGS);
        else if (oc)              krp_k_image<false, true, true><<<pers, tb, 0, st>>>(KRP_IMG_ARGS);
        else if (!zt)             krp_k_image<false, false, false><<<pers, tb, smem, st>>>(KRP_IMG_ARGS);
        else                      krp_k_image<false, false, true><<<pers, tb, smem, st>>>(KRP_IMG_ARGS);
#undef KRP_IMG_ARGS
        g->launches++;
    }
    krp_k_events_clear<<<1, 1, 0, st>>>(g->d_ctl);
    g->ev_has_emission = 0;
    g->launches++;
    CK(cudaGetLastError());
    // counters of this pass for the ordering decision of a later one (never waited for)
    if (g->order_policy == 1 && !g->order_decided && !g->ray_stats_pending) {
        if (!g->h_ray_stats) {
            CK(cudaMallocHost(&g->h_ray_stats, 3 * sizeof(unsigned long long)));
            g->h_ray_stats[0] = g->h_ray_stats[1] = g->h_ray_stats[2] = 0;
            CK(cudaEventCreateWithFlags(&g->ray_stats_ev, cudaEventDisableTiming));
        }
        // steps_image, contributions, dropped are consecutive in KrpStatsDev
        CK(cudaMemcpyAsync(g->h_ray_stats, &g->d_ctl->stats.steps_image, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
        CK(cudaEventRecord(g->ray_stats_ev, st));
        g->ray_stats_pending = true;
        g->req_pn = g->acc_pn;
    }
    return KRP_OK;
}

// every synchronising call reports a past overflow of the event buffer, not only krp_stats_get
static int overflow_code(krp_grid* g, const KrpCtl& c)
{
    if (c.stats.overflow)
        return fail(KRP_ERR_EVENT_FULL, "event buffer overflowed: %llu events lost (capacity %llu)",
                    (unsigned long long)c.stats.overflow, (unsigned long long)g->ev_cap);
    return KRP_OK;
}

extern "C" int krp_image_get(krp_grid* g, double* out, int mem, void* stream)
{
    if (!g || !out) return fail(KRP_ERR_ARG, "grid or out is NULL");
    if (!g->d_img) return fail(KRP_ERR_STATE, "krp_image has not been called");
    cudaStream_t st = (cudaStream_t)stream;
    size_t bytes = sizeof(double) * 4 * (size_t)g->n_obs * g->npx * g->npy;
    if (mem == KRP_MEM_HOST) {
        CK(cudaMemcpyAsync(out, g->d_img, bytes, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        KrpCtl c;      // a synchronising call: report a past overflow (the maps are delivered all the same)
        CK(cudaMemcpy(&c, g->d_ctl, sizeof(c), cudaMemcpyDeviceToHost));
        return overflow_code(g, c);
    } else if (mem == KRP_MEM_DEVICE) {
        CK(cudaMemcpyAsync(out, g->d_img, bytes, cudaMemcpyDeviceToDevice, st));
    } else {
        return fail(KRP_ERR_ARG, "mem must be KRP_MEM_DEVICE or KRP_MEM_HOST");
    }
    return KRP_OK;
}

extern "C" int krp_image_reset(krp_grid* g, void* stream)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    if (!g->d_img) return KRP_OK;
    size_t bytes = sizeof(double) * 4 * (size_t)g->n_obs * g->npx * g->npy;
    CK(cudaMemsetAsync(g->d_img, 0, bytes, (cudaStream_t)stream));
    return KRP_OK;
}

extern "C" int krp_stats_get(krp_grid* g, krp_stats* out)
{
    if (!g || !out) return fail(KRP_ERR_ARG, "grid or out is NULL");
    CK(cudaDeviceSynchronize());
    KrpCtl c;
    CK(cudaMemcpy(&c, g->d_ctl, sizeof(c), cudaMemcpyDeviceToHost));
    out->packets = c.stats.packets; out->events = c.stats.events; out->records = c.stats.records;
    out->steps_transport = c.stats.steps_transport; out->steps_image = c.stats.steps_image;
    out->contributions = c.stats.contributions; out->dropped = c.stats.dropped; out->overflow = c.stats.overflow;
    out->segments = c.sg_segments;
    out->w_emitted = c.stats.w_emitted; out->w_escaped = c.stats.w_escaped;
    out->w_absorbed = c.stats.w_absorbed; out->w_cut = c.stats.w_cut;
    return overflow_code(g, c);
}

extern "C" int krp_stats_reset(krp_grid* g, void* stream)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    CK(cudaMemsetAsync(&g->d_ctl->stats, 0, sizeof(KrpStatsDev), (cudaStream_t)stream));
    CK(cudaMemsetAsync(&g->d_ctl->sg_segments, 0, sizeof(unsigned long long), (cudaStream_t)stream));
    return KRP_OK;
}

// krp_events_get / krp_events_select: download the buffer in slices of 2^22 events and keep those whose packet id
// lies in [id_first, id_first + id_count)
static int events_download(krp_grid* g, uint64_t id_first, uint64_t id_count, uint64_t cap, uint64_t* n, uint64_t* id, int32_t* k,
                           int64_t* cell, float* pos, float* dir, float* stokes)
{
    CK(cudaDeviceSynchronize());
    KrpCtl c;
    CK(cudaMemcpy(&c, g->d_ctl, sizeof(c), cudaMemcpyDeviceToHost));
    const uint64_t have = c.n_events < g->ev_cap ? c.n_events : g->ev_cap;
    const bool all = id_count == UINT64_MAX;
    const uint64_t slice = 1ull << 22;
    std::vector<float4> pc, nk, S;
    std::vector<unsigned long long> ids;
    uint64_t found = 0;
    for (uint64_t e0 = 0; e0 < have; e0 += slice) {
        const uint64_t m = have - e0 < slice ? have - e0 : slice;
        ids.resize(m);
        CK(cudaMemcpy(ids.data(), g->ev.id + e0, m * sizeof(unsigned long long), cudaMemcpyDeviceToHost));
        if (cap == 0) {      // count only
            if (all) found += m;
            else for (uint64_t i = 0; i < m; ++i) found += (ids[i] - id_first < id_count) ? 1 : 0;
            continue;
        }
        pc.resize(m); nk.resize(m); S.resize(m);
        CK(cudaMemcpy(pc.data(), g->ev.pc + e0, m * sizeof(float4), cudaMemcpyDeviceToHost));
        CK(cudaMemcpy(nk.data(), g->ev.nk + e0, m * sizeof(float4), cudaMemcpyDeviceToHost));
        CK(cudaMemcpy(S.data(), g->ev.S + e0, m * sizeof(float4), cudaMemcpyDeviceToHost));
        for (uint64_t i = 0; i < m; ++i) {
            if (!all && !(ids[i] - id_first < id_count)) continue;
            const uint64_t o = found++;
            if (o >= cap) continue;
            uint32_t cb, kb;
            memcpy(&cb, &pc[i].w, 4); memcpy(&kb, &nk[i].w, 4);
            if (id) id[o] = ids[i];
            if (k) k[o] = (int32_t)(kb & ~KRP_TERM_BIT);
            if (cell) {
                const KrpModel& mm = g->m;
                uint32_t t = cb / (uint32_t)mm.px, hx = cb - t * (uint32_t)mm.px, hz = t / (uint32_t)mm.py, hy = t - hz * (uint32_t)mm.py;
                cell[o] = ((int64_t)(hz - 1) * mm.ny + (int64_t)(hy - 1)) * mm.nx + (int64_t)(hx - 1);
            }
            if (pos) { pos[3 * o] = pc[i].x; pos[3 * o + 1] = pc[i].y; pos[3 * o + 2] = pc[i].z; }
            if (dir) { dir[3 * o] = nk[i].x; dir[3 * o + 1] = nk[i].y; dir[3 * o + 2] = nk[i].z; }
            if (stokes) {
                stokes[4 * o] = S[i].x; stokes[4 * o + 1] = S[i].x * S[i].y;
                stokes[4 * o + 2] = S[i].x * S[i].z; stokes[4 * o + 3] = S[i].x * S[i].w;
            }
        }
    }
    *n = found;
    return overflow_code(g, c);
}

extern "C" int krp_events_get(krp_grid* g, uint64_t cap, uint64_t* n, uint64_t* id, int32_t* k, int64_t* cell, float* pos,
                              float* dir, float* stokes)
{
    if (!g || !n) return fail(KRP_ERR_ARG, "grid or n is NULL");
    return events_download(g, 0, UINT64_MAX, cap, n, id, k, cell, pos, dir, stokes);
}

extern "C" int krp_events_select(krp_grid* g, uint64_t id_first, uint64_t id_count, uint64_t cap, uint64_t* n, uint64_t* id,
                                 int32_t* k, int64_t* cell, float* pos, float* dir, float* stokes)
{
    if (!g || !n) return fail(KRP_ERR_ARG, "grid or n is NULL");
    if (id_count == UINT64_MAX) return fail(KRP_ERR_ARG, "id_count must be below 2^64-1");
    return events_download(g, id_first, id_count, cap, n, id, k, cell, pos, dir, stokes);
}

extern "C" int krp_events_clear(krp_grid* g, void* stream)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    krp_k_events_clear<<<1, 1, 0, (cudaStream_t)stream>>>(g->d_ctl);
    g->ev_has_emission = 0;
    g->launches++;
    CK(cudaGetLastError());
    return KRP_OK;
}

extern "C" int krp_tune(krp_grid* g, int transport_block, int image_block, int blocks_per_sm, int flight_burst)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    auto okb = [](int b) { return b == 0 || (b >= 32 && b <= 256 && b % 32 == 0); };
    if (!okb(transport_block) || !okb(image_block)) return fail(KRP_ERR_ARG, "block sizes must be multiples of 32 in 32..256");
    if (blocks_per_sm < 0 || blocks_per_sm > 64) return fail(KRP_ERR_ARG, "blocks_per_sm must be in 0..64");
    if (transport_block) g->transport_block = transport_block;
    if (image_block) g->image_block = image_block;
    if (blocks_per_sm) { g->blocks_per_sm = blocks_per_sm; g->bps_tuned = 1; }
    if (flight_burst < 0 || flight_burst > 4096) return fail(KRP_ERR_ARG, "flight_burst must be in 0..4096");
    if (flight_burst) { g->burst = flight_burst; g->burst_auto = false; }
    return KRP_OK;
}

extern "C" int krp_tune_fused(krp_grid* g, long long max_packets)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    if (max_packets < 0) return fail(KRP_ERR_ARG, "max_packets must be >= 0");
    g->fused_max = max_packets;
    return KRP_OK;
}

extern "C" int krp_tune_schedule(krp_grid* g, int dir_sort, int obs_cells, int order_policy)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    if (dir_sort < -1 || dir_sort > 1 || obs_cells < -1 || obs_cells > 1 || order_policy < -1 || order_policy > 2)
        return fail(KRP_ERR_ARG, "dir_sort, obs_cells must be -1, 0 or 1 and order_policy -1..2");
    if (dir_sort >= 0) g->dir_sort = dir_sort;
    if (obs_cells >= 0 && obs_cells != g->obs_pre) { g->obs_pre = obs_cells; g->obs_host.clear(); }   // rebuilt at the next krp_image
    if (order_policy >= 0) { g->order_policy = order_policy; g->order_events = order_policy != 0; g->ray_stats_pending = false; g->order_decided = false; }
    return KRP_OK;
}

// ------------------------------------------------------------------------------------------
// the paper's two-step form (include/krp.h)
// ------------------------------------------------------------------------------------------
extern "C" int krp_sgrid_end(krp_grid* g)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    CK(cudaDeviceSynchronize());
    cudaFree(g->d_sgrid); g->d_sgrid = nullptr;
    cudaFree(g->d_sg_obs); g->d_sg_obs = nullptr;
    g->sg_n_obs = 0; g->sg_obs_host.clear();
    return KRP_OK;
}

extern "C" int krp_sgrid_begin(krp_grid* g, const krp_observer* obs, int n_obs, void* stream)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    int rc = check_observers(obs, n_obs, 1, 1);
    if (rc) return rc;
    if (n_obs > KRP_SG_MAX_OBS) return fail(KRP_ERR_ARG, "a source grid holds at most %d cameras", KRP_SG_MAX_OBS);
    if (g->m.periodic) return fail(KRP_ERR_STATE, "a source grid cannot be opened on a model with periodic boundaries");
    if (g->m.z.zt) return fail(KRP_ERR_STATE, "a source grid cannot be opened while a full Z table is set");
    cudaStream_t st = (cudaStream_t)stream;
    rc = krp_sgrid_end(g);
    if (rc) return rc;
    const size_t bytes = sizeof(float) * 4 * (size_t)g->npad * (size_t)n_obs;
    if (cudaMalloc(&g->d_sgrid, bytes) != cudaSuccess) {
        cudaGetLastError(); g->d_sgrid = nullptr;
        return fail(KRP_ERR_OOM, "source grid of %zu bytes does not fit", bytes);
    }
    CK(cudaMemsetAsync(g->d_sgrid, 0, bytes, st));
    std::vector<KrpObserverDev> od(n_obs);
    for (int o = 0; o < n_obs; ++o) od[o] = make_observer_dev(g, obs[o]);
    CK(cudaMalloc(&g->d_sg_obs, sizeof(KrpObserverDev) * n_obs));
    CK(cudaMemcpyAsync(g->d_sg_obs, od.data(), sizeof(KrpObserverDev) * n_obs, cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));
    g->sg_n_obs = n_obs;
    g->sg_obs_host.assign(obs, obs + n_obs);
    const int smem_d = n_obs * 2 * 128 * (int)sizeof(float4);
    CK(cudaFuncSetAttribute(krp_k_deposit<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_d));
    CK(cudaFuncSetAttribute(krp_k_deposit<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_d));
    return KRP_OK;
}

extern "C" int krp_sgrid_reset(krp_grid* g, void* stream)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    if (!g->d_sgrid) return fail(KRP_ERR_STATE, "no source grid is open");
    CK(cudaMemsetAsync(g->d_sgrid, 0, sizeof(float) * 4 * (size_t)g->npad * (size_t)g->sg_n_obs, (cudaStream_t)stream));
    return KRP_OK;
}

extern "C" int krp_sgrid_get(krp_grid* g, float* out, int mem, void* stream)
{
    if (!g || !out) return fail(KRP_ERR_ARG, "grid or out is NULL");
    if (!g->d_sgrid) return fail(KRP_ERR_STATE, "no source grid is open");
    if (mem != KRP_MEM_DEVICE && mem != KRP_MEM_HOST) return fail(KRP_ERR_ARG, "mem must be KRP_MEM_DEVICE or KRP_MEM_HOST");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n4 = (size_t)g->m.ncell * (size_t)g->sg_n_obs;
    float4* tmp = nullptr;
    float4* dst = (float4*)out;
    if (mem == KRP_MEM_HOST) { CK(cudaMalloc(&tmp, sizeof(float4) * n4)); dst = tmp; }
    krp_k_sgrid_unpad<<<(unsigned)((n4 + 255) / 256), 256, 0, st>>>(g->m, (const float4*)g->d_sgrid, g->sg_n_obs, dst);
    g->launches++;
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && mem == KRP_MEM_HOST) {
        e = cudaMemcpyAsync(out, tmp, sizeof(float4) * n4, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    }
    cudaFree(tmp);
    if (e != cudaSuccess) return fail(KRP_ERR_CUDA, "krp_sgrid_get: %s", cudaGetErrorString(e));
    return KRP_OK;
}

extern "C" int krp_image_rays(krp_grid* g, const krp_observer* obs, int n_obs, int npix_x, int npix_y, const float* emis, int mem,
                              void* stream)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    int rc = check_observers(obs, n_obs, npix_x, npix_y);
    if (rc) return rc;
    if (!g->d_sgrid && !emis) return fail(KRP_ERR_STATE, "krp_image_rays needs an open source grid or a thermal source");
    if (emis && mem != KRP_MEM_DEVICE && mem != KRP_MEM_HOST) return fail(KRP_ERR_ARG, "mem must be KRP_MEM_DEVICE or KRP_MEM_HOST");
    if (g->d_sgrid && (n_obs != g->sg_n_obs || memcmp(g->sg_obs_host.data(), obs, sizeof(krp_observer) * n_obs) != 0))
        return fail(KRP_ERR_ARG, "the observers must be the cameras of the open source grid");
    if ((size_t)npix_x * npix_y >= (1ull << 31)) return fail(KRP_ERR_ARG, "too many pixels");
    cudaStream_t st = (cudaStream_t)stream;
    rc = setup_maps(g, obs, n_obs, npix_x, npix_y, st, false);
    if (rc) return rc;
    const float* d_em = nullptr;
    if (emis) {
        // the caller's [nz][ny][nx] array into the padded order of the cells
        if (!g->d_emis) CK(cudaMalloc(&g->d_emis, sizeof(float) * (size_t)g->npad));
        const float* src = emis;
        float* stage = nullptr;
        if (mem == KRP_MEM_HOST) {
            CK(cudaMalloc(&stage, sizeof(float) * (size_t)g->m.ncell));
            CK(cudaMemcpyAsync(stage, emis, sizeof(float) * (size_t)g->m.ncell, cudaMemcpyHostToDevice, st));
            src = stage;
        }
        krp_k_pad_scalar<<<(unsigned)((g->npad + 255u) / 256u), 256, 0, st>>>(g->m, src, g->npad, g->d_emis);
        g->launches++;
        if (stage) { CK(cudaStreamSynchronize(st)); cudaFree(stage); }
        d_em = g->d_emis;
    }
    const int npix = npix_x * npix_y;
    for (int o = 0; o < n_obs; ++o) {
        KrpRayObs ro;
        const double st_ = std::sin(obs[o].theta), ct_ = std::cos(obs[o].theta);
        const double n[3] = { st_ * std::cos(obs[o].phi), st_ * std::sin(obs[o].phi), ct_ };
        double th[3], ph[3];
        host_basis(n, th, ph);
        for (int a = 0; a < 3; ++a) { ro.n[a] = n[a]; ro.th[a] = th[a]; ro.ph[a] = ph[a]; ro.center[a] = obs[o].center[a]; }
        ro.half_w = obs[o].half_w; ro.half_h = obs[o].half_h;
        TimedLaunch tl(g, st, KRP_T_RAYS);
        if (g->m.scalar) krp_k_image_rays<true><<<(npix + 127) / 128, 128, 0, st>>>(g->m, g->d_ctl, ro, o, n_obs, npix_x, npix_y, g->d_sgrid, d_em, g->d_img);
        else             krp_k_image_rays<false><<<(npix + 127) / 128, 128, 0, st>>>(g->m, g->d_ctl, ro, o, n_obs, npix_x, npix_y, g->d_sgrid, d_em, g->d_img);
        g->launches++;
    }
    CK(cudaGetLastError());
    return KRP_OK;
}

// ------------------------------------------------------------------------------------------
// frequency bins (include/krp.h)
// ------------------------------------------------------------------------------------------
static int apply_scale(krp_grid* g, float k, cudaStream_t st)
{
    if (k == g->cur_scale) return KRP_OK;
    const unsigned nb = (unsigned)((g->npad + 255u) / 256u);
    if (!g->d_base) {
        CK(cudaMalloc(&g->d_base, sizeof(float) * (size_t)g->npad));
        krp_k_save_base<<<nb, 256, 0, st>>>(g->npad, g->d_kr, g->d_cell, g->d_base);
        g->launches++;
    }
    krp_k_rescale<<<nb, 256, 0, st>>>(g->npad, g->d_base, k, g->d_kr, g->d_cell);
    g->launches++;
    CK(cudaGetLastError());
    g->cur_scale = k;
    g->obs_cells_stale = true;
    return KRP_OK;
}

extern "C" int krp_freq_select(krp_grid* g, int bin, void* stream)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    if (bin < 0 || bin >= (int)g->bins.size()) return fail(KRP_ERR_ARG, "bin must be in 0..%d", (int)g->bins.size() - 1);
    cudaStream_t st = (cudaStream_t)stream;
    if (bin == g->cur_bin) return KRP_OK;
    CK(cudaStreamSynchronize(st));
    KrpCtl c;
    CK(cudaMemcpy(&c, g->d_ctl, sizeof(c), cudaMemcpyDeviceToHost));
    if (c.n_events != 0) return fail(KRP_ERR_STATE, "image (or clear) the buffered events before selecting another frequency bin");
    // an open source grid holds the deposits of the current bin's opacities: mixing bins in it would be silent nonsense
    if (g->d_sgrid) return fail(KRP_ERR_STATE, "close the source grid (krp_sgrid_end) before selecting another frequency bin");
    g->bins[g->cur_bin].d_img = g->d_img;            // park the maps of the bin we leave
    double* img = g->bins[bin].d_img;
    if (!img && g->d_img) {                           // same observer set and size for every bin
        const size_t bytes = sizeof(double) * 4 * (size_t)g->n_obs * g->npx * g->npy;
        CK(cudaMalloc(&img, bytes));
        CK(cudaMemsetAsync(img, 0, bytes, st));
    }
    g->d_img = img;
    g->bins[bin].d_img = nullptr;                     // owned through g->d_img while current
    apply_tables(g, bin);
    return apply_scale(g, g->bins[bin].kscale, st);
}

extern "C" int krp_freq_define(krp_grid* g, int n_freq, const krp_tables* tables, const float* kappa_scale, void* stream)
{
    if (!g || !tables || !kappa_scale) return fail(KRP_ERR_ARG, "grid, tables or kappa_scale is NULL");
    if (n_freq < 1 || n_freq > 4096) return fail(KRP_ERR_ARG, "n_freq must be in 1..4096");
    cudaStream_t st = (cudaStream_t)stream;
    for (int b = 0; b < n_freq; ++b) {
        int rc = check_tables(tables + b);
        if (rc) return rc;
        if (!(kappa_scale[b] > 0.f) || !std::isfinite(kappa_scale[b])) return fail(KRP_ERR_ARG, "kappa_scale[%d] must be positive and finite", b);
    }
    CK(cudaStreamSynchronize(st));
    KrpCtl c;
    CK(cudaMemcpy(&c, g->d_ctl, sizeof(c), cudaMemcpyDeviceToHost));
    if (c.n_events != 0) return fail(KRP_ERR_STATE, "krp_freq_define with a non-empty event buffer");
    std::vector<TableSet> nb(n_freq);
    for (int b = 0; b < n_freq; ++b) {
        int rc = build_tables(tables + b, nb[b], st);
        if (!rc && g->m.scalar && !(nb[b].constant && !nb[b].dichroic))
            rc = fail(KRP_ERR_ARG, "bin %d needs the 16-byte cell layout: create the model with a field or a direction-dependent table", b);
        if (rc) { for (TableSet& t : nb) free_tables(t); return rc; }
        nb[b].kscale = kappa_scale[b];
    }
    // the maps of the old bins go; those of the current one are g->d_img
    cudaFree(g->d_img); g->d_img = nullptr; g->obs_host.clear();
    g->bins[g->cur_bin].d_img = nullptr;
    for (TableSet& t : g->bins) free_tables(t);
    g->bins.swap(nb);
    apply_tables(g, 0);
    return apply_scale(g, g->bins[0].kscale, st);
}

// ------------------------------------------------------------------------------------------
// full scattering matrix of aligned grains (include/krp.h)
// ------------------------------------------------------------------------------------------
extern "C" int krp_zmatrix_set(krp_grid* g, int n_ti, int n_to, int n_dp, const float* Z, void* stream)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaStreamSynchronize(st));
    cudaFree(g->d_zt); cudaFree(g->d_zt_norm); cudaFree(g->d_zt_bound);
    g->d_zt = nullptr; g->d_zt_norm = nullptr; g->d_zt_bound = nullptr;
    g->m.z = KrpZt{ nullptr, nullptr, nullptr, 0, 0, 0 };
    if (!Z) return KRP_OK;
    if (g->m.scalar) return fail(KRP_ERR_ARG, "a Z table needs the 16-byte cell layout: create the model with a field or a direction-dependent table");
    if (g->d_sgrid) return fail(KRP_ERR_STATE, "close the source grid before setting a Z table");
    if (n_ti < 2 || n_to < 2 || n_dp < 2 || (uint64_t)n_ti * n_to * n_dp > (1ull << 26)) return fail(KRP_ERR_ARG, "Z table: need n_ti, n_to, n_dp >= 2 and at most 2^26 nodes");
    const size_t nn = (size_t)n_ti * n_to * n_dp;
    std::vector<double> norm(4 * (size_t)n_ti, 0.0), bound(n_ti, 0.0);
    // per incidence node: (1/4pi) integral over outgoing directions of row 1 (trapezoid in vartheta_out with sin, mean over dphi),
    // and the bound of the rejection sampler max(Z11 + |(Z12, Z13, Z14)|)
    const double dth = KRP_PI_D / (n_to - 1);
    for (int i = 0; i < n_ti; ++i)
        for (int o = 0; o < n_to; ++o) {
            const double w = (o == 0 || o == n_to - 1 ? 0.5 : 1.0) * std::sin(o * dth) * dth * 0.5;
            for (int d = 0; d < n_dp; ++d) {
                const float* e = Z + (((size_t)i * n_to + o) * n_dp + d) * 16;
                for (int k = 0; k < 16; ++k) if (!std::isfinite(e[k])) return fail(KRP_ERR_ARG, "Z table: entry is not finite");
                if (!(e[0] > 0.f)) return fail(KRP_ERR_ARG, "Z table: Z11 must be positive (node %d,%d,%d)", i, o, d);
                for (int s = 0; s < 4; ++s) norm[4 * i + s] += w * (double)e[s] / n_dp;
                const double b = (double)e[0] + std::sqrt((double)e[1] * e[1] + (double)e[2] * e[2] + (double)e[3] * e[3]);
                if (b > bound[i]) bound[i] = b;
            }
        }
    CK(cudaMalloc(&g->d_zt, sizeof(float) * 16 * nn));
    CK(cudaMalloc(&g->d_zt_norm, sizeof(double) * 4 * n_ti));
    CK(cudaMalloc(&g->d_zt_bound, sizeof(double) * n_ti));
    CK(cudaMemcpyAsync(g->d_zt, Z, sizeof(float) * 16 * nn, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(g->d_zt_norm, norm.data(), sizeof(double) * 4 * n_ti, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(g->d_zt_bound, bound.data(), sizeof(double) * n_ti, cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));
    g->m.z = KrpZt{ g->d_zt, g->d_zt_norm, g->d_zt_bound, n_ti, n_to, n_dp };
    return KRP_OK;
}

extern "C" int krp_timing_enable(krp_grid* g, int on)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    g->timing = on != 0;
    if (!g->timing) g->t_cls.clear();
    return KRP_OK;
}

extern "C" int krp_timing_get(krp_grid* g, double* ms, uint64_t* launches)
{
    if (!g) return fail(KRP_ERR_ARG, "grid is NULL");
    CK(cudaDeviceSynchronize());
    double acc[KRP_T_COUNT] = { 0 };
    uint64_t cnt[KRP_T_COUNT] = { 0 };
    for (size_t k = 0; k < g->t_cls.size(); ++k) {
        float t = 0.f;
        CK(cudaEventElapsedTime(&t, g->t_ev[2 * k], g->t_ev[2 * k + 1]));
        acc[g->t_cls[k]] += (double)t; cnt[g->t_cls[k]]++;
    }
    g->t_cls.clear();
    for (int c = 0; c < KRP_T_COUNT; ++c) { if (ms) ms[c] = acc[c]; if (launches) launches[c] = cnt[c]; }
    return KRP_OK;
}

extern "C" uint64_t krp_launch_count(const krp_grid* g) { return g ? g->launches : 0; }

#include "krp_noalloc.cuh"
