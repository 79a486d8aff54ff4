/*
 * krp.h -- C ABI of the B200-native polarized Monte-Carlo radiative-transfer hot path
 * (Kratos-polrad, arxiv 2512.01283; citations are PAPER.md:<line> of the extracted paper
 * text, "R<n>" are the readings listed in DESIGN.md).
 *
 * The library computes, on one GPU and entirely in its own CUDA kernels:
 *   transport  photon packets through a uniform Cartesian grid (cell interface to cell
 *              interface) with Stokes-dependent extinction solved analytically
 *              inside each cell (App. A), scattering in the grain frame
 *              reached through the quaternion q_B (eq. 1-7) with angles
 *              sampled from the tabulated Mueller matrix;
 *   imaging    the second step of the two-step scheme (eq. 10-11): every
 *              recorded scattering event sends its Stokes vector toward every observer and
 *              is attenuated cell by cell to the grid edge, then summed into I,Q,U,V maps.
 *
 * Conventions
 *   - every function returns KRP_OK (0) or a negative error code; it never throws or exits.
 *     krp_last_error() gives a thread-local message for the last failing call.
 *   - "DEVICE" pointers are CUDA device pointers valid on the current device, "HOST" pointers
 *     are ordinary host memory.  The library copies what it needs: the caller keeps
 *     ownership of every array it passes and may free it once the call's stream work is done
 *     (for HOST inputs: as soon as the call returns).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All
 *     work is enqueued on it; only the calls marked "synchronises" wait for the device.
 *   - arrays over cells are [nz][ny][nx] (x fastest).
 *   - one krp_grid may be used from one host thread at a time.
 */
#ifndef KRP_H_
#define KRP_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    KRP_OK = 0,
    KRP_ERR_ARG = -1,        /* invalid argument (message says which) */
    KRP_ERR_CUDA = -2,       /* a CUDA runtime call failed */
    KRP_ERR_OOM = -3,        /* device allocation failed */
    KRP_ERR_STATE = -4,      /* call made in the wrong order (e.g. image_get before image) */
    KRP_ERR_EVENT_FULL = -5  /* the event buffer overflowed; see krp_stats.overflow */
};

enum { KRP_MEM_DEVICE = 0, KRP_MEM_HOST = 1 };

const char* krp_last_error(void);
/* library identification: "krp <version> sm_100a <build id>", the build id being a hash of the sources the library
 * was compiled from (the binding refuses a library whose id differs from the sources beside it) */
const char* krp_version(void);

typedef struct krp_grid krp_grid; /* opaque; owns all device memory of one model */

/* Lookup tables ("interpolation tables"; R8, R13).  HOST pointers, copied.
 *   mueller  [n_ang][4] = S11,S12,S33,S34 on Theta_j = j*180/(n_ang-1) degrees, n_ang >= 2,
 *            S11 > 0 and S11^2 >= S12^2+S33^2+S34^2 on every node; S11 need not be normalised
 *            for sampling, but image units assume (1/2) int S11 sin(Theta) dTheta = 1.
 *   opacity  [n_inc][4] = alpha1, alpha2, alpha3, albedo on mu_m = m/(n_inc-1),
 *            mu = |cos(angle between n^ and B^)|, n_inc >= 1 (n_inc = 1: constant);
 *            alpha1 > |alpha2|, 0 <= albedo <= 1.  The alphas are the elements of the App. A
 *            matrix (R1) per unit of density*length.
 *   w_min, max_scatter   a packet stops after a scattering that leaves its weight below
 *            w_min or after max_scatter scatterings (R12; deterministic, no roulette). */
typedef struct krp_tables {
    int n_ang;
    const float* mueller;
    int n_inc;
    const float* opacity;
    float w_min;
    int max_scatter;
    int periodic;     /* bit a set: axis a (0 x, 1 y, 2 z) is periodic (reading R20): packets and imaging rays
                         that leave through a face of that axis re-enter through the opposite face; after 4096 such crossings a
                         ray counts as having left the grid.  A periodic model uses the 16-byte cell layout.  A source grid
                         (krp_sgrid_begin) cannot be opened on a periodic model (KRP_ERR_STATE). */
} krp_tables;

/* Build a model.  bounds = xlo,xhi,ylo,yhi,zlo,zhi (HOST).  density [nz][ny][nx] >= 0 is
 * kappa*rho per unit length (PAPER.md:101 lambda_ext^-1).  bfield [nz][ny][nx][3], any
 * norm, zero vector = unaligned cell (B^ = z^), may be NULL (B^ = z^ everywhere).
 * `mem` says where density/bfield live (KRP_MEM_DEVICE or KRP_MEM_HOST).  Cells are packed
 * into the library's own layout here (not timed as part of the hot path).
 * Errors: KRP_ERR_ARG for non-positive dims, non-increasing bounds, bad tables. */
int krp_grid_create(krp_grid** out, int nx, int ny, int nz, const double bounds[6],
                    const float* density, const float* bfield, int mem,
                    const krp_tables* tables, void* stream);
int krp_grid_destroy(krp_grid* g);

/* Replace the density (and field) of an existing model, e.g. the next snapshot of the simulation the dust
 * belongs to (the method runs inside a hydrodynamics code): same dimensions, bounds and tables,
 * arrays laid out as for krp_grid_create, bfield non-NULL exactly when the model was created with one.
 * Re-packs the cells without re-allocating anything; buffered events and image maps are left as they are.
 * Synchronises (it reports bad densities).  Errors as krp_grid_create. */
int krp_grid_update(krp_grid* g, const float* density, const float* bfield, int mem, void* stream);
/* The same for HOST snapshots, in two halves, so that the host-to-device copy of the NEXT snapshot runs while the current one
 * is still being transported and imaged: krp_grid_stage starts the copy of density/bfield (host arrays; pinned memory makes it
 * asynchronous) into the model's staging buffers on `copy_stream` and returns at once; krp_grid_update_staged makes `stream`
 * wait for that copy, re-packs the cells from it (after whatever `stream` still runs on the old cells) and synchronises like
 * krp_grid_update.  One snapshot can be staged at a time: stage the next one only after the last krp_grid_update /
 * krp_grid_update_staged has returned; a krp_grid_update with KRP_MEM_HOST in between overwrites a staged snapshot.
 * Errors: KRP_ERR_ARG as krp_grid_update; KRP_ERR_STATE from krp_grid_update_staged when nothing is staged. */
int krp_grid_stage(krp_grid* g, const float* density, const float* bfield, void* copy_stream);
int krp_grid_update_staged(krp_grid* g, void* stream);

/* Source of packets (PAPER.md:107 emission; R17).
 *   kind bit0: 0 = all packets start at pos (a pos outside the box is moved to the nearest point of the box, coordinate by
 *              coordinate: reading R24), 1 = start uniformly inside a cell drawn with
 *              probability proportional to cell_weight (DEVICE, [ncell]; NULL = uniform);
 *   kind bit1: 0 = isotropic directions, 1 = all along dir (need not be normalised).
 *   kind bit2 (only as kind = 5): thermal emission of the grains themselves (eq. 8, alpha_abs B; reading R22):
 *              positions as for bit0 (cell_weight = kappa*rho*B*V of the cell makes the cells emit in proportion), directions
 *              drawn with density (1 - albedo(mu)) alpha1(mu), mu = |n^ . B^| of the emitting cell, Stokes vector
 *              (1, alpha2/alpha1, 0, 0) in the grain-frame reference.  One packet then stands for L_tot / N with
 *              L_tot = 4 pi <(1 - albedo) alpha1>_mu sum(kappa*rho*B*V); the direct thermal light is krp_image_rays' `emis`.
 *              No emission records.  Set it again after krp_freq_select (it depends on the bin's table).
 *   emit_records != 0 also appends an "emission record" (event index k = 0) per packet so
 *   that krp_image(flags bit0) can add the direct, unscattered light.
 * Every packet starts unpolarised, Stokes (1,0,0,0), weight 1. */
typedef struct krp_source {
    int kind;
    double pos[3];
    double dir[3];
    const float* cell_weight;
    int emit_records;
} krp_source;
int krp_source_set(krp_grid* g, const krp_source* src, void* stream);

/* Capacity of the event buffer (events held between krp_transport and krp_image).
 * Optional: krp_transport grows it to 4 events per packet (at least 2^20) when unset.
 * Events beyond the capacity are dropped, the packet stops, krp_stats.overflow counts them, and from then on until
 * krp_stats_reset every call that reads results back to the host -- krp_stats_get, krp_events_get, krp_events_select,
 * krp_image_get to HOST memory -- delivers what it has and returns KRP_ERR_EVENT_FULL (krp_image itself does not
 * synchronise: it images the truncated buffer). */
int krp_events_reserve(krp_grid* g, uint64_t max_events);

/* Transport packets with global ids [next_id, next_id + n_packets) (next_id starts at 0 and
 * persists across calls; krp_packet_id_set changes it), Philox4x32-10 keyed by `seed` with the
 * counter schedule R11, so results do not depend on how the caller batches.  Appends one
 * record per scattering event: position, cell, incoming direction, albedo*weight and the
 * normalised Stokes state in the lab reference.  Does not synchronise (it does once, when a
 * larger batch than any before makes it grow its queues).  The order in which packets are processed and
 * events are appended is not defined (an isotropic point source is processed in direction order). */
int krp_transport(krp_grid* g, uint64_t n_packets, uint64_t seed, void* stream);
int krp_packet_id_set(krp_grid* g, uint64_t next_id);

/* Observer: direction toward the observer (theta, phi in radians, global spherical angles),
 * image plane centred on `center` with half extents half_w (along phi^_obs, image x) and
 * half_h (along -theta^_obs, image y); orthographic (R14). */
typedef struct krp_observer {
    double theta, phi;
    double center[3];
    double half_w, half_h;
} krp_observer;

/* Image every buffered event toward every observer (obs: HOST array) and add the result to
 * the internal fp64 maps [n_obs][4][npix_y][npix_x] (I,Q,U,V relative to theta^_obs, sum of
 * contributions per pixel, no area normalisation, R14).  flags bit0: include emission
 * records (direct light).  Clears the event buffer afterwards.  The maps are (re)allocated
 * and zeroed when the observer set or the pixel counts differ from the previous call; with a field
 * (16-byte cells) the call then also tabulates 16 bytes per cell and observer if that fits in device memory.
 * Does not synchronise except on such a change.  The order in which the events are imaged is not defined
 * (they are ordered by cell when the rays of earlier passes were long enough for that to pay). */
int krp_image(krp_grid* g, const krp_observer* obs, int n_obs, int npix_x, int npix_y,
              int flags, void* stream);
/* Copy the maps to out ([n_obs][4][npix_y][npix_x] doubles; `mem` = where out lives).
 * Synchronises when out is HOST memory. */
int krp_image_get(krp_grid* g, double* out, int mem, void* stream);
int krp_image_reset(krp_grid* g, void* stream);

/* ---- Imaging without any allocation (for callers that cannot reach cudaMalloc: code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it) --------------------------------------------------------------------------
 * The per-event imaging of PAPER.md:121 (peel-off, attenuation march with the in-cell solution of App. A, orthographic
 * projection; what krp_image does) for n events the CALLER holds, toward ONE observer, ADDED to the caller's map.
 *   k, cell, pos, dir, stokes   DEVICE arrays in the format of krp_events_get: event index (0 = emission record, imaged only
 *                               with flags bit0), linear cell index (x fastest), cell-local position [n][3], incoming
 *                               direction [n][3], albedo*weight*(1,q,u,v) [n][4] in the lab reference of dir;
 *   obs                         HOST, one observer;    img   DEVICE, [4][npix_y][npix_x] doubles, the caller zeroes it;
 *   rejected                    NULL, or HOST: receives the number of events that were left out (cell outside the grid,
 *                               negative k, non-finite values); asking for it makes the call synchronise.
 * The call makes no cudaMalloc, cudaFree or allocating library call and, with rejected = NULL, does not synchronise: it
 * launches two kernels and one memset on `stream`.  Its event records and control block live in one fixed device array
 * inside the library, KRP_NOALLOC_MAX_EVENTS events (12 MiB, held by every GPU that has loaded the library until the process
 * ends): n beyond that is KRP_ERR_ARG.  All calls on a device share that array: calls that overlap on the GPU (two streams,
 * two threads) race on it and must be serialised by the caller; nothing is carried from one call to the next.  The grid's
 * own event buffer, maps, krp_stats and timing classes are not touched.  General mode marches over the 16-byte cells
 * themselves (krp_image's per-observer coefficient arrays are an allocation) and the events are taken in the given order,
 * so maps equal krp_image's up to the rounding of the fp32 march.  The grid must have been created on the current device. */
#define KRP_NOALLOC_MAX_EVENTS 262144
int krp_image_events_noalloc(krp_grid* g, uint64_t n, const int32_t* k, const int64_t* cell, const float* pos,
                             const float* dir, const float* stokes, const krp_observer* obs, int npix_x, int npix_y,
                             int flags, double* img, uint64_t* rejected, void* stream);

/* ---- The paper's own two-step imaging (eq. 11) -------------------------------
 * Step 1: while a source grid is open, krp_transport also deposits, for every path segment of every flight (not only at
 * scattering events), the segment's expected scattered Stokes vector toward every camera,
 * S_pp = Z(Omega_cam; Omega_pp) I_pp (reading R18), into S(Omega_cam, x): fp32, [cell][camera][I,Q,U,V],
 * reference theta^_cam, including albedo, packet weight and the 1/(4 pi) of the phase matrix, not attenuated, not divided
 * by the cell volume.  The packets and their scattering events are exactly those of a run without a source grid.
 * Step 2: krp_image_rays marches ONE ray per pixel through the pixel centre from the far side of the grid toward the
 * camera and integrates eq. 8 cell by cell with the analytic in-cell solution INCLUDING source terms (App. A,
 * PAPER.md:296-328): the scattering source S / (V_cell kappa rho) of an open source grid and, when `emis` is given, the
 * thermal source alpha_abs B of eq. 8 with alpha_abs = (1 - albedo) alpha (reading R19) and B = emis[cell] (array
 * [nz][ny][nx], `mem` says where it lives; NULL = no thermal emission).  The result, radiance times pixel area (the unit
 * of krp_image's maps, R14), is ADDED to the maps krp_image_get returns.
 *   krp_sgrid_begin   opens (allocates and zeroes) the source grid for these cameras (n_obs <= 16); KRP_ERR_OOM if
 *                     16 bytes x cells x n_obs do not fit.  Synchronises.
 *   krp_sgrid_get     copies the grid to out ([nz][ny][nx][n_obs][4] floats), parity / debug.  Synchronises for HOST.
 *   krp_sgrid_reset   zeroes it;  krp_sgrid_end  closes it and frees its memory.
 *   krp_image_rays    obs must be the cameras of the open source grid (when one is open), else any cameras.
 * Errors: KRP_ERR_STATE without an open grid (get/reset) or with neither a grid nor emis (image_rays). */
int krp_sgrid_begin(krp_grid* g, const krp_observer* obs, int n_obs, void* stream);
int krp_sgrid_get(krp_grid* g, float* out, int mem, void* stream);
int krp_sgrid_reset(krp_grid* g, void* stream);
int krp_sgrid_end(krp_grid* g);
int krp_image_rays(krp_grid* g, const krp_observer* obs, int n_obs, int npix_x, int npix_y, const float* emis, int mem,
                   void* stream);

/* ---- Frequency bins ("For each frequency bin ... the transfer equation reads": eq. 8 holds per bin, the bins
 * do not exchange energy) -------------------------------------------------------------------------------------------
 * krp_freq_define gives the model n_freq bins, each with its own tables (tables[b], HOST, as for krp_grid_create; the
 * `periodic` field is ignored) and its own density factor: kappa*rho of bin b = kappa_scale[b] x the model's (the dust
 * is the same, its opacity per unit mass differs).  All bins use the cell layout chosen at krp_grid_create, so a model
 * whose first table was direction-independent and non-dichroic and that has no field accepts only such tables
 * (KRP_ERR_ARG otherwise).  krp_freq_select makes bin b the current one: krp_transport, krp_image, krp_image_rays,
 * krp_image_get and krp_image_reset then act on that bin (its tables, its density, its own maps; the observer set and
 * the pixel counts are common to all bins).  Buffered events belong to the bin they were transported in: image them before
 * selecting another bin (KRP_ERR_STATE if the buffer is not empty; it synchronises to check); an open source grid holds
 * deposits of the current bin only: close it first (KRP_ERR_STATE otherwise).  Bin 0 is current after
 * krp_freq_define.  A model without krp_freq_define has the single bin of krp_grid_create. */
int krp_freq_define(krp_grid* g, int n_freq, const krp_tables* tables, const float* kappa_scale, void* stream);
int krp_freq_select(krp_grid* g, int bin, void* stream);

/* ---- Full scattering matrix of aligned grains (eq. 10: "Z(Omega; Omega') depends on both the scattering angle
 * and the local magnetic field orientation"; :107-109, :129 rejection sampling, reading R21) ------------
 * Z (HOST, copied): [n_ti][n_to][n_dp][4][4] floats on the incidence angle vartheta_in = i 180/(n_ti-1) degrees, the outgoing
 * polar angle vartheta_out = o 180/(n_to-1) and the azimuth difference dphi = phi_out - phi_in = d 360/n_dp (periodic), all in the
 * Grain Frame (z_GF = B^ of the event cell, eq. 2-3); incoming and outgoing Stokes vectors are referenced to (theta^', phi^') of
 * their own direction in that frame (eq. 4-5).  Trilinear interpolation.  Z[..][0][0] > 0 and row 1 must keep the scattered
 * intensity positive for every physical Stokes vector.  With a Z table set, krp_transport samples the outgoing direction by
 * rejection against row 1 of Z . s and applies Z (instead of the Theta, phi sampling and F(Theta) of krp_tables.mueller), and
 * krp_image peels every event off with Z / (4 pi N), N the table's own integral of the scattered intensity.  The opacity table,
 * albedo and event location are unchanged.  Needs the 16-byte cell layout (a field or a direction-dependent table at
 * krp_grid_create; KRP_ERR_ARG otherwise) and no open source grid (KRP_ERR_STATE).  Z = NULL returns to F(Theta). */
int krp_zmatrix_set(krp_grid* g, int n_ti, int n_to, int n_dp, const float* Z, void* stream);

/* Counters (also the numerators of the roofline figures). */
typedef struct krp_stats {
    uint64_t packets;         /* packets emitted */
    uint64_t events;          /* scattering events recorded */
    uint64_t records;         /* emission records recorded */
    uint64_t steps_transport; /* cell steps taken by transport flights */
    uint64_t steps_image;     /* cell steps taken by imaging rays (a ray stops once its attenuation is 0 in fp32) */
    uint64_t contributions;   /* image contributions deposited */
    uint64_t dropped;         /* contributions that fell outside the frame */
    uint64_t overflow;        /* events lost to a full event buffer */
    uint64_t segments;        /* path segments deposited into an open source grid (two-step form) */
    double w_emitted, w_escaped, w_absorbed, w_cut;
} krp_stats;
int krp_stats_get(krp_grid* g, krp_stats* out);  /* synchronises */
int krp_stats_reset(krp_grid* g, void* stream);

/* Debug / parity: dump the buffered events (HOST arrays of capacity cap, any may be NULL).
 *   id[i], k[i]  packet id and event index (0 = emission record, k >= 1 = k-th scattering)
 *   cell[i]      linear cell index (x fastest)
 *   pos[i][3]    cell-local position in [0,1]^3
 *   dir[i][3]    incoming direction n^_in
 *   stokes[i][4] albedo*weight*(1,q,u,v), lab reference of n^_in
 * *n receives the number of buffered events (which may exceed cap; only min(*n,cap) are
 * written).  Order is not defined (the buffer is filled with atomics).  Synchronises. */
int krp_events_get(krp_grid* g, uint64_t cap, uint64_t* n, uint64_t* id, int32_t* k,
                   int64_t* cell, float* pos, float* dir, float* stokes);
/* The same for the events of packets id_first <= id < id_first + id_count only (a sample of a large batch: the parity
 * tests compare such a sample with the oracle); the buffer is read in slices, so host memory stays small. */
int krp_events_select(krp_grid* g, uint64_t id_first, uint64_t id_count, uint64_t cap, uint64_t* n, uint64_t* id, int32_t* k,
                      int64_t* cell, float* pos, float* dir, float* stokes);
int krp_events_clear(krp_grid* g, void* stream);

/* Launch-shape knobs, for measurement only (0 keeps the current value): threads per block of the
 * flight and imaging kernels (multiples of 32 up to 256; defaults 256, general-mode flights 128),
 * persistent blocks per SM (default: 8; the general-mode flight fills an SM once, 640 threads), and
 * the number of cell steps a flight kernel takes between two points where idle lanes take new packets
 * (default: scalar mode 1 = static assignment; general mode 32 until the library has seen the mean flight
 * length of a batch, then 1, 8 or 16 for flights shorter than 3, shorter than 24, or longer; setting it
 * here switches that choice off).  Results do not depend on any of these. */
int krp_tune(krp_grid* g, int transport_block, int image_block, int blocks_per_sm, int flight_burst);
/* Scheduling features, for A/B measurement and for the tests that show results do not depend on them (-1 keeps the
 * current value): dir_sort 1/0 = first flights of an isotropic point source taken in direction order / in id order;
 * obs_cells 1/0 = per-observer cell coefficient arrays in the general-mode imaging march / look-ups in the march (takes
 * effect at the next change of the observer set); order_policy 0 never / 1 by the measured ray length (not below 12 cell
 * steps per ray) and the size of the pass (not for fewer than 2^18 events over a cell array of at most 12 MiB) / 2 always
 * order the events by cell before imaging. */
int krp_tune_schedule(krp_grid* g, int dir_sort, int obs_cells, int order_policy);
/* Small batches in scalar mode (no field, constant non-dichroic opacity, F(Theta) scattering, no open source grid): a
 * krp_transport call of at most max_packets packets runs as ONE kernel in which a thread follows a packet from emission to its
 * end (flight, record, scattering, next flight: the kernel shape of PAPER.md:123) instead of one flight and one scattering
 * launch per scattering order -- a batch that small is bound by launch latency as a wavefront.  Records are bit-identical to
 * the wavefront's; their order in the event buffer differs.  Default 1048576 (measured on B200: the one kernel wins up to ~1.5e6
 * packets on a 128^3 disk and beyond 4e6 on a 32^3 sphere); 0 = always the wavefront.  KRP_ERR_ARG if negative. */
int krp_tune_fused(krp_grid* g, long long max_packets);
/* Device time per kernel class, for measurement (bench.py's roofline): when enabled, every launch of a
 * flight, scattering, ordering or imaging kernel is bracketed by CUDA events on the caller's stream.
 * krp_timing_get synchronises, adds up the elapsed times since the last call into ms[KRP_T_COUNT] and the
 * launch counts into launches[KRP_T_COUNT] (either may be NULL), and rearms.  At most 4096 launches are kept
 * between two krp_timing_get calls; later ones go untimed. */
enum { KRP_T_FLIGHT = 0, KRP_T_SCATTER = 1, KRP_T_ORDER = 2, KRP_T_IMAGE = 3, KRP_T_EMIT = 4, KRP_T_DEPOSIT = 5, KRP_T_RAYS = 6,
       KRP_T_COUNT = 7 };
int krp_timing_enable(krp_grid* g, int on);
int krp_timing_get(krp_grid* g, double* ms, uint64_t* launches);

/* Number of kernels the library has launched on behalf of g since creation. */
uint64_t krp_launch_count(const krp_grid* g);

#ifdef __cplusplus
}
#endif
#endif /* KRP_H_ */
