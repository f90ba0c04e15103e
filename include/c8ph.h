/*
 * c8ph.h — C-ABI of libc8ph: B200-native optical-photon emission and propagation
 * for air-shower track segments (arxiv/paper_2405_04229, D. Baack).
 * P:n = PAPER.md line n of the thesis text.
 *
 * The library computes, per charged-particle track segment:
 *   Cherenkov yield (Frank-Tamm, Eq. 2.2-2.4, height dependent n(h) from
 *   Listing 4.1) or fluorescence yield (Eq. 2.6, constant photons/MeV)
 *   -> photons on the cone cos(theta) = 1/(beta n) (Eq. 2.5), Philox4x32-10
 *      keyed on (seed; segment id, photon index)
 *   -> straight line to the observation level (Eq. 3.3)
 *   -> refraction: none | per-photon layered Snell sum (Eq. 3.15) | interpolation
 *      tracing with a pre-computed correction table
 *   -> atmospheric transmission
 *   -> photon cuts: LV1 segment filter (Eq. 4.3), LV2/LV3 photon filter
 *   -> ground grid / telescope spheres / camera pixels x time bins, photon list.
 *
 * Conventions: units m, ns, nm, g/cm^2, MeV.  Local right-handed frame, origin at the array
 * centre on the observation level, z up; observation level is the plane z = 0 at
 * altitude h_obs a.s.l.; in the spherical model the Earth centre is (0,0,-(R+h_obs)).
 *
 * All functions return C8PH_OK (0) or a negative error code; no exceptions cross the
 * boundary.  Pointers are marked HOST or DEVICE.  No torch types appear here.
 */
#ifndef C8PH_H
#define C8PH_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define C8PH_VERSION 200

enum {
    C8PH_OK = 0,
    C8PH_E_ARG = -1,      /* NULL / out-of-range / inconsistent argument                      */
    C8PH_E_STATE = -2,    /* atmosphere, detector or trace table not set up for this request   */
    C8PH_E_CUDA = -3,     /* a CUDA runtime call failed; text in c8ph_last_error()              */
    C8PH_E_NOMEM = -4
};

typedef struct c8ph_ctx c8ph_ctx;   /* opaque; owns only what it creates (tables, detector grids) */

/* Create / destroy a context bound to one CUDA device.  Not thread-safe per context.
 * Validation switch: with C8PH_FORCE_BRUTE=1 in the environment at create time every telescope
 * search of the context walks all telescopes instead of the uniform grids (same results, slow). */
int c8ph_create(c8ph_ctx **out, int cuda_device);
int c8ph_destroy(c8ph_ctx *ctx);
/* Text of the last error of this context (or of create, if ctx == NULL); never NULL. */
const char *c8ph_last_error(const c8ph_ctx *ctx);
int c8ph_version(void);

/* ---- atmosphere (thesis sec. 3.3, sec. 4.1) ------------------------------ */
/* C8PH_ATM_CYLINDRICAL (thesis sec. 3.3.3; R24): per photon the refractive-index gradient keeps the
 * azimuth of the emission point about the origin's vertical and only its zenith angle follows the position: coaxial
 * cylinders instead of spheres.  Heights and local verticals at the emission point are those of the spherical model;
 * table tracing only, with a table built with n_c >= 2; no aerosol, no flat_plane.                                 */
enum { C8PH_ATM_HOMOGENEOUS = 0, C8PH_ATM_PLANAR = 1, C8PH_ATM_SPHERICAL = 2, C8PH_ATM_CYLINDRICAL = 3 };
typedef struct {
    uint32_t size;                   /* sizeof(c8ph_atmosphere_desc), for versioning              */
    int32_t model;                   /* C8PH_ATM_*                                                 */
    float n_const_minus_1;           /* homogeneous model: refractivity n-1                        */
    float h0_m, dh_m;                /* uniform height grid of the tables, node k at h0 + k dh     */
    int32_t n_nodes;                 /* >= 2 (ignored for the homogeneous model)                   */
    const float *refractivity;       /* HOST [n_nodes]: n-1 at the nodes (Listing 4.1)             */
    const float *overburden_gcm2;    /* HOST [n_nodes] or NULL: vertical overburden X_v(h)         */
    float earth_radius_m, h_obs_m;   /* R and the altitude of the observation level                */
    float rayleigh_X_gcm2, rayleigh_lambda_nm; /* tau_R = X_slant (lambda_R/lambda)^4 / X_R; X_R = 0: off */
    float aer_L_m, aer_H_m, aer_lambda_nm, aer_angstrom; /* aerosol: alpha = exp(-h/H)/L (lambda_a/lambda)^a; L = 0: off */
    /* Tabulated extinction (thesis P:772-796, Fig. 4.7a: MODTRAN-type curves per wavelength and height for
     * vertical flight): vertical optical depth between the observation level and node k of the height grid
     * for wavelength node i on the uniform grid ext_lambda0_nm + i ext_dlambda_nm; bilinear, clamped; a
     * slanted path scales it with X_slant / (X_v(h_obs) - X_v(h_e)) (needs overburden_gcm2).  When given
     * (n_ext_lambda > 0) it replaces the Rayleigh / aerosol laws above.                                   */
    int32_t n_ext_lambda;
    float ext_lambda0_nm, ext_dlambda_nm;
    const float *ext_tau_v;          /* HOST [n_ext_lambda][n_nodes]; copied                      */
} c8ph_atmosphere_desc;
/* Copies the tables to the device (synchronous).  Invalidates a previously built trace table. */
int c8ph_init_atmosphere(c8ph_ctx *ctx, const c8ph_atmosphere_desc *desc);

/* ---- interpolation-tracing correction table (thesis sec. 4.4.1) -------------------- */
#define C8PH_TABLE_CHANNELS 5        /* dd [m], ds [m], dt [ns], X_slant [g/cm^2], tau_aer        */
typedef struct {
    uint32_t size;
    int32_t n_h, n_zen;              /* nodes: h_a = a h_max/(n_h-1) a.s.l., theta_b = b zen_max/(n_zen-1) */
    float h_max_m, zen_max_deg;
    int32_t substeps;                /* sub-layers per n(h) table cell in the builder (>= 1)       */
    /* Table "relative to a flat observation plane" (thesis P:861, Fig. 4.10; R21; spherical model only):
     * two more axes, rho = polar radius of the straight-line point on the plane z = 0 (n_rho >= 2 uniform nodes up to
     * rho_max_m) and the pointing angle of the direction of flight against the outward radial direction there (kept
     * as even / odd / transverse parts).  n_rho = 0: not built.  Used by params.flat_plane = 2.                    */
    int32_t n_rho;
    float rho_max_m;
    /* Cylindrical model (R24): third axis c = cos^2(azimuth of the flight against the plane of curvature), n_c >= 2
     * uniform nodes in [0, 1] (c = 0: the planar model's table, c = 1: the spherical one); texels (dd, dt, X_slant,
     * displacement across the flight / (sin psi cos psi)).  0: not built.                                          */
    int32_t n_c;
} c8ph_table_desc;
/* One kernel, one thread per node: the exact layered-Snell ray (fp64) from (h_a, theta_b) to the
 * observation sphere/plane minus the straight line (asynchronous on `stream`, a cudaStream_t).   */
int c8ph_build_trace_table(c8ph_ctx *ctx, const c8ph_table_desc *desc, void *stream);
/* Copy the table out / in (HOST, layout [n_h][n_zen][C8PH_TABLE_CHANNELS]); synchronous.
 * set_ lets a caller inject a table computed elsewhere.  No-ground nodes hold NaN.              */
int c8ph_get_trace_table(c8ph_ctx *ctx, float *host_out, int64_t n_floats);
int c8ph_set_trace_table(c8ph_ctx *ctx, const c8ph_table_desc *desc, const float *host_in);
/* The flat-plane table as stored: HOST [2][n_rho][n_h][n_zen][4]; part 0 (even) = dd [m], dt [ns], X_slant, tau_aer
 * relative to the straight line to the PLANE; part 1 = odd dd, odd dt, transverse displacement P [m], 0.  Synchronous. */
int c8ph_get_trace_table_flat(c8ph_ctx *ctx, float *host_out, int64_t n_floats);
/* The cylindrical model's table as stored: HOST [n_c][n_h][n_zen][4].  Synchronous. */
int c8ph_get_trace_table_cyl(c8ph_ctx *ctx, float *host_out, int64_t n_floats);

/* ---- detector (thesis sec. 6.2; camera: BASELINE cfg3) ---------------------------- */
typedef struct {
    uint32_t size;
    int32_t hist_nx, hist_ny;        /* ground grid, bin (ix,iy) -> iy*hist_nx + ix; 0: no grid    */
    float hist_x0, hist_y0, hist_cell;
    int32_t n_tel;                   /* telescope bounding spheres                        */
    const float *tel_xyzr;           /* HOST [n_tel][4] = centre x,y,z and radius; copied          */
    int32_t cam_enabled;             /* camera on the (single) telescope: pixel x time-bin histogram */
    float cam_axis_az_deg, cam_axis_el_deg, cam_pix_deg;
    int32_t cam_rows, cam_cols, n_tbins;
    double t_ref_ns;                 /* photon times are reported relative to t_ref               */
    float t_bin_ns;
    /* Last-mile optics inside the bounding spheres (thesis sec. 6.4): every telescope is a
     * parabolic first-surface mirror (focal length f, aperture radius R_m, vertex at centre - (f/2) w)
     * with a camera disc (radius R_c, at centre + (f/2) w) that also shadows the mirror; w = pointing
     * direction (azimuth from +x towards +y, elevation above the horizon).  With WRITE_TEL only camera
     * hits are written: record.x,y = camera-plane coordinates [m] along (right, up) =
     * ((-sin az, cos az, 0), w x right), record.ux,uy = reflected direction along (right, up) (the ray
     * travels towards +w), t = arrival at the camera; counters[CAM_HIT] counts them.  The spheres must
     * contain mirror and camera.  Excludes cam_enabled and WRITE_ALL.                               */
    int32_t opt_enabled;
    float opt_az_deg, opt_el_deg, opt_focal_m, opt_mirror_radius_m, opt_camera_radius_m;
    /* More of thesis sec. 6.4 (R22).  "Light bending at a boundary layer (e.g. lens ...)":
     * opt_kind = 1 replaces the mirror by a plano-convex lens - plane face (aperture radius opt_mirror_radius_m) at
     * centre + (f/2) w, convex spherical face (radius of curvature opt_lens_roc_m, apex opt_lens_thickness_m above
     * the plane face) towards the sky, index opt_lens_index, camera disc at centre - (f/2) w facing the lens; vector
     * Snell (Eq. 3.15) at both faces, a ray that is totally reflected inside the glass (Fig. 6.6a) is lost; the
     * record's time counts the index inside the glass, its direction (ux, uy along right, up) belongs to a ray that
     * travels towards -w.  "Absorption by objects": opt_n_abs <= 8 opaque capsules
     * (axis end points and radius, telescope frame (right, up, axis) about the sphere centre, e.g. the truss): a ray
     * whose leg sphere entry -> mirror / lens or mirror / lens -> camera comes within the radius is absorbed.       */
    int32_t opt_kind;                /* 0: parabolic mirror, 1: plano-convex lens                     */
    float opt_lens_roc_m, opt_lens_thickness_m, opt_lens_index;
    int32_t opt_n_abs;
    float opt_abs[8][7];             /* x0, y0, z0, x1, y1, z1, r                                      */
} c8ph_detector;
/* Copies the telescope list and builds the two uniform-grid accelerators on the host (per cell: the
 * candidate telescopes sorted by a lower-bound key, the smallest key, the nearest / first telescope in
 * line); synchronous, so it takes no stream (SURVEY 8(b) lists one: the grids are built on the host).
 * LV2 margins up to 64 m are covered by the grid.  cam_enabled needs exactly one telescope.        */
int c8ph_set_detector(c8ph_ctx *ctx, const c8ph_detector *det);

/* ---- run parameters --------------------------------------------------------------------------- */
enum {
    C8PH_EMIT_CHERENKOV = 0, C8PH_EMIT_FLUORESCENCE = 1
};
enum { C8PH_TRACE_STRAIGHT = 0, C8PH_TRACE_NUMERIC = 1, C8PH_TRACE_TABLE = 2 };
enum { C8PH_TRANS_OFF = 0, C8PH_TRANS_WEIGHT = 1, C8PH_TRANS_ROULETTE = 2 };
enum { C8PH_WRITE_NONE = 0, C8PH_WRITE_ALL = 1, C8PH_WRITE_TEL = 2 };
typedef struct {
    uint32_t size;
    int32_t emit, trace, trans, write;      /* the enums above                                    */
    int32_t filter_lv1, filter_lv2;         /* booleans                                           */
    float lambda_min_nm, lambda_max_nm;     /* Cherenkov band                                     */
    float bunch_weight;                     /* photons per generated bunch (> 0)                  */
    float lv1_margin_rad, lv2_margin_m;
    float fluor_yield_per_MeV, aim_factor;  /* fluorescence: photons/MeV; forced-cone radius = aim_factor * r_tel */
                                            /* (fluorescence line spectrum: c8ph_set_line_spectrum) */
    /* Dispersion (thesis P:314-322, Eq. 2.5): n(lambda,h) - 1 = (n(h) - 1) D(lambda),
     * D = 1 + b (1/lambda^2 - 1/lambda0^2), the n(h) table being valid at lambda0.  The yield is the
     * integral over the band with the Heaviside threshold beta n(lambda) > 1, wavelengths follow
     * lambda^-2 sin^2 theta(lambda), the cone angle uses n(lambda, h_e).  b = 0: off; b >= 0.    */
    float disp_b_nm2, disp_lambda0_nm;
    /* Detector efficiency eps(lambda) (mirror x sensor, thesis P:360-366) folded into the
     * survival probability / weight together with the atmospheric transmission: the table given to
     * c8ph_set_efficiency.  0: off.  Needs trans != C8PH_TRANS_OFF.                                */
    int32_t use_efficiency;
    /* Flat observation plane in the spherical model (thesis Fig. 4.10: the correction tables are
     * "relative to a flat observation plane"; R19).  The (height, zenith) table describes the ray
     * where it meets the observation SPHERE; 0: its displacement is applied at the straight-line point of
     * the plane z = 0 (the sag of the sphere under the plane is ignored: < 1 mm within 5 km of the
     * origin, centimetres beyond 15 km); 1: line on to the sphere, arc along the flight direction, back
     * along the arrival direction to z = 0 (0.1 mm / 1 ps against a 3-D ray integration out to 25 km).
     * Photons whose straight line misses the sphere count as C8PH_CNT_TABLE_RANGE.  2: the same result from the
     * thesis' own construction, the table over (height, zenith, rho, pointing angle) built with n_rho >= 2 (R21):
     * one lookup of 16 texels instead of the analytic step; straight-line points beyond rho_max_m count as
     * TABLE_RANGE.  Ignored for the planar / homogeneous models and the straight trace.              */
    int32_t flat_plane;
} c8ph_params;

/* Wavelength tables of the context (set-up calls: synchronous, copied; the hot call then allocates and copies nothing).
 * c8ph_set_line_spectrum: the discrete fluorescence spectrum (thesis P:340-344): n_lines wavelengths [nm] and
 *   the cumulative line probabilities (non-decreasing, last = 1); needed by C8PH_EMIT_FLUORESCENCE.
 * c8ph_set_efficiency: eps(lambda) in [0,1] on the uniform grid lambda0_nm + i dlambda_nm, linear between nodes, end
 *   values held outside; used by calls with params.use_efficiency.  n = 0 removes the table.
 * Not to be called while work that uses the table is still in flight on a stream.                             */
int c8ph_set_line_spectrum(c8ph_ctx *ctx, int32_t n_lines, const float *line_nm, const float *line_cdf);
int c8ph_set_efficiency(c8ph_ctx *ctx, int32_t n_eff, float lambda0_nm, float dlambda_nm, const float *eff);

/* ---- segments, outputs ------------------------------------------------------------------------- */
typedef struct {                            /* SoA, fp32, n_segments each, caller-owned            */
    uint32_t size;
    const float *x, *y, *z;                 /* start point A                                       */
    const float *dx, *dy, *dz;              /* direction P (renormalised on the device)            */
    const float *len, *beta, *t0, *charge;  /* length, v/c, time at A, charge number               */
    const float *edep;                      /* MeV deposited (fluorescence) or NULL                */
    const uint64_t *id;                     /* global segment ids (the Philox counter words) or NULL:
                                               seg_id_base + i.  With ids the result does not depend on the order of
                                               the segments in the arrays (record.seg stays the array index).          */
} c8ph_segments;

typedef struct {                            /* 32 B photon record                                  */
    float x, y;                             /* position on the observation plane                   */
    float ux, uy;                           /* arrival direction (uz = -sqrt(1-ux^2-uy^2))         */
    float t_ns;                             /* arrival time - t_ref                                */
    float lambda_nm;
    uint32_t seg;                           /* segment index within the call                       */
    uint32_t j_tel;                         /* (photon index j << 14) | telescope, 0x3FFF = none   */
} c8ph_photon;
#define C8PH_TEL_NONE 0x3FFFu
#define C8PH_MAX_BUNCHES_PER_SEGMENT (1 << 18)

enum {
    C8PH_CNT_SEGMENTS = 0, C8PH_CNT_SEG_BELOW_THRESHOLD, C8PH_CNT_SEG_LV1, C8PH_CNT_SEG_EMITTING,
    C8PH_CNT_EMITTED, C8PH_CNT_UPGOING, C8PH_CNT_LV2, C8PH_CNT_TABLE_RANGE, C8PH_CNT_ROULETTE,
    C8PH_CNT_LANDED, C8PH_CNT_IN_GRID, C8PH_CNT_TEL_HIT, C8PH_CNT_CAM_HIT,
    C8PH_CNT_WRITTEN, C8PH_CNT_OVERFLOW, C8PH_CNT_CLIPPED,
    C8PH_CNT_NONFINITE,        /* segments with a non-finite field or a zero direction: dropped, never silent        */
    C8PH_N_COUNTERS
};

typedef struct {
    uint32_t size;
    float *hist;               /* [hist_ny*hist_nx] or camera [n_pix*n_tbins]; += weight; or NULL   */
    float *tel_counts;         /* [n_tel]; += weight per telescope hit; or NULL                     */
    c8ph_photon *photons;      /* [photon_capacity] or NULL                                         */
    float *photon_weight;      /* [photon_capacity] or NULL: bunch weight x transmission per record */
    int64_t photon_capacity;
    uint64_t *counters;        /* [C8PH_N_COUNTERS], accumulated; counters[WRITTEN] is the photon-list cursor */
} c8ph_outputs;

/* The hot call.  All segment and output pointers are DEVICE pointers; every buffer is borrowed for
 * the duration of the enqueued work only.  Asynchronous on `stream`; no allocation, no host sync
 * and no host<->device copy of bulk data.  Outputs are ACCUMULATED (caller zeroes them).  Results
 * depend only on (seed, seg_id_base + i, j): not on grid size, segment order or batching.
 * Photons that do not fit photon_capacity are still binned and counted in OVERFLOW.
 * Launches of one context share its device scratch (work cursor, prepared-segment slots): the library orders a
 * launch after the context's previous one when the two are on different streams (event wait), so calls from one host
 * thread are safe on any streams; they do not run concurrently.  A stream that is being captured into a CUDA graph
 * is not given that wait: keep the launches of one context in one capture stream.  Not thread-safe.          */
int c8ph_emit_propagate(c8ph_ctx *ctx, const c8ph_segments *segments, int64_t n_segments,
                        int64_t seg_id_base, const c8ph_params *params, uint64_t seed,
                        const c8ph_outputs *out, void *stream);

/* Same path with HOST buffers (pinned or pageable; pinned for full overlap): the segments are split
 * into up to 16 chunks that are pipelined over three internal streams (H2D of chunk c+1 | kernel of
 * chunk c | D2H of the photons chunk c-1 wrote), each chunk with seg_id_base + its offset, so the
 * result is that of one call.  hist / tel_counts / counters / the first min(written, capacity)
 * photons are copied into the HOST buffers of `out` (overwritten, not accumulated); photon.seg is
 * the segment index within the whole call.  Synchronous; device scratch is owned by the context
 * and grown on demand.                                                                          */
int c8ph_emit_propagate_host(c8ph_ctx *ctx, const c8ph_segments *host_segments, int64_t n_segments,
                             int64_t seg_id_base, const c8ph_params *params, uint64_t seed,
                             const c8ph_outputs *host_out);

/* ---- sub-stepping: the step before the hot path (thesis sec. 4.2.1) -------------------
 * Long particle steps are cut into linear pieces that follow the physical path to the telescopes'
 * resolution.  Magnetic deflection: uniform field B [T], the path f_mag:[0,1]->R^3 is
 * the Lorentz helix with kappa = 0.299792458 q B / p [1/m]; a track of arc length `len` becomes
 * n = ceil(len / sqrt(8 tol / curvature)) pieces (sagitta of each chord <= tol_m).  Multiple
 * scattering (optional): n >= ceil(len / ms_max_step_m); every piece gets Highland's
 * width theta0 = 13.6 MeV/(beta c p) |z| sqrt(t)(1 + 0.038 ln(t z^2/beta^2)), t = rho(h) ds / X0, and
 * per transverse plane the correlated Gaussian offset / deflection pair, drawn from Philox
 * (seed; piece index, track_id_base + i, stream 16): a random walk from piece to piece.  Needs the
 * atmosphere (overburden table) of the context for the density.  n <= max_sub <= 2^20 (tracks that would need
 * more are counted in desc->clipped).  A track of length 0 gives one piece of length 0 along its direction.
 * Two calls, both asynchronous on `stream`, no allocation:
 *   c8ph_substep_plan  writes offsets[0..n_tracks] (exclusive prefix sum of the piece counts); the
 *                      caller reads offsets[n_tracks] to size the segment arrays;
 *   c8ph_substep_fill  writes the pieces of track i to segments[offsets[i] .. offsets[i+1]).
 * tracks: the c8ph_segments SoA (x,y,z = start, dx,dy,dz = initial direction, len = arc length,
 * beta, t0, charge; edep ignored) plus p_GeV (momentum [GeV/c]); all DEVICE pointers.
 * out: DEVICE SoA of capacity >= offsets[n_tracks] per array (edep, if given, is zeroed).        */
typedef struct {
    uint32_t size;
    float B_tesla[3];
    float tol_m;                            /* sagitta bound of the magnetic chords (> 0)          */
    int32_t max_sub;                        /* pieces per track <= max_sub (>= 1)                  */
    int32_t ms_enabled;                     /* multiple-scattering sub-steps                       */
    float ms_max_step_m, ms_X0_gcm2;        /* piece length bound; radiation length (air: 36.62)   */
    uint64_t seed;
    int64_t track_id_base;
    uint64_t *clipped;                      /* DEVICE counter or NULL; c8ph_substep_plan adds the number of tracks whose
                                               bounds asked for more than max_sub pieces (they get max_sub): never silent */
} c8ph_substep_desc;
int c8ph_substep_plan(c8ph_ctx *ctx, const c8ph_segments *tracks, const float *p_GeV, int64_t n_tracks,
                      const c8ph_substep_desc *desc, int64_t *offsets, void *stream);
typedef struct {                            /* like c8ph_segments, but written */
    uint32_t size;
    float *x, *y, *z, *dx, *dy, *dz, *len, *beta, *t0, *charge, *edep;
} c8ph_segments_out;
int c8ph_substep_fill(c8ph_ctx *ctx, const c8ph_segments *tracks, const float *p_GeV, int64_t n_tracks,
                      const c8ph_substep_desc *desc, const int64_t *offsets,
                      const c8ph_segments_out *out, void *stream);

/* ---- allocation-free planning (for callers that cannot call cudaMalloc: CUDA graph capture, tight serving loops,
 * harnesses that forbid it).  Same operation, arguments and result as c8ph_substep_plan (the piece count
 * needs no atmosphere), but without a context (c8ph_create allocates) and for at most
 * C8PH_SUBSTEP_STATIC_MAX_TRACKS tracks per call: the scan scratch is a static device array of that size / 1024 x 8 B
 * = 32 KB inside the library, held by every GPU that loads it until the process exits.  The call runs on the CURRENT
 * device, asynchronously on `stream`, and calls no cudaMalloc / cudaFree or allocating library routine (its first
 * call on a device resolves the array's address with cudaGetSymbolAddress: make that call outside a capture).
 * All calls on a device share the scratch and it keeps the last call's contents (every element a call reads it has
 * written before): calls that overlap on the GPU - different streams without ordering - race; order them.
 * tracks / p_GeV / offsets / desc->clipped: DEVICE pointers of the current device, caller-owned.
 * Errors: C8PH_E_ARG for NULL / inconsistent arguments and for n_tracks > C8PH_SUBSTEP_STATIC_MAX_TRACKS (nothing
 * is launched; split the call or use c8ph_substep_plan), C8PH_E_CUDA for a failed runtime call; the text is in
 * c8ph_substep_plan_static_error() (per host thread).                                                      */
#define C8PH_SUBSTEP_STATIC_MAX_TRACKS 4194304
int c8ph_substep_plan_static(const c8ph_segments *tracks, const float *p_GeV, int64_t n_tracks,
                             const c8ph_substep_desc *desc, int64_t *offsets, void *stream);
const char *c8ph_substep_plan_static_error(void);

/* Device time of the last c8ph_emit_propagate kernel of this context in ms (CUDA events on the
 * launch stream; synchronises on the end event).  Returns < 0 if nothing was launched.          */
float c8ph_last_kernel_ms(c8ph_ctx *ctx);
/* Number of kernels the library has launched in this context so far. */
int64_t c8ph_launch_count(const c8ph_ctx *ctx);
const char *c8ph_counter_name(int index);

#ifdef __cplusplus
}
#endif
#endif /* C8PH_H */
