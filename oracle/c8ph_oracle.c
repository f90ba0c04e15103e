/*
 * c8ph_oracle.c — CPU ORACLE for the optical-photon hot path of
 * arxiv/paper_2405_04229 (D. Baack, "Optical Photon Emission in Extended
 * Airshowers").  P:n below = /root/reference/PAPER.md line n.
 *
 * THIS IS TEST INFRASTRUCTURE.  It is a plain, slow, fp64, step-by-step
 * restatement of what the path computes, written from the paper.  Only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load it.  It shares no code, header, table or constant
 * with the CUDA library (paper_2405_04229_b200/csrc); neither includes the
 * other.  No blocking, fusion or reordering beyond what the cited passages
 * state; OpenMP only distributes independent track segments over cores.
 *
 * Units: m, ns, nm, g/cm^2.  Frame: local Cartesian, origin at the array
 * centre on the observation level, z up (plane normal parallel to z),
 * observation plane z = 0 at altitude h_obs a.s.l.; Earth centre at
 * (0,0,-(R+h_obs)).  Readings of silent / garbled passages are listed in
 * DESIGN.md ("Readings"); each function cites the passage it follows.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"):
 *   orc_philox4x32_10   published Random123 known-answer vectors
 *   orc_cherenkov_yield Frank-Tamm closed form (Eq. 2.4), threshold beta = 1/n
 *   orc_rodrigues       M D = P, M = M^T = M^-1
 *   orc_cone_direction  u.P = cos(theta_c), |u| = 1, azimuth uniformity
 *   orc_straight_line   constant-n ring radius Z tan(theta_c)
 *   orc_trace           Snell / Bouguer invariants, constant-n limit, R->inf
 *                       limit, corrected Eq. 3.23 closed form (linear n),
 *                       brute-force fine-step ray integration
 *   orc_table_lookup    node values, exactness on bilinear functions
 *   orc_transmission    single-exponential closed form
 *   orc_run             photon-count conservation, filter losslessness,
 *                       ray-sphere analytic cases
 *   fluorescence / camera (cfg3): isotropy moments, line frequencies,
 *                       pixel-centre round trip.
 *   orc_substep_track (R16) chord end points vs an independent RK4 Lorentz integration, sagitta <= tol
 *                       with the smallest piece count, lengths / clocks, zero-field and stiff limits.
 *   orc_substep_track_ms (R18) Highland width values, Var(theta), Var(y), Cov(y, theta) of one piece,
 *                       accumulation over pieces, zero-density identity with R16, id-keyed draws.
 *   orc_run photon geometry (R9 application, R19 flat plane) landed position, time and direction of whole
 *                       photons vs an independent 3-D RK4 ray integration to the plane z = 0 (off-centre
 *                       emission, any azimuth): mm agreement out to 30 km with flat_plane, and the size
 *                       of the sag error without it.
 *   orc_last_mile (R15) focus and constant path of axis-parallel rays, camera shadow fraction,
 *                       vertex-ray shadow rule, independent numerical intersection of skew rays.
 *   tabulated extinction (R17) table filled from the Rayleigh law reproduces orc_transmission (nodes,
 *                       slant scaling, whole runs), tau linear in the table.
 *   efficiency (R14)    lookup values, eps = 1 identity, constant eps scaling, step curve.
 *   dispersion (R13)    b -> 0 limit, closed form of the yield integral incl. threshold
 *                       inside the band, u.P = 1/(beta n(lambda)), KS test of the spectrum.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_C_M_PER_NS 0.299792458
#define ORC_ALPHA (1.0 / 137.035999)
#define ORC_PI 3.14159265358979323846

/* ------------------------------------------------------------------ types */
typedef struct {
    int32_t model;            /* 0 homogeneous, 1 planar, 2 spherical */
    int32_t n_nodes;
    double n_const_minus_1;   /* homogeneous refractivity */
    double h0, dh;            /* uniform height grid (Listing 4.1) */
    const float *refractivity;/* n-1 at the nodes (fp32 input bytes) */
    const float *overburden;  /* vertical overburden X_v at the nodes [g/cm^2] or NULL */
    double earth_radius, h_obs;
    double rayleigh_X, rayleigh_lambda;            /* X_R [g/cm^2] at lambda_R [nm]; 0 = off */
    double aer_L, aer_H, aer_lambda, aer_angstrom; /* aer_L = 0 => no aerosol */
    /* tabulated extinction (reading R17): vertical optical depth from the observation level up to the
     * nodes of the height grid, per wavelength node; replaces the Rayleigh / aerosol laws when given */
    int32_t n_ext_lambda, pad4;
    double ext_lambda0, ext_dlambda;
    const float *ext_tau_v;                        /* [n_ext_lambda][n_nodes] or NULL */
} orc_atmosphere;

typedef struct {
    int32_t n_h, n_zen, n_ch;      /* n_ch = 5: dd, ds, dt, X_slant, tau_aer */
    int32_t pad;
    double h_max, zen_max_rad;
    const float *data;             /* [n_h][n_zen][n_ch], fp32 as stored */
    /* reading R21: the table "relative to a flat observation plane" (Fig. 4.10): third axis rho (polar radius of
     * the straight-line point on the plane z = 0, uniform, n_rho >= 2), fourth axis cos(pointing angle) as even / odd part */
    int32_t n_rho, pad3;
    double rho_max;
    const float *data3;            /* [2][n_rho][n_h][n_zen][n_ch] or NULL */
} orc_table;

typedef struct {
    const float *x, *y, *z, *dx, *dy, *dz, *len, *beta, *t0, *charge, *edep;
    const uint64_t *id;            /* global segment ids (Philox counter words) or NULL: seg_id_base + i */
} orc_segments;

typedef struct {
    int32_t hist_nx, hist_ny;
    double hist_x0, hist_y0, hist_cell;
    int32_t n_tel, cam_enabled;
    const float *tel_xyzr;         /* [n_tel][4] */
    double cam_az_deg, cam_el_deg, cam_pix_deg;
    int32_t cam_rows, cam_cols, n_tbins, pad;
    double t_ref_ns, t_bin_ns;
    /* last-mile optics (thesis sec. 6.4, reading R15): one parabolic mirror + camera disc per telescope */
    int32_t opt_enabled, pad3;
    double opt_az_deg, opt_el_deg;         /* pointing direction of every telescope */
    double opt_focal_m, opt_mirror_radius_m, opt_camera_radius_m;
    /* reading R22 (thesis sec. 6.4: "light bending at a boundary layer (e.g. lens ...)", "absorption by objects") */
    int32_t opt_kind, opt_n_abs;           /* 0: parabolic mirror (R15); 1: plano-convex lens.  absorbing capsules (<= 8) */
    double opt_lens_roc_m, opt_lens_thickness_m, opt_lens_index;
    double opt_abs[8][7];                  /* capsule axis end points and radius (x0,y0,z0,x1,y1,z1,r) in the telescope
                                              frame (right, up, axis) about the bounding-sphere centre */
} orc_detector;

enum { ORC_EMIT_CHERENKOV = 0, ORC_EMIT_FLUOR = 1 };
enum { ORC_TRACE_STRAIGHT = 0, ORC_TRACE_NUMERIC = 1, ORC_TRACE_TABLE = 2 };
enum { ORC_TRANS_OFF = 0, ORC_TRANS_WEIGHT = 1, ORC_TRANS_ROULETTE = 2 };

typedef struct {
    int32_t emit, trace, trans;
    int32_t lv1, lv2, substeps;
    double lambda_min_nm, lambda_max_nm, bunch_weight;
    double lv1_margin_rad, lv2_margin_m;
    double fluor_yield_per_MeV, aim_factor;
    int32_t n_lines, pad;
    const float *line_nm, *line_cdf;
    double disp_b_nm2, disp_lambda0_nm;   /* dispersion n-1 = eta(h) D(lambda); b = 0: off (reading R13) */
    int32_t n_eff;                        /* detector efficiency eps(lambda) folded into the transmission (R14) */
    int32_t flat_plane;                   /* spherical model: exact step from the observation sphere to the plane z = 0 (R19) */
    double eff_lambda0_nm, eff_dlambda_nm;
    const float *eff;                     /* [n_eff] on the uniform grid lambda0 + i dlambda, in [0,1] */
} orc_params;

/* photon status */
enum { ORC_ST_LANDED = 0, ORC_ST_UPGOING = 1, ORC_ST_LV2 = 2, ORC_ST_TABLE_RANGE = 3,
       ORC_ST_ROULETTE = 4 };

typedef struct {
    int64_t seg;                  /* index within the call */
    int32_t j, status;
    double x, y, ux, uy, uz, t, lambda_nm, T, weight;
    double x_line, y_line;        /* straight-line point (before the correction) */
    int32_t bin, tel, pix, tbin;
} orc_photon;

enum { ORC_CNT_SEGMENTS = 0, ORC_CNT_SEG_BELOW_THRESHOLD, ORC_CNT_SEG_LV1, ORC_CNT_SEG_EMITTING,
       ORC_CNT_EMITTED, ORC_CNT_UPGOING, ORC_CNT_LV2, ORC_CNT_TABLE_RANGE, ORC_CNT_ROULETTE,
       ORC_CNT_LANDED, ORC_CNT_IN_GRID, ORC_CNT_TEL_HIT, ORC_CNT_CAM_HIT,
       ORC_CNT_NONFINITE,          /* segments with a non-finite field or a zero direction: dropped and counted */
       ORC_N_COUNTERS };

/* ------------------------------------------------------------------ O0 RNG
 * Philox4x32-10, Salmon et al. (the thesis' ref. [66], "counter
 * based ... easily parallelized ... without losing the deterministic
 * sequence").  Restated from the published algorithm: ten rounds of two
 * 32x32->64 multiplications with the round key bumped by Weyl constants. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* uniform in (0,1): (2m+1) 2^-24 with m the top 23 bits — exactly
 * representable in fp32 and fp64, so oracle and device start from identical
 * uniforms (reading R0). */
double orc_uniform(uint32_t r) { return ((double)(r >> 9) + 0.5) * (1.0 / 8388608.0); }

/* counter = (j, id_lo, id_hi, stream); key = (seed_lo, seed_hi); id = global
 * segment id; j = 0xFFFFFFFF is the per-segment draw. */
static void orc_draw(uint64_t seed, uint64_t seg_id, uint32_t j, uint32_t stream, double u[4])
{
    uint32_t ctr[4] = { j, (uint32_t)seg_id, (uint32_t)(seg_id >> 32), stream };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) }, r[4];
    orc_philox4x32_10(ctr, key, r);
    for (int k = 0; k < 4; ++k) u[k] = orc_uniform(r[k]);
}

/* ------------------------------------------------------------------ A3 n(h)
 * Listing 4.1: idx = floor(h/step), linear between idx, idx+1.
 * lookups must not leave the table -> h clamped to the table range. */
static double table_lerp(const float *data, int32_t n_nodes, double h0, double dh, double h)
{
    double f = (h - h0) / dh;
    if (f < 0.0) f = 0.0;
    if (f > (double)(n_nodes - 1)) f = (double)(n_nodes - 1);
    int idx = (int)floor(f);
    if (idx > n_nodes - 2) idx = n_nodes - 2;
    double frac = f - idx;
    return (1.0 - frac) * (double)data[idx] + frac * (double)data[idx + 1];
}

double orc_refractivity(const orc_atmosphere *atm, double h)
{
    if (atm->model == 0) return atm->n_const_minus_1;
    return table_lerp(atm->refractivity, atm->n_nodes, atm->h0, atm->dh, h);
}

double orc_overburden(const orc_atmosphere *atm, double h)
{
    if (!atm->overburden) return 0.0;
    return table_lerp(atm->overburden, atm->n_nodes, atm->h0, atm->dh, h);
}

/* height a.s.l. of a local-frame point (planar h = h_obs + z;
 * spherical h = |A - C| - R with C = (0,0,-(R+h_obs))). */
double orc_height(const orc_atmosphere *atm, const double A[3])
{
    if (atm->model < 2) return atm->h_obs + A[2];        /* cylindrical (3): every point lies in its own plane of curvature */
    double Rg = atm->earth_radius + atm->h_obs;
    double zz = A[2] + Rg;
    return sqrt(A[0] * A[0] + A[1] * A[1] + zz * zz) - atm->earth_radius;
}

/* ------------------------------------------------------------------ A1 yield
 * Eq. 2.2-2.4: d2N/dxdlambda = 2 pi alpha z^2 lambda^-2 sin^2(theta),
 * cos(theta) = 1/(beta n), integrated over [lambda1, lambda2] for a
 * non-dispersive n; Heaviside threshold of P:316-318 -> max(0, .). */
double orc_cherenkov_yield(double charge, double len_m, double beta, double n,
                           double lambda1_nm, double lambda2_nm)
{
    double sin2 = 1.0 - 1.0 / (beta * beta * n * n);
    if (!(sin2 > 0.0)) return 0.0;
    double inv_l = 1.0 / (lambda1_nm * 1e-9) - 1.0 / (lambda2_nm * 1e-9);
    return 2.0 * ORC_PI * ORC_ALPHA * charge * charge * len_m * inv_l * sin2;
}

/* ------------------------------------------------------------------ dispersion (row f4, reading R13)
 * "wavelength dependence of the refractive index, called dispersion ... only for a part
 * of the light spectrum the condition beta > 1/n(lambda) may be fulfilled"; the yield integral with
 * the Heaviside function (unnumbered equation before Eq. 2.5) and theta = arccos(1/(beta n(lambda,l))).
 * The thesis gives no dispersion law (Sellmeier / Edlen are only named); reading: a
 * Cauchy-type law on the refractivity, n(lambda,h) - 1 = eta(h) D(lambda),
 * D(lambda) = 1 + b (1/lambda^2 - 1/lambda0^2), eta tabulated at lambda0. */
double orc_dispersion_factor(double b_nm2, double lambda0_nm, double lambda_nm)
{
    return 1.0 + b_nm2 * (1.0 / (lambda_nm * lambda_nm) - 1.0 / (lambda0_nm * lambda0_nm));
}

/* sin^2(theta) = max(0, 1 - 1/(beta n)^2) at wave number k = 1/lambda [1/nm] */
static double disp_sin2(double beta, double eta, double b, double lambda0, double k)
{
    double n = 1.0 + eta * (1.0 + b * (k * k - 1.0 / (lambda0 * lambda0)));
    double s = 1.0 - 1.0 / (beta * beta * n * n);
    return s > 0.0 ? s : 0.0;
}

/* N = 2 pi alpha z^2 L int_{1/l2}^{1/l1} Theta(beta n(k) - 1) (1 - 1/(beta n(k))^2) dk,
 * plain composite Simpson rule, 8192 panels. */
double orc_cherenkov_yield_dispersive(double charge, double len_m, double beta, double eta,
                                      double lambda1_nm, double lambda2_nm, double b_nm2, double lambda0_nm)
{
    const int n = 8192;
    double k_lo = 1.0 / lambda2_nm, k_hi = 1.0 / lambda1_nm, h = (k_hi - k_lo) / n;
    double acc = disp_sin2(beta, eta, b_nm2, lambda0_nm, k_lo) + disp_sin2(beta, eta, b_nm2, lambda0_nm, k_hi);
    for (int i = 1; i < n; ++i)
        acc += (i & 1 ? 4.0 : 2.0) * disp_sin2(beta, eta, b_nm2, lambda0_nm, k_lo + i * h);
    return 2.0 * ORC_PI * ORC_ALPHA * charge * charge * len_m * (acc * h / 3.0) * 1e9;
}

/* ------------------------------------------------------------------ A9 rotation
 * 180 deg Euler-Rodrigues rotation about the bisector A = D + P of
 * D = (0,0,-1) and P: M = 2 A A^T / |A|^2 - 1.  P -> (0,0,1)
 * makes A -> 0: there M = diag(1,-1,-1) (reading R4). M row-major. */
void orc_rodrigues(const double P[3], double M[9])
{
    double A[3] = { P[0], P[1], P[2] - 1.0 };
    double a2 = A[0] * A[0] + A[1] * A[1] + A[2] * A[2];
    if (P[2] > 1.0 - 1e-6 || a2 <= 0.0) {
        double d[9] = { 1, 0, 0, 0, -1, 0, 0, 0, -1 };
        memcpy(M, d, sizeof d);
        return;
    }
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c)
            M[3 * r + c] = 2.0 * A[r] * A[c] / a2 - (r == c ? 1.0 : 0.0);
}

/* local cone vector p = (cos(phi) sin(th), sin(phi) sin(th), -cos(th))
 * rotated into the particle direction, u = M p. */
void orc_cone_direction(const double M[9], double cos_th, double sin_th, double phi, double u[3])
{
    double p[3] = { cos(phi) * sin_th, sin(phi) * sin_th, -cos_th };
    for (int r = 0; r < 3; ++r) u[r] = M[3 * r] * p[0] + M[3 * r + 1] * p[1] + M[3 * r + 2] * p[2];
}

/* ------------------------------------------------------------------ A6 straight line
 * Eq. 3.3 for the plane z = 0 with the sign fixed (reading R7):
 * t* = -A_z/u_z, I = A + t* u.  Returns t* (the geometric distance D). */
double orc_straight_line(const double A[3], const double u[3], double I[3])
{
    double t = -A[2] / u[2];
    I[0] = A[0] + t * u[0];
    I[1] = A[1] + t * u[1];
    I[2] = 0.0;
    return t;
}

/* ------------------------------------------------------------------ A7 numerical tracing
 * Layered atmosphere, Snell's law in vector form, Eq. 3.15:
 *   A2' = A1' + ( sqrt(n2^2 - n1^2 + n1^2 cos^2(a1)) - n1 cos(a1) ) N,
 * A' = n * direction ("optical length" vector), N = unit normal of the
 * layer boundary along the direction of travel.  Layers are the cells of the
 * n(h) table split into `sub` equal sub-layers; each layer is homogeneous
 * with n taken at its mid height from Listing 4.1 (reading R8).  Planar: the
 * boundaries are horizontal planes, N = (0,-1).  Spherical: boundaries are
 * spheres about the Earth centre, N = -r/|r| at the crossing point.
 * Worked in the 2-D plane of the ray: coordinates (horizontal, up),
 * spherical origin at the Earth centre.
 *
 * in : h_e [m a.s.l.], zenith angle of travel measured from the local
 *      downward vertical (sin_z, cos_z > 0), target height h_g.
 * out: [0] horizontal displacement (planar) or Earth-central angle psi (spherical)
 *      [1] geometric path S  [2] optical path c*T = sum n s  [3] X_slant = int rho ds
 *      [4] aerosol optical depth at aer_lambda  [5] sin of arrival zenith angle
 * returns 0, or 1 if the ray never reaches h_g ("no-ground").
 */
int orc_trace(const orc_atmosphere *atm, int spherical, double h_e, double sin_z, double cos_z,
              double h_g, int sub, double out[6])
{
    for (int k = 0; k < 6; ++k) out[k] = 0.0;
    if (sub < 1) sub = 1;
    const double R = atm->earth_radius;
    double px = 0.0, py = spherical ? R + h_e : h_e;        /* position */
    double n_prev = 1.0 + orc_refractivity(atm, h_e);
    double Ax = n_prev * sin_z, Ay = -n_prev * cos_z;       /* A' = n * direction */
    double h_cur = h_e;
    double S = 0, cT = 0, X = 0, tau = 0;
    const double step = atm->model == 0 ? 1.0e30 : atm->dh / sub;
    while (h_cur > h_g) {
        /* next boundary below h_cur on the sub-layer grid */
        double h_next;
        if (atm->model == 0) h_next = h_g;
        else {
            double g = floor((h_cur - atm->h0) / step);
            h_next = atm->h0 + g * step;
            if (!(h_next < h_cur - 1e-9 * step)) h_next = atm->h0 + (g - 1.0) * step;
            if (h_next < h_g) h_next = h_g;
        }
        double n_l = 1.0 + orc_refractivity(atm, 0.5 * (h_cur + h_next));
        /* boundary normal along the travel direction at the current point */
        double Nx, Ny;
        if (spherical) { double r = sqrt(px * px + py * py); Nx = -px / r; Ny = -py / r; }
        else { Nx = 0.0; Ny = -1.0; }
        double n1cos = Ax * Nx + Ay * Ny;                    /* n1 cos(a1) */
        double rad = n_l * n_l - n_prev * n_prev + n1cos * n1cos;
        if (!(rad > 0.0) || !(n1cos > 0.0)) return 1;        /* total reflection / turning ray */
        double c = sqrt(rad) - n1cos;
        Ax += c * Nx; Ay += c * Ny;                          /* Eq. 3.15 */
        double dx = Ax / n_l, dy = Ay / n_l;                 /* unit direction in the layer */
        double s;
        if (spherical) {
            /* |p + s d| = R + h_next, nearest root, cancellation-free form */
            double rt = R + h_next;
            double b = px * dx + py * dy;                    /* < 0 going down */
            double cc = px * px + py * py - rt * rt;         /* >= 0 */
            double disc = b * b - cc;
            if (!(disc >= 0.0) || !(b < 0.0)) return 1;      /* misses the lower shell */
            s = cc / (-b + sqrt(disc));
        } else {
            s = (h_cur - h_next) / (-dy);
        }
        double dhl = h_cur - h_next;
        S += s;
        cT += n_l * s;
        X += (orc_overburden(atm, h_next) - orc_overburden(atm, h_cur)) * (s / dhl);
        if (atm->aer_L > 0.0)
            tau += (atm->aer_H / atm->aer_L) * (exp(-h_next / atm->aer_H) - exp(-h_cur / atm->aer_H)) * (s / dhl);
        px += s * dx; py += s * dy;
        n_prev = n_l;
        h_cur = h_next;
    }
    /* leave the last layer into the medium at the target height */
    {
        double n_g = 1.0 + orc_refractivity(atm, h_g);
        double Nx, Ny;
        if (spherical) { double r = sqrt(px * px + py * py); Nx = -px / r; Ny = -py / r; }
        else { Nx = 0.0; Ny = -1.0; }
        double n1cos = Ax * Nx + Ay * Ny;
        double rad = n_g * n_g - n_prev * n_prev + n1cos * n1cos;
        if (!(rad > 0.0)) return 1;
        double c = sqrt(rad) - n1cos;
        Ax += c * Nx; Ay += c * Ny;
        /* sine of the angle between the direction and the local downward vertical */
        double tx = -Ny, ty = Nx;                            /* horizontal unit vector */
        out[5] = fabs(Ax * tx + Ay * ty) / n_g;
    }
    out[0] = spherical ? atan2(px, py) : px;
    out[1] = S; out[2] = cT; out[3] = X; out[4] = tau;
    return 0;
}

/* R19 (Fig. 4.10: the correction is "relative to a flat observation plane"): dd, dt and the arrival
 * direction ua describe the ray where it meets the observation SPHERE r = Rg; the detector plane z = 0 touches that
 * sphere at the origin and lies above it elsewhere.  Line from the emission point Ae along u to the sphere, arc dd
 * along the direction of flight on the sphere, then back along the arrival direction (straight, at the ground index)
 * to z = 0.  Returns 1 if the straight line misses the sphere.  t_rel = arrival time - emission time [ns]. */
/* ------------------------------------------------------------------ A5 cylindrical atmosphere model (reading R24)
 * Thesis sec. 3.3.3: besides the height "the horizontal distance d from the coordinate systems origin ... to
 * the emission point, with d^2 = x^2 + y^2, is added.  Afterwards, the refractive index gradient only changes in its
 * Zenith angle theta where the rotation angle phi is kept constant" - the spherical model "requires an additional change
 * of the refractive index gradient rotation angle in every step".  Reading: per photon the rotation angle phi of the
 * gradient is frozen at the azimuth of its emission point about the origin's vertical; the gradient stays in the vertical
 * plane of that azimuth and its zenith angle follows the position along it: the atmosphere is a set of coaxial CYLINDERS
 * whose axis passes through the Earth's centre, horizontal and perpendicular to that plane.  At the emission point
 * height and local vertical are those of the spherical model; along the path the curvature across the plane is missing.
 * Numerical tracing = the layered construction of orc_trace (Eq. 3.15, layers = table cells split in `sub`, n at the
 * layer mid height) in three dimensions with N = the in-plane radial direction at the crossing point.
 * Frame: x' along the frozen azimuth, y' along the cylinder axis, z' from the axis through the emission point (x' = 0).
 * in : h_e, local zenith (sin_z, cos_z > 0), psi = azimuth of the horizontal direction of flight against x', h_g
 * out: [0] central angle about the axis (x' arc / (R + h_g))  [1] S  [2] c T  [3] X_slant  [4] tau_aer  [5] y' displacement
 *      [6..8] arrival direction (x', y', z')
 * returns 0, or 1 if the ray never reaches h_g. */
int orc_trace_cyl(const orc_atmosphere *atm, double h_e, double sin_z, double cos_z, double psi, double h_g, int sub, double out[9])
{
    for (int k = 0; k < 9; ++k) out[k] = 0.0;
    if (sub < 1) sub = 1;
    const double R = atm->earth_radius;
    double p[3] = { 0.0, 0.0, R + h_e };
    double n_prev = 1.0 + orc_refractivity(atm, h_e);
    double A[3] = { n_prev * sin_z * cos(psi), n_prev * sin_z * sin(psi), -n_prev * cos_z };   /* A' = n * direction */
    double h_cur = h_e, S = 0, cT = 0, X = 0, tau = 0;
    const double step = atm->dh / sub;
    while (h_cur > h_g) {
        double g = floor((h_cur - atm->h0) / step);
        double h_next = atm->h0 + g * step;
        if (!(h_next < h_cur - 1e-9 * step)) h_next = atm->h0 + (g - 1.0) * step;
        if (h_next < h_g) h_next = h_g;
        double n_l = 1.0 + orc_refractivity(atm, 0.5 * (h_cur + h_next));
        double r = sqrt(p[0]*p[0] + p[2]*p[2]);
        double N[3] = { -p[0] / r, 0.0, -p[2] / r };             /* gradient: in the plane of curvature only */
        double n1cos = A[0]*N[0] + A[2]*N[2];
        double rad = n_l*n_l - n_prev*n_prev + n1cos*n1cos;
        if (!(rad > 0.0) || !(n1cos > 0.0)) return 1;
        double c = sqrt(rad) - n1cos;
        A[0] += c * N[0]; A[2] += c * N[2];                      /* Eq. 3.15; the component along the axis is untouched */
        double d[3] = { A[0] / n_l, A[1] / n_l, A[2] / n_l };
        /* |(p_x + s d_x, p_z + s d_z)| = R + h_next, nearest root */
        double rt = R + h_next;
        double a2 = d[0]*d[0] + d[2]*d[2];
        double b = p[0]*d[0] + p[2]*d[2];
        double cc = p[0]*p[0] + p[2]*p[2] - rt*rt;
        double disc = b*b - a2*cc;
        if (!(disc >= 0.0) || !(b < 0.0)) return 1;
        double s = cc / (-b + sqrt(disc));
        double dhl = h_cur - h_next;
        S += s; cT += n_l * s;
        X += (orc_overburden(atm, h_next) - orc_overburden(atm, h_cur)) * (s / dhl);
        if (atm->aer_L > 0.0)
            tau += (atm->aer_H / atm->aer_L) * (exp(-h_next / atm->aer_H) - exp(-h_cur / atm->aer_H)) * (s / dhl);
        for (int k = 0; k < 3; ++k) p[k] += s * d[k];
        n_prev = n_l; h_cur = h_next;
    }
    {   /* into the medium at the target height */
        double n_g = 1.0 + orc_refractivity(atm, h_g);
        double r = sqrt(p[0]*p[0] + p[2]*p[2]);
        double N[3] = { -p[0] / r, 0.0, -p[2] / r };
        double n1cos = A[0]*N[0] + A[2]*N[2];
        double rad = n_g*n_g - n_prev*n_prev + n1cos*n1cos;
        if (!(rad > 0.0)) return 1;
        double c = sqrt(rad) - n1cos;
        A[0] += c * N[0]; A[2] += c * N[2];
        out[6] = A[0] / n_g; out[7] = A[1] / n_g; out[8] = A[2] / n_g;
    }
    out[0] = atan2(p[0], p[2]); out[1] = S; out[2] = cT; out[3] = X; out[4] = tau; out[5] = p[1];
    return 0;
}

/* the cylindrical ray against the straight line to the same cylinder surface r' = R + h_g: corr[0] displacement along the
 * horizontal direction of flight e_h, corr[1] across it (along e_h turned by +90 deg), corr[2] time [ns], corr[3] X_slant,
 * corr[4] tau_aer.  (The sag of that surface under the plane z = 0 is ignored as in the spherical model, R9 (i).) */
int orc_cyl_correction(const orc_atmosphere *atm, double h_e, double sin_z, double cos_z, double psi, int sub, double corr[5])
{
    double r[9];
    if (orc_trace_cyl(atm, h_e, sin_z, cos_z, psi, atm->h_obs, sub, r)) return 1;
    const double Rg = atm->earth_radius + atm->h_obs, re = atm->earth_radius + h_e;
    const double ux = sin_z * cos(psi), uy = sin_z * sin(psi), uz = -cos_z;
    /* straight line: in the plane of curvature a chord from radius re to radius Rg */
    const double up = sqrt(ux*ux + uz*uz);                      /* in-plane part of the unit direction */
    const double sp = ux / up, cp = -uz / up;                   /* in-plane zenith angle */
    const double pp = re * sp;
    if (!(fabs(pp) < Rg)) return 1;
    const double chord = re * cp - sqrt(Rg*Rg - pp*pp);         /* in-plane length */
    const double S_line = chord / up;
    const double psi_line = asin(pp / Rg) - atan2(sp, cp);      /* central angle of the straight line */
    const double dxp = Rg * (r[0] - psi_line), dyp = r[5] - uy * S_line;
    corr[0] = dxp * cos(psi) + dyp * sin(psi);
    corr[1] = -dxp * sin(psi) + dyp * cos(psi);
    corr[2] = (r[2] - S_line) / ORC_C_M_PER_NS;
    corr[3] = r[3]; corr[4] = r[4];
    return 0;
}

/* Interpolation tracing in the cylindrical model: the table of P:861 with its third axis.  By the symmetry of the
 * cylinders the distance d drops out once the observation surface is the cylinder r' = R + h_obs, and what remains
 * besides (height, zenith) is the azimuth psi of the flight against the plane of curvature: axis uniform in
 * c = cos^2(psi) (the curvature the ray sees along its ground track is c / R, Euler's theorem), n_c >= 2 nodes.
 * Channels: ch0 dd along e_h, ch1 the across displacement divided by sin(psi) cos(psi) (smooth in c; evaluated 1e-3 rad
 * inside the ends), ch2 dt [ns], ch3 X_slant, ch4 tau_aer.  Layout [n_c][n_h][n_zen][5]; c = 0 is the planar model's
 * table, c = 1 the spherical one. */
void orc_build_table_cyl(const orc_atmosphere *atm, int n_h, int n_zen, int n_c, double h_max, double zen_max_rad,
                         int sub, float *out)
{
    #pragma omp parallel for schedule(dynamic, 4)
    for (int a = 0; a < n_h; ++a) {
        double h = a * h_max / (n_h - 1);
        for (int b = 0; b < n_zen; ++b) {
            double th = b * zen_max_rad / (n_zen - 1);
            for (int k = 0; k < n_c; ++k) {
                float *o = out + (((size_t)k * n_h + a) * n_zen + b) * 5;
                if (h <= atm->h_obs) { for (int q = 0; q < 5; ++q) o[q] = 0.0f; continue; }
                double c = (double)k / (n_c - 1);
                double psi = acos(sqrt(c));
                psi = fmin(fmax(psi, 1e-3), 0.5 * ORC_PI - 1e-3);
                double corr[5];
                if (orc_cyl_correction(atm, h, sin(th), cos(th), psi, sub, corr)) { for (int q = 0; q < 5; ++q) o[q] = NAN; continue; }
                o[0] = (float)corr[0];
                o[1] = (float)(corr[1] / (sin(psi) * cos(psi)));
                o[2] = (float)corr[2]; o[3] = (float)corr[3]; o[4] = (float)corr[4];
            }
        }
    }
}

static void norm3(double v[3]);
static int flat_plane_step(const orc_atmosphere *atm, const double Ae[3], const double u[3], double h_e,
                           double sin_zen, double cos_zen, double dd, double dt_ns, const double ua[3],
                           double *x, double *y, double *t_rel, double *path)
{
    const double Rg = atm->earth_radius + atm->h_obs;
    const double n_ground = 1.0 + orc_refractivity(atm, atm->h_obs);
    double re = atm->earth_radius + h_e, pp = re * sin_zen;
    if (!(pp < Rg)) return 1;
    double S_line = re * cos_zen - sqrt(Rg*Rg - pp*pp);
    double w[3] = { Ae[0] + S_line*u[0], Ae[1] + S_line*u[1], Ae[2] + S_line*u[2] + Rg };
    norm3(w);
    double cw = u[0]*w[0] + u[1]*w[1] + u[2]*w[2];
    double et[3] = { u[0] - cw*w[0], u[1] - cw*w[1], u[2] - cw*w[2] };
    double en = sqrt(et[0]*et[0] + et[1]*et[1] + et[2]*et[2]);
    if (en < 1e-12) { et[0] = et[1] = et[2] = 0.0; } else { et[0] /= en; et[1] /= en; et[2] /= en; }
    double ca = cos(dd / Rg), sa = sin(dd / Rg);
    double Pr[3] = { Rg*(ca*w[0] + sa*et[0]), Rg*(ca*w[1] + sa*et[1]), Rg*(ca*w[2] + sa*et[2]) - Rg };
    double s_back = Pr[2] / ua[2];
    *x = Pr[0] - s_back * ua[0];
    *y = Pr[1] - s_back * ua[1];
    *t_rel = S_line / ORC_C_M_PER_NS + dt_ns - n_ground * s_back / ORC_C_M_PER_NS;
    if (path) *path = S_line - s_back;
    return 0;
}

/* arrival direction: u turned in the ray plane (u, local vertical rv at the emission point) by delta (R9) */
static void rotate_in_ray_plane(const double u[3], const double rv[3], double sin_zen, double cos_zen, double delta, double ua[3])
{
    for (int k = 0; k < 3; ++k) ua[k] = u[k];
    if (sin_zen > 1e-9 && delta != 0.0) {
        double ep[3];
        for (int k = 0; k < 3; ++k) ep[k] = (cos_zen*u[k] + rv[k]) / sin_zen;
        for (int k = 0; k < 3; ++k) ua[k] = cos(delta)*u[k] + sin(delta)*ep[k];
    }
}

/* rotation of the direction between emission and arrival from the Bouguer invariant (spherical model, R9) */
static double bouguer_delta(const orc_atmosphere *atm, double h_e, double sin_zen, double cos_zen, double dd)
{
    const double Rg = atm->earth_radius + atm->h_obs;
    const double n_ground = 1.0 + orc_refractivity(atm, atm->h_obs), n_ray = 1.0 + orc_refractivity(atm, h_e);
    double re = atm->earth_radius + h_e;
    double a_line = re * sin_zen / Rg;
    double a_true = n_ray * re * sin_zen / (n_ground * Rg);
    double psi_line = asin(a_line) - acos(cos_zen);
    return asin(a_true) - (psi_line + dd / Rg) - acos(cos_zen);
}

/* R21, the thesis' table "relative to a flat observation plane" for the spherical model (Fig. 4.10: height, zenith
 * angle, distance d = "the radius in the polar coordinate frame of reference", and "an additional pointing angle": four
 * dimensions).  Axes here: emission height and local zenith (as the 2-D table), rho = polar radius of the straight-line
 * point on the plane z = 0 (uniform), and cos(chi), chi = angle between the horizontal direction of flight and the
 * outward radial direction at that point, with its two end nodes -1 / +1 stored as even and odd part:
 *     value(rho, chi) = E(rho) + cos(chi) O(rho),  E = (T(+rho) + T(-rho))/2,  O = (T(+rho) - T(-rho))/2,
 * T(x) = the photon of Fig. 4.10: emitted at height h_a in the vertical plane through the origin with local zenith
 * theta_b, flying towards +x on the straight line that meets the plane at the signed coordinate x, traced exactly to
 * the observation sphere (orc_trace) and taken on to the plane by R19's construction.  Two things distinguish the plane
 * from the sphere at distance rho: it lies rho^2/2Rg higher (E, even in x) and it is tilted by rho/Rg against the
 * sphere's tangent along the direction of flight (O, odd in x, proportional to cos(chi)); terms of second order in
 * rho/Rg (1e-5 of the correction) are not represented.  Channels as in the 2-D table, relative to the straight line to
 * the PLANE: ch0 displacement along the horizontal direction of flight, ch1 path, ch2 time [ns], ch3 X_slant, ch4 tau_aer.
 * Layout [2][n_rho][n_h][n_zen][5] (E then O; ch3 of O holds the transverse displacement P, see flat_node_tangential).
 * E(rho = 0) is the 2-D table.  Nodes without such a photon hold NaN. */
static int flat_node(const orc_atmosphere *atm, double h, double th, double sz, double cz, const double r[6], double x_target, double T[5])
{
    const double rg = atm->earth_radius + atm->h_obs, re = atm->earth_radius + h;
    const double p = re * sz;
    const double S_line_sph = re * cz - sqrt(rg * rg - p * p);
    const double dd = rg * r[0] - rg * (asin(p / rg) - th);
    /* emission point E = (re sin(beta), 0, re cos(beta) - rg), direction (sin(th - beta), 0, -cos(th - beta)): its
     * straight line meets z = 0 at x(beta) = E_x + E_z tan(th - beta); solve x(beta) = x_target by bisection */
    double lo = -0.2, hi = 0.2, beta = 0.0;                   /* central angle of the emission point, +-1270 km */
    for (int it = 0; it < 64; ++it) {
        beta = 0.5 * (lo + hi);
        double Ex = re * sin(beta), Ez = re * cos(beta) - rg;
        if (Ex + Ez * tan(th - beta) < x_target) lo = beta; else hi = beta;
    }
    double Ae[3] = { re * sin(beta), 0.0, re * cos(beta) - rg };
    if (!(Ae[2] > 0.0) || !(cos(th - beta) > 1e-3) || fabs(Ae[0] + Ae[2] * tan(th - beta) - x_target) > 1e-6 * (1.0 + fabs(x_target))) return 1;
    double u[3] = { sin(th - beta), 0.0, -cos(th - beta) };
    double rv[3] = { sin(beta), 0.0, cos(beta) };
    double ua[3], x, y, t_rel, path;
    rotate_in_ray_plane(u, rv, sz, cz, bouguer_delta(atm, h, sz, cz, dd), ua);
    if (flat_plane_step(atm, Ae, u, h, sz, cz, dd, (r[2] - S_line_sph) / ORC_C_M_PER_NS, ua, &x, &y, &t_rel, &path)) return 1;
    const double D = Ae[2] / cos(th - beta);                   /* straight line to the plane */
    T[0] = x - x_target;
    T[1] = path + (r[1] - S_line_sph) - D;
    T[2] = t_rel - D / ORC_C_M_PER_NS;
    T[3] = r[3];
    T[4] = r[4];
    return 0;
}

/* The tilt of the plane against the sphere also has a component across the direction of flight: on the sphere the
 * refraction displacement dd runs along the geodesic, whose projection on the plane leans towards the radial direction
 * by cot(zenith) rho/Rg.  P(rho) = displacement towards the outward radial direction r^ of a photon in tangential flight
 * (chi = 90 deg: straight-line point (rho, 0, 0), flying along +y); for any chi the transverse part is
 * P (r^ - cos(chi) e_h).  Emission point in closed form: cos^2(global zenith) = (re^2 cos^2(theta) + rho^2 + Rg^2 - re^2)/Rg^2. */
static int flat_node_tangential(const orc_atmosphere *atm, double h, double th, double sz, double cz, const double r[6], double rho, double *P)
{
    const double rg = atm->earth_radius + atm->h_obs, re = atm->earth_radius + h;
    const double p = re * sz;
    const double S_line_sph = re * cz - sqrt(rg * rg - p * p);
    const double dd = rg * r[0] - rg * (asin(p / rg) - th);
    const double c2 = (re * re * cz * cz + rho * rho + rg * rg - re * re) / (rg * rg);
    if (!(c2 > 1e-6 && c2 <= 1.0)) return 1;
    const double cg = sqrt(c2), sg = sqrt(1.0 - c2);
    const double sdist = -rg * cg + re * cz;                   /* distance from the emission point to the plane point */
    if (!(sdist > 0.0)) return 1;
    double Ae[3] = { rho, -sdist * sg, sdist * cg };
    double u[3] = { 0.0, sg, -cg };
    double rv[3] = { Ae[0] / re, Ae[1] / re, (Ae[2] + rg) / re };
    double ua[3], x, y, t_rel;
    rotate_in_ray_plane(u, rv, sz, cz, bouguer_delta(atm, h, sz, cz, dd), ua);
    if (flat_plane_step(atm, Ae, u, h, sz, cz, dd, (r[2] - S_line_sph) / ORC_C_M_PER_NS, ua, &x, &y, &t_rel, NULL)) return 1;
    *P = x - rho;
    return 0;
}

void orc_build_table_flat(const orc_atmosphere *atm, int n_h, int n_zen, int n_rho, double h_max, double zen_max_rad,
                          double rho_max, int sub, float *out /* [2][n_rho][n_h][n_zen][5] */)
{
    const size_t half = (size_t)n_rho * n_h * n_zen * 5;
    #pragma omp parallel for schedule(dynamic, 4)
    for (int a = 0; a < n_h; ++a) {
        double h = a * h_max / (n_h - 1);
        for (int b = 0; b < n_zen; ++b) {
            double th = b * zen_max_rad / (n_zen - 1);
            double r[6];
            double sz = sin(th), cz = cos(th);
            int zero = h <= atm->h_obs, bad = 0;
            if (!zero) bad = orc_trace(atm, 1, h, sz, cz, atm->h_obs, sub, r);
            for (int c = 0; c < n_rho; ++c) {
                float *e = out + (((size_t)c * n_h + a) * n_zen + b) * 5, *o = e + half;
                if (zero) { for (int k = 0; k < 5; ++k) e[k] = o[k] = 0.0f; continue; }
                const double rho = rho_max * c / (n_rho - 1);
                double Tp[5], Tm[5], P = 0.0;
                if (bad || flat_node(atm, h, th, sz, cz, r, rho, Tp) || flat_node(atm, h, th, sz, cz, r, -rho, Tm) ||
                    flat_node_tangential(atm, h, th, sz, cz, r, rho, &P)) {
                    for (int k = 0; k < 5; ++k) e[k] = o[k] = NAN;
                    continue;
                }
                for (int k = 0; k < 5; ++k) { e[k] = (float)(0.5 * (Tp[k] + Tm[k])); o[k] = (float)(0.5 * (Tp[k] - Tm[k])); }
                o[3] = (float)P;                                /* odd part, ch3: transverse displacement (X_slant has no odd part) */
                o[4] = 0.0f;
            }
        }
    }
}

/* lookup in the flat-plane table: trilinear in (height, zenith, rho) on E and on O (indices clamped), then
 * E + cos(chi) O; cos_chi = (horizontal direction of flight) . (outward radial direction at the straight-line point);
 * *perp = P, the displacement along (r^ - cos(chi) e_h) */
int orc_table_flat_lookup(const orc_table *t, double h, double zen, double rho, double cos_chi, double out[5], double *perp)
{
    if (!t->data3 || t->n_rho < 2) return 1;
    if (!(h >= 0.0) || h > t->h_max || !(zen >= 0.0) || zen > t->zen_max_rad || !(rho >= 0.0) || rho > t->rho_max) return 1;
    double f = h / (t->h_max / (t->n_h - 1)), g = zen / (t->zen_max_rad / (t->n_zen - 1));
    double e = rho / (t->rho_max / (t->n_rho - 1));
    int a = (int)floor(f), b = (int)floor(g), c = (int)floor(e);
    if (a > t->n_h - 2) a = t->n_h - 2;
    if (b > t->n_zen - 2) b = t->n_zen - 2;
    if (c > t->n_rho - 2) c = t->n_rho - 2;
    double ff = f - a, gg = g - b, ee = e - c;
    int bad = 0;
    const size_t s = (size_t)t->n_ch, plane = (size_t)t->n_h * t->n_zen * s, half = plane * t->n_rho;
    for (int k = 0; k < 5; ++k) {
        double part[2];
        for (int eo = 0; eo < 2; ++eo) {
            double v[2];
            for (int q = 0; q < 2; ++q) {
                const float *d = t->data3 + eo * half + (size_t)(c + q) * plane;
                double v00 = d[((size_t)a * t->n_zen + b) * s + k], v01 = d[((size_t)a * t->n_zen + b + 1) * s + k];
                double v10 = d[((size_t)(a + 1) * t->n_zen + b) * s + k], v11 = d[((size_t)(a + 1) * t->n_zen + b + 1) * s + k];
                v[q] = (1 - ff) * ((1 - gg) * v00 + gg * v01) + ff * ((1 - gg) * v10 + gg * v11);
            }
            part[eo] = (1 - ee) * v[0] + ee * v[1];
        }
        if (k >= 3) { out[k] = part[0]; if (k == 3 && perp) *perp = part[1]; }   /* X_slant, tau_aer: even part only */
        else out[k] = part[0] + cos_chi * part[1];
        if (isnan(out[k]) || isnan(part[1])) bad = 1;
    }
    return bad;
}

/* trilinear lookup in the cylindrical model's table [n_c][n_h][n_zen][5] (data3, n_rho = n_c, third axis c = cos^2(psi)
 * in [0, 1]); indices clamped as in orc_table_lookup */
int orc_table_cyl_lookup(const orc_table *t, double h, double zen, double c, double out[5])
{
    if (!t->data3 || t->n_rho < 2) return 1;
    if (!(h >= 0.0) || h > t->h_max || !(zen >= 0.0) || zen > t->zen_max_rad || !(c >= 0.0) || !(c <= 1.0)) return 1;
    double f = h / (t->h_max / (t->n_h - 1)), g = zen / (t->zen_max_rad / (t->n_zen - 1)), e = c * (t->n_rho - 1);
    int a = (int)floor(f), b = (int)floor(g), k = (int)floor(e);
    if (a > t->n_h - 2) a = t->n_h - 2;
    if (b > t->n_zen - 2) b = t->n_zen - 2;
    if (k > t->n_rho - 2) k = t->n_rho - 2;
    double ff = f - a, gg = g - b, ee = e - k;
    int bad = 0;
    const size_t s = (size_t)t->n_ch, plane = (size_t)t->n_h * t->n_zen * s;
    for (int ch = 0; ch < 5; ++ch) {
        double v[2];
        for (int q = 0; q < 2; ++q) {
            const float *d = t->data3 + (size_t)(k + q) * plane;
            double v00 = d[((size_t)a * t->n_zen + b) * s + ch], v01 = d[((size_t)a * t->n_zen + b + 1) * s + ch];
            double v10 = d[((size_t)(a + 1) * t->n_zen + b) * s + ch], v11 = d[((size_t)(a + 1) * t->n_zen + b + 1) * s + ch];
            v[q] = (1 - ff) * ((1 - gg) * v00 + gg * v01) + ff * ((1 - gg) * v10 + gg * v11);
        }
        out[ch] = (1 - ee) * v[0] + ee * v[1];
        if (isnan(out[ch])) bad = 1;
    }
    return bad;
}

/* ------------------------------------------------------------------ A15 interpolation tracing
 * a correction table "calculated in advance from the difference
 * between the swift linear propagation and the slower but more accurate
 * iterative propagation".  Node (a,b): emission height h_a = a h_max/(n_h-1)
 * a.s.l., local zenith theta_b = b theta_max/(n_zen-1); value = orc_trace to
 * the sphere r_g = R + h_obs minus the straight line in the same direction to
 * the same sphere (readings R9): ch0 dd = r_g (psi_true - psi_line) [m],
 * ch1 ds = S - S_line [m], ch2 dt = (cT - S_line)/c [ns], ch3 X_slant,
 * ch4 tau_aer.  h_a <= h_obs -> zeros.  No-ground nodes hold NaN.
 * Planar model: psi -> horizontal displacement, sphere -> plane.  */
void orc_build_table(const orc_atmosphere *atm, int n_h, int n_zen, double h_max, double zen_max_rad,
                     int sub, float *out /* [n_h][n_zen][5] */)
{
    const int spherical = atm->model == 2;
    const double rg = atm->earth_radius + atm->h_obs;
    #pragma omp parallel for schedule(dynamic, 4)
    for (int a = 0; a < n_h; ++a) {
        double h = a * h_max / (n_h - 1);
        for (int b = 0; b < n_zen; ++b) {
            float *o = out + ((size_t)a * n_zen + b) * 5;
            double th = b * zen_max_rad / (n_zen - 1);
            if (h <= atm->h_obs) { for (int k = 0; k < 5; ++k) o[k] = 0.0f; continue; }
            double r[6];
            double sz = sin(th), cz = cos(th);
            if (orc_trace(atm, spherical, h, sz, cz, atm->h_obs, sub, r)) {
                for (int k = 0; k < 5; ++k) o[k] = NAN;
                continue;
            }
            double S_line, d_line, d_true;
            if (spherical) {
                double re = atm->earth_radius + h;
                double p = re * sz;
                S_line = re * cz - sqrt(rg * rg - p * p);
                d_line = rg * (asin(p / rg) - th);
                d_true = rg * r[0];
            } else {
                S_line = (h - atm->h_obs) / cz;
                d_line = (h - atm->h_obs) * sz / cz;
                d_true = r[0];
            }
            o[0] = (float)(d_true - d_line);
            o[1] = (float)(r[1] - S_line);
            o[2] = (float)((r[2] - S_line) / ORC_C_M_PER_NS);
            o[3] = (float)r[3];
            o[4] = (float)r[4];
        }
    }
}

/* bilinear lookup, indices clamped to [0, n-2] (P:947 hardware-style linear
 * interpolation between support points).  Returns 1 (TABLE_RANGE) if the
 * point is outside the table or the 2x2 stencil touches a no-ground node. */
int orc_table_lookup(const orc_table *t, double h, double zen, double out[5])
{
    if (!(h >= 0.0) || h > t->h_max || !(zen >= 0.0) || zen > t->zen_max_rad) return 1;
    double f = h / (t->h_max / (t->n_h - 1)), g = zen / (t->zen_max_rad / (t->n_zen - 1));
    int a = (int)floor(f), b = (int)floor(g);
    if (a > t->n_h - 2) a = t->n_h - 2;
    if (b > t->n_zen - 2) b = t->n_zen - 2;
    double ff = f - a, gg = g - b;
    int bad = 0;
    for (int k = 0; k < t->n_ch; ++k) {
        const float *d = t->data;
        size_t s = (size_t)t->n_ch;
        double v00 = d[((size_t)a * t->n_zen + b) * s + k], v01 = d[((size_t)a * t->n_zen + b + 1) * s + k];
        double v10 = d[((size_t)(a + 1) * t->n_zen + b) * s + k], v11 = d[((size_t)(a + 1) * t->n_zen + b + 1) * s + k];
        double v = (1 - ff) * ((1 - gg) * v00 + gg * v01) + ff * ((1 - gg) * v10 + gg * v11);
        if (isnan(v)) bad = 1;
        if (k < 5) out[k] = v;
    }
    return bad;
}

/* ------------------------------------------------------------------ A12 transmission
 * P:360-366, P:772-796 with the analytic stand-in of DESIGN.md (R11):
 * tau = X_slant (lambda_R/lambda)^4 / X_R + tau_aer(lambda_a) (lambda_a/lambda)^angstrom. */
double orc_transmission(const orc_atmosphere *atm, double x_slant, double tau_aer, double lambda_nm)
{
    double tau = 0.0;
    if (atm->rayleigh_X > 0.0) {
        double q = atm->rayleigh_lambda / lambda_nm;
        tau += x_slant * q * q * q * q / atm->rayleigh_X;
    }
    if (atm->aer_L > 0.0) tau += tau_aer * pow(atm->aer_lambda / lambda_nm, atm->aer_angstrom);
    return exp(-tau);
}

/* Tabulated atmospheric extinction (transmission curves per wavelength and emission height
 * "with vertical flight direction", Fig. 4.7a, generated with MODTRAN).  Reading R17: the user gives the
 * vertical optical depth tau_v(lambda_i, h_k) between the observation level and the height nodes of
 * Listing 4.1's grid on a uniform wavelength grid; bilinear in (lambda, h), both clamped; a slanted,
 * refracted path scales it with the air-mass factor X_slant / (X_v(h_obs) - X_v(h_e)). */
double orc_ext_tau_vertical(const orc_atmosphere *atm, double lambda_nm, double h)
{
    if (atm->n_ext_lambda <= 0 || !atm->ext_tau_v) return 0.0;
    double g = atm->n_ext_lambda > 1 ? (lambda_nm - atm->ext_lambda0) / atm->ext_dlambda : 0.0;
    if (g < 0.0) g = 0.0;
    if (g > (double)(atm->n_ext_lambda - 1)) g = (double)(atm->n_ext_lambda - 1);
    int il = (int)floor(g);
    if (il > atm->n_ext_lambda - 2) il = atm->n_ext_lambda - 2;
    if (il < 0) il = 0;
    double gl = g - il;
    int il1 = il + 1 < atm->n_ext_lambda ? il + 1 : il;
    double lo = table_lerp(atm->ext_tau_v + (size_t)il * atm->n_nodes, atm->n_nodes, atm->h0, atm->dh, h);
    double hi = table_lerp(atm->ext_tau_v + (size_t)il1 * atm->n_nodes, atm->n_nodes, atm->h0, atm->dh, h);
    return (1.0 - gl) * lo + gl * hi;
}

double orc_transmission_tabulated(const orc_atmosphere *atm, double x_slant, double h_e, double lambda_nm)
{
    double dxv = orc_overburden(atm, atm->h_obs) - orc_overburden(atm, h_e);
    if (!(dxv > 0.0)) return 1.0;
    return exp(-orc_ext_tau_vertical(atm, lambda_nm, h_e) * (x_slant / dxv));
}

/* detector efficiency eps(lambda) ("reduce the number of photons by one to two orders of
 * magnitude ... atmosphere and detector efficiencies", Fig. 4.7b: mirror reflectivity x
 * sensor efficiency): user table on a uniform wavelength grid, linear between nodes, end values
 * held outside (reading R14).  Folded into the survival probability: p = T_atm eps. */
double orc_efficiency(const orc_params *par, double lambda_nm)
{
    if (par->n_eff <= 0 || !par->eff) return 1.0;
    if (par->n_eff == 1) return (double)par->eff[0];
    double f = (lambda_nm - par->eff_lambda0_nm) / par->eff_dlambda_nm;
    if (f < 0.0) f = 0.0;
    if (f > (double)(par->n_eff - 1)) f = (double)(par->n_eff - 1);
    int i = (int)floor(f);
    if (i > par->n_eff - 2) i = par->n_eff - 2;
    double fr = f - i;
    return (1.0 - fr) * (double)par->eff[i] + fr * (double)par->eff[i + 1];
}

/* ------------------------------------------------------------------ A14 ray / sphere
 * P:1068 "hitting the bounding sphere": the line I + s u passes within r of c.
 * Returns 1 and the entry parameter s_in if hit. */
int orc_ray_sphere(const double I[3], const double u[3], const double c[3], double r, double *s_in)
{
    double d[3] = { c[0] - I[0], c[1] - I[1], c[2] - I[2] };
    double du = d[0] * u[0] + d[1] * u[1] + d[2] * u[2];
    double d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    double m2 = d2 - du * du;
    if (m2 > r * r) return 0;
    *s_in = du - sqrt(r * r - m2);
    return 1;
}

/* hex camera (cfg3, reading R12): pixel centres
 * (a,e)_rc = ((c - (cols-1)/2 + (r mod 2)/2) p, (r - (rows-1)/2) p sqrt(3)/2);
 * nearest centre wins (brute force), must lie within the hexagon's circumradius p/sqrt(3). */
int orc_camera_pixel(const orc_detector *det, const double u_arr[3])
{
    const double d2r = ORC_PI / 180.0;
    double az = det->cam_az_deg * d2r, el = det->cam_el_deg * d2r, p = det->cam_pix_deg * d2r;
    /* camera frame: w = optical axis, right = horizontal, up completes it */
    double w[3] = { cos(el) * cos(az), cos(el) * sin(az), sin(el) };
    double rgt[3] = { -sin(az), cos(az), 0.0 };
    double up[3] = { w[1] * rgt[2] - w[2] * rgt[1], w[2] * rgt[0] - w[0] * rgt[2], w[0] * rgt[1] - w[1] * rgt[0] };
    double v[3] = { -u_arr[0], -u_arr[1], -u_arr[2] };       /* where the photon comes from */
    double vw = v[0] * w[0] + v[1] * w[1] + v[2] * w[2];
    if (!(vw > 0.0)) return -1;
    double a = atan2(v[0] * rgt[0] + v[1] * rgt[1] + v[2] * rgt[2], vw);
    double e = atan2(v[0] * up[0] + v[1] * up[1] + v[2] * up[2], vw);
    int best = -1; double bd = 1e300;
    for (int r = 0; r < det->cam_rows; ++r)
        for (int c = 0; c < det->cam_cols; ++c) {
            double ca = (c - 0.5 * (det->cam_cols - 1) + 0.5 * (r % 2)) * p;
            double ce = (r - 0.5 * (det->cam_rows - 1)) * p * sqrt(3.0) / 2.0;
            double dd = (a - ca) * (a - ca) + (e - ce) * (e - ce);
            if (dd < bd) { bd = dd; best = r * det->cam_cols + c; }
        }
    if (bd > p * p / 3.0) return -1;
    return best;
}

/* ------------------------------------------------------------------ last mile (row f3, reading R15)
 * Thesis sec. 6.4: "a raytracer can replace the photon propagator in a defined area
 * around the experiment": reflection on a (first-surface) mirror and absorption by objects, shown
 * for "a MAGIC like telescope with 17 m diameter parabola and focal point distance of 17 m" and a
 * camera of 1.47 m diameter, angular acceptance not considered.  Reading: inside the bounding
 * sphere of a telescope (centre c) the photon's arrival ray I + s u meets
 *   the camera disc  (radius R_c, centre c + (f/2) w, normal w)   from behind: absorbed (shadow),
 *   the paraboloid   z = rho^2/(4f) about the axis w with vertex V = c - (f/2) w, rho <= R_m:
 *                    mirror reflection  u' = u - 2 (u.n) n,
 *   the camera disc  again, now from the mirror side: a camera hit at (x_c, y_c) in the plane
 *                    coordinates (right, up) = (e_r, e_u), e_r = (-sin az, cos az, 0), e_u = w x e_r.
 * w = (cos el cos az, cos el sin az, sin el) is the common pointing direction.
 * in : I (point on the arrival ray, any), u (unit direction), c (sphere centre)
 * out: res[0..1] camera-plane coordinates, res[2..4] reflected direction (e_r, e_u, w components),
 *      res[5] path length from I to the camera along the ray (may start before I: s < 0 allowed)
 * returns 1 camera hit, 0 missed mirror / camera, -1 shadowed by the camera. */
/* Snell's law in vector form (Eq. 3.15) at a surface with unit normal N (pointing against the incoming ray or
 * along it: the sign is taken from u.N), from index n1 into n2: u2 = (n1 u + (sqrt(n2^2 - n1^2 + (n1 u.N)^2) - n1 |u.N|) N')/n2
 * with N' = N turned along the direction of propagation.  Returns 0 on total internal reflection (Fig. 6.6a). */
int orc_refract(const double u[3], const double N[3], double n1, double n2, double out[3])
{
    double c = u[0]*N[0] + u[1]*N[1] + u[2]*N[2];
    double sgn = c < 0.0 ? -1.0 : 1.0;                           /* N' = sgn N points along the ray */
    double ca = fabs(c);
    double q = n2*n2 - n1*n1 + n1*n1*ca*ca;
    if (q < 0.0) return 0;
    double k = sqrt(q) - n1 * ca;
    for (int i = 0; i < 3; ++i) out[i] = (n1 * u[i] + k * sgn * N[i]) / n2;
    return 1;
}

/* smallest distance between the segments P0 + s (P1 - P0), s in [0,1], and Q0 + t (Q1 - Q0), t in [0,1] */
double orc_segment_distance(const double P0[3], const double P1[3], const double Q0[3], const double Q1[3])
{
    double d1[3], d2[3], r[3];
    for (int k = 0; k < 3; ++k) { d1[k] = P1[k] - P0[k]; d2[k] = Q1[k] - Q0[k]; r[k] = P0[k] - Q0[k]; }
    double a = d1[0]*d1[0] + d1[1]*d1[1] + d1[2]*d1[2], e = d2[0]*d2[0] + d2[1]*d2[1] + d2[2]*d2[2];
    double f = d2[0]*r[0] + d2[1]*r[1] + d2[2]*r[2], cc = d1[0]*r[0] + d1[1]*r[1] + d1[2]*r[2];
    double b = d1[0]*d2[0] + d1[1]*d2[1] + d1[2]*d2[2];
    double sN, tN;
    if (a <= 1e-300 && e <= 1e-300) { sN = tN = 0.0; }
    else if (a <= 1e-300) { sN = 0.0; tN = fmin(fmax(f / e, 0.0), 1.0); }
    else if (e <= 1e-300) { tN = 0.0; sN = fmin(fmax(-cc / a, 0.0), 1.0); }
    else {
        double den = a * e - b * b;
        sN = den > 1e-300 * a * e ? fmin(fmax((b * f - cc * e) / den, 0.0), 1.0) : 0.0;
        tN = (b * sN + f) / e;
        if (tN < 0.0) { tN = 0.0; sN = fmin(fmax(-cc / a, 0.0), 1.0); }
        else if (tN > 1.0) { tN = 1.0; sN = fmin(fmax((b - cc) / a, 0.0), 1.0); }
    }
    double dx = r[0] + sN*d1[0] - tN*d2[0], dy = r[1] + sN*d1[1] - tN*d2[1], dz = r[2] + sN*d1[2] - tN*d2[2];
    return sqrt(dx*dx + dy*dy + dz*dz);
}

/* "absorption by objects": is the leg A -> B (telescope frame about the sphere centre) within reach of a capsule? */
static int leg_absorbed(const orc_detector *det, const double A[3], const double B[3])
{
    for (int k = 0; k < det->opt_n_abs && k < 8; ++k) {
        const double *o = det->opt_abs[k];
        if (orc_segment_distance(A, B, o, o + 3) <= o[6]) return 1;
    }
    return 0;
}

/* in : I (point on the arrival ray, any), u (unit direction), c (sphere centre), r_sphere (its radius: the incoming leg
 *      starts where the ray enters the sphere)
 * out: res[0..1] camera-plane coordinates, res[2..4] direction at the camera (e_r, e_u, w components),
 *      res[5] optical path length from I to the camera along the ray (may start before I: s < 0 allowed)
 * returns 1 camera hit, 0 missed mirror / lens / camera, -1 shadowed by the camera, -2 absorbed by an object (R22),
 *         -3 total internal reflection in the lens (R22).
 * opt_kind 1 (R22, "light bending at a boundary layer (e.g. lens ...)"): instead of the mirror a plano-convex lens, plane
 * face (radius R_m) at centre + (f/2) w, convex spherical face (radius of curvature R_l, apex t above the plane face)
 * towards the sky; camera disc at centre - (f/2) w facing the lens.  Vector Snell at both faces. */
int orc_last_mile(const orc_detector *det, const double I[3], const double u[3], const double c[3], double r_sphere, double res[6])
{
    const double d2r = ORC_PI / 180.0;
    const double az = det->opt_az_deg * d2r, el = det->opt_el_deg * d2r;
    const double f = det->opt_focal_m, Rm = det->opt_mirror_radius_m, Rc = det->opt_camera_radius_m;
    const double w[3] = { cos(el) * cos(az), cos(el) * sin(az), sin(el) };
    const double er[3] = { -sin(az), cos(az), 0.0 };
    const double eu[3] = { w[1]*er[2] - w[2]*er[1], w[2]*er[0] - w[0]*er[2], w[0]*er[1] - w[1]*er[0] };
    double pc[3], g[3], dr, du, dw;
    for (int k = 0; k < 3; ++k) pc[k] = I[k] - c[k];                           /* relative to the sphere centre */
    g[0] = pc[0]*er[0] + pc[1]*er[1] + pc[2]*er[2];
    g[1] = pc[0]*eu[0] + pc[1]*eu[1] + pc[2]*eu[2];
    g[2] = pc[0]*w[0] + pc[1]*w[1] + pc[2]*w[2];
    dr = u[0]*er[0] + u[1]*er[1] + u[2]*er[2];
    du = u[0]*eu[0] + u[1]*eu[1] + u[2]*eu[2];
    dw = u[0]*w[0] + u[1]*w[1] + u[2]*w[2];
    if (!(dw < 0.0)) return 0;                                  /* not travelling towards the mirror / lens */
    const double d[3] = { dr, du, dw };
    /* entry into the bounding sphere: start of the incoming leg */
    double bq = g[0]*d[0] + g[1]*d[1] + g[2]*d[2], cq = g[0]*g[0] + g[1]*g[1] + g[2]*g[2] - r_sphere*r_sphere;
    double s_in = -bq - sqrt(fmax(bq*bq - cq, 0.0));
    double E[3] = { g[0] + s_in*d[0], g[1] + s_in*d[1], g[2] + s_in*d[2] };
    if (det->opt_kind == 1) {
        const double Rl = det->opt_lens_roc_m, th = det->opt_lens_thickness_m, nl = det->opt_lens_index;
        const double zc = 0.5 * f + th - Rl;                    /* centre of curvature on the axis */
        /* convex face: |g + s d - (0,0,zc)|^2 = Rl^2, the first (upper) intersection */
        double oc[3] = { g[0], g[1], g[2] - zc };
        double b2 = oc[0]*d[0] + oc[1]*d[1] + oc[2]*d[2], c2 = oc[0]*oc[0] + oc[1]*oc[1] + oc[2]*oc[2] - Rl*Rl;
        double disc = b2*b2 - c2;
        if (disc < 0.0) return 0;
        double s1 = -b2 - sqrt(disc);
        double P1[3] = { g[0] + s1*d[0], g[1] + s1*d[1], g[2] + s1*d[2] };
        if (P1[0]*P1[0] + P1[1]*P1[1] > Rm*Rm || P1[2] < 0.5 * f) return 0;     /* outside the aperture / below the plane face */
        if (leg_absorbed(det, E, P1)) return -2;
        double N1[3] = { P1[0] / Rl, P1[1] / Rl, (P1[2] - zc) / Rl }, v[3], v2[3];
        if (!orc_refract(d, N1, 1.0, nl, v)) return -3;
        if (!(v[2] < 0.0)) return 0;
        double s2 = (0.5 * f - P1[2]) / v[2];                   /* plane face z = f/2 */
        double P2[3] = { P1[0] + s2*v[0], P1[1] + s2*v[1], 0.5 * f };
        if (P2[0]*P2[0] + P2[1]*P2[1] > Rm*Rm) return 0;        /* leaves through the rim */
        const double Nz[3] = { 0.0, 0.0, 1.0 };
        if (!orc_refract(v, Nz, nl, 1.0, v2)) return -3;        /* total internal reflection at the plane face */
        if (!(v2[2] < 0.0)) return 0;
        double s3 = (-0.5 * f - P2[2]) / v2[2];                 /* camera plane z = -f/2 */
        double P3[3] = { P2[0] + s3*v2[0], P2[1] + s3*v2[1], -0.5 * f };
        if (leg_absorbed(det, P2, P3)) return -2;
        if (P3[0]*P3[0] + P3[1]*P3[1] > Rc*Rc) return 0;
        res[0] = P3[0]; res[1] = P3[1]; res[2] = v2[0]; res[3] = v2[1]; res[4] = v2[2];
        res[5] = s1 + nl * s2 + s3;
        return 1;
    }
    /* parabolic mirror (R15), coordinates relative to the vertex V = centre - (f/2) w */
    double a = g[0], b = g[1], z0 = g[2] + 0.5 * f;
    /* camera disc from behind */
    double sc = (f - z0) / dw, xs = a + sc * dr, ys = b + sc * du;
    if (xs * xs + ys * ys <= Rc * Rc) return -1;
    /* paraboloid: (a + s dr)^2 + (b + s du)^2 = 4 f (z0 + s dw); the ray leaves the bowl at the larger root */
    double A = dr * dr + du * du, B = 2.0 * (a * dr + b * du) - 4.0 * f * dw, C = a * a + b * b - 4.0 * f * z0;
    double sh;
    if (A < 1e-18) sh = -C / B;
    else {
        double disc = B * B - 4.0 * A * C;
        if (disc < 0.0) return 0;
        double q = -0.5 * (B + (B >= 0.0 ? sqrt(disc) : -sqrt(disc)));
        double s1 = q / A, s2 = (q != 0.0) ? C / q : s1;
        sh = s1 > s2 ? s1 : s2;
    }
    double x = a + sh * dr, y = b + sh * du, z = z0 + sh * dw;
    if (x * x + y * y > Rm * Rm) return 0;
    /* mirror normal (towards the focus) and reflection */
    double n[3] = { -x / (2.0 * f), -y / (2.0 * f), 1.0 };
    double nn = sqrt(n[0]*n[0] + n[1]*n[1] + 1.0);
    n[0] /= nn; n[1] /= nn; n[2] /= nn;
    double dn = dr * n[0] + du * n[1] + dw * n[2];
    double r[3] = { dr - 2.0 * dn * n[0], du - 2.0 * dn * n[1], dw - 2.0 * dn * n[2] };
    if (!(r[2] > 0.0)) return 0;
    double s2c = (f - z) / r[2];
    double xc = x + s2c * r[0], yc = y + s2c * r[1];
    if (det->opt_n_abs > 0) {                                   /* R22: truss between the sphere entry, the mirror and the camera */
        double M[3] = { x, y, z - 0.5 * f }, K[3] = { xc, yc, 0.5 * f };
        if (leg_absorbed(det, E, M) || leg_absorbed(det, M, K)) return -2;
    }
    if (xc * xc + yc * yc > Rc * Rc) return 0;
    res[0] = xc; res[1] = yc; res[2] = r[0]; res[3] = r[1]; res[4] = r[2]; res[5] = sh + s2c;
    return 1;
}

/* ------------------------------------------------------------------ per-segment quantities */
typedef struct {
    double A[3], P[3], L, beta, t0, M[9];
    double n_exp; int64_t n_bunch; int lv1_dropped;
    double eta_mid;               /* refractivity at the segment mid height (dispersive sampling) */
    /* fluorescence */
    double aim[3], cos_psi;
} orc_segprep;

static void norm3(double v[3]) { double n = sqrt(v[0]*v[0]+v[1]*v[1]+v[2]*v[2]); v[0]/=n; v[1]/=n; v[2]/=n; }

/* bounding radius of telescopes and histogram about the array centre (origin) */
static double array_radius(const orc_detector *det)
{
    double r = 0.0;
    for (int k = 0; k < det->n_tel; ++k) {
        const float *t = det->tel_xyzr + 4 * k;
        double d = sqrt((double)t[0]*t[0] + (double)t[1]*t[1] + (double)t[2]*t[2]) + t[3];
        if (d > r) r = d;
    }
    if (det->hist_nx > 0 && det->hist_ny > 0 && !det->cam_enabled) {
        double xs[2] = { det->hist_x0, det->hist_x0 + det->hist_nx * det->hist_cell };
        double ys[2] = { det->hist_y0, det->hist_y0 + det->hist_ny * det->hist_cell };
        for (int i = 0; i < 2; ++i) for (int j = 0; j < 2; ++j) {
            double d = sqrt(xs[i]*xs[i] + ys[j]*ys[j]);
            if (d > r) r = d;
        }
    }
    return r;
}

/* SURVEY 8(b) "NONFINITE": a segment with a non-finite input field or a direction of zero length is dropped. */
static int segment_is_finite(const orc_segments *sg, int64_t i, int fluor)
{
    const double v[10] = { sg->x[i], sg->y[i], sg->z[i], sg->dx[i], sg->dy[i], sg->dz[i], sg->len[i], sg->beta[i],
                           sg->t0[i], sg->charge[i] };
    for (int k = 0; k < 10; ++k) if (!isfinite(v[k])) return 0;
    if (fluor && sg->edep && !isfinite((double)sg->edep[i])) return 0;
    return v[3]*v[3] + v[4]*v[4] + v[5]*v[5] > 0.0;
}

/* a1-a4 for one segment: ingest, LV1, yield, bunch count, rotation. */
static void prepare_segment(const orc_atmosphere *atm, const orc_detector *det, const orc_params *par,
                            const orc_table *tab, const orc_segments *sg, int64_t i,
                            uint64_t seed, uint64_t seg_id, double r_arr, orc_segprep *o)
{
    o->A[0] = sg->x[i]; o->A[1] = sg->y[i]; o->A[2] = sg->z[i];
    o->P[0] = sg->dx[i]; o->P[1] = sg->dy[i]; o->P[2] = sg->dz[i];
    norm3(o->P);
    o->L = sg->len[i]; o->beta = sg->beta[i]; o->t0 = sg->t0[i];
    o->lv1_dropped = 0; o->n_bunch = 0; o->n_exp = 0.0;
    double mid[3] = { o->A[0] + 0.5*o->L*o->P[0], o->A[1] + 0.5*o->L*o->P[1], o->A[2] + 0.5*o->L*o->P[2] };
    double h_mid = orc_height(atm, mid);
    double u_seg[4];
    orc_draw(seed, seg_id, 0xFFFFFFFFu, 0, u_seg);
    if (par->emit == ORC_EMIT_CHERENKOV) {
        double n_mid = 1.0 + orc_refractivity(atm, h_mid);
        o->eta_mid = n_mid - 1.0;
        /* O1 (R1): midpoint rule for the height dependence of Eq. 2.2 */
        if (par->disp_b_nm2 != 0.0) {
            o->eta_mid = orc_refractivity(atm, h_mid);
            o->n_exp = orc_cherenkov_yield_dispersive(sg->charge[i], o->L, o->beta, o->eta_mid,
                                                      par->lambda_min_nm, par->lambda_max_nm,
                                                      par->disp_b_nm2, par->disp_lambda0_nm);
            /* LV1 and the threshold use the largest n of the band (blue end for b > 0) */
            double Dmax = fmax(orc_dispersion_factor(par->disp_b_nm2, par->disp_lambda0_nm, par->lambda_min_nm),
                               orc_dispersion_factor(par->disp_b_nm2, par->disp_lambda0_nm, par->lambda_max_nm));
            n_mid = 1.0 + o->eta_mid * Dmax;
        } else
        o->n_exp = orc_cherenkov_yield(sg->charge[i], o->L, o->beta, n_mid,
                                       par->lambda_min_nm, par->lambda_max_nm);
        if (o->n_exp > 0.0 && par->lv1) {
            /* O10 LV1: Eq. 4.3 with point of interest = array centre widened by the
             * array's angular radius (options 1/2) and the Cherenkov angle */
            double d[3] = { -mid[0], -mid[1], -mid[2] };
            double dist = sqrt(d[0]*d[0] + d[1]*d[1] + d[2]*d[2]);
            double cosa = (o->P[0]*d[0] + o->P[1]*d[1] + o->P[2]*d[2]) / dist;
            if (cosa > 1.0) cosa = 1.0;
            if (cosa < -1.0) cosa = -1.0;
            double theta_c = acos(fmin(1.0, 1.0 / (o->beta * n_mid)));
            double ratio = r_arr / dist; if (ratio > 1.0) ratio = 1.0;
            if (acos(cosa) > theta_c + asin(ratio) + par->lv1_margin_rad) o->lv1_dropped = 1;
        }
        orc_rodrigues(o->P, o->M);
    } else {
        /* O5 fluorescence: N = Y E_dep Omega/4pi, forced cone about the line to the
         * pre-corrected aim point ("favors the direction pointing to the experiment ...
         * number of photons scaled accordingly") */
        const float *t = det->tel_xyzr;                      /* aperture = telescope 0 */
        double c[3] = { t[0], t[1], t[2] };
        double d[3] = { c[0]-mid[0], c[1]-mid[1], c[2]-mid[2] };
        double dist = sqrt(d[0]*d[0] + d[1]*d[1] + d[2]*d[2]);
        o->aim[0] = c[0]; o->aim[1] = c[1]; o->aim[2] = c[2];
        if (tab && par->trace == ORC_TRACE_TABLE) {
            double dir[3] = { d[0]/dist, d[1]/dist, d[2]/dist };
            double Rg = atm->earth_radius + atm->h_obs;
            double rv[3] = { mid[0], mid[1], mid[2] + (atm->model >= 2 ? Rg : 0.0) };
            if (atm->model < 2) { rv[0] = 0; rv[1] = 0; rv[2] = 1; }
            norm3(rv);
            double cz = -(dir[0]*rv[0] + dir[1]*rv[1] + dir[2]*rv[2]);
            double corr[5];
            double hn = sqrt(dir[0]*dir[0] + dir[1]*dir[1]);
            if (cz > 0 && hn > 1e-9 && !orc_table_lookup(tab, h_mid, acos(fmin(1.0, cz)), corr)) {
                o->aim[0] -= corr[0] * dir[0] / hn;
                o->aim[1] -= corr[0] * dir[1] / hn;
            }
        }
        double rho_aim = par->aim_factor * t[3];
        double sin_psi = rho_aim / dist; if (sin_psi > 1.0) sin_psi = 1.0;
        o->cos_psi = sqrt(1.0 - sin_psi * sin_psi);
        o->n_exp = par->fluor_yield_per_MeV * sg->edep[i] * 0.5 * (1.0 - o->cos_psi);
    }
    if (o->n_exp > 0.0 && !o->lv1_dropped)
        o->n_bunch = (int64_t)floor(o->n_exp / par->bunch_weight + u_seg[0]);   /* R1(iv) */
}

/* number of bunches each segment emits (used to size the photon buffer) */
int64_t orc_count(const orc_atmosphere *atm, const orc_detector *det, const orc_params *par,
                  const orc_table *tab, const orc_segments *sg, int64_t n_seg, int64_t seg_id_base,
                  uint64_t seed, int64_t *n_bunch /* [n_seg] or NULL */)
{
    double r_arr = array_radius(det);
    int64_t total = 0;
    #pragma omp parallel for schedule(static) reduction(+:total)
    for (int64_t i = 0; i < n_seg; ++i) {
        orc_segprep sp;
        if (!segment_is_finite(sg, i, par->emit == ORC_EMIT_FLUOR)) { if (n_bunch) n_bunch[i] = 0; continue; }
        prepare_segment(atm, det, par, tab, sg, i, seed, sg->id ? sg->id[i] : (uint64_t)(seg_id_base + i), r_arr, &sp);
        if (n_bunch) n_bunch[i] = sp.n_bunch;
        total += sp.n_bunch;
    }
    return total;
}

/* ------------------------------------------------------------------ the whole path
 * record_mode 0: histogram/counters only; 1: every emitted photon is written
 * to `photons` at offset[segment] + j (offsets = exclusive prefix sum of
 * orc_count's n_bunch), with its status. */
int orc_run(const orc_atmosphere *atm, const orc_detector *det, const orc_params *par,
            const orc_table *tab, const orc_segments *sg, int64_t n_seg, int64_t seg_id_base,
            uint64_t seed, double *hist, double *tel_counts, uint64_t *counters,
            int record_mode, const int64_t *offsets, orc_photon *photons)
{
    const double r_arr = array_radius(det);
    const double Rg = atm->earth_radius + atm->h_obs;
    const double n_ground = 1.0 + orc_refractivity(atm, atm->h_obs);
    uint64_t cnt[ORC_N_COUNTERS];
    memset(cnt, 0, sizeof cnt);
    int err = 0;
    if (par->trace == ORC_TRACE_TABLE && !tab) return -1;

    #pragma omp parallel
    {
        uint64_t lc[ORC_N_COUNTERS];
        memset(lc, 0, sizeof lc);
        #pragma omp for schedule(dynamic, 16)
        for (int64_t i = 0; i < n_seg; ++i) {
            orc_segprep sp;
            uint64_t seg_id = sg->id ? sg->id[i] : (uint64_t)(seg_id_base + i);
            lc[ORC_CNT_SEGMENTS]++;
            if (!segment_is_finite(sg, i, par->emit == ORC_EMIT_FLUOR)) { lc[ORC_CNT_NONFINITE]++; continue; }
            prepare_segment(atm, det, par, tab, sg, i, seed, seg_id, r_arr, &sp);
            if (!(sp.n_exp > 0.0)) { lc[ORC_CNT_SEG_BELOW_THRESHOLD]++; continue; }
            if (sp.lv1_dropped) { lc[ORC_CNT_SEG_LV1]++; continue; }
            if (sp.n_bunch <= 0) continue;
            lc[ORC_CNT_SEG_EMITTING]++;
            for (int64_t j = 0; j < sp.n_bunch; ++j) {
                orc_photon ph;
                memset(&ph, 0, sizeof ph);
                ph.seg = i; ph.j = (int32_t)j; ph.bin = ph.tel = ph.pix = ph.tbin = -1;
                ph.weight = par->bunch_weight; ph.T = 1.0;
                lc[ORC_CNT_EMITTED]++;
                double u4[4];
                orc_draw(seed, seg_id, (uint32_t)j, 0, u4);
                /* O2: random position along the track, particle clock */
                double s = u4[1] * sp.L;
                double Ae[3] = { sp.A[0] + s*sp.P[0], sp.A[1] + s*sp.P[1], sp.A[2] + s*sp.P[2] };
                double t_e = sp.t0 + s / (sp.beta * ORC_C_M_PER_NS);
                double h_e = orc_height(atm, Ae);
                double eta_e = orc_refractivity(atm, h_e);
                double n_e = 1.0 + eta_e;
                double u[3];
                if (par->emit == ORC_EMIT_CHERENKOV) {
                    /* O3: 1/lambda uniform (spectrum ~ 1/lambda^2, Eq. 2.4) */
                    double il1 = 1.0 / par->lambda_min_nm, il2 = 1.0 / par->lambda_max_nm;
                    ph.lambda_nm = 1.0 / (il1 - u4[2] * (il1 - il2));
                    if (par->disp_b_nm2 != 0.0) {
                        /* R13: the spectrum is 1/lambda^2 sin^2 theta(lambda): rejection from the
                         * 1/lambda-uniform law with the envelope max sin^2, n at the segment mid height;
                         * trial t takes the uniforms (2 (t&1), 2 (t&1) + 1) of draw stream 2 + t/2 */
                        double b = par->disp_b_nm2, l0 = par->disp_lambda0_nm;
                        double smax = fmax(disp_sin2(sp.beta, sp.eta_mid, b, l0, il1), disp_sin2(sp.beta, sp.eta_mid, b, l0, il2));
                        double k = il1;
                        for (int t = 0; t < 32; ++t) {
                            double ut[4];
                            orc_draw(seed, seg_id, (uint32_t)j, 2u + (uint32_t)(t >> 1), ut);
                            k = il1 - ut[2 * (t & 1)] * (il1 - il2);
                            if (ut[2 * (t & 1) + 1] * smax < disp_sin2(sp.beta, sp.eta_mid, b, l0, k)) break;
                        }
                        ph.lambda_nm = 1.0 / k;
                        n_e = 1.0 + eta_e * orc_dispersion_factor(b, l0, ph.lambda_nm);
                    }
                    /* O4: Eq. 2.5 — the angle depends on the location (and, with dispersion, on lambda) */
                    double cos_th = 1.0 / (sp.beta * n_e);
                    double sin2 = 1.0 - cos_th * cos_th;
                    if (sin2 < 0.0) { sin2 = 0.0; cos_th = 1.0; }
                    orc_cone_direction(sp.M, cos_th, sqrt(sin2), 2.0 * ORC_PI * u4[0], u);
                } else {
                    /* O5: wavelength from the discrete line CDF, direction uniform in
                     * the cone about (aim - A_e); cos(polar) uniform => isotropic density */
                    int li = 0;
                    while (li < par->n_lines - 1 && u4[2] >= (double)par->line_cdf[li]) ++li;
                    ph.lambda_nm = par->line_nm[li];
                    double ub[4];
                    orc_draw(seed, seg_id, (uint32_t)j, 1, ub);
                    double ax[3] = { sp.aim[0]-Ae[0], sp.aim[1]-Ae[1], sp.aim[2]-Ae[2] };
                    norm3(ax);
                    double cp = 1.0 - ub[0] * (1.0 - sp.cos_psi);
                    double spn = sqrt(fmax(0.0, 1.0 - cp * cp));
                    double phi = 2.0 * ORC_PI * u4[0];
                    /* orthonormal basis about ax: e1 = normalised (ax x z), e2 = ax x e1 */
                    double e1[3] = { ax[1], -ax[0], 0.0 };
                    double e1n = sqrt(e1[0]*e1[0] + e1[1]*e1[1]);
                    if (e1n < 1e-12) { e1[0] = 1; e1[1] = 0; e1n = 1; }
                    e1[0] /= e1n; e1[1] /= e1n;
                    double e2[3] = { ax[1]*e1[2]-ax[2]*e1[1], ax[2]*e1[0]-ax[0]*e1[2], ax[0]*e1[1]-ax[1]*e1[0] };
                    for (int k = 0; k < 3; ++k) u[k] = cp*ax[k] + spn*(cos(phi)*e1[k] + sin(phi)*e2[k]);
                }
                /* O6: discard up-going / horizontal photons */
                /* reading R7: Eq. 3.3 needs t* = -A_z/u_z > 0; a photon emitted at or below the observation
                 * level cannot reach it going down and is dropped with the up-going ones */
                if (u[2] >= -1e-6 || !(Ae[2] > 0.0)) { ph.status = ORC_ST_UPGOING; lc[ORC_CNT_UPGOING]++; goto store; }
                /* O7 straight line to the observation level */
                double I[3];
                double D = orc_straight_line(Ae, u, I);
                ph.x_line = I[0]; ph.y_line = I[1];
                double hn = sqrt(u[0]*u[0] + u[1]*u[1]);
                double eh[2] = { 0.0, 0.0 };
                if (hn >= 1e-9) { eh[0] = u[0]/hn; eh[1] = u[1]/hn; }
                /* O10 LV2/LV3: on the straight-line point, before the correction */
                if (par->lv2) {
                    int keep = 0;
                    double m = par->lv2_margin_m;
                    if (det->hist_nx > 0 && !det->cam_enabled) {
                        double x1 = det->hist_x0 + det->hist_nx*det->hist_cell, y1 = det->hist_y0 + det->hist_ny*det->hist_cell;
                        if (I[0] >= det->hist_x0 - m && I[0] < x1 + m && I[1] >= det->hist_y0 - m && I[1] < y1 + m) keep = 1;
                    }
                    for (int k = 0; k < det->n_tel && !keep; ++k) {
                        const float *t = det->tel_xyzr + 4*k;
                        double ddx = I[0]-t[0], ddy = I[1]-t[1];
                        double reach = t[3] / fabs(u[2]) + m;
                        if (ddx*ddx + ddy*ddy <= reach*reach) keep = 1;
                    }
                    if (!keep) { ph.status = ORC_ST_LV2; lc[ORC_CNT_LV2]++; goto store; }
                }
                /* O8/O9 refraction */
                double dd = 0, dt_ns = 0, x_slant = 0, tau_aer = 0, sin_arr, cos_zen, sin_zen;
                double rv[3] = { 0, 0, 1 };                  /* local vertical at A_e */
                if (atm->model >= 2) { rv[0] = Ae[0]; rv[1] = Ae[1]; rv[2] = Ae[2] + Rg; norm3(rv); }
                cos_zen = -(u[0]*rv[0] + u[1]*rv[1] + u[2]*rv[2]);
                if (cos_zen > 1.0) cos_zen = 1.0;
                sin_zen = sqrt(fmax(0.0, 1.0 - cos_zen*cos_zen));
                sin_arr = sin_zen;
                double delta = 0.0;                          /* rotation of the direction in the ray plane */
                double perp_flat = 0.0, rho_I = 0.0, cos_chi = 0.0;   /* R21: transverse displacement of the flat-plane table */
                double perp_cyl = 0.0;                       /* R24: displacement across the direction of flight */
                if (par->trace == ORC_TRACE_STRAIGHT) {
                    dt_ns = eta_e * D / ORC_C_M_PER_NS;      /* homogeneous: t = t_e + n D / c */
                    if (atm->model != 0) {
                        /* straight line through a stratified medium: no delay model beyond n_e */
                    }
                } else if (atm->model == 3) {
                    /* R24 cylindrical model: the plane of curvature is the vertical plane through the origin's vertical and
                     * the emission point (frozen per photon); psi = azimuth of the flight against it */
                    double d_e = sqrt(Ae[0]*Ae[0] + Ae[1]*Ae[1]);
                    double ephi[2] = { 1.0, 0.0 };
                    if (d_e > 1e-6) { ephi[0] = Ae[0] / d_e; ephi[1] = Ae[1] / d_e; }
                    else if (hn > 1e-12) { ephi[0] = eh[0]; ephi[1] = eh[1]; }
                    double cpsi = eh[0]*ephi[0] + eh[1]*ephi[1], spsi = ephi[0]*eh[1] - ephi[1]*eh[0];
                    if (!(hn > 1e-12)) { cpsi = 1.0; spsi = 0.0; }
                    double corr[5];
                    int bad;
                    if (par->trace == ORC_TRACE_NUMERIC) {
                        bad = cos_zen <= 0.0 || orc_cyl_correction(atm, h_e, sin_zen, cos_zen, atan2(spsi, cpsi), par->substeps, corr);
                    } else {
                        bad = cos_zen <= 0.0 || orc_table_cyl_lookup(tab, h_e, acos(cos_zen), cpsi * cpsi, corr);
                        corr[1] *= spsi * cpsi;                  /* the table holds the across displacement / (sin psi cos psi) */
                    }
                    if (bad) { ph.status = ORC_ST_TABLE_RANGE; lc[ORC_CNT_TABLE_RANGE]++; goto store; }
                    dd = corr[0]; perp_cyl = corr[1]; dt_ns = corr[2]; x_slant = corr[3]; tau_aer = corr[4];
                } else if (par->trace == ORC_TRACE_NUMERIC) {
                    double r[6];
                    if (cos_zen <= 0.0 || orc_trace(atm, atm->model == 2, h_e, sin_zen, cos_zen, atm->h_obs, par->substeps, r)) {
                        ph.status = ORC_ST_TABLE_RANGE; lc[ORC_CNT_TABLE_RANGE]++; goto store;
                    }
                    double d_line, S_line;
                    if (atm->model == 2) {
                        double re = atm->earth_radius + h_e, p = re * sin_zen;
                        S_line = re*cos_zen - sqrt(Rg*Rg - p*p);
                        d_line = Rg * (asin(p/Rg) - acos(cos_zen));
                        dd = Rg * r[0] - d_line;
                    } else {
                        S_line = (h_e - atm->h_obs) / cos_zen;
                        d_line = (h_e - atm->h_obs) * sin_zen / cos_zen;
                        dd = r[0] - d_line;
                    }
                    dt_ns = (r[2] - S_line) / ORC_C_M_PER_NS;
                    x_slant = r[3]; tau_aer = r[4];
                } else {
                    double corr[5];
                    /* R21: with flat_plane = 2 the flat-plane table (polar radius of the straight-line point, pointing
                     * angle of the horizontal direction of flight against the outward radial direction there) gives the
                     * correction relative to the plane z = 0 directly */
                    const int t3 = par->flat_plane == 2 && atm->model == 2;
                    rho_I = sqrt(I[0]*I[0] + I[1]*I[1]);
                    cos_chi = rho_I > 1e-9 ? (eh[0]*I[0] + eh[1]*I[1]) / rho_I : 0.0;
                    if (cos_zen <= 0.0 || (t3 ? orc_table_flat_lookup(tab, h_e, acos(cos_zen), rho_I, cos_chi, corr, &perp_flat)
                                              : orc_table_lookup(tab, h_e, acos(cos_zen), corr))) {
                        ph.status = ORC_ST_TABLE_RANGE; lc[ORC_CNT_TABLE_RANGE]++; goto store;
                    }
                    dd = corr[0]; dt_ns = corr[2]; x_slant = corr[3]; tau_aer = corr[4];
                }
                if (par->trace != ORC_TRACE_STRAIGHT) {
                    /* arrival direction from the Snell / Bouguer invariant: the direction
                     * turns in the ray plane by delta = theta_arr - psi_true - theta_z  (R9).  The ray is the
                     * one the n(h) table defines (dd, dt come from it), so the invariant takes the table's
                     * index at both ends, also when the cone angle is dispersive (R13: the table is valid at
                     * lambda0 and refraction is not dispersive) */
                    const double n_ray = 1.0 + eta_e;
                    if (atm->model >= 2) {                   /* cylindrical: the spherical formula (differs by < 1e-6 rad, R24) */
                        double re = atm->earth_radius + h_e;
                        double a_line = re * sin_zen / Rg;
                        double a_true = n_ray * re * sin_zen / (n_ground * Rg);
                        double psi_line = asin(a_line) - acos(cos_zen);
                        delta = asin(a_true) - (psi_line + dd / Rg) - acos(cos_zen);
                    } else {
                        delta = asin(n_ray * sin_zen / n_ground) - acos(cos_zen);
                    }
                }
                /* O11 transmission */
                if (par->trans != ORC_TRANS_OFF) {
                    ph.T = (atm->n_ext_lambda > 0 ? orc_transmission_tabulated(atm, x_slant, h_e, ph.lambda_nm)
                                                  : orc_transmission(atm, x_slant, tau_aer, ph.lambda_nm))
                           * orc_efficiency(par, ph.lambda_nm);
                    if (par->trans == ORC_TRANS_ROULETTE) {
                        if (!(u4[3] < ph.T)) { ph.status = ORC_ST_ROULETTE; lc[ORC_CNT_ROULETTE]++; goto store; }
                    } else ph.weight = par->bunch_weight * ph.T;
                }
                /* landed: corrected position, time, direction */
                ph.x = I[0] + dd * eh[0];
                ph.y = I[1] + dd * eh[1];
                if (perp_cyl != 0.0) {                           /* R24: along e_h turned by +90 degrees */
                    ph.x += perp_cyl * (-eh[1]);
                    ph.y += perp_cyl * eh[0];
                }
                if (perp_flat != 0.0 && rho_I > 1e-9) {          /* R21: across the direction of flight, towards r^ */
                    ph.x += perp_flat * (I[0] / rho_I - cos_chi * eh[0]);
                    ph.y += perp_flat * (I[1] / rho_I - cos_chi * eh[1]);
                }
                ph.t = t_e + D / ORC_C_M_PER_NS + dt_ns;
                {
                    double ua[3] = { u[0], u[1], u[2] };
                    if (sin_zen > 1e-9 && delta != 0.0) {
                        double ep[3];
                        for (int k = 0; k < 3; ++k) ep[k] = (cos_zen*u[k] + rv[k]) / sin_zen;
                        for (int k = 0; k < 3; ++k) ua[k] = cos(delta)*u[k] + sin(delta)*ep[k];
                    }
                    ph.ux = ua[0]; ph.uy = ua[1]; ph.uz = ua[2];
                    if (par->flat_plane == 1 && atm->model == 2 && par->trace != ORC_TRACE_STRAIGHT) {
                        /* R19: from the observation sphere to the plane z = 0 (flat_plane_step above) */
                        double t_rel;
                        if (flat_plane_step(atm, Ae, u, h_e, sin_zen, cos_zen, dd, dt_ns, ua, &ph.x, &ph.y, &t_rel, NULL)) {
                            ph.status = ORC_ST_TABLE_RANGE; lc[ORC_CNT_TABLE_RANGE]++; goto store;
                        }
                        ph.t = t_e + t_rel;
                    }
                }
                (void)sin_arr;
                ph.status = ORC_ST_LANDED;
                lc[ORC_CNT_LANDED]++;
                /* O12 binning: ground grid */
                if (det->hist_nx > 0 && !det->cam_enabled) {
                    double fx = floor((ph.x - det->hist_x0) / det->hist_cell);
                    double fy = floor((ph.y - det->hist_y0) / det->hist_cell);
                    if (fx >= 0 && fx < det->hist_nx && fy >= 0 && fy < det->hist_ny) {
                        ph.bin = (int32_t)fy * det->hist_nx + (int32_t)fx;
                        lc[ORC_CNT_IN_GRID]++;
                        if (hist) {
                            #pragma omp atomic
                            hist[ph.bin] += ph.weight;
                        }
                    }
                }
                /* O12 telescopes: brute force over all spheres; earliest entry, then lowest k */
                {
                    double Ip[3] = { ph.x, ph.y, 0.0 }, ua[3] = { ph.ux, ph.uy, ph.uz };
                    double best = 1e300;
                    for (int k = 0; k < det->n_tel; ++k) {
                        const float *t = det->tel_xyzr + 4*k;
                        double c[3] = { t[0], t[1], t[2] }, s_in;
                        if (orc_ray_sphere(Ip, ua, c, t[3], &s_in) && s_in < best) { best = s_in; ph.tel = k; }
                    }
                    if (ph.tel >= 0) {
                        lc[ORC_CNT_TEL_HIT]++;
                        if (tel_counts) {
                            #pragma omp atomic
                            tel_counts[ph.tel] += ph.weight;
                        }
                        if (det->opt_enabled) {
                            /* R15 last mile: the record becomes the camera-plane hit (x_c, y_c), the
                             * reflected direction in the telescope frame (stored as (r, u, -w) so that the
                             * third component keeps the record's sign convention) and the camera time */
                            const float *t = det->tel_xyzr + 4*ph.tel;
                            double c[3] = { t[0], t[1], t[2] }, res[6];
                            if (orc_last_mile(det, Ip, ua, c, t[3], res) == 1) {
                                ph.pix = 0;
                                lc[ORC_CNT_CAM_HIT]++;
                                ph.x = res[0]; ph.y = res[1];
                                ph.ux = res[2]; ph.uy = res[3];
                                ph.uz = det->opt_kind == 1 ? res[4] : -res[4];    /* mirror: towards +w; lens: towards -w */
                                ph.t += res[5] / ORC_C_M_PER_NS;
                            }
                        }
                        if (det->cam_enabled) {
                            ph.pix = orc_camera_pixel(det, ua);
                            double tb = floor((ph.t - det->t_ref_ns) / det->t_bin_ns);
                            if (ph.pix >= 0 && tb >= 0 && tb < det->n_tbins) {
                                ph.tbin = (int32_t)tb;
                                lc[ORC_CNT_CAM_HIT]++;
                                if (hist) {
                                    #pragma omp atomic
                                    hist[(size_t)ph.pix * det->n_tbins + ph.tbin] += ph.weight;
                                }
                            }
                        }
                    }
                }
            store:
                if (record_mode == 1 && photons && offsets) photons[offsets[i] + j] = ph;
            }
        }
        #pragma omp critical
        for (int k = 0; k < ORC_N_COUNTERS; ++k) cnt[k] += lc[k];
    }
    if (counters) for (int k = 0; k < ORC_N_COUNTERS; ++k) counters[k] += cnt[k];
    return err;
}

int orc_sizeof_photon(void) { return (int)sizeof(orc_photon); }
/* harness only (no arithmetic): threads of the next orc_run; n <= 0 restores the OpenMP default; returns what is in force */
#ifdef _OPENMP
#include <omp.h>
int orc_set_threads(int n) { omp_set_num_threads(n > 0 ? n : omp_get_num_procs()); return omp_get_max_threads(); }
#else
int orc_set_threads(int n) { (void)n; return 1; }
#endif
int orc_n_counters(void) { return ORC_N_COUNTERS; }

/* ------------------------------------------------------------------ sub-stepping (row f2, reading R16)
 * Thesis sec. 4.2.1: the photon generation needs linear track pieces that follow the
 * physical path to the resolution of the telescopes (0.02 deg ~ 34.9 cm per km, 500 ps ~ 15 cm,
 * P:716); "a secondary loop was introduced to step through the physically calculated particle path to
 * generate a sequence of linear tracks with sufficient accuracy", with the magnetic deflection given
 * by f_mag : [0,1] -> R^3.  Reading: uniform field B, so f_mag is the helix
 *   P(s) = P_par + |P_perp| (e1 cos(kappa s) + e2 sin(kappa s)),
 *   X(s) = A + P_par s + (|P_perp| / kappa) (e1 sin(kappa s) + e2 (1 - cos(kappa s))),
 * kappa = 0.299792458 q B[T] / p[GeV/c] per metre, e1 = P_perp/|P_perp|, e2 = e1 x B/|B|;
 * the arc of length L is cut into n = ceil(L / sqrt(8 tol / curvature)) equal pieces (sagitta of each
 * chord <= tol, curvature = |kappa| |P_perp|), each piece becoming the chord from X(s_i) to X(s_i+1)
 * with the clock t0 + s_i/(beta c).  Multiple scattering sub-steps are not built.
 * Returns the number of pieces (1..max_sub); if seg_out != NULL writes 10 floats per piece:
 * x y z dx dy dz len beta t0 charge. */
int32_t orc_substep_track(const double A[3], const double Pin[3], double L, double beta, double t0, double charge,
                          double p_GeV, const double B[3], double tol_m, int32_t max_sub, float *seg_out)
{
    double P[3] = { Pin[0], Pin[1], Pin[2] };
    norm3(P);
    double Bn = sqrt(B[0]*B[0] + B[1]*B[1] + B[2]*B[2]);
    double kappa = (Bn > 0.0 && p_GeV > 0.0) ? 0.299792458 * charge * Bn / p_GeV : 0.0;
    double bh[3] = { 0, 0, 1 };
    if (Bn > 0.0) { bh[0] = B[0]/Bn; bh[1] = B[1]/Bn; bh[2] = B[2]/Bn; }
    double ppar = P[0]*bh[0] + P[1]*bh[1] + P[2]*bh[2];
    double Pp[3] = { P[0] - ppar*bh[0], P[1] - ppar*bh[1], P[2] - ppar*bh[2] };
    double pperp = sqrt(Pp[0]*Pp[0] + Pp[1]*Pp[1] + Pp[2]*Pp[2]);
    double curv = fabs(kappa) * pperp;
    int32_t n = 1;
    if (curv > 0.0 && L > 0.0) {
        double lmax = sqrt(8.0 * tol_m / curv);
        double nn = ceil(L / lmax);
        n = nn < 1.0 ? 1 : (nn > (double)max_sub ? max_sub : (int32_t)nn);
    }
    if (!seg_out) return n;
    double e1[3] = { 1, 0, 0 }, e2[3] = { 0, 1, 0 };
    if (pperp > 0.0) {
        for (int k = 0; k < 3; ++k) e1[k] = Pp[k] / pperp;
        e2[0] = e1[1]*bh[2] - e1[2]*bh[1]; e2[1] = e1[2]*bh[0] - e1[0]*bh[2]; e2[2] = e1[0]*bh[1] - e1[1]*bh[0];
    }
    double Xp[3], Xn[3];
    for (int i = 0; i <= n; ++i) {
        double s = L * (double)i / (double)n;
        for (int k = 0; k < 3; ++k) {
            double bend = (curv > 0.0) ? (pperp / kappa) * (e1[k] * sin(kappa * s) + e2[k] * (1.0 - cos(kappa * s)))
                                       : pperp * e1[k] * s;
            Xn[k] = A[k] + ppar * bh[k] * s + bend;
        }
        if (i > 0) {
            double d[3] = { Xn[0]-Xp[0], Xn[1]-Xp[1], Xn[2]-Xp[2] };
            double len = sqrt(d[0]*d[0] + d[1]*d[1] + d[2]*d[2]);
            float *o = seg_out + 10 * (size_t)(i - 1);
            double s0 = L * (double)(i - 1) / (double)n;
            o[0] = (float)Xp[0]; o[1] = (float)Xp[1]; o[2] = (float)Xp[2];
            o[3] = (float)(d[0]/len); o[4] = (float)(d[1]/len); o[5] = (float)(d[2]/len);
            o[6] = (float)len; o[7] = (float)beta; o[8] = (float)(t0 + s0 / (beta * ORC_C_M_PER_NS)); o[9] = (float)charge;
        }
        for (int k = 0; k < 3; ++k) Xp[k] = Xn[k];
    }
    return n;
}

/* ------------------------------------------------------------------ multiple-scattering sub-steps (R18)
 * Thesis P:738-746: "instead of calculating the multiple scattering path deviation to the next
 * interaction in a single step, several substeps could be sampled according to the required precision
 * and stored ... the first approach is used ... due to the additional displacement included, which
 * emulates a random walk between each substep"; the angular law comes from an approximation "which
 * employs the initial energy and the particles traversed grammage", Highland or Moliere.  The thesis
 * calls PROPOSAL for it; reading: Highland's width in the PDG (Lynch-Dahl) form
 *   theta0 = 13.6 MeV / (beta c p) |z| sqrt(t) (1 + 0.038 ln(t z^2 / beta^2)),  t = x / X0,
 * per sub-step of arc length ds and grammage x = rho(h_mid) ds, and per transverse plane the correlated
 * Gaussian pair  theta = z2 theta0,  y = (z1/sqrt(12) + z2/2) ds theta0  (z1, z2 ~ N(0,1), Box-Muller on
 * the uniforms of Philox counter (piece, track id, stream 16)).  The magnetic step of R16 is applied
 * first (exact rotation about B), then the offset and the deflection. */
double orc_highland_theta0(double beta, double p_GeV, double charge, double t)
{
    if (!(t > 0.0) || !(p_GeV > 0.0)) return 0.0;
    double corr = 1.0 + 0.038 * log(t * charge * charge / (beta * beta));
    if (corr < 0.0) corr = 0.0;
    return 0.0136 / (beta * p_GeV) * fabs(charge) * sqrt(t) * corr;
}

/* density [g/cm^2 per m] of the cell of the overburden table that holds height h (X_v is linear per cell) */
static double cell_density(const orc_atmosphere *atm, double h)
{
    if (!atm->overburden || atm->model == 0) return 0.0;
    double f = (h - atm->h0) / atm->dh;
    if (f < 0.0) f = 0.0;
    if (f > (double)(atm->n_nodes - 1)) f = (double)(atm->n_nodes - 1);
    int k = (int)floor(f);
    if (k > atm->n_nodes - 2) k = atm->n_nodes - 2;
    return ((double)atm->overburden[k] - (double)atm->overburden[k + 1]) / atm->dh;
}

int32_t orc_substep_track_ms(const orc_atmosphere *atm, const double A[3], const double Pin[3], double L, double beta,
                             double t0, double charge, double p_GeV, const double B[3], double tol_m,
                             double ms_max_step_m, double ms_X0, uint64_t seed, uint64_t track_id,
                             int32_t max_sub, float *seg_out)
{
    int32_t n = orc_substep_track(A, Pin, L, beta, t0, charge, p_GeV, B, tol_m, max_sub, NULL);
    if (ms_max_step_m > 0.0 && L > 0.0) {
        double nn = ceil(L / ms_max_step_m);
        int32_t n2 = nn > (double)max_sub ? max_sub : (int32_t)nn;
        if (n2 > n) n = n2;
    }
    if (!seg_out) return n;
    double P[3] = { Pin[0], Pin[1], Pin[2] }, X[3] = { A[0], A[1], A[2] };
    norm3(P);
    double Bn = sqrt(B[0]*B[0] + B[1]*B[1] + B[2]*B[2]);
    double kappa = (Bn > 0.0 && p_GeV > 0.0) ? 0.299792458 * charge * Bn / p_GeV : 0.0;
    double bh[3] = { 0, 0, 1 };
    if (Bn > 0.0) { bh[0] = B[0]/Bn; bh[1] = B[1]/Bn; bh[2] = B[2]/Bn; }
    const double ds = L / (double)n;
    for (int i = 0; i < n; ++i) {
        /* magnetic step: P' = P_par + cos(k ds) P_perp + sin(k ds) (P_perp x b), displacement = its integral */
        double ppar = P[0]*bh[0] + P[1]*bh[1] + P[2]*bh[2];
        double Pp[3] = { P[0] - ppar*bh[0], P[1] - ppar*bh[1], P[2] - ppar*bh[2] };
        double Pc[3] = { Pp[1]*bh[2] - Pp[2]*bh[1], Pp[2]*bh[0] - Pp[0]*bh[2], Pp[0]*bh[1] - Pp[1]*bh[0] };
        double dX[3], Pn[3];
        double sn = sin(kappa * ds), cs = cos(kappa * ds);
        for (int k = 0; k < 3; ++k) {
            if (kappa != 0.0) {
                dX[k] = ppar * bh[k] * ds + (sn * Pp[k] + (1.0 - cs) * Pc[k]) / kappa;
                Pn[k] = ppar * bh[k] + cs * Pp[k] + sn * Pc[k];
            } else { dX[k] = P[k] * ds; Pn[k] = P[k]; }
        }
        /* multiple scattering of the piece */
        double mid[3] = { X[0] + 0.5*dX[0], X[1] + 0.5*dX[1], X[2] + 0.5*dX[2] };
        double rho = cell_density(atm, orc_height(atm, mid));
        double th0 = orc_highland_theta0(beta, p_GeV, charge, rho * ds / ms_X0);
        double u[4];
        orc_draw(seed, track_id, (uint32_t)i, 16u, u);
        double r1 = sqrt(-2.0 * log(u[0])), r2 = sqrt(-2.0 * log(u[2]));
        double z1 = r1 * cos(2.0 * ORC_PI * u[1]), z2 = r1 * sin(2.0 * ORC_PI * u[1]);
        double z3 = r2 * cos(2.0 * ORC_PI * u[3]), z4 = r2 * sin(2.0 * ORC_PI * u[3]);
        double ea[3] = { Pn[1], -Pn[0], 0.0 };                        /* P' x z */
        double na = sqrt(ea[0]*ea[0] + ea[1]*ea[1]);
        if (na < 1e-12) { ea[0] = 1.0; ea[1] = 0.0; na = 1.0; }
        ea[0] /= na; ea[1] /= na;
        double eb[3] = { Pn[1]*ea[2] - Pn[2]*ea[1], Pn[2]*ea[0] - Pn[0]*ea[2], Pn[0]*ea[1] - Pn[1]*ea[0] };
        double ya = (z1 / sqrt(12.0) + 0.5 * z2) * ds * th0, yb = (z3 / sqrt(12.0) + 0.5 * z4) * ds * th0;
        double Xe[3], Pe[3];
        for (int k = 0; k < 3; ++k) {
            Xe[k] = X[k] + dX[k] + ya * ea[k] + yb * eb[k];
            Pe[k] = Pn[k] + z2 * th0 * ea[k] + z4 * th0 * eb[k];
        }
        norm3(Pe);
        double d[3] = { Xe[0]-X[0], Xe[1]-X[1], Xe[2]-X[2] };
        double len = sqrt(d[0]*d[0] + d[1]*d[1] + d[2]*d[2]);
        float *o = seg_out + 10 * (size_t)i;
        o[0] = (float)X[0]; o[1] = (float)X[1]; o[2] = (float)X[2];
        o[3] = (float)(d[0]/len); o[4] = (float)(d[1]/len); o[5] = (float)(d[2]/len);
        o[6] = (float)len; o[7] = (float)beta; o[8] = (float)(t0 + (double)i * ds / (beta * ORC_C_M_PER_NS)); o[9] = (float)charge;
        for (int k = 0; k < 3; ++k) { X[k] = Xe[k]; P[k] = Pe[k]; }
    }
    return n;
}
