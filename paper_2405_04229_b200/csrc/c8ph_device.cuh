// c8ph_device.cuh — launch-argument structs shared by the host API and the kernels of libc8ph.
// (Internal to the CUDA library; the CPU oracle under oracle/ shares nothing with this.)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "../../include/c8ph.h"

namespace c8ph {


struct DevAtm {
    int model;              // C8PH_ATM_*
    int n_nodes;            // nodes of the n(h) grid (>= 2; homogeneous: 2 identical nodes)
    int n_pad;              // floats per table array, multiple of 4 (16 B, bulk-copy granule)
    float h0, dh, inv_dh, h_top;
    float f_max;            // (float)(n_nodes - 1)
    const float *eta;       // DEVICE [n_pad] refractivity n-1 at the nodes
    const float *xv;        // DEVICE [n_pad] vertical overburden at the nodes (zeros if none)
    const float *dxv;       // DEVICE [n_pad] X_v(node k) - X_v(node k+1)
    double R, h_obs, Rg;    // Earth radius, observation altitude, R + h_obs
    float eta_g;            // refractivity at the observation level
    float ray_inv_X;        // 1 / X_R, 0 = Rayleigh off
    float ray_lambda;       // lambda_R [nm]
    float aer_L, aer_H, aer_lambda, aer_angstrom;
    const float *aexp;      // DEVICE [n_pad] aerosol column A(h_k) = (H/L) exp(-h_k/H) at the nodes (zeros without aerosol)
    float aer_HL, aer_invH, aer_Ag;   // H/L, 1/H, A(h_obs)
    // planar layered sum in closed form: mom[q * n_pad + k] = sum over the layers between the observation level and
    // node k of thickness * nu_l^(q+1) (q = 0..3) and of dX_v * n_l * nu_l^(q-4) (q = 4..7), nu_l = n_l^2 - 1 at the
    // layer's mid height (c8ph_init_atmosphere)
    const float *mom;
    float nu_span;                    // max nu - min nu over the table: bounds the expansion parameter
    int n_ext;              // tabulated extinction: wavelength nodes (0: off)
    float ext_l0, ext_inv_dl;
    const float *ext;       // DEVICE [n_ext][n_nodes] vertical optical depth obs level -> node
    float xv_g;             // X_v at the observation level
};

struct DevTable {
    int n_h, n_zen;
    float h_max, zen_max;           // [m], [rad]
    float inv_dh, inv_dz;           // (n_h-1)/h_max, (n_zen-1)/zen_max
    float f_max, g_max;             // (float)(n_h-1), (float)(n_zen-1)
    const float4 *hot;              // DEVICE [n_h][n_zen] = (dd, dt, X_slant, tau_aer)
    const float *full;              // DEVICE [n_h][n_zen][5]
    cudaTextureObject_t tex;        // the hot texels as a 2-D float4 texture (x: zenith node, y: height node), linear filter
    // flat-plane table (R21): [n_rho][n_h][n_zen] texels; E = (dd, dt, X_slant, tau_aer) even in the pointing angle,
    // O = (dd odd, dt odd, transverse displacement P, 0)
    int n_rho;
    float rho_max, inv_drho, e_max;
    const float4 *flatE, *flatO;
    // cylindrical model (R24): [n_c][n_h][n_zen] texels (dd, dt, X_slant, across displacement / (sin psi cos psi))
    int n_c;
    float c_max;                    // (float)(n_c - 1)
    const float4 *cyl;
};

// Uniform grid over the telescope array.  Every cell lists the telescopes that a point of the cell
// can reach, SORTED by a lower-bound key, together with the smallest key of the cell, so that the
// common "nothing near" case exits after one load (hit grid: one byte per cell, the key quantised
// downwards, so that the cells under a shower stay in L1) and a search stops at the first key above
// the photon's threshold.
//   hit grid: key = dist(cell rectangle, centre_xy) / (r + |z|);  a photon with direction u at a
//             point of the cell can hit the sphere only if key <= 1/|u_z|
//   LV2 grid: key = dist(cell rectangle, centre_xy) [m];  the point can be within r/|u_z| + margin
//             of the centre only if key <= r_max/|u_z| + margin
constexpr float kHitKeyScale = 64.f;    // quantisation of the hit grid's per-cell smallest key (one byte per cell)

struct DevGrid {
    float x0, y0, inv_cs;
    int nx, ny;
    const float *kmin;              // DEVICE [nx*ny]   smallest key of the cell (+inf: empty)
    const uint8_t *kq;              // hit grid only, DEVICE [nx*ny]: floor(kmin * kHitKeyScale), 254 at most; 255: empty
    const float4 *knear;            // LV2 grid only, DEVICE [nx*ny]: (kmin, x, y, r) = smallest key of the cell and the telescope
                                    // nearest to the cell (least dist(cell centre, centre_k) - r_k), tested in line before any list
                                    // walk; empty cell: (+inf, far away, far away, 0)
    const float4 *first;            // hit grid only, DEVICE [nx*ny]: (x, y, z, r) of the cell's first listed telescope (smallest key)
    const int2 *first_kn;           // hit grid only, DEVICE [nx*ny]: (its index, number of telescopes listed for the cell); finish()
                                    // issues both loads before its arithmetic, so the usual one-telescope cell costs one memory latency
    const int *start;               // DEVICE [nx*ny+1] CSR offsets into items
    const float2 *items;            // DEVICE (key, telescope index as int bits), ascending key per cell
};

struct DevDet {
    int hist_nx, hist_ny;
    float hist_x0, hist_y0, hist_cell, hist_inv_cell;
    int n_tel;
    const float4 *tel;              // DEVICE [n_tel]
    int use_grid;                   // 0: brute force over all telescopes
    float grid_min_cos;             // the grids are valid for |u_z| >= grid_min_cos
    float r_max;                    // largest telescope radius (LV2 threshold)
    DevGrid lv2, hit;
    double r_array;                 // bounding radius of telescopes + histogram about the origin
    int cam_enabled, cam_rows, cam_cols, n_tbins;
    float cam_w[3], cam_r[3], cam_u[3];   // camera frame: axis, right, up
    float cam_pitch, cam_inv_pitch;       // [rad]
    double t_ref;
    float t_bin, inv_t_bin;
    int opt_enabled;                      // last-mile optics inside the bounding spheres
    float opt_w[3], opt_r[3], opt_u[3];   // telescope frame: pointing axis, right, up
    float opt_f, opt_rm2, opt_rc2;        // focal length, mirror radius^2, camera radius^2
    int opt_kind, opt_n_abs;              // R22: 1 = plano-convex lens instead of the mirror; absorbing capsules
    float opt_lens_roc, opt_lens_t, opt_lens_n;
    float opt_abs[8][7];                  // capsule axis end points and radius, telescope frame about the sphere centre
};

struct DevRun {
    int emit, trace, trans, write, lv1, lv2;
    float il1, il2;                 // 1/lambda_min, 1/lambda_max  [1/nm]
    float w;                        // bunch weight
    double yield_k;                 // Cherenkov: 2 pi alpha (1/l1 - 1/l2) [1/m]
    double lv1_margin;
    float lv2_margin;
    float box_x0, box_x1, box_y0, box_y1;   // LV2: histogram extent widened by the margin (empty if no grid)
    float inv_Rg;                   // 1 / (R + h_obs)
    float hit_infl;                 // telescope pre-test: 1/|u_z| inflated to cover the refraction rotation
    int hit_brute;                  // 1: the rotation can exceed what the hit grid lists cover -> search all
    double fluor_yield, aim_factor;
    int n_lines;
    const float *line_nm, *line_cdf;      // DEVICE
    float disp_b, disp_c0;          // dispersion D(k) = disp_c0 + disp_b k^2, k = 1/lambda [1/nm]; disp_b = 0: off
    double disp_k0sq;               // 1/lambda0^2
    double il1_d, il2_d;            // 1/lambda_min, 1/lambda_max in fp64 (dispersive yield integral)
    int force_generic;              // validation / timing: use the generic kernel variant even for the production setting
    int flat_plane;                 // spherical model: exact step from the observation sphere to the plane z = 0 (R19)
    int n_eff;                      // detector efficiency table (0: off)
    float eff_l0, eff_inv_dl;       // grid origin [nm], 1 / spacing
    const float *eff;               // DEVICE [n_eff]
    uint32_t key0[10], key1[10];    // Philox round keys
    int64_t n_seg, seg_id_base;
    uint32_t local_base;            // added to the call-local segment index written into photon records
    c8ph_segments seg;              // DEVICE pointers
    c8ph_outputs out;               // DEVICE pointers
    unsigned long long *cursor;     // DEVICE work cursor (segments)
    void *slots;                    // DEVICE scratch: 32 prepared-segment slots per resident warp
    void *qring;                    // DEVICE scratch: candidate queues of the resident warps when they live in global memory (C8PH_QUEUE_GLOBAL)
    int segs_per_grab;              // segments one warp prepares per grab (1..32)
};

// Constants every photon reads, copied by the host from the structs below into 16-byte groups in
// the order of use, so the kernel fetches them with few wide constant loads.
struct alignas(16) HotConst {
    uint2 key[10];                                      // Philox round keys (k0, k1) per round
    float eta_h0, eta_inv_dh, eta_fmax; int eta_kmax;   // n(h) lookup: origin, 1/dh, n_nodes-1, n_nodes-2
    const float *eta; float il1, dil;                   // n(h) nodes; 1/lambda_min, 1/lambda_min - 1/lambda_max
    float box_x0, box_x1, box_y0, box_y1;               // LV2 keep-box
    float lv2_margin, r_max, grid_min_cos, hit_infl_q;  // hit_infl_q = DevRun::hit_infl * kHitKeyScale
    float ray_lambda, ray_k, w, pad0;                   // ray_k = log2(e) / X_R
    float hit_x0, hit_y0, hit_inv_cs; int hit_nx;       // hit grid
    int hit_ny; float hist_inv_cell; int hist_nx, hist_ny;
    const uint8_t *hit_kq; float *hist;
};

struct KArgs {
    HotConst hc;
    DevAtm atm;
    DevTable tab;
    DevDet det;
    DevRun run;
};

struct TableBuildArgs {
    DevAtm atm;
    int n_h, n_zen, substeps;
    double h_max, zen_max;
    float *full;                    // [n_h][n_zen][5]
    float4 *hot;                    // [n_h][n_zen]
    int n_rho;                      // flat-plane table (R21): nodes in rho, 0: none
    double rho_max;
    float4 *flatE, *flatO;          // [n_rho][n_h][n_zen] each
    int n_c;                        // cylindrical model's table (R24): nodes in c = cos^2(psi), 0: none
    float4 *cyl;                    // [n_c][n_h][n_zen]
};

struct SubstepArgs {
    c8ph_segments trk;              // DEVICE
    const float *p_GeV;
    long long n;
    double B[3], Bn;                // field [T] and its norm
    double tol;
    int max_sub;
    long long *offsets;             // [n+1]
    unsigned long long *clipped;    // DEVICE counter (plan only) or NULL: += tracks clipped to max_sub pieces
    c8ph_segments_out out;          // DEVICE (fill only)
    int ms_enabled;                 // multiple-scattering sub-steps (R18)
    double ms_max_step, ms_X0;
    uint2 key[10];                  // Philox round keys
    long long id_base;
    DevAtm atm;                     // density from the overburden table
};

// kernels / launchers (c8ph_kernels.cu)
cudaError_t launch_emit_propagate(const KArgs &a, int n_sm, cudaStream_t st);
cudaError_t launch_build_table(const TableBuildArgs &a, cudaStream_t st);
size_t emit_smem_bytes(const KArgs &a);
size_t segment_slot_bytes(int n_sm);
size_t queue_ring_bytes(int n_sm);
cudaError_t launch_substep_plan(const SubstepArgs &a, long long *block_sums, cudaStream_t st);
cudaError_t launch_substep_fill(const SubstepArgs &a, int n_sm, cudaStream_t st);
size_t substep_scratch_elems(long long n);

}  // namespace c8ph
