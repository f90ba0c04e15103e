// c8ph_substep.cu — sub-stepping of particle tracks along the magnetically deflected path
// (thesis sec. 4.2.1): the step before the hot path.  Three small kernels plan the pieces
// (count per track + exclusive prefix sum), one fills them (a warp expands 32 tracks cooperatively).  fp64: the pieces
// must reproduce km-scale positions to well below the 15 cm resolution the thesis quotes.
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <cmath>
#include "c8ph_device.cuh"
#include "c8ph_philox.cuh"

namespace c8ph {

namespace {

constexpr int kScanThreads = 1024;
constexpr float kMsFp32Theta0 = 0.03f;      // multiple scattering: fp32 normal deviates below this theta_0 [rad]

struct Helix {
    double A[3], bh[3], e1[3], e2[3];
    double ppar, pperp, kappa, curv, L, beta, t0, charge;
};

// helix of track i (R16): P(s) = P_par + |P_perp| (e1 cos(kappa s) + e2 sin(kappa s))
__device__ __forceinline__ Helix helix_of(const SubstepArgs &a, long long i)
{
    Helix h;
    h.A[0] = a.trk.x[i]; h.A[1] = a.trk.y[i]; h.A[2] = a.trk.z[i];
    double P[3] = {a.trk.dx[i], a.trk.dy[i], a.trk.dz[i]};
    const double pn = 1.0 / sqrt(P[0] * P[0] + P[1] * P[1] + P[2] * P[2]);
    P[0] *= pn; P[1] *= pn; P[2] *= pn;
    h.L = a.trk.len[i]; h.beta = a.trk.beta[i]; h.t0 = a.trk.t0[i]; h.charge = a.trk.charge[i];
    const double p = a.p_GeV[i];
    h.kappa = (a.Bn > 0.0 && p > 0.0) ? 0.299792458 * h.charge * a.Bn / p : 0.0;
    h.bh[0] = 0.0; h.bh[1] = 0.0; h.bh[2] = 1.0;
    if (a.Bn > 0.0) { h.bh[0] = a.B[0] / a.Bn; h.bh[1] = a.B[1] / a.Bn; h.bh[2] = a.B[2] / a.Bn; }
    h.ppar = P[0] * h.bh[0] + P[1] * h.bh[1] + P[2] * h.bh[2];
    const double Pp[3] = {P[0] - h.ppar * h.bh[0], P[1] - h.ppar * h.bh[1], P[2] - h.ppar * h.bh[2]};
    h.pperp = sqrt(Pp[0] * Pp[0] + Pp[1] * Pp[1] + Pp[2] * Pp[2]);
    h.curv = fabs(h.kappa) * h.pperp;
    h.e1[0] = 1.0; h.e1[1] = 0.0; h.e1[2] = 0.0; h.e2[0] = 0.0; h.e2[1] = 1.0; h.e2[2] = 0.0;
    if (h.pperp > 0.0) {
        for (int k = 0; k < 3; ++k) h.e1[k] = Pp[k] / h.pperp;
        h.e2[0] = h.e1[1] * h.bh[2] - h.e1[2] * h.bh[1];
        h.e2[1] = h.e1[2] * h.bh[0] - h.e1[0] * h.bh[2];
        h.e2[2] = h.e1[0] * h.bh[1] - h.e1[1] * h.bh[0];
    }
    return h;
}

// number of pieces: sagitta L_piece^2 curvature / 8 <= tol, and (multiple scattering) L_piece <= ms_max_step
// `clipped` is set when the bounds ask for more than max_sub pieces (the track then gets max_sub: counted, never silent)
__device__ __forceinline__ int pieces_of(const Helix &h, const SubstepArgs &a, bool *clipped = nullptr)
{
    int n = 1;
    bool cl = false;
    if (h.curv > 0.0 && h.L > 0.0) {
        const double nn = ceil(h.L / sqrt(8.0 * a.tol / h.curv));
        cl = nn > (double)a.max_sub;
        n = nn < 1.0 ? 1 : (cl ? a.max_sub : (int)nn);
    }
    if (a.ms_enabled && a.ms_max_step > 0.0 && h.L > 0.0) {
        const double nn = ceil(h.L / a.ms_max_step);
        cl = cl || nn > (double)a.max_sub;
        const int n2 = nn > (double)a.max_sub ? a.max_sub : (int)nn;
        if (n2 > n) n = n2;
    }
    if (clipped) *clipped = cl;
    return n;
}

__device__ __forceinline__ void point_on(const Helix &h, double s, double X[3])
{
    double sn, cs;
    sincos(h.kappa * s, &sn, &cs);
    for (int k = 0; k < 3; ++k) {
        const double bend = h.curv > 0.0 ? (h.pperp / h.kappa) * (h.e1[k] * sn + h.e2[k] * (1.0 - cs)) : h.pperp * h.e1[k] * s;
        X[k] = h.A[k] + h.ppar * h.bh[k] * s + bend;
    }
}

// K1: piece count per track, inclusive scan inside the block, block totals
__global__ void __launch_bounds__(kScanThreads) k_substep_count(const __grid_constant__ SubstepArgs a, long long *block_sums)
{
    __shared__ long long s_warp[32];
    const long long i = (long long)blockIdx.x * kScanThreads + threadIdx.x;
    long long v = 0;
    bool cl = false;
    if (i < a.n) v = pieces_of(helix_of(a, i), a, &cl);
    if (a.clipped) {                                              // tracks that needed more than max_sub pieces
        const unsigned m = __ballot_sync(0xFFFFFFFFu, cl);
        if (m && (threadIdx.x & 31) == 0) atomicAdd(a.clipped, (unsigned long long)__popc(m));
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int d = 1; d < 32; d <<= 1) {
        const long long t = __shfl_up_sync(0xFFFFFFFFu, v, d);
        if (lane >= d) v += t;
    }
    if (lane == 31) s_warp[warp] = v;
    __syncthreads();
    if (warp == 0) {
        long long w = s_warp[lane];
        for (int d = 1; d < 32; d <<= 1) {
            const long long t = __shfl_up_sync(0xFFFFFFFFu, w, d);
            if (lane >= d) w += t;
        }
        s_warp[lane] = w;
    }
    __syncthreads();
    if (warp > 0) v += s_warp[warp - 1];
    if (i < a.n) a.offsets[i + 1] = v;
    if (threadIdx.x == kScanThreads - 1) block_sums[blockIdx.x] = v;
}

// K2: exclusive scan of the block totals (one block, chunks of 1024 with a carry)
__global__ void __launch_bounds__(kScanThreads) k_substep_scan_blocks(long long *block_sums, long long n_blocks)
{
    __shared__ long long s_warp[32];
    __shared__ long long s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (long long base = 0; base < n_blocks; base += kScanThreads) {
        const long long i = base + threadIdx.x;
        const long long own = i < n_blocks ? block_sums[i] : 0;
        long long v = own;
        for (int d = 1; d < 32; d <<= 1) {
            const long long t = __shfl_up_sync(0xFFFFFFFFu, v, d);
            if (lane >= d) v += t;
        }
        if (lane == 31) s_warp[warp] = v;
        __syncthreads();
        if (warp == 0) {
            long long w = s_warp[lane];
            for (int d = 1; d < 32; d <<= 1) {
                const long long t = __shfl_up_sync(0xFFFFFFFFu, w, d);
                if (lane >= d) w += t;
            }
            s_warp[lane] = w;
        }
        __syncthreads();
        if (warp > 0) v += s_warp[warp - 1];
        const long long carry = s_carry;
        if (i < n_blocks) block_sums[i] = carry + v - own;             // exclusive
        __syncthreads();
        if (threadIdx.x == kScanThreads - 1) s_carry = carry + v;
        __syncthreads();
    }
}

// K3: add the block offsets
__global__ void __launch_bounds__(kScanThreads) k_substep_add_blocks(const __grid_constant__ SubstepArgs a, const long long *block_sums)
{
    const long long i = (long long)blockIdx.x * kScanThreads + threadIdx.x;
    if (i < a.n) a.offsets[i + 1] += block_sums[blockIdx.x];
    if (i == 0) a.offsets[0] = 0;
}

// fill: a warp takes 32 consecutive tracks and expands them cooperatively.  First every lane prepares ONE track (helix,
// piece length, the half-angle of a piece, chord length and the constant part of the chord direction: everything that
// is the same for all pieces of a track) into the warp's shared-memory table; then lane l writes the pieces base + l,
// base + l + 32, ... of the group (coalesced), the owner track of a piece found by a five-step search over the group's
// 32 start offsets held one per lane (shuffles, no global binary search).  A piece costs one fp64 sincos:
//   X(s) = A + v_b s + R (e1 sin(kappa s) + e2 (1 - cos(kappa s))),  v_b = P_par b, R = |P_perp| / kappa,
//   piece j of m: D = L / m, s0 = j D, delta = kappa D / 2,
//   X1 - X0 = v_b D + 2 R sin(delta) (e1 cos(kappa s0 + delta) + e2 sin(kappa s0 + delta)),
//   |X1 - X0|^2 = (P_par D)^2 + (2 R sin(delta))^2          (b, e1, e2 orthonormal: the same for every piece),
// with sin / 1 - cos of kappa s0 from the half angle (2 Sh Ch, 2 Sh^2: no cancellation for stiff tracks).
constexpr int kFillThreads = 128;
enum { TF_AX, TF_AY, TF_AZ, TF_VX, TF_VY, TF_VZ, TF_R1X, TF_R1Y, TF_R1Z, TF_R2X, TF_R2Y, TF_R2Z, TF_UX, TF_UY, TF_UZ,
       TF_HK, TF_D, TF_SD, TF_CD, TF_Q, TF_T0, TF_IBC, TF_N };

__global__ void __launch_bounds__(kFillThreads, 6) k_substep_fill(const __grid_constant__ SubstepArgs a)
{
    __shared__ double s_trk[kFillThreads / 32][TF_N][32];
    __shared__ float s_trkf[kFillThreads / 32][3][32];                 // chord length, beta, charge
    const unsigned FULL = 0xFFFFFFFFu;
    const int lane = threadIdx.x & 31;
    double (*T)[32] = s_trk[threadIdx.x >> 5];
    float (*Tf)[32] = s_trkf[threadIdx.x >> 5];
    const long long n_groups = (a.n + 31) >> 5;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long grp = warp0; grp < n_groups; grp += n_warps) {
        const long long i0 = grp << 5;
        const long long base = a.offsets[i0];
        const long long i_me = i0 + lane < a.n ? i0 + lane : a.n;
        const long long i_end = i0 + 32 < a.n ? i0 + 32 : a.n;
        const int rel = (int)(a.offsets[i_me] - base);                 // start of my track within the group (<= 32 * max_sub)
        const int total = (int)(a.offsets[i_end] - base);              // lanes beyond the last track hold `total`
        __syncwarp();                                                  // the table of the previous group is no longer read
        if (i0 + lane < a.n) {
            const Helix h = helix_of(a, i0 + lane);
            const int m = (int)(a.offsets[i0 + lane + 1] - a.offsets[i0 + lane]);
            const double D = h.L / (double)m;
            const bool bent = h.curv > 0.0;
            const double R = bent ? h.pperp / h.kappa : 0.0;
            double sd = 0.0, cd = 1.0;
            if (bent) sincos(0.5 * h.kappa * D, &sd, &cd);
            const double chord = 2.0 * R * sd;                         // signed
            const double len = bent ? sqrt(h.ppar * h.ppar * D * D + chord * chord) : D;
            const double il = len > 0.0 ? 1.0 / len : 0.0;
            for (int k = 0; k < 3; ++k) {
                const double P = h.ppar * h.bh[k] + h.pperp * h.e1[k];  // direction of flight at the track start
                T[TF_AX + k][lane] = h.A[k];
                T[TF_VX + k][lane] = bent ? h.ppar * h.bh[k] : P;
                T[TF_R1X + k][lane] = R * h.e1[k];
                T[TF_R2X + k][lane] = R * h.e2[k];
                T[TF_UX + k][lane] = len > 0.0 ? (bent ? h.ppar * h.bh[k] * D * il : P) : P;   // zero length: direction of flight
            }
            T[TF_HK][lane] = bent ? 0.5 * h.kappa : 0.0;
            T[TF_D][lane] = D;
            T[TF_SD][lane] = sd; T[TF_CD][lane] = cd;
            T[TF_Q][lane] = 2.0 * sd * il;
            T[TF_T0][lane] = h.t0;
            T[TF_IBC][lane] = 1.0 / (h.beta * 0.299792458);
            Tf[0][lane] = (float)len; Tf[1][lane] = (float)h.beta; Tf[2][lane] = (float)h.charge;
        }
        __syncwarp();
        for (int p0 = 0; p0 < total; p0 += 32) {
            const int p = p0 + lane;
            int lo = 0;                                                // largest t with rel[t] <= p
#pragma unroll
            for (int step = 16; step >= 1; step >>= 1) {
                const int v = __shfl_sync(FULL, rel, (lo + step) & 31);
                if (v <= p) lo += step;
            }
            const int r0 = __shfl_sync(FULL, rel, lo);
            if (p < total) {
                const double s0 = T[TF_D][lo] * (double)(p - r0);
                double Sh, Ch;
                sincos(T[TF_HK][lo] * s0, &Sh, &Ch);
                const double sn0 = 2.0 * Sh * Ch, omc = 2.0 * Sh * Sh, cs0 = 1.0 - omc;
                const double sd = T[TF_SD][lo], cd = T[TF_CD][lo], q = T[TF_Q][lo];
                const double Sm = fma(sn0, cd, cs0 * sd), Cm = fma(cs0, cd, -sn0 * sd);
                const long long g = base + p;
                a.out.x[g] = (float)fma(T[TF_R2X][lo], omc, fma(T[TF_R1X][lo], sn0, fma(T[TF_VX][lo], s0, T[TF_AX][lo])));
                a.out.y[g] = (float)fma(T[TF_R2Y][lo], omc, fma(T[TF_R1Y][lo], sn0, fma(T[TF_VY][lo], s0, T[TF_AY][lo])));
                a.out.z[g] = (float)fma(T[TF_R2Z][lo], omc, fma(T[TF_R1Z][lo], sn0, fma(T[TF_VZ][lo], s0, T[TF_AZ][lo])));
                a.out.dx[g] = (float)fma(q, fma(T[TF_R1X][lo], Cm, T[TF_R2X][lo] * Sm), T[TF_UX][lo]);
                a.out.dy[g] = (float)fma(q, fma(T[TF_R1Y][lo], Cm, T[TF_R2Y][lo] * Sm), T[TF_UY][lo]);
                a.out.dz[g] = (float)fma(q, fma(T[TF_R1Z][lo], Cm, T[TF_R2Z][lo] * Sm), T[TF_UZ][lo]);
                a.out.len[g] = Tf[0][lo];
                a.out.beta[g] = Tf[1][lo];
                a.out.t0[g] = (float)fma(s0, T[TF_IBC][lo], T[TF_T0][lo]);
                a.out.charge[g] = Tf[2][lo];
                if (a.out.edep) a.out.edep[g] = 0.f;
            }
        }
    }
}

// fill with multiple scattering (R18): the pieces of a track are a random walk, so one thread walks one
// track: exact magnetic rotation of the piece, then Highland's correlated offset / deflection per plane.
// Positions, directions and the rotation are fp64 (km-scale coordinates, errors accumulate along the walk); the four
// standard-normal deviates are formed in fp32 (accurate logf / sqrtf / sincospif, ~2e-7 relative; the uniforms are
// 23-bit values, exact in fp32) where Highland's theta_0 of the piece is below kMsFp32Theta0: their rounding
// multiplies theta_0, so a piece's direction moves by < 1e-8 rad; stiffer kicks (0.35 rad for a 10 MeV electron over
// 25 m of air at sea level) take the fp64 functions.  theta_0 itself is fp32 arithmetic on fp64-derived inputs.
//
// The lanes of a warp walk in lock step, so a warp costs its longest track: a CTA takes 512 consecutive tracks,
// orders them by piece count in shared memory (counting sort, 63 and more pieces in one class; the order inside a
// class is arbitrary and does not matter: every piece has its own place in the output) and hands each warp 32 tracks
// that are neighbours in that order.  Measured on 1e7 tracks with a log-uniform momentum spectrum: 11.6 -> 20.4 active
// lanes per warp instruction.  The chunk size trades balance against the output footprint in flight: a track's run is
// ~40 B per array, so most 32-byte sectors are completed by a neighbouring track that another warp walks later, and
// sectors evicted from L2 half written cost a DRAM read-modify-write (chunks of 256 / 512 / 1024 tracks: 11.1 / 14.3 /
// 18.7 GB of DRAM traffic for 4.7 GB of input + output, 7.7 / 6.9 / 8.0 ms; staging a 256-track chunk's whole output
// in shared memory and writing it as one range brings the traffic to 5.0 GB but costs a CTA-wide barrier per chunk
// behind its longest track: 10.9 ms).
constexpr int kMsThreads = 128, kMsChunk = 512, kMsBins = 64;

// the whole warp calls this; lanes without a track pass valid = false.  Pieces are staged in the warp's shared-memory
// tile (10 fields x 32 tracks x 8 pieces, row pitch 9 floats: conflict-free for lane = track and for the flush) and
// written every 8 pieces by the warp together: a lane's 8 pieces are 32 contiguous bytes per field, so the stores
// fill sectors instead of touching one float of 32 different sectors each.
constexpr int kMsStage = 8, kMsPitch = kMsStage + 1, kMsFields = 10;

__device__ __forceinline__ void ms_walk(const SubstepArgs &a, long long i, bool valid, float *stage)
{
    const unsigned FULL = 0xFFFFFFFFu;
    const int lane = threadIdx.x & 31;
    const DevAtm &atm = a.atm;
    const double inv_dh = 1.0 / (double)atm.dh;
    if (!valid) i = 0;                                               // any readable track; its pieces are not produced
    {
        const Helix h = helix_of(a, i);
        const long long g0 = a.offsets[i];
        const int n_own = (int)(a.offsets[i + 1] - g0);
        const int n = valid ? n_own : 0;
        const int n_max = __reduce_max_sync(FULL, n);
        const double ds = h.L / (double)n_own;
        const double p = a.p_GeV[i];
        const unsigned long long tid = (unsigned long long)(a.id_base + i);
        double X[3] = {h.A[0], h.A[1], h.A[2]};
        double P[3];
        for (int k = 0; k < 3; ++k) P[k] = h.ppar * h.bh[k] + h.pperp * h.e1[k];
        double sn, cs;
        sincos(h.kappa * ds, &sn, &cs);
        const bool bent = h.kappa != 0.0;
        const double ik = bent ? 1.0 / h.kappa : 0.0;
        const double a_s = sn * ik, a_c = (1.0 - cs) * ik;
        // Highland: theta_0 = 0.0136 / (beta p) |z| sqrt(t) (1 + 0.038 ln(t z^2 / beta^2)), t = rho ds / X0
        const bool scat = p > 0.0;
        const double hl_cd = scat ? 0.0136 / (h.beta * p) * fabs(h.charge) : 0.0, hl_zd = h.charge * h.charge / (h.beta * h.beta);
        const float hl_c = (float)hl_cd, hl_z = (float)hl_zd;
        const double t_per_rho = ds / a.ms_X0;
        const double dt_piece = ds / (h.beta * 0.299792458);
        const float beta_f = (float)h.beta, charge_f = (float)h.charge;
        float *mine = stage + lane * kMsPitch;
        for (int j0 = 0; j0 < n_max; j0 += kMsStage) {
          for (int jr = 0; jr < kMsStage && j0 + jr < n_max; ++jr) {
            const int j = j0 + jr;
            if (j >= n) continue;
            const double ppar = P[0] * h.bh[0] + P[1] * h.bh[1] + P[2] * h.bh[2];
            double dX[3], Pn[3];
            if (bent) {
                const double Pp[3] = {P[0] - ppar * h.bh[0], P[1] - ppar * h.bh[1], P[2] - ppar * h.bh[2]};
                const double Pc[3] = {Pp[1] * h.bh[2] - Pp[2] * h.bh[1], Pp[2] * h.bh[0] - Pp[0] * h.bh[2], Pp[0] * h.bh[1] - Pp[1] * h.bh[0]};
                for (int k = 0; k < 3; ++k) {
                    const double par = ppar * h.bh[k];
                    dX[k] = fma(par, ds, fma(a_s, Pp[k], a_c * Pc[k]));
                    Pn[k] = fma(cs, Pp[k], fma(sn, Pc[k], par));
                }
            } else {
                for (int k = 0; k < 3; ++k) { dX[k] = P[k] * ds; Pn[k] = P[k]; }
            }
            // density of the overburden-table cell at the piece's mid height
            const double mz = fma(0.5, dX[2], X[2]);
            double hm = atm.h_obs + mz;
            if (atm.model == C8PH_ATM_SPHERICAL) {
                const double mx = fma(0.5, dX[0], X[0]), my = fma(0.5, dX[1], X[1]);
                hm = sqrt(mx * mx + my * my + (mz + atm.Rg) * (mz + atm.Rg)) - atm.R;
            }
            double th0 = 0.0;
            bool stiff = false;                                   // theta_0 above kMsFp32Theta0: everything in fp64
            if (atm.model != C8PH_ATM_HOMOGENEOUS && scat) {
                double f = (hm - (double)atm.h0) * inv_dh;
                f = fmin(fmax(f, 0.0), (double)(atm.n_nodes - 1));
                const int k = min((int)f, atm.n_nodes - 2);
                const double td = ((double)__ldg(atm.xv + k) - (double)__ldg(atm.xv + k + 1)) * inv_dh * t_per_rho;
                const float t = (float)td;
                if (t > 0.f) {
                    const float th0f = hl_c * sqrtf(t) * fmaxf(fmaf(0.038f, logf(t * hl_z), 1.f), 0.f);
                    stiff = th0f > kMsFp32Theta0;
                    th0 = stiff ? hl_cd * sqrt(td) * fmax(fma(0.038, log(td * hl_zd), 1.0), 0.0) : (double)th0f;
                }
            }
            const uint4 r = philox4x32_10((uint32_t)j, (uint32_t)tid, (uint32_t)(tid >> 32), 16u, a.key);
            // Box-Muller; sin / cos of 2 pi u through sincospi, whose argument 2 u is exact
            double z1, z2, z3, z4;
            if (stiff) {
                auto u01d = [](uint32_t v) { return ((double)(v >> 9) + 0.5) * (1.0 / 8388608.0); };
                const double r1 = sqrt(-2.0 * log(u01d(r.x))), r2 = sqrt(-2.0 * log(u01d(r.z)));
                double s1, c1, s2, c2;
                sincospi(2.0 * u01d(r.y), &s1, &c1);
                sincospi(2.0 * u01d(r.w), &s2, &c2);
                z1 = r1 * c1; z2 = r1 * s1; z3 = r2 * c2; z4 = r2 * s2;
            } else {
                auto u01f = [](uint32_t v) { return ((float)(v >> 9) + 0.5f) * (1.0f / 8388608.0f); };
                const float r1 = sqrtf(-2.0f * logf(u01f(r.x))), r2 = sqrtf(-2.0f * logf(u01f(r.z)));
                float s1, c1, s2, c2;
                sincospif(2.0f * u01f(r.y), &s1, &c1);
                sincospif(2.0f * u01f(r.w), &s2, &c2);
                z1 = (double)(r1 * c1); z2 = (double)(r1 * s1); z3 = (double)(r2 * c2); z4 = (double)(r2 * s2);
            }
            // transverse frame of the rotated direction
            double ea0 = Pn[1], ea1 = -Pn[0];
            const double na2 = ea0 * ea0 + ea1 * ea1;
            if (na2 < 1e-24) { ea0 = 1.0; ea1 = 0.0; }
            else { const double ina = rsqrt(na2); ea0 *= ina; ea1 *= ina; }
            const double eb[3] = {-Pn[2] * ea1, Pn[2] * ea0, Pn[0] * ea1 - Pn[1] * ea0};
            const double dsth = ds * th0;
            const double ya = fma(z1, 0.28867513459481287, 0.5 * z2) * dsth, yb = fma(z3, 0.28867513459481287, 0.5 * z4) * dsth;
            const double ka = z2 * th0, kb = z4 * th0;
            const double d[3] = {fma(ya, ea0, fma(yb, eb[0], dX[0])), fma(ya, ea1, fma(yb, eb[1], dX[1])), fma(yb, eb[2], dX[2])};
            const double Pe[3] = {fma(ka, ea0, fma(kb, eb[0], Pn[0])), fma(ka, ea1, fma(kb, eb[1], Pn[1])), fma(kb, eb[2], Pn[2])};
            const double pn = rsqrt(Pe[0] * Pe[0] + Pe[1] * Pe[1] + Pe[2] * Pe[2]);
            const double len2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            float *o = mine + jr;
            constexpr int F = 32 * kMsPitch;                      // floats per field
            o[0] = (float)X[0]; o[F] = (float)X[1]; o[2 * F] = (float)X[2];
            if (!(len2 > 0.0)) {                                  // zero-length track: keep the direction of flight
                o[3 * F] = (float)P[0]; o[4 * F] = (float)P[1]; o[5 * F] = (float)P[2];
                o[6 * F] = 0.f;
            } else {
                const double il = rsqrt(len2);
                o[3 * F] = (float)(d[0] * il); o[4 * F] = (float)(d[1] * il); o[5 * F] = (float)(d[2] * il);
                o[6 * F] = (float)(len2 * il);
            }
            o[7 * F] = beta_f;
            o[8 * F] = (float)fma((double)j, dt_piece, h.t0);
            o[9 * F] = charge_f;
            for (int k = 0; k < 3; ++k) { X[k] += d[k]; P[k] = Pe[k] * pn; }
          }
          __syncwarp();
          // flush: lane = (track of a quartet, piece); eight quartets
          const int cnt = min(max(n - j0, 0), kMsStage);
          const long long gs = g0 + j0;
          float *const outs[kMsFields] = {a.out.x, a.out.y, a.out.z, a.out.dx, a.out.dy, a.out.dz, a.out.len, a.out.beta, a.out.t0, a.out.charge};
          const int tq = lane >> 3, pr = lane & 7;
#pragma unroll 1
          for (int q = 0; q < 8; ++q) {
              const int trk = 4 * q + tq;
              const int c = __shfl_sync(FULL, cnt, trk);
              const long long g = __shfl_sync(FULL, gs, trk) + pr;
              if (pr < c) {
                  const float *src = stage + trk * kMsPitch + pr;
#pragma unroll
                  for (int f = 0; f < kMsFields; ++f) outs[f][g] = src[f * 32 * kMsPitch];
                  if (a.out.edep) a.out.edep[g] = 0.f;
              }
          }
          __syncwarp();
        }
    }
}

__global__ void __launch_bounds__(kMsThreads) k_substep_fill_ms(const __grid_constant__ SubstepArgs a)
{
    __shared__ int s_hist[kMsBins], s_start[kMsBins];
    __shared__ unsigned short s_perm[kMsChunk];
    __shared__ float s_stage[kMsThreads / 32][kMsFields * 32 * kMsPitch];
    constexpr int kPer = kMsChunk / kMsThreads;
    const long long n_chunks = (a.n + kMsChunk - 1) / kMsChunk;
    for (long long chunk = blockIdx.x; chunk < n_chunks; chunk += gridDim.x) {
        const long long c0 = chunk * kMsChunk;
        const int cn = (int)(a.n - c0 < kMsChunk ? a.n - c0 : kMsChunk);
        if (threadIdx.x < kMsBins) s_hist[threadIdx.x] = 0;
        __syncthreads();
        int bin[kPer], rank[kPer];
#pragma unroll
        for (int r = 0; r < kPer; ++r) {
            const int t = threadIdx.x + kMsThreads * r;
            bin[r] = -1;
            if (t < cn) {
                const long long m = a.offsets[c0 + t + 1] - a.offsets[c0 + t];
                bin[r] = kMsBins - 1 - (int)(m < kMsBins - 1 ? m : kMsBins - 1);        // longest tracks first
                rank[r] = atomicAdd(&s_hist[bin[r]], 1);
            }
        }
        __syncthreads();
        if (threadIdx.x < 32) {                                       // exclusive scan of the 64 class sizes
            const int lane = threadIdx.x;
            const int h0 = s_hist[2 * lane], h1 = s_hist[2 * lane + 1];
            int v = h0 + h1;
            for (int d = 1; d < 32; d <<= 1) {
                const int u = __shfl_up_sync(0xFFFFFFFFu, v, d);
                if (lane >= d) v += u;
            }
            s_start[2 * lane] = v - h0 - h1;
            s_start[2 * lane + 1] = v - h1;
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < kPer; ++r)
            if (bin[r] >= 0) s_perm[s_start[bin[r]] + rank[r]] = (unsigned short)(threadIdx.x + kMsThreads * r);
        __syncthreads();
        for (int r = 0; r < kPer; ++r) {
            const int pos = threadIdx.x + kMsThreads * r;
            if ((pos & ~31) < cn) ms_walk(a, pos < cn ? c0 + s_perm[pos] : 0, pos < cn, s_stage[threadIdx.x >> 5]);
        }
        __syncthreads();
    }
}

}  // namespace

size_t substep_scratch_elems(long long n) { return (size_t)((n + kScanThreads - 1) / kScanThreads); }

cudaError_t launch_substep_plan(const SubstepArgs &a, long long *block_sums, cudaStream_t st)
{
    const long long nb = (a.n + kScanThreads - 1) / kScanThreads;
    k_substep_count<<<(unsigned)nb, kScanThreads, 0, st>>>(a, block_sums);
    k_substep_scan_blocks<<<1, kScanThreads, 0, st>>>(block_sums, nb);
    k_substep_add_blocks<<<(unsigned)nb, kScanThreads, 0, st>>>(a, block_sums);
    return cudaGetLastError();
}

cudaError_t launch_substep_fill(const SubstepArgs &a, int n_sm, cudaStream_t st)
{
    if (a.ms_enabled) k_substep_fill_ms<<<n_sm * 8, kMsThreads, 0, st>>>(a);
    else k_substep_fill<<<n_sm * 16, kFillThreads, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace c8ph

// ------------------------------------------------------------------------------------------------------------------
// c8ph_substep_plan_static: the planning step for callers that must not allocate (code under CUDA graph capture,
// tight serving loops, harnesses that forbid cudaMalloc).  No context (c8ph_create allocates): the scan scratch - one
// block total per 1024 tracks - is the file-scope device array below, C8PH_SUBSTEP_STATIC_MAX_TRACKS / 1024 x 8 B =
// 32 KB that every GPU loading the library holds until exit.  In host code `g_static_bsums` is a host-side stand-in,
// not a device address: the address the kernels get comes from cudaGetSymbolAddress, resolved once per device with
// that device current.  All calls on a device share the array: two calls that overlap on the GPU (different streams,
// no ordering) race on it.  Nothing in it has to start at zero: k_substep_count writes every block total a call reads
// before k_substep_scan_blocks reads it, so the contents the previous call left behind are never seen.
static __device__ __align__(256) long long g_static_bsums[C8PH_SUBSTEP_STATIC_MAX_TRACKS / 1024];
static_assert(c8ph::kScanThreads == 1024, "the static scratch is sized for 1024-track scan blocks");

namespace {
constexpr int kStaticMaxDevices = 64;
long long *g_static_ptr[kStaticMaxDevices];          // device address of g_static_bsums, per device (0: not resolved yet)
thread_local char g_static_err[256] = "";

int static_fail(int code, const char *msg, cudaError_t e = cudaSuccess)
{
    if (e != cudaSuccess) snprintf(g_static_err, sizeof g_static_err, "%s: %s", msg, cudaGetErrorString(e));
    else snprintf(g_static_err, sizeof g_static_err, "%s", msg);
    return code;
}
}  // namespace

extern "C" const char *c8ph_substep_plan_static_error(void) { return g_static_err; }

extern "C" int c8ph_substep_plan_static(const c8ph_segments *t, const float *p_GeV, int64_t n, const c8ph_substep_desc *d,
                                        int64_t *offsets, void *stream)
{
    if (!t || t->size != sizeof(c8ph_segments) || !d || d->size != sizeof(c8ph_substep_desc))
        return static_fail(C8PH_E_ARG, "substep_plan_static: NULL struct or size mismatch");
    if (n < 0) return static_fail(C8PH_E_ARG, "substep_plan_static: n_tracks < 0");
    if (n > (int64_t)C8PH_SUBSTEP_STATIC_MAX_TRACKS) {
        snprintf(g_static_err, sizeof g_static_err,
                 "substep_plan_static: n_tracks = %lld exceeds C8PH_SUBSTEP_STATIC_MAX_TRACKS = %lld (split the call, or use "
                 "c8ph_substep_plan with a context)", (long long)n, (long long)C8PH_SUBSTEP_STATIC_MAX_TRACKS);
        return C8PH_E_ARG;
    }
    if (!offsets) return static_fail(C8PH_E_ARG, "substep_plan_static: offsets is NULL");
    if (n > 0 && (!t->x || !t->y || !t->z || !t->dx || !t->dy || !t->dz || !t->len || !t->beta || !t->t0 || !t->charge || !p_GeV))
        return static_fail(C8PH_E_ARG, "substep_plan_static: NULL track array");
    if (!(d->tol_m > 0.f) || d->max_sub < 1 || d->max_sub > (1 << 20))
        return static_fail(C8PH_E_ARG, "substep_plan_static: tol_m > 0 and 1 <= max_sub <= 2^20 required");
    if (d->ms_enabled && !(d->ms_max_step_m >= 0.f)) return static_fail(C8PH_E_ARG, "substep_plan_static: ms_max_step_m >= 0 required");
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e;
    if (n == 0) {
        if ((e = cudaMemsetAsync(offsets, 0, sizeof(int64_t), st)) != cudaSuccess) return static_fail(C8PH_E_CUDA, "substep_plan_static: memset", e);
        return C8PH_OK;
    }
    // set-up, once per device, with that device current: the device address of the scratch array
    int dev = -1;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return static_fail(C8PH_E_CUDA, "substep_plan_static: cudaGetDevice", e);
    if (dev < 0 || dev >= kStaticMaxDevices) return static_fail(C8PH_E_ARG, "substep_plan_static: device ordinal out of range");
    long long *scratch = __atomic_load_n(&g_static_ptr[dev], __ATOMIC_ACQUIRE);
    if (!scratch) {
        if ((e = cudaGetSymbolAddress((void **)&scratch, g_static_bsums)) != cudaSuccess || !scratch)
            return static_fail(C8PH_E_CUDA, "substep_plan_static: cudaGetSymbolAddress", e);
        __atomic_store_n(&g_static_ptr[dev], scratch, __ATOMIC_RELEASE);      // every thread resolves the same address
    }
    c8ph::SubstepArgs a{};
    a.trk = *t; a.p_GeV = p_GeV; a.n = n;
    for (int k = 0; k < 3; ++k) a.B[k] = d->B_tesla[k];
    a.Bn = sqrt(a.B[0] * a.B[0] + a.B[1] * a.B[1] + a.B[2] * a.B[2]);
    a.tol = d->tol_m; a.max_sub = d->max_sub;
    a.ms_enabled = d->ms_enabled ? 1 : 0; a.ms_max_step = d->ms_max_step_m; a.ms_X0 = d->ms_X0_gcm2;
    a.id_base = d->track_id_base;
    a.clipped = reinterpret_cast<unsigned long long *>(d->clipped);
    a.offsets = reinterpret_cast<long long *>(offsets);
    if ((e = c8ph::launch_substep_plan(a, scratch, st)) != cudaSuccess) return static_fail(C8PH_E_CUDA, "substep_plan_static: launch", e);
    return C8PH_OK;
}
