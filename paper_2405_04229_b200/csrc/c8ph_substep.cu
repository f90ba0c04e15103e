// c8ph_substep.cu — sub-stepping of particle tracks along the magnetically deflected path
// (thesis sec. 4.2.1): the step before the hot path.  Three small kernels plan the pieces
// (count per track + exclusive prefix sum), one fills them (a warp expands 32 tracks cooperatively).  fp64: the pieces
// must reproduce km-scale positions to well below the 15 cm resolution the thesis quotes.
#include <cuda_runtime.h>
#include <cstdint>
#include "c8ph_device.cuh"
#include "c8ph_philox.cuh"

namespace c8ph {

namespace {

constexpr int kScanThreads = 1024;

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

// fill: a warp takes 32 consecutive tracks and expands them cooperatively - lane l writes the pieces
// base + l, base + l + 32, ... of the group (coalesced), the owner track of a piece by a five-step
// search over the group's 32 start offsets held one per lane (shuffles, no global binary search)
__global__ void __launch_bounds__(256) k_substep_fill(const __grid_constant__ SubstepArgs a)
{
    const unsigned FULL = 0xFFFFFFFFu;
    const int lane = threadIdx.x & 31;
    const long long n_groups = (a.n + 31) >> 5;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long grp = warp0; grp < n_groups; grp += n_warps) {
        const long long i0 = grp << 5;
        const long long base = a.offsets[i0];
        const long long i_me = i0 + lane < a.n ? i0 + lane : a.n;
        const long long i_end = i0 + 32 < a.n ? i0 + 32 : a.n;
        const int rel = (int)(a.offsets[i_me] - base);                 // start of my track within the group (<= 32 * max_sub)
        const int total = (int)(a.offsets[i_end] - base);              // lanes beyond the last track hold `total`
        for (int p0 = 0; p0 < total; p0 += 32) {
            __syncwarp();                                              // lanes that skipped the tail of the last pass rejoin
            const int p = p0 + lane;
            int lo = 0;                                                // largest t with rel[t] <= p
#pragma unroll
            for (int step = 16; step >= 1; step >>= 1) {
                const int v = __shfl_sync(FULL, rel, (lo + step) & 31);
                if (v <= p) lo += step;
            }
            const int r0 = __shfl_sync(FULL, rel, lo);
            int r1 = __shfl_sync(FULL, rel, (lo + 1) & 31);
            if (lo == 31) r1 = total;
            if (p >= total) continue;
            const Helix h = helix_of(a, i0 + lo);
            const int m = r1 - r0, j = p - r0;
            const double s0 = h.L * (double)j / (double)m, s1 = h.L * (double)(j + 1) / (double)m;
            double X0[3], X1[3];
            point_on(h, s0, X0);
            point_on(h, s1, X1);
            double d[3] = {X1[0] - X0[0], X1[1] - X0[1], X1[2] - X0[2]};
            double len = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            const long long g = base + p;
            a.out.x[g] = (float)X0[0]; a.out.y[g] = (float)X0[1]; a.out.z[g] = (float)X0[2];
            if (!(len > 0.0)) {                                   // zero-length track: a piece of length 0 along the direction of flight
                for (int k = 0; k < 3; ++k) d[k] = h.ppar * h.bh[k] + h.pperp * h.e1[k];
                a.out.dx[g] = (float)d[0]; a.out.dy[g] = (float)d[1]; a.out.dz[g] = (float)d[2];
            } else {
                a.out.dx[g] = (float)(d[0] / len); a.out.dy[g] = (float)(d[1] / len); a.out.dz[g] = (float)(d[2] / len);
            }
            a.out.len[g] = (float)len;
            a.out.beta[g] = (float)h.beta;
            a.out.t0[g] = (float)(h.t0 + s0 / (h.beta * 0.299792458));
            a.out.charge[g] = (float)h.charge;
            if (a.out.edep) a.out.edep[g] = 0.f;
        }
    }
}

// fill with multiple scattering (R18): the pieces of a track are a random walk, so one thread walks one
// track: exact magnetic rotation of the piece, then Highland's correlated offset / deflection per plane
__global__ void __launch_bounds__(128) k_substep_fill_ms(const __grid_constant__ SubstepArgs a)
{
    const DevAtm &atm = a.atm;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < a.n; i += (long long)gridDim.x * blockDim.x) {
        const Helix h = helix_of(a, i);
        const long long g0 = a.offsets[i];
        const int n = (int)(a.offsets[i + 1] - g0);
        const double ds = h.L / (double)n;
        const double p = a.p_GeV[i];
        const unsigned long long tid = (unsigned long long)(a.id_base + i);
        double X[3] = {h.A[0], h.A[1], h.A[2]};
        double P[3];
        for (int k = 0; k < 3; ++k) P[k] = h.ppar * h.bh[k] + h.pperp * h.e1[k];
        double sn, cs;
        sincos(h.kappa * ds, &sn, &cs);
        for (int j = 0; j < n; ++j) {
            const double ppar = P[0] * h.bh[0] + P[1] * h.bh[1] + P[2] * h.bh[2];
            const double Pp[3] = {P[0] - ppar * h.bh[0], P[1] - ppar * h.bh[1], P[2] - ppar * h.bh[2]};
            const double Pc[3] = {Pp[1] * h.bh[2] - Pp[2] * h.bh[1], Pp[2] * h.bh[0] - Pp[0] * h.bh[2], Pp[0] * h.bh[1] - Pp[1] * h.bh[0]};
            double dX[3], Pn[3];
            for (int k = 0; k < 3; ++k) {
                if (h.kappa != 0.0) {
                    dX[k] = ppar * h.bh[k] * ds + (sn * Pp[k] + (1.0 - cs) * Pc[k]) / h.kappa;
                    Pn[k] = ppar * h.bh[k] + cs * Pp[k] + sn * Pc[k];
                } else { dX[k] = P[k] * ds; Pn[k] = P[k]; }
            }
            // density of the overburden-table cell at the piece's mid height
            const double mx = X[0] + 0.5 * dX[0], my = X[1] + 0.5 * dX[1], mz = X[2] + 0.5 * dX[2];
            double hm = atm.h_obs + mz;
            if (atm.model == C8PH_ATM_SPHERICAL) hm = sqrt(mx * mx + my * my + (mz + atm.Rg) * (mz + atm.Rg)) - atm.R;
            double rho = 0.0;
            if (atm.model != C8PH_ATM_HOMOGENEOUS) {
                double f = (hm - (double)atm.h0) / (double)atm.dh;
                f = fmin(fmax(f, 0.0), (double)(atm.n_nodes - 1));
                const int k = min((int)f, atm.n_nodes - 2);
                rho = ((double)__ldg(atm.xv + k) - (double)__ldg(atm.xv + k + 1)) / (double)atm.dh;
            }
            double th0 = 0.0;
            const double t = rho * ds / a.ms_X0;
            if (t > 0.0 && p > 0.0) {
                const double corr = fmax(1.0 + 0.038 * log(t * h.charge * h.charge / (h.beta * h.beta)), 0.0);
                th0 = 0.0136 / (h.beta * p) * fabs(h.charge) * sqrt(t) * corr;
            }
            const uint4 r = philox4x32_10((uint32_t)j, (uint32_t)tid, (uint32_t)(tid >> 32), 16u, a.key);
            auto u01d = [](uint32_t v) { return ((double)(v >> 9) + 0.5) * (1.0 / 8388608.0); };
            const double r1 = sqrt(-2.0 * log(u01d(r.x))), r2 = sqrt(-2.0 * log(u01d(r.z)));
            double s1, c1, s2, c2;
            sincos(2.0 * 3.14159265358979323846 * u01d(r.y), &s1, &c1);
            sincos(2.0 * 3.14159265358979323846 * u01d(r.w), &s2, &c2);
            const double z1 = r1 * c1, z2 = r1 * s1, z3 = r2 * c2, z4 = r2 * s2;
            double ea[3] = {Pn[1], -Pn[0], 0.0};
            double na = sqrt(ea[0] * ea[0] + ea[1] * ea[1]);
            if (na < 1e-12) { ea[0] = 1.0; ea[1] = 0.0; na = 1.0; }
            ea[0] /= na; ea[1] /= na;
            const double eb[3] = {Pn[1] * ea[2] - Pn[2] * ea[1], Pn[2] * ea[0] - Pn[0] * ea[2], Pn[0] * ea[1] - Pn[1] * ea[0]};
            const double ya = (z1 / sqrt(12.0) + 0.5 * z2) * ds * th0, yb = (z3 / sqrt(12.0) + 0.5 * z4) * ds * th0;
            double Xe[3], Pe[3];
            for (int k = 0; k < 3; ++k) {
                Xe[k] = X[k] + dX[k] + ya * ea[k] + yb * eb[k];
                Pe[k] = Pn[k] + z2 * th0 * ea[k] + z4 * th0 * eb[k];
            }
            const double pn = 1.0 / sqrt(Pe[0] * Pe[0] + Pe[1] * Pe[1] + Pe[2] * Pe[2]);
            const double d[3] = {Xe[0] - X[0], Xe[1] - X[1], Xe[2] - X[2]};
            const double len = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            const long long g = g0 + j;
            a.out.x[g] = (float)X[0]; a.out.y[g] = (float)X[1]; a.out.z[g] = (float)X[2];
            if (!(len > 0.0)) {                                   // zero-length track: keep the direction of flight
                a.out.dx[g] = (float)P[0]; a.out.dy[g] = (float)P[1]; a.out.dz[g] = (float)P[2];
            } else {
                a.out.dx[g] = (float)(d[0] / len); a.out.dy[g] = (float)(d[1] / len); a.out.dz[g] = (float)(d[2] / len);
            }
            a.out.len[g] = (float)len;
            a.out.beta[g] = (float)h.beta;
            a.out.t0[g] = (float)(h.t0 + (double)j * ds / (h.beta * 0.299792458));
            a.out.charge[g] = (float)h.charge;
            if (a.out.edep) a.out.edep[g] = 0.f;
            for (int k = 0; k < 3; ++k) { X[k] = Xe[k]; P[k] = Pe[k] * pn; }
        }
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
    if (a.ms_enabled) k_substep_fill_ms<<<n_sm * 8, 128, 0, st>>>(a);
    else k_substep_fill<<<n_sm * 8, 256, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace c8ph
