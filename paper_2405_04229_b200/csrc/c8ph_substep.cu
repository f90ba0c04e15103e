// c8ph_substep.cu — sub-stepping of particle tracks along the magnetically deflected path
// (thesis sec. 4.2.1): the step before the hot path.  Three small kernels plan the pieces
// (count per track + exclusive prefix sum), one fills them (one thread per piece).  fp64: the pieces
// must reproduce km-scale positions to well below the 15 cm resolution the thesis quotes.
#include <cuda_runtime.h>
#include <cstdint>
#include "c8ph_device.cuh"

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

// number of chords: sagitta L_piece^2 curvature / 8 <= tol
__device__ __forceinline__ int pieces_of(const Helix &h, double tol, int max_sub)
{
    if (!(h.curv > 0.0) || !(h.L > 0.0)) return 1;
    const double nn = ceil(h.L / sqrt(8.0 * tol / h.curv));
    return nn < 1.0 ? 1 : (nn > (double)max_sub ? max_sub : (int)nn);
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
    if (i < a.n) v = pieces_of(helix_of(a, i), a.tol, a.max_sub);
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

// fill: one thread per piece (grid-stride over offsets[n] pieces), owner track by binary search
__global__ void __launch_bounds__(256) k_substep_fill(const __grid_constant__ SubstepArgs a)
{
    const long long total = a.offsets[a.n];
    for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < total; g += (long long)gridDim.x * blockDim.x) {
        long long lo = 0, hi = a.n;                                    // largest i with offsets[i] <= g
        while (hi - lo > 1) {
            const long long mid = (lo + hi) >> 1;
            if (a.offsets[mid] <= g) lo = mid; else hi = mid;
        }
        const Helix h = helix_of(a, lo);
        const long long m = a.offsets[lo + 1] - a.offsets[lo], j = g - a.offsets[lo];
        const double s0 = h.L * (double)j / (double)m, s1 = h.L * (double)(j + 1) / (double)m;
        double X0[3], X1[3];
        point_on(h, s0, X0);
        point_on(h, s1, X1);
        const double d[3] = {X1[0] - X0[0], X1[1] - X0[1], X1[2] - X0[2]};
        const double len = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        a.out.x[g] = (float)X0[0]; a.out.y[g] = (float)X0[1]; a.out.z[g] = (float)X0[2];
        a.out.dx[g] = (float)(d[0] / len); a.out.dy[g] = (float)(d[1] / len); a.out.dz[g] = (float)(d[2] / len);
        a.out.len[g] = (float)len;
        a.out.beta[g] = (float)h.beta;
        a.out.t0[g] = (float)(h.t0 + s0 / (h.beta * 0.299792458));
        a.out.charge[g] = (float)h.charge;
        if (a.out.edep) a.out.edep[g] = 0.f;
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

cudaError_t launch_substep_fill(const SubstepArgs &a, cudaStream_t st)
{
    k_substep_fill<<<148 * 8, 256, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace c8ph
