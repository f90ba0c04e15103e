// c8ph_kernels.cu — sm_100a kernels of libc8ph.
//
//  * k_emit_propagate: the fused hot path  segment -> yield -> photons -> straight line -> cuts ->
//    refraction (none | layered Snell sum | interpolation-tracing table) -> transmission ->
//    ground grid / telescope spheres / camera -> compacted photon list.   (thesis sec. 5.3)
//  * k_build_table: the interpolation-tracing correction table (thesis sec. 4.4.1).
//
// Design (DESIGN.md section 5 has the long version and the measurements behind each choice):
//  - persistent grid, one warp owns a group of segments taken from a global cursor; the 32 lanes
//    first PREPARE up to 32 segments in parallel, one per lane, in fp64 (yield, bunch count, LV1,
//    Rodrigues basis, axis-landing anchor) and park them in the warp's slots of a global scratch
//    array; then the warp walks the emitting segments and the lanes stride over the photons of one
//    segment, photon state in registers only;
//  - per-photon arithmetic is fp32 in cancellation-free "anchor + offset" form: the landing point
//    of the particle axis and its clock are computed once per segment in fp64, the photon only
//    adds small offsets, which keeps bin flips against the fp64 oracle below 1e-4;
//  - Philox4x32-10 keyed on (seed; segment id, photon index): results are independent of grid
//    size, segment order and batching;
//  - n(h) through L1 (lanes of a warp emit from one short segment: one cache line); only the
//    layered-sum variant stages n(h) and the overburden steps per CTA in shared memory with one
//    TMA bulk copy each (cp.async.bulk + mbarrier);
//  - the correction table (float4 texels dd, dt, X_slant, tau_aer) is read with 4 x LDG.128
//    through L1: the lanes of a warp share (height, zenith) to within the Cherenkov angle;
//  - telescope searches on uniform grids whose cells list candidates sorted by a lower-bound key
//    (one 4 B load decides "nothing in reach"); the few photons that pass the pre-test are queued
//    in a per-warp shared-memory ring and a full warp finishes 32 of them at a time (arrival time
//    and direction, exact sphere test, ballot-ranked record store);
//  - the ground histogram takes one RED.ADD.F32 per binned photon into the L2-resident grid.
#include <cuda_runtime.h>
#include <math_constants.h>
#include <cstdint>
#include <cstdlib>
#include <type_traits>
#include "c8ph_device.cuh"
#include "c8ph_philox.cuh"

// ---- compile-time A/B knobs (`python -m paper_2405_04229_b200.build --define NAME=VALUE --out lib.so`, then
// C8PH_LIB=lib.so).  The defaults are what the measurements on cfg4 chose; profiles/r2_ab.md has one row per knob.
#ifndef C8PH_SINCOS_MUFU
#define C8PH_SINCOS_MUFU 1      // 1: azimuth sin / cos by MUFU.SIN / MUFU.COS (sin.approx), 0: polynomial from the uniform's bits
#endif
#ifndef C8PH_TABLE_TEX
#define C8PH_TABLE_TEX 0        // 1: correction table through a 2-D float4 texture object with hardware bilinear filtering
#endif
#ifndef C8PH_HIST_MATCH
#define C8PH_HIST_MATCH 0       // 1: lanes of a warp that hit the same ground bin are aggregated (match.any) into one RED
#endif
#ifndef C8PH_ETA_STAGED
#define C8PH_ETA_STAGED 0       // 1: n(h) staged in shared memory by a TMA bulk copy also for the table-tracing variants
#endif
#ifndef C8PH_ETA_SEGFIT
#define C8PH_ETA_SEGFIT 0       // 1: n(h_e) along a segment from a per-segment quadratic in s, fitted in fp64 and checked against the
#endif                          //    piecewise-linear table (Listing 4.1) to 4e-7 relative; segments that fail it read the table per photon
#ifndef C8PH_TABLE_EXIT
#define C8PH_TABLE_EXIT 1       // 1: the table lookup leaves before its loads when (h, zenith) is out of range, instead of clamping the node coordinates
#endif
#ifndef C8PH_HIT_RING
#define C8PH_HIT_RING 1         // 1: a point outside the hit grid is clamped into the grid's ring of empty border cells instead of being tested
#endif
#ifndef C8PH_SLOT_PREFETCH
#define C8PH_SLOT_PREFETCH 0    // 1: the next emitting segment's slot (two 128 B lines) is prefetched into L1 while the current one runs (measured: +0.3 % time)
#endif
#ifndef C8PH_HIT_PREFETCH
#define C8PH_HIT_PREFETCH 0     // 1: a lane that queues a telescope candidate prefetches the hit cell's first-telescope record (finish() reads it)
#endif
#ifndef C8PH_QUEUE_VOTE
#define C8PH_QUEUE_VOTE 1       // 1: "32 candidates wait" is decided by a vote of the lanes that pushed; 0: by reading the fill count
#endif
#ifndef C8PH_TABLE_EARLY
#define C8PH_TABLE_EARLY 0      // 1 (production variants): the four texel loads of the correction table are issued before the straight
#endif                          //    line and the LV2 test and combined after them, so that their latency overlaps that arithmetic
#ifndef C8PH_QUEUE_CONVERGED
#define C8PH_QUEUE_CONVERGED 0  // 1: candidates are queued after the photon body's reconvergence point (one ballot, fill count in a
#endif                          //    register); 0: inside the body, where the few candidate lanes are
#ifndef C8PH_QUEUE_LANE_ATOMS
#define C8PH_QUEUE_LANE_ATOMS 1 // (inside the body) 1: every candidate lane takes its slot with its own ATOMS; 0: one ATOMS per group of
#endif                          //    lanes that arrive together, slot = base + rank (activemask, leader, shuffle)
#ifndef C8PH_PROD_ONLY
#define C8PH_PROD_ONLY 0        // 1: instantiate only the generic variants and SPEC = base (fast A/B builds)
#endif

namespace c8ph {

namespace {

// Launch shape.  Table / straight tracing: ONE CTA per SM whose per-warp candidate queues plus static and reserved shared
// memory fit the 100 KB carve-out, which leaves 156 KB of L1 (124 KB with three CTAs of 256 threads: +4 % time; measured
// in profiles/r2_ab.md): 768 threads (24 warps at 80 registers, 4 KB queues) by default, 896 / 640 threads for the
// variants kernel_threads() names.  The layered-sum variant stages 80-120 KB of tables per CTA and runs two CTAs of 256
// threads.
#ifndef C8PH_THREADS
#define C8PH_THREADS 768
#endif
#ifndef C8PH_MIN_BLOCKS
#define C8PH_MIN_BLOCKS 1
#endif
constexpr int kMaxWarpsPerSM = 64;                             // hardware limit; the segment-slot scratch is sized for it
#ifndef C8PH_THREADS_WIDE
#define C8PH_THREADS_WIDE 640   // variants that spill at 80 registers: 20 warps at 96 registers (5 x 128 threads; 672 / 704 are rounded up to 768 by ptxas)
#endif
// Cherenkov variants with every switch at run time (SPEC = 0) and the 16-texel flat-plane table variant run 640 threads:
// 15.8 -> 14.1 ms and 16.1 -> 13.4 ms on 2e6 cfg4 segments; every other compiled variant and fluorescence are faster at 768
// (profiles/r2_extras.md)
#ifndef C8PH_THREADS_DENSE
#define C8PH_THREADS_DENSE 896  // 28 warps at 72 registers: the compiled variants with 56-byte queue entries
#endif
#ifndef C8PH_QUEUE_GLOBAL
#define C8PH_QUEUE_GLOBAL 0     // 1: the compact candidate queues live in global memory (L2, st/ld .cg) instead of shared memory: no carve-out
#endif
#ifndef C8PH_QUEUE_COMPACT
#define C8PH_QUEUE_COMPACT 1    // 1: 56-byte queue entries in the SPEC != 0 variants (needs the default queue knobs)
#endif
__host__ __device__ constexpr bool queue_compact(int spec)
{
    return C8PH_QUEUE_COMPACT && C8PH_QUEUE_LANE_ATOMS && C8PH_QUEUE_VOTE && !C8PH_QUEUE_CONVERGED && spec != 0;
}
__host__ __device__ constexpr int queue_words(int spec) { return queue_compact(spec) ? 14 : 16; }
__host__ __device__ constexpr int kernel_threads(int emit, int trace, int spec)
{
    // 896 threads: the compiled variants without the analytic flat-plane step (bit 2) and the optics (bit 32), which
    // gain nothing from it (profiles/r2_extras.md)
    return trace == C8PH_TRACE_NUMERIC ? 256
         : ((spec == 0 && emit == C8PH_EMIT_CHERENKOV) || (spec & 64) != 0) ? C8PH_THREADS_WIDE
         : (queue_compact(spec) && (spec & (2 | 32)) == 0) ? C8PH_THREADS_DENSE : C8PH_THREADS;
}
__host__ __device__ constexpr int kernel_min_blocks(int trace) { return trace == C8PH_TRACE_NUMERIC ? 2 : C8PH_MIN_BLOCKS; }
constexpr float kInvC = 1.0f / 0.299792458f;     // ns per metre
constexpr double kC = 0.299792458;               // m / ns
constexpr double kAlphaFS = 1.0 / 137.035999;    // fine-structure constant (Eq. 2.3)
constexpr float kUpCut = -1.0e-6f;               // drop photons with u_z >= kUpCut

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

// ---- TMA bulk copy global -> shared, completion on an mbarrier ---------------------------------
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

// (2m+1) 2^-24, m = top 23 bits: exact in fp32; built from the mantissa bits without an I2F
__device__ __forceinline__ float u01(uint32_t r)
{
    return __uint_as_float(0x3F800000u | (r >> 9)) - 0.99999994f;
}

__device__ __forceinline__ double u01d(uint32_t r)
{
    return (static_cast<double>(r >> 9) + 0.5) * (1.0 / 8388608.0);
}

// ---- per-segment state: prepared by one lane in fp64, parked in the warp's slot of a global
// scratch array (L2-resident), then read back by all lanes (uniform address).  HOT = used by every
// photon, kept in registers while the warp walks the segment; COLD = used by landed photons /
// rare branches, re-read through L1 where it is needed (keeps the register count down).
struct alignas(16) SegHot {                       // 28 words = 7 x 16 B
    float Px, Py, Pz, e1x, e1y, e2y;                  // direction and the Rodrigues columns (M symmetric, third column -P:
                                                      // e2x = e1y, e1z = -P_x, e2z = -P_y)
    float q0, q1, q2;                                 // n(h_e) - 1 = q0 + s (q1 + s q2) along the segment (anchor bit 1 set)
    float L, beta, delta;                             // length, beta, 1 - beta
    float hA, cA, k2;                                 // height of A, dh/ds, second-order term
    float Az, AzP;                                    // A_z, A_z / P_z (anchor form)
    float Gx, Gy;                                     // axis landing point (anchor) or unused
    float a1, a2, inv_rA;                             // e1.r, e2.r, 1/|A - C|
    uint32_t id_lo, id_hi;                            // global segment id (Philox counter words)
    int N, anchor;                                    // bunches to emit; bit 0: anchor form valid, bit 1: q0..q2 valid
    float dob, inv_beta;                              // (1 - beta)/beta, 1/beta (read from the slot, not kept in registers)
};
struct alignas(16) SegCold {                      // 16 words = 4 x 16 B
    float fbx, fby;                                   // fractional grid coordinate of the anchor
    int ibx, iby;                                     // integer grid coordinate of the anchor
    float rx, ry, rz;                                 // local vertical at A
    float Ax, Ay;                                     // start point (non-anchor form); anchor form: G - (float)G
    float aimx, aimy, aimz, omc;                      // fluorescence: aim point - A, 1 - cos(psi)
    float Tg;                                         // anchor clock - t_ref  (or t0 - t_ref)
    uint32_t local;                                   // segment index within the call
    float eta_mid;                                    // refractivity at the segment mid height (dispersion)
};
struct alignas(16) SegSlot { SegHot h; SegCold c; };
static_assert(sizeof(SegHot) == 112 && sizeof(SegCold) == 64 && sizeof(SegSlot) == 176, "segment slot layout");

// candidate queue entry (64 B in shared memory, written / read with four 16 B accesses): what finish()
// needs of a photon
// entry = 4 x float4: (x, y, ux, uy) (uz, s, q w_z, dt) (1/lambda, weight, eta_e, h_e) (dd, cos zenith, cell, j<<5|slot)
constexpr int Q_WORDS = 16;
constexpr int kQueue = 64;                       // ring entries per warp (a drain leaves < 32)
// compact entry of the production variants (56 B, three float4 planes + one float2 plane per warp): the weight is the
// bunch weight (roulette mode) and h_e is recomputed from s and the segment slot in finish(), bit for bit:
// (x, y, ux, uy) (uz, s, q w_z, dt) (1/lambda, eta_e, dd, cos zenith) (cell, j<<5|slot)
// 28 queues of 3.5 KB = 98 KB fit the 100 KB carve-out that 24 queues of 4 KB fill: 28 warps per SM with the same L1
constexpr int Q_WORDS_COMPACT = 14;

template <typename T>
__device__ __forceinline__ void copy16(T *dst, const T *src)
{
    const float4 *s = reinterpret_cast<const float4 *>(src);
    float4 *d = reinterpret_cast<float4 *>(dst);
#pragma unroll
    for (int i = 0; i < (int)(sizeof(T) / 16); ++i) d[i] = s[i];
}

// n-1 at height h from the global table in fp64 (Listing 4.1), clamped to the table
__device__ __forceinline__ double eta_lookup_d(const DevAtm &atm, double h)
{
    double f = (h - (double)atm.h0) / (double)atm.dh;
    f = fmin(fmax(f, 0.0), (double)(atm.n_nodes - 1));
    int k = min((int)f, atm.n_nodes - 2);
    double fr = f - k;
    return (1.0 - fr) * (double)__ldg(atm.eta + k) + fr * (double)__ldg(atm.eta + k + 1);
}

// ---- single-instruction special functions (MUFU, max relative error 2^-23; PTX ISA "rcp.approx",
// "sqrt.approx", "rsqrt.approx").  The IEEE versions add a range check, a branch and a Newton step
// per call; one ulp more on these quantities is far inside the parity budget.
__device__ __forceinline__ float rcp_fast(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float sqrt_fast(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float exp2_fast(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rsqrt_fast(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// acos(x) for x in [0,1]: sqrt(1-x) * p6(x) (least-squares fit on Chebyshev nodes, max error
// 3.3e-7 rad in fp32 = 5e-5 of a zenith cell of the correction table)
__device__ __forceinline__ float acos01(float x)
{
    float p = 0.002251368248835206f;
    p = fmaf(p, x, -0.011012386530637741f);
    p = fmaf(p, x, 0.02674933150410652f);
    p = fmaf(p, x, -0.048724401742219925f);
    p = fmaf(p, x, 0.08873733133077621f);
    p = fmaf(p, x, -0.21458369493484497f);
    p = fmaf(p, x, 1.5707961320877075f);
    return sqrt_fast(1.f - x) * p;
}

// sin and cos of phi = 2 pi u, u = (2m+1) 2^-24 with m = r >> 9 the uniform's 23 mantissa bits
// (a6: azimuth on the cone).  Octant from the top three bits of m, the remaining 20 bits give the
// angle a in (0, pi/4) exactly (odd octants reflected), degree-7/8 polynomials in a (max error
// 7e-8), then swap / sign by octant.
__device__ __forceinline__ void sincos_2pi_u(uint32_t r, float &sphi, float &cphi)
{
#if C8PH_SINCOS_MUFU
    // u - 1/2 = (v - 1.5) + 2^-24 with v = 1.m in [1, 2): exact in fp32; sin(2 pi u) = -sin(2 pi (u - 1/2)), same for cos.
    // sin.approx = FMUL.RZ by 1/(2 pi) + MUFU.SIN on [-pi, pi] (PTX ISA: max absolute error 2^-20.9)
    const float a = __uint_as_float(0x3F800000u | (r >> 9)) - 1.5f;
    const float ph = fmaf(a, 6.2831853071795865f, 3.7450702829e-07f);       // 2 pi (u - 1/2)
    float sv, cv;
    asm("sin.approx.ftz.f32 %0, %1;" : "=f"(sv) : "f"(ph));
    asm("cos.approx.ftz.f32 %0, %1;" : "=f"(cv) : "f"(ph));
    sphi = -sv; cphi = -cv;
#else
    const uint32_t m = r >> 9, o = m >> 20;
    uint32_t ml = m & 0xFFFFFu;
    if (o & 1u) ml ^= 0xFFFFFu;
    const float a = (float)(int)(2u * ml + 1u) * 3.7450702829e-07f;        // pi / 2^23
    const float z = a * a;
    float sp = -0.0001958794891834259f;
    sp = fmaf(sp, z, 0.008332748897373676f);
    sp = fmaf(sp, z, -0.166666641831398f);
    const float sv = fmaf(a * z, sp, a);
    float cp = 2.4463915906380862e-05f;
    cp = fmaf(cp, z, -0.001388759003020823f);
    cp = fmaf(cp, z, 0.04166664928197861f);
    cp = fmaf(cp, z, -0.5f);
    const float cv = fmaf(z, cp, 1.f);
    const bool swap = ((o + 1u) & 2u) != 0u;
    const float s0 = swap ? cv : sv, c0 = swap ? sv : cv;
    sphi = __uint_as_float(__float_as_uint(s0) ^ ((o & 4u) << 29));
    cphi = __uint_as_float(__float_as_uint(c0) ^ (((o + 2u) & 4u) << 29));
#endif
}

// Dispersive Cherenkov yield integral (thesis P:318, unnumbered equation before Eq. 2.5):
//   int_{k_lo}^{k_hi} Theta(beta n(k) - 1) (1 - 1/(beta n(k))^2) dk,  n(k) = 1 + eta (c0 + b k^2),  k = 1/lambda,
// b >= 0 so n grows towards the blue: the threshold k_th (beta n = 1) is a lower limit.  8-point
// Gauss-Legendre on the smooth part; sin^2 in the cancellation-free form x(2+x)/(1+x)^2, x = beta n - 1.
__device__ __forceinline__ double disp_yield_integral(double beta, double eta, double b, double k0sq,
                                                      double k_lo, double k_hi)
{
    const double delta = 1.0 - beta;
    auto D = [&](double k) { return 1.0 + b * (k * k - k0sq); };
    if (!(beta * eta * D(k_hi) > delta)) return 0.0;                  // below threshold over the whole band
    double ka = k_lo;
    if (!(beta * eta * D(k_lo) > delta)) ka = sqrt(k0sq + (delta / (beta * eta) - 1.0) / b);
    const double xs[4] = {0.1834346424956498, 0.5255324099163290, 0.7966664774136267, 0.9602898564975363};
    const double ws[4] = {0.3626837833783620, 0.3137066458778873, 0.2223810344533745, 0.1012285362903763};
    const double c = 0.5 * (k_hi + ka), hw = 0.5 * (k_hi - ka);
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
#pragma unroll
        for (int sgn = -1; sgn <= 1; sgn += 2) {
            const double x = fmax(beta * eta * D(c + sgn * hw * xs[i]) - delta, 0.0);
            acc += ws[i] * x * (2.0 + x) / ((1.0 + x) * (1.0 + x));
        }
    }
    return acc * hw;
}

struct TabVal { float dd, dt, X, ta; bool bad; };
struct TabRaw { float4 v00, v01, v10, v11; float ff, gg; bool bad; };

// the two halves of table_lookup below: issue the four texel loads / combine them
__device__ __forceinline__ TabRaw table_issue(const DevTable &t, float h, float thz)
{
    TabRaw r;
    r.bad = !(h <= t.h_max) || !(thz <= t.zen_max) || !(h >= 0.f);
    const float f = fminf(fmaxf(h * t.inv_dh, 0.f), t.f_max);
    const float g = fminf(fmaxf(thz * t.inv_dz, 0.f), t.g_max);
    const int ia = min((int)f, t.n_h - 2), ib = min((int)g, t.n_zen - 2);
    r.ff = f - (float)ia; r.gg = g - (float)ib;
    const float4 *p = t.hot + (unsigned)(ia * t.n_zen + ib);
    const float4 *p1 = p + (unsigned)t.n_zen;
    r.v00 = __ldg(p); r.v01 = __ldg(p + 1); r.v10 = __ldg(p1); r.v11 = __ldg(p1 + 1);
    return r;
}
__device__ __forceinline__ TabVal table_combine(const TabRaw &r)
{
    TabVal o;
    const float w11 = r.ff * r.gg, w10 = r.ff - w11, w01 = r.gg - w11, w00 = (1.f - r.ff) - w01;
    o.dd = fmaf(w11, r.v11.x, fmaf(w10, r.v10.x, fmaf(w01, r.v01.x, w00 * r.v00.x)));
    o.dt = fmaf(w11, r.v11.y, fmaf(w10, r.v10.y, fmaf(w01, r.v01.y, w00 * r.v00.y)));
    o.X = fmaf(w11, r.v11.z, fmaf(w10, r.v10.z, fmaf(w01, r.v01.z, w00 * r.v00.z)));
    o.ta = fmaf(w11, r.v11.w, fmaf(w10, r.v10.w, fmaf(w01, r.v01.w, w00 * r.v00.w)));
    o.bad = r.bad || (o.dd != o.dd);
    return o;
}

// bilinear lookup in the correction table (linear interpolation between support points):
// four LDG.128 texels (dd, dt, X_slant, tau_aer); indices clamped; out of range / no-ground -> bad
__device__ __forceinline__ TabVal table_lookup(const DevTable &t, float h, float thz)
{
    TabVal o;
    o.bad = !(h <= t.h_max) || !(thz <= t.zen_max) || !(h >= 0.f);
#if C8PH_TABLE_TEX
    {
        // texel (b, a) = node (height a, zenith b); unnormalised coordinates, clamped addressing, linear filter
        const float4 v = tex2D<float4>(t.tex, fmaf(thz, t.inv_dz, 0.5f), fmaf(h, t.inv_dh, 0.5f));
        o.dd = v.x; o.dt = v.y; o.X = v.z; o.ta = v.w;
        o.bad = o.bad || (o.dd != o.dd);
        return o;
    }
#endif
#if C8PH_TABLE_EXIT
    // out of range (or NaN): the photon is dropped, nothing is read; inside the range 0 <= h <= h_max and
    // 0 <= thz <= zen_max bound the node coordinates, so only the top node needs the integer clamp
    if (o.bad) { o.dd = o.dt = o.X = o.ta = 0.f; return o; }
    const float f = h * t.inv_dh, g = thz * t.inv_dz;
#else
    const float f = fminf(fmaxf(h * t.inv_dh, 0.f), t.f_max);
    const float g = fminf(fmaxf(thz * t.inv_dz, 0.f), t.g_max);
#endif
    const int ia = min((int)f, t.n_h - 2), ib = min((int)g, t.n_zen - 2);
    const float ff = f - (float)ia, gg = g - (float)ib;
    const float4 *p = t.hot + (unsigned)(ia * t.n_zen + ib);
    const float4 *p1 = p + (unsigned)t.n_zen;
    const float4 v00 = __ldg(p), v01 = __ldg(p + 1), v10 = __ldg(p1), v11 = __ldg(p1 + 1);
    const float w11 = ff * gg, w10 = ff - w11, w01 = gg - w11, w00 = (1.f - ff) - w01;
    o.dd = fmaf(w11, v11.x, fmaf(w10, v10.x, fmaf(w01, v01.x, w00 * v00.x)));
    o.dt = fmaf(w11, v11.y, fmaf(w10, v10.y, fmaf(w01, v01.y, w00 * v00.y)));
    o.X = fmaf(w11, v11.z, fmaf(w10, v10.z, fmaf(w01, v01.z, w00 * v00.z)));
    o.ta = fmaf(w11, v11.w, fmaf(w10, v10.w, fmaf(w01, v01.w, w00 * v00.w)));
    o.bad = o.bad || (o.dd != o.dd);
    return o;
}

// R21: lookup in the flat-plane table: trilinear in (height, zenith, rho) on the even and the odd texels (16 LDG.128),
// value = E + cos(chi) O along the direction of flight; perp = P, the displacement along (r^ - cos(chi) e_h)
__device__ __forceinline__ TabVal table_lookup_flat(const DevTable &t, float h, float thz, float rho, float cos_chi, float &perp)
{
    TabVal o;
    o.bad = !(h <= t.h_max) || !(thz <= t.zen_max) || !(h >= 0.f) || !(rho <= t.rho_max);
    const float f = fminf(fmaxf(h * t.inv_dh, 0.f), t.f_max);
    const float g = fminf(fmaxf(thz * t.inv_dz, 0.f), t.g_max);
    const float e = fminf(fmaxf(rho * t.inv_drho, 0.f), t.e_max);
    const int ia = min((int)f, t.n_h - 2), ib = min((int)g, t.n_zen - 2), ic = min((int)e, t.n_rho - 2);
    const float ff = f - (float)ia, gg = g - (float)ib, ee = e - (float)ic;
    const unsigned plane = (unsigned)(t.n_h * t.n_zen);
    const unsigned base = (unsigned)ic * plane + (unsigned)(ia * t.n_zen + ib);
    const float w11 = ff * gg, w10 = ff - w11, w01 = gg - w11, w00 = (1.f - ff) - w01;
    float4 acc[2];
#pragma unroll
    for (int part = 0; part < 2; ++part) {
        const float4 *p = (part ? t.flatO : t.flatE) + base;
        float4 lay[2];
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const float4 *pq = p + (unsigned)q * plane;
            const float4 v00 = __ldg(pq), v01 = __ldg(pq + 1), v10 = __ldg(pq + t.n_zen), v11 = __ldg(pq + t.n_zen + 1);
            lay[q].x = fmaf(w11, v11.x, fmaf(w10, v10.x, fmaf(w01, v01.x, w00 * v00.x)));
            lay[q].y = fmaf(w11, v11.y, fmaf(w10, v10.y, fmaf(w01, v01.y, w00 * v00.y)));
            lay[q].z = fmaf(w11, v11.z, fmaf(w10, v10.z, fmaf(w01, v01.z, w00 * v00.z)));
            lay[q].w = fmaf(w11, v11.w, fmaf(w10, v10.w, fmaf(w01, v01.w, w00 * v00.w)));
        }
        acc[part].x = fmaf(ee, lay[1].x - lay[0].x, lay[0].x);
        acc[part].y = fmaf(ee, lay[1].y - lay[0].y, lay[0].y);
        acc[part].z = fmaf(ee, lay[1].z - lay[0].z, lay[0].z);
        acc[part].w = fmaf(ee, lay[1].w - lay[0].w, lay[0].w);
    }
    o.dd = fmaf(cos_chi, acc[1].x, acc[0].x);
    o.dt = fmaf(cos_chi, acc[1].y, acc[0].y);
    o.X = acc[0].z;
    o.ta = acc[0].w;
    perp = acc[1].z;
    o.bad = o.bad || (o.dd != o.dd) || (perp != perp);
    return o;
}

// R24: lookup in the cylindrical model's table: trilinear in (height, zenith, c = cos^2 psi), 8 LDG.128;
// texel = (dd, dt, X_slant, across displacement / (sin psi cos psi))
__device__ __forceinline__ TabVal table_lookup_cyl(const DevTable &t, float h, float thz, float c, float &ptilde)
{
    TabVal o;
    o.bad = !(h <= t.h_max) || !(thz <= t.zen_max) || !(h >= 0.f) || !(c >= 0.f) || !(c <= 1.f);
    const float f = fminf(fmaxf(h * t.inv_dh, 0.f), t.f_max);
    const float g = fminf(fmaxf(thz * t.inv_dz, 0.f), t.g_max);
    const float e = fminf(fmaxf(c * t.c_max, 0.f), t.c_max);
    const int ia = min((int)f, t.n_h - 2), ib = min((int)g, t.n_zen - 2), ic = min((int)e, t.n_c - 2);
    const float ff = f - (float)ia, gg = g - (float)ib, ee = e - (float)ic;
    const unsigned plane = (unsigned)(t.n_h * t.n_zen);
    const float4 *p = t.cyl + (unsigned)ic * plane + (unsigned)(ia * t.n_zen + ib);
    const float w11 = ff * gg, w10 = ff - w11, w01 = gg - w11, w00 = (1.f - ff) - w01;
    float4 lay[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const float4 *pq = p + (unsigned)q * plane;
        const float4 v00 = __ldg(pq), v01 = __ldg(pq + 1), v10 = __ldg(pq + t.n_zen), v11 = __ldg(pq + t.n_zen + 1);
        lay[q].x = fmaf(w11, v11.x, fmaf(w10, v10.x, fmaf(w01, v01.x, w00 * v00.x)));
        lay[q].y = fmaf(w11, v11.y, fmaf(w10, v10.y, fmaf(w01, v01.y, w00 * v00.y)));
        lay[q].z = fmaf(w11, v11.z, fmaf(w10, v10.z, fmaf(w01, v01.z, w00 * v00.z)));
        lay[q].w = fmaf(w11, v11.w, fmaf(w10, v10.w, fmaf(w01, v01.w, w00 * v00.w)));
    }
    o.dd = fmaf(ee, lay[1].x - lay[0].x, lay[0].x);
    o.dt = fmaf(ee, lay[1].y - lay[0].y, lay[0].y);
    o.X = fmaf(ee, lay[1].z - lay[0].z, lay[0].z);
    o.ta = 0.f;
    ptilde = fmaf(ee, lay[1].w - lay[0].w, lay[0].w);
    o.bad = o.bad || (o.dd != o.dd) || (ptilde != ptilde);
    return o;
}

// ---- telescope search (DevGrid: sorted candidate lists with a per-cell smallest key) -----------
// cell of (x,y), or -1 outside the grid (outside => no telescope within reach)
__device__ __forceinline__ int grid_cell(const DevGrid &g, float x, float y)
{
    const int cx = __float2int_rd((x - g.x0) * g.inv_cs), cy = __float2int_rd((y - g.y0) * g.inv_cs);
    if ((unsigned)cx >= (unsigned)g.nx || (unsigned)cy >= (unsigned)g.ny) return -1;
    return cy * g.nx + cx;
}

// exact ray / bounding-sphere test of one telescope; updates the nearest entry
__device__ __forceinline__ void sphere_test_rec(const float4 t, int k, float x, float y, float ux, float uy, float uz,
                                                float &best_s, int &best_k);
__device__ __forceinline__ void sphere_test(const DevDet &det, int k, float x, float y, float ux, float uy, float uz,
                                            float &best_s, int &best_k)
{
    sphere_test_rec(__ldg(det.tel + k), k, x, y, ux, uy, uz, best_s, best_k);
}
__device__ __forceinline__ void sphere_test_rec(const float4 t, int k, float x, float y, float ux, float uy, float uz,
                                                float &best_s, int &best_k)
{
    // every product is written as an explicit fma / rounded multiply: the function is inlined at several places and the
    // tie-break between duplicate spheres (lowest index) needs the same bits from each of them
    const float dx = t.x - x, dy = t.y - y, dz = t.z;
    const float du = fmaf(dx, ux, fmaf(dy, uy, __fmul_rn(dz, uz)));
    // squared miss distance from the perpendicular part of (centre - point): |d|^2 - du^2 cancels when a grazing ray
    // meets the plane kilometres from the telescope (10 cm at 2 km in fp32)
    const float qx = fmaf(-du, ux, dx), qy = fmaf(-du, uy, dy), qz = fmaf(-du, uz, dz);
    const float m2 = fmaf(qx, qx, fmaf(qy, qy, __fmul_rn(qz, qz)));
    const float r2 = __fmul_rn(t.w, t.w);
    if (m2 <= r2) {
        const float s_in = __fsub_rn(du, sqrtf(__fsub_rn(r2, m2)));
        if (s_in < best_s || (s_in == best_s && k < best_k)) { best_s = s_in; best_k = k; }
    }
}

// nearest entry along the arrival ray, lowest index on ties.  `cell` < -1: brute force over all
// telescopes; otherwise the sorted candidates of the cell while key <= thr (thr >= 1/|u_z|).
// (t0, kn0) = the cell's first listed telescope and (its index, list length), loaded by the caller ahead of time.
__device__ __forceinline__ int tel_hit_search(const DevDet &det, int cell, float thr, float x, float y,
                                           float ux, float uy, float uz, const float4 t0, const int2 kn0)
{
    int best_k = -1;
    float best_s = CUDART_INF_F;
    if (cell < -1) {
        for (int k = 0; k < det.n_tel; ++k) sphere_test(det, k, x, y, ux, uy, uz, best_s, best_k);
        return best_k;
    }
    if (cell < 0 || kn0.y <= 0) return -1;
    // the first entry has the smallest key; the pre-test already compared it (rounded down) with the threshold
    sphere_test_rec(t0, kn0.x, x, y, ux, uy, uz, best_s, best_k);
    if (kn0.y == 1) return best_k;
    const int hi = __ldg(det.hit.start + cell + 1);
    for (int i = __ldg(det.hit.start + cell) + 1; i < hi; ++i) {
        const float2 e = __ldg(det.hit.items + i);
        if (e.x > thr) break;
        sphere_test(det, __float_as_int(e.y), x, y, ux, uy, uz, best_s, best_k);
    }
    return best_k;
}

// LV2/LV3 proximity: is (x,y) within r_k/|u_z| + margin of any telescope centre?  (single exit)
__device__ __forceinline__ bool tel_near_search(const DevDet &det, int cell, float thr, float x, float y,
                                                float inv_abs_uz, float margin)
{
    bool found = false;
    if (cell < -1) {
        for (int k = 0; k < det.n_tel && !found; ++k) {
            const float4 t = __ldg(det.tel + k);
            const float dx = x - t.x, dy = y - t.y, reach = fmaf(t.w, inv_abs_uz, margin);
            found = dx * dx + dy * dy <= reach * reach;
        }
    } else if (cell >= 0) {
        const int hi = __ldg(det.lv2.start + cell + 1);
        for (int i = __ldg(det.lv2.start + cell); i < hi && !found; ++i) {
            const float2 e = __ldg(det.lv2.items + i);
            if (e.x > thr) break;
            const float4 t = __ldg(det.tel + __float_as_int(e.y));
            const float dx = x - t.x, dy = y - t.y, reach = fmaf(t.w, inv_abs_uz, margin);
            found = dx * dx + dy * dy <= reach * reach;
        }
    }
    return found;
}

// ---- R22 (thesis sec. 6.4): refraction at a boundary (vector Snell, Eq. 3.15) and absorbing capsules ----------------
// u -> out across a surface with unit normal N from index n1 into n2; false: total internal reflection
__device__ __forceinline__ bool refract_vec(float ux, float uy, float uz, float Nx, float Ny, float Nz, float n1, float n2,
                                            float &ox, float &oy, float &oz)
{
    const float c = ux * Nx + uy * Ny + uz * Nz;
    const float sgn = c < 0.f ? -1.f : 1.f, ca = fabsf(c);
    const float q = fmaf(n2, n2, fmaf(n1 * n1, ca * ca, -n1 * n1));
    if (q < 0.f) return false;
    const float k = (sqrtf(q) - n1 * ca) * sgn, in2 = 1.f / n2;
    ox = fmaf(k, Nx, n1 * ux) * in2; oy = fmaf(k, Ny, n1 * uy) * in2; oz = fmaf(k, Nz, n1 * uz) * in2;
    return true;
}

// squared distance between the segments P0 -> P1 and Q0 -> Q1
__device__ float segment_dist2(const float3 P0, const float3 P1, const float3 Q0, const float3 Q1)
{
    const float3 d1 = make_float3(P1.x - P0.x, P1.y - P0.y, P1.z - P0.z), d2 = make_float3(Q1.x - Q0.x, Q1.y - Q0.y, Q1.z - Q0.z);
    const float3 r = make_float3(P0.x - Q0.x, P0.y - Q0.y, P0.z - Q0.z);
    const float a = d1.x * d1.x + d1.y * d1.y + d1.z * d1.z, e = d2.x * d2.x + d2.y * d2.y + d2.z * d2.z;
    const float f = d2.x * r.x + d2.y * r.y + d2.z * r.z, c = d1.x * r.x + d1.y * r.y + d1.z * r.z;
    const float b = d1.x * d2.x + d1.y * d2.y + d1.z * d2.z;
    float sN = 0.f, tN = 0.f;
    if (a <= 1e-30f && e <= 1e-30f) { }
    else if (a <= 1e-30f) tN = fminf(fmaxf(f / e, 0.f), 1.f);
    else if (e <= 1e-30f) sN = fminf(fmaxf(-c / a, 0.f), 1.f);
    else {
        const float den = a * e - b * b;
        sN = den > 1e-12f * a * e ? fminf(fmaxf((b * f - c * e) / den, 0.f), 1.f) : 0.f;
        tN = (b * sN + f) / e;
        if (tN < 0.f) { tN = 0.f; sN = fminf(fmaxf(-c / a, 0.f), 1.f); }
        else if (tN > 1.f) { tN = 1.f; sN = fminf(fmaxf((b - c) / a, 0.f), 1.f); }
    }
    const float dx = r.x + sN * d1.x - tN * d2.x, dy = r.y + sN * d1.y - tN * d2.y, dz = r.z + sN * d1.z - tN * d2.z;
    return dx * dx + dy * dy + dz * dz;
}

__device__ bool leg_absorbed(const DevDet &det, const float3 A, const float3 B)
{
    for (int k = 0; k < det.opt_n_abs; ++k) {
        const float *o = det.opt_abs[k];
        if (segment_dist2(A, B, make_float3(o[0], o[1], o[2]), make_float3(o[3], o[4], o[5])) <= o[6] * o[6]) return true;
    }
    return false;
}

// hexagonal camera pixel of an arrival direction (cfg3); -1 outside.  Nearest centre among the
// rows/columns adjacent to the point (equivalent to the brute-force nearest centre).
__device__ __forceinline__ int camera_pixel(const DevDet &det, float ux, float uy, float uz)
{
    const float vx = -ux, vy = -uy, vz = -uz;
    const float vw = vx * det.cam_w[0] + vy * det.cam_w[1] + vz * det.cam_w[2];
    if (!(vw > 0.f)) return -1;
    const float a = atan2f(vx * det.cam_r[0] + vy * det.cam_r[1] + vz * det.cam_r[2], vw);
    const float e = atan2f(vx * det.cam_u[0] + vy * det.cam_u[1] + vz * det.cam_u[2], vw);
    const float p = det.cam_pitch, rp = p * 0.8660254037844386f;
    const float fr = e / rp + 0.5f * (float)(det.cam_rows - 1);
    const int r0 = (int)floorf(fr);
    int best = -1;
    float bd = CUDART_INF_F;
#pragma unroll
    for (int dr = 0; dr < 2; ++dr) {
        const int r = r0 + dr;
        if (r < 0 || r >= det.cam_rows) continue;
        const float ce = ((float)r - 0.5f * (float)(det.cam_rows - 1)) * rp;
        const float fc = a * det.cam_inv_pitch + 0.5f * (float)(det.cam_cols - 1) - 0.5f * (float)(r & 1);
        const int c0 = (int)floorf(fc);
#pragma unroll
        for (int dc = 0; dc < 2; ++dc) {
            const int c = c0 + dc;
            if (c < 0 || c >= det.cam_cols) continue;
            const float ca = ((float)c - 0.5f * (float)(det.cam_cols - 1) + 0.5f * (float)(r & 1)) * p;
            const float d2 = (a - ca) * (a - ca) + (e - ce) * (e - ce);
            const int idx = r * det.cam_cols + c;
            if (d2 < bd || (d2 == bd && idx < best)) { bd = d2; best = idx; }
        }
    }
    if (bd > p * p * (1.0f / 3.0f)) return -1;
    return best;
}

// 1: the planar layered Snell sum (TRACE_NUMERIC) in closed form from per-node layer moments where its series
//    converges to fp32 accuracy (no aerosol, nu_span / (n_e cos z)^2 < kLayerSeriesMax), the per-layer loop elsewhere;
//    0: always the loop
#ifndef C8PH_LAYER_MOMENTS
#define C8PH_LAYER_MOMENTS 1
#endif
constexpr float kLayerSeriesMax = 0.02f;

// a9 for a segment without a valid axis anchor (P_z >= -0.05: near-horizontal or up-going particle):
// plain Eq. 3.3 from the emission point.  Rare; kept out of line so the common path does not pay.
#ifndef C8PH_LINE_BY_VALUE
#define C8PH_LINE_BY_VALUE 1    // 1: the out-of-line general straight line returns its point in registers (no local-memory out-parameters)
#endif
#if C8PH_LINE_BY_VALUE
__device__ __noinline__ float2 line_general(const SegCold *sc, float s, float D, float Px, float Py, float ux, float uy)
{
    return make_float2(fmaf(D, ux, fmaf(s, Px, sc->Ax)), fmaf(D, uy, fmaf(s, Py, sc->Ay)));
}
#else
__device__ __noinline__ void line_general(const SegCold *sc, float s, float D, float Px, float Py, float ux, float uy,
                                          float &ox, float &oy)
{
    ox = fmaf(D, ux, fmaf(s, Px, sc->Ax));
    oy = fmaf(D, uy, fmaf(s, Py, sc->Ay));
}
#endif

// event counters of the CTA kept in shared memory (u64, shared-memory atomics once per segment group / counter flush),
// flushed to the global counters at the end
enum { WC_BELOW = 0, WC_LV1, WC_EMITTING, WC_CLIPPED, WC_NONFINITE, WC_EMITTED, WC_UP, WC_LV2, WC_TR, WC_ROUL, WC_GRID, WC_TEL,
       WC_CAM, WC_WRITTEN, WC_OVERFLOW, WC_N };

// ================================================================================================
// SPEC != 0 fixes the run-time switches to the array-detector production setting (LV2 on, Rayleigh
// roulette without aerosol, ground histogram + telescope grid, WRITE_TEL, all outputs present) and
// compiles in the optional features whose bits are set; the host picks the variant when the call
// matches one that is instantiated (launch_emit_propagate).  SPEC = 0 reads every switch at run time.
constexpr int kSpecBase = 1, kSpecFlat = 2, kSpecExt = 4, kSpecDisp = 8, kSpecEff = 16, kSpecOpt = 32, kSpecFlatTab = 64,
              kSpecNoGrid = 128;     // production setting without a ground histogram (telescope spheres only: BASELINE configs[2])
template <int EMIT, int TRACE, bool SPH, int SPEC>
__global__ void __launch_bounds__(kernel_threads(EMIT, TRACE, SPEC), kernel_min_blocks(TRACE))
k_emit_propagate(const __grid_constant__ KArgs a)
{
    static_assert(kSpecFlat == 2 && kSpecOpt == 32 && kSpecFlatTab == 64, "kernel_threads() names the feature bits by value");
    constexpr int kWarps = kernel_threads(EMIT, TRACE, SPEC) / 32;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t s_bar;
    __shared__ unsigned long long s_cnt[WC_N];               // event counters of the CTA (shared-memory atomics, rare)

    const HotConst &hc = a.hc;
    const DevAtm &atm = a.atm;
    const DevDet &det = a.det;
    const DevRun &run = a.run;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned FULL = 0xFFFFFFFFu;
    unsigned long long *cntp = reinterpret_cast<unsigned long long *>(run.out.counters);
    constexpr bool STAGED = TRACE == C8PH_TRACE_NUMERIC;     // n(h), overburden steps (and aerosol column) in shared memory
    constexpr bool STAGE_ETA = STAGED || (C8PH_ETA_STAGED && TRACE == C8PH_TRACE_TABLE);   // n(h) in shared memory

    // ---- shared memory carve-up: [n(h) tables] | per-warp candidate queue (SoA, kQueue entries)
    float *s_eta = reinterpret_cast<float *>(smem_raw);
    float *s_dxv = s_eta + (STAGE_ETA ? atm.n_pad : 0);
    float *s_aexp = s_dxv + (STAGED ? atm.n_pad : 0);       // aerosol column A(h_k) = (H/L) exp(-h_k/H), staged only with aerosol
    const bool aer_staged = STAGED && atm.aer_L > 0.f;
    float *s_end = s_aexp + (aer_staged ? atm.n_pad : 0);
    constexpr bool QC = queue_compact(SPEC);
    constexpr int QW = queue_words(SPEC);
    static_assert(QW == (QC ? Q_WORDS_COMPACT : Q_WORDS), "queue entry size");
    static_assert(kQueue == 64, "the push's plane offsets (16 + 1024 k, 3088) are written for 64 entries");
    // 16-word entries: s_q[slot * 4 + part]; compact: planes s_q[part * kQueue + slot] (part 0..2) and s_q3[slot]
    // compact layout: the warp's fill count sits in the 16 bytes in front of its planes, so that the push forms every
    // address from the one register that holds the count's shared-memory address (kQueueHead bytes per warp)
    constexpr int kQueueHead = QC ? 16 : 0;
    constexpr bool QG = QC && C8PH_QUEUE_GLOBAL;
    constexpr uint32_t kQBlock = kQueue * QW * 4 + kQueueHead;      // bytes per warp
    unsigned char *const q_cta = QG ? static_cast<unsigned char *>(run.qring) + (size_t)blockIdx.x * (kWarps * kQBlock)
                                    : reinterpret_cast<unsigned char *>(s_end);
    unsigned char *s_qblock = q_cta + (size_t)warp * kQBlock;
    float4 *s_q = reinterpret_cast<float4 *>(s_qblock + kQueueHead);
    float2 *s_q3 = reinterpret_cast<float2 *>(s_q + 3 * kQueue);
#if !C8PH_QUEUE_CONVERGED
    __shared__ int s_qn_static[(QC && !QG) ? 1 : kWarps];     // entries waiting in the warp's queue (16-word layout, global queues)
    int *const s_qn_w = (QC && !QG) ? reinterpret_cast<int *>(s_qblock) : &s_qn_static[warp];
    const uint32_t qn_addr = smem_u32(s_qn_w);
#endif
    // segment slots of this warp: global scratch owned by the context (L2-resident, re-read through L1)
    SegSlot *g_slot = static_cast<SegSlot *>(run.slots) + ((size_t)blockIdx.x * kWarps + warp) * 32;

    if (threadIdx.x < WC_N) s_cnt[threadIdx.x] = 0ull;
    __syncthreads();
#if !C8PH_QUEUE_CONVERGED
    if (lane == 0) *s_qn_w = 0;
#endif
    // ---- layered-sum variant: stage the atmosphere tables with one TMA bulk copy per array
    if (STAGE_ETA) {
        if (threadIdx.x == 0) {
            mbar_init(&s_bar, 1);
            const uint32_t bytes = (uint32_t)atm.n_pad * 4u;
            mbar_expect_tx(&s_bar, bytes * (STAGED ? (aer_staged ? 3u : 2u) : 1u));
            bulk_g2s(s_eta, atm.eta, bytes, &s_bar);
            if (STAGED) bulk_g2s(s_dxv, atm.dxv, bytes, &s_bar);
            if (aer_staged) bulk_g2s(s_aexp, atm.aexp, bytes, &s_bar);
        }
        __syncthreads();
        mbar_wait(&s_bar, 0);
    }
    __syncwarp();
    // n(h) node: shared memory when staged, otherwise through L1 (the lanes of a warp emit from one
    // short segment: 1-3 adjacent words, one cache line)
    auto eta_node = [&](int k) -> float { return STAGE_ETA ? s_eta[k] : __ldg(hc.eta + k); };

    // per-lane event counters of the photon loop, two 16-bit fields per register, flushed to
    // s_cnt before a field can overflow
    uint32_t pkA = 0, pkB = 0, pkC = 0;          // up | lv2<<16 ; tr | roul<<16 ; grid | tel<<16
    int iters_pending = 0;
    auto flush_counts = [&]() {
        const uint32_t v0 = __reduce_add_sync(FULL, pkA & 0xFFFFu), v1 = __reduce_add_sync(FULL, pkA >> 16);
        const uint32_t v2 = __reduce_add_sync(FULL, pkB & 0xFFFFu), v3 = __reduce_add_sync(FULL, pkB >> 16);
        const uint32_t v4 = __reduce_add_sync(FULL, pkC & 0xFFFFu), v5 = __reduce_add_sync(FULL, pkC >> 16);
        if (lane == 0) {
            auto bump = [&](int idx, uint32_t v) { if (v) atomicAdd(&s_cnt[idx], (unsigned long long)v); };
            bump(WC_UP, v0); bump(WC_LV2, v1); bump(WC_TR, v2); bump(WC_ROUL, v3); bump(WC_GRID, v4); bump(WC_TEL, v5);
        }
        pkA = pkB = pkC = 0;
        iters_pending = 0;
    };

    const bool has_hist = SPEC ? !(SPEC & kSpecNoGrid) : (det.hist_nx > 0 && !det.cam_enabled && run.out.hist != nullptr);
    const bool has_grid_geom = SPEC ? !(SPEC & kSpecNoGrid) : (det.hist_nx > 0 && !det.cam_enabled);
    const bool f_lv2 = SPEC ? true : run.lv2 != 0;
    const bool f_tel = SPEC ? true : det.n_tel > 0;
    const bool f_grid = SPEC ? true : det.use_grid != 0;
    const bool f_hit_brute = SPEC ? false : run.hit_brute != 0;
    const int f_trans = SPEC ? (int)C8PH_TRANS_ROULETTE : run.trans;
    const bool f_ray = SPEC ? true : atm.ray_inv_X > 0.f;
    const bool f_aer = SPEC ? false : atm.aer_L > 0.f;
    const bool f_disp = SPEC ? (SPEC & kSpecDisp) != 0 : run.disp_b != 0.f;
    const bool f_eff = SPEC ? (SPEC & kSpecEff) != 0 : run.n_eff > 0;
    const bool f_opt = SPEC ? (SPEC & kSpecOpt) != 0 : det.opt_enabled != 0;
    const bool f_ext = SPEC ? (SPEC & kSpecExt) != 0 : atm.n_ext > 0;
    // flat observation plane: 1 = analytic step from the sphere (R19), 2 = the thesis' table with rho and pointing axes (R21)
    const int f_flat_mode = (!SPH || TRACE == C8PH_TRACE_STRAIGHT) ? 0 : (SPEC ? ((SPEC & kSpecFlat) ? 1 : ((SPEC & kSpecFlatTab) ? 2 : 0)) : run.flat_plane);
    const bool f_flat = f_flat_mode == 1;
    // cylindrical model (R24): generic variant only; geometry at the emission point as in the spherical model
    const bool f_cyl = SPEC ? false : (SPH && TRACE == C8PH_TRACE_TABLE && atm.model == C8PH_ATM_CYLINDRICAL);
    const bool f_flat_tab = TRACE == C8PH_TRACE_TABLE && f_flat_mode == 2;
    const int f_write = SPEC ? (int)C8PH_WRITE_TEL : run.write;
    const bool f_cam = SPEC ? false : det.cam_enabled != 0;
    const bool f_photons = SPEC ? true : run.out.photons != nullptr;
    const bool f_telc = SPEC ? true : run.out.tel_counts != nullptr;
    const float inv_ng = 1.0f / (1.0f + atm.eta_g);
    int q_head = 0;                                           // ring position of the oldest queue entry
#if C8PH_QUEUE_CONVERGED
    int q_n = 0;                                              // entries waiting in the warp's queue (warp-uniform register)
#endif

    // arrival direction: u turned in the ray plane (u, local vertical) by the angle that follows from the
    // Snell / Bouguer invariant (R9), small-angle form
    auto arrival_dir = [&](const SegCold *sc, float ux, float uy, float uz, float cz, float eta_e, float h_e, float dd,
                           float &uax, float &uay, float &uaz) {
        uax = ux; uay = uy; uaz = uz;
        const float sinz = sqrt_fast(fmaxf(1.f - cz * cz, 0.f));
        if (TRACE != C8PH_TRACE_STRAIGHT && sinz >= 1e-6f) {
            const float eps = (eta_e - atm.eta_g) * inv_ng;
            const float scale = SPH ? 1.f + (h_e - (float)atm.h_obs) * run.inv_Rg : 1.f;
            const float al = sinz * scale;
            const float cyy = sqrt_fast(fmaxf(1.f - al * al, 0.f));
            const float at = al * (1.f + eps);
            const float cxx = sqrt_fast(fmaxf(1.f - at * at, 0.f));
            float dl = al * (eps * cyy + al * al * eps * (2.f + eps) * rcp_fast(cyy + cxx));
            if (SPH) dl -= dd * run.inv_Rg;
            const float k2 = dl * rcp_fast(sinz), k1 = fmaf(k2, cz, fmaf(-0.5f * dl, dl, 1.f));
            uax = fmaf(k1, ux, k2 * sc->rx);
            uay = fmaf(k1, uy, k2 * sc->ry);
            uaz = fmaf(k1, uz, k2 * sc->rz);
        }
    };

    // ---- a13/a14/a16 for photons that may hit a telescope or are written anyway: arrival direction
    // (rotation in the ray plane by the Snell / Bouguer invariant), exact sphere search, counters,
    // ballot-compacted record store.  Called warp-converged; `act` marks the lanes that carry a photon.
    auto finish = [&](bool act, float4 q0, float4 q1, float4 q2, float4 q3) {
        const float ux = q0.z, uy = q0.w, uz = q1.x, s = q1.y, qw = q1.z, dt = q1.w;
        const float lam_inv = q2.x, wgt = q2.y, eta_e = q2.z, dd = q3.x, cz = q3.y;
        int cell = __float_as_int(q3.z);
        const uint32_t jslot = __float_as_uint(q3.w);
        float h_e = q2.w;
        if (QC) {                                             // compact entry: the emission height from s, as the photon loop formed it
            const SegHot *shq = &(g_slot + (jslot & 31u))->h;
            h_e = fmaf(s, fmaf(s, shq->k2, shq->cA), shq->hA);
        }
        int tel = -1;
        float uax = ux, uay = uy, uaz = uz, t_arr = 0.f;
        float rx_out = 0.f, ry_out = 0.f;                     // record position (ground plane, or camera plane with optics)
        // a14: the first listed telescope of the photon's hit cell; loaded first so that the latency overlaps a13
        float4 t0 = make_float4(0.f, 0.f, 0.f, 0.f);
        int2 kn0 = make_int2(-1, 0);
        if (act && f_tel && cell >= 0) { t0 = __ldg(det.hit.first + cell); kn0 = __ldg(det.hit.first_kn + cell); }
        bool opt_hit = false;
        const SegSlot *sl = g_slot + (jslot & 31u);
        const SegHot *sh = &sl->h;
        const SegCold *sc = &sl->c;
        // with optics the entry carries the offset from the segment anchor, so that the ray's position on the
        // mirror does not go through an fp32 ground coordinate (0.24 mm at 3 km is 1.4e-5 rad after the mirror)
        const float xg = (f_opt && act) ? sh->Gx + q0.x : q0.x, yg = (f_opt && act) ? sh->Gy + q0.y : q0.y;
        rx_out = xg; ry_out = yg;
        if (act) {
            // a13: arrival time relative to t_ref
            if (sh->anchor & 1) {
                // (t - T_G) c = s delta/beta + (s + A_z/P_z)(q w_z - bn1 P_z)/(P_z + q w_z) + c dt
                const float Pz = sh->Pz;
                const float eta_c = f_disp ? eta_e * fmaf(run.disp_b, lam_inv * lam_inv, run.disp_c0) : eta_e;
                const float bn1 = fmaxf(fmaf(sh->beta, eta_c, -sh->delta), 0.f);
                const float num = fmaf(-bn1, Pz, qw);
                const float geo = (s + sh->AzP) * num * rcp_fast(Pz + qw);
                t_arr = sc->Tg + fmaf(fmaf(s, sh->dob, geo), kInvC, dt);
            } else {
                const float D = -fmaf(s, sh->Pz, sh->Az) * rcp_fast(uz);
                t_arr = sc->Tg + fmaf(fmaf(s, sh->inv_beta, D), kInvC, dt);
            }
            arrival_dir(sc, ux, uy, uz, cz, eta_e, h_e, dd, uax, uay, uaz);
            if (f_tel && cell != -1) {
                // the pre-test threshold must cover the rotated direction; if it does not (never in
                // air), search all telescopes
                const float thr = -rcp_fast(uz) * run.hit_infl;
                if (cell >= 0 && !(-uaz * thr >= 1.f)) cell = -2;
                tel = tel_hit_search(det, cell, thr, xg, yg, uax, uay, uaz, t0, kn0);
            }
            if (tel >= 0) {
                pkC += 0x10000u;
                if (f_telc) atomicAdd(run.out.tel_counts + tel, wgt);
                if (f_opt) {
                    // last mile (thesis sec. 6.4): camera shadow, parabolic mirror z = rho^2/(4f) about the
                    // pointing axis (vertex at centre - (f/2) w), reflection, camera disc at z = f
                    const float4 tc = __ldg(det.tel + tel);
                    const float f = det.opt_f, hf = 0.5f * f;
                    const float lox = (sh->anchor & 1) ? sc->Ax : 0.f, loy = (sh->anchor & 1) ? sc->Ay : 0.f;
                    const float px = (sh->Gx - tc.x) + (q0.x + lox) + hf * det.opt_w[0];
                    const float py = (sh->Gy - tc.y) + (q0.y + loy) + hf * det.opt_w[1], pz = -(tc.z - hf * det.opt_w[2]);
                    const float a0 = px * det.opt_r[0] + py * det.opt_r[1] + pz * det.opt_r[2];
                    const float b0 = px * det.opt_u[0] + py * det.opt_u[1] + pz * det.opt_u[2];
                    const float z0 = px * det.opt_w[0] + py * det.opt_w[1] + pz * det.opt_w[2];
                    const float dr = uax * det.opt_r[0] + uay * det.opt_r[1] + uaz * det.opt_r[2];
                    const float du = uax * det.opt_u[0] + uay * det.opt_u[1] + uaz * det.opt_u[2];
                    const float dw = uax * det.opt_w[0] + uay * det.opt_w[1] + uaz * det.opt_w[2];
                    // R22: start of the incoming leg = entry into the bounding sphere (frame about the sphere centre)
                    const float3 g0 = make_float3(a0, b0, z0 - hf);
                    float3 Een = g0;
                    if (det.opt_n_abs > 0 || det.opt_kind == 1) {
                        const float bq = g0.x * dr + g0.y * du + g0.z * dw, cq = g0.x * g0.x + g0.y * g0.y + g0.z * g0.z - tc.w * tc.w;
                        const float s_in = -bq - sqrtf(fmaxf(bq * bq - cq, 0.f));
                        Een = make_float3(fmaf(s_in, dr, g0.x), fmaf(s_in, du, g0.y), fmaf(s_in, dw, g0.z));
                    }
                    if (det.opt_kind == 1) {
                        // plano-convex lens (R22): convex face towards the sky, plane face at +f/2, camera at -f/2 (about the centre)
                        const float Rl = det.opt_lens_roc, nl = det.opt_lens_n, zc = hf + det.opt_lens_t - Rl;
                        const float ocz = g0.z - zc;
                        const float b2 = g0.x * dr + g0.y * du + ocz * dw, c2 = g0.x * g0.x + g0.y * g0.y + ocz * ocz - Rl * Rl;
                        const float disc = b2 * b2 - c2;
                        if (dw < 0.f && disc >= 0.f) {
                            const float s1 = -b2 - sqrtf(disc);
                            const float3 P1 = make_float3(fmaf(s1, dr, g0.x), fmaf(s1, du, g0.y), fmaf(s1, dw, g0.z));
                            float vx, vy, vz, v2x, v2y, v2z;
                            if (P1.x * P1.x + P1.y * P1.y <= det.opt_rm2 && P1.z >= hf && !leg_absorbed(det, Een, P1) &&
                                refract_vec(dr, du, dw, P1.x / Rl, P1.y / Rl, (P1.z - zc) / Rl, 1.f, nl, vx, vy, vz) && vz < 0.f) {
                                const float s2 = (hf - P1.z) / vz;
                                const float3 P2 = make_float3(fmaf(s2, vx, P1.x), fmaf(s2, vy, P1.y), hf);
                                if (P2.x * P2.x + P2.y * P2.y <= det.opt_rm2 && refract_vec(vx, vy, vz, 0.f, 0.f, 1.f, nl, 1.f, v2x, v2y, v2z) && v2z < 0.f) {
                                    const float s3 = (-hf - P2.z) / v2z;
                                    const float3 P3 = make_float3(fmaf(s3, v2x, P2.x), fmaf(s3, v2y, P2.y), -hf);
                                    if (!leg_absorbed(det, P2, P3) && P3.x * P3.x + P3.y * P3.y <= det.opt_rc2) {
                                        opt_hit = true;
                                        atomicAdd(&s_cnt[WC_CAM], 1ull);
                                        rx_out = P3.x; ry_out = P3.y; uax = v2x; uay = v2y;
                                        t_arr = fmaf(s1 + nl * s2 + s3, kInvC, t_arr);
                                    }
                                }
                            }
                        }
                    } else
                    if (dw < 0.f) {
                        const float sc0 = (f - z0) * rcp_fast(dw);
                        const float xs = fmaf(sc0, dr, a0), ys = fmaf(sc0, du, b0);
                        if (xs * xs + ys * ys > det.opt_rc2) {                       // not shadowed by the camera
                            const float A = dr * dr + du * du, B = 2.f * (a0 * dr + b0 * du) - 4.f * f * dw;
                            const float C = a0 * a0 + b0 * b0 - 4.f * f * z0;
                            float sh = 0.f;
                            bool ok = true;
                            if (A < 1e-12f) sh = -C * rcp_fast(B);
                            else {
                                const float disc = B * B - 4.f * A * C;
                                ok = disc >= 0.f;
                                const float sq = sqrt_fast(fmaxf(disc, 0.f));
                                const float qq = -0.5f * (B + (B >= 0.f ? sq : -sq));
                                const float s1 = qq * rcp_fast(A), s2 = qq != 0.f ? C * rcp_fast(qq) : s1;
                                sh = fmaxf(s1, s2);                                  // the ray leaves the bowl at the larger root
                            }
                            const float x = fmaf(sh, dr, a0), y = fmaf(sh, du, b0), z = fmaf(sh, dw, z0);
                            if (ok && x * x + y * y <= det.opt_rm2) {
                                const float i2f = 0.5f * rcp_fast(f);
                                float nx = -x * i2f, ny = -y * i2f;
                                const float inn = rsqrt_fast(nx * nx + ny * ny + 1.f);
                                nx *= inn; ny *= inn;
                                const float dn = dr * nx + du * ny + dw * inn;
                                const float r0 = fmaf(-2.f * dn, nx, dr), r1 = fmaf(-2.f * dn, ny, du), r2 = fmaf(-2.f * dn, inn, dw);
                                if (r2 > 0.f) {
                                    const float s2c = (f - z) * rcp_fast(r2);
                                    const float xc = fmaf(s2c, r0, x), yc = fmaf(s2c, r1, y);
                                    bool absorbed = false;                            // R22: truss shadowing on both legs
                                    if (det.opt_n_abs > 0) {
                                        const float3 Mp = make_float3(x, y, z - hf), Kp = make_float3(xc, yc, hf);
                                        absorbed = leg_absorbed(det, Een, Mp) || leg_absorbed(det, Mp, Kp);
                                    }
                                    if (!absorbed && xc * xc + yc * yc <= det.opt_rc2) {
                                        opt_hit = true;
                                        atomicAdd(&s_cnt[WC_CAM], 1ull);
                                        rx_out = xc; ry_out = yc; uax = r0; uay = r1;
                                        t_arr = fmaf(sh + s2c, kInvC, t_arr);
                                    }
                                }
                            }
                        }
                    }
                }
                if (f_cam) {
                    const int pix = camera_pixel(det, uax, uay, uaz);
                    const float tb = floorf(t_arr * det.inv_t_bin);
                    if (pix >= 0 && tb >= 0.f && tb < (float)det.n_tbins) {
                        atomicAdd(&s_cnt[WC_CAM], 1ull);
                        if (run.out.hist) atomicAdd(run.out.hist + (size_t)pix * det.n_tbins + (int)tb, wgt);
                    }
                }
            }
        }
        // a16: survivors are ranked by warp ballot and stored straight from registers: one cursor
        // atomic per call, consecutive 32 B records
        const bool write = act && (f_write == C8PH_WRITE_ALL || (f_write == C8PH_WRITE_TEL && (f_opt ? opt_hit : tel >= 0)));
        if (f_photons) {
            const unsigned wm = __ballot_sync(FULL, write);
            if (wm) {
                unsigned long long base = 0;
                if (lane == 0) base = atomicAdd(&cntp[C8PH_CNT_WRITTEN], (unsigned long long)__popc(wm));
                base = __shfl_sync(FULL, base, 0);
                if (write) {
                    const long long idx = (long long)base + __popc(wm & ((1u << lane) - 1u));
                    if (idx < run.out.photon_capacity) {
                        uint4 *dst = reinterpret_cast<uint4 *>(run.out.photons + idx);
                        // records are written once and never read here: streaming stores (evict first)
                        __stcs(dst, make_uint4(__float_as_uint(rx_out), __float_as_uint(ry_out), __float_as_uint(uax), __float_as_uint(uay)));
                        __stcs(dst + 1, make_uint4(__float_as_uint(t_arr), __float_as_uint(rcp_fast(lam_inv)), sc->local,
                                                   ((jslot >> 5) << 14) | (tel >= 0 ? (uint32_t)tel : C8PH_TEL_NONE)));
                        if (run.out.photon_weight) __stcs(run.out.photon_weight + idx, wgt);
                    } else {
                        atomicAdd(&s_cnt[WC_OVERFLOW], 1ull);
                    }
                }
            }
        }
    };

    // take up to 32 queued candidates (all of them if `all`) through finish()
    auto drain = [&](bool all) {
        __syncwarp();
#if C8PH_QUEUE_CONVERGED
        int n = q_n;
#else
        int n = *s_qn_w;
#endif
        while (n >= 32 || (all && n > 0)) {
            const int take = n < 32 ? n : 32;
            const bool act = lane < take;
            if (QC) {
                const int qi = (q_head + lane) & (kQueue - 1);
                float4 p0, p1, p2;
                float2 p3;
                if (QG) { p0 = __ldcg(s_q + qi); p1 = __ldcg(s_q + kQueue + qi); p2 = __ldcg(s_q + 2 * kQueue + qi); p3 = __ldcg(s_q3 + qi); }
                else { p0 = s_q[qi]; p1 = s_q[kQueue + qi]; p2 = s_q[2 * kQueue + qi]; p3 = s_q3[qi]; }
                finish(act, p0, p1, make_float4(p2.x, hc.w, p2.y, 0.f), make_float4(p2.z, p2.w, p3.x, p3.y));
            } else {
                const float4 *e = s_q + ((q_head + lane) & (kQueue - 1)) * 4;
                finish(act, e[0], e[1], e[2], e[3]);
            }
            q_head = (q_head + take) & (kQueue - 1);
            n -= take;
            __syncwarp();
#if C8PH_QUEUE_CONVERGED
            q_n = n;
#else
            if (lane == 0) *s_qn_w = n;
            __syncwarp();
#endif
        }
    };

    for (;;) {
        // ---- grab a group of segments for this warp
        unsigned long long g0 = 0;
        if (lane == 0) g0 = atomicAdd(run.cursor, (unsigned long long)run.segs_per_grab);
        g0 = __shfl_sync(FULL, g0, 0);
        if ((long long)g0 >= run.n_seg) break;

        // ---- a1-a4: one lane prepares one segment (fp64) and parks it in its shared-memory slot
        int myN = 0;
        {
            const long long i = (long long)g0 + lane;
            bool below = false, lv1_drop = false, clipped = false, nonfinite = false;
            if (lane < run.segs_per_grab && i < run.n_seg) {
                SegHot me;
                SegCold mc;
                // inputs are read once: streaming loads, so that they do not push the tables out of L2
                const double Ax = __ldcs(run.seg.x + i), Ay = __ldcs(run.seg.y + i), Az = __ldcs(run.seg.z + i);
                double Px = __ldcs(run.seg.dx + i), Py = __ldcs(run.seg.dy + i), Pz = __ldcs(run.seg.dz + i);
                const double L = __ldcs(run.seg.len + i), beta = __ldcs(run.seg.beta + i), t0 = __ldcs(run.seg.t0 + i);
                const double pn = 1.0 / sqrt(Px * Px + Py * Py + Pz * Pz);
                Px *= pn; Py *= pn; Pz *= pn;
                // a non-finite input field or a zero direction: the segment is dropped and counted (C8PH_CNT_NONFINITE)
                {
                    double chk = Ax + Ay + Az + Px + Py + Pz + L + beta + t0 + (double)__ldcs(run.seg.charge + i);
                    if (EMIT == C8PH_EMIT_FLUORESCENCE && run.seg.edep) chk += (double)run.seg.edep[i];
                    nonfinite = !(fabs(chk) < CUDART_INF);
                }
                const unsigned long long gid = run.seg.id ? (unsigned long long)__ldcs(run.seg.id + i) : (unsigned long long)(run.seg_id_base + i);
                me.id_lo = (uint32_t)gid; me.id_hi = (uint32_t)(gid >> 32); mc.local = run.local_base + (uint32_t)i;
                // local vertical and height at A and at the midpoint
                double rx = 0.0, ry = 0.0, rz = 1.0, rA = 1.0, hA, h_mid;
                const double mx = Ax + 0.5 * L * Px, my = Ay + 0.5 * L * Py, mz = Az + 0.5 * L * Pz;
                if (SPH) {
                    const double zz = Az + atm.Rg;
                    rA = sqrt(Ax * Ax + Ay * Ay + zz * zz);
                    rx = Ax / rA; ry = Ay / rA; rz = zz / rA;
                    hA = rA - atm.R;
                    const double zm = mz + atm.Rg;
                    h_mid = sqrt(mx * mx + my * my + zm * zm) - atm.R;
                } else {
                    hA = atm.h_obs + Az;
                    h_mid = atm.h_obs + mz;
                }
                const double cA = Px * rx + Py * ry + Pz * rz;
                double n_exp = 0.0;
                const uint4 rs = philox4x32_10(0xFFFFFFFFu, me.id_lo, me.id_hi, 0u, hc.key);
                float e1x, e1y, e1z, e2x, e2y, e2z;
                mc.aimx = mc.aimy = mc.aimz = mc.omc = 0.f;
                if (EMIT == C8PH_EMIT_CHERENKOV) {
                    // Frank-Tamm, Eq. 2.2-2.4, n at the segment mid height
                    const double eta_mid = eta_lookup_d(atm, h_mid);
                    double n_mid = 1.0 + eta_mid;
                    const double zq = __ldcs(run.seg.charge + i);
                    mc.eta_mid = (float)eta_mid;                      // eta at the mid height (dispersive sampling)
                    if (run.disp_b != 0.f) {
                        // dispersion: yield integral over the band with the threshold;
                        // LV1 below uses the largest n of the band (blue end)
                        const double k1 = run.il1_d, k2 = run.il2_d, b = run.disp_b;
                        n_exp = (2.0 * 3.14159265358979323846 * kAlphaFS * 1.0e9) * zq * zq * L *
                                disp_yield_integral(beta, eta_mid, b, run.disp_k0sq, k2, k1);
                        n_mid = 1.0 + eta_mid * (1.0 + b * (k1 * k1 - run.disp_k0sq));
                    }
                    const double bn = beta * n_mid;
                    const double sin2 = 1.0 - 1.0 / (bn * bn);
                    if (run.disp_b == 0.f && sin2 > 0.0) n_exp = run.yield_k * zq * zq * L * sin2;
                    if (n_exp > 0.0 && run.lv1) {
                        // LV1, Eq. 4.3: angle between P and the direction to the array centre
                        const double dist = sqrt(mx * mx + my * my + mz * mz);
                        double cosa = -(Px * mx + Py * my + Pz * mz) / dist;
                        cosa = fmin(1.0, fmax(-1.0, cosa));
                        const double theta_c = acos(fmin(1.0, 1.0 / bn));
                        const double ratio = fmin(1.0, det.r_array / dist);
                        lv1_drop = acos(cosa) > theta_c + asin(ratio) + run.lv1_margin;
                    }
                    // Rodrigues half-turn about the bisector of D = (0,0,-1) and P
                    const double Bx = Px, By = Py, Bz = Pz - 1.0;
                    const double b2 = Bx * Bx + By * By + Bz * Bz;
                    if (Pz > 1.0 - 1e-6 || b2 <= 0.0) {
                        e1x = 1.f; e1y = 0.f; e1z = 0.f; e2x = 0.f; e2y = -1.f; e2z = 0.f;
                    } else {
                        const double k = 2.0 / b2;
                        e1x = (float)(k * Bx * Bx - 1.0); e1y = (float)(k * Bx * By); e1z = (float)(k * Bx * Bz);
                        e2x = (float)(k * By * Bx); e2y = (float)(k * By * By - 1.0); e2z = (float)(k * By * Bz);
                    }
                } else {
                    // fluorescence: N = Y E_dep Omega/4pi, forced cone towards the pre-corrected aim point
                    const float4 t0v = __ldg(det.tel);
                    const double dx = t0v.x - mx, dy = t0v.y - my, dz = t0v.z - mz;
                    const double dist = sqrt(dx * dx + dy * dy + dz * dz);
                    double aimx = t0v.x, aimy = t0v.y;
                    if (TRACE == C8PH_TRACE_TABLE) {
                        const double ux = dx / dist, uy = dy / dist, uz = dz / dist;
                        double vx = 0, vy = 0, vz = 1;
                        if (SPH) {
                            const double zm = mz + atm.Rg, rm = sqrt(mx * mx + my * my + zm * zm);
                            vx = mx / rm; vy = my / rm; vz = zm / rm;
                        }
                        const double cz = -(ux * vx + uy * vy + uz * vz);
                        const double hn = sqrt(ux * ux + uy * uy);
                        if (cz > 0.0 && hn > 1e-9) {
                            // same bilinear rule as the per-photon lookup, in fp64 on the stored fp32 nodes
                            const DevTable &t = a.tab;
                            const double thz = acos(fmin(1.0, cz));
                            if (h_mid >= 0.0 && h_mid <= (double)t.h_max && thz <= (double)t.zen_max) {
                                const double f = h_mid / ((double)t.h_max / (t.n_h - 1)), g = thz / ((double)t.zen_max / (t.n_zen - 1));
                                const int ia = min((int)f, t.n_h - 2), ib = min((int)g, t.n_zen - 2);
                                const double ff = f - ia, gg = g - ib;
                                const float4 *p = t.hot + (size_t)ia * t.n_zen + ib;
                                const double v = (1 - ff) * ((1 - gg) * (double)__ldg(p).x + gg * (double)__ldg(p + 1).x)
                                               + ff * ((1 - gg) * (double)__ldg(p + t.n_zen).x + gg * (double)__ldg(p + t.n_zen + 1).x);
                                if (v == v) { aimx -= v * ux / hn; aimy -= v * uy / hn; }
                            }
                        }
                    }
                    // relative to the start point, in fp64: the cone axis must not go through fp32 ground coordinates
                    // (2 mm at 20 km is 2e-4 rad for an emission point 10 m from the telescope)
                    mc.aimx = (float)(aimx - Ax); mc.aimy = (float)(aimy - Ay); mc.aimz = (float)((double)t0v.z - Az);
                    const double rho = run.aim_factor * (double)t0v.w;
                    const double sp = fmin(1.0, rho / dist);
                    const double cps = sqrt(1.0 - sp * sp);
                    const double omc = sp * sp / (1.0 + cps);                 // 1 - cos(psi), cancellation-free
                    mc.omc = (float)omc;
                    const float *ed = run.seg.edep;
                    n_exp = run.fluor_yield * (ed ? (double)ed[i] : 0.0) * 0.5 * omc;
                    e1x = e1y = e1z = e2x = e2y = e2z = 0.f;
                    mc.eta_mid = 0.f;
                }
                long long N = 0;
                if (nonfinite) { n_exp = 0.0; lv1_drop = false; }
                else if (!(n_exp > 0.0)) below = true;
                else if (!lv1_drop) {
                    N = (long long)floor(n_exp / (double)run.w + u01d(rs.x));
                    if (N >= C8PH_MAX_BUNCHES_PER_SEGMENT) { clipped = true; N = C8PH_MAX_BUNCHES_PER_SEGMENT - 1; }
                }
                myN = (int)N;
                if (myN > 0) {
                    me.N = myN;
                    me.Px = (float)Px; me.Py = (float)Py; me.Pz = (float)Pz;
                    me.e1x = e1x; me.e1y = e1y; me.e2y = e2y;
                    me.q0 = me.q1 = me.q2 = 0.f;
                    mc.Ax = (float)Ax; mc.Ay = (float)Ay; me.Az = (float)Az;
                    me.L = (float)L; me.beta = (float)beta; me.delta = 1.0f - (float)beta;
                    me.hA = (float)hA; me.cA = (float)cA; me.k2 = SPH ? (float)((1.0 - cA * cA) / (2.0 * rA)) : 0.f;
                    mc.rx = (float)rx; mc.ry = (float)ry; mc.rz = (float)rz; me.inv_rA = SPH ? (float)(1.0 / rA) : 0.f;
                    me.a1 = e1x * mc.rx + e1y * mc.ry + e1z * mc.rz;
                    me.a2 = e2x * mc.rx + e2y * mc.ry + e2z * mc.rz;
                    // axis landing anchor (fp64): G = A - A_z P / P_z, its clock, its grid coordinate
                    // (a segment that reaches z <= 0 takes the general form, which checks every emission point)
                    me.anchor = (EMIT == C8PH_EMIT_CHERENKOV && Pz < -0.05 && Az > 0.0 && Az + L * Pz > 0.0) ? 1 : 0;
#if C8PH_ETA_SEGFIT
                    if (EMIT == C8PH_EMIT_CHERENKOV && TRACE != C8PH_TRACE_NUMERIC) {
                        // Listing 4.1 along the segment: eta(h(s)) is piecewise quadratic in s (linear in h between nodes,
                        // h quadratic in s).  One quadratic through s = 0, L/2, L replaces the per-photon lookup if it
                        // reproduces the table at every node the segment crosses and half-way between them.
                        const double hA32 = (double)me.hA, cA32 = (double)me.cA, k232 = (double)me.k2;   // what the photon uses
                        auto h_of = [&](double sv) { return hA32 + sv * (cA32 + sv * k232); };
                        const double f0 = eta_lookup_d(atm, h_of(0.0)), fm = eta_lookup_d(atm, h_of(0.5 * L)), f1 = eta_lookup_d(atm, h_of(L));
                        const double c2 = L > 0.0 ? 2.0 * (f1 - 2.0 * fm + f0) / (L * L) : 0.0;
                        const double c1 = L > 0.0 ? (-3.0 * f0 + 4.0 * fm - f1) / L : 0.0;
                        const float q0f = (float)f0, q1f = (float)c1, q2f = (float)c2;
                        auto fit = [&](double sv) { return (double)q0f + sv * ((double)q1f + sv * (double)q2f); };
                        const double ha = h_of(0.0), hb = h_of(L), dhn = (double)atm.dh;
                        const double ka = (fmin(ha, hb) - (double)atm.h0) / dhn, kb = (fmax(ha, hb) - (double)atm.h0) / dhn;
                        bool ok = fabs(cA32) > 1e-3 && kb - ka < 8.0;                 // monotonic height, a few nodes at most
                        if (ok) {
                            const double tol = 4e-7 * fmax(fabs(fm), 1e-12);
                            double s_prev = 0.0, err = fmax(fabs(fit(0.5 * L) - fm), fabs(fit(L) - f1));
                            const int k_lo = (int)ceil(ka), k_hi = (int)floor(kb);
                            // nodes in the order the particle meets them
                            for (int t = 0; t <= k_hi - k_lo + 1; ++t) {
                                double s_k = L;
                                if (t <= k_hi - k_lo) {
                                    const int kn = cA32 < 0.0 ? k_hi - t : k_lo + t;
                                    s_k = fmin(fmax((((double)atm.h0 + kn * dhn) - hA32) / cA32, 0.0), L);
                                }
                                const double sm = 0.5 * (s_prev + s_k);
                                err = fmax(err, fmax(fabs(fit(sm) - eta_lookup_d(atm, h_of(sm))), fabs(fit(s_k) - eta_lookup_d(atm, h_of(s_k)))));
                                s_prev = s_k;
                            }
                            ok = err <= tol;
                        }
                        if (ok) { me.q0 = q0f; me.q1 = q1f; me.q2 = q2f; me.anchor |= 2; }
                    }
#endif
                    me.Gx = me.Gy = me.AzP = 0.f;
                    mc.fbx = mc.fby = 0.f; mc.ibx = mc.iby = 0;
                    me.dob = (float)((double)me.delta / beta); me.inv_beta = (float)(1.0 / beta);
                    if (me.anchor & 1) {
                        const double azp = Az / Pz;
                        const double Gx = Ax - azp * Px, Gy = Ay - azp * Py;
                        me.Gx = (float)Gx; me.Gy = (float)Gy; me.AzP = (float)azp;
                        // anchor form: Ax, Ay are free and carry what fp32 loses of the anchor (last-mile optics)
                        mc.Ax = (float)(Gx - (double)me.Gx); mc.Ay = (float)(Gy - (double)me.Gy);
                        mc.Tg = (float)(t0 - azp / kC - det.t_ref);
                        if (has_grid_geom) {
                            const double bx = (Gx - (double)det.hist_x0) / (double)det.hist_cell;
                            const double by = (Gy - (double)det.hist_y0) / (double)det.hist_cell;
                            const double fx = fmin(fmax(floor(bx), -1.0e9), 1.0e9), fy = fmin(fmax(floor(by), -1.0e9), 1.0e9);
                            mc.ibx = (int)fx; mc.iby = (int)fy;
                            mc.fbx = (float)(bx - fx); mc.fby = (float)(by - fy);
                        }
                    } else {
                        mc.Tg = (float)(t0 - det.t_ref);
                        if (has_grid_geom) {                         // bin = floor(x / cell + fb) with G = 0
                            mc.fbx = (float)(-(double)det.hist_x0 / (double)det.hist_cell);
                            mc.fby = (float)(-(double)det.hist_y0 / (double)det.hist_cell);
                        }
                    }
                    copy16(&g_slot[lane].h, &me);
                    copy16(&g_slot[lane].c, &mc);
                }
            }
            // segment-level counters of the group: one ballot each, lane 0 books them
            const unsigned mb = __ballot_sync(FULL, below), ml = __ballot_sync(FULL, lv1_drop), mcl = __ballot_sync(FULL, clipped);
            const unsigned me_ = __ballot_sync(FULL, myN > 0), mnf = __ballot_sync(FULL, nonfinite);
            const uint32_t nsum = __reduce_add_sync(FULL, (uint32_t)myN);
            if (lane == 0) {
                auto bump = [&](int idx, unsigned v) { if (v) atomicAdd(&s_cnt[idx], (unsigned long long)v); };
                bump(WC_BELOW, __popc(mb)); bump(WC_LV1, __popc(ml)); bump(WC_CLIPPED, __popc(mcl));
                bump(WC_EMITTING, __popc(me_)); bump(WC_NONFINITE, __popc(mnf)); bump(WC_EMITTED, nsum);
            }
        }
        unsigned emask = __ballot_sync(FULL, myN > 0);
        __syncwarp();

        // ---- a5-a16: the warp walks the emitting segments; lanes stride over the photons
        while (emask) {
            const int src = __ffs(emask) - 1;
            emask &= emask - 1;
            const SegSlot *sl = g_slot + src;
            asm volatile("" : "+l"(sl));                              // keep the slot address in registers
            SegHot sg;
            copy16(&sg, &sl->h);                                      // uniform address: one sector per LDG.128
            const SegCold *sc = &sl->c;                               // cold fields are re-read (L1) where used
#if C8PH_SLOT_PREFETCH
            if (emask && lane < 3)                                    // next emitting segment of the group: 176 B from L2 into L1
                asm volatile("prefetch.global.L1 [%0];" ::"l"(reinterpret_cast<const char *>(g_slot + (__ffs(emask) - 1)) + lane * 88 - (lane >> 1)));
#endif
            const int n_iter = (sg.N + 31) >> 5;
            if (iters_pending + n_iter > 60000) flush_counts();
            iters_pending += n_iter;
            // the loop variable is the queue entry's last word, js = j << 5 | slot of the segment (j = 32 it + lane): the photon
            // index is one shift away and neither the lane index nor the slot number needs a register of its own
            for (uint32_t js = ((uint32_t)lane << 5) | (uint32_t)src; js < ((uint32_t)n_iter << 10); js += 1024u) {
                const int j = (int)(js >> 5);
#if C8PH_QUEUE_VOTE && C8PH_QUEUE_LANE_ATOMS && !C8PH_QUEUE_CONVERGED
                bool qfull = false;
#endif
#if C8PH_QUEUE_CONVERGED
                bool qpush = false;
                float4 qe0, qe1, qe2, qe3;                            // defined where qpush is set
#endif
                // one photon per lane; every cut leaves through the same exit (one reconvergence point)
                if (js < ((uint32_t)sg.N << 5)) do {                  // j < N
                    const uint4 rn = philox4x32_10((uint32_t)j, sg.id_lo, sg.id_hi, 0u, hc.key);
                    const float u1 = u01(rn.y), u2 = u01(rn.z);
                    // a6: emission point on the track, its height and n(h_e) (Listing 4.1)
                    const float s = u1 * sg.L;
                    const float h_e = fmaf(s, fmaf(s, sg.k2, sg.cA), sg.hA);
                    float eta_e;
#if C8PH_ETA_SEGFIT
                    if (sg.anchor & 2) eta_e = fmaf(s, fmaf(s, sg.q2, sg.q1), sg.q0);     // warp-uniform branch
                    else
#endif
                    {
                        float f = (h_e - hc.eta_h0) * hc.eta_inv_dh;
                        f = fminf(fmaxf(f, 0.f), hc.eta_fmax);
                        const int k = min((int)f, hc.eta_kmax);
                        const float e0 = eta_node(k), e1 = eta_node(k + 1);
                        eta_e = fmaf(f - (float)k, e1 - e0, e0);
                    }
                    float ux, uy, uz, lam_inv, cth = 1.f, q = 0.f, pqz = 0.f, wx = 0.f, wy = 0.f, wz = 0.f;
                    float sphi, cphi;
                    sincos_2pi_u(rn.x, sphi, cphi);                       // phi = 2 pi u0
                    if (EMIT == C8PH_EMIT_CHERENKOV) {
                        // a6/a7: cos(theta_c) = 1/(beta n(h_e)) (Eq. 2.5), beta n - 1 without cancellation
                        lam_inv = fmaf(-u2, hc.dil, hc.il1);            // 1/lambda uniform
                        float eta_c = eta_e;                            // refractivity that sets the cone angle
                        if (f_disp) {
                            // dispersion (Eq. 2.5): spectrum lambda^-2 sin^2 theta(lambda) by rejection from
                            // the 1/lambda-uniform law (n at the segment mid height); trial t takes uniforms
                            // (2 (t&1), 2 (t&1) + 1) of Philox stream 2 + t/2; then n(lambda, h_e) for the angle
                            const float em = sc->eta_mid * sg.beta;
                            auto sin2 = [&](float k) {
                                const float x = fmaxf(fmaf(em, fmaf(run.disp_b, k * k, run.disp_c0), -sg.delta), 0.f);
                                return x * (2.f + x) * rcp_fast((1.f + x) * (1.f + x));
                            };
                            const float smax = fmaxf(sin2(hc.il1), sin2(hc.il1 - hc.dil));
                            uint4 rt = make_uint4(0u, 0u, 0u, 0u);
                            for (int t = 0; t < 32; ++t) {
                                if (!(t & 1)) rt = philox4x32_10((uint32_t)j, sg.id_lo, sg.id_hi, 2u + (uint32_t)(t >> 1), hc.key);
                                lam_inv = fmaf(-u01((t & 1) ? rt.z : rt.x), hc.dil, hc.il1);
                                if (u01((t & 1) ? rt.w : rt.y) * smax < sin2(lam_inv)) break;
                            }
                            eta_c = eta_e * fmaf(run.disp_b, lam_inv * lam_inv, run.disp_c0);
                        }
                        const float bn1 = fmaxf(fmaf(sg.beta, eta_c, -sg.delta), 0.f);
                        q = sqrt_fast(bn1 * (2.f + bn1));               // tan(theta_c)
                        cth = rcp_fast(1.f + bn1);                      // cos(theta_c)
                        // M = 2 A A^T - 1 is symmetric with third column -P: e2x = e1y, e1z = -P_x, e2z = -P_y
                        wx = cphi * sg.e1x + sphi * sg.e1y;
                        wy = cphi * sg.e1y + sphi * sg.e2y;
                        wz = -(cphi * sg.Px + sphi * sg.Py);
                        pqz = fmaf(q, wz, sg.Pz);
                        ux = cth * fmaf(q, wx, sg.Px);
                        uy = cth * fmaf(q, wy, sg.Py);
                        uz = cth * pqz;
                    } else {
                        // fluorescence: uniform in the cone about (aim - A_e)
                        int li = 0;
                        while (li < run.n_lines - 1 && u2 >= __ldg(run.line_cdf + li)) ++li;
                        lam_inv = 1.0f / __ldg(run.line_nm + li);
                        const uint4 rb = philox4x32_10((uint32_t)j, sg.id_lo, sg.id_hi, 1u, hc.key);
                        float ax = fmaf(-s, sg.Px, sc->aimx), ay = fmaf(-s, sg.Py, sc->aimy), az = fmaf(-s, sg.Pz, sc->aimz);
                        const float an = rsqrtf(ax * ax + ay * ay + az * az);
                        ax *= an; ay *= an; az *= an;
                        const float tt = u01(rb.x) * sc->omc;            // 1 - cos(polar)
                        const float cp = 1.f - tt, sp2 = sqrtf(tt * (2.f - tt));
                        float e1x = ay, e1y = -ax;
                        float e1n = e1x * e1x + e1y * e1y;
                        if (e1n < 1e-24f) { e1x = 1.f; e1y = 0.f; e1n = 1.f; }
                        const float ie = rsqrtf(e1n);
                        e1x *= ie; e1y *= ie;
                        const float e2x = -az * e1y, e2y = az * e1x, e2z = ax * e1y - ay * e1x;
                        ux = cp * ax + sp2 * (cphi * e1x + sphi * e2x);
                        uy = cp * ay + sp2 * (cphi * e1y + sphi * e2y);
                        uz = cp * az + sp2 * (sphi * e2z);
                    }
                    // (production variants) zenith angle and the table's texel loads ahead of a8-a10
                    constexpr bool EARLY_TAB = C8PH_TABLE_EARLY && SPEC != 0 && EMIT == C8PH_EMIT_CHERENKOV && TRACE == C8PH_TRACE_TABLE;
                    TabRaw traw;
                    float cz_e = 0.f;
                    if (EARLY_TAB) {
                        if (SPH) {
                            const float ur = cth * fmaf(q, fmaf(cphi, sg.a1, sphi * sg.a2), sg.cA);
                            const float sr = s * sg.inv_rA;
                            cz_e = -(fmaf(-sr * sg.cA, ur, ur) + sr * cth);
                        } else cz_e = -uz;
                        cz_e = fminf(cz_e, 1.f);
                        traw = table_issue(a.tab, h_e, acos01(fmaxf(cz_e, 0.f)));
                    }
                    // a8: up-going / horizontal photons are discarded
                    if (uz >= kUpCut) { pkA += 1u; break; }
                    // a9: straight line to z = 0 (Eq. 3.3), anchor + offset form
                    // (segments without a valid anchor carry G = 0 and the offset is the whole position)
                    float ox, oy;
                    const float inv_uz = rcp_fast(uz);
                    const float Z = fmaf(s, sg.Pz, sg.Az);
                    const float D = -Z * inv_uz;
                    if (sg.anchor & 1) {
                        const float zq = -Z * q * rcp_fast(sg.Pz * pqz);
                        ox = zq * (wx * sg.Pz - sg.Px * wz);
                        oy = zq * (wy * sg.Pz - sg.Py * wz);
                    } else {
                        if (!(Z > 0.f)) { pkA += 1u; break; }           // emitted at or below the observation level (R7: t* > 0)
#if C8PH_LINE_BY_VALUE
                        const float2 o2 = line_general(sc, s, D, sg.Px, sg.Py, ux, uy);
                        ox = o2.x; oy = o2.y;
#else
                        line_general(sc, s, D, sg.Px, sg.Py, ux, uy, ox, oy);
#endif
                    }
                    const float xl = sg.Gx + ox, yl = sg.Gy + oy;
                    // a10: LV2/LV3 on the straight-line point, before the correction: keep iff
                    // inside the histogram extent + margin or within r/|u_z| + margin of a telescope
                    if (f_lv2) {
                        const unsigned conv = __activemask();            // lanes that reach the filter together
                        bool keep = xl >= hc.box_x0 && xl < hc.box_x1 && yl >= hc.box_y0 && yl < hc.box_y1;
                        if (!keep && f_tel) {
                            const bool brute = !f_grid || -uz < hc.grid_min_cos;
                            const float thr = fmaf(hc.r_max, -inv_uz, hc.lv2_margin);
                            const int cell = brute ? -2 : grid_cell(det.lv2, xl, yl);
                            // per cell: (smallest key, x, y, r of the telescope nearest to the cell): that one is tested
                            // in line; if it is out of reach and the smallest key <= thr the sorted list is walked
                            float4 ka = make_float4(CUDART_INF_F, 3.0e18f, 3.0e18f, 0.f);
                            if (cell >= 0) ka = __ldg(det.lv2.knear + cell);
                            {
                                const float dx = xl - ka.y, dy = yl - ka.z, reach = fmaf(ka.w, -inv_uz, hc.lv2_margin);
                                keep = dx * dx + dy * dy <= reach * reach;
                            }
                            if (!keep && (cell < -1 || ka.x <= thr))
                                keep = tel_near_search(det, cell, thr, xl, yl, -inv_uz, hc.lv2_margin);
                        }
                        __syncwarp(conv);                                // rejoin the lanes that searched a list
                        if (!keep) { pkA += 0x10000u; break; }
                    }
                    // local zenith angle of the photon at the emission point
                    float dd = 0.f, dt = 0.f, Xs = 0.f, ta = 0.f, cz;
                    float flat_perp = 0.f, flat_px = 0.f, flat_py = 0.f;      // R21: transverse displacement and its direction
                    if (EARLY_TAB) cz = cz_e;
                    else if (SPH) {
                        float ur;
                        if (EMIT == C8PH_EMIT_CHERENKOV) ur = cth * fmaf(q, fmaf(cphi, sg.a1, sphi * sg.a2), sg.cA);
                        else ur = ux * sc->rx + uy * sc->ry + uz * sc->rz;
                        const float sr = s * sg.inv_rA;
                        const float uP = (EMIT == C8PH_EMIT_CHERENKOV) ? cth : (ux * sg.Px + uy * sg.Py + uz * sg.Pz);
                        cz = -(fmaf(-sr * sg.cA, ur, ur) + sr * uP);
                    } else {
                        cz = -uz;
                    }
                    cz = fminf(cz, 1.f);
                    // a11: refraction
                    if (TRACE == C8PH_TRACE_STRAIGHT) {
                        dt = eta_e * D * kInvC;                          // homogeneous: t = t_e + n D / c
                    } else if (TRACE == C8PH_TRACE_TABLE) {
                        TabVal v;
                        if (f_cyl) {
                            // plane of curvature = vertical plane through the origin's vertical and the emission point
                            // (xl - D u): psi = azimuth of the flight against it
                            const float xe = fmaf(-D, ux, xl), ye = fmaf(-D, uy, yl);
                            const float hn2c = ux * ux + uy * uy, de2 = fmaf(xe, xe, ye * ye);
                            const float ihc = hn2c >= 1e-24f ? rsqrt_fast(hn2c) : 0.f;
                            const float ehx_ = ux * ihc, ehy_ = uy * ihc;
                            float epx = ehx_, epy = ehy_;
                            if (de2 > 1e-12f) { const float id = rsqrt_fast(de2); epx = xe * id; epy = ye * id; }
                            float cps = ehx_ * epx + ehy_ * epy, sps = epx * ehy_ - epy * ehx_;
                            if (ihc == 0.f) { cps = 1.f; sps = 0.f; }
                            float ptilde;
                            v = table_lookup_cyl(a.tab, h_e, acos01(fmaxf(cz, 0.f)), fminf(cps * cps, 1.f), ptilde);
                            flat_perp = ptilde * sps * cps;              // across the flight: along e_h turned by +90 degrees
                            flat_px = -ehy_; flat_py = ehx_;
                        } else
                        if (f_flat_tab) {
                            // R21: polar radius of the straight-line point and pointing angle of the direction of flight
                            const float hn2f = ux * ux + uy * uy, rho2 = fmaf(xl, xl, yl * yl);
                            const float ihf = hn2f >= 1e-18f ? rsqrt_fast(hn2f) : 0.f, irho = rho2 >= 1e-18f ? rsqrt_fast(rho2) : 0.f;
                            const float rx = xl * irho, ry = yl * irho;          // outward radial direction
                            const float cchi = (ux * rx + uy * ry) * ihf;
                            v = table_lookup_flat(a.tab, h_e, acos01(fmaxf(cz, 0.f)), rho2 * irho, cchi, flat_perp);
                            flat_px = fmaf(-cchi * ihf, ux, rx); flat_py = fmaf(-cchi * ihf, uy, ry);
                        } else
                            v = EARLY_TAB ? table_combine(traw) : table_lookup(a.tab, h_e, acos01(fmaxf(cz, 0.f)));
                        if (v.bad || !(cz > 0.f)) { pkB += 1u; break; }
                        dd = v.dd; dt = v.dt; Xs = v.X; ta = v.ta;
                    } else {
                        // layered Snell sum (Eq. 3.15 in its invariant form K = n sin(theta)),
                        // accumulated as the difference to the straight line
                        const float sinz = sqrtf(fmaxf(1.f - cz * cz, 0.f));
                        const float n_e = 1.f + eta_e;
                        const float K = n_e * sinz;
                        const float r_e = __frcp_rn(n_e * cz);
                        const float fe = fminf(fmaxf((h_e - atm.h0) * atm.inv_dh, 0.f), (float)(atm.n_nodes - 1));
                        const float fg = fminf(fmaxf(((float)atm.h_obs - atm.h0) * atm.inv_dh, 0.f), (float)(atm.n_nodes - 1));
                        const int ke = min((int)fe, atm.n_nodes - 2), kg = min((int)fg, atm.n_nodes - 2);
                        const float fre = fe - (float)ke, frg = fg - (float)kg;
                        float aX = 0.f, aT = 0.f, aS = 0.f, aA = 0.f;
                        bool ok = cz > 0.f;
                        // da = A(layer bottom) - A(layer top), A(h) = (H/L) exp(-h/H): the layer's vertical aerosol depth
                        auto layer = [&](auto aer, float eta_l, float thick, float dxv_l, float da) {
                            const float n_l = 1.f + eta_l;
                            const float ql = fmaf(n_l, n_l, -K * K);
                            ok = ok && (ql > 0.f);
                            const float r_l = rsqrt_fast(ql);
                            const float dq = (eta_e - eta_l) * (2.f + eta_e + eta_l);       // q_e - q_l
                            const float dr = dq * r_l * r_l * r_e * r_e * rcp_fast(r_l + r_e);  // r_l - r_e
                            aX = fmaf(thick * K, dr, aX);
                            aT = fmaf(thick, fmaf(n_l * n_l, dr, r_e * (fmaf(eta_l, eta_l, 2.f * eta_l) - eta_e)), aT);
                            aS = fmaf(dxv_l * n_l, r_l, aS);
                            if (decltype(aer)::value) aA = fmaf(da * n_l, r_l, aA);
                        };
                        auto walk = [&](auto aer) {
                            float Ae = 0.f, Ag = 0.f;                   // A at the emission height and at the observation level
                            if (decltype(aer)::value) {
                                Ae = atm.aer_HL * exp2_fast(-1.4426950408889634f * h_e * atm.aer_invH);
                                Ag = atm.aer_Ag;
                            }
                            auto A = [&](int k) { return decltype(aer)::value ? s_aexp[k] : 0.f; };
                            if (ke == kg) {
                                const float fm = 0.5f * (fre + frg);
                                layer(aer, fmaf(fm, s_eta[ke + 1] - s_eta[ke], s_eta[ke]), (fre - frg) * atm.dh, (fre - frg) * s_dxv[ke], Ag - Ae);
                            } else {
                                if (fre > 0.f)
                                    layer(aer, fmaf(0.5f * fre, s_eta[ke + 1] - s_eta[ke], s_eta[ke]), fre * atm.dh, fre * s_dxv[ke], A(ke) - Ae);
                                for (int k = ke - 1; k > kg; --k)             // n at the layer mid height
                                    layer(aer, 0.5f * (s_eta[k] + s_eta[k + 1]), atm.dh, s_dxv[k], A(k) - A(k + 1));
                                layer(aer, fmaf(0.5f * (1.f + frg), s_eta[kg + 1] - s_eta[kg], s_eta[kg]), (1.f - frg) * atm.dh, (1.f - frg) * s_dxv[kg], Ag - A(kg + 1));
                            }
                        };
                        const float re2 = r_e * r_e;
                        if (C8PH_LAYER_MOMENTS && !aer_staged && ke > kg && ok && atm.nu_span * re2 < kLayerSeriesMax) {
                            // The same sum in closed form.  With nu = n^2 - 1: n_l^2 - K^2 = (1 + x_l) / r_e^2,
                            // x_l = (nu_l - nu_e) r_e^2, so r_l = r_e (1 + x_l)^(-1/2) and every term of the three sums
                            // is a power series in x_l (|x_l| < 0.02 here: the p = 5 term is below 1e-9 of the first).
                            // sum thickness x_l^p follows from the binomial expansion of (nu_l - nu_e)^p and the layer
                            // moments mom[] (c8ph_init_atmosphere) up to the node below the emission cell, plus the
                            // partial layer of the emission cell itself.
                            const float eta_p = fmaf(0.5f * fre, s_eta[ke + 1] - s_eta[ke], s_eta[ke]);
                            const float nu_p = eta_p * (2.f + eta_p), th_p = fre * atm.dh, g_p = fre * s_dxv[ke] * (1.f + eta_p);
                            const float *mk = atm.mom + ke;
                            const int np = atm.n_pad;
                            const float nu_p2 = nu_p * nu_p;
                            const float M1 = fmaf(th_p, nu_p, __ldg(mk)), M2 = fmaf(th_p, nu_p2, __ldg(mk + np));
                            const float M3 = fmaf(th_p * nu_p, nu_p2, __ldg(mk + 2 * np)), M4 = fmaf(th_p * nu_p2, nu_p2, __ldg(mk + 3 * np));
                            const float G0 = __ldg(mk + 4 * np) + g_p, G1 = fmaf(g_p, nu_p, __ldg(mk + 5 * np)), G2 = fmaf(g_p, nu_p2, __ldg(mk + 6 * np));
                            const float G3 = fmaf(g_p * nu_p, nu_p2, __ldg(mk + 7 * np));
                            const float Hh = (fe - fg) * atm.dh;                     // sum of the layer thicknesses
                            const float d = -eta_e * (2.f + eta_e);                  // -nu_e
                            // S_p = sum thickness x_l^p
                            const float S1 = re2 * fmaf(d, Hh, M1);
                            const float S2 = re2 * re2 * fmaf(d, fmaf(d, Hh, 2.f * M1), M2);
                            const float S3 = re2 * re2 * re2 * fmaf(d, fmaf(d, fmaf(d, Hh, 3.f * M1), 3.f * M2), M3);
                            const float S4 = (re2 * re2) * (re2 * re2) * fmaf(d, fmaf(d, fmaf(d, fmaf(d, Hh, 4.f * M1), 6.f * M2), 4.f * M3), M4);
                            const float Am = fmaf(0.2734375f, S4, fmaf(-0.3125f, S3, fmaf(0.375f, S2, -0.5f * S1)));       // sum thickness ((1+x)^(-1/2) - 1)
                            const float Ap = fmaf(-0.0390625f, S4, fmaf(0.0625f, S3, fmaf(-0.125f, S2, 0.5f * S1)));      // sum thickness ((1+x)^(+1/2) - 1)
                            aX = K * r_e * Am;
                            // sum thickness (n_l^2 r_l - n_e r_e), n_l^2 r_l = (1+x)^(1/2) / r_e + K^2 r_e (1+x)^(-1/2)
                            aT = fmaf(Hh * r_e * n_e, eta_e, fmaf(Ap, n_e * cz, K * K * r_e * Am));
                            // sum dX_v n_l r_l
                            const float T1 = re2 * fmaf(d, G0, G1), T2 = re2 * re2 * fmaf(d, fmaf(d, G0, 2.f * G1), G2);
                            const float T3 = re2 * re2 * re2 * fmaf(d, fmaf(d, fmaf(d, G0, 3.f * G1), 3.f * G2), G3);
                            aS = r_e * fmaf(-0.3125f, T3, fmaf(0.375f, T2, fmaf(-0.5f, T1, G0)));
                        } else
                        if (aer_staged) walk(std::true_type{}); else walk(std::false_type{});
                        if (!ok) { pkB += 1u; break; }
                        dd = aX; dt = aT * kInvC; Xs = aS; ta = aA;
                    }
                    float wgt = hc.w;
                    if (f_trans != C8PH_TRANS_OFF) {
                        // a12: transmission, Rayleigh ~ lambda^-4 scaled by slant depth (+ aerosol)
                        float tau = 0.f;
                        if (f_ext) {
                            // tabulated extinction (Fig. 4.7a): vertical optical depth tau_v(lambda, h_e),
                            // bilinear, times the air-mass factor X_slant / (X_v(h_obs) - X_v(h_e)); in units of ln 2
                            const float fh = fminf(fmaxf((h_e - atm.h0) * atm.inv_dh, 0.f), atm.f_max);
                            const int kh = min((int)fh, atm.n_nodes - 2);
                            const float wh = fh - (float)kh;
                            const float gl = fminf(fmaxf((rcp_fast(lam_inv) - atm.ext_l0) * atm.ext_inv_dl, 0.f), (float)(atm.n_ext - 1));
                            const int kl = min((int)gl, max(atm.n_ext - 2, 0));
                            const float wl = gl - (float)kl;
                            const float *r0 = atm.ext + (size_t)kl * atm.n_nodes + kh;
                            const float *r1 = atm.ext + (size_t)min(kl + 1, atm.n_ext - 1) * atm.n_nodes + kh;
                            const float t0 = fmaf(wh, __ldg(r0 + 1) - __ldg(r0), __ldg(r0)), t1 = fmaf(wh, __ldg(r1 + 1) - __ldg(r1), __ldg(r1));
                            const float xe = fmaf(wh, __ldg(atm.xv + kh + 1) - __ldg(atm.xv + kh), __ldg(atm.xv + kh));
                            const float dxv = atm.xv_g - xe;
                            tau = dxv > 0.f ? 1.4426950408889634f * fmaf(wl, t1 - t0, t0) * Xs * rcp_fast(dxv) : 0.f;
                        } else
                        if (f_ray) {
                            float qq = hc.ray_lambda * lam_inv;
                            qq *= qq; qq *= qq;
                            tau = Xs * qq * hc.ray_k;                        // optical depth in units of ln 2
                        }
                        if (f_aer && !f_ext) tau = fmaf(1.4426950408889634f * ta, __powf(atm.aer_lambda * lam_inv, atm.aer_angstrom), tau);
                        float T = exp2_fast(-tau);
                        if (f_eff) {
                            // detector efficiency eps(lambda): linear on a uniform grid, ends held
                            const float fl = fminf(fmaxf((rcp_fast(lam_inv) - run.eff_l0) * run.eff_inv_dl, 0.f), (float)(run.n_eff - 1));
                            const int ie = min((int)fl, max(run.n_eff - 2, 0));
                            const float e0 = __ldg(run.eff + ie), e1 = __ldg(run.eff + min(ie + 1, run.n_eff - 1));
                            T *= fmaf(fl - (float)ie, e1 - e0, e0);
                        }
                        if (f_trans == C8PH_TRANS_ROULETTE) {
                            if (!(u01(rn.w) < T)) { pkB += 0x10000u; break; }
                        } else wgt = hc.w * T;
                    }
                    // landed: corrected position (dd along the horizontal direction of flight)
                    const float hn2 = ux * ux + uy * uy;
                    const float ih = hn2 >= 1e-18f ? rsqrt_fast(hn2) : 0.f;            // vertical photon: no correction
                    const float ehx = ux * ih, ehy = uy * ih;
                    float cx = fmaf(dd, ehx, ox), cy = fmaf(dd, ehy, oy);               // offset from the anchor
                    if (f_flat_tab || f_cyl) { cx = fmaf(flat_perp, flat_px, cx); cy = fmaf(flat_perp, flat_py, cy); }
                    if (f_flat) {
                        // R19, flat observation plane (thesis Fig. 4.10): dd, dt and the rotation hold where
                        // the ray meets the observation sphere; the plane z = 0 lies h_I above it at the line point.
                        // Line on to the sphere (s1), arc dd along the flight direction on the sphere, back along
                        // the arrival direction to z = 0; all in cancellation-free perturbation form about I.
                        const float Rg = (float)atm.Rg;
                        const float rho2 = fmaf(xl, xl, yl * yl);
                        const float hI = rho2 * rcp_fast(Rg + sqrt_fast(fmaf(Rg, Rg, rho2)));
                        const float m = hI * fmaf(2.f, Rg, hI);                         // |I - C|^2 - Rg^2
                        const float uw = fmaf(ux, xl, fmaf(uy, yl, uz * Rg));           // u . (I - C)
                        const float disc = fmaf(uw, uw, -m);
                        if (!(disc > 0.f) || !(uw < 0.f)) { pkB += 1u; break; }         // the line misses the sphere
                        const float s1 = m * rcp_fast(sqrt_fast(disc) - uw);
                        const float rwx = fmaf(s1, ux, xl) * run.inv_Rg, rwy = fmaf(s1, uy, yl) * run.inv_Rg;
                        const float rwz = fmaf(s1 * uz, run.inv_Rg, 1.f);               // unit radial at the sphere point
                        const float cw = fmaf(ux, rwx, fmaf(uy, rwy, uz * rwz));
                        const float st2 = fmaf(-cw, cw, 1.f);
                        const float ie = st2 >= 1e-18f ? rsqrt_fast(st2) : 0.f;
                        const float etx = fmaf(-cw, rwx, ux) * ie, ety = fmaf(-cw, rwy, uy) * ie, etz = fmaf(-cw, rwz, uz) * ie;
                        float uax, uay, uaz;
                        arrival_dir(sc, ux, uy, uz, cz, eta_e, h_e, dd, uax, uay, uaz);
                        const float sb = fmaf(dd, etz, s1 * uz) * rcp_fast(uaz);
                        cx = ox + fmaf(dd, etx, fmaf(s1, ux, -sb * uax));
                        cy = oy + fmaf(dd, ety, fmaf(s1, uy, -sb * uay));
                        dt = fmaf(fmaf(-(1.f + atm.eta_g), sb, s1), kInvC, dt);
                    }
                    const float xg = sg.Gx + cx, yg = sg.Gy + cy;
                    // a14 pre-test: the photon can hit a sphere of its grid cell only if the cell's
                    // smallest key <= 1/|u_z| (inflated for the refraction rotation of the direction); the
                    // load is issued before the binning arithmetic so its latency overlaps
                    int cell = -1;
                    float kmin = 255.f;                               // quantised smallest key of the cell (255: empty)
                    if (f_tel) {
                        const bool brute = f_hit_brute || !f_grid || -uz < hc.grid_min_cos;
                        if (f_grid) {
#if C8PH_HIT_RING
                            // the grid has a border ring of empty cells (c8ph_set_detector): a point outside it is
                            // clamped into the ring (negative coordinates wrap to large unsigned values) and finds "empty"
                            const unsigned gx = min((unsigned)__float2int_rd((xg - hc.hit_x0) * hc.hit_inv_cs), (unsigned)(hc.hit_nx - 1));
                            const unsigned gy = min((unsigned)__float2int_rd((yg - hc.hit_y0) * hc.hit_inv_cs), (unsigned)(hc.hit_ny - 1));
                            cell = (int)(gy * (unsigned)hc.hit_nx + gx);
                            kmin = (float)__ldg(hc.hit_kq + cell);
#else
                            const int gx = __float2int_rd((xg - hc.hit_x0) * hc.hit_inv_cs), gy = __float2int_rd((yg - hc.hit_y0) * hc.hit_inv_cs);
                            cell = ((unsigned)gx < (unsigned)hc.hit_nx && (unsigned)gy < (unsigned)hc.hit_ny) ? gy * hc.hit_nx + gx : -1;
                            kmin = (float)__ldg(hc.hit_kq + max(cell, 0));  // cell -1 (outside): never a candidate
                            if (cell < 0) kmin = 255.f;
#endif
                        }
                        if (brute) cell = -2;
                    }
                    // a15: ground grid
                    if (has_grid_geom) {
                        const float4 fb = *reinterpret_cast<const float4 *>(sc);         // fbx, fby, ibx, iby
                        const int ix = __float_as_int(fb.z) + __float2int_rd(fmaf(cx, hc.hist_inv_cell, fb.x));
                        const int iy = __float_as_int(fb.w) + __float2int_rd(fmaf(cy, hc.hist_inv_cell, fb.y));
                        if ((unsigned)ix < (unsigned)hc.hist_nx && (unsigned)iy < (unsigned)hc.hist_ny) {
                            pkC += 1u;
#if C8PH_HIST_MATCH
                            if (SPEC) {                                  // roulette mode: every bunch has weight w
                                const int bin = iy * hc.hist_nx + ix;
                                const unsigned peers = __match_any_sync(__activemask(), bin);
                                if (lane == __ffs(peers) - 1) atomicAdd(hc.hist + bin, wgt * (float)__popc(peers));
                            } else
#endif
                            if (has_hist) atomicAdd(hc.hist + (iy * hc.hist_nx + ix), wgt);
                        }
                    }
                    const bool cand = cell < -1 || (kmin <= -inv_uz * hc.hit_infl_q && kmin < 255.f);
                    if (!cand) {
                        if (f_write != C8PH_WRITE_ALL) break;
                        cell = -1;
                    }
                    // queue the photon for finish() (a13/a14/a16)
#if C8PH_QUEUE_CONVERGED
                    // the entry leaves the body in registers and is stored after the reconvergence point
                    qe0 = f_opt ? make_float4(cx, cy, ux, uy) : make_float4(xg, yg, ux, uy);
                    qe1 = make_float4(uz, s, q * wz, dt);
                    qe2 = make_float4(lam_inv, wgt, eta_e, h_e);
                    qe3 = make_float4(dd, cz, __int_as_float(cell), __uint_as_float(js));
                    qpush = true;
#else
                    // slots are handed out per group of lanes
                    // that arrive here together (one shared-memory atomic per group), four 16 B stores
#if C8PH_HIT_PREFETCH
                    if (f_tel && cell >= 0) {
                        asm volatile("prefetch.global.L1 [%0];" ::"l"(det.hit.first + cell));
                        asm volatile("prefetch.global.L1 [%0];" ::"l"(det.hit.first_kn + cell));
                    }
#endif
#if C8PH_QUEUE_LANE_ATOMS
                    int qb;                                              // inline asm: no compiler-generated warp aggregation
                    asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(qb) : "r"(qn_addr) : "memory");
#if C8PH_QUEUE_VOTE
                    qfull = qb >= 31;
#endif
                    if (QC) {
                        const uint32_t qi = (uint32_t)(q_head + qb) & (uint32_t)(kQueue - 1);
                        if (QG) {
                            // the warp's block from the count's address: (qn_addr - &s_qn_static[0]) / 4 = warp
                            const uint32_t woff = (qn_addr - smem_u32(&s_qn_static[0])) * (kQBlock / 4u);
                            unsigned char *g4 = q_cta + (woff + qi * 16u), *g2 = q_cta + (woff + qi * 8u);
                            const float e0x = f_opt ? cx : xg, e0y = f_opt ? cy : yg;
                            asm volatile("st.global.cg.v4.f32 [%0+16], {%1, %2, %3, %4};" ::"l"(g4), "f"(e0x), "f"(e0y), "f"(ux), "f"(uy) : "memory");
                            asm volatile("st.global.cg.v4.f32 [%0+1040], {%1, %2, %3, %4};" ::"l"(g4), "f"(uz), "f"(s), "f"(q * wz), "f"(dt) : "memory");
                            asm volatile("st.global.cg.v4.f32 [%0+2064], {%1, %2, %3, %4};" ::"l"(g4), "f"(lam_inv), "f"(eta_e), "f"(dd), "f"(cz) : "memory");
                            asm volatile("st.global.cg.v2.b32 [%0+3088], {%1, %2};" ::"l"(g2), "r"(cell), "r"(js) : "memory");
                            break;
                        }
                        const uint32_t a4 = qn_addr + qi * 16u, a2 = qn_addr + qi * 8u;     // + 16: past the fill count
                        const float e0x = f_opt ? cx : xg, e0y = f_opt ? cy : yg;
                        asm volatile("st.shared.v4.f32 [%0+16], {%1, %2, %3, %4};" ::"r"(a4), "f"(e0x), "f"(e0y), "f"(ux), "f"(uy) : "memory");
                        asm volatile("st.shared.v4.f32 [%0+1040], {%1, %2, %3, %4};" ::"r"(a4), "f"(uz), "f"(s), "f"(q * wz), "f"(dt) : "memory");
                        asm volatile("st.shared.v4.f32 [%0+2064], {%1, %2, %3, %4};" ::"r"(a4), "f"(lam_inv), "f"(eta_e), "f"(dd), "f"(cz) : "memory");
                        asm volatile("st.shared.v2.b32 [%0+3088], {%1, %2};" ::"r"(a2), "r"(cell), "r"(js) : "memory");
                        break;
                    }
                    float4 *e = s_q + ((q_head + qb) & (kQueue - 1)) * 4;
#else
                    const unsigned am = __activemask();
                    const int leader = __ffs(am) - 1;
                    int qb = 0;
                    if (lane == leader)                                  // plain ATOMS: the group is already aggregated
                        asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(qb) : "r"(qn_addr), "r"(__popc(am)) : "memory");
                    qb = __shfl_sync(am, qb, leader);
                    float4 *e = s_q + ((q_head + qb + __popc(am & ((1u << lane) - 1u))) & (kQueue - 1)) * 4;
#endif
                    e[0] = f_opt ? make_float4(cx, cy, ux, uy) : make_float4(xg, yg, ux, uy);
                    e[1] = make_float4(uz, s, q * wz, dt);
                    e[2] = make_float4(lam_inv, wgt, eta_e, h_e);
                    e[3] = make_float4(dd, cz, __int_as_float(cell), __uint_as_float(js));
#endif
                } while (false);
#if C8PH_QUEUE_CONVERGED
                // all lanes are back together: one ballot ranks the candidates, four 16 B stores each, the fill count
                // stays in a (warp-uniform) register
                {
                    const unsigned pm = __ballot_sync(FULL, qpush);
                    if (pm) {
                        if (qpush) {
                            float4 *e = s_q + ((q_head + q_n + __popc(pm & ((1u << lane) - 1u))) & (kQueue - 1)) * 4;
                            e[0] = qe0; e[1] = qe1; e[2] = qe2; e[3] = qe3;
                        }
                        q_n += __popc(pm);
                        // a14/a16: once 32 candidates wait, a full warp takes them through finish()
                        if (q_n >= 32) drain(false);
                    }
                }
#else
                // a14/a16: once 32 candidates wait, a full warp takes them through finish()
#if C8PH_QUEUE_VOTE && C8PH_QUEUE_LANE_ATOMS
                if (__any_sync(FULL, qfull)) drain(false);
#else
                drain(false);
#endif
#endif
            }
        }
        drain(true);                                                  // slots are rewritten by the next group
    }
    flush_counts();
    __syncthreads();

    // ---- counters: one global atomic per CTA and non-zero counter
    if (run.out.counters && threadIdx.x == 0) {
        const unsigned long long *c = s_cnt;
        auto add = [&](int idx, unsigned long long v) { if (v) atomicAdd(&cntp[idx], v); };
        if (blockIdx.x == 0) add(C8PH_CNT_SEGMENTS, (unsigned long long)run.n_seg);
        add(C8PH_CNT_SEG_BELOW_THRESHOLD, c[WC_BELOW]);
        add(C8PH_CNT_SEG_LV1, c[WC_LV1]);
        add(C8PH_CNT_SEG_EMITTING, c[WC_EMITTING]);
        add(C8PH_CNT_CLIPPED, c[WC_CLIPPED]);
        add(C8PH_CNT_NONFINITE, c[WC_NONFINITE]);
        add(C8PH_CNT_EMITTED, c[WC_EMITTED]);
        add(C8PH_CNT_UPGOING, c[WC_UP]);
        add(C8PH_CNT_LV2, c[WC_LV2]);
        add(C8PH_CNT_TABLE_RANGE, c[WC_TR]);
        add(C8PH_CNT_ROULETTE, c[WC_ROUL]);
        add(C8PH_CNT_IN_GRID, c[WC_GRID]);
        add(C8PH_CNT_TEL_HIT, c[WC_TEL]);
        add(C8PH_CNT_CAM_HIT, c[WC_CAM]);
        add(C8PH_CNT_OVERFLOW, c[WC_OVERFLOW]);
        add(C8PH_CNT_LANDED, c[WC_EMITTED] - c[WC_UP] - c[WC_LV2] - c[WC_TR] - c[WC_ROUL]);
    }
}

// ================================================================================================
// Correction table: one thread per node, exact layered ray in fp64 by the Snell (planar) or
// Bouguer (spherical) invariant, layer by layer on the n(h) grid (layers = table cells split in
// `substeps`, n at the layer mid height), minus the straight line to the same sphere / plane.
struct NodeRay { bool ground; double psi, S, cT, X, tau; };

// exact layered ray from (h_e, zenith th) down to the observation level: central angle (spherical) or horizontal
// displacement (planar), geometric path, optical path, slant depth, aerosol optical depth
__device__ NodeRay trace_node(const DevAtm &atm, double h_e, double th, int substeps)
{
    NodeRay o;
    o.ground = true; o.psi = o.S = o.cT = o.X = o.tau = 0.0;
    const bool sph = atm.model >= C8PH_ATM_SPHERICAL;     // the cylindrical model's 2-D table is the spherical one
    const double h_g = atm.h_obs;
    const double sz = sin(th);
    const double n_e = 1.0 + eta_lookup_d(atm, h_e);
    const double K = sph ? n_e * (atm.R + h_e) * sz : n_e * sz;     // Bouguer / Snell invariant
    const double step = atm.model == C8PH_ATM_HOMOGENEOUS ? 1.0e30 : (double)atm.dh / substeps;
    double h_cur = h_e;
    auto xv_at = [&](double h) {
        double f = (h - (double)atm.h0) / (double)atm.dh;
        f = fmin(fmax(f, 0.0), (double)(atm.n_nodes - 1));
        const int k = min((int)f, atm.n_nodes - 2);
        const double fr = f - k;
        return (1.0 - fr) * (double)__ldg(atm.xv + k) + fr * (double)__ldg(atm.xv + k + 1);
    };
    double xv_cur = xv_at(h_cur);
    double ea_cur = atm.aer_L > 0.f ? exp(-h_cur / (double)atm.aer_H) : 0.0;
    while (h_cur > h_g) {
        double h_next;
        if (atm.model == C8PH_ATM_HOMOGENEOUS) h_next = h_g;
        else {
            const double g = floor((h_cur - (double)atm.h0) / step);
            h_next = (double)atm.h0 + g * step;
            if (!(h_next < h_cur - 1e-9 * step)) h_next = (double)atm.h0 + (g - 1.0) * step;
            if (h_next < h_g) h_next = h_g;
        }
        const double n_l = 1.0 + eta_lookup_d(atm, 0.5 * (h_cur + h_next));
        const double dhl = h_cur - h_next;
        double s;
        if (sph) {
            const double p = K / n_l;                                // impact parameter of the chord
            const double rt = atm.R + h_cur, rb = atm.R + h_next;
            if (!(rb > p)) { o.ground = false; break; }
            const double at = sqrt(rt * rt - p * p), ab = sqrt(rb * rb - p * p);
            s = dhl * (rt + rb) / (at + ab);                         // at - ab, cancellation-free
            const double x = p * s / (rt * rb);                      // sin of the central-angle step
            o.psi += x * (1.0 + x * x * (1.0 / 6.0 + x * x * (3.0 / 40.0)));
        } else {
            const double q2 = n_l * n_l - K * K;
            if (!(q2 > 0.0)) { o.ground = false; break; }
            const double iq = 1.0 / sqrt(q2);
            s = dhl * n_l * iq;
            o.psi += dhl * K * iq;                                   // horizontal displacement
        }
        o.S += s;
        o.cT += n_l * s;
        const double xv_next = xv_at(h_next);
        o.X += (xv_next - xv_cur) * (s / dhl);
        xv_cur = xv_next;
        if (atm.aer_L > 0.f) {
            const double ea_next = exp(-h_next / (double)atm.aer_H);
            o.tau += ((double)atm.aer_H / (double)atm.aer_L) * (ea_next - ea_cur) * (s / dhl);
            ea_cur = ea_next;
        }
        h_cur = h_next;
    }
    return o;
}

__global__ void __launch_bounds__(128) k_build_table(const __grid_constant__ TableBuildArgs a)
{
    const int node = blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= a.n_h * a.n_zen) return;
    const int ia = node / a.n_zen, ib = node % a.n_zen;
    const DevAtm &atm = a.atm;
    const double h_e = ia * a.h_max / (a.n_h - 1);
    const double th = ib * a.zen_max / (a.n_zen - 1);
    float out[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
    const bool sph = atm.model >= C8PH_ATM_SPHERICAL;     // the cylindrical model's 2-D table is the spherical one
    const double h_g = atm.h_obs;
    if (h_e > h_g) {
        const double sz = sin(th), cz = cos(th);
        const NodeRay r = trace_node(atm, h_e, th, a.substeps);
        if (r.ground) {
            double S_line, d_line, d_true;
            if (sph) {
                const double re = atm.R + h_e, rg = atm.Rg, p = re * sz;
                S_line = re * cz - sqrt(rg * rg - p * p);
                d_line = rg * (asin(p / rg) - th);
                d_true = rg * r.psi;
            } else {
                S_line = (h_e - h_g) / cz;
                d_line = (h_e - h_g) * sz / cz;
                d_true = r.psi;
            }
            out[0] = (float)(d_true - d_line);
            out[1] = (float)(r.S - S_line);
            out[2] = (float)((r.cT - S_line) / kC);
            out[3] = (float)r.X;
            out[4] = (float)r.tau;
        } else {
            const float nanv = __int_as_float(0x7FC00000);
            for (int k = 0; k < 5; ++k) out[k] = nanv;
        }
    }
    for (int k = 0; k < 5; ++k) a.full[(size_t)node * 5 + k] = out[k];
    a.hot[node] = make_float4(out[0], out[2], out[3], out[4]);
}

// ------------------------------------------------------------------------------------------------
// R21: the thesis' table "relative to a flat observation plane" (Fig. 4.10; spherical model): axes height,
// local zenith, rho = polar radius of the straight-line point on the plane z = 0, and the pointing angle chi of the
// horizontal direction of flight against the outward radial direction there, kept as even part E (texels as the 2-D
// table: dd, dt, X_slant, tau_aer), odd part O (dd, dt) and transverse displacement P in one more texel (O.dd, O.dt, P, 0):
// value = E + cos(chi) O along the direction of flight, P (r^ - cos(chi) e_h) across it.  One thread per (height,
// zenith) node traces the ray once and takes it from the observation sphere on to the plane for every rho.
struct Vec3d { double x, y, z; };
__device__ __forceinline__ double dot3(const Vec3d &a, const Vec3d &b) { return a.x * b.x + a.y * b.y + a.z * b.z; }

// from the sphere to the plane: line from A along u to the sphere r = Rg, arc dd along the direction of flight, back
// along the arrival direction ua (straight, ground index) to z = 0.  Returns false if the line misses the sphere.
__device__ bool sphere_to_plane(const DevAtm &atm, const Vec3d &A, const Vec3d &u, double h_e, double sz, double cz, double dd,
                                double dt_ns, const Vec3d &ua, double &x, double &y, double &t_rel)
{
    const double Rg = atm.Rg, re = atm.R + h_e, pp = re * sz;
    if (!(pp < Rg)) return false;
    const double S_line = re * cz - sqrt(Rg * Rg - pp * pp);
    Vec3d w = {A.x + S_line * u.x, A.y + S_line * u.y, A.z + S_line * u.z + Rg};
    const double wn = 1.0 / sqrt(dot3(w, w));
    w.x *= wn; w.y *= wn; w.z *= wn;
    const double cw = dot3(u, w);
    Vec3d et = {u.x - cw * w.x, u.y - cw * w.y, u.z - cw * w.z};
    const double en = sqrt(dot3(et, et));
    if (en < 1e-12) et.x = et.y = et.z = 0.0; else { et.x /= en; et.y /= en; et.z /= en; }
    const double ca = cos(dd / Rg), sa = sin(dd / Rg);
    const Vec3d Pr = {Rg * (ca * w.x + sa * et.x), Rg * (ca * w.y + sa * et.y), Rg * (ca * w.z + sa * et.z) - Rg};
    const double s_back = Pr.z / ua.z;
    x = Pr.x - s_back * ua.x;
    y = Pr.y - s_back * ua.y;
    t_rel = S_line / kC + dt_ns - (1.0 + (double)atm.eta_g) * s_back / kC;
    return true;
}

// the photon of Fig. 4.10 with its arrival direction: emission point A, direction u, local vertical rv
__device__ bool flat_photon(const DevAtm &atm, const Vec3d &A, const Vec3d &u, const Vec3d &rv, double h_e, double th, double dd,
                            double dt_ns, double &x, double &y, double &t_rel)
{
    const double sz = sin(th), cz = cos(th);
    // rotation of the direction in the ray plane from the Bouguer invariant (R9), n at the observation level = 1 + eta_g
    const double re = atm.R + h_e, Rg = atm.Rg, n_ray = 1.0 + eta_lookup_d(atm, h_e), n_g = 1.0 + (double)atm.eta_g;
    const double psi_line = asin(re * sz / Rg) - th;
    const double delta = asin(n_ray * re * sz / (n_g * Rg)) - (psi_line + dd / Rg) - th;
    Vec3d ua = u;
    if (sz > 1e-9 && delta != 0.0) {
        const double cd = cos(delta), sd = sin(delta);
        ua.x = cd * u.x + sd * (cz * u.x + rv.x) / sz;
        ua.y = cd * u.y + sd * (cz * u.y + rv.y) / sz;
        ua.z = cd * u.z + sd * (cz * u.z + rv.z) / sz;
    }
    return sphere_to_plane(atm, A, u, h_e, sz, cz, dd, dt_ns, ua, x, y, t_rel);
}

__global__ void __launch_bounds__(128) k_build_table_flat(const __grid_constant__ TableBuildArgs a)
{
    const int node = blockIdx.x * blockDim.x + threadIdx.x;
    if (node >= a.n_h * a.n_zen) return;
    const int ia = node / a.n_zen, ib = node % a.n_zen;
    const DevAtm &atm = a.atm;
    const double h_e = ia * a.h_max / (a.n_h - 1);
    const double th = ib * a.zen_max / (a.n_zen - 1);
    const size_t plane = (size_t)a.n_h * a.n_zen;
    const float nanv = __int_as_float(0x7FC00000);
    const bool zero = !(h_e > atm.h_obs);
    NodeRay r;
    r.ground = false;
    double dd = 0.0, dt_sph = 0.0, S_line_sph = 0.0;
    const double sz = sin(th), cz = cos(th), Rg = atm.Rg, re = atm.R + h_e;
    if (!zero) {
        r = trace_node(atm, h_e, th, a.substeps);
        if (r.ground) {
            const double p = re * sz;
            S_line_sph = re * cz - sqrt(Rg * Rg - p * p);
            dd = Rg * r.psi - Rg * (asin(p / Rg) - th);
            dt_sph = (r.cT - S_line_sph) / kC;
        }
    }
    for (int c = 0; c < a.n_rho; ++c) {
        float4 E = make_float4(0.f, 0.f, 0.f, 0.f), O = E;
        if (!zero) {
            bool ok = r.ground;
            const double rho = a.rho_max * c / (a.n_rho - 1);
            double T[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, P = 0.0;
            for (int sgn = 0; sgn < 2 && ok; ++sgn) {
                // radial flight: emission point (re sin(beta), 0, re cos(beta) - Rg), direction (sin(th - beta), 0, -cos(th - beta));
                // its straight line meets z = 0 at x(beta) = E_x + E_z tan(th - beta) = +-rho (bisection)
                const double xt = sgn ? -rho : rho;
                double lo = -0.2, hi = 0.2, beta = 0.0;
                for (int it = 0; it < 64; ++it) {
                    beta = 0.5 * (lo + hi);
                    if (re * sin(beta) + (re * cos(beta) - Rg) * tan(th - beta) < xt) lo = beta; else hi = beta;
                }
                const Vec3d A = {re * sin(beta), 0.0, re * cos(beta) - Rg};
                ok = A.z > 0.0 && cos(th - beta) > 1e-3 && fabs(A.x + A.z * tan(th - beta) - xt) <= 1e-6 * (1.0 + fabs(xt));
                if (!ok) break;
                const Vec3d u = {sin(th - beta), 0.0, -cos(th - beta)}, rv = {sin(beta), 0.0, cos(beta)};
                double x, y, t_rel;
                ok = flat_photon(atm, A, u, rv, h_e, th, dd, dt_sph, x, y, t_rel);
                const double D = A.z / cos(th - beta);
                T[sgn][0] = x - xt;
                T[sgn][1] = t_rel - D / kC;
            }
            if (ok) {
                // tangential flight: straight-line point (rho, 0, 0), flying along +y; emission point in closed form
                const double c2 = (re * re * cz * cz + rho * rho + Rg * Rg - re * re) / (Rg * Rg);
                ok = c2 > 1e-6 && c2 <= 1.0;
                if (ok) {
                    const double cg = sqrt(c2), sg = sqrt(1.0 - c2), sd = -Rg * cg + re * cz;
                    ok = sd > 0.0;
                    const Vec3d A = {rho, -sd * sg, sd * cg}, u = {0.0, sg, -cg};
                    const Vec3d rv = {A.x / re, A.y / re, (A.z + Rg) / re};
                    double x, y, t_rel;
                    ok = ok && flat_photon(atm, A, u, rv, h_e, th, dd, dt_sph, x, y, t_rel);
                    P = x - rho;
                }
            }
            if (ok) {
                E = make_float4((float)(0.5 * (T[0][0] + T[1][0])), (float)(0.5 * (T[0][1] + T[1][1])), (float)r.X, (float)r.tau);
                O = make_float4((float)(0.5 * (T[0][0] - T[1][0])), (float)(0.5 * (T[0][1] - T[1][1])), (float)P, 0.f);
            } else {
                E = O = make_float4(nanv, nanv, nanv, nanv);
            }
        }
        a.flatE[(size_t)c * plane + node] = E;
        a.flatO[(size_t)c * plane + node] = O;
    }
}

// ------------------------------------------------------------------------------------------------
// R24, cylindrical model (thesis sec. 3.3.3): coaxial cylinders about a horizontal axis through the Earth's centre.  The
// gradient has no component along the axis, so kappa = n u_axis is conserved and the motion in the plane of curvature is
// Bouguer's with the effective index n_eff = sqrt(n^2 - kappa^2): the layer loop of trace_node with n_eff in the
// geometry, the real path s n / n_eff per in-plane chord s, and the advance along the axis kappa s / n_eff.
// One thread per (height, zenith, c) node, psi = acos(sqrt(c)) kept 1e-3 rad inside the ends.
__global__ void __launch_bounds__(128) k_build_table_cyl(const __grid_constant__ TableBuildArgs a)
{
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    const int plane = a.n_h * a.n_zen;
    if (idx >= plane * a.n_c) return;
    const int k = idx / plane, node = idx % plane;
    const int ia = node / a.n_zen, ib = node % a.n_zen;
    const DevAtm &atm = a.atm;
    const double h_e = ia * a.h_max / (a.n_h - 1);
    const double th = ib * a.zen_max / (a.n_zen - 1);
    const float nanv = __int_as_float(0x7FC00000);
    float4 out = make_float4(0.f, 0.f, 0.f, 0.f);
    if (h_e > atm.h_obs) {
        const double c = (double)k / (a.n_c - 1);
        double psi = acos(sqrt(c));
        psi = fmin(fmax(psi, 1e-3), 0.5 * 3.14159265358979323846 - 1e-3);
        const double sz = sin(th), cz = cos(th), cps = cos(psi), sps = sin(psi);
        const double ux = sz * cps, uy = sz * sps, up = sqrt(ux * ux + cz * cz);
        const double sin_par = ux / up, cos_par = cz / up;             // zenith angle of the in-plane motion
        const double n_e = 1.0 + eta_lookup_d(atm, h_e);
        const double kappa = n_e * uy;
        const double K = n_e * up * (atm.R + h_e) * sin_par;           // n_eff r sin(theta_par)
        const double h_g = atm.h_obs, step = (double)atm.dh / a.substeps;
        double h_cur = h_e, psi_c = 0.0, S = 0.0, cT = 0.0, X = 0.0, yax = 0.0;
        bool ground = true;
        auto xv_at = [&](double h) {
            double f = (h - (double)atm.h0) / (double)atm.dh;
            f = fmin(fmax(f, 0.0), (double)(atm.n_nodes - 1));
            const int kk = min((int)f, atm.n_nodes - 2);
            const double fr = f - kk;
            return (1.0 - fr) * (double)__ldg(atm.xv + kk) + fr * (double)__ldg(atm.xv + kk + 1);
        };
        double xv_cur = xv_at(h_cur);
        while (h_cur > h_g) {
            const double g = floor((h_cur - (double)atm.h0) / step);
            double h_next = (double)atm.h0 + g * step;
            if (!(h_next < h_cur - 1e-9 * step)) h_next = (double)atm.h0 + (g - 1.0) * step;
            if (h_next < h_g) h_next = h_g;
            const double n_l = 1.0 + eta_lookup_d(atm, 0.5 * (h_cur + h_next));
            const double ne2 = n_l * n_l - kappa * kappa;
            if (!(ne2 > 0.0)) { ground = false; break; }
            const double n_eff = sqrt(ne2), p = K / n_eff;
            const double rt = atm.R + h_cur, rb = atm.R + h_next, dhl = h_cur - h_next;
            if (!(rb > fabs(p))) { ground = false; break; }
            const double at = sqrt(rt * rt - p * p), ab = sqrt(rb * rb - p * p);
            const double s_par = dhl * (rt + rb) / (at + ab);
            const double x = p * s_par / (rt * rb);
            psi_c += x * (1.0 + x * x * (1.0 / 6.0 + x * x * (3.0 / 40.0)));
            const double s = s_par * n_l / n_eff;
            yax += kappa / n_eff * s_par;
            S += s; cT += n_l * s;
            const double xv_next = xv_at(h_next);
            X += (xv_next - xv_cur) * (s / dhl);
            xv_cur = xv_next;
            h_cur = h_next;
        }
        const double Rg = atm.Rg, re = atm.R + h_e, pp = re * sin_par;
        if (ground && fabs(pp) < Rg) {
            const double chord = re * cos_par - sqrt(Rg * Rg - pp * pp), S_line = chord / up;
            const double psi_line = asin(pp / Rg) - atan2(sin_par, cos_par);
            const double dxp = Rg * (psi_c - psi_line), dyp = yax - uy * S_line;
            out = make_float4((float)(dxp * cps + dyp * sps), (float)((cT - S_line) / kC), (float)X,
                              (float)((-dxp * sps + dyp * cps) / (sps * cps)));
        } else {
            out = make_float4(nanv, nanv, nanv, nanv);
        }
    }
    a.cyl[idx] = out;
}

// dynamic shared memory of a variant with `threads` threads: [staged n(h) tables] + one candidate queue per warp
size_t smem_for(const KArgs &a, int threads, int q_words)
{
    size_t tables = a.run.trace == C8PH_TRACE_NUMERIC ? (size_t)a.atm.n_pad * 4u * (a.atm.aer_L > 0.f ? 3u : 2u) : 0u;
    if (C8PH_ETA_STAGED && a.run.trace == C8PH_TRACE_TABLE) tables = (size_t)a.atm.n_pad * 4u;
    if (C8PH_QUEUE_GLOBAL && q_words == Q_WORDS_COMPACT) return tables;
    return tables + (size_t)(threads / 32) * ((size_t)kQueue * q_words * sizeof(float) + (q_words == Q_WORDS_COMPACT ? 16u : 0u));
}

template <int EMIT, int TRACE, bool SPH, int SPEC>
cudaError_t launch_one(const KArgs &a, int n_sm, cudaStream_t st)
{
    auto kern = k_emit_propagate<EMIT, TRACE, SPH, SPEC>;
    const size_t smem = smem_for(a, kernel_threads(EMIT, TRACE, SPEC), queue_words(SPEC));
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    {
        static const char *cv = getenv("C8PH_CARVEOUT");               // experiment: shared-memory carve-out in percent
        if (cv) cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, atoi(cv));
    }
    int per_sm = 0;
    constexpr int kThreads = kernel_threads(EMIT, TRACE, SPEC), kWarps = kThreads / 32;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kThreads, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    if (per_sm * kWarps > kMaxWarpsPerSM) per_sm = kMaxWarpsPerSM / kWarps;   // the segment-slot scratch is sized for this
    long long warps_needed = (a.run.n_seg + a.run.segs_per_grab - 1) / a.run.segs_per_grab;
    long long blocks = (warps_needed + kWarps - 1) / kWarps;
    const long long max_blocks = (long long)n_sm * per_sm;          // persistent: one resident wave
    if (blocks > max_blocks) blocks = max_blocks;
    if (blocks < 1) blocks = 1;
    kern<<<(unsigned)blocks, kThreads, smem, st>>>(a);
    return cudaGetLastError();
}

}  // namespace

size_t queue_ring_bytes(int n_sm)
{
    return C8PH_QUEUE_GLOBAL ? (size_t)n_sm * kMaxWarpsPerSM * (kQueue * Q_WORDS_COMPACT * 4 + 16) : 0;
}

size_t segment_slot_bytes(int n_sm)
{
    return (size_t)n_sm * kMaxWarpsPerSM * 32 * sizeof(SegSlot);
}

size_t emit_smem_bytes(const KArgs &a)               // upper bound over the variants of this (emit, trace): host-side validation
{
    return std::max(smem_for(a, kernel_threads(a.run.emit, a.run.trace, 0), queue_words(0)),
                    smem_for(a, kernel_threads(a.run.emit, a.run.trace, kSpecBase), queue_words(kSpecBase)));
}

// SPEC mask of the call: 0 unless it matches the switches the SPEC != 0 variants are compiled for,
// else kSpecBase | the optional features that are on
static int array_production_setting(const KArgs &a)
{
    const DevRun &r = a.run;
    const DevDet &d = a.det;
    const bool base = a.atm.model != C8PH_ATM_CYLINDRICAL &&          // the cylindrical model runs the generic variant
           r.emit == C8PH_EMIT_CHERENKOV && r.trace == C8PH_TRACE_TABLE && r.lv2 && r.trans == C8PH_TRANS_ROULETTE &&
           (a.atm.ray_inv_X > 0.f || a.atm.n_ext > 0) && !(a.atm.aer_L > 0.f) && !d.cam_enabled &&
           ((d.hist_nx > 0 && r.out.hist != nullptr) || d.hist_nx == 0) &&
           d.n_tel > 0 && d.use_grid && !r.hit_brute && r.write == C8PH_WRITE_TEL && r.out.photons != nullptr &&
           r.out.tel_counts != nullptr && !r.force_generic;
    if (!base) return 0;
    return kSpecBase | (d.hist_nx == 0 ? kSpecNoGrid : 0) | (r.flat_plane == 1 ? kSpecFlat : 0) | (r.flat_plane == 2 ? kSpecFlatTab : 0) | (a.atm.n_ext > 0 ? kSpecExt : 0) | (r.disp_b != 0.f ? kSpecDisp : 0) |
           (r.n_eff > 0 ? kSpecEff : 0) | (d.opt_enabled ? kSpecOpt : 0);
}

cudaError_t launch_emit_propagate(const KArgs &a, int n_sm, cudaStream_t st)
{
    const bool sph = a.atm.model >= C8PH_ATM_SPHERICAL;
    const int spec = array_production_setting(a);
    if (spec == kSpecBase)
        return sph ? launch_one<C8PH_EMIT_CHERENKOV, C8PH_TRACE_TABLE, true, kSpecBase>(a, n_sm, st)
                   : launch_one<C8PH_EMIT_CHERENKOV, C8PH_TRACE_TABLE, false, kSpecBase>(a, n_sm, st);
    // production setting + optional features (spherical model): the combinations that are compiled
#if C8PH_PROD_ONLY
#define C8_SPEC(M)
#else
#define C8_SPEC(M) \
    if (sph && spec == (kSpecBase | (M))) return launch_one<C8PH_EMIT_CHERENKOV, C8PH_TRACE_TABLE, true, kSpecBase | (M)>(a, n_sm, st);
#endif
    C8_SPEC(kSpecNoGrid)
    C8_SPEC(kSpecFlat)
    C8_SPEC(kSpecFlatTab)
    C8_SPEC(kSpecExt)
    C8_SPEC(kSpecDisp)
    C8_SPEC(kSpecEff)
    C8_SPEC(kSpecOpt)
    C8_SPEC(kSpecEff | kSpecOpt)
    C8_SPEC(kSpecExt | kSpecEff)
    C8_SPEC(kSpecExt | kSpecEff | kSpecOpt)
    C8_SPEC(kSpecDisp | kSpecEff | kSpecOpt)
    C8_SPEC(kSpecDisp | kSpecExt | kSpecEff | kSpecOpt)
    C8_SPEC(kSpecFlat | kSpecExt | kSpecEff | kSpecOpt)
    C8_SPEC(kSpecFlat | kSpecDisp | kSpecExt | kSpecEff | kSpecOpt)
#undef C8_SPEC
#define C8_CASE(E, T)                                                             \
    if (a.run.emit == E && a.run.trace == T)                                      \
        return sph ? launch_one<E, T, true, 0>(a, n_sm, st) : launch_one<E, T, false, 0>(a, n_sm, st);
    C8_CASE(C8PH_EMIT_CHERENKOV, C8PH_TRACE_STRAIGHT)
    C8_CASE(C8PH_EMIT_CHERENKOV, C8PH_TRACE_NUMERIC)
    C8_CASE(C8PH_EMIT_CHERENKOV, C8PH_TRACE_TABLE)
    C8_CASE(C8PH_EMIT_FLUORESCENCE, C8PH_TRACE_STRAIGHT)
    C8_CASE(C8PH_EMIT_FLUORESCENCE, C8PH_TRACE_TABLE)
#undef C8_CASE
    return cudaErrorInvalidValue;
}

cudaError_t launch_build_table(const TableBuildArgs &a, cudaStream_t st)
{
    const int n = a.n_h * a.n_zen;
    k_build_table<<<(n + 127) / 128, 128, 0, st>>>(a);
    if (a.n_rho >= 2 && a.flatE && a.flatO) k_build_table_flat<<<(n + 127) / 128, 128, 0, st>>>(a);
    if (a.n_c >= 2 && a.cyl) k_build_table_cyl<<<(n * a.n_c + 127) / 128, 128, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace c8ph
