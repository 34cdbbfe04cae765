// a3: exact-adjoint backprojector G = P^T y as a race-free gather (O2 in DESIGN.md).
//
// The paper rejects the transpose form because a ray-driven scatter races and replaces it
// by the voxel-driven eq. 2.  Here the transpose itself is evaluated voxel-driven: a thread owns a
// column of KC voxels (fixed major index i = slab, fixed minor index j, KC consecutive k) and
// gathers, for every angle, from the few rays that can touch it:
//   * in-plane: the rays u whose slab-i traversal touches minor row j.  Candidates come from
//     projecting the column's x-y square onto the detector; each is then tested with the
//     projector's own minor_split(), giving its lambda-interval [l0,l1] inside row j;
//   * axially: within the slab a ray (u,v) lies in at most two z rows, split at lambda = b(u,v).
//     The rays of column u that ENTER the slab in row k are a contiguous run of v, bounded by the
//     first ray at or above plane k and the first at or above plane k+1, so
//         sum_v [entry row = k] y(u,v) = C(u, vT(k+1)) - C(u, vT(k))
//     with C the prefix sums of y along v (built once per call by prefix_kernel, compensated so
//     that the difference carries fp32 accuracy).  That is the whole weight (l1 - l0) of every ray
//     that does not cross a z plane inside the slab (most of them).  A ray that does cross plane k
//     (its v lies between vT(k) and the same bound taken at the slab's exit plane) moves
//         max(0, l1 - max(l0, b))        (= its exit-row fraction among the projector's four)
//     from its entry z row to its exit z row, with b from the projector's own expression.
//     The cost per (column, ray u) is therefore O(KC), independent of how many detector rows fall
//     into one voxel row (4.8 at c3's 2.5 mm slices).
// The projections handed in are pre-multiplied by the slab chord length l(u,v).
// One launch per ray class; class 0 accumulates into a [k][x][y] array, class 1 into [k][y][x],
// so lanes (adjacent minor index) write contiguously; op_combine() adds the two.
#include <type_traits>

#include "cbct_internal.h"
#include "ray_common.cuh"

// 1/x to 1 ulp by one MUFU instruction; denormal x is flushed to zero (the result, +-inf, is saturated by the caller)
__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// base + row * pitch (bytes): 32-bit row and pitch (either sign), 64-bit base -> one IMAD.WIDE
__device__ __forceinline__ const char *row_ptr(const char *base, int row, int pitch) { return base + (long long)row * pitch; }
// hides how a value was computed from the optimiser, so that an address formed from it is not re-derived from its parts
// (ptxas would otherwise share the product row * pitch between a row and its mirror image and pay two 64-bit adds for each)
__device__ __forceinline__ int opaque(int x) { asm("" : "+r"(x)); return x; }
__device__ __forceinline__ const char *opaque(const char *p)
{
    long long x = reinterpret_cast<long long>(p);
    asm("" : "+l"(x));
    return reinterpret_cast<const char *>(x);
}

// a + b = s + two_sum_err(a, b, s) exactly, for s = fl(a + b) (Knuth's two-sum; no assumption on the magnitudes)
__device__ __forceinline__ float two_sum_err(float a, float b, float s)
{
    const float bb = __fsub_rn(s, a);
    return __fadd_rn(__fsub_rn(a, __fsub_rn(s, bb)), __fsub_rn(b, bb));
}

#ifndef CBCT_BP_FIXED
#define CBCT_BP_FIXED 0
#endif
#ifndef CBCT_BP_PACKED
#define CBCT_BP_PACKED 1
#endif
// Prefix sums along v in one of two forms.  kFixed = false: (sum, two-sum compensation) float pairs.  kFixed = true: 32-bit
// fixed point with wrap-around: every column (a, u) is scaled by a power of two s(a,u) such that any run of at most
// `run_max` detector rows sums to less than 2^30 in magnitude, rounded to integers and summed modulo 2^32, so the difference
// of two prefix values is the EXACT sum of the rounded run whatever the prefix has grown to; 1/s(a,u) sits in a float table
// behind the prefix values.  Half the bytes per lookup and one integer subtraction per run.
constexpr bool kFixed = CBCT_BP_FIXED != 0;
using PrefixT = std::conditional_t<kFixed, int, float2>;
__device__ __forceinline__ float run_sum(const float2 hi, const float2 lo) { return (hi.x - lo.x) + (hi.y - lo.y); }
__device__ __forceinline__ float run_sum(const int hi, const int lo) { return (float)(hi - lo); }
__device__ __forceinline__ void put_prefix(float2 *p, float s, float e, unsigned) { *p = make_float2(s, e); }
__device__ __forceinline__ void put_prefix(int *p, float, float, unsigned si) { *p = (int)si; }

// C[a][v][u] = sum_{v' < v} y[a][v'][u] for v = 0..nv as (sum, compensation) pairs: the rounding
// error of every addition is carried in the second float (two-sum), so C(v2) - C(v1) evaluated as
// (s2 - s1) + (c2 - c1) has the accuracy of summing the run directly.
// scale != 0: y = l(u,v) * in (and the scaled projections are also written to rs_out).
__global__ void __launch_bounds__(128) prefix_kernel(const DevGeom d, const float *__restrict__ in, const int scale,
                                                     float *__restrict__ rs_out, PrefixT *__restrict__ C, float *__restrict__ inv_s,
                                                     const float run_max)
{
    const int u = blockIdx.x * blockDim.x + threadIdx.x, a = blockIdx.y;
    if (u >= d.nu) return;
    RayXY r = load_ray(d, a, u);
    const float *p = in + (size_t)a * d.nv * d.nu + u;
    float *po = rs_out ? rs_out + (size_t)a * d.nv * d.nu + u : nullptr;
    PrefixT *c = C + (size_t)a * (d.nv + 1) * d.nu + u;
    constexpr int PF = 8;
    float sc = 1.f;                                        // kFixed: the column's power-of-two scale
    if constexpr (kFixed) {
        float m = 0.f;
        for (int v0 = 0; v0 < d.nv; v0 += PF) {
            float y[PF];
#pragma unroll
            for (int q = 0; q < PF; ++q) y[q] = (v0 + q < d.nv) ? __ldg(p + (size_t)(v0 + q) * d.nu) : 0.f;
#pragma unroll
            for (int q = 0; q < PF; ++q) {
                if (v0 + q >= d.nv) break;
                m = fmaxf(m, fabsf(scale ? y[q] * chord_scale(r, __ldg(d.dz_mm + v0 + q)) : y[q]));
            }
        }
        int e = 0;
        frexpf(m * run_max, &e);                           // m run_max = f 2^e, f in [0.5, 1): f 2^30 < 2^30
        sc = (m > 0.f && m < 3e38f) ? ldexpf(1.f, max(min(30 - e, 120), -120)) : 1.f;
        inv_s[(size_t)a * d.nu + u] = 1.f / sc;
    }
    float s = 0.f, e = 0.f;
    unsigned si = 0u;
    put_prefix(c, 0.f, 0.f, 0u);
    for (int v0 = 0; v0 < d.nv; v0 += PF) {
        float y[PF];
#pragma unroll
        for (int q = 0; q < PF; ++q) y[q] = (v0 + q < d.nv) ? __ldg(p + (size_t)(v0 + q) * d.nu) : 0.f;
#pragma unroll
        for (int q = 0; q < PF; ++q) {
            if (v0 + q >= d.nv) break;
            float yy = y[q];
            if (scale) {
                yy *= chord_scale(r, __ldg(d.dz_mm + v0 + q));
                if (po) po[(size_t)(v0 + q) * d.nu] = yy;
            }
            if constexpr (kFixed) {
                si += (unsigned)__float2int_rn(yy * sc);
            } else {
                const float t = s + yy;
                const float bp = t - s;
                e += (s - (t - bp)) + (yy - bp);
                s = t;
            }
            put_prefix(c + (size_t)(v0 + q + 1) * d.nu, s, e, si);
        }
    }
}


// The same prefix sums with the column cut into SEG segments of detector rows, one thread per (column, segment): a column
// scanned by one thread leaves the GPU at 160 CTAs of 128 threads (c2) waiting on its own loads.  Pass 1 sums every segment
// (compensated), the segment totals meet in shared memory, pass 2 rescans the segment (its rows now come from L1 / L2) on top
// of the two-float total of the segments before it.  C(v).x + C(v).y is the sum of the rows below v to ~2^-48 as before; only
// the rounding of the .x parts differs from the one-thread scan.
template <int SEG>
__global__ void __launch_bounds__(32 * SEG) prefix_seg_kernel(const DevGeom d, const float *__restrict__ in, const int scale,
                                                              float *__restrict__ rs_out, float2 *__restrict__ C)
{
    __shared__ float2 tot[SEG][32];
    const int lane = threadIdx.x, seg = threadIdx.y;
    const int u = blockIdx.x * 32 + lane, a = blockIdx.y;
    const bool in_range = u < d.nu;
    const int len = (d.nv + SEG - 1) / SEG, v_lo = min(seg * len, d.nv), v_hi = min(v_lo + len, d.nv);
    const int uc = min(u, d.nu - 1);
    const RayXY r = load_ray(d, a, uc);
    const float *p = in + (size_t)a * d.nv * d.nu + uc;
    constexpr int PF = 8;
    auto value = [&](float y, int v) { return scale ? y * chord_scale(r, __ldg(d.dz_mm + v)) : y; };
    // pass 1: compensated sum of the segment
    float s = 0.f, e = 0.f;
    for (int v0 = v_lo; v0 < v_hi; v0 += PF) {
        float y[PF];
#pragma unroll
        for (int q = 0; q < PF; ++q) y[q] = (v0 + q < v_hi) ? __ldg(p + (size_t)(v0 + q) * d.nu) : 0.f;
#pragma unroll
        for (int q = 0; q < PF; ++q) {
            if (v0 + q >= v_hi) break;
            const float yy = value(y[q], v0 + q);
            const float t = __fadd_rn(s, yy);
            e += two_sum_err(s, yy, t);
            s = t;
        }
    }
    tot[seg][lane] = make_float2(s, e);
    __syncthreads();
    // two-float total of the segments below this one
    float os = 0.f, oe = 0.f;
    for (int g = 0; g < seg; ++g) {
        const float2 t2 = tot[g][lane];
        const float t = __fadd_rn(os, t2.x);
        oe += two_sum_err(os, t2.x, t) + t2.y;
        os = t;
    }
    if (!in_range) return;
    float *po = rs_out ? rs_out + (size_t)a * d.nv * d.nu + u : nullptr;
    float2 *c = C + (size_t)a * (d.nv + 1) * d.nu + u;
    if (seg == 0) *c = make_float2(0.f, 0.f);
    // pass 2: the running sum of the segment on top of the offset
    s = os; e = oe;
    for (int v0 = v_lo; v0 < v_hi; v0 += PF) {
        float y[PF];
#pragma unroll
        for (int q = 0; q < PF; ++q) y[q] = (v0 + q < v_hi) ? __ldg(p + (size_t)(v0 + q) * d.nu) : 0.f;
#pragma unroll
        for (int q = 0; q < PF; ++q) {
            if (v0 + q >= v_hi) break;
            const float yy = value(y[q], v0 + q);
            if (scale && po) po[(size_t)(v0 + q) * d.nu] = yy;
            const float t = __fadd_rn(s, yy);
            e += two_sum_err(s, yy, t);
            s = t;
            c[(size_t)(v0 + q + 1) * d.nu] = make_float2(s, e);
        }
    }
}

#ifndef CBCT_BP_MINB
#define CBCT_BP_MINB 8          // resident CTAs per SM the plain gather is compiled for (64 registers)
#endif
#ifndef CBCT_BP_MINB_M
#define CBCT_BP_MINB_M 5        // the same for the mirrored gather (two accumulator columns)
#endif

// MIRROR: the scan is symmetric about the central plane z = 0 (nz even, detector centred in v: cv = (nv-1)/2), so ray
// (u, nv-1-v) is the mirror image of ray (u, v) and voxel row nz-1-k that of row k.  A thread then owns a column chunk of
// the UPPER half (planes zk >= 0) together with its mirror image: the run bounds of plane -zk are nv - vT and nv - vTn, its
// crossing ray is nv-1-vs with the same b, and the direction of every crossing ray is the sign of dt (zeta > 0 above the
// central plane), so the bound / crossing arithmetic of a plane (17 of its ~30 instructions) is done once for two voxel rows.
template <int KC, int BI, bool MIRROR>
__global__ void __launch_bounds__(32 * BI, MIRROR ? CBCT_BP_MINB_M : CBCT_BP_MINB)
backproject_kernel(const DevGeom d, const int cls, const unsigned char *__restrict__ angle_has,
                   const float *__restrict__ rs, const PrefixT *__restrict__ C, const float *__restrict__ inv_s, float *__restrict__ G,
                   const int parts)
{
    const ClassGrid cg = d.cls[cls];
    const int j = blockIdx.x * 32 + threadIdx.x;      // minor index
    const int i = blockIdx.y * BI + threadIdx.y;      // major index = slab
    // small volumes: the angle list is dealt out over `parts` CTAs per column chunk (part p takes angles p, p + parts, ...),
    // each writing its own partial volume; op_combine adds the partial volumes in the order of p
    const int kchunks = gridDim.z / parts, part = blockIdx.z / kchunks;
    const int k0 = (MIRROR ? d.koff : 0) + (blockIdx.z - part * kchunks) * KC;
    G += (size_t)part * d.nx * d.ny * d.nz;
    if (i >= cg.nmaj) return;                          // warp-uniform
    const bool valid = j < cg.nmin;

    // kPacked (MIRROR, float prefix sums): a voxel row and its mirror image accumulate as the two halves of one float2, updated
    // by sm_100's packed fp32 instructions (FFMA2: two fused multiply-adds, one issue slot) — the kernel is bound by issue slots
    constexpr bool kPacked = MIRROR && !kFixed && CBCT_BP_PACKED != 0;
    float2 accP[kPacked ? KC : 1];
    if constexpr (kPacked) {
#pragma unroll
        for (int q = 0; q < KC; ++q) accP[q] = make_float2(0.f, 0.f);
    }
    float acc[kPacked ? 1 : KC], accL[MIRROR && !kPacked ? KC : 1];
    if constexpr (!kPacked) {
#pragma unroll
        for (int q = 0; q < KC; ++q) acc[q] = 0.f;
        if constexpr (MIRROR) {
#pragma unroll
            for (int q = 0; q < KC; ++q) accL[q] = 0.f;
        }
    }

    // the column's x-y square in mm (candidate search only; the accept test is exact)
    const float maj0 = ((float)i - 0.5f * (float)cg.nmaj) * cg.hmaj, maj1 = maj0 + cg.hmaj;
    const float mn0 = ((float)min(j, cg.nmin - 1) - 0.5f * (float)cg.nmin) * cg.hmin, mn1 = mn0 + cg.hmin;
    const float x0 = cls == 0 ? maj0 : mn0, x1 = cls == 0 ? maj1 : mn1;
    const float y0 = cls == 0 ? mn0 : maj0, y1 = cls == 0 ? mn1 : maj1;
    const float ef = (float)(i - cg.ioff);
    const float cu = d.cu, cv = d.cv;                  // detector index of the central ray (shifted panels: not the middle)
    const float sdd_du = d.sdd / d.du;
    const int npitchC = opaque(-d.nu * (int)sizeof(PrefixT)), npitchR = opaque(-d.nu * (int)sizeof(float));   // MIRROR: rows counted down
    const float inv_hzdv = rcp_approx(d.hzdv_hi);
    const float zk0 = (float)(k0 - d.koff) - d.zfrac;  // plane k0 in the units of z_entry(), minus zfrac (MIRROR: >= 0, an integer)

    for (int a = part; a < d.na; a += parts) {
        if (!angle_has[a]) continue;                   // uniform
        const float2 cs = __ldg(d.cs + a);
        float umin = 3e38f, umax = -3e38f;
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const float x = (m & 1) ? x1 : x0, y = (m & 2) ? y1 : y0;
            const float num = fmaf(-x, cs.y, y * cs.x);
            const float den = d.sad - fmaf(x, cs.x, y * cs.y);
            const float uu = fmaf(sdd_du, num * rcp_approx(den), cu);      // den = depth of the corner > 0
            umin = fminf(umin, uu);
            umax = fmaxf(umax, uu);
        }
        const int uA = max(0, (int)floorf(umin - 0.02f));
        const int uB = valid ? min(d.nu - 1, (int)ceilf(umax + 0.02f)) : -1;
        for (int u = uA; u <= uB; ++u) {
            const RayXY r = load_ray(d, a, u);
            if (ray_cls(r.range) != cls) continue;
            // the projector's minor_split() with the minor coordinate Ya = mc + ef sm carried as two floats (exact product and
            // sum, plus what the table's floats drop of mc and sm): the split a = (row boundary - Ya) / sm amplifies an error of
            // Ya by 1 / |sm|, and fp32 leaves 1.5e-5 of a voxel in Ya at |ef| = 256
            const float4 rlo = __ldg(d.rays_lo + (a * d.nu + u));
            const float pm = __fmul_rn(ef, r.sm), pm_lo = fmaf(ef, r.sm, -pm);
            const float Ya = __fadd_rn(r.mc, pm);
            const float Ya_lo = fmaf(ef, rlo.y, __fadd_rn(__fadd_rn(two_sum_err(r.mc, pm, Ya), pm_lo), rlo.x));
            const float fl = floorf(Ya);
            const float a_ = __saturatef(__fsub_rn(__fsub_rn(fl + (r.sm >= 0.f ? 1.f : 0.f), Ya), Ya_lo) * r.inv_sm);
            const int ja = (int)fl + cg.joff;
            float l0, l1;
            if (ja == j) { l0 = 0.f; l1 = a_; }
            else if (ja + (r.sm >= 0.f ? 1 : -1) == j) { l0 = a_; l1 = 1.f; }
            else continue;
            const float w = l1 - l0;
            if (!(w > 0.f)) continue;

            // Entry ray parameter T = tc + ef dt and the detector rows per z plane at the entry plane, cT = (hz / dv) / T, as
            // unevaluated sums of two floats: a z plane zk meets the detector at row cv + zk cT, |zk cT| up to several hundred
            // rows, and the crossing fraction of a ray amplifies an error in that position by (T / dt) / |v - cv| (4 at c5):
            // plain fp32 leaves 1e-4 of a chord there.  The exit plane only detects crossings; fp32 is enough for it.
            // (__fmul_rn / __fadd_rn / __fsub_rn are never contracted into FMAs, which would break the error-free sums)
            const float p_hi = __fmul_rn(ef, r.dt), p_lo = fmaf(ef, r.dt, -p_hi);
            const float T = __fadd_rn(r.tc, p_hi);
            const float T_lo = (two_sum_err(r.tc, p_hi, T) + p_lo) + rlo.z;
            const float Tn = fmaf(ef + 1.f, r.dt, r.tc);
            const float rT = rcp_approx(T);
            const float cT = __fmul_rn(d.hzdv_hi, rT), cTn = d.hzdv_hi * rcp_approx(Tn);          // d v / d z at entry / exit (T > 0)
            // rho = (true cT - cT) / cT from the exact remainder hz/dv - cT (T + T_lo)
            const float rho = __fadd_rn(fmaf(-cT, T_lo, fmaf(-cT, T, d.hzdv_hi)), d.hzdv_lo) * inv_hzdv;
            // 32-bit element offsets of (a, v = 0, u) in the prefix sums and in the projections (checked at geometry creation)
            // byte offsets: one IMAD.WIDE (row * pitch + base) forms the address of a row's element
            const char *Cu = reinterpret_cast<const char *>(C + (a * (d.nv + 1) * d.nu + u));
            const float wr = kFixed ? w * __ldg(inv_s + (a * d.nu + u)) : w;          // weight of a run sum (fixed point: unscaled)
            const char *Ru = reinterpret_cast<const char *>(rs + (a * d.nv * d.nu + u));
            const int pitchC = d.nu * (int)sizeof(PrefixT), pitchR = d.nu * (int)sizeof(float);
            // b = lambda at which ray v meets plane zk: (T + b dt) (v - cv) dv / hz = zk.  With delta = (v - cv) - zk cT, the
            // distance of the ray from where the plane meets the detector at the slab's entry, b = -(T / dt) delta / (v - cv).
            const float TD = T * r.inv_dt;
            const float l1c = fmaf(-TD, rho, l1);
            // entry and exit bounds of a plane less than one detector row apart on every plane of the chunk: at most one
            // ray crosses a plane inside the slab, and the loop over further crossing rays is compiled out
            const bool single = fmaxf(fabsf(zk0), fabsf(zk0 + (float)KC)) * fabsf(cT - cTn) < 0.999f;
            // all run bounds of the chunk fall on the detector: no clamping needed (MIRROR: zk >= 0, so the bounds lie between cv
            // and the top plane's, and their mirror images do the same below)
            bool inside;
            if constexpr (MIRROR) inside = fmaf(zk0 + (float)KC, fmaxf(cT, cTn), cv) <= (float)(d.nv - 1);
            else inside = fminf(fminf(fmaf(zk0, cT, cv), fmaf(zk0, cTn, cv)), fminf(fmaf(zk0 + (float)KC, cT, cv), fmaf(zk0 + (float)KC, cTn, cv))) >= 0.f &&
                          fmaxf(fmaxf(fmaf(zk0, cT, cv), fmaf(zk0, cTn, cv)), fmaxf(fmaf(zk0 + (float)KC, cT, cv), fmaf(zk0 + (float)KC, cTn, cv))) <= (float)(d.nv - 1);
            // bounds of plane k0 (plane k0+q: + q cT, q a literal); the entry bound as xT0 + x_lo, x_lo = what the float drops of
            // cv + zk0 cT (exact product by FMA, exact sum by two-sum).  The plane really sits at cv + zk cT (1 + rho): with
            // delta' = (v - cv) - zk cT, delta = delta' - rho zk cT = delta' - rho (v - cv) to first order, so
            // l1 - b = (l1 - (T / dt) rho) + (T / dt) delta' / (v - cv): the correction costs nothing per plane.
            const float P_hi = __fmul_rn(zk0, cT), P_lo = fmaf(zk0, cT, -P_hi);
            const float xT0 = __fadd_rn(cv, P_hi), xTn0 = fmaf(zk0, cTn, cv);
            // reference row on a 2^-8 grid, so that vs - xTc is exact for every detector row vs (both multiples of 2^-8 below 2^15),
            // and what it drops of cv + zk0 cT
            const float xTc = rintf(xT0 * 256.f) * (1.f / 256.f);
            const float x_lo = __fadd_rn((two_sum_err(cv, P_hi, xT0) + P_lo) + d.cv_lo, __fsub_rn(xT0, xTc));
            // MIRROR: prefix row nv and projection row nv-1 of this (a, u): the mirrored bound nv - vT and ray nv-1-vs are one
            // IMAD.WIDE with the negated pitch away
            const char *CuT = opaque(Cu + (long long)d.nv * pitchC), *RuT = opaque(Ru + (long long)(d.nv - 1) * pitchR);
            const int up_sign = __float_as_int(r.dt) & 0x80000000;                     // MIRROR: rising iff dt > 0
            auto planes = [&](auto multi_tag, auto clamp_tag) {
                constexpr bool MULTI = decltype(multi_tag)::value, CLAMP = decltype(clamp_tag)::value;
                PrefixT c1{}, c1L{};
#pragma unroll
                for (int q = 0; q <= KC; ++q) {
                    // first ray at or above plane k0+q at the slab's entry / exit plane
                    // (plain gather: from zk itself, so that the central plane zk = 0 sits at cv exactly, its two bounds agree and a
                    // ray lying in it — odd nv, even nz — crosses nothing and belongs to the row above; the mirrored gather meets that
                    // plane only as q = 0 of the chunk with zk0 = 0, where xT0 = xTn0 = cv)
                    int vT, vTn;
                    if constexpr (kPacked) {                   // both bounds by one packed FMA
                        const float2 xb = __ffma2_rn(make_float2((float)q, (float)q), make_float2(cT, cTn), make_float2(xT0, xTn0));
                        vT = (int)ceilf(xb.x);
                        vTn = (int)ceilf(xb.y);
                    } else if constexpr (MIRROR) {
                        vT = (int)ceilf(fmaf((float)q, cT, xT0));
                        vTn = (int)ceilf(fmaf((float)q, cTn, xTn0));
                    } else {
                        const float zk = zk0 + (float)q;
                        vT = (int)ceilf(fmaf(zk, cT, cv));
                        vTn = (int)ceilf(fmaf(zk, cTn, cv));
                    }
                    if constexpr (CLAMP) {
                        vT = min(max(vT, 0), d.nv);
                        vTn = min(max(vTn, 0), d.nv);
                    }
                    const PrefixT c2 = __ldg(reinterpret_cast<const PrefixT *>(row_ptr(Cu, vT, pitchC)));
                    // rays crossing plane k0+q inside the slab: v in [min(vT,vTn), max(vT,vTn)) (y = 0 stands in if there is none).
                    // The part of such a ray's chord in this minor row that lies beyond the plane is
                    //   max(0, l1 - max(l0, sat(b))) = min(sat(l1 - b), l1 - l0)       (0 <= l0 <= l1 <= 1)
                    // — its exit-row fraction among the projector's four.  A ray in the central plane (v = cv, only met at zk = 0)
                    // crosses nothing: its 0 * inf is a NaN that the saturation turns into 0.
                    const int dlt = vTn - vT, vs = min(vT, vTn);
                    const float vsf = (float)vs, vf = vsf - cv;
                    // delta = vs - (cv + (zk0 + q) cT): vs - xTc is exact, the FMA rounds a number of a few rows at most, x_lo restores
                    // what xTc dropped
                    const float dl = __fsub_rn(fmaf(-(float)q, cT, __fsub_rn(vsf, xTc)), x_lo);
                    const float fr = fminf(__saturatef(fmaf(TD, dl * rcp_approx(vf), l1c)), w);
                    // signed: positive = the ray rises across the plane (dt zeta(v) > 0), so the fraction moves from the row below
                    // the plane to the row above it
                    const int sgn = MIRROR ? up_sign : ((__float_as_int(vf) ^ __float_as_int(r.dt)) & 0x80000000);
                    const float fs = __int_as_float(__float_as_int(fr) ^ sgn);
                    float yq = 0.f;
                    if (dlt != 0) yq = __ldg(reinterpret_cast<const float *>(row_ptr(Ru, vs, pitchR)));
                    float up = fs * yq;                // moved up across the plane (negative: moved down)
                    // the mirror image: plane -zk, bounds nv - vT (plane 0 is its own image: the same bound, so that a ray lying
                    // in it belongs to the row above it on both sides), crossing ray nv-1-vs, rising <-> falling
                    [[maybe_unused]] PrefixT c2L;
                    [[maybe_unused]] float dn = 0.f;                    // moved DOWN across the mirrored plane
                    [[maybe_unused]] float yL = 0.f;
                    if constexpr (MIRROR) {
                        c2L = (q == 0 && zk0 == 0.f) ? c2 : __ldg(reinterpret_cast<const PrefixT *>(row_ptr(CuT, vT, npitchC)));
                        if (dlt != 0) yL = __ldg(reinterpret_cast<const float *>(row_ptr(RuT, vs, npitchR)));
                        dn = fs * yL;
                    }
                    if constexpr (MULTI) {
                        for (int v = vs + 1; v < vs + abs(dlt); ++v) {   // further rays crossing this plane (fine detector rows)
                            const float dl2 = __fsub_rn(fmaf(-(float)q, cT, __fsub_rn((float)v, xTc)), x_lo);
                            const float fr2 = fminf(__saturatef(fmaf(TD, dl2 * rcp_approx((float)v - cv), l1c)), w);
                            const float f2 = __int_as_float(__float_as_int(fr2) ^ sgn);
                            up = fmaf(f2, __ldg(reinterpret_cast<const float *>(row_ptr(Ru, v, pitchR))), up);
                            if constexpr (MIRROR) dn = fmaf(f2, __ldg(reinterpret_cast<const float *>(row_ptr(RuT, v, npitchR))), dn);
                        }
                    }
                    if constexpr (kPacked && !MULTI) {
                        // (upper row, mirrored row) side by side: c2 - c1 and c1L - c2L as packed FMAs with -1, the run sums, then
                        // three packed FMAs move w run - up into row q-1 and up into row q on both sides
                        const float2 m1 = make_float2(-1.f, -1.f), yy = make_float2(yq, yL);
                        if (q > 0) {
                            const float2 dU = __ffma2_rn(c1, m1, c2), dL = __ffma2_rn(c2L, m1, c1L);
                            const float2 run = make_float2(dU.x + dU.y, dL.x + dL.y);
                            accP[q > 0 ? q - 1 : 0] = __ffma2_rn(make_float2(wr, wr), run, accP[q > 0 ? q - 1 : 0]);
                            accP[q > 0 ? q - 1 : 0] = __ffma2_rn(make_float2(-fs, -fs), yy, accP[q > 0 ? q - 1 : 0]);
                        }
                        if (q < KC) accP[q < KC ? q : 0] = __ffma2_rn(make_float2(fs, fs), yy, accP[q < KC ? q : 0]);
                    } else if constexpr (kPacked) {           // the rare several-crossings loop: the same rows, one half at a time
                        if (q > 0) {
                            accP[q > 0 ? q - 1 : 0].x = fmaf(wr, run_sum(c2, c1), accP[q > 0 ? q - 1 : 0].x) - up;
                            accP[q > 0 ? q - 1 : 0].y = fmaf(wr, run_sum(c1L, c2L), accP[q > 0 ? q - 1 : 0].y) - dn;
                        }
                        if (q < KC) {
                            accP[q < KC ? q : 0].x += up;
                            accP[q < KC ? q : 0].y += dn;
                        }
                    } else {
                        if (q > 0) {
                            acc[q > 0 ? q - 1 : 0] = fmaf(wr, run_sum(c2, c1), acc[q > 0 ? q - 1 : 0]) - up;
                            if constexpr (MIRROR) {
                                accL[q > 0 ? q - 1 : 0] = fmaf(wr, run_sum(c1L, c2L), accL[q > 0 ? q - 1 : 0]) - dn;
                            }
                        }
                        if (q < KC) {
                            acc[q < KC ? q : 0] += up;
                            if constexpr (MIRROR) accL[q < KC ? q : 0] += dn;
                        }
                    }
                    c1 = c2;
                    if constexpr (MIRROR) c1L = c2L;
                }
            };
            if (single && inside) planes(std::false_type{}, std::false_type{});
            else if (single) planes(std::false_type{}, std::true_type{});
            else planes(std::true_type{}, std::true_type{});
        }
    }
    if (!valid) return;
#pragma unroll
    for (int q = 0; q < KC; ++q) {
        const int k = k0 + q;
        if (k < d.nz) {
            G[((size_t)k * cg.nmaj + i) * cg.nmin + j] = kPacked ? accP[kPacked ? q : 0].x : acc[kPacked ? 0 : q];
            if constexpr (MIRROR) G[((size_t)(d.nz - 1 - k) * cg.nmaj + i) * cg.nmin + j] = kPacked ? accP[kPacked ? q : 0].y : accL[kPacked ? 0 : q];
        }
    }
}

cbct_status op_backproject_prefix(cbct_geometry *g, const float *d_in, int scale, float *d_rs_out, cudaStream_t st)
{
    CBCT_TRY(ensure(g, &g->proj_prefix, (size_t)g->na * (g->nv + 1) * g->nu));
    ProfileScope ps(2, st);
    dim3 grid((g->nu + 127) / 128, g->na);
    // kFixed: the column scales 1/s(a,u) sit behind the (half-size) integer prefix values in the same buffer
    PrefixT *Cp = reinterpret_cast<PrefixT *>(g->proj_prefix);
    float *inv_s = kFixed ? reinterpret_cast<float *>(Cp + (size_t)g->na * (g->nv + 1) * g->nu) : nullptr;
#ifndef CBCT_BP_PREFIX_SEG
#define CBCT_BP_PREFIX_SEG 8
#endif
    if constexpr (!kFixed && CBCT_BP_PREFIX_SEG > 1) {
        if (g->nv >= 8 * CBCT_BP_PREFIX_SEG) {
            dim3 sgrid((g->nu + 31) / 32, g->na), sblock(32, CBCT_BP_PREFIX_SEG);
            prefix_seg_kernel<CBCT_BP_PREFIX_SEG><<<sgrid, sblock, 0, st>>>(g->dev, d_in, scale, d_rs_out, reinterpret_cast<float2 *>(g->proj_prefix));
            CBCT_LAUNCH_CHECK();
            return CBCT_OK;
        }
    }
    prefix_kernel<<<grid, 128, 0, st>>>(g->dev, d_in, scale, d_rs_out, Cp, inv_s, g->bp_run_max);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

template <int KC, int BI, bool MIRROR>
static cbct_status launch_gather(cbct_geometry *g, const float *d_scaled, cudaStream_t st)
{
    // A small volume has too few voxel columns to fill the GPU (c1: 16 CTAs per class, 70 us per launch whatever the clock):
    // the angles are then dealt out over up to 8 CTAs per column chunk, aiming at two CTAs per SM
    const int rows = MIRROR ? g->nz / 2 : g->nz;       // voxel rows the chunks cover (MIRROR: the upper half)
    const int kchunks = (rows + KC - 1) / KC;
    g->bp_parts = 1;
    {
        int dev = 0, sms = 148;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        const ClassGrid &cg = g->dev.cls[0];
        const long ctas = (long)((cg.nmin + 31) / 32) * ((cg.nmaj + BI - 1) / BI) * kchunks;
        while (g->bp_parts < 8 && ctas * g->bp_parts < 2L * sms && 2 * g->bp_parts <= g->na) g->bp_parts *= 2;
    }
    for (int c = 0; c < 2; ++c) {
        if (g->n_tiles[c] == 0) continue;
        if (g->G_parts_alloc[c] < g->bp_parts) {
            if (g->G_cls[c]) { CBCT_CUDA(cudaStreamSynchronize(st)); cbct_dev_free(g, g->G_cls[c]); g->bytes -= g->n_vox() * sizeof(float) * g->G_parts_alloc[c]; g->G_cls[c] = nullptr; }
            CBCT_TRY(ensure(g, &g->G_cls[c], g->n_vox() * g->bp_parts));
            g->G_parts_alloc[c] = g->bp_parts;
        }
        const ClassGrid &cg = g->dev.cls[c];
        dim3 grid((cg.nmin + 31) / 32, (cg.nmaj + BI - 1) / BI, kchunks * g->bp_parts), block(32, BI);
        const PrefixT *Cp = reinterpret_cast<const PrefixT *>(g->proj_prefix);
        const float *inv_s = kFixed ? reinterpret_cast<const float *>(Cp + (size_t)g->na * (g->nv + 1) * g->nu) : nullptr;
        backproject_kernel<KC, BI, MIRROR><<<grid, block, 0, st>>>(g->dev, c, g->d_angle_has[c], d_scaled, Cp, inv_s, g->G_cls[c], g->bp_parts);
        CBCT_LAUNCH_CHECK();
    }
    return CBCT_OK;
}

// the scan is its own mirror image about the central plane: an even number of slices and a detector centred in v
bool gather_is_mirrored(const cbct_geometry *g)
{
    return g->use_mirror && g->nz % 2 == 0 && g->off_v == 0.0;
}

cbct_status op_backproject_gather(cbct_geometry *g, const float *d_scaled, cudaStream_t st)
{
    // z rows per thread and slabs per CTA: compile-time tuning knobs (measured best of a sweep on B200)
#ifndef CBCT_BP_KC
#define CBCT_BP_KC 16
#define CBCT_BP_BI 4
#endif
#ifndef CBCT_BP_KC_M
#define CBCT_BP_KC_M 16
#endif
    ProfileScope ps(3, st);
    if (gather_is_mirrored(g)) return launch_gather<CBCT_BP_KC_M, CBCT_BP_BI, true>(g, d_scaled, st);
    return launch_gather<CBCT_BP_KC, CBCT_BP_BI, false>(g, d_scaled, st);
}

// out = G1 + G0^T  or  out = f - c (G1 + G0^T) [clamped]  — fuses a4 (and a6 when n_inner = 0) into the
// transpose-add that the two-class gather needs anyway.
template <bool PARTS>
__global__ void __launch_bounds__(256) combine_kernel(const float *__restrict__ G0, const float *__restrict__ G1,
                                                      const float *__restrict__ f, float c, int clamp,
                                                      float *__restrict__ out, int nx, int ny, int parts, size_t nvox)
{
    __shared__ float tile[32][33];
    const int k = blockIdx.z;
    const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
    const size_t plane = (size_t)k * nx * ny;
    // all of a thread's loads (4 of G0 for the transpose, 4 of G1, 4 of f) are requested before the first use: the kernel is
    // latency-bound, so what counts is the bytes in flight
    float g1[4], fv[4], g0[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int r = threadIdx.y + 8 * q;
        const int j = j0 + r, i = i0 + threadIdx.x;
        const bool in = j < ny && i < nx;
        const size_t o = plane + (size_t)j * nx + i;
        g1[q] = 0.f;
        if (G1 && in) {
            g1[q] = __ldg(G1 + o);
            if constexpr (PARTS)
                for (int p = 1; p < parts; ++p) g1[q] += __ldg(G1 + p * nvox + o);
        }
        fv[q] = (f && in) ? __ldg(f + o) : 0.f;
        g0[q] = 0.f;
        if (G0) {                                  // G0 is [k][x][y]: read rows of constant x
            const int ii = i0 + r, jj = j0 + threadIdx.x;
            if (ii < nx && jj < ny) {
                g0[q] = __ldg(G0 + plane + (size_t)ii * ny + jj);
                if constexpr (PARTS)
                    for (int p = 1; p < parts; ++p) g0[q] += __ldg(G0 + p * nvox + plane + (size_t)ii * ny + jj);
            }
        }
    }
    if (G0) {
#pragma unroll
        for (int q = 0; q < 4; ++q) tile[threadIdx.y + 8 * q][threadIdx.x] = g0[q];
        __syncthreads();
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int r = threadIdx.y + 8 * q;
        const int j = j0 + r, i = i0 + threadIdx.x;
        if (j < ny && i < nx) {
            const float gsum = (G0 ? tile[threadIdx.x][r] : 0.f) + g1[q];
            float val = gsum;
            if (f) {
                val = fmaf(-c, gsum, fv[q]);
                if (clamp) val = fmaxf(val, 0.f);
            }
            out[plane + (size_t)j * nx + i] = val;
        }
    }
}

cbct_status op_combine(cbct_geometry *g, const float *f, float c, int clamp, float *out, cudaStream_t st)
{
    ProfileScope ps(4, st);
    const float *G0 = g->n_tiles[0] > 0 ? g->G_cls[0] : nullptr;
    const float *G1 = g->n_tiles[1] > 0 ? g->G_cls[1] : nullptr;
    dim3 grid((g->nx + 31) / 32, (g->ny + 31) / 32, g->nz), block(32, 8);
    if (g->bp_parts > 1) combine_kernel<true><<<grid, block, 0, st>>>(G0, G1, f, c, clamp, out, g->nx, g->ny, g->bp_parts, g->n_vox());
    else combine_kernel<false><<<grid, block, 0, st>>>(G0, G1, f, c, clamp, out, g->nx, g->ny, 1, g->n_vox());
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}
