// a1/a2, staged variant: the ray-driven exact-chord projector of projector.cu with the volume brought to the rays through
// shared memory by the TMA unit (BASELINE.json north_star: "a ray-driven projector kernel that stages volume bricks through
// TMA/shared memory and shares detector-row work across a warp"; "we first perform the forward x-ray projection
// operation ... for all (u,v) and theta").
//
// Same rays, same arithmetic, same order of the fp32 sums as forward_kernel (projector.cu): a CTA is one 32-wide detector
// column tile x (V * WARPS) detector rows of one angle; a thread marches V rays of one column; per slab a ray touches two
// minor rows and at most two z rows with the four chord fractions of ray_common.cuh.  What differs is where the voxels come
// from.  The CTA walks its slab range in blocks of SB slabs; for each block ONE brick of the class' padded volume copy
//     SB major rows  x  BJ minor columns  x  BK z planes
// holds every voxel any of its rays touches there.  Its corner (cj, i0, ck) follows the ray fan and is found by warp 0 from
// the extremes of the tile's rays (minor coordinate is linear in the slab index and monotone in u; z is monotone in v); BJ and
// BK are the geometry's worst-case spans, found at handle creation.  The bricks travel by cp.async.bulk.tensor (3-D box,
// out-of-range parts read as zero) into a ring of shared-memory stages, completion on an mbarrier, two blocks ahead of the
// march; all voxel reads of the march are 32-bit-addressed LDS.
#include "cbct_internal.h"
#include "ray_common.cuh"
#include "tma.cuh"

namespace {
#ifndef CBCT_FWT_SB
#define CBCT_FWT_SB 8           // measured on B200 (c2 / c3, ms per projection; __ldg march: 1.97 / 2.45):
#define CBCT_FWT_STAGES 2       //   SB 8, 3 stages, 4 warps 2.63 / 3.60 (3 CTAs per SM by shared memory); SB 8, 2 stages 1.97 / 2.69;
#define CBCT_FWT_WARPS 4        //   SB 4, 3 stages 1.98 / 2.67; SB 4, 8 warps 2.04 / 2.89; SB 2, 4 stages 2.38 / 3.41
#endif
constexpr int SB = CBCT_FWT_SB;            // slabs per brick
constexpr int kStages = CBCT_FWT_STAGES;

template <int V, int WARPS>
__global__ void __launch_bounds__(32 * WARPS)
forward_tma_kernel(const DevGeom d, const int cls, const int2 *__restrict__ tiles, const __grid_constant__ CUtensorMap tm_vol,
                   const int BJ, const int BK, float *__restrict__ out, const float *__restrict__ Y, const int mode)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    const int brick_floats = BK * SB * BJ;
    const size_t brick_bytes = ((size_t)brick_floats * sizeof(float) + 127) & ~(size_t)127;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + kStages * brick_bytes);            // [kStages]
    int *meta = reinterpret_cast<int *>(smem + kStages * brick_bytes + 64);                 // [kStages][2]: cj, ck
    int *range = meta + 2 * kStages;                                                         // [WARPS][2]: lo_w, hi_w

    const ClassGrid cg = d.cls[cls];
    const int lane = threadIdx.x, wid = threadIdx.y;
    const int2 tile = tiles[blockIdx.x];
    const int a = tile.x, u = tile.y + lane;
    const int vg0 = blockIdx.y * WARPS * V;                    // first detector row of the CTA
    const int v0 = vg0 + wid * V;
    const bool warp_has_rows = v0 < d.nv;

    RayXY r = load_ray(d, a, min(u, d.nu - 1));
    int ilo = ray_ilo(r.range), ihi = ray_ihi(r.range);
    const bool xy_ok = (u < d.nu) && (ray_cls(r.range) == cls) && ihi > ilo;   // the ray meets the volume's x-y footprint (same in every warp)
    const bool mine = (u < d.nu) && (ray_cls(r.range) == cls) && warp_has_rows;
    bool active = mine && ihi > ilo;
    // z clip (as forward_kernel): the ray of this thread closest to the central plane stays inside longest
    if (warp_has_rows) {
        const float za = __ldg(d.zeta + v0), zb = __ldg(d.zeta + min(v0 + V - 1, d.nv - 1));
        float tmax = 3.0e38f;
        if (za > 0.f && zb > 0.f) tmax = ((float)(d.nz - d.koff) + 1.f - d.zfrac) / fminf(za, zb);
        else if (za < 0.f && zb < 0.f) tmax = (-(float)d.koff - 1.f - d.zfrac) / fmaxf(za, zb);
        if (tmax < 2.f) {
            float e = (tmax - r.tc) * r.inv_dt;
            if (r.dt > 0.f) ihi = min(ihi, cg.ioff + (int)floorf(e) + 2);
            else            ilo = max(ilo, cg.ioff + (int)ceilf(e) - 2);
        }
        active = active && ihi > ilo;
    }
    const int lo_w = __reduce_min_sync(0xffffffffu, active ? ilo : 0x7fffffff);
    const int hi_w = __reduce_max_sync(0xffffffffu, active ? ihi : -1);
    // a lane without a ray through the footprint marches a copy of a neighbour's ray (its loads then stay inside the brick);
    // it stores 0 if the ray is its own (a miss) and nothing otherwise.  The choice depends on x-y geometry only, so all
    // warps of the CTA march the same 32 x-y traversals and warp 0 can place the bricks for everyone.
    {
        const unsigned am = __ballot_sync(0xffffffffu, xy_ok);
        if (am) {
            const int src = __ffs(am) - 1;
            RayXY s;
            s.mc = __shfl_sync(0xffffffffu, r.mc, src); s.sm = __shfl_sync(0xffffffffu, r.sm, src);
            s.inv_sm = __shfl_sync(0xffffffffu, r.inv_sm, src); s.tc = __shfl_sync(0xffffffffu, r.tc, src);
            s.dt = __shfl_sync(0xffffffffu, r.dt, src); s.inv_dt = __shfl_sync(0xffffffffu, r.inv_dt, src);
            s.lxy2 = __shfl_sync(0xffffffffu, r.lxy2, src); s.range = r.range;
            if (!xy_ok) r = s;
        }
    }
    if (lane == 0) { range[2 * wid] = lo_w; range[2 * wid + 1] = hi_w; }
    if (threadIdx.x == 0 && threadIdx.y == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(full + s, 1);
        mbar_fence_init();
    }
    __syncthreads();
    int lo_c = 0x7fffffff, hi_c = -1;
#pragma unroll
    for (int q = 0; q < WARPS; ++q) { lo_c = min(lo_c, range[2 * q]); hi_c = max(hi_c, range[2 * q + 1]); }
    const int nblk = hi_c > lo_c ? (hi_c - lo_c + SB - 1) / SB : 0;

    const float dirpos = r.sm >= 0.f ? 1.f : 0.f;
    const int dneg = r.sm >= 0.f ? 0 : 1;
    const int vlast = min(vg0 + WARPS * V, d.nv) - 1;
    const float zeta_first = __ldg(d.zeta + min(vg0, d.nv - 1)), zeta_last = __ldg(d.zeta + vlast);

    // warp 0: corner of the brick of block b (padded-copy coordinates) and its TMA
    auto issue = [&](int b) {
        const int st = b % kStages;
        const int i0 = lo_c + b * SB, i1 = min(i0 + SB, hi_c) - 1;       // first and last slab of the block
        int jmn = 0x7fffffff, kmn = 0x7fffffff;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const float ef = (float)((e ? i1 : i0) - cg.ioff);
            float a_, fl;
            minor_split(ef, r, dirpos, a_, fl);
            jmn = min(jmn, min(max((int)fl + cg.joff - dneg, -2), cg.nmin));
            // z rows at the entry plane of the first and the exit plane of the last slab, for the CTA's extreme detector rows
            const float T = fmaf(ef + (e ? 1.f : 0.f), r.dt, r.tc);
            const float z1 = floorf(fmaf(T, zeta_first, d.zfrac)), z2 = floorf(fmaf(T, zeta_last, d.zfrac));
            kmn = min(kmn, (int)fminf(z1, z2));
        }
        jmn = __reduce_min_sync(0xffffffffu, jmn);
        kmn = __reduce_min_sync(0xffffffffu, kmn);
        // column in the padded row, rounded down to a 16-byte boundary (jmn >= -2): cp.async.bulk.tensor raises "illegal
        // instruction" on B200 when the box does not start on one in the contiguous dimension (measured; the other two are free)
        const int cj = (jmn + kPadLo) & ~3;
        const int ck = min(max(kmn + d.koff - 1, -kPadK), d.nz + kPadK - 1) + kPadK;       // plane in the padded copy (1 row of slack)
        if (lane == 0) {
            meta[2 * st] = cj; meta[2 * st + 1] = ck;
            mbar_arrive_expect_tx(full + st, (uint32_t)(brick_floats * sizeof(float)));
            tma_load_3d(smem + st * brick_bytes, &tm_vol, full + st, cj, i0, ck);
        }
    };
    if (wid == 0)
        for (int b = 0; b < nblk && b < kStages; ++b) issue(b);

    float acc[V];
#pragma unroll
    for (int q = 0; q < V; ++q) acc[q] = 0.f;

    if (nblk > 0 && warp_has_rows) {
        float zeta[V], inv_sz[V], zbnd[V];
        int krow[V];
        {
            const float T0 = fmaf((float)(lo_c - cg.ioff), r.dt, r.tc);
#pragma unroll
            for (int q = 0; q < V; ++q) {
                const int v = min(v0 + q, d.nv - 1);
                zeta[q] = __ldg(d.zeta + v);
                inv_sz[q] = r.inv_dt * __ldg(d.inv_zeta + v);
                const float kf = floorf(fmaf(T0, zeta[q], d.zfrac));
                zbnd[q] = kf + (inv_sz[q] >= 0.f ? 1.f : 0.f);
                krow[q] = (int)kf + d.koff;
            }
        }
        const int pstride = SB * BJ;                                   // floats per z plane of a brick
        for (int b = 0; b < nblk; ++b) {
            const int st = b % kStages;
            if (b > 0) {
                __syncthreads();                                       // every warp is done with the stage of block b-1
                if (wid == 0 && b - 1 + kStages < nblk) issue(b - 1 + kStages);
            }
            mbar_wait(full + st, (uint32_t)(b / kStages) & 1u);
            const int cj = meta[2 * st], ck = meta[2 * st + 1];
            const float *brick = reinterpret_cast<const float *>(smem + st * brick_bytes);
            const int i0 = lo_c + b * SB, i1 = min(i0 + SB, hi_c);
            int rowoff[V];
#pragma unroll
            for (int q = 0; q < V; ++q) rowoff[q] = (min(max(krow[q], -kPadK), d.nz + kPadK - 1) + kPadK - ck) * pstride;
            const float *base = brick + (kPadLo - cj);
            for (int i = i0; i < i1; ++i) {
                const float ef = (float)(i - cg.ioff);
                const float T = fmaf(ef, r.dt, r.tc);
                float a_, fl;
                minor_split(ef, r, dirpos, a_, fl);
                const int ja = (int)fl + cg.joff;
                const int jlo = min(max(ja - dneg, -2), cg.nmin);
                const float oma = 1.f - a_;
                const float wlo = dneg ? oma : a_;
                const float whi = dneg ? a_ : oma;
                const int off_i = (i - i0) * BJ + jlo;
                float bb[V];
#pragma unroll
                for (int q = 0; q < V; ++q) {
                    const float Za = fmaf(T, zeta[q], d.zfrac);
                    bb[q] = __saturatef((zbnd[q] - Za) * inv_sz[q]);
                    const float *p = base + (rowoff[q] + off_i);
                    acc[q] = fmaf(wlo, p[0], acc[q]);
                    acc[q] = fmaf(whi, p[1], acc[q]);
                }
#pragma unroll
                for (int q = 0; q < V; ++q) {
                    if (bb[q] < 1.f) {
                        const bool upz = inv_sz[q] >= 0.f;
                        krow[q] += upz ? 1 : -1;
                        const int rowoff1 = (min(max(krow[q], -kPadK), d.nz + kPadK - 1) + kPadK - ck) * pstride;
                        const float *p = base + (rowoff[q] + off_i), *p1 = base + (rowoff1 + off_i);
                        const float c_r0 = a_ - fminf(a_, bb[q]), c_r1 = 1.f - fmaxf(a_, bb[q]);
                        const float c_lo = dneg ? c_r1 : c_r0, c_hi = dneg ? c_r0 : c_r1;
                        acc[q] = fmaf(c_lo, p1[0] - p[0], acc[q]);
                        acc[q] = fmaf(c_hi, p1[1] - p[1], acc[q]);
                        zbnd[q] += upz ? 1.f : -1.f;
                        rowoff[q] = rowoff1;
                    }
                }
            }
        }
    } else {
        // a warp without rows (ragged last row group) still takes part in the block barriers
        for (int b = 1; b < nblk; ++b) {
            __syncthreads();
            if (wid == 0 && b - 1 + kStages < nblk) issue(b - 1 + kStages);
        }
    }
    if (!mine) return;
    const RayXY ro = load_ray(d, a, u);                                // the lane's own ray (r may be a neighbour's copy)
#pragma unroll
    for (int q = 0; q < V; ++q) {
        const int v = v0 + q;
        if (v < d.nv) {
            const float len = chord_scale(ro, __ldg(d.dz_mm + v));
            const size_t o = ((size_t)a * d.nv + v) * d.nu + u;
            float val = active ? __fmul_rn(len, acc[q]) : 0.f;           // uncontracted, as in projector.cu
            if (mode == 1) val = __fmul_rn(len, __fsub_rn(val, __ldg(Y + o)));
            else if (mode == 2) val = __fsub_rn(val, __ldg(Y + o));
            out[o] = val;
        }
    }
}
}  // namespace

// Worst-case brick spans of a class over all tiles (host, fp64, with slack): BJ minor columns, BK z planes.
static void brick_spans(const cbct_geometry *g, int c, int V, int WARPS, int *BJ, int *BK)
{
    const ClassGrid &cg = g->dev.cls[c];
    double maxsm = 0.0, maxspread = 0.0, maxT = 0.0, maxdt = 0.0;
    const double hmin = c == 0 ? g->hy : g->hx;
    for (int a = 0; a < g->na; ++a) {
        const double th = g->angles[a], co = std::cos(th), si = std::sin(th);
        const double Sx = g->sad * co, Sy = g->sad * si;
        for (int u0 = 0; u0 < g->nu; u0 += 32) {
            double lo[2] = {1e300, 1e300}, hi[2] = {-1e300, -1e300};
            bool any = false;
            for (int u = u0; u < std::min(u0 + 32, g->nu); ++u) {
                const double uc = (u - 0.5 * (g->nu - 1)) * g->du + g->off_u;
                const double Dx = -(g->sdd - g->sad) * co - uc * si, Dy = -(g->sdd - g->sad) * si + uc * co;
                const double dXv = (Dx - Sx) / g->hx, dYv = (Dy - Sy) / g->hy;
                if ((std::fabs(dXv) >= std::fabs(dYv) ? 0 : 1) != c) continue;
                any = true;
                const double Smaj = c == 0 ? Sx : Sy, Smin = c == 0 ? Sy : Sx;
                const double dmaj = c == 0 ? Dx - Sx : Dy - Sy, dmin = c == 0 ? Dy - Sy : Dx - Sx;
                const double hmaj = c == 0 ? g->hx : g->hy;
                const double sm = (dmin / hmin) / (dmaj / hmaj);
                maxsm = std::fmax(maxsm, std::fabs(sm));
                maxdt = std::fmax(maxdt, std::fabs(hmaj / dmaj));
                for (int e = 0; e < 2; ++e) {                           // minor coordinate at the two ends of the volume
                    const double maj = (e ? 0.5 : -0.5) * cg.nmaj * hmaj;
                    const double t = (maj - Smaj) / dmaj;
                    const double y = (Smin + t * dmin) / hmin;
                    lo[e] = std::fmin(lo[e], y); hi[e] = std::fmax(hi[e], y);
                    maxT = std::fmax(maxT, t);
                }
            }
            if (any) maxspread = std::fmax(maxspread, std::fmax(hi[0] - lo[0], hi[1] - lo[1]));
        }
    }
    *BJ = (((int)std::ceil(maxspread + SB * maxsm) + 5 + 3) + 3) / 4 * 4;                // + 3: the brick starts on a 16-byte boundary
    const double rows = (double)(V * WARPS - 1) * g->dv / g->hz * maxT;           // z spread of the CTA's detector rows
    const double rise = SB * maxdt * (0.5 * g->nv * g->dv + std::fabs(g->off_v)) / g->hz;
    *BK = (int)std::ceil(rows + rise) + 4;
}

cbct_status op_forward_padded_tma(cbct_geometry *g, float *d_out, const float *d_Y, int mode, cudaStream_t st, int *done)
{
    constexpr int V = 4, WARPS = CBCT_FWT_WARPS;
    *done = 0;
    for (int c = 0; c < 2; ++c) {
        if (g->n_tiles[c] == 0 || g->fw_bj[c] > 0) continue;
        brick_spans(g, c, V, WARPS, &g->fw_bj[c], &g->fw_bk[c]);
    }
    size_t smem[2] = {0, 0};
    for (int c = 0; c < 2; ++c) {
        if (g->n_tiles[c] == 0) continue;
        if (g->fw_bj[c] > 256 || g->fw_bk[c] > 256) return CBCT_OK;
        smem[c] = kStages * ((((size_t)g->fw_bk[c] * SB * g->fw_bj[c] * sizeof(float)) + 127) & ~(size_t)127) + 256;
        if (smem[c] > 100 * 1024) return CBCT_OK;                       // bricks too large to keep two CTAs per SM: use the __ldg path
    }
    *done = 1;
    ProfileScope ps(1, st);
    auto kern = forward_tma_kernel<V, WARPS>;
    static size_t smem_set = 0;
    for (int c = 0; c < 2; ++c) {
        if (g->n_tiles[c] == 0) continue;
        if (smem[c] > smem_set) {
            CBCT_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem[c]));
            smem_set = smem[c];
        }
        const ClassGrid &cg = g->dev.cls[c];
        CUtensorMap tm;
        CBCT_TRY(cbct_tensor_map_3d(&tm, g->vol_pad[c], (unsigned long long)cg.row_stride, (unsigned long long)cg.nmaj,
                                    (unsigned long long)(g->nz + 2 * kPadK), (unsigned long long)cg.row_stride * sizeof(float),
                                    (unsigned long long)cg.plane_stride * sizeof(float), (unsigned)g->fw_bj[c], SB, (unsigned)g->fw_bk[c]));
        dim3 grid(g->n_tiles[c], (g->nv + V * WARPS - 1) / (V * WARPS)), block(32, WARPS);
        kern<<<grid, block, smem[c], st>>>(g->dev, c, g->d_tiles[c], tm, g->fw_bj[c], g->fw_bk[c], d_out, d_Y, mode);
        CBCT_LAUNCH_CHECK();
    }
    return CBCT_OK;
}
