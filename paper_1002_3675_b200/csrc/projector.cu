// a1/a2: ray-driven exact-chord cone-beam projector (definition O1 in DESIGN.md).
//
// One thread marches V rays that share a detector column u (and therefore share their whole
// x-y traversal: the detector's v axis is parallel to the rotation axis, so the t-parameters of
// all x- and y-plane crossings are independent of v).  A warp is 32 adjacent u of one
// detector-row group, so in every slab its lanes read ~contiguous minor-axis addresses of the
// class' padded volume copy (class 0 reads the [k][x][y] transposed copy, class 1 the [k][y][x]
// copy).  Per slab (one voxel of the major axis) a ray touches at most two minor rows, split at
// lambda = a, and at most two z rows, split at lambda = b (lambda = position inside the slab
// in [0,1]); the four chord fractions are
//      (r0,k0) min(a,b)   (r1,k0) b - min(a,b)   (r0,k1) a - min(a,b)   (r1,k1) 1 - max(a,b)
// and the backprojector (backprojector.cu) evaluates exactly the same expressions.
#include "cbct_internal.h"
#include "ray_common.cuh"

// ------------------------------------------------------------------------------------------
// Padded copies: class 1 copy is [k+K][j][PadLo+i], class 0 copy is the transpose [k+K][i][PadLo+j].
// Pads are zeroed once at allocation and never written, which is what makes "f = 0 outside
// the volume" exact without bounds checks in the march.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) pad_copy_kernel(const float *__restrict__ vol, float *__restrict__ pad_x,
                                                       float *__restrict__ pad_y, int nx, int ny,
                                                       int rs_x, long long ps_x, int rs_y, long long ps_y)
{
    __shared__ float tile[32][33];
    const int k = blockIdx.z;
    const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
    const float *src = vol + (size_t)k * ny * nx;
    for (int r = threadIdx.y; r < 32; r += 8) {
        int j = j0 + r, i = i0 + threadIdx.x;
        float v = (j < ny && i < nx) ? __ldg(src + (size_t)j * nx + i) : 0.f;
        tile[r][threadIdx.x] = v;
        if (pad_y && j < ny && i < nx) pad_y[(size_t)(k + kPadK) * ps_y + (size_t)j * rs_y + kPadLo + i] = v;
    }
    if (!pad_x) return;
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += 8) {
        int i = i0 + r, j = j0 + threadIdx.x;
        if (i < nx && j < ny) pad_x[(size_t)(k + kPadK) * ps_x + (size_t)i * rs_x + kPadLo + j] = tile[threadIdx.x][r];
    }
}

cbct_status op_pad_copies(cbct_geometry *g, const float *d_vol, cudaStream_t st)
{
    for (int c = 0; c < 2; ++c)
        if (g->n_tiles[c] > 0) CBCT_TRY(ensure_zeroed(g, &g->vol_pad[c], pad_elems(g, c), st));
    float *px = g->n_tiles[0] > 0 ? g->vol_pad[0] : nullptr;
    float *py = g->n_tiles[1] > 0 ? g->vol_pad[1] : nullptr;
    if (!px && !py) return CBCT_OK;
    const DevGeom &d = g->dev;
    ProfileScope ps(0, st);
    dim3 grid((g->nx + 31) / 32, (g->ny + 31) / 32, g->nz), block(32, 8);
    pad_copy_kernel<<<grid, block, 0, st>>>(d_vol, px, py, g->nx, g->ny, d.cls[0].row_stride, d.cls[0].plane_stride,
                                            d.cls[1].row_stride, d.cls[1].plane_stride);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

// ------------------------------------------------------------------------------------------
// Forward march.
// ------------------------------------------------------------------------------------------
// MIRROR: the scan is its own mirror image about the central plane z = 0 (nz even, nv even, detector centred in v).  Ray
// (u, nv-1-v) is then the mirror image of ray (u, v): same x-y traversal, same crossing positions b, z rows nz-1-k.  A thread
// marches V rays of the UPPER half of the detector (v >= nv/2) together with their V mirror images, so the z arithmetic of a
// slab (entry position, b, the row advance and its clamps) is done once for two rays.
// TWIN (with MIRROR): the angle list is closed under theta -> theta + 180 degrees (angle a + na/2 = angle a + pi).  Turning
// the whole scan by 180 degrees about the rotation axis maps ray (a, u, v) onto ray (a + na/2, u, v) and voxel (i, j, k) onto
// (nx-1-i, ny-1-j, k): the twin ray has the same slabs, splits a and b and chord fractions, met in the point-reflected
// voxels, i.e. at padded offset (nmaj-1) row_stride + nmin-2 minus the ray's own, with the two minor rows swapped.  A thread
// then marches V rays, their z-mirror images and the twins of both: 4 V rays from one evaluation of all the ray arithmetic.
template <int V, int WARPS, bool MIRROR, bool TWIN = false>
__global__ void __launch_bounds__(32 * WARPS)
forward_kernel(const DevGeom d, const int cls, const int2 *__restrict__ tiles, const float *__restrict__ vol,
               float *__restrict__ out, const float *__restrict__ Y, const int mode)
{
    const ClassGrid cg = d.cls[cls];
    const int lane = threadIdx.x;
    const int2 tile = tiles[blockIdx.x];
    const int a = tile.x, u = tile.y + lane;
    const int vbase = MIRROR ? d.nv / 2 : 0;                  // first detector row this launch marches directly
    const int v0 = vbase + (blockIdx.y * WARPS + threadIdx.y) * V;
    if (v0 >= d.nv) return;                                   // warp-uniform

    RayXY r = load_ray(d, a, min(u, d.nu - 1));
    int ilo = ray_ilo(r.range), ihi = ray_ihi(r.range);
    const bool mine = (u < d.nu) && (ray_cls(r.range) == cls);
    bool active = mine && ihi > ilo;

    // z clip: the ray of this thread closest to the central plane stays inside longest
    {
        const float za = __ldg(d.zeta + v0), zb = __ldg(d.zeta + min(v0 + V - 1, d.nv - 1));
        float tmax = 3.0e38f;
        if (za > 0.f && zb > 0.f) tmax = ((float)(d.nz - d.koff) + 1.f - d.zfrac) / fminf(za, zb);
        else if (za < 0.f && zb < 0.f) tmax = (-(float)d.koff - 1.f - d.zfrac) / fmaxf(za, zb);
        if (tmax < 2.f) {                                     // t <= tmax, t = tc + (i - ioff) dt
            float e = (tmax - r.tc) * r.inv_dt;
            if (r.dt > 0.f) ihi = min(ihi, cg.ioff + (int)floorf(e) + 2);
            else            ilo = max(ilo, cg.ioff + (int)ceilf(e) - 2);
        }
        active = active && ihi > ilo;
    }
    if (!active) { r.mc = -30000.f; r.sm = 0.f; r.inv_sm = 1e30f; }   // clamps to the zero pad
    const int lo_w = __reduce_min_sync(0xffffffffu, active ? ilo : 0x7fffffff);
    const int hi_w = __reduce_max_sync(0xffffffffu, active ? ihi : -1);

    static_assert(!TWIN || MIRROR, "the twin march is built on the mirrored one");
    float acc[V], accM[MIRROR ? V : 1], accT[TWIN ? V : 1], accMT[TWIN ? V : 1];
#pragma unroll
    for (int q = 0; q < V; ++q) acc[q] = 0.f;
    if constexpr (MIRROR) {
#pragma unroll
        for (int q = 0; q < V; ++q) accM[q] = 0.f;
    }
    if constexpr (TWIN) {
#pragma unroll
        for (int q = 0; q < V; ++q) accT[q] = accMT[q] = 0.f;
    }

    if (lo_w < hi_w) {
        const float dirpos = r.sm >= 0.f ? 1.f : 0.f;
        const int dneg = r.sm >= 0.f ? 0 : 1;
        float zeta[V], inv_sz[V], zbnd[V];
        int krow[V], rowoff[V];                                          // element offsets fit 32 bits (checked at geometry creation)
        const int pstride = (int)cg.plane_stride;
        // MIRROR: padded row of the mirror image = (nz - 1 + 2 kPadK) - padded row (the clamp range is symmetric)
        const int row_top = (d.nz - 1 + 2 * kPadK) * pstride;
        // TWIN: offset of the point-reflected row pair inside a padded plane = off_top - (the ray's own offset)
        const int off_top = (cg.nmaj - 1) * cg.row_stride + cg.nmin - 2;
        const float e0 = (float)(lo_w - cg.ioff);
        const float T0 = fmaf(e0, r.dt, r.tc);
#pragma unroll
        for (int q = 0; q < V; ++q) {
            const int v = min(v0 + q, d.nv - 1);
            zeta[q] = __ldg(d.zeta + v);
            inv_sz[q] = r.inv_dt * __ldg(d.inv_zeta + v);      // sign = direction of the ray in z
            const float Za = fmaf(T0, zeta[q], d.zfrac);
            const float kf = floorf(Za);
            zbnd[q] = kf + (inv_sz[q] >= 0.f ? 1.f : 0.f);
            krow[q] = (int)kf + d.koff;
            rowoff[q] = (min(max(krow[q], -kPadK), d.nz + kPadK - 1) + kPadK) * pstride;
        }
        const float *base = vol + kPadLo;
        for (int i = lo_w; i < hi_w; ++i) {
            const float ef = (float)(i - cg.ioff);
            const float T = fmaf(ef, r.dt, r.tc);
            float a_, fl;
            minor_split(ef, r, dirpos, a_, fl);
            const int ja = (int)fl + cg.joff;
            const int jlo = min(max(ja - dneg, -2), cg.nmin);
            const float oma = 1.f - a_;
            const float wlo = dneg ? oma : a_;                 // fraction [0,a] belongs to row ja, [a,1] to ja+dir
            const float whi = dneg ? a_ : oma;
            const int off_i = i * cg.row_stride + jlo;
            // Pass 1, branch-free: every ray as if it stayed in its entry z row for the whole slab
            // (all 2V loads are independent and in flight together).
            float b[V];
#pragma unroll
            for (int q = 0; q < V; ++q) {
                const float Za = fmaf(T, zeta[q], d.zfrac);
                b[q] = __saturatef((zbnd[q] - Za) * inv_sz[q]);
                const float *p = base + (rowoff[q] + off_i);
                acc[q] = fmaf(wlo, __ldg(p), acc[q]);
                acc[q] = fmaf(whi, __ldg(p + 1), acc[q]);
                if constexpr (MIRROR) {
                    const float *pm = base + ((row_top - rowoff[q]) + off_i);
                    accM[q] = fmaf(wlo, __ldg(pm), accM[q]);
                    accM[q] = fmaf(whi, __ldg(pm + 1), accM[q]);
                }
                if constexpr (TWIN) {                          // reflected rows: [0] is the twin of p[1], [1] the twin of p[0]
                    const float *pt = base + (rowoff[q] + (off_top - off_i));
                    accT[q] = fmaf(whi, __ldg(pt), accT[q]);
                    accT[q] = fmaf(wlo, __ldg(pt + 1), accT[q]);
                    const float *pmt = base + ((row_top - rowoff[q]) + (off_top - off_i));
                    accMT[q] = fmaf(whi, __ldg(pmt), accMT[q]);
                    accMT[q] = fmaf(wlo, __ldg(pmt + 1), accMT[q]);
                }
            }
            // Pass 2: a ray that crosses a z plane inside the slab (b < 1) moves its exit-row fractions
            // a - min(a,b) (row ja) and 1 - max(a,b) (row ja+dir) to the next z row, and continues there.
#pragma unroll
            for (int q = 0; q < V; ++q) {
                if (b[q] < 1.f) {
                    const bool upz = inv_sz[q] >= 0.f;
                    const float zs = upz ? 1.f : -1.f;
                    krow[q] += upz ? 1 : -1;                   // true z row (rows outside the pad read the outermost zero plane)
                    const int rowoff1 = (min(max(krow[q], -kPadK), d.nz + kPadK - 1) + kPadK) * pstride;
                    const float *p = base + (rowoff[q] + off_i), *p1 = base + (rowoff1 + off_i);
                    const float c_r0 = a_ - fminf(a_, b[q]), c_r1 = 1.f - fmaxf(a_, b[q]);
                    const float c_lo = dneg ? c_r1 : c_r0, c_hi = dneg ? c_r0 : c_r1;
                    acc[q] = fmaf(c_lo, __ldg(p1) - __ldg(p), acc[q]);
                    acc[q] = fmaf(c_hi, __ldg(p1 + 1) - __ldg(p + 1), acc[q]);
                    if constexpr (MIRROR) {
                        const float *pm = base + ((row_top - rowoff[q]) + off_i), *pm1 = base + ((row_top - rowoff1) + off_i);
                        accM[q] = fmaf(c_lo, __ldg(pm1) - __ldg(pm), accM[q]);
                        accM[q] = fmaf(c_hi, __ldg(pm1 + 1) - __ldg(pm + 1), accM[q]);
                    }
                    if constexpr (TWIN) {
                        const int offt = off_top - off_i;
                        const float *pt = base + (rowoff[q] + offt), *pt1 = base + (rowoff1 + offt);
                        accT[q] = fmaf(c_hi, __ldg(pt1) - __ldg(pt), accT[q]);
                        accT[q] = fmaf(c_lo, __ldg(pt1 + 1) - __ldg(pt + 1), accT[q]);
                        const float *pmt = base + ((row_top - rowoff[q]) + offt), *pmt1 = base + ((row_top - rowoff1) + offt);
                        accMT[q] = fmaf(c_hi, __ldg(pmt1) - __ldg(pmt), accMT[q]);
                        accMT[q] = fmaf(c_lo, __ldg(pmt1 + 1) - __ldg(pmt + 1), accMT[q]);
                    }
                    zbnd[q] += zs;
                    rowoff[q] = rowoff1;
                }
            }
        }
    }
    if (!mine) return;
#pragma unroll
    for (int q = 0; q < V; ++q) {
        const int v = v0 + q;
        if (v < d.nv) {
            const float len = chord_scale(r, __ldg(d.dz_mm + v));
#pragma unroll
            for (int m = 0; m < (TWIN ? 4 : MIRROR ? 2 : 1); ++m) {          // the ray, its z-mirror image, the twins of both
                const int aa = (m & 2) ? a + d.na / 2 : a, vv = (m & 1) ? d.nv - 1 - v : v;
                const size_t o = ((size_t)aa * d.nv + vv) * d.nu + u;
                const float ac = m == 0 ? acc[q] : m == 1 ? accM[MIRROR ? q : 0] : m == 2 ? accT[TWIN ? q : 0] : accMT[TWIN ? q : 0];
                // uncontracted (no FMA across the subtraction), so that op_residual applied to a stored mode-0 value is bit-identical
                float val = __fmul_rn(len, ac);
                if (mode == 1) val = __fmul_rn(len, __fsub_rn(val, __ldg(Y + o)));
                else if (mode == 2) val = __fsub_rn(val, __ldg(Y + o));
                out[o] = val;
            }
        }
    }
}

bool march_is_mirrored(const cbct_geometry *g);

// a2 alone: turns a plain projection q = P f (mode 0 of the march) into the residual the march's mode 1 / mode 2 would have
// stored, with the very same operations (val = len * acc was stored; here len * (val - Y) or val - Y), so the result is bit
// for bit the fused one.  Used by the host-buffer path, whose first projection starts before Y has arrived on the device.
__global__ void __launch_bounds__(256) residual_kernel(const DevGeom d, float *__restrict__ q, const float *__restrict__ Y, const int mode,
                                                       const int twin)
{
    const int u = blockIdx.x * blockDim.x + threadIdx.x, v = blockIdx.y, a = blockIdx.z;
    if (u >= d.nu) return;
    const size_t o = ((size_t)a * d.nv + v) * d.nu + u;
    float val = q[o];
    // (the twin march takes the chord length of a second-half ray from its first-half twin's table entry; so does this)
    const int at = twin && a >= d.na / 2 ? a - d.na / 2 : a;
    if (mode == 1) val = __fmul_rn(chord_scale(load_ray(d, at, u), __ldg(d.dz_mm + v)), __fsub_rn(val, __ldg(Y + o)));
    else val = __fsub_rn(val, __ldg(Y + o));
    q[o] = val;
}

cbct_status op_residual(cbct_geometry *g, float *d_q, const float *d_Y, int mode, cudaStream_t st)
{
    ProfileScope ps(1, st);
    dim3 grid((g->nu + 255) / 256, g->nv, g->na);
    residual_kernel<<<grid, 256, 0, st>>>(g->dev, d_q, d_Y, mode, g->last_march_twin);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}

// the scan is its own mirror image about the central plane: even slice and detector-row counts, detector centred in v
bool march_is_mirrored(const cbct_geometry *g)
{
    return g->use_mirror && g->nz % 2 == 0 && g->nv % 2 == 0 && g->off_v == 0.0;
}

cbct_status op_forward_padded(cbct_geometry *g, float *d_out, const float *d_Y, int mode, cudaStream_t st)
{
    // rays per thread and warps per CTA: compile-time tuning knobs (measured best of a sweep on B200: 4 x 4)
#ifndef CBCT_FW_V
#define CBCT_FW_V 4
#define CBCT_FW_WARPS 4
#endif
#ifndef CBCT_FW_VM
#define CBCT_FW_VM 3
#endif
#ifndef CBCT_FW_VT
#define CBCT_FW_VT 2
#endif
    constexpr int V = CBCT_FW_V, WARPS = CBCT_FW_WARPS;
    g->last_march_twin = 0;
    if (g->fw_staged) {
        int done = 0;
        CBCT_TRY(op_forward_padded_tma(g, d_out, d_Y, mode, st, &done));
        if (done) return CBCT_OK;
    }
    ProfileScope ps(1, st);
    // every ray belongs to a tile of its class (geometry.cu), so every output element is written: 0 / -Y / -l Y for a
    // ray that misses the volume
    const bool mirror = march_is_mirrored(g);
    g->last_march_twin = mirror && g->twin_ok;           // op_residual follows the march that made the projection
    for (int c = 0; c < 2; ++c) {
        if (g->n_tiles[c] == 0) continue;
        if (mirror && g->twin_ok) {
            constexpr int VT = CBCT_FW_VT;                    // ray quadruples per thread; only the tiles of the first half turn
            dim3 grid(g->n_tiles_half[c], (g->nv / 2 + VT * WARPS - 1) / (VT * WARPS)), block(32, WARPS);
            if (grid.x > 0)
                forward_kernel<VT, WARPS, true, true><<<grid, block, 0, st>>>(g->dev, c, g->d_tiles[c], g->vol_pad[c], d_out, d_Y, mode);
        } else if (mirror) {
            constexpr int VM = CBCT_FW_VM;                    // ray pairs per thread
            dim3 grid(g->n_tiles[c], (g->nv / 2 + VM * WARPS - 1) / (VM * WARPS)), block(32, WARPS);
            forward_kernel<VM, WARPS, true><<<grid, block, 0, st>>>(g->dev, c, g->d_tiles[c], g->vol_pad[c], d_out, d_Y, mode);
        } else {
            dim3 grid(g->n_tiles[c], (g->nv + V * WARPS - 1) / (V * WARPS)), block(32, WARPS);
            forward_kernel<V, WARPS, false><<<grid, block, 0, st>>>(g->dev, c, g->d_tiles[c], g->vol_pad[c], d_out, d_Y, mode);
        }
        CBCT_LAUNCH_CHECK();
    }
    return CBCT_OK;
}
