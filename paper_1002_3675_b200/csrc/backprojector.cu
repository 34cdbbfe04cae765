// a3: exact-adjoint backprojector G = P^T y as a race-free gather (O2 in DESIGN.md).
//
// The paper rejects the transpose form because a ray-driven scatter races and replaces it
// by the voxel-driven eq. 2.  Here the transpose itself is evaluated voxel-driven: a thread owns a
// column of KC voxels (fixed major index i = slab, fixed minor index j, KC consecutive k) and
// gathers, for every angle, from the few rays that can touch it:
//   * in-plane: the rays u whose slab-i traversal touches minor row j.  Candidates come from
//     projecting the column's x-y square onto the detector; each is then tested with the
//     projector's own minor_split(), giving its lambda-interval [l0,l1] inside row j;
//   * axially: for row k the rays v whose z-interval meets [l0,l1]; with p0,p1 the (saturated)
//     lambdas at which ray v meets planes k and k+1, the chord fraction is
//         w = max(0, min(l1, max(p0,p1)) - max(l0, min(p0,p1)))
//     which reproduces the projector's four fractions term by term (see ray_common.cuh).
// The projections handed in are pre-multiplied by the slab chord length l(u,v).
// One launch per ray class; class 0 accumulates into a [k][x][y] array, class 1 into [k][y][x],
// so lanes (adjacent minor index) write contiguously; op_combine() adds the two.
#include "cbct_internal.h"
#include "ray_common.cuh"

template <int KC, int BI>
__global__ void __launch_bounds__(32 * BI)
backproject_kernel(const DevGeom d, const int cls, const unsigned char *__restrict__ angle_has,
                   const float *__restrict__ rs, float *__restrict__ G)
{
    const ClassGrid cg = d.cls[cls];
    const int j = blockIdx.x * 32 + threadIdx.x;      // minor index
    const int i = blockIdx.y * BI + threadIdx.y;      // major index = slab
    const int k0 = blockIdx.z * KC;
    if (i >= cg.nmaj) return;                          // warp-uniform
    const bool valid = j < cg.nmin;

    float acc[KC];
#pragma unroll
    for (int q = 0; q < KC; ++q) acc[q] = 0.f;

    // the column's x-y square in mm (candidate search only; the accept test is exact)
    const float maj0 = ((float)i - 0.5f * (float)cg.nmaj) * cg.hmaj, maj1 = maj0 + cg.hmaj;
    const float mn0 = ((float)min(j, cg.nmin - 1) - 0.5f * (float)cg.nmin) * cg.hmin, mn1 = mn0 + cg.hmin;
    const float x0 = cls == 0 ? maj0 : mn0, x1 = cls == 0 ? maj1 : mn1;
    const float y0 = cls == 0 ? mn0 : maj0, y1 = cls == 0 ? mn1 : maj1;
    const float ef = (float)(i - cg.ioff);
    const float cu = 0.5f * (float)(d.nu - 1), cv = 0.5f * (float)(d.nv - 1);
    const float sdd_du = d.sdd / d.du;
    const float dzeta = d.dv / d.hz;

    for (int a = 0; a < d.na; ++a) {
        if (!angle_has[a]) continue;                   // uniform
        const float2 cs = __ldg(d.cs + a);
        float umin = 3e38f, umax = -3e38f;
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const float x = (m & 1) ? x1 : x0, y = (m & 2) ? y1 : y0;
            const float num = fmaf(-x, cs.y, y * cs.x);
            const float den = d.sad - fmaf(x, cs.x, y * cs.y);
            const float uu = fmaf(sdd_du, __fdividef(num, den), cu);
            umin = fminf(umin, uu);
            umax = fmaxf(umax, uu);
        }
        const int uA = max(0, (int)floorf(umin - 0.02f));
        const int uB = valid ? min(d.nu - 1, (int)ceilf(umax + 0.02f)) : -1;
        for (int u = uA; u <= uB; ++u) {
            const RayXY r = load_ray(d, a, u);
            if (ray_cls(r.range) != cls || i < ray_ilo(r.range) || i >= ray_ihi(r.range)) continue;
            const float dirpos = r.sm >= 0.f ? 1.f : 0.f;
            float a_, fl;
            minor_split(ef, r, dirpos, a_, fl);
            const int ja = (int)fl + cg.joff;
            float l0, l1;
            if (ja == j) { l0 = 0.f; l1 = a_; }
            else if (ja + (r.sm >= 0.f ? 1 : -1) == j) { l0 = a_; l1 = 1.f; }
            else continue;
            if (!(l1 > l0)) continue;

            const float T = fmaf(ef, r.dt, r.tc);
            const float invB = __fdividef(1.f, T * dzeta);            // d v / d Z at this slab
            const float absdt_T = fabsf(r.dt) / T;
            const float *rsa = rs + (size_t)a * d.nv * d.nu + u;
#pragma unroll
            for (int q = 0; q < KC; ++q) {
                const int k = k0 + q;
                if (k >= d.nz) break;
                const float kf = (float)(k - d.koff);
                const float sb = absdt_T * (fabsf(kf - d.zfrac) + 2.f) + 1e-3f;   // bound on |sz| near this row (+ slack)
                const float zlo = kf - sb - d.zfrac, zhi = kf + 1.f + sb - d.zfrac;
                const int vs = max(0, (int)ceilf(fmaf(zlo, invB, cv) - 1e-3f));
                const int ve = min(d.nv - 1, (int)floorf(fmaf(zhi, invB, cv) + 1e-3f));
                float s = 0.f;
                for (int v = vs; v <= ve; ++v) {
                    const float Za = z_entry(T, __ldg(d.zeta + v), d.zfrac);
                    const float inv_sz = r.inv_dt * __ldg(d.inv_zeta + v);
                    const float p0 = __saturatef((kf - Za) * inv_sz);
                    const float p1 = __saturatef(((kf + 1.f) - Za) * inv_sz);
                    const float w = fmaxf(0.f, fminf(l1, fmaxf(p0, p1)) - fmaxf(l0, fminf(p0, p1)));
                    s = fmaf(w, __ldg(rsa + (size_t)v * d.nu), s);
                }
                acc[q] += s;
            }
        }
    }
    if (!valid) return;
#pragma unroll
    for (int q = 0; q < KC; ++q) {
        const int k = k0 + q;
        if (k < d.nz) G[((size_t)k * cg.nmaj + i) * cg.nmin + j] = acc[q];
    }
}

cbct_status op_backproject_gather(cbct_geometry *g, const float *d_scaled, cudaStream_t st)
{
    constexpr int KC = 16, BI = 4;
    ProfileScope ps(3, st);
    for (int c = 0; c < 2; ++c) {
        if (g->n_tiles[c] == 0) continue;
        CBCT_TRY(ensure(g, &g->G_cls[c], g->n_vox()));
        const ClassGrid &cg = g->dev.cls[c];
        dim3 grid((cg.nmin + 31) / 32, (cg.nmaj + BI - 1) / BI, (g->nz + KC - 1) / KC), block(32, BI);
        backproject_kernel<KC, BI><<<grid, block, 0, st>>>(g->dev, c, g->d_angle_has[c], d_scaled, g->G_cls[c]);
        CBCT_LAUNCH_CHECK();
    }
    return CBCT_OK;
}

// out = G1 + G0^T  or  out = f - c (G1 + G0^T) [clamped]  — fuses a4 (and a6 when n_inner = 0) into the
// transpose-add that the two-class gather needs anyway.
__global__ void __launch_bounds__(256) combine_kernel(const float *__restrict__ G0, const float *__restrict__ G1,
                                                      const float *__restrict__ f, float c, int clamp,
                                                      float *__restrict__ out, int nx, int ny)
{
    __shared__ float tile[32][33];
    const int k = blockIdx.z;
    const int i0 = blockIdx.x * 32, j0 = blockIdx.y * 32;
    const size_t plane = (size_t)k * nx * ny;
    if (G0) {
        // G0 is [k][x][y]: read rows of constant x
        for (int r = threadIdx.y; r < 32; r += 8) {
            int i = i0 + r, j = j0 + threadIdx.x;
            tile[r][threadIdx.x] = (i < nx && j < ny) ? __ldg(G0 + plane + (size_t)i * ny + j) : 0.f;
        }
        __syncthreads();
    }
    for (int r = threadIdx.y; r < 32; r += 8) {
        int j = j0 + r, i = i0 + threadIdx.x;
        if (j < ny && i < nx) {
            const size_t o = plane + (size_t)j * nx + i;
            float gsum = G0 ? tile[threadIdx.x][r] : 0.f;
            if (G1) gsum += __ldg(G1 + o);
            float val = gsum;
            if (f) {
                val = fmaf(-c, gsum, __ldg(f + o));
                if (clamp) val = fmaxf(val, 0.f);
            }
            out[o] = val;
        }
    }
}

cbct_status op_combine(cbct_geometry *g, const float *f, float c, int clamp, float *out, cudaStream_t st)
{
    ProfileScope ps(4, st);
    const float *G0 = g->n_tiles[0] > 0 ? g->G_cls[0] : nullptr;
    const float *G1 = g->n_tiles[1] > 0 ? g->G_cls[1] : nullptr;
    dim3 grid((g->nx + 31) / 32, (g->ny + 31) / 32, g->nz), block(32, 8);
    combine_kernel<<<grid, block, 0, st>>>(G0, G1, f, c, clamp, out, g->nx, g->ny);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}
