// NEXT-1: the paper's own voxel-driven backprojector, eq. 2, without its prefactor 2/(N_theta A):
//   (B r)(x) = sum_theta L^3(u*,v*) / (L0 l^2(x)) r^theta(u*,v*),
// x the voxel centre, (u*,v*) where the line source -> x meets the imager, L0 = SDD, l = |x - S|,
// L = |(u*,v*) - S|; r bilinear between pixel centres, 0 outside the detector (reading Q4 of DESIGN.md).
// "Each thread on GPU can independently evaluate the functional variation at a (x,y,z) coordinate":
// one thread per z column of KC voxels, lanes along x.  By similar triangles L = l SDD/t with t the depth
// of x along the central ray, so the weight is (SDD/t)^2 (l/t); t, the lateral offset and u* are shared by
// the column, v* and l change with z.  Not the transpose of cbct_forward (see cbct_backproject for that).
#include "cbct_internal.h"

template <int KC>
__global__ void __launch_bounds__(128)
backproject_eq2_kernel(const DevGeom d, const float *__restrict__ proj, const float *__restrict__ f, const float c,
                       const int clamp, float *__restrict__ out)
{
    const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 4 + threadIdx.y, k0 = blockIdx.z * KC;
    if (i >= d.nx || j >= d.ny) return;
    const float x = ((float)i - 0.5f * (float)(d.nx - 1)) * d.hx, y = ((float)j - 0.5f * (float)(d.ny - 1)) * d.hy;
    const float cu = d.cu, cv = d.cv;
    const float z0 = ((float)k0 - 0.5f * (float)(d.nz - 1)) * d.hz;
    const float inv_du = 1.f / d.du, inv_dv = 1.f / d.dv;
    float acc[KC];
#pragma unroll
    for (int q = 0; q < KC; ++q) acc[q] = 0.f;

    for (int a = 0; a < d.na; ++a) {
        const float2 cs = __ldg(d.cs + a);
        const float t = d.sad - fmaf(x, cs.x, y * cs.y);          // depth along the central ray (> 0: checked at creation)
        const float lat = fmaf(-x, cs.y, y * cs.x);               // offset along the detector's u axis
        const float inv_t = 1.f / t, M = d.sdd * inv_t;
        const float pu = fmaf(M * lat, inv_du, cu);
        const float fu = floorf(pu), au = pu - fu;
        const int iu = (int)fu;
        const bool u0ok = (unsigned)iu < (unsigned)d.nu, u1ok = (unsigned)(iu + 1) < (unsigned)d.nu;
        if (!u0ok && !u1ok) continue;
        const float w0 = u0ok ? 1.f - au : 0.f, w1 = u1ok ? au : 0.f;
        const float *img = proj + (size_t)a * d.nv * d.nu;                             // one image: 32-bit offsets below
        const int c0 = min(max(iu, 0), d.nu - 1), c1 = min(max(iu + 1, 0), d.nu - 1);   // clamped columns (weight 0 if outside)
        const float M2 = M * M * inv_t, r2 = fmaf(t, t, lat * lat);
        const float Mv = M * inv_dv;
#pragma unroll
        for (int q = 0; q < KC; ++q) {
            const float z = fmaf((float)q, d.hz, z0);
            const float pv = fmaf(Mv, z, cv);
            const float fv = floorf(pv), av = pv - fv;
            const int iv = (int)fv;
            const bool v0ok = (unsigned)iv < (unsigned)d.nv, v1ok = (unsigned)(iv + 1) < (unsigned)d.nv;
            const int row0 = min(max(iv, 0), d.nv - 1) * d.nu, row1 = min(max(iv + 1, 0), d.nv - 1) * d.nu;
            const float b0 = fmaf(w0, __ldg(img + (row0 + c0)), w1 * __ldg(img + (row0 + c1)));
            const float b1 = fmaf(w0, __ldg(img + (row1 + c0)), w1 * __ldg(img + (row1 + c1)));
            const float val = fmaf(v0ok ? 1.f - av : 0.f, b0, (v1ok ? av : 0.f) * b1);
            const float l2 = fmaf(z, z, r2);                              // l^2 > 0
            acc[q] = fmaf(M2 * (l2 * rsqrtf(l2)), val, acc[q]);           // (SDD/t)^2 (l/t); rsqrt: 2 ulp, far below the tolerance
        }
    }
#pragma unroll
    for (int q = 0; q < KC; ++q) {
        const int k = k0 + q;
        if (k >= d.nz) break;
        const size_t o = ((size_t)k * d.ny + j) * d.nx + i;
        float v = acc[q];
        if (f) {
            v = fmaf(-c, v, __ldg(f + o));
            if (clamp) v = fmaxf(v, 0.f);
        }
        out[o] = v;
    }
}

// out = B r  (f == nullptr)   or   out = f - c (B r), optionally clamped at 0 (the gradient step a4 fused)
cbct_status op_backproject_eq2(cbct_geometry *g, const float *d_proj, const float *f, float c, int clamp, float *out,
                               cudaStream_t st)
{
    constexpr int KC = 8;
    ProfileScope ps(3, st);
    dim3 grid((g->nx + 31) / 32, (g->ny + 3) / 4, (g->nz + KC - 1) / KC), block(32, 4);
    backproject_eq2_kernel<KC><<<grid, block, 0, st>>>(g->dev, d_proj, f, c, clamp, out);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}
