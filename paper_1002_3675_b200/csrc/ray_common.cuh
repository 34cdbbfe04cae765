// Arithmetic shared by the projector and its exact-adjoint gather.  Both kernels MUST evaluate
// the chord fractions with these very expressions: that is what makes the gather the transpose
// of the march entry by entry (up to the order of the fp32 sums) and not merely "an adjoint-like"
// operator.
#pragma once
#include "cbct_internal.h"

__device__ __forceinline__ RayXY load_ray(const DevGeom &d, int a, int u)
{
    const float4 *p = reinterpret_cast<const float4 *>(d.rays + (size_t)a * d.nu + u);
    const float4 x = __ldg(p), y = __ldg(p + 1);
    RayXY r;
    r.mc = x.x; r.sm = x.y; r.inv_sm = x.z; r.tc = x.w;
    r.dt = y.x; r.inv_dt = y.y; r.lxy2 = y.z; r.range = __float_as_int(y.w);
    return r;
}

// Slab whose entry plane is the major plane with centred index ef = i - ioff.  The ray enters it
// in minor row floor(Ya) =: fl (relative to joff) and stays there for lambda in [0,a]; for
// lambda in [a,1] it is in row fl + dir (dir = sign of sm).  a = 1 when it does not cross.
__device__ __forceinline__ void minor_split(float ef, const RayXY &r, float dirpos, float &a, float &fl)
{
    const float Ya = fmaf(ef, r.sm, r.mc);
    fl = floorf(Ya);
    a = __saturatef(((fl + dirpos) - Ya) * r.inv_sm);
}

// z coordinate (voxel units, minus koff) of ray (u,v) at the slab's entry plane.
__device__ __forceinline__ float z_entry(float T, float zeta, float zfrac) { return fmaf(T, zeta, zfrac); }

// Chord length (mm) of one full slab for ray (u,v): sqrt(hmaj^2 + (sm hmin)^2 + (sz hz)^2), sz hz = dt Dz.
__device__ __forceinline__ float chord_scale(const RayXY &r, float dz_mm)
{
    const float s = r.dt * dz_mm;
    return sqrtf(fmaf(s, s, r.lxy2));
}
